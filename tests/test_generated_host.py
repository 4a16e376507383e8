"""The emitted matrix elements, compiled for the host with g++ (no GPU), against the oracle.

The device library and the generated code are plain templated C++ on the host (HG_HD = inline, HostStage instead of
shared memory), so the generator's output -- diagram list, signs, colour flows, helicity-zero analysis, closing by
current, staging slots -- is checked here on CPU; the `-m gpu` tests then check the kernels that wrap it.
"""
import os
import subprocess

import numpy as np
import pytest

from oracle import phase_space as ops
from oracle import processes as opr
from oracle import sm as osm

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, 'tests', 'hostcheck.cpp')
N = {1: 64, 2: 48, 3: 24, 4: 4, 5: 6, 6: 64, 7: 48, 8: 48, 9: 3, 10: 48, 11: 48}


@pytest.fixture(scope='module')
def exe(tmp_path_factory):
    out = str(tmp_path_factory.mktemp('hostcheck') / 'hostcheck')
    subprocess.check_call(['g++', '-O1', '-std=c++17', SRC, '-o', out, '-lm'])
    return out


@pytest.mark.parametrize('cfg', [1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11])
def test_generated_code_matches_oracle(exe, cfg):
    par = osm.default_params()
    p, _ = ops.generate(cfg, 7, 0, N[cfg], opr.SQRT_S[cfg], par)
    ref = opr.me2(opr.config(cfg), p, par)
    text = '\n'.join('%d ' % cfg + ' '.join('%.17g' % x for x in ev.reshape(-1)) for ev in p) + '\n'
    out = subprocess.run([exe], input=text, capture_output=True, text=True, check=True).stdout.split()
    got = np.array([float(x) for x in out])
    assert got.shape == ref.shape
    rel = np.abs(got - ref) / ref
    assert rel.max() <= 1e-11, (cfg, rel.max())
