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
    subprocess.check_call(['g++', '-O1', '-std=c++17', '-pthread', SRC, '-o', out, '-lm'])
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


@pytest.mark.parametrize('cfg', [4, 5, 9])
def test_pair_and_team_execution_matches_oracle(exe, cfg):
    """The staged matrix elements evaluated the way the kernels do it: by the two warps of a pair (configs 4, 5) or the
    four warps of a team (W + 4 jets: two halves of the innermost helicity loop x two groups of closings), played by
    host threads that share one staging area and meet at every st.sync().  Checks what the single-threaded run
    cannot: the dealing of the shared phases (st.own), the partition of the closings with its duplicated sub-currents
    (st.grp), the per-warp accumulator sets, and that every rendezvous is reached by every warp."""
    par = osm.default_params()
    p, _ = ops.generate(cfg, 9, 0, N[cfg], opr.SQRT_S[cfg], par)
    ref = opr.me2(opr.config(cfg), p, par)
    text = '\n'.join('%d ' % cfg + ' '.join('%.17g' % x for x in ev.reshape(-1)) for ev in p) + '\n'
    out = subprocess.run([exe, 'team'], input=text, capture_output=True, text=True, check=True, timeout=600).stdout.split()
    got = np.array([float(x) for x in out])
    assert got.shape == ref.shape
    assert (np.abs(got - ref) / ref).max() <= 1e-11


@pytest.mark.parametrize('cfg', [1, 3, 6, 7, 8, 10, 11])
def test_complex_mass_option_matches_oracle(exe, cfg):
    """hg_params.complex_mass = 1 (Eq. 55-56): complex m_V^2 in the q q / m_V^2 terms and in the
    couplings g_W m_W, g_Z m_Z, 1/v; Gamma_W from Eq. 56.  The option changes the result (by O(Gamma/m)), and the
    generated code follows the oracle's implementation of the same option."""
    par = dict(osm.default_params(), complex_mass=1)
    p, _ = ops.generate(cfg, 8, 0, N[cfg], opr.SQRT_S[cfg], par)
    ref = opr.me2(opr.config(cfg), p, par)
    ref0 = opr.me2(opr.config(cfg), p, osm.default_params())
    text = '\n'.join('%d ' % -cfg + ' '.join('%.17g' % x for x in ev.reshape(-1)) for ev in p) + '\n'
    out = subprocess.run([exe], input=text, capture_output=True, text=True, check=True).stdout.split()
    got = np.array([float(x) for x in out])
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max() and (np.abs(got - ref) / ref).max() <= 1e-11
    if cfg != 3:
        assert (np.abs(ref0 - ref) / ref).max() > 1e-6      # the option is not a no-op


def test_host_step_tool_matches_oracle(tmp_path):
    """gen/hoststep.cpp (bench.py's `cpu_generated_code`: the generated code on the CPU cores) runs the whole path;
    its sums equal the oracle's on the same Philox stream."""
    import math
    from oracle import integrate as oint
    exe = str(tmp_path / 'hoststep')
    subprocess.check_call(['g++', '-O1', '-fopenmp', '-std=c++17',
                           os.path.join(ROOT, 'paper_1305_0708_b200', 'gen', 'hoststep.cpp'), '-o', exe, '-lm'])
    par = osm.default_params()
    for cfg, n in ((3, 1500), (10, 800)):
        out = subprocess.check_output([exe, str(cfg), repr(opr.SQRT_S[cfg]), '77', '11', str(n)], text=True).split()
        w, ok = oint.weights(cfg, 77, 11, n, opr.SQRT_S[cfg], par)
        ref = oint.accumulate(w, ok)
        assert float(out[2]) == ref[3]
        assert abs(float(out[0]) - ref[0]) <= 1e-10 * ref[0] and abs(float(out[1]) - ref[1]) <= 2e-10 * ref[1]
