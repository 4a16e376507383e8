"""The C-ABI library loads on a CPU-only box and exports every symbol include/hg.h declares; host-only calls work."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope='module')
def api():
    from paper_1305_0708_b200 import build
    build.build()
    from paper_1305_0708_b200 import api
    return api


def test_exports_every_declared_symbol(api):
    lib = api.load()
    for header, symbols in (('hg.h', api.SYMBOLS), ('hg_bench.h', api.BENCH_SYMBOLS)):
        hdr = open(os.path.join(ROOT, 'include', header)).read()
        hdr = re.sub(r'/\*.*?\*/', '', hdr, flags=re.S)
        declared = set(re.findall(r'\b(hg_[a-z0-9_]+)\s*\(', hdr))
        assert declared == set(symbols), header
        for s in declared:
            assert hasattr(lib, s), s
    assert sorted(os.listdir(os.path.join(ROOT, 'include'))) == ['hg.h', 'hg_bench.h']


def test_process_info_matches_survey_table(api):
    # SURVEY.md 8a per-config table: (n_ext, hel total / non-zero, diagrams / amplitudes, flows)
    expect = {1: (4, 16, 1, 1, 1, 1), 2: (5, 32, 8, 4, 4, 1), 3: (6, 64, 4, 8, 8, 2), 4: (9, 512, 8, 16, 18, 6),
              5: (7, 128, 8, 50, 54, 6),
              # NEXT-1 / NEXT-4 processes; a scalar leg has one state
              6: (5, 16, 1, 1, 1, 1), 7: (6, 16, 4, 4, 4, 1), 8: (5, 16, 16, 8, 8, 2), 9: (8, 256, 16, 428, 516, 24),
              # weak-boson fusion, two quark lines: W W and Z Z fusion = two colour flows
              10: (5, 16, 4, 2, 2, 2), 11: (6, 16, 4, 8, 8, 2)}
    avg = {1: 1 / 36, 2: 1 / 36, 3: 1 / 72, 4: 1 / 256, 5: 1 / 216, 6: 1 / 36, 7: 1 / 72, 8: 1 / 256, 9: 1 / 864,
           10: 1 / 36, 11: 1 / 72}
    for pid, e in expect.items():
        i = api.hg_process_info(pid)
        assert (i['n_ext'], i['n_hel_total'], i['n_hel_nonzero'], i['n_diagrams'], i['n_amplitudes'],
                i['n_flows']) == e
        assert abs(i['avg_factor'] - avg[pid]) < 1e-15
        assert i['flops_f64'] > 100 and i['n_draws'] in (8, 12, 16, 24, 20)
    with pytest.raises(api.HgError):
        api.hg_process_info(0)


def test_defaults(api):
    p = api.hg_default_params()
    assert (p.mz, p.mw, p.gz, p.gw, p.mt, p.gt, p.alpha_em_inv, p.alpha_s) == \
        (91.1876, 80.419, 2.441, 2.048, 174.3, 1.5, 132.507, 0.118)
    c = api.hg_default_cuts(5)
    assert (c.pt_jet_min, c.eta_jet_max, c.eta_lep_max, c.dr_jj_min) == (20.0, 2.5, 0.0, 0.4)


def test_no_cpu_fallback(api):
    import torch
    if torch.cuda.is_available():
        pytest.skip('GPU present')
    with pytest.raises(RuntimeError):
        api.Context(0)


def test_grid_refine_matches_oracle(api):
    """hg_grid_refine (host C++) against oracle.vegas.refine on random histograms, peaked ones, and empty rows."""
    import numpy as np
    import torch
    from oracle import vegas
    rng = np.random.default_rng(3)
    for nb in (2, 16, 50, 64):
        ndim = 5
        grid = np.sort(np.concatenate([np.zeros((ndim, 1)), rng.uniform(0, 1, (ndim, nb - 1)), np.ones((ndim, 1))], 1), 1)
        hist = rng.uniform(0, 1, (ndim, nb)) ** 8
        hist[1] = 0.0                      # nothing accumulated: row unchanged
        hist[2, : nb // 2] = 0.0           # empty bins
        hist[3] = 0.0
        hist[3, nb // 3] = 7.0             # everything in one bin
        for alpha in (1.5, 1.0, 0.3):
            want = vegas.refine(grid, hist, alpha)
            got = torch.from_numpy(grid.copy())
            api.hg_grid_refine(torch.from_numpy(hist.copy()), alpha, got)
            got = got.numpy()
            assert np.array_equal(got[1], grid[1])
            assert np.allclose(got, want, rtol=0, atol=1e-14), (nb, alpha, np.abs(got - want).max())
            assert np.all(np.diff(got, axis=1) > 0) and np.all(got[:, 0] == 0) and np.all(got[:, -1] == 1)
    with pytest.raises(api.HgError):
        api.hg_grid_refine(torch.zeros((2, 100), dtype=torch.float64), 1.5, torch.zeros((2, 101), dtype=torch.float64))
