"""Event weights and BASES-style accumulation (oracle; test infrastructure).

Step a9/a10 of SURVEY.md 8a:  w = Theta_cuts * 1/(2 s_hat) * |Mbar|^2 * w_ps * (hbar c)^2  [pb]
(Eq. 4), accumulated as sum w, sum w^2, N, N_pass.
sigma = sum w / N,  delta sigma = sqrt((sum w^2 / N - sigma^2) / (N - 1)).
"""
import math
import numpy as np

from . import phase_space as ps
from . import processes as pr
from . import sm


def weights(cfg, seed, first_event, n, rs, par, cuts=None, batch=1024, skip_failed=True, grid=None, bins_out=None):
    """Per-event weights [n] in pb and pass flags, for events first_event.. of config cfg.  grid: adaptive grid of
    oracle.vegas (None = flat); bins_out [n, n_draws] receives the bin of every draw."""
    proc = pr.config(cfg)
    w = np.zeros(n)
    ok_all = np.zeros(n, dtype=bool)
    for i in range(0, n, batch):
        m = min(batch, n - i)
        p, wps, bins = ps.generate(cfg, seed, first_event + i, m, rs, par, grid=grid, with_bins=True)
        if bins_out is not None and bins is not None:
            bins_out[i:i + m] = bins
        ok = ps.passes(cfg, p, cuts)
        ok_all[i:i + m] = ok
        idx = np.nonzero(ok)[0] if skip_failed else np.arange(m)
        if len(idx):
            me = pr.me2(proc, p[idx], par)
            w[i + idx] = me * wps[idx] / (2.0 * rs * rs) * sm.HBARC2_PB * ok[idx]
    return w, ok_all


def accumulate(w, ok):
    """(sum w, sum w^2, N, N_pass) with exact (math.fsum) summation."""
    return math.fsum(w), math.fsum(w * w), float(len(w)), float(np.count_nonzero(ok))


def sigma(acc):
    sw, sw2, n, _ = acc
    s = sw / n
    var = max(sw2 / n - s * s, 0.0) / (n - 1.0)
    return s, math.sqrt(var)
