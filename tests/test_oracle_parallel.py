"""oracle.parallel cuts a batch into slices for worker processes: same numbers as the single-process calls."""
import numpy as np

from oracle import integrate as oint
from oracle import parallel
from oracle import phase_space as ops
from oracle import processes as opr
from oracle import sm as osm


def test_parallel_equals_serial():
    par = osm.default_params()
    try:
        for cfg, n in ((3, 1300), (4, 40)):
            p, _ = ops.generate(cfg, 5, 7, n, opr.SQRT_S[cfg], par)
            a = parallel.me2(cfg, p, par, slice_events=n // 5)
            b = opr.me2(opr.config(cfg), p, par)
            assert a.shape == b.shape and np.array_equal(a, b)
            w, ok = parallel.weights(cfg, 5, 7, n, opr.SQRT_S[cfg], par, slice_events=n // 5)
            w0, ok0 = oint.weights(cfg, 5, 7, n, opr.SQRT_S[cfg], par)
            assert np.array_equal(ok, ok0) and np.array_equal(w, w0)
        p, _ = ops.generate(3, 5, 0, 64, 1000.0, par)
        e = parallel.me2(3, p, par, extended=True, slice_events=16)
        assert np.array_equal(e, opr.me2_extended(opr.config(3), p, par))
        assert np.abs(e / opr.me2(opr.config(3), p, par) - 1).max() < 1e-12
    finally:
        parallel.close()
