"""Runs the oracle over the host cores (oracle; test infrastructure): the oracle is vectorised over events and
events are independent (one phase-space point at a time), so a batch is cut into slices that
worker processes evaluate with the unchanged single-process functions.  Nothing of the method lives here.

Workers are spawned (not forked): the parent may hold a CUDA context."""
import multiprocessing as mp
import os

import numpy as np

_POOL = None


def _init():
    for v in ('OMP_NUM_THREADS', 'OPENBLAS_NUM_THREADS', 'MKL_NUM_THREADS'):
        os.environ[v] = '1'


def _weights_slice(args):
    cfg, seed, first, n, rs, par = args
    from oracle import integrate as oint
    w, ok = oint.weights(cfg, seed, first, n, rs, par)
    return w, ok


def _me2_slice(args):
    cfg, p, par, extended = args
    from oracle import processes as opr
    proc = opr.config(cfg)
    if extended:
        return opr.me2_extended(proc, p, par, on_shell=(extended != 'given'))
    return opr.me2(proc, p, par)


def n_workers():
    return max(1, min(32, os.cpu_count() or 1))


def pool():
    global _POOL
    if _POOL is None:
        _POOL = mp.get_context('spawn').Pool(n_workers(), initializer=_init)
    return _POOL


def close():
    global _POOL
    if _POOL is not None:
        _POOL.terminate()
        _POOL = None


def me2(cfg, p, par, extended=False, slice_events=None):
    """oracle.processes.me2 (or me2_extended: extended=True, or 'given' for on_shell=False) of config cfg on momenta
    p [N, n_ext, 4], over all host cores."""
    n = len(p)
    if n == 0:
        return np.zeros(0)
    workers = n_workers()
    if slice_events is None:
        slice_events = max(1, min(512, -(-n // (4 * workers))))
    if n <= slice_events or workers == 1:
        return _me2_slice((cfg, p, par, extended))
    jobs = [(cfg, p[i:i + slice_events], par, extended) for i in range(0, n, slice_events)]
    return np.concatenate(pool().map(_me2_slice, jobs, chunksize=1))


def weights(cfg, seed, first_event, n, rs, par, slice_events=None):
    """oracle.integrate.weights (Philox -> momenta -> cuts -> |Mbar|^2 -> weight) for events first_event ..
    first_event + n - 1, over all host cores.  Returns (w [n], pass flags [n])."""
    workers = n_workers()
    if slice_events is None:
        slice_events = max(1, min(512, -(-n // (4 * workers))))
    if n <= slice_events or workers == 1:
        return _weights_slice((cfg, seed, first_event, n, rs, par))
    jobs = [(cfg, seed, first_event + i, min(slice_events, n - i), rs, par) for i in range(0, n, slice_events)]
    res = pool().map(_weights_slice, jobs, chunksize=1)
    return np.concatenate([r[0] for r in res]), np.concatenate([r[1] for r in res])
