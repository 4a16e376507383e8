"""Thin ctypes binding of libhg.so (include/hg.h): argument marshalling only, same names as the C ABI.

PyTorch supplies device memory and streams (`tensor.data_ptr()`, `torch.cuda.current_stream().cuda_stream`); every
step of the path runs in the library's kernels.  There is no CPU fallback: importing works without a GPU (the
library loads and its host-only calls work), any compute call without a CUDA device fails loudly.
"""
import ctypes as C
import os

import torch

HG_F64, HG_F32 = 0, 1
HG_UDX_EPVE, HG_UUX_EPEMG, HG_UDX_EPVEGG, HG_GG_TTXG_DILEP, HG_UDX_EPVEGGG = 1, 2, 3, 4, 5
PROCESSES = (1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11)
HG_OK, HG_EINVAL, HG_ENOPROC, HG_ECUDA, HG_ENOTSET = 0, -1, -2, -3, -4

# symbols include/hg.h declares (checked by tests/test_abi.py)
SYMBOLS = ('hg_create', 'hg_destroy', 'hg_last_error', 'hg_default_params', 'hg_default_cuts', 'hg_process_info',
           'hg_set_params', 'hg_gen_phase_space', 'hg_matrix_element', 'hg_matrix_element_host',
           'hg_matrix_element_host_cm', 'hg_accumulate', 'hg_accumulate_noalloc',
           'hg_integrate_step', 'hg_set_grid', 'hg_grid_refine', 'hg_default_hadronic', 'hg_set_hadronic')
HG_GRID_MAX_BINS = 64
# measurement helpers of include/hg_bench.h (bench.py only)
BENCH_SYMBOLS = ('hg_set_profiling', 'hg_last_step_info', 'hg_measure_fma_peak')


class hg_params(C.Structure):
    _fields_ = [(n, C.c_double) for n in ('mz', 'mw', 'gz', 'gw', 'mt', 'gt', 'mb', 'mh', 'gh', 'alpha_em_inv',
                                          'alpha_s')] + [('ckm_diagonal', C.c_int), ('complex_mass', C.c_int)]


class hg_cuts(C.Structure):
    _fields_ = [(n, C.c_double) for n in ('pt_jet_min', 'eta_jet_max', 'eta_lep_max', 'dr_jj_min')]


class hg_hadronic(C.Structure):
    _fields_ = [('y_res_max', C.c_double), ('pdf_norm', C.c_double * 2), ('pdf_a', C.c_double * 2),
                ('pdf_b', C.c_double * 2)]


class hg_process_info_t(C.Structure):
    _fields_ = [(n, C.c_int) for n in ('n_ext', 'n_final', 'n_hel_total', 'n_hel_nonzero', 'n_diagrams',
                                       'n_amplitudes', 'n_flows', 'n_draws')] + \
               [(n, C.c_double) for n in ('avg_factor', 'flops_f64', 'flops_ps')]


class HgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__('hg error %d: %s' % (code, msg))
        self.code = code


_LIB = None


def lib_path():
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), 'libhg.so')


def load():
    """Load libhg.so (built in-tree by paper_1305_0708_b200.build).  Raises if it is missing: no fallback."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError('%s not found: run `python -m paper_1305_0708_b200.build` (nvcc, sm_100a)' % path)
    L = C.CDLL(path)
    vp, i32, i64, u64, dbl = C.c_void_p, C.c_int, C.c_int64, C.c_uint64, C.c_double
    L.hg_create.argtypes = [C.POINTER(vp), i32]
    L.hg_destroy.argtypes = [vp]
    L.hg_destroy.restype = None
    L.hg_last_error.argtypes = [vp]
    L.hg_last_error.restype = C.c_char_p
    L.hg_default_params.argtypes = [C.POINTER(hg_params)]
    L.hg_default_params.restype = None
    L.hg_default_cuts.argtypes = [i32, C.POINTER(hg_cuts)]
    L.hg_process_info.argtypes = [i32, C.POINTER(hg_process_info_t)]
    L.hg_set_params.argtypes = [vp, C.POINTER(hg_params), C.POINTER(hg_cuts)]
    L.hg_gen_phase_space.argtypes = [vp, i32, i32, u64, u64, i64, dbl, vp, vp, vp, vp]
    L.hg_matrix_element.argtypes = [vp, i32, i32, i64, vp, vp, vp]
    L.hg_matrix_element_host.argtypes = [vp, i32, i32, i64, vp, vp, vp]
    L.hg_matrix_element_host_cm.argtypes = [vp, i32, i32, i64, dbl, vp, vp, vp]
    L.hg_accumulate.argtypes = [vp, i32, i64, vp, vp, vp, dbl, C.POINTER(dbl), vp]
    L.hg_accumulate_noalloc.argtypes = [i32, i64, vp, vp, vp, dbl, vp, vp]
    L.hg_integrate_step.argtypes = [vp, i32, i32, u64, u64, i64, dbl, C.POINTER(dbl), vp]
    L.hg_default_hadronic.argtypes = [i32, C.POINTER(hg_hadronic)]
    L.hg_set_hadronic.argtypes = [vp, C.POINTER(hg_hadronic)]
    L.hg_set_grid.argtypes = [vp, vp, i32, i32, vp]
    L.hg_grid_refine.argtypes = [i32, i32, vp, dbl, vp]
    L.hg_measure_fma_peak.argtypes = [vp, i32, C.POINTER(dbl), vp]
    L.hg_set_profiling.argtypes = [vp, i32]
    L.hg_last_step_info.argtypes = [vp, C.POINTER(dbl)]
    _LIB = L
    return L


def hg_default_params():
    p = hg_params()
    load().hg_default_params(C.byref(p))
    return p


def hg_default_cuts(process):
    c = hg_cuts()
    rc = load().hg_default_cuts(process, C.byref(c))
    if rc != HG_OK:
        raise HgError(rc, 'unknown process id')
    return c


def hg_default_hadronic(process):
    h = hg_hadronic()
    rc = load().hg_default_hadronic(process, C.byref(h))
    if rc != HG_OK:
        raise HgError(rc, 'unknown process id')
    return h


def hg_process_info(process):
    info = hg_process_info_t()
    rc = load().hg_process_info(process, C.byref(info))
    if rc != HG_OK:
        raise HgError(rc, 'unknown process id')
    return {n: getattr(info, n) for n, _ in hg_process_info_t._fields_}


def hg_grid_refine(hist, alpha, grid):
    """One refinement of the grid [n_dim, n_bins + 1] (host float64 tensor, updated in place) from hist [n_dim, n_bins]."""
    n_dim, nb1 = grid.shape
    for t, shape in ((grid, (n_dim, nb1)), (hist, (n_dim, nb1 - 1))):
        if t.device.type != 'cpu' or t.dtype != torch.float64 or not t.is_contiguous() or tuple(t.shape) != shape:
            raise ValueError('grid / hist must be contiguous host float64 tensors [n_dim, n_bins + 1] / [n_dim, n_bins]')
    rc = load().hg_grid_refine(n_dim, nb1 - 1, C.c_void_p(hist.data_ptr()), float(alpha), C.c_void_p(grid.data_ptr()))
    if rc != HG_OK:
        raise HgError(rc, 'hg_grid_refine: bad argument')
    return grid


def _dtype(precision):
    return torch.float64 if precision == HG_F64 else torch.float32


HG_NOALLOC_MAX_EVENTS = 1 << 24


def hg_accumulate_noalloc(precision, me2, wps, passed, sqrt_s_hat, acc, stream=None):
    """hg_accumulate without a context and without any allocation (include/hg.h): acc is a CUDA float64 tensor of 4
    elements that the CALLER provides; it receives (sum w, sum w^2, n, n_pass) asynchronously on the stream.  The
    tensors must live on the current CUDA device."""
    n = me2.numel()
    dt = _dtype(precision)
    for t, name, want in ((me2, 'me2', dt), (wps, 'wps', dt), (passed, 'pass', torch.uint8)):
        if t is None and name == 'pass':
            continue
        if t.device.type != 'cuda' or t.dtype != want or not t.is_contiguous() or t.numel() != n:
            raise ValueError('%s must be a contiguous CUDA %s tensor with %d elements' % (name, want, n))
    if acc.device.type != 'cuda' or acc.dtype != torch.float64 or not acc.is_contiguous() or acc.numel() != 4:
        raise ValueError('acc must be a contiguous CUDA float64 tensor with 4 elements')
    L = load()
    rc = L.hg_accumulate_noalloc(precision, n, _ptr(me2), _ptr(wps), _ptr(passed), float(sqrt_s_hat), _ptr(acc),
                                 _stream(stream))
    if rc != 0:
        raise HgError(rc, L.hg_last_error(None).decode())
    return acc


def _stream(stream):
    if stream is None:
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, 'cuda_stream') else int(stream)


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


class Context:
    """hg_ctx with the C calls as methods of the same names."""

    def __init__(self, device=0, params=None, cuts=None):
        self._L = load()
        if not torch.cuda.is_available():
            raise RuntimeError('paper_1305_0708_b200 needs a CUDA device: there is no CPU path')
        h = C.c_void_p()
        rc = self._L.hg_create(C.byref(h), int(device))
        if rc != HG_OK:
            raise HgError(rc, self._L.hg_last_error(None).decode())
        self._h = h
        self.device = torch.device('cuda', int(device))
        self.hg_set_params(params if params is not None else hg_default_params(), cuts)

    def close(self):
        if getattr(self, '_h', None):
            self._L.hg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc != HG_OK:
            raise HgError(rc, self._L.hg_last_error(self._h).decode())

    def hg_set_params(self, params, cuts=None):
        self._check(self._L.hg_set_params(self._h, C.byref(params), C.byref(cuts) if cuts is not None else None))

    def _check_tensor(self, t, precision, numel, name, dtype=None):
        dtype = dtype or _dtype(precision)
        if t.device.type != 'cuda' or t.dtype != dtype or not t.is_contiguous() or t.numel() != numel:
            raise ValueError('%s must be a contiguous CUDA %s tensor with %d elements' % (name, dtype, numel))

    def hg_gen_phase_space(self, process, precision, seed, first_event, n, sqrt_s_hat, p=None, wps=None,
                           passed=None, stream=None, want_pass=True):
        """Returns (p [n_ext,4,n], wps [n], pass [n] uint8).  Buffers are allocated with torch if not given."""
        n_ext = hg_process_info(process)['n_ext']
        dt = _dtype(precision)
        if p is None:
            p = torch.empty((n_ext, 4, n), dtype=dt, device=self.device)
        if wps is None:
            wps = torch.empty((n,), dtype=dt, device=self.device)
        if passed is None and want_pass:
            passed = torch.empty((n,), dtype=torch.uint8, device=self.device)
        self._check_tensor(p, precision, n_ext * 4 * n, 'p')
        self._check_tensor(wps, precision, n, 'wps')
        if passed is not None:
            self._check_tensor(passed, precision, n, 'pass', torch.uint8)
        self._check(self._L.hg_gen_phase_space(self._h, process, precision, seed, first_event, n, sqrt_s_hat,
                                               _ptr(p), _ptr(wps), _ptr(passed), _stream(stream)))
        return p, wps, passed

    def hg_matrix_element(self, process, precision, p, me2=None, stream=None):
        """p: CUDA tensor [n_ext, 4, n] (SoA).  Returns me2 [n]."""
        n_ext = hg_process_info(process)['n_ext']
        n = p.numel() // (4 * n_ext)
        self._check_tensor(p, precision, n_ext * 4 * n, 'p')
        if me2 is None:
            me2 = torch.empty((n,), dtype=_dtype(precision), device=p.device)
        self._check_tensor(me2, precision, n, 'me2')
        self._check(self._L.hg_matrix_element(self._h, process, precision, n, _ptr(p), _ptr(me2), _stream(stream)))
        return me2

    def hg_matrix_element_host(self, process, precision, p, me2=None, stream=None):
        """p: HOST tensor [n_ext, 4, n] (pinned for full speed).  Returns a host tensor me2 [n]; synchronises."""
        n_ext = hg_process_info(process)['n_ext']
        n = p.numel() // (4 * n_ext)
        dt = _dtype(precision)
        if p.device.type != 'cpu' or p.dtype != dt or not p.is_contiguous():
            raise ValueError('p must be a contiguous host %s tensor' % dt)
        if me2 is None:
            me2 = torch.empty((n,), dtype=dt).pin_memory()
        if me2.device.type != 'cpu' or me2.dtype != dt or not me2.is_contiguous() or me2.numel() != n:
            raise ValueError('me2 must be a contiguous host %s tensor with %d elements' % (dt, n))
        self._check(self._L.hg_matrix_element_host(self._h, process, precision, n, _ptr(p), _ptr(me2),
                                                   _stream(stream)))
        return me2

    def hg_matrix_element_host_cm(self, process, precision, sqrt_s_hat, pfinal, me2=None, stream=None):
        """pfinal: HOST tensor [n_ext - 2, 4, n] of the final-state momenta in the partonic centre-of-mass frame (the
        incoming legs are sqrt_s_hat/2 (1, 0, 0, +-1) and are not shipped).  Returns a host tensor me2 [n]."""
        n_fin = hg_process_info(process)['n_ext'] - 2
        n = pfinal.numel() // (4 * n_fin)
        dt = _dtype(precision)
        if pfinal.device.type != 'cpu' or pfinal.dtype != dt or not pfinal.is_contiguous() or \
                pfinal.numel() != 4 * n_fin * n:
            raise ValueError('pfinal must be a contiguous host %s tensor [n_ext - 2, 4, n]' % dt)
        if me2 is None:
            me2 = torch.empty((n,), dtype=dt).pin_memory()
        if me2.device.type != 'cpu' or me2.dtype != dt or not me2.is_contiguous() or me2.numel() != n:
            raise ValueError('me2 must be a contiguous host %s tensor with %d elements' % (dt, n))
        self._check(self._L.hg_matrix_element_host_cm(self._h, process, precision, n, sqrt_s_hat, _ptr(pfinal),
                                                      _ptr(me2), _stream(stream)))
        return me2

    def hg_accumulate(self, precision, me2, wps, passed, sqrt_s_hat, stream=None):
        n = me2.numel()
        self._check_tensor(me2, precision, n, 'me2')
        self._check_tensor(wps, precision, n, 'wps')
        if passed is not None:
            self._check_tensor(passed, precision, n, 'pass', torch.uint8)
        acc = (C.c_double * 4)()
        self._check(self._L.hg_accumulate(self._h, precision, n, _ptr(me2), _ptr(wps), _ptr(passed), sqrt_s_hat,
                                          acc, _stream(stream)))
        return tuple(acc)

    def hg_integrate_step(self, process, precision, seed, first_event, n, sqrt_s_hat, stream=None):
        """Returns (sum w, sum w^2, n, n_pass), w in pb."""
        acc = (C.c_double * 4)()
        self._check(self._L.hg_integrate_step(self._h, process, precision, seed, first_event, n, sqrt_s_hat, acc,
                                              _stream(stream)))
        return tuple(acc)

    def hg_set_hadronic(self, had):
        """had: hg_hadronic (the paper's hadronic phase space with toy parton densities) or None (RAMBO at fixed s_hat)."""
        self._check(self._L.hg_set_hadronic(self._h, C.byref(had) if had is not None else None))

    def hg_set_grid(self, grid, hist=None):
        """grid: CUDA float64 tensor [n_draws, n_bins + 1] (kept alive by the context wrapper) or None for flat
        sampling; hist: CUDA float64 tensor [n_draws, n_bins] that hg_integrate_step adds sum w^2 per bin to."""
        if grid is None:
            self._grid = self._hist = None
            self._check(self._L.hg_set_grid(self._h, None, 0, 0, None))
            return
        n_dim, nb1 = grid.shape
        self._check_tensor(grid, HG_F64, n_dim * nb1, 'grid', torch.float64)
        if hist is not None:
            self._check_tensor(hist, HG_F64, n_dim * (nb1 - 1), 'hist', torch.float64)
        self._grid, self._hist = grid, hist
        self._check(self._L.hg_set_grid(self._h, _ptr(grid), n_dim, nb1 - 1, _ptr(hist)))

    def hg_set_profiling(self, on):
        self._check(self._L.hg_set_profiling(self._h, 1 if on else 0))

    def hg_last_step_info(self):
        """(ms in phase-space kernels, ms in matrix-element kernels, kernels launched) of the last step."""
        out = (C.c_double * 3)()
        self._check(self._L.hg_last_step_info(self._h, out))
        return out[0], out[1], int(out[2])

    def hg_measure_fma_peak(self, precision, stream=None):
        out = C.c_double()
        self._check(self._L.hg_measure_fma_peak(self._h, precision, C.byref(out), _stream(stream)))
        return out.value

