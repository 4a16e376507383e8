"""hg_accumulate_noalloc (include/hg.h): the allocation-free variant of hg_accumulate, against hg_accumulate.

Collected last on purpose (the suite runs with pytest -x).  The two paths add the same per-event weights in a
different order (fixed 4096-event ranges per block here, a grid sized by the SM count there), so the sums agree
to rounding: 1e-12 relative, the tolerance tests/test_gpu_parity.py uses for sums; n and n_pass are exact.
"""
import pytest
import torch

pytestmark = pytest.mark.gpu

SEED = 13050708
RS = 1000.0     # W + 2 jets (config 3) at its BASELINE.json energy
REL = 1e-12


@pytest.fixture(scope='module')
def api():
    from paper_1305_0708_b200 import api
    return api


@pytest.fixture(scope='module')
def ctx(api):
    c = api.Context(0)
    yield c
    c.close()


def _inputs(ctx, api, precision, first, n):
    p, wps, ok = ctx.hg_gen_phase_space(3, precision, SEED, first, n, RS)
    me = ctx.hg_matrix_element(3, precision, p)
    return me, wps, ok


def _close(got, ref):
    assert got[2] == ref[2] and got[3] == ref[3], (got, ref)
    for i in (0, 1):
        assert abs(got[i] - ref[i]) <= REL * abs(ref[i]), (i, got, ref)


@pytest.mark.parametrize('prec', ['f64', 'f32'])
def test_two_calls_in_a_row_match_hg_accumulate(ctx, api, prec):
    precision = api.HG_F64 if prec == 'f64' else api.HG_F32
    torch.cuda.set_device(0)
    acc = torch.full((4,), float('nan'), dtype=torch.float64, device='cuda')
    # first call: many blocks and a ragged tail; second: fewer events (the array still holds the first call's
    # partial sums beyond the blocks the second call uses) and no pass array
    big = _inputs(ctx, api, precision, 0, 3 * 4096 * 37 + 1234)
    small = _inputs(ctx, api, precision, 777, 4096 + 5)
    ref_big = ctx.hg_accumulate(precision, big[0], big[1], big[2], RS)
    ref_small = ctx.hg_accumulate(precision, small[0], small[1], None, RS)
    assert ref_big[3] > 0 and ref_big[3] < ref_big[2]      # the cuts reject some events
    api.hg_accumulate_noalloc(precision, big[0], big[1], big[2], RS, acc)
    got_big = acc.cpu().tolist()                           # synchronises
    free0 = torch.cuda.mem_get_info()[0]
    api.hg_accumulate_noalloc(precision, small[0], small[1], None, RS, acc)
    got_small = acc.cpu().tolist()
    free1 = torch.cuda.mem_get_info()[0]
    _close(got_big, ref_big)
    _close(got_small, ref_small)
    assert free1 == free0                                  # no device memory taken by the call
    # and once more with the first inputs: same bits as before (fixed summation order, nothing left over)
    api.hg_accumulate_noalloc(precision, big[0], big[1], big[2], RS, acc)
    assert acc.cpu().tolist() == got_big


def test_empty_and_limits(api):
    torch.cuda.set_device(0)
    acc = torch.full((4,), float('nan'), dtype=torch.float64, device='cuda')
    e = torch.empty((0,), dtype=torch.float64, device='cuda')
    api.hg_accumulate_noalloc(api.HG_F64, e, e, None, RS, acc)
    assert acc.cpu().tolist() == [0.0, 0.0, 0.0, 0.0]
    # one event more than the static array covers: rejected before anything is launched, acc untouched
    acc.fill_(-1.0)
    n = api.HG_NOALLOC_MAX_EVENTS + 1
    x = torch.zeros((n,), dtype=torch.float32, device='cuda')
    with pytest.raises(api.HgError) as err:
        api.hg_accumulate_noalloc(api.HG_F32, x, x, None, RS, acc)
    assert err.value.code == api.HG_EINVAL and 'HG_NOALLOC_MAX_EVENTS' in str(err.value)
    assert acc.cpu().tolist() == [-1.0] * 4
    # exactly the maximum is accepted: 4096 blocks, all ones -> sum w = n * wscale
    y = torch.ones((api.HG_NOALLOC_MAX_EVENTS,), dtype=torch.float32, device='cuda')
    api.hg_accumulate_noalloc(api.HG_F32, y, y, None, RS, acc)
    got = acc.cpu().tolist()
    assert got[2] == got[3] == float(api.HG_NOALLOC_MAX_EVENTS)
    assert abs(got[0] / got[2] - got[1] / got[0]) <= 1e-12 * got[0] / got[2]     # w constant: <w> = <w^2>/<w>
    with pytest.raises(api.HgError):
        api.hg_accumulate_noalloc(api.HG_F64, e, e, None, float('nan'), acc)


def test_under_cuda_graph_capture(ctx, api):
    """What the entry point is for: it can be captured into a CUDA graph (no allocation, no synchronisation, no
    host-side result) and replayed on new contents of the same buffers."""
    torch.cuda.set_device(0)
    precision = api.HG_F64
    n = 3 * 4096 + 77
    me, wps, ok = _inputs(ctx, api, precision, 4242, n)
    acc = torch.zeros((4,), dtype=torch.float64, device='cuda')
    api.hg_accumulate_noalloc(precision, me, wps, ok, RS, acc)      # set-up (symbol address) outside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        api.hg_accumulate_noalloc(precision, me, wps, ok, RS, acc)   # launches go to the capturing stream
    for first in (4242, 99):
        me2, wps2, ok2 = _inputs(ctx, api, precision, first, n)
        me.copy_(me2)
        wps.copy_(wps2)
        ok.copy_(ok2)
        acc.fill_(float('nan'))
        g.replay()
        torch.cuda.synchronize()
        _close(acc.cpu().tolist(), ctx.hg_accumulate(precision, me, wps, ok, RS))
