"""Small run of every entry point of libhg.so for every process and both precisions -- the target of
`compute-sanitizer` (memcheck / racecheck / synccheck) and a quick installation check.

    python -m paper_1305_0708_b200.selfcheck [--n 300] [--processes 4,5,9] [--big]

It checks internal consistency only (no oracle): hg_integrate_step == hg_gen_phase_space -> hg_matrix_element ->
hg_accumulate on the same counter range, finite positive |Mbar|^2, fp32 close to fp64.  --big adds one multi-chunk
case per process (n = 2^20 + 777) so that the chunked code paths run under the tool as well (slow under racecheck).
"""
import argparse
import sys

import torch

from . import api

SQRT_S = {1: 80.0, 2: 500.0, 3: 1000.0, 4: 1500.0, 5: 2000.0, 6: 500.0, 7: 1000.0, 8: 1000.0, 9: 3000.0, 10: 1000.0,
          11: 1000.0}


def run(processes, n, big=False, seed=13050708):
    ctx = api.Context(0)
    bad = 0
    for pid in processes:
        rs = SQRT_S.get(pid, 2000.0)
        for n_ev in ([n] + ([(1 << 20) + 777] if big else [])):
            p, wps, ok = ctx.hg_gen_phase_space(pid, api.HG_F64, seed, 3, n_ev, rs)
            me = ctx.hg_matrix_element(pid, api.HG_F64, p)
            me32 = ctx.hg_matrix_element(pid, api.HG_F32, p.float())
            acc = ctx.hg_accumulate(api.HG_F64, me, wps, ok, rs)
            st = ctx.hg_integrate_step(pid, api.HG_F64, seed, 3, n_ev, rs)
            st32 = ctx.hg_integrate_step(pid, api.HG_F32, seed, 3, n_ev, rs)
            hme = ctx.hg_matrix_element_host(pid, api.HG_F64, p.cpu().pin_memory())
            torch.cuda.synchronize()
            good = bool(torch.isfinite(me).all() and (me > 0).all())
            good &= torch.equal(hme.cuda(), me)
            good &= acc[3] == st[3] == st32[3] and abs(acc[0] - st[0]) <= 1e-12 * abs(st[0])
            good &= abs(st32[0] - st[0]) <= 1e-3 * abs(st[0])
            sel = ok.bool()
            if sel.any():
                rel = ((me32.double() - me).abs() / me)[sel]
                good &= bool(rel.median() <= 1e-5)
            print('process %d  n=%d  pass %d  sum w %.6e  %s' % (pid, n_ev, int(st[3]), st[0], 'ok' if good else 'FAILED'))
            bad += 0 if good else 1
    ctx.close()
    return bad


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument('--n', type=int, default=300)
    ap.add_argument('--processes', default=','.join(str(p) for p in api.PROCESSES))
    ap.add_argument('--big', action='store_true')
    a = ap.parse_args()
    sys.exit(1 if run([int(x) for x in a.processes.split(',')], a.n, a.big) else 0)


if __name__ == '__main__':
    main()
