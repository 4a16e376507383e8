"""bench.py -- helicity+colour-summed |M|^2 events/s on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference] [--all-configs]

A step is one pass of the whole hot path over one batch of BASELINE.json's size:
hg_integrate_step = Philox -> RAMBO/Breit-Wigner momenta -> cuts -> |Mbar|^2 -> weight -> (sum w, sum w^2, n_pass);
one fused kernel for configs 1-3, a phase-space kernel and a |M|^2 + reduction kernel per 2^20-event chunk for
configs 4-5; fp64.  Default workload: config 5 (u d~ -> e+ ve g g g, 2^22 events, 2 TeV), the
largest one, which is also the config that asks for the BASES-style accumulation.  `value` counts ALL generated
events per second (events failing the cuts are generated, tested and counted, their matrix element is skipped,
PAPER.md:1168); the pass fraction is reported.  `e2e` is hg_matrix_element_host: momenta in pinned HOST memory ->
H2D -> |Mbar|^2 kernel -> D2H of the per-event results, inside the timed region.  Extra keys give, per config and
precision, the three timings SURVEY.md 8d asks for (matrix element alone on device-resident momenta, fused step,
phase space alone) with their FLOP/s fractions.

--impl reference times the oracle (oracle/, numpy fp64, as it stands) on the host cores over bounded samples.
With N > 1 (torchrun) every rank integrates its own 2^22-event counter range (weak scaling) and the accumulators
are summed with one all-reduce of 4 doubles per step.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = 'helicity+colour-summed |M|^2 events/s on 1 B200; % of FP64/FP32 peak'
UNIT = 'events/s'
SQRT_S = {1: 80.0, 2: 500.0, 3: 1000.0, 4: 1500.0, 5: 2000.0, 6: 500.0, 7: 1000.0, 8: 1000.0, 9: 3000.0, 10: 1000.0,
          11: 1000.0}
N_EVENTS = {1: 1 << 16, 2: 1 << 20, 3: 1 << 22, 4: 1 << 22, 5: 1 << 22, 6: 1 << 20, 7: 1 << 20, 8: 1 << 20, 9: 1 << 20,
            10: 1 << 20, 11: 1 << 20}
NAMES = {1: 'u d~ -> e+ ve', 2: 'u u~ -> e+ e- g', 3: 'u d~ -> e+ ve g g',
         4: 'g g -> t t~ g -> b e+ ve b~ mu- vm~ g', 5: 'u d~ -> e+ ve g g g',
         6: 'u d~ -> e+ ve h', 7: 'u u~ -> e+ e- h h', 8: 'g g -> t t~ h',   # 6-8: Higgs-sector (NEXT-1)
         9: 'u d~ -> e+ ve g g g g',                                          # W + 4 jets (NEXT-4)
         10: 'u d -> h u d', 11: 'u d -> h h u d'}                            # weak-boson fusion (NEXT-1)
SEED = 13050708
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel come from the ncu --set full
# captures summarised in profiles/: profiles/dram_traffic.csv lists (kernel, config, dtype, events per launch, bytes
# read, bytes written, source file); a run whose dominant-kernel launch matches no row reports traffic = null.
def dram_traffic(kernel, cfg, dtype, events_per_launch):
    path = os.path.join(ROOT, 'profiles', 'dram_traffic.csv')
    try:
        with open(path) as f:
            rows = [ln.strip().split(',') for ln in f if ln.strip() and not ln.startswith('#')]
    except OSError:
        return None, 'profiles/dram_traffic.csv not found'
    for r in rows[1:]:
        if r[0] == kernel and int(r[1]) == cfg and r[2] == dtype and int(r[3]) == events_per_launch:
            return int(r[4]) + int(r[5]), r[6]
    return None, 'no ncu capture of %s for config %d %s at %d events per launch' % (kernel, cfg, dtype, events_per_launch)


# nominal non-tensor peaks of B200: 148 SMs x 4 SMSP x 16 lanes x 2 flop x 1.965 GHz for
# FP64 (one DFMA warp instruction per SMSP every 2 cycles) and twice that for FP32
PEAK_NOMINAL_TFLOPS = {'f64': 148 * 64 * 2 * 1.965e9 / 1e12, 'f32': 148 * 128 * 2 * 1.965e9 / 1e12}


def workload_name(cfg, n):
    return 'config %d: %s, %d events, sqrt(s_hat) = %g GeV, Philox->RAMBO, BASELINE.json cuts' % (
        cfg, NAMES[cfg], n, SQRT_S[cfg])


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ('clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,'
         'clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,'
         'clocks_event_reasons.sw_power_cap')

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(['nvidia-smi', '-i', str(self.index), '--query-gpu=' + self.Q,
                                          '--format=csv,noheader,nounits', '-lms', '20'],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def wait_first(self, timeout=5.0):
        """Block until nvidia-smi has delivered its first sample (its start-up can exceed a short timed region)."""
        t0 = time.time()
        while self.proc is not None and not self.rows and time.time() - t0 < timeout:
            time.sleep(0.02)

    def n_between(self, t0, t1):
        return sum(1 for t, _ in self.rows if t0 <= t <= t1)

    def stop(self, t0, t1):
        if self.proc is None:
            return {'sm_mhz': None, 'sm_max_mhz': None, 'reasons': ['nvidia-smi unavailable']}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ('hw_slowdown', 'hw_thermal_slowdown', 'sw_thermal_slowdown', 'sw_power_cap')
        rows = [r for t, r in self.rows if t0 <= t <= t1]
        for r in rows:
            f = [x.strip() for x in r.split(',')]
            try:
                sm.append(float(f[0]))
                smax = float(f[1])
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith('active'):
                    reasons.add(nm)
        return {'sm_mhz': statistics.median(sm) if sm else None, 'sm_max_mhz': smax, 'reasons': sorted(reasons),
                'samples': len(sm)}


# ------------------------------------------------------------------------------------------ oracle timing
ORACLE_SAMPLE = {1: 65536, 2: 8192, 3: 2048, 4: 48, 5: 48, 6: 8192, 7: 4096, 8: 1024, 9: 4, 10: 8192, 11: 2048}   # events per oracle step (about 1-3 s each)


def oracle_step(cfg, first, n, all_cores):
    """One pass of the hot path in the oracle: Philox -> momenta -> cuts -> |Mbar|^2 -> weights -> sums; on one
    thread, or cut into slices over the host cores (oracle/parallel.py: the same functions per slice)."""
    from oracle import integrate as oint
    from oracle import parallel as opar
    from oracle import sm as osm
    if all_cores:
        w, ok = opar.weights(cfg, SEED, first, n, SQRT_S[cfg], osm.default_params(),
                             slice_events=max(1, n // opar.n_workers()))
    else:
        w, ok = oint.weights(cfg, SEED, first, n, SQRT_S[cfg], osm.default_params())
    return oint.accumulate(w, ok)


def time_oracle(cfg, steps, warmup, n=None, all_cores=True):
    """The oracle as it stands on the host: events/s on all cores (worker processes) and on one thread."""
    from oracle import parallel as opar
    cores = opar.n_workers() if all_cores else 1
    n1 = n or ORACLE_SAMPLE[cfg]
    n = n1 * (cores if all_cores else 1)
    for i in range(warmup):
        oracle_step(cfg, i * n, n, all_cores)
    t0 = time.perf_counter()
    for i in range(steps):
        oracle_step(cfg, (warmup + i) * n, n, all_cores)
    wall = time.perf_counter() - t0
    # one thread, one step of the per-core sample
    os.environ.setdefault('OMP_NUM_THREADS', '1')
    t1 = time.perf_counter()
    oracle_step(cfg, 0, n1, False)
    wall1 = time.perf_counter() - t1
    opar.close()
    return {'value': steps * n / wall, 'unit': UNIT, 'cores': cores, 'kind': 'oracle',
            'value_1_process': n1 / wall1,
            'sample': '%d steps of %d events of the same Philox stream (numpy fp64 oracle, all 2^n_ext helicities, '
                      'brute-force colour) cut into slices over %d worker processes; value_1_process = one step of %d '
                      'events in this process; %d host cores present' % (steps, n, cores, n1, os.cpu_count() or 1)}, \
        wall / steps


def time_generated_host(cfg, n_events):
    """The generated matrix elements + phase space compiled for the host (gen/hoststep.cpp, g++ -O3 -fopenmp) on all
    cores: a compiled CPU implementation of the same algorithm, the counterpart of the paper's Fortran HELAS baseline.
    An extra, labelled figure; `cpu_baseline` stays the oracle."""
    import tempfile
    src = os.path.join(ROOT, 'paper_1305_0708_b200', 'gen', 'hoststep.cpp')
    try:
        with tempfile.TemporaryDirectory() as tmp:
            exe = os.path.join(tmp, 'hoststep')
            subprocess.check_call(['g++', '-O3', '-march=native', '-fopenmp', '-std=c++17', src, '-o', exe, '-lm'],
                                  stderr=subprocess.DEVNULL)
            env = {k_: v_ for k_, v_ in os.environ.items() if k_ != 'OMP_NUM_THREADS'}      # all cores
            subprocess.check_output([exe, str(cfg), repr(SQRT_S[cfg]), str(SEED), '0', str(n_events // 8)], env=env)
            out = subprocess.check_output([exe, str(cfg), repr(SQRT_S[cfg]), str(SEED), '0', str(n_events)],
                                          text=True, env=env).split()
            env1 = dict(os.environ, OMP_NUM_THREADS='1')
            out1 = subprocess.check_output([exe, str(cfg), repr(SQRT_S[cfg]), str(SEED), '0', str(n_events // 8)],
                                           text=True, env=env1).split()
    except (OSError, subprocess.CalledProcessError) as e:
        return {'unavailable': 'g++ build or run of gen/hoststep.cpp failed: %r' % (e,)}
    sec, threads = float(out[3]), int(out[4])
    return {'value': n_events / sec, 'unit': UNIT, 'cores': threads, 'kind': 'generated code on the host',
            'value_1_thread': (n_events // 8) / float(out1[3]), 'sum_w_pb': float(out[0]), 'n_pass': float(out[2]),
            'sample': '%d events of the same Philox stream, gen/hoststep.cpp built with g++ -O3 -march=native -fopenmp '
                      '(fp64; shared sub-currents, non-zero helicities only, colour-flow basis: the algorithm of the '
                      'kernels, on CPU cores)' % n_events}


def run_reference(args):
    rank = int(os.environ.get('RANK', '0'))
    if rank != 0:
        return
    cfg = args.config
    base, sec = time_oracle(cfg, args.steps, args.warmup)
    line = {'impl': 'reference', 'metric': METRIC, 'value': base['value'], 'unit': UNIT, 'n_gpus': args.gpus,
            'steps': args.steps, 'warmup': args.warmup, 'ms_per_step': sec * 1e3, 'higher_is_better': True,
            'scaling': 'weak', 'vs_baseline': None, 'dtype': 'f64', 'data': 'synthetic',
            'config': {'workload': workload_name(cfg, N_EVENTS[cfg]),
                       'sample_per_step': ORACLE_SAMPLE[cfg] * base['cores']},
            'cpu_baseline': base,
            'e2e': {'value': base['value'], 'unit': UNIT, 'h2d_bytes_per_step': 0, 'd2h_bytes_per_step': 0},
            'gpu_launches': 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------ GPU arm
def _events_ms(torch, fn, reps):
    """CUDA-event time of each of `reps` calls of fn on the current stream (the stream the library launches on)."""
    out = []
    for _ in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        b.synchronize()
        out.append(a.elapsed_time(b))
    return out


def measure_config(torch, api, ctx, cfg, prec, n, reps, peaks):
    """The three timings of SURVEY.md 8d for one config and precision (median of reps after 3 warm-up calls)."""
    info = api.hg_process_info(cfg)
    rs = SQRT_S[cfg]
    pname = 'f64' if prec == api.HG_F64 else 'f32'
    p, wps, ok = ctx.hg_gen_phase_space(cfg, prec, SEED, 0, n, rs)
    me = torch.empty((n,), dtype=p.dtype, device=p.device)
    res = {}
    fns = {'matrix_element': lambda: ctx.hg_matrix_element(cfg, prec, p, me),
           'integrate_step': lambda: ctx.hg_integrate_step(cfg, prec, SEED, 0, n, rs),
           'gen_phase_space': lambda: ctx.hg_gen_phase_space(cfg, prec, SEED, 0, n, rs, p, wps, ok)}
    acc = ctx.hg_integrate_step(cfg, prec, SEED, 0, n, rs)
    pass_frac = acc[3] / acc[2]
    for name, fn in fns.items():
        for _ in range(3):
            fn()
        ms = statistics.median(_events_ms(torch, fn, reps))
        flops = {'matrix_element': info['flops_f64'] * n,
                 'integrate_step': info['flops_f64'] * acc[3] + info['flops_ps'] * n,
                 'gen_phase_space': info['flops_ps'] * n}[name]
        r = {'ms': ms, 'events_per_s': n / (ms * 1e-3), 'tflops': flops / (ms * 1e-3) / 1e12}
        # the matrix element computes in `prec`; the phase space is always fp64
        pk = 'f64' if name == 'gen_phase_space' else pname
        r['frac_of_nominal_peak'] = r['tflops'] / PEAK_NOMINAL_TFLOPS[pk]
        r['frac_of_measured_fma_peak'] = r['tflops'] / peaks[pk]
        if name == 'matrix_element':
            el = 8 if prec == api.HG_F64 else 4
            r['hbm_gbs'] = n * (4 * info['n_ext'] + 1) * el / (ms * 1e-3) / 1e9
        res[name] = r
    res['pass_fraction'] = pass_frac
    res['flops_per_event'] = info['flops_f64']
    res['n'] = n
    del p, wps, ok, me
    return res


def _sig(acc):
    s = acc[0] / acc[2]
    return s, (max(acc[1] / acc[2] - s * s, 0.0) / max(acc[2] - 1.0, 1.0)) ** 0.5


def measure_paper_phase_space(torch, api, ctx, cfg, n, reps):
    """the step in the paper's own phase space (hadronic sqrt(s) = 14 TeV, toy parton
    densities, A23), flat and after a BASES-style grid optimisation (5 iterations of n points, A22):
    events/s, pass fraction and relative Monte-Carlo error per step, beside flat RAMBO at fixed s_hat."""
    import numpy as np
    rs_had, nb, alpha, iters = 14000.0, 50, 1.0, 5
    nd = api.hg_process_info(cfg)['n_draws']
    prec = api.HG_F64
    out = {}

    def timed(fn):
        for _ in range(2):
            fn()
        return statistics.median(_events_ms(torch, fn, reps))

    acc = ctx.hg_integrate_step(cfg, prec, SEED, 0, n, SQRT_S[cfg])
    s, e = _sig(acc)
    out['rambo_fixed_shat'] = {'pass_fraction': acc[3] / acc[2], 'rel_error': e / s, 'sigma_pb': s}
    try:
        ctx.hg_set_hadronic(api.hg_default_hadronic(cfg))
        acc = ctx.hg_integrate_step(cfg, prec, SEED, 0, n, rs_had)
        ms = timed(lambda: ctx.hg_integrate_step(cfg, prec, SEED, 0, n, rs_had))
        s, e = _sig(acc)
        out['paper_flat'] = {'ms': ms, 'events_per_s': n / (ms * 1e-3), 'pass_fraction': acc[3] / acc[2],
                             'rel_error': e / s, 'sigma_pb': s}
        grid = torch.from_numpy(np.tile(np.linspace(0.0, 1.0, nb + 1), (nd, 1))).contiguous()
        t_opt = []
        for it in range(iters):
            d_grid = grid.cuda()
            d_hist = torch.zeros((nd, nb), dtype=torch.float64, device='cuda')
            ctx.hg_set_grid(d_grid, d_hist)
            t_opt += _events_ms(torch, lambda: ctx.hg_integrate_step(cfg, prec, SEED, (it + 1) * n, n, rs_had), 1)
            api.hg_grid_refine(d_hist.cpu(), alpha, grid)
        d_grid = grid.cuda()
        ctx.hg_set_grid(d_grid, None)
        acc = ctx.hg_integrate_step(cfg, prec, SEED, (iters + 2) * n, n, rs_had)
        ms = timed(lambda: ctx.hg_integrate_step(cfg, prec, SEED, (iters + 2) * n, n, rs_had))
        s, e = _sig(acc)
        out['paper_adapted'] = {'ms': ms, 'events_per_s': n / (ms * 1e-3), 'pass_fraction': acc[3] / acc[2],
                                'rel_error': e / s, 'sigma_pb': s, 'grid_optimisation_ms_per_iteration':
                                statistics.median(t_opt), 'iterations': iters, 'bins': nb, 'alpha': alpha}
        out['error_reduction_by_grid'] = out['paper_flat']['rel_error'] / out['paper_adapted']['rel_error']
    finally:
        ctx.hg_set_grid(None)
        ctx.hg_set_hadronic(None)
    out['n'] = n
    return out


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_1305_0708_b200 import api, shard

    rank = int(os.environ.get('RANK', '0'))
    world = int(os.environ.get('WORLD_SIZE', '1'))
    local = int(os.environ.get('LOCAL_RANK', '0'))
    if not torch.cuda.is_available():
        raise SystemExit('bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle')
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group('nccl', device_id=torch.device('cuda', local))
    ctx = api.Context(local)
    ctx.hg_set_profiling(True)
    cfg, rs = args.config, SQRT_S[args.config]
    n = args.events or N_EVENTS[cfg]
    info = api.hg_process_info(cfg)
    prec = api.HG_F64 if args.dtype == 'f64' else api.HG_F32
    first = rank * n                                  # weak scaling: every rank its own n-event counter range
    dev = torch.device('cuda', local)

    def step():
        acc = ctx.hg_integrate_step(cfg, prec, SEED, first, n, rs)
        return shard.combine_acc(acc, device=dev) if world > 1 else acc

    def sync():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        acc = step()
    sampler = ClockSampler(local)
    sampler.start()
    sampler.wait_first()
    sync()
    t0 = time.time()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    per_step = []
    ps_ms = me_ms = 0.0
    launches = 0
    for _ in range(args.steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        acc = step()
        b.record()
        per_step.append((a, b))
        t_ps, t_me, nl = ctx.hg_last_step_info()   # CUDA events recorded by the library around its kernels
        ps_ms += t_ps
        me_ms += t_me
        launches += nl
    e1.record()
    sync()
    t1 = time.time()
    total_ms = e0.elapsed_time(e1)
    kern_ms = statistics.mean(a.elapsed_time(b) for a, b in per_step)
    # K steps of a few ms can be shorter than a handful of 20 ms samples: keep the same load running (untimed) until the
    # sampler has seen at least 5 samples under it, and say how many fell inside the timed region itself
    in_region = sampler.n_between(t0, t1)
    t_load = t1
    while sampler.proc is not None and sampler.n_between(t0, t_load) < 5 and time.time() - t1 < 3.0:
        step()
        torch.cuda.synchronize()
        t_load = time.time()
    clocks = sampler.stop(t0, t_load)
    clocks['samples_in_timed_region'] = in_region
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = t.item()
    ms_per_step = total_ms / args.steps
    value = world * n / (ms_per_step * 1e-3)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- rank 0: end-to-end leg, per-config table, peaks, oracle baseline
    peaks = {'f64': ctx.hg_measure_fma_peak(api.HG_F64) / 1e12, 'f32': ctx.hg_measure_fma_peak(api.HG_F32) / 1e12}
    pname = args.dtype
    el = 8 if prec == api.HG_F64 else 4
    p, _, _ = ctx.hg_gen_phase_space(cfg, prec, SEED, first, n, rs, want_pass=False)
    pf = p[2:].contiguous()                      # the events are in the partonic CM frame: ship the final-state legs
    hp = torch.empty(pf.shape, dtype=p.dtype).pin_memory()
    hp.copy_(pf)
    hme = torch.empty((n,), dtype=p.dtype).pin_memory()
    del p, pf
    for _ in range(3):
        ctx.hg_matrix_element_host_cm(cfg, prec, rs, hp, hme)
    e2e_ms = statistics.mean(_events_ms(torch, lambda: ctx.hg_matrix_element_host_cm(cfg, prec, rs, hp, hme),
                                        args.steps))
    e2e = {'value': n / (e2e_ms * 1e-3), 'unit': UNIT, 'h2d_bytes_per_step': hp.numel() * el,
           'd2h_bytes_per_step': hme.numel() * el,
           'what': 'hg_matrix_element_host_cm: pinned host momenta of the final-state legs (the incoming ones follow '
                   'from sqrt(s_hat)) -> H2D -> |Mbar|^2 kernel -> D2H per step, pipelined in 2^19-event chunks (copy of '
                   'chunk i+1 overlaps the kernel of chunk i)'}
    del hp, hme

    n_pass = acc[3] / world if world > 1 else acc[3]
    staged = ps_ms > 0.0          # two-kernel step (configs 4, 5): the dominant kernel is me_acc_kernel
    n_chunks = max(1, (launches // args.steps - 1) // 3) if staged else 1
    me_ms_step = me_ms / args.steps                      # all launches of the dominant kernel in one step
    flops_kernel = info['flops_f64'] * n_pass + (0.0 if staged else info['flops_ps'] * n)
    achieved = flops_kernel / (me_ms_step * 1e-3) / 1e12
    tname = 'double' if pname == 'f64' else 'float'
    kname = 'me_acc_kernel' if staged else 'integrate_kernel'
    traffic, traffic_src = dram_traffic(kname, cfg, pname, min(n, 1 << 20) if staged else n)
    roofline = {'bound': 'alu',
                'kernel': ('me_acc_kernel<P%d,%s>' if staged else 'integrate_kernel<P%d,%s>') % (cfg, tname),
                'achieved': achieved, 'peak': PEAK_NOMINAL_TFLOPS[pname], 'unit': 'TFLOP/s',
                'frac': achieved / PEAK_NOMINAL_TFLOPS[pname], 'traffic': traffic, 'traffic_source': traffic_src,
                'peak_kind': 'nominal non-tensor %s peak (148 SM x %d lanes x 2 x 1.965 GHz, DESIGN.md); '
                             'MEASURED_PEAKS.json has no ALU figure' % (pname, 64 if pname == 'f64' else 128),
                'peak_measured_fma_chain': peaks[pname], 'frac_of_measured_fma_chain': achieved / peaks[pname],
                'launches_per_step': n_chunks, 'algorithmic_flops_per_launch': flops_kernel / n_chunks,
                'launch_ms': me_ms_step / n_chunks, 'kernel_ms_per_step': me_ms_step,
                'phase_space_ms_per_step': ps_ms / args.steps, 'share_of_step': me_ms_step / kern_ms,
                'flops_per_event': info['flops_f64']}

    per_config = {}
    if not args.no_table:
        for c in (1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11):
            for pr, nm in ((api.HG_F64, 'f64'), (api.HG_F32, 'f32')):
                per_config['cfg%d_%s' % (c, nm)] = measure_config(torch, api, ctx, c, pr, N_EVENTS[c], 7, peaks)
        per_config['cfg1_f64_4M'] = measure_config(torch, api, ctx, 1, api.HG_F64, 1 << 22, 7, peaks)
        per_config['cfg1_f32_4M'] = measure_config(torch, api, ctx, 1, api.HG_F32, 1 << 22, 7, peaks)

    paper_ps = None if args.no_table else measure_paper_phase_space(torch, api, ctx, cfg, n, 5)
    cpu_base, _ = time_oracle(cfg, 4, 1)
    cpu_gen = time_generated_host(cfg, {9: 1 << 14}.get(cfg, 1 << 19))
    s = acc[0] / acc[2]
    ds = (max(acc[1] / acc[2] - s * s, 0.0) / max(acc[2] - 1.0, 1.0)) ** 0.5
    line = {'metric': METRIC, 'value': value, 'unit': UNIT, 'n_gpus': world, 'steps': args.steps,
            'warmup': max(args.warmup, 3), 'ms_per_step': ms_per_step, 'higher_is_better': True, 'scaling': 'weak',
            'vs_baseline': None, 'dtype': pname, 'data': 'synthetic',
            'config': {'workload': workload_name(cfg, n), 'events_per_gpu': n,
                       'step': 'hg_integrate_step: Philox -> RAMBO -> cuts -> |M|^2 -> weight -> sums; ' + (
                           'per chunk of 2^20 events a phase-space kernel and a |M|^2 + reduction kernel' if staged
                           else 'one fused kernel'),
                       'l2': 'every step regenerates its events; the chunk buffer (%d MB) and the e2e / matrix_element '
                             'inputs (%d MB) exceed the 126 MB L2' % (
                                 min(n, 1 << 20) * (4 * info['n_ext'] * el + 9) >> 20, n * 4 * info['n_ext'] * el >> 20),
                       'pass_fraction': acc[3] / acc[2], 'sigma_pb': s, 'sigma_err_pb': ds},
            'clocks': clocks, 'e2e': e2e, 'gpu_launches': launches, 'roofline': roofline,
            'cpu_baseline': cpu_base, 'fma_peak_measured_tflops': peaks, 'per_config': per_config,
            'paper_phase_space': paper_ps, 'cpu_generated_code': cpu_gen}
    print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument('--gpus', type=int, default=1)
    ap.add_argument('--steps', type=int, default=20)
    ap.add_argument('--warmup', type=int, default=3)
    ap.add_argument('--config', type=int, default=5, choices=[1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11])
    ap.add_argument('--dtype', default='f64', choices=['f64', 'f32'])
    ap.add_argument('--events', type=int, default=0, help='events per GPU per step (default: BASELINE.json size)')
    ap.add_argument('--impl', default='graft', choices=['graft', 'reference'])
    ap.add_argument('--no-table', action='store_true', help='skip the per-config table')
    args = ap.parse_args()
    if args.impl == 'reference':
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == '__main__':
    main()
