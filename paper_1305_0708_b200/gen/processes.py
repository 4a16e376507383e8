"""The five processes of BASELINE.json (workloads of PAPER.md:147-256) and the generator driver.

`python -m paper_1305_0708_b200.gen` writes csrc/generated/me2_<name>.cuh for every process and
csrc/generated/hg_processes.inc (the table the C-ABI layer includes).
"""
import os

from .diagrams import Diagrams, ProcessSpec
from .emit import CodeGen

# Leg order = include/hg.h.  Decay groups (reading A13): legs that must come from one resonance.
SPECS = [
    ProcessSpec('udx_epve', 1, ['u', 'd~'], ['e+', 've']),
    ProcessSpec('uux_epemg', 2, ['u', 'u~'], ['e+', 'e-', 'g']),
    ProcessSpec('udx_epvegg', 3, ['u', 'd~'], ['e+', 've', 'g', 'g']),
    ProcessSpec('gg_ttxg_dilep', 4, ['g', 'g'], ['b', 'e+', 've', 'b~', 'mu-', 'vm~', 'g'],
                decays=[('t', (2, 3, 4)), ('w+', (3, 4)), ('t', (5, 6, 7)), ('w+', (6, 7))]),
    ProcessSpec('udx_epveggg', 5, ['u', 'd~'], ['e+', 've', 'g', 'g', 'g']),
    # Higgs-sector processes: VVS; VVS + VVSS + SSS; FFS with massive external fermions
    ProcessSpec('udx_epveh', 6, ['u', 'd~'], ['e+', 've', 'h']),
    ProcessSpec('uux_epemhh', 7, ['u', 'u~'], ['e+', 'e-', 'h', 'h']),
    ProcessSpec('gg_ttxh', 8, ['g', 'g'], ['t', 't~', 'h']),
    # next size up: W + 4 jets, 428 diagrams / 516 amplitudes, 24 colour flows
    ProcessSpec('udx_epvegggg', 9, ['u', 'd~'], ['e+', 've', 'g', 'g', 'g', 'g']),
    # weak-boson fusion, two quark lines (Eq. 21a, 22a): W W and Z Z
    # fusion interfere (different colour flows, relative Fermi sign); VVS, and VVS + VVSS + SSS
    ProcessSpec('ud_hud', 10, ['u', 'd'], ['h', 'u', 'd']),
    ProcessSpec('ud_hhud', 11, ['u', 'd'], ['h', 'h', 'u', 'd']),
]

# resonance of the W/Z + jets family in the paper's hadronic phase space: suffix of PsConst::m?, mg?, tmax_?
HADRONIC = {1: 'w', 2: 'z', 3: 'w', 5: 'w', 9: 'w'}

# uniform random numbers per event used by the phase-space generator
N_DRAWS = {1: 8, 2: 12, 3: 16, 4: 24, 5: 20, 6: 12, 7: 16, 8: 12, 9: 24, 10: 12, 11: 16}

# rough per-call cost (flops) used only to choose the closing leg; the reported flop counts are measured by
# running the generated code on a counting type (gen/flopcount.py)
_COST = {'FFV': 70, 'VVV': 150, 'VVVV': 90}


def _estimate(cg):
    """Estimated flops per event = sum over emitted values of cost x loop multiplicity."""
    mult = [1]
    for l in cg.dynamic:
        mult.append(mult[-1] * len(cg.nhel[l]))
    depth_of = {l: i + 1 for i, l in enumerate(cg.dynamic)}
    total = 0
    for hel, roots in cg.variants:
        seen = set()

        def visit(nd):
            nonlocal total
            if nd.uid in seen or nd.is_leaf:
                return
            seen.add(nd.uid)
            for ch in nd.children:
                visit(ch)
            d = max([depth_of.get(l, 0) for l in range(cg.dg.n) if nd.mask >> l & 1])
            cost = 8 if nd.is_sum else _COST.get(nd.vertex.kind, 100)
            total += cost * mult[d] * (2 if nd.particle.mass and nd.particle.spin == 'F' else 1)

        for r in roots:
            for ch in r.children:
                visit(ch)
            total += _COST.get(r.vertex.kind, 100) * mult[-1]
    return total


# processes whose loop-crossing values are kept in the shared-memory staging area (csrc/hg_stage.cuh).
# Measured for W + 2 jets too: staged 0.88 ms against 0.66 ms unstaged for 2^22 events -- small processes stay
# in registers.
STAGED = {4, 5, 9}
# unstaged processes whose step is nevertheless run as separate kernels: the phase-space code runs at full occupancy
# instead of inside a 250-register kernel (measured per 2^22 events, fp64: config 2 1.13 -> 1.05 ms, Z H H
# 1.95 -> 1.48 ms, t t~ H 4.04 -> 3.79 ms; W + 2 jets 1.17 -> 1.16 ms in fp64 but 0.82 -> 0.88 ms in fp32, so
# it stays fused, like the tiny matrix elements of configs 1 and 6)
SPLIT_STEP = {2, 7, 8}
# add currents with the same legs, field and colour structure before use (gen/diagrams.py)
MERGE = True
# of those, processes that rebuild internal momenta from staged external momenta inside the loops (fewer slots,
# more shared-memory loads)
KFROMP = set()
# processes whose FFV closings do NOT go through dressed spinors (gen/emit.py DRESS): config 4 would need 174 staged
# words instead of 142 and fall from 12 to 8 warps per SM
NO_DRESS = {4}
# staged processes whose staging area lives in GLOBAL memory (csrc/hg_stage.cuh GmemStage).  Measured for W + 4 jets
# (738 words per event: one pair of warps per SM in shared memory): 8 warps per SM through L2 are SLOWER than 2 warps
# through shared memory, 34.9 ms against 26.5 ms per 2^18 events in fp64, 27.2 against 12.9 ms in fp32, whether the
# 8 warps sit in one block or four (profiles/r02_notes.md): the option stays off.
STAGE_GLOBAL = set()
# staged processes evaluated by a TEAM of four warps per 32 events: the closings of the innermost loop body are dealt
# to two groups of warps (gen/emit.py groups).  W + 4 jets keeps 711 words per event, i.e. one pair of warps per SM in
# fp64 with two of the four schedulers idle; the second set of accumulators (+192 words) still fits
# (measured for config 5 too: three teams = 12 warps per SM at 168 registers with the accumulators in the staging area,
# 9.8 % duplicated sub-currents: |M|^2 of 2^22 events 4.67 -> 7.97 ms in fp64, 2.66 -> 5.29 ms in fp32 -- pairs stay)
GROUPS = {9: 2}
# staged processes whose innermost loop body calls one real function per shape of vertex call instead of inlining
# the arithmetic of every call (gen/emit.py opcalls).  Measured on B200, |M|^2 of 2^22 events (2^18 for W + 4 jets):
#   W + 4 jets  fp64 18.59 -> 14.56 ms, fp32 9.02 -> 6.13 ms   (4 warps per SM in fp64: nothing else hides the fetch)
#   config 5    fp64  4.60 ->  5.83 ms, fp32 2.66 -> 3.40 ms   (8-12 warps per SM hide it; the calls only cost)
#   config 4    fp64  4.43 ->  5.02 ms, fp32 2.71 -> 3.20 ms
OPCALLS = {9}
# staged processes whose fp64 rendezvous is a named barrier per pair instead of __syncthreads().  bench.py, B200,
# 2^22 events, step / dominant kernel per 2^20 events: config 5 fp64 5.097 -> 4.978 ms / 1.077 -> 1.047 ms, config 4
# fp64 5.662 -> 5.539 ms / 1.125 -> 1.100 ms; in fp32 the named barrier is SLOWER (config 5 3.274 -> 3.334 ms,
# config 4 3.943 -> 4.081 ms), so fp32 keeps __syncthreads (hg_process_impl.cuh me2_event); W + 4 jets: no difference
NAMED_BARRIER = {4, 5}
# staged processes whose fp32 staging area keeps the words of an event two by two (csrc/hg_stage.cuh PAIRS), with every
# value of two or more words at an even slot (gen/emit.py align_pairs): a complex number is one 8-byte shared-memory
# access.  Not W + 4 jets: its 903 words fill the SM exactly, the padding would cost a team.  bench.py, B200, fp32,
# dominant kernel per 2^20-event launch: config 5 0.6233 -> 0.6088 ms (LDS + STS 17 % -> 9 % of the instructions of
# an issue-bound kernel), config 4 0.7000 -> 0.7530 ms (slower: stays with single words)
STAGE_PAIRS = {5}


def build(spec, last=None):
    """Enumerate the diagrams of `spec` closing on leg `last` (default: the leg with the lowest estimated cost)."""
    stage = spec.pid in STAGED
    if last is None:
        last = spec.last
    def make(leg):
        cg_ = CodeGen(Diagrams(spec, merge=MERGE).build(leg), stage, spec.pid in KFROMP,
                      dress=spec.pid not in NO_DRESS, groups=GROUPS.get(spec.pid, 1), opcalls=spec.pid in OPCALLS,
                      align_pairs=spec.pid in STAGE_PAIRS)
        cg_.count_dg = Diagrams(spec).build(leg)   # Feynman-diagram counts: the unmerged enumeration
        return cg_

    if last is not None and last >= 0:
        return make(last)
    best = None
    for cand in range(len(spec.initial) + len(spec.final)):
        cg = make(cand)
        if stage:
            try:
                cg.generate()       # staged mode needs a two-state innermost loop: not every closing leg has one
            except NotImplementedError:
                continue
        est = _estimate(cg)
        if best is None or est < best[0]:
            best = (est, cg)
    return best[1]


def render(cg):
    spec = cg.dg.spec
    lines = cg.generate()
    flows, cmat, cden = cg.colour_matrix()
    head = [
        '// GENERATED by paper_1305_0708_b200/gen (python -m paper_1305_0708_b200.gen) -- do not edit.',
        '// process %d: %s -> %s' % (spec.pid, ' '.join(spec.initial), ' '.join(spec.final)),
        '// closing leg %d; %d topological diagrams, %d amplitudes, %d colour flows %s;' % (
            cg.dg.last, cg.count_dg.n_topological(), cg.count_dg.n_amplitudes(), len(flows), flows),
        '// helicity combinations: %d of %d are not identically zero; colour matrix = (1/%d) x %s' % (
            cg.n_hel_nonzero, cg.n_hel_total, cden, cmat),
        '#pragma once',
        '#include "../hg_helas.cuh"',
        '#include "../hg_params.cuh"',
        '#include "../hg_stage.cuh"',
        'namespace hg {',
    ] + list(cg.prelude) + [
        'template <class T, class St>',
        'HG_HD T me2_%s(const Mom<T>* p, const Coup<T>& c, const St& st) {' % spec.name,
    ]
    return '\n'.join(head + lines + ['}', '}  // namespace hg', ''])


def info_row(cg):
    spec = cg.dg.spec
    flows, cmat, cden = cg.colour_matrix()
    return dict(pid=spec.pid, name=spec.name, n_ext=cg.dg.n, n_final=len(spec.final), n_hel_total=cg.n_hel_total,
                n_hel_nonzero=cg.n_hel_nonzero, n_diagrams=cg.count_dg.n_topological(), n_amplitudes=cg.count_dg.n_amplitudes(),
                n_flows=len(flows), n_draws=N_DRAWS[spec.pid], avg_factor=float(cg.avg_factor()))


def generated_dir():
    return os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), 'csrc', 'generated')


# legs the cuts look at (scope: SURVEY.md 8c-A11/A12): gluon jets, charged leptons
def _cut_legs(spec):
    names = spec.initial + spec.final
    n_in = len(spec.initial)
    jets = [i for i, nm in enumerate(names) if i >= n_in and nm == 'g']
    leps = [i for i, nm in enumerate(names) if i >= n_in and nm in ('e+', 'e-', 'mu+', 'mu-')]
    return jets, leps


def _ps_flops(spec):
    """Operation count of phase-space generation + cuts (add, mul = 1; div, sqrt, log, sincos, tan, atan2,
    asinh = 1 each), from the formulas of csrc/hg_phase_space.cuh; an estimate (Philox is integer work)."""
    n = 3 if spec.decays else len(spec.final)
    f = 49 * n + 17
    if spec.decays:
        f += 4 * 12 + 12 * (3 * 7 + 2) + 3 * 9 + 10 + 4 * (2 * 22 + 30)
    jets, leps = _cut_legs(spec)
    f += 10 * len(jets) + 7 * len(leps) + 25 * (len(jets) * (len(jets) - 1) // 2)
    return float(f)


def render_descriptor(cg):
    """generated/hg_proc_<pid>.cuh: the static description of the process used by csrc/hg_process_impl.cuh."""
    spec = cg.dg.spec
    row = info_row(cg)
    jets, leps = _cut_legs(spec)
    arr = lambda xs: ', '.join(str(x) for x in (xs or [-1]))
    n_rambo = 3 if spec.decays else len(spec.final)
    from .model import PARTICLES
    fmass = [PARTICLES[nm].mass for nm in spec.final]
    if spec.decays:
        gen_call = 'gen_ttxg_dilep<GRID>(k, seed, event, %d, p, bins)' % spec.pid
    elif any(fmass):
        # massive final-state particles: massive RAMBO with the masses taken from the call's constants
        gen_call = 'gen_massive<%d, GRID>(k, seed, event, %d, {%s}, p, bins)' % (
            len(spec.final), spec.pid, ', '.join('k.%s' % m if m else '0.0' for m in fmass))
    else:
        gen_call = 'gen_massless<%d, GRID>(k, seed, event, %d, p, bins)' % (len(spec.final), spec.pid)
    # the paper's hadronic phase space (hg_set_hadronic, reading A23): W/Z + jets family and config 4
    res = HADRONIC.get(spec.pid)
    if spec.decays:
        had_call = 'gen_had_ttxg_dilep<GRID>(k, seed, event, %d, p, bins)' % spec.pid
    elif res:
        had_call = 'gen_had_vjets<%d, %d, GRID>(k, seed, event, %d, k.m%s, k.mg%s, k.tmax_%s, p, bins)' % (
            len(jets), N_DRAWS[spec.pid], spec.pid, res, res, res)
    else:
        had_call = None
    return """// GENERATED by paper_1305_0708_b200/gen (python -m paper_1305_0708_b200.gen) -- do not edit.
// process %(pid)d: %(proc)s
#pragma once
#include "../hg_phase_space.cuh"
#include "me2_%(name)s.cuh"
namespace hg {
struct P%(pid)d {
  static constexpr int pid = %(pid)d, n_ext = %(n_ext)d, n_final = %(n_final)d, n_rambo = %(n_rambo)d;
  static constexpr int n_hel_total = %(n_hel_total)d, n_hel_nonzero = %(n_hel_nonzero)d;
  static constexpr int n_diagrams = %(n_diagrams)d, n_amplitudes = %(n_amplitudes)d, n_flows = %(n_flows)d;
  static constexpr int n_draws = %(n_draws)d;
  static constexpr int n_stage = %(n_stage)d;  // words per event of the staging area (0: not staged)
  static constexpr bool stage_global = %(stage_global)s;  // the staging area is global memory, not shared
  static constexpr int n_split = %(n_split)d;  // warps that share an event of a staged process: pair, or team of four
  static constexpr bool named_barrier = %(named_barrier)s;  // rendezvous per pair / team, not per block (hg_stage.cuh)
  static constexpr bool stage_pairs = %(stage_pairs)s;  // fp32: staged words two by two, complex numbers in one access
  // hg_integrate_step as phase-space kernel + compaction + |M|^2 kernel per chunk (true) or one fused kernel
  static constexpr bool split_step = %(split_step)s;
  static constexpr double avg_factor = %(avg)s;
  static constexpr int me_threads = %(me_threads)d;
  static constexpr int n_jets = %(n_jets)d, n_leps = %(n_leps)d;
  HG_HD static constexpr int jet(int i) {
    constexpr int t[] = {%(jets)s};
    return t[i];
  }
  HG_HD static constexpr int lep(int i) {
    constexpr int t[] = {%(leps)s};
    return t[i];
  }
  // GRID: sample through the adaptive grid k.grid; bins (or NULL) then receives the grid bin of every draw
  // HAD: the paper's hadronic phase space (k.rs = hadronic sqrt(s)) instead of RAMBO at fixed s_hat
  static constexpr bool has_hadronic = %(has_had)s;
  template <bool GRID = false, bool HAD = false>
  HG_HD static double gen(const PsConst& k, uint64_t seed, uint64_t event, Mom<double>* p, uint8_t* bins = nullptr) {
    if constexpr (HAD) {
      %(had_call)s
    } else {
      return %(gen_call)s;
    }
  }
  template <class T, class St>
  HG_HD static T me2(const Mom<T>* p, const Coup<T>& c, const St& st) {
    return me2_%(name)s<T>(p, c, st);
  }
};
}  // namespace hg
""" % dict(pid=spec.pid, proc='%s -> %s' % (' '.join(spec.initial), ' '.join(spec.final)), name=spec.name,
           n_ext=row['n_ext'], n_final=row['n_final'], n_rambo=n_rambo, n_hel_total=row['n_hel_total'],
           n_hel_nonzero=row['n_hel_nonzero'], n_diagrams=row['n_diagrams'], n_amplitudes=row['n_amplitudes'],
           n_flows=row['n_flows'], n_draws=row['n_draws'], n_stage=cg.n_stage,
           stage_global='true' if spec.pid in STAGE_GLOBAL else 'false',
           n_split=2 * GROUPS.get(spec.pid, 1),
           named_barrier='true' if spec.pid in NAMED_BARRIER else 'false',
           stage_pairs='true' if spec.pid in STAGE_PAIRS else 'false',
           split_step='true' if (cg.n_stage > 0 or spec.pid in SPLIT_STEP) else 'false', avg=repr(row['avg_factor']),
           me_threads=ME_THREADS.get(spec.pid, 128), n_jets=len(jets), n_leps=len(leps), jets=arr(jets),
           leps=arr(leps), gen_call=gen_call, has_had='true' if had_call else 'false',
           had_call=('return %s;' % had_call) if had_call else 'return 0.0;  // not implemented: rejected by the C ABI')


def render_unit(spec, flops_me, flops_ps):
    """generated/hg_proc_<pid>.cu: one translation unit per process (they compile in parallel)."""
    return """// GENERATED by paper_1305_0708_b200/gen (python -m paper_1305_0708_b200.gen) -- do not edit.
#include "hg_proc_%(pid)d.cuh"
#include "../hg_process_impl.cuh"
namespace hg {
// flops per event: matrix element counted by gen/flopcount.cpp on the counting type; phase space estimated
extern const ProcVTable hg_proc_%(pid)d = make_vtable<P%(pid)d>(%(fme)r, %(fps)r);
}  // namespace hg
""" % dict(pid=spec.pid, fme=float(flops_me), fps=float(flops_ps))


# threads per block of the matrix-element kernel (tuned with ncu)
ME_THREADS = {1: 256, 2: 128, 3: 128, 4: 128, 5: 128, 6: 128, 7: 128, 8: 128, 9: 128, 10: 128, 11: 128}


def count_flops(outdir):
    """Compile gen/flopcount.cpp against the freshly generated headers with g++ and run it."""
    import subprocess
    import tempfile
    here = os.path.dirname(os.path.abspath(__file__))
    with tempfile.TemporaryDirectory() as tmp:
        exe = os.path.join(tmp, 'flopcount')
        subprocess.check_call(['g++', '-O1', '-std=c++17', '-x', 'c++', os.path.join(here, 'flopcount.cpp'),
                               '-o', exe, '-lm'])
        out = subprocess.check_output([exe], text=True)
    res = {}
    for line in out.strip().splitlines():
        f = line.split()
        res[int(f[0])] = dict(min=int(f[1]), mean=float(f[2]), max=int(f[3]), me2_double=float(f[4]),
                              me2_counted=float(f[5]))
    return res


def write_all(outdir=None):
    outdir = outdir or generated_dir()
    os.makedirs(outdir, exist_ok=True)
    rows, cgs = [], []
    for spec in SPECS:
        cg = build(spec)
        with open(os.path.join(outdir, 'me2_%s.cuh' % spec.name), 'w') as f:
            f.write(render(cg))
        with open(os.path.join(outdir, 'hg_proc_%d.cuh' % spec.pid), 'w') as f:
            f.write(render_descriptor(cg))
        rows.append(info_row(cg))
        cgs.append(cg)
    flops = count_flops(outdir)
    for spec, row in zip(SPECS, rows):
        row['flops_me'] = flops[spec.pid]['mean']
        row['flops_me_range'] = (flops[spec.pid]['min'], flops[spec.pid]['max'])
        row['flops_ps'] = _ps_flops(spec)
        with open(os.path.join(outdir, 'hg_proc_%d.cu' % spec.pid), 'w') as f:
            f.write(render_unit(spec, row['flops_me'], row['flops_ps']))
    return rows
