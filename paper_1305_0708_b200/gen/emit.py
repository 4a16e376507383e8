"""CUDA emitter: diagram list -> one fused per-process device function (steps a5-a8).

Role of MG2CUDA's output stage (section 5.1, 5.4, 5.5), re-designed:
  * helicity combinations that vanish identically are found at generation time by propagating chirality masks
    through the diagrams (massless fermions keep one Weyl half; W couples to the left half only) and are never
    evaluated;
  * helicities of massless fermions are unrolled at generation time (they change the sparsity of the code),
    helicities of gluons / massive particles are run-time loops, nested so that a sub-current is evaluated at the
    loop depth of the deepest leg it depends on (values that depend on no looped leg are computed once);
  * momenta of internal lines, their invariants and the propagator factors are helicity independent and are
    computed once per event, before the helicity loops; invariants of massless pairs are formed from unit vectors
    so that fp32 does not cancel for collinear pairs;
  * amplitudes are added into colour-flow partial amplitudes jamp[f] with integer coefficients, and the colour
    matrix (integers over a common denominator) is contracted per helicity combination.
The paper's temporary-variable recycling is left to nvcc's register allocator: values are
emitted in SSA form inside the loop scope where they live.
"""
import itertools
import re
from fractions import Fraction
from math import factorial, gcd

from . import colour as C
from .diagrams import Diagrams, bits
from .model import PARTICLES

A, B, AB = 1, 2, 3
GL, GR = 1, 2


def _lcm(a, b):
    return a * b // gcd(a, b)


class Emitter:
    def __init__(self, diag: Diagrams):
        self.dg = diag
        self.legs = diag.legs
        self.static = [l.index for l in self.legs if l.particle.spin == 'F' and not l.particle.mass]
        self.dynamic = [l.index for l in self.legs if l.index not in self.static]
        if diag.last in self.dynamic:      # the closing leg is the innermost one
            self.dynamic.remove(diag.last)
            self.dynamic.append(diag.last)
        self.nhel = {}
        for l in self.legs:
            p = l.particle
            if p.spin == 'S':
                self.nhel[l.index] = (0,)
            elif p.spin == 'V' and p.mass:
                self.nhel[l.index] = (-1, 0, 1)
            else:
                self.nhel[l.index] = (-1, 1)
        self._analyse()

    # ------------------------------------------------------------------ chirality masks
    def _gmask(self, v):
        return (GL if v.coup[0] else 0) | (GR if v.coup[1] else 0)

    def _leaf_mask(self, nd, hel):
        lg = self.legs[nd.leg]
        p = lg.particle
        if p.spin != 'F':
            return AB
        if p.mass:
            return AB
        nsf = self._nsf(lg)
        colslot = A if hel[nd.leg] * nsf < 0 else B
        if nd.wtype == 'col':
            return colslot
        return B if colslot == A else A

    @staticmethod
    def _nsf(lg):
        return -1 if PARTICLES[lg.name].is_anti else +1

    def _node_mask(self, nd, hel, memo):
        """Non-zero slot mask of a node for the static helicity assignment hel (dict leg -> +-1); 0 = vanishes."""
        key = (nd.uid, tuple(hel[l] for l in bits(nd.mask) if l in hel))
        if key in memo:
            return memo[key]
        if nd.is_leaf:
            r = self._leaf_mask(nd, hel)
        elif nd.is_sum:
            r = 0
            for ch in nd.members:
                r |= self._node_mask(ch, hel, memo)
        else:
            cm = [self._node_mask(ch, hel, memo) for ch in nd.children]
            if 0 in cm:
                r = 0
            elif nd.vertex.kind in ('FFV', 'FFS'):
                r = self._ff_mask(nd.vertex, dict(zip(nd.slots, cm)), nd.out_slot, bool(nd.particle.mass))
            else:
                r = AB
        memo[key] = r
        return r

    def _ff_mask(self, v, by_slot, out_slot, massive):
        g = self._gmask(v)
        # FFV: gL pairs column slot A with row slot B; gR pairs column B with row A.
        # FFS (Eq. 39): psibar (gL PL + gR PR) psi: gL pairs column A with row A; gR column B, row B.
        scalar = v.kind == 'FFS'
        if 0 in by_slot and 1 in by_slot:  # row and column given -> boson (or closed amplitude)
            mo, mi = by_slot[0], by_slot[1]
            rowL, rowR = (A, B) if scalar else (B, A)
            ok = ((mi & A) and (mo & rowL) and (g & GL)) or ((mi & B) and (mo & rowR) and (g & GR))
            return AB if ok else 0
        if 1 in by_slot:  # column continues
            mi = by_slot[1]
            l, r = bool((mi & A) and (g & GL)), bool((mi & B) and (g & GR))
            if not (l or r):
                return 0
            if massive:
                return AB
            if scalar:   # PL psi stays in A, then qslash moves it to B
                return (B if l else 0) | (A if r else 0)
            return (A if l else 0) | (B if r else 0)
        mo = by_slot[0]  # row continues
        if scalar:
            l, r = bool((mo & A) and (g & GL)), bool((mo & B) and (g & GR))
        else:
            l, r = bool((mo & B) and (g & GL)), bool((mo & A) and (g & GR))
        if not (l or r):
            return 0
        if massive:
            return AB
        if scalar:
            return (B if l else 0) | (A if r else 0)
        return (B if l else 0) | (A if r else 0)

    def _root_nonzero(self, rt, hel, memo):
        cm = [self._node_mask(ch, hel, memo) for ch in rt.children]
        if 0 in cm:
            return False
        if rt.vertex.kind in ('FFV', 'FFS'):
            return self._ff_mask(rt.vertex, dict(zip(rt.slots, cm)), -1, False) != 0
        return True

    def _analyse(self):
        self.memo = {}
        self.variants = []  # (hel dict for static legs, [non-zero roots])
        for combo in itertools.product(*[self.nhel[l] for l in self.static]):
            hel = dict(zip(self.static, combo))
            roots = [r for r in self.dg.roots if self._root_nonzero(r, hel, self.memo)]
            if roots:
                self.variants.append((hel, roots))
        ndyn = 1
        for l in self.dynamic:
            ndyn *= len(self.nhel[l])
        self.n_hel_nonzero = len(self.variants) * ndyn
        self.n_hel_total = 1
        for l in self.legs:
            self.n_hel_total *= len(self.nhel[l.index])

    # ------------------------------------------------------------------ normalisation (Eq. 4; A7)
    def avg_factor(self):
        f = Fraction(1)
        for l in self.legs:
            if l.state == 'in':
                f /= len(self.nhel[l.index])
                f /= abs(l.particle.colour)
        names = [l.name for l in self.legs if l.state == 'out']
        for nm in set(names):
            f /= factorial(names.count(nm))
        return f

    def colour_matrix(self):
        flows = self.dg.flows()
        cm = C.colour_matrix(flows)
        den = 1
        for row in cm:
            for x in row:
                den = _lcm(den, x.denominator)
        return flows, [[int(x * den) for x in row] for row in cm], den


# ====================================================================================== code generation
def _popcount(m):
    return bin(m).count('1')


class CodeGen(Emitter):
    """Emits `template <class T, class St> HG_HD T me2_<name>(const Mom<T>* p, const Coup<T>& c, const St& st)`.

    stage=True: every value produced outside a helicity loop and consumed inside one is kept in the staging area
    `st` (csrc/hg_stage.cuh; shared memory on the device) and reloaded at each use; stage=False: plain SSA values,
    liveness left to nvcc (small processes)."""

    SIZES = {'T': 1, 'cx<T>': 2, 'Mom<T>': 4, 'Vc<T>': 8, 'pol': 5}
    # staged mode: extra block rendezvous after this many calls inside a loop body.  Tuned on B200: 1, 4, 16 and
    # none gave 13.35 / 12.90 ms (before the merged currents) and 5.50 / 5.38 / 5.34 ms (after) for cfg 5 fp64, so
    # only the rendezvous at the top of each loop iteration remains (needed by the pair split, hg_stage.cuh).
    SYNC_EVERY = 1000
    ACC_IN_REGS_MAX = 8   # colour-flow accumulators stay in registers up to this many flows
    SPLIT_SHARED = True   # deal the phases outside the innermost loop to the two warps of a pair
    # closing by spinor: an FFV vertex that closes on the massless vector leg with one of its spinors independent of
    # every looped helicity is evaluated as a dot product with that spinor dressed once per event (hg_helas.cuh
    # dress_row / dress_col / sdot) instead of current + projection
    DRESS = True
    # scaled momenta: on a massless single-chirality fermion line coupling x propagator factor are folded into the
    # momentum once per event, kept in light-cone components (hg_helas.cuh lc_scaled / fvixx0 / fvoxx0)
    SCALED_K = True
    # polarisation vectors of looped gluons reach FFV vertices in light-cone form (12 instead of 24 fp64 instructions
    # for the matrix product eps-slash x spinor); staged processes only (measured: configs 4 / 5 / W + 4 jets 2.4 / 0.9 /
    # 1.5 % faster, the fused fp32 step of W + 2 jets 15 % slower)
    POL_LC = True

    def __init__(self, diag, stage=False, kfromp=False, dress=None, groups=1, opcalls=False, align_pairs=False):
        super().__init__(diag)
        if dress is not None:
            self.DRESS = dress
        self.stage = stage
        self.kfromp = stage and kfromp   # inside loops rebuild internal momenta from staged external momenta
        # group split (staged processes with the accumulators in the staging area): the closings of the innermost
        # loop body are dealt to `groups` warps (with the currents each needs; a current two groups need is
        # evaluated by both), each with its own set of accumulators, so that a TEAM of 2 x groups warps evaluates an
        # event; the colour contraction adds the sets up, one helicity of the closing leg per group.
        self.groups = groups if stage else 1
        # op calls (staged processes with the accumulators in the staging area): the arithmetic of every vertex call
        # of the innermost loop body becomes a call of a REAL function, one per distinct shape of call (routine,
        # template arguments, kinds of operands); operands and results travel by value (the ABI keeps them in
        # registers) and the loads from the staging area stay at the call site.  The inlined body of W + 4 jets is
        # 600 KB of SASS, far beyond the instruction caches, and with one warp per scheduler nothing hides the
        # fetch latency; a dozen arithmetic-only functions stay cached (DESIGN.md section 9 NEXT-4).
        self.opcalls = stage and opcalls
        # every staged value of two or more words starts at an EVEN slot (a skipped slot is kept for a later one-word
        # value): with the paired fp32 layout of hg_stage.cuh a complex number is then one 8-byte access
        self.align_pairs = stage and align_pairs

    # ------------------------------------------------------------------ value registry / operand access
    def _reg(self, name, ctype, depth, mask=AB, region=None, pol_of=None, hvar=None):
        if name not in self.vals:
            self.vals[name] = dict(name=name, ctype=ctype, depth=depth, mask=mask, slot=None,
                                   region=(0 if depth == 0 else 1) if region is None else region,
                                   pol_of=pol_of, hvar=hvar)
        return self.vals[name]

    def _size(self, v):
        if v['ctype'] == 'Sp<T>':
            return 8 if v['mask'] == AB else 4
        return self.SIZES[v['ctype']]

    def _slot(self, v):
        """Slot expression of a staged value (allocated on first use)."""
        if v['slot'] is None:
            r = v['region']
            size = self._size(v)
            if self.align_pairs and size == 1 and self.holes[r]:
                v['slot'] = self.holes[r].pop()
            else:
                if self.align_pairs and size > 1 and self.n_slots[r] % 2:
                    self.holes[r].append(self.n_slots[r])
                    self.n_slots[r] += 1
                v['slot'] = self.n_slots[r]
                self.n_slots[r] += size
            self.max_slots[r] = max(self.max_slots[r], self.n_slots[r])
        return str(v['slot']) if v['region'] == 0 else 'L + %d' % v['slot']

    def _load_expr(self, v):
        ct = v['ctype']
        if ct == 'Sp<T>':
            return 'ld_sp<%d, T>(st, %s)' % (v['mask'], self._slot(v))
        fn = {'T': 'ld_T', 'cx<T>': 'ld_cx', 'Mom<T>': 'ld_mom', 'Vc<T>': 'ld_vec'}[ct]
        return '%s<T>(st, %s)' % (fn, self._slot(v))

    def _store_line(self, v):
        ct = v['ctype']
        if ct == 'pol':
            return 'st_pol<T>(st, %s, %s);' % (self._slot(v), v['name'])
        if ct == 'Sp<T>':
            return 'st_sp<%d, T>(st, %s, %s);' % (v['mask'], self._slot(v), v['name'])
        fn = {'T': 'st_T', 'cx<T>': 'st_cx', 'Mom<T>': 'st_mom', 'Vc<T>': 'st_vec'}[ct]
        return '%s<T>(st, %s, %s);' % (fn, self._slot(v), v['name'])

    def _ref(self, name, as_pol=False):
        """Text by which the op being emitted (at loop depth self.cur_depth) reads value `name`.  as_pol: the reader is
        an FFV vertex and `name` the helicity state of a looped massless vector leg: hand it over in light-cone form
        (hg_helas.cuh Pol<T>: eps^0 = 0, real eps^3, V1 -+ i V2 formed once)."""
        v = self.vals[name]
        as_pol = as_pol and self.POL_LC and self.stage and v['pol_of'] is not None
        if not self.stage or v['depth'] >= self.cur_depth:
            return 'y' + name[1:] if as_pol else name
        alias = 'a%d' % len(self.cur_loads)
        if as_pol:
            e = self.vals[v['pol_of']]
            self.cur_loads.append('const Pol<T> %s = ld_pol_lc<T>(st, %s, %s);' % (alias, self._slot(e), v['hvar']))
        elif v['pol_of'] is not None:      # helicity state of a looped massless vector leg: from its eps(+1)
            e = self.vals[v['pol_of']]
            self.cur_loads.append('const Vc<T> %s = ld_pol<T>(st, %s, %s);' % (alias, self._slot(e), v['hvar']))
        elif v['ctype'] == 'pol':
            self.cur_loads.append('const Vc<T> %s = ld_pol<T>(st, %s, 0);' % (alias, self._slot(v)))
        else:
            self.cur_loads.append('const %s %s = %s;' % (v['ctype'], alias, self._load_expr(v)))
        return alias

    def _begin(self, depth):
        self.cur_depth = depth
        self.cur_loads = []

    # ------------------------------------------------------------------ driver
    def generate(self):
        self.vals = {}
        self.n_slots = [0, 0]
        self.max_slots = [0, 0]
        self.holes = [[], []]
        self.need_K = set()       # masks whose summed momentum is needed
        self.need_P = set()       # external legs whose momentum is read inside loops (kfromp)
        self.dup_names = set()    # cheap depth-0 values evaluated by both warps of a pair
        self.need_d = {}          # (mask, field) -> variable name of the propagator factor
        self.need_rm2 = set()     # mass names whose 1/m^2 is needed
        self.need_Q = {}          # name -> (mask, negate, coupling text, propagator-factor name): scaled momenta
        self.need_ratio = set()   # ratios of couplings 'r_<coupling>_mgs'
        self.shared = {}          # key -> name of depth-0 values already emitted
        self.shared_items = []
        self.op_funcs = {}        # shape -> name of the op function
        self.prelude = []         # lines emitted before the me2 function (the op functions)
        dyn = self.dynamic
        self.depth_of_leg = {l: i + 1 for i, l in enumerate(dyn)}
        for l in dyn:
            lg = self.legs[l]
            if lg.particle.spin == 'V' and not lg.particle.mass:
                self._reg('e%d' % l, 'pol', 0)
                if self.stage:
                    self._slot(self.vals['e%d' % l])
                self._reg('x%d' % l, 'Vc<T>', self.depth_of_leg[l], pol_of='e%d' % l, hvar='h%d' % l)
            elif self.stage:
                raise NotImplementedError('staged mode: looped legs must be massless vector bosons')
            else:
                self._reg('x%d' % l, {'V': 'Vc<T>', 'F': 'Sp<T>', 'S': 'cx<T>'}[lg.particle.spin],
                          self.depth_of_leg[l])
        flows, cmat, cden = self.colour_matrix()
        self.flows = flows
        if self.stage:
            # the kernels split the innermost loop over a pair of warps (csrc/hg_process_impl.cuh)
            nloops = len(dyn) - 1 if self.closes_by_current() else len(dyn)
            if nloops < 1 or len(self.nhel[dyn[nloops - 1]]) != 2:
                raise NotImplementedError('staged mode needs an innermost helicity loop of two states')
        variants = []
        for vi, (hel, roots) in enumerate(self.variants):
            self.n_slots[1] = 0       # loop-level slots are reused by every static-helicity variant
            self.holes[1] = []
            variants.append(self._emit_variant(vi, hel, roots, cmat))
        pre = self._preamble()
        out = []
        if self.stage:
            if self.align_pairs:
                self.max_slots[0] += self.max_slots[0] % 2
            out.append('  constexpr int L = %d;  // first slot of the loop-level values' % self.max_slots[0])
        out += self._render_shared(pre + self.shared_items, '  ')
        out.append('  T me = T(0);')
        for var in variants:
            out += self._render_variant(var)
        scale = self.avg_factor() / cden
        out.append('  return me * T(%s);' % _lit(scale))
        self.n_stage = self.max_slots[0] + self.max_slots[1] if self.stage else 0
        return out

    # rough cost (flops) of an emitted call, used only to balance the two halves of a shared phase
    _CALL_COST = (('dress_', 45), ('lc_scaled', 8), ('fvixx0', 55), ('fvoxx0', 55), ('fvixxx', 63), ('fvoxxx', 63), ('fsixxx', 40), ('fsoxxx', 40), ('jioxx', 45), ('jvvxxx', 110),
                  ('jgggxx', 70), ('vxxxxx', 40), ('ixxxx0', 25), ('oxxxx0', 25), ('crcp', 25), ('hrcp', 15),
                  ('unit0', 18), ('two_dot0', 8))

    def _render_shared(self, items, ind):
        """A phase that both warps of a pair would execute (everything outside the innermost helicity loop).  Its
        items are partitioned into groups that do not read each other's registers (values of other loop depths
        come through the staging area anyway) and the groups are dealt to the two warps, st.own(0) / st.own(1),
        balanced by estimated cost.  The rendezvous at the top of the next loop makes all results visible."""
        if not (self.stage and self.SPLIT_SHARED) or any(it[0] != 'def' for it in items) or len(items) < 2:
            return self._render_items(items, ind)
        both = [it for it in items if it[1] in self.dup_names]
        items = [it for it in items if it[1] not in self.dup_names]
        index = {it[1]: i for i, it in enumerate(items)}
        parent = list(range(len(items)))

        def find(i):
            while parent[i] != i:
                parent[i] = parent[parent[i]]
                i = parent[i]
            return i

        cost = []
        for i, it in enumerate(items):
            for tok in set(re.findall(r'[A-Za-z_]\w*', it[2])):
                j = index.get(tok)
                if j is not None and j != i:
                    parent[find(i)] = find(j)
            c = 4
            for fn, w in self._CALL_COST:
                if fn in it[2]:
                    c = w
                    break
            cost.append(c)
        groups = {}
        for i in range(len(items)):
            groups.setdefault(find(i), []).append(i)
        nown = 2 * self.groups       # warps that share an event: pair, or team of four
        load = [0] * nown
        owner = {}
        for root, members in sorted(groups.items(), key=lambda kv: -sum(cost[i] for i in kv[1])):
            h = load.index(min(load))
            load[h] += sum(cost[i] for i in members)
            for i in members:
                owner[i] = h
        out = self._render_items(both, ind)
        for h in range(nown):
            mine = [items[i] for i in range(len(items)) if owner[i] == h]
            if not mine:
                continue
            out.append(ind + 'if (st.own(%d)) {  // estimated %d of %d flops of this phase' % (h, load[h], sum(load)))
            body = self._render_items(mine, ind + '  ', no_sync=True)
            assert not any('st.sync' in ln for ln in body), 'block barrier under st.own()'
            out += body
            out.append(ind + '}')
        return out

    def _render_items(self, items, ind, no_sync=False):
        """items: ('raw', text) | ('def', name, expr, loads) | ('blk', [lines], loads).  no_sync: the items sit under a
        warp-divergent condition (st.own): a block barrier there would hang the block."""
        out = []
        nsince = 0
        for it in items:
            if self.stage and it[0] != 'raw' and not no_sync:
                nsince += 1
                if nsince > self.SYNC_EVERY:
                    out.append(ind + 'st.sync();')
                    nsince = 1
            if it[0] == 'raw':
                out.append(ind + it[1])
            elif it[0] == 'def':
                _, name, expr, loads = it
                v = self.vals[name]
                ct = 'Vc<T>' if v['ctype'] == 'pol' else v['ctype']
                if loads:
                    out.append(ind + '%s %s;' % (ct, name))
                    out.append(ind + '{ ' + ' '.join(loads))
                    out.append(ind + '  %s = %s; }' % (name, expr))
                else:
                    out.append(ind + 'const %s %s = %s;' % (ct, name, expr))
                if self.stage and v['slot'] is not None:
                    out.append(ind + self._store_line(v))
            else:
                _, lines, loads = it
                out.append(ind + '{ ' + ' '.join(loads))
                for ln in lines:
                    out.append(ind + '  ' + ln)
                out.append(ind + '}')
        return out

    # ------------------------------------------------------------------ op calls (innermost loop body)
    _RE_REG = re.compile(r'\b(v\d+_\d+|[xya]\d+)\b')
    _RE_CPL = re.compile(r'\bc\.\w+\b')
    _RE_ACC = re.compile(r'^(acc_add<T>\(st, A \+ \d+, T\(-?\d+\), rb, ib\);|X\d+ = X\d+ |j\d+ = j\d+ )')
    _RE_ALIAS = re.compile(r'^const ([A-Za-z]+(?:<T>)?) (a\d+) = (\w+)(?:<(\d), T>)?')

    def _reg_ctype(self, name):
        if name[0] == 'y':
            return 'Pol<T>'
        if name[0] == 'x':
            return 'Vc<T>'
        v = self.vals[name]
        return 'Vc<T>' if v['ctype'] == 'pol' else v['ctype']

    def _op_call(self, ret, loads, body, ret_mask=AB):
        """Call expression of the op function with the shape of `body` (created on first use).  Couplings become T
        parameters (one per occurrence), register operands and the aliases of `loads` by-value parameters (one per
        distinct operand); a single-chirality spinor travels as its non-zero half (hg_stage.cuh Sh<T>)."""
        params, args, regs, unpack = [], [], {}, []
        count = {'g': 0, 'r': 0}
        alias = {}
        for ln in loads:
            m = self._RE_ALIAS.match(ln)
            assert m, ln
            alias[m.group(2)] = (m.group(1), int(m.group(4)) if m.group(3) == 'ld_sp' else AB)

        def param(kind, ctype, actual):
            if kind == 'r' and actual in regs:
                return regs[actual]
            pname = '%s%d' % (kind, count[kind])
            count[kind] += 1
            m = AB
            if kind == 'r' and ctype == 'Sp<T>':
                m = alias[actual][1] if actual in alias else self.vals[actual]['mask']
            if m != AB:
                params.append('Sh<T> %sh' % pname)
                args.append('sp_half<%d>(%s)' % (m, actual))
                unpack.append('const Sp<T> %s = sp_full<%d>(%sh);' % (pname, m, pname))
            else:
                params.append('%s %s' % (ctype, pname))
                args.append(actual)
            if kind == 'r':
                regs[actual] = pname
            return pname

        def ctype_of(name):
            return alias[name][0] if name in alias else self._reg_ctype(name)

        out = []
        for ln in body:
            assert '(st' not in ln, ln
            ln = self._RE_REG.sub(lambda m: param('r', ctype_of(m.group(1)), m.group(1)), ln)
            ln = self._RE_CPL.sub(lambda m: param('g', 'T', m.group(0)), ln)
            out.append(ln)
        out = unpack + out
        half = None
        if ret == 'Sp<T>' and ret_mask != AB:
            half = ret_mask
            ret = 'Sh<T>'
            assert out[-1].startswith('return ')
            out[-1] = 'return sp_half<%d>(%s);' % (half, out[-1][len('return '):-1])
        key = (ret, tuple(params), tuple(out))
        if key not in self.op_funcs:
            name = 'op_%s_%d' % (self.dg.spec.name, len(self.op_funcs))
            self.op_funcs[key] = name
            self.prelude.append('template <class T>')
            self.prelude.append('HG_OPCALL %s %s(%s) {' % (ret, name, ', '.join(params)))
            self.prelude += ['  ' + ln for ln in out]
            self.prelude.append('}')
        call = '%s<T>(%s)' % (self.op_funcs[key], ', '.join(args))
        return 'sp_full<%d>(%s)' % (half, call) if half else call

    # Prefetch: the loads of call i + 1 issued BEFORE call i, so that their latency overlaps the arithmetic of call i.
    # Measured on B200 for W + 4 jets and switched off: the prefetched operands live across the call, ptxas spills
    # more (fp64 1.7 -> 3.0 KB of spill loads per thread) and the kernel is SLOWER, 14.2 -> 17.7 ms per 2^18 events in
    # fp64, 5.98 -> 6.26 ms in fp32.
    OP_PREFETCH = False

    # accumulator updates of one closing in batches of this many flows: all loads of a batch are issued before its
    # first add (acc_add_batch, hg_stage.cuh).  One acc_add per flow left every update waiting for its own
    # shared-memory load (ncu source view: one DADD per flow with the stall samples of a whole LDS latency).
    # Measured for W + 4 jets, 2^18 events: one flow at a time 14.15 ms (fp64) / 5.96 ms (fp32), batches of 4
    # 13.50 / 5.55 ms, batches of 8 13.52 / 5.61 ms.
    # (The batch as a call of a real function -- offsets at run time, signs as a bit mask -- makes the call sites a
    # quarter smaller but was measured SLOWER for W + 4 jets: 13.3 -> 15.4 ms in fp64, 5.6 -> 7.5 ms in fp32.)
    ACC_BATCH = 4
    _RE_ACC_SMEM = re.compile(r'^acc_add<T>\(st, A \+ (\d+), T\((-?\d+)\), rb, ib\);$')

    def _batch_accs(self, accs):
        ms = [self._RE_ACC_SMEM.match(ln) for ln in accs]
        if self.ACC_BATCH < 2 or not all(ms) or len(ms) < 2:
            return accs
        out = []
        for i in range(0, len(ms), self.ACC_BATCH):
            part = ms[i:i + self.ACC_BATCH]
            if len(part) == 1:
                out.append(part[0].group(0))
                continue
            out.append('{ const int o[%d] = {%s}; const T k[%d] = {%s}; acc_add_batch<%d, T>(st, A, o, k, rb, ib); }' % (
                len(part), ', '.join(m.group(1) for m in part), len(part),
                ', '.join('T(%s)' % m.group(2) for m in part), len(part)))
        return out

    def _render_calls(self, items, ind):
        """The innermost loop body with the arithmetic of every vertex call in an op function (see __init__)."""
        steps = []      # (loads, lines after the loads)
        for n, it in enumerate(items):
            ren = lambda t: re.sub(r'\ba(\d+)\b', r'a%d_\1' % n, t)
            if it[0] == 'raw':
                steps.append(([], [it[1]]))
            elif it[0] == 'def':
                _, name, expr, loads = it
                v = self.vals[name]
                ct = 'Vc<T>' if v['ctype'] == 'pol' else v['ctype']
                if '(' not in expr:          # a sum of register values: stays in line
                    assert not loads
                    after = ['const %s %s = %s;' % (ct, name, expr)]
                else:
                    call = self._op_call(ct, loads, ['return %s;' % expr], v['mask'])
                    after = ['const %s %s = %s;' % (ct, name, ren(call))]
                if v['slot'] is not None:
                    after.append(self._store_line(v))
                steps.append(([ren(ln) for ln in loads], after))
            else:
                _, lines, loads = it
                work = [ln for ln in lines if not self._RE_ACC.match(ln)]
                accs = [ln for ln in lines if self._RE_ACC.match(ln)]
                assert accs and len(work) + len(accs) == len(lines), lines
                if any(' rb' in ln for ln in work):     # closing by current: projections on eps(+) and its conjugate
                    call = self._op_call('RbIb<T>', loads, work + ['return RbIb<T>{rb, ib};'])
                    first = 'const RbIb<T> q = %s; const cx<T> rb = q.rb, ib = q.ib;' % ren(call)
                else:                                   # closing by amplitude
                    assert len(work) == 1 and work[0].startswith('const cx<T> a = '), work
                    call = self._op_call('cx<T>', loads, ['return ' + work[0][len('const cx<T> a = '):]])
                    first = 'const cx<T> a = %s;' % ren(call)
                steps.append(([ren(ln) for ln in loads], ['{ ' + first] + ['  ' + ln for ln in self._batch_accs(accs)]
                              + ['}']))
        out = []
        if not self.OP_PREFETCH:
            for loads, after in steps:
                out += [ind + ln for ln in loads + after]
            return out
        out += [ind + ln for ln in (steps[0][0] if steps else [])]
        for i, (loads, after) in enumerate(steps):
            if i + 1 < len(steps):
                out += [ind + ln for ln in steps[i + 1][0]]
            out += [ind + ln for ln in after]
        return out

    # ------------------------------------------------------------------ helpers
    def _depth(self, mask):
        d = 0
        for l in bits(mask):
            d = max(d, self.depth_of_leg.get(l, 0))
        return d

    def _helcode(self, mask, hel):
        return ''.join('p' if hel[l] > 0 else 'm' for l in bits(mask) if l in hel)

    def _K(self, mask, neg=False):
        if self.kfromp and self.cur_depth > 0:
            # sum of at most n/2 external momenta (momentum conservation: K(mask) = -K(complement))
            n = self.dg.n
            use, sg = (mask, 1) if _popcount(mask) <= n - _popcount(mask) else (self.dg.full & ~mask, -1)
            if neg:
                sg = -sg
            terms = []
            for l in bits(use):
                self.need_P.add(l)
                self._reg('P%d' % l, 'Mom<T>', 0)
                s_l = sg * (1 if self.legs[l].state == 'in' else -1)
                terms.append(('+' if s_l > 0 else '-', self._ref('P%d' % l)))
            txt = ('-' if terms[0][0] == '-' else '') + terms[0][1]
            for sign, t in terms[1:]:
                txt += ' %s %s' % (sign, t)
            return '(%s)' % txt if len(terms) > 1 or terms[0][0] == '-' else txt
        self.need_K.add(mask)
        self._reg('K%d' % mask, 'Mom<T>', 0)
        return ('-' if neg else '') + self._ref('K%d' % mask)

    def _Kn(self, mask):
        return self._K(mask, neg=True)

    def _d_name(self, nd):
        p = nd.particle
        key = (nd.mask, p.mass, p.width, p.spin)
        if key not in self.need_d:
            self.need_d[key] = 'd%d_%s%s' % (nd.mask, p.spin.lower(), p.mass or '0')
            self._reg(self.need_d[key], 'cx<T>' if p.width else 'T', 0)
        return self.need_d[key]

    def _d(self, nd):
        return self._ref(self._d_name(nd))

    def _Q(self, nd, neg, coup):
        """Scaled light-cone momentum of the massless fermion line nd: (coupling x propagator factor) x (+-K)."""
        dname = self._d_name(nd)          # the propagator factor, used at depth 0 only
        self.need_K.add(nd.mask)
        self._reg('K%d' % nd.mask, 'Mom<T>', 0)
        name = 'Q%d_%s%s' % (nd.mask, 'm' if neg else 'p', coup)
        if name not in self.need_Q:
            self.need_Q[name] = (nd.mask, neg, coup, dname)
            self._reg(name, 'Mom<T>', 0)
        return self._ref(name)

    def _mass(self, p):
        return 'c.%s' % p.mass if p.mass else 'T(0)'

    def _rm2(self, p):
        if not p.mass:
            return 'T(0)'
        self.need_rm2.add(p.mass)
        self._reg('rm2_%s' % p.mass, 'cx<T>', 0)
        return self._ref('rm2_%s' % p.mass)

    # couplings that contain m_W or m_Z: complex in the paper's complex-mass option (Eq. 55)
    COMPLEX_COUPLINGS = ('gtth', 'gwwh', 'gzzh', 'ghhh')

    @classmethod
    def _cpl(cls, name):
        if name in cls.COMPLEX_COUPLINGS:
            return 'mk<T>(c.%s, c.%s_i)' % (name, name)
        return 'c.%s' % name if name else 'T(0)'

    def _name(self, nd, vi, hel):
        if nd.is_leaf and nd.leg in self.depth_of_leg:
            return 'x%d' % nd.leg
        if self._depth(nd.mask) == 0:
            return 's%d_%s' % (nd.uid, self._helcode(nd.mask, hel))
        return 'v%d_%d' % (vi, nd.uid)

    def _wtype_decl(self, nd):
        return {'col': 'Sp<T>', 'row': 'Sp<T>', 'vec': 'Vc<T>', 'sca': 'cx<T>'}[nd.wtype]

    # ------------------------------------------------------------------ one node
    def _leaf_expr(self, nd, hel):
        lg = self.legs[nd.leg]
        p = lg.particle
        if p.spin == 'F':
            fn = 'ixxxx0' if nd.wtype == 'col' else 'oxxxx0'
            return '%s<T>(p[%d], %d, %d)' % (fn, nd.leg, hel[nd.leg], self._nsf(lg))
        raise NotImplementedError

    def _sum_expr(self, nd, vi, hel):
        """Sum of the member currents that do not vanish for this helicity assignment."""
        txt = ''
        for ch, sg in zip(nd.members, nd.msigns):
            if self._node_mask(ch, hel, self.memo) == 0:
                continue
            r = self._ref(self._name(ch, vi, hel))
            txt += (' + ' if sg > 0 else ' - ') + r if txt else ('-' if sg < 0 else '') + r
        return txt

    def _node_expr(self, nd, vi, hel):
        v = nd.vertex
        by_slot = dict(zip(nd.slots, nd.children))
        nm = lambda ch: self._ref(self._name(ch, vi, hel))
        mk = lambda ch: self._node_mask(ch, hel, self.memo)
        p = nd.particle
        massive = 'true' if p.mass else 'false'
        if v.kind == 'FFV':
            g = self._gmask(v)
            gl, gr = self._cpl(v.coup[0]), self._cpl(v.coup[1])
            if self.SCALED_K and nd.out_slot in (0, 1) and not p.mass and not p.width:
                cont = by_slot[1] if nd.out_slot == 0 else by_slot[0]
                m_in = mk(cont)
                if nd.out_slot == 0:
                    left, right = bool((m_in & A) and (g & GL)), bool((m_in & B) and (g & GR))
                else:
                    left, right = bool((m_in & B) and (g & GL)), bool((m_in & A) and (g & GR))
                coup = v.coup[0] if left else v.coup[1]
                # staged processes are short of staging words: one scaled momentum per line, for the strong coupling
                # (the W attaches once per diagram, gluons everywhere)
                if left != right:
                    fn = 'fvixx0' if nd.out_slot == 0 else 'fvoxx0'
                    vec = by_slot[2]
                    a_f, a_v = nm(cont), self._ref(self._name(vec, vi, hel), as_pol=True)
                    if self.stage and coup != 'mgs':
                        # staged processes are short of staging words: ONE scaled momentum per line, for the strong
                        # coupling (gluons attach everywhere, the W once per diagram); other couplings rescale
                        ratio = 'r_%s_mgs' % coup
                        if ratio not in self.need_ratio:
                            self.need_ratio.add(ratio)
                            self._reg(ratio, 'T', 0)
                        return '%ss<%d, %d>(%s, %s, %s, %s)' % (fn, m_in, g, a_f, a_v,
                                                               self._Q(nd, nd.out_slot == 1, 'mgs'), self._ref(ratio))
                    return '%s<%d, %d>(%s, %s, %s)' % (fn, m_in, g, a_f, a_v, self._Q(nd, nd.out_slot == 1, coup))
            if nd.out_slot == 0:    # remaining field is the row slot -> the column continues
                col, vec = by_slot[1], by_slot[2]
                return 'fvixxx<%d, %d, %s>(%s, %s, %s, %s, %s, %s, %s)' % (
                    mk(col), g, massive, nm(col), self._ref(self._name(vec, vi, hel), as_pol=True), gl, gr,
                    self._K(nd.mask), self._mass(p), self._d(nd))
            if nd.out_slot == 1:    # the row continues
                row, vec = by_slot[0], by_slot[2]
                return 'fvoxxx<%d, %d, %s>(%s, %s, %s, %s, %s, %s, %s)' % (
                    mk(row), g, massive, nm(row), self._ref(self._name(vec, vi, hel), as_pol=True), gl, gr,
                    self._Kn(nd.mask), self._mass(p), self._d(nd))
            row, col = by_slot[0], by_slot[1]
            if p.mass:
                return 'jioxxx<%d, %d, %d, true>(%s, %s, %s, %s, %s, %s, %s)' % (
                    mk(col), mk(row), g, nm(col), nm(row), gl, gr, self._K(nd.mask), self._rm2(p), self._d(nd))
            return 'jioxx0<%d, %d, %d>(%s, %s, %s, %s, %s)' % (
                mk(col), mk(row), g, nm(col), nm(row), gl, gr, self._d(nd))
        if v.kind == 'VVV':
            a, b = by_slot[(nd.out_slot + 1) % 3], by_slot[(nd.out_slot + 2) % 3]
            return 'jvvxxx<%s>(%s, %s, %s, %s, %s, %s, %s)' % (
                massive, nm(a), nm(b), self._cpl(v.coup[0]), self._K(a.mask), self._K(b.mask), self._rm2(p),
                self._d(nd))
        if v.kind == 'VVVV':
            if v.colour != 'ff':
                raise NotImplementedError('electroweak four-boson vertex (K13, out of scope)')
            kids = [by_slot[s] for s in sorted(by_slot)]
            a, b, c3 = kids
            x, y, z = {1: (a, b, c3), 2: (a, c3, b), 3: (b, c3, a)}[nd.struct]
            return 'jgggxx(%s, %s, %s, %s, %s)' % (nm(x), nm(y), nm(z), self._cpl(v.coup[0]), self._d(nd))
        if v.kind == 'FFS':
            g = self._gmask(v)
            gl, gr = self._cpl(v.coup[0]), self._cpl(v.coup[1])
            if nd.out_slot == 0:    # the column continues
                col, sca = by_slot[1], by_slot[2]
                return 'fsixxx<%d, %d, %s>(%s, %s, %s, %s, %s, %s, %s)' % (
                    mk(col), g, massive, nm(col), nm(sca), gl, gr, self._K(nd.mask), self._mass(p), self._d(nd))
            if nd.out_slot == 1:    # the row continues
                row, sca = by_slot[0], by_slot[2]
                return 'fsoxxx<%d, %d, %s>(%s, %s, %s, %s, %s, %s, %s)' % (
                    mk(row), g, massive, nm(row), nm(sca), gl, gr, self._Kn(nd.mask), self._mass(p), self._d(nd))
            row, col = by_slot[0], by_slot[1]
            return 'hioxxx<%d, %d, %d>(%s, %s, %s, %s, %s)' % (
                mk(col), mk(row), g, nm(col), nm(row), gl, gr, self._d(nd))
        if v.kind in ('VVS', 'VVSS'):
            # slots 0, 1: vectors; 2 (, 3): scalars
            g = self._cpl(v.coup[0])
            scas = [nm(by_slot[s_]) for s_ in sorted(by_slot) if s_ >= 2]
            if nd.out_slot >= 2:    # scalar from the two vectors (and the other scalar)
                fn = 'hvvxxx' if v.kind == 'VVS' else 'hvvsxx'
                return '%s(%s)' % (fn, ', '.join([nm(by_slot[0]), nm(by_slot[1])] + scas + [g, self._d(nd)]))
            vec = by_slot[1 - nd.out_slot]
            fn = 'jvsxxx' if v.kind == 'VVS' else 'jvssxx'
            return '%s<%s>(%s)' % (fn, massive, ', '.join([nm(vec)] + scas + [g, self._K(nd.mask), self._rm2(p),
                                                                             self._d(nd)]))
        if v.kind == 'SSS':
            a, b = [by_slot[s_] for s_ in sorted(by_slot)]
            return 'hssxxx(%s, %s, %s, %s)' % (nm(a), nm(b), self._cpl(v.coup[0]), self._d(nd))
        raise NotImplementedError(v.kind)

    def _root_expr(self, rt, vi, hel):
        v = rt.vertex
        by_slot = dict(zip(rt.slots, rt.children))
        nm = lambda ch: self._ref(self._name(ch, vi, hel))
        mk = lambda ch: self._node_mask(ch, hel, self.memo)
        if v.kind == 'FFV':
            row, col, vec = by_slot[0], by_slot[1], by_slot[2]
            return 'iovxxx<%d, %d, %d>(%s, %s, %s, %s, %s)' % (
                mk(col), mk(row), self._gmask(v), nm(col), nm(row), nm(vec), self._cpl(v.coup[0]),
                self._cpl(v.coup[1]))
        if v.kind == 'VVV':
            a, b, c3 = by_slot[0], by_slot[1], by_slot[2]
            return 'vvvxxx(%s, %s, %s, %s, %s, %s, %s)' % (
                nm(a), nm(b), nm(c3), self._cpl(v.coup[0]), self._K(a.mask), self._K(b.mask), self._K(c3.mask))
        if v.kind == 'VVVV':
            if v.colour != 'ff':
                raise NotImplementedError('electroweak four-boson vertex (K13, out of scope)')
            a, b, c3, d4 = [by_slot[s] for s in sorted(by_slot)]
            x, y, z = {1: (a, b, c3), 2: (a, c3, b), 3: (b, c3, a)}[rt.struct]
            return 'ggggxx(%s, %s, %s, %s, %s)' % (nm(x), nm(y), nm(z), nm(d4), self._cpl(v.coup[0]))
        if v.kind == 'FFS':
            row, col, sca = by_slot[0], by_slot[1], by_slot[2]
            return 'iosxxx<%d, %d, %d>(%s, %s, %s, %s, %s)' % (
                mk(col), mk(row), self._gmask(v), nm(col), nm(row), nm(sca), self._cpl(v.coup[0]),
                self._cpl(v.coup[1]))
        if v.kind in ('VVS', 'VVSS', 'SSS'):
            fn = {'VVS': 'vvsxxx', 'VVSS': 'vvssxx', 'SSS': 'sssxxx'}[v.kind]
            return '%s(%s)' % (fn, ', '.join([nm(by_slot[s_]) for s_ in sorted(by_slot)] + [self._cpl(v.coup[0])]))
        raise NotImplementedError(v.kind)

    def closes_by_current(self):
        """True if the last leg is a massless vector boson: the roots are then evaluated as bare currents projected
        on eps(+1) of that leg (hg_helas.cuh "closing on a massless vector leg") and its helicity is not looped."""
        if not self.dynamic or self.dynamic[-1] != self.dg.last:
            return False
        p = self.legs[self.dg.last].particle
        return p.spin == 'V' and not p.mass

    def _root_current_expr(self, rt, vi, hel):
        v = rt.vertex
        by_slot = dict(zip(rt.slots, rt.children))
        nm = lambda ch: self._ref(self._name(ch, vi, hel))
        mk = lambda ch: self._node_mask(ch, hel, self.memo)
        last = self.dg.last
        is_last = lambda ch: ch.is_leaf and ch.leg == last
        if v.kind == 'FFV':
            row, col, vec = by_slot[0], by_slot[1], by_slot[2]
            assert is_last(vec)
            return 'ffv_current<%d, %d, %d>(%s, %s, %s, %s)' % (
                mk(col), mk(row), self._gmask(v), nm(col), nm(row), self._cpl(v.coup[0]), self._cpl(v.coup[1]))
        if v.kind == 'VVV':
            (sl,) = [s_ for s_, ch in by_slot.items() if is_last(ch)]
            a, b = by_slot[(sl + 1) % 3], by_slot[(sl + 2) % 3]
            return 'jvv_bare(%s, %s, %s, %s, %s)' % (nm(a), nm(b), self._cpl(v.coup[0]), self._K(a.mask),
                                                     self._K(b.mask))
        if v.kind == 'VVVV':
            if v.colour != 'ff':
                raise NotImplementedError('electroweak four-boson vertex (K13, out of scope)')
            a, b, c3, d4 = [by_slot[s_] for s_ in sorted(by_slot)]
            x, y, z = {1: (a, b, c3), 2: (a, c3, b), 3: (b, c3, a)}[rt.struct]
            # ggggxx(x, y, z, d4) = g2 [(x.z)(y.d4) - (y.z)(x.d4)], solved for the closing leg
            if is_last(d4):
                t = (x, y, z)
            elif is_last(z):
                t = (y, x, d4)
            elif is_last(y):
                t = (z, d4, x)
            else:
                assert is_last(x)
                t = (d4, z, y)
            return 'jggg_bare(%s, %s, %s, %s)' % (nm(t[0]), nm(t[1]), nm(t[2]), self._cpl(v.coup[0]))
        raise NotImplementedError(v.kind)

    # ------------------------------------------------------------------ one static-helicity variant
    def _emit_variant(self, vi, hel, roots, cmat):
        dyn = self.dynamic
        cbc = self.closes_by_current()
        k = len(dyn) - 1 if cbc else len(dyn)   # number of helicity loops
        levels = [[] for _ in range(k + 1)]     # items per loop depth
        done = set()

        def need(nd):
            """Emit nd (and, first, its children) in post-order."""
            if nd.is_leaf and nd.leg in self.depth_of_leg:
                return                      # dynamic leaf: declared by its loop header
            dep = self._depth(nd.mask)
            name = self._name(nd, vi, hel)
            if dep == 0:
                if name in self.shared:
                    return
            elif nd.uid in done:
                return
            for ch in nd.children:
                need(ch)
            self._reg(name, self._wtype_decl(nd), dep, mask=self._node_mask(nd, hel, self.memo))
            self._begin(dep)
            if nd.is_leaf:
                expr = self._leaf_expr(nd, hel)
            elif nd.is_sum:
                expr = self._sum_expr(nd, vi, hel)
            else:
                expr = self._node_expr(nd, vi, hel)
            item = ('def', name, expr, self.cur_loads)
            if dep == 0:
                self.shared[name] = True
                self.shared_items.append(item)
            else:
                done.add(nd.uid)
                levels[dep].append(item)

        nf = len(self.flows)
        fidx = {w: i for i, w in enumerate(self.flows)}
        inner = levels[k]
        last = self.dg.last
        # Many colour flows (W + 4 jets: 24): the 2 nf complex accumulators would take 8 nf registers of fp64, so
        # they live in the staging area instead, one set per warp of the pair.
        acc_smem = cbc and self.stage and (nf > self.ACC_IN_REGS_MAX or self.groups > 1)
        G = self.groups
        if not (G == 1 or (G == 2 and acc_smem)):
            raise NotImplementedError('group split needs the accumulators in the staging area (closing by current)')
        if acc_smem:
            accbase = self.n_slots[1]
            self.n_slots[1] += 8 * nf * G
            self.max_slots[1] = max(self.max_slots[1], self.n_slots[1])
        for rt in roots:
            for ch in rt.children:
                need(ch)
            self._begin(k)
            lines = []
            if cbc:
                dressed = self._dressed_closing(rt, vi, hel, k)
                if dressed:
                    lines += dressed
                else:
                    lines.append('const Vc<T> b = %s;' % self._root_current_expr(rt, vi, hel))
                    lines.append('cx<T> rb, ib;')
                    lines.append('close_proj(%s, b, rb, ib);' % self._ref('e%d' % last))
                for w, cf in sorted(rt.colour.terms.items()):
                    f = fidx[w]
                    if acc_smem:
                        lines.append('acc_add<T>(st, A + %d, T(%d), rb, ib);' % (4 * f, cf))
                    elif cf == 1:
                        lines.append('X%d = X%d + rb; Y%d = Y%d + ib;' % (f, f, f, f))
                    elif cf == -1:
                        lines.append('X%d = X%d - rb; Y%d = Y%d - ib;' % (f, f, f, f))
                    else:
                        lines.append('X%d = X%d + T(%d) * rb; Y%d = Y%d + T(%d) * ib;' % (f, f, cf, f, f, cf))
            else:
                lines.append('const cx<T> a = %s;' % self._root_expr(rt, vi, hel))
                for w, cf in sorted(rt.colour.terms.items()):
                    f = fidx[w]
                    if cf == 1:
                        lines.append('j%d = j%d + a;' % (f, f))
                    elif cf == -1:
                        lines.append('j%d = j%d - a;' % (f, f))
                    else:
                        lines.append('j%d = j%d + T(%d) * a;' % (f, f, cf))
            inner.append(('blk', lines, self.cur_loads))
        if G == 2:
            levels[k] = inner = [('grp', self._partition(inner))]
        # colour contraction (symmetric form)
        tail = []
        if cbc:
            tail.append('#pragma unroll')
            tail.append('for (int h%d = 0; h%d < 2; ++h%d) {' % (last, last, last))
            tail.append('  const T sg = h%d ? T(-1) : T(1);' % last)
            if acc_smem and G == 2:
                o = 4 * nf
                tail.append('  const cx<T> ' + ', '.join(
                    'j%d = close_amp(ld_cx<T>(st, A + %d) + ld_cx<T>(st, A + %d), ld_cx<T>(st, A + %d) + '
                    'ld_cx<T>(st, A + %d), sg)' % (f, 4 * f, o + 4 * f, 4 * f + 2, o + 4 * f + 2)
                    for f in range(nf)) + ';')
            elif acc_smem:
                tail.append('  const cx<T> ' + ', '.join(
                    'j%d = close_amp(ld_cx<T>(st, A + %d), ld_cx<T>(st, A + %d), sg)' % (f, 4 * f, 4 * f + 2)
                    for f in range(nf)) + ';')
            else:
                tail.append('  const cx<T> ' + ', '.join('j%d = close_amp(X%d, Y%d, sg)' % (f, f, f)
                                                         for f in range(nf)) + ';')
        pre = '  ' if cbc else ''
        for f in range(nf):
            terms = []
            for g in range(f, nf):
                cval = cmat[f][g] * (1 if g == f else 2)
                if cval == 0:
                    continue
                terms.append('T(%d) * j%d' % (cval, g))
            tail.append(pre + '{ const cx<T> t = %s; me += j%d.re * t.re + j%d.im * t.im; }' % (
                ' + '.join(terms), f, f))
        if cbc and acc_smem and G == 2:
            # the sets of the two groups are complete after a rendezvous of the team; group g contracts helicity g
            tail[0] = '#pragma unroll 1'
            tail[1] = 'for (int h%d = 0; h%d < 2; ++h%d) if (st.grp(h%d)) {' % (last, last, last, last)
            tail.append('}')
            tail = ['st.sync();', 'const int A = L + %d + st.lo() * %d;' % (accbase, 8 * nf)] + tail
            accdecl = ('const int A = L + %d + (st.lo() * 2 + %%d) * %d; for (int i = 0; i < %d; ++i) '
                       'st.put(A + i, T(0));' % (accbase, 4 * nf, 4 * nf))
        elif cbc and acc_smem:
            tail.append('}')
            accdecl = ('const int A = L + %d + st.lo() * %d; for (int i = 0; i < %d; ++i) st.put(A + i, T(0));'
                       % (accbase, 4 * nf, 4 * nf))
        elif cbc:
            tail.append('}')
            accdecl = 'cx<T> ' + ', '.join('X%d = czero<T>(), Y%d = czero<T>()' % (f, f) for f in range(nf)) + ';'
        else:
            accdecl = 'cx<T> ' + ', '.join('j%d = czero<T>()' % f for f in range(nf)) + ';'
        return dict(hel=hel, levels=levels, tail=tail, k=k, accdecl=accdecl, groups=G,
                    calls=bool(self.opcalls and k > 0))

    # (A cost table with the closings' own flops -- jvv_bare 140, jggg_bare 110, ffv_current 80, sdot 32, 8 per
    # accumulator update -- balances the four warps of W + 4 jets to 2 % instead of 11 % in counted flops but
    # duplicates more sub-currents: 14.15 -> 14.30 ms in fp64, 5.96 -> 5.80 ms in fp32 per 2^18 events; not adopted.)
    def _partition(self, inner):
        """Deals the closings ('blk' items) of the innermost loop body to two groups, each with the 'def' items its
        closings need (in the original order).  Greedy, in order (neighbouring closings share currents): a closing
        goes to the group whose estimated cost grows less, with the running totals as the balance."""
        index = {it[1]: i for i, it in enumerate(inner) if it[0] == 'def'}
        deps, cost = [], []
        for i, it in enumerate(inner):
            text = it[2] if it[0] == 'def' else ' '.join(it[1])
            deps.append({index[n] for n in re.findall(r'v\d+_\d+', text) if n in index and index[n] != i})
            c = 8
            for fn, w in self._CALL_COST:
                if fn in text:
                    c = w
                    break
            cost.append(c + 4 * text.count('acc_add'))
        memo = {}

        def closure(i):
            if i not in memo:
                r = {i}
                for j in deps[i]:
                    r |= closure(j)
                memo[i] = r
            return memo[i]

        have, total = [set(), set()], [0, 0]
        for i, it in enumerate(inner):
            if it[0] != 'blk':
                continue
            need = closure(i)
            add = [sum(cost[j] for j in need - have[g]) for g in (0, 1)]
            g = 0 if total[0] + add[0] <= total[1] + add[1] else 1
            have[g] |= need
            total[g] += add[g]
        assert all(i in have[0] or i in have[1] for i in range(len(inner)))
        self.group_cost = total
        return [[inner[i] for i in sorted(h)] for h in have]

    def _dressed_closing(self, rt, vi, hel, k):
        """Lines that compute rb, ib of an FFV root as spinor dot products, or None if neither spinor is helicity-loop
        independent (or the option is off).  The dressed spinors are depth-0 values, defined once and shared."""
        if not self.DRESS or rt.vertex.kind != 'FFV' or k == 0:
            return None
        v = rt.vertex
        by_slot = dict(zip(rt.slots, rt.children))
        row, col = by_slot[0], by_slot[1]
        drow, dcol = self._depth(row.mask), self._depth(col.mask)
        if min(drow, dcol) != 0 or max(drow, dcol) == 0:
            return None
        g = self._gmask(v)
        mrow, mcol = self._node_mask(row, hel, self.memo), self._node_mask(col, hel, self.memo)
        left = bool((mcol & A) and (mrow & B) and (g & GL))
        right = bool((mcol & B) and (mrow & A) and (g & GR))
        if not (left or right):
            return None
        last = self.dg.last
        gl, gr = self._cpl(v.coup[0]), self._cpl(v.coup[1])
        if drow == 0:     # dress the row spinor; its L part lands in slots A (meets the column's slots A)
            base, fn, m_in = self._name(row, vi, hel), 'dress_row', mrow
            dmask = (A if left else 0) | (B if right else 0)
            other = col
        else:             # dress the column spinor; its L part lands in slots B (meets the row's slots B)
            base, fn, m_in = self._name(col, vi, hel), 'dress_col', mcol
            dmask = (B if left else 0) | (A if right else 0)
            other = row
        names = []
        for part, tag in ((0, 'zr'), (1, 'zi')):
            name = '%s_%s_%s' % (tag, base, (v.coup[0] or '0') + (v.coup[1] or '0'))
            if name not in self.shared:
                self._reg(name, 'Sp<T>', 0, mask=dmask)
                self._begin(0)
                expr = '%s<%d, %d, %d>(%s, %s, %s, %s)' % (fn, m_in, g, part, self._ref(base), self._ref('e%d' % last),
                                                          gl, gr)
                self.shared[name] = True
                self.shared_items.append(('def', name, expr, self.cur_loads))
            names.append(name)
        self._begin(k)
        o = self._ref(self._name(other, vi, hel))
        zr, zi = self._ref(names[0]), self._ref(names[1])
        return ['const cx<T> rb = sdot<%d>(%s, %s), ib = sdot<%d>(%s, %s);' % (dmask, zr, o, dmask, zi, o)]

    def _render_variant(self, var):
        dyn = self.dynamic
        k, levels = var['k'], var['levels']
        b = []
        ind = '  '
        b.append(ind + '{  // static helicities: ' +
                 ', '.join('%s(%d)=%+d' % (self.legs[l].name, l, h) for l, h in sorted(var['hel'].items())))
        ind += '  '
        if k == 0:
            b.append(ind + var['accdecl'])
        b += self._render_items(levels[0], ind)
        for d in range(1, k + 1):
            leg = dyn[d - 1]
            lg = self.legs[leg]
            nh = len(self.nhel[leg])
            b.append(ind + '#pragma unroll 1')
            if self.stage and d == k and nh == 2:
                # innermost loop: on the device its two iterations run in the two warps of a pair (st.lo/st.hi)
                b.append(ind + 'for (int h%d = st.lo(); h%d < st.hi(); ++h%d) {' % (leg, leg, leg))
            else:
                b.append(ind + 'for (int h%d = 0; h%d < %d; ++h%d) {' % (leg, leg, nh, leg))
            ind += '  '
            if self.stage:
                b.append(ind + 'st.sync();')
            b.append(ind + self._dyn_leaf_decl(lg))
            render = self._render_calls if var['calls'] else self._render_items
            if d == k and var['groups'] == 2:
                for g, items in enumerate(levels[d][0][1]):
                    b.append(ind + 'if (st.grp(%d)) {  // estimated %d flops' % (g, self.group_cost[g]))
                    b.append(ind + '  ' + var['accdecl'] % g)
                    body = render(items, ind + '  ')
                    assert not any('st.sync' in ln for ln in body), 'block barrier under st.grp()'
                    b += body
                    b.append(ind + '}')
            elif d == k:
                b.append(ind + var['accdecl'])
                b += render(levels[d], ind)
            else:
                b += self._render_shared(levels[d], ind)
        for line in var['tail']:
            b.append(ind + line)
        for d in range(k):
            ind = ind[:-2]
            b.append(ind + '}')
        ind = ind[:-2]
        b.append(ind + '}')
        return b

    def _dyn_leaf_decl(self, lg):
        p = lg.particle
        i = lg.index
        if p.spin == 'V' and not p.mass:
            lc = ' const Pol<T> y%d = to_pol(x%d);' % (i, i) if (self.POL_LC and self.stage) else ''
            if self.stage:
                return 'const Vc<T> x%d = ld_pol<T>(st, %s, h%d);%s' % (i, self._slot(self.vals['e%d' % i]), i, lc)
            return 'const Vc<T> x%d = h%d ? vflip(e%d) : e%d;%s' % (i, i, i, i, lc)
        if p.spin == 'V':
            nsv = -1 if lg.state == 'in' else 1
            return 'const Vc<T> x%d = vxxxxx<T>(p[%d], c.%s, h%d - 1, %d);' % (i, i, p.mass, i, nsv)
        if p.spin == 'F':
            fn = 'oxxxxx' if p.is_anti else 'ixxxxx'
            return 'const Sp<T> x%d = %s<T>(p[%d], c.%s, 2 * h%d - 1, %d);' % (i, fn, i, p.mass, i, self._nsf(lg))
        return 'const cx<T> x%d = sxxxxx<T>();' % i

    # ------------------------------------------------------------------ per-event, helicity independent part
    def _preamble(self):
        """Items of loop depth 0: momenta of internal lines, invariants, propagator factors, eps(+1) of looped legs."""
        self._begin(0)
        L = []
        raw = lambda t: L.append(('raw', t))

        def define(name, ctype, expr, cheap=False):
            self._reg(name, ctype, 0)
            if cheap:   # a few adds / one reciprocal: evaluated by both warps of a pair (see _render_shared)
                self.dup_names.add(name)
            L.append(('def', name, expr, []))

        n = self.dg.n
        sgn = {l.index: (1 if l.state == 'in' else -1) for l in self.legs}
        for l in sorted(self.need_P):
            define('P%d' % l, 'Mom<T>', 'p[%d]' % l, cheap=True)
        # momenta of sub-sets (all-incoming: initial +p, final -p)
        have = {}
        for m in sorted(self.need_K, key=lambda m: (_popcount(m), m)):
            self._emit_K(m, have, define, sgn)
        # invariants
        pairs = set()
        q2 = {}
        for (m, mass, width, spin), name in sorted(self.need_d.items()):
            if m not in q2:
                use = m if _popcount(m) <= n - _popcount(m) else (self.dg.full & ~m)
                q2[m] = use
                ls = list(bits(use))
                for a in range(len(ls)):
                    for b2 in range(a + 1, len(ls)):
                        pairs.add((ls[a], ls[b2]))
        units = sorted({l for pr in pairs for l in pr if not self.legs[l].particle.mass})
        for l in units:
            define('n%d' % l, 'Mom<T>', 'unit0(p[%d])' % l, cheap=True)
        for (a, b2) in sorted(pairs):
            s = '' if sgn[a] * sgn[b2] > 0 else '-'
            if not self.legs[a].particle.mass and not self.legs[b2].particle.mass:
                define('t%d_%d' % (a, b2), 'T', '%stwo_dot0(n%d, n%d)' % (s, a, b2), cheap=True)
            else:
                define('t%d_%d' % (a, b2), 'T', '%sT(2) * mdot(p[%d], p[%d])' % (s, a, b2), cheap=True)
        for m, use in sorted(q2.items()):
            ls = list(bits(use))
            terms = ['t%d_%d' % (ls[a], ls[b2]) for a in range(len(ls)) for b2 in range(a + 1, len(ls))]
            for l in ls:
                if self.legs[l].particle.mass:
                    terms.append('c.%s * c.%s' % (self.legs[l].particle.mass, self.legs[l].particle.mass))
            define('q2_%d' % m, 'T', ' + '.join(terms), cheap=True)
        for mass in sorted(self.need_rm2):
            # 1 / m_V^2, or 1 / (m_V^2 - i m_V Gamma_V) in the complex-mass option (c.cms = 1)
            width = {'mw': 'ww', 'mz': 'wz'}.get(mass)
            if width:
                define('rm2_%s' % mass, 'cx<T>', 'crcp(c.%s * c.%s, -(c.cms * c.%s * c.%s))' % (mass, mass, mass, width),
                       cheap=True)
            else:
                define('rm2_%s' % mass, 'cx<T>', 'mk<T>(hrcp(c.%s * c.%s), T(0))' % (mass, mass), cheap=True)
        for (m, mass, width, spin), name in sorted(self.need_d.items()):
            sign = '' if spin == 'V' else '-'
            den = 'q2_%d' % m if not mass else '(q2_%d - c.%s * c.%s)' % (m, mass, mass)
            if width:
                define(name, 'cx<T>', '%scrcp(%s, c.%s * c.%s)' % (sign, den, mass, width))
            else:
                define(name, 'T', '%shrcp(%s)' % (sign, den))
        for ratio in sorted(self.need_ratio):
            define(ratio, 'T', 'c.%s * hrcp(c.mgs)' % ratio.split('_')[1], cheap=True)
        # scaled light-cone momenta of massless single-chirality fermion lines
        for name, (m, neg, coup, dname) in sorted(self.need_Q.items()):
            define(name, 'Mom<T>', 'lc_scaled(K%d, %sc.%s * %s)' % (m, '-' if neg else '', coup, dname))
        # polarisation vectors of looped massless vector legs (helicity +1; -1 by vflip)
        for l in self.dynamic:
            lg = self.legs[l]
            if lg.particle.spin == 'V' and not lg.particle.mass:
                define('e%d' % l, 'pol', 'vxxxxx<T>(p[%d], T(0), 1, %d)' % (l, -1 if lg.state == 'in' else 1))
        return L

    def _emit_K(self, m, have, define, sgn):
        if m in have:
            return
        hi = max(bits(m))
        rest = m & ~(1 << hi)
        if rest == 0:
            define('K%d' % m, 'Mom<T>', '%sp[%d]' % ('' if sgn[hi] > 0 else '-', hi), cheap=True)
        else:
            self._emit_K(rest, have, define, sgn)
            define('K%d' % m, 'Mom<T>', 'K%d %s p[%d]' % (rest, '+' if sgn[hi] > 0 else '-', hi), cheap=True)
        have[m] = True


def _lit(fr):
    """Fraction -> C literal with full double precision."""
    return repr(float(fr))
