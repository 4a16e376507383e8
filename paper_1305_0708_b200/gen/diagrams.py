"""Tree-diagram enumeration from the SM vertex set, with shared sub-currents (step a0).

Role of MG2CUDA's input stage (section 5.1-5.2): the paper converts MadGraph's `matrix.f`
(a HELAS call sequence) to HEGET calls.  No `matrix.f` exists here, so the diagrams are enumerated directly:
every subtree over a subset of the external legs is built once (memoised) and shared by all diagrams that
contain it -- the same wavefunction sharing MadGraph's call sequence has.

A subtree ("Node") delivers an off-shell field to its parent vertex; its value is the product of a vertex
function and a propagator (an off-shell HEGET function).  A diagram ("Root") is a vertex whose
children cover all legs; its value is an amplitude function.  Four-gluon vertices are split into their three
colour structures (C.47-C.52), each a node / root of its own.
"""
import itertools
from dataclasses import dataclass, field as dc_field

from . import colour as C
from .model import PARTICLES, VERTICES, anti


@dataclass
class Leg:
    index: int
    name: str       # physical particle name as written in the process
    state: str      # 'in' | 'out'
    field: str      # all-incoming field

    @property
    def particle(self):
        return PARTICLES[self.field]


@dataclass(eq=False)
class Node:
    uid: int
    mask: int                 # bit set of external legs
    field: str                # field delivered to the parent (all-incoming, as the parent vertex sees it)
    vertex: object = None     # None for a leaf
    children: tuple = ()      # in the slot order of `slots`
    slots: tuple = ()         # vertex slot index of each child
    out_slot: int = -1        # vertex slot of the delivered (propagating) field
    struct: int = 0           # 1..3 for the colour structures of a four-gluon vertex
    colour: object = None
    leg: int = -1             # leaf only
    members: tuple = ()       # sum node: the currents added up (= children), with relative signs msigns
    msigns: tuple = ()

    @property
    def is_leaf(self):
        return self.vertex is None and not self.members

    @property
    def is_sum(self):
        return bool(self.members)

    @property
    def particle(self):
        return PARTICLES[self.field]

    @property
    def wtype(self):
        p = self.particle
        if p.spin == 'F':
            return 'row' if p.is_anti else 'col'
        return 'vec' if p.spin == 'V' else 'sca'


@dataclass(eq=False)
class Root:
    uid: int
    vertex: object
    children: tuple
    slots: tuple
    struct: int
    colour: object            # Col('line' or 'none')
    topo: int                 # index of the topological diagram this term belongs to


@dataclass
class ProcessSpec:
    name: str
    pid: int
    initial: list
    final: list
    decays: list = dc_field(default_factory=list)   # [(particle name, (leg indices))]
    last: int = -1                                  # leg used to close the diagrams (-1: choose)


def bits(mask):
    i = 0
    while mask:
        if mask & 1:
            yield i
        mask >>= 1
        i += 1


def _partitions(items, nparts):
    items = tuple(items)
    if nparts == 1:
        yield (items,)
        return
    first, rest = items[0], items[1:]
    for r in range(0, len(rest) - nparts + 2):
        for extra in itertools.combinations(rest, r):
            g1 = (first,) + extra
            left = tuple(x for x in rest if x not in extra)
            for sub in _partitions(left, nparts - 1):
                yield (g1,) + sub


def _mask(legs):
    m = 0
    for l in legs:
        m |= 1 << l
    return m


def _match(vertex, fields):
    """Assign the given child fields to distinct slots of `vertex`; return (slots, remaining slots) or None.
    Identical fields take slots in increasing order (children are given in canonical order)."""
    free = list(range(len(vertex.fields)))
    slots = []
    for f in fields:
        for s in free:
            if vertex.fields[s] == f:
                slots.append(s)
                free.remove(s)
                break
        else:
            return None
    return tuple(slots), tuple(free)


class Diagrams:
    def __init__(self, spec, merge=False):
        """merge=True: off-shell currents over the same legs with the same field and the same colour structure (up
        to a sign) are added into one current before they are used -- by linearity every vertex that would be
        evaluated once per member is evaluated once for the sum (e.g. the W emitted before or after a gluon on the
        quark line).  The amplitude is unchanged; the diagram COUNTS are those of the unmerged enumeration."""
        self.spec = spec
        self.merge = merge
        self.legs = []
        for nm in spec.initial:
            self.legs.append(Leg(len(self.legs), nm, 'in', nm))
        for nm in spec.final:
            self.legs.append(Leg(len(self.legs), nm, 'out', anti(nm)))
        self.n = len(self.legs)
        self.full = (1 << self.n) - 1
        self.decays = [(nm, _mask(ls)) for nm, ls in spec.decays]
        self._uid = 0
        self.nodes = []
        self.roots = []
        self.n_topo = 0

    # ------------------------------------------------------------------ decay-chain constraint (reading A13)
    def _line_ok(self, mask, fld):
        comp = self.full & ~mask
        for nm, d in self.decays:
            inter = mask & d
            if not (inter == 0 or inter == mask or inter == d or (comp & ~d) == 0):
                return False
            if (mask == d or comp == d) and fld not in (nm, anti(nm)):
                return False
        return True

    def _merge(self, m, nodes):
        groups = {}
        for nd in nodes:
            key = (nd.field,) + nd.colour.key()
            groups.setdefault(key, []).append(nd)
        out = []
        for key, grp in groups.items():
            # split the group into classes of proportional colour (ratio +-1)
            classes = []
            for nd in grp:
                for cl in classes:
                    ref = cl[0][0].colour.terms
                    ratios = {nd.colour.terms[w] / ref[w] for w in ref}
                    if len(ratios) == 1 and abs(next(iter(ratios))) == 1:
                        cl.append((nd, int(next(iter(ratios)))))
                        break
                else:
                    classes.append([(nd, 1)])
            for cl in classes:
                if len(cl) == 1:
                    out.append(cl[0][0])
                else:
                    mem = tuple(nd for nd, _ in cl)
                    out.append(self._new_node(mask=m, field=mem[0].field, children=mem, members=mem,
                                              msigns=tuple(sg for _, sg in cl), colour=mem[0].colour))
        return out

    def _new_node(self, **kw):
        nd = Node(uid=self._uid, **kw)
        self._uid += 1
        self.nodes.append(nd)
        return nd

    # ------------------------------------------------------------------ colour of a vertex application
    @staticmethod
    def _vertex_colour(vertex, slots, cols, struct):
        """Colour object of the remaining slot (or of the closed amplitude if all slots are filled)."""
        by_slot = dict(zip(slots, cols))
        nslot = len(vertex.fields)
        if vertex.colour == '1':
            return C.singlet(cols)
        if vertex.colour == 'T':  # slots: 0 row, 1 column, 2 gluon
            return C.qqg(by_slot.get(1), by_slot.get(0), by_slot.get(2))
        if vertex.colour == 'f':
            if len(cols) == 2:  # cyclic: the pair in cyclic order (s, s+1) -> free slot s+2
                free = [s for s in range(3) if s not in by_slot][0]
                a, b = by_slot[(free + 1) % 3], by_slot[(free + 2) % 3]
                return C.f3(a, b)
            x = C.f3(by_slot[0], by_slot[1])
            return C.contract(x, by_slot[2])
        if vertex.colour == 'ff':
            # children occupy slots in order (A, B, C[, D]); structure s: see DESIGN.md "four-gluon vertex"
            vals = [by_slot[s] for s in sorted(by_slot)]
            a, b, c = vals[0], vals[1], vals[2]
            trip = {1: (a, b, c), 2: (a, c, b), 3: (b, c, a)}[struct]
            x = C.f3(C.f3(trip[0], trip[1]), trip[2])
            if len(vals) == 3:
                return x
            return C.contract(x, vals[3])
        raise ValueError(vertex.colour)

    def _leaf_colour(self, leg):
        p = leg.particle
        if p.colour == 8:
            return C.leaf('adj', leg.index)
        if abs(p.colour) == 3:
            return C.leaf('row' if p.is_anti else 'col', leg.index)
        return C.leaf('none')

    # ------------------------------------------------------------------ enumeration
    def build(self, last):
        self.last = last
        others = tuple(i for i in range(self.n) if i != last)
        memo = {}

        def subtrees(legs):
            m = _mask(legs)
            if m in memo:
                return memo[m]
            res = []
            if len(legs) == 1:
                lg = self.legs[legs[0]]
                res.append(self._new_node(mask=m, field=lg.field, leg=lg.index, colour=self._leaf_colour(lg)))
            else:
                for npart in (2, 3):
                    if len(legs) < npart:
                        continue
                    for groups in _partitions(legs, npart):
                        lists = [subtrees(g) for g in groups]
                        for combo in itertools.product(*lists):
                            fields = [nd.field for nd in combo]
                            for v in VERTICES:
                                if len(v.fields) != npart + 1:
                                    continue
                                mt = _match(v, fields)
                                if mt is None:
                                    continue
                                slots, free = mt
                                out_field = anti(v.fields[free[0]])
                                if not self._line_ok(m, out_field):
                                    continue
                                for struct in ((1, 2, 3) if v.kind == 'VVVV' else (0,)):
                                    try:
                                        col = self._vertex_colour(v, slots, [nd.colour for nd in combo], struct)
                                    except ValueError:
                                        continue
                                    if not col.terms:
                                        continue
                                    res.append(self._new_node(mask=m, field=out_field, vertex=v, children=combo,
                                                              slots=slots, out_slot=free[0], struct=struct,
                                                              colour=col))
            if self.merge and len(res) > 1:
                res = self._merge(m, res)
            memo[m] = res
            return res

        lastleaf = self._new_node(mask=1 << last, field=self.legs[last].field, leg=last,
                                  colour=self._leaf_colour(self.legs[last]))
        for npart in (2, 3):
            if len(others) < npart:
                continue
            for groups in _partitions(others, npart):
                lists = [subtrees(g) for g in groups]
                for combo in itertools.product(*lists):
                    kids = tuple(combo) + (lastleaf,)
                    # canonical child order: by lowest leg, so identical-field slots are filled consistently
                    kids = tuple(sorted(kids, key=lambda nd: min(bits(nd.mask))))
                    fields = [nd.field for nd in kids]
                    for v in VERTICES:
                        if len(v.fields) != npart + 1:
                            continue
                        mt = _match(v, fields)
                        if mt is None or mt[1]:
                            continue
                        topo = None
                        for struct in ((1, 2, 3) if v.kind == 'VVVV' else (0,)):
                            try:
                                col = C.closed_flow(self._vertex_colour(v, mt[0], [nd.colour for nd in kids],
                                                                        struct))
                            except ValueError:
                                continue
                            if not col.terms:
                                continue
                            if topo is None:
                                topo = self.n_topo
                                self.n_topo += 1
                            self.roots.append(Root(uid=len(self.roots), vertex=v, children=kids, slots=mt[0],
                                                   struct=struct, colour=col, topo=topo))
        self._prune()
        return self

    def _prune(self):
        """Keep only nodes reachable from a root."""
        keep = set()

        def visit(nd):
            if nd.uid in keep:
                return
            keep.add(nd.uid)
            for ch in nd.children:
                visit(ch)

        for r in self.roots:
            for ch in r.children:
                visit(ch)
        self.nodes = [nd for nd in self.nodes if nd.uid in keep]

    # ------------------------------------------------------------------ counting
    def n_topological(self):
        """Number of Feynman diagrams: each root term expands into the product of its children's four-gluon
        structure choices; a topological diagram is counted once for all of them."""

        def shape(nd):
            if nd.is_leaf:
                return ('L', nd.leg)
            return (nd.field, id(nd.vertex), tuple(sorted(shape(c) for c in nd.children)))

        shapes = set()
        for r in self.roots:
            shapes.add((id(r.vertex), tuple(sorted(shape(c) for c in r.children))))
        return len(shapes)

    def n_amplitudes(self):
        return len(self.roots)

    def flows(self):
        """Sorted list of colour words appearing in any amplitude."""
        ws = set()
        for r in self.roots:
            ws.update(r.colour.terms.keys())
        return sorted(ws)
