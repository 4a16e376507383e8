"""Tree-level Feynman diagrams, one by one, with textbook Feynman rules (oracle; test infrastructure).

What is computed (Eq. 4 and Eq. 6):

    |Mbar|^2 = 1/(2*2) * 1/(n_a n_b) * 1/S_ident * sum_lambda sum_colours | sum_diagrams M |^2

How (plain definition, nothing shared with the CUDA path):
  * every tree diagram that can be built from the process' vertex list is enumerated
    explicitly (a diagram = nested tuple of vertices);
  * each diagram is evaluated on its own, from its leaves up, by explicit 4x4 Dirac-matrix /
    Lorentz-tensor contraction with the textbook rules below, every factor of i kept;
  * the colour factor of each diagram is an explicit tensor over the external colour indices
    (quarks 1..3, gluons 1..8) built from Gell-Mann T^a and f^{abc}; the colour
    sum is the brute-force index sum  CM[l,l'] = sum_{ext colours} c_l conj(c_l');
  * all helicity combinations are summed (2 per external leg), no zero skipping.

Feynman rules (all momenta incoming at a vertex; derived from the paper's Lagrangians):
  FFV   Eq. 35   i gamma^mu (gL PL + gR PR)
  qqg   Eq. 36   -i g_s gamma^mu T^a_{ji}      (gL = gR = -g_s, colour T^a)
  ggg   Eq. 42   -g_s f^{abc} [ g^{mu nu}(k1-k2)^rho + g^{nu rho}(k2-k3)^mu + g^{rho mu}(k3-k1)^nu ]
  gggg  Eq. 48   -i g_s^2 [ f^{abe}f^{cde}(g^{mu rho}g^{nu sigma}-g^{mu sigma}g^{nu rho})
                                          + f^{ace}f^{bde}(g^{mu nu}g^{rho sigma}-g^{mu sigma}g^{nu rho})
                                          + f^{ade}f^{bce}(g^{mu nu}g^{rho sigma}-g^{mu rho}g^{nu sigma}) ]
  FFS   Eq. 39   i (gL PL + gR PR)             t t H: gL = gR = -m_t / v
  VVS   Eq. 50   i g g^{mu nu}                   W W H: g_W m_W,  Z Z H: g_Z m_Z   (v = 2 m_W / g_W)
  VVSS  Eq. 51   i g g^{mu nu}                   W W H H: g_W^2 / 2,  Z Z H H: g_Z^2 / 2
  SSS   Eq. 52   i g                             H H H: -3 m_H^2 / v
        (the coefficients are those of the Feynman rules that follow from |D Phi|^2, the Higgs potential and the
        Yukawa term with Phi = (0, (v + H)/sqrt2); the scalar wavefunction is 1, Eq. 34)
  propagators (widths PAPER.md:1591, 1637; reading SURVEY 8c-A4):
        fermion  i (pslash + m) / (p^2 - m^2 + i m Gamma)
        massless vector (Feynman gauge)  -i g_{mu nu} / q^2
        massive vector (unitary gauge)   -i (g_{mu nu} - q_mu q_nu / m^2) / (q^2 - m^2 + i m Gamma)
        scalar   i / (q^2 - m^2 + i m Gamma)
"""
import itertools
import numpy as np

from . import dirac as D
from . import su3
from . import sm

# ----------------------------------------------------------------------------- fields
# name: (spin, colour dimension, mass key, width key, antiparticle)
_F = {}


def _add(name, spin, col, mkey, wkey, anti):
    _F[name] = (spin, col, mkey, wkey, anti)
    if anti != name:
        _F[anti] = (spin, col, mkey, wkey, name)


_add('u', 'F', 3, None, None, 'u~')
_add('d', 'F', 3, None, None, 'd~')
_add('t', 'F', 3, 'mt', 'gt', 't~')
_add('b', 'F', 3, 'mb', None, 'b~')
_add('e-', 'F', 1, None, None, 'e+')
_add('mu-', 'F', 1, None, None, 'mu+')
_add('ve', 'F', 1, None, None, 've~')
_add('vm', 'F', 1, None, None, 'vm~')
_add('g', 'V', 8, None, None, 'g')
_add('a', 'V', 1, None, None, 'a')
_add('z', 'V', 1, 'mz', 'gz', 'z')
_add('w+', 'V', 1, 'mw', 'gw', 'w-')
_add('h', 'S', 1, 'mh', 'gh', 'h')
PARTICLES = {'u', 'd', 't', 'b', 'e-', 'mu-', 've', 'vm'}  # fermion (not anti-fermion) names


def spin(f):
    return _F[f][0]


def coldim(f):
    return _F[f][1]


def anti(f):
    return _F[f][4]


def mass_width(f, par):
    mk, wk = _F[f][2], _F[f][3]
    if wk == 'gw':
        return par[mk], sm.effective_widths(par)[0]      # Eq. 56 in the complex-mass option
    return (par[mk] if mk else 0.0), (par[wk] if wk else 0.0)


def is_row(f):
    """An incoming anti-fermion line is a row spinor (psibar), an incoming fermion a column."""
    return spin(f) == 'F' and f not in PARTICLES


# ----------------------------------------------------------------------------- vertices
class Vertex:
    def __init__(self, kind, fields, **kw):
        self.kind = kind  # 'FFV', 'VVV', 'VVVV'
        self.fields = tuple(fields)  # all-incoming field names
        self.__dict__.update(kw)

    def __repr__(self):
        return 'V' + repr(self.fields)


def ffv(f1_out, f2_in, v_in, gl, gr):
    """L = psibar_F1 gamma^mu (gl PL + gr PR) psi_F2 V : fermion F2 absorbs V_in and leaves as F1."""
    return Vertex('FFV', (anti(f1_out), f2_in, v_in), row=anti(f1_out), col=f2_in, vec=v_in, gl=gl, gr=gr)


def build_vertices(par, names):
    """names: iterable of vertex keys, e.g. 'uug', 'udw', 'ggg', 'gggg', 'uua', 'eez' ..."""
    c = sm.couplings(par)
    gs = c['gs']
    # complex-mass option (Eq. 55): m_V -> mu_V = sqrt(m_V^2 - i m_V Gamma_V) in the couplings
    muw2, muz2 = sm.complex_masses(par)
    cms = bool(par.get('complex_mass'))
    mw_c = np.sqrt(muw2) if cms else par['mw']
    mz_c = np.sqrt(muz2) if cms else par['mz']
    vev = 2.0 * mw_c / c['gw']
    out = []
    for n in names:
        if n == 'ggg':
            out.append(Vertex('VVV', ('g', 'g', 'g'), g=gs))
        elif n == 'gggg':
            out.append(Vertex('VVVV', ('g', 'g', 'g', 'g'), g=gs))
        elif n in ('uug', 'ddg', 'ttg', 'bbg'):
            out.append(ffv(n[0], n[0], 'g', -gs, -gs))
        elif n in ('uua', 'dda', 'tta', 'bba', 'uuz', 'ddz', 'ttz', 'bbz'):
            gl, gr = c[(n[2], n[0])]
            out.append(ffv(n[0], n[0], n[2], gl, gr))
        elif n in ('eea', 'eez', 'mma', 'mmz'):
            f = {'e': 'e-', 'm': 'mu-'}[n[0]]
            gl, gr = c[(n[2], f)]
            out.append(ffv(f, f, n[2], gl, gr))
        elif n in ('udw', 'tbw', 'enw', 'mnw'):
            up, dn = {'udw': ('u', 'd'), 'tbw': ('t', 'b'), 'enw': ('ve', 'e-'), 'mnw': ('vm', 'mu-')}[n]
            gl, gr = c['w']
            out.append(ffv(up, dn, 'w+', gl, gr))  # dn + W+ -> up
            out.append(ffv(dn, up, 'w-', gl, gr))  # up + W- -> dn   (hermitian conjugate, real coupling)
        elif n == 'tth':
            y = -par['mt'] / vev
            out.append(Vertex('FFS', ('t~', 't', 'h'), row='t~', col='t', sca='h', gl=y, gr=y))
        elif n == 'wwh':
            out.append(Vertex('VVS', ('w-', 'w+', 'h'), g=c['gw'] * mw_c))
        elif n == 'zzh':
            out.append(Vertex('VVS', ('z', 'z', 'h'), g=c['gz'] * mz_c))
        elif n == 'wwhh':
            out.append(Vertex('VVSS', ('w-', 'w+', 'h', 'h'), g=0.5 * c['gw'] ** 2))
        elif n == 'zzhh':
            out.append(Vertex('VVSS', ('z', 'z', 'h', 'h'), g=0.5 * c['gz'] ** 2))
        elif n == 'hhh':
            out.append(Vertex('SSS', ('h', 'h', 'h'), g=-3.0 * par['mh'] ** 2 / vev))
        else:
            raise ValueError(n)
    return out


# ----------------------------------------------------------------------------- diagrams
class Leaf:
    def __init__(self, leg, field):
        self.leg, self.field, self.legs = leg, field, (leg,)
        self.sig = 'L%d' % leg


class Node:
    """vertex + children; `field` = the off-shell field this subtree delivers to its parent vertex."""

    def __init__(self, vertex, children, field):
        self.vertex, self.children, self.field = vertex, children, field
        self.legs = tuple(sorted(l for ch in children for l in ch.legs))
        # structural name of the subtree: equal subtrees of different diagrams have equal names (used only to
        # avoid evaluating the same sub-diagram twice, see kin_terms)
        self.sig = '(%s|%s:%s)' % (field, ','.join(vertex.fields), ' '.join(ch.sig for ch in children))


def _grow(shape, leg):
    """All shapes obtained from `shape` by attaching `leg`.  A shape is what hangs below a line: an external leg
    (an int) or a vertex (a tuple of the shapes below its 2 or 3 other lines).  The new leg goes on the line above
    `shape` (a new three-point vertex), on a three-point vertex (making it a four-point vertex), or anywhere
    further down."""
    yield (shape, leg)
    if isinstance(shape, tuple):
        if len(shape) == 2:
            yield shape + (leg,)
        for i, sub in enumerate(shape):
            for g in _grow(sub, leg):
                yield shape[:i] + (g,) + shape[i + 1:]


def topologies(n):
    """All tree topologies with n labelled external legs and vertices of degree 3 and 4, hung from leg n-1, by the
    textbook recursion: the topologies with one more leg are obtained by attaching the new leg to every line
    (external lines included) and to every three-point vertex.  Removing that leg again undoes exactly one such
    step, so every topology is produced once: 1, 4, 25, 220, 2485, 34300 for n = 3 .. 8."""
    shapes = [(0, 1)]
    for leg in range(2, n - 1):
        shapes = [g for s in shapes for g in _grow(s, leg)]
    return shapes


def _vertex_tables(vertices):
    """closed[sorted fields] = vertex;  open_[sorted fields but one] = [(vertex, the missing field), ...]."""
    closed, open_ = {}, {}
    for v in vertices:
        closed[tuple(sorted(v.fields))] = v
        for f in set(v.fields):
            rest = list(v.fields)
            rest.remove(f)
            open_.setdefault(tuple(sorted(rest)), []).append((v, f))
    return closed, open_


def enumerate_diagrams(ext_fields, vertices):
    """All tree diagrams for external all-incoming fields `ext_fields` (Eq. 6: the sum runs over
    "all Feynman diagrams of the subprocess").

    Two steps: (1) every topology of `topologies(n)`; (2) every way of putting fields of the model on its internal
    lines such that each point is a vertex of the model: going through the topology from the outside inwards, the
    fields arriving at a point fix, through the vertex table, the fields the point can send on; the point that
    carries the last leg must close.

    Returns a list of root Nodes whose children include Leaf(n-1) as the LAST child."""
    n = len(ext_fields)
    closed, open_ = _vertex_tables(vertices)

    def dressed(shape):
        if not isinstance(shape, tuple):
            return [Leaf(shape, ext_fields[shape])]
        parts = []
        for sub in shape:
            d = dressed(sub)
            if not d:
                return []
            parts.append(d)
        found = []
        for kids in itertools.product(*parts):
            for v, missing in open_.get(tuple(sorted(t.field for t in kids)), ()):
                found.append(Node(v, list(kids), anti(missing)))
        return found

    last = Leaf(n - 1, ext_fields[n - 1])
    roots = []
    for top in topologies(n):
        parts = [dressed(sub) for sub in top]
        if all(parts):
            for kids in itertools.product(*parts):
                v = closed.get(tuple(sorted([t.field for t in kids] + [last.field])))
                if v is not None:
                    roots.append(Node(v, list(kids) + [last], None))
    return roots


def n_colour_terms(tree):
    """Number of (kinematic, colour) terms a diagram splits into (3 per four-gluon vertex)."""
    if isinstance(tree, Leaf):
        return 1
    n = 3 if tree.vertex.kind == 'VVVV' else 1
    for ch in tree.children:
        n *= n_colour_terms(ch)
    return n


# ----------------------------------------------------------------------------- colour
_OWN = 20  # einsum label of a subtree's own colour index; inner labels 21..


def _ffv_colour(v):
    nf, nv = coldim(v.col), coldim(v.vec)
    if nf == 3 and nv == 8:
        return np.transpose(su3.T, (1, 2, 0)).copy()  # c[j,i,a] = T^a_{ji}
    if nf == 3 and nv == 1:
        return np.eye(3, dtype=complex)[:, :, None]
    if nf == 1 and nv == 1:
        return np.ones((1, 1, 1), dtype=complex)
    raise ValueError('colour structure')


def _vertex_colour_tensors(v):
    """List of (tensor, axis roles).  FFV axes (row j, col i, vec a); VVV (a,b,c); VVVV (a,b,c,d) x3."""
    if v.kind == 'FFV':
        return [_ffv_colour(v)]
    if v.kind == 'FFS':
        return [np.eye(coldim(v.col), dtype=complex)[:, :, None]]
    if v.kind in ('VVS', 'VVSS', 'SSS'):
        return [np.ones((1,) * len(v.fields), dtype=complex)]
    f = su3.F.astype(complex)
    if v.kind == 'VVV':
        return [f]
    return [np.einsum('abe,cde->abcd', f, f), np.einsum('ace,bde->abcd', f, f), np.einsum('ade,bce->abcd', f, f)]


def _slot_order(v, child_fields):
    """Map children (and the remaining line) to the vertex tensor's axes.

    Returns (axes of the children, axis of the remaining line)."""
    if v.kind in ('FFV', 'FFS'):
        roles = {v.row: 0, v.col: 1, (v.vec if v.kind == 'FFV' else v.sca): 2}
        ax = [roles[f] for f in child_fields]
        rem = [a for a in (0, 1, 2) if a not in ax]
        return ax, (rem[0] if rem else None)
    k = len(child_fields)
    return list(range(k)), (k if k < len(v.fields) else None)


def colour_terms(tree):
    """List of colour tensors, axes = [own] + sorted external legs of the subtree."""
    if isinstance(tree, Leaf):
        return [np.eye(coldim(tree.field), dtype=complex)]
    v = tree.vertex
    chs = tree.children
    ax, rem = _slot_order(v, [c.field for c in chs])
    out = []
    child_lists = [colour_terms(c) for c in chs]
    out_legs = list(tree.legs)
    for combo in itertools.product(*child_lists):
        for ct in _vertex_colour_tensors(v):
            labels = [0] * ct.ndim
            for i, a in enumerate(ax):
                labels[a] = _OWN + 1 + i
            if rem is not None:
                labels[rem] = _OWN
            args = [ct, labels]
            for i, (c, cv) in enumerate(zip(chs, combo)):
                if isinstance(c, Leaf):
                    args += [cv, [_OWN + 1 + i, c.leg]]
                else:
                    args += [cv, [_OWN + 1 + i] + list(c.legs)]
            res_labels = ([_OWN] if rem is not None else []) + out_legs
            out.append(np.einsum(*args, res_labels))
    return out


# ----------------------------------------------------------------------------- kinematics
class Kinematics:
    """External momenta (all-incoming convention) and wavefunctions for one batch of events."""

    def __init__(self, process, p, par):
        # p: [N, n_ext, 4] physical momenta (E>0); process.legs: list of (name, 'in'|'out')
        self.par = par
        self.n = p.shape[0]
        self.k = []  # all-incoming momenta
        self.fields = process.ext_fields
        self.wf = {}
        for i, (name, state) in enumerate(process.legs):
            pi = p[:, i, :]
            self.k.append(pi if state == 'in' else -pi)
            m, _ = mass_width(name, par)
            s = spin(name)
            for lam in process.helicities(i):
                if s == 'F':
                    is_part = name in PARTICLES
                    if state == 'in':
                        w = D.u_spinor(pi, m, lam) if is_part else D.bar(D.v_spinor(pi, m, lam))
                    else:
                        w = D.bar(D.u_spinor(pi, m, lam)) if is_part else D.v_spinor(pi, m, lam)
                elif s == 'S':
                    w = np.ones(self.n, dtype=complex)
                else:
                    e = D.polvec(pi, m, lam)
                    w = e if state == 'in' else np.conj(e)
                self.wf[(i, lam)] = w

    def momentum(self, legs):
        return sum(self.k[l] for l in legs)


def _gamma_coupling(v):
    """gamma^mu (gL PL + gR PR) as [4(mu),4,4]."""
    return np.einsum('mab,bc->mac', D.GAM, v.gl * D.PL + v.gr * D.PR)


def _vslash_coupled(v, vec):
    """V_mu gamma^mu (gL PL + gR PR): [N,4,4] for vec = V^mu [N,4]."""
    return np.einsum('nm,mab->nab', vec * D.METRIC, _gamma_coupling(v))


def _vertex_currents(v, child_fields, child_vals, child_moms):
    """Unpropagated current(s) on the remaining line of vertex v, = (i x Lagrangian vertex) contracted
    with the children.  One entry per colour structure of the vertex."""
    if v.kind == 'FFV':
        vals = dict(zip(child_fields, child_vals))
        if v.row in vals and v.col in vals:  # -> vector J^mu = psibar i gamma^mu (..) psi
            G = _gamma_coupling(v)
            return [1j * np.einsum('na,mab,nb->nm', vals[v.row], G, vals[v.col])]
        if v.col in vals:  # column continues: i Vslash (..) psi
            return [1j * np.einsum('nab,nb->na', _vslash_coupled(v, vals[v.vec]), vals[v.col])]
        return [1j * np.einsum('na,nab->nb', vals[v.row], _vslash_coupled(v, vals[v.vec]))]
    if v.kind == 'FFS':
        vals = dict(zip(child_fields, child_vals))
        G = v.gl * D.PL + v.gr * D.PR
        if v.row in vals and v.col in vals:  # -> scalar
            return [1j * np.einsum('na,ab,nb->n', vals[v.row], G, vals[v.col])]
        if v.col in vals:
            return [1j * vals[v.sca][:, None] * np.einsum('ab,nb->na', G, vals[v.col])]
        return [1j * vals[v.sca][:, None] * np.einsum('na,ab->nb', vals[v.row], G)]
    if v.kind in ('VVS', 'VVSS', 'SSS'):
        vecs = [x for f, x in zip(child_fields, child_vals) if spin(f) == 'V']
        scas = [x for f, x in zip(child_fields, child_vals) if spin(f) == 'S']
        c = 1j * v.g
        for x in scas:
            c = c * x
        nvec = sum(1 for f in v.fields if spin(f) == 'V')
        if len(vecs) == nvec == 2:      # both vectors given -> scalar line (or closed on a scalar)
            return [c * D.mdot(vecs[0], vecs[1])]
        if nvec == 2:                   # one vector given -> the other vector, index raised by g^{mu nu}
            return [c[:, None] * vecs[0]] if np.ndim(c) else [c * vecs[0]]
        return [c if np.ndim(c) else c * np.ones(child_vals[0].shape[0], dtype=complex)]  # SSS
    if v.kind == 'VVV':
        v1, v2 = child_vals
        k1, k2 = child_moms
        k3 = -(k1 + k2)
        j = (D.mdot(v1, v2)[:, None] * (k1 - k2) + v2 * D.mdot(k2 - k3, v1)[:, None]
             + v1 * D.mdot(k3 - k1, v2)[:, None])
        return [-v.g * j]
    v1, v2, v3 = child_vals
    d12, d13, d23 = D.mdot(v1, v2)[:, None], D.mdot(v1, v3)[:, None], D.mdot(v2, v3)[:, None]
    c = -1j * v.g ** 2
    return [c * (d13 * v2 - d23 * v1), c * (d12 * v3 - d23 * v1), c * (d12 * v3 - d13 * v2)]


def _propagate(field, K, cur, par):
    """Attach the propagator of the line that delivers `field` (incoming to the parent) with momentum K."""
    m, w = mass_width(field, par)
    den = D.mdot(K, K) - m * m + 1j * m * w
    s = spin(field)
    if s == 'S':
        return 1j * cur / den
    if s == 'V':
        if m == 0.0:
            return -1j * cur / den[:, None]
        m2 = m * m
        if par.get('complex_mass'):       # Eq. 55 also in the q q / m_V^2 term
            m2 = m * m - 1j * m * w
        return -1j * (cur - K * (D.mdot(K, cur) / m2)[:, None]) / den[:, None]
    if not is_row(field):  # column spinor, fermion number flows with K
        num = D.slash(K) + m * D.ONE4
        return 1j * np.einsum('nab,nb->na', num, cur) / den[:, None]
    num = -D.slash(K) + m * D.ONE4  # row spinor, fermion number flows against K
    return 1j * np.einsum('na,nab->nb', cur, num) / den[:, None]


def kin_terms(tree, hel, kin, memo=None):
    """List of kinematic values (same term order as colour_terms) for helicity assignment `hel`."""
    if isinstance(tree, Leaf):
        return [kin.wf[(tree.leg, hel[tree.leg])]]
    key = None
    if memo is not None:
        key = (tree.sig, tuple(hel[l] for l in tree.legs))
        if key in memo:
            return memo[key]
    v = tree.vertex
    chs = tree.children
    lists = [kin_terms(c, hel, kin, memo) for c in chs]
    moms = [kin.momentum(c.legs) for c in chs]
    fields = [c.field for c in chs]
    K = kin.momentum(tree.legs)
    out = []
    for combo in itertools.product(*lists):
        for cur in _vertex_currents(v, fields, list(combo), moms):
            out.append(_propagate(tree.field, K, cur, kin.par))
    if memo is not None:
        memo[key] = out
    return out


def root_amplitudes(root, hel, kin, memo=None):
    """Amplitude terms of one full diagram: vertex current from all children but the last,
    contracted with the last external wavefunction."""
    chs = root.children[:-1]
    last = root.children[-1]
    v = root.vertex
    lists = [kin_terms(c, hel, kin, memo) for c in chs]
    moms = [kin.momentum(c.legs) for c in chs]
    fields = [c.field for c in chs]
    wl = kin.wf[(last.leg, hel[last.leg])]
    sign = fermion_sign(root)
    out = []
    for combo in itertools.product(*lists):
        for cur in _vertex_currents(v, fields, list(combo), moms):
            if spin(last.field) == 'S':
                out.append(sign * cur * wl)
            elif spin(last.field) == 'V':
                out.append(sign * D.mdot(cur, wl))
            else:
                out.append(sign * np.einsum('na,na->n', cur, wl))
    return out


def fermion_lines(root):
    """The fermion lines of a diagram as (row leg, column leg) pairs: the external leg at the END of the fermion
    arrow (its wavefunction is a row spinor, psibar) and the one at its START (a column spinor)."""
    lines = []

    def walk(tree):
        """Returns the open end ('row' | 'col', leg) of the fermion line that leaves `tree` towards its parent."""
        if isinstance(tree, Leaf):
            if spin(tree.field) != 'F':
                return None
            return ('row' if is_row(tree.field) else 'col', tree.leg)
        ends = [e for e in (walk(ch) for ch in tree.children) if e is not None]
        if len(ends) == 2:                       # both ends meet at this vertex: the line is complete
            (k1, l1), (k2, l2) = ends
            assert {k1, k2} == {'row', 'col'}
            lines.append((l1, l2) if k1 == 'row' else (l2, l1))
            return None
        assert len(ends) <= 1
        return ends[0] if ends else None

    assert walk(root) is None
    return sorted(lines)


def fermion_sign(root):
    """Relative sign of a diagram from Fermi statistics: the diagram is a product of spinor chains
    (psibar_r1 ... psi_c1)(psibar_r2 ... psi_c2)...; its sign is the parity of the permutation that brings
    (r1, c1, r2, c2, ...) to the reference order of the external fermion legs (increasing leg number).  Diagrams
    with a single fermion line all have the same sign."""
    seq = [l for pair in fermion_lines(root) for l in pair]
    sign = 1
    for i in range(len(seq)):
        for j in range(i + 1, len(seq)):
            if seq[i] > seq[j]:
                sign = -sign
    return sign


def root_colour(root):
    """Colour tensors of one full diagram over ALL external legs (axes = legs 0..n-1)."""
    chs = root.children[:-1]
    last = root.children[-1]
    tmp = Node(root.vertex, chs, last.field)  # `own` axis = the last leg's colour index
    # the remaining slot must be the last leg's: _slot_order assigns it from the fields
    res = []
    for t in colour_terms(tmp):
        res.append(np.moveaxis(t, 0, -1))  # legs sorted: the last leg has the highest index
    return res
