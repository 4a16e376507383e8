"""Process definitions and the helicity+colour summed, averaged |Mbar|^2 (oracle; test infrastructure).

The five BASELINE.json configs plus the 2->2 processes used as pins.
|Mbar|^2 follows Eq. 4 with the identical-particle factor of SURVEY 8c-A7.
"""
import itertools
import math
import numpy as np

from . import feynman as fy


_DIAGRAM_CACHE = {}   # diagram lists are built once per (process, parameters) and session


class Process:
    def __init__(self, name, initial, final, vertex_names):
        self.name = name
        self.initial, self.final = list(initial), list(final)
        self.legs = [(x, 'in') for x in initial] + [(x, 'out') for x in final]
        self.ext_fields = [x for x in initial] + [fy.anti(x) for x in final]
        self.vertex_names = list(vertex_names)

    @property
    def n_ext(self):
        return len(self.legs)

    def helicities(self, leg):
        name = self.legs[leg][0]
        if fy.spin(name) == 'S':
            return (0,)
        if fy.spin(name) == 'V' and fy._F[name][2] is not None:
            return (-1, 0, 1)  # massive vector (never external in the configs)
        return (-1, 1)

    def ident_factor(self):
        f = 1
        for x in set(self.final):
            f *= math.factorial(self.final.count(x))
        return f

    def avg_factor(self):
        """1/(2*2) * 1/(n_a n_b) * 1/S_ident   (Eq. 4; A7)."""
        f = 1.0
        for i, x in enumerate(self.initial):
            f /= len(self.helicities(i)) * fy.coldim(x)
        return f / self.ident_factor()

    def diagrams(self, par):
        """Diagram list and the brute-force colour matrix between all (diagram, colour-structure) terms."""
        key = (self.name, tuple(self.legs), tuple(self.vertex_names), tuple(sorted(par.items())))
        if key not in _DIAGRAM_CACHE:
            verts = fy.build_vertices(par, self.vertex_names)
            roots = fy.enumerate_diagrams(self.ext_fields, verts)
            cols = []
            for r in roots:
                cols += [c.reshape(-1) for c in fy.root_colour(r)]
            cmat = np.array(cols)  # [n_terms, prod(colour dims)]
            cm = cmat @ np.conj(cmat.T)  # CM[l,l'] = sum_ext c_l conj(c_l')
            _DIAGRAM_CACHE[key] = (roots, cm, cmat)
        return _DIAGRAM_CACHE[key]


def amplitudes(proc, p, par, hel, memo=None, kin=None):
    """Kinematic amplitude of every (diagram, colour-structure) term for one helicity assignment: [n_terms, N]."""
    roots, _, _ = proc.diagrams(par)
    if kin is None:
        kin = fy.Kinematics(proc, p, par)
    out = []
    for r in roots:
        out += fy.root_amplitudes(r, hel, kin, memo)
    return np.array(out)


def me2(proc, p, par, per_helicity=False, batch=2048, wf_hook=None):
    """|Mbar|^2 for momenta p [N, n_ext, 4] (GeV, physical E>0 for every leg).

    wf_hook(kin), if given, may replace external wavefunctions in kin.wf before evaluation (used by the
    Ward-identity pins: polarisation vector -> momentum)."""
    p = np.asarray(p)
    if p.dtype != np.longdouble:
        p = p.astype(float)
    N = p.shape[0]
    if N > batch:
        parts = [me2(proc, p[i:i + batch], par, per_helicity, batch, wf_hook) for i in range(0, N, batch)]
        return np.concatenate(parts, axis=-1)
    roots, cm, _ = proc.diagrams(par)
    kin = fy.Kinematics(proc, p, par)
    if wf_hook is not None:
        wf_hook(kin)
    memo = {}
    total = np.zeros(N, dtype=p.dtype)
    per = {}
    for hel in itertools.product(*[proc.helicities(i) for i in range(proc.n_ext)]):
        a = amplitudes(proc, p, par, hel, memo, kin)  # [n_terms, N]
        m2 = np.einsum('ln,lm,mn->n', a, cm, np.conj(a)).real
        total += m2
        if per_helicity:
            per[hel] = m2 * proc.avg_factor()
    if per_helicity:
        return per
    return total * proc.avg_factor()


def me2_extended(proc, p, par, on_shell=True, batch=512):
    """|Mbar|^2 with the same plain formulas evaluated in extended precision (numpy.longdouble: the x87 80-bit
    format, eps = 1.1e-19, about 3.3 decimal digits more than fp64).  The arbiter when the fp64 oracle and the
    kernel differ by more than the tolerance (reading A21).

    on_shell=True (reading A21): an external leg is on its mass shell by definition (Eq. 29-33, PAPER.md:412-447,
    are functions of an on-shell momentum), so its energy is a function of its 3-momentum, E = sqrt(|p|^2 + m^2),
    taken here in extended precision; the fp64 energy that came with the input is that value rounded.  With
    on_shell=False the energies are used as given (then p^2 - m^2 = O(eps E^2) enters every invariant that
    contains the leg).  Returns float64."""
    p = np.asarray(p).astype(np.longdouble)
    if on_shell:
        p = p.copy()
        for i, (name, _) in enumerate(proc.legs):
            m, _w = fy.mass_width(name, par)
            p[:, i, 0] = np.sqrt(p[:, i, 1] ** 2 + p[:, i, 2] ** 2 + p[:, i, 3] ** 2 + np.longdouble(m) ** 2)
    return me2(proc, p, par, batch=batch).astype(np.float64)


def me2_explicit_colour(proc, p, par):
    """Same number by the literal double sum of Eq. 4: for every helicity AND every explicit external colour
    assignment, add up the diagrams and square.  (Slower; used as a cross-check of the colour matrix.)"""
    p = np.asarray(p, dtype=float)
    roots, _, cmat = proc.diagrams(par)
    kin = fy.Kinematics(proc, p, par)
    total = np.zeros(p.shape[0])
    for hel in itertools.product(*[proc.helicities(i) for i in range(proc.n_ext)]):
        a = amplitudes(proc, p, par, hel, None, kin)  # [n_terms, N]
        full = np.einsum('ln,lc->cn', a, cmat)  # amplitude for each explicit colour assignment c
        total += np.sum(np.abs(full) ** 2, axis=0)
    return total * proc.avg_factor()


# ----------------------------------------------------------------------------- the five configs
def config(i):
    """BASELINE.json configs[i-1]; external leg order = initial then final as written there."""
    if i == 1:
        return Process('udx_epve', ['u', 'd~'], ['e+', 've'], ['udw', 'enw'])
    if i == 2:
        return Process('uux_epemg', ['u', 'u~'], ['e+', 'e-', 'g'], ['uug', 'uua', 'uuz', 'eea', 'eez'])
    if i == 3:
        return Process('udx_epvegg', ['u', 'd~'], ['e+', 've', 'g', 'g'],
                       ['udw', 'enw', 'uug', 'ddg', 'ggg', 'gggg'])
    if i == 4:
        # decay-chain subset (A13): no gluon radiation off b, no non-resonant diagrams -> b has no g/a/z vertex
        return Process('gg_ttxg_dilep', ['g', 'g'], ['b', 'e+', 've', 'b~', 'mu-', 'vm~', 'g'],
                       ['ttg', 'ggg', 'gggg', 'tbw', 'enw', 'mnw'])
    if i == 5:
        return Process('udx_epveggg', ['u', 'd~'], ['e+', 've', 'g', 'g', 'g'],
                       ['udw', 'enw', 'uug', 'ddg', 'ggg', 'gggg'])
    # Higgs-sector processes: every scalar vertex of the library in a small process
    if i == 6:   # VVS: W* -> W H (Eq. 18a)
        return Process('udx_epveh', ['u', 'd~'], ['e+', 've', 'h'], ['udw', 'enw', 'wwh'])
    if i == 7:   # VVS twice, VVSS, SSS: Z* -> Z H H
        return Process('uux_epemhh', ['u', 'u~'], ['e+', 'e-', 'h', 'h'],
                       ['uuz', 'eez', 'zzh', 'zzhh', 'hhh'])
    if i == 8:   # FFS with massive external fermions: g g -> t t~ H (Eq. 20d)
        return Process('gg_ttxh', ['g', 'g'], ['t', 't~', 'h'], ['ttg', 'ggg', 'tth'])
    if i == 9:   # next size up: W + 4 jets, 428 diagrams, 516 colour-split terms
        return Process('udx_epvegggg', ['u', 'd~'], ['e+', 've', 'g', 'g', 'g', 'g'],
                       ['udw', 'enw', 'uug', 'ddg', 'ggg', 'gggg'])
    # weak-boson fusion: two quark lines (Eq. 21a, 22a)
    if i == 10:
        return Process('ud_hud', ['u', 'd'], ['h', 'u', 'd'], ['uuz', 'ddz', 'udw', 'zzh', 'wwh'])
    if i == 11:
        return Process('ud_hhud', ['u', 'd'], ['h', 'h', 'u', 'd'],
                       ['uuz', 'ddz', 'udw', 'zzh', 'wwh', 'zzhh', 'wwhh', 'hhh'])
    raise ValueError(i)


# sqrt(s_hat) [GeV] and number of events of each config (BASELINE.json)
SQRT_S = {1: 80.0, 2: 500.0, 3: 1000.0, 4: 1500.0, 5: 2000.0, 6: 500.0, 7: 1000.0, 8: 1000.0, 9: 3000.0, 10: 1000.0,
          11: 1000.0}
N_EVENTS = {1: 1 << 16, 2: 1 << 20, 3: 1 << 22, 4: 1 << 22, 5: 1 << 22, 6: 1 << 20, 7: 1 << 20, 8: 1 << 20, 9: 1 << 20,
            10: 1 << 20, 11: 1 << 20}
