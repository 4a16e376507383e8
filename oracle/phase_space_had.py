"""The paper's own phase-space parameterisation for hadron collisions (oracle; test infrastructure).

Section 3 and Appendix A of the paper, followed step by step:

  * generalised phase space including the parton momentum fractions, Eq. 24 / A.7:

        dSigma_n = dx_a dx_b dPhi_n
                 = Theta(1 - x_a) Theta(1 - x_b) / (2 s (4 pi)^(2n-3))  dy_n  prod_{i<n} dy_i dpT_i^2 dphi_i/(2 pi)

    integration variables y_i (i = 1..n), ln(pT_i^2 + m_i^2) and phi_i (i = 1..n-1), Eq. 28 / A.11
    (PAPER.md:388-391, 1170-1172):  dpT^2 = (pT^2 + m^2) d ln(pT^2 + m^2);
  * the n-th transverse momentum and the momentum fractions follow from momentum conservation, A.9
    (PAPER.md:1153-1161); a point with x_a >= 1 or x_b >= 1 gets a null weight, A.10;
  * resonances: dSigma = dSigma_n prod_k ds_k/(2 pi) dPhi(R_k -> f_k), Eq. 26 / A.12, with the
    Breit-Wigner map of Eq. 27 / A.13-A.15 (oracle.phase_space.bw_mass) and isotropic two-body decays
    (oracle.phase_space.two_body).

Readings (A23): the DEPENDENT particle n is the resonance (no pT cut applies to it), so every jet's pT
and rapidity cut is built into the ranges, y_jet in +-eta_jet_max (5 if the config has no eta cut),
pT_jet in [pT_min, sqrt(s)/2]; the resonance rapidity is uniform in +-y_res_max.  CTEQ6L1 is not available: the parton
densities are the documented toy  f(x) = N x^-a (1 - x)^b  per beam.  The returned weight is

        w = dSigma-weight * f_a(x_a) f_b(x_b) * s / s_hat

so that the event weight keeps the form of the fixed-s_hat path,  w_event = |Mbar|^2 w (hbar c)^2 / (2 s),  with s the
HADRONIC centre-of-mass energy squared.

Draw layout (Philox draw index; the unused draws of a config's n_draws are ignored):
  W/Z + nj jets (configs 1, 2, 3, 5, 9):  0: s_R;  1+3j, 2+3j, 3+3j: y, ln pT^2, phi of jet j;  1+3nj: y_R;
                                          2+3nj, 3+3nj: cos theta*, phi* of R -> l l'
  config 4 (t t~ g, dileptons):  0-3: s_t, s_t~, s_W+, s_W-;  4, 5, 6: y, ln pT^2, phi of the gluon;
                                 7, 8, 9: y, ln(pT^2 + s_t), phi of t*;  10: y of t~*;  11-18: the four decays as in
                                 oracle.phase_space (t*, W+*, t~*, W-*).
"""
import math

import numpy as np

from . import phase_space as ps
from . import philox

TWO_PI = 2.0 * math.pi

# resonance of the W/Z + jets family: (mass key, width key, legs of its decay products)
RESONANCE = {1: ('mw', 'gw'), 2: ('mz', 'gz'), 3: ('mw', 'gw'), 5: ('mw', 'gw'), 9: ('mw', 'gw')}
N_JETS = {1: 0, 2: 1, 3: 2, 5: 3, 9: 4}


def default_hadronic(cfg):
    """Toy parton densities f(x) = N x^-a (1 - x)^b of the two incoming partons (valence-like u, sea-like d~ / u~,
    gluon) and the rapidity range of the resonance."""
    val = (2.2, 0.5, 3.0)
    sea = (0.2, 1.2, 7.0)
    glu = (3.0, 1.2, 5.0)
    a, b = (glu, glu) if cfg == 4 else (val, sea)
    return dict(y_res_max=4.0, pdf_norm=(a[0], b[0]), pdf_a=(a[1], b[1]), pdf_b=(a[2], b[2]))


def pdf(x, norm, a, b):
    return norm * x ** (-a) * (1.0 - x) ** b


def generalised(y, lnpt2m, phi, m2, s):
    """Eq. 24 with A.9 for n particles of masses^2 m2 [N, n]: y [N, n], ln(pT^2 + m^2) [N, n-1], phi [N, n-1].
    Returns momenta k [N, n, 4], x_a, x_b and the weight factor  1/(2 s (4 pi)^(2n-3)) prod_{i<n} (pT_i^2 + m_i^2)
    (the ranges of the integration variables are multiplied in by the caller)."""
    N, n = y.shape
    k = np.empty((N, n, 4))
    w = np.full(N, 1.0 / (2.0 * s * (4.0 * math.pi) ** (2 * n - 3)))
    px = np.zeros(N)
    py = np.zeros(N)
    for i in range(n):
        if i < n - 1:
            mt2 = np.exp(lnpt2m[:, i])
            pt = np.sqrt(np.maximum(mt2 - m2[:, i], 0.0))
            kx, ky = pt * np.cos(phi[:, i]), pt * np.sin(phi[:, i])
            px += kx
            py += ky
            w = w * mt2
        else:
            kx, ky = -px, -py                                   # A.9a
            mt2 = m2[:, i] + kx * kx + ky * ky
        mt = np.sqrt(mt2)
        k[:, i, 0] = mt * np.cosh(y[:, i])
        k[:, i, 1] = kx
        k[:, i, 2] = ky
        k[:, i, 3] = mt * np.sinh(y[:, i])
    rs = math.sqrt(s)
    xa = (k[:, :, 0] + k[:, :, 3]).sum(1) / rs                  # A.9b
    xb = (k[:, :, 0] - k[:, :, 3]).sum(1) / rs                  # A.9c
    return k, xa, xb, w


def _ranges(cfg, rs, cuts):
    ptmin, etaj, _, _ = cuts if cuts is not None else ps.default_cuts(cfg)
    ymax = etaj if etaj > 0 else 5.0
    ptmin = ptmin if ptmin > 0 else 1.0
    return ymax, math.log(ptmin * ptmin), math.log(0.25 * rs * rs)


def from_uniforms(cfg, u, rs, par, had, cuts=None):
    """Momenta [N, n_ext, 4] (lab frame: incoming x_a, x_b along +-z), weight (module docstring) and the validity
    flag x_a < 1 and x_b < 1 (a point that violates it has weight 0)."""
    N = u.shape[0]
    s = rs * rs
    ymax, l0, l1 = _ranges(cfg, rs, cuts)
    p = np.zeros((N, ps.N_EXT[cfg], 4))
    if cfg in RESONANCE:
        nj = N_JETS[cfg]
        mk, wk = RESONANCE[cfg]
        sR, w = ps.bw_mass(u[:, 0], par[mk], par[wk])
        n = nj + 1
        y = np.empty((N, n))
        lnpt = np.empty((N, n - 1))
        phi = np.empty((N, n - 1))
        for j in range(nj):
            y[:, j] = ymax * (2.0 * u[:, 1 + 3 * j] - 1.0)
            lnpt[:, j] = l0 + (l1 - l0) * u[:, 2 + 3 * j]
            phi[:, j] = TWO_PI * u[:, 3 + 3 * j]
            w = w * (2.0 * ymax) * (l1 - l0)
        y[:, nj] = had['y_res_max'] * (2.0 * u[:, 1 + 3 * nj] - 1.0)
        w = w * 2.0 * had['y_res_max']
        m2 = np.zeros((N, n))
        m2[:, nj] = sR
        k, xa, xb, wg = generalised(y, lnpt, phi, m2, s)
        w = w * wg
        zero = np.zeros(N)
        l1_, l2_, d = ps.two_body(k[:, nj], sR, zero, zero, u[:, 2 + 3 * nj], u[:, 3 + 3 * nj])
        w = w * d
        p[:, 2], p[:, 3] = l1_, l2_
        for j in range(nj):
            p[:, 4 + j] = k[:, j]
    elif cfg == 4:
        st, j1 = ps.bw_mass(u[:, 0], par['mt'], par['gt'])
        stb, j2 = ps.bw_mass(u[:, 1], par['mt'], par['gt'])
        swp, j3 = ps.bw_mass(u[:, 2], par['mw'], par['gw'])
        swm, j4 = ps.bw_mass(u[:, 3], par['mw'], par['gw'])
        w = j1 * j2 * j3 * j4
        y = np.empty((N, 3))
        lnpt = np.empty((N, 2))
        phi = np.empty((N, 2))
        y[:, 0] = ymax * (2.0 * u[:, 4] - 1.0)
        lnpt[:, 0] = l0 + (l1 - l0) * u[:, 5]
        phi[:, 0] = TWO_PI * u[:, 6]
        w = w * (2.0 * ymax) * (l1 - l0)
        yr = had['y_res_max']
        y[:, 1] = yr * (2.0 * u[:, 7] - 1.0)
        lt0 = np.log(st)                                         # Eq. 28: ln(pT^2 + s_k) from pT = 0 ...
        lt1 = np.log(st + 0.25 * s)                              # ... to pT = sqrt(s)/2
        lnpt[:, 1] = lt0 + (lt1 - lt0) * u[:, 8]
        phi[:, 1] = TWO_PI * u[:, 9]
        y[:, 2] = yr * (2.0 * u[:, 10] - 1.0)
        w = w * (2.0 * yr) * (lt1 - lt0) * (2.0 * yr)
        m2 = np.stack([np.zeros(N), st, stb], axis=1)
        k, xa, xb, wg = generalised(y, lnpt, phi, m2, s)
        w = w * wg
        mb2 = par['mb'] ** 2
        zero = np.zeros(N)
        b, wp, d1 = ps.two_body(k[:, 1], st, mb2 + zero, swp, u[:, 11], u[:, 12])
        ep, ve, d2 = ps.two_body(wp, swp, zero, zero, u[:, 13], u[:, 14])
        bb, wm, d3 = ps.two_body(k[:, 2], stb, mb2 + zero, swm, u[:, 15], u[:, 16])
        mu, vm, d4 = ps.two_body(wm, swm, zero, zero, u[:, 17], u[:, 18])
        w = w * d1 * d2 * d3 * d4
        for i, x in enumerate([b, ep, ve, bb, mu, vm, k[:, 0]]):
            p[:, 2 + i] = x
    else:
        raise ValueError('hadronic phase space: process %d not implemented' % cfg)
    valid = (xa < 1.0) & (xb < 1.0)
    xa_c = np.where(valid, xa, 0.5)
    xb_c = np.where(valid, xb, 0.5)
    ea, eb = 0.5 * rs * xa, 0.5 * rs * xb
    p[:, 0, 0], p[:, 0, 3] = ea, ea
    p[:, 1, 0], p[:, 1, 3] = eb, -eb
    fa = pdf(xa_c, had['pdf_norm'][0], had['pdf_a'][0], had['pdf_b'][0])
    fb = pdf(xb_c, had['pdf_norm'][1], had['pdf_a'][1], had['pdf_b'][1])
    w = np.where(valid, w * fa * fb / (xa_c * xb_c), 0.0)
    return p, w, valid


def generate(cfg, seed, first_event, n, rs, par, had=None, cuts=None, grid=None, with_bins=False):
    """Events first_event .. of the stream (same Philox layout as the fixed-s_hat generator, A15)."""
    had = had if had is not None else default_hadronic(cfg)
    u = philox.uniforms(seed, first_event, n, ps.N_DRAWS[cfg], cfg)
    bins, jac = None, 1.0
    if grid is not None:
        from . import vegas
        u, jac, bins = vegas.apply_grid(np.asarray(grid, dtype=float), u)
    p, w, valid = from_uniforms(cfg, u, rs, par, had, cuts)
    w = w * jac
    return (p, w, valid, bins) if with_bins else (p, w, valid)
