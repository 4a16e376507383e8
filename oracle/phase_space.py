"""Phase-space points, weights and cuts for the five configs (oracle; test infrastructure).

Steps a1-a4 of SURVEY.md 8a, written out in order:
  * uniforms from Philox (oracle/philox.py, layout A15);
  * flat RAMBO for massless final states at fixed sqrt(s_hat) (BASELINE.json; algorithm as read in
    SURVEY 8c-A16), draws per particle i: (4i: cos theta, 4i+1: phi, 4i+2, 4i+3: energy);
  * config 4: Breit-Wigner mapped invariant masses (Eq. 27; A.13-A.15),
    massive RAMBO for (t*, t~*, g), then nested isotropic two-body decays (Eq. 26):
        draws 0..3 : s_t, s_t~, s_W+, s_W-          (theta_k uniform in +-atan(min(20, m/Gamma)))
        draws 4..15: RAMBO for t*, t~*, g
        draws 16,17: t* -> b W+*  (cos theta, phi in the t* rest frame);  18,19: W+* -> e+ ve
        draws 20,21: t~* -> b~ W-*;                                        22,23: W-* -> mu- vm~
  * incoming momenta p_a,b = sqrt(s_hat)/2 (1, 0, 0, +-1);
  * cuts (Eq. 8-11, values from BASELINE.json, scope A11/A12): a failing event has weight 0
    ("null value") and is counted in N.
"""
import math
import numpy as np

from . import philox

TWO_PI = 2.0 * math.pi


def _iso(c, f, e):
    st = np.sqrt(1.0 - c * c)
    return np.stack([e, e * st * np.cos(f), e * st * np.sin(f), e * c], axis=1)


def rambo_massless(u, n, rs):
    """u: [N, 4n] uniforms -> p [N, n, 4], weight (constant V_n)."""
    N = u.shape[0]
    q = np.empty((N, n, 4))
    for i in range(n):
        c = 2.0 * u[:, 4 * i] - 1.0
        f = TWO_PI * u[:, 4 * i + 1]
        e = -np.log(u[:, 4 * i + 2] * u[:, 4 * i + 3])
        q[:, i, :] = _iso(c, f, e)
    Q = q.sum(axis=1)
    M = np.sqrt(Q[:, 0] ** 2 - Q[:, 1] ** 2 - Q[:, 2] ** 2 - Q[:, 3] ** 2)
    b = -Q[:, 1:] / M[:, None]
    x = rs / M
    g = Q[:, 0] / M
    a = 1.0 / (1.0 + g)
    p = np.empty_like(q)
    for i in range(n):
        bq = np.sum(b * q[:, i, 1:], axis=1)
        p[:, i, 0] = x * (g * q[:, i, 0] + bq)
        p[:, i, 1:] = x[:, None] * (q[:, i, 1:] + b * q[:, i, 0][:, None] + (a * bq)[:, None] * b)
    # Reading A16b.  The conformal map above is ill-conditioned (~ (Q0/M)^2 roundings) when the q_i are
    # nearly collinear, so its output satisfies sum p = (rs, 0) and p_i^2 = 0 only to that accuracy.  The point is
    # put back on the constraint surface exactly: the last 3-momentum closes the sum, every energy is |p_i|, and
    # one common factor restores sum E = rs.  This moves the point by no more than the rounding it already had.
    p[:, n - 1, 1:] = -p[:, :n - 1, 1:].sum(axis=1)
    p[:, :, 0] = np.sqrt(np.sum(p[:, :, 1:] ** 2, axis=2))
    p *= (rs / p[:, :, 0].sum(axis=1))[:, None, None]
    vol = (math.pi / 2.0) ** (n - 1) * rs ** (2 * n - 4) / (math.factorial(n - 1) * math.factorial(n - 2)) \
        * TWO_PI ** (4 - 3 * n)
    return p, np.full(N, vol)


def rambo_massive(u, masses, rs):
    """masses: [N, n] array.  Massless RAMBO followed by the rescaling of the 3-momenta by xi with
    sum_i sqrt(m_i^2 + xi^2 E_i^2) = sqrt(s) solved by Newton iteration (A16)."""
    N, n = masses.shape
    p, w = rambo_massless(u, n, rs)
    e0 = p[:, :, 0]
    m2 = masses ** 2
    xi = np.sqrt(1.0 - (masses.sum(axis=1) / rs) ** 2)
    for _ in range(12):
        en = np.sqrt(m2 + (xi ** 2)[:, None] * e0 ** 2)
        f = en.sum(axis=1) - rs
        df = (xi[:, None] * e0 ** 2 / en).sum(axis=1)
        xi = xi - f / df
    k = np.empty_like(p)
    k[:, :, 0] = np.sqrt(m2 + (xi ** 2)[:, None] * e0 ** 2)
    k[:, :, 1:] = xi[:, None, None] * p[:, :, 1:]
    kabs = xi[:, None] * e0
    wt = (kabs.sum(axis=1) / rs) ** (2 * n - 3) * np.prod(kabs / k[:, :, 0], axis=1) \
        * rs / (kabs ** 2 / k[:, :, 0]).sum(axis=1)
    return k, w * wt


def bw_mass(u, m, gam):
    """s = m^2 + m Gamma tan(theta), theta uniform in +-atan(min(20, m/Gamma)); returns s and ds/(2 pi)."""
    tmax = math.atan(min(20.0, m / gam))
    th = -tmax + 2.0 * tmax * u
    s = m * m + m * gam * np.tan(th)
    jac = ((s - m * m) ** 2 + (m * gam) ** 2) / (m * gam) * (2.0 * tmax) / TWO_PI
    return s, jac


def boost(pr, P, M, msq):
    """Boost pr (given in the rest frame of a particle of mass M) to the frame where that particle has momentum P.
    The boosted energy (P.pr)/M fixes the 3-momentum; the returned energy is then taken from the mass-shell
    condition E = sqrt(|p|^2 + msq) (reading A16b), equal to it up to rounding."""
    e = (P[:, 0] * pr[:, 0] + np.sum(P[:, 1:] * pr[:, 1:], axis=1)) / M
    fac = (e + pr[:, 0]) / (P[:, 0] + M)
    out = np.empty_like(pr)
    out[:, 1:] = pr[:, 1:] + fac[:, None] * P[:, 1:]
    out[:, 0] = np.sqrt(np.sum(out[:, 1:] ** 2, axis=1) + msq)
    return out


def two_body(P, M2, m1sq, m2sq, uc, uf):
    """Isotropic decay of momentum P (mass^2 = M2) into masses^2 (m1sq, m2sq); weight = |p*| / (4 pi M)."""
    M = np.sqrt(M2)
    lam = (M2 - m1sq - m2sq) ** 2 - 4.0 * m1sq * m2sq
    pst = np.sqrt(lam) / (2.0 * M)
    c = 2.0 * uc - 1.0
    f = TWO_PI * uf
    st = np.sqrt(1.0 - c * c)
    d = np.stack([st * np.cos(f), st * np.sin(f), c], axis=1) * pst[:, None]
    p1 = np.concatenate([np.sqrt(pst ** 2 + m1sq)[:, None], d], axis=1)
    p2 = np.concatenate([np.sqrt(pst ** 2 + m2sq)[:, None], -d], axis=1)
    return boost(p1, P, M, m1sq), boost(p2, P, M, m2sq), pst / (4.0 * math.pi * M)


N_FINAL = {1: 2, 2: 3, 3: 4, 5: 5, 6: 3, 7: 4, 8: 3, 9: 6, 10: 3, 11: 4}
N_DRAWS = {1: 8, 2: 12, 3: 16, 4: 24, 5: 20, 6: 12, 7: 16, 8: 12, 9: 24, 10: 12, 11: 16}
N_EXT = {1: 4, 2: 5, 3: 6, 4: 9, 5: 7, 6: 5, 7: 6, 8: 5, 9: 8, 10: 5, 11: 6}
# masses of the final-state legs of the Higgs-sector processes (parameter names; None = massless)
FINAL_MASSES = {6: (None, None, 'mh'), 7: (None, None, 'mh', 'mh'), 8: ('mt', 'mt', 'mh'), 10: ('mh', None, None),
                11: ('mh', 'mh', None, None)}


def generate(cfg, seed, first_event, n, rs, par, grid=None, with_bins=False):
    """Momenta [n, n_ext, 4] (leg order of oracle.processes.config) and phase-space weight [n].

    grid [n_draws, NB + 1] (oracle.vegas): the Philox uniforms are mapped through the adaptive grid before they are
    used and the weight carries the Jacobian; with_bins=True also returns the bin of every draw [n, n_draws]."""
    u = philox.uniforms(seed, first_event, n, N_DRAWS[cfg], cfg)
    if grid is None:
        p, w = from_uniforms(cfg, u, rs, par)
        return (p, w, None) if with_bins else (p, w)
    from . import vegas
    x, jac, bins = vegas.apply_grid(np.asarray(grid, dtype=float), u)
    p, w = from_uniforms(cfg, x, rs, par)
    return (p, w * jac, bins) if with_bins else (p, w * jac)


def from_uniforms(cfg, u, rs, par):
    """Steps a2-a3 for given numbers u [n, n_draws] in (0, 1)."""
    n = u.shape[0]
    p = np.zeros((n, N_EXT[cfg], 4))
    p[:, 0, 0] = p[:, 1, 0] = p[:, 0, 3] = 0.5 * rs
    p[:, 1, 3] = -0.5 * rs
    if cfg in FINAL_MASSES:
        masses = np.stack([np.full(n, par[m] if m else 0.0) for m in FINAL_MASSES[cfg]], axis=1)
        pf, w = rambo_massive(u, masses, rs)
        p[:, 2:, :] = pf
        return p, w
    if cfg != 4:
        pf, w = rambo_massless(u, N_FINAL[cfg], rs)
        p[:, 2:, :] = pf
        return p, w
    st, j1 = bw_mass(u[:, 0], par['mt'], par['gt'])
    stb, j2 = bw_mass(u[:, 1], par['mt'], par['gt'])
    swp, j3 = bw_mass(u[:, 2], par['mw'], par['gw'])
    swm, j4 = bw_mass(u[:, 3], par['mw'], par['gw'])
    masses = np.stack([np.sqrt(st), np.sqrt(stb), np.zeros(n)], axis=1)
    k, w = rambo_massive(u[:, 4:16], masses, rs)
    mb2 = par['mb'] ** 2
    zero = np.zeros(n)
    b, wp, d1 = two_body(k[:, 0], st, mb2 + zero, swp, u[:, 16], u[:, 17])
    ep, ve, d2 = two_body(wp, swp, zero, zero, u[:, 18], u[:, 19])
    bb, wm, d3 = two_body(k[:, 1], stb, mb2 + zero, swm, u[:, 20], u[:, 21])
    mu, vm, d4 = two_body(wm, swm, zero, zero, u[:, 22], u[:, 23])
    for i, x in enumerate([b, ep, ve, bb, mu, vm, k[:, 2]]):
        p[:, 2 + i, :] = x
    return p, w * j1 * j2 * j3 * j4 * d1 * d2 * d3 * d4


# ----------------------------------------------------------------------------- cuts
def default_cuts(cfg):
    """(pt_jet_min, eta_jet_max, eta_lep_max, dr_jj_min); <= 0 disables.  BASELINE.json configs, scope A11/A12."""
    return {1: (0.0, 0.0, 0.0, 0.0), 2: (20.0, 2.5, 2.5, 0.0), 3: (20.0, 0.0, 0.0, 0.4),
            4: (20.0, 2.5, 0.0, 0.0), 5: (20.0, 2.5, 0.0, 0.4), 9: (20.0, 2.5, 0.0, 0.4)}.get(cfg, (0.0, 0.0, 0.0, 0.0))


JETS = {1: [], 2: [4], 3: [4, 5], 4: [8], 5: [4, 5, 6], 6: [], 7: [], 8: [], 9: [4, 5, 6, 7], 10: [], 11: []}  # gluon legs
CHARGED_LEPTONS = {1: [2], 2: [2, 3], 3: [2], 4: [3, 6], 5: [2], 6: [2], 7: [2, 3], 8: [], 9: [2], 10: [], 11: []}


def pt(p):
    return np.sqrt(p[:, 1] ** 2 + p[:, 2] ** 2)


def eta(p):
    """Pseudorapidity = asinh(pz / pT)."""
    return np.arcsinh(p[:, 3] / pt(p))


def delta_r(p1, p2):
    """Eq. 9b."""
    dphi = np.arctan2(p1[:, 2], p1[:, 1]) - np.arctan2(p2[:, 2], p2[:, 1])
    dphi = np.where(dphi > math.pi, dphi - TWO_PI, dphi)
    dphi = np.where(dphi < -math.pi, dphi + TWO_PI, dphi)
    deta = eta(p1) - eta(p2)
    return np.sqrt(deta ** 2 + dphi ** 2)


def passes(cfg, p, cuts=None):
    ptmin, etaj, etal, drmin = cuts if cuts is not None else default_cuts(cfg)
    ok = np.ones(p.shape[0], dtype=bool)
    jets = JETS[cfg]
    for j in jets:
        if ptmin > 0:
            ok &= pt(p[:, j]) > ptmin
        if etaj > 0:
            ok &= np.abs(eta(p[:, j])) < etaj
    if etal > 0:
        for l in CHARGED_LEPTONS[cfg]:
            ok &= np.abs(eta(p[:, l])) < etal
    if drmin > 0:
        for a in range(len(jets)):
            for b in range(a + 1, len(jets)):
                ok &= delta_r(p[:, jets[a]], p[:, jets[b]]) > drmin
    return ok
