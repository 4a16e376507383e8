"""Pins of the oracle's |Mbar|^2 against closed forms (SURVEY.md 8c 'Pins'; Eq. 4, Eq. 35 PAPER.md:506,
Eq. 36-49).  Every Feynman rule used by configs 1-5 is exercised by at least one 2->2 form."""
import math
import os

import numpy as np
import pytest

from oracle import processes as P
from oracle import sm
from oracle import phase_space as ps
from oracle import integrate
import inputs

PAR = sm.default_params()
C = sm.couplings(PAR)
GOLD = os.path.join(os.path.dirname(__file__), 'golden', 'cfg1_closed_form.txt')


def _gold():
    rows = {}
    for line in open(GOLD):
        if line.startswith('#') or not line.strip():
            continue
        k, a, v = line.split()
        rows[(k, float(a))] = float(v)
    return rows


def test_cfg1_printed_values():
    """Values printed in SURVEY 8c for cos(theta) = 0, 0.5, 1, -1 at sqrt(s_hat) = 80 GeV (7 digits)."""
    g = _gold()
    ct = np.array([0.0, 0.5, 1.0, -1.0])
    # theta = angle between u (leg 0, +z) and ve (leg 3): two_to_two_at puts leg 2 at ct, so leg 3 is at -ct
    p = inputs.two_to_two_at(80.0, 0.0, 0.0, -ct, 0.3)
    m = P.me2(P.config(1), p, PAR)
    for c, v in zip(ct, m):
        want = g[('me2', float(c))]
        assert abs(v - want) <= 6e-7 * max(want, 1.0)
    assert abs(C['gw'] ** 2 - g[('gw2', 0.0)]) < 6e-8


def test_cfg1_closed_form_random():
    p = inputs.two_to_two(80.0, 0, 0, 200, seed=11, cmax=1.0)
    s = 80.0 ** 2
    ct = p[:, 3, 3] / p[:, 3, 0]
    cf = C['gw'] ** 4 * s * s * (1 + ct) ** 2 / (48 * ((s - PAR['mw'] ** 2) ** 2 + (PAR['mw'] * PAR['gw']) ** 2))
    # equivalently 16 (p_u.p_e+)(p_d~.p_ve) g_W^4 / (4*12*|D|^2)
    cf2 = 16 * inputs.mdot(p[:, 0], p[:, 2]) * inputs.mdot(p[:, 1], p[:, 3]) * C['gw'] ** 4 / \
        (48 * ((s - PAR['mw'] ** 2) ** 2 + (PAR['mw'] * PAR['gw']) ** 2))
    m = P.me2(P.config(1), p, PAR)
    assert np.allclose(m, cf, rtol=1e-12, atol=1e-13)
    assert np.allclose(m, cf2, rtol=1e-12, atol=1e-13)


def test_cfg1_only_one_helicity_nonzero():
    p = inputs.two_to_two(80.0, 0, 0, 20, seed=2)
    per = P.me2(P.config(1), p, PAR, per_helicity=True)
    nz = [h for h, v in per.items() if np.max(v) > 1e-20]
    assert nz == [(-1, 1, 1, -1)]  # u_L d~_R -> e+_R ve_L
    assert len(per) == 16


def test_cfg1_cross_section_analytic_vs_mc():
    """sigma_hat = g_W^4 s/(576 pi |D|^2) = 7924.94 pb; oracle MC over all 65,536 RAMBO points of config 1."""
    g = _gold()
    s = 80.0 ** 2
    sig = C['gw'] ** 4 * s / (576 * math.pi * ((s - PAR['mw'] ** 2) ** 2 + (PAR['mw'] * PAR['gw']) ** 2))
    assert abs(sig - g[('sigma_gev2', 0.0)]) < 5e-12
    assert abs(sig * sm.HBARC2_PB - g[('sigma_pb', 0.0)]) < 0.006
    w, ok = integrate.weights(1, 13050708_1, 0, 1 << 16, 80.0, PAR)
    est, err = integrate.sigma(integrate.accumulate(w, ok))
    assert ok.all()
    assert abs(est - sig * sm.HBARC2_PB) < 3 * err
    assert 0.0030 < err / est < 0.0040  # std/mean of (1+c)^2 is 0.894 -> 0.35 % at N = 65,536


def _ratio(proc, p, par, want):
    got = P.me2(proc, p, par)
    return np.max(np.abs(got / want - 1))


def test_qqbar_to_photons():
    p = inputs.two_to_two(300.0, 0, 0, 20)
    s, t, u = inputs.mandelstam(p)
    want = (2.0 / 3) * C['e'] ** 4 * (2.0 / 3) ** 4 * (t / u + u / t) * 0.5  # 1/2: identical photons
    assert _ratio(P.Process('x', ['u', 'u~'], ['a', 'a'], ['uua']), p, PAR, want) < 1e-12


def test_uubar_to_epem_gamma_z_interference():
    p = inputs.two_to_two(200.0, 0, 0, 20)
    sh = 200.0 ** 2
    A = {}
    for lq, gq in enumerate(C[('z', 'u')]):
        for le, ge in enumerate(C[('z', 'e-')]):
            A[(lq, le)] = C['e'] ** 2 * (2.0 / 3) * (-1) / sh + gq * ge / (sh - PAR['mz'] ** 2 + 1j * PAR['mz'] * PAR['gz'])
    pu, pub, pep, pem = p[:, 0], p[:, 1], p[:, 2], p[:, 3]
    d = inputs.mdot
    tot = 16 * ((abs(A[0, 0]) ** 2 + abs(A[1, 1]) ** 2) * d(pu, pep) * d(pub, pem)
                + (abs(A[0, 1]) ** 2 + abs(A[1, 0]) ** 2) * d(pu, pem) * d(pub, pep))
    pr = P.Process('x', ['u', 'u~'], ['e+', 'e-'], ['uua', 'uuz', 'eea', 'eez'])
    assert _ratio(pr, p, PAR, tot * 3 / 36.0) < 1e-12


def test_qcd_two_to_two_massless():
    p = inputs.two_to_two(300.0, 0, 0, 20)
    s, t, u = inputs.mandelstam(p)
    gs = C['gs']
    want = gs ** 4 * ((32.0 / 27) * (t * t + u * u) / (t * u) - (8.0 / 3) * (t * t + u * u) / s ** 2) * 0.5
    assert _ratio(P.Process('x', ['u', 'u~'], ['g', 'g'], ['uug', 'ggg']), p, PAR, want) < 1e-12
    want = gs ** 4 * 4.5 * (3 - t * u / s ** 2 - s * u / t ** 2 - s * t / u ** 2) * 0.5
    assert _ratio(P.Process('x', ['g', 'g'], ['g', 'g'], ['ggg', 'gggg']), p, PAR, want) < 1e-12


def test_heavy_quark_production():
    par0 = dict(PAR, gt=0.0)
    mt = PAR['mt']
    gs = C['gs']
    p = inputs.two_to_two(600.0, mt, mt, 20)
    s, t, u = inputs.mandelstam(p)
    want = gs ** 4 * (4.0 / 9) * ((t - mt ** 2) ** 2 + (u - mt ** 2) ** 2 + 2 * mt ** 2 * s) / s ** 2
    assert _ratio(P.Process('x', ['u', 'u~'], ['t', 't~'], ['uug', 'ttg']), p, par0, want) < 1e-12
    t1, t2, rho = (mt ** 2 - t) / s, (mt ** 2 - u) / s, 4 * mt ** 2 / s
    want = gs ** 4 * (1 / (6 * t1 * t2) - 3.0 / 8) * (t1 ** 2 + t2 ** 2 + rho - rho ** 2 / (4 * t1 * t2))
    assert _ratio(P.Process('x', ['g', 'g'], ['t', 't~'], ['ttg', 'ggg']), p, par0, want) < 1e-12


def _with_soft_gluon(rs, eg, n, seed, n_hard_final=2):
    """2 -> 2 (massless) + one gluon of energy eg appended as the LAST leg; the hard pair recoils."""
    rng = np.random.default_rng(seed)
    ct, ph = rng.uniform(-0.8, 0.8, n), rng.uniform(0, 2 * np.pi, n)
    st = np.sqrt(1 - ct * ct)
    k = eg * np.stack([np.ones(n), st * np.cos(ph), st * np.sin(ph), ct], 1)
    P0 = np.zeros((n, 4))
    P0[:, 0] = rs
    Q = P0 - k
    Q2 = inputs.mdot(Q, Q)
    z = np.zeros(n)
    a, b, _ = ps.two_body(Q, Q2, z, z, rng.uniform(0.2, 0.8, n), rng.uniform(0, 1, n))
    p = np.zeros((n, 5, 4))
    p[:, 0] = [rs / 2, 0, 0, rs / 2]
    p[:, 1] = [rs / 2, 0, 0, -rs / 2]
    p[:, 2], p[:, 3], p[:, 4] = a, b, k
    return p


def test_cfg2_soft_gluon_limit():
    """|M(u u~ -> e+ e- g)|^2 -> g_s^2 C_F 2 p_u.p_u~ / ((p_u.k)(p_u~.k)) |M(u u~ -> e+ e-)|^2, ratio -> 1 linearly in E_g."""
    born = P.Process('x', ['u', 'u~'], ['e+', 'e-'], ['uua', 'uuz', 'eea', 'eez'])
    devs = []
    for eg in (1.0, 1e-2, 1e-4):
        p = _with_soft_gluon(500.0, eg, 10, seed=4)
        m3 = P.me2(P.config(2), p, PAR)
        d = inputs.mdot
        eik = C['gs'] ** 2 * (4.0 / 3) * 2 * d(p[:, 0], p[:, 1]) / (d(p[:, 0], p[:, 4]) * d(p[:, 1], p[:, 4]))
        # Born at the recoiled lepton momenta, in the lepton-pair rest frame with rescaled beams
        Q = p[:, 2] + p[:, 3]
        rs2 = np.sqrt(d(Q, Q))
        pb = np.zeros((len(p), 4, 4))
        pb[:, 0, 0] = pb[:, 0, 3] = rs2 / 2
        pb[:, 1, 0] = rs2 / 2
        pb[:, 1, 3] = -rs2 / 2
        pb[:, 2], pb[:, 3] = p[:, 2], p[:, 3]  # O(E_g) mismatch of frames only
        m2 = P.me2(born, pb, PAR)
        devs.append(np.max(np.abs(m3 / (eik * m2) - 1)))
    assert devs[0] < 5e-2 and devs[1] < 5e-4 and devs[2] < 5e-6
    assert devs[1] < devs[0] / 30 and devs[2] < 1e-7  # approaches 1 at least linearly, down to rounding


def test_cfg3_soft_gluon_limit_pins_normalisation():
    """Soft limit of u d~ -> e+ ve g g onto u d~ -> e+ ve g with the colour-correlated eikonal factor
    (one colour structure T^a_ij, so <T_i.T_j> = (C_k - C_i - C_j)/2 |M|^2):
        |M_gg|^2 -> 1/2 * g_s^2 [ 3 S_qg + 3 S_q~g - (1/3) S_qq~ ] |M_g|^2 ,  S_ij = p_i.p_j / (p_i.k p_j.k).
    Together with the soft limit of u d~ -> e+ ve g onto the closed form of config 1 this fixes the absolute
    normalisation of config 3."""
    d = inputs.mdot
    one_g = P.Process('x', ['u', 'd~'], ['e+', 've', 'g'], ['udw', 'enw', 'uug', 'ddg'])
    rng = np.random.default_rng(9)
    n = 6
    # hard configuration: u d~ -> e+ ve g from RAMBO, then a soft gluon k; recoil absorbed by rescaling the beams
    from oracle import philox
    u = philox.uniforms(99, 0, n, 12, 7)
    devs = []
    for eg in (1e-1, 1e-3, 1e-5):
        rs = 1000.0
        pf, _ = ps.rambo_massless(u, 3, rs)
        ct, ph = rng.uniform(-0.5, 0.5, n), rng.uniform(0, 2 * np.pi, n)
        st = np.sqrt(1 - ct * ct)
        k = eg * np.stack([np.ones(n), st * np.cos(ph), st * np.sin(ph), ct], 1)
        tot = pf.sum(1) + k
        # go to the rest frame of (hard system + soft gluon) and put massless beams along +-z there
        M = np.sqrt(d(tot, tot))
        Pm = tot.copy()
        Pm[:, 1:] *= -1.0  # boosting with -P brings P to rest
        pf = np.stack([ps.boost(pf[:, i], Pm, M, 0.0) for i in range(3)], 1)
        k = ps.boost(k, Pm, M, 0.0)
        pa = np.stack([M / 2, 0 * M, 0 * M, M / 2], 1)
        pb = np.stack([M / 2, 0 * M, 0 * M, -M / 2], 1)
        p4 = np.stack([pa, pb, pf[:, 0], pf[:, 1], pf[:, 2], k], 1)
        m4 = P.me2(P.config(3), p4, PAR)
        p3 = p4[:, :5].copy()  # momentum not conserved by O(E_g): fine for the limit
        m3 = P.me2(one_g, p3, PAR)
        S = lambda i, j: d(p4[:, i], p4[:, j]) / (d(p4[:, i], k) * d(p4[:, j], k))
        eik = 0.5 * C['gs'] ** 2 * (3 * S(0, 4) + 3 * S(1, 4) - S(0, 1) / 3.0)
        devs.append(np.max(np.abs(m4 / (eik * m3) - 1)))
    assert devs[0] < 5e-2 and devs[1] < 5e-4 and devs[2] < 5e-6, devs


def test_w_plus_one_gluon_soft_limit_onto_cfg1():
    d = inputs.mdot
    one_g = P.Process('x', ['u', 'd~'], ['e+', 've', 'g'], ['udw', 'enw', 'uug', 'ddg'])
    devs = []
    for eg in (1e-2, 1e-4):
        p = _with_soft_gluon(80.0, eg, 10, seed=6)
        m3 = P.me2(one_g, p, PAR)
        eik = C['gs'] ** 2 * (4.0 / 3) * 2 * d(p[:, 0], p[:, 1]) / (d(p[:, 0], p[:, 4]) * d(p[:, 1], p[:, 4]))
        s = d(p[:, 2] + p[:, 3], p[:, 2] + p[:, 3])
        cf = 16 * d(p[:, 0], p[:, 2]) * d(p[:, 1], p[:, 3]) * C['gw'] ** 4 / \
            (48 * ((s - PAR['mw'] ** 2) ** 2 + (PAR['mw'] * PAR['gw']) ** 2))
        devs.append(np.max(np.abs(m3 / (eik * cf) - 1)))
    assert devs[0] < 5e-3 and devs[1] < 5e-5, devs


def test_four_quark_closed_forms_fix_the_fermi_sign():
    """Two quark lines: textbook massless QCD 2 -> 2 results.  q q' -> q q' has one diagram; q q -> q q and
    q q~ -> q q~ have two whose fermion lines pair the external legs differently: their interference carries the
    relative Fermi sign (oracle.feynman.fermion_sign) and the colour-suppressed factor.  With the wrong sign the
    interference term flips: the ratios below are off by 20-60 %."""
    from oracle import feynman as fy
    gs4 = sm.couplings(PAR)['gs'] ** 4
    p = inputs.two_to_two(500.0, 0.0, 0.0, 16, seed=3, cmax=0.8)
    s, t, u = inputs.mandelstam(p)
    cases = [
        (P.Process('ud_ud', ['u', 'd'], ['u', 'd'], ['uug', 'ddg']), (4 / 9) * (s * s + u * u) / (t * t)),
        (P.Process('uu_uu', ['u', 'u'], ['u', 'u'], ['uug']),
         ((4 / 9) * ((s * s + u * u) / (t * t) + (s * s + t * t) / (u * u)) - (8 / 27) * s * s / (t * u)) / 2),
        (P.Process('uux_uux', ['u', 'u~'], ['u', 'u~'], ['uug']),
         (4 / 9) * ((s * s + u * u) / (t * t) + (t * t + u * u) / (s * s)) - (8 / 27) * u * u / (s * t)),
        (P.Process('uux_ddx', ['u', 'u~'], ['d', 'd~'], ['uug', 'ddg']), (4 / 9) * (t * t + u * u) / (s * s)),
    ]
    for proc, want in cases:
        got = P.me2(proc, p, PAR)
        assert np.allclose(got, gs4 * want, rtol=1e-12), proc.name
        assert np.allclose(P.me2_explicit_colour(proc, p[:3], PAR), got[:3], rtol=1e-12)
    roots = cases[2][0].diagrams(PAR)[0]
    assert sorted(fy.fermion_sign(r) for r in roots) == [-1, 1]
    assert [len(fy.fermion_lines(r)) for r in roots] == [2, 2]


def test_ww_fusion_closed_form():
    """u b -> h d t is pure t-channel W W fusion (one diagram: Z Z fusion would leave u b in the final state).  With
    the W W H coupling g_W m_W and left-handed currents,
        sum |M|^2 = (g_W^2/2)^2 (g_W m_W)^2 16 (p_u.p_b)(p_d.p_t) / (|D_1|^2 |D_2|^2),
    colour 9, average 1/36; D_i = q_i^2 - m_W^2 + i m_W Gamma_W on the space-like lines.  The top is taken massless
    here (t and b merely stand for a second quark doublet): with m_t != 0 the q_mu q_nu / m_W^2 term of the
    unitary-gauge propagator contributes through the non-conserved t b current."""
    par = dict(PAR, mt=0.0, gt=0.0)
    proc = P.Process('ub_hdt', ['u', 'b'], ['h', 'd', 't'], ['udw', 'tbw', 'wwh'])
    assert len(proc.diagrams(par)[0]) == 1
    from oracle import phase_space as ops
    from oracle import philox
    n, rs = 32, 1000.0
    u = philox.uniforms(5, 0, n, 12, 3)
    masses = np.stack([np.full(n, PAR['mh']), np.zeros(n), np.zeros(n)], 1)
    k, _ = ops.rambo_massive(u, masses, rs)
    p = np.zeros((n, 5, 4))
    p[:, 0] = [rs / 2, 0, 0, rs / 2]
    p[:, 1] = [rs / 2, 0, 0, -rs / 2]
    p[:, 2:] = k
    gw, mw, gam = sm.couplings(PAR)['gw'], PAR['mw'], PAR['gw']
    q1 = p[:, 0] - p[:, 3]
    q2 = p[:, 1] - p[:, 4]
    d1 = (inputs.mdot(q1, q1) - mw * mw) ** 2 + (mw * gam) ** 2
    d2 = (inputs.mdot(q2, q2) - mw * mw) ** 2 + (mw * gam) ** 2
    want = (gw ** 2 / 2) ** 2 * (gw * mw) ** 2 * 16 * inputs.mdot(p[:, 0], p[:, 1]) * inputs.mdot(p[:, 3], p[:, 4]) \
        / (d1 * d2) * 9 / 36
    assert np.allclose(P.me2(proc, p, par), want, rtol=1e-11)
