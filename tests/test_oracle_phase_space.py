"""Pins of the oracle's Philox, RAMBO, Breit-Wigner mapping, decays and cuts (SURVEY.md 8c 'Phase space', A14-A16)."""
import math

import numpy as np
import pytest
from scipy import integrate as sci

from oracle import philox
from oracle import phase_space as ps
from oracle import sm
import inputs

PAR = sm.default_params()


def test_philox_known_answers():
    """Known-answer vectors of the published Philox4x32-10 algorithm (Random123 KAT file)."""
    kat = [((0, 0, 0, 0), (0, 0), '6627e8d5 e169c58d bc57ac4c 9b00dbd8'),
           ((0xffffffff,) * 4, (0xffffffff,) * 2, '408f276d 41c83b0e a20bc7c6 6d5451fd'),
           ((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0),
            'd16cfe09 94fdcceb 5001e420 24126ea1')]
    for c, k, want in kat:
        r = philox.philox4x32_10([np.array([x], dtype=np.uint64) for x in c], [np.uint64(x) for x in k])
        assert ' '.join('%08x' % int(x[0]) for x in r) == want


def test_uniform_layout_and_range():
    u = philox.uniforms(42, 1000, 4096, 24, 4)
    assert u.shape == (4096, 24) and u.min() > 0 and u.max() < 1
    # counter-based: a split batch reproduces the same numbers (determinism contract)
    v = philox.uniforms(42, 1000 + 100, 50, 24, 4)
    assert np.array_equal(u[100:150], v)
    # draw d of event k = words (2d mod 4, 2d+1 mod 4) of block d//2, 52-bit mantissa + 1/2
    w = philox.philox4x32_10([np.array([1003], dtype=np.uint64), np.array([0], dtype=np.uint64),
                              np.array([1], dtype=np.uint64), np.array([4], dtype=np.uint64)], (42, 0))
    lo, hi = int(w[2][0]), int(w[3][0])
    assert u[3, 3] == ((hi >> 6) * (1 << 26) + (lo >> 6) + 0.5) / float(1 << 52)
    # moments of U(0,1)
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12.0 / u.size)
    assert abs((u ** 2).mean() - 1 / 3.0) < 4 * math.sqrt(4 / 45.0 / u.size)


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_rambo_massless(n):
    N = 20000
    rs = 1000.0
    u = philox.uniforms(7, 0, N, 4 * n, n)
    p, w = ps.rambo_massless(u, n, rs)
    tot = p.sum(1)
    # conservation and mass shell to 1e-13 sqrt(s_hat) for every event (SURVEY.md 8c 'Phase space' pin): reading A16b
    # puts the point back on the constraint surface after the ill-conditioned conformal map
    dev = np.maximum(np.abs(tot[:, 0] - rs), np.abs(tot[:, 1:]).max(1))
    assert dev.max() < 1e-13 * rs
    assert np.abs(inputs.mdot(p, p)).max() < 1e-13 * rs * rs
    assert (p[:, :, 0] > 0).all()
    # flat weight = n-body massless phase-space volume; n=2: 1/(8 pi); n=3: s/(256 pi^3)
    vol = {2: 1 / (8 * math.pi), 3: rs ** 2 / (256 * math.pi ** 3),
           4: rs ** 4 / (24576 * math.pi ** 5), 5: rs ** 6 / (4718592 * math.pi ** 7)}[n]
    assert np.allclose(w, vol, rtol=1e-13)
    if n >= 3:
        # energy fraction x = 2E/sqrt(s) of any particle is distributed as x (1-x)^(n-3): <x^2> = 6/(n(n+1))
        for i in range(n):
            x = 2 * p[:, i, 0] / rs
            m2 = 6.0 / (n * (n + 1))
            assert abs((x ** 2).mean() - m2) < 5 * (x ** 2).std() / math.sqrt(N)
        # isotropy: <cos^2 theta> = 1/3
        c = p[:, 0, 3] / p[:, 0, 0]
        assert abs((c ** 2).mean() - 1 / 3.0) < 5 * (c ** 2).std() / math.sqrt(N)


def test_rambo_massive_two_body_weight():
    """n=2 massive weight = lambda^(1/2)(s, m1^2, m2^2) / (8 pi s)."""
    N = 64
    rs = 500.0
    m = np.stack([np.full(N, 174.3), np.full(N, 80.4)], 1)
    u = philox.uniforms(3, 0, N, 8, 2)
    k, w = ps.rambo_massive(u, m, rs)
    s = rs * rs
    lam = (s - m[0, 0] ** 2 - m[0, 1] ** 2) ** 2 - 4 * m[0, 0] ** 2 * m[0, 1] ** 2
    assert np.allclose(w, math.sqrt(lam) / (8 * math.pi * s), rtol=1e-12)
    assert np.abs(k.sum(1) - np.array([rs, 0, 0, 0])).max() < 1e-10
    assert np.allclose(inputs.mdot(k, k), m ** 2, rtol=1e-11)


def test_rambo_massive_three_body_volume():
    """MC mean of the massive-RAMBO weight = Phi_3(s; m1, m2, 0) = int ds12/(2 pi) Phi_2(s; s12, 0) Phi_2(s12; m1, m2)."""
    N = 40000
    rs = 1500.0
    m1, m2 = 174.3, 160.0
    m = np.stack([np.full(N, m1), np.full(N, m2), np.zeros(N)], 1)
    u = philox.uniforms(11, 0, N, 12, 3)
    k, w = ps.rambo_massive(u, m, rs)
    assert np.abs(k.sum(1) - np.array([rs, 0, 0, 0])).max() < 1e-9
    assert np.allclose(inputs.mdot(k, k), m ** 2, atol=1e-6)
    s = rs * rs

    def phi2(M2, a, b):
        return math.sqrt(max((M2 - a - b) ** 2 - 4 * a * b, 0.0)) / (8 * math.pi * M2)

    vol, _ = sci.quad(lambda s12: phi2(s, s12, 0.0) * phi2(s12, m1 * m1, m2 * m2) / (2 * math.pi),
                      (m1 + m2) ** 2, s, epsabs=0, epsrel=1e-10)
    assert abs(w.mean() - vol) < 4 * w.std() / math.sqrt(N)
    assert abs(w.mean() / vol - 1) < 0.01


def test_breit_wigner_map():
    """int over the window of m Gamma / ((s-m^2)^2 + m^2 Gamma^2) ds = 2 atan(min(20, m/Gamma))  (A.13-A.15)."""
    for m, g, lim in ((PAR['mt'], PAR['gt'], 20.0), (PAR['mw'], PAR['gw'], 20.0), (10.0, 2.0, 5.0)):
        u = (np.arange(200000) + 0.5) / 200000
        s, jac = ps.bw_mass(u, m, g)
        assert abs((abs(s - m * m) / (m * g)).max() - lim) < 1e-2
        integrand = m * g / ((s - m * m) ** 2 + (m * g) ** 2) * jac * 2 * math.pi
        assert np.allclose(integrand, 2 * math.atan(lim), rtol=1e-12)  # the map flattens the Breit-Wigner exactly
    st, _ = ps.bw_mass(np.array([1e-12, 1 - 1e-12]), PAR['mt'], PAR['gt'])
    sw, _ = ps.bw_mass(np.array([1e-12, 1 - 1e-12]), PAR['mw'], PAR['gw'])
    assert np.allclose(np.sqrt(st), [158.6, 188.7], atol=0.1) and np.allclose(np.sqrt(sw), [56.3, 98.8], atol=0.1)  # A14


def test_two_body_decay():
    N = 1000
    rng = np.random.default_rng(0)
    P = np.zeros((N, 4))
    P[:, 1:] = rng.normal(size=(N, 3)) * 200
    M2 = np.full(N, 174.3 ** 2)
    P[:, 0] = np.sqrt(M2 + (P[:, 1:] ** 2).sum(1))
    m2sq = np.full(N, 80.0 ** 2)
    a, b, w = ps.two_body(P, M2, np.zeros(N), m2sq, rng.uniform(size=N), rng.uniform(size=N))
    assert np.abs(a + b - P).max() < 1e-10
    assert np.abs(inputs.mdot(a, a)).max() < 1e-8 and np.allclose(inputs.mdot(b, b), m2sq, rtol=1e-11)
    pst = (174.3 ** 2 - 80.0 ** 2) / (2 * 174.3)
    assert np.allclose(w, pst / (4 * math.pi * 174.3))  # = lambda^(1/2) / (8 pi M^2)


def test_cfg4_generation():
    N = 5000
    p, w = ps.generate(4, 9, 0, N, 1500.0, PAR)
    assert np.abs(p[:, 0] + p[:, 1] - p[:, 2:].sum(1)).max() < 1e-9
    assert np.abs(inputs.mdot(p[:, 2:], p[:, 2:])).max() < 1e-6
    st = inputs.mdot(p[:, 2] + p[:, 3] + p[:, 4], p[:, 2] + p[:, 3] + p[:, 4])
    sw = inputs.mdot(p[:, 3] + p[:, 4], p[:, 3] + p[:, 4])
    stb = inputs.mdot(p[:, 5:8].sum(1), p[:, 5:8].sum(1))
    assert (np.sqrt(st) > 158.5).all() and (np.sqrt(st) < 188.8).all() and (np.sqrt(stb) > 158.5).all()
    assert (np.sqrt(sw) > 56.2).all() and (np.sqrt(sw) < 98.9).all()
    assert (w > 0).all()
    # half of the BW-mapped points lie within |s - m^2| < m Gamma  (atan 1 / atan 20 = 0.5158)
    frac = np.mean(np.abs(st - PAR['mt'] ** 2) < PAR['mt'] * PAR['gt'])
    assert abs(frac - math.atan(1) / math.atan(20)) < 4 * 0.5 / math.sqrt(N)


def test_cuts():
    # hand-made momenta: leg order of config 3 (u d~ e+ ve g g)
    def v(pt, eta, phi):
        return [pt * math.cosh(eta), pt * math.cos(phi), pt * math.sin(phi), pt * math.sinh(eta)]
    p = np.zeros((4, 6, 4))
    p[:, 2] = v(30, 0, 0)
    p[:, 3] = v(30, 0, 1)
    p[0, 4], p[0, 5] = v(25, 0.0, 0.0), v(25, 0.0, 1.0)  # pass
    p[1, 4], p[1, 5] = v(19.9, 0.0, 0.0), v(25, 0.0, 1.0)  # pT fail
    p[2, 4], p[2, 5] = v(25, 0.0, 0.0), v(25, 0.3, 0.2)  # dR = 0.36 fail
    p[3, 4], p[3, 5] = v(25, 0.0, 3.1), v(25, 0.0, -3.1)  # dphi wraps: dR = 0.083 fail
    assert list(ps.passes(3, p)) == [True, False, False, False]
    assert np.isclose(ps.delta_r(p[2:3, 4], p[2:3, 5])[0], math.hypot(0.3, 0.2))
    assert np.isclose(ps.delta_r(p[3:4, 4], p[3:4, 5])[0], 2 * math.pi - 6.2)
    assert np.isclose(ps.eta(np.array([v(10, 1.7, 0.4)]))[0], 1.7)
    # eta cut of config 5
    q = np.zeros((2, 7, 4))
    q[:, 2] = v(30, 0, 0)
    q[0, 4], q[0, 5], q[0, 6] = v(25, 0, 0), v(25, 0, 2), v(25, 2.4, 4)
    q[1, 4], q[1, 5], q[1, 6] = v(25, 0, 0), v(25, 0, 2), v(25, -2.6, 4)
    assert list(ps.passes(5, q)) == [True, False]


def test_cfg4_nested_volume():
    """Pin of oracle.phase_space.generate(cfg=4) as a whole (SURVEY.md 8c 'cfg4 total volume vs nested closed form';
    Eq. 25-27): the Monte-Carlo mean of  w * prod_k BW_k(s_k),  BW_k(s) = m G / ((s - m^2)^2 + m^2 G^2)
    with the s_k re-measured from the generated momenta, equals the nested integral

        int prod_k ds_k/(2 pi) BW_k(s_k)  Phi_3(s_hat; s_t, s_t~, 0)  Phi_2(s_t; 0, s_W+) Phi_2(s_W+; 0, 0)
                                                                      Phi_2(s_t~; 0, s_W-) Phi_2(s_W-; 0, 0)

    over the four Breit-Wigner windows (A14), evaluated here by independent quadrature.  The Breit-Wigner test
    function cancels the Jacobian of the mapping, so the Monte-Carlo variance is that of the phase-space factors
    only and 4e4 points give 0.3 %: a missing 1/(2 pi) of one resonance, a dropped two-body factor or a wrong power
    of the massive-RAMBO weight changes the mean by tens of per cent or more."""
    N, rs = 40000, 1500.0
    p, w = ps.generate(4, 77, 0, N, rs, PAR)
    mt, gt, mw, gw = PAR['mt'], PAR['gt'], PAR['mw'], PAR['gw']

    def bw(s, m, g):
        return m * g / ((s - m * m) ** 2 + (m * g) ** 2)

    def inv(legs):
        q = p[:, legs].sum(1)
        return inputs.mdot(q, q)

    f = w * bw(inv([2, 3, 4]), mt, gt) * bw(inv([5, 6, 7]), mt, gt) * bw(inv([3, 4]), mw, gw) * bw(inv([6, 7]), mw, gw)

    def phi2(M2, a, b):
        return math.sqrt(max((M2 - a - b) ** 2 - 4 * a * b, 0.0)) / (8 * math.pi * M2)

    def window(m, g):
        lim = min(20.0, m / g)
        return m * m - lim * m * g, m * m + lim * m * g

    def h(s_top):
        """int ds_W/(2 pi) BW_W(s_W) Phi_2(s_top; 0, s_W) Phi_2(s_W; 0, 0)."""
        lo, hi = window(mw, gw)
        v, _ = sci.quad(lambda sw: bw(sw, mw, gw) * phi2(s_top, 0.0, sw) * phi2(sw, 0.0, 0.0) / (2 * math.pi),
                        lo, hi, points=[mw * mw], epsabs=0, epsrel=1e-10)
        return v

    def phi3(s1, s2):
        """Phi_3(s_hat; s1, s2, 0) = int ds12/(2 pi) Phi_2(s_hat; s12, 0) Phi_2(s12; s1, s2)."""
        v, _ = sci.quad(lambda s12: phi2(rs * rs, s12, 0.0) * phi2(s12, s1, s2) / (2 * math.pi),
                        (math.sqrt(s1) + math.sqrt(s2)) ** 2, rs * rs, epsabs=0, epsrel=1e-9)
        return v

    # outer two integrals over s_t, s_t~: Gauss-Legendre in theta = atan((s - m^2)/(m G)), which resolves the peaks
    # (ds BW(s) = d theta); the integrand left over is smooth
    x, wt = np.polynomial.legendre.leggauss(12)
    tmax = math.atan(min(20.0, mt / gt))
    s_nodes = mt * mt + mt * gt * np.tan(tmax * x)
    hv = np.array([h(s) for s in s_nodes])
    total = 0.0
    for i in range(len(x)):
        for j in range(len(x)):
            total += wt[i] * wt[j] * phi3(s_nodes[i], s_nodes[j]) * hv[i] * hv[j]
    exact = total * (tmax / (2 * math.pi)) ** 2
    err = f.std() / math.sqrt(N)
    assert err / f.mean() < 0.01
    assert abs(f.mean() - exact) < 4 * err, (f.mean(), exact, err)
    assert abs(f.mean() / exact - 1) < 0.02
