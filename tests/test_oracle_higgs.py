"""Pins of the oracle's Higgs-sector Feynman rules (FFS, VVS, VVSS, SSS).

None of these retypes the oracle's formulas: decay |M|^2 of H -> W W, Z Z, t t~ (textbook closed forms), the
Higgs-strahlung cross section q q~ -> Z H (textbook closed form in G_F), and the high-energy behaviour of
longitudinal amplitudes, which stays bounded only if the contact (VVSS), Higgs-exchange (SSS x VVS), Yukawa (FFS)
and gauge (VVS) terms have the right relative signs and sizes.
"""
import math

import numpy as np

from oracle import processes as opr
from oracle import sm as osm
from inputs import two_to_two_at


def _decay_momenta(M, m1, m2):
    pst = math.sqrt((M * M - (m1 + m2) ** 2) * (M * M - (m1 - m2) ** 2)) / (2 * M)
    d = np.array([0.3, -0.5, math.sqrt(1 - 0.09 - 0.25)]) * pst
    return np.array([[[M, 0, 0, 0], [math.hypot(pst, m1), *d], [math.hypot(pst, m2), *(-d)]]])


def test_higgs_decay_matrix_elements():
    par = dict(osm.default_params(), mh=500.0)
    c = osm.couplings(par)
    vev = 2 * par['mw'] / c['gw']
    mh = par['mh']
    # H -> W+ W-:  sum |M|^2 = (g mW)^2 [2 + (p1.p2)^2 / mW^4],  p1.p2 = (mH^2 - 2 mW^2)/2
    for vv, vtx, m, g in (('w+', 'wwh', par['mw'], c['gw'] * par['mw']), ('z', 'zzh', par['mz'], c['gz'] * par['mz'])):
        proc = opr.Process('h_vv', ['h'], [vv, 'w-' if vv == 'w+' else 'z'], [vtx])
        got = opr.me2(proc, _decay_momenta(mh, m, m), par)[0] * proc.ident_factor()
        p12 = 0.5 * (mh * mh - 2 * m * m)
        want = g * g * (2 + p12 * p12 / m ** 4)
        assert abs(got - want) <= 1e-12 * want, (vv, got, want)
    # H -> t t~:  sum |M|^2 = Nc (mt/v)^2 4 (p1.p2 - mt^2) = Nc (mt/v)^2 2 mH^2 beta^2
    proc = opr.Process('h_tt', ['h'], ['t', 't~'], ['tth'])
    got = opr.me2(proc, _decay_momenta(mh, par['mt'], par['mt']), dict(par, gt=0.0))[0]
    beta2 = 1 - 4 * par['mt'] ** 2 / mh ** 2
    want = 3 * (par['mt'] / vev) ** 2 * 2 * mh * mh * beta2
    assert abs(got - want) <= 1e-12 * want, (got, want)
    # H H H vertex: |M|^2 = (3 mH^2 / v)^2 whatever the momenta
    proc = opr.Process('h_hh', ['h'], ['h', 'h'], ['hhh'])
    got = opr.me2(proc, _decay_momenta(mh, 10.0, 20.0), par)[0] * 2
    assert abs(got - (3 * mh * mh / vev) ** 2) <= 1e-12 * got


def test_higgs_strahlung_cross_section():
    """sigma(q q~ -> Z H) = G_F^2 mZ^4 / (96 pi s) (v_q^2 + a_q^2) sqrt(lam) (lam + 12 mZ^2/s) / (1 - mZ^2/s)^2 / 3,
    v_q = 2 T3 - 4 Q sw2, a_q = 2 T3, lam = (1 - (mH+mZ)^2/s)(1 - (mH-mZ)^2/s), G_F/sqrt2 = gW^2 / (8 mW^2);
    1/3 is the colour average (the e+ e- formula has none).  Narrow: the s-channel Z width is set to 0."""
    par = dict(osm.default_params(), gz=0.0)
    c = osm.couplings(par)
    rs = 400.0
    s = rs * rs
    mz, mh = par['mz'], par['mh']
    proc = opr.Process('uux_zh', ['u', 'u~'], ['z', 'h'], ['uuz', 'zzh'])
    x, w = np.polynomial.legendre.leggauss(24)
    p = two_to_two_at(rs, mz, mh, x, 0.4)
    me = opr.me2(proc, p, par)
    lam = (1 - (mh + mz) ** 2 / s) * (1 - (mh - mz) ** 2 / s)
    pst = 0.5 * rs * math.sqrt(lam)
    sigma = (me * w).sum() * pst / (16 * math.pi * s * rs)      # int dcos |M|^2 p*/(16 pi s sqrt s)
    gf = math.sqrt(2) * c['gw'] ** 2 / (8 * par['mw'] ** 2)
    vq, aq = 2 * 0.5 - 4 * (2 / 3) * c['sw2'], 2 * 0.5
    want = gf * gf * mz ** 4 / (96 * math.pi * s) * (vq * vq + aq * aq) * math.sqrt(lam) * (lam + 12 * mz * mz / s) \
        / (1 - mz * mz / s) ** 2 / 3
    assert abs(sigma - want) <= 1e-10 * want, (sigma, want)


def _longitudinal(proc, rs, m3, m4, par, hel_idx):
    p = two_to_two_at(rs, m3, m4, np.array([0.3]), 0.7)
    per = opr.me2(proc, p, par, per_helicity=True)
    return sum(v[0] for h, v in per.items() if all(h[i] == 0 for i in hel_idx))


def test_unitarity_cancellations_fix_relative_couplings():
    par = dict(osm.default_params(), gw=0.0, gz=0.0, gh=0.0, gt=0.0)
    # H H -> W_L W_L: contact (VVSS) + t/u-channel W (VVS^2) + s-channel H (SSS x VVS); each grows like s/v^2
    proc = opr.Process('hh_ww', ['h', 'h'], ['w+', 'w-'], ['wwh', 'wwhh', 'hhh'])
    lo = _longitudinal(proc, 3.0e3, par['mw'], par['mw'], par, (2, 3))
    hi = _longitudinal(proc, 3.0e4, par['mw'], par['mw'], par, (2, 3))
    assert 0.5 < hi / lo < 2.0, (lo, hi)
    # a wrong contact term is seen: without it the same ratio is ~ (s_hi/s_lo)^2 = 1e4
    bad = opr.Process('hh_ww_bad', ['h', 'h'], ['w+', 'w-'], ['wwh', 'hhh'])
    assert _longitudinal(bad, 3.0e4, par['mw'], par['mw'], par, (2, 3)) > \
        1e3 * _longitudinal(bad, 3.0e3, par['mw'], par['mw'], par, (2, 3))
    # t t~ -> Z_L H: Z-exchange (VVS) against Higgs emission off the top (FFS): the m_t sqrt(s)/v^2 growth cancels
    proc = opr.Process('ttx_zh', ['t', 't~'], ['z', 'h'], ['ttz', 'tth', 'zzh'])
    lo = _longitudinal(proc, 3.0e3, par['mz'], par['mh'], par, (2,))
    hi = _longitudinal(proc, 3.0e4, par['mz'], par['mh'], par, (2,))
    assert 0.3 < hi / lo < 3.0, (lo, hi)
    bad = opr.Process('ttx_zh_bad', ['t', 't~'], ['z', 'h'], ['ttz', 'zzh'])
    assert _longitudinal(bad, 3.0e4, par['mz'], par['mh'], par, (2,)) > \
        30 * _longitudinal(bad, 3.0e3, par['mz'], par['mh'], par, (2,))
