"""Pins of the paper's hadronic phase-space parameterisation (oracle/phase_space_had.py; Eq. 24-28, App. A).

The weight formula is checked against INDEPENDENT Monte-Carlo evaluations of the same restricted integrals: momentum
fractions drawn flat, the final state from the textbook two-body formula or from flat RAMBO (itself pinned in
tests/test_oracle_phase_space.py), the ranges of the paper's variables applied as cuts afterwards."""
import math

import numpy as np

from oracle import phase_space as ops
from oracle import phase_space_had as had
from oracle import philox
from oracle import sm
import inputs

PAR = sm.default_params()
RS = 1000.0


def _rap(k):
    with np.errstate(invalid='ignore', divide='ignore'):
        return 0.5 * np.log((k[..., 0] + k[..., 3]) / (k[..., 0] - k[..., 3]))


def _pt(k):
    return np.hypot(k[..., 1], k[..., 2])


def _paper_estimate(n, m_last, ymax, yres, ptmin, N, seed):
    """Mean of the generalised phase-space weight over the box |y_i| < ymax (i < n), pT_i in [ptmin, sqrt(s)/2],
    |y_n| < yres, with x_a, x_b < 1."""
    s = RS * RS
    u = philox.uniforms(seed, 0, N, 3 * n - 2, 77)
    y = np.empty((N, n))
    y[:, :n - 1] = ymax * (2 * u[:, :n - 1] - 1)
    y[:, n - 1] = yres * (2 * u[:, n - 1] - 1)
    l0, l1 = math.log(ptmin ** 2), math.log(s / 4)
    lnpt = l0 + (l1 - l0) * u[:, n:2 * n - 1]
    phi = had.TWO_PI * u[:, 2 * n - 1:3 * n - 2]
    m2 = np.zeros((N, n))
    m2[:, n - 1] = m_last ** 2
    k, xa, xb, w = had.generalised(y, lnpt, phi, m2, s)
    w = w * (2 * ymax) ** (n - 1) * (2 * yres) * (l1 - l0) ** (n - 1) * ((xa < 1) & (xb < 1))
    # the point really is a point of phase space: momentum conservation with the incoming partons, mass shells
    tot = k.sum(1)
    assert np.allclose(tot[:, 0], 0.5 * RS * (xa + xb)) and np.allclose(tot[:, 3], 0.5 * RS * (xa - xb))
    assert np.abs(tot[:, 1:3]).max() < 1e-9 * RS
    assert np.allclose(inputs.mdot(k, k), m2, atol=1e-6 * s)
    return w.mean(), w.std() / math.sqrt(N), np.mean(w > 0)


def _box(k, ymax, yres, ptmin):
    n = k.shape[1]
    ok = np.abs(_rap(k[:, n - 1])) < yres
    for i in range(n - 1):
        ok &= (np.abs(_rap(k[:, i])) < ymax) & (_pt(k[:, i]) > ptmin)
    return ok


def _boost_z(k, xa, xb):
    """Partonic CM frame -> lab: boost along z with rapidity ln(xa/xb)/2."""
    yc = 0.5 * np.log(xa / xb)
    ch, sh = np.cosh(yc)[:, None], np.sinh(yc)[:, None]
    out = k.copy()
    out[..., 0] = ch * k[..., 0] + sh * k[..., 3]
    out[..., 3] = sh * k[..., 0] + ch * k[..., 3]
    return out


def test_two_body_against_textbook():
    """n = 2, masses (0, M): int dx_a dx_b dPhi_2 over the box, dPhi_2 = (s_hat - M^2)/(8 pi s_hat) dcos/2 dphi/2pi."""
    M, ymax, yres, ptmin, N = 80.0, 2.5, 3.0, 20.0, 1500000
    est, err, eff = _paper_estimate(2, M, ymax, yres, ptmin, N, 5)
    rng = np.random.default_rng(12)
    xa, xb = rng.uniform(0, 1, N), rng.uniform(0, 1, N)
    sh = xa * xb * RS * RS
    live = sh > M * M
    pst = np.where(live, (sh - M * M) / (2 * np.sqrt(np.where(live, sh, 1.0))), 0.0)
    c, f = rng.uniform(-1, 1, N), rng.uniform(0, 2 * math.pi, N)
    st = np.sqrt(1 - c * c)
    d = np.stack([st * np.cos(f), st * np.sin(f), c], 1) * pst[:, None]
    k = np.empty((N, 2, 4))
    k[:, 0, 0], k[:, 0, 1:] = pst, d
    k[:, 1, 0], k[:, 1, 1:] = np.sqrt(pst ** 2 + M * M), -d
    k = _boost_z(k, xa, xb)
    wt = np.where(live, (sh - M * M) / (8 * math.pi * np.where(live, sh, 1.0)), 0.0) * _box(k, ymax, yres, ptmin)
    ref, rerr = wt.mean(), wt.std() / math.sqrt(N)
    assert err / est < 0.01 and rerr / ref < 0.01
    assert abs(est - ref) < 4 * math.hypot(err, rerr), (est, err, ref, rerr)
    assert 0.3 < eff < 1.0


def test_three_body_against_rambo():
    """n = 3, masses (0, 0, M): the power of 4 pi, the product over i < n and A.9 for more than one free particle."""
    M, ymax, yres, ptmin, N = 80.0, 2.5, 3.0, 20.0, 1500000
    est, err, eff = _paper_estimate(3, M, ymax, yres, ptmin, N, 6)
    rng = np.random.default_rng(13)
    xa, xb = rng.uniform(0, 1, N), rng.uniform(0, 1, N)
    rsh = np.sqrt(xa * xb) * RS
    live = rsh > M + 1.0
    idx = np.nonzero(live)[0]
    u = rng.uniform(0, 1, (len(idx), 12))
    masses = np.stack([np.zeros(len(idx)), np.zeros(len(idx)), np.full(len(idx), M)], 1)
    # oracle.rambo_massive takes one sqrt(s) for the whole batch: generate at sqrt(s) = 1 with masses m / sqrt(s_hat)
    # and scale the momenta back (dPhi_3 has the dimension energy^2)
    kk, ww = ops.rambo_massive(u, masses / rsh[idx][:, None], 1.0)
    k = kk * rsh[idx][:, None, None]
    w = ww * rsh[idx] ** 2
    klab = _boost_z(k, xa[idx], xb[idx])
    wt = np.zeros(N)
    wt[idx] = w * _box(klab, ymax, yres, ptmin)
    ref, rerr = wt.mean(), wt.std() / math.sqrt(N)
    assert err / est < 0.015 and rerr / ref < 0.015
    assert abs(est - ref) < 4 * math.hypot(err, rerr), (est, err, ref, rerr)


def test_w_plus_two_jets_generator():
    """from_uniforms(cfg 3) with unit parton densities: mean of w * (s_hat / s) * BW(s_W) against the same integral
    done by hand: flat x_a, x_b, flat s_W in the Breit-Wigner window, flat RAMBO for (g, g, W*), the decay factor
    1/(8 pi), ranges as cuts.  The Breit-Wigner test function cancels the Jacobian of the mapping (small variance)."""
    cfg, N = 3, 1000000
    hd = dict(y_res_max=3.0, pdf_norm=(1.0, 1.0), pdf_a=(0.0, 0.0), pdf_b=(0.0, 0.0))
    cuts = (20.0, 2.5, 0.0, 0.0)
    u = philox.uniforms(9, 0, N, 16, cfg)
    p, w, valid = had.from_uniforms(cfg, u, RS, PAR, hd, cuts)
    mw, gw = PAR['mw'], PAR['gw']
    bw = lambda s_: mw * gw / ((s_ - mw * mw) ** 2 + (mw * gw) ** 2)
    sW = inputs.mdot(p[:, 2] + p[:, 3], p[:, 2] + p[:, 3])
    xa, xb = p[:, 0, 0] / (0.5 * RS), p[:, 1, 0] / (0.5 * RS)
    f = w * xa * xb * bw(sW)                        # w carries s / s_hat = 1 / (x_a x_b)
    est, err = f.mean(), f.std() / math.sqrt(N)
    # valid points are physical events: momentum conservation, massless legs, inside the ranges
    v = valid
    assert np.abs((p[v, 0] + p[v, 1] - p[v, 2:].sum(1))).max() < 1e-8 * RS
    assert np.abs(inputs.mdot(p[v, 2:], p[v, 2:])).max() < 1e-7 * RS * RS
    assert np.all(_pt(p[v, 4:]) > 20.0 * (1 - 1e-12)) and np.all(np.abs(_rap(p[v, 4:])) < 2.5 + 1e-9)
    assert np.all(w[~v] == 0) and 0.2 < v.mean() < 1.0
    # by hand
    rng = np.random.default_rng(21)
    M = N
    xa2, xb2 = rng.uniform(0, 1, M), rng.uniform(0, 1, M)
    lim = min(20.0, mw / gw)
    s_lo, s_hi = mw * mw - lim * mw * gw, mw * mw + lim * mw * gw
    sw2 = rng.uniform(s_lo, s_hi, M)
    rsh = np.sqrt(xa2 * xb2) * RS
    live = rsh > np.sqrt(sw2) + 1.0
    idx = np.nonzero(live)[0]
    uu = rng.uniform(0, 1, (len(idx), 12))
    masses = np.stack([np.zeros(len(idx)), np.zeros(len(idx)), np.sqrt(sw2[idx])], 1)
    kk, ww = ops.rambo_massive(uu, masses / rsh[idx][:, None], 1.0)
    klab = _boost_z(kk * rsh[idx][:, None, None], xa2[idx], xb2[idx])
    wt = np.zeros(M)
    wt[idx] = ww * rsh[idx] ** 2 * _box(klab, 2.5, 3.0, 20.0) * bw(sw2[idx]) * (s_hi - s_lo) / (2 * math.pi) / (8 * math.pi)
    ref, rerr = wt.mean(), wt.std() / math.sqrt(M)
    assert err / est < 0.02 and rerr / ref < 0.02
    assert abs(est - ref) < 4 * math.hypot(err, rerr), (est, err, ref, rerr)


def test_parton_densities_and_null_weight():
    cfg, N = 5, 20000
    hd = had.default_hadronic(cfg)
    p, w, valid = had.generate(cfg, 3, 0, N, 14000.0, PAR, hd)
    flat = dict(hd, pdf_norm=(1.0, 1.0), pdf_a=(0.0, 0.0), pdf_b=(0.0, 0.0))
    p1, w1, valid1 = had.generate(cfg, 3, 0, N, 14000.0, PAR, flat)
    assert np.array_equal(p, p1) and np.array_equal(valid, valid1)
    xa, xb = p[:, 0, 0] / 7000.0, p[:, 1, 0] / 7000.0
    want = w1[valid] * had.pdf(xa[valid], 2.2, 0.5, 3.0) * had.pdf(xb[valid], 0.2, 1.2, 7.0)
    assert np.allclose(w[valid], want, rtol=1e-13)
    assert np.all(w[~valid] == 0.0) and np.all((xa[valid] < 1) & (xb[valid] < 1))
    # generation efficiency under the cuts, the reason for this parameterisation (42 % and 29 % of
    # the points survive for 3 and 4 massless particles); here W + 3 jets with the Delta R cuts applied afterwards
    ok = ops.passes(cfg, p) & valid
    assert 0.2 < ok.mean() < 0.6, ok.mean()
