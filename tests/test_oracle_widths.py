"""Pins of the oracle's treatment of unstable particles (widths, decay chains):  the position of the propagator
pole (sign of +i m Gamma) and the exact factorisation of the decayed amplitude at
the resonance poles (config 4 against undecayed g g -> t t~ g, SURVEY.md 8c 'cfg4 decays')."""
import itertools
import math

import numpy as np
import pytest

from oracle import feynman as fy
from oracle import processes as opr
from oracle import sm
import inputs

PAR = sm.default_params()


@pytest.mark.parametrize('field', ['h', 'z', 'w+', 't', 't~'])
def test_propagator_pole_is_in_the_lower_half_plane(field):
    """A state of mass m and width Gamma evolves as exp(-i m t - Gamma t / 2): as a function of complex energy (at
    rest) its propagator has the pole of the positive-energy state at E = sqrt(m^2 - i m Gamma) ~ m - i Gamma/2,
    BELOW the real axis.  This fixes the sign of the width term in 1/(q^2 - m^2 + i m Gamma), which no helicity-
    summed |M|^2 pin sees (|D|^2 and the gamma/Z interference are even in Gamma).  With the other sign the pole of
    _propagate moves to m + i Gamma/2 and both assertions fail."""
    m, w = fy.mass_width(field, PAR)
    assert m > 0 and w > 0
    pole = np.sqrt(complex(m * m, -m * w))
    assert pole.imag < 0 and abs(pole.imag + w / 2) < 1e-3 * w

    def size(E):
        K = np.array([[E, 0, 0, 0]], dtype=complex)
        cur = np.ones(1, dtype=complex) if fy.spin(field) == 'S' else np.ones((1, 4), dtype=complex)
        return float(np.abs(fy._propagate(field, K, cur, PAR)).max())

    on_axis = size(pole.real)                      # a distance Gamma/2 from the pole
    near = size(pole + 1e-3 * w)                   # 500 times closer
    mirrored = size(np.conj(pole) + 1e-3 * w)      # the same point reflected above the axis: twice as far
    assert near > 100 * on_axis          # the pole is there ...
    assert mirrored < on_axis            # ... and not at the mirror point


def _event(n_t, n_wp, n_tb, n_wm, rs=1500.0):
    """g g -> t t~ g with on-shell tops, then t -> b W+ (W+ along -n_t... b along n_t in the t frame), W+ -> e+ ve
    (e+ along n_wp in the W frame), same for t~; every resonance exactly on its pole."""
    mt, mw = PAR['mt'], PAR['mw']
    tot = np.array([rs, 0.0, 0.0, 0.0])
    g_dir = np.array([0.3, -0.5, 0.4])
    g_dir /= np.linalg.norm(g_dir)
    eg = 210.0
    mtt = math.sqrt(rs * rs - 2 * rs * eg)
    g, tt = decay(tot, 0.0, mtt, g_dir)
    d = np.array([0.6, 0.2, -0.7])
    d /= np.linalg.norm(d)
    t, tb = decay(tt, mt, mt, d)
    b, wp = decay(t, 0.0, mw, n_t)
    ep, ve = decay(wp, 0.0, 0.0, n_wp)
    bb, wm = decay(tb, 0.0, mw, n_tb)
    mu, vm = decay(wm, 0.0, 0.0, n_wm)
    pa = np.array([rs / 2, 0, 0, rs / 2])
    pb = np.array([rs / 2, 0, 0, -rs / 2])
    full = np.array([pa, pb, b, ep, ve, bb, mu, vm, g])
    prod = np.array([pa, pb, t, tb, g])
    return full, prod


decay = inputs.decay


def test_cfg4_factorises_on_the_poles():
    """With s_t = s_t~ = m_t^2 and s_W+- = m_W^2 exactly, every resonant propagator numerator is the spin sum of
    on-shell wavefunctions, so the config-4 amplitude is  sum_spins M_prod * M_dec(t) * M_dec(t~) / (i m_t G_t)^2.
    Averaged over the decay directions the spin correlations drop out (rotational invariance in the top rest frame):

        < |Mbar(g g -> b e+ ve b~ mu- vm~ g)|^2 >  =  |Mbar(g g -> t t~ g)|^2 * prod_{t, t~} [ 1/2 <sum|M_dec|^2> / (m_t G_t)^2 ]

    with the textbook  sum_spins |M(t -> b e+ ve)|^2 = 4 g_W^4 (p_t.p_e+)(p_b.p_ve) / (m_W G_W)^2  on the W pole.
    The averages are exact sums over spherical 2-designs (the decay matrix is quadratic in the lepton momentum), so
    the identity holds to rounding, not to O(Gamma/m): it pins the relative signs and factors of the 16 decayed
    diagrams, the fermion and W propagators with widths, and the t b W / l nu W vertices against the undecayed
    process (itself pinned by the g g -> t t~ closed form, Ward identity and soft limit)."""
    mt, gt, mw, gw = PAR['mt'], PAR['gt'], PAR['mw'], PAR['gw']
    gW = sm.couplings(PAR)['gw']
    d1, d2 = inputs.tetrahedron(0.3), inputs.tetrahedron(1.1)
    fulls, decs = [], []
    for a, b, c, d in itertools.product(range(4), repeat=4):
        full, prod = _event(d1[a], d2[b], d2[c], d1[d])
        fulls.append(full)
        pt_, ptb = prod[2], prod[3]
        dec_t = 4 * gW ** 4 * inputs.mdot(pt_, full[3]) * inputs.mdot(full[2], full[4]) / (mw * gw) ** 2
        dec_tb = 4 * gW ** 4 * inputs.mdot(ptb, full[6]) * inputs.mdot(full[5], full[7]) / (mw * gw) ** 2
        decs.append((dec_t, dec_tb))
    fulls = np.array(fulls)
    decs = np.array(decs)
    lhs = opr.me2(opr.config(4), fulls, PAR).mean()
    undecayed = opr.Process('gg_ttxg', ['g', 'g'], ['t', 't~', 'g'], ['ttg', 'ggg', 'gggg'])
    prod_me = opr.me2(undecayed, prod[None], PAR)[0]
    rhs = prod_me * (0.5 * decs[:, 0].mean() / (mt * gt) ** 2) * (0.5 * decs[:, 1].mean() / (mt * gt) ** 2)
    assert abs(lhs / rhs - 1) < 1e-9, (lhs, rhs)
    # the directions matter event by event (spin correlations are there): the identity is not trivially true
    per_event = opr.me2(opr.config(4), fulls[:8], PAR) / (prod_me * 0.25 * decs[:8, 0] * decs[:8, 1] / (mt * gt) ** 4)
    assert np.abs(per_event - 1).max() > 0.05


# ---------------------------------------------------------------------------------------- complex-mass option
def test_complex_mass_is_the_analytic_continuation_in_the_masses():
    """Eq. 55-56: replacing m_V^2 by m_V^2 - i m_V Gamma_V everywhere (propagator denominators,
    q q / m_V^2 numerators, couplings) with mu_W^2 / mu_Z^2 = cos^2 theta_W is the same as evaluating the ZERO-WIDTH
    formulas at the complex masses m_V sqrt(1 - i Gamma_Z / m_Z).  The oracle's explicit option branches
    (complex_mass = 1) are compared with its plain formulas fed with complex mass parameters, for the processes whose
    W and Z lines are all internal and end on conserved or non-conserved currents alike (Z* -> Z H H, W W / Z Z
    fusion to H and H H).  A term that keeps the real mass (numerator, a coupling, the W width of Eq. 56) breaks the
    equality at O(Gamma / m) = 3e-2 x its weight."""
    from oracle import phase_space as ops
    cms = dict(PAR, complex_mass=1)
    fac = np.sqrt(complex(1.0, -PAR['gz'] / PAR['mz']))
    cont = dict(PAR, mw=PAR['mw'] * fac, mz=PAR['mz'] * fac, gw=0.0, gz=0.0)
    for cfg in (7, 10, 11):
        p, _ = ops.generate(cfg, 4, 0, 6, opr.SQRT_S[cfg], PAR)
        a = opr.me2(opr.config(cfg), p, cms)
        b = opr.me2(opr.config(cfg), p, cont)
        assert np.allclose(a, b, rtol=1e-12), (cfg, a, b)
        plain = opr.me2(opr.config(cfg), p, PAR)
        assert np.abs(a / plain - 1).max() > 1e-5          # the option does something
    # Eq. 56 fixes the W width; in the narrow limit the option changes nothing
    assert abs(sm.effective_widths(cms)[0] - PAR['mw'] * PAR['gz'] / PAR['mz']) < 1e-15
    narrow = dict(PAR, gw=1e-12, gz=1e-12)
    p, _ = ops.generate(11, 4, 0, 4, opr.SQRT_S[11], PAR)
    assert np.allclose(opr.me2(opr.config(11), p, dict(narrow, complex_mass=1)), opr.me2(opr.config(11), p, narrow),
                       rtol=1e-12)


def test_complex_mass_ww_fusion_closed_form():
    """The W W fusion closed form (tests/test_oracle_closed_forms.py) with the complex-mass option: the W W H coupling
    becomes g_W mu_W, |mu_W|^2 = m_W^2 sqrt(1 + (Gamma_W/m_W)^2), and both space-like propagators carry Eq. 56's
    width."""
    from oracle import phase_space as ops
    from oracle import philox
    par = dict(PAR, mt=0.0, gt=0.0, complex_mass=1)
    proc = opr.Process('ub_hdt', ['u', 'b'], ['h', 'd', 't'], ['udw', 'tbw', 'wwh'])
    n, rs = 16, 1000.0
    u = philox.uniforms(5, 0, n, 12, 3)
    masses = np.stack([np.full(n, PAR['mh']), np.zeros(n), np.zeros(n)], 1)
    k, _ = ops.rambo_massive(u, masses, rs)
    p = np.zeros((n, 5, 4))
    p[:, 0] = [rs / 2, 0, 0, rs / 2]
    p[:, 1] = [rs / 2, 0, 0, -rs / 2]
    p[:, 2:] = k
    gw, mw = sm.couplings(par)['gw'], par['mw']
    gam = par['mw'] * par['gz'] / par['mz']
    q1 = p[:, 0] - p[:, 3]
    q2 = p[:, 1] - p[:, 4]
    d1 = (inputs.mdot(q1, q1) - mw * mw) ** 2 + (mw * gam) ** 2
    d2 = (inputs.mdot(q2, q2) - mw * mw) ** 2 + (mw * gam) ** 2
    mu2 = mw * mw * math.sqrt(1 + (gam / mw) ** 2)
    want = (gw ** 2 / 2) ** 2 * gw ** 2 * mu2 * 16 * inputs.mdot(p[:, 0], p[:, 1]) * inputs.mdot(p[:, 3], p[:, 4]) \
        / (d1 * d2) * 9 / 36
    assert np.allclose(opr.me2(proc, p, par), want, rtol=1e-11)
