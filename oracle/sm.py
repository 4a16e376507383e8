"""Standard Model inputs and derived couplings for the oracle (test infrastructure).

Inputs: BASELINE.json configs[0] (MZ, MW, GZ, GW, 1/alpha), configs[3] (mt, Gt, mb=0),
configs[1] (alpha_s=0.118).  Derivation of the couplings: SURVEY.md 8c-A5 (tree-level
relations; the paper's own inputs are at PAPER.md:1075).  FFV couplings are the gc[0]
(left) and gc[1] (right) of the Lagrangian Eq. 35.
"""
import math

HBARC2_PB = 0.3893793721e9  # (hbar c)^2 in pb GeV^2


def default_params():
    return dict(mz=91.1876, mw=80.419, gz=2.441, gw=2.048, mt=174.3, gt=1.5, mb=0.0,
                mh=125.0, gh=0.00407, alpha_em_inv=132.507, alpha_s=0.118, complex_mass=0)


def complex_masses(par):
    """The paper's complex-mass option (Eq. 54-56; reading A4b in DESIGN.md): every m_V^2
    (V = W, Z) in propagators AND couplings is replaced by mu_V^2 = m_V^2 - i m_V Gamma_V, with
    mu_W^2 = (g_W^2 / g_Z^2) mu_Z^2 imposed (Eq. 56).  g_W^2 / g_Z^2 = cos^2 theta_W = m_W^2 / m_Z^2 is real here
    (sw2 is derived from the real masses), so Eq. 56 fixes the W width: Gamma_W = m_W Gamma_Z / m_Z replaces the
    input.  Returns (mu_W^2, mu_Z^2) as complex numbers; with complex_mass = 0 the real masses squared."""
    if not par.get('complex_mass'):
        return complex(par['mw'] ** 2), complex(par['mz'] ** 2)
    muz2 = complex(par['mz'] ** 2, -par['mz'] * par['gz'])
    muw2 = (par['mw'] ** 2 / par['mz'] ** 2) * muz2
    return muw2, muz2


def effective_widths(par):
    """Widths in the propagator denominators: the inputs, or Eq. 56's W width in the complex-mass option."""
    if not par.get('complex_mass'):
        return par['gw'], par['gz']
    return par['mw'] * par['gz'] / par['mz'], par['gz']


# electric charge and weak isospin of the left-handed component
_Q = {'u': 2.0 / 3, 'd': -1.0 / 3, 't': 2.0 / 3, 'b': -1.0 / 3, 'e-': -1.0, 'mu-': -1.0,
      've': 0.0, 'vm': 0.0}
_T3 = {'u': 0.5, 'd': -0.5, 't': 0.5, 'b': -0.5, 'e-': -0.5, 'mu-': -0.5, 've': 0.5, 'vm': 0.5}


def couplings(par):
    """Return a dict of real couplings derived from the inputs (tree-level relations)."""
    ratio = par['mw'] ** 2 / par['mz'] ** 2
    if isinstance(ratio, complex):      # complex masses of equal phase (analytic-continuation pin): the ratio is real
        assert abs(ratio.imag) < 1e-14 * abs(ratio.real)
        ratio = ratio.real
    sw2 = 1.0 - ratio
    sw = math.sqrt(sw2)
    cw = math.sqrt(1.0 - sw2)
    e = math.sqrt(4.0 * math.pi / par['alpha_em_inv'])
    gw = e / sw
    gzz = e / (sw * cw)
    gs = math.sqrt(4.0 * math.pi * par['alpha_s'])
    c = dict(sw2=sw2, e=e, gw=gw, gz=gzz, gs=gs)
    # L = psibar gamma^mu (gL PL + gR PR) psi V_mu  with D = d + i e Q A + i gz (T3 - Q sw2) Z
    for f in _Q:
        c[('a', f)] = (-e * _Q[f], -e * _Q[f])
        c[('z', f)] = (-gzz * (_T3[f] - _Q[f] * sw2), gzz * _Q[f] * sw2)
    c['w'] = (-gw / math.sqrt(2.0), 0.0)
    return c
