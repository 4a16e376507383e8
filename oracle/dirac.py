"""Explicit Dirac algebra, external spinors and polarisation vectors (oracle; test infrastructure).

Follows the definitions of PAPER.md:412-447 (Eq. 29-33): u(p,lambda), v(p,lambda) are
helicity eigenstates for arbitrary mass, eps^mu(p,lambda) the helicity-basis polarisation
vectors (conjugated for final-state bosons).  The *Dirac* representation of the gamma
matrices is used here on purpose (the device library uses the chiral one);
helicity-summed |M|^2 does not depend on the choice.

All functions are vectorised over a leading event axis: p has shape [N,4] = (E,px,py,pz),
metric (+,-,-,-).  The arithmetic runs in the dtype of p: float64 normally, numpy.longdouble (x87 80-bit,
eps = 1.1e-19) when the caller passes extended-precision momenta (oracle.processes.me2_extended).
"""
import numpy as np

I2 = np.eye(2, dtype=complex)
SIG = np.array([[[0, 1], [1, 0]], [[0, -1j], [1j, 0]], [[1, 0], [0, -1]]], dtype=complex)
Z2 = np.zeros((2, 2), dtype=complex)

G0 = np.block([[I2, Z2], [Z2, -I2]])
GAM = np.array([G0] + [np.block([[Z2, SIG[k]], [-SIG[k], Z2]]) for k in range(3)])  # gamma^mu
G5 = np.block([[Z2, I2], [I2, Z2]])
ONE4 = np.eye(4, dtype=complex)
PL = 0.5 * (ONE4 - G5)
PR = 0.5 * (ONE4 + G5)
METRIC = np.array([1.0, -1.0, -1.0, -1.0])


def mdot(a, b):
    """Minkowski product a.b of [N,4] arrays (no complex conjugation)."""
    return a[..., 0] * b[..., 0] - a[..., 1] * b[..., 1] - a[..., 2] * b[..., 2] - a[..., 3] * b[..., 3]


def slash(v):
    """v_mu gamma^mu for v = v^mu of shape [N,4] -> [N,4,4]."""
    vl = v * METRIC  # lower the index
    return np.einsum('nm,mab->nab', vl + 0j, GAM)


def _chi(p, lam):
    """Two-component helicity eigenstate chi_lam(p^), (sigma.p^) chi = lam chi, lam = +-1."""
    px, py, pz = p[:, 1], p[:, 2], p[:, 3]
    pabs = np.sqrt(px * px + py * py + pz * pz)
    pt = np.sqrt(px * px + py * py)
    safe = pabs > 0
    pa = np.where(safe, pabs, 1.0)
    pzs = np.where(safe, pz, 1.0)
    big = pa + np.abs(pzs)  # |p| + |pz|: no cancellation
    cs_big = np.sqrt(big / (2 * pa))  # the larger of cos(theta/2), sin(theta/2)
    cs_small = pt / np.sqrt(2 * pa * big)  # the smaller one, = sqrt((|p| - |pz|) / 2|p|) without cancellation
    c2 = np.where(pzs >= 0, cs_big, cs_small)  # cos(theta/2)
    s2 = np.where(pzs >= 0, cs_small, cs_big)  # sin(theta/2)
    ptsafe = pt > 0
    eiphi = np.where(ptsafe, (px + 1j * py) / np.where(ptsafe, pt, 1.0), 1.0 + 0j)
    if lam == +1:
        return np.stack([c2 + 0j, eiphi * s2], axis=1)
    return np.stack([-np.conj(eiphi) * s2, c2 + 0j], axis=1)


def u_spinor(p, m, lam):
    """u(p, lam/2): column spinor [N,4], (pslash - m) u = 0, ubar u = 2m  (Eq. 29a)."""
    E = p[:, 0]
    pabs = np.sqrt(p[:, 1] ** 2 + p[:, 2] ** 2 + p[:, 3] ** 2)
    chi = _chi(p, lam)
    up = np.sqrt(np.clip(E + m, 0, None))[:, None] * chi
    dn = (lam * np.sqrt(np.clip(E - m, 0, None)))[:, None] * chi  # |p|/sqrt(E+m) = sqrt(E-m)
    del pabs
    return np.concatenate([up, dn], axis=1)


def v_spinor(p, m, lam):
    """v(p, lam/2): column spinor [N,4], (pslash + m) v = 0, vbar v = -2m  (Eq. 29b).

    The antiparticle of helicity lam/2 is built on chi_{-lam}.
    """
    E = p[:, 0]
    chi = _chi(p, -lam)
    up = (-lam * np.sqrt(np.clip(E - m, 0, None)))[:, None] * chi
    dn = np.sqrt(np.clip(E + m, 0, None))[:, None] * chi
    return np.concatenate([up, dn], axis=1)


def bar(psi):
    """psibar = psi^dagger gamma^0, row spinor [N,4]."""
    return np.conj(psi) @ G0


def polvec(p, m, lam):
    """eps^mu(p, lam) with upper index, [N,4]; lam = +1, -1, or 0 (massive only)  (Eq. 32b)."""
    E, px, py, pz = p[:, 0], p[:, 1], p[:, 2], p[:, 3]
    pabs = np.sqrt(px * px + py * py + pz * pz)
    pt = np.sqrt(px * px + py * py)
    safe = pabs > 0
    pa = np.where(safe, pabs, 1.0)
    ct = np.where(safe, pz / pa, 1.0)
    st = np.where(safe, pt / pa, 0.0)
    ptsafe = pt > 0
    cphi = np.where(ptsafe, px / np.where(ptsafe, pt, 1.0), 1.0)
    sphi = np.where(ptsafe, py / np.where(ptsafe, pt, 1.0), 0.0)
    zero = np.zeros_like(E)
    if lam == 0:
        return np.stack([pabs / m, E / m * st * cphi, E / m * st * sphi, E / m * ct], axis=1) + 0j
    e1 = np.stack([zero, ct * cphi, ct * sphi, -st], axis=1)  # theta^ direction
    e2 = np.stack([zero, -sphi, cphi, zero], axis=1)  # phi^ direction
    return (-lam * e1 - 1j * e2) / np.sqrt(E.dtype.type(2))
