"""Seeded synthetic inputs shared by oracle pins and CUDA parity tests.  No method arithmetic here:
only plain kinematic constructions of momenta (numpy), so that neither side's code is involved."""
import numpy as np


def two_to_two(rs, m3, m4, n, seed=1, cmax=0.95):
    """[n,4,4] momenta for a+b -> 3+4 in the CM frame, incoming along +-z, random angles."""
    rng = np.random.default_rng(seed)
    ct = rng.uniform(-cmax, cmax, n)
    ph = rng.uniform(0, 2 * np.pi, n)
    return two_to_two_at(rs, m3, m4, ct, ph)


def two_to_two_at(rs, m3, m4, ct, ph):
    ct = np.asarray(ct, dtype=float)
    ph = np.broadcast_to(np.asarray(ph, dtype=float), ct.shape)
    n = len(ct)
    p = np.zeros((n, 4, 4))
    E = rs / 2
    p[:, 0] = [E, 0, 0, E]
    p[:, 1] = [E, 0, 0, -E]
    e3 = (rs * rs + m3 * m3 - m4 * m4) / (2 * rs)
    k = np.sqrt(e3 * e3 - m3 * m3)
    st = np.sqrt(1 - ct * ct)
    p[:, 2, 0] = e3
    p[:, 2, 1] = k * st * np.cos(ph)
    p[:, 2, 2] = k * st * np.sin(ph)
    p[:, 2, 3] = k * ct
    p[:, 3, 0] = rs - e3
    p[:, 3, 1:] = -p[:, 2, 1:]
    return p


def mdot(a, b):
    return a[..., 0] * b[..., 0] - (a[..., 1:] * b[..., 1:]).sum(-1)


def mandelstam(p):
    s = mdot(p[:, 0] + p[:, 1], p[:, 0] + p[:, 1])
    t = mdot(p[:, 0] - p[:, 2], p[:, 0] - p[:, 2])
    u = mdot(p[:, 0] - p[:, 3], p[:, 0] - p[:, 3])
    return s, t, u


def lorentz(p, beta=(0.3, -0.2, 0.4), angles=(0.7, 1.1)):
    """Common boost (velocity beta) followed by a rotation, applied to every 4-vector in p[..., 4]."""
    bx = np.array(beta)
    g = 1 / np.sqrt(1 - bx @ bx)
    E = p[..., 0]
    v = p[..., 1:]
    bp = v @ bx
    E2 = g * (E + bp)
    v2 = v + ((g - 1) * bp / (bx @ bx) + g * E)[..., None] * bx
    a, b = angles
    R = np.array([[1, 0, 0], [0, np.cos(a), -np.sin(a)], [0, np.sin(a), np.cos(a)]]) @ \
        np.array([[np.cos(b), -np.sin(b), 0], [np.sin(b), np.cos(b), 0], [0, 0, 1]])
    return np.concatenate([E2[..., None], v2 @ R.T], -1)


def boost_from_rest(pr, P):
    """pr[..., 4] given in the rest frame of a particle with momentum P[4] (mass from P) -> the frame of P (pure boost)."""
    P = np.asarray(P, dtype=float)
    M = np.sqrt(mdot(P, P))
    e = (P[0] * pr[..., 0] + pr[..., 1:] @ P[1:]) / M
    fac = (e + pr[..., 0]) / (P[0] + M)
    return np.concatenate([e[..., None], pr[..., 1:] + fac[..., None] * P[1:]], -1)


def decay(P, m1, m2, nhat):
    """Two-body decay of momentum P into masses (m1, m2); particle 1 leaves along the unit vector nhat in the rest
    frame of P.  Returns (p1, p2) in the frame of P."""
    P = np.asarray(P, dtype=float)
    M = np.sqrt(mdot(P, P))
    k = np.sqrt(max((M * M - m1 * m1 - m2 * m2) ** 2 - 4 * m1 * m1 * m2 * m2, 0.0)) / (2 * M)
    nhat = np.asarray(nhat, dtype=float)
    p1 = np.concatenate([[np.sqrt(k * k + m1 * m1)], k * nhat])
    p2 = np.concatenate([[np.sqrt(k * k + m2 * m2)], -k * nhat])
    return boost_from_rest(p1, P), boost_from_rest(p2, P)


def tetrahedron(rot=0.0):
    """Four unit vectors forming a spherical 2-design (sums of polynomials of degree <= 2 over them equal the sphere
    average), rotated about the z axis by `rot` and tilted so that no vector is along an axis."""
    v = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=float) / np.sqrt(3.0)
    c, s = np.cos(rot), np.sin(rot)
    Rz = np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]])
    a = 0.4
    Rx = np.array([[1, 0, 0], [0, np.cos(a), -np.sin(a)], [0, np.sin(a), np.cos(a)]])
    return v @ (Rz @ Rx).T
