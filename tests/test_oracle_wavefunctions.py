"""Pins for the oracle's spinors, polarisation vectors (Eq. 29-33; A2, A3) and SU(3)."""
import numpy as np
import pytest

from oracle import dirac as D
from oracle import su3


def _momenta(m, n=40, seed=3):
    rng = np.random.default_rng(seed)
    v = rng.normal(size=(n, 3)) * 50.0
    v[0] = [0, 0, 30.0]  # along +z
    v[1] = [0, 0, -30.0]  # along -z (special branch)
    v[2] = [1e-9, 0, -30.0]
    if m > 0:
        v[3] = [0, 0, 0]  # at rest
    E = np.sqrt(m * m + (v ** 2).sum(1))
    return np.concatenate([E[:, None], v], 1)


@pytest.mark.parametrize("m", [0.0, 4.7, 174.3])
def test_dirac_equation_and_normalisation(m):
    p = _momenta(m)
    ps = D.slash(p)
    scale = p[:, 0:1] ** 1.5
    for lam in (-1, 1):
        u, v = D.u_spinor(p, m, lam), D.v_spinor(p, m, lam)
        assert np.abs(np.einsum('nab,nb->na', ps, u) - m * u).max() < 1e-12 * scale.max()
        assert np.abs(np.einsum('nab,nb->na', ps, v) + m * v).max() < 1e-12 * scale.max()
        assert np.allclose(np.einsum('na,na->n', D.bar(u), u), 2 * m, atol=1e-9)
        assert np.allclose(np.einsum('na,na->n', D.bar(v), v), -2 * m, atol=1e-9)


@pytest.mark.parametrize("m", [0.0, 4.7, 174.3])
def test_spinor_completeness(m):
    p = _momenta(m)
    ps = D.slash(p)
    su = sum(np.einsum('na,nb->nab', D.u_spinor(p, m, l), D.bar(D.u_spinor(p, m, l))) for l in (-1, 1))
    sv = sum(np.einsum('na,nb->nab', D.v_spinor(p, m, l), D.bar(D.v_spinor(p, m, l))) for l in (-1, 1))
    tol = 1e-12 * p[:, 0].max()
    assert np.abs(su - (ps + m * D.ONE4)).max() < tol
    assert np.abs(sv - (ps - m * D.ONE4)).max() < tol


def test_helicity_eigenstates():
    m = 4.7
    p = _momenta(m)[4:]
    pabs = np.sqrt((p[:, 1:] ** 2).sum(1))
    # spin operator along p:  Sigma.p^ = diag(sigma.p^, sigma.p^) in the Dirac representation
    sp = np.einsum('nk,kab->nab', p[:, 1:] / pabs[:, None], D.SIG)
    S = np.zeros((len(p), 4, 4), dtype=complex)
    S[:, :2, :2] = sp
    S[:, 2:, 2:] = sp
    for lam in (-1, 1):
        u = D.u_spinor(p, m, lam)
        assert np.allclose(np.einsum('nab,nb->na', S, u), lam * u, atol=1e-10)
        v = D.v_spinor(p, m, lam)  # antiparticle of helicity lam has spin projection -lam in v
        assert np.allclose(np.einsum('nab,nb->na', S, v), -lam * v, atol=1e-10)


def test_massless_limit_is_chiral():
    p = _momenta(0.0)
    for lam in (-1, 1):
        u = D.u_spinor(p, 0.0, lam)
        proj = D.PR if lam == 1 else D.PL
        assert np.allclose(u @ proj.T, u, atol=1e-12)


@pytest.mark.parametrize("m", [0.0, 80.419])
def test_polarisation_vectors(m):
    p = _momenta(m)
    if m > 0:
        p = p[[0, 1, 2] + list(range(4, len(p)))]
    lams = (-1, 1) if m == 0 else (-1, 0, 1)
    eps = {l: D.polvec(p, m, l) for l in lams}
    for l in lams:
        assert np.abs(D.mdot(eps[l], p.astype(complex))).max() < 1e-12 * p[:, 0].max()
        for l2 in lams:
            d = D.mdot(eps[l], np.conj(eps[l2]))
            assert np.allclose(d, -1.0 if l == l2 else 0.0, atol=1e-12)
    if m > 0:
        g = np.diag(D.METRIC)
        tot = sum(np.einsum('nm,nv->nmv', eps[l], np.conj(eps[l])) for l in lams)
        want = -g[None] + np.einsum('nm,nv->nmv', p, p) / m ** 2
        assert np.abs(tot - want).max() < 1e-10 * (p[:, 0].max() / m) ** 2
    else:
        # e(-) = -conj(e(+)) in this basis, and both are purely spatial
        assert np.allclose(eps[-1], -np.conj(eps[1]))
        assert np.allclose(eps[1][:, 0], 0)


def test_gamma_algebra():
    g = np.diag(D.METRIC)
    for m in range(4):
        for n in range(4):
            ac = D.GAM[m] @ D.GAM[n] + D.GAM[n] @ D.GAM[m]
            assert np.allclose(ac, 2 * g[m, n] * D.ONE4)
        assert np.allclose(D.G5 @ D.GAM[m] + D.GAM[m] @ D.G5, 0)
    assert np.allclose(D.G5, 1j * D.GAM[0] @ D.GAM[1] @ D.GAM[2] @ D.GAM[3])


def test_su3_identities():
    T, F = su3.T, su3.F
    for a in range(8):
        assert np.allclose(T[a], np.conj(T[a].T))
        for b in range(8):
            assert np.isclose(np.trace(T[a] @ T[b]), 0.5 * (a == b))
            assert np.allclose(T[a] @ T[b] - T[b] @ T[a], 1j * np.einsum('c,cij->ij', F[a, b], T))
    assert np.allclose(np.einsum('aij,ajk->ik', T, T), 4.0 / 3.0 * np.eye(3))  # C_F
    assert np.allclose(np.einsum('acd,bcd->ab', F, F), 3.0 * np.eye(8))  # C_A
    assert np.allclose(F, -np.transpose(F, (1, 0, 2)))
    assert np.isclose(F[0, 1, 2], 1.0) and np.isclose(F[3, 4, 7], np.sqrt(3) / 2)
    # Jacobi
    jac = np.einsum('abe,ecd->abcd', F, F) + np.einsum('bce,ead->abcd', F, F) + np.einsum('cae,ebd->abcd', F, F)
    assert np.abs(jac).max() < 1e-14


def test_colour_matrices_closed_form():
    """SURVEY 8c 'Colour matrices': brute force over Gell-Mann matrices of the permutation strings."""
    import itertools
    T = su3.T
    # 2 gluons: C = (1/3)[[16,-2],[-2,16]]
    s = [np.einsum('aij,bjk->ikab', T, T), np.einsum('bij,ajk->ikab', T, T)]
    C = np.array([[np.sum(x * np.conj(y)).real for y in s] for x in s])
    assert np.allclose(C, np.array([[16, -2], [-2, 16]]) / 3.0)
    perms = list(itertools.permutations(range(3)))
    s = []
    for pm in perms:
        lab = 'abc'
        s.append(np.einsum('%sij,%sjk,%skl->ilabc' % (lab[pm[0]], lab[pm[1]], lab[pm[2]]), T, T, T))
    C = np.array([[np.sum(x * np.conj(y)).real for y in s] for x in s])
    want = np.array([[64, -8, -8, 1, 1, 10], [-8, 64, 1, 10, -8, 1], [-8, 1, 64, -8, 10, 1],
                     [1, 10, -8, 64, 1, -8], [1, -8, 10, 1, 64, -8], [10, 1, 1, -8, -8, 64]]) / 9.0
    assert np.allclose(C, want)
