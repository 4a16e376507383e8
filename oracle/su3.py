"""Explicit SU(3): Gell-Mann generators T^a = lambda^a / 2 and structure constants f^{abc}.

Oracle / test infrastructure.  Colour indices as in PAPER.md:88 (1..3 quarks, 1..8 gluons);
T^a_{ij} of Eq. 36, f^{abc} of Eq. 42.
"""
import numpy as np

_l = np.zeros((8, 3, 3), dtype=complex)
_l[0] = [[0, 1, 0], [1, 0, 0], [0, 0, 0]]
_l[1] = [[0, -1j, 0], [1j, 0, 0], [0, 0, 0]]
_l[2] = [[1, 0, 0], [0, -1, 0], [0, 0, 0]]
_l[3] = [[0, 0, 1], [0, 0, 0], [1, 0, 0]]
_l[4] = [[0, 0, -1j], [0, 0, 0], [1j, 0, 0]]
_l[5] = [[0, 0, 0], [0, 0, 1], [0, 1, 0]]
_l[6] = [[0, 0, 0], [0, 0, -1j], [0, 1j, 0]]
_l[7] = np.diag([1, 1, -2]) / np.sqrt(3.0)

T = _l / 2.0  # T[a, i, j]

# f^{abc} = -2i Tr([T^a, T^b] T^c)   (from [T^a,T^b] = i f^{abc} T^c, Tr T^a T^b = delta/2)
F = np.zeros((8, 8, 8))
for _a in range(8):
    for _b in range(8):
        _comm = T[_a] @ T[_b] - T[_b] @ T[_a]
        for _c in range(8):
            F[_a, _b, _c] = (-2j * np.trace(_comm @ T[_c])).real
