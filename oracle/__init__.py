"""Oracle for arXiv:1305.0708 hot path -- TEST INFRASTRUCTURE ONLY.

A plain, slow, fp64 CPU (numpy) statement of what the hot path computes:
tree-level Standard Model |M|^2 summed over helicities and colours (PAPER.md:75-88,
Eq. 4-6), phase-space points and weights, cuts, and the Monte-Carlo accumulation.

Rules this package obeys:
  * It shares no code with the CUDA path (`paper_1305_0708_b200/`): neither imports the
    other.  Only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline` /
    `--impl reference` legs of `bench.py` may import it.
  * Different formulation from the CUDA path on purpose: Dirac representation of the
    gamma matrices (the device library is chiral), explicit 4x4 matrix algebra, textbook
    Feynman rules with every factor of i, one term per Feynman diagram (no shared
    sub-currents), all 2^n helicity combinations (no zero skipping), colour summed by brute
    force over explicit Gell-Mann matrices and f^{abc} (no colour-flow basis).
  * Everything is vectorised over the event axis only; there is no blocking, fusion or
    reordering beyond that.

Pins (tests/test_oracle_*.py, `-m "not gpu"`): Dirac equation / completeness of the
spinors and polarisation vectors, SU(3) identities, closed-form 2->2 |M|^2
(u d~ -> e+ ve, q q~ -> a a, u u~ -> e+ e-, q q~ -> t t~, g g -> t t~, q q~ -> g g,
g g -> g g), Ward identities, Lorentz invariance, Bose symmetry, soft-gluon limit,
diagram counts, Philox known-answer vectors, RAMBO volumes and energy moments,
Breit-Wigner integral, analytic sigma(u d~ -> e+ ve), the nested phase-space volume of config 4, the position
of the propagator pole (sign of the width term), the exact factorisation of config 4 on the resonance poles
into undecayed g g -> t t~ g times the textbook top-decay matrix elements.

Parity status: configs 1 and 2 are pinned to closed forms.  Configs 3, 4, 5 have no printed
number in the paper: they are pinned by Ward identity + Lorentz/Bose invariance + the
2->2 closed forms that exercise every Feynman rule they use + soft limits; their
absolute normalisation against an external number is "parity unpinned".
"""
