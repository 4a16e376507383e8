"""Standard Model particle and vertex tables for the process generator (step a0).

The vertex set is the one of PAPER.md:456-649 (section 4.2): FFV (Eq. 35; qqg Eq. 36), VVV (Eq. 40; ggg Eq. 42),
VVVV (gggg Eq. 47-48), FFS (Eq. 39), VVS (Eq. 50), VVSS (Eq. 51), SSS (Eq. 52).  Light fermions are massless,
the CKM matrix is diagonal (BASELINE.json).  Couplings are *names* of members of the device struct
`hg::Coup<T>` (csrc/hg_params.cuh); their values are derived in csrc/hg_api.cu:hg_set_params.

All vertices are written with ALL-INCOMING fields.  For a fermion bilinear  psibar_F1 Gamma psi_F2  the incoming
fields are (anti(F1), F2): the row spinor belongs to anti(F1), the column spinor to F2.
"""
from dataclasses import dataclass


@dataclass(frozen=True)
class Particle:
    name: str
    spin: str      # 'F', 'V', 'S'
    colour: int    # 1, 3 (fundamental; the antiparticle is listed with -3), 8
    mass: str      # name of the mass member of Coup ('' = massless)
    width: str     # name of the width member ('' = none)
    anti: str
    is_anti: bool  # True for the antifermion (row spinor when incoming)


PARTICLES = {}


def _add(name, spin, colour, mass, width, anti):
    PARTICLES[name] = Particle(name, spin, colour, mass, width, anti, False)
    if anti != name:
        PARTICLES[anti] = Particle(anti, spin, -colour if colour == 3 else colour, mass, width, name, spin == 'F')


_add('u', 'F', 3, '', '', 'u~')
_add('d', 'F', 3, '', '', 'd~')
_add('t', 'F', 3, 'mt', 'wt', 't~')
_add('b', 'F', 3, '', '', 'b~')        # mb = 0 in every config (BASELINE.json configs[3])
_add('e-', 'F', 1, '', '', 'e+')
_add('mu-', 'F', 1, '', '', 'mu+')
_add('ve', 'F', 1, '', '', 've~')
_add('vm', 'F', 1, '', '', 'vm~')
_add('g', 'V', 8, '', '', 'g')
_add('a', 'V', 1, '', '', 'a')
_add('z', 'V', 1, 'mz', 'wz', 'z')
_add('w+', 'V', 1, 'mw', 'ww', 'w-')
_add('h', 'S', 1, 'mh', 'wh', 'h')


def anti(name):
    return PARTICLES[name].anti


@dataclass(frozen=True)
class Vertex:
    kind: str        # 'FFV', 'VVV', 'VVVV', 'FFS', 'VVS', 'VVSS', 'SSS'
    fields: tuple    # all-incoming particle names; FFV/FFS: (row = antifermion, column = fermion, boson)
    coup: tuple      # names of Coup members: FFV (gL, gR) ('' = zero); others (g,)
    colour: str      # '1' colourless/delta, 'T' = T^a_{ji}, 'f' = i f^{abc}, 'ff' = four-gluon


VERTICES = []


def _ffv(f_out, f_in, boson, gl, gr, colour='1'):
    """L = psibar_{f_out} gamma^mu (gl PL + gr PR) psi_{f_in} V_mu(boson annihilated)."""
    VERTICES.append(Vertex('FFV', (anti(f_out), f_in, boson), (gl, gr), colour))


# strong interaction: gL = gR = -g_s with colour factor T^a (Eq. 36-38)
for _q in ('u', 'd', 't', 'b'):
    _ffv(_q, _q, 'g', 'mgs', 'mgs', 'T')
# photon and Z (Eq. 35; couplings SURVEY.md 8c-A5)
for _f, _tag in (('u', 'u'), ('d', 'd'), ('t', 'u'), ('b', 'd'), ('e-', 'l'), ('mu-', 'l')):
    _ffv(_f, _f, 'a', 'ga' + _tag, 'ga' + _tag)
    _ffv(_f, _f, 'z', 'gz' + _tag + 'L', 'gz' + _tag + 'R')
for _f in ('ve', 'vm'):
    _ffv(_f, _f, 'z', 'gznL', '')
# W: psibar_up gamma^mu PL psi_dn W+_mu + h.c.
for _up, _dn in (('u', 'd'), ('t', 'b'), ('ve', 'e-'), ('vm', 'mu-')):
    _ffv(_up, _dn, 'w+', 'gwf', '')
    _ffv(_dn, _up, 'w-', 'gwf', '')
# gauge self-interactions
VERTICES.append(Vertex('VVV', ('g', 'g', 'g'), ('gs',), 'f'))
VERTICES.append(Vertex('VVVV', ('g', 'g', 'g', 'g'), ('gs2',), 'ff'))
VERTICES.append(Vertex('VVV', ('w-', 'w+', 'a'), ('gwwa',), '1'))   # Table 16 ordering
VERTICES.append(Vertex('VVV', ('w-', 'w+', 'z'), ('gwwz',), '1'))
# Higgs sector of the library (Eq. 39, 50-52): exercised only by NEXT-1 processes
VERTICES.append(Vertex('FFS', ('t~', 't', 'h'), ('gtth', 'gtth'), '1'))
VERTICES.append(Vertex('VVS', ('w-', 'w+', 'h'), ('gwwh',), '1'))
VERTICES.append(Vertex('VVS', ('z', 'z', 'h'), ('gzzh',), '1'))
VERTICES.append(Vertex('VVSS', ('w-', 'w+', 'h', 'h'), ('gwwhh',), '1'))
VERTICES.append(Vertex('VVSS', ('z', 'z', 'h', 'h'), ('gzzhh',), '1'))
VERTICES.append(Vertex('SSS', ('h', 'h', 'h'), ('ghhh',), '1'))
