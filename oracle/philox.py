"""Philox4x32-10 counter-based generator and the uniform layout of SURVEY.md 8c-A15 (oracle side).

The paper's per-thread xorshift is replaced by Philox as BASELINE.json
mandates.  This is the oracle's own implementation (numpy uint64 arithmetic); the CUDA path
implements the same published algorithm independently.

Layout: key = (seed_lo, seed_hi); counter = (event_lo, event_hi, block j, process id);
draw d uses words (2d mod 4, 2d+1 mod 4) of block floor(d/2):
    u = ((hi >> 6) * 2^26 + (lo >> 6) + 1/2) * 2^-52    in the open interval (0,1),
with lo = word 2d mod 4, hi = word (2d+1) mod 4.  (A15 proposes a 53-bit mantissa; with 53 bits the
"+1/2" is not exactly representable for the largest mantissas and u could round to 1.0, so 52 bits are
used: every step is exact in fp64 and u is strictly inside (0,1) -- RAMBO takes log u.)
"""
import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = np.uint64(0x9E3779B9)
_W1 = np.uint64(0xBB67AE85)
_MASK = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)


def philox4x32_10(ctr, key):
    """ctr: 4 uint64 arrays holding 32-bit words, key: 2 (arrays or scalars).  Returns 4 arrays of 32-bit words."""
    c0, c1, c2, c3 = [np.asarray(c, dtype=np.uint64) & _MASK for c in ctr]
    k0 = np.asarray(key[0], dtype=np.uint64) & _MASK
    k1 = np.asarray(key[1], dtype=np.uint64) & _MASK
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        hi0, lo0 = p0 >> _S32, p0 & _MASK
        hi1, lo1 = p1 >> _S32, p1 & _MASK
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0) & _MASK, lo1, (hi0 ^ c3 ^ k1) & _MASK, lo0
        k0 = (k0 + _W0) & _MASK
        k1 = (k1 + _W1) & _MASK
    return c0, c1, c2, c3


def uniforms(seed, first_event, n, ndraw, process_id):
    """[n, ndraw] doubles in (0,1) for events first_event .. first_event+n-1."""
    ev = np.uint64(first_event) + np.arange(n, dtype=np.uint64)
    key = (np.uint64(seed & 0xFFFFFFFF), np.uint64((seed >> 32) & 0xFFFFFFFF))
    out = np.empty((n, ndraw))
    nblk = (ndraw + 1) // 2
    for j in range(nblk):
        w = philox4x32_10((ev & _MASK, ev >> _S32, np.full(n, j, dtype=np.uint64),
                           np.full(n, process_id, dtype=np.uint64)), key)
        for h in range(2):
            d = 2 * j + h
            if d >= ndraw:
                break
            lo, hi = w[2 * h], w[2 * h + 1]
            mant = (hi >> np.uint64(6)) * np.uint64(1 << 26) + (lo >> np.uint64(6))
            out[:, d] = (mant.astype(np.float64) + 0.5) * 2.0 ** -52
    return out
