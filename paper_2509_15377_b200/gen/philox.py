"""Counter-based random numbers for the *input generators* (numpy, vectorised).

Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11) with the counter/key layout of SURVEY.md §8(c)
"Uniforms": counter (c0,c1,c2,c3) = (n, block, id_lo, id_hi), key = (seed_lo, seed_hi); two doubles per
block, u = ((x >> 12) + 0.5) * 2^-52 with x the 64-bit word (w0 << 32 | w1) resp. (w2 << 32 | w3).

This module belongs to the seeded input generators only (primaries, gas-table seeds, map seeds).  The
oracle (oracle/avmo.cpp) and the CUDA path (csrc/) each carry their own implementation of the same
generator and import nothing from here.
"""
from __future__ import annotations

import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = np.uint32(0x9E3779B9)
_W1 = np.uint32(0xBB67AE85)
_MASK32 = np.uint64(0xFFFFFFFF)
_S32 = np.uint64(32)

BLOCK_CHILD_ID = 0xFFFFFFFF      # block used for secondary-electron ids
N_PRIMARY = 0xFFFFFFFE           # reserved collision index used to draw primaries


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Ten rounds; all arguments broadcastable uint32 arrays. Returns four uint32 arrays."""
    c0, c1, c2, c3, k0, k1 = np.broadcast_arrays(*[np.asarray(a, dtype=np.uint32) for a in (c0, c1, c2, c3, k0, k1)])
    c0, c1, c2, c3, k0, k1 = (a.copy() for a in (c0, c1, c2, c3, k0, k1))
    with np.errstate(over="ignore"):
        for r in range(10):
            p0 = _M0 * c0.astype(np.uint64)
            p1 = _M1 * c2.astype(np.uint64)
            hi0 = (p0 >> _S32).astype(np.uint32)
            lo0 = (p0 & _MASK32).astype(np.uint32)
            hi1 = (p1 >> _S32).astype(np.uint32)
            lo1 = (p1 & _MASK32).astype(np.uint32)
            c0, c1, c2, c3 = hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0
            if r < 9:
                k0 = k0 + _W0
                k1 = k1 + _W1
    return c0, c1, c2, c3


def words(seed, ident, n, block, key_xor_hi=0):
    """Philox block for (seed, electron id, collision index n, block)."""
    seed = np.asarray(seed, dtype=np.uint64)
    ident = np.asarray(ident, dtype=np.uint64)
    k0 = (seed & _MASK32).astype(np.uint32)
    k1 = ((seed >> _S32) & _MASK32).astype(np.uint32) ^ np.uint32(key_xor_hi)
    i_lo = (ident & _MASK32).astype(np.uint32)
    i_hi = ((ident >> _S32) & _MASK32).astype(np.uint32)
    return philox4x32_10(np.asarray(n, dtype=np.uint32), np.asarray(block, dtype=np.uint32), i_lo, i_hi, k0, k1)


def _to_unit(hi, lo):
    x = (hi.astype(np.uint64) << _S32) | lo.astype(np.uint64)
    return ((x >> np.uint64(12)).astype(np.float64) + 0.5) * 2.0 ** -52


def uniform_pair(seed, ident, n, block, key_xor_hi=0):
    """Two doubles strictly inside (0, 1), exactly representable."""
    w0, w1, w2, w3 = words(seed, ident, n, block, key_xor_hi)
    return _to_unit(w0, w1), _to_unit(w2, w3)
