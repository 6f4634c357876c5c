"""Philox4x32-10 and Gumbel noise (oracle; test infrastructure only).

north_star (BASELINE.json): "Gumbel-max sampling from counter-based Philox keyed
on (seed, prompt, sample, step)".  The paper itself only says "sampling"
(§4.1.1: "M'_i independent trajectories"); R4 fixes the
counter/key assignment:

    counter = (v >> 2, step s, sample j, prompt i)      key = (seed_lo32, seed_hi32)
    x       = output word (v & 3) of Philox4x32-10(counter, key)
    u       = ((x >> 9) + 0.5) * 2^-23                   in (0, 1), exact in float32
    g       = -ln(-ln u)                                  standard Gumbel

Philox4x32-10 is the published algorithm of Salmon, Moraes, Dror, Shaw,
"Parallel random numbers: as easy as 1, 2, 3" (SC'11): ten rounds of
    (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0))
with M0 = 0xD2511F53, M1 = 0xCD9E8D57, and the key bumped between rounds by the
Weyl constants (0x9E3779B9, 0xBB67AE85).
Pin: tests/golden/philox4x32_10_kat.txt (Random123 known-answer vectors).
"""
import numpy as np

M0 = np.uint64(0xD2511F53)
M1 = np.uint64(0xCD9E8D57)
W0 = np.uint64(0x9E3779B9)
W1 = np.uint64(0xBB67AE85)
MASK = np.uint64(0xFFFFFFFF)
S32 = np.uint64(32)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Vectorised over numpy arrays of equal (broadcastable) shape; returns 4 uint32 arrays."""
    c0, c1, c2, c3, k0, k1 = [np.asarray(a, dtype=np.uint64) & MASK for a in (c0, c1, c2, c3, k0, k1)]
    c0, c1, c2, c3, k0, k1 = np.broadcast_arrays(c0, c1, c2, c3, k0, k1)
    for r in range(10):
        p0 = M0 * c0            # 64-bit product of two 32-bit values
        p1 = M1 * c2
        hi0, lo0 = p0 >> S32, p0 & MASK
        hi1, lo1 = p1 >> S32, p1 & MASK
        c0, c1, c2, c3 = (hi1 ^ c1 ^ k0), lo1, (hi0 ^ c3 ^ k1), lo0
        k0 = (k0 + W0) & MASK
        k1 = (k1 + W1) & MASK
    return tuple(a.astype(np.uint32) for a in (c0, c1, c2, c3))


def uniform_from_bits(x):
    """u = ((x >> 9) + 0.5) * 2^-23: 24 significant bits, so exactly representable in float32
    (the GPU forms the same u in fp32) and never 0 or 1."""
    return ((np.asarray(x, dtype=np.uint32) >> np.uint32(9)).astype(np.float64) + 0.5) * 2.0 ** -23


def gumbel_noise(V, seed, i, j, s):
    """g[0..V) for prompt i, sample j, step s (float64)."""
    v = np.arange(V, dtype=np.uint64)
    seed = int(seed) & 0xFFFFFFFFFFFFFFFF
    words = philox4x32_10(v >> np.uint64(2), s, j, i, seed & 0xFFFFFFFF, seed >> 32)
    lane = (v & np.uint64(3)).astype(np.int64)
    x = np.choose(lane, words)
    u = uniform_from_bits(x)
    return -np.log(-np.log(u))
