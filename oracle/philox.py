"""Oracle: seed -> Philox4x32-10 words -> Box-Muller normals (TEST INFRASTRUCTURE, fp64).

Follows PAPER.md:59 ("starts from random Gaussian noise"), :61 ("K distinct noise
seeds") and :251 ("we assign each sample a deterministic random seed").  The paper
does not name the generator; BASELINE.json's north_star (a) does: Philox4x32-10
with Box-Muller.  Layout readings S1-S3 of DESIGN.md:

  key     = (lo32(seed), hi32(seed))
  counter = (lo32(j), hi32(j), stream_id, 0) for 4-element block j = e // 4
  round r = 0..9:  (r > 0: k0 += 0x9E3779B9, k1 += 0xBB67AE85)
            p0 = 0xD2511F53 * c0, p1 = 0xCD9E8D57 * c2   (64-bit products)
            (c0,c1,c2,c3) <- (hi(p1)^c1^k0, lo(p1), hi(p0)^c3^k1, lo(p0))
  u1 = ((wa >> 8) + 1) * 2**-24 in (0,1],  u2 = (wb >> 8) * 2**-24 in [0,1)
  za = sqrt(-2 ln u1) cos(2 pi u2),  zb = sqrt(-2 ln u1) sin(2 pi u2)
  lanes: (z0,z1) from (w0,w1), (z2,z3) from (w2,w3)

Pinned by tests/test_oracle_philox.py against the cuRAND *host* generator
(an independent implementation), a bijection check and moment/KS statistics.
"""
from __future__ import annotations

import numpy as np

M0 = np.uint64(0xD2511F53)
M1 = np.uint64(0xCD9E8D57)
W0 = 0x9E3779B9
W1 = 0xBB67AE85
MASK32 = np.uint64(0xFFFFFFFF)
S32 = np.uint64(32)


def philox4x32_10(c0, c1, c2, c3, k0: int, k1: int):
    """Ten Philox rounds on arrays of 32-bit counter words (held in uint64); returns 4 uint32 arrays."""
    c0 = np.asarray(c0, dtype=np.uint64) & MASK32
    c1 = np.asarray(c1, dtype=np.uint64) & MASK32
    c2 = np.asarray(c2, dtype=np.uint64) & MASK32
    c3 = np.asarray(c3, dtype=np.uint64) & MASK32
    k0 = int(k0) & 0xFFFFFFFF
    k1 = int(k1) & 0xFFFFFFFF
    for r in range(10):
        if r > 0:
            k0 = (k0 + W0) & 0xFFFFFFFF
            k1 = (k1 + W1) & 0xFFFFFFFF
        p0 = M0 * c0                     # < 2**64, exact in uint64
        p1 = M1 * c2
        n0 = (p1 >> S32) ^ c1 ^ np.uint64(k0)
        n1 = p1 & MASK32
        n2 = (p0 >> S32) ^ c3 ^ np.uint64(k1)
        n3 = p0 & MASK32
        c0, c1, c2, c3 = n0, n1, n2, n3
    return tuple(c.astype(np.uint32) for c in (c0, c1, c2, c3))


def words_for_seed(seed: int, n_elems: int, stream_id: int = 0, first_elem: int = 0) -> np.ndarray:
    """Raw 32-bit words for flat elements [first_elem, first_elem + n_elems) of one seed's tensor."""
    assert first_elem % 4 == 0 and n_elems % 4 == 0
    seed = int(seed) & 0xFFFFFFFFFFFFFFFF
    j = np.arange(first_elem // 4, (first_elem + n_elems) // 4, dtype=np.uint64)
    w = philox4x32_10(j & MASK32, j >> S32, np.full_like(j, stream_id), np.zeros_like(j),
                      seed & 0xFFFFFFFF, seed >> 32)
    return np.stack(w, axis=1).reshape(-1)          # word i of block j at flat index 4*j + i


def box_muller(words: np.ndarray) -> np.ndarray:
    """uint32 words (length multiple of 2) -> fp64 normals, pair (w[2i], w[2i+1]) -> (z[2i], z[2i+1])."""
    w = words.reshape(-1, 2).astype(np.uint64)
    u1 = ((w[:, 0] >> np.uint64(8)).astype(np.float64) + 1.0) * 2.0 ** -24
    u2 = (w[:, 1] >> np.uint64(8)).astype(np.float64) * 2.0 ** -24
    rho = np.sqrt(-2.0 * np.log(u1))
    phi = 2.0 * np.pi * u2
    return np.stack([rho * np.cos(phi), rho * np.sin(phi)], axis=1).reshape(-1)


def noise_from_seeds(seeds, elems_per_seed: int, stream_id: int = 0) -> np.ndarray:
    """[n_seeds, elems_per_seed] fp64 N(0,1); row b depends on (seeds[b], stream_id) only."""
    return np.stack([box_muller(words_for_seed(s, elems_per_seed, stream_id)) for s in seeds], axis=0)
