"""Pins for oracle/philox.py (CPU only).  O1-O2 of DESIGN.md "Oracle pins".

O1: Philox4x32-10 vs the cuRAND HOST generator (independent implementation, CPU-only): rounds,
    multipliers, Weyl key schedule, key = (lo,hi)(seed), roles of counter words c0, c1, c2.
    Bijection on 2^20 consecutive counters and single-bit avalanche (structure).
O2: Box-Muller: identity z_a^2 + z_b^2 = -2 ln u1, the range bound |z| <= sqrt(48 ln 2), moments and
    a Kolmogorov-Smirnov distance against the normal CDF on 2^22 samples.
"""
import os

import numpy as np
import pytest
from scipy import stats

from oracle import philox

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox_curand_host.txt")


def _oracle_block(seed, n, stream=None):
    """Oracle words for host-generator block n: c2 = n % 65536 plays the stream slot, (c1:c0) = n // 65536."""
    c2 = n % 65536
    j = n // 65536
    return philox.words_for_seed(seed, 4, stream_id=c2, first_elem=4 * j)


def test_philox_matches_curand_host_golden():
    rows = [l.split() for l in open(GOLDEN) if not l.startswith("#")]
    assert len(rows) == 42
    for r in rows:
        seed, off = int(r[0], 16), int(r[1], 16)
        want = np.array([int(x, 16) for x in r[2:]], dtype=np.uint32)
        got = np.concatenate([_oracle_block(seed, off // 4), _oracle_block(seed, off // 4 + 1)])
        assert (got == want).all(), (hex(seed), off)


def test_philox_matches_curand_host_live():
    mk = pytest.importorskip("tests.golden.make_philox_curand", reason="golden script not importable")
    try:
        lib = mk.load_curand()
    except OSError:
        pytest.skip("libcurand not present")
    seed = 0x9E3779B97F4A7C15
    n_blocks = 3 * 65536                      # covers c0 in {0,1,2} and every c2 in [0, 65536)
    w = mk.curand_words(lib, seed, 0, 4 * n_blocks).reshape(n_blocks, 4)
    c2 = np.arange(n_blocks, dtype=np.uint64) % 65536
    c0 = np.arange(n_blocks, dtype=np.uint64) // 65536
    mine = np.stack(philox.philox4x32_10(c0, np.zeros_like(c0), c2, np.zeros_like(c0),
                                         seed & 0xFFFFFFFF, seed >> 32), axis=1)
    assert (mine == w).all()


def test_philox_bijection_and_avalanche():
    n = 1 << 20
    w = philox.words_for_seed(12345, 4 * n).reshape(n, 4).astype(np.uint64)
    packed = np.stack([(w[:, 0] << np.uint64(32)) | w[:, 1], (w[:, 2] << np.uint64(32)) | w[:, 3]], axis=1)
    assert np.unique(packed, axis=0).shape[0] == n            # injective on 2^20 counters
    a = philox.words_for_seed(99, 4 * 4096)
    for flipped in (philox.words_for_seed(99 ^ 1, 4 * 4096), philox.words_for_seed(99, 4 * 4096, stream_id=1)):
        bits = np.unpackbits((a ^ flipped).view(np.uint8)).sum() / 4096.0
        assert 60.0 < bits < 68.0                              # ~64 of 128 bits flip


def test_words_layout_is_position_pure():
    full = philox.words_for_seed(7, 4096)
    part = philox.words_for_seed(7, 1024, first_elem=2048)
    assert (full[2048:3072] == part).all()
    # counter word c1 = hi32(block index): element 4 * 2^32 uses counter (0, 1, stream, 0)
    far = philox.words_for_seed(7, 4, first_elem=4 * (1 << 32))
    direct = np.stack(philox.philox4x32_10([0], [1], [0], [0], 7, 0), 1)[0]
    assert (far == direct).all()


def test_box_muller_identity_and_bounds():
    w = philox.words_for_seed(3, 1 << 16)
    z = philox.box_muller(w).reshape(-1, 2)
    u1 = ((w.reshape(-1, 2)[:, 0] >> 8).astype(np.float64) + 1.0) / 2 ** 24
    assert np.allclose(z[:, 0] ** 2 + z[:, 1] ** 2, -2.0 * np.log(u1), rtol=1e-12, atol=1e-12)
    assert np.abs(z).max() <= np.sqrt(48 * np.log(2.0)) + 1e-12
    # extreme words: u1 = 2^-24 (largest radius), u1 = 1 (zero radius), u2 = 0 -> angle 0
    ext = philox.box_muller(np.array([0x000000FF, 0, 0xFFFFFFFF, 0], dtype=np.uint32))
    assert abs(ext[0] - np.sqrt(48 * np.log(2.0))) < 1e-12 and ext[1] == 0.0
    assert ext[2] == 0.0 and ext[3] == 0.0
    # quarter turn: u2 = 1/4 -> (cos, sin) = (0, 1)
    q = philox.box_muller(np.array([0x7FFFFF00, 0x40000000], dtype=np.uint32))
    assert abs(q[0]) < 1e-15 and abs(q[1] - np.sqrt(-2 * np.log(0.5))) < 1e-12


def test_box_muller_statistics():
    z = philox.noise_from_seeds([11], 1 << 22)[0]
    assert abs(z.mean()) < 2e-3 and abs(z.var() - 1.0) < 3e-3
    assert abs(stats.skew(z)) < 5e-3 and abs(stats.kurtosis(z)) < 1e-2
    assert stats.kstest(z, "norm").statistic < 1.5e-3
    # the two lanes of a pair are uncorrelated, and so are neighbouring seeds
    pairs = z.reshape(-1, 2)
    assert abs(np.corrcoef(pairs[:, 0], pairs[:, 1])[0, 1]) < 3e-3
    a, b = philox.noise_from_seeds([0, 1], 1 << 18)
    assert abs(np.corrcoef(a, b)[0, 1]) < 1e-2


def test_noise_is_batch_independent():
    a = philox.noise_from_seeds([5, 6, 7], 256)
    b = philox.noise_from_seeds([7], 256)
    assert (a[2] == b[0]).all()
