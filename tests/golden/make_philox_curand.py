"""Writes tests/golden/philox_curand_host.txt from the cuRAND HOST generator (CPU only, no GPU).

This is a pin for the ORACLE's Philox4x32-10 (oracle/philox.py), taken from an independent
implementation: NVIDIA's libcurand host generator CURAND_RNG_PSEUDO_PHILOX4_32_10.  It calls
neither oracle/ nor the CUDA library.  Observed ordering of the host generator (see
tests/test_oracle_philox.py): with generator offset `off` (in 32-bit outputs), the i-th
4-word block is Philox(counter = (c0, c1, c2, 0), key = (lo32(seed), hi32(seed))) with
n = off/4 + i, c2 = n % 65536, (c1:c0) = n // 65536.

Each line: seed offset w0 w1 w2 w3 w4 w5 w6 w7   (hex; the first 8 outputs at that offset)
Run:  python tests/golden/make_philox_curand.py
"""
import ctypes
import glob
import os
import site

import numpy as np

SEEDS = [0, 1, 2, 3, 0x0123456789ABCDEF, 0xDEADBEEFCAFEF00D, 2 ** 64 - 1]
OFFSETS = [0, 4 * 17, 4 * 65536, 4 * 65536 * 12345 + 4 * 77, 4 * 65536 * (2 ** 32), 4 * 65536 * (3 * 2 ** 32 + 9) + 4 * 17]


def load_curand():
    for sp in site.getsitepackages():
        hits = glob.glob(os.path.join(sp, "nvidia", "curand", "lib", "libcurand.so*"))
        if hits:
            return ctypes.CDLL(hits[0])
    return ctypes.CDLL("libcurand.so.10")


def curand_words(lib, seed, offset, n):
    gen = ctypes.c_void_p()
    assert lib.curandCreateGeneratorHost(ctypes.byref(gen), 161) == 0      # PHILOX4_32_10
    assert lib.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
    assert lib.curandSetGeneratorOffset(gen, ctypes.c_ulonglong(offset)) == 0
    out = np.zeros(n, dtype=np.uint32)
    assert lib.curandGenerate(gen, out.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(n)) == 0
    lib.curandDestroyGenerator(gen)
    return out


if __name__ == "__main__":
    lib = load_curand()
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "philox_curand_host.txt"), "w") as f:
        f.write("# written by tests/golden/make_philox_curand.py from libcurand's host Philox4_32_10\n")
        for s in SEEDS:
            for off in OFFSETS:
                w = curand_words(lib, s, off, 8)
                f.write(f"{s:016x} {off:x} " + " ".join(f"{int(x):08x}" for x in w) + "\n")
    print("ok")
