"""Pins for the oracle's Philox4x32-10 (ref. [60]; R10).

1. NVIDIA cuRAND *host* generator CURAND_RNG_PSEUDO_PHILOX4_32_10 (a library routine,
   runs on the CPU): element n of its stream is PX(c0 = n // 2^18, 0, c2 = (n // 4) % 2^16, 0)
   [n % 4] with key = seed -- exercises rounds, multipliers, key schedule, c0 and c2.
2. An independent implementation with Python big ints (different code shape: no 64-bit
   products split by casts) on random counters/keys -- exercises c1, c3.
3. Known-answer vectors (tests/golden/philox4x32_10_kat.txt).
"""
import ctypes as C
import os
import random

import numpy as np
import pytest

from oracle import philox4x32_10

M32 = 0xFFFFFFFF


def philox_py(ctr, key, rounds=10):
    c = list(ctr)
    k = list(key)
    for _ in range(rounds):
        p0 = 0xD2511F53 * c[0]
        p1 = 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & M32, (p0 >> 32) ^ c[3] ^ k[1], p0 & M32]
        k = [(k[0] + 0x9E3779B9) & M32, (k[1] + 0xBB67AE85) & M32]
    return tuple(c)


def test_kat_vectors():
    path = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")
    n = 0
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(x, 16) for x in line.split()]
        assert philox4x32_10(*v[:6]) == tuple(v[6:])
        assert philox_py(v[:4], v[4:6]) == tuple(v[6:])
        n += 1
    assert n == 3


def test_against_python_bigint():
    rnd = random.Random(1311)
    for _ in range(2000):
        v = [rnd.getrandbits(32) for _ in range(6)]
        assert philox4x32_10(*v) == philox_py(v[:4], v[4:])
    # rounds matter: 7 rounds (the paper's philox4x32_7) must differ
    assert philox_py((1, 2, 3, 4), (5, 6), 7) != philox4x32_10(1, 2, 3, 4, 5, 6)


def _curand_host():
    for name in ("libcurand.so", "libcurand.so.10", "/usr/local/cuda/lib64/libcurand.so"):
        try:
            return C.CDLL(name)
        except OSError:
            continue
    return None


def test_against_curand_host_generator():
    lib = _curand_host()
    if lib is None:
        pytest.skip("libcurand not loadable")
    gen = C.c_void_p()
    assert lib.curandCreateGeneratorHost(C.byref(gen), 161) == 0  # PHILOX4_32_10
    for seed in (0, 4, 0x0123456789ABCDEF, 0xFFFFFFFFFFFFFFFF):
        assert lib.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
        assert lib.curandSetGeneratorOffset(gen, C.c_ulonglong(0)) == 0
        n = (1 << 18) + 64
        out = np.zeros(n, dtype=np.uint32)
        assert lib.curandGenerate(gen, out.ctypes.data_as(C.c_void_p), C.c_size_t(n)) == 0
        k0, k1 = seed & M32, seed >> 32
        for pos in list(range(0, 64)) + [4 * 65535, 4 * 65535 + 3, 1 << 18, (1 << 18) + 7,
                                         4 * 12345 + 2]:
            c0, c2, lane = pos >> 18, (pos >> 2) & 0xFFFF, pos & 3
            assert philox4x32_10(c0, 0, c2, 0, k0, k1)[lane] == int(out[pos]), (seed, pos)
    lib.curandDestroyGenerator(gen)
