"""Pins P1/P2: the oracle's SHA-256 and frame hash H.

FIPS 180-4 published digests (tests/golden/sha256_fips180.txt), the standard's
definition of its constants (fractional parts of cube / square roots of the
first primes, FIPS 180-4 sections 4.2.2 and 5.3.3), hashlib on random lengths
spanning every padding boundary, and PAPER.md:45's H = h_1 xor ... xor h_n.
"""
import hashlib
from math import isqrt

import numpy as np
import pytest

from conftest import read_golden


def _msg(spec: str) -> bytes:
    kind, _, rest = spec.partition(":")
    if kind == "lit":
        return rest.encode()
    text, _, count = rest.partition(":")
    return text.encode() * int(count)


@pytest.mark.parametrize("spec,digest", read_golden("sha256_fips180.txt"))
def test_fips_vectors(orc, spec, digest):
    m = _msg(spec)
    assert hashlib.sha256(m).hexdigest() == digest  # the fixture itself is sound
    assert orc.sha256(m).hex() == digest


def _primes(n):
    out, k = [], 2
    while len(out) < n:
        if all(k % p for p in out if p * p <= k):
            out.append(k)
        k += 1
    return out


def _icbrt(x):
    r = int(round(x ** (1 / 3)))
    while r * r * r > x:
        r -= 1
    while (r + 1) ** 3 <= x:
        r += 1
    return r


def test_constants_from_primes(orc):
    k, h0 = orc.sha256_constants()
    ps = _primes(64)
    # K_t = first 32 bits of the fractional part of cbrt(p_t): floor(cbrt(p * 2^96)) mod 2^32
    want_k = [_icbrt(p << 96) & 0xFFFFFFFF for p in ps]
    want_h = [isqrt(p << 64) & 0xFFFFFFFF for p in ps[:8]]
    assert [int(v) for v in k] == want_k
    assert [int(v) for v in h0] == want_h


def test_random_lengths_vs_hashlib(orc):
    rng = np.random.default_rng(7)
    lengths = list(range(0, 301)) + [511, 512, 513, 1000, 4095, 4096, 65537]
    for n in lengths:
        m = rng.integers(0, 256, n, dtype=np.uint8).tobytes()
        assert orc.sha256(m) == hashlib.sha256(m).digest(), n


def test_H_n1_is_sha256_of_frame(orc):
    f = np.random.default_rng(1).integers(0, 256, (17, 13, 3), dtype=np.uint8)
    assert orc.frame_hash(f, 1) == hashlib.sha256(f.tobytes()).digest()


@pytest.mark.parametrize("h,w,n", [(16, 8, 4), (17, 5, 4), (7, 3, 32), (1080 // 8, 16, 32), (5, 4, 5)])
def test_H_is_xor_of_row_band_hashes(orc, h, w, n):
    f = np.random.default_rng(h * 100 + n).integers(0, 256, (h, w, 3), dtype=np.uint8)
    acc = np.zeros(32, np.uint8)
    covered = 0
    for m in range(n):
        r0, r1 = (m * h) // n, ((m + 1) * h) // n
        covered += r1 - r0
        acc ^= np.frombuffer(hashlib.sha256(f[r0:r1].tobytes()).digest(), np.uint8)
    assert covered == h
    assert orc.frame_hash(f, n) == acc.tobytes()


def test_H_one_bit_avalanche(orc):
    f = np.random.default_rng(3).integers(0, 256, (64, 48, 3), dtype=np.uint8)
    base = np.frombuffer(orc.frame_hash(f, 8), np.uint8)
    flips = []
    rng = np.random.default_rng(4)
    for _ in range(64):
        g = f.copy()
        g[rng.integers(64), rng.integers(48), rng.integers(3)] ^= np.uint8(1 << rng.integers(8))
        d = np.frombuffer(orc.frame_hash(g, 8), np.uint8) ^ base
        flips.append(int(np.unpackbits(d).sum()))
    # one sub-hash changes completely: ~128 of 256 bits, sigma = 8; mean of 64 within 5 sigma/8
    assert 123 < np.mean(flips) < 133
    assert min(flips) > 80
