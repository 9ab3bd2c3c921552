"""Pins of the statistics oracle (oracle/stats_oracle.py; Eq. 4-11, 14-16) against library routines, closed forms
and special cases, so that a wrong sign, index, normalisation or log base fails one of them."""
import numpy as np
import pytest

from oracle import stats_oracle as so


def rnd(h, w, seed):
    return np.random.default_rng(seed).integers(0, 256, (h, w), dtype=np.uint8)


def test_hist_variance_is_the_population_variance_of_the_histogram():
    a = rnd(64, 48, 1)
    z = np.bincount(a.ravel(), minlength=256).astype(np.float64)
    assert np.isclose(so.hist_variance(a), np.var(z), rtol=1e-12)
    assert so.hist_variance(np.repeat(np.arange(256, dtype=np.uint8), 4).reshape(32, 32)) == 0.0  # flat histogram
    n = 64 * 64
    const = np.full((64, 64), 7, np.uint8)  # one bin holds everything: var = N^2 (1/256)(255/256)
    assert np.isclose(so.hist_variance(const), n * n * (1 / 256) * (255 / 256), rtol=1e-12)


def test_chi2_matches_scipy_and_closed_forms():
    from scipy.stats import chisquare

    a = rnd(96, 80, 2)
    z = np.bincount(a.ravel(), minlength=256)
    assert np.isclose(so.chi2(a), chisquare(z).statistic, rtol=1e-12)
    assert np.isclose(so.chi2(np.full((32, 32), 200, np.uint8)), 255.0 * 32 * 32, rtol=1e-12)  # constant frame: 255 N
    # i.i.d. uniform bytes: E = 255, sd = sqrt(510); PAPER.md:179 critical value 293.25 at alpha = 0.05
    vals = [so.chi2(rnd(256, 256, s)) for s in range(20)]
    assert abs(np.mean(vals) - 255.0) < 4 * np.sqrt(510 / 20)


def test_entropy_matches_scipy_and_special_cases():
    from scipy.stats import entropy as sp_entropy

    a = rnd(50, 70, 3)
    z = np.bincount(a.ravel(), minlength=256)
    assert np.isclose(so.entropy(a), sp_entropy(z, base=2), rtol=1e-12)
    assert so.entropy(np.repeat(np.arange(256, dtype=np.uint8), 4).reshape(32, 32)) == 8.0
    assert so.entropy(np.full((8, 8), 3, np.uint8)) == 0.0
    two = np.zeros((8, 8), np.uint8); two[:4] = 9
    assert so.entropy(two) == 1.0
    n = 512 * 512  # PAPER.md Tab. IV: encrypted ~ 7.9993 = 8 - 255 / (2 N ln 2)
    assert abs(so.entropy(rnd(512, 512, 4)) - (8 - 255 / (2 * n * np.log(2)))) < 2e-4


@pytest.mark.parametrize("direction", [0, 1, 2])
def test_correlation_matches_numpy_corrcoef_and_pair_geometry(direction):
    i, j = np.meshgrid(np.arange(40), np.arange(56), indexing="ij")
    a = ((3 * i + 5 * j + rnd(40, 56, 5) // 16) % 256).astype(np.uint8)
    x, y = so._pairs(a, direction)
    assert np.isclose(so.correlation(a, direction), np.corrcoef(x, y)[0, 1], rtol=1e-10)
    di, dj = [(0, 1), (1, 0), (1, 1)][direction]
    assert x.size == (40 - di) * (56 - dj)
    assert x[0] == a[0, 0] and y[0] == a[di, dj]  # (i, j) pairs with (i + di, j + dj)
    ramp = np.tile(np.arange(56, dtype=np.uint8), (40, 1))  # depends on j only: r = 1 horizontally and diagonally
    if direction != 1:
        assert np.isclose(so.correlation(ramp, direction), 1.0)
    else:
        assert np.isclose(so.correlation(ramp, direction), 1.0)  # identical pairs vertically
    assert np.isnan(so.correlation(np.full((4, 4), 1, np.uint8), direction))  # zero variance
    assert abs(so.correlation(rnd(300, 300, 6), direction)) < 5 / np.sqrt(299 * 299)


def test_local_entropy_is_the_mean_of_block_entropies():
    a = rnd(128, 128, 7)
    blocks = [(0, 0), (44, 0), (0, 44), (80, 80)]
    assert np.isclose(so.local_entropy(a, blocks, 44), np.mean([so.entropy(a[y:y + 44, x:x + 44]) for x, y in blocks]))
    b = a.copy(); b[0:44, 0:44] = 5  # one constant block of four: its entropy 0
    assert np.isclose(so.local_entropy(b, blocks, 44), 0.75 * np.mean([so.entropy(a[y:y + 44, x:x + 44]) for x, y in blocks[1:]]))
    # ideal H(30, 1936) = 7.902469317 for uniform bytes
    vals = []
    for s in range(8):
        f = rnd(512, 512, 100 + s)
        vals.append(so.local_entropy(f, [(44 * (k % 10), 44 * (k // 10)) for k in range(30)], 44))
    assert abs(np.mean(vals) - 7.902469317) < 1e-3


def test_npcr_uaci_special_cases_and_closed_forms():
    a = rnd(64, 64, 8)
    assert so.npcr(a, a) == 0.0 and so.uaci(a, a) == 0.0
    z, o = np.zeros((16, 16), np.uint8), np.full((16, 16), 255, np.uint8)
    assert so.npcr(z, o) == 100.0 and so.uaci(z, o) == 100.0 and so.uaci(o, z) == 100.0  # |a - b|, not a - b
    b = a.copy(); b[3, 5] ^= 1
    assert np.isclose(so.npcr(a, b), 100.0 / a.size) and np.isclose(so.uaci(a, b), 100.0 / (a.size * 255.0))
    x, y = rnd(512, 512, 9), rnd(512, 512, 10)  # independent uniform: PAPER.md:493 expectations
    assert abs(so.npcr(x, y) - 100 * 255 / 256) < 5 * 100 * np.sqrt(255 / 256 / 256 / x.size)
    assert abs(so.uaci(x, y) - 100 * (256 ** 2 - 1) / (3 * 256 * 255)) < 5 * 0.0462
