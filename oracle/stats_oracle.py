"""oracle/stats_oracle.py -- plain numpy statements of the paper's evaluation metrics (PAPER.md sections III-IV).

TEST INFRASTRUCTURE ONLY (like oracle/vcrypt_oracle.c): only tests/ may import it; it shares nothing with the product.
Each function is the equation as printed, in binary64, with no blocking or algebraic shortcut:
  hist_variance  Eq. 4     chi2      Eq. 5  (:177)
  correlation    Eq. 6-9 (:283-294), over ALL adjacent pairs of a direction (the paper samples 6 000 / 10 000 of them at
                 random, :269, :294; taking all of them is the deterministic limit of that sampling)
  entropy        Eq. 10 (:345), log base 2   local_entropy Eq. 11 (:394)
  npcr, uaci     Eq. 14-16 (:482-491)
Pins (tests/test_oracle_stats.py): Eq. 4 == population variance of the histogram (numpy.var), Eq. 5 == scipy.stats.chisquare,
Eq. 6 == numpy.corrcoef, Eq. 10 == scipy.stats.entropy(base=2) and 8 bits for a flat histogram, closed forms for constant /
complementary / independent uniform frames.
"""
import numpy as np


def histogram(channel: np.ndarray) -> np.ndarray:
    """z_i = number of pixels of intensity i, i = 0..255."""
    return np.bincount(np.asarray(channel, dtype=np.uint8).ravel(), minlength=256).astype(np.float64)


def hist_variance(channel: np.ndarray) -> float:
    z = histogram(channel)
    return float(np.sum(0.5 * (z[:, None] - z[None, :]) ** 2) / 256.0 ** 2)  # Eq. 4


def chi2(channel: np.ndarray) -> float:
    z = histogram(channel)
    e = channel.size / 256.0
    return float(np.sum((z - e) ** 2 / e))  # Eq. 5


def entropy(channel: np.ndarray) -> float:
    z = histogram(channel)
    p = z[z > 0] / channel.size
    return float(np.sum(p * np.log2(1.0 / p)))  # Eq. 10


def _pairs(channel: np.ndarray, direction: int):
    a = np.asarray(channel, dtype=np.float64)
    if direction == 0:  # horizontal: (i, j) - (i, j+1)
        return a[:, :-1].ravel(), a[:, 1:].ravel()
    if direction == 1:  # vertical: (i, j) - (i+1, j)
        return a[:-1, :].ravel(), a[1:, :].ravel()
    return a[:-1, :-1].ravel(), a[1:, 1:].ravel()  # diagonal: (i, j) - (i+1, j+1)


def correlation(channel: np.ndarray, direction: int) -> float:
    x, y = _pairs(channel, direction)
    if x.size == 0:
        return float("nan")
    ex, ey = np.sum(x) / x.size, np.sum(y) / y.size                     # Eq. 9
    cov = np.sum((x - ex) * (y - ey)) / x.size                           # Eq. 7
    dx, dy = np.sum((x - ex) ** 2) / x.size, np.sum((y - ey) ** 2) / y.size  # Eq. 8
    if dx == 0 or dy == 0:
        return float("nan")
    return float(cov / np.sqrt(dx * dy))                                 # Eq. 6


def local_entropy(channel: np.ndarray, blocks_xy, side: int) -> float:
    hs = [entropy(channel[y:y + side, x:x + side]) for x, y in blocks_xy]
    return float(np.sum(hs) / len(hs))  # Eq. 11


def npcr(a: np.ndarray, b: np.ndarray) -> float:
    d = (np.asarray(a) != np.asarray(b))  # Eq. 16
    return float(np.sum(d) / d.size * 100.0)  # Eq. 14


def uaci(a: np.ndarray, b: np.ndarray) -> float:
    d = np.abs(np.asarray(a, dtype=np.float64) - np.asarray(b, dtype=np.float64))
    return float(np.sum(d) / (d.size * 255.0) * 100.0)  # Eq. 15
