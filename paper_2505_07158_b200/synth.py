"""Seeded synthetic video for the five BASELINE.json configs.

This module serves BOTH the oracle-side tests and the CUDA-side tests / bench,
so it holds none of the method's arithmetic: it only draws pixels.  It imports
neither the oracle nor the CUDA binding.

The clips stand in for the paper's Akiyo / Coastguard / Hall / Rhinos / Train /
Waterfall videos, which are not available offline.  Shapes
follow Tab. VIII's resolutions; the value structure (smooth
gradient + blocks + noise) gives the strongly correlated neighbours of natural
frames (Tab. III V_o rows).  Recipe: DESIGN.md "Inputs".
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass

import numpy as np

# fixed test key for all configs: four doubles = 256 bits, gamma, n
KEY = (3.141592653589793, 2.718281828459045, 1.4142135623730951, 1.7320508075688772)
GAMMA = -1.0
N_WORKERS = 32  # the paper's server setting


@dataclass(frozen=True)
class Config:
    name: str
    w: int
    h: int
    frames: int
    seed: int
    kind: str  # "uniform" | "gradient" | "blocks"
    sigma: float = 0.0
    batch: int = 8
    n_streams: int = 3


CONFIGS = {
    "C1": Config("C1", 256, 256, 1, 0, "uniform", batch=1),
    "C2": Config("C2", 640, 480, 24, 1, "gradient", 6.0),
    "C3": Config("C3", 1920, 1080, 30, 2, "blocks", 8.0, batch=1),
    "C4": Config("C4", 1920, 1080, 300, 3, "blocks", 8.0, batch=8, n_streams=3),
    "C5": Config("C5", 3840, 2160, 120, 4, "blocks", 8.0, batch=8, n_streams=3),
}


def _base(cfg: Config, t: int, total: int) -> np.ndarray:
    i = np.arange(cfg.h, dtype=np.float32)[:, None, None]
    j = np.arange(cfg.w, dtype=np.float32)[None, :, None]
    c = np.arange(3, dtype=np.float32)[None, None, :]
    return (255.0 * (i + j + 2.0 * t) / float(cfg.h + cfg.w + 2 * total)) * (1.0 - 0.2 * c)


def frame_iter(cfg: Config, frames: int | None = None, out: np.ndarray | None = None):
    """Yield the clip's frames in order (uint8, H x W x 3).  Taking a prefix of a
    clip gives the same frames as the full clip (one generator, drawn in order)."""
    total = cfg.frames
    count = total if frames is None else frames
    rng = np.random.default_rng(cfg.seed)
    for t in range(count):
        if cfg.kind == "uniform":
            f = rng.integers(0, 256, (cfg.h, cfg.w, 3), dtype=np.uint8)
        else:
            f = _base(cfg, t, total)
            if cfg.kind == "blocks":
                for _ in range(64):
                    y = int(rng.integers(0, cfg.h - 32))
                    x = int(rng.integers(0, cfg.w - 32))
                    colour = rng.integers(0, 256, 3).astype(np.float32)
                    f[y:y + 32, x:x + 32, :] = colour
            f = f + rng.standard_normal((cfg.h, cfg.w, 3), dtype=np.float32) * np.float32(cfg.sigma)
            f = np.clip(np.rint(f), 0, 255).astype(np.uint8)
        if out is not None:
            out[t] = f
        yield f


def video(cfg: Config | str, frames: int | None = None, out: np.ndarray | None = None) -> np.ndarray:
    """The clip as one (T, H, W, 3) uint8 array (optionally written into `out`,
    e.g. a pinned buffer)."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    count = cfg.frames if frames is None else frames
    if out is None:
        out = np.empty((count, cfg.h, cfg.w, 3), np.uint8)
    for _ in frame_iter(cfg, count, out):
        pass
    return out[:count]


def one_bit_pairs(cfg: Config | str, pairs: int, seed: int = 1003):
    """Config 4's plaintext pairs differing in one random bit (NPCR / UACI,
    PAPER.md:473-495): yields (frame, modified_frame, (i, j, c, bit))."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    rng = np.random.default_rng(seed)
    for p, f in enumerate(frame_iter(cfg, pairs)):
        i = int(rng.integers(0, cfg.h))
        j = int(rng.integers(0, cfg.w))
        c = int(rng.integers(0, 3))
        bit = int(rng.integers(0, 8))
        g = f.copy()
        g[i, j, c] ^= np.uint8(1 << bit)
        yield f, g, (i, j, c, bit)


def random_blocks(w: int, h: int, k: int, side: int, seed: int) -> np.ndarray:
    """k non-overlapping side x side blocks inside a w x h frame (top-left (x, y), uint32), for the local Shannon entropy
    test ("randomly selected, non-overlapping sub-blocks"); rejection sampling on a seeded generator."""
    rng = np.random.default_rng(seed)
    out = []
    tries = 0
    while len(out) < k:
        tries += 1
        if tries > 100000:
            raise ValueError("cannot place the blocks")
        x, y = int(rng.integers(0, w - side + 1)), int(rng.integers(0, h - side + 1))
        if all(abs(x - a) >= side or abs(y - b) >= side for a, b in out):
            out.append((x, y))
    return np.array(out, dtype=np.uint32)


def random_frames(w: int, h: int, frames: int, seed: int) -> np.ndarray:
    """i.i.d. uniform bytes, for odd shapes and edge cases."""
    return np.random.default_rng(seed).integers(0, 256, (frames, h, w, 3), dtype=np.uint8)


def random_DB(w: int, h: int, seed: int):
    """Random shift distances (u16, 3(h+w)) and keystream bytes (h, w, 3) for
    kernel-level tests that bypass the derivation."""
    rng = np.random.default_rng(seed)
    D = rng.integers(0, 65536, 3 * (h + w), dtype=np.uint16)
    B = rng.integers(0, 256, (h, w, 3), dtype=np.uint8)
    return D, B


def digest(a: np.ndarray) -> str:
    """SHA-256 of the generated bytes (logged so a numpy stream change cannot
    silently alter a run); hashlib here is bookkeeping, not the method."""
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


# ------------------------------------------------------------------------------------------------------
# channel damage applied to CIPHERTEXT before decryption (Fig. 8 - 9: cropping, salt-and-pepper and
# Gaussian noise).  Inputs of the robustness harness only: no cipher arithmetic here.  The paper's figure gives no noise
# levels; DESIGN.md states the ones used (densities 0.01 / 0.05 / 0.1 per byte, Gaussian variances 0.001 / 0.01 of full scale).
# ------------------------------------------------------------------------------------------------------
def salt_and_pepper(cipher: np.ndarray, density: float, seed: int) -> np.ndarray:
    """A copy of `cipher` in which a fraction `density` of the bytes is forced to 0 or 255 (equal odds)."""
    rng = np.random.default_rng(seed)
    out = cipher.copy()
    hit = rng.random(cipher.shape) < density
    salt = rng.random(cipher.shape) < 0.5
    out[hit & salt] = 255
    out[hit & ~salt] = 0
    return out


def gaussian_noise(cipher: np.ndarray, variance: float, seed: int) -> np.ndarray:
    """A copy of `cipher` with additive zero-mean Gaussian noise of the given variance (full scale = 1), rounded and clipped."""
    rng = np.random.default_rng(seed)
    noisy = cipher.astype(np.float64) + rng.normal(0.0, 255.0 * np.sqrt(variance), cipher.shape)
    return np.clip(np.rint(noisy), 0, 255).astype(np.uint8)


def crop(cipher: np.ndarray, fraction: float) -> np.ndarray:
    """A copy of `cipher` whose top-left rectangle covering `fraction` of the frame area is blanked (Fig. 8)."""
    out = cipher.copy()
    h, w = cipher.shape[-3], cipher.shape[-2]
    s = float(np.sqrt(fraction))
    out[..., : int(round(h * s)), : int(round(w * s)), :] = 0
    return out
