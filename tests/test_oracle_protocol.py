"""Pins P6-P9, P11: Algorithm 1 end to end on the oracle.

Round trip on the configs and odd shapes, closed-form NPCR / UACI for one-bit plaintext changes
(Eq. 14-16), the frame-to-frame chain of Fig. 12 (:614-620), key sensitivity of
Fig. 6 (:463-469), and the ciphertext statistics of section III (:164-439) against the values an
i.i.d. uniform byte source gives.
"""
import numpy as np
import pytest

from paper_2505_07158_b200 import synth

NPCR_IDEAL = 255 / 256 * 100                         # 99.609375 %
UACI_IDEAL = (256**2 - 1) / (3 * 256 * 255) * 100    # 33.463542 %


def npcr_uaci(a, b):
    a = a.astype(np.int32).ravel(); b = b.astype(np.int32).ravel()
    return 100.0 * np.mean(a != b), 100.0 * np.mean(np.abs(a - b)) / 255.0


def test_closed_form_constants():
    # Eq. 14-16 for two independent uniform bytes: P(a != b) = 255/256, E|a-b| = (256^2-1)/(3*256)
    v = np.arange(256)
    d = np.abs(v[:, None] - v[None, :])
    assert abs(100 * (d != 0).mean() - NPCR_IDEAL) < 1e-12
    assert abs(100 * d.mean() / 255 - UACI_IDEAL) < 1e-12
    assert round(NPCR_IDEAL, 6) == 99.609375 and round(UACI_IDEAL, 6) == 33.463542


@pytest.mark.parametrize("name,frames", [("C1", 1), ("C2", 3)])
def test_round_trip_configs(orc, name, frames):
    cfg = synth.CONFIGS[name]
    v = synth.video(cfg, frames)
    enc = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h)
    dec = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h)
    E, H = enc.encrypt_frames(v)
    assert (dec.decrypt_frames(E, H) == v).all()
    for t in range(frames):
        assert H[t].tobytes() == orc.frame_hash(v[t], synth.N_WORKERS)
        assert npcr_uaci(E[t], v[t])[0] > 99.0


@pytest.mark.parametrize("w,h,n", [(1, 1, 1), (1, 7, 2), (7, 1, 3), (5, 3, 32), (31, 17, 4), (100, 37, 6)])
def test_round_trip_odd_shapes(orc, w, h, n):
    v = synth.random_frames(w, h, 3, seed=w * 1000 + h)
    enc = orc.ctx(synth.KEY, -0.5, n, w, h)
    dec = orc.ctx(synth.KEY, -0.5, n, w, h)
    E, H = enc.encrypt_frames(v)
    assert (dec.decrypt_frames(E, H) == v).all()


def test_frames_must_be_decrypted_in_order(orc):
    """frame f's initial conditions come from frame f-1's x_2n..w_2n."""
    w, h = 32, 24
    v = synth.random_frames(w, h, 2, seed=9)
    enc = orc.ctx(synth.KEY, -1.0, 4, w, h)
    E, H = enc.encrypt_frames(v)
    dec = orc.ctx(synth.KEY, -1.0, 4, w, h)
    wrong = dec.decrypt_frames(E[1:], H[1:])       # second frame first: garbage
    assert np.mean(wrong[0] != v[1]) > 0.98


def test_npcr_uaci_one_bit_pairs(orc):
    """P7: 20 one-bit pairs at 256x256 (N = 196608 bytes per frame).  Per-pair sigma:
    NPCR sqrt(p(1-p)/N) = 0.0141 %, UACI 0.2366/sqrt(N) = 0.0534 %; accept each pair within
    5 sigma and the mean within 3 sigma/sqrt(20)."""
    cfg = synth.CONFIGS["C1"]
    N = 3 * cfg.w * cfg.h
    s_n, s_u = 100 * np.sqrt(255 / 256 / 256 / N), 100 * 0.2366 / np.sqrt(N)
    res = []
    base = synth.random_frames(cfg.w, cfg.h, 20, seed=77)
    rng = np.random.default_rng(1003)
    for p in range(20):
        f = base[p]
        g = f.copy()
        g[rng.integers(cfg.h), rng.integers(cfg.w), rng.integers(3)] ^= np.uint8(1 << rng.integers(8))
        e1, _ = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h).encrypt_frames(f[None])
        e2, _ = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h).encrypt_frames(g[None])
        n_, u_ = npcr_uaci(e1, e2)
        assert abs(n_ - NPCR_IDEAL) < 5 * s_n and abs(u_ - UACI_IDEAL) < 5 * s_u, (p, n_, u_)
        res.append((n_, u_))
        for c in range(3):  # every channel changes (Fig. 12 (e)-(g))
            assert npcr_uaci(e1[0, :, :, c], e2[0, :, :, c])[0] > 99.3
    m = np.mean(res, axis=0)
    assert abs(m[0] - NPCR_IDEAL) < 3 * s_n / np.sqrt(20)
    assert abs(m[1] - UACI_IDEAL) < 3 * s_u / np.sqrt(20)
    # the paper's 512x512 critical values hold a fortiori for the mean
    assert m[0] > 99.5893 and 33.3730 < m[1] < 33.5541


def test_chain_next_frame_changes_although_its_hash_does_not(orc):
    """P8 / Fig. 12(h): a one-bit change in frame 0 changes ~99.6 % of frame 1's ciphertext."""
    w, h = 96, 64
    v = synth.random_frames(w, h, 2, seed=5)
    v2 = v.copy()
    v2[0, 10, 20, 1] ^= 4
    E1, H1 = orc.ctx(synth.KEY, -1.0, 8, w, h).encrypt_frames(v)
    E2, H2 = orc.ctx(synth.KEY, -1.0, 8, w, h).encrypt_frames(v2)
    assert (H1[1] == H2[1]).all() and (H1[0] != H2[0]).any()
    assert abs(npcr_uaci(E1[1], E2[1])[0] - NPCR_IDEAL) < 0.3


@pytest.mark.parametrize("which", [0, 1, 2, 3])
def test_key_sensitivity_1e14(orc, which):
    """P9 / Fig. 6: decrypting with x0 (y0, z0, w0) + 1e-14 leaves ~99.6 % of the bytes wrong."""
    w, h = 96, 64
    v = synth.random_frames(w, h, 1, seed=6)
    E, H = orc.ctx(synth.KEY, -1.0, 8, w, h).encrypt_frames(v)
    key = list(synth.KEY)
    key[which] += 1e-14
    assert key[which] != synth.KEY[which]
    P = orc.ctx(key, -1.0, 8, w, h).decrypt_frames(E, H)
    assert abs(100 * np.mean(P != v) - NPCR_IDEAL) < 0.5


def test_ciphertext_statistics_512(orc):
    """P11: a smooth 512x512 frame (adjacent-pixel correlation > 0.95, as Tab. III's V_o rows)
    encrypts to bytes whose chi-square (Eq. 5), entropy (Eq. 10) and adjacent-pixel correlation
    (Eq. 6-9) match an i.i.d. uniform source: chi-square ~ 255 +- 22.6 (paper's bound 293.25 is
    the 5 % point; 340 used here is ~3.8 sigma), entropy ~ 8 - 255/(2 N ln 2) = 7.99930,
    mean |r| of 10000 pairs ~ 0.008."""
    w = h = 512
    i = np.arange(h)[:, None, None]; j = np.arange(w)[None, :, None]; c = np.arange(3)[None, None, :]
    rng = np.random.default_rng(12)
    F = np.clip(np.rint(255.0 * (i + j) / (h + w) * (1 - 0.2 * c) + rng.normal(0, 3, (h, w, 3))), 0, 255).astype(np.uint8)
    assert np.corrcoef(F[:, :-1, 0].ravel(), F[:, 1:, 0].ravel())[0, 1] > 0.95
    E, _ = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, w, h).encrypt_frames(F[None])
    E = E[0]
    N = w * h
    for ch in range(3):
        cnt = np.bincount(E[:, :, ch].ravel(), minlength=256)
        chi = ((cnt - N / 256) ** 2 / (N / 256)).sum()
        assert chi < 340, (ch, chi)
        p = cnt / N
        ent = -(p[p > 0] * np.log2(p[p > 0])).sum()
        assert 7.9990 < ent < 8.0, (ch, ent)
        ys = rng.integers(0, h - 1, 10000); xs = rng.integers(0, w - 1, 10000)
        a = E[ys, xs, ch].astype(float)
        for dy, dx in ((0, 1), (1, 0), (1, 1)):
            r = np.corrcoef(a, E[ys + dy, xs + dx, ch].astype(float))[0, 1]
            assert abs(r) < 0.04, (ch, dy, dx, r)
