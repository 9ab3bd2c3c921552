"""NEXT-4: the robustness experiments of PAPER.md section IV as a harness through the C ABI, on synthetic
video (the paper's clips are not available): key sensitivity (Fig. 6), cropping (Fig. 8, :547-551),
salt-and-pepper and Gaussian channel noise (Fig. 9, :553-557).  Every decryption runs in vcrypt_decrypt_frames on the
GPU and is compared element by element with the oracle's decryption of the same bytes with the same (possibly wrong)
key; the damage counts come from vcrypt_npcr_uaci_device and are held against what the absence of diffusion promises
(a damaged ciphertext byte reaches at most two plaintext bytes, same channel)."""
import numpy as np
import pytest

from paper_2505_07158_b200 import synth

pytestmark = pytest.mark.gpu

NPCR_IDEAL = 100.0 * 255 / 256
W, H, NF = 640, 480, 3  # config 2's shape (Tab. VIII); three chained frames


@pytest.fixture(scope="module")
def vb():
    from paper_2505_07158_b200 import binding

    return binding


@pytest.fixture(scope="module")
def clip(vb, orc):
    """Plaintext, ciphertext and hashes of a strongly correlated clip (C2's generator), encrypted on the GPU path and
    checked against the oracle once."""
    cfg = synth.CONFIGS["C2"]
    frames = synth.video(cfg, NF)
    C, Hs = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, W, H).encrypt_frames(frames)
    Co, Ho = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, W, H).encrypt_frames(frames)
    assert np.array_equal(C, Co) and np.array_equal(Hs, Ho)
    return frames, C, Hs


def gpu_decrypt(vb, key, C, Hs):
    return vb.Vcrypt(key, synth.GAMMA, synth.N_WORKERS, W, H).decrypt_frames(C, Hs)


def differing(vb, a, b):
    """Percentage of differing bytes per frame: (all channels, c0, c1, c2) from vcrypt_npcr_uaci_device."""
    import torch

    v = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, W, H)
    npcr, _ = v.npcr_uaci_device(torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda())
    return npcr


@pytest.mark.parametrize("which", [0, 1, 2, 3])
def test_key_sensitivity_through_decrypt_frames(vb, orc, clip, which):
    """Fig. 6: x0 (y0, z0, w0) + 1e-14 at the receiver -> about 99.6 % of the bytes of every frame wrong, and exactly the
    bytes the oracle gets with the same wrong key."""
    frames, C, Hs = clip
    key = list(synth.KEY)
    key[which] += 1e-14
    assert key[which] != synth.KEY[which]
    P = gpu_decrypt(vb, key, C, Hs)
    assert np.array_equal(P, orc.ctx(key, synth.GAMMA, synth.N_WORKERS, W, H).decrypt_frames(C, Hs))
    npcr = differing(vb, P, frames)
    n = 3 * W * H
    sigma = 100.0 * np.sqrt((255 / 256) * (1 / 256) / n)
    for k in range(NF):
        assert abs(npcr[k, 0] - NPCR_IDEAL) < 6 * sigma + 0.02, (k, npcr[k])
    assert np.array_equal(gpu_decrypt(vb, synth.KEY, C, Hs), frames)  # the right key still opens it


def check_damage(vb, orc, frames, C, Hs, damaged):
    """Decrypt damaged ciphertext on the GPU; same bytes as the oracle; damage stays local (no diffusion)."""
    P = gpu_decrypt(vb, synth.KEY, damaged, Hs)
    assert np.array_equal(P, orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, W, H).decrypt_frames(damaged, Hs))
    hit = differing(vb, damaged, C)      # % of ciphertext bytes the channel changed
    bad = differing(vb, P, frames)       # % of plaintext bytes that came out wrong
    for k in range(NF):
        assert hit[k, 0] > 0
        for c in range(4):  # all channels together, then each channel: damage never crosses channels
            assert 0 < bad[k, c] <= 2.0 * hit[k, c] + 1e-12, (k, c, hit[k], bad[k])
    return hit, bad


@pytest.mark.parametrize("density", [0.01, 0.05, 0.1])
def test_salt_and_pepper_on_ciphertext(vb, orc, clip, density):
    frames, C, Hs = clip
    hit, bad = check_damage(vb, orc, frames, C, Hs, synth.salt_and_pepper(C, density, seed=int(density * 1000)))
    # a forced byte differs from a uniform ciphertext byte with probability 255/256
    assert abs(hit[:, 0].mean() - 100.0 * density * 255 / 256) < 0.1
    # an 8-bit window straddles two bytes unless the rotation is a whole number of bytes: close to 2 plaintext bytes per hit
    assert bad[:, 0].mean() > 1.5 * hit[:, 0].mean() * (1 - density)


@pytest.mark.parametrize("variance", [0.001, 0.01])
def test_gaussian_noise_on_ciphertext(vb, orc, clip, variance):
    frames, C, Hs = clip
    check_damage(vb, orc, frames, C, Hs, synth.gaussian_noise(C, variance, seed=7))


@pytest.mark.parametrize("fraction", [1 / 16, 1 / 4, 1 / 2])
def test_cropping_of_ciphertext(vb, orc, clip, fraction):
    frames, C, Hs = clip
    hit, bad = check_damage(vb, orc, frames, C, Hs, synth.crop(C, fraction))
    assert abs(hit[:, 0].mean() - 100.0 * fraction * 255 / 256) < 1.0
    assert bad[:, 0].max() < 100.0 * (1 - (1 - fraction) ** 2) + 1.0  # a plaintext byte is wrong only if one of its two sources was cropped
