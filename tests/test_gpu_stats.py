"""GPU parity of the statistical evaluation kernels (Eq. 4-11, 14-16) against
oracle/stats_oracle.py: histograms bit for bit, the floating-point quantities to rounding (the device produces exact
integer sums, the last binary64 steps run on the host: tolerance 1e-9 relative, derived from ~1e3 accumulated roundings of
the oracle's literal sums at 1e-16 each), on random and strongly correlated frames, odd shapes and ciphertext."""
import numpy as np
import pytest

from oracle import stats_oracle as so
from paper_2505_07158_b200 import synth

pytestmark = pytest.mark.gpu
RTOL = 1e-9


@pytest.fixture(scope="module")
def torch_cuda():
    import torch

    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def vb():
    from paper_2505_07158_b200 import binding

    return binding


def frames_for(kind, w, h, nf, seed):
    if kind == "random":
        return synth.random_frames(w, h, nf, seed)
    i, j = np.meshgrid(np.arange(h), np.arange(w), indexing="ij")
    rng = np.random.default_rng(seed)
    out = np.empty((nf, h, w, 3), np.uint8)
    for f in range(nf):
        for c in range(3):
            out[f, :, :, c] = np.clip(0.7 * i + 0.4 * j * (1 + c) / 2 + 10 * f + rng.normal(0, 4, (h, w)), 0, 255).astype(np.uint8)
    return out


@pytest.mark.parametrize("kind", ["random", "smooth"])
# w % 4 == 0: DP4A fast path (incl. a single item per row, a single row, a single column of items); others: byte path
@pytest.mark.parametrize("w,h,nf", [(64, 48, 2), (4, 6, 2), (8, 1, 2), (4, 1, 1), (132, 33, 1), (640, 480, 2), (1920, 1080, 1),
                                    (17, 9, 3), (1, 7, 1), (5, 1, 2), (130, 33, 1)])
def test_frame_stats_match_oracle(torch_cuda, vb, kind, w, h, nf):
    F = frames_for(kind, w, h, nf, seed=w * 7 + h)
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, 4, w, h)
    r = v.frame_stats_device(torch_cuda.from_numpy(F).cuda())
    for f in range(nf):
        for c in range(3):
            ch = F[f, :, :, c]
            assert np.array_equal(r["hist"][f, c], np.bincount(ch.ravel(), minlength=256))
            assert np.isclose(r["hist_variance"][f, c], so.hist_variance(ch), rtol=RTOL, atol=1e-9)
            assert np.isclose(r["chi2"][f, c], so.chi2(ch), rtol=RTOL)
            assert np.isclose(r["entropy"][f, c], so.entropy(ch), rtol=RTOL, atol=1e-12)
            for d in range(3):
                ref = so.correlation(ch, d)
                if np.isnan(ref):
                    assert np.isnan(r["corr"][f, c, d])
                else:
                    assert np.isclose(r["corr"][f, c, d], ref, rtol=RTOL, atol=1e-9), (c, d)


@pytest.mark.parametrize("w,h,nf", [(64, 48, 2), (17, 9, 2), (1, 1, 1), (640, 480, 1)])
def test_npcr_uaci_match_oracle(torch_cuda, vb, w, h, nf):
    A, B = synth.random_frames(w, h, nf, 1), synth.random_frames(w, h, nf, 2)
    B[0, 0, 0, 0] = A[0, 0, 0, 0]
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, 4, w, h)
    npcr, uaci = v.npcr_uaci_device(torch_cuda.from_numpy(A).cuda(), torch_cuda.from_numpy(B).cuda())
    for f in range(nf):
        assert np.isclose(npcr[f, 0], so.npcr(A[f], B[f]), rtol=1e-12) and np.isclose(uaci[f, 0], so.uaci(A[f], B[f]), rtol=1e-12)
        for c in range(3):
            assert np.isclose(npcr[f, 1 + c], so.npcr(A[f, :, :, c], B[f, :, :, c]), rtol=1e-12)
            assert np.isclose(uaci[f, 1 + c], so.uaci(A[f, :, :, c], B[f, :, :, c]), rtol=1e-12)
    z, _ = v.npcr_uaci_device(torch_cuda.from_numpy(A).cuda(), torch_cuda.from_numpy(A).cuda())
    assert np.all(z == 0.0)


def test_local_entropy_matches_oracle_and_rejects_blocks_outside(torch_cuda, vb):
    w, h, nf = 512, 512, 2
    F = synth.random_frames(w, h, nf, 3)
    blocks = synth.random_blocks(w, h, 30, 44, seed=5)
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, 4, w, h)
    out = v.local_entropy_device(torch_cuda.from_numpy(F).cuda(), blocks, 44)
    for f in range(nf):
        for c in range(3):
            assert np.isclose(out[f, c], so.local_entropy(F[f, :, :, c], blocks, 44), rtol=RTOL)
    bad = blocks.copy(); bad[3] = (500, 10)
    res = np.empty((nf, 3))
    rc = v.L.vcrypt_local_entropy_device(v._p, torch_cuda.from_numpy(F).cuda().data_ptr(), nf, bad.ctypes.data, 30, 44, res.ctypes.data, 0)
    assert rc == vb.E_ARG


def test_ciphertext_statistics_512(torch_cuda, vb):
    """The paper's acceptance ranges on OUR ciphertext at 512 x 512 (Tab. I-VII; closed forms for uniform
    bytes in SURVEY.md section 4): chi^2 < 293.25 on average, entropy ~ 7.9993, |r| ~ 0.002 over all pairs, local
    entropy inside (7.9015, 7.9034) on average, NPCR / UACI of a one-bit pair inside the 512^2 critical values."""
    torch = torch_cuda
    cfg = synth.Config("S", 512, 512, 8, 77, "blocks", 8.0, 8, 3)
    frames = synth.video(cfg, 8)
    enc = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, 512, 512, batch=8)
    C, _ = enc.encrypt_frames(frames)
    dC = torch.from_numpy(C).cuda()
    r = enc.frame_stats_device(dC)
    plain = enc.frame_stats_device(torch.from_numpy(frames).cuda())
    assert np.mean(r["chi2"]) < 293.25 and np.mean(plain["chi2"]) > 10000
    assert abs(np.mean(r["entropy"]) - 7.9993) < 2e-4
    assert np.mean(np.abs(r["corr"])) < 0.004 and np.mean(np.abs(plain["corr"])) > 0.9
    le = enc.local_entropy_device(dC, synth.random_blocks(512, 512, 30, 44, 9), 44)
    assert 7.9005 < np.mean(le) < 7.9044
    g = frames[:1].copy(); g[0, 100, 200, 1] ^= 4
    C2, _ = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, 512, 512, batch=1).encrypt_frames(g)
    C1, _ = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, 512, 512, batch=1).encrypt_frames(frames[:1])
    npcr, uaci = enc.npcr_uaci_device(torch.from_numpy(C1).cuda(), torch.from_numpy(C2).cuda())
    assert npcr[0, 0] > 99.5893 and 33.3730 < uaci[0, 0] < 33.5541
