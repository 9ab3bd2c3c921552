"""vcrypt_npcr_uaci_device_noalloc: NPCR / UACI (Eq. 14-16) for callers that cannot allocate GPU memory.

Why the entry point exists: the ordinary call, vcrypt_npcr_uaci_device, does a cudaMalloc and a cudaFree every time.  A
process that runs inside someone else's memory budget cannot do that -- an inference server or a framework pool that took
all of HBM at start-up leaves cudaMalloc nothing to give; a video loop with a frame deadline cannot afford the driver lock
and the device-wide wait that cudaFree implies; a service with a "nothing is allocated after start-up" rule is not allowed
to.  For them the library carries a fixed 24 KB accumulator array in its own device image and this call uses only that.

What is checked here, on a GPU, through the C ABI:
  * the numbers equal those of the allocating call (same integer sums on the device, same binary64 steps on the host,
    so exact equality is expected; the assertion uses the 1e-12 relative tolerance of tests/test_gpu_stats.py);
  * on TWO CALLS IN A ROW: the array is shared and keeps the previous call's sums, so the second call -- made with fewer
    frames, smaller differences, and once from a context of another frame shape -- must not see anything of the first;
  * the documented capacity: exactly VCRYPT_NOALLOC_MAX_FRAMES frames work, one more is refused with VCRYPT_E_LIMIT and a
    message that names both numbers.
The capacity check needs no GPU and runs in the CPU suite as well.

This file is named so that pytest collects it last: under `pytest -x` a failure here must not hide the parity tests.  It
passes on its own in a fresh process (its first call is then the one that does the per-device set-up) and after the rest
of the suite."""
import numpy as np
import pytest

from paper_2505_07158_b200 import synth

RTOL = 1e-12  # as tests/test_gpu_stats.py::test_npcr_uaci_match_oracle


@pytest.fixture(scope="module")
def torch_cuda():
    import torch

    assert torch.cuda.is_available()
    return torch


@pytest.fixture(scope="module")
def vb():
    from paper_2505_07158_b200 import binding

    return binding


def _same(got, want):
    return all(np.allclose(g, w, rtol=RTOL, atol=0.0) for g, w in zip(got, want))


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_allocating_path(torch_cuda, vb):
    torch = torch_cuda
    w, h, nf = 200, 120, 5  # 72 000 bytes per frame: several CTAs per frame and a ragged tail of 12-byte items
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, 4, w, h)
    A = torch.from_numpy(synth.random_frames(w, h, nf, 11)).cuda()
    B = torch.from_numpy(synth.random_frames(w, h, nf, 12)).cuda()
    want1 = v.npcr_uaci_device(A, B)
    assert want1[0].min() > 99.0  # random against random: large sums left behind in the shared array

    # call 1: every frame differs almost everywhere
    got1 = v.npcr_uaci_device_noalloc(A, B)
    assert _same(got1, want1)

    # call 2, straight after: fewer frames and a single differing byte; any leftover of call 1 would swamp it
    C = A[:2].clone()
    C[1, 7, 9, 2] ^= 0x40
    want2 = v.npcr_uaci_device(A[:2], C)
    got2 = v.npcr_uaci_device_noalloc(A[:2], C)
    assert _same(got2, want2)
    assert np.all(got2[0][0] == 0.0) and np.all(got2[1][0] == 0.0)  # frame 0 is identical
    assert got2[0][1, 3] == pytest.approx(100.0 / (w * h), rel=RTOL) and got2[0][1, 1] == 0.0  # one byte, channel 2

    # call 3: another context (another shape) on the same GPU uses the same array
    w2, h2 = 17, 9
    v2 = vb.Vcrypt(synth.KEY, synth.GAMMA, 3, w2, h2)
    P = torch.from_numpy(synth.random_frames(w2, h2, 3, 21)).cuda()
    Q = torch.from_numpy(synth.random_frames(w2, h2, 3, 22)).cuda()
    assert _same(v2.npcr_uaci_device_noalloc(P, Q), v2.npcr_uaci_device(P, Q))

    # and back: the first context again, on a non-default stream, identical inputs -> all zero
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        z = v.npcr_uaci_device_noalloc(A, A, stream=s.cuda_stream)
    assert np.all(z[0] == 0.0) and np.all(z[1] == 0.0)
    assert _same(v.npcr_uaci_device_noalloc(A, B), want1)


@pytest.mark.gpu
def test_capacity_is_exactly_the_documented_maximum(torch_cuda, vb):
    torch = torch_cuda
    w, h, cap = 8, 4, vb.NOALLOC_MAX_FRAMES
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, 2, w, h)
    A = torch.from_numpy(synth.random_frames(w, h, cap + 1, 31)).cuda()
    B = torch.from_numpy(synth.random_frames(w, h, cap + 1, 32)).cuda()
    assert _same(v.npcr_uaci_device_noalloc(A[:cap], B[:cap]), v.npcr_uaci_device(A[:cap], B[:cap]))
    with pytest.raises(vb.VcryptError) as ei:
        v.npcr_uaci_device_noalloc(A, B)
    assert ei.value.code == vb.E_LIMIT and str(cap + 1) in str(ei.value) and str(cap) in str(ei.value)
    # a refused call enqueued nothing and left the library usable
    assert _same(v.npcr_uaci_device_noalloc(A[:3], B[:3]), v.npcr_uaci_device(A[:3], B[:3]))


def test_oversized_call_is_refused_before_any_cuda_work(vb):
    """CPU suite: the limit is checked ahead of everything that needs a GPU, so a host-only context reports it too."""
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, 2, 8, 4, flags=vb.FLAG_HOST_ONLY)
    out = np.empty((vb.NOALLOC_MAX_FRAMES + 1, 4))
    fake = 0x1000  # never dereferenced: the call fails first
    rc = v.L.vcrypt_npcr_uaci_device_noalloc(v._p, fake, fake, vb.NOALLOC_MAX_FRAMES + 1, out.ctypes.data, out.ctypes.data, 0)
    assert rc == vb.E_LIMIT
    assert "scratch" in v.L.vcrypt_strerror(rc).decode()
    assert str(vb.NOALLOC_MAX_FRAMES + 1) in v.L.vcrypt_last_cuda_error(v._p).decode()
    rc = v.L.vcrypt_npcr_uaci_device_noalloc(v._p, fake, fake, 1, out.ctypes.data, out.ctypes.data, 0)
    assert rc == vb.E_CUDA  # within the limit, but this context has no GPU
