"""GPU parity (run with -m gpu on the B200 box): the CUDA path, called through the C ABI, against the CPU
oracle, bit for bit (integer / byte work: the bar is exact equality).

Kernel level  : vcrypt_encrypt_device / vcrypt_decrypt_device with random D, B (rows a6-a10, a12) against the
                oracle's literal bit-matrix Algorithms 3-7, over tiled shapes, ragged any-shape cases, special
                distances and in-place calls.
Whole path    : vcrypt_encrypt_frames / vcrypt_decrypt_frames (rows a1-a12) against the oracle's Algorithm 1
                on the BASELINE.json configs, every frame element by element: C1 and C2 in full, and the whole
                clips of C3 (30 frames), C4 (300 frames) and C5 (120 frames of 4K) at full size in bench's launch
                configuration, with every hash compared and the round trip checked on every frame.
"""
import numpy as np
import pytest

from paper_2505_07158_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch

    assert torch.cuda.is_available(), "these tests need the B200"
    return torch


@pytest.fixture(scope="module")
def vb():
    from paper_2505_07158_b200 import binding

    return binding


def gpu_ctx(vb, w, h, n=synth.N_WORKERS, **kw):
    return vb.Vcrypt(synth.KEY, synth.GAMMA, n, w, h, **kw)


def run_device(torch, v, F, D, B, decrypt=False, inplace=False):
    dF = torch.from_numpy(F).cuda()
    dD = torch.from_numpy(D.view(np.int16)).cuda()
    dB = torch.from_numpy(B).cuda()
    dO = dF if inplace else torch.empty_like(dF)
    (v.decrypt_device if decrypt else v.encrypt_device)(dF, dD, dB, dO)
    torch.cuda.synchronize()
    return dO.cpu().numpy()


def rnd_case(w, h, nf, seed, dmode="random"):
    rng = np.random.default_rng(seed)
    F = rng.integers(0, 256, (nf, h, w, 3), dtype=np.uint8)
    B = rng.integers(0, 256, (nf, h, w, 3), dtype=np.uint8)
    nD = 3 * (h + w)
    if dmode == "random":
        D = rng.integers(0, 65536, (nf, nD), dtype=np.uint16)
    elif dmode == "zero":
        D = np.zeros((nf, nD), np.uint16)
    elif dmode == "max":
        D = np.full((nf, nD), 65535, np.uint16)
    elif dmode == "bytes":  # horizontal distances multiples of 8: pure byte rolls
        D = (rng.integers(0, 8192, (nf, nD)) * 8).astype(np.uint16)
    elif dmode == "wrap":  # distances at the modulus boundaries
        D = rng.choice(np.array([0, 1, 7, 8, 8 * w - 1, 8 * w, 8 * w + 1, h - 1, h, h + 1, 31, 32, 33], np.int64) % 65536,
                       (nf, nD)).astype(np.uint16)
    return F, D, B


def oracle_frames(orc, F, D, B, inverse=False):
    return np.stack([orc.confuse_xor(F[k], D[k], B[k], inverse=inverse) for k in range(F.shape[0])])


# shapes on the tiled path (w % 16 == 0, w >= 64, h % 4 == 0, h >= 16): several column strips, a ragged last strip
# (3w % 64 != 0: TMA out-of-bounds columns), h % 8 == 4 (half row group at the bottom), h not a multiple of the TMA
# tile height, a single 4-row block per CTA, more quads than compute threads (w = 2048); and w % 16 == 0 shapes
# that fall back to the any-shape kernels (w < 64 or h % 4 != 0)
TILED = [(256, 256, 1), (64, 48, 3), (80, 32, 2), (112, 20, 3), (1008, 36, 1), (64, 16, 5), (2048, 24, 1), (144, 1028, 1),
         (640, 480, 2), (16, 1, 2), (16, 5, 1), (48, 33, 2), (80, 7, 4), (1008, 19, 1)]
# shapes only the any-shape kernels take
RAGGED = [(1, 1, 1), (1, 7, 2), (5, 1, 1), (17, 9, 3), (33, 20, 2), (100, 37, 1), (15, 64, 1), (250, 3, 2)]


@pytest.mark.parametrize("w,h,nf", TILED + RAGGED)
@pytest.mark.parametrize("dmode", ["random", "wrap"])
def test_kernels_match_oracle(torch_cuda, vb, orc, w, h, nf, dmode):
    F, D, B = rnd_case(w, h, nf, seed=w * 131 + h * 7 + nf, dmode=dmode)
    v = gpu_ctx(vb, w, h)
    E = run_device(torch_cuda, v, F, D, B)
    assert np.array_equal(E, oracle_frames(orc, F, D, B))
    assert v.launch_count()[0] >= 1
    P = run_device(torch_cuda, v, E, D, B, decrypt=True)
    assert np.array_equal(P, oracle_frames(orc, E, D, B, inverse=True))
    assert np.array_equal(P, F)


@pytest.mark.parametrize("dmode", ["zero", "max", "bytes"])
@pytest.mark.parametrize("w,h", [(64, 48), (17, 9), (256, 64)])
def test_special_distances(torch_cuda, vb, orc, w, h, dmode):
    F, D, B = rnd_case(w, h, 2, seed=5, dmode=dmode)
    v = gpu_ctx(vb, w, h)
    E = run_device(torch_cuda, v, F, D, B)
    assert np.array_equal(E, oracle_frames(orc, F, D, B))
    if dmode == "zero":
        assert np.array_equal(E, F ^ B)  # identity confusion: Algorithm 6 alone
    assert np.array_equal(run_device(torch_cuda, v, E, D, B, decrypt=True), F)


@pytest.mark.parametrize("w,h,nf", [(64, 48, 3), (256, 256, 2), (17, 9, 2)])
@pytest.mark.parametrize("generic", [False, True])
def test_in_place_and_forced_generic(torch_cuda, vb, orc, w, h, nf, generic):
    F, D, B = rnd_case(w, h, nf, seed=11)
    v = gpu_ctx(vb, w, h, flags=vb.FLAG_FORCE_GENERIC if generic else 0)
    ref = oracle_frames(orc, F, D, B)
    assert np.array_equal(run_device(torch_cuda, v, F, D, B), ref)
    assert np.array_equal(run_device(torch_cuda, v, F, D, B, inplace=True), ref)
    assert np.array_equal(run_device(torch_cuda, v, ref, D, B, decrypt=True, inplace=True), F)


# Row pass variants: the default plan takes the register-landing row pass (256 threads up to w = 1024, 512 threads up to 2048, 512
# threads with two items per thread up to 4096; the inverse direction too, except for frames 1537 to 2048 pixels wide) and the
# TMA-staged one beyond;
# VCRYPT_FLAG_ROW_TMA keeps the TMA-staged row pass at every width.  Widths on both sides of every boundary, widths whose items do
# not fill the last warp, several blocks per CTA (nf * h / 4 above the resident CTAs), in place.
@pytest.mark.parametrize("w,h,nf", [(64, 16, 2), (1024, 16, 2), (1040, 20, 1), (1536, 16, 2), (1552, 16, 2), (2048, 16, 2), (2064, 20, 2), (3840, 16, 1), (4096, 16, 1),
                                    (4112, 16, 1), (640, 480, 12), (1920, 64, 40)])
@pytest.mark.parametrize("row_tma", [False, True])
def test_row_pass_variants_match_oracle(torch_cuda, vb, orc, w, h, nf, row_tma):
    F, D, B = rnd_case(w, h, nf, seed=w + 3 * h + nf)
    v = gpu_ctx(vb, w, h, flags=vb.FLAG_ROW_TMA if row_tma else 0)
    ref = oracle_frames(orc, F, D, B)
    assert np.array_equal(run_device(torch_cuda, v, F, D, B), ref)
    assert np.array_equal(run_device(torch_cuda, v, F, D, B, inplace=True), ref)
    assert np.array_equal(run_device(torch_cuda, v, ref, D, B, decrypt=True), F)
    assert np.array_equal(run_device(torch_cuda, v, ref, D, B, decrypt=True, inplace=True), F)


@pytest.mark.parametrize("w,h,nf", [(256, 256, 1), (64, 48, 3), (112, 20, 3), (64, 16, 5), (2048, 24, 1), (144, 1028, 1), (640, 480, 7),
                                    (64, 48, 40), (720, 480, 2), (1920, 1080, 3)])
@pytest.mark.parametrize("tune", [(0, 0, 0, 0), (1, 1, 1, 3), (2, 7, 2, 1)])
def test_persistent_kernel_matches_oracle(torch_cuda, vb, orc, w, h, nf, tune):
    """VCRYPT_FLAG_PERSISTENT: the whole call as ONE persistent kernel (row team + strip team per SM, work by ticket, per-frame
    counters between the passes; cipher.cu) -- the same bytes as the oracle in both directions and in place, whatever the
    tuning (row stages, blocks per ticket, window, keystream ring), over strips with a ragged end, a half row group at the
    bottom, more frames than the window, and 40 frames of a tiny shape (many tickets per CTA)."""
    F, D, B = rnd_case(w, h, nf, seed=w + h + nf)
    v = gpu_ctx(vb, w, h, flags=vb.FLAG_PERSISTENT, tune=tune)
    want = oracle_frames(orc, F, D, B)
    E = run_device(torch_cuda, v, F, D, B)
    assert v.launch_count()[0] == 1
    assert np.array_equal(E, want)
    assert np.array_equal(run_device(torch_cuda, v, E, D, B, decrypt=True), F)
    assert np.array_equal(run_device(torch_cuda, v, F, D, B, inplace=True), want)
    assert np.array_equal(run_device(torch_cuda, v, want, D, B, decrypt=True, inplace=True), F)
    # the launch state is left clean: the same context again, other data
    F2, D2, B2 = rnd_case(w, h, nf, seed=w + h + nf + 1)
    assert np.array_equal(run_device(torch_cuda, v, F2, D2, B2), oracle_frames(orc, F2, D2, B2))


def test_persistent_kernel_4k_narrow_strips(torch_cuda, vb, orc):
    """At 3840 x 2160 a 64-byte strip leaves no room for the row team: the persistent kernel takes 32-byte strips (eight
    sub-warps per warp), one row stage, no keystream ring.  Two frames against the oracle, and back."""
    w, h, nf = 3840, 2160, 2
    F, D, B = rnd_case(w, h, nf, seed=99)
    v = gpu_ctx(vb, w, h, flags=vb.FLAG_PERSISTENT)
    E = run_device(torch_cuda, v, F, D, B)
    assert v.launch_count()[0] == 1
    for k in range(nf):
        assert np.array_equal(E[k], orc.confuse_xor(F[k], D[k], B[k])), k
    assert np.array_equal(run_device(torch_cuda, v, E, D, B, decrypt=True), F)


def test_persistent_kernel_whole_path(vb, orc):
    """vcrypt_encrypt_frames / vcrypt_decrypt_frames with VCRYPT_FLAG_PERSISTENT on config 2 (batches over the slots' streams,
    one launch state per stream): every frame against the oracle."""
    cfg = synth.CONFIGS["C2"]
    frames = synth.video(cfg)
    enc = gpu_ctx(vb, cfg.w, cfg.h, batch=5, n_streams=3, flags=vb.FLAG_PERSISTENT)
    C, Hs = enc.encrypt_frames(frames)
    Co, Ho = oracle_clip(orc, "C2", cfg.frames)
    assert np.array_equal(C, Co) and np.array_equal(Hs, Ho)
    dec = gpu_ctx(vb, cfg.w, cfg.h, batch=7, n_streams=2, flags=vb.FLAG_PERSISTENT)
    assert np.array_equal(dec.decrypt_frames(C, Hs), frames)


# NEXT-4: the other resolutions of the paper's Tab. VIII: 360 x 240 takes the any-shape
# kernels (w % 16 != 0), the others the tiled path (720 x 480 and 1280 x 720 with a ragged last column strip)
@pytest.mark.parametrize("w,h", [(320, 240), (360, 240), (640, 360), (720, 480), (1280, 720)])
def test_table_viii_resolutions(torch_cuda, vb, orc, w, h):
    F, D, B = rnd_case(w, h, 2, seed=w + h)
    v = gpu_ctx(vb, w, h)
    E = run_device(torch_cuda, v, F, D, B)
    assert np.array_equal(E[0], orc.confuse_xor(F[0], D[0], B[0]))
    assert np.array_equal(E[1], orc.confuse_xor(F[1], D[1], B[1]))
    assert np.array_equal(run_device(torch_cuda, v, E, D, B, decrypt=True), F)


@pytest.mark.parametrize("w,h", [(640, 480), (100, 37)])
def test_error_locality_without_diffusion(torch_cuda, vb, w, h):
    """NEXT-4 / pin P10 on the GPU path (cropping and channel noise do not spread): a corrupted
    ciphertext byte changes at most 2 plaintext bytes, in the same channel, horizontally adjacent (mod w); a cropped
    rectangle of the ciphertext damages at most that many bytes + one neighbour each."""
    F, D, B = rnd_case(w, h, 1, seed=3)
    v = gpu_ctx(vb, w, h)
    E = run_device(torch_cuda, v, F, D, B)
    rng = np.random.default_rng(9)
    for _ in range(8):
        i, j, c = int(rng.integers(0, h)), int(rng.integers(0, w)), int(rng.integers(0, 3))
        E2 = E.copy()
        E2[0, i, j, c] ^= np.uint8(1 + rng.integers(0, 255))
        P = run_device(torch_cuda, v, E2, D, B, decrypt=True)
        diff = np.argwhere(P[0] != F[0])
        assert 1 <= len(diff) <= 2
        assert set(diff[:, 2]) == {diff[0, 2]} and len(set(diff[:, 0])) == 1
        if len(diff) == 2:
            assert (diff[1, 1] - diff[0, 1]) % w in (1, w - 1)
    E3 = E.copy()
    E3[0, 5:15, 10:30, :] = 0  # cropping attack (Fig. 8): 10 x 20 pixels blanked
    P = run_device(torch_cuda, v, E3, D, B, decrypt=True)
    assert 0 < np.count_nonzero(P[0] != F[0]) <= 2 * 10 * 20 * 3


def test_many_frames_per_call_split_into_l2_sized_launches(torch_cuda, vb, orc):
    """More frames than one L2-resident launch holds: the call splits, results unchanged."""
    w, h, nf = 640, 480, 120  # 110.6 MB of frames: two launch pairs (113 + 7 frames)
    F, D, B = rnd_case(w, h, nf, seed=21)
    v = gpu_ctx(vb, w, h, pipe_streams=1)  # every launch on the caller's stream
    E = run_device(torch_cuda, v, F, D, B)
    assert v.launch_count()[0] == 4
    for k in (0, 1, 37, 112, 113, 114, 119):
        assert np.array_equal(E[k], orc.confuse_xor(F[k], D[k], B[k])), k
    assert np.array_equal(run_device(torch_cuda, v, E, D, B, decrypt=True), F)


@pytest.mark.parametrize("w,h,nf,pf,ps", [(64, 48, 11, 2, 2), (80, 32, 13, 3, 3), (256, 256, 9, 1, 4), (112, 20, 17, 4, 2),
                                          (64, 16, 14, 3, 9)])
def test_resident_clip_schedule_over_streams(torch_cuda, vb, orc, w, h, nf, pf, ps):
    """A call that brings >= 4 * pipe_frames frames alternates its launch pairs over pipe_streams streams (forked from and
    joined into the caller's stream): balanced pairs with a ragged count, every frame bit-exact, both directions, in place
    too, and ordered with respect to the caller's stream (the very next operation on it reads the result)."""
    F, D, B = rnd_case(w, h, nf, seed=31 + nf)
    want = oracle_frames(orc, F, D, B)
    v = gpu_ctx(vb, w, h, pipe_frames=pf, pipe_streams=ps)
    E = run_device(torch_cuda, v, F, D, B)
    npairs = -(-nf // pf)
    assert v.launch_count()[0] == 2 * npairs
    assert np.array_equal(E, want)
    assert np.array_equal(run_device(torch_cuda, v, F, D, B, inplace=True), want)
    assert np.array_equal(run_device(torch_cuda, v, E, D, B, decrypt=True), F)
    # stream order: on a side stream, the copy enqueued right after the call must see the finished ciphertext
    torch = torch_cuda
    dF, dB = torch.from_numpy(F).cuda(), torch.from_numpy(B).cuda()
    dD = torch.from_numpy(D.view(np.int16)).cuda()
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        for _ in range(3):
            dE = torch.zeros_like(dF)
            v.encrypt_device(dF, dD, dB, dE, side.cuda_stream)
            host = torch.empty(dE.shape, dtype=dE.dtype).pin_memory()
            host.copy_(dE, non_blocking=True)
            side.synchronize()
            assert np.array_equal(host.numpy(), want)
    # a single-stream context gives the same bytes
    v1 = gpu_ctx(vb, w, h, pipe_streams=1)
    assert np.array_equal(run_device(torch_cuda, v1, F, D, B), want)


def test_resident_clip_schedule_under_stream_capture(torch_cuda, vb, orc):
    """The fork / join over the internal stream is a legal capture pattern: the call is recorded into a CUDA graph and the
    replays (on new inputs in the same buffers) are bit-exact."""
    torch = torch_cuda
    w, h, nf = 64, 48, 12
    v = gpu_ctx(vb, w, h, pipe_frames=3, pipe_streams=2)
    F, D, B = rnd_case(w, h, nf, seed=77)
    dF, dB = torch.from_numpy(F).cuda(), torch.from_numpy(B).cuda()
    dD = torch.from_numpy(D.view(np.int16)).cuda()
    dE = torch.zeros_like(dF)
    v.encrypt_device(dF, dD, dB, dE)  # warm-up outside the capture: creates the internal stream and events
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        v.encrypt_device(dF, dD, dB, dE, torch.cuda.current_stream().cuda_stream)
    for seed in (78, 79):
        F2, D2, B2 = rnd_case(w, h, nf, seed=seed)
        dF.copy_(torch.from_numpy(F2))
        dB.copy_(torch.from_numpy(B2))
        dD.copy_(torch.from_numpy(D2.view(np.int16)))
        dE.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert np.array_equal(dE.cpu().numpy(), oracle_frames(orc, F2, D2, B2)), seed


def test_resident_clip_schedule_defaults(torch_cuda, vb, orc):
    """Default pipe_frames (about 31 MB of frames per launch pair when encrypting): 640 x 480 -> 35 frames; 160 frames >= 4 x 35
    = 5 pairs of 32, while 120 frames stay on the caller's stream (test_many_frames_per_call... covers the split by L2 budget)."""
    w, h, nf = 640, 480, 160
    F, D, B = rnd_case(w, h, nf, seed=22)
    v = gpu_ctx(vb, w, h)
    E = run_device(torch_cuda, v, F, D, B)
    assert v.launch_count()[0] == 10
    for k in (0, 31, 32, 63, 64, 95, 96, 127, 128, 159):
        assert np.array_equal(E[k], orc.confuse_xor(F[k], D[k], B[k])), k
    assert np.array_equal(run_device(torch_cuda, v, E, D, B, decrypt=True), F)
    E2 = run_device(torch_cuda, v, F[:120], D[:120], B[:120])
    assert v.launch_count()[0] == 4 and np.array_equal(E2, E[:120])


@pytest.mark.parametrize("w,h,nf", [(640, 480, 6), (1920, 1080, 3), (64, 48, 9), (100, 37, 3)])
def test_calls_chained_on_one_stream_without_host_sync(torch_cuda, vb, orc, w, h, nf):
    """Every kernel of the library starts under programmatic dependent launch: a call's first kernel may be scheduled while the
    last kernel of the call before it (which lets its dependents launch early) is still running.  Producer -> consumer chains on one
    stream with no host synchronisation in between: the inputs D and B written by device copies right before the call, encrypt ->
    decrypt -> encrypt in place on the same buffers, repeated; the result must be what the oracle gives for the last inputs."""
    torch = torch_cuda
    F, D, B = rnd_case(w, h, nf, seed=77)
    F2, D2, B2 = rnd_case(w, h, nf, seed=78)
    v = gpu_ctx(vb, w, h)
    src = [torch.from_numpy(a).cuda() for a in (F, D.view(np.int16), B)]
    src2 = [torch.from_numpy(a).cuda() for a in (F2, D2.view(np.int16), B2)]
    dF, dD, dB = (torch.empty_like(t) for t in src)
    dE, dP = torch.empty_like(dF), torch.empty_like(dF)
    torch.cuda.synchronize()
    for rep in range(6):
        cur = src if rep % 2 == 0 else src2
        dF.copy_(cur[0]); dD.copy_(cur[1]); dB.copy_(cur[2])  # producers of every input, same stream, no sync
        v.encrypt_device(dF, dD, dB, dE)
        v.decrypt_device(dE, dD, dB, dP)                       # consumes the ciphertext the call before produced
        v.encrypt_device(dP, dD, dB, dP)                       # ... and its plaintext, in place
    torch.cuda.synchronize()
    want = oracle_frames(orc, F2, D2, B2)
    assert np.array_equal(dE.cpu().numpy(), want)
    assert np.array_equal(dP.cpu().numpy(), want)


def test_two_live_contexts_of_different_shapes(torch_cuda, vb, orc):
    """The opt-in shared-memory limit of a kernel is state of the FUNCTION in the whole process, not of a context: a large
    shape's context must keep working after a smaller shape's context (same kernel instantiations, smaller strips and rings)
    has been created later, in every order and for every kernel family (kernel pairs, TMA-staged row pass, persistent)."""
    shapes = [(1920, 1080), (640, 480), (1280, 720)]
    cases = {wh: rnd_case(wh[0], wh[1], 2, seed=sum(wh)) for wh in shapes}
    want = {wh: oracle_frames(orc, *cases[wh]) for wh in shapes}
    for flags in (0, vb.FLAG_ROW_TMA, vb.FLAG_PERSISTENT):
        big = gpu_ctx(vb, 1920, 1080, flags=flags)
        assert np.array_equal(run_device(torch_cuda, big, *cases[(1920, 1080)]), want[(1920, 1080)])
        small = gpu_ctx(vb, 640, 480, flags=flags)   # created AFTER the large one: must not lower its limits
        mid = gpu_ctx(vb, 1280, 720, flags=flags)
        for _ in range(2):
            for v, wh in ((big, (1920, 1080)), (small, (640, 480)), (mid, (1280, 720)), (big, (1920, 1080))):
                E = run_device(torch_cuda, v, *cases[wh])
                assert np.array_equal(E, want[wh]), (flags, wh)
                assert np.array_equal(run_device(torch_cuda, v, E, cases[wh][1], cases[wh][2], decrypt=True), cases[wh][0]), (flags, wh)


def test_persistent_kernel_first_launch_on_a_non_blocking_stream(torch_cuda, vb, orc):
    """The persistent kernel's launch state is zeroed once per context; that must have happened before the first launch also
    when the launch goes to a stream that does not synchronise with the default stream and nothing else precedes it there."""
    torch = torch_cuda
    w, h, nf = 640, 480, 6
    F, D, B = rnd_case(w, h, nf, seed=4242)
    dF, dD, dB = torch.from_numpy(F).cuda(), torch.from_numpy(D.view(np.int16)).cuda(), torch.from_numpy(B).cuda()
    dE = torch.empty_like(dF)
    want = oracle_frames(orc, F, D, B)
    for _ in range(3):  # a fresh context each time: its very first GPU work is the kernel on the side stream
        st = torch.cuda.Stream()  # torch's streams are created non-blocking
        torch.cuda.synchronize()
        v = gpu_ctx(vb, w, h, flags=vb.FLAG_PERSISTENT)
        v.encrypt_device(dF, dD, dB, dE, st.cuda_stream)
        st.synchronize()
        assert np.array_equal(dE.cpu().numpy(), want)


def test_device_call_argument_errors(torch_cuda, vb):
    torch = torch_cuda
    v = gpu_ctx(vb, 64, 48)
    F, D, B = rnd_case(64, 48, 2, seed=1)
    dF, dD, dB = torch.from_numpy(F).cuda(), torch.from_numpy(D.view(np.int16)).cuda(), torch.from_numpy(B).cuda()
    L = v.L
    st = torch.cuda.current_stream().cuda_stream
    assert L.vcrypt_encrypt_device(v._p, None, dD.data_ptr(), dB.data_ptr(), 2, dF.data_ptr(), st) == vb.E_ARG
    assert L.vcrypt_encrypt_device(v._p, dF.data_ptr() + 1, dD.data_ptr(), dB.data_ptr(), 1, dF.data_ptr(), st) == vb.E_ARG
    # partial overlap of input and output
    assert L.vcrypt_encrypt_device(v._p, dF.data_ptr(), dD.data_ptr(), dB.data_ptr(), 2, dF.data_ptr() + 64 * 48 * 3, st) == vb.E_ARG
    assert L.vcrypt_encrypt_device(v._p, dF.data_ptr(), dD.data_ptr(), dB.data_ptr(), 0, dF.data_ptr(), st) == vb.OK


@pytest.mark.parametrize("cfgname,nf,pairs_enc,pairs_dec", [("C4", 30, 6, 6), ("C5", 8, 8, 8)])
def test_full_size_resident_clip_as_bench_times_it(torch_cuda, vb, orc, cfgname, nf, pairs_enc, pairs_dec):
    """The launch configuration bench.py's kernel leg times -- ONE *_device call on a resident clip with the default schedule
    (FHD: launch pairs of 5 frames; 4K: 1) -- at full frame size, every frame
    against the oracle and through the inverse."""
    torch = torch_cuda
    cfg = synth.CONFIGS[cfgname]
    w, h = cfg.w, cfg.h
    F, D, B = rnd_case(w, h, nf, seed=41)
    v = gpu_ctx(vb, w, h)
    dF, dB = torch.from_numpy(F).cuda(), torch.from_numpy(B).cuda()
    dD = torch.from_numpy(D.view(np.int16)).cuda()
    dE = torch.empty_like(dF)
    v.encrypt_device(dF, dD, dB, dE)
    torch.cuda.synchronize()
    assert v.launch_count()[0] == 2 * pairs_enc
    E = dE.cpu().numpy()
    for k in range(nf):  # every frame against the oracle
        assert np.array_equal(E[k], orc.confuse_xor(F[k], D[k], B[k])), k
    dP = torch.empty_like(dF)
    v.decrypt_device(dE, dD, dB, dP)
    torch.cuda.synchronize()
    assert v.launch_count()[0] == 2 * pairs_dec
    assert bool(torch.equal(dP, dF))
    # the same call repeated in place gives the same bytes (no dependence on what the streams did before)
    dG = dF.clone()
    v.encrypt_device(dG, dD, dB, dG)
    torch.cuda.synchronize()
    assert bool(torch.equal(dG, dE))


# ------------------------------------------------------------------------------------------------------
# whole path
# ------------------------------------------------------------------------------------------------------
def test_config1_full(vb, orc):
    cfg = synth.CONFIGS["C1"]
    frames = synth.video(cfg)
    assert synth.digest(frames) == synth.digest(synth.video(cfg))  # generator is deterministic
    enc = gpu_ctx(vb, cfg.w, cfg.h, batch=cfg.batch)
    C, Hs = enc.encrypt_frames(frames)
    oc = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h)
    Co, Ho = oc.encrypt_frames(frames)
    assert np.array_equal(Hs, Ho)
    assert np.array_equal(C, Co)
    dec = gpu_ctx(vb, cfg.w, cfg.h, batch=cfg.batch)
    assert np.array_equal(dec.decrypt_frames(C, Hs), frames)


def test_config2_full(vb, orc):
    cfg = synth.CONFIGS["C2"]
    frames = synth.video(cfg)
    enc = gpu_ctx(vb, cfg.w, cfg.h, batch=cfg.batch, n_streams=cfg.n_streams)
    C, Hs = enc.encrypt_frames(frames)
    oc = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h)
    Co, Ho = oc.encrypt_frames(frames)
    assert np.array_equal(Hs, Ho)
    assert np.array_equal(C, Co)
    od = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h)
    dec = gpu_ctx(vb, cfg.w, cfg.h, batch=5, n_streams=2)  # another pipeline shape: results must not change
    P = dec.decrypt_frames(C, Hs)
    assert np.array_equal(P, od.decrypt_frames(Co, Ho))
    assert np.array_equal(P, frames)


def full_parity(vb, orc, cfg, nframes, pinned, chunk_batches=3):
    """Full-size config in bench's launch configuration (batches of cfg.batch frames over cfg.n_streams streams): every hash
    and every frame's ciphertext element by element against the oracle (its D, B follow the whole chain), round trip on every
    frame.  The clip is streamed through in chunks of chunk_batches batches -- drawn, encrypted (the context carries the chain
    from call to call), checked, decrypted, dropped -- so host memory stays bounded at 4K; the oracle's per-frame work (hash,
    literal bit-matrix confusion) runs on a few host threads, its chain step stays serial."""
    import os
    from concurrent.futures import ThreadPoolExecutor

    import torch

    chunk = chunk_batches * cfg.batch
    shape = (chunk, cfg.h, cfg.w, 3)
    if pinned:
        tin, tout, tpl = (torch.empty(shape, dtype=torch.uint8).pin_memory() for _ in range(3))
        fin, C, P = tin.numpy(), tout.numpy(), tpl.numpy()
    else:
        fin, C, P = (np.empty(shape, np.uint8) for _ in range(3))
    Hs = np.empty((chunk, 32), np.uint8)
    enc = gpu_ctx(vb, cfg.w, cfg.h, batch=cfg.batch, n_streams=cfg.n_streams)
    dec = gpu_ctx(vb, cfg.w, cfg.h, batch=cfg.batch, n_streams=cfg.n_streams)
    oc = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h)
    frames = synth.frame_iter(cfg, nframes)
    done = 0
    with ThreadPoolExecutor(max(1, min(8, (os.cpu_count() or 2) - 1))) as pool:
        while done < nframes:
            m = min(chunk, nframes - done)
            for k in range(m):
                fin[k] = next(frames)
            enc.encrypt_frames(fin[:m], C[:m], Hs[:m])
            want_H = list(pool.map(lambda k: orc.frame_hash(fin[k], synth.N_WORKERS), range(m)))
            DB = []
            for k in range(m):
                assert want_H[k] == Hs[k].tobytes(), done + k
                DB.append(oc.derive(want_H[k]))
            same = list(pool.map(lambda k: bool(np.array_equal(C[k], orc.confuse_xor(fin[k], *DB[k]))), range(m)))
            assert all(same), [done + k for k in range(m) if not same[k]]
            dec.decrypt_frames(C[:m], Hs[:m], P[:m])
            assert np.array_equal(P[:m], fin[:m]), done
            done += m
    assert done == nframes
    return enc


def test_config3_fhd_batch1(vb, orc):
    cfg = synth.CONFIGS["C3"]
    full_parity(vb, orc, cfg, cfg.frames, pinned=False)  # all 30 frames


def test_config4_fhd_batches_of_8_three_streams(vb, orc):
    """Long test (about a minute): the WHOLE clip of config 4, all 300 frames against the oracle."""
    cfg = synth.CONFIGS["C4"]
    enc = full_parity(vb, orc, cfg, cfg.frames, pinned=True)
    assert cfg.frames == 300 and enc.launch_count()[1] >= 2 * 38  # 37 full batches + 4 frames, a launch pair each


def test_config5_4k(vb, orc):
    """Long test (about two minutes): the WHOLE clip of config 5, all 120 frames of 3840 x 2160 against the oracle."""
    cfg = synth.CONFIGS["C5"]
    full_parity(vb, orc, cfg, cfg.frames, pinned=True)
    assert cfg.frames == 120


def test_config4_one_bit_pairs_npcr_uaci(vb, torch_cuda):
    """Pin P7 on the GPU path, config 4's 100 pairs: one flipped plaintext bit -> NPCR ~ 255/256, UACI ~
    (256^2-1)/(3*256*255) (Eq. 14-16; closed forms for independent uniform ciphertexts), over all
    three channels and per channel; every pair within 5 sigma, the mean within 3 sigma / sqrt(pairs)."""
    torch = torch_cuda
    cfg = synth.CONFIGS["C4"]
    pairs = 100
    npcr, uaci, npcr_c, uaci_c = [], [], [], []
    for f, g, _ in synth.one_bit_pairs(cfg, pairs):
        c1, _ = gpu_ctx(vb, cfg.w, cfg.h, batch=1, n_streams=1, host_threads=8).encrypt_frames(f[None])
        c2, _ = gpu_ctx(vb, cfg.w, cfg.h, batch=1, n_streams=1, host_threads=8).encrypt_frames(g[None])
        a = torch.from_numpy(c1[0]).cuda().to(torch.int16)
        b = torch.from_numpy(c2[0]).cuda().to(torch.int16)
        ne = (a != b).to(torch.float64)
        ad = (a - b).abs().to(torch.float64)
        npcr.append(100.0 * float(ne.mean()))
        uaci.append(100.0 * float(ad.mean()) / 255.0)
        npcr_c.append([100.0 * float(ne[..., c].mean()) for c in range(3)])
        uaci_c.append([100.0 * float(ad[..., c].mean()) / 255.0 for c in range(3)])
    n = 3 * cfg.w * cfg.h
    e_npcr, e_uaci = 100.0 * 255 / 256, 100.0 * (256 ** 2 - 1) / (3 * 256 * 255)
    s_npcr = 100.0 * np.sqrt((255 / 256) * (1 / 256) / n)
    # |a - b| / 255 for independent uniform bytes: E = (256^2-1)/(3*256*255), E[d^2] = (256^2-1)/6
    var_d = (256 ** 2 - 1) / 6.0 - ((256 ** 2 - 1) / (3 * 256.0)) ** 2
    s_uaci = 100.0 * np.sqrt(var_d / n) / 255.0
    assert all(abs(x - e_npcr) < 5 * s_npcr for x in npcr), npcr
    assert all(abs(x - e_uaci) < 5 * s_uaci for x in uaci), uaci
    assert abs(np.mean(npcr) - e_npcr) < 3 * s_npcr / np.sqrt(pairs)
    assert abs(np.mean(uaci) - e_uaci) < 3 * s_uaci / np.sqrt(pairs)
    s3 = np.sqrt(3.0)  # a channel has a third of the bytes
    assert all(abs(x - e_npcr) < 5 * s_npcr * s3 for row in npcr_c for x in row)
    assert all(abs(x - e_uaci) < 5 * s_uaci * s3 for row in uaci_c for x in row)


@pytest.mark.parametrize("w,h,n", [(64, 48, 32), (64, 48, 1), (17, 9, 3), (80, 32, 7), (256, 256, 32), (33, 5, 8), (640, 480, 6)])
def test_device_derivation_matches_oracle(torch_cuda, vb, orc, w, h, n):
    """NEXT-1: the worker systems on the GPU give the oracle's D and B bit for bit (fp64 RK4 without FMA
    contraction), over ragged worker slices (n not dividing h or 3(h+w), empty bands when n > h), and keep the chain in
    step with the host derivation."""
    torch = torch_cuda
    v = gpu_ctx(vb, w, h, n=n)
    vh = gpu_ctx(vb, w, h, n=n)
    oc = orc.ctx(synth.KEY, synth.GAMMA, n, w, h)
    dD = torch.zeros(3 * (h + w), dtype=torch.int16, device="cuda")
    dB = torch.zeros((h, w, 3), dtype=torch.uint8, device="cuda")
    rng = np.random.default_rng(w + h + n)
    for _ in range(3):  # three chained frames
        H = rng.integers(0, 256, 32, dtype=np.uint8).tobytes()
        D_or, B_or = oc.derive(H)
        v.derive_device(H, dD, dB)
        assert np.array_equal(dD.cpu().numpy().view(np.uint16), D_or)
        assert np.array_equal(dB.cpu().numpy(), B_or)
        vh.derive(H)
        assert np.array_equal(v.get_state()[0], vh.get_state()[0]) and v.get_state()[1] == vh.get_state()[1]


@pytest.mark.parametrize("w,h,n,nf", [(64, 48, 32, 3), (64, 48, 1, 2), (16, 5, 8, 2), (80, 33, 7, 2), (256, 256, 32, 1), (640, 480, 6, 2),
                                      (1920, 1080, 32, 2)])
def test_device_hashing_matches_oracle(torch_cuda, vb, orc, w, h, n, nf):
    """NEXT-2: H = xor of the band SHA-256 digests computed on the GPU equals the oracle's (and hashlib's for
    n = 1), over bands of unequal height, empty bands (n > h), tails of 0 / 16 / 32 / 48 bytes."""
    import hashlib

    torch = torch_cuda
    F = synth.random_frames(w, h, nf, seed=w + h + n)
    v = gpu_ctx(vb, w, h, n=n)
    Hs = v.frame_hash_device(torch.from_numpy(F).cuda())
    for k in range(nf):
        assert Hs[k].tobytes() == orc.frame_hash(F[k], n), k
        assert Hs[k].tobytes() == v.frame_hash(F[k])
        if n == 1:
            assert Hs[k].tobytes() == hashlib.sha256(F[k].tobytes()).digest()


def test_device_hashing_rejects_unaligned_rows(torch_cuda, vb):
    torch = torch_cuda
    v = gpu_ctx(vb, 17, 9, n=3)
    F = torch.zeros((1, 9, 17, 3), dtype=torch.uint8, device="cuda")
    out = np.empty((1, 32), np.uint8)
    assert v.L.vcrypt_frame_hash_device(v._p, F.data_ptr(), 1, out.ctypes.data, 0) == vb.E_SHAPE


_oracle_clips = {}


def oracle_clip(orc, cfgname, nframes):
    """The oracle's ciphertext and hashes of the first frames of a config's clip (computed once per module run)."""
    key = (cfgname, nframes)
    if key not in _oracle_clips:
        cfg = synth.CONFIGS[cfgname]
        _oracle_clips[key] = orc.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h).encrypt_frames(synth.video(cfg, nframes))
    return _oracle_clips[key]


@pytest.mark.parametrize("flags", ["derive", "hash", "both"])
@pytest.mark.parametrize("cfgname,nframes", [("C1", 1), ("C2", 24), ("C4", 20)])
def test_whole_path_with_device_derivation(vb, orc, cfgname, nframes, flags):
    """vcrypt_encrypt_frames / vcrypt_decrypt_frames with VCRYPT_FLAG_DEVICE_DERIVE and / or VCRYPT_FLAG_DEVICE_HASH
    (two-stage pipeline, hashing running ahead): same ciphertext, hashes and plaintext."""
    cfg = synth.CONFIGS[cfgname]
    frames = synth.video(cfg, nframes)
    fl = {"derive": vb.FLAG_DEVICE_DERIVE, "hash": vb.FLAG_DEVICE_HASH, "both": vb.FLAG_DEVICE_DERIVE | vb.FLAG_DEVICE_HASH}[flags]
    enc = gpu_ctx(vb, cfg.w, cfg.h, batch=cfg.batch, n_streams=cfg.n_streams if flags == "derive" else 0, flags=fl)
    C, Hs = enc.encrypt_frames(frames)
    ref = gpu_ctx(vb, cfg.w, cfg.h, batch=cfg.batch, n_streams=cfg.n_streams)
    C2, H2 = ref.encrypt_frames(frames)
    assert np.array_equal(Hs, H2) and np.array_equal(C, C2)
    Co, Ho = oracle_clip(orc, cfgname, nframes)  # every frame against the oracle
    assert np.array_equal(C, Co) and np.array_equal(Hs, Ho)
    dec = gpu_ctx(vb, cfg.w, cfg.h, batch=3, n_streams=2, flags=fl)
    assert np.array_equal(dec.decrypt_frames(C, Hs), frames)
    assert enc.get_state()[1] == nframes and np.array_equal(enc.get_state()[0], ref.get_state()[0])


def test_failed_call_leaves_chain_untouched(vb):
    v = gpu_ctx(vb, 64, 48)
    s0 = v.get_state()
    f = synth.random_frames(64, 48, 2, 1)
    rc = v.L.vcrypt_encrypt_frames(v._p, f.ctypes.data, 2, None, None)
    assert rc == vb.E_ARG
    s1 = v.get_state()
    assert s0[1] == s1[1] and np.array_equal(s0[0], s1[0])
    v.encrypt_frames(f)
    assert v.get_state()[1] == 2
