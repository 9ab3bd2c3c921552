"""CPU-side tests of libvcrypt (no GPU needed): the library loads, exports every symbol include/vcrypt.h
declares, validates its arguments, and its production host derivation (SHA-NI / portable SHA-256, AVX-512 /
AVX2 / scalar LHCS lanes, thread pool) gives the oracle's H, D and B bit for bit.
"""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2505_07158_b200 import binding as vb
from paper_2505_07158_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HO = vb.FLAG_HOST_ONLY


def host_ctx(w, h, n, flags=0, **kw):
    return vb.Vcrypt(synth.KEY, synth.GAMMA, n, w, h, flags=HO | flags, **kw)


def test_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "vcrypt.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = sorted(set(re.findall(r"\b(vcrypt_[a-z_0-9]+)\s*\(", hdr)))
    assert len(names) >= 16, names
    L = vb.lib()
    for nm in names:
        assert hasattr(L, nm), f"{nm} declared in vcrypt.h but not exported"


def test_params_struct_matches_header():
    hdr = open(os.path.join(ROOT, "include", "vcrypt.h")).read()
    body = re.search(r"typedef struct vcrypt_params \{(.*?)\} vcrypt_params;", hdr, re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if decl:
            fields += [f.strip() for f in decl.split(None, 1)[1].split(",")]
    assert fields == [f[0] for f in vb.Params._fields_]


def test_strerror_and_describe():
    L = vb.lib()
    seen = set()
    for code in range(0, -7, -1):
        s = L.vcrypt_strerror(code).decode()
        assert s and s not in seen
        seen.add(s)
    assert "unknown" in L.vcrypt_strerror(-99).decode()
    d = vb.describe()
    for token in ("dt=0.005", "N0=20000", "K_m=16", "u=40"):
        assert token in d


@pytest.mark.parametrize("bad,code", [
    (dict(gamma=-0.05), vb.E_KEY), (dict(gamma=-1.53), vb.E_KEY), (dict(gamma=float("nan")), vb.E_KEY),
    (dict(key=(float("inf"), 1, 1, 1)), vb.E_KEY), (dict(key=(1e300, 1, 1, 1)), vb.E_KEY),
    (dict(n=0), vb.E_SHAPE), (dict(w=0), vb.E_SHAPE), (dict(h=0), vb.E_SHAPE), (dict(w=70000), vb.E_SHAPE),
    (dict(w=32768, h=32768), vb.E_SHAPE),  # 3wh >= 2^31: byte offsets inside a frame are 32-bit in the kernels
    (dict(w=26760, h=26760), vb.E_SHAPE),  # just above 2^31 / 3 pixels
])
def test_init_rejects_bad_parameters(bad, code):
    kw = dict(key=synth.KEY, gamma=synth.GAMMA, n=4, w=16, h=8)
    kw.update(bad)
    with pytest.raises(vb.VcryptError) as ei:
        vb.Vcrypt(kw["key"], kw["gamma"], kw["n"], kw["w"], kw["h"], flags=HO)
    assert ei.value.code == code


def test_null_arguments_and_host_only_gpu_calls():
    L = vb.lib()
    assert L.vcrypt_init(None, None) == vb.E_ARG
    L.vcrypt_destroy(None)  # allowed
    v = host_ctx(16, 8, 2)
    buf = np.zeros(16 * 8 * 3, np.uint8)
    hs = np.zeros(32, np.uint8)
    assert L.vcrypt_frame_hash(v._p, None, hs.ctypes.data) == vb.E_ARG
    assert L.vcrypt_derive(v._p, hs.ctypes.data, None, buf.ctypes.data) == vb.E_ARG
    assert L.vcrypt_encrypt_frames(v._p, None, 1, buf.ctypes.data, hs.ctypes.data) == vb.E_ARG
    # a host-only context has no GPU path and no CPU fallback
    assert L.vcrypt_encrypt_frames(v._p, buf.ctypes.data, 1, buf.ctypes.data, hs.ctypes.data) == vb.E_CUDA
    assert L.vcrypt_decrypt_frames(v._p, buf.ctypes.data, hs.ctypes.data, 1, buf.ctypes.data) == vb.E_CUDA
    assert L.vcrypt_encrypt_device(v._p, C.c_void_p(256), C.c_void_p(256), C.c_void_p(256), 1, C.c_void_p(256), None) == vb.E_CUDA


def test_init_without_gpu_fails_loudly():
    """No CPU fallback: on a box without a CUDA device a normal context cannot be created."""
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(vb.VcryptError) as ei:
        vb.Vcrypt(synth.KEY, synth.GAMMA, 4, 16, 8)
    assert ei.value.code == vb.E_CUDA


SHAPES = [(256, 256, 32), (64, 48, 5), (17, 9, 3), (1, 1, 1), (3, 2, 7), (640, 480, 32), (100, 37, 12), (33, 20, 9)]


@pytest.mark.parametrize("w,h,n", SHAPES)
@pytest.mark.parametrize("flags", [0, vb.FLAG_HOST_SCALAR])
def test_hash_and_derivation_match_oracle(orc, w, h, n, flags):
    """Rows a1-a4: three frames in a row (the chain), every ISA path."""
    v = host_ctx(w, h, n, flags)
    oc = orc.ctx(synth.KEY, synth.GAMMA, n, w, h)
    frames = synth.random_frames(w, h, 3, seed=w * 1000 + h)
    for f in frames:
        H = v.frame_hash(f)
        assert H == orc.frame_hash(f, n)
        D, B = v.derive(H)
        Do, Bo = oc.derive(H)
        assert np.array_equal(D, Do)
        assert np.array_equal(B, Bo)
    s, k = v.get_state()
    assert k == 3 and np.array_equal(s, oc.state)


@pytest.mark.parametrize("flags", [0, vb.FLAG_HOST_SCALAR])
def test_host_derivation_reproduces_frozen_vector(flags):
    """tests/golden/derive_tiny.txt (written from oracle/ alone by tests/golden/make_derive_tiny.py and reproduced by the
    pure-Python restatement in tests/test_oracle_derivation.py): the product's host derivation arrives at the same base
    states, D and B over the two chained frames without the oracle being involved in this test at all."""
    import struct

    from conftest import read_golden

    key = (3.141592653589793, 2.718281828459045, 1.4142135623730951, 1.7320508075688772)
    v = vb.Vcrypt(key, -1.0, 2, 5, 7, flags=HO | flags)
    rows = read_golden("derive_tiny.txt")
    nframes = 0
    for i, row in enumerate(rows):
        if row[0] != "H":
            continue
        S, D, B = rows[i + 1], rows[i + 3], rows[i + 4]
        assert S[0] == "S" and D[0] == "D" and B[0] == "B"
        s, k = v.get_state()
        assert k == nframes and struct.pack("<4d", *s) == struct.pack("<4Q", *[int(x, 16) for x in S[1:]])
        Dv, Bv = v.derive(bytes.fromhex(row[1]))
        assert Dv.tolist() == [int(x, 16) for x in D[1:]]
        assert Bv.tobytes() == bytes.fromhex(B[1])
        nframes += 1
    assert nframes == 2


def test_lane_paths_agree_on_ragged_worker_slices(orc):
    """n that does not divide h or 3(h+w), and n not a multiple of the lane count: padded lanes, ragged tails,
    and the split into single-lane runs when D iteration counts differ inside a lane group."""
    for (w, h, n) in [(40, 30, 13), (24, 50, 11), (7, 5, 9), (50, 13, 16)]:
        outs = []
        for flags in (0, vb.FLAG_HOST_SCALAR):
            v = host_ctx(w, h, n, flags, host_threads=3)
            outs.append(v.derive(bytes(range(32))))
        oc = orc.ctx(synth.KEY, synth.GAMMA, n, w, h)
        Do, Bo = oc.derive(bytes(range(32)))
        for D, B in outs:
            assert np.array_equal(D, Do) and np.array_equal(B, Bo), (w, h, n)


def test_results_do_not_depend_on_thread_count():
    f = synth.random_frames(64, 48, 1, 3)[0]
    ref = None
    for nt in (1, 2, 5, 16):
        v = host_ctx(64, 48, 32, host_threads=nt)
        assert v.host_threads() == nt
        H = v.frame_hash(f)
        D, B = v.derive(H)
        cur = (H, D.tobytes(), B.tobytes())
        ref = ref or cur
        assert cur == ref


def test_state_checkpoint_resume():
    """The chain state (4 doubles + counter) is all a caller needs to resume a stream."""
    a = host_ctx(32, 16, 4)
    hashes = [bytes([i] * 32) for i in range(4)]
    outs = [a.derive(hh) for hh in hashes]
    b = host_ctx(32, 16, 4)
    b.derive(hashes[0]); b.derive(hashes[1])
    s, k = b.get_state()
    c = host_ctx(32, 16, 4)
    c.set_state(s, k)
    for i in (2, 3):
        D, B = c.derive(hashes[i])
        assert np.array_equal(D, outs[i][0]) and np.array_equal(B, outs[i][1])
    assert c.get_state()[1] == 4
    with pytest.raises(vb.VcryptError) as ei:
        c.set_state([float("nan"), 0, 0, 0], 0)
    assert ei.value.code == vb.E_STATE
    with pytest.raises(vb.VcryptError) as ei:  # same bound as the key: |v| < 2^53, so that the integer part stays exact
        c.set_state([2.0 ** 53, 0, 0, 0], 0)
    assert ei.value.code == vb.E_STATE
    c.set_state([2.0 ** 53 - 1, 0, 0, 0], 0)


def test_production_sha256_fips_vectors():
    """The production SHA-256 (not the oracle's) against FIPS 180-4 examples, through vcrypt_frame_hash with
    n = 1 (H = SHA-256(frame), pin P2): messages are frames of 3wh bytes."""
    import hashlib

    for (w, h) in [(1, 1), (21, 1), (64, 1), (1, 37), (40, 40), (333, 3)]:
        for flags in (0, vb.FLAG_HOST_SCALAR):
            v = host_ctx(w, h, 1, flags)
            f = synth.random_frames(w, h, 1, w + h)[0]
            assert v.frame_hash(f) == hashlib.sha256(f.tobytes()).digest()
    # "abc" = one 1x1 RGB pixel (FIPS 180-4 / NIST example B.1)
    v = host_ctx(1, 1, 1)
    assert v.frame_hash(np.frombuffer(b"abc", np.uint8).reshape(1, 1, 3).copy()).hex() == \
        "ba7816bf8f01cfea414140de5dae2223b00361a396177a9cb410ff61f20015ad"
