"""ctypes front-end of the CPU oracle (oracle/vcrypt_oracle.c).

TEST INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py may import this module.
It imports nothing from the product package and the product imports nothing
from here.

Every function is a thin marshalling layer; the arithmetic lives in the C
file, where each function cites the PAPER.md passage it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vcrypt_oracle.c")
# -ffp-contract=off: no FMA contraction, so the RK4 expression order of the C
# source is the arithmetic that runs.
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c99", "-shared", "-fPIC"]


def build(opt: str = "-O2", out: str | None = None, force: bool = False) -> str:
    """Compile the oracle with gcc; returns the path of the shared object."""
    out = out or os.path.join(_HERE, "liboracle.so")
    if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
        return out
    flags = [opt if f == "-O2" else f for f in CFLAGS]
    tmp = out + ".tmp.%d" % os.getpid()
    subprocess.run(["gcc", *flags, "-o", tmp, _SRC, "-lm"], check=True)
    os.replace(tmp, out)
    return out


_u8p = C.POINTER(C.c_uint8)
_u16p = C.POINTER(C.c_uint16)
_f64p = C.POINTER(C.c_double)


def _p8(a):
    return a.ctypes.data_as(_u8p)


def _p16(a):
    return a.ctypes.data_as(_u16p)


def _pf(a):
    return a.ctypes.data_as(_f64p)


def _u8(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    if a.dtype != np.uint8:
        raise TypeError("expected uint8")
    return a


class OracleError(RuntimeError):
    pass


def _check(rc: int, what: str):
    if rc != 0:
        raise OracleError(f"{what} failed with code {rc}")


class Lib:
    """One loaded build of the oracle (tests load an -O0 and an -O2 build)."""

    def __init__(self, path: str | None = None):
        self.path = path or build()
        L = self.L = C.CDLL(self.path)
        L.orc_sha256.argtypes = [_u8p, C.c_size_t, _u8p]
        L.orc_sha256.restype = None
        L.orc_sha256_k.restype = C.POINTER(C.c_uint32)
        L.orc_sha256_h0.restype = C.POINTER(C.c_uint32)
        L.orc_frame_hash.argtypes = [_u8p, C.c_uint32, C.c_uint32, C.c_uint32, _u8p]
        L.orc_lhcs_rhs.argtypes = [_f64p, C.c_double, _f64p]
        L.orc_lhcs_rhs.restype = None
        L.orc_rk4_step.argtypes = [_f64p, C.c_double]
        L.orc_rk4_step.restype = None
        L.orc_reconstruct.argtypes = [C.c_double, _u8p]
        L.orc_reconstruct.restype = C.c_double
        L.orc_init.argtypes = [C.POINTER(C.c_void_p)] + [C.c_double] * 5 + [C.c_uint32] * 3
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_destroy.restype = None
        L.orc_get_state.argtypes = [C.c_void_p, _f64p]
        L.orc_get_state.restype = None
        L.orc_set_state.argtypes = [C.c_void_p, _f64p]
        L.orc_set_state.restype = None
        L.orc_derive.argtypes = [C.c_void_p, _u8p, _u16p, _u8p, _f64p]
        for name in ("orc_bit_extract",):
            getattr(L, name).argtypes = [_u8p, C.c_uint32, C.c_uint32, _u8p]
            getattr(L, name).restype = None
        for name in ("orc_hshift", "orc_vshift"):
            getattr(L, name).argtypes = [_u8p, _u8p, C.c_uint32, C.c_uint32, _u16p, C.c_int]
            getattr(L, name).restype = None
        L.orc_xor_bits.argtypes = [_u8p, _u8p, C.c_uint32, C.c_uint32, _u8p]
        L.orc_xor_bits.restype = None
        L.orc_pack.argtypes = [_u8p, C.c_uint32, C.c_uint32, _u8p]
        L.orc_pack.restype = None
        for name in ("orc_confuse_xor", "orc_unconfuse_xor"):
            getattr(L, name).argtypes = [_u8p, C.c_uint32, C.c_uint32, _u16p, _u8p, _u8p]
        L.orc_encrypt_frames.argtypes = [C.c_void_p, _u8p, C.c_size_t, _u8p, _u8p]
        L.orc_decrypt_frames.argtypes = [C.c_void_p, _u8p, _u8p, C.c_size_t, _u8p]

    # -- SHA-256 ---------------------------------------------------------
    def sha256(self, msg: bytes | np.ndarray) -> bytes:
        a = np.frombuffer(bytes(msg), dtype=np.uint8) if not isinstance(msg, np.ndarray) else _u8(msg).ravel()
        buf = a if a.size else np.zeros(1, np.uint8)
        out = np.zeros(32, np.uint8)
        self.L.orc_sha256(_p8(buf), a.size, _p8(out))
        return out.tobytes()

    def sha256_constants(self):
        k = np.ctypeslib.as_array(self.L.orc_sha256_k(), shape=(64,)).copy()
        h0 = np.ctypeslib.as_array(self.L.orc_sha256_h0(), shape=(8,)).copy()
        return k, h0

    def frame_hash(self, frame: np.ndarray, n: int) -> bytes:
        f = _u8(frame)
        h, w, c = f.shape
        assert c == 3
        out = np.zeros(32, np.uint8)
        _check(self.L.orc_frame_hash(_p8(f), w, h, n, _p8(out)), "orc_frame_hash")
        return out.tobytes()

    # -- LHCS ------------------------------------------------------------
    def lhcs_rhs(self, s, gamma: float) -> np.ndarray:
        s = np.ascontiguousarray(s, dtype=np.float64)
        d = np.zeros(4)
        self.L.orc_lhcs_rhs(_pf(s), gamma, _pf(d))
        return d

    def rk4(self, s, gamma: float, steps: int = 1) -> np.ndarray:
        s = np.array(s, dtype=np.float64)
        for _ in range(steps):
            self.L.orc_rk4_step(_pf(s), gamma)
        return s

    def reconstruct(self, v: float, hb: bytes) -> float:
        a = np.frombuffer(bytes(hb), dtype=np.uint8).copy()
        assert a.size == 8
        return float(self.L.orc_reconstruct(v, _p8(a)))

    # -- Algorithms 3..7 on explicit bit matrices --------------------------
    def bit_extract(self, F: np.ndarray) -> np.ndarray:
        F = _u8(F)
        h, w, _ = F.shape
        M = np.zeros((3, h, 8 * w), np.uint8)
        self.L.orc_bit_extract(_p8(F), w, h, _p8(M))
        return M

    def _shift(self, fn, M: np.ndarray, D: np.ndarray, inverse: bool) -> np.ndarray:
        M = _u8(M)
        _, h, w8 = M.shape
        D = np.ascontiguousarray(D, dtype=np.uint16)
        assert D.size == 3 * (h + w8 // 8)
        out = np.zeros_like(M)
        fn(_p8(M), _p8(out), w8 // 8, h, _p16(D), int(inverse))
        return out

    def hshift(self, M, D, inverse=False):
        return self._shift(self.L.orc_hshift, M, D, inverse)

    def vshift(self, M, D, inverse=False):
        return self._shift(self.L.orc_vshift, M, D, inverse)

    def xor_bits(self, M: np.ndarray, B: np.ndarray) -> np.ndarray:
        M = _u8(M)
        _, h, w8 = M.shape
        B = _u8(B)
        assert B.size == 3 * h * (w8 // 8)
        out = np.zeros_like(M)
        self.L.orc_xor_bits(_p8(M), _p8(out), w8 // 8, h, _p8(B))
        return out

    def pack(self, M: np.ndarray) -> np.ndarray:
        M = _u8(M)
        _, h, w8 = M.shape
        F = np.zeros((h, w8 // 8, 3), np.uint8)
        self.L.orc_pack(_p8(M), w8 // 8, h, _p8(F))
        return F

    def confuse_xor(self, F: np.ndarray, D: np.ndarray, B: np.ndarray, inverse: bool = False) -> np.ndarray:
        F = _u8(F)
        h, w, _ = F.shape
        D = np.ascontiguousarray(D, dtype=np.uint16)
        B = _u8(B)
        assert D.size == 3 * (h + w) and B.size == F.size
        out = np.zeros_like(F)
        fn = self.L.orc_unconfuse_xor if inverse else self.L.orc_confuse_xor
        _check(fn(_p8(F), w, h, _p16(D), _p8(B), _p8(out)), "orc_confuse_xor")
        return out

    def ctx(self, key, gamma: float, n: int, w: int, h: int) -> "Ctx":
        return Ctx(self, key, gamma, n, w, h)


class Ctx:
    """Algorithm 1's frame-to-frame state (encrypt side or decrypt side)."""

    def __init__(self, lib: Lib, key, gamma: float, n: int, w: int, h: int):
        self.lib, self.n, self.w, self.h = lib, n, w, h
        self._p = C.c_void_p()
        x0, y0, z0, w0 = (float(v) for v in key)
        _check(lib.L.orc_init(C.byref(self._p), x0, y0, z0, w0, float(gamma), n, w, h), "orc_init")

    def close(self):
        if self._p:
            self.lib.L.orc_destroy(self._p)
            self._p = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def state(self) -> np.ndarray:
        s = np.zeros(4)
        self.lib.L.orc_get_state(self._p, _pf(s))
        return s

    @state.setter
    def state(self, s):
        s = np.ascontiguousarray(s, dtype=np.float64)
        self.lib.L.orc_set_state(self._p, _pf(s))

    def derive(self, H: bytes, want_ir: bool = False):
        Hh = np.frombuffer(bytes(H), dtype=np.uint8).copy()
        assert Hh.size == 32
        D = np.zeros(3 * (self.h + self.w), np.uint16)
        B = np.zeros((self.h, self.w, 3), np.uint8)
        IR = np.zeros((2 * self.n, 4)) if want_ir else None
        _check(self.lib.L.orc_derive(self._p, _p8(Hh), _p16(D), _p8(B), _pf(IR) if want_ir else None), "orc_derive")
        return (D, B, IR) if want_ir else (D, B)

    def encrypt_frames(self, frames: np.ndarray):
        f = _u8(frames)
        assert f.ndim == 4 and f.shape[1:] == (self.h, self.w, 3)
        out = np.zeros_like(f)
        hashes = np.zeros((f.shape[0], 32), np.uint8)
        _check(self.lib.L.orc_encrypt_frames(self._p, _p8(f), f.shape[0], _p8(out), _p8(hashes)), "orc_encrypt_frames")
        return out, hashes

    def decrypt_frames(self, cipher: np.ndarray, hashes: np.ndarray):
        f = _u8(cipher)
        hs = _u8(hashes)
        assert f.ndim == 4 and f.shape[1:] == (self.h, self.w, 3) and hs.shape == (f.shape[0], 32)
        out = np.zeros_like(f)
        _check(self.lib.L.orc_decrypt_frames(self._p, _p8(f), _p8(hs), f.shape[0], _p8(out)), "orc_decrypt_frames")
        return out


_default: Lib | None = None


def lib() -> Lib:
    global _default
    if _default is None:
        _default = Lib()
    return _default
