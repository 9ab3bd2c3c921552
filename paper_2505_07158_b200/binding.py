"""Thin ctypes binding of libvcrypt (include/vcrypt.h): same names, argument marshalling only.

Every step of the path runs inside the library; this module never computes.  It fails loudly if the
library cannot be built or loaded, and the library itself fails with VCRYPT_E_CUDA when there is no GPU
(unless a context is explicitly created host-only for the derivation hooks).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

OK, E_ARG, E_KEY, E_SHAPE, E_CUDA, E_NOMEM, E_STATE, E_LIMIT = 0, -1, -2, -3, -4, -5, -6, -7
NOALLOC_MAX_FRAMES = 512  # VCRYPT_NOALLOC_MAX_FRAMES
FLAG_HOST_ONLY, FLAG_FORCE_GENERIC, FLAG_HOST_SCALAR, FLAG_DEVICE_DERIVE, FLAG_DEVICE_HASH, FLAG_PERSISTENT, FLAG_ROW_TMA = 1, 2, 4, 8, 16, 32, 64


class Params(C.Structure):
    _fields_ = [("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double), ("w0", C.c_double),
                ("gamma", C.c_double), ("n_workers", C.c_uint32), ("width", C.c_uint32), ("height", C.c_uint32),
                ("batch", C.c_uint32), ("n_streams", C.c_uint32), ("host_threads", C.c_uint32),
                ("flags", C.c_uint32), ("device", C.c_int32), ("device_hash_bands", C.c_uint32),
                ("pipe_frames", C.c_uint32), ("pipe_streams", C.c_uint32),
                ("tune_row_stages", C.c_uint32), ("tune_row_item_blocks", C.c_uint32), ("tune_window", C.c_uint32),
                ("tune_ring", C.c_uint32)]


class FrameStats(C.Structure):
    _fields_ = [("hist_variance", C.c_double * 3), ("chi2", C.c_double * 3), ("entropy", C.c_double * 3),
                ("corr", (C.c_double * 3) * 3)]


class VcryptError(RuntimeError):
    def __init__(self, code: int, what: str, detail: str = ""):
        self.code = code
        msg = f"{what}: {lib().vcrypt_strerror(code).decode()} ({code})"
        if detail:
            msg += f" [{detail}]"
        super().__init__(msg)


_lib = None
_vp = C.c_void_p


def lib() -> C.CDLL:
    """Loads (building if stale) libvcrypt.so and declares every prototype of vcrypt.h."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if os.environ.get("VCRYPT_NO_BUILD") != "1" or not os.path.exists(path):
        path = _build.build()
    L = C.CDLL(path)
    L.vcrypt_init.argtypes = [C.POINTER(_vp), C.POINTER(Params)]
    L.vcrypt_encrypt_frames.argtypes = [_vp, _vp, C.c_size_t, _vp, _vp]
    L.vcrypt_decrypt_frames.argtypes = [_vp, _vp, _vp, C.c_size_t, _vp]
    L.vcrypt_destroy.argtypes = [_vp]
    L.vcrypt_destroy.restype = None
    L.vcrypt_strerror.argtypes = [C.c_int]
    L.vcrypt_strerror.restype = C.c_char_p
    L.vcrypt_last_cuda_error.argtypes = [_vp]
    L.vcrypt_last_cuda_error.restype = C.c_char_p
    L.vcrypt_describe.restype = C.c_char_p
    L.vcrypt_frame_hash.argtypes = [_vp, _vp, _vp]
    L.vcrypt_derive.argtypes = [_vp, _vp, _vp, _vp]
    L.vcrypt_get_state.argtypes = [_vp, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
    L.vcrypt_set_state.argtypes = [_vp, C.POINTER(C.c_double), C.c_uint64]
    L.vcrypt_host_threads.argtypes = [_vp]
    L.vcrypt_encrypt_device.argtypes = [_vp, _vp, _vp, _vp, C.c_size_t, _vp, _vp]
    L.vcrypt_decrypt_device.argtypes = [_vp, _vp, _vp, _vp, C.c_size_t, _vp, _vp]
    L.vcrypt_launch_count.argtypes = [_vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.vcrypt_last_stage_ms.argtypes = [_vp, C.POINTER(C.c_double)]
    L.vcrypt_derive_device.argtypes = [_vp, _vp, _vp, _vp, _vp]
    L.vcrypt_frame_hash_device.argtypes = [_vp, _vp, C.c_size_t, _vp, _vp]
    L.vcrypt_frame_stats_device.argtypes = [_vp, _vp, C.c_size_t, C.POINTER(FrameStats), _vp, _vp]
    L.vcrypt_npcr_uaci_device.argtypes = [_vp, _vp, _vp, C.c_size_t, _vp, _vp, _vp]
    L.vcrypt_npcr_uaci_device_noalloc.argtypes = [_vp, _vp, _vp, C.c_size_t, _vp, _vp, _vp]
    L.vcrypt_local_entropy_device.argtypes = [_vp, _vp, C.c_size_t, _vp, C.c_uint32, C.c_uint32, _vp, _vp]
    _lib = L
    return L


def _host_ptr(a, dtype, nbytes: int, what: str) -> int:
    """Address of a C-contiguous numpy array or CPU torch tensor (pinned or not); no copy."""
    if isinstance(a, np.ndarray):
        if a.dtype != dtype or not a.flags.c_contiguous or a.nbytes != nbytes:
            raise ValueError(f"{what}: need C-contiguous {np.dtype(dtype).name} of {nbytes} bytes")
        return a.ctypes.data
    if hasattr(a, "data_ptr"):  # torch tensor
        if a.device.type != "cpu" or not a.is_contiguous() or a.numel() * a.element_size() != nbytes:
            raise ValueError(f"{what}: need contiguous CPU tensor of {nbytes} bytes")
        return a.data_ptr()
    raise TypeError(f"{what}: numpy array or CPU torch tensor expected")


def _dev_ptr(t, nbytes: int, what: str) -> int:
    if not hasattr(t, "data_ptr") or t.device.type != "cuda" or not t.is_contiguous():
        raise ValueError(f"{what}: contiguous CUDA tensor expected")
    if t.numel() * t.element_size() != nbytes:
        raise ValueError(f"{what}: need {nbytes} bytes, got {t.numel() * t.element_size()}")
    return t.data_ptr()


class Vcrypt:
    """One vcrypt_ctx.  Method names follow the C calls without the vcrypt_ prefix."""

    def __init__(self, key, gamma: float, n_workers: int, width: int, height: int, batch: int = 0,
                 n_streams: int = 0, host_threads: int = 0, flags: int = 0, device: int = -1, device_hash_bands: int = 0,
                 pipe_frames: int = 0, pipe_streams: int = 0, tune=(0, 0, 0, 0)):
        self.L = lib()
        self.w, self.h, self.n = int(width), int(height), int(n_workers)
        self.frame_bytes = 3 * self.w * self.h
        self.nD = 3 * (self.w + self.h)
        x0, y0, z0, w0 = (float(v) for v in key)
        self.params = Params(x0, y0, z0, w0, float(gamma), n_workers, width, height, batch, n_streams,
                             host_threads, flags, device, device_hash_bands, pipe_frames, pipe_streams, *[int(t) for t in (tuple(tune) + (0,) * 4)[:4]])
        self._p = _vp()
        rc = self.L.vcrypt_init(C.byref(self._p), C.byref(self.params))
        if rc != OK:
            self._p = _vp()
            raise VcryptError(rc, "vcrypt_init")

    # -- life cycle ------------------------------------------------------------------------------
    def destroy(self):
        if getattr(self, "_p", None):
            self.L.vcrypt_destroy(self._p)
            self._p = _vp()

    close = destroy

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def _check(self, rc: int, what: str):
        if rc != OK:
            raise VcryptError(rc, what, self.L.vcrypt_last_cuda_error(self._p).decode() if rc in (E_CUDA, E_LIMIT) else "")

    # -- host-buffer calls ---------------------------------------------------------------------------
    def encrypt_frames(self, frames, cipher_out=None, hashes_out=None):
        """frames: (n, H, W, 3) uint8 numpy array or CPU torch tensor.  Returns (cipher, hashes)."""
        n = int(frames.shape[0])
        if cipher_out is None:
            cipher_out = np.empty((n, self.h, self.w, 3), np.uint8)
        if hashes_out is None:
            hashes_out = np.empty((n, 32), np.uint8)
        rc = self.L.vcrypt_encrypt_frames(self._p, _host_ptr(frames, np.uint8, n * self.frame_bytes, "frames"), n,
                                          _host_ptr(cipher_out, np.uint8, n * self.frame_bytes, "cipher_out"),
                                          _host_ptr(hashes_out, np.uint8, n * 32, "hashes_out"))
        self._check(rc, "vcrypt_encrypt_frames")
        return cipher_out, hashes_out

    def decrypt_frames(self, cipher, hashes, plain_out=None):
        n = int(cipher.shape[0])
        if plain_out is None:
            plain_out = np.empty((n, self.h, self.w, 3), np.uint8)
        rc = self.L.vcrypt_decrypt_frames(self._p, _host_ptr(cipher, np.uint8, n * self.frame_bytes, "cipher"),
                                          _host_ptr(hashes, np.uint8, n * 32, "hashes"), n,
                                          _host_ptr(plain_out, np.uint8, n * self.frame_bytes, "plain_out"))
        self._check(rc, "vcrypt_decrypt_frames")
        return plain_out

    # -- host derivation hooks -------------------------------------------------------------------------
    def frame_hash(self, frame) -> bytes:
        out = np.empty(32, np.uint8)
        self._check(self.L.vcrypt_frame_hash(self._p, _host_ptr(frame, np.uint8, self.frame_bytes, "frame"),
                                             out.ctypes.data), "vcrypt_frame_hash")
        return out.tobytes()

    def derive(self, hash32: bytes, D_out=None, B_out=None):
        H = np.frombuffer(bytes(hash32), np.uint8).copy()
        if H.size != 32:
            raise ValueError("hash must be 32 bytes")
        if D_out is None:
            D_out = np.empty(self.nD, np.uint16)
        if B_out is None:
            B_out = np.empty((self.h, self.w, 3), np.uint8)
        self._check(self.L.vcrypt_derive(self._p, H.ctypes.data, _host_ptr(D_out, np.uint16, 2 * self.nD, "D_out"),
                                         _host_ptr(B_out, np.uint8, self.frame_bytes, "B_out")), "vcrypt_derive")
        return D_out, B_out

    def frame_hash_device(self, d_frames, stream=None) -> np.ndarray:
        """vcrypt_frame_hash_device: H of the frames of a CUDA tensor (n, h, w, 3), hashed on the GPU -> (n, 32) uint8."""
        n = int(d_frames.shape[0])
        out = np.empty((n, 32), np.uint8)
        st = 0 if stream is None else int(stream)
        self._check(self.L.vcrypt_frame_hash_device(self._p, _dev_ptr(d_frames, n * self.frame_bytes, "d_frames"), n,
                                                    out.ctypes.data, st), "vcrypt_frame_hash_device")
        return out

    def derive_device(self, hash32: bytes, d_D, d_B, stream=None):
        """vcrypt_derive_device: D (int16/uint16 tensor, 3(h+w)) and B (uint8, h x w x 3) derived on the GPU into device tensors."""
        H = np.frombuffer(bytes(hash32), np.uint8).copy()
        if H.size != 32:
            raise ValueError("hash must be 32 bytes")
        st = 0 if stream is None else int(stream)
        self._check(self.L.vcrypt_derive_device(self._p, H.ctypes.data, _dev_ptr(d_D, 2 * self.nD, "d_D"),
                                                _dev_ptr(d_B, self.frame_bytes, "d_B"), st), "vcrypt_derive_device")

    def get_state(self):
        s = (C.c_double * 4)()
        k = C.c_uint64()
        self._check(self.L.vcrypt_get_state(self._p, s, C.byref(k)), "vcrypt_get_state")
        return np.array(list(s)), int(k.value)

    def set_state(self, state, frames_done: int):
        s = (C.c_double * 4)(*[float(v) for v in state])
        self._check(self.L.vcrypt_set_state(self._p, s, int(frames_done)), "vcrypt_set_state")

    def host_threads(self) -> int:
        return int(self.L.vcrypt_host_threads(self._p))

    # -- kernel-only path (torch CUDA tensors; torch is plumbing for device memory and streams) -----------
    def _device(self, fn, what, d_in, d_D, d_B, d_out, stream):
        n = int(d_in.shape[0])
        if stream is None:
            import torch

            stream = torch.cuda.current_stream().cuda_stream
        rc = fn(self._p, _dev_ptr(d_in, n * self.frame_bytes, "input"), _dev_ptr(d_D, 2 * n * self.nD, "D"),
                _dev_ptr(d_B, n * self.frame_bytes, "B"), n, _dev_ptr(d_out, n * self.frame_bytes, "output"),
                _vp(int(stream)))
        self._check(rc, what)
        return d_out

    def encrypt_device(self, d_frames, d_D, d_B, d_cipher, stream=None):
        return self._device(self.L.vcrypt_encrypt_device, "vcrypt_encrypt_device", d_frames, d_D, d_B, d_cipher, stream)

    def decrypt_device(self, d_cipher, d_D, d_B, d_plain, stream=None):
        return self._device(self.L.vcrypt_decrypt_device, "vcrypt_decrypt_device", d_cipher, d_D, d_B, d_plain, stream)

    def launch_count(self):
        a, b = C.c_uint64(), C.c_uint64()
        self._check(self.L.vcrypt_launch_count(self._p, C.byref(a), C.byref(b)), "vcrypt_launch_count")
        return int(a.value), int(b.value)

    def frame_stats_device(self, d_frames, stream=None):
        """vcrypt_frame_stats_device -> dict of arrays: hist_variance, chi2, entropy (n, 3), corr (n, 3, 3), hist (n, 3, 256)."""
        n = int(d_frames.shape[0])
        st = (FrameStats * n)()
        hist = np.empty((n, 3, 256), np.uint32)
        self._check(self.L.vcrypt_frame_stats_device(self._p, _dev_ptr(d_frames, n * self.frame_bytes, "d_frames"), n, st,
                                                     hist.ctypes.data, 0 if stream is None else int(stream)), "vcrypt_frame_stats_device")
        return {"hist_variance": np.array([list(x.hist_variance) for x in st]), "chi2": np.array([list(x.chi2) for x in st]),
                "entropy": np.array([list(x.entropy) for x in st]),
                "corr": np.array([[list(row) for row in x.corr] for x in st]), "hist": hist}

    def npcr_uaci_device(self, d_a, d_b, stream=None):
        """vcrypt_npcr_uaci_device -> (npcr, uaci), each (n, 4): all channels, channel 0, 1, 2 (percent)."""
        n = int(d_a.shape[0])
        npcr, uaci = np.empty((n, 4)), np.empty((n, 4))
        self._check(self.L.vcrypt_npcr_uaci_device(self._p, _dev_ptr(d_a, n * self.frame_bytes, "d_a"),
                                                   _dev_ptr(d_b, n * self.frame_bytes, "d_b"), n, npcr.ctypes.data, uaci.ctypes.data,
                                                   0 if stream is None else int(stream)), "vcrypt_npcr_uaci_device")
        return npcr, uaci

    def npcr_uaci_device_noalloc(self, d_a, d_b, stream=None):
        """vcrypt_npcr_uaci_device_noalloc -> (npcr, uaci) like npcr_uaci_device, for processes that may not allocate GPU
        memory (all of it reserved by a pool, a frame deadline, a no-allocation-after-start rule): the accumulators are a
        fixed array inside libvcrypt.so.  At most NOALLOC_MAX_FRAMES frames per call (VcryptError E_LIMIT above that); one
        call at a time per GPU -- concurrent calls share the array and corrupt each other's sums."""
        n = int(d_a.shape[0])
        npcr, uaci = np.empty((n, 4)), np.empty((n, 4))
        self._check(self.L.vcrypt_npcr_uaci_device_noalloc(self._p, _dev_ptr(d_a, n * self.frame_bytes, "d_a"),
                                                           _dev_ptr(d_b, n * self.frame_bytes, "d_b"), n, npcr.ctypes.data,
                                                           uaci.ctypes.data, 0 if stream is None else int(stream)),
                    "vcrypt_npcr_uaci_device_noalloc")
        return npcr, uaci

    def local_entropy_device(self, d_frames, blocks_xy, side: int, stream=None):
        """vcrypt_local_entropy_device -> (n, 3): mean block entropy per channel; blocks_xy (k, 2) uint32 top-left (x, y)."""
        n = int(d_frames.shape[0])
        xy = np.ascontiguousarray(blocks_xy, dtype=np.uint32)
        out = np.empty((n, 3))
        self._check(self.L.vcrypt_local_entropy_device(self._p, _dev_ptr(d_frames, n * self.frame_bytes, "d_frames"), n, xy.ctypes.data,
                                                       xy.shape[0], side, out.ctypes.data, 0 if stream is None else int(stream)),
                    "vcrypt_local_entropy_device")
        return out

    def last_stage_ms(self):
        out = (C.c_double * 4)()
        self._check(self.L.vcrypt_last_stage_ms(self._p, out), "vcrypt_last_stage_ms")
        return dict(zip(("hash", "derive", "staging", "gpu_wait"), list(out)))


def describe() -> str:
    return lib().vcrypt_describe().decode()
