"""Small timing probes of the individual device entry points (what profiles/ cites next to bench.py):

  python -m paper_2505_07158_b200.probe kernels [--config C4] [--batch 8] [--batches 6] [--streams 1] | [--clip 96 --pipe-frames 0 --pipe-streams 0]   encrypt / decrypt kernels, CUDA events
  python -m paper_2505_07158_b200.probe derive  [--config C4] [--frames 8]                device hashing + worker systems, wall clock
  python -m paper_2505_07158_b200.probe stats   [--config C4] [--frames 32]               evaluation metrics, wall clock
  python -m paper_2505_07158_b200.probe dsmem                                             all-to-all through distributed shared memory

Inputs are random device tensors (the kernels' time does not depend on the values); results are only timed here --
parity lives in tests/.  Needs a CUDA device.
"""
from __future__ import annotations

import argparse
import time

import numpy as np

from . import binding as vb
from . import synth


def _hbm_peak() -> float:
    import json
    import os

    try:
        with open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"])
    except Exception:
        return 6650.0


def kernels(cfg, batch: int, batches: int, streams: int = 1, clip: int = 0, pipe_frames: int = 0, pipe_streams: int = 0):
    import torch

    if clip:  # one call on a resident clip of `clip` frames: the library's own launch schedule (pipe_frames, pipe_streams)
        batch, batches = clip, 1
    w, h, T = cfg.w, cfg.h, batch * batches
    g = torch.Generator(device="cuda")
    g.manual_seed(1)
    F = torch.randint(0, 256, (T, h, w, 3), dtype=torch.uint8, device="cuda", generator=g)
    B = torch.randint(0, 256, (T, h, w, 3), dtype=torch.uint8, device="cuda", generator=g)
    D = torch.randint(-32768, 32767, (T, 3 * (h + w)), dtype=torch.int16, device="cuda", generator=g)
    E, P = torch.empty_like(F), torch.empty_like(F)
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, w, h, pipe_frames=pipe_frames, pipe_streams=pipe_streams)
    # calls go round-robin over `streams` streams (independent batches: no ordering is needed between them);
    # the timed region is bracketed on the current stream, which the side streams fork from and join into
    cur = torch.cuda.current_stream()
    side = [torch.cuda.Stream() for _ in range(streams)] if streams > 1 else [cur]
    alg = (9 * w * h + 6 * (w + h)) * T
    for name, fn, src, dst in (("encrypt", v.encrypt_device, F, E), ("decrypt", v.decrypt_device, E, P)):
        def run():
            for k, b0 in enumerate(range(0, T, batch)):
                fn(src[b0:b0 + batch], D[b0:b0 + batch], B[b0:b0 + batch], dst[b0:b0 + batch], side[k % len(side)].cuda_stream)
        for _ in range(3):
            run()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(cur)
        if streams > 1:
            for s_ in side:
                s_.wait_event(e0)
        for _ in range(10):
            run()
        if streams > 1:
            for s_ in side:
                cur.wait_stream(s_)
        e1.record(cur)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 10
        print(f"{cfg.name} {name}: {ms * 1e3 / T:.3f} us/frame, {alg / ms / 1e6:.0f} GB/s algorithmic, {alg / ms / 1e6 / _hbm_peak():.3f} of the HBM copy rate")
    print("decrypt(encrypt(x)) == x:", bool(torch.equal(P, F)))


def derive(cfg, frames: int):
    import torch

    w, h = cfg.w, cfg.h
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, w, h)
    F = torch.randint(0, 256, (frames, h, w, 3), dtype=torch.uint8, device="cuda")
    v.frame_hash_device(F)
    t0 = time.perf_counter()
    for _ in range(3):
        v.frame_hash_device(F)
    dt = (time.perf_counter() - t0) / 3
    print(f"{cfg.name} device hashing of {frames} frames ({frames * synth.N_WORKERS} band messages): {dt * 1e3:.2f} ms per call")
    dD = torch.zeros(3 * (h + w), dtype=torch.int16, device="cuda")
    dB = torch.zeros((h, w, 3), dtype=torch.uint8, device="cuda")
    v.derive_device(bytes(32), dD, dB)
    t0 = time.perf_counter()
    for _ in range(3):
        v.derive_device(bytes(32), dD, dB)
    print(f"{cfg.name} device worker systems of 1 frame ({2 * synth.N_WORKERS} chains): {(time.perf_counter() - t0) / 3 * 1e3:.2f} ms per call")


def stats(cfg, frames: int):
    import torch

    w, h = cfg.w, cfg.h
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, w, h)
    F = torch.randint(0, 256, (frames, h, w, 3), dtype=torch.uint8, device="cuda")
    G = torch.randint(0, 256, (frames, h, w, 3), dtype=torch.uint8, device="cuda")
    blocks = synth.random_blocks(w, h, 30, 44, 1)
    for name, fn, mult in (("frame_stats", lambda: v.frame_stats_device(F), 1), ("npcr_uaci", lambda: v.npcr_uaci_device(F, G), 2),
                           ("local_entropy", lambda: v.local_entropy_device(F, blocks, 44), 0)):
        fn()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(5):
            fn()
        dt = (time.perf_counter() - t0) / 5
        extra = f", {mult * frames * 3 * w * h / dt / 1e9:.0f} GB/s" if mult else ""
        print(f"{cfg.name} {name}: {dt * 1e3:.3f} ms per call of {frames} frames (device + host finish){extra}")


def dsmem(cfg):
    """What an all-to-all between the CTAs of a cluster costs through distributed shared memory."""
    v = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h)
    for cs in (2, 4, 8, 16):
        for kb in (64, 96, 110):
            own = kb * 1024 // (16 * cs) * (16 * cs)
            for mode, name in ((0, "st.shared::cluster.v4"), (1, "cp.async.bulk to peer")):
                try:
                    us, nc = v.dsmem_probe(cs, own, mode, 20)
                except vb.VcryptError as e:
                    print(f"cluster {cs:2d} x {kb:3d} KB {name}: {e}")
                    continue
                tot = own * cs * nc
                print(f"cluster {cs:2d} x {kb:3d} KB per CTA, {nc:2d} resident clusters ({cs * nc:3d} SMs), {name:22s}: "
                      f"{us:6.2f} us per all-to-all, {tot / us / 1e6:5.2f} TB/s chip-wide, {own / (us * 1e-6) / 1.965e9:5.1f} B/clk/SM at 1965 MHz")


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("what", choices=["kernels", "derive", "stats", "dsmem"])
    ap.add_argument("--config", default="C4", choices=sorted(synth.CONFIGS))
    ap.add_argument("--batch", type=int, default=8)
    ap.add_argument("--batches", type=int, default=6)
    ap.add_argument("--frames", type=int, default=0)
    ap.add_argument("--streams", type=int, default=1, help="kernels: streams the calls go round-robin over")
    ap.add_argument("--clip", type=int, default=0, help="kernels: one call on a resident clip of this many frames")
    ap.add_argument("--pipe-frames", type=int, default=0, help="kernels: vcrypt_params.pipe_frames (0: library default)")
    ap.add_argument("--pipe-streams", type=int, default=0, help="kernels: vcrypt_params.pipe_streams (0: library default, 1: off)")
    a = ap.parse_args()
    cfg = synth.CONFIGS[a.config]
    if a.what == "kernels":
        kernels(cfg, a.batch, a.batches, a.streams, a.clip, a.pipe_frames, a.pipe_streams)
    elif a.what == "dsmem":
        dsmem(cfg)
    elif a.what == "derive":
        derive(cfg, a.frames or 8)
    else:
        stats(cfg, a.frames or 32)


if __name__ == "__main__":
    _ = np  # numpy is a dependency of the binding; imported for clarity
    main()
