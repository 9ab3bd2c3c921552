#!/usr/bin/env python
"""bench.py -- FHD frames/s encrypted on B200 (BASELINE.json metric), kernel-only and end to end.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4|C5|C3|C2|C1] [--impl ours|reference]

One "step" = one pass of the whole hot path over the clip of the chosen config (default C4: 300 frames of
1920x1080x3, batches of 8 frames per call, 3 streams).
  value : frames/s with F_o, D, B already resident in HBM -- vcrypt_encrypt_device calls only (rows a6-a10),
          timed with CUDA events on the launching stream.
  e2e   : frames/s through vcrypt_encrypt_frames with pinned HOST buffers: sub-frame SHA-256, chain, worker
          LHCS -> D, B, H2D, kernels, D2H all inside the timed region (rows a1-a11), wall clock.  By default the band
          hashes and the worker systems run on the GPU (--hash device --derive device, pipeline 12 deep); --hash host
          --derive host is the all-host derivation with the config's 3 streams: same bytes.
  roofline : algorithmic bytes (9wh per frame + D) / CUDA-event time of the encrypt kernels vs the measured HBM peak.
  cpu_baseline : the oracle as it stands on a bounded sample, one core.
Prints ONE JSON line (rank 0).  Under torchrun (N > 1) every rank encrypts its own clip (weak scaling, no
collective on the data path: frames are independent once the host chain step is done).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2505_07158_b200 import parallel, synth  # noqa: E402

METRIC = "FHD frames/s encrypted"
UNIT = "frames/s"
FALLBACK_HBM_GBS = 6650.0  # B200_PROFILING.md fallback
# dram__bytes_read.sum + dram__bytes_write.sum of the two kernels of one launch pair (5 FHD frames: row pass 30.9 + 2.9 MB,
# column pass 27.0 + 3.2 MB), from the ncu --set full capture summarised in profiles/r1n_ncu_full_summary.csv; below the
# 93.4 MB of algorithmic bytes of a pair because most of its output is still dirty in L2 when the kernel ends
NCU_TRAFFIC_PER_CALL = {"C4": 64.0e6}
NCU_COL_SHARE = 0.544  # column pass's share of a launch pair's serialised time in the same capture (19.6 of 36.1 us)


def hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                       "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_lib():
    from oracle import oracle  # only the cpu_baseline / reference legs and the result check use it

    return oracle.lib()


def time_oracle(cfg, frames_np, nframes):
    O = oracle_lib()
    oc = O.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h)
    t0 = time.perf_counter()
    C, H = oc.encrypt_frames(frames_np[:nframes])
    dt = time.perf_counter() - t0
    return nframes / dt, C, H


def run_reference(args, cfg):
    """--impl reference: the oracle, as it stands, on the host cores (one thread), bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    per_step = {"C1": 1, "C2": 8, "C3": 2, "C4": 2, "C5": 1}[cfg.name]
    frames = synth.video(cfg, per_step)
    O = oracle_lib()
    oc = O.ctx(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h)
    for _ in range(args.warmup):
        oc.encrypt_frames(frames)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oc.encrypt_frames(frames)
    dt = time.perf_counter() - t0
    v = per_step * args.steps / dt
    sample = f"first {per_step} frame(s) of {cfg.name} per step, chain carried across steps"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "frames_per_step": per_step},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def workload_name(cfg):
    return (f"{cfg.name}: {cfg.w}x{cfg.h}x3 uint8 synthetic video (moving gradient + blocks + noise), {cfg.frames} frames, "
            f"end-to-end leg in batches of {cfg.batch} per launch pair over e2e.n_streams streams; kernel-only leg = one call on the "
            f"resident clip (launch pairs of about 31 MB of frames over 2 streams), "
            f"key = 4 doubles, n_workers = {synth.N_WORKERS}")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C4", choices=sorted(synth.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--frames", type=int, default=0, help="frames per step (default: the config's clip length)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--derive", default="auto", choices=["auto", "host", "device"],
                    help="where the worker systems (D, B) of the end-to-end leg run: host lanes or the GPU (same bytes)")
    ap.add_argument("--hash", default="auto", choices=["auto", "host", "device"],
                    help="where the sub-frame SHA-256 of the end-to-end leg runs (same H)")
    ap.add_argument("--hash-bands", type=int, default=0, help="with --hash device: row bands per frame hashed on the GPU (0: all)")
    ap.add_argument("--e2e-batch", type=int, default=0, help="frames per pipeline slot of the end-to-end leg (0: the config's)")
    ap.add_argument("--e2e-streams", type=int, default=0, help="pipeline depth of the end-to-end leg (0: the config's)")
    args = ap.parse_args()
    cfg = synth.CONFIGS[args.config]
    # auto: throughput configs (batches of several frames) put band hashing and worker systems on the GPU; the one-frame-
    # per-call latency config (C3) keeps them on the host threads (a GPU thread needs 6 ms per band, 2.6 ms per chain)
    for k in ("derive", "hash"):
        if getattr(args, k) == "auto":
            setattr(args, k, "device" if (args.e2e_batch or cfg.batch) >= 4 else "host")
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import torch.distributed as dist

    from paper_2505_07158_b200 import binding as vb

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    W = max(3, args.warmup)
    K = args.steps
    T = args.frames or cfg.frames
    fb, nD = 3 * cfg.w * cfg.h, 3 * (cfg.w + cfg.h)
    ncores = os.cpu_count() or 1
    threads = max(1, ncores // world)

    # ---- inputs: rank r gets its own clip (seed + r) in pinned host memory --------------------------------
    rcfg = parallel.rank_clip_config(cfg, rank, T)
    h_in = torch.empty((T, cfg.h, cfg.w, 3), dtype=torch.uint8).pin_memory()
    distinct = min(T, 48)  # drawing pixels is slow: the clip repeats its first frames with a per-frame stamp
    synth.video(rcfg, distinct, out=h_in.numpy())
    for t in range(distinct, T):
        h_in[t].copy_(h_in[t % distinct])
        h_in[t, 0, 0, 0] = t % 251  # every frame distinct -> distinct hash, D, B
    h_out = torch.empty_like(h_in).pin_memory()
    h_hash = torch.empty((T, 32), dtype=torch.uint8)
    frames_np = h_in.numpy()

    # ---- device-resident inputs for the kernel-only number: D, B from the production host derivation -------
    ctx = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h, batch=cfg.batch, n_streams=cfg.n_streams,
                    host_threads=threads, device=local)
    D_all = np.empty((T, nD), np.uint16)
    B_all = torch.empty((T, cfg.h, cfg.w, 3), dtype=torch.uint8).pin_memory()
    for t in range(T):
        ctx.derive(ctx.frame_hash(frames_np[t]), D_all[t], B_all.numpy()[t])
    d_F = h_in.cuda(non_blocking=True)
    d_B = B_all.cuda(non_blocking=True)
    d_D = torch.from_numpy(D_all.view(np.int16)).cuda()
    d_E = torch.empty_like(d_F)
    torch.cuda.synchronize()
    del B_all
    kctx = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h, batch=cfg.batch, n_streams=cfg.n_streams,
                     host_threads=threads, device=local)
    stream = torch.cuda.current_stream().cuda_stream

    def kernel_step():
        # one call on the resident clip: the library cuts it into launch pairs (row pass + column pass) of about 31 MB of
        # frames and alternates them over two streams forked from / joined into `stream` (vcrypt_params.pipe_*)
        kctx.encrypt_device(d_F, d_D, d_B, d_E, stream)
        return kctx.launch_count()[0]

    def kernel_step_batches():
        # context figure: one call per batch of cfg.batch frames, every launch on `stream` (the schedule before pipe_*)
        for b0 in range(0, T, cfg.batch):
            b1 = min(T, b0 + cfg.batch)
            kctx.encrypt_device(d_F[b0:b1], d_D[b0:b1], d_B[b0:b1], d_E[b0:b1], stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- kernel-only: CUDA events on the launching stream -----------------------------------------------
    # W untimed steps; a kernel-only step lasts about a millisecond, so the warm-up is also held for at least 50 ms of GPU
    # work: the timed steps must not see the clock ramp of a GPU that idled during the host-side set-up.  (Measured: 3 steps
    # or 50 ms of warm-up -> 0.600 - 0.604 of the copy rate; 250 ms of warm-up -> 0.594 with sw_power_cap reported: the
    # timed region of 10 steps is 14 ms, a burst like the copy the peak was measured with.)
    warm_steps, t_warm = 0, time.perf_counter()
    while warm_steps < W or (time.perf_counter() - t_warm < 0.05 and warm_steps < 2000):
        kernel_step()
        warm_steps += 1
        if warm_steps >= W:
            torch.cuda.synchronize()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    launches = 0
    ev[0].record()
    for k in range(K):
        launches += kernel_step()
        ev[k + 1].record()
    barrier()
    step_ms = [ev[k].elapsed_time(ev[k + 1]) for k in range(K)]
    kern_ms_total = ev[0].elapsed_time(ev[K])
    kernel_out_digest = synth.digest(d_E[:2].cpu().numpy())
    kernel_all_digest = synth.digest(d_E.cpu().numpy())
    pairs_per_step = max(1, launches // (2 * K))

    # ---- context figure: the same frames in calls of cfg.batch frames on one stream ----------------------------------
    KB = max(1, min(K, 5))
    d_E.zero_()
    for _ in range(2):
        kernel_step_batches()
    barrier()
    bv = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    bv[0].record()
    for _ in range(KB):
        kernel_step_batches()
    bv[1].record()
    barrier()
    batches_ms_frame = bv[0].elapsed_time(bv[1]) / KB / T
    batches_same = bool(synth.digest(d_E.cpu().numpy()) == kernel_all_digest)

    # ---- context figures: the inverse kernels on the same clip, and what the memory system allows for these bytes ----
    def decrypt_step():
        kctx.decrypt_device(d_E, d_D, d_B, d_P, stream)

    d_P = torch.empty_like(d_F)
    for _ in range(2):
        decrypt_step()
    barrier()
    dv = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    KD = max(1, min(K, 5))
    dv[0].record()
    for _ in range(KD):
        decrypt_step()
    dv[1].record()
    barrier()
    dec_ms_frame = dv[0].elapsed_time(dv[1]) / KD / T
    decrypt_ok = bool(torch.equal(d_P, d_F))
    del d_P
    probes = {}
    if rank == 0:
        nb = min(cfg.batch, T)
        for which, name in ((0, "sequential_copy"), (1, "two_pass_traffic_sequential"), (2, "column_strips_read_write")):
            probes[name] = kctx.memory_probe(which, nb, 20) / nb  # us per frame

    # pipeline depth of the end-to-end leg: the config's 3 streams with host hashing; device hashing (6 ms per band on a
    # GPU thread) needs a deeper pipeline to be hidden (results do not depend on it)
    e2e_streams = args.e2e_streams or (12 if args.hash == "device" else cfg.n_streams)
    # ---- end to end through the host-buffer call -----------------------------------------------------------
    ectx = None
    e2e_s = []
    for k in range(W + K):
        ectx = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h, batch=args.e2e_batch or cfg.batch,
                         n_streams=e2e_streams, host_threads=threads, device=local,
                         flags=(vb.FLAG_DEVICE_DERIVE if args.derive == "device" else 0) |
                         (vb.FLAG_DEVICE_HASH if args.hash == "device" else 0),
                         device_hash_bands=args.hash_bands) if ectx is None else ectx
        if k == W:
            barrier()
            t_e2e0 = time.perf_counter()
        t0 = time.perf_counter()
        ectx.encrypt_frames(h_in, h_out, h_hash)
        if k >= W:
            e2e_s.append(time.perf_counter() - t0)
        if k == 0:
            first_out = h_out[:2].numpy().copy()
            first_hash = h_hash[:2].numpy().copy()
            first_all_digest = synth.digest(h_out.numpy())
    barrier()
    e2e_total = time.perf_counter() - t_e2e0
    stage = ectx.last_stage_ms()
    clocks = sampler.stop() if sampler else None

    # ---- context: the receiver's side end to end (vcrypt_decrypt_frames: no hashing, H is transmitted) -----------------------
    h_plain = torch.empty_like(h_in).pin_memory()
    fresh = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h, batch=args.e2e_batch or cfg.batch, n_streams=e2e_streams,
                      host_threads=threads, device=local, flags=(vb.FLAG_DEVICE_DERIVE if args.derive == "device" else 0) |
                      (vb.FLAG_DEVICE_HASH if args.hash == "device" else 0), device_hash_bands=args.hash_bands)
    fresh.encrypt_frames(h_in, h_out, h_hash)  # the clip from the start of the chain (the timed calls carried the chain on)
    fresh.destroy()
    dec_s = []
    dctx = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h, batch=args.e2e_batch or cfg.batch,
                     n_streams=e2e_streams, host_threads=threads, device=local,
                     flags=vb.FLAG_DEVICE_DERIVE if args.derive == "device" else 0)
    state0 = dctx.get_state()[0].copy()
    for k in range(4):  # the first call allocates the pipeline's buffers: not timed
        dctx.set_state(state0, 0)  # back to the start of the chain (checkpoint / resume hook)
        barrier()
        t0 = time.perf_counter()
        dctx.decrypt_frames(h_out, h_hash, h_plain)
        if k:
            dec_s.append(time.perf_counter() - t0)
    dctx.destroy()
    e2e_decrypt_ok = bool(torch.equal(h_plain, h_in))
    del h_plain

    # max over ranks
    kern_ms_total, e2e_total = parallel.max_over_ranks([kern_ms_total, e2e_total], device="cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- no number for a wrong result: first pass of the e2e path (fresh chain) against the oracle -----------
    check = {"frames_vs_oracle": 2}
    cpu_baseline = None
    n_or = {"C1": 1, "C2": 24, "C3": 16, "C4": 16, "C5": 4}[cfg.name]
    n_or = min(n_or, T) if not args.no_cpu_baseline else min(2, T)
    fps_or, C_or, H_or = time_oracle(cfg, frames_np, n_or)
    m = min(2, n_or)
    check["e2e_vs_oracle"] = bool(np.array_equal(C_or[:m], first_out[:m]) and np.array_equal(H_or[:m], first_hash[:m]))
    check["kernels_vs_e2e_first_frames"] = bool(kernel_out_digest == synth.digest(first_out))
    check["kernels_vs_e2e_all_frames"] = bool(kernel_all_digest == first_all_digest)
    check["kernels_in_batches_same_bytes"] = batches_same
    check["decrypt_kernels_invert"] = decrypt_ok
    check["e2e_decrypt_returns_clip"] = e2e_decrypt_ok
    ok = all(v for k, v in check.items() if k != "frames_vs_oracle")
    check["ok"] = bool(ok)
    if not ok:
        print(json.dumps({"metric": METRIC, "error": "GPU output does not match the oracle", "check": check}))
        raise SystemExit(1)
    if not args.no_cpu_baseline:
        cpu_baseline = {"value": fps_or, "unit": UNIT, "cores": 1, "kind": "oracle",
                        "sample": f"first {n_or} frames of the clip, oracle/vcrypt_oracle.c single-threaded, "
                                  f"{ncores} host cores present"}

    peak, peak_src = hbm_peak()
    alg_bytes_frame = 3 * fb + 2 * nD  # read F_o + read B + write F_e + read D (~9wh)
    value = parallel.whole_job_rate(world, T, K, kern_ms_total * 1e-3)
    achieved = alg_bytes_frame * T * K / (kern_ms_total * 1e-3) / 1e9
    e2e_value = parallel.whole_job_rate(world, T, K, e2e_total)
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": kern_ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u8", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "frames_per_step": T, "ms_per_frame_kernel": kern_ms_total / K / T,
                   "l2": f"inputs larger than L2: {3 * fb * T / 1e6:.0f} MB streamed per step, no flush needed",
                   "host_threads": threads, "host_cores": ncores, "warmup_steps_run": warm_steps, "describe": vb.describe()},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": T * ((fb + 64 * synth.N_WORKERS) if args.derive == "device" else (2 * fb + 2 * nD)),
                "d2h_bytes_per_step": T * fb,
                "ms_per_frame": 1e3 * e2e_total / (K * T), "ms_per_step_median": 1e3 * statistics.median(e2e_s),
                "stage_ms_last_call": stage, "derive": args.derive, "hash": args.hash, "hash_bands_on_gpu": (args.hash_bands or synth.N_WORKERS) if args.hash == "device" else 0, "batch": args.e2e_batch or cfg.batch, "n_streams": e2e_streams,
                "timer": "wall clock around vcrypt_encrypt_frames, pinned host in/out"},
        "gpu_launches": launches,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": NCU_TRAFFIC_PER_CALL.get(cfg.name),
                     "kernel": "row_pass_kernel<false> + col_enc_kernel<64> = one launch pair of vcrypt_encrypt_device "
                               f"(col_enc_kernel is the larger share, {NCU_COL_SHARE:.0%} in profiles/); the step is ONE call on the "
                               f"resident clip = {pairs_per_step} launch pairs alternating over 2 streams, so achieved = the step's "
                               "algorithmic bytes / its duration (CUDA events on the calling stream, which the internal stream "
                               "forks from and joins); single_stream_batches = the same frames as one call per batch on one stream",
                     "algorithmic_bytes_per_frame": alg_bytes_frame,
                     "launch_pairs_per_step": pairs_per_step,
                     "frames_per_launch_pair": T / pairs_per_step,
                     "algorithmic_bytes_per_launch_pair": alg_bytes_frame * T / pairs_per_step,
                     "us_per_launch_pair": 1e3 * kern_ms_total / K / pairs_per_step,
                     "single_stream_batches": {"frames_per_call": min(cfg.batch, T), "us_per_frame": 1e3 * batches_ms_frame,
                                               "us_per_call": 1e3 * batches_ms_frame * min(cfg.batch, T),
                                               "frac": alg_bytes_frame / (batches_ms_frame * 1e-3) / 1e9 / peak, "steps": KB},
                     "peak_source": peak_src, "frac_of_8TBs_nominal": achieved / 8000.0,
                     "step_ms_median": statistics.median(step_ms), "step_ms_min": min(step_ms),
                     # what the memory system allows for the same bytes (vcrypt_memory_probe, us per frame): a plain
                     # copy, the 5-trips-through-L2 traffic of any two-pass design, the column pass's strided DRAM side
                     "memory_probes_us_per_frame": probes,
                     "two_pass_ceiling_frac": (alg_bytes_frame / (probes["two_pass_traffic_sequential"] * 1e-6) / 1e9 / peak)
                     if probes.get("two_pass_traffic_sequential") else None},
        "e2e_decrypt": {"value": world * T / min(dec_s), "unit": UNIT, "ms_per_frame": 1e3 * min(dec_s) / T,
                        "note": "vcrypt_decrypt_frames from the start of the chain, best of 3 after one warm-up call, pinned host in/out, rank 0's time"},
        "decrypt_kernels": {"value": 1e3 / dec_ms_frame, "unit": UNIT, "us_per_frame": 1e3 * dec_ms_frame,
                            "frac": alg_bytes_frame / (dec_ms_frame * 1e-3) / 1e9 / peak, "steps": KD},
        "cpu_baseline": cpu_baseline, "clocks": clocks, "check": check,
        "context": {"paper_ms_per_fhd_frame": 25.84, "paper_hw": "Xeon Gold 6226R + RTX 3090 (PAPER.md:5, :568); not a target"},
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
