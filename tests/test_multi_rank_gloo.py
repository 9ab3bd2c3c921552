"""N > 1 host logic on CPU: world_size 2 over gloo.

The path shards by frame with no data-path collective, so what there is to test is: every rank gets its own clip,
derives its own hashes / D / B through the production host path, the timing reduction is a max over ranks, the
whole-job rate counts every rank's frames, and the reference arm runs on rank 0 only.
"""
import json
import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    from paper_2505_07158_b200 import binding as vb
    from paper_2505_07158_b200 import parallel, synth

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        cfg = synth.CONFIGS["C2"]
        rcfg = parallel.rank_clip_config(cfg, rank, 3)
        frames = synth.video(rcfg, 3)
        v = vb.Vcrypt(synth.KEY, synth.GAMMA, synth.N_WORKERS, cfg.w, cfg.h, flags=vb.FLAG_HOST_ONLY, host_threads=2)
        hashes = [v.frame_hash(frames[k]) for k in range(3)]
        D, B = v.derive(hashes[0])
        # every rank's clip, hashes and key material differ
        mine = torch.tensor(list(hashes[0]) + list(B.reshape(-1)[:32]), dtype=torch.uint8)
        got = [torch.empty_like(mine) for _ in range(world)]
        dist.all_gather(got, mine)
        distinct = len({bytes(g.numpy().tobytes()) for g in got}) == world
        # timing reduction: max over ranks, element-wise
        red = parallel.max_over_ranks([1.0 + rank, 10.0 - rank])
        dist.barrier()
        q.put((rank, distinct, red, parallel.whole_job_rate(world, 3, 2, red[0]), synth.digest(frames)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_own_clips_and_max_reduction():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1]
    assert all(r[1] for r in res), "ranks produced identical clips or key material"
    for r in res:
        assert r[2] == [2.0, 10.0]              # max(1, 2), max(10, 9) on every rank
        assert r[3] == 2 * 3 * 2 / 2.0          # whole-job frames / slowest rank's time
    assert res[0][4] != res[1][4]               # different synthetic clips


def test_single_process_reduction_is_identity():
    from paper_2505_07158_b200 import parallel

    assert parallel.max_over_ranks([3.5, 1.25]) == [3.5, 1.25]
    assert parallel.whole_job_rate(1, 300, 10, 2.0) == 1500.0


def test_reference_arm_runs_on_rank_zero_only():
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(_free_port()))
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
           "--config", "C1"]
    r1 = subprocess.run(cmd, env=dict(env, RANK="1", LOCAL_RANK="1"), capture_output=True, text=True, timeout=300)
    assert r1.returncode == 0 and r1.stdout.strip() == ""
    r0 = subprocess.run(cmd, env=dict(env, RANK="0", LOCAL_RANK="0"), capture_output=True, text=True, timeout=300)
    assert r0.returncode == 0, r0.stderr
    line = json.loads(r0.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert np.isclose(line["value"], line["cpu_baseline"]["value"])
