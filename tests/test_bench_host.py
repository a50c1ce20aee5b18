"""Host logic of bench.py without a GPU: the N>1 reduction (world-size-2 gloo), the byte model, the reference arm."""
import json
import os
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local_ms = [40.0, 50.0][rank]                      # rank 1 is the slow replica
    total = bench.max_over_ranks(local_ms, world)
    q.put((rank, total, bench.job_gedges(1_000_000, 10, world, total)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregate_uses_slowest_rank():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in procs]
    res = sorted(q.get(timeout=120) for _ in range(2))
    [p.join(timeout=60) for p in procs]
    for _, total, value in res:
        assert total == 50.0
        assert abs(value - 2 * 1_000_000 * 10 / 0.050 * 1e-9) < 1e-12
    assert bench.max_over_ranks(7.0, 1) == 7.0


def test_byte_model_counts():
    n, e, H, d = 100, 1000, 4, 64
    c = dict(n=n, e=e, heads=H, head_dim=d, dtype="bf16", layer="gt")
    deg = np.full(n, 10, np.int64)
    perm = np.arange(n)
    cnt = dict(n_hub=1, n_cta=9, n_group=90, n_chunks=3, n_hub_t=0, n_cta_t=0, n_group_t=100, n_chunks_t=0)
    alg, comp = bench.byte_model(c, cnt, deg, deg, perm, perm)
    R, b = H * d, 2
    assert alg["gt_fwd/group"] == 900 * (4 + 2 * R * b) + 90 * (8 + 2 * R * b + 4 * H)
    assert alg["gt_fwd/segment"] == 100 * (4 + 2 * R * b) + 12 * (8 + 2 * R * b + 4 * H)
    assert alg["gt_bwd_src/group"] == 1000 * (4 + 2 * R * b + 8 * H) + 100 * (8 + 2 * R * b + 8 * R)
    assert comp["fwd"] == 4 * (n + 1) + 4 * e + 4 * n * R * b + 4 * n * H


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--cfg", "1", "--steps", "2",
                          "--warmup", "1", "--cpu-seconds", "1"], capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "GEdges/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["config"]["workload"] == "cfg1_gt_er1k_f32"
