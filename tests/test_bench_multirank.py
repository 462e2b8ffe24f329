"""The N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only, so the multi-rank
logic is the max-over-ranks timing, the whole-job aggregation and "rank 0 alone prints"."""
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [3.0, 7.5][rank]                       # rank 1 is the slow one
    slowest = bench.max_over_ranks(ms, device="cpu")
    dist.barrier()
    out.put((rank, slowest, bench.whole_job_value(world, 1000, 10, slowest)))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, slowest, value in got:
        assert slowest == 7.5                                  # every rank reports the slowest rank's time
        assert value == pytest.approx(2 * 1000 * 10 / 7.5e-3)  # both replicas' cell-solves over that time


def test_single_process_helpers_need_no_process_group():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.max_over_ranks(4.25, device="cpu") == 4.25
    assert bench.whole_job_value(1, 65536, 20, 10.0) == pytest.approx(65536 * 20 / 0.01)
    assert bench.algorithmic_bytes_per_cell_solve(64, 1) == 8 * 64 * 64 + 24 * 64 + 64
    assert bench.structured_bytes_per_cell_solve(64, 1) == 36 * 64 + 136 + 64 + 8


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "3", "--ref-cells", "64"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["value"] > 0
