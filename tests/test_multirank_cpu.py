"""N > 1 path on the CPU (gloo, world_size 2).  The hot path does not shard (north_star: one GPU, no collectives), so
bench.py --gpus N runs N independent replicas; what the ranks share is the timing reduction
(max over ranks), the whole-job rate, the per-rank seeds, and the rule that only rank 0 prints."""
import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import pytest

torch = pytest.importorskip("torch")
ROOT = Path(__file__).resolve().parents[1]


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    import torch.distributed as dist

    sys.path.insert(0, str(ROOT))
    import bench

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        # rank r is "slower" by r ms in the first slot and faster in the second
        got = bench.max_over_ranks([10.0 + rank, 5.0 - rank, 1.0], world, "cpu")
        p = bench.make_problem("config1", rank)
        Path(out_dir, f"r{rank}.json").write_text(json.dumps({
            "max": got, "seed": p.meta["seed"], "n": p.N, "x0": float(p.pos[1, 0]),
            "rate": bench.whole_job_rate(world, 4, 100, got[0] * 1e-3)}))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_replica_seeds_world2(tmp_path):
    import torch.multiprocessing as mp

    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    r0, r1 = (json.loads((tmp_path / f"r{r}.json").read_text()) for r in (0, 1))
    assert r0["max"] == r1["max"] == [11.0, 5.0, 1.0]  # the slowest rank decides, on every rank
    assert r0["rate"] == pytest.approx(2 * 4 * 100 / 11e-3)  # whole job: both replicas' pairs over the slowest time
    assert r0["n"] == r1["n"] and r0["seed"] != r1["seed"] and r0["x0"] != r1["x0"]  # same recipe, different draw


def test_reference_arm_under_torchrun_prints_once(tmp_path):
    """bench.py --impl reference launched as the driver does for N = 2: rank 0 alone runs the oracle and prints."""
    env = dict(os.environ, OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "config1"]
    out = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
