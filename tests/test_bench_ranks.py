"""The N > 1 path of bench.py on CPU: world_size 2 over gloo (replicas only).

The CUDA path itself cannot run here; what runs is the rank plumbing around
it: per-rank replica seeds, MAX-over-ranks times and SUM-over-ranks counts,
and the reference arm under torch.distributed.run (rank 0 alone works and
prints the JSON line, the other rank exits 0 without output).
"""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str) -> None:
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        # rank r took (1 + r) s for its steps and (0.5 - 0.1 r) s for the probe; it did 100 (r + 1) updates, 7 launches
        times, counts = bench.combine_over_ranks([1.0 + rank, 0.5 - 0.1 * rank], [100.0 * (rank + 1), 7.0])
        with open(os.path.join(out_dir, f"rank{rank}.json"), "w") as f:
            json.dump({"times": times, "counts": counts, "seed": bench.replica_seed(3004, rank)}, f)
    finally:
        dist.destroy_process_group()


def test_combine_over_two_gloo_ranks(tmp_path):
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    got = [json.load(open(tmp_path / f"rank{r}.json")) for r in range(world)]
    for g in got:                       # every rank sees the whole-job numbers
        assert g["times"] == [2.0, 0.5]             # MAX over ranks
        assert g["counts"] == [300.0, 14.0]         # SUM over ranks
    assert got[0]["seed"] != got[1]["seed"]         # independent replicas


def test_combine_without_a_process_group_is_the_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.combine_over_ranks([1.5, 2.5], [3, 4]) == ([1.5, 2.5], [3.0, 4.0])


@pytest.mark.timeout(600)
def test_reference_arm_under_torchrun_prints_one_line_from_rank_0():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(port),
           os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1",
           "--workload", "cfg1"]
    env = dict(os.environ, OMP_NUM_THREADS="2")
    r = subprocess.run(cmd, cwd=ROOT, env=env, capture_output=True, text=True, timeout=580)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"] == "cfg1"
