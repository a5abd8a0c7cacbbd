"""The transport of the row-block decomposition (include/mpr.h, mpr_create_slab) on CPU: three gloo
ranks run DistSlabComm's all-reduce and halo exchange on host tensors (the path taken when the backend is not nccl).
The slab contexts themselves need a GPU: tests/test_gpu_slab.py runs them against a single context."""
import os
import socket
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class _NoStream:
    def synchronize(self):
        pass


def _worker(rank: int, world: int, port: int, out_dir: str) -> None:
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1811_01604_b200 import mpr
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        comm = mpr.DistSlabComm()
        assert comm.host and comm.rank == rank and comm.world == world
        res = {"sum": comm.allreduce([1.0 + rank, 0.5], 0), "min": comm.allreduce([10.0 - rank], 1),
               "max": comm.allreduce([float(rank), -float(rank)], 2)}
        n = 64
        up, down = rank > 0, rank < world - 1
        mk = lambda on, v: torch.full((n,), v, dtype=torch.uint8) if on else None
        send_up, send_down = mk(up, 10 * rank + 1), mk(down, 10 * rank + 2)
        recv_up, recv_down = mk(up, 255), mk(down, 255)
        for _ in range(3):                               # repeated exchanges do not cross
            comm.exchange(send_up, recv_up, send_down, recv_down, _NoStream())
        res["recv_up"] = None if recv_up is None else sorted(set(recv_up.tolist()))
        res["recv_down"] = None if recv_down is None else sorted(set(recv_down.tolist()))
        np.save(os.path.join(out_dir, f"rank{rank}.npy"), np.array([res], dtype=object), allow_pickle=True)
    finally:
        dist.destroy_process_group()


def test_dist_slab_comm_over_three_gloo_ranks(tmp_path):
    import torch.multiprocessing as mp
    world, port = 3, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    got = [np.load(tmp_path / f"rank{r}.npy", allow_pickle=True)[0] for r in range(world)]
    for r, g in enumerate(got):
        assert g["sum"] == [6.0, 1.5] and g["min"] == [8.0] and g["max"] == [2.0, 0.0]
        # the upper neighbour's send_down (its value 10 (r - 1) + 2), the lower neighbour's send_up (10 (r + 1) + 1)
        assert g["recv_up"] == (None if r == 0 else [10 * (r - 1) + 2])
        assert g["recv_down"] == (None if r == world - 1 else [10 * (r + 1) + 1])


def test_slab_geometry_host_checks():
    sys.path.insert(0, ROOT)
    import pytest
    from paper_1811_01604_b200 import build as mpr_build
    from paper_1811_01604_b200 import mpr
    mpr_build.build()                        # a fresh checkout has no library yet (nvcc cross-compiles without a GPU)
    mpr.lib()
    assert mpr.slab_local_rows(4096, 4096, 0, 2048) == (0, 2056)
    assert mpr.slab_local_rows(4096, 4096, 2048, 4096) == (2040, 2056)
    assert mpr.slab_local_rows(300, 64, 100, 200) == (92, 116)
    assert mpr.slab_local_rows(300, 64, 0, 300) == (0, 300)
    assert mpr.lib().mpr_slab_halo_bytes(4096) == 8 * 4096 * 8 and mpr.lib().mpr_slab_halo_bytes(51) == 8 * 52 * 8
    for bad in ((300, 64, 100, 90), (300, 64, -2, 90), (300, 64, 200, 302), (300, 64, 4, 296 + 8)):
        with pytest.raises(mpr.MprError) as e:
            mpr.slab_local_rows(*bad)
        assert e.value.name == "MPR_ERR_ARG"
