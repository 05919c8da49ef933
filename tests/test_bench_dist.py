"""World-size-2 gloo test (CPU) of bench.py's rank logic.  The path does not shard ("replicas only"):
ranks exchange timing scalars only -- barrier, max of the device time, sum of the processed units --
and the reference arm runs on rank 0 alone."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    r = bench.Ranks(world, "cpu")
    r.barrier()
    units, ms = [1.0e9, 3.0e9][rank], [2.0, 5.0][rank]       # rank 1 is slower and did more
    value, ms_max = r.job_value(units, ms)
    ref_rc = None
    if rank != 0:                                              # reference arm: other ranks do no work and exit 0
        class A:
            steps, warmup, config, coulomb, lj_rc, water_nside = 1, 0, 0, "ewald", 0.0, 0
        ref_rc = bench.run_reference(A())
    out.put((rank, value, ms_max, r.max(float(rank)), r.sum(1.0), ref_rc))
    r.barrier()
    dist.destroy_process_group()


def test_rank_aggregation_world2_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, ms_max, mx, sm, ref_rc in res:
        assert ms_max == 5.0
        assert abs(value - 4.0e9 / 5.0e-3) < 1e-3             # sum of units / max time, identical on both ranks
        assert mx == 1.0 and sm == 2.0
        assert ref_rc == (None if rank == 0 else 0)


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    r = bench.Ranks(1, "cpu")
    r.barrier()
    assert r.job_value(10.0, 2.0) == (10.0 / 2.0e-3, 2.0)
