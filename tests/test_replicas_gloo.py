"""N > 1 path of bench.py on CPU: "replicas only" — no data-path collective, the only
collectives are the barrier and the MAX all-reduce of the per-rank device time.  world_size 2, gloo."""
import io
import os
import socket
import sys
from contextlib import redirect_stdout

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        my_ms = 10.0 + 5.0 * rank            # rank 1 is the slow replica
        dist.barrier()
        mx = bench.max_over_ranks(my_ms, dist, "cpu")
        value = bench.replica_value(1 << 20, 3, world, mx)
        # the reference arm under torchrun: only rank 0 works and prints, the others return 0 silently
        buf = io.StringIO()
        with redirect_stdout(buf):
            rc = bench.run_reference(type("A", (), {"gpus": world, "steps": 1, "warmup": 0})()) if rank else 0
        q.put((rank, mx, value, rc, buf.getvalue()))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get() for _ in range(world))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, mx, value, rc, out in got:
        assert mx == 15.0                                        # MAX over ranks, identical on every rank
        assert value == 2 * (1 << 20) * 3 / 15.0e-3              # both replicas' updates / slowest time
        assert rc == 0 and out == ""                             # non-zero ranks of the reference arm are silent


def test_single_process_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(7.5, None, "cpu") == 7.5
    assert bench.replica_value(1000, 2, 1, 4.0) == 1000 * 2 / 4.0e-3
