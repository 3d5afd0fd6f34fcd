"""Row f4, the N > 1 path on CPU: one process per shard, world_size 2, gloo.  Each rank replays ITS shard with the
exact-integer model of tests/shard_sim.py, following the library's phase list and exchange list, and the edge
messages really travel between the processes through the package's own transport function
(`paper_1705_03162_b200._transport`: torch.distributed point-to-point; NCCL on a GPU node, gloo here).  What is
covered: who sends what to whom after which phase, message sizes, both directions, the per-step remainder's two-way
exchange, and that every own point of every rank ends at the final tier with no garbage from the ghost-zone tiles."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CASES = [(64, 32, 1, 1, 16 * 6 + 7), (128, 64, 2, 2, 16 * 7 + 8 + 6), (256, 128, 2, 3, 3 * 77)]


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import paper_1705_03162_b200 as sw
    from shard_sim import ShardSim
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        out = []
        for n_local, n, h, sigma, nsub in CASES:
            plan = sw.swept_plan(nsub, n, h, sigma)
            xch = sw.swept_shard_exchanges(plan, h, sigma, n_local)
            sim = ShardSim(n_local, n, h, sigma)
            # a second message names its sender, so that one delivered to the wrong rank, or back to its sender, fails
            ix, sent = 0, 0
            for i in range(-1, len(plan)):
                if i >= 0:
                    sim.phase(plan[i])
                while ix < len(xch) and xch[ix][0] == i:
                    msg = torch.tensor(sim.pack(xch[ix]), dtype=torch.int64)
                    sender = torch.tensor([rank, ix], dtype=torch.int64)
                    recv, who = torch.empty_like(msg), torch.empty_like(sender)
                    sw._transport(msg, recv, xch[ix][1], rank, world)
                    sw._transport(sender, who, xch[ix][1], rank, world)
                    assert who.tolist() == [(rank - xch[ix][1]) % world, ix], "message from the wrong neighbour"
                    sim.unpack(xch[ix], recv.tolist())
                    sent += msg.numel()
                    ix += 1
            out.append((sim.own_level() == [nsub] * n_local, ix, sent))
        q.put((rank, out))
    finally:
        dist.destroy_process_group()


def test_two_shards_two_processes_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get() for _ in range(world))
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert [r for r, _ in got] == [0, 1]
    for (_, a), (_, b) in [(got[0], got[1])]:
        assert a == b, "both ranks follow the same plan and move the same volume"
        for ok, nx, sent in a:
            assert ok and nx > 0 and sent > 0
