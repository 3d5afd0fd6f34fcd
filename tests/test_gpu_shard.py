"""GPU parity for row f4: the swept cycle cut into shards with one edge exchange per phase
(PAPER.md:21, 283, 303).  One GPU is all a test run has, so the shards of a problem live on the same device:
  * `swept_shard_run` — all shards in one process, each message one cudaMemcpyAsync between staging buffers;
  * one process per shard (world_size 2, gloo, both on cuda:0; their kernels never wait on one another — every
    message is a host-synchronised copy), through the phase-wise C ABI and the package's transport function, the only
    piece an 8-GPU node replaces (NCCL).
Either way the result must equal the unsharded oracle bit for bit: sharding only moves where tiles are computed.
SWEPT_POISON fills every slab (ghost zones included) with NaNs first, so garbage leaking from a ghost-zone tile shows."""
import os
import socket
import sys

import numpy as np
import pytest

import oracle
import paper_1705_03162_b200 as sw
import swept_inputs as si

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(autouse=True)
def poison(monkeypatch):
    monkeypatch.setenv("SWEPT_POISON", "1")


def sharded(w, nshards, n, flavor=sw.FLAVOR_AUTO, group=0):
    s = sw.SweptShards.from_workload(w, nshards, n)
    try:
        s.run(w.nsteps, flavor, group)
        return s.read(), s.last_launches
    finally:
        s.close()


@pytest.mark.parametrize("nshards", [1, 2, 4])
@pytest.mark.parametrize("flavor,group", [(sw.FLAVOR_TIER, 1), (sw.FLAVOR_CHAR, 32), (sw.FLAVOR_AUTO, 0)])
def test_heat_shards_match_oracle(nshards, flavor, group):
    w = si.heat_sines(4096, 8, 41, 1000 + 37)   # 8 cycles of n = 256 and a multi-level remainder
    ref = oracle.run_workload(w)
    got, _ = sharded(w, nshards, 256, flavor, group)
    assert np.array_equal(got, ref)


@pytest.mark.parametrize("make,n,flavor,group", [
    (lambda: si.ks_cos(8192, 42, 333), 256, sw.FLAVOR_CHAR, 32),
    (lambda: si.ks_cos(8192, 42, 333), 512, sw.FLAVOR_TIER, 2),
    (lambda: si.ks3_cos(4096, 43, 211), 256, sw.FLAVOR_TIER, 1),
    (lambda: si.euler_double_sod(2048, 150), 128, sw.FLAVOR_TIER, 1),
    (lambda: si.euler_double_sod(2048, 150, rk2=si.RK2_MIDPOINT), 256, sw.FLAVOR_AUTO, 0)])
def test_other_problems_two_and_four_shards(make, n, flavor, group):
    w = make()
    ref = oracle.run_workload(w)
    for nshards in (2, 4):
        got, _ = sharded(w, nshards, n, flavor, group)
        assert np.array_equal(got, ref), nshards


def test_shards_equal_the_unsharded_library_run_at_config_size():
    # heat N = 2^20 cut into 8 shards of 2^17 points (the per-GPU size of an 8-GPU node), 2000 steps, n = 512
    w = si.heat_sines(1 << 20, 16, 44, 2000)
    s = sw.Swept.from_workload(w)
    s.run(w.nsteps, 512, sw.SWEPT, sw.FLAVOR_CHAR, 32)
    whole = s.read()
    s.close()
    got, launches = sharded(w, 8, 512, sw.FLAVOR_CHAR, 32)
    assert np.array_equal(got, whole)
    plan = sw.swept_plan(w.nsteps, 512, 1)
    xch = sw.swept_shard_exchanges(plan, 1, 1, (1 << 20) // 8)
    assert launches <= 8 * (len(plan) + 16 + 2 * len(xch))


def test_shard_argument_checks():
    w = si.heat_sines(4096, 8, 45, 10)
    with pytest.raises(sw.SweptError):
        sw.SweptShards.from_workload(w, 3, 256)            # N not a multiple of nshards * tile_width
    s = sw.SweptShards.from_workload(w, 2, 256)
    try:
        with pytest.raises(sw.SweptError):
            s.run(10, sw.FLAVOR_FLOW)                       # persistent flavour: no phase boundary to exchange at
        with pytest.raises(sw.SweptError):
            sw.swept_run(s._states[0], 10, 256, sw.SWEPT)   # a shard cannot advance alone
    finally:
        s.close()


# ---------------------------------------------------------------- one process per shard
def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      SWEPT_POISON="1")
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import paper_1705_03162_b200 as sw_
    import swept_inputs as si_
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        out = {}
        for name, w, n in (("heat", si_.heat_sines(4096, 8, 41, 500 + 21), 256), ("ks", si_.ks_cos(4096, 42, 100), 256)):
            s = sw_.SweptShards.from_workload(w, world, n, ranks=(rank, world))
            s.run(w.nsteps)
            out[name] = s.read()
            s.close()
        q.put((rank, out))
    finally:
        dist.destroy_process_group()


def test_one_process_per_shard_gloo_transport():
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_rank_main, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = dict(q.get() for _ in range(world))
    for p in procs:
        p.join(300)
        assert p.exitcode == 0
    for name, w in (("heat", si.heat_sines(4096, 8, 41, 500 + 21)), ("ks", si.ks_cos(4096, 42, 100))):
        ref = oracle.run_workload(w)
        glued = np.concatenate([got[r][name] for r in range(world)])
        assert np.array_equal(glued, ref), name
