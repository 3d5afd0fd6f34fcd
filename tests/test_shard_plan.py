"""Row f4: sharding the swept cycle with ONE edge exchange per phase.
Host-side bookkeeping only (no GPU): the library's phase list and exchange list, replayed by the exact-integer shard
model of tests/shard_sim.py for R shards in one process.  The multi-process version of the same check is
tests/test_shard_gloo.py; the kernels are checked in tests/test_gpu_shard.py."""
import pytest

import paper_1705_03162_b200 as sw
from shard_sim import GARBAGE, REM, ShardSim

CASES = [  # nshards, n_local, n, h, sigma, nsub
    (2, 64, 32, 1, 1, 16 * 5), (2, 64, 32, 1, 1, 16 * 6 + 7), (3, 32, 32, 1, 1, 100), (4, 128, 64, 2, 2, 16 * 7 + 8 + 6),
    (2, 128, 128, 2, 2, 32 * 4), (1, 128, 64, 1, 1, 200), (2, 256, 128, 2, 3, 3 * 77), (2, 128, 64, 2, 3, 16 * 6),
    (2, 64, 64, 1, 1, 0), (2, 64, 64, 1, 1, 5)]


def run_sharded(nshards, n_local, n, h, sigma, nsub):
    plan = sw.swept_plan(nsub, n, h, sigma)
    xch = sw.swept_shard_exchanges(plan, h, sigma, n_local)
    shards = [ShardSim(n_local, n, h, sigma) for _ in range(nshards)]
    ix = 0
    for i in range(-1, len(plan)):
        if i >= 0:
            for s in shards:
                s.phase(plan[i])
        while ix < len(xch) and xch[ix][0] == i:
            msgs = [s.pack(xch[ix]) for s in shards]           # everybody packs, then everybody receives
            for k, s in enumerate(shards):
                s.unpack(xch[ix], msgs[(k - xch[ix][1]) % nshards])
            ix += 1
    assert ix == len(xch)
    return plan, xch, shards


@pytest.mark.parametrize("nshards,n_local,n,h,sigma,nsub", CASES)
def test_sharded_schedule_is_exact(nshards, n_local, n, h, sigma, nsub):
    plan, xch, shards = run_sharded(nshards, n_local, n, h, sigma, nsub)
    for s in shards:
        assert s.own_level() == [nsub] * n_local, "every own point must reach the final tier; no garbage may leak in"
    # one message per swept phase that has a successor in its cycle (and per neighbour pair), alternating direction
    swept_phases = [i for i, p in enumerate(plan) if p[0] != REM]
    per_phase = {i: [x for x in xch if x[0] == i and x[5] > 1] for i in swept_phases}
    assert all(len(v) <= 1 for v in per_phase.values())
    dirs = [v[0][1] for i, v in sorted(per_phase.items()) if v]
    assert all(a != b for a, b in zip(dirs, dirs[1:])) or len({p[4] for p in plan if p[0] != REM}) > 1
    for x in xch:
        assert x[4] <= n // 2 + h, "an edge is at most half a tile plus the halo (SURVEY.md §8(e))"


def test_a_wrong_exchange_is_caught():
    # the model must be able to fail: drop one message and garbage reaches an own point
    n_local, n, h, sigma, nsub = 64, 32, 1, 1, 16 * 5
    plan = sw.swept_plan(nsub, n, h, sigma)
    xch = sw.swept_shard_exchanges(plan, h, sigma, n_local)
    for drop in range(len(xch)):
        shards = [ShardSim(n_local, n, h, sigma) for _ in range(2)]
        ix = 0
        for i in range(-1, len(plan)):
            if i >= 0:
                for s in shards:
                    s.phase(plan[i])
            while ix < len(xch) and xch[ix][0] == i:
                if ix != drop:
                    msgs = [s.pack(xch[ix]) for s in shards]
                    for k, s in enumerate(shards):
                        s.unpack(xch[ix], msgs[(k - xch[ix][1]) % 2])
                ix += 1
        assert any(GARBAGE in s.own_level() or s.own_level() != [nsub] * n_local for s in shards), drop


def test_message_volume_per_phase_matches_the_survey():
    # per phase one hand-off of 2 rows x n/2 x w bytes (plus the h halo points) each way
    n, h, n_local = 512, 1, 1 << 17
    plan = sw.swept_plan(10000, n, h, 1)
    xch = sw.swept_shard_exchanges(plan, h, 1, n_local)
    top = [x for x in xch if x[5] == 2 and x[4] == n // 2 + h]
    assert len(top) == sum(1 for p in plan if p[4] == n and p[0] != 3)
    per_step_messages = 2 * 10000          # a per-step scheme exchanges its halo every sub-timestep, both ways
    assert len(xch) < per_step_messages / 100


def test_exchange_list_rejects_bad_arguments():
    plan = sw.swept_plan(64, 32, 1)
    with pytest.raises(sw.SweptError):
        sw.swept_shard_exchanges(plan, 3, 1, 64)      # h must be 1 or 2
    with pytest.raises(sw.SweptError):
        sw.swept_shard_exchanges(plan, 1, 4, 64)      # sigma must be 1, 2 or 3
    with pytest.raises(sw.SweptError):
        sw.swept_shard_exchanges(plan, 1, 1, 0)       # n_local must be positive
    assert sw.swept_shard_exchanges([], 1, 1, 64) == []
