"""P10 — exact-integer simulation of the swept schedule, driven by the phase list the
LIBRARY's host-side planner (`swept_plan`, C ABI, no GPU needed) produces.

State: two ping-pong buffers of R global rows (R = 2 for one or two sub-timesteps per timestep, R = 3 for the
three-sub-timestep scheme of row f3); row p holds, per point, the tier index of the latest value
with tier = p (mod R) (or None).  Each phase does what a tile kernel does: load rows over [S-h, S+n+h) from the input
buffer, compute its tiers, write rows over [S, S+n) to the output buffer.  Every stencil read is asserted to
carry exactly the tier the scheme needs (t-1 for the 2h+1 window, t-2 for the own-point base of a final
stage), so a wrong range, shift, tier count or parity anywhere fails.  Counts are pinned to the paper's
printed numbers (65 792 values for n = 512; KS n = 32 -> 4 timesteps per cycle).
"""
import pytest

import paper_1705_03162_b200 as sw

UP, SPLIT, WHOLE, DOWN, REM = 0, 1, 2, 3, 4


def active_range(kind, t, n, h):
    m = n // (2 * h)
    if kind == UP:
        return h * t, n - h * t
    w = h * t if (kind == DOWN or t <= m) else h * (2 * m - t)
    return n // 2 - w, n // 2 + w


def simulate(N, n, h, sigma, nsub):
    R = 3 if sigma == 3 else 2
    plan = sw.swept_plan(nsub, n, h, sigma)
    bufs = [[[None] * N for _ in range(R)] for _ in range(2)]
    bufs[0][0] = [0] * N  # tier 0 everywhere in row 0
    cur, updates, launches = 0, 0, 0
    field_tier = 0
    for kind, shift, tier0, ntiers, n_ph in plan:
        if kind == REM:
            assert tier0 == field_tier and ntiers % sigma == 0
            field_tier += ntiers
            updates += N * ntiers
            launches += ntiers
            continue
        launches += 1
        assert n_ph <= n and n % n_ph == 0
        n = n_ph  # remainder cycles use narrower tiles (reading G5)
        src, dst = bufs[cur], bufs[1 - cur]
        new_dst = [list(row) for row in dst]
        assert N % n == 0 and shift in (0, n // 2)
        for tile in range(N // n):
            S = (shift + tile * n) % N
            # local copy of [S-h, S+n+h)
            loc = [[src[r][(S - h + j) % N] for j in range(n + 2 * h)] for r in range(R)]
            if kind == UP:
                assert tier0 % sigma == 0, "a cycle starts from a full time level"
                for r in range(1, R):
                    loc[r] = [None] * (n + 2 * h)
            for t in range(1, ntiers + 1):
                g = tier0 + t  # global tier
                par = g % R
                if R == 2:
                    assert par == t % 2, "phases of the two-row schemes must start on even tiers"
                stage = g % sigma  # 1 = first stage ... 0 = final stage of the timestep
                lo, hi = active_range(kind, t, n, h)
                assert 0 <= lo < hi <= n
                new_vals = {}
                for j in range(lo, hi):
                    for d in range(-h, h + 1):
                        assert loc[(g - 1) % R][h + j + d] == g - 1, (kind, t, j, d, loc[(g - 1) % R][h + j + d], g - 1)
                    if sigma >= 2 and stage != 1:
                        # own-point value at the start of the timestep (u^n): always in row 0
                        back = sigma if stage == 0 else stage
                        assert (g - back) % R == 0 and loc[0][h + j] == g - back, (kind, t, j, loc[0][h + j], g - back)
                    new_vals[j] = g
                for j, v in new_vals.items():
                    loc[par][h + j] = v
                updates += hi - lo
            rows_out = (0,) if kind == DOWN else tuple(range(R))
            for r in rows_out:
                for j in range(n):
                    new_dst[r][(S + j) % N] = loc[r][h + j]
        bufs[1 - cur] = new_dst
        cur = 1 - cur
        if kind == DOWN:
            field_tier = tier0 + ntiers
            assert field_tier % sigma == 0 and field_tier % R == 0
            assert all(v == field_tier for v in bufs[cur][0]), "Down must leave a full time level in row 0"
    assert field_tier == nsub
    assert updates == N * nsub, "the swept schedule performs exactly the per-step work (PAPER.md:37)"
    return plan, launches


@pytest.mark.parametrize("N,n,h,sigma,D", [
    (64, 16, 1, 1, 0), (64, 16, 1, 1, 1), (64, 16, 1, 1, 2), (64, 16, 1, 1, 3), (128, 32, 2, 2, 1),
    (128, 32, 2, 2, 2), (128, 32, 2, 2, 3), (64, 32, 2, 2, 3), (32, 32, 2, 2, 3), (256, 64, 2, 2, 5),
    (64, 32, 1, 1, 4), (32, 32, 1, 1, 2)])
def test_schedule_exact(N, n, h, sigma, D):
    m = n // (2 * h)
    plan, _ = simulate(N, n, h, sigma, (D + 1) * m)
    kinds = [p[0] for p in plan]
    assert kinds[0] == UP and kinds[-1] == DOWN and len(plan) == D + 2
    assert kinds[1:-1] == [SPLIT if k % 2 == 1 else WHOLE for k in range(1, D + 1)]


@pytest.mark.parametrize("nsub", [0, 2, 14, 16, 18, 46, 100])
def test_remainder_policy_g5(nsub):
    # nsub not a multiple of m: largest T = (D+1) m <= nsub by swept phases, the rest per-step (reading G5)
    N, n, h, sigma = 64, 32, 1, 1
    plan, _ = simulate(N, n, h, sigma, nsub)
    m = n // (2 * h)
    swept_part = sum(1 for p in plan if p[0] != REM)
    if nsub < m:
        assert swept_part == 0
    else:
        assert swept_part == nsub // m + 1
    rem = [p for p in plan if p[0] == REM]
    assert (len(rem) == 1 and rem[0][3] == nsub % m) if nsub % m else not rem


@pytest.mark.parametrize("N,n,h,sigma,nsub", [(256, 128, 1, 1, 64 + 32 + 16 + 5), (256, 128, 1, 1, 3 * 64 + 16),
                                              (256, 256, 2, 2, 64 + 2 * 16 + 8 + 6), (512, 128, 2, 2, 5 * 32 + 30),
                                              (128, 128, 1, 1, 1000)])
def test_multi_level_remainder_g5(N, n, h, sigma, nsub):
    # what a cycle of width n cannot cover goes to cycles of width n/2, n/4, ... >= 32, then per-step
    plan, launches = simulate(N, n, h, sigma, nsub)
    widths = [p[4] for p in plan if p[0] != REM]
    assert widths == sorted(widths, reverse=True) and widths[0] == n
    rem = sum(p[3] for p in plan if p[0] == REM)
    assert rem < 32 // (2 * h), "only less than the narrowest tile's m sub-timesteps go per-step"
    for w in set(widths):  # every cycle is Up, diamonds, Down
        kinds = [p[0] for p in plan if p[4] == w and p[0] != REM]
        assert kinds[0] == UP and kinds[-1] == DOWN and all(k in (SPLIT, WHOLE) for k in kinds[1:-1])
    assert launches < nsub or nsub < 32 // (2 * h)


def paper_values():
    """tests/golden/paper_values.txt: the numbers the paper itself prints, each with its citation."""
    import os
    out = {}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_values.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                out[k.strip()] = int(v)
    return out


def test_paper_counts():
    gold = paper_values()
    # the triangle of a 512-point node holds 65 792 values (incl. the initial row), h = 1
    n, h = 512, 1
    m = n // (2 * h)
    total = n + sum(active_range(UP, t, n, h)[1] - active_range(UP, t, n, h)[0] for t in range(1, m))
    assert total == gold["triangle_values_n512"] == 65792
    assert 2 * n == gold["triangle_two_row_values_n512"]
    # a 32-point node needs four times the launches of a 128-point node for the same timesteps (KS)
    nsub = 2 * 4096
    launches = {w: sum(1 for p in sw.swept_plan(nsub, w, 2) if p[4] == w) for w in (32, 128)}
    assert (launches[32] - 1) == gold["ks_launch_ratio_n32_vs_n128"] * (launches[128] - 1)
    # two global accesses (one read, one write of the edges) per n sub-timesteps: one launch per n/(2h)
    assert gold["global_accesses_per_n_substeps"] == 2 and launches[128] - 1 == nsub // (128 // 4)
    # KS with n = 32: four timesteps per cycle (m = n/(2h) = 8 sub-timesteps)
    plan = sw.swept_plan(2 * 4 * 3, 32, 2)
    assert plan[1][3] == 15 and plan[2][2] - plan[1][2] == 8
    # n sub-timesteps per pair of global accesses: a diamond advances n/h - 1 tiers at its centre
    assert sw.swept_plan(64 * 10, 64, 1)[1][3] == 63
    # launch counts: heat N=2^20 n=256, 50 000 steps: D + 2 launches (~392)
    plan = sw.swept_plan(50000, 256, 1)
    assert sum(1 for p in plan if p[4] == 256) == 50000 // 128 + 1 == 391


def test_plan_rejects_bad_arguments():
    with pytest.raises(sw.SweptError):
        sw.swept_plan(10, 48, 1)  # not a power of two
    with pytest.raises(sw.SweptError):
        sw.swept_plan(10, 64, 3)


@pytest.mark.parametrize("N,n,h,D", [(128, 32, 2, 2), (128, 32, 2, 5), (64, 32, 2, 8), (32, 32, 2, 2), (256, 64, 2, 5),
                                     (256, 128, 2, 2)])
def test_schedule_three_subtimesteps(N, n, h, D):
    # Row f3: three sub-timesteps per timestep on a three-row state.  m = n/(2h) is a power of two,
    # so a cycle ends on a full timestep only when (D+1) is a multiple of 3, and diamonds start on any stage.
    m = n // (2 * h)
    plan, _ = simulate(N, n, h, 3, (D + 1) * m)
    kinds = [p[0] for p in plan]
    assert kinds[0] == UP and kinds[-1] == DOWN and len(plan) == D + 2
    assert {p[2] % 3 for p in plan[1:]} == {0, 1, 2} or D < 3


@pytest.mark.parametrize("nsub", [0, 3, 21, 24, 27, 48, 3 * 61, 3 * 200])
def test_three_subtimesteps_remainder(nsub):
    # the widest cycle takes the largest multiple of 3 rows of tiles; narrower cycles and per-step stages the rest
    N, n, h = 128, 64, 2
    plan, _ = simulate(N, n, h, 3, nsub)
    for w in {p[4] for p in plan if p[0] != REM}:
        rows = [p for p in plan if p[4] == w and p[0] != REM]
        assert (len(rows) - 1) % 3 == 0
    rem = sum(p[3] for p in plan if p[0] == REM)
    assert rem % 3 == 0 and rem < 3 * (32 // (2 * h))


def test_plan_sigma_rejects_bad_arguments():
    with pytest.raises(sw.SweptError):
        sw.swept_plan(10, 64, 2, 3)   # nsub must be a whole number of timesteps (a multiple of sigma)
    with pytest.raises(sw.SweptError):
        sw.swept_plan(12, 64, 2, 4)   # sigma must be 1, 2 or 3
    # sigma = 3: every cycle has a multiple of 3 rows after the Up row
    plan = sw.swept_plan(3 * 100, 64, 2, 3)
    for w in {p[4] for p in plan if p[0] != REM}:
        assert (sum(1 for p in plan if p[4] == w and p[0] != REM) - 1) % 3 == 0
