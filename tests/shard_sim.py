"""Exact-integer model of ONE shard of a sharded swept run, driven by the library's own
phase list (`swept_plan`) and exchange list (`swept_shard_exchanges`).  Test infrastructure, used by
tests/test_shard_plan.py (all shards in one process) and tests/test_shard_gloo.py (one process per shard, gloo).

A shard holds n_local own points and a ghost zone of n points behind them; its arrays are periodic in
Next = n_local + n, exactly as the library lays them out.  A value is the tier index it carries, or GARBAGE (-1).
Every tile of the extended array is computed, as the kernels do, but a point whose stencil inputs do not carry
exactly the tiers the scheme needs becomes GARBAGE instead of failing an assertion: the tiles inside the ghost zone
legitimately compute garbage, and the claim under test is that none of it ever reaches an own point — i.e. that the
exchange list (ranges, direction, rows, order) is right.
"""
GARBAGE = -1
UP, SPLIT, WHOLE, DOWN, REM = 0, 1, 2, 3, 4


def active_range(kind, t, n, h):
    m = n // (2 * h)
    if kind == UP:
        return h * t, n - h * t
    w = h * t if (kind == DOWN or t <= m) else h * (2 * m - t)
    return n // 2 - w, n // 2 + w


class ShardSim:
    def __init__(self, n_local, n_top, h, sigma):
        self.nl, self.ghost, self.h, self.sigma = n_local, n_top, h, sigma
        self.R = 3 if sigma == 3 else 2
        self.Next = n_local + n_top
        self.rows = [[GARBAGE] * self.Next for _ in range(self.R)]   # rows written by the last phase
        self.level = [0] * n_local + [GARBAGE] * n_top               # current full time level (tier 0 on own points)
        self.tier = 0
        self.updates_own = 0

    # ---- one entry of the phase list
    def phase(self, ph):
        kind, shift, tier0, ntiers, n = ph
        h, R, Next, sigma = self.h, self.R, self.Next, self.sigma
        if kind == REM:
            assert tier0 == self.tier
            for _ in range(ntiers):
                g = self.tier + 1
                old = self.level
                self.level = [g if all(old[(x + d) % Next] == g - 1 for d in range(-h, h + 1)) else GARBAGE
                              for x in range(Next)]
                self.tier = g
            return
        assert Next % n == 0
        src = [self.level] + [[GARBAGE] * Next for _ in range(R - 1)] if kind == UP else self.rows
        dst = [[GARBAGE] * Next for _ in range(R)]
        for tile in range(Next // n):
            S = (shift + tile * n) % Next
            loc = [[src[r][(S - h + j) % Next] for j in range(n + 2 * h)] for r in range(R)]
            for t in range(1, ntiers + 1):
                g = tier0 + t
                stage = g % sigma
                lo, hi = active_range(kind, t, n, h)
                new = {}
                for j in range(lo, hi):
                    ok = all(loc[(g - 1) % R][h + j + d] == g - 1 for d in range(-h, h + 1))
                    if sigma >= 2 and stage != 1:
                        ok = ok and loc[0][h + j] == g - (sigma if stage == 0 else stage)
                    new[j] = g if ok else GARBAGE
                for j, v in new.items():
                    loc[g % R][h + j] = v
            for r in ((0,) if kind == DOWN else range(R)):
                for j in range(n):
                    dst[r][(S + j) % Next] = loc[r][h + j]
        self.rows = dst
        if kind == DOWN:
            self.tier = tier0 + ntiers
            self.level = list(dst[0])

    # ---- one entry of the exchange list: what this shard sends, and where a received message lands
    def pack(self, x):
        _, _, src_off, _, count, rows = x
        srcs = [self.level] if rows == 1 else self.rows[:rows]
        return [row[(src_off + j) % self.Next] for row in srcs for j in range(count)]

    def unpack(self, x, msg):
        _, _, _, dst_off, count, rows = x
        dsts = [self.level] if rows == 1 else self.rows[:rows]
        for r, row in enumerate(dsts):
            for j in range(count):
                row[(dst_off + j) % self.Next] = msg[r * count + j]

    def own_level(self):
        return self.level[:self.nl]
