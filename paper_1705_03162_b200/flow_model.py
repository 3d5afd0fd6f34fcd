"""Discrete-event model of one persistent FLOW launch: is the measured throughput explained by the issue
rate of the sweep and the tile dependencies alone?

    python -m paper_1705_03162_b200.flow_model [--K 2048] [--rows 40] [--B 16]

Model: 148 x 4 schedulers; `wps` resident warps per scheduler, each a task loop (ticket -> wait for the two parent tiles
of the previous row -> stage -> sweep m + L super-steps -> publish); the warps of a scheduler that are sweeping share it:
with `a` of them active each advances one super-step per cycles[a] SM cycles — the table `swept_probe_sweep` measures
(profiles/r2_probes.csv; heat FP64).  Tickets are row-major; tile (r, k) needs tiles k, k+1 (r odd) or k-1, k (r even) of
row r-1.  Per-tile overheads are the instrumented kernel's (profiles/r2_flow_phases.csv): ticket + flag reads ~1.7 k cycles,
staging + publishing ~6 k.  Output: updates per second at 1965 MHz and the share of warp time spent waiting for parents.
A measurement-analysis tool like sweep.py; no library code, nothing here runs on the GPU.
"""
from __future__ import annotations

import argparse
import heapq

#: SM cycles per super-step with `a` warps of a scheduler active (all of them advance one step), heat FP64
CYCLES = {8: {1: 197.4, 2: 208.6, 3: 232.7, 4: 267.8, 6: 360.0, 8: 469.5},
          16: {1: 202.2, 2: 260.2, 3: 349.2, 4: 447.6, 6: 653.8},
          32: {1: 631.4, 2: 656.6, 3: 735.3}}


def simulate(K: int, rows: int, B: int, wps: int, nsched: int = 592, flag_cost: float = 1700.0, io_cost: float = 6000.0):
    cyc = CYCLES[B]
    steps = 32 * B // 2 + 32  # m + L super-steps of a heat tile (h = 1)

    def rate(a):
        if a in cyc:
            return 1.0 / cyc[a]
        lo = max(x for x in cyc if x <= a)
        return 1.0 / (cyc[lo] * a / lo)

    ntasks, W = K * rows, nsched * wps
    done = [False] * ntasks
    active = [dict() for _ in range(nsched)]  # scheduler -> {warp: remaining super-steps}
    last = [0.0] * nsched
    waiting, kids, since, task = {}, {}, {}, {}
    ev, nxt, waited = [], 0, 0.0

    def parents(t):
        r, k = divmod(t, K)
        if r == 0:
            return []
        p = (k, (k + 1) % K) if r & 1 else ((k - 1) % K, k)
        return [(r - 1) * K + p[0], (r - 1) * K + p[1]]

    def advance(s, now):
        a = len(active[s])
        if a:
            d = (now - last[s]) * rate(a)
            for w in active[s]:
                active[s][w] -= d
        last[s] = now

    def next_finish(s, now):
        if active[s]:
            w = min(active[s], key=active[s].get)
            heapq.heappush(ev, (now + max(active[s][w], 0.0) / rate(len(active[s])), 1, s, w))

    def take(w, now):
        nonlocal nxt
        if nxt >= ntasks:
            return
        t, nxt = nxt, nxt + 1
        ps = [p for p in parents(t) if not done[p]]
        if ps:
            since[w] = now
            waiting[w] = [t, set(ps)]
            for p in ps:
                kids.setdefault(p, []).append(w)
        else:
            heapq.heappush(ev, (now + flag_cost + io_cost / 2, 2, w, t))

    for w in range(W):
        take(w, 0.0)
    now = 0.0
    while ev:
        now, kind, x, y = heapq.heappop(ev)
        if kind == 1:  # a warp of scheduler x may have finished its sweep
            if y not in active[x]:
                continue
            advance(x, now)
            if active[x][y] > 1e-6:
                next_finish(x, now)
                continue
            del active[x][y]
            next_finish(x, now)
            heapq.heappush(ev, (now + io_cost / 2, 3, y, 0))
        elif kind == 2:  # staged: start sweeping
            s = x % nsched
            advance(s, now)
            active[s][x] = float(steps)
            task[x] = y
            next_finish(s, now)
        else:  # published
            t = task[x]
            done[t] = True
            for cw in kids.pop(t, []):
                waiting[cw][1].discard(t)
                if not waiting[cw][1]:
                    ct = waiting.pop(cw)[0]
                    waited += now - since.pop(cw)
                    heapq.heappush(ev, (now + flag_cost + io_cost / 2, 2, cw, ct))
            take(x, now)
    return now, waited / (W * now)


def main(argv=None) -> int:
    ap = argparse.ArgumentParser()
    ap.add_argument("--K", type=int, default=2048, help="tiles per row (N / n)")
    ap.add_argument("--rows", type=int, default=40, help="rows of tiles in the launch (D + 2)")
    ap.add_argument("--B", type=int, default=16, help="lines per lane (n / 32)")
    args = ap.parse_args(argv)
    n, m = 32 * args.B, 16 * args.B
    print(f"heat FP64, N = {args.K * n}, n = {n}, {args.rows} rows ({(args.rows - 1) * m} timesteps per launch)")
    print("CTAs/SM, resident warps, model ms, model updates/s, waiting share")
    for wps in (1, 2, 3, 4, 6):
        if wps not in CYCLES[args.B] and wps > max(CYCLES[args.B]):
            continue
        cycles, wait = simulate(args.K, args.rows, args.B, wps)
        sec = cycles / 1.965e9
        print(f"{wps},{592 * wps},{sec * 1e3:.3f},{args.K * n * (args.rows - 1) * m / sec:.3e},{wait:.3f}")
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
