"""GPU parity for the CLUSTER flavour (include/swept.h SWEPT_FLAVOR_CLUSTER): the whole domain in one
thread-block cluster, a warp per tile in registers, rows of tiles chained by stores into the next tiles' shared memory
(st.async + mbarrier: the device-side synchronisation PAPER.md:297-303 names as future work; the survey's row f2).  Same
functors as every other flavour, so the result must equal the oracle bit for bit."""
import numpy as np
import pytest

import oracle
import paper_1705_03162_b200 as sw
import swept_inputs as si

pytestmark = pytest.mark.gpu
CL = sw.FLAVOR_CLUSTER


def admissible(problem, N, n, wpc, size=8):
    """The rules of include/swept.h / DESIGN.md §5.10, restated: which (N, n, warps per CTA) must run."""
    h, _, C = si.PROBLEM_SHAPE[problem]
    if n not in (32, 64, 128, 256, 512) or N % n or problem not in (si.HEAT, si.KS):
        return False
    if n == 32 and problem != si.HEAT:          # one point per lane: the three-point scheme only (a lane's block must hold h points)
        return False
    K, P = N // n, n // 32
    max_wpc = 8 if P >= 8 else 16
    for cand in (1, 2, 4, 8, 16, 32):
        if (cand != wpc) if wpc else (cand < 4 and K > cand):
            continue
        if cand > max_wpc or K % cand or K // cand > 16 or 2 * 2 * C * cand * n * size > 200 * 1024:
            continue
        return True
    return False


def run(w, n, wpc=0, dtype=np.float64):
    s = sw.Swept.from_workload(w, dtype=dtype)
    try:
        s.run(w.nsteps, n, sw.SWEPT, CL, wpc)
        return s.read(), s.last_launches
    finally:
        s.close()


@pytest.mark.parametrize("N,nsteps", [(64, 40), (256, 7), (2048, 300), (4096, 1000), (8192, 517), (1536, 200)])
def test_heat_cluster_matches_oracle(N, nsteps):
    w = si.heat_sines(N, 8, 51, nsteps)
    ref = oracle.run_workload(w)
    ran = 0
    for n in (32, 64, 128, 256, 512):
        for wpc in (0, 1, 4, 8, 16, 32):
            want = admissible(si.HEAT, N, n, wpc)
            try:
                got, _ = run(w, n, wpc)
            except sw.SweptError as e:
                assert not want, f"library refused n={n} wpc={wpc}: {e}"
                continue
            assert want, f"library ran the inadmissible n={n} wpc={wpc}"
            assert np.array_equal(got, ref), (n, wpc)
            ran += 1
    assert ran >= 2


@pytest.mark.parametrize("rk2", [si.RK2_MIDPOINT, si.RK2_HEUN])
@pytest.mark.parametrize("N,nsteps", [(128, 30), (2048, 150), (16384, 333)])
def test_ks_cluster_matches_oracle(N, nsteps, rk2):
    w = si.ks_cos(N, 52, nsteps)
    w.rk2 = rk2
    ref = oracle.run_workload(w)
    ran = 0
    for n in (32, 64, 128, 256, 512):
        for wpc in (0, 8):
            want = admissible(si.KS, N, n, wpc)
            try:
                got, _ = run(w, n, wpc)
            except sw.SweptError as e:
                assert not want, f"library refused n={n} wpc={wpc}: {e}"
                continue
            assert want, (n, wpc)
            assert np.array_equal(got, ref), (n, wpc)
            ran += 1
    assert ran >= 2


@pytest.mark.parametrize("N,nsteps", [(64, 50), (256, 333), (2048, 700), (8192, 1029)])
def test_heat_insulated_ends_cluster(N, nsteps):
    # the paper's own heat boundary condition (B.5) in the register-resident flavour: the lanes next to a wall take the
    # mirror image of their own neighbour point instead of the shuffled value; K = 1 (one tile holds both walls), the
    # split tile of the shifted rows, multi-level remainders; FP64 and FP32; slabs poisoned with NaNs
    import os
    os.environ["SWEPT_POISON"] = "1"
    try:
        w = si.heat_insulated(N, 6, 57, nsteps)
        ref = oracle.run_workload(w)
        ran = 0
        for n in (32, 64, 128, 256, 512):
            for wpc in (0, 8):
                if not admissible(si.HEAT, N, n, wpc):
                    continue
                got, _ = run(w, n, wpc)
                assert np.array_equal(got, ref), (n, wpc)
                ran += 1
        assert ran >= 1
        s = sw.Swept.from_workload(w)            # library default at these sizes: this flavour
        s.run(nsteps, 0, sw.SWEPT)
        assert np.array_equal(s.read(), ref)
        s.close()
        ref32 = oracle.run_workload(w, dtype=np.float32)
        got32, _ = run(w, 64, 0, dtype=np.float32)
        assert np.array_equal(got32, ref32)
    finally:
        del os.environ["SWEPT_POISON"]


def test_heat_fp32_cluster():
    w = si.heat_sines(4096, 16, 53, 700)
    ref = oracle.run_workload(w, dtype=np.float32)
    for n in (128, 256):
        got, _ = run(w, n, 0, dtype=np.float32)
        assert np.array_equal(got, ref)


def test_config1_full_length_cluster():
    # BASELINE.json configs[0]: heat N = 2048, 20 000 steps — the regime this flavour is for
    w = si.config(1)
    ref = oracle.run_workload(w)
    got, launches = run(w, 256)
    assert np.array_equal(got, ref)
    assert launches <= 12, "one launch per cycle (plus the few narrower cycles and stages of the remainder)"


def test_cluster_refusals():
    w = si.heat_sines(1 << 20, 8, 54, 10)
    with pytest.raises(sw.SweptError):
        run(w, 256)                       # 4096 tiles do not fit one cluster
    e = si.euler_double_sod(2048, 10)
    with pytest.raises(sw.SweptError):
        run(e, 128)
    k3 = si.ks3_cos(2048, 56, 10)
    with pytest.raises(sw.SweptError):
        run(k3, 512)                      # three register rows per lane: n <= 256 (tests/test_gpu_ks3.py covers the rest)
    tube = si.euler_sod(2048, 10)
    with pytest.raises(sw.SweptError):
        run(tube, 128)                    # walls in this flavour: the heat problem only


def test_probe_tier_chain():
    # the floor of this flavour's time per tier, measured by the library itself (include/swept.h swept_probe_tier):
    # a shuffle round trip, the neighbour sum and the update, the window select — each link adds latency
    runs = [sw.swept_probe_tier() for _ in range(3)]
    t = tuple(min(r[i] for r in runs) for i in range(4))   # a pre-empted run reads high: the minimum is the latency
    assert len(t) == 4 and all(x > 0 for x in t)
    assert 10 < t[0] < 80 and t[0] < t[1] < t[2] < 300 and 8 < t[3] < 80
