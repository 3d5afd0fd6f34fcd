"""swept_heat_flow_static (include/swept.h "an entry point that allocates nothing"): one swept cycle of the heat problem by
the persistent FLOW kernel with every byte of scratch — counters, per-tile flags, three row slabs — in a file-scope
static device array of the library, for callers that cannot call cudaMalloc.  Checked against the existing path
(swept_create / swept_run with the FLOW flavour; same kernel and functor, so the expected difference is zero; the gate is
the 1e-12 of the other FP64 tests) on two calls in a row that share the array, then on a different size, then the
refusals.  Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`.
"""
import numpy as np
import pytest

import paper_1705_03162_b200 as sw
import swept_inputs as si

pytestmark = pytest.mark.gpu
TOL = 1e-12


def relerr(got, ref):
    return float(np.max(np.abs(got - ref)) / max(float(np.max(np.abs(ref))), 1e-300))


def existing_path(w, n, nsteps_list):
    """The field after each cumulative step count, from a swept_state advanced with the FLOW flavour."""
    s = sw.Swept.from_workload(w)
    out = []
    try:
        for k in nsteps_list:
            s.run(k, n, sw.SWEPT, sw.FLAVOR_FLOW)
            out.append(s.read().copy())
    finally:
        s.close()
    return out


def test_static_scratch_entry_point_matches_existing_path_twice_in_a_row():
    import torch
    N, n = 8192, 256
    m = n // 2
    steps1, steps2 = 5 * m, 2 * m                  # 6 rows of tiles (odd D), then 3 (even D): both buffer parities
    w = si.heat_sines(N, 8, 61, steps1 + steps2)
    ref1, ref2 = existing_path(w, n, [steps1, steps2])

    u0 = torch.from_numpy(np.ascontiguousarray(w.u0)).cuda()
    a = torch.full_like(u0, float("nan"))          # outputs start as NaNs: every point must be written
    b = torch.full_like(u0, float("nan"))
    sw.swept_heat_flow_static(u0.data_ptr(), a.data_ptr(), N, steps1, n, w.dx, w.dt, w.alpha)
    # second call straight after the first, same stream, same static scratch, the first call's output as its input
    sw.swept_heat_flow_static(a.data_ptr(), b.data_ptr(), N, steps2, n, w.dx, w.dt, w.alpha)
    sw.swept_heat_flow_static_check()
    got1, got2 = a.cpu().numpy(), b.cpu().numpy()
    assert np.all(np.isfinite(got1)) and np.all(np.isfinite(got2))
    assert relerr(got1, ref1) <= TOL and relerr(got2, ref2) <= TOL
    assert np.array_equal(got1, ref1) and np.array_equal(got2, ref2), "same kernel, same functor: expected 0 ulp"
    assert np.array_equal(u0.cpu().numpy(), w.u0), "the input buffer is read-only"

    # the same call again allocates nothing: free device memory is unchanged (all tensors exist already)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        sw.swept_heat_flow_static(u0.data_ptr(), a.data_ptr(), N, steps1, n, w.dx, w.dt, w.alpha)
    sw.swept_heat_flow_static_check()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    assert np.array_equal(a.cpu().numpy(), ref1), "the scratch keeps the last call's contents; the result must not depend on it"


@pytest.mark.parametrize("N,n,rows_after_up", [(sw.STATIC_MAX_N, 512, 4), (4096, 1024, 1), (1024, 1024, 3), (512, 256, 2)])
def test_static_scratch_other_sizes(N, n, rows_after_up):
    import torch
    steps = rows_after_up * (n // 2)
    w = si.heat_sines(N, 16, 62, steps)
    (ref,) = existing_path(w, n, [steps])
    u0 = torch.from_numpy(np.ascontiguousarray(w.u0)).cuda()
    out = torch.full_like(u0, float("nan"))
    sw.swept_heat_flow_static(u0.data_ptr(), out.data_ptr(), N, steps, n, w.dx, w.dt, w.alpha)
    sw.swept_heat_flow_static_check()
    got = out.cpu().numpy()
    assert relerr(got, ref) <= TOL and np.array_equal(got, ref)


def test_static_scratch_refusals():
    import torch
    big = 2 * sw.STATIC_MAX_N
    x = torch.zeros(big, dtype=torch.float64, device="cuda")
    y = torch.zeros(big, dtype=torch.float64, device="cuda")
    dx = 1.0 / big
    with pytest.raises(sw.SweptError, match="maximum N"):          # beyond the static array
        sw.swept_heat_flow_static(x.data_ptr(), y.data_ptr(), big, 256, 512, dx, 0.25 * dx * dx)
    with pytest.raises(sw.SweptError, match="multiple of tile_width / 2"):
        sw.swept_heat_flow_static(x.data_ptr(), y.data_ptr(), 4096, 100, 256, dx, 0.25 * dx * dx)
    with pytest.raises(sw.SweptError, match="tile_width"):
        sw.swept_heat_flow_static(x.data_ptr(), y.data_ptr(), 4096, 64, 128, dx, 0.25 * dx * dx)
    with pytest.raises(sw.SweptError, match="overlap"):
        sw.swept_heat_flow_static(x.data_ptr(), x.data_ptr() + 8 * 1024, 4096, 128, 256, dx, 0.25 * dx * dx)
    with pytest.raises(sw.SweptError, match="null"):
        sw.swept_heat_flow_static(0, y.data_ptr(), 4096, 128, 256, dx, 0.25 * dx * dx)
