// kernels_euler.cu — Euler equations / Sod tube (App. D) host dispatch, FP64.
// The swept kernels themselves are instantiated in kernels_euler_inst.cu, compiled once per
// (flavour, integrator) slice so that the slices build in parallel (see build.py).
#include "kernels_persist_impl.cuh"
namespace swept {
extern template int tier_T<Euler<double, 0>, 4>(const TileLaunch&);
extern template int tier_T<Euler<double, 1>, 4>(const TileLaunch&);
extern template int char_L<Euler<double, 0>, 8>(const TileLaunch&);
extern template int char_L<Euler<double, 1>, 8>(const TileLaunch&);

int launch_per_step_euler(int dtype, int rk2, const PerStepLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  if (a.N < 8) return NO_KERNEL;
  return rk2 == 0 ? per_step_lane_go<Euler<double, 0>>(a) : per_step_lane_go<Euler<double, 1>>(a);
}
bool tile_config_ok_euler(int dtype, int flavor, int64_t N, int n, int P) {
  if (dtype != 0) return false;
  if (flavor == SWEPT_FLAVOR_TIER) return tier_ok<Euler<double, 0>>(n, P, 4);
  // CHAR for Euler: B = 8 lines per lane only (24 state registers per lane on top of ~250 live ones of the flux; the
  // B = 16 instantiations took 7 minutes each to compile and never won a sweep)
  if (flavor == SWEPT_FLAVOR_CHAR) return char_ok<Euler<double, 0>, 8>(N, n, P);
  return false;
}
int launch_tile_euler(int dtype, int rk2, const TileLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  if (a.flavor == SWEPT_FLAVOR_TIER)
    return rk2 == 0 ? tier_T<Euler<double, 0>, 4>(a) : tier_T<Euler<double, 1>, 4>(a);
  if (a.flavor == SWEPT_FLAVOR_CHAR)
    return rk2 == 0 ? char_T<Euler<double, 0>, 8>(a) : char_T<Euler<double, 1>, 8>(a);
  return NO_KERNEL;
}
int launch_resident_euler(int dtype, int rk2, const ResidentLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  return rk2 == 0 ? resident_T<Euler<double, 0>, 2>(a) : resident_T<Euler<double, 1>, 2>(a);
}
}  // namespace swept
