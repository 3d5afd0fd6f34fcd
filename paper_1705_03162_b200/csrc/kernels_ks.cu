// kernels_ks.cu — Kuramoto-Sivashinsky (App. C) kernel instantiations, FP64.
#include "kernels_persist_impl.cuh"
namespace swept {
int launch_per_step_ks(int dtype, int rk2, const PerStepLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  return rk2 == 0 ? per_step_T<KS<double, 0>, 4>(a) : per_step_T<KS<double, 1>, 4>(a);
}
// one launch per timestep: in = u^n, out = u^{n+1} (a.base and a.odd unused); P = 4 or 2 or 1 by divisibility
int launch_per_step_ks_fused(int dtype, int rk2, const PerStepLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  if (a.P == 4) return rk2 == 0 ? per_step_fused_go<KS<double, 0>, 4>(a) : per_step_fused_go<KS<double, 1>, 4>(a);
  if (a.P == 2) return rk2 == 0 ? per_step_fused_go<KS<double, 0>, 2>(a) : per_step_fused_go<KS<double, 1>, 2>(a);
  return NO_KERNEL;
}
bool tile_config_ok_ks(int dtype, int flavor, int64_t N, int n, int P) {
  if (dtype != 0) return false;
  if (flavor == SWEPT_FLAVOR_TIER) return tier_ok<KS<double, 0>>(n, P, 4);
  if (flavor == SWEPT_FLAVOR_CHAR) return char_ok<KS<double, 0>, 32>(N, n, P);
  if (flavor == SWEPT_FLAVOR_FLOW) return flow_ok<KS<double, 0>, 32>(N, n);
  if (flavor == SWEPT_FLAVOR_CLUSTER) return cluster_ok<KS<double, 0>>(N, n, P);
  return false;
}
int launch_tile_ks(int dtype, int rk2, const TileLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  if (a.flavor == SWEPT_FLAVOR_TIER) return rk2 == 0 ? tier_T<KS<double, 0>, 4>(a) : tier_T<KS<double, 1>, 4>(a);
  if (a.flavor == SWEPT_FLAVOR_CHAR) return rk2 == 0 ? char_T<KS<double, 0>, 32>(a) : char_T<KS<double, 1>, 32>(a);
  return NO_KERNEL;
}
int launch_flow_ks(int dtype, int rk2, const FlowLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  return rk2 == 0 ? flow_T<KS<double, 0>, 32>(a) : flow_T<KS<double, 1>, 32>(a);
}
int launch_cluster_ks(int dtype, int rk2, const ClusterLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  return rk2 == 0 ? cluster_T<KS<double, 0>>(a) : cluster_T<KS<double, 1>>(a);
}
int launch_resident_ks(int dtype, int rk2, const ResidentLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  return rk2 == 0 ? resident_T<KS<double, 0>, 8>(a) : resident_T<KS<double, 1>, 8>(a);
}
}  // namespace swept
