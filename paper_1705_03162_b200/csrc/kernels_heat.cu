// kernels_heat.cu — heat equation (App. B) kernel instantiations, FP64 and FP32.
#include "kernels_persist_impl.cuh"
namespace swept {
int launch_per_step_heat(int dtype, const PerStepLaunch& a) {
  return dtype == 0 ? per_step_T<Heat<double>, 4>(a) : per_step_T<Heat<float>, 4>(a);
}
bool tile_config_ok_heat(int dtype, int flavor, int64_t N, int n, int P) {
  if (flavor == SWEPT_FLAVOR_TIER) return dtype == 0 ? tier_ok<Heat<double>>(n, P, 4) : tier_ok<Heat<float>>(n, P, 4);
  if (flavor == SWEPT_FLAVOR_CHAR) return dtype == 0 ? char_ok<Heat<double>, 32>(N, n, P) : char_ok<Heat<float>, 32>(N, n, P);
  if (flavor == SWEPT_FLAVOR_FLOW) return dtype == 0 ? flow_ok<Heat<double>, 32>(N, n) : flow_ok<Heat<float>, 32>(N, n);
  if (flavor == SWEPT_FLAVOR_CLUSTER) return dtype == 0 ? cluster_ok<Heat<double>>(N, n, P) : cluster_ok<Heat<float>>(N, n, P);
  return false;
}
int launch_tile_heat(int dtype, const TileLaunch& a) {
  if (a.flavor == SWEPT_FLAVOR_TIER) return dtype == 0 ? tier_T<Heat<double>, 4>(a) : tier_T<Heat<float>, 4>(a);
  if (a.flavor == SWEPT_FLAVOR_CHAR) return dtype == 0 ? char_T<Heat<double>, 32>(a) : char_T<Heat<float>, 32>(a);
  return NO_KERNEL;
}
int launch_flow_heat(int dtype, const FlowLaunch& a) {
  return dtype == 0 ? flow_T<Heat<double>, 32>(a) : flow_T<Heat<float>, 32>(a);
}
int launch_cluster_heat(int dtype, const ClusterLaunch& a) {
  return dtype == 0 ? cluster_T<Heat<double>>(a) : cluster_T<Heat<float>>(a);
}
int launch_resident_heat(int dtype, const ResidentLaunch& a) {
  return dtype == 0 ? resident_T<Heat<double>, 16>(a) : resident_T<Heat<float>, 16>(a);
}
}  // namespace swept
