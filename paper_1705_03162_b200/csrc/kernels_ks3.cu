// kernels_ks3.cu — KS with three sub-timesteps per timestep (SSP-RK3 on Eq. (C.2); SURVEY.md §8(f) row f3,
// PAPER.md:131) kernel instantiations, FP64: the per-step kernel (one launch per stage) and the swept TIER flavour
// on a three-row state.
#include "kernels_persist_impl.cuh"
namespace swept {
int launch_per_step_ks3(int dtype, const PerStepLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  return per_step_T<KS3<double>, 4>(a);
}
bool tile_config_ok_ks3(int dtype, int flavor, int64_t N, int n, int P) {
  if (dtype != 0) return false;
  if (flavor == SWEPT_FLAVOR_TIER) return tier_ok<KS3<double>>(n, P, 4);
  if (flavor == SWEPT_FLAVOR_CLUSTER) return cluster_ok<KS3<double>>(N, n, P);
  return false;
}
int launch_cluster_ks3(int dtype, const ClusterLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  return cluster_T<KS3<double>>(a);
}
int launch_tile_ks3(int dtype, const TileLaunch& a) {
  if (dtype != 0) return NO_KERNEL;
  if (a.flavor == SWEPT_FLAVOR_TIER) return tier_T<KS3<double>, 4>(a);
  return NO_KERNEL;
}
}  // namespace swept
