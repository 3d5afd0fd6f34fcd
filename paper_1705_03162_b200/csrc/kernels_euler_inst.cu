// kernels_euler_inst.cu — one slice of the Euler swept-kernel instantiations per compilation:
//   -DSWEPT_INST=0  TIER flavour (P = 1, 2, 4; Up/Split/Whole/Down)
//   -DSWEPT_INST=1  CHAR flavour, B = 8 lines per lane (L = 8, 16, 32)
//   -DSWEPT_RK2=0 midpoint, =1 Heun (BASELINE.json config 4)
#include "kernels_impl.cuh"
#ifndef SWEPT_INST
#error "compile with -DSWEPT_INST=0|1 -DSWEPT_RK2=0|1 (see build.py)"
#endif
namespace swept {
#if SWEPT_INST == 0
template int tier_T<Euler<double, SWEPT_RK2>, 4>(const TileLaunch&);
#else
template int char_L<Euler<double, SWEPT_RK2>, 8>(const TileLaunch&);
#endif
}  // namespace swept
