// pz_fft_xy_inv.cu -- inverse instantiations of the fused y/x transform (pz_fft_xy_impl.cuh).
#include "pz_fft_xy_impl.cuh"

namespace pz {
int launch_fft_xy_inv(pz_plan *pl, double *p, cudaStream_t st) { return dispatch_xy<true>(pl, p, st); }
} // namespace pz
