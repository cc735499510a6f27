// pz_fft_xy_fwd.cu -- forward instantiations of the fused x/y transform (pz_fft_xy_impl.cuh).
#include "pz_fft_xy_impl.cuh"

namespace pz {
int launch_fft_xy_fwd(pz_plan *pl, double *p, cudaStream_t st) { return dispatch_xy<false>(pl, p, st); }
} // namespace pz
