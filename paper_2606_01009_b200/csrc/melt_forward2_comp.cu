// melt_forward2_comp.cu -- instantiations of the CTA-pair forward kernel for one operand precision (one translation unit per
// precision, so that the three sets of template instantiations compile in parallel).
#include "melt_forward2_kernel.cuh"

namespace melt {

int launch_forward2_comp(const K2Params &kp, int grid, int sigma, cudaStream_t stream) {
    return sigma ? launch_one<P2_COMP, 1>(kp, grid, stream) : launch_one<P2_COMP, 0>(kp, grid, stream);
}

}  // namespace melt

#ifdef MELT_TRACE
// development builds only: event trace of the compensated-mode kernels (this translation unit's copy of the pointer)
extern "C" int melt_debug_set_trace(long long *buf) {
    return (int)cudaMemcpyToSymbol(melt::g_melt_trace, &buf, sizeof(buf));
}
#endif
