// melt_forward2_bf16.cu -- instantiations of the CTA-pair forward kernel for one operand precision (one translation unit per
// precision, so that the three sets of template instantiations compile in parallel).
#include "melt_forward2_kernel.cuh"

namespace melt {

int launch_forward2_bf16(const K2Params &kp, int grid, int sigma, cudaStream_t stream) {
    return sigma ? launch_one<P2_BF16, 1>(kp, grid, stream) : launch_one<P2_BF16, 0>(kp, grid, stream);
}

}  // namespace melt
