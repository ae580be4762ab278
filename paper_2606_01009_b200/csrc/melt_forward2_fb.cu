// melt_forward2_fb.cu -- instantiations of the CTA-pair forward kernel for the conventional front end (MODE 4: DFT bins, power, a
// second tensor-core product with the triangular Mel filterbank, log).  A translation unit of its own so
// that it compiles in parallel with the MelT / MFCCT instantiations.
#include "melt_forward2_kernel.cuh"

namespace melt {

int launch_forward2_fb(const K2Params &kp, int grid, int sigma, cudaStream_t stream) {
    if (!kp.fb_mels || kp.b_resident || kp.direct || kp.offsets) return fail(MELT_ERR_UNSUPPORTED, "internal: filterbank kernel needs a dense batch and a streamed basis");
    return sigma ? launch_one_s<P2_COMP, 1, false, 4, true, false>(kp, grid, stream)
                 : launch_one_s<P2_COMP, 0, false, 4, true, false>(kp, grid, stream);
}

}  // namespace melt
