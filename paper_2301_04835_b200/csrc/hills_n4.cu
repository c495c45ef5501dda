// k_hills instantiations for 4 CVs (binary32 terms; any periodic CV -> the all-periodic kernel, where a
// non-periodic dim has inv_period = 0 and its wrap is the identity) and the binary64-term kernels of all sizes.
#include "hills_launch.cuh"

cudaError_t psg_hills_dispatch_n4(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid) {
    if (c->md.hc.pmask) PSG_NEQ_SWITCH(4, 15, false, 1, 1, 0, 1)
    PSG_NEQ_SWITCH(4, 0, false, 1, 1, 0, 1)
}

cudaError_t psg_hills_dispatch_f64(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid) {
    switch (c->sys.n_cv) {
    case 1: return launch_k<1, 0, 1, true>(c, A, smem, grid);
    case 2: return launch_k<2, 0, 1, true>(c, A, smem, grid);
    case 3: return launch_k<3, 0, 1, true>(c, A, smem, grid);
    case 4: return launch_k<4, 0, 1, true>(c, A, smem, grid);
    }
    return cudaErrorInvalidValue;
}
