// k_hills instantiations for 1 and 2 CVs (binary32 terms).
#include "hills_launch.cuh"

cudaError_t psg_hills_dispatch_n12(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid) {
    const int pm = c->md.hc.pmask;
    if (c->sys.n_cv == 1) {
        if (pm & 1) return launch_k<1, 1, 1, false>(c, A, smem, grid);
        return launch_k<1, 0, 1, false>(c, A, smem, grid);
    }
    switch (pm & 3) {
    case 0: PSG_NEQ_SWITCH(2, 0, false, 1, 1, 0, 0)
    case 1: PSG_NEQ_SWITCH(2, 1, false, 1, 1, 0, 0)
    case 2: PSG_NEQ_SWITCH(2, 2, false, 1, 1, 0, 0)
    default: PSG_NEQ_SWITCH(2, 3, false, 1, 1, 0, 0)
    }
}
