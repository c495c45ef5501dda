// k_hills instantiations for 3 CVs, periodic masks 4..7 (binary32 terms).
#include "hills_launch.cuh"

cudaError_t psg_hills_dispatch_n3b(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid) {
    switch (c->md.hc.pmask & 7) {
    case 4: PSG_NEQ_SWITCH(3, 4, false, 1, 1, 1, 0)
    case 5: PSG_NEQ_SWITCH(3, 5, false, 1, 1, 1, 0)
    case 6: PSG_NEQ_SWITCH(3, 6, false, 1, 1, 1, 0)
    default: PSG_NEQ_SWITCH(3, 7, false, 1, 1, 1, 0)
    }
}
