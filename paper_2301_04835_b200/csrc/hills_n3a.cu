// k_hills instantiations for 3 CVs, periodic masks 0..3 (binary32 terms).
#include "hills_launch.cuh"

cudaError_t psg_hills_dispatch_n3a(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid) {
    switch (c->md.hc.pmask & 7) {
    case 0: PSG_NEQ_SWITCH(3, 0, false, 1, 1, 1, 0)
    case 1: PSG_NEQ_SWITCH(3, 1, false, 1, 1, 1, 0)
    case 2: PSG_NEQ_SWITCH(3, 2, false, 1, 1, 1, 0)
    default: PSG_NEQ_SWITCH(3, 3, false, 1, 1, 1, 0)
    }
}
