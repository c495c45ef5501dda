// hills_launch.cuh -- launch helper shared by the translation units that instantiate k_hills.
#pragma once
#include "hills.cuh"

template <int NCV, int PM, int NEQ, bool F64>
static cudaError_t launch_k(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid) {
    auto kern = k_hills<NCV, PM, NEQ, F64>;
    static size_t attr_bytes[PSG_MAX_DEVICES] = {};   // function attributes are per device: one process may hold ctxs on several
    size_t& have = attr_bytes[c->device % PSG_MAX_DEVICES];
    if (smem > have) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        have = smem;
    }
    kern<<<grid, HWARPS * 32, smem, c->stream>>>(c->sys, c->md.hc, A);
    c->launches++;
    return cudaGetLastError();
}

// NEQ handled: the largest instantiated value <= the run-time one (fewer leading dims merged is always valid)
#define PSG_NEQ_SWITCH(NCV, PM, F64, A1, A2, A3, A4)                                                           \
    {                                                                                                          \
        int neq = c->md.hc.neq;                                                                                \
        if ((A4) && neq >= 4) return launch_k<NCV, PM, (A4) ? 4 : 1, F64>(c, A, smem, grid);                    \
        if ((A3) && neq >= 3) return launch_k<NCV, PM, (A3) ? 3 : 1, F64>(c, A, smem, grid);                    \
        if ((A2) && neq >= 2) return launch_k<NCV, PM, (A2) ? 2 : 1, F64>(c, A, smem, grid);                    \
        return launch_k<NCV, PM, 1, F64>(c, A, smem, grid);                                                     \
    }
