// abf.cuh -- device-side pieces of the ABF grid update, shared by the separate
// kernels (bias.cu) and the fused ABF step (abf_step.cu).
#pragma once
#include "internal.h"

// ABF bin of one replica, DEFINED IN BINARY32 (reading R-ABF-1): per CV
//   t = fl32(fl32(xi - lower) * invd), I = (int)floorf(t); two separately rounded operations (no FMA contraction).
__device__ __forceinline__ int abf_flat_bin(const AbfState& G, int n_cv, const float* __restrict__ xi_r) {
    long long flat = 0;
    for (int k = 0; k < n_cv; ++k) {
        float t = __fmul_rn(__fsub_rn(xi_r[k], G.lower[k]), G.invd[k]);
        float f = floorf(t);
        if (!(f == f)) return -1;   // NaN
        int i;
        if (G.periodic[k]) {
            float m = fmodf(f, (float)G.shape[k]);
            if (m < 0.f) m += (float)G.shape[k];
            i = (int)m;
            if (i >= G.shape[k]) i = 0;
        } else {
            if (f < 0.f || f >= (float)G.shape[k]) return -1;
            i = (int)f;
        }
        flat = flat * G.shape[k] + i;
    }
    return (int)flat;
}

// Phase 1 for one replica: bin xi; hist[bin] += 1 (int32 atomic, exact); Fsum[bin][k] += f_k (red.global.add.v2.f32
// when n_cv == 2, v4 when n_cv == 4, else scalar float atomics). Returns the bin (-1 = outside, nothing updated).
__device__ __forceinline__ int abf_accumulate_one(const AbfState& G, int n_cv, const float* __restrict__ xi_r,
                                                  const float* __restrict__ f) {
    const int b = abf_flat_bin(G, n_cv, xi_r);
    if (b < 0) return b;
    atomicAdd(G.hist + b, 1);
    float* dst = G.fsum + (long long)b * n_cv;
    if (n_cv == 2) {
        atomicAdd(reinterpret_cast<float2*>(dst), make_float2(f[0], f[1]));
    } else if (n_cv == 4) {
        atomicAdd(reinterpret_cast<float4*>(dst), make_float4(f[0], f[1], f[2], f[3]));
    } else {
        for (int k = 0; k < n_cv; ++k) atomicAdd(dst + k, f[k]);
    }
    return b;
}

// Phase 2 for one replica (after ALL replicas accumulated): Fbar_k = Fsum[bin][k] / max(hist[bin], N); outside: 0.
__device__ __forceinline__ void abf_mean_one(const AbfState& G, int n_cv, int b, float* __restrict__ dVdxi_r) {
    float cnt_eff = 1.f;
    if (b >= 0) {
        int cnt = __ldcg(G.hist + b);
        cnt_eff = (float)(cnt > G.n_threshold ? cnt : G.n_threshold);
    }
    for (int k = 0; k < n_cv; ++k) {
        float m = 0.f;
        if (b >= 0) m = __fdiv_rn(__ldcg(G.fsum + (long long)b * n_cv + k), cnt_eff);
        dVdxi_r[k] = m;
    }
}
