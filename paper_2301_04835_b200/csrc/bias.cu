// bias.cu -- harmonic bias and the ABF grid update.
#include "internal.h"

// V = 1/2 sum_k k_k D_k^2, dV/dxi_k = k_k D_k; D wrapped to the nearest image for periodic CVs.
// One thread per replica; binary64 registers, rounded once on store.
__global__ void __launch_bounds__(256) k_harmonic(const __grid_constant__ SysParams P, const float* __restrict__ xi,
                                                   const float* __restrict__ kspring, const float* __restrict__ centers,
                                                   float* __restrict__ V, double* __restrict__ V64, float* __restrict__ dVdxi) {
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= P.R) return;
    double v = 0.0;
    for (int k = 0; k < P.n_cv; ++k) {
        double d = (double)xi[(long long)r * P.n_cv + k] - (double)centers[(long long)r * P.n_cv + k];
        double per = (double)P.cv[k].period;
        if (per > 0.0) d -= per * rint(d / per);
        double ks = (double)kspring[k];
        v += 0.5 * ks * d * d;
        dVdxi[(long long)r * P.n_cv + k] = (float)(ks * d);
    }
    if (V) V[r] = (float)v;
    if (V64) V64[r] = v;
}

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

// Phase 1: every replica bins its xi and accumulates: hist[bin] += 1 (int32 atomic, exact),
// Fsum[bin][k] += f_k (red.global.add.v2.f32 when n_cv == 2, else scalar float atomics).
__global__ void __launch_bounds__(256) k_abf_accumulate(const __grid_constant__ AbfState G, int R, int n_cv, const float* __restrict__ xi,
                                                         const float* __restrict__ fsample, int* __restrict__ bin_out) {
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    int b = abf_flat_bin(G, n_cv, xi + (long long)r * n_cv);
    bin_out[r] = b;
    if (b < 0) return;
    atomicAdd(G.hist + b, 1);
    const float* f = fsample + (long long)r * n_cv;
    float* dst = G.fsum + (long long)b * n_cv;
    if (n_cv == 2) {
        atomicAdd(reinterpret_cast<float2*>(dst), make_float2(f[0], f[1]));
    } else if (n_cv == 4) {
        atomicAdd(reinterpret_cast<float4*>(dst), make_float4(f[0], f[1], f[2], f[3]));
    } else {
        for (int k = 0; k < n_cv; ++k) atomicAdd(dst + k, f[k]);
    }
}

// Phase 2 (after ALL replicas accumulated): Fbar_k = Fsum[bin][k] / max(hist[bin], N); outside: 0.
__global__ void __launch_bounds__(256) k_abf_mean(const __grid_constant__ AbfState G, int R, int n_cv, const int* __restrict__ bin,
                                                   int* __restrict__ bin_user, float* __restrict__ dVdxi) {
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    int b = bin[r];
    if (bin_user) bin_user[r] = b;
    float cnt_eff = 1.f;
    if (b >= 0) {
        int cnt = __ldcg(G.hist + b);
        cnt_eff = (float)(cnt > G.n_threshold ? cnt : G.n_threshold);
    }
    for (int k = 0; k < n_cv; ++k) {
        float m = 0.f;
        if (b >= 0) m = __fdiv_rn(__ldcg(G.fsum + (long long)b * n_cv + k), cnt_eff);
        dVdxi[(long long)r * n_cv + k] = m;
    }
}

cudaError_t psg_launch_harmonic(psg_ctx* c, const float* d_xi, float* d_V, float* d_dVdxi) {
    k_harmonic<<<(c->sys.R + 255) / 256, 256, 0, c->stream>>>(c->sys, d_xi, c->d_kspring, c->d_centers, d_V, c->d_V64, d_dVdxi);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t psg_launch_abf(psg_ctx* c, const float* d_xi, const float* d_fsample, int* d_bin, float* d_dVdxi) {
    int R = c->sys.R, g = (R + 255) / 256;
    k_abf_accumulate<<<g, 256, 0, c->stream>>>(c->abf, R, c->sys.n_cv, d_xi, d_fsample, c->d_bin);
    k_abf_mean<<<g, 256, 0, c->stream>>>(c->abf, R, c->sys.n_cv, c->d_bin, d_bin, d_dVdxi);
    c->launches += 2;
    return cudaGetLastError();
}
