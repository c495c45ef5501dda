// bias.cu -- harmonic bias and the ABF grid update.
#include "abf.cuh"

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

// Phase 1: every replica bins its xi and accumulates: hist[bin] += 1 (int32 atomic, exact),
// Fsum[bin][k] += f_k (red.global.add.v2.f32 when n_cv == 2, else scalar float atomics).
__global__ void __launch_bounds__(256) k_abf_accumulate(const __grid_constant__ AbfState G, int R, int n_cv, const float* __restrict__ xi,
                                                         const float* __restrict__ fsample, int* __restrict__ bin_out) {
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    bin_out[r] = abf_accumulate_one(G, n_cv, xi + (long long)r * n_cv, fsample + (long long)r * n_cv);
}

// Phase 2 (after ALL replicas accumulated): Fbar_k = Fsum[bin][k] / max(hist[bin], N); outside: 0.
__global__ void __launch_bounds__(256) k_abf_mean(const __grid_constant__ AbfState G, int R, int n_cv, const int* __restrict__ bin,
                                                   int* __restrict__ bin_user, float* __restrict__ dVdxi) {
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    int b = bin[r];
    if (bin_user) bin_user[r] = b;
    abf_mean_one(G, n_cv, b, dVdxi + (long long)r * n_cv);
}

cudaError_t psg_launch_harmonic(psg_ctx* c, const float* d_xi, float* d_V, float* d_dVdxi) {
    k_harmonic<<<(c->sys.R + 255) / 256, 256, 0, c->stream>>>(c->sys, d_xi, c->d_kspring, c->d_centers, d_V, c->d_V64, d_dVdxi);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t psg_launch_abf_accumulate(psg_ctx* c, const float* d_xi, const float* d_fsample, int* hist, float* fsum) {
    AbfState G = c->abf;
    G.hist = hist; G.fsum = fsum;
    k_abf_accumulate<<<(c->sys.R + 255) / 256, 256, 0, c->stream>>>(G, c->sys.R, c->sys.n_cv, d_xi, d_fsample, c->d_bin);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t psg_launch_abf_mean(psg_ctx* c, int* d_bin, float* d_dVdxi) {
    k_abf_mean<<<(c->sys.R + 255) / 256, 256, 0, c->stream>>>(c->abf, c->sys.R, c->sys.n_cv, c->d_bin, d_bin, d_dVdxi);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t psg_launch_abf(psg_ctx* c, const float* d_xi, const float* d_fsample, int* d_bin, float* d_dVdxi) {
    cudaError_t e = psg_launch_abf_accumulate(c, d_xi, d_fsample, c->abf.hist, c->abf.fsum);
    if (e != cudaSuccess) return e;
    return psg_launch_abf_mean(c, d_bin, d_dVdxi);
}
