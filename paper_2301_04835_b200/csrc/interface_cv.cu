// interface_cv.cu -- DistanceToInterface, the paper's own worked collective variable (Eq. 4-8;
// listing of Appendix A), batched over replicas:
//   xi = barycenter(mobile)[axis] - sum_j softmax(coeff |mass_{j+1} - mass_j|)_j (c_{j+1} + c_j)/2,
//   mass_j = sum_i exp(-(x_i - c_j)^2 / (2 sigma^2)) over the interface atoms,  c = linspace(scope0, scope1, bins).
// Three kernels, all binary64 (the softmax of DIFFERENCES of nearly equal masses amplifies rounding: binary32 masses
// put the interface off by ~1e-4 nm, far outside the parity bar; the paper's JAX code runs in binary32):
//   k_dti_mass   grid (chunks of 1,024 atoms, R): coordinates of the chunk -> shared memory; thread j sums bin j
//   k_dti_finish block per replica: chunk partials in fixed order; softmax, interface and G_j = d interface / d mass_j by the
//                whole block (fixed-order block reductions); xi
//   k_dti_apply  grid (chunks, R): thread per atom, F_i[axis] += dV/dxi * sum_j G_j d mass_j / d x_i; mobile atoms too
// A first version: exp-bound (bins x atoms binary64 exponentials per pass), not tuned.
#include "internal.h"

#define DTI_CHUNK 1024
#define DTI_MAX_BINS 1024

struct DtiParams {
    int R, ps, fs, axis, bins, n_mobile;
    long long N, rstride, ibegin, isize;
    int n_chunks;
    double sigma, scope0, scope1, coeff;
    int mobile_idx[PSG_MAX_SLOTS];
    float mobile_w[PSG_MAX_SLOTS];
};

__device__ __forceinline__ double dti_center(const DtiParams& D, int j) {
    return D.bins > 1 ? D.scope0 + (D.scope1 - D.scope0) * (double)j / (double)(D.bins - 1) : D.scope0;
}

__global__ void __launch_bounds__(128) k_dti_mass(const __grid_constant__ DtiParams D, const float* __restrict__ pos,
                                                  double* __restrict__ part /*[R][n_chunks][bins]*/) {
    __shared__ double x[DTI_CHUNK];
    const int r = blockIdx.y, ch = blockIdx.x, tid = threadIdx.x;
    const float* p = pos + (long long)r * D.rstride * D.ps;
    const long long a0 = D.ibegin + (long long)ch * DTI_CHUNK;
    long long cnt = D.ibegin + D.isize - a0;
    if (cnt > DTI_CHUNK) cnt = DTI_CHUNK;
    for (int i = tid; i < cnt; i += 128) x[i] = (double)__ldg(p + (a0 + i) * D.ps + D.axis);
    __syncthreads();
    const double is = 1.0 / D.sigma;
    for (int j = tid; j < D.bins; j += 128) {
        const double c = dti_center(D, j);
        double m = 0.0;
        for (int i = 0; i < cnt; ++i) {
            const double d = (x[i] - c) * is;
            m += exp(-0.5 * d * d);
        }
        part[((long long)r * D.n_chunks + ch) * D.bins + j] = m;
    }
}

__global__ void __launch_bounds__(128) k_dti_finish(const __grid_constant__ DtiParams D, const float* __restrict__ pos,
                                                    const double* __restrict__ part, double* __restrict__ G /*[R][bins]*/,
                                                    float* __restrict__ xi_out, int xi_stride, int xi_col) {
    __shared__ double mass[DTI_MAX_BINS], prob[DTI_MAX_BINS];
    const int r = blockIdx.x, tid = threadIdx.x;
    for (int j = tid; j < D.bins; j += 128) {
        double m = 0.0;
        for (int ch = 0; ch < D.n_chunks; ++ch) m += part[((long long)r * D.n_chunks + ch) * D.bins + j];   // fixed order
        mass[j] = m;
    }
    __syncthreads();
    // softmax over the nb = bins - 1 bin boundaries, the interface position and its derivative with respect to every bin
    // mass, by the whole block: maximum, partition sum and interface are block reductions in a fixed order (lanes by an
    // xor tree, the four warps in sequence), everything else is one bin boundary per thread
    __shared__ double red[4];
    __shared__ double bc[3];   // mx, Z, I
    const int nb = D.bins - 1, lane = tid & 31, wid = tid >> 5;
    auto block_reduce = [&](double v, bool is_max, int slot) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double u = __shfl_xor_sync(0xffffffffu, v, o);
            v = is_max ? fmax(v, u) : v + u;
        }
        if (lane == 0) red[wid] = v;
        __syncthreads();
        if (tid == 0) {
            double t = red[0];
            for (int w = 1; w < 4; ++w) t = is_max ? fmax(t, red[w]) : t + red[w];
            bc[slot] = t;
        }
        __syncthreads();
    };
    double mx = -1e300;
    for (int j = tid; j < nb; j += 128) {
        const double v = fabs(mass[j + 1] - mass[j]) * D.coeff;
        prob[j] = v;
        mx = fmax(mx, v);
    }
    block_reduce(mx, true, 0);
    double z = 0.0;
    for (int j = tid; j < nb; j += 128) { prob[j] = exp(prob[j] - bc[0]); z += prob[j]; }
    block_reduce(z, false, 1);
    double it = 0.0;
    for (int j = tid; j < nb; j += 128) {
        prob[j] /= bc[1];
        it += prob[j] * 0.5 * (dti_center(D, j + 1) + dti_center(D, j));
    }
    block_reduce(it, false, 2);
    const double I = bc[2];
    // d interface / d mass_j: boundary j - 1 pulls bin j one way, boundary j the other
    auto pull = [&](int j) {   // boundary j in [0, nb)
        const double diff = mass[j + 1] - mass[j];
        const double sg = diff > 0.0 ? 1.0 : (diff < 0.0 ? -1.0 : 0.0);
        return D.coeff * sg * prob[j] * (0.5 * (dti_center(D, j + 1) + dti_center(D, j)) - I);
    };
    double* g = G + (long long)r * D.bins;
    for (int j = tid; j < D.bins; j += 128) g[j] = (j >= 1 ? pull(j - 1) : 0.0) - (j < nb ? pull(j) : 0.0);
    if (tid == 0) {
        const float* p = pos + (long long)r * D.rstride * D.ps;
        double W = 0.0, mob = 0.0;
        for (int m = 0; m < D.n_mobile; ++m) {
            const double w = (double)D.mobile_w[m];
            mob += w * (double)p[(long long)D.mobile_idx[m] * D.ps + D.axis];
            W += w;
        }
        xi_out[(long long)r * xi_stride + xi_col] = (float)(mob / W - I);
    }
}

__global__ void __launch_bounds__(256) k_dti_apply(const __grid_constant__ DtiParams D, const float* __restrict__ pos,
                                                   const double* __restrict__ G, const float* __restrict__ dVdxi, int dv_stride,
                                                   int dv_col, float* __restrict__ force) {
    __shared__ double g[DTI_MAX_BINS];
    const int r = blockIdx.y, ch = blockIdx.x, tid = threadIdx.x;
    for (int j = tid; j < D.bins; j += 256) g[j] = G[(long long)r * D.bins + j];
    __syncthreads();
    const float* p = pos + (long long)r * D.rstride * D.ps;
    float* f = force + (long long)r * D.rstride * D.fs;
    const double dv = (double)dVdxi[(long long)r * dv_stride + dv_col], is2 = 1.0 / (D.sigma * D.sigma);
    const long long a0 = D.ibegin + (long long)ch * DTI_CHUNK;
    for (int i = tid; i < DTI_CHUNK; i += 256) {
        const long long a = a0 + i;
        if (a >= D.ibegin + D.isize) break;
        const double x = (double)__ldg(p + a * D.ps + D.axis);
        double dI = 0.0;
        for (int j = 0; j < D.bins; ++j) {
            const double d = x - dti_center(D, j);
            dI -= g[j] * exp(-0.5 * d * d * is2) * d * is2;
        }
        // d xi / d x_i = -dI;  F_i = -dV/dxi * d xi / d x_i
        const float add = (float)(dv * dI);
        // always a reduction: block 0 adds the mobile atoms' term in this same launch and a mobile atom may lie inside the
        // interface range (a plain += racing that atomic could lose one of the two); free next to the exp loop above
        atomicAdd(f + a * D.fs + D.axis, add);
    }
    if (ch == 0 && tid < D.n_mobile) {   // mobile atoms: d xi / d r_m = (w_m / W) e_axis; they may coincide with interface atoms
        double W = 0.0;
        for (int m = 0; m < D.n_mobile; ++m) W += (double)D.mobile_w[m];
        atomicAdd(f + (long long)D.mobile_idx[tid] * D.fs + D.axis, (float)(-dv * (double)D.mobile_w[tid] / W));
    }
}

struct DtiState {
    DtiParams D;
    double* part;
    double* G;
};

static DtiState* dti(psg_ctx* c) { return reinterpret_cast<DtiState*>(c->dti); }

extern "C" int psg_interface_cv_set(psg_ctx* c, int n_mobile, const int* mobile_idx, const float* mobile_w, long long iface_begin,
                                    long long iface_size, int axis, double sigma, double scope0, double scope1, int bins,
                                    double coeff) {
    if (!c) return PSG_EINVAL;
    auto bad = [&](const char* m) { c->err = m; return PSG_EINVAL; };
    if (!c->have_layout) { c->err = "psg_interface_cv_set: call psg_set_layout first"; return PSG_ESTATE; }
    const SysParams& P = c->sys;
    if (n_mobile < 1 || n_mobile > PSG_MAX_SLOTS || !mobile_idx) return bad("psg_interface_cv_set: 1 <= n_mobile <= PSG_MAX_SLOTS");
    if (iface_begin < 0 || iface_size < 1 || iface_begin + iface_size > P.N) return bad("psg_interface_cv_set: interface range outside [0, n_atoms)");
    if (axis < 0 || axis > 2 || !(sigma > 0.0) || bins < 2 || bins > DTI_MAX_BINS || !(scope1 > scope0))
        return bad("psg_interface_cv_set: need axis in 0..2, sigma > 0, 2 <= bins <= 1024, scope1 > scope0");
    for (int m = 0; m < n_mobile; ++m) {
        if (mobile_idx[m] < 0 || mobile_idx[m] >= P.N) return bad("psg_interface_cv_set: mobile atom index out of range");
        if (mobile_w && !(mobile_w[m] > 0.f)) return bad("psg_interface_cv_set: weights must be > 0");
    }
    cudaSetDevice(c->device);
    DtiState* S = dti(c);
    if (!S) { S = new DtiState(); S->part = nullptr; S->G = nullptr; c->dti = S; }
    DtiParams& D = S->D;
    D.R = P.R; D.ps = P.ps; D.fs = P.fs; D.axis = axis; D.bins = bins; D.n_mobile = n_mobile;
    D.N = P.N; D.rstride = P.rstride; D.ibegin = iface_begin; D.isize = iface_size;
    D.n_chunks = (int)((iface_size + DTI_CHUNK - 1) / DTI_CHUNK);
    D.sigma = sigma; D.scope0 = scope0; D.scope1 = scope1; D.coeff = coeff;
    for (int m = 0; m < PSG_MAX_SLOTS; ++m) { D.mobile_idx[m] = m < n_mobile ? mobile_idx[m] : 0; D.mobile_w[m] = m < n_mobile ? (mobile_w ? mobile_w[m] : 1.f) : 0.f; }
    if (S->part) cudaFree(S->part);
    if (S->G) cudaFree(S->G);
    if (cudaMalloc((void**)&S->part, sizeof(double) * (size_t)P.R * D.n_chunks * bins) != cudaSuccess ||
        cudaMalloc((void**)&S->G, sizeof(double) * (size_t)P.R * bins) != cudaSuccess) { c->err = "psg_interface_cv_set: out of device memory"; return PSG_ENOMEM; }
    return PSG_OK;
}

extern "C" int psg_interface_cv_eval(psg_ctx* c, const float* d_pos, float* d_xi) {
    if (!c) return PSG_EINVAL;
    DtiState* S = dti(c);
    if (!S) { c->err = "psg_interface_cv_eval: call psg_interface_cv_set first"; return PSG_ESTATE; }
    if (!d_pos || !d_xi) { c->err = "psg_interface_cv_eval: NULL pointer"; return PSG_EINVAL; }
    if (psg_launch_dti_eval(c, d_pos, d_xi, 1, 0) != cudaSuccess) { c->err = "psg_interface_cv_eval: launch failed"; return PSG_ECUDA; }
    return PSG_OK;
}

extern "C" int psg_interface_cv_apply(psg_ctx* c, const float* d_pos, const float* d_dVdxi, float* d_force) {
    if (!c) return PSG_EINVAL;
    DtiState* S = dti(c);
    if (!S) { c->err = "psg_interface_cv_apply: call psg_interface_cv_set and psg_interface_cv_eval first"; return PSG_ESTATE; }
    if (!d_pos || !d_dVdxi || !d_force) { c->err = "psg_interface_cv_apply: NULL pointer"; return PSG_EINVAL; }
    if (psg_launch_dti_apply(c, d_pos, d_dVdxi, 1, 0, d_force) != cudaSuccess) { c->err = "psg_interface_cv_apply: launch failed"; return PSG_ECUDA; }
    return PSG_OK;
}

// value into column xi_col of a [R][xi_stride] array (psg_cv_eval: the CV's own column of xi) ...
cudaError_t psg_launch_dti_eval(psg_ctx* c, const float* d_pos, float* d_xi, int xi_stride, int xi_col) {
    DtiState* S = dti(c);
    const DtiParams& D = S->D;
    k_dti_mass<<<dim3(D.n_chunks, D.R), 128, 0, c->stream>>>(D, d_pos, S->part);
    k_dti_finish<<<D.R, 128, 0, c->stream>>>(D, d_pos, S->part, S->G, d_xi, xi_stride, xi_col);
    c->launches += 2;
    return cudaGetLastError();
}
// ... and the forces of that CV from column dv_col of dV/dxi (psg_apply_bias_forces)
cudaError_t psg_launch_dti_apply(psg_ctx* c, const float* d_pos, const float* d_dVdxi, int dv_stride, int dv_col, float* d_force) {
    DtiState* S = dti(c);
    const DtiParams& D = S->D;
    k_dti_apply<<<dim3(D.n_chunks, D.R), 256, 0, c->stream>>>(D, d_pos, S->G, d_dVdxi, dv_stride, dv_col, d_force);
    c->launches += 1;
    return cudaGetLastError();
}

void psg_interface_cv_free(psg_ctx* c) {
    DtiState* S = dti(c);
    if (!S) return;
    if (S->part) cudaFree(S->part);
    if (S->G) cudaFree(S->G);
    delete S;
    c->dti = nullptr;
}
