// hills.cu -- metadynamics: the hill sum, hill deposition, and the fused step.
//
// Hill sum  V(xi) = sum_h W_h exp(-1/2 sum_k (d_hk/sigma_k)^2),  dV/dxi_k = -sum_h W_h exp(..) d_hk/sigma_k^2,
// d_hk = nearest image of xi_k - s_hk.  Not a dense contraction (the wrap breaks bilinearity): FP32-pipe + MUFU work.
//
// Decomposition: CTA = (tile of 64 replicas) x (chunk of hills). Warp w owns 8 replicas whose xi sit in registers;
// its 32 lanes stride over the hills of the chunk, which is streamed through shared memory by 1-D TMA bulk copies
// (cp.async.bulk + mbarrier, 3 stages). Each hill record (one LDS.128) is reused for 8 replica evaluations.
// Terms are binary32; every 8 hills the binary32 partial sums are flushed into binary64 accumulators. Lanes are
// combined with warp shuffles, chunks through a scratch array summed IN FIXED ORDER by the last CTA of the tile
// (ticket counter), so results are bitwise reproducible. The same kernel, FUSED, first evaluates the CVs of its
// tile from the engine's positions and, in the last CTA, scatters -dV/dxi * J into the engine's forces:
// one launch per MD step.
#include "geom.cuh"

#define RT PSG_HILL_RT
#define HWARPS PSG_HILL_WARPS
#define TILE_R PSG_HILL_TILE_R
#define SUB PSG_HILL_SUB
#define STAGES PSG_HILL_STAGES
#define FLUSH_EVERY 8
#define MAGIC_RN 12582912.0f   // 1.5 * 2^23: (x + M) - M = rint(x) for |x| < 2^22

// ---------------------------------------------------------------- mbarrier / TMA (1-D bulk) helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---------------------------------------------------------------- per-thread accumulation over one smem sub-tile
template <int NCV>
struct Acc {
    double V[RT];
    double g[RT][NCV];
};

template <int NCV>
__device__ __forceinline__ void load_rec(const float4* __restrict__ sm, int h, float (&s)[NCV], float& W) {
    if (NCV <= 3) {
        float4 v = sm[h];
        s[0] = v.x;
        if (NCV > 1) s[1 % NCV] = v.y;
        if (NCV > 2) s[2 % NCV] = v.z;
        W = v.w;
    } else {
        float4 a = sm[2 * h], b = sm[2 * h + 1];
        s[0] = a.x; s[1 % NCV] = a.y; s[2 % NCV] = a.z; s[3 % NCV] = a.w;
        W = b.x;
    }
}

// binary32 terms. PM = bitmask of periodic CVs (compile time, so non-periodic dims pay no wrap).
template <int NCV, int PM>
__device__ __forceinline__ void accumulate_f32(const float4* __restrict__ sm, int n_sub, int lane,
                                               const float (&xi)[RT][NCV], const HillConsts& hc, Acc<NCV>& acc) {
    for (int base = 0; base < n_sub; base += 32 * FLUSH_EVERY) {
        float aV[RT], ag[RT][NCV];
#pragma unroll
        for (int j = 0; j < RT; ++j) {
            aV[j] = 0.f;
#pragma unroll
            for (int k = 0; k < NCV; ++k) ag[j][k] = 0.f;
        }
#pragma unroll 2
        for (int u = 0; u < FLUSH_EVERY; ++u) {
            int h = base + u * 32 + lane;
            if (h < n_sub) {
                float s[NCV], W;
                load_rec<NCV>(sm, h, s, W);
#pragma unroll
                for (int j = 0; j < RT; ++j) {
                    float a[NCV];
                    float x = 0.f;
#pragma unroll
                    for (int k = 0; k < NCV; ++k) {
                        float d = __fsub_rn(xi[j][k], s[k]);
                        if (PM & (1 << k)) {
                            // nearest image: d -= P*rint(d/P); P = p_hi + p_lo (Cody-Waite) so the wrap adds no bias
                            float t = __fmaf_rn(d, hc.inv_period[k], MAGIC_RN);
                            float kf = __fsub_rn(t, MAGIC_RN);
                            d = __fmaf_rn(-kf, hc.p_hi[k], d);
                            d = __fmaf_rn(-kf, hc.p_lo[k], d);
                        }
                        a[k] = __fmul_rn(d, hc.cscale[k]);
                        x = __fmaf_rn(-a[k], a[k], x);
                    }
                    float ew = __fmul_rn(ex2_approx(x), W);
                    aV[j] = __fadd_rn(aV[j], ew);
#pragma unroll
                    for (int k = 0; k < NCV; ++k) ag[j][k] = __fmaf_rn(ew, a[k], ag[j][k]);
                }
            }
        }
#pragma unroll
        for (int j = 0; j < RT; ++j) {
            acc.V[j] += (double)aV[j];
#pragma unroll
            for (int k = 0; k < NCV; ++k) acc.g[j][k] += (double)ag[j][k];
        }
    }
}

// binary64 terms (PSG_HILLS_F64): the definition, evaluated in double on the FP64 pipe.
template <int NCV, int PM>
__device__ __forceinline__ void accumulate_f64(const float4* __restrict__ sm, int n_sub, int lane,
                                               const float (&xi)[RT][NCV], const HillConsts& hc, Acc<NCV>& acc) {
    for (int h = lane; h < n_sub; h += 32) {
        float s[NCV], W;
        load_rec<NCV>(sm, h, s, W);
#pragma unroll 2
        for (int j = 0; j < RT; ++j) {
            double q[NCV], e2 = 0.0;
#pragma unroll
            for (int k = 0; k < NCV; ++k) {
                double d = (double)xi[j][k] - (double)s[k];
                if (PM & (1 << k)) d -= hc.period_d[k] * rint(d / hc.period_d[k]);
                q[k] = d * hc.inv_sigma_d[k];
                e2 += q[k] * q[k];
            }
            double w = (double)W * exp(-0.5 * e2);
            acc.V[j] += w;
#pragma unroll
            for (int k = 0; k < NCV; ++k) acc.g[j][k] += w * q[k];   // scaled by -1/sigma_k at the end
        }
    }
}

// lane-local CV of (replica r, CV k) for systems with explicit groups only; JAC: dc[g] = dxi/dc_g / W_g.
template <bool JAC>
__device__ __forceinline__ double thread_cv(const SysParams& P, int r, int k, const float* __restrict__ pos, D3* dc) {
    const CvDev& C = P.cv[k];
    const float* p = pos + (long long)r * P.rstride * P.ps;
    const int* sa = P.slot_atom + (P.per_rep ? (long long)r * P.n_slots : 0);
    D3 c[4];
    double W[4];
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        c[g] = d3(0, 0, 0);
        W[g] = 1.0;
        if (g < C.n_groups) {
            const GroupDev& G = P.grp[C.gid0 + g];
            double sx = 0, sy = 0, sz = 0, sw = 0;
            for (int i = 0; i < G.size; ++i) {
                int s = G.begin + i;
                D3 x = load_pos(p, sa[s], P.ps);
                double w = P.slot_weight ? (double)P.slot_weight[s] : 1.0;
                sx += w * x.x; sy += w * x.y; sz += w * x.z; sw += w;
            }
            double iw = 1.0 / sw;
            c[g] = d3(sx * iw, sy * iw, sz * iw);
            W[g] = sw;
        }
    }
    double xi = cv_from_centers<JAC>(C.type, C.axis, c, dc);
    if (JAC) {
#pragma unroll
        for (int g = 0; g < 4; ++g) dc[g] = (1.0 / W[g]) * dc[g];
    }
    return xi;
}

struct HillKernelArgs {
    const float4* hills;
    const int* n_hills;
    double* part;
    unsigned* ticket;
    const float* xi_in;     // non-fused: [R][n_cv]
    float* V_out;           // nullable
    double* V64_out;        // nullable
    float* dV_out;          // nullable
    float* xi_out;          // fused: step outputs
    const float* pos;       // fused
    float* force;           // fused
    int R;
};

// One kernel for psg_bias_eval (FUSED = false) and the whole metadynamics step (FUSED = true).
template <int NCV, int PM, bool F64, bool FUSED>
__global__ void __launch_bounds__(HWARPS * 32) k_hills(const __grid_constant__ SysParams P, const __grid_constant__ HillConsts hc,
                                                         const __grid_constant__ HillKernelArgs A) {
    constexpr int REC = NCV <= 3 ? 1 : 2;
    constexpr int NV = 1 + NCV;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* stage = reinterpret_cast<float4*>(smem_raw);                          // STAGES * SUB * REC float4
    uint64_t* full = reinterpret_cast<uint64_t*>(stage + STAGES * SUB * REC);     // STAGES barriers
    float* s_xi = reinterpret_cast<float*>(full + STAGES);                        // TILE_R * NCV
    double* s_out = reinterpret_cast<double*>(s_xi + TILE_R * PSG_MAX_CV);        // TILE_R * NV
    __shared__ int s_last;

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int R = A.R;
    const int n_rt = (R + TILE_R - 1) / TILE_R;
    const int n_h = *A.n_hills;
    // chunking: as many chunks per tile as the grid allows, chunk length a multiple of 32
    int cpt = (int)gridDim.x / n_rt;
    if (cpt < 1) cpt = 1;
    int Lc = (n_h + cpt - 1) / cpt;
    Lc = ((Lc + 31) / 32) * 32;
    if (Lc < 32) Lc = 32;
    int n_chunks = (n_h + Lc - 1) / Lc;
    if (n_chunks < 1) n_chunks = 1;
    const int items = n_rt * n_chunks;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned seq = 0;   // sub-tiles consumed so far by this CTA (stage = seq % STAGES, parity = (seq / STAGES) & 1)

    for (int item = blockIdx.x; item < items; item += gridDim.x) {
        const int tile = item % n_rt, chunk = item / n_rt;
        const int r0 = tile * TILE_R;
        const int h0 = chunk * Lc;
        int len = n_h - h0;
        if (len > Lc) len = Lc;
        if (len < 0) len = 0;
        const int n_st = (len + SUB - 1) / SUB;
        // producer prologue
        if (tid == 0) {
            for (int t = 0; t < n_st && t < STAGES; ++t) {
                int s = (seq + t) % STAGES;
                int cnt = min(SUB, len - t * SUB);
                mbar_expect_tx(&full[s], (uint32_t)cnt * REC * 16u);
                tma_load_1d(stage + s * SUB * REC, A.hills + (size_t)(h0 + t * SUB) * REC, (uint32_t)cnt * REC * 16u, &full[s]);
            }
        }
        // CV values of this tile's replicas (overlaps the first TMA loads)
        if (FUSED) {
            for (int t = tid; t < TILE_R * NCV; t += blockDim.x) {
                int rr = t / NCV, k = t % NCV, r = r0 + rr;
                float v = 0.f;
                if (r < R) v = (float)thread_cv<false>(P, r, k, A.pos, nullptr);
                s_xi[rr * NCV + k] = v;
            }
        } else {
            for (int t = tid; t < TILE_R * NCV; t += blockDim.x) {
                int r = r0 + t / NCV;
                s_xi[t] = r < R ? A.xi_in[(long long)r0 * NCV + t] : 0.f;
            }
        }
        __syncthreads();
        float xi[RT][NCV];
#pragma unroll
        for (int j = 0; j < RT; ++j)
#pragma unroll
            for (int k = 0; k < NCV; ++k) xi[j][k] = s_xi[(wid * RT + j) * NCV + k];
        Acc<NCV> acc;
#pragma unroll
        for (int j = 0; j < RT; ++j) {
            acc.V[j] = 0.0;
#pragma unroll
            for (int k = 0; k < NCV; ++k) acc.g[j][k] = 0.0;
        }
        const bool warp_active = r0 + wid * RT < R;
        for (int t = 0; t < n_st; ++t) {
            int s = seq % STAGES;
            mbar_wait(&full[s], (seq / STAGES) & 1);
            int cnt = min(SUB, len - t * SUB);
            if (warp_active) {
                if (F64) accumulate_f64<NCV, PM>(stage + s * SUB * REC, cnt, lane, xi, hc, acc);
                else accumulate_f32<NCV, PM>(stage + s * SUB * REC, cnt, lane, xi, hc, acc);
            }
            __syncthreads();   // everyone is done with stage s
            if (tid == 0 && t + STAGES < n_st) {
                int cn = min(SUB, len - (t + STAGES) * SUB);
                mbar_expect_tx(&full[s], (uint32_t)cn * REC * 16u);
                tma_load_1d(stage + s * SUB * REC, A.hills + (size_t)(h0 + (t + STAGES) * SUB) * REC, (uint32_t)cn * REC * 16u,
                            &full[s]);
            }
            ++seq;
        }
        // lanes -> warp totals (each warp owns its replicas: no cross-warp reduction)
        double* dst = A.part + ((size_t)(chunk * n_rt + tile) * TILE_R + wid * RT) * NV;
#pragma unroll
        for (int j = 0; j < RT; ++j) {
            double v = warp_sum(acc.V[j]);
            if (lane == 0) dst[j * NV] = v;
#pragma unroll
            for (int k = 0; k < NCV; ++k) {
                double gk = warp_sum(acc.g[j][k]);
                if (lane == 0) dst[j * NV + 1 + k] = gk;
            }
        }
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            unsigned old = atomicAdd(&A.ticket[tile], 1u);
            s_last = (old == (unsigned)(n_chunks - 1));
        }
        __syncthreads();
        if (s_last) {   // block-uniform: this CTA finishes the tile
            __threadfence();
            for (int t = tid; t < TILE_R * NV; t += blockDim.x) {
                double sum = 0.0;
                for (int c = 0; c < n_chunks; ++c) sum += __ldcg(A.part + ((size_t)(c * n_rt + tile) * TILE_R) * NV + t);
                int v = t % NV;
                if (v > 0) sum *= -(F64 ? hc.inv_sigma_d[v - 1] : hc.gscale[v - 1]);
                s_out[t] = sum;
                int r = r0 + t / NV;
                if (r < R) {
                    if (v == 0) {
                        if (A.V_out) A.V_out[r] = (float)sum;
                        if (A.V64_out) A.V64_out[r] = sum;
                    } else if (A.dV_out) {
                        A.dV_out[(long long)r * NCV + v - 1] = (float)sum;
                    }
                }
            }
            if (tid == 0) A.ticket[tile] = 0u;   // ready for the next launch
            if (FUSED) {
                __syncthreads();
                // forces: lane <-> (replica, CV); each lane scatters its CV's atoms
                for (int t = tid; t < TILE_R * NCV; t += blockDim.x) {
                    int rr = t / NCV, k = t % NCV, r = r0 + rr;
                    if (r >= R) continue;
                    D3 dc[4];
                    double xv = thread_cv<true>(P, r, k, A.pos, dc);
                    if (A.xi_out) A.xi_out[(long long)r * NCV + k] = (float)xv;
                    // same rounding as the unfused path: dV/dxi passes through binary32
                    double dv = -(double)(float)s_out[rr * NV + 1 + k];
                    const CvDev& C = P.cv[k];
                    const int* sa = P.slot_atom + (P.per_rep ? (long long)r * P.n_slots : 0);
                    float* f = A.force + (long long)r * P.rstride * P.fs;
#pragma unroll
                    for (int g = 0; g < 4; ++g) {
                        if (g < C.n_groups) {
                            const GroupDev& G = P.grp[C.gid0 + g];
                            for (int i = 0; i < G.size; ++i) {
                                int s = G.begin + i;
                                double w = P.slot_weight ? (double)P.slot_weight[s] : 1.0;
                                // J rounded to binary32 first, like the cached Jacobian of the unfused path
                                float jx = (float)(w * dc[g].x), jy = (float)(w * dc[g].y), jz = (float)(w * dc[g].z);
                                float fdv = (float)dv;
                                float* fa = f + (long long)sa[s] * P.fs;
                                atomicAdd(fa, fdv * jx);
                                atomicAdd(fa + 1, fdv * jy);
                                atomicAdd(fa + 2, fdv * jz);
                            }
                        }
                    }
                }
            }
        }
        __syncthreads();   // s_xi / s_out / s_last reused by the next item
    }
}

// ---------------------------------------------------------------- deposition
// Single block. Replica r deposits (mask == NULL or mask[r]) at slot n_h + (#depositing replicas before r):
// replica order. W = w0 exp(-V_old/(kB dT)) in binary64, stored binary32 (well-tempered) or W = w0.
__global__ void __launch_bounds__(1024) k_deposit(int R, int n_cv, int rec, const float* __restrict__ xi, const double* __restrict__ Vold,
                                                   const unsigned char* __restrict__ mask, double w0, double kBdT, float4* __restrict__ hills,
                                                   int* __restrict__ n_hills, int capacity) {
    __shared__ int s_warp[32];
    __shared__ int s_base;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) s_base = *n_hills;
    __syncthreads();
    for (int r0 = 0; r0 < R; r0 += 1024) {
        int r = r0 + tid;
        int dep = (r < R) && (!mask || mask[r]);
        unsigned b = __ballot_sync(0xffffffffu, dep);
        int pre = __popc(b & ((1u << lane) - 1u));
        if (lane == 0) s_warp[wid] = __popc(b);
        __syncthreads();
        int off = 0, tot = 0;
        for (int w = 0; w < 32; ++w) {
            if (w < wid) off += s_warp[w];
            tot += s_warp[w];
        }
        if (dep) {
            int slot = s_base + off + pre;
            if (slot < capacity) {
                float W = (float)(kBdT > 0.0 ? w0 * exp(-Vold[r] / kBdT) : w0);
                float s[4] = {0.f, 0.f, 0.f, 0.f};
                for (int k = 0; k < n_cv; ++k) s[k] = xi[(long long)r * n_cv + k];
                if (rec == 1) hills[slot] = make_float4(s[0], s[1], s[2], W);
                else {
                    hills[2 * slot] = make_float4(s[0], s[1], s[2], s[3]);
                    hills[2 * slot + 1] = make_float4(W, 0.f, 0.f, 0.f);
                }
            }
        }
        __syncthreads();
        if (tid == 0) s_base = min(s_base + tot, capacity);
        __syncthreads();
    }
    if (tid == 0) *n_hills = s_base;
}

__global__ void k_pack_hills(int n, int n_cv, int rec, const float* __restrict__ centers, const float* __restrict__ heights,
                             float4* __restrict__ hills) {
    int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n) return;
    float s[4] = {0.f, 0.f, 0.f, 0.f};
    for (int k = 0; k < n_cv; ++k) s[k] = centers[(long long)h * n_cv + k];
    if (rec == 1) hills[h] = make_float4(s[0], s[1], s[2], heights[h]);
    else {
        hills[2 * h] = make_float4(s[0], s[1], s[2], s[3]);
        hills[2 * h + 1] = make_float4(heights[h], 0.f, 0.f, 0.f);
    }
}

__global__ void k_unpack_hills(int n, int n_cv, int rec, const float4* __restrict__ hills, float* __restrict__ centers,
                               float* __restrict__ heights) {
    int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n) return;
    float4 a = hills[rec * h];
    float s[4] = {a.x, a.y, a.z, a.w};
    float W = rec == 1 ? a.w : hills[2 * h + 1].x;
    for (int k = 0; k < n_cv; ++k) centers[(long long)h * n_cv + k] = s[k];
    heights[h] = W;
}

// ---------------------------------------------------------------- host side
static size_t hills_smem_bytes(int n_cv) {
    int rec = n_cv <= 3 ? 1 : 2;
    return (size_t)STAGES * SUB * rec * 16 + STAGES * 8 + TILE_R * PSG_MAX_CV * 4 + TILE_R * (1 + PSG_MAX_CV) * 8 + 64;
}

static int hills_grid(const psg_ctx* c) { return c->sm_count * 2; }

size_t psg_hill_part_doubles(const psg_ctx* c, int* max_chunks_out, int* n_rtiles_out) {
    int n_rt = (c->sys.R + TILE_R - 1) / TILE_R;
    int cpt = hills_grid(c) / n_rt;
    if (cpt < 1) cpt = 1;
    if (max_chunks_out) *max_chunks_out = cpt;
    if (n_rtiles_out) *n_rtiles_out = n_rt;
    return (size_t)cpt * n_rt * TILE_R * (1 + PSG_MAX_CV);
}

template <int NCV, int PM, bool F64, bool FUSED>
static cudaError_t launch_k(psg_ctx* c, const HillKernelArgs& A) {
    auto kern = k_hills<NCV, PM, F64, FUSED>;
    size_t smem = hills_smem_bytes(NCV);
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    int n_rt = (c->sys.R + TILE_R - 1) / TILE_R;
    int grid = hills_grid(c);
    (void)n_rt;
    kern<<<grid, HWARPS * 32, smem, c->stream>>>(c->sys, c->md.hc, A);
    c->launches++;
    return cudaGetLastError();
}

template <int NCV, bool F64, bool FUSED>
static cudaError_t dispatch_pm(psg_ctx* c, const HillKernelArgs& A) {
    int pm = c->md.hc.pmask;
    if (NCV == 4) {   // 4 CVs: one generic instantiation per "any periodic" (mask handled at run time via inv_period = 0)
        return pm ? launch_k<4, 15, F64, FUSED>(c, A) : launch_k<4, 0, F64, FUSED>(c, A);
    }
    switch (pm) {
#define PMCASE(m) \
    case m:       \
        if ((m) < (1 << NCV)) return launch_k<NCV, ((m) < (1 << NCV) ? (m) : 0), F64, FUSED>(c, A); \
        break;
        PMCASE(0) PMCASE(1) PMCASE(2) PMCASE(3) PMCASE(4) PMCASE(5) PMCASE(6) PMCASE(7)
#undef PMCASE
    }
    return cudaErrorInvalidValue;
}

template <bool FUSED>
static cudaError_t dispatch(psg_ctx* c, const HillKernelArgs& A) {
    bool f64 = c->md.precision == PSG_HILLS_F64;
    switch (c->sys.n_cv) {
    case 1: return f64 ? dispatch_pm<1, true, FUSED>(c, A) : dispatch_pm<1, false, FUSED>(c, A);
    case 2: return f64 ? dispatch_pm<2, true, FUSED>(c, A) : dispatch_pm<2, false, FUSED>(c, A);
    case 3: return f64 ? dispatch_pm<3, true, FUSED>(c, A) : dispatch_pm<3, false, FUSED>(c, A);
    case 4: return f64 ? dispatch_pm<4, true, FUSED>(c, A) : dispatch_pm<4, false, FUSED>(c, A);
    }
    return cudaErrorInvalidValue;
}

cudaError_t psg_launch_hillsum(psg_ctx* c, const float* d_xi, float* d_V, float* d_dVdxi) {
    HillKernelArgs A{};
    A.hills = c->md.hills; A.n_hills = c->md.n_hills; A.part = c->md.part; A.ticket = c->md.ticket;
    A.xi_in = d_xi; A.V_out = d_V; A.V64_out = c->d_V64; A.dV_out = d_dVdxi; A.R = c->sys.R;
    return dispatch<false>(c, A);
}

bool psg_metad_step_supported(const psg_ctx* c) { return c->sys.n_ranges == 0 && !c->sys.any_rgyr; }

cudaError_t psg_launch_metad_step(psg_ctx* c, const float* d_pos, float* d_force) {
    HillKernelArgs A{};
    A.hills = c->md.hills; A.n_hills = c->md.n_hills; A.part = c->md.part; A.ticket = c->md.ticket;
    A.V_out = c->d_V; A.V64_out = c->d_V64; A.dV_out = c->d_dVdxi; A.xi_out = c->d_xi;
    A.pos = d_pos; A.force = d_force; A.R = c->sys.R;
    return dispatch<true>(c, A);
}

cudaError_t psg_launch_deposit(psg_ctx* c, const float* d_xi, const unsigned char* d_mask) {
    if (c->md.kB_deltaT > 0.0) {
        cudaError_t e = psg_launch_hillsum(c, d_xi, nullptr, nullptr);   // V_old -> d_V64
        if (e != cudaSuccess) return e;
    }
    k_deposit<<<1, 1024, 0, c->stream>>>(c->sys.R, c->sys.n_cv, c->md.rec, d_xi, c->d_V64, d_mask, c->md.w0, c->md.kB_deltaT,
                                         c->md.hills, c->md.n_hills, c->md.capacity);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t psg_launch_pack_hills(psg_ctx* c, int n, const float* d_centers, const float* d_heights) {
    if (n > 0) {
        k_pack_hills<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->sys.n_cv, c->md.rec, d_centers, d_heights, c->md.hills);
        c->launches++;
    }
    return cudaGetLastError();
}

cudaError_t psg_launch_unpack_hills(psg_ctx* c, int n, float* d_centers, float* d_heights) {
    if (n > 0) {
        k_unpack_hills<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->sys.n_cv, c->md.rec, c->md.hills, d_centers, d_heights);
        c->launches++;
    }
    return cudaGetLastError();
}
