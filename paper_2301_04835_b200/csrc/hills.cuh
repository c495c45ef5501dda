// hills.cuh -- the metadynamics hill-sum kernel, also the fused metadynamics step.
//
//   V(xi) = sum_h W_h exp(-1/2 sum_k (d_hk/sigma_k)^2),   dV/dxi_k = -(1/sigma_k^2) sum_h W_h exp(..) d_hk,
//   d_hk = nearest image of xi_k - s_hk.
// Not a dense contraction (the wrap breaks bilinearity; the exp dominates): FP32-pipe + MUFU work, no tensor cores.
//
// Decomposition. CTA = (tile of 64 replicas) x (chunk of hills); ONE CTA of 16 warps per SM. Warps w and w + 8 own the
// same 8 replicas, whose xi sit in registers as 4 packed f32x2 pairs; the 64 lanes of the pair stride over the hills of
// the chunk, which is streamed through shared memory by 1-D TMA bulk copies (cp.async.bulk + mbarrier). One LDS.128
// hill record feeds 8 evaluations. (Two independent 8-warp CTAs per SM were measured to run unevenly -- the scheduler favours one,
// which finishes at half time -- with the same total time; one 16-warp CTA per SM ends all its warps together.)
// All arithmetic of an evaluation is PACKED binary32 (FADD2/FMUL2/FFMA2: two replicas per instruction), which
// halves the issue slots per evaluation and leaves the FMA pipe as the only bound:
//     per periodic dim  d = xi - s; t = d/P + M; k = t - M; d -= k P_hi; d -= k P_lo   (5)
//     exponent          q = d0^2 (+ d1^2 ...);  x = log2(W) - c q                        (NCV + 1 if the sigmas agree)
//     MUFU.EX2 (one per replica), V += e, g_k += e d_k                                   (1 + NCV)
// Binary32 partial sums are flushed into binary64 accumulators (shared memory, thread-private slots) after every
// sub-tile (<= 32 hills per lane); lanes, then chunks, are combined in binary64 in FIXED order (the last CTA of
// a tile, found with a ticket counter, sums the chunk partials), so results are bitwise reproducible.
// FUSED: the CTA first evaluates the CVs (and Jacobians, kept in shared memory) of its tile from the engine's
// positions; the last CTA of the tile scatters -dV/dxi * J into the engine's forces: one launch per MD step.
#pragma once
#include "geom.cuh"

#define RT PSG_HILL_RT
#define HWARPS PSG_HILL_WARPS
#define TILE_R PSG_HILL_TILE_R
#define SUB PSG_HILL_SUB
#ifndef PSG_FLUSH_EVERY
#define PSG_FLUSH_EVERY 2        // sub-tiles (32 hills per lane each) between binary32 -> binary64 flushes
#endif
#define MAGIC_RN 12582912.0f   // 1.5 * 2^23: (x + M) - M = rint(x) for |x| < 2^22

typedef unsigned long long u64;

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

// ---------------------------------------------------------------- packed binary32 (two replicas per instruction)
__device__ __forceinline__ u64 pk(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 sub2(u64 a, u64 b) {
    u64 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

template <int NCV>
__device__ __forceinline__ void load_rec(const float4* __restrict__ sm, int h, float (&s)[NCV], float& lw) {
    if (NCV <= 3) {
        float4 v = sm[h];
        s[0] = v.x;
        if (NCV > 1) s[1 % NCV] = v.y;
        if (NCV > 2) s[2 % NCV] = v.z;
        lw = v.w;
    } else {
        float4 a = sm[2 * h], b = sm[2 * h + 1];
        s[0] = a.x; s[1 % NCV] = a.y; s[2 % NCV] = a.z; s[3 % NCV] = a.w;
        lw = b.x;
    }
}

// One hill against the thread's RT replicas (RT/2 packed pairs). PM = bitmask of periodic CVs; NEQ = number of
// leading CVs sharing sigma_0.  a32[p][0] += e, a32[p][1 + k] += e * d_k for the replica pair p.
template <int NCV, int PM, int NEQ>
struct HillBody {
    u64 INVP[NCV], NPHI[NCV], NPLO[NCV], NC[NCV];
    __device__ __forceinline__ HillBody(const HillConsts& hc) {
#pragma unroll
        for (int k = 0; k < NCV; ++k) {
            INVP[k] = pk(hc.inv_period[k], hc.inv_period[k]);
            NPHI[k] = pk(hc.np_hi[k], hc.np_hi[k]);
            NPLO[k] = pk(hc.np_lo[k], hc.np_lo[k]);
            NC[k] = pk(hc.nc[k], hc.nc[k]);
        }
    }
    __device__ __forceinline__ void operator()(const float4* __restrict__ sm, int h, const u64 (&X)[RT / 2][NCV],
                                               u64 (&a32)[RT / 2][1 + NCV]) const {
        const u64 MG = pk(MAGIC_RN, MAGIC_RN), NMG = pk(-MAGIC_RN, -MAGIC_RN);
        float s[NCV], lw;
        load_rec<NCV>(sm, h, s, lw);
        u64 S[NCV];
#pragma unroll
        for (int k = 0; k < NCV; ++k) S[k] = pk(s[k], s[k]);
        const u64 LW = pk(lw, lw);
#pragma unroll
        for (int p = 0; p < RT / 2; ++p) {
            u64 D[NCV];
#pragma unroll
            for (int k = 0; k < NCV; ++k) {
                u64 d = sub2(X[p][k], S[k]);
                if (PM & (1 << k)) {
                    // nearest image: d -= P rint(d / P), -P = np_hi + np_lo (two constants: the wrap adds no bias)
                    u64 t = fma2(d, INVP[k], MG);
                    u64 kf = add2(t, NMG);
                    d = fma2(kf, NPHI[k], d);
                    d = fma2(kf, NPLO[k], d);
                }
                D[k] = d;
            }
            u64 q = mul2(D[0], D[0]);
#pragma unroll
            for (int k = 1; k < NEQ; ++k) q = fma2(D[k], D[k], q);
            u64 x = fma2(q, NC[0], LW);   // base-2 exponent: log2(W) - sum_k d_k^2 log2(e) / (2 sigma_k^2)
#pragma unroll
            for (int k = NEQ; k < NCV; ++k) x = fma2(mul2(D[k], D[k]), NC[k], x);
            float x0, x1;
            upk(x, x0, x1);
            const u64 E = pk(ex2_approx(x0), ex2_approx(x1));
            a32[p][0] = add2(a32[p][0], E);
#pragma unroll
            for (int k = 0; k < NCV; ++k) a32[p][1 + k] = fma2(E, D[k], a32[p][1 + k]);
        }
    }
};

// binary32 terms over one shared-memory sub-tile: the 64 lanes of a warp pair stride the hills; full groups of 64 run unpredicated
template <int NCV, int PM, int NEQ>
__device__ __forceinline__ void accumulate_f32(const float4* __restrict__ sm, int n_sub, int off, const u64 (&X)[RT / 2][NCV],
                                               const HillConsts& hc, u64 (&a32)[RT / 2][1 + NCV]) {
    // off = lane + 32 * half in [0, 64): this thread takes hills off, off + 64, ...
    const HillBody<NCV, PM, NEQ> body(hc);
    const int n_full = n_sub >> 6;
#pragma unroll 2
    for (int i = 0; i < n_full; ++i) body(sm, off + 64 * i, X, a32);
    if (off + 64 * n_full < n_sub) body(sm, off + 64 * n_full, X, a32);
}

// binary64 terms (PSG_HILLS_F64): the definition, evaluated in double on the FP64 pipe; heights read from the
// exported height array (global). Accumulates straight into the thread's binary64 slots.
template <int NCV>
__device__ __forceinline__ void accumulate_f64(const float4* __restrict__ sm, const float* __restrict__ W, int n_sub, int off,
                                               const float (&xi)[RT][NCV], const HillConsts& hc, double* __restrict__ acc,
                                               int acc_stride) {
    constexpr int NV = 1 + NCV;
    for (int j0 = 0; j0 < RT; j0 += 2) {
        double a[2][NV];
#pragma unroll
        for (int jj = 0; jj < 2; ++jj)
#pragma unroll
            for (int v = 0; v < NV; ++v) a[jj][v] = 0.0;
        for (int h = off; h < n_sub; h += 64) {
            float s[NCV], lw;
            load_rec<NCV>(sm, h, s, lw);
            const double w = (double)__ldg(W + h);
#pragma unroll
            for (int jj = 0; jj < 2; ++jj) {
                double d[NCV], e2 = 0.0;
#pragma unroll
                for (int k = 0; k < NCV; ++k) {
                    d[k] = (double)xi[j0 + jj][k] - (double)s[k];
                    d[k] -= hc.period_d[k] * rint(d[k] / hc.period_d[k]);   // period_d = 1e300 when not periodic
                    double qk = d[k] * hc.inv_sigma_d[k];
                    e2 += qk * qk;
                }
                const double t = w * exp(-0.5 * e2);
                a[jj][0] += t;
#pragma unroll
                for (int k = 0; k < NCV; ++k) a[jj][1 + k] += t * d[k];
            }
        }
#pragma unroll
        for (int jj = 0; jj < 2; ++jj)
#pragma unroll
            for (int v = 0; v < NV; ++v) acc[((j0 + jj) * NV + v) * acc_stride] += a[jj][v];
    }
}

// lane-local CV of (replica r, CV k) for systems with explicit groups only; dc[g] = d xi / d c_g / W_g.
template <bool JAC>
__device__ __forceinline__ double thread_cv(const SysParams& P, int r, int k, const float* __restrict__ pos, D3* dc) {
    const CvDev& C = P.cv[k];
    const float* p = pos + (long long)r * P.rstride * P.ps;
    const int* sa = P.slot_atom + (P.per_rep ? (long long)r * P.n_slots : 0);
    D3 c[4];
    double W[4];
    // Fast path (measured: the gather, not the arithmetic, was half of the prologue): every group a single unweighted
    // atom -- a single atom is its own barycenter -- so all indices are formed first and the four position loads are in
    // flight together instead of one dependent (index -> position) chain per group.
    bool single = !P.slot_weight;
#pragma unroll
    for (int g = 0; g < 4; ++g)
        if (g < C.n_groups) single = single && P.grp[C.gid0 + g].size == 1;
    if (single) {
        long long a[4];
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            const int s = P.grp[C.gid0 + (g < C.n_groups ? g : 0)].begin;   // unused groups re-read group 0 (no branch)
            a[g] = P.per_rep ? sa[s] : P.slot_atom_c[s];                    // shared index lists come from kernel parameters
        }
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            c[g] = load_pos(p, a[g], P.ps);
            W[g] = 1.0;
        }
    } else {
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            c[g] = d3(0, 0, 0);
            W[g] = 1.0;
            if (g < C.n_groups) {
                const GroupDev& G = P.grp[C.gid0 + g];
                double sx = 0, sy = 0, sz = 0, sw = 0;
                const D3 first = load_pos(p, P.per_rep ? sa[G.begin] : P.slot_atom_c[G.begin], P.ps);
                for (int i = 0; i < G.size; ++i) {
                    int s = G.begin + i;
                    D3 x = load_pos(p, P.per_rep ? sa[s] : P.slot_atom_c[s], P.ps);
                    if (P.has_box) x = first + min_image(x - first, P.box);   // the image nearest to the group's first atom
                    double w = P.slot_weight ? (double)P.slot_weight[s] : 1.0;
                    sx += w * x.x; sy += w * x.y; sz += w * x.z; sw += w;
                }
                double iw = 1.0 / sw;
                c[g] = d3(sx * iw, sy * iw, sz * iw);
                W[g] = sw;
            }
        }
    }
    double xi = cv_from_centers<JAC>(C.type, C.axis, c, dc, sys_box(P));
    if (JAC) {
#pragma unroll
        for (int g = 0; g < 4; ++g)
            if (W[g] != 1.0) dc[g] = (1.0 / W[g]) * dc[g];
    }
    return xi;
}

// The force records the final scatter will update, requested into L2 while the hill loop runs: with a cold L2 the
// atomics at the end of the step otherwise wait for DRAM.
__device__ __forceinline__ void prefetch_force_lines(const SysParams& P, int r, int k, const float* force) {
    const CvDev& C = P.cv[k];
    const int* sa = P.slot_atom + (P.per_rep ? (long long)r * P.n_slots : 0);
    for (int g = 0; g < C.n_groups; ++g) {
        const GroupDev& G = P.grp[C.gid0 + g];
        for (int i = 0; i < G.size; ++i) {
            const long long atom = sa[G.begin + i];
            asm volatile("prefetch.global.L2 [%0];" ::"l"(force + ((long long)r * P.rstride + atom) * P.fs));
        }
    }
}

struct HillKernelArgs {
    const float4* hills;     // packed records {s0, s1, s2, log2 W} (n_cv == 4: two float4)
    const float* heights;    // W, as exported
    const int* n_hills;      // device counter (exact), read only when n_h_host < 0 (stream capture)
    int n_h_host;            // host upper bound of the count; records beyond the exact count are null (contribute 0)
    double* part;
    unsigned* ticket;
    const float* xi_in;      // not fused: [R][n_cv]
    float* V_out;            // nullable
    double* V64_out;         // nullable
    float* dV_out;           // nullable
    float* xi_out;           // fused: step outputs
    const float* pos;        // fused
    float* force;            // fused
    int R;
    int fused;
    int stages;              // shared-memory stages of SUB x 16 bytes
#ifdef PSG_TRACE
    long long* trace;        // [grid][8] clock64 stamps of the first item of every CTA (debug builds only)
#endif
};
#ifdef PSG_TRACE
#define PSG_STAMP(i) do { if (threadIdx.x == 0 && item == (int)blockIdx.x && A.trace) { long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); A.trace[blockIdx.x * 8 + (i)] = t_; } } while (0)
#else
#define PSG_STAMP(i) do { } while (0)
#endif

__host__ __device__ inline size_t hills_smem_bytes(int n_cv, int stages, int n_groups, bool fused) {
    int rec = n_cv <= 3 ? 1 : 2;
    (void)rec;
    size_t b = (size_t)stages * SUB * 16;                          // hill stages (SUB / rec hills each)
    b += (size_t)RT * (1 + n_cv) * HWARPS * 32 * 8;                // binary64 accumulators [RT*NV][256]
    b += (size_t)3 * TILE_R * (1 + n_cv) * 8;                      // s_out, s_half[2]
    b += (size_t)TILE_R * n_cv * 4;                                // s_xi
    b += fused ? (size_t)TILE_R * n_groups * 3 * 4 : 0;            // s_jv
    b += 8 * 8 + 64;                                               // barriers, pad
    return b;
}

// One kernel for psg_bias_eval and the whole metadynamics step (A.fused).
template <int NCV, int PM, int NEQ, bool F64>
__global__ void __launch_bounds__(HWARPS * 32, 1) k_hills(const __grid_constant__ SysParams P, const __grid_constant__ HillConsts hc,
                                                           const __grid_constant__ HillKernelArgs A) {
    constexpr int REC = NCV <= 3 ? 1 : 2;
    constexpr int SUBH = SUB / REC;   // hills per stage: a stage is always SUB x 16 bytes
    constexpr int NV = 1 + NCV;
    constexpr int NT = HWARPS * 32;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int STG = A.stages;
    float4* stage = reinterpret_cast<float4*>(smem_raw);                          // STG * SUBH * REC float4
    double* s_acc = reinterpret_cast<double*>(stage + STG * SUBH * REC);           // [RT*NV][NT]
    double* s_out = s_acc + RT * NV * NT;                                         // [TILE_R][NV]
    double* s_half = s_out + TILE_R * NV;                                         // [2][TILE_R][NV]: per-half / per-part sums
    uint64_t* full = reinterpret_cast<uint64_t*>(s_half + 2 * TILE_R * NV);       // 8 barriers
    float* s_xi = reinterpret_cast<float*>(full + 8);                             // [NCV][TILE_R] (pairs of replicas adjacent)
    float* s_jv = s_xi + TILE_R * NCV;                                            // fused: [TILE_R][n_groups][3]
    __shared__ int s_last;
    __shared__ int s_cnt[8];   // warps that have left a stage

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int half = wid >> 3, w8 = wid & 7;   // warps w8 and w8 + 8 own the same replicas; half picks the hills
    const int R = A.R;
    const int n_rt = (R + TILE_R - 1) / TILE_R;
    const int n_h = A.n_h_host >= 0 ? A.n_h_host : *A.n_hills;
    // chunking: as many chunks per tile as the grid allows, chunk length a multiple of 32
    int cpt = (int)gridDim.x / n_rt;
    if (cpt < 1) cpt = 1;
    int Lc = (n_h + cpt - 1) / cpt;
    Lc = ((Lc + 31) / 32) * 32;
    if (Lc < 32) Lc = 32;
    int n_chunks = (n_h + Lc - 1) / Lc;
    if (n_chunks < 1) n_chunks = 1;
    const int items = n_rt * n_chunks;

    if (tid < 8) s_cnt[tid] = 0;
    if (tid == 0) {
        for (int s = 0; s < STG; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // no CTA-wide sync here: thread 0 issues the first TMA loads itself; everybody else first meets the barriers
    // after the __syncthreads that follows the CV prologue
    unsigned seq = 0;   // sub-tiles consumed so far by this CTA (stage = seq % STG, parity = (seq / STG) & 1)

    for (int item = blockIdx.x; item < items; item += gridDim.x) {
        const int tile = item % n_rt, chunk = item / n_rt;
        const int r0 = tile * TILE_R;
        const int h0 = chunk * Lc;
        int len = n_h - h0;
        if (len > Lc) len = Lc;
        if (len < 0) len = 0;
        const int n_st = (len + SUBH - 1) / SUBH;
        PSG_STAMP(0);
        // producer prologue
        if (tid == 0) {
            for (int t = 0; t < n_st && t < STG; ++t) {
                int s = (seq + t) % STG;
                int cnt = min(SUBH, len - t * SUBH);
                mbar_expect_tx(&full[s], (uint32_t)cnt * REC * 16u);
                tma_load_1d(stage + s * SUBH * REC, A.hills + (size_t)(h0 + t * SUBH) * REC, (uint32_t)cnt * REC * 16u, &full[s]);
            }
        }
        // binary64 accumulators of this item
#pragma unroll
        for (int i = 0; i < RT * NV; ++i) s_acc[i * NT + tid] = 0.0;
        // CV values (and per-group Jacobian vectors) of this tile's replicas; overlaps the first TMA loads
        if (A.fused) {
            // the value (gather, cross products, atan2) and the Jacobian (gather, cross products, divisions) of one CV are
            // two serial binary64 chains: different threads (different warps) take them, which shortens the prologue
            for (int t2 = tid; t2 < 2 * TILE_R * NCV; t2 += NT) {
                const bool want_j = t2 >= TILE_R * NCV;
                const int t = want_j ? t2 - TILE_R * NCV : t2;
                const int rr = t / NCV, k = t % NCV, r = r0 + rr;
                if (!want_j) {
                    float v = 0.f;
                    if (r < R) {
                        D3 dc[4];
                        v = (float)thread_cv<false>(P, r, k, A.pos, dc);
                        if (chunk == 0 && A.xi_out) A.xi_out[(long long)r * NCV + k] = v;
                    }
                    s_xi[k * TILE_R + rr] = v;
                } else if (r < R) {
                    D3 dc[4];
                    if (chunk == 0) prefetch_force_lines(P, r, k, A.force);
                    (void)thread_cv<true>(P, r, k, A.pos, dc);
                    const CvDev& C = P.cv[k];
#pragma unroll
                    for (int g = 0; g < 4; ++g)
                        if (g < C.n_groups) {
                            float* j = s_jv + (rr * P.n_groups + C.gid0 + g) * 3;
                            j[0] = (float)dc[g].x; j[1] = (float)dc[g].y; j[2] = (float)dc[g].z;
                        }
                }
            }
        } else {
            for (int t = tid; t < TILE_R * NCV; t += NT) {
                int rr = t / NCV, k = t % NCV;
                s_xi[k * TILE_R + rr] = r0 + rr < R ? A.xi_in[(long long)r0 * NCV + t] : 0.f;
            }
        }
        __syncthreads();
        PSG_STAMP(1);
        const bool warp_active = r0 + w8 * RT < R;
        if (!F64) {
            u64 X[RT / 2][NCV], a32[RT / 2][NV];
#pragma unroll
            for (int p = 0; p < RT / 2; ++p) {
#pragma unroll
                for (int k = 0; k < NCV; ++k)
                    X[p][k] = *reinterpret_cast<const u64*>(s_xi + k * TILE_R + w8 * RT + 2 * p);   // {xi[2p][k], xi[2p+1][k]}
#pragma unroll
                for (int v = 0; v < NV; ++v) a32[p][v] = 0ull;
            }
            for (int t = 0; t < n_st; ++t) {
                int s = seq % STG;
                mbar_wait(&full[s], (seq / STG) & 1);
                int cnt = min(SUBH, len - t * SUBH);
                if (warp_active) {
                    // a full sub-tile gets a compile-time trip count (the compiler then schedules across iterations)
                    if (cnt == SUBH) accumulate_f32<NCV, PM, NEQ>(stage + s * SUBH * REC, SUBH, lane + 32 * half, X, hc, a32);
                    else accumulate_f32<NCV, PM, NEQ>(stage + s * SUBH * REC, cnt, lane + 32 * half, X, hc, a32);
                }
                if (warp_active && ((t % PSG_FLUSH_EVERY) == PSG_FLUSH_EVERY - 1 || t == n_st - 1)) {
                    // flush the binary32 partial sums (<= 64 hills per lane: 4 sub-tiles of 16) into the binary64 slots
#pragma unroll
                    for (int p = 0; p < RT / 2; ++p)
#pragma unroll
                        for (int v = 0; v < NV; ++v) {
                            float lo, hi;
                            upk(a32[p][v], lo, hi);
                            s_acc[((2 * p) * NV + v) * NT + tid] += (double)lo;
                            s_acc[((2 * p + 1) * NV + v) * NT + tid] += (double)hi;
                            a32[p][v] = 0ull;
                        }
                }
                // No CTA-wide barrier per sub-tile (measured: the bare loop reaches 0.95 of the FFMA peak, the loop with a
                // barrier per 1,024 hills 0.80): warps drift freely, and the warp that leaves a stage LAST refills it.
                __syncwarp();
                if (lane == 0) {
                    if (atomicAdd(&s_cnt[s], 1) == HWARPS - 1) {
                        s_cnt[s] = 0;
                        if (t + STG < n_st) {
                            int cn = min(SUBH, len - (t + STG) * SUBH);
                            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                            mbar_expect_tx(&full[s], (uint32_t)cn * REC * 16u);
                            tma_load_1d(stage + s * SUBH * REC, A.hills + (size_t)(h0 + (t + STG) * SUBH) * REC,
                                        (uint32_t)cn * REC * 16u, &full[s]);
                        }
                    }
                }
                ++seq;
            }
        } else {
            float xi[RT][NCV];
#pragma unroll
            for (int j = 0; j < RT; ++j)
#pragma unroll
                for (int k = 0; k < NCV; ++k) xi[j][k] = s_xi[k * TILE_R + w8 * RT + j];
            for (int t = 0; t < n_st; ++t) {
                int s = seq % STG;
                mbar_wait(&full[s], (seq / STG) & 1);
                int cnt = min(SUBH, len - t * SUBH);
                if (warp_active)
                    accumulate_f64<NCV>(stage + s * SUBH * REC, A.heights + h0 + t * SUBH, cnt, lane + 32 * half, xi, hc, s_acc + tid, NT);
                __syncwarp();
                if (lane == 0) {
                    if (atomicAdd(&s_cnt[s], 1) == HWARPS - 1) {
                        s_cnt[s] = 0;
                        if (t + STG < n_st) {
                            int cn = min(SUBH, len - (t + STG) * SUBH);
                            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                            mbar_expect_tx(&full[s], (uint32_t)cn * REC * 16u);
                            tma_load_1d(stage + s * SUBH * REC, A.hills + (size_t)(h0 + (t + STG) * SUBH) * REC,
                                        (uint32_t)cn * REC * 16u, &full[s]);
                        }
                    }
                }
                ++seq;
            }
        }
        PSG_STAMP(2);
        // lanes -> warp totals through the shared accumulators: lane v (< RT*NV) sums value v over the 32 lanes
        // (rotated start => no bank conflicts; the order is fixed per lane => deterministic)
        __syncwarp();
        constexpr int TV = TILE_R * NV;
        double* dst = s_half + half * TV + w8 * RT * NV;
        for (int v = lane; v < RT * NV; v += 32) {
            const double* src = s_acc + v * NT + wid * 32;
            double sum = 0.0;
#pragma unroll 8
            for (int i = 0; i < 32; ++i) sum += src[(i + lane) & 31];
            dst[v] = sum;
        }
        __syncthreads();
        // the two warp halves in fixed order -> this chunk's partial of the tile
        for (int t = tid; t < TV; t += NT) A.part[(size_t)(chunk * n_rt + tile) * TV + t] = s_half[t] + s_half[TV + t];
        __syncthreads();
        PSG_STAMP(3);
        if (tid == 0) {
            // release: the CTA's partials (ordered before this by the barrier) are visible to whoever acquires the ticket
            unsigned old;
            asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(A.ticket + tile) : "memory");
            s_last = (old == (unsigned)(n_chunks - 1));
        }
        __syncthreads();
        PSG_STAMP(4);
        if (s_last) {   // block-uniform: this CTA finishes the tile
            // chunk partials in fixed order; two thread groups split the chunks so that more loads are in flight
            constexpr int PARTS = NT >= 2 * TV ? 2 : 1;
            const size_t cstride = (size_t)n_rt * TV;
            const int cn = (n_chunks + PARTS - 1) / PARTS;
            for (int t = tid; t < PARTS * TV; t += NT) {
                const int pt = t / TV, v = t - pt * TV;
                const double* src = A.part + (size_t)tile * TV + v;
                const int c1 = min(n_chunks, (pt + 1) * cn);
                double sum = 0.0;
#pragma unroll 9
                for (int c = pt * cn; c < c1; ++c) sum += __ldcg(src + c * cstride);
                s_half[pt * TV + v] = sum;
            }
            __syncthreads();
            for (int t = tid; t < TV; t += NT) {
                double sum = s_half[t];
                if (PARTS == 2) sum += s_half[TV + t];
                int v = t % NV;
                if (v > 0) sum *= -hc.gscale[v - 1];
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
            if (A.fused) {
                __syncthreads();
                PSG_STAMP(5);
                // forces: one thread per (replica, slot); red.global.add (atoms shared by CVs / walkers collide)
                for (int t = tid; t < TILE_R * P.n_slots; t += NT) {
                    int rr = t / P.n_slots, s = t % P.n_slots, r = r0 + rr;
                    if (r >= R) continue;
                    int gid = P.slot_gid[s];
                    // same rounding as the unfused path: dV/dxi and J pass through binary32
                    float fdv = -(float)s_out[rr * NV + 1 + P.grp[gid].cv];
                    float w = P.slot_weight ? P.slot_weight[s] : 1.f;
                    const float* j = s_jv + (rr * P.n_groups + gid) * 3;
                    int atom = P.slot_atom[(P.per_rep ? (long long)r * P.n_slots : 0) + s];
                    float* fa = A.force + ((long long)r * P.rstride + atom) * P.fs;
                    force_add(fa, fdv * (w * j[0]), fdv * (w * j[1]), fdv * (w * j[2]), P.fs);
                }
            }
        }
        __syncthreads();   // s_xi / s_out / s_acc / s_last are reused by the next item
        PSG_STAMP(6);
#ifdef PSG_TRACE
        if (threadIdx.x == 0 && item == (int)blockIdx.x && A.trace) {
            unsigned smid; asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
            A.trace[blockIdx.x * 8 + 7] = smid;
        }
#endif
    }
}
