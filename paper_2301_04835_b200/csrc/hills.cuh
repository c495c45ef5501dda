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
// Binary32 partial sums (<= 64 hills per lane) are flushed into binary64 by a warp-wide transpose-reduction (31 shuffle +
// add steps turn 32 per-lane values into one warp total per lane): the binary64 accumulators are ONE slot per lane (4 KB per CTA), not
// 98-131 KB of shared memory, which leaves the SM's shared memory to the hill stages (3 x 64 KB in flight).  Lanes (butterfly),
// warps, then chunks are combined in binary64 in FIXED order (the CTA of a tile's chunk 0 collects the other chunks'
// published partials, each word carrying its own valid flag), so results are bitwise reproducible.
// FUSED: the CTA first evaluates the CVs (and Jacobians, kept in shared memory) of its tile from the engine's
// positions; the finishing CTA of the tile scatters -dV/dxi * J into the engine's forces: one launch per MD step.
#pragma once
#include "geom.cuh"

#define RT PSG_HILL_RT
#define HWARPS PSG_HILL_WARPS
#define HHALF PSG_HILL_HALF
#define TILE_R PSG_HILL_TILE_R
#define SUB PSG_HILL_SUB
#ifndef PSG_FLUSH_EVERY
#define PSG_FLUSH_EVERY 1        // sub-tiles (64 hills per lane each; 32 with 4 CVs) between binary32 -> binary64 flushes
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

// non-blocking poll (acquire): true if the phase with this parity has completed
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 P1, [%1], %2;\n"
        "selp.u32 %0, 1, 0, P1;\n"
        "}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}

// ---------------------------------------------------------------- packed binary32 (two replicas per instruction)
__device__ __forceinline__ u64 pk(float lo, float hi) {
    u64 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
// the same, opaque to common-subexpression elimination: every call is its own mov.b64 in the PTX (see HillBody)
__device__ __forceinline__ u64 pk_once(float lo, float hi) {
    u64 r;
    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
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
// accumulate in place (read-write operand): biases the register allocator towards updating the accumulator's own pair
// instead of rotating it through a copy at the loop's back edge
__device__ __forceinline__ void acc_add2(u64& a, u64 b) { asm("add.rn.f32x2 %0, %0, %1;" : "+l"(a) : "l"(b)); }
__device__ __forceinline__ void acc_fma2(u64& a, u64 b, u64 c) { asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(a) : "l"(b), "l"(c)); }
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
        // (the {s, s} pairs are formed at every use, not once per hill: a single-use pair is what ptxas reliably folds
        // into the scalar-broadcast operand form of the packed instruction; a shared one it sometimes materialises with
        // two MOVs per value -- +10 % instructions in the loop)
#pragma unroll
        for (int p = 0; p < RT / 2; ++p) {
            u64 D[NCV];
#pragma unroll
            for (int k = 0; k < NCV; ++k) {
                u64 d = sub2(X[p][k], pk_once(s[k], s[k]));
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
            u64 x = fma2(q, NC[0], pk_once(lw, lw));   // base-2 exponent: log2(W) - sum_k d_k^2 log2(e) / (2 sigma_k^2)
#pragma unroll
            for (int k = NEQ; k < NCV; ++k) x = fma2(mul2(D[k], D[k]), NC[k], x);
            float x0, x1;
            upk(x, x0, x1);
            const u64 E = pk(ex2_approx(x0), ex2_approx(x1));
            acc_add2(a32[p][0], E);
#pragma unroll
            for (int k = 0; k < NCV; ++k) acc_fma2(a32[p][1 + k], E, D[k]);
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

#ifndef PSG_ACC_IN_REGS
#define PSG_ACC_IN_REGS(NCV) 0
#endif
#ifndef PSG_PEND_VARS
#define PSG_PEND_VARS(NCV) ((NCV) >= 3)
#endif
// Warp-wide transpose-reduction of the thread's binary32 partial sums into binary64: value i = (2 p + h) NV + v of the
// thread's RT replicas (padded with zeros to 32 per pass); after the steps xor 16, 8, 4, 2, 1 lane l holds the sum over the
// warp's 32 lanes of value 32 pass + l, which it adds to its own slot of the warp's binary64 accumulators wacc[32 pass + l] (shared
// memory; a register would be taken from the hill loop, which needs all 128).  Every addition is binary64, in an order fixed
// by the lane numbers.  a32 is cleared.
template <int NCV>
__device__ __forceinline__ void butterfly_flush(u64 (&a32)[RT / 2][1 + NCV], double (&accd)[(RT * (1 + NCV) + 31) / 32],
                                                double* __restrict__ wacc, int lane) {
    constexpr int NV = 1 + NCV, NVAL = RT * NV, PASSES = (NVAL + 31) / 32;
    float f[32 * PASSES];
#pragma unroll
    for (int i = 0; i < 32 * PASSES; ++i) f[i] = 0.f;
#pragma unroll
    for (int p = 0; p < RT / 2; ++p)
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            upk(a32[p][v], f[(2 * p) * NV + v], f[(2 * p + 1) * NV + v]);
            a32[p][v] = 0ull;
        }
#pragma unroll
    for (int ps = 0; ps < PASSES; ++ps) {
        double w[16];
        const bool up16 = (lane & 16) != 0;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            // the first step exchanges binary32 (one shuffle) and converts after: the sum itself is binary64
            const float a = f[32 * ps + i], b = f[32 * ps + i + 16];
            const float keep = up16 ? b : a, send = up16 ? a : b;
            w[i] = (double)keep + (double)__shfl_xor_sync(0xffffffffu, send, 16);
        }
#pragma unroll
        for (int m = 8; m >= 1; m >>= 1) {
            const bool up = (lane & m) != 0;
#pragma unroll
            for (int i = 0; i < m; ++i) {
                const double keep = up ? w[i + m] : w[i], send = up ? w[i] : w[i + m];
                w[i] = keep + __shfl_xor_sync(0xffffffffu, send, m);
            }
        }
        // the lane's running total: a register where the hill loop can spare one (measured per NCV: the loop's schedule is
        // sensitive to a single register at the 128-register limit), else its own slot of the warp's shared-memory accumulators
        if (PSG_ACC_IN_REGS(NCV)) accd[ps] += w[0];
        else wacc[32 * ps + lane] += w[0];
    }
}

// binary64 terms (PSG_HILLS_F64): the definition, evaluated in double on the FP64 pipe; heights read from the
// exported height array (global).  Two replicas at a time over the sub-tile; their sums are reduced over the warp by
// shuffles (binary64, fixed order) and lane 0 adds them to the warp's accumulators wacc[RT * NV] in shared memory.
template <int NCV>
__device__ __forceinline__ void accumulate_f64(const float4* __restrict__ sm, const float* __restrict__ W, int n_sub, int off,
                                               const float (&xi)[RT][NCV], const HillConsts& hc, double* __restrict__ wacc, int lane) {
    constexpr int NV = 1 + NCV;
#pragma unroll   // (static replica indices keep xi in registers; a rolled loop puts it in local memory)
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
            for (int v = 0; v < NV; ++v) {
                const double t = warp_sum(a[jj][v]);
                if (lane == 0) wacc[(j0 + jj) * NV + v] += t;
            }
    }
    __syncwarp();
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
    int n_long;              // > 0: uneven chunking (hills_spare_chunking): CTA b < n_long runs item b only, the grid - n_long CTAs
                             // behind them share the short last chunks of all tiles: items b, b + (grid - n_long), ...  (It sits in
                             // the padding after n_h_host: the struct must not grow into another constant-cache line, whose cold
                             // miss after an L2 flush costs the fused step 2 us.)
    double* part;
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
    int Lc_host, n_chunks_host;   // the chunking for n_h_host (computed on the host: three integer divisions off the kernel's entry path)
    float inv_n_rt;          // 1 / (number of replica tiles), for the item -> (tile, chunk) split
    int simple;              // fused: every group one unweighted atom, no box: the lean gather (SysParams::cv_slot / cv_atom)
};

// chunk length (a multiple of 32, at least 32) and number of chunks per replica tile for n_h hills on `grid` CTAs
__host__ __device__ inline void hills_chunking(int n_h, int grid, int n_rt, int& Lc, int& n_chunks) {
    int cpt = grid / n_rt;
    if (cpt < 1) cpt = 1;
    Lc = (n_h + cpt - 1) / cpt;
    Lc = ((Lc + 31) / 32) * 32;
    if (Lc < 32) Lc = 32;
    n_chunks = (n_h + Lc - 1) / Lc;
    if (n_chunks < 1) n_chunks = 1;
}
// Which instantiations take the uneven chunking below.  The hill loop sits at the 128-register limit and its code changes with
// anything that is live across it: the 1- and 2-CV kernels lost 2 % to two extra moves with this in (config 1, whose chunks are
// too short to gain anyway), the 3-CV kernel gained; the binary64-term kernels are left as they were measured.
#ifndef PSG_SPARE_CHUNKS
#define PSG_SPARE_CHUNKS(NCV, F64) ((NCV) >= 3 && !(F64))
#endif
// When the grid is not a multiple of the tile count, grid - cpt * n_rt CTAs would idle (config 4: 16 tiles x 9 chunks = 144 of
// 148).  Host only: shorten the cpt long chunks of every tile and add one SHORT last chunk per tile; the spare CTAs run those,
// m = ceil(n_rt / spare) each.  The short length x balances m (x + o) = (n_h - x) / cpt + o, o = the fixed cost of one item
// (launch-to-loop, flushes, publish) in hills.  Returns false (nothing changed) when the long chunks are too short to gain.
__host__ inline bool hills_spare_chunking(int n_h, int grid, int n_rt, int& Lc, int& n_chunks, int& n_long) {
    const int cpt = grid / n_rt, spare = grid - cpt * n_rt;
    if (cpt < 2 || spare <= 0 || n_chunks != cpt || Lc < 8192) return false;
    const int m = (n_rt + spare - 1) / spare;
    const double o = 600.0;
    const double x = ((double)n_h / cpt + o - m * o) / (m + 1.0 / cpt);
    if (x < 64.0) return false;
    int L = (int)(((double)n_h - x) / cpt);
    L = ((L + 31) / 32) * 32;
    if (L >= Lc || n_h - cpt * L < 32) return false;
    Lc = L; n_chunks = cpt + 1; n_long = cpt * n_rt;
    return true;
}
__host__ __device__ inline size_t hills_wacc_doubles(int n_cv) { return (size_t)((RT * (1 + n_cv) + 31) / 32) * 32; }
__host__ __device__ inline size_t hills_smem_bytes(int n_cv, int stages, int n_groups, bool fused) {
    size_t b = (size_t)stages * SUB * 16;                          // hill stages (SUB / rec hills each)
    b += (size_t)HWARPS * hills_wacc_doubles(n_cv) * 8;            // per-warp binary64 totals
    b += (size_t)3 * TILE_R * (1 + n_cv) * 8;                      // s_out, s_half[2]
    b += (size_t)TILE_R * n_cv * 4;                                // s_xi
    b += fused ? (size_t)TILE_R * n_groups * 4 * 4 : 0;            // s_jv, s_ja
    b += 8 * 8 + 64;                                               // barriers, pad
    return b;
}
#ifndef PSG_HILL_MAX_STAGES
#define PSG_HILL_MAX_STAGES 3
#endif

// item -> (tile, chunk) without an integer division: a binary32 quotient, corrected by one (item < 2^24)
__device__ __forceinline__ void hills_item(int item, int n_rt, float inv_n_rt, int& tile, int& chunk) {
    chunk = (int)((float)item * inv_n_rt);
    if (chunk * n_rt > item) --chunk;
    else if ((chunk + 1) * n_rt <= item) ++chunk;
    tile = item - chunk * n_rt;
}
// the atoms of CV k of replica r in the lean gather (every group one atom): one table look-up per group
__device__ __forceinline__ void hills_cv_atoms(const SysParams& P, int r, int k, int (&a)[4]) {
    if (P.per_rep) {
        const int* sa = P.slot_atom + (long long)r * P.n_slots;
#pragma unroll
        for (int g = 0; g < 4; ++g) a[g] = __ldg(sa + P.cv_slot[k * PSG_MAX_GROUPS + g]);
    } else {
#pragma unroll
        for (int g = 0; g < 4; ++g) a[g] = P.cv_atom[k * PSG_MAX_GROUPS + g];
    }
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
    constexpr int WACC = ((RT * NV + 31) / 32) * 32;   // per-warp binary64 totals (padded to whole butterfly passes)
    constexpr int PASSES = WACC / 32;
    const int STG = A.stages;
    float4* stage = reinterpret_cast<float4*>(smem_raw);                          // STG * SUBH * REC float4
    double* s_wacc = reinterpret_cast<double*>(stage + STG * SUBH * REC);          // [HWARPS][WACC]
    double* s_out = s_wacc + HWARPS * WACC;                                       // [TILE_R][NV]
    double* s_half = s_out + TILE_R * NV;                                         // [2][TILE_R][NV]: per-part sums of the last CTA
    uint64_t* full = reinterpret_cast<uint64_t*>(s_half + 2 * TILE_R * NV);       // 8 barriers
    float* s_xi = reinterpret_cast<float*>(full + 8);                             // [NCV][TILE_R] (pairs of replicas adjacent)
    float* s_jv = s_xi + TILE_R * NCV;                                            // fused: [TILE_R][n_groups][3]
    int* s_ja = reinterpret_cast<int*>(s_jv + TILE_R * P.n_groups * 3);           // fused, lean gather: [TILE_R][n_groups] atom of the group
    __shared__ int s_cnt[8];   // warps that have left a stage

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int half = wid / HHALF, w8 = wid % HHALF;   // warps w8 and w8 + HHALF own the same replicas; half picks the hills
    const int R = A.R;
    const int n_rt = (R + TILE_R - 1) / TILE_R;
    // Lean gather, FIRST thing in the kernel: the position loads of this CTA's first item are on the critical path of
    // the launch (measured: ~250 set-up instructions at a cold instruction cache otherwise precede them), so they are
    // issued before anything else.  They are consumed BEFORE the item loop (lean_finish below): registers that stayed live
    // into the loop would be taken from the hill loop.
    static_assert(2 * TILE_R * NCV <= NT, "one pass of the CV prologue covers a tile");
    static_assert(sizeof(HillKernelArgs) == 128, "HillKernelArgs is two 64-byte constant lines");
    const bool early = A.fused && A.simple && A.n_h_host >= 0 && (int)blockIdx.x < n_rt * A.n_chunks_host;   // CTA-uniform
    float4 pre[4];
    int pre_a[4];
    int tile0 = 0, chunk0 = 0;
    if (early) {
        hills_item((int)blockIdx.x, n_rt, A.inv_n_rt, tile0, chunk0);
        const int t = tid >= TILE_R * NCV ? tid - TILE_R * NCV : tid;
        const int r = tile0 * TILE_R + t / NCV;
        if (tid < 2 * TILE_R * NCV && r < R) {
            hills_cv_atoms(P, r, t % NCV, pre_a);
            const float* p = A.pos + (long long)r * P.rstride * P.ps;
#pragma unroll
            for (int g = 0; g < 4; ++g) pre[g] = load_pos_raw(p, pre_a[g], P.ps);
        }
    }
    // chunking: as many chunks per tile as the grid allows, chunk length a multiple of 32 (hills_chunking: the host did
    // these divisions when it knows the hill count; under stream capture the count is the device counter's)
    int n_h, Lc, n_chunks;
    if (A.n_h_host >= 0) {
        n_h = A.n_h_host; Lc = A.Lc_host; n_chunks = A.n_chunks_host;
    } else {
        n_h = *A.n_hills;
        hills_chunking(n_h, (int)gridDim.x, n_rt, Lc, n_chunks);
    }
    const int items = n_rt * n_chunks;
    // One thread with no CV work of its own (lane 0 of the last warp) owns the barriers and the first TMA loads of an item;
    // nobody else touches them before the __syncthreads that follows the CV prologue.
    const bool producer = tid == NT - 32;
    if (producer) {
        for (int i = 0; i < 8; ++i) s_cnt[i] = 0;
        for (int s = 0; s < STG; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    unsigned seq = 0;   // sub-tiles consumed so far by this CTA (stage = seq % STG, parity = (seq / STG) & 1)

    // Lean gather (every group a single unweighted atom, no box: the ADP dihedrals of PAPER.md:L81 and every BASELINE.json
    // metadynamics config): a single atom is its own barycenter, so a thread forms its four atom indices from one table
    // look-up each and has all four position loads in flight at once.  The value (cross products, atan2) and the Jacobian
    // (cross products, reciprocals without subroutine calls) of a CV are taken by different threads; both chains are a few
    // hundred cycles once the loads are back.  lean_finish: positions -> xi (shared memory, step output) or Jacobian
    // vectors + atoms (shared memory, for the scatter).
    auto lean_finish = [&](bool want_j, int rr, int k, int r, bool first_chunk, const int (&a)[4], const float4 (&raw)[4]) {
        if (r < R) {
            D3 c[4], dc[4];
#pragma unroll
            for (int g = 0; g < 4; ++g) c[g] = d3((double)raw[g].x, (double)raw[g].y, (double)raw[g].z);
            const CvDev& C = P.cv[k];
            if (!want_j) {
                const float v = (float)cv_from_centers<false>(C.type, C.axis, c, dc, nullptr);
                if (first_chunk && A.xi_out) A.xi_out[(long long)r * NCV + k] = v;
                s_xi[k * TILE_R + rr] = v;
            } else {
                if (first_chunk) {   // the force records the final scatter will update, requested into L2 now
#pragma unroll
                    for (int g = 0; g < 4; ++g)
                        if (g < C.n_groups)
                            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.force + ((long long)r * P.rstride + a[g]) * P.fs));
                }
                cv_jacobian_only(C.type, C.axis, c, dc);
#pragma unroll
                for (int g = 0; g < 4; ++g)
                    if (g < C.n_groups) {
                        float* j = s_jv + (rr * P.n_groups + C.gid0 + g) * 3;
                        j[0] = (float)dc[g].x; j[1] = (float)dc[g].y; j[2] = (float)dc[g].z;
                        s_ja[rr * P.n_groups + C.gid0 + g] = a[g];   // the scatter needs no index load of its own
                    }
            }
        } else if (!want_j) {
            s_xi[k * TILE_R + rr] = 0.f;
        }
    };
    bool lean_done = false;
    if (early) {   // the first item's prologue, from the loads issued at the top of the kernel
        if (tid < 2 * TILE_R * NCV) {
            const bool want_j = tid >= TILE_R * NCV;
            const int t = want_j ? tid - TILE_R * NCV : tid;
            lean_finish(want_j, t / NCV, t % NCV, tile0 * TILE_R + t / NCV, chunk0 == 0, pre_a, pre);
        }
        lean_done = true;
    }

    // (the step is recomputed from the kernel parameters at the end of an item: a value kept live across the hill loop costs it
    // moves; and only the instantiations that use the uneven chunking compile it: PSG_SPARE_CHUNKS)
    for (int item = blockIdx.x; item < items;
         item += (PSG_SPARE_CHUNKS(NCV, F64) && A.n_long > 0) ? ((int)blockIdx.x < A.n_long ? items : (int)gridDim.x - A.n_long) : (int)gridDim.x) {
        int tile, chunk;
        hills_item(item, n_rt, A.inv_n_rt, tile, chunk);
        const int r0 = tile * TILE_R;
        const int h0 = chunk * Lc;
        int len = n_h - h0;
        if (len > Lc) len = Lc;
        if (len < 0) len = 0;
        const int n_st = (len + SUBH - 1) / SUBH;
        if (producer) {
            for (int t = 0; t < n_st && t < STG; ++t) {
                int s = (seq + t) % STG;
                int cnt = min(SUBH, len - t * SUBH);
                mbar_expect_tx(&full[s], (uint32_t)cnt * REC * 16u);
                tma_load_1d(stage + s * SUBH * REC, A.hills + (size_t)(h0 + t * SUBH) * REC, (uint32_t)cnt * REC * 16u, &full[s]);
            }
        }
        // CV values (and per-group Jacobian vectors) of this tile's replicas; overlaps the first TMA loads
        if (A.fused && A.simple) {
            if (!lean_done) {
                for (int t2 = tid; t2 < 2 * TILE_R * NCV; t2 += NT) {
                    const bool want_j = t2 >= TILE_R * NCV;
                    const int t = want_j ? t2 - TILE_R * NCV : t2;
                    const int rr = t / NCV, k = t % NCV, r = r0 + rr;
                    int a[4];
                    float4 raw[4];
                    if (r < R) {
                        hills_cv_atoms(P, r, k, a);
                        const float* p = A.pos + (long long)r * P.rstride * P.ps;
#pragma unroll
                        for (int g = 0; g < 4; ++g) raw[g] = load_pos_raw(p, a[g], P.ps);
                    }
                    lean_finish(want_j, rr, k, r, chunk == 0, a, raw);
                }
            }
            lean_done = false;
        } else if (A.fused) {
            // the general gather (groups of several atoms, weights, minimum image): value and Jacobian again in different threads
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
        const bool warp_active = r0 + w8 * RT < R;
        // Stage hand-back without a CTA-wide barrier (measured: the bare loop reaches 0.95 of the FFMA peak, the loop with a
        // barrier per 1,024 hills 0.80): warps drift freely; lane 0 counts its warp out of the stage with a shared-memory
        // atomic, and the warp that left LAST refills it.  The atomic's result is only looked at one sub-tile LATER, so
        // nobody waits for its round trip (STG >= 3 keeps the refill two sub-tiles ahead of its use); likewise the barrier
        // of the NEXT stage is polled (test_wait) before the bookkeeping, and the blocking wait is skipped when it was ready.
        // (whether the previous sub-tile's stage and index are kept in registers or re-derived from seq and t changes the
        // register allocation of the hill loop, hence PSG_PEND_VARS, chosen per NCV like PSG_ACC_IN_REGS)
        int pend_old = -1;      // lane 0: the count-out of the previous sub-tile (stage (seq - 1) % STG, sub-tile t - 1)
        int pend_s = 0, pend_t = 0;
        bool ready = false;
        auto hand_back = [&](int s, int t) {
            if (lane == 0) {
                if (pend_old == HWARPS - 1) {
                    const int ps = PSG_PEND_VARS(NCV) ? pend_s : (int)((seq + STG - 1) % STG), pt = PSG_PEND_VARS(NCV) ? pend_t : t - 1;
                    s_cnt[ps] = 0;
                    if (pt + STG < n_st) {
                        const int cn = min(SUBH, len - (pt + STG) * SUBH);
                        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                        mbar_expect_tx(&full[ps], (uint32_t)cn * REC * 16u);
                        tma_load_1d(stage + ps * SUBH * REC, A.hills + (size_t)(h0 + (pt + STG) * SUBH) * REC, (uint32_t)cn * REC * 16u,
                                    &full[ps]);
                    }
                }
                pend_old = atomicAdd(&s_cnt[s], 1);
                if (PSG_PEND_VARS(NCV)) { pend_s = s; pend_t = t; }
            }
        };
        if (!F64) {
            u64 X[RT / 2][NCV], a32[RT / 2][NV];
            double accd[PASSES];
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps) {
                accd[ps] = 0.0;
                s_wacc[wid * WACC + 32 * ps + lane] = 0.0;
            }
#pragma unroll
            for (int p = 0; p < RT / 2; ++p) {
#pragma unroll
                for (int k = 0; k < NCV; ++k)
                    X[p][k] = *reinterpret_cast<const u64*>(s_xi + k * TILE_R + w8 * RT + 2 * p);   // {xi[2p][k], xi[2p+1][k]}
#pragma unroll
                for (int v = 0; v < NV; ++v) a32[p][v] = 0ull;
            }
            for (int t = 0; t < n_st; ++t) {
                const int s = seq % STG;
                if (!ready) mbar_wait(&full[s], (seq / STG) & 1);
                const int cnt = min(SUBH, len - t * SUBH);
                if (warp_active) {
                    // a full sub-tile gets a compile-time trip count (the compiler then schedules across iterations)
                    if (cnt == SUBH) accumulate_f32<NCV, PM, NEQ>(stage + s * SUBH * REC, SUBH, lane + 32 * half, X, hc, a32);
                    else accumulate_f32<NCV, PM, NEQ>(stage + s * SUBH * REC, cnt, lane + 32 * half, X, hc, a32);
                }
#ifndef PSG_NO_EARLY_POLL
                ready = t + 1 < n_st && mbar_test(&full[(seq + 1) % STG], ((seq + 1) / STG) & 1);
#endif
                // flush the binary32 partial sums (<= 64 hills per lane) into the lanes' binary64 registers (with
                // PSG_FLUSH_EVERY > 1 the four warps of a scheduler, wid mod 4, flush at different sub-tiles; with one flush per
                // 64-hill sub-tile the warps drift apart by themselves)
#ifdef PSG_NO_STAGGER
                const int ph = 0;
#else
                const int ph = (wid >> 2) % PSG_FLUSH_EVERY;
#endif
                if (warp_active && (((t + ph) % PSG_FLUSH_EVERY) == PSG_FLUSH_EVERY - 1 || t == n_st - 1)) butterfly_flush<NCV>(a32, accd, s_wacc + wid * WACC, lane);
                __syncwarp();
                hand_back(s, t);
                ++seq;
            }
            if (PSG_ACC_IN_REGS(NCV)) {
#pragma unroll
                for (int ps = 0; ps < PASSES; ++ps) s_wacc[wid * WACC + 32 * ps + lane] = accd[ps];
            }
        } else {
            float xi[RT][NCV];
#pragma unroll
            for (int j = 0; j < RT; ++j)
#pragma unroll
                for (int k = 0; k < NCV; ++k) xi[j][k] = s_xi[k * TILE_R + w8 * RT + j];
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps) s_wacc[wid * WACC + 32 * ps + lane] = 0.0;
            __syncwarp();
            for (int t = 0; t < n_st; ++t) {
                const int s = seq % STG;
                mbar_wait(&full[s], (seq / STG) & 1);
                const int cnt = min(SUBH, len - t * SUBH);
                if (warp_active)
                    accumulate_f64<NCV>(stage + s * SUBH * REC, A.heights + h0 + t * SUBH, cnt, lane + 32 * half, xi, hc, s_wacc + wid * WACC, lane);
                __syncwarp();
                hand_back(s, t);
                ++seq;
            }
        }
        if (lane == 0 && pend_old == HWARPS - 1) s_cnt[PSG_PEND_VARS(NCV) ? pend_s : (int)((seq + STG - 1) % STG)] = 0;   // the item's last count-out (nothing left to refill)
        constexpr int TV = TILE_R * NV;
        __syncthreads();
        // Warps w8 and w8 + HHALF (the two halves of the chunk's hills) in fixed order -> this chunk's partial of the tile.
        // The CTA of chunk 0 FINISHES the tile: the others publish their partials and are done; it keeps its own on chip
        // and collects theirs.  A published value is ONE 64-bit word that carries its own valid flag -- the lowest mantissa
        // bit, forced to 1 (a deterministic perturbation of at most 1 ulp of binary64; a cleared word is 0) -- so a single
        // relaxed 8-byte load either sees the new value or knows it is not there yet: no ticket, no fence, one L2 round trip
        // between the end of the hill loop and the sums.  The finisher clears what it consumed for the next launch.  (A
        // launch runs one item per CTA whenever a tile has several chunks, and only finishers wait, so nothing can deadlock.)
        const bool finisher = chunk == 0;   // block-uniform
        u64* const part_bits = reinterpret_cast<u64*>(A.part);
        for (int t = tid; t < TV; t += NT) {
            const int rr = t / NV, v = t - rr * NV, ww = rr / RT, j = rr - ww * RT;
            const double val = s_wacc[ww * WACC + j * NV + v] + s_wacc[(ww + HHALF) * WACC + j * NV + v];
            if (finisher) s_out[t] = val;
            else __stcg(part_bits + (size_t)(chunk * n_rt + tile) * TV + t, (u64)__double_as_longlong(val) | 1ull);
        }
        if (finisher) {
            __syncthreads();
            // chunk partials in fixed order; two thread groups split the chunks so that more loads are in flight
            constexpr int PARTS = NT >= 2 * TV ? 2 : 1;
            constexpr int BATCH = 9;   // words in flight per thread (config 1: 18 chunks per tile = 2 groups x 9: one round trip)
            const size_t cstride = (size_t)n_rt * TV;
            const int cn = (n_chunks + PARTS - 1) / PARTS;
            for (int t = tid; t < PARTS * TV; t += NT) {
                const int pt = t / TV, v = t - pt * TV;
                u64* src = part_bits + (size_t)tile * TV + v;
                const int c1 = min(n_chunks, (pt + 1) * cn);
                double sum = 0.0;
                for (int c = pt * cn; c < c1; c += BATCH) {
                    u64 w[BATCH];
#pragma unroll
                    for (int i = 0; i < BATCH; ++i) {
                        w[i] = 1ull;   // (own chunk / beyond the range: nothing to wait for)
                        if (c + i < c1 && c + i > 0) w[i] = __ldcg(src + (size_t)(c + i) * cstride);
                    }
                    // words that were not there yet are re-read TOGETHER, one round trip per pass (re-reading them one after
                    // the other cost the finisher a round trip per late word)
                    for (;;) {
                        u64 all = ~0ull;
#pragma unroll
                        for (int i = 0; i < BATCH; ++i) all &= w[i];
                        if (all & 1ull) break;
#pragma unroll
                        for (int i = 0; i < BATCH; ++i)
                            if (!(w[i] & 1ull))
                                asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(w[i]) : "l"(src + (size_t)(c + i) * cstride) : "memory");
                    }
#pragma unroll
                    for (int i = 0; i < BATCH; ++i) {
                        if (c + i >= c1) break;
                        if (c + i == 0) {
                            sum += s_out[v];   // this CTA's own chunk
                        } else {
                            sum += __longlong_as_double((long long)w[i]);
                            __stcg(src + (size_t)(c + i) * cstride, 0ull);
                        }
                    }
                }
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
            if (A.fused) {
                __syncthreads();
                // forces: L2 reductions (atoms shared by CVs / walkers collide).  Lean gather: one thread per (replica, group),
                // atom and Jacobian out of shared memory -- no global load between the last sum and the reductions
                if (A.simple) {
                    for (int t = tid; t < TILE_R * P.n_groups; t += NT) {
                        const int rr = t / P.n_groups, gid = t - rr * P.n_groups, r = r0 + rr;
                        if (r >= R) continue;
                        const float fdv = -(float)s_out[rr * NV + 1 + P.grp[gid].cv];   // dV/dxi and J pass through binary32, as unfused
                        const float* j = s_jv + t * 3;
                        float* fa = A.force + ((long long)r * P.rstride + s_ja[t]) * P.fs;
                        force_add(fa, fdv * j[0], fdv * j[1], fdv * j[2], P.fs);
                    }
                } else
                // general gather: one thread per (replica, slot)
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
        __syncthreads();   // s_xi / s_out / s_wacc are reused by the next item
    }
}
