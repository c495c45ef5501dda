// range_step.cu -- the fused umbrella-sampling step over LARGE contiguous atom groups (SURVEY.md 8(a) rows
// A1, A3a, A3b, A4, A8, A9; the paper's measured instance of this path is a COM-distance CV over 1,600-bead
// groups with a harmonic bias).  ONE persistent, warp-specialised launch per MD step;
// one CTA per SM; item = (window r, slice s of RS_SLICE atoms); CTA b owns items b, b + grid, b + 2 grid, ...
//
//   producer warp : positions of the CTA's next items -> a ring of RS_STAGES shared-memory stages, one 1-D TMA
//                   bulk copy per slice (cp.async.bulk + mbarrier, SASS UBLKCP), up to RS_STAGES - 1 items ahead.
//   A group (8 warps): weighted moments {W, sum w r, sum w |r|^2} of every range group over the slice, binary64,
//                   reduced in fixed order -> rpart; one acq_rel ticket per item.  Whoever takes the LAST ticket
//                   of a window hands the window to its CTA's window warp and moves on.
//   window warp   : combines the window's partials in fixed order, evaluates the CVs (center-of-mass distance /
//                   angle / dihedral / component, radius of gyration) and the harmonic bias in binary64, and
//                   publishes per-group force descriptors (16-byte records carrying a valid tag).
//   B groups (2 x 8 warps, alternating items): wait for the window's descriptors, then
//                   F_i += -dV/dxi_k * w_i (v_g + coef_g (r_i - c_g))  with r_i from the stage STILL RESIDENT in
//                   shared memory and the force streamed through registers (ld.global.cs / st.global.cs float4);
//                   then the stage is handed back to the producer.
//   Positions cross HBM once, forces are read once and written once = 48 B/atom, the algorithmic minimum.  The
//   three roles are decoupled by the stage ring, so the inter-CTA dependency (B needs every A of its window) is
//   absorbed by the A group running several items ahead of the B groups.
// A never waits on another CTA, so the wait in B cannot deadlock as long as the grid is co-resident and a window
// has at most `grid` slices: the kernel is launched cooperatively (the launch fails instead of hanging).
// Results are bitwise reproducible and equal to the unfused calls: fixed thread -> atom map, fixed reduction
// order, one writer per atom.
#include <stdlib.h>

#include "geom.cuh"

#define RS_SLICE PSG_RANGE_TILE   // atoms per slice (2048): 32 KB of float4 positions per stage
#define RS_STAGES 6
#define RS_GT 256                 // threads of the A group and of each B group
#define RS_NB 2                   // B groups
#define RS_LEAD 64                 // producer warp + window warp
#define RS_THREADS (RS_LEAD + RS_GT * (1 + RS_NB))
#define RS_WQ 8                    // ring of windows handed from the A group to the window warp
#define RS_PER (RS_SLICE / RS_GT)
#define RS_DESC 4                 // float4 records per (window, range group): {v, tag} {c_hi, tag} {c_lo, tag} {k, 0, 0, tag}
#define RS_TAG 1.0f

struct RangeStepArgs {
    const float* pos;
    float* force;
    const float* kspring;   // [n_cv]
    const float* centers;   // [R][n_cv]
    float* xi_out;          // [R][n_cv]
    float* V_out;           // [R]
    double* V64_out;        // [R]
    float* dV_out;          // [R][n_cv]
    double* rpart;          // [R][n_ranges][n_slices][PSG_MOM]
    unsigned* arrive;       // [R]  tickets of phase A
    unsigned* done;         // [R]  finished phase B
    float4* desc;           // [R][n_ranges][RS_DESC]
#ifdef PSG_TRACE
    long long* trace;
#endif
};

__device__ __forceinline__ uint32_t rs_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void rs_mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(rs_smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void rs_mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(rs_smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void rs_mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(rs_smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void rs_tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(rs_smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(rs_smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void rs_mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "RS_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra RS_DONE;\n"
        "bra RS_WAIT;\n"
        "RS_DONE:\n"
        "}" ::"r"(rs_smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void rs_group_sync(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(RS_GT) : "memory"); }
__device__ __forceinline__ float4 rs_ld_relaxed_f4(const float4* p) {   // one 16-byte access, always from L2
    float4 v;
    asm volatile("ld.relaxed.gpu.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
    return v;
}

struct RsShared {
    double red[2][RS_GT / 32][PSG_MAX_RANGE_GROUPS][PSG_MOM];    // A: per-warp partial moments, double-buffered by item parity
    double mom[PSG_MAX_RANGE_GROUPS][PSG_MOM];                    // window warp: moments
    double cen[PSG_MAX_RANGE_GROUPS][4];                          // window warp: centre, W per range group
    double gv[PSG_MAX_RANGE_GROUPS][3], gcoef[PSG_MAX_RANGE_GROUPS];   // d xi / d c_g / W_g,  Rg: 1/(W Rg)
    double dv[PSG_MAX_CV];                                        // -(dV/dxi_k), through binary32 like the unfused path
    double vk[PSG_MAX_CV];                                        // 1/2 k_k D_k^2
    float4 desc[RS_NB][PSG_MAX_RANGE_GROUPS][RS_DESC];            // B groups: the window's force descriptors
    uint64_t full[RS_STAGES], empty[RS_STAGES];
    int wq[RS_WQ];                    // windows waiting for the window warp
    volatile int wq_head, wq_tail;    // written by A's warp 0 / by the window warp
    volatile int a_done;              // the A group has processed its last item
};

struct RsItem {
    int r, s;
    long long a0;       // first atom of the slice in the flat arrays
    uint32_t bytes;     // 16 * atoms in the slice
};
__device__ __forceinline__ RsItem rs_item(const SysParams& P, long long it, long long G) {
    RsItem I;
    const long long j = blockIdx.x + it * G;
    I.r = (int)(j / P.range_blocks); I.s = (int)(j % P.range_blocks);
    const long long b = P.span_begin + (long long)I.s * RS_SLICE;
    I.a0 = (long long)I.r * P.rstride + b;
    long long cnt = P.span_end - b;
    if (cnt > RS_SLICE) cnt = RS_SLICE;
    I.bytes = (uint32_t)cnt * 16u;
    return I;
}

// Window-level work, done ONCE per window by warp 0 of the A group of the CTA that took its last ticket: combine
// partials, CVs, harmonic bias, outputs, and the per-group force descriptors published for every CTA of the window.
__device__ __forceinline__ void rs_window(const SysParams& P, const RangeStepArgs& A, RsShared& S, int r, int lane) {
    const int n_slices = P.range_blocks;
    // fixed-order combination per value: lanes stride the slices (increasing), then an xor tree
    for (int q = 0; q < P.n_ranges; ++q) {
        const double* src = A.rpart + (((long long)r * P.n_ranges + q) * n_slices) * PSG_MOM;
        double sum[PSG_MOM] = {0, 0, 0, 0, 0};
        for (int b = lane; b < n_slices; b += 32) {
#pragma unroll
            for (int i = 0; i < PSG_MOM; ++i) sum[i] += __ldcg(src + (long long)b * PSG_MOM + i);
        }
#pragma unroll
        for (int i = 0; i < PSG_MOM; ++i) {
            sum[i] = warp_sum(sum[i]);
            if (lane == 0) S.mom[q][i] = sum[i];
        }
    }
    __syncwarp();
    if (lane < P.n_ranges) {
        const double iw = 1.0 / S.mom[lane][0];
        S.cen[lane][0] = S.mom[lane][1] * iw; S.cen[lane][1] = S.mom[lane][2] * iw; S.cen[lane][2] = S.mom[lane][3] * iw;
        S.cen[lane][3] = S.mom[lane][0];
    }
    __syncwarp();
    if (lane < P.n_cv) {
        const CvDev& C = P.cv[lane];
        double xi;
        if (C.type == PSG_CV_RGYR) {
            const int q = P.grp[C.gid0].range_id;
            const D3 c = d3(S.cen[q][0], S.cen[q][1], S.cen[q][2]);
            const double W = S.cen[q][3];
            const double rg2 = S.mom[q][4] / W - dot(c, c);
            xi = rg2 > 0.0 ? sqrt(rg2) : 0.0;
            S.gcoef[q] = xi > 0.0 ? 1.0 / (W * xi) : 0.0;
            S.gv[q][0] = S.gv[q][1] = S.gv[q][2] = 0.0;
        } else {
            D3 c[4], dc[4];
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                c[g] = d3(0, 0, 0);
                if (g < C.n_groups) {
                    const int q = P.grp[C.gid0 + g].range_id;
                    c[g] = d3(S.cen[q][0], S.cen[q][1], S.cen[q][2]);
                }
            }
            xi = cv_from_centers<true>(C.type, C.axis, c, dc);
#pragma unroll
            for (int g = 0; g < 4; ++g)
                if (g < C.n_groups) {
                    const int q = P.grp[C.gid0 + g].range_id;
                    const double iw = 1.0 / S.cen[q][3];
                    S.gv[q][0] = dc[g].x * iw; S.gv[q][1] = dc[g].y * iw; S.gv[q][2] = dc[g].z * iw;
                    S.gcoef[q] = 0.0;
                }
        }
        // harmonic bias at the CV rounded to binary32, as the unfused calls see it
        const float xif = (float)xi;
        double d = (double)xif - (double)A.centers[(long long)r * P.n_cv + lane];
        const double per = C.period;
        if (per > 0.0) d -= per * rint(d / per);
        const double ks = (double)A.kspring[lane];
        const float dVf = (float)(ks * d);
        S.dv[lane] = -(double)dVf;
        S.vk[lane] = 0.5 * ks * d * d;
        A.xi_out[(long long)r * P.n_cv + lane] = xif;
        A.dV_out[(long long)r * P.n_cv + lane] = dVf;
    }
    __syncwarp();
    if (lane == 0) {
        double V = 0.0;
        for (int k = 0; k < P.n_cv; ++k) V += S.vk[k];
        if (A.V_out) A.V_out[r] = (float)V;
        if (A.V64_out) A.V64_out[r] = V;
    }
    if (lane < P.n_ranges) {
        const GroupDev& G = P.grp[P.range_gid[lane]];
        const double dv = S.dv[G.cv];
        float v[3], hi[3], lo[3];
#pragma unroll
        for (int x = 0; x < 3; ++x) {
            v[x] = (float)(dv * S.gv[lane][x]);
            hi[x] = (float)S.cen[lane][x];
            lo[x] = (float)(S.cen[lane][x] - (double)hi[x]);   // centre as hi + lo: (r - hi) - lo keeps r - c accurate
        }
        float4* d = A.desc + ((long long)r * P.n_ranges + lane) * RS_DESC;
        // every 16-byte record is one store and carries its own valid tag
        __stcg(d + 0, make_float4(v[0], v[1], v[2], RS_TAG));
        __stcg(d + 1, make_float4(hi[0], hi[1], hi[2], RS_TAG));
        __stcg(d + 2, make_float4(lo[0], lo[1], lo[2], RS_TAG));
        __stcg(d + 3, make_float4((float)(dv * S.gcoef[lane]), 0.f, 0.f, RS_TAG));
    }
    __syncwarp();
}

// A group, one item: moments of the slice in shared memory -> rpart -> ticket (-> window work)
__device__ __forceinline__ void rs_phase_a(const SysParams& P, const RangeStepArgs& A, RsShared& S, const float4* __restrict__ sp,
                                           const RsItem& I, int buf, int tid) {
    const int lane = tid & 31, wid = tid >> 5;
    const int n_slices = P.range_blocks;
    const long long t0 = P.span_begin + (long long)I.s * RS_SLICE;
    const long long t1 = t0 + (I.bytes >> 4);
    bool have_full = false;           // moments over the WHOLE slice, shared by every group that contains it
    double mf[PSG_MOM] = {0, 0, 0, 0, 0};
    for (int q = 0; q < P.n_ranges; ++q) {
        const GroupDev& G = P.grp[P.range_gid[q]];
        const long long gb = G.rbegin, ge = G.rbegin + G.rsize;
        double m[PSG_MOM] = {0, 0, 0, 0, 0};
        if (t0 < ge && t1 > gb) {     // group-uniform
            const bool inside = gb <= t0 && t1 <= ge;
            if (inside && have_full) {
#pragma unroll
                for (int i = 0; i < PSG_MOM; ++i) m[i] = mf[i];
            } else {
#pragma unroll
                for (int i = 0; i < RS_PER; ++i) {
                    const long long a = t0 + tid + i * RS_GT;
                    if (a >= gb && a < ge && a < t1) {
                        // (re-read from shared memory per group pass: registers are the scarce resource here)
                        const float4 v = sp[tid + i * RS_GT];
                        const double wd = P.atom_weight ? (double)__ldg(P.atom_weight + a) : 1.0;
                        // products of binary32 inputs are exact in binary64
                        const double xd = (double)v.x, yd = (double)v.y, zd = (double)v.z;
                        m[0] += wd; m[1] += wd * xd; m[2] += wd * yd; m[3] += wd * zd;
                        m[4] += wd * (xd * xd + yd * yd + zd * zd);
                    }
                }
#pragma unroll
                for (int i = 0; i < PSG_MOM; ++i) m[i] = warp_sum(m[i]);
                if (inside) {
                    have_full = true;
#pragma unroll
                    for (int i = 0; i < PSG_MOM; ++i) mf[i] = m[i];
                }
            }
        }
        if (lane == 0) {
#pragma unroll
            for (int i = 0; i < PSG_MOM; ++i) S.red[buf][wid][q][i] = m[i];
        }
    }
    rs_group_sync(1);
    if (wid == 0) {
        // warp 0 finishes the item while warps 1..7 move on (S.red is double-buffered)
        for (int t = lane; t < P.n_ranges * PSG_MOM; t += 32) {
            const int q = t / PSG_MOM, i = t % PSG_MOM;
            double sum = 0.0;
#pragma unroll
            for (int wq = 0; wq < RS_GT / 32; ++wq) sum += S.red[buf][wq][q][i];
            A.rpart[(((long long)I.r * P.n_ranges + q) * n_slices + I.s) * PSG_MOM + i] = sum;
        }
        __syncwarp();
        unsigned old = 0;
        if (lane == 0) {
            // release: the warp's partials (ordered before this by the warp barrier) become visible to whoever
            // acquires the ticket
            asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(A.arrive + I.r) : "memory");
        }
        if (lane == 0 && old == (unsigned)(n_slices - 1)) {
            // last ticket of the window: hand it to the window warp (the ring cannot realistically fill: a CTA
            // closes a window every few items; wait if it does)
            const int h = S.wq_head;
            while (h - S.wq_tail >= RS_WQ) __nanosleep(100);
            S.wq[h % RS_WQ] = I.r;
            __threadfence_block();
            S.wq_head = h + 1;
        }
    }
}

// B group, one item: force update of the slice; positions from shared memory, forces streamed through registers
__device__ __forceinline__ void rs_phase_b(const SysParams& P, const RangeStepArgs& A, RsShared& S, const float4* __restrict__ sp,
                                           const RsItem& I, int g, int tid) {
    const int bar_id = 2 + g;
    float4* f = reinterpret_cast<float4*>(A.force) + I.a0;
    const int cnt = (int)(I.bytes >> 4);
    // forces first: their latency overlaps the descriptor poll
    float4 fv[RS_PER];
#pragma unroll
    for (int i = 0; i < RS_PER; ++i) {
        const int o = tid + i * RS_GT;
        fv[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (o < cnt) fv[i] = __ldcs(f + o);   // streamed: read once, written once
    }
    if (tid < P.n_ranges * RS_DESC) {
        const float4* src = A.desc + (long long)I.r * P.n_ranges * RS_DESC + tid;
        float4 d = rs_ld_relaxed_f4(src);
        while (d.w != RS_TAG) {   // window not finished yet: only at pipeline start-up or if the A groups lag
            __nanosleep(200);
            d = rs_ld_relaxed_f4(src);
        }
        S.desc[g][tid / RS_DESC][tid % RS_DESC] = d;
    }
    rs_group_sync(bar_id);
    const long long t0 = P.span_begin + (long long)I.s * RS_SLICE;
#pragma unroll
    for (int i = 0; i < RS_PER; ++i) {
        const int o = tid + i * RS_GT;
        if (o >= cnt) continue;
        const long long a = t0 + o;
        const float4 p = sp[o];
        float ax = 0.f, ay = 0.f, az = 0.f;
        bool any = false;
        for (int q = 0; q < P.n_ranges; ++q) {
            const GroupDev& G = P.grp[P.range_gid[q]];
            if (a >= G.rbegin && a < G.rbegin + G.rsize) {
                any = true;
                const float4 v = S.desc[g][q][0], hi = S.desc[g][q][1], lo = S.desc[g][q][2];
                const float k = S.desc[g][q][3].x;
                ax += v.x + k * ((p.x - hi.x) - lo.x);
                ay += v.y + k * ((p.y - hi.y) - lo.y);
                az += v.z + k * ((p.z - hi.z) - lo.z);
            }
        }
        if (!any) continue;   // an atom of the span that belongs to no group is not written
        const float w = P.atom_weight ? __ldg(P.atom_weight + a) : 1.f;
        // (no contraction: same bits as the unfused path); the record's w keeps its bits
        fv[i].x += __fmul_rn(ax, w); fv[i].y += __fmul_rn(ay, w); fv[i].z += __fmul_rn(az, w);
        __stcs(f + o, fv[i]);
    }
}

__global__ void __launch_bounds__(RS_THREADS, 1) k_range_step(const __grid_constant__ SysParams P, const __grid_constant__ RangeStepArgs A) {
    extern __shared__ __align__(128) unsigned char rs_smem[];
    float4* stage = reinterpret_cast<float4*>(rs_smem);   // RS_STAGES x RS_SLICE positions
    RsShared& S = *reinterpret_cast<RsShared*>(rs_smem + (size_t)RS_STAGES * RS_SLICE * 16);
    const int tid = threadIdx.x;
    const long long items = (long long)P.R * P.range_blocks;
    const long long G = gridDim.x;
    const long long n_mine = blockIdx.x < items ? (items - blockIdx.x + G - 1) / G : 0;

    if (tid == 0) {
        for (int st = 0; st < RS_STAGES; ++st) {
            rs_mbar_init(&S.full[st], 1);
            rs_mbar_init(&S.empty[st], RS_GT / 32);   // one arrival per warp of the B group that used the stage
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid == 0) { S.wq_head = 0; S.wq_tail = 0; S.a_done = 0; }
    __syncthreads();

    if (tid < 32) {
        // ---------------- producer warp
        if (tid == 0) {
            for (long long it = 0; it < n_mine; ++it) {
                const int st = (int)(it % RS_STAGES);
                if (it >= RS_STAGES) rs_mbar_wait(&S.empty[st], (uint32_t)((it / RS_STAGES - 1) & 1));
                const RsItem I = rs_item(P, it, G);
                rs_mbar_expect_tx(&S.full[st], I.bytes);
                rs_tma_load_1d(stage + (size_t)st * RS_SLICE, reinterpret_cast<const float4*>(A.pos) + I.a0, I.bytes, &S.full[st]);
            }
        }
    } else if (tid < RS_LEAD) {
        // ---------------- window warp: serves the windows whose last ticket was taken by this CTA
        const int lane = tid & 31;
        int tail = 0;
        for (;;) {
            int head = S.wq_head;
            const int fin = S.a_done;   // read AFTER head: a_done is set after the last hand-over
            if (head == tail) {
                if (fin && S.wq_head == tail) break;
                __nanosleep(100);
                continue;
            }
            __threadfence_block();
            const int r = S.wq[tail % RS_WQ];
            __threadfence();            // acquire side of the ticket (taken by another warp of this CTA)
            rs_window(P, A, S, r, lane);
            ++tail;
            if (lane == 0) S.wq_tail = tail;
            __syncwarp();
        }
    } else if (tid < RS_LEAD + RS_GT) {
        // ---------------- A group
        const int t = tid - RS_LEAD;
        for (long long it = 0; it < n_mine; ++it) {
            const int st = (int)(it % RS_STAGES);
            const RsItem I = rs_item(P, it, G);
            rs_mbar_wait(&S.full[st], (uint32_t)((it / RS_STAGES) & 1));
            rs_phase_a(P, A, S, stage + (size_t)st * RS_SLICE, I, (int)(it & 1), t);
        }
        rs_group_sync(1);               // warp 0 has handed over its last window
        if (t == 0) { __threadfence_block(); S.a_done = 1; }
    } else {
        // ---------------- B groups: group g takes the items it = g, g + RS_NB, ...
        const int g = (tid - RS_LEAD - RS_GT) / RS_GT, t = (tid - RS_LEAD - RS_GT) % RS_GT;
        for (long long it = g; it < n_mine; it += RS_NB) {
            const int st = (int)(it % RS_STAGES);
            const RsItem I = rs_item(P, it, G);
            rs_mbar_wait(&S.full[st], (uint32_t)((it / RS_STAGES) & 1));   // the stage's bytes are visible to this thread
            rs_phase_b(P, A, S, stage + (size_t)st * RS_SLICE, I, g, t);
            __syncwarp();
            if ((t & 31) == 0) rs_mbar_arrive(&S.empty[st]);   // this warp is done reading the stage
            rs_group_sync(2 + g);                              // S.desc[g] may be overwritten by the next item
            if (t == 0) {
                // the last CTA to finish a window re-arms its counters and descriptor tags for the next launch
                const unsigned old = atomicAdd(A.done + I.r, 1u);
                if (old == (unsigned)(P.range_blocks - 1)) {
                    A.arrive[I.r] = 0u; A.done[I.r] = 0u;
                    for (int i = 0; i < P.n_ranges * RS_DESC; ++i)
                        __stcg(A.desc + (long long)I.r * P.n_ranges * RS_DESC + i, make_float4(0.f, 0.f, 0.f, 0.f));
                }
            }
        }
    }
}

static const size_t kRsSmem = (size_t)RS_STAGES * RS_SLICE * 16 + sizeof(RsShared);

// co-resident CTAs per SM (0 if the kernel cannot be configured)
static int rs_blocks_per_sm() {
    static int n = -1;
    if (n < 0) {
        n = 0;
        if (cudaFuncSetAttribute(k_range_step, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRsSmem) == cudaSuccess) {
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_range_step, RS_THREADS, kRsSmem) != cudaSuccess) n = 0;
        }
        (void)cudaGetLastError();
    }
    return n;
}

// The fused step covers: harmonic bias; every group a contiguous range; float4 positions and forces, 16-byte
// aligned (the position slices are TMA bulk copies); one array per window; windows of at most `grid` slices (so
// that every A a waiting B depends on belongs to the same or the next round of items). Anything else takes the
// separate kernels of cv.cu / bias.cu.
bool psg_range_step_supported(const psg_ctx* c, const float* d_pos, const float* d_force) {
    const SysParams& P = c->sys;
    static const bool disabled = getenv("PSG_DISABLE_RANGE_STEP") != nullptr;   // profiling aid: take the separate kernels
    if (disabled) return false;
    if (!(c->method == PSG_METHOD_HARMONIC && P.n_ranges > 0 && P.n_slots == 0 && P.ps == 4 && P.fs == 4 && P.rstride > 0 &&
          ((reinterpret_cast<uintptr_t>(d_pos) | reinterpret_cast<uintptr_t>(d_force)) & 15u) == 0 &&
          c->d_arrive != nullptr))
        return false;
    const long long grid = (long long)c->sm_count * rs_blocks_per_sm();
    return grid >= 1 && P.range_blocks <= grid;
}

cudaError_t psg_launch_range_step(psg_ctx* c, const float* d_pos, float* d_force) {
    const int max_blocks_per_sm = rs_blocks_per_sm();
    if (max_blocks_per_sm < 1) return cudaErrorLaunchOutOfResources;
    const SysParams& P = c->sys;
    RangeStepArgs A{};
    A.pos = d_pos; A.force = d_force; A.kspring = c->d_kspring; A.centers = c->d_centers;
    A.xi_out = c->d_xi; A.V_out = c->d_V; A.V64_out = c->d_V64; A.dV_out = c->d_dVdxi;
    A.rpart = c->d_rpart; A.arrive = c->d_arrive; A.done = c->d_arrive + P.R; A.desc = c->d_rdesc;
#ifdef PSG_TRACE
    A.trace = psg_trace_buffer();
#endif
    long long items = (long long)P.R * P.range_blocks;
    long long grid = (long long)c->sm_count * max_blocks_per_sm;
    if (grid > items) grid = items;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(RS_THREADS); cfg.dynamicSmemBytes = kRsSmem; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;   // co-residency is what makes the inter-CTA wait safe
    attr[0].val.cooperative = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, k_range_step, P, A);
    if (e == cudaSuccess) c->launches++;
    return e;
}
