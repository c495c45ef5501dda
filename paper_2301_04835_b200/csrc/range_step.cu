// range_step.cu -- the fused umbrella-sampling step over LARGE contiguous atom groups (SURVEY.md 8(a) rows
// A1, A3a, A3b, A4, A8, A9; the paper's measured instance of this path is a COM-distance CV over 1,600-bead
// groups with a harmonic bias).  ONE persistent, warp-specialised launch per MD step;
// one CTA per SM; item = (window r, slice s of RS_SLICE atoms); CTA b owns items b, b + grid, b + 2 grid, ...
// Every byte of the two big arrays enters the SM by 1-D TMA bulk copies (cp.async.bulk + mbarrier, SASS UBLKCP).
//
//   PA warp  : positions of the next items -> ring A (L2 policy evict_last), throttled to stay at most `lag`
//              items ahead of the B group, so the slices it brought in are still in L2 when B wants them.
//   A group  (8 warps): weighted moments {W, sum w r, sum w |r|^2} of every range group over the slice, binary64,
//              per-warp partials -> a small shared-memory ring; the stage goes straight back to PA.
//   T warps  (2, alternating items): sum the 8 warp partials in fixed order -> rpart (global); one release
//              ticket per item on the window's counter.
//   W warp   : owns the windows r = b, b + grid, ... (an even share, whoever finishes them): waits until a window
//              has all its tickets (acquire), combines its partials in fixed order, evaluates the CVs (center-of-mass distance / angle /
//              dihedral / component, radius of gyration) and the harmonic bias in binary64, publishes per-group
//              force descriptors (16-byte records carrying a valid tag).
//   PB warp  : positions (now an L2 hit) and forces of the B group's next items -> ring B.
//   B group  (16 warps): takes the window's descriptors (requested one item earlier with cp.async; polls only if the
//              window is not finished), then
//              F_i += -dV/dxi_k * w_i (v_g + coef_g (r_i - c_g))  out of shared memory, st.global.cs float4.
//   HBM traffic: positions once (the second read is served by L2 while `lag` x grid x 32 KB fits), forces read
//   once and written once = 48 B/atom, the algorithmic minimum; 64 B/atom if L2 keeps nothing.
// The window dependency (B needs every A of its window, from ~49 other CTAs, plus the window warp's work) is a
// chain of several L2 round trips; it is absorbed by B simply running `lag` items behind A -- no shared-memory
// stage is held across it.  A, T and W never wait on another CTA, so the wait in B cannot deadlock as long as the
// grid is co-resident and a window has at most `grid` slices: the kernel is launched cooperatively (the launch
// fails instead of hanging).  Results are bitwise reproducible and equal to the unfused calls: fixed
// thread -> atom map, fixed reduction order, one writer per atom.
#include "geom.cuh"

#define RS_SLICE PSG_RANGE_TILE   // atoms per slice (2048): 32 KB of float4 per array and stage
#define RS_ASTAGES 2              // ring A: positions
#define RS_BSTAGES 2              // ring B: positions + forces
#define RS_RED 4                  // ring of per-warp partial moments between the A group and the T warps
#define RS_NT 2                   // T warps
#define RS_GT PSG_RANGE_THREADS   // threads of the A group (256; fixes the reduction order: same map as k_range_moments)
#define RS_GTB 512                // threads of the B group
#define RS_LEAD (32 * (3 + RS_NT))   // PA, PB, W, T warps
#define RS_THREADS (RS_LEAD + RS_GT + RS_GTB)
#define RS_PER (RS_SLICE / RS_GT)
#define RS_PERB (RS_SLICE / RS_GTB)
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
    unsigned* arrive;       // [R]  tickets
    unsigned* done;         // [R]  slices whose forces are written
    float4* desc;           // [R][n_ranges][RS_DESC]
    int lag;                // items PA may run ahead of the B group
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
__device__ __forceinline__ uint64_t rs_policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t rs_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void rs_tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                     rs_smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(rs_smem_u32(bar)), "l"(policy)
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
__device__ __forceinline__ void rs_b_sync() { asm volatile("bar.sync 2, %0;" ::"n"(RS_GTB) : "memory"); }
__device__ __forceinline__ float4 rs_ld_relaxed_f4(const float4* p) {   // one 16-byte access, always from L2
    float4 v;
    asm volatile("ld.relaxed.gpu.global.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p) : "memory");
    return v;
}


struct RsShared {
    double red[RS_RED][RS_GT / 32][PSG_MAX_RANGE_GROUPS][PSG_MOM];   // A group -> T warps: per-warp partial moments
    double mom[PSG_MAX_RANGE_GROUPS][PSG_MOM];                    // W warp: the window's moments
    double cen[PSG_MAX_RANGE_GROUPS][4];                          // W warp: centre, W per range group
    double gv[PSG_MAX_RANGE_GROUPS][3], gcoef[PSG_MAX_RANGE_GROUPS];   // d xi / d c_g / W_g,  Rg: 1/(W Rg)
    double dv[PSG_MAX_CV];                                        // -(dV/dxi_k), through binary32 like the unfused path
    double vk[PSG_MAX_CV];                                        // 1/2 k_k D_k^2
    // B group, three buffers indexed by item % 3: item it computes from [it % 3] while the descriptors of item it + 1 are
    // already arriving in [(it + 1) % 3] (cp.async) and slow warps may still read item it - 1's in [(it - 1) % 3]
    float4 desc[3][PSG_MAX_RANGE_GROUPS][RS_DESC];                // the window's force descriptors
    int blo[3][PSG_MAX_RANGE_GROUPS], bhi[3][PSG_MAX_RANGE_GROUPS];   // slice-local atom bounds of every group
    int bfast[3];                                                 // the item takes the straight-line path
    long long g_b[PSG_MAX_RANGE_GROUPS], g_e[PSG_MAX_RANGE_GROUPS];   // atom range of every range group (copied once from the
                                                                  // kernel parameters)
    uint64_t a_full[RS_ASTAGES], a_empty[RS_ASTAGES], b_full[RS_BSTAGES], b_empty[RS_BSTAGES];
    uint64_t red_full[RS_RED], red_empty[RS_RED];
    volatile long long b_prog;                  // items the B group has finished
};

struct RsItem {
    int r, s;
    long long a0;       // first atom of the slice in the flat arrays
    uint32_t bytes;     // 16 * atoms in the slice
};
__device__ __forceinline__ RsItem rs_item(const SysParams& P, long long it, long long G) {
    RsItem I;
    // R <= 65535 and range_blocks <= grid, so the item index fits 32 bits: one 32-bit division, not two 64-bit ones
    const unsigned j = (unsigned)(blockIdx.x + it * G);
    const unsigned nb = (unsigned)P.range_blocks;
    const unsigned r = j / nb;
    I.r = (int)r; I.s = (int)(j - r * nb);
    const long long b = P.span_begin + (long long)I.s * RS_SLICE;
    I.a0 = (long long)I.r * P.rstride + b;
    long long cnt = P.span_end - b;
    if (cnt > RS_SLICE) cnt = RS_SLICE;
    I.bytes = (uint32_t)cnt * 16u;
    return I;
}

// Window-level work, done ONCE per window by the W warp of the CTA that took its last ticket: combine partials,
// CVs, harmonic bias, outputs, and the per-group force descriptors published for every CTA of the window.
__device__ __forceinline__ void rs_window(const SysParams& P, const RangeStepArgs& A, RsShared& S, int r, int lane) {
    const int n_slices = P.range_blocks;
    // operands of the bias, requested early: their latency hides behind the combination
    float h_center = 0.f, h_k = 0.f;
    if (lane < P.n_cv) {
        h_center = __ldg(A.centers + (long long)r * P.n_cv + lane);
        h_k = __ldg(A.kspring + lane);
    }
    // fixed-order combination per value: lanes stride the slices (increasing), then an xor tree. Three groups
    // at a time, so that all their loads (L2, written by other SMs) are in flight together: this latency is
    // what every CTA of the window waits for.
    for (int q0 = 0; q0 < P.n_ranges; q0 += 3) {
        double sum[3][PSG_MOM];
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int i = 0; i < PSG_MOM; ++i) sum[j][i] = 0.0;
#pragma unroll 2
        for (int b = lane; b < n_slices; b += 32) {
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                if (q0 + j < P.n_ranges) {
                    const double* src = A.rpart + (((long long)r * P.n_ranges + q0 + j) * n_slices + b) * PSG_MOM;
#pragma unroll
                    for (int i = 0; i < PSG_MOM; ++i) sum[j][i] += __ldcg(src + i);
                }
            }
        }
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int i = 0; i < PSG_MOM; ++i) {
                const double t = warp_sum(sum[j][i]);
                if (lane == 0 && q0 + j < P.n_ranges) S.mom[q0 + j][i] = t;
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
        double d = (double)xif - (double)h_center;
        const double per = C.period;
        if (per > 0.0) d -= per * rint(d / per);
        const double ks = (double)h_k;
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

// A group, one item: per-warp moments of the slice in shared memory -> S.red[buf]. Warps do not synchronise with
// each other: each reports to the T warp (red_full) and hands the stage back (a_empty) on its own.
__device__ __forceinline__ void rs_phase_a(const SysParams& P, RsShared& S, const float4* __restrict__ sp, const RsItem& I, int buf,
                                           int tid) {
    const int lane = tid & 31, wid = tid >> 5;
    const long long t0 = P.span_begin + (long long)I.s * RS_SLICE;
    const long long t1 = t0 + (I.bytes >> 4);
    bool have_full = false;           // moments over the WHOLE slice, shared by every group that contains it
    double mf[PSG_MOM] = {0, 0, 0, 0, 0};
    for (int q = 0; q < P.n_ranges; ++q) {
        const long long gb = S.g_b[q], ge = S.g_e[q];
        double m[PSG_MOM] = {0, 0, 0, 0, 0};
        if (t0 < ge && t1 > gb) {     // uniform over the group
            const bool inside = gb <= t0 && t1 <= ge;
            if (inside && have_full) {
#pragma unroll
                for (int i = 0; i < PSG_MOM; ++i) m[i] = mf[i];
            } else {
                if (inside && (t1 - t0 == RS_SLICE) && !P.atom_weight) {
                    // the common case, straight-line: a whole slice inside the group, unit weights
                    // (1.0 * x + m rounds exactly like x + m: same bits as the general loop)
#pragma unroll
                    for (int i = 0; i < RS_PER; ++i) {
                        const float4 v = sp[tid + i * RS_GT];
                        const double xd = (double)v.x, yd = (double)v.y, zd = (double)v.z;
                        m[0] += 1.0; m[1] += xd; m[2] += yd; m[3] += zd;
                        m[4] += xd * xd + yd * yd + zd * zd;
                    }
                } else {
                    // branch-free: an atom outside the group (or past the end of a ragged slice) enters with w = 0
                    // and r = 0, which adds exactly +0 to every moment -- the same bits as skipping it
#pragma unroll
                    for (int i = 0; i < RS_PER; ++i) {
                        const int o = tid + i * RS_GT;
                        const long long a = t0 + o;
                        const bool in = a >= gb && a < ge && a < t1;
                        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                        float wf = 0.f;
                        if (in) {   // predicated loads, no divergence
                            v = sp[o];
                            wf = P.atom_weight ? __ldg(P.atom_weight + a) : 1.f;
                        }
                        // products of binary32 inputs are exact in binary64
                        const double wd = (double)wf, xd = (double)v.x, yd = (double)v.y, zd = (double)v.z;
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
    __syncwarp();
}

// T warp, one item: the slice's moments (8 warp partials, fixed order) -> rpart; ticket on the window's counter
__device__ __forceinline__ void rs_tail(const SysParams& P, const RangeStepArgs& A, RsShared& S, const RsItem& I, int buf,
                                        int lane) {
    const int n_slices = P.range_blocks;
    for (int t = lane; t < P.n_ranges * PSG_MOM; t += 32) {
        const int q = t / PSG_MOM, i = t % PSG_MOM;
        double sum = 0.0;
#pragma unroll
        for (int wq = 0; wq < RS_GT / 32; ++wq) sum += S.red[buf][wq][q][i];
        A.rpart[(((long long)I.r * P.n_ranges + q) * n_slices + I.s) * PSG_MOM + i] = sum;
    }
    __syncwarp();
    if (lane == 0) {
        rs_mbar_arrive(&S.red_empty[buf]);
        // release: the warp's partials (ordered before this by the warp barrier) become visible to the W warp that
        // acquires the counter
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(A.arrive + I.r) : "memory");
    }
    __syncwarp();
}

// B group, one item: force update of the slice; positions and forces out of shared memory, result streamed to global
__device__ __forceinline__ void rs_phase_b(const SysParams& P, const RangeStepArgs& A, RsShared& S, const float4* __restrict__ sp,
                                           const float4* __restrict__ sf, const RsItem& I, int tid, int db, int r_next) {
    if (tid < P.n_ranges * RS_DESC) {
        // this thread's record was requested one item ago (cp.async, no registers held): in steady state it is already
        // here and the L2 round trip is off the critical path; poll only if the window was not finished yet
        asm volatile("cp.async.wait_all;" ::: "memory");
        float4* mine = &S.desc[db][tid / RS_DESC][tid % RS_DESC];
        const float4* src = A.desc + (long long)I.r * P.n_ranges * RS_DESC + tid;
        float4 d = *mine;
        while (d.w != RS_TAG) {
            d = rs_ld_relaxed_f4(src);
            if (d.w != RS_TAG) __nanosleep(200);
        }
        *mine = d;
        if (r_next >= 0) {
            float4* nxt = &S.desc[(db + 1) % 3][tid / RS_DESC][tid % RS_DESC];
            *nxt = make_float4(0.f, 0.f, 0.f, 0.f);   // (an unpublished or skipped copy must read as invalid)
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(rs_smem_u32(nxt)),
                         "l"(A.desc + (long long)r_next * P.n_ranges * RS_DESC + tid)
                         : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
    }
    if (tid >= 32 && tid < 32 + P.n_ranges) {
        // slice-local bounds of every group: the atom loop compares 32-bit offsets held in shared memory
        const long long t0 = P.span_begin + (long long)I.s * RS_SLICE;
        long long lo = S.g_b[tid - 32] - t0, hi = S.g_e[tid - 32] - t0;
        const long long cnt = (long long)(I.bytes >> 4);
        if (lo < 0) lo = 0;
        if (hi > cnt) hi = cnt;
        S.blo[db][tid - 32] = (int)lo;
        S.bhi[db][tid - 32] = hi > lo ? (int)hi : (int)lo;
    }
    if (tid == 64) {
        // fast path: a whole slice that every group either covers completely or does not touch, and is touched at all
        const long long t0 = P.span_begin + (long long)I.s * RS_SLICE;
        const long long t1 = t0 + (long long)(I.bytes >> 4);
        bool fast = (I.bytes >> 4) == RS_SLICE, any = false;
        for (int q = 0; q < P.n_ranges; ++q) {
            const long long gb = S.g_b[q], ge = S.g_e[q];
            const bool touch = t0 < ge && t1 > gb, cover = gb <= t0 && t1 <= ge;
            if (touch && !cover) fast = false;
            any |= cover;
        }
        S.bfast[db] = fast && any;
    }
    rs_b_sync();
    float4* f = reinterpret_cast<float4*>(A.force) + I.a0;
    const long long t0 = P.span_begin + (long long)I.s * RS_SLICE;
    // group-major, the thread's RS_PERB atoms side by side (independent chains); per atom the groups are still
    // accumulated in increasing order, as in the unfused kernel
    float ax[RS_PERB], ay[RS_PERB], az[RS_PERB];
#pragma unroll
    for (int i = 0; i < RS_PERB; ++i) ax[i] = ay[i] = az[i] = 0.f;
    if (S.bfast[db] && !P.atom_weight) {
        // the common case, straight-line: a whole slice, every group either covers all of it or none of it, unit
        // weights (x * 1.0f is x: same bits as the general loop)
        for (int q = 0; q < P.n_ranges; ++q) {
            if (S.blo[db][q] >= S.bhi[db][q]) continue;   // uniform
            const float4 v = S.desc[db][q][0], hi = S.desc[db][q][1], lo = S.desc[db][q][2];
            const float k = S.desc[db][q][3].x;
#pragma unroll
            for (int i = 0; i < RS_PERB; ++i) {
                const float4 p = sp[tid + i * RS_GTB];   // re-read per group: registers are the scarce resource
                ax[i] += v.x + k * ((p.x - hi.x) - lo.x);
                ay[i] += v.y + k * ((p.y - hi.y) - lo.y);
                az[i] += v.z + k * ((p.z - hi.z) - lo.z);
            }
        }
#pragma unroll
        for (int i = 0; i < RS_PERB; ++i) {
            const int o = tid + i * RS_GTB;
            float4 fv = sf[o];
            fv.x += ax[i]; fv.y += ay[i]; fv.z += az[i];   // the record's w keeps its bits
            __stcs(f + o, fv);
        }
        return;
    }
    unsigned anym = 0u;
    for (int q = 0; q < P.n_ranges; ++q) {
        const int lo_o = S.blo[db][q], hi_o = S.bhi[db][q];
        if (lo_o >= hi_o) continue;   // uniform: the slice does not touch this group
        const float4 v = S.desc[db][q][0], hi = S.desc[db][q][1], lo = S.desc[db][q][2];
        const float k = S.desc[db][q][3].x;
#pragma unroll
        for (int i = 0; i < RS_PERB; ++i) {
            const int o = tid + i * RS_GTB;
            if (o >= lo_o && o < hi_o) {
                const float4 p = sp[o];
                anym |= 1u << i;
                ax[i] += v.x + k * ((p.x - hi.x) - lo.x);
                ay[i] += v.y + k * ((p.y - hi.y) - lo.y);
                az[i] += v.z + k * ((p.z - hi.z) - lo.z);
            }
        }
    }
#pragma unroll
    for (int i = 0; i < RS_PERB; ++i) {
        if (!((anym >> i) & 1u)) continue;   // an atom of the span that belongs to no group is not written
        const int o = tid + i * RS_GTB;
        const float w = P.atom_weight ? __ldg(P.atom_weight + t0 + o) : 1.f;
        float4 fv = sf[o];
        // (no contraction: same bits as the unfused path); the record's w keeps its bits
        fv.x += __fmul_rn(ax[i], w); fv.y += __fmul_rn(ay[i], w); fv.z += __fmul_rn(az[i], w);
        __stcs(f + o, fv);
    }
}

__global__ void __launch_bounds__(RS_THREADS, 1) k_range_step(const __grid_constant__ SysParams P, const __grid_constant__ RangeStepArgs A) {
    extern __shared__ __align__(128) unsigned char rs_smem[];
    float4* ring_a = reinterpret_cast<float4*>(rs_smem);                       // RS_ASTAGES x RS_SLICE positions
    float4* ring_b = ring_a + (size_t)RS_ASTAGES * RS_SLICE;                   // RS_BSTAGES x {RS_SLICE positions, RS_SLICE forces}
    RsShared& S = *reinterpret_cast<RsShared*>(ring_b + (size_t)RS_BSTAGES * 2 * RS_SLICE);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long items = (long long)P.R * P.range_blocks;
    const long long G = gridDim.x;
    const long long n_mine = blockIdx.x < items ? (items - blockIdx.x + G - 1) / G : 0;
    if (tid == 0) {
        for (int st = 0; st < RS_ASTAGES; ++st) { rs_mbar_init(&S.a_full[st], 1); rs_mbar_init(&S.a_empty[st], RS_GT / 32); }
        for (int st = 0; st < RS_BSTAGES; ++st) { rs_mbar_init(&S.b_full[st], 1); rs_mbar_init(&S.b_empty[st], RS_GTB / 32); }
        for (int b = 0; b < RS_RED; ++b) { rs_mbar_init(&S.red_full[b], RS_GT / 32); rs_mbar_init(&S.red_empty[b], 1); }
        S.b_prog = 0;
        for (int q = 0; q < PSG_MAX_RANGE_GROUPS; ++q)
            for (int i = 0; i < RS_DESC; ++i) S.desc[0][q][i] = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int q = 0; q < P.n_ranges; ++q) {
            const GroupDev& G = P.grp[P.range_gid[q]];
            S.g_b[q] = G.rbegin; S.g_e[q] = G.rbegin + G.rsize;
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == 0) {
        // ---------------- PA: positions -> ring A, at most `lag` items ahead of the B group
        if (lane == 0) {
            const uint64_t keep = rs_policy_evict_last();
            for (long long it = 0; it < n_mine; ++it) {
                const int st = (int)(it % RS_ASTAGES);
                if (it >= RS_ASTAGES) rs_mbar_wait(&S.a_empty[st], (uint32_t)((it / RS_ASTAGES - 1) & 1));
                while (it - S.b_prog > A.lag) __nanosleep(200);
                const RsItem I = rs_item(P, it, G);
                rs_mbar_expect_tx(&S.a_full[st], I.bytes);
                rs_tma_load_1d(ring_a + (size_t)st * RS_SLICE, reinterpret_cast<const float4*>(A.pos) + I.a0, I.bytes, &S.a_full[st], keep);
            }
        }
    } else if (warp == 1) {
        // ---------------- PB: positions (L2) + forces -> ring B
        if (lane == 0) {
            const uint64_t once = rs_policy_evict_first();
            for (long long it = 0; it < n_mine; ++it) {
                const int st = (int)(it % RS_BSTAGES);
                if (it >= RS_BSTAGES) rs_mbar_wait(&S.b_empty[st], (uint32_t)((it / RS_BSTAGES - 1) & 1));
                const RsItem I = rs_item(P, it, G);
                float4* dst = ring_b + (size_t)st * 2 * RS_SLICE;
                rs_mbar_expect_tx(&S.b_full[st], 2u * I.bytes);
                rs_tma_load_1d(dst, reinterpret_cast<const float4*>(A.pos) + I.a0, I.bytes, &S.b_full[st], once);
                rs_tma_load_1d(dst + RS_SLICE, reinterpret_cast<const float4*>(A.force) + I.a0, I.bytes, &S.b_full[st], once);
            }
        }
    } else if (warp == 2) {
        // ---------------- W: windows b, b + grid, ...
        for (long long r = blockIdx.x; r < P.R; r += G) {
            if (lane == 0) {
                unsigned n;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(n) : "l"(A.arrive + r) : "memory");
                    if (n < (unsigned)P.range_blocks) __nanosleep(200);
                } while (n < (unsigned)P.range_blocks);
            }
            __syncwarp();
            __threadfence();
            rs_window(P, A, S, (int)r, lane);
        }
    } else if (warp < 3 + RS_NT) {
        // ---------------- T warp j: items j, j + RS_NT, ...
        const int j = warp - 3;
        for (long long it = j; it < n_mine; it += RS_NT) {
            const int buf = (int)(it % RS_RED);
            const RsItem I = rs_item(P, it, G);
            rs_mbar_wait(&S.red_full[buf], (uint32_t)((it / RS_RED) & 1));
            rs_tail(P, A, S, I, buf, lane);
        }
    } else if (tid < RS_LEAD + RS_GT) {
        // ---------------- A group
        const int t = tid - RS_LEAD;
        for (long long it = 0; it < n_mine; ++it) {
            const int st = (int)(it % RS_ASTAGES), buf = (int)(it % RS_RED);
            const RsItem I = rs_item(P, it, G);
            rs_mbar_wait(&S.a_full[st], (uint32_t)((it / RS_ASTAGES) & 1));
            if (it >= RS_RED) rs_mbar_wait(&S.red_empty[buf], (uint32_t)((it / RS_RED - 1) & 1));
            rs_phase_a(P, S, ring_a + (size_t)st * RS_SLICE, I, buf, t);
            if ((t & 31) == 0) {
                rs_mbar_arrive(&S.red_full[buf]);   // this warp's partials are in S.red[buf]
                rs_mbar_arrive(&S.a_empty[st]);     // and it is done reading the stage
            }
        }
    } else {
        // ---------------- B group
        const int t = tid - RS_LEAD - RS_GT;
        for (long long it = 0; it < n_mine; ++it) {
            const int st = (int)(it % RS_BSTAGES);
            const RsItem I = rs_item(P, it, G);
            const float4* sp = ring_b + (size_t)st * 2 * RS_SLICE;
            rs_mbar_wait(&S.b_full[st], (uint32_t)((it / RS_BSTAGES) & 1));
            const int r_next = it + 1 < n_mine ? rs_item(P, it + 1, G).r : -1;
            rs_phase_b(P, A, S, sp, sp + RS_SLICE, I, t, (int)(it % 3), r_next);
            __syncwarp();
            if ((t & 31) == 0) rs_mbar_arrive(&S.b_empty[st]);   // this warp is done reading the stage
            if (t == 0) {
                S.b_prog = it + 1;
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

static const size_t kRsSmem = (size_t)(RS_ASTAGES + 2 * RS_BSTAGES) * RS_SLICE * 16 + sizeof(RsShared);

// co-resident CTAs per SM (0 if the kernel cannot be configured)
static int rs_blocks_per_sm(int device) {
    static int cache[PSG_MAX_DEVICES];
    static bool have[PSG_MAX_DEVICES] = {};
    int& n = cache[device % PSG_MAX_DEVICES];
    if (!have[device % PSG_MAX_DEVICES]) {
        have[device % PSG_MAX_DEVICES] = true;
        n = 0;
        if (cudaFuncSetAttribute(k_range_step, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kRsSmem) == cudaSuccess) {
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_range_step, RS_THREADS, kRsSmem) != cudaSuccess) n = 0;
        }
        (void)cudaGetLastError();
    }
    return n;
}

// The fused step covers: harmonic bias; every group a contiguous range; float4 positions and forces, 16-byte
// aligned (the position slices are TMA bulk copies); no minimum-image box; one array per window; windows of at most `grid` slices (so
// that every A a waiting B depends on belongs to the same or the next round of items). Anything else takes the
// separate kernels of cv.cu / bias.cu.
bool psg_range_step_supported(const psg_ctx* c, const float* d_pos, const float* d_force) {
    const SysParams& P = c->sys;
    if (c->range_step_off) return false;   // psg_set_tuning: take the separate kernels
    if (!(c->method == PSG_METHOD_HARMONIC && !P.has_box && !P.any_shape_range && P.n_ranges > 0 && P.n_slots == 0 && P.ps == 4 && P.fs == 4 && P.rstride > 0 &&
          ((reinterpret_cast<uintptr_t>(d_pos) | reinterpret_cast<uintptr_t>(d_force)) & 15u) == 0 &&
          c->d_arrive != nullptr))
        return false;
    const long long grid = (long long)c->sm_count * rs_blocks_per_sm(c->device);
    return grid >= 1 && P.range_blocks <= grid;
}

cudaError_t psg_launch_range_step(psg_ctx* c, const float* d_pos, float* d_force) {
    const int max_blocks_per_sm = rs_blocks_per_sm(c->device);
    if (max_blocks_per_sm < 1) return cudaErrorLaunchOutOfResources;
    const SysParams& P = c->sys;
    RangeStepArgs A{};
    A.pos = d_pos; A.force = d_force; A.kspring = c->d_kspring; A.centers = c->d_centers;
    A.xi_out = c->d_xi; A.V_out = c->d_V; A.V64_out = c->d_V64; A.dV_out = c->d_dVdxi;
    A.rpart = c->d_rpart; A.arrive = c->d_arrive; A.done = c->d_arrive + P.R; A.desc = c->d_rdesc;
    // B runs `lag` items behind A: long enough to cover the window dependency (several L2 round trips), short
    // enough that lag x grid x 32 KB of positions stays in L2 (10 x 148 x 32 KB = 47 MB of 126 MB; measured optimum)
    A.lag = c->range_lag > 0 ? c->range_lag : 10;
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
