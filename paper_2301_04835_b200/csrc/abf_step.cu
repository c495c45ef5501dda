// abf_step.cu -- the fused ABF step: ONE launch
// per MD step instead of four.  A step of config 2 moves < 4 MB, so launch latency, not bandwidth, is what it costs.
//
//   phase 1  warp per replica: gather the CV atoms in place, CVs + Jacobians (binary64 registers), bin xi in
//            binary32, hist[bin] += 1 (int32 atomic), Fsum[bin] += f (vector float atomic)
//   grid barrier (all replicas have accumulated: the two-phase reading R-ABF-2 of DESIGN.md)
//   phase 2  the same warp: Fbar = Fsum[bin] / max(hist[bin], N)  ->  dV/dxi;  force[i] += -Fbar_k * dxi_k/dr_i
//            (red.global.add.f32: atoms shared between CVs or walkers collide)
// The barrier is a counter in global memory, so the grid must be co-resident: the kernel is launched cooperatively
// (the launch fails instead of hanging) with at most occupancy x SM-count CTAs; warps loop over replicas.
// k_abf_step_lean (below) takes the whole step for the common layout: two threads per (replica, CV) instead of a warp per
// replica.
// Same arithmetic as k_cv_eval + k_abf_accumulate + k_abf_mean + k_apply_sparse: bins, counts, xi, dV/dxi and the
// Jacobian are bit-identical to the separate calls; Fsum and forces differ only by the order of the atomics.
#include "abf.cuh"
#include "geom.cuh"

struct AbfStepArgs {
    const float* pos;
    const float* fsample;   // [R][n_cv]
    float* force;
    float* xi_out;          // [R][n_cv]
    int* bin_out;           // [R]
    float* dV_out;          // [R][n_cv]
    float* jac;             // [R][n_slots][3] (the ctx cache, as after psg_cv_eval)
    unsigned* bar;          // [2] arrive / depart counters, zero between launches
    int phase;              // 0: the whole step; 1: phase 1 only (G then points at per-step DELTA arrays, psg_abf_accumulate_delta);
                            // 2: phase 2 only (bins and Jacobians of an earlier phase-1 launch, psg_abf_apply_grid_delta)
};

__global__ void __launch_bounds__(256, 4) k_abf_step(const __grid_constant__ SysParams P, const __grid_constant__ AbfState G,
                                                  const __grid_constant__ AbfStepArgs A) {
    __shared__ WarpCvSmem sm[8];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int warps = gridDim.x * 8, gw = blockIdx.x * 8 + wid;
    WarpCvSmem& S = sm[wid];

    // With at most one replica per warp (R <= resident warps: config 2's 4,096 on 4,736) the warp keeps what phase 2 needs ON
    // CHIP across the barrier: lane 0 the bin, lane s the Jacobian of slot s (the first 32 slots; more go through the ctx
    // cache).  Phase 2 is then ONE L2 round trip (the grid entry) instead of three (bin, grid entry, dV + Jacobian).
    const bool one = A.phase == 0 && P.R <= warps;   // grid-uniform
    int my_bin = -1;
    float jx = 0.f, jy = 0.f, jz = 0.f;
    for (int r = gw; A.phase != 2 && r < P.R; r += warps) {
        warp_cv_eval<true>(P, r, A.pos, nullptr, S, lane);
        if (lane < P.n_cv) A.xi_out[(long long)r * P.n_cv + lane] = (float)S.xi[lane];
        for (int s = lane; s < P.n_slots; s += 32) {
            const D3 j = slot_jacobian(P, r, A.pos, S, s);
            const long long o = ((long long)r * P.n_slots + s) * 3;
            A.jac[o] = (float)j.x; A.jac[o + 1] = (float)j.y; A.jac[o + 2] = (float)j.z;
            if (s == lane) { jx = (float)j.x; jy = (float)j.y; jz = (float)j.z; }
            // the force record phase 2 will update, requested into L2 now (the arrays are GBs: a cold miss otherwise)
            const int atom = slot_atom_of(P, r, s);
            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.force + ((long long)r * P.rstride + atom) * P.fs));
        }
        if (lane == 0) {
            float xi[PSG_MAX_CV];
#pragma unroll
            for (int k = 0; k < PSG_MAX_CV; ++k) xi[k] = k < P.n_cv ? (float)S.xi[k] : 0.f;
            my_bin = abf_accumulate_one(G, P.n_cv, xi, A.fsample + (long long)r * P.n_cv);
            A.bin_out[r] = my_bin;
        }
        __syncwarp();
    }

    if (A.phase == 1) return;
    // ---- grid barrier: every replica's atomics are performed before anyone reads the grid
    __syncthreads();
    if (A.phase == 0 && tid == 0) {
        __threadfence();
        atomicAdd(A.bar, 1u);
        unsigned n;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(n) : "l"(A.bar) : "memory");
        } while (n < gridDim.x);
    }
    __syncthreads();

    for (int r = gw; r < P.R; r += warps) {
        float* dV = A.dV_out + (long long)r * P.n_cv;
        if (one) {
            float* sdv = reinterpret_cast<float*>(&S.xi[0]);   // this warp's scratch: phase 1 is over
            if (lane == 0) {
                abf_mean_one(G, P.n_cv, my_bin, sdv);
                for (int k = 0; k < P.n_cv; ++k) dV[k] = sdv[k];
            }
            __syncwarp();
            for (int s = lane; s < P.n_slots; s += 32) {
                const int gid = P.slot_gid_c[s];
                const float dv = -sdv[P.grp[gid].cv];
                const int atom = slot_atom_of(P, r, s);
                float* f = A.force + ((long long)r * P.rstride + atom) * P.fs;
                if (s < 32) {
                    force_add(f, dv * jx, dv * jy, dv * jz, P.fs);
                } else {
                    const float* j = A.jac + ((long long)r * P.n_slots + s) * 3;
                    force_add(f, dv * j[0], dv * j[1], dv * j[2], P.fs);
                }
            }
            continue;
        }
        if (lane == 0) abf_mean_one(G, P.n_cv, A.bin_out[r], dV);
        __syncwarp();
        for (int s = lane; s < P.n_slots; s += 32) {
            const int gid = P.slot_gid_c[s];
            const float dv = -dV[P.grp[gid].cv];
            const int atom = slot_atom_of(P, r, s);
            float* f = A.force + ((long long)r * P.rstride + atom) * P.fs;
            const float* j = A.jac + ((long long)r * P.n_slots + s) * 3;
            force_add(f, dv * j[0], dv * j[1], dv * j[2], P.fs);
        }
    }

    // ---- the last CTA to leave re-arms the barrier for the next launch
    __syncthreads();
    if (A.phase == 0 && tid == 0) {
        const unsigned old = atomicAdd(A.bar + 1, 1u);
        if (old == gridDim.x - 1) { A.bar[0] = 0u; A.bar[1] = 0u; }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// The same step for the common layout (explicit groups, no box, point-group CVs): TWO THREADS per
// (replica, CV) instead of a warp per replica.  One thread takes the value (sqrt / atan2 chain), another (in another warp) the
// derivative (cv_jacobian_only: Newton-refined hardware reciprocals), so the two binary64 chains run side by side and a warp
// instruction carries 32 of them: the warp-per-replica kernel issues every binary64 instruction for 2 live lanes, and with
// 32 such warps per SM the FP64 pipe (16 lanes/clk per scheduler) is what phase 1 waits for (measured: 5.3-7.3 us of a
// 13 us launch).  Each thread gathers the (few) atoms of its CV's groups itself.  The thread that owns the derivative keeps it
// in registers across the barrier and scatters it.
// LEAN_RB replicas per CTA; block = LEAN_RB x n_cv value threads followed by as many derivative threads (whole warps each: the
// two roles are different code and would serialise inside a warp); grid = ceil(R / LEAN_RB), co-resident (cooperative launch).
#define LEAN_RB 32
__global__ void __launch_bounds__(LEAN_RB * PSG_MAX_CV * 2) k_abf_step_lean(const __grid_constant__ SysParams P, const __grid_constant__ AbfState G,
                                                                          const __grid_constant__ AbfStepArgs A) {
    __shared__ float s_xi[LEAN_RB][PSG_MAX_CV], s_dv[LEAN_RB][PSG_MAX_CV];
    __shared__ int s_bin[LEAN_RB];
    const int tid = threadIdx.x, n_cv = P.n_cv;
    const int role = tid >= LEAN_RB * n_cv ? 1 : 0;   // role 0: value, 1: derivative
    const int t = tid - role * LEAN_RB * n_cv, rl = t / n_cv, k = t - rl * n_cv;
    const int r = blockIdx.x * LEAN_RB + rl;
    const bool live = r < P.R;
    const CvDev& C = P.cv[k];
    float jf[4][3];   // derivative thread: d xi_k / d c_g / W_g, rounded to binary32 like the ctx cache
    if (live) {
        const float* p = A.pos + (long long)r * P.rstride * P.ps;
        D3 c[4], dc[4];
        double Wg[4];
        thread_group_centres(P, r, C, p, c, Wg);   // (the arithmetic of warp_cv_eval's gather: xi keeps its bits)
        if (role == 0) {
            const float v = (float)cv_from_centers<false>(C.type, C.axis, c, dc, nullptr);
            s_xi[rl][k] = v;
            A.xi_out[(long long)r * n_cv + k] = v;
        } else {
            cv_jacobian_only(C.type, C.axis, c, dc);
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                const double iw = fast_rcp(Wg[g]);
                jf[g][0] = (float)(dc[g].x * iw); jf[g][1] = (float)(dc[g].y * iw); jf[g][2] = (float)(dc[g].z * iw);
                if (g < C.n_groups) {
                    const GroupDev& Gd = P.grp[C.gid0 + g];
                    for (int i = 0; i < Gd.size; ++i) {
                        // the ctx cache, as after psg_cv_eval; and the force record phase 2 will update, requested into L2 now
                        const int s = Gd.begin + i;
                        const double w = P.slot_weight ? (double)P.slot_weight[s] : 1.0;
                        const long long o = ((long long)r * P.n_slots + s) * 3;
                        A.jac[o] = (float)(w * (dc[g].x * iw)); A.jac[o + 1] = (float)(w * (dc[g].y * iw)); A.jac[o + 2] = (float)(w * (dc[g].z * iw));
                        asm volatile("prefetch.global.L2 [%0];" ::"l"(A.force + ((long long)r * P.rstride + slot_atom_of(P, r, s)) * P.fs));
                    }
                }
            }
        }
    }
    __syncthreads();
    const bool owner = live && k == 0 && role == 0;   // one thread per replica bins and reads the grid
    if (owner) {
        float xi[PSG_MAX_CV];
#pragma unroll
        for (int q = 0; q < PSG_MAX_CV; ++q) xi[q] = q < n_cv ? s_xi[rl][q] : 0.f;
        const int b = abf_accumulate_one(G, n_cv, xi, A.fsample + (long long)r * n_cv);
        s_bin[rl] = b;
        A.bin_out[r] = b;
    }
    // ---- grid barrier: every replica's atomics are performed before anyone reads the grid
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        atomicAdd(A.bar, 1u);
        unsigned n;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(n) : "l"(A.bar) : "memory");
        } while (n < gridDim.x);
    }
    __syncthreads();
    if (owner) {
        abf_mean_one(G, n_cv, s_bin[rl], s_dv[rl]);
        for (int q = 0; q < n_cv; ++q) A.dV_out[(long long)r * n_cv + q] = s_dv[rl][q];
    }
    __syncthreads();
    if (live && role == 1) {
        const float dv = -s_dv[rl][k];
#pragma unroll
        for (int g = 0; g < 4; ++g)
            if (g < C.n_groups) {
                const GroupDev& Gd = P.grp[C.gid0 + g];
                for (int i = 0; i < Gd.size; ++i) {
                    const int s = Gd.begin + i;
                    const float w = P.slot_weight ? P.slot_weight[s] : 1.f;
                    force_add(A.force + ((long long)r * P.rstride + slot_atom_of(P, r, s)) * P.fs, dv * (w * jf[g][0]), dv * (w * jf[g][1]),
                              dv * (w * jf[g][2]), P.fs);
                }
            }
    }
    // ---- the last CTA to leave re-arms the barrier for the next launch
    if (tid == 0) {
        const unsigned old = atomicAdd(A.bar + 1, 1u);
        if (old == gridDim.x - 1) { A.bar[0] = 0u; A.bar[1] = 0u; }
    }
}

// CTAs of the lean kernel that can be co-resident on the device (0 if it cannot be configured)
static long long abf_lean_capacity(const psg_ctx* c, int threads) {
    int n = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_abf_step_lean, threads, 0) != cudaSuccess) n = 0;
    (void)cudaGetLastError();
    return (long long)n * c->sm_count;
}

static int abf_blocks_per_sm(int device) {
    static int cache[PSG_MAX_DEVICES];
    static bool have[PSG_MAX_DEVICES] = {};
    int& n = cache[device % PSG_MAX_DEVICES];
    if (!have[device % PSG_MAX_DEVICES]) {
        have[device % PSG_MAX_DEVICES] = true;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, k_abf_step, 256, 0) != cudaSuccess) n = 0;
        (void)cudaGetLastError();
    }
    return n;
}

bool psg_abf_step_supported(const psg_ctx* c) {
    return c->method == PSG_METHOD_ABF && c->sys.n_ranges == 0 && c->dti_cv < 0 && c->d_gbar != nullptr && abf_blocks_per_sm(c->device) >= 1;
}

// grid[b] += delta[b] for every bin (the all-reduced contribution of one step, psg_abf_apply_grid_delta)
__global__ void __launch_bounds__(256) k_abf_add_delta(long long n_bins, int n_cv, int* __restrict__ hist, float* __restrict__ fsum,
                                                        const int* __restrict__ dh, const float* __restrict__ df) {
    const long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_bins) return;
    hist[b] += dh[b];
    for (int k = 0; k < n_cv; ++k) fsum[b * n_cv + k] += df[b * n_cv + k];
}

cudaError_t psg_launch_abf_add_delta(psg_ctx* c, const int* d_hist_delta, const float* d_fsum_delta) {
    const long long nb = c->abf.n_bins;
    k_abf_add_delta<<<(unsigned)((nb + 255) / 256), 256, 0, c->stream>>>(nb, c->sys.n_cv, c->abf.hist, c->abf.fsum, d_hist_delta,
                                                                         d_fsum_delta);
    c->launches++;
    return cudaGetLastError();
}

// one half of the step on its own (phase 1 into `hist` / `fsum`, which may be per-step delta arrays; phase 2 from the ctx grid):
// no inter-CTA wait, so an ordinary launch
cudaError_t psg_launch_abf_phase(psg_ctx* c, int phase, const float* d_pos, const float* d_fsample, float* d_force, int* hist,
                                 float* fsum) {
    const SysParams& P = c->sys;
    AbfStepArgs A{};
    A.pos = d_pos; A.fsample = d_fsample; A.force = d_force;
    A.xi_out = c->d_xi; A.bin_out = c->d_bin; A.dV_out = c->d_dVdxi; A.jac = c->d_jac; A.bar = c->d_gbar; A.phase = phase;
    AbfState G = c->abf;
    G.hist = hist; G.fsum = fsum;
    long long grid = (P.R + 7) / 8;
    const long long cap = (long long)c->sm_count * 8;
    if (grid > cap) grid = cap;
    k_abf_step<<<(unsigned)grid, 256, 0, c->stream>>>(P, G, A);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t psg_launch_abf_step(psg_ctx* c, const float* d_pos, const float* d_fsample, float* d_force) {
    const SysParams& P = c->sys;
    AbfStepArgs A{};
    A.pos = d_pos; A.fsample = d_fsample; A.force = d_force;
    A.xi_out = c->d_xi; A.bin_out = c->d_bin; A.dV_out = c->d_dVdxi; A.jac = c->d_jac; A.bar = c->d_gbar; A.phase = 0;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;   // co-residency is what makes the grid barrier safe
    attr[0].val.cooperative = 1;
    if (psg_lean_layout(c)) {
        const int threads = LEAN_RB * P.n_cv * 2;
        const long long lgrid = (P.R + LEAN_RB - 1) / LEAN_RB;
        if (lgrid <= abf_lean_capacity(c, threads)) {
            cudaLaunchConfig_t cfg{};
            cfg.gridDim = dim3((unsigned)lgrid); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = 0; cfg.stream = c->stream;
            cfg.attrs = attr; cfg.numAttrs = 1;
            cudaError_t e = cudaLaunchKernelEx(&cfg, k_abf_step_lean, P, c->abf, A);
            if (e == cudaSuccess) c->launches++;
            return e;
        }
    }
    long long grid = (P.R + 7) / 8;
    const long long cap = (long long)c->sm_count * abf_blocks_per_sm(c->device);
    if (grid > cap) grid = cap;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3(256); cfg.dynamicSmemBytes = 0; cfg.stream = c->stream;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cudaError_t e = cudaLaunchKernelEx(&cfg, k_abf_step, P, c->abf, A);
    if (e == cudaSuccess) c->launches++;
    return e;
}
