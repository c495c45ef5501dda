// hills.cu -- metadynamics: host side of the hill sum, hill deposition, pack / unpack.
// The kernel itself is hills.cuh; its instantiations live in hills_n*.cu.
#include <math.h>

#include "hills.cuh"

cudaError_t psg_hills_dispatch_n12(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid);
cudaError_t psg_hills_dispatch_n3a(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid);
cudaError_t psg_hills_dispatch_n3b(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid);
cudaError_t psg_hills_dispatch_n4(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid);
cudaError_t psg_hills_dispatch_f64(psg_ctx* c, const HillKernelArgs& A, size_t smem, int grid);

// ---------------------------------------------------------------- deposition
// Single block. Replica r deposits (mask == NULL or mask[r]) at slot n_h + (#depositing replicas before r):
// replica order. W = w0 exp(-V_old/(kB dT)) in binary64, stored binary32 (well-tempered) or W = w0.
// The kernel-side record carries log2 of the STORED (binary32) height, so that the exported list and the
// list the hill sum uses are the same numbers.
__device__ __forceinline__ void store_hill(float4* __restrict__ hills, float* __restrict__ heights, int rec, int slot, const float (&s)[4],
                                           float W) {
    float lw = (float)log2((double)W);   // W = 0 -> -inf -> contributes exactly 0
    heights[slot] = W;
    if (rec == 1) hills[slot] = make_float4(s[0], s[1], s[2], lw);
    else {
        hills[2 * slot] = make_float4(s[0], s[1], s[2], s[3]);
        hills[2 * slot + 1] = make_float4(lw, 0.f, 0.f, 0.f);
    }
}

// W_in == nullptr: one deposit event of this ctx's R walkers (heights from Vold).  W_in != nullptr: append R ready-made hills
// (centres xi, heights W_in; the other ranks' included, psg_append_hills), skipping the zero heights of masked-out walkers.
__global__ void __launch_bounds__(1024) k_deposit(int R, int n_cv, int rec, const float* __restrict__ xi, const double* __restrict__ Vold,
                                                   const unsigned char* __restrict__ mask, double w0, double kBdT, float4* __restrict__ hills,
                                                   float* __restrict__ heights, int* __restrict__ n_hills, int capacity,
                                                   const float* __restrict__ W_in) {
    __shared__ int s_warp[32];
    __shared__ int s_base;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) s_base = *n_hills;
    __syncthreads();
    for (int r0 = 0; r0 < R; r0 += 1024) {
        int r = r0 + tid;
        int dep = (r < R) && (W_in ? W_in[r] != 0.f : (!mask || mask[r]));
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
                float W = W_in ? W_in[r] : (float)(kBdT > 0.0 ? w0 * exp(-Vold[r] / kBdT) : w0);
                float s[4] = {0.f, 0.f, 0.f, 0.f};
                for (int k = 0; k < n_cv; ++k) s[k] = xi[(long long)r * n_cv + k];
                store_hill(hills, heights, rec, slot, s, W);
            }
        }
        __syncthreads();
        if (tid == 0) {
            if (s_base + tot > capacity) n_hills[1] = 1;   // sticky: hills were dropped (reported by psg_sync_check / psg_get_hills)
            s_base = min(s_base + tot, capacity);
        }
        __syncthreads();
    }
    if (tid == 0) *n_hills = s_base;
}

__global__ void k_pack_hills(int n, int n_cv, int rec, const float* __restrict__ centers, const float* __restrict__ heights_in,
                             float4* __restrict__ hills, float* __restrict__ heights) {
    int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n) return;
    float s[4] = {0.f, 0.f, 0.f, 0.f};
    for (int k = 0; k < n_cv; ++k) s[k] = centers[(long long)h * n_cv + k];
    store_hill(hills, heights, rec, h, s, heights_in[h]);
}

__global__ void k_unpack_hills(int n, int n_cv, int rec, const float4* __restrict__ hills, const float* __restrict__ heights_in,
                               float* __restrict__ centers, float* __restrict__ heights) {
    int h = blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= n) return;
    float4 a = hills[rec * h];
    float s[4] = {a.x, a.y, a.z, a.w};
    if (rec == 2 && n_cv > 3) s[3] = a.w;
    for (int k = 0; k < n_cv; ++k) centers[(long long)h * n_cv + k] = s[k];
    heights[h] = heights_in[h];
}

// null records: centre 0, log2 W = -inf, W = 0: ex2(-inf) = 0, so they add exactly 0 to V and to the gradient
__global__ void k_null_hills(int begin, int end, int rec, float4* __restrict__ hills, float* __restrict__ heights) {
    int h = begin + blockIdx.x * blockDim.x + threadIdx.x;
    if (h >= end) return;
    const float ninf = __int_as_float(0xff800000);
    heights[h] = 0.f;
    if (rec == 1) hills[h] = make_float4(0.f, 0.f, 0.f, ninf);
    else {
        hills[2 * h] = make_float4(0.f, 0.f, 0.f, 0.f);
        hills[2 * h + 1] = make_float4(ninf, 0.f, 0.f, 0.f);
    }
}

// ---------------------------------------------------------------- host side
bool psg_stream_capturing(const psg_ctx* c) {
    cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(c->stream, &st) != cudaSuccess) { st = cudaStreamCaptureStatusNone; (void)cudaGetLastError(); }
    return st != cudaStreamCaptureStatusNone;
}
static int hills_grid(const psg_ctx* c) { return c->sm_count; }   // one 16-warp CTA per SM

size_t psg_hill_part_doubles(const psg_ctx* c, int* max_chunks_out, int* n_rtiles_out) {
    int n_rt = (c->sys.R + TILE_R - 1) / TILE_R;
    int cpt = hills_grid(c) / n_rt;
    if (cpt < 1) cpt = 1;
    if (max_chunks_out) *max_chunks_out = cpt + 1;
    if (n_rtiles_out) *n_rtiles_out = n_rt;
    return (size_t)(cpt + 1) * n_rt * TILE_R * (1 + PSG_MAX_CV);   // + 1: the short last chunk of hills_spare_chunking
}

static cudaError_t launch_hills(psg_ctx* c, HillKernelArgs& A) {
    const int n_cv = c->sys.n_cv;
    const bool fused = A.fused != 0;
    // stages of 64 KB: three of them fit the SM's 227 KB beside the per-warp totals for every n_cv and group count (the hand-back
    // scheme wants 3: the refill of a stage is issued one sub-tile after its last reader left)
    int stages = PSG_HILL_MAX_STAGES;
    for (; stages > 3; --stages)
        if (hills_smem_bytes(n_cv, stages, c->sys.n_groups, fused) + 1024 <= 227 * 1024) break;
    A.stages = stages;
    const size_t smem = hills_smem_bytes(n_cv, stages, c->sys.n_groups, fused);
    const int grid = hills_grid(c);
    const int n_rt = (c->sys.R + TILE_R - 1) / TILE_R;
    A.inv_n_rt = 1.0f / (float)n_rt;
    A.Lc_host = A.n_chunks_host = 0;
    A.n_long = 0;
    if (A.n_h_host >= 0) {
        hills_chunking(A.n_h_host, grid, n_rt, A.Lc_host, A.n_chunks_host);
        if (PSG_SPARE_CHUNKS(n_cv, c->md.precision == PSG_HILLS_F64)) hills_spare_chunking(A.n_h_host, grid, n_rt, A.Lc_host, A.n_chunks_host, A.n_long);
    }
    A.simple = fused && c->sys.simple_groups && !c->sys.slot_weight && !c->sys.has_box;
    if (c->md.precision == PSG_HILLS_F64) return psg_hills_dispatch_f64(c, A, smem, grid);
    switch (n_cv) {
    case 1:
    case 2: return psg_hills_dispatch_n12(c, A, smem, grid);
    case 3: return (c->md.hc.pmask & 4) ? psg_hills_dispatch_n3b(c, A, smem, grid) : psg_hills_dispatch_n3a(c, A, smem, grid);
    case 4: return psg_hills_dispatch_n4(c, A, smem, grid);
    }
    return cudaErrorInvalidValue;
}

static HillKernelArgs base_args(psg_ctx* c) {
    HillKernelArgs A{};
    A.hills = c->md.hills; A.heights = c->md.heights; A.n_hills = c->md.n_hills; A.part = c->md.part;
    A.R = c->sys.R;
    // The host's upper bound of the hill count saves the kernel a dependent global load. Under stream capture the
    // launch may be replayed with a longer list than the one seen now, and after a CAPTURED deposit the replays grow the
    // list behind the host's back: in both cases the kernel reads the device counter.
    A.n_h_host = (psg_stream_capturing(c) || c->count_unknown) ? -1 : (int)c->nh_bound;
    return A;
}

cudaError_t psg_launch_null_hills(psg_ctx* c, int begin, int end) {
    if (end > begin) {
        k_null_hills<<<(end - begin + 255) / 256, 256, 0, c->stream>>>(begin, end, c->md.rec, c->md.hills, c->md.heights);
        c->launches++;
    }
    return cudaGetLastError();
}

cudaError_t psg_launch_hillsum(psg_ctx* c, const float* d_xi, float* d_V, float* d_dVdxi) {
    HillKernelArgs A = base_args(c);
    A.xi_in = d_xi; A.V_out = d_V; A.V64_out = c->d_V64; A.dV_out = d_dVdxi; A.fused = 0;
    return launch_hills(c, A);
}

bool psg_metad_step_supported(const psg_ctx* c) { return c->sys.n_ranges == 0 && !c->sys.any_rgyr; }

cudaError_t psg_launch_metad_step(psg_ctx* c, const float* d_pos, float* d_force) {
    HillKernelArgs A = base_args(c);
    A.V_out = c->d_V; A.V64_out = c->d_V64; A.dV_out = c->d_dVdxi; A.xi_out = c->d_xi;
    A.pos = d_pos; A.force = d_force; A.fused = 1;
    return launch_hills(c, A);
}

cudaError_t psg_launch_deposit(psg_ctx* c, const float* d_xi, const unsigned char* d_mask) {
    if (c->md.kB_deltaT > 0.0) {
        cudaError_t e = psg_launch_hillsum(c, d_xi, nullptr, nullptr);   // V_old -> d_V64
        if (e != cudaSuccess) return e;
    }
    k_deposit<<<1, 1024, 0, c->stream>>>(c->sys.R, c->sys.n_cv, c->md.rec, d_xi, c->d_V64, d_mask, c->md.w0, c->md.kB_deltaT,
                                         c->md.hills, c->md.heights, c->md.n_hills, c->md.capacity, nullptr);
    c->launches++;
    return cudaGetLastError();
}

// the height every walker of this ctx would deposit now (0 where masked out); nothing is appended
__global__ void __launch_bounds__(256) k_hill_heights(int R, const double* __restrict__ Vold, const unsigned char* __restrict__ mask,
                                                       double w0, double kBdT, float* __restrict__ W_out) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    float W = 0.f;
    if (!mask || mask[r]) W = (float)(kBdT > 0.0 ? w0 * exp(-Vold[r] / kBdT) : w0);   // the expression of k_deposit
    W_out[r] = W;
}

cudaError_t psg_launch_hill_heights(psg_ctx* c, const float* d_xi, const unsigned char* d_mask, float* d_heights) {
    if (c->md.kB_deltaT > 0.0) {
        cudaError_t e = psg_launch_hillsum(c, d_xi, nullptr, nullptr);   // V_old -> d_V64
        if (e != cudaSuccess) return e;
    }
    k_hill_heights<<<(c->sys.R + 255) / 256, 256, 0, c->stream>>>(c->sys.R, c->d_V64, d_mask, c->md.w0, c->md.kB_deltaT, d_heights);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t psg_launch_append_hills(psg_ctx* c, int n, const float* d_centers, const float* d_heights) {
    k_deposit<<<1, 1024, 0, c->stream>>>(n, c->sys.n_cv, c->md.rec, d_centers, nullptr, nullptr, c->md.w0, c->md.kB_deltaT,
                                         c->md.hills, c->md.heights, c->md.n_hills, c->md.capacity, d_heights);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t psg_launch_pack_hills(psg_ctx* c, int n, const float* d_centers, const float* d_heights) {
    if (n > 0) {
        k_pack_hills<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->sys.n_cv, c->md.rec, d_centers, d_heights, c->md.hills,
                                                             c->md.heights);
        c->launches++;
    }
    return cudaGetLastError();
}

cudaError_t psg_launch_unpack_hills(psg_ctx* c, int n, float* d_centers, float* d_heights) {
    if (n > 0) {
        k_unpack_hills<<<(n + 255) / 256, 256, 0, c->stream>>>(n, c->sys.n_cv, c->md.rec, c->md.hills, c->md.heights, d_centers,
                                                               d_heights);
        c->launches++;
    }
    return cudaGetLastError();
}
