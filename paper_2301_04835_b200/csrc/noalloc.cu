// noalloc.cu -- psg_range_rgyr_static (include/psg_static.h): the range-moment reduction of cv.cu's k_range_moments for one
// contiguous group, with its scratch (the per-block partial moments) in a file-scope static __device__ array instead of
// ctx memory, so that the call allocates nothing.  Two kernels: block partials -> scratch, one warp per replica combines.
// The thread -> atom map and every summation order are those of k_range_moments / warp_cv_eval (open boundaries).
#include <mutex>
#include <string>

#include "geom.cuh"
#include "psg_static.h"

static_assert(PSG_STATIC_TILE == PSG_RANGE_TILE, "the static variant keeps k_range_moments' tile");

// The scratch.  Every device that loads the library holds its own copy until the process exits.  In HOST code this name is
// a host-side stand-in, not a device address: host code below only ever hands it to cudaGetSymbolAddress.
static __device__ __align__(256) double g_static_rpart[(size_t)PSG_STATIC_MAX_BLOCKS * PSG_MOM];

struct StaticRangeArgs {
    const float* pos;
    const float* weight;   // nullable
    long long rstride, first, count;
    int ps, blocks, R;
};

// grid (blocks, R), block b of replica r: atoms [first + b*TILE, +TILE) of the range -> rpart[r][b][5], binary64
__global__ void __launch_bounds__(PSG_RANGE_THREADS, 4) k_range_moments_static(const StaticRangeArgs A, double* __restrict__ rpart) {
    constexpr int NT = PSG_RANGE_THREADS, PER = PSG_RANGE_TILE / NT;
    const int r = blockIdx.y, b = blockIdx.x, tid = threadIdx.x;
    const float* p = A.pos + (long long)r * A.rstride * A.ps;
    const long long t0 = A.first + (long long)b * PSG_RANGE_TILE, end = A.first + A.count;
    double m[PSG_MOM] = {0, 0, 0, 0, 0};
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        const long long a = t0 + tid + (long long)i * NT;
        float x = 0.f, y = 0.f, z = 0.f, wf = 0.f;
        if (a < end) {
            if (A.ps == 4) {
                const float4 v = __ldg(reinterpret_cast<const float4*>(p) + a);
                x = v.x; y = v.y; z = v.z;
            } else {
                x = __ldg(p + a * 3); y = __ldg(p + a * 3 + 1); z = __ldg(p + a * 3 + 2);
            }
            wf = A.weight ? __ldg(A.weight + a) : 1.f;
        }
        // an atom past the end enters with w = 0 and r = 0, which adds exactly +0
        const double xd = (double)x, yd = (double)y, zd = (double)z, wd = (double)wf;
        m[0] += wd; m[1] += wd * xd; m[2] += wd * yd; m[3] += wd * zd;
        m[4] += wd * (xd * xd + yd * yd + zd * zd);
    }
    __shared__ double red[NT / 32][PSG_MOM];
#pragma unroll
    for (int i = 0; i < PSG_MOM; ++i) m[i] = warp_sum(m[i]);
    if ((tid & 31) == 0) {
#pragma unroll
        for (int i = 0; i < PSG_MOM; ++i) red[tid >> 5][i] = m[i];
    }
    __syncthreads();
    if (tid < PSG_MOM) {
        double s = 0;
#pragma unroll
        for (int wq = 0; wq < NT / 32; ++wq) s += red[wq][tid];
        rpart[((long long)r * A.blocks + b) * PSG_MOM + tid] = s;   // every record the finisher reads is written here, each call
    }
}

// one warp per replica: block partials in lane-strided order, then Rg^2 = sum w|r|^2 / W - |c|^2 (as warp_cv_eval)
__global__ void __launch_bounds__(256) k_rgyr_static(const StaticRangeArgs A, const double* __restrict__ rpart, float* __restrict__ xi,
                                                     double* __restrict__ center) {
    const int lane = threadIdx.x & 31, r = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (r >= A.R) return;
    const double* src = rpart + (long long)r * A.blocks * PSG_MOM;
    double a[PSG_MOM] = {0, 0, 0, 0, 0};
    for (int b = lane; b < A.blocks; b += 32) {
#pragma unroll
        for (int i = 0; i < PSG_MOM; ++i) a[i] += __ldcg(src + (long long)b * PSG_MOM + i);
    }
#pragma unroll
    for (int i = 0; i < PSG_MOM; ++i) a[i] = warp_sum(a[i]);
    if (lane == 0) {
        const double iw = 1.0 / a[0];
        const D3 c = d3(a[1] * iw, a[2] * iw, a[3] * iw);
        const double rg2 = a[4] / a[0] - dot(c, c);
        xi[r] = (float)(rg2 > 0.0 ? sqrt(rg2) : 0.0);
        if (center) {
            center[4 * r] = c.x; center[4 * r + 1] = c.y; center[4 * r + 2] = c.z; center[4 * r + 3] = a[0];
        }
    }
}

// ------------------------------------------------------------------------------------------------ host side
static thread_local std::string g_static_err;
static std::mutex g_static_mu;
static double* g_static_ptr[PSG_MAX_DEVICES];   // DEVICE address of g_static_rpart on each device, looked up once per device

static int sfail(int code, const std::string& msg) {
    g_static_err = msg;
    return code;
}

// with `device` current: the device address of the scratch array on that device (cudaGetSymbolAddress, once per device)
static int static_scratch(int device, double** out) {
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_rpart);
        if (e != cudaSuccess || !p)
            return sfail(PSG_ECUDA, std::string("psg_range_rgyr_static: cudaGetSymbolAddress(g_static_rpart): ") + cudaGetErrorString(e));
        g_static_ptr[device] = static_cast<double*>(p);
    }
    *out = g_static_ptr[device];
    return PSG_OK;
}

namespace {
struct DeviceRestore {   // the caller's current device comes back on every return path
    int prev = -1;
    ~DeviceRestore() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};
}   // namespace

extern "C" const char* psg_static_last_error(void) { return g_static_err.c_str(); }

extern "C" int psg_range_rgyr_static(int device, void* cuda_stream, const float* d_pos, int pos_stride, int n_replicas,
                                     long long replica_stride_atoms, long long first_atom, long long n_group_atoms,
                                     const float* d_weight, float* d_xi, double* d_center) {
    if (device < 0 || device >= PSG_MAX_DEVICES) return sfail(PSG_EINVAL, "psg_range_rgyr_static: device must be in [0, 64)");
    if (!d_pos || !d_xi) return sfail(PSG_EINVAL, "psg_range_rgyr_static: d_pos and d_xi must not be NULL");
    if (pos_stride != 3 && pos_stride != 4) return sfail(PSG_EINVAL, "psg_range_rgyr_static: pos_stride must be 3 or 4");
    if (pos_stride == 4 && (reinterpret_cast<uintptr_t>(d_pos) & 15))
        return sfail(PSG_EINVAL, "psg_range_rgyr_static: pos_stride 4 needs 16-byte aligned positions");
    if (n_replicas < 1 || n_replicas > 65535) return sfail(PSG_EINVAL, "psg_range_rgyr_static: n_replicas must be in [1, 65535]");
    if (first_atom < 0 || n_group_atoms < 1 || first_atom > replica_stride_atoms ||
        n_group_atoms > replica_stride_atoms - first_atom)
        return sfail(PSG_EINVAL, "psg_range_rgyr_static: the range must lie inside [0, replica_stride_atoms)");
    const long long blocks = (n_group_atoms + PSG_STATIC_TILE - 1) / PSG_STATIC_TILE;
    if (blocks * n_replicas > PSG_STATIC_MAX_BLOCKS)
        return sfail(PSG_ECAPACITY, "psg_range_rgyr_static: n_replicas * ceil(n_group_atoms / " + std::to_string(PSG_STATIC_TILE) + ") = " +
                                        std::to_string(blocks * n_replicas) + " exceeds the static scratch array (PSG_STATIC_MAX_BLOCKS = " +
                                        std::to_string(PSG_STATIC_MAX_BLOCKS) + "); use psg_cv_eval on a context");
    DeviceRestore guard;
    cudaError_t e = cudaGetDevice(&guard.prev);
    if (e != cudaSuccess) {
        guard.prev = -1;
        return sfail(PSG_ECUDA, std::string("psg_range_rgyr_static: no usable CUDA device, and there is no CPU fallback: ") + cudaGetErrorString(e));
    }
    if ((e = cudaSetDevice(device)) != cudaSuccess)
        return sfail(PSG_ECUDA, std::string("psg_range_rgyr_static: cudaSetDevice: ") + cudaGetErrorString(e));
    double* scratch = nullptr;
    if (int rc = static_scratch(device, &scratch)) return rc;

    StaticRangeArgs A;
    A.pos = d_pos; A.weight = d_weight; A.rstride = replica_stride_atoms; A.first = first_atom; A.count = n_group_atoms;
    A.ps = pos_stride; A.blocks = (int)blocks; A.R = n_replicas;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    k_range_moments_static<<<dim3((unsigned)blocks, (unsigned)n_replicas), PSG_RANGE_THREADS, 0, st>>>(A, scratch);
    k_rgyr_static<<<(n_replicas + 7) / 8, 256, 0, st>>>(A, scratch, d_xi, d_center);
    if ((e = cudaGetLastError()) != cudaSuccess)
        return sfail(PSG_ECUDA, std::string("psg_range_rgyr_static: kernel launch: ") + cudaGetErrorString(e));
    return PSG_OK;
}
