// api.cu -- the C ABI of libpsg.so (include/psg.h): context, setup, argument validation, dispatch.
// Hot-path calls validate on the host, enqueue on the ctx stream, never synchronise.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <vector>

#include <nvtx3/nvToolsExt.h>

#include "internal.h"

static thread_local std::string g_create_err;

// NVTX range around a hot-path call: visible in Nsight Systems timelines, a few ns when no tool listens
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

#define CK(ctx, expr)                                                                  \
    do {                                                                               \
        cudaError_t e__ = (expr);                                                      \
        if (e__ != cudaSuccess) {                                                      \
            (ctx)->err = std::string(#expr) + ": " + cudaGetErrorString(e__);           \
            return e__ == cudaErrorMemoryAllocation ? PSG_ENOMEM : PSG_ECUDA;          \
        }                                                                              \
    } while (0)

static int fail(psg_ctx* c, int code, const char* msg) {
    if (c) c->err = msg;
    return code;
}

template <class T>
static void dfree(T*& p) {
    if (p) cudaFree(p);
    p = nullptr;
}

template <class T>
static cudaError_t dalloc(T*& p, size_t n) {
    dfree(p);
    if (n == 0) n = 1;
    return cudaMalloc((void**)&p, n * sizeof(T));
}

// Host-side admission of a deposit of up to n hills: the exact count lives on the device; the host keeps a
// lower and an upper bound (equal while no mask was used).  Refused, nothing launched, when overflow is CERTAIN (lower bound
// + the hills this call surely adds > capacity; exact for unmasked calls).  A masked call that might overflow is launched:
// the kernel clamps at capacity and raises the sticky flag psg_sync_check / psg_get_hills report.  After a deposit captured
// in a CUDA graph the host knows nothing (replays append behind its back): admission is left to the device clamp.
static int deposit_admit(psg_ctx* c, long long n, bool masked, const char* msg) {
    if (c->count_unknown) return PSG_OK;
    const long long sure = masked ? 0 : n;
    if (c->nh_lo + sure > c->md.capacity) {
        c->err = msg;
        return PSG_ECAPACITY;
    }
    return PSG_OK;
}
static void deposit_account(psg_ctx* c, long long n, bool masked) {
    const long long cap = c->md.capacity;
    if (c->nh_bound + n > cap || c->count_unknown) c->overflow_possible = true;   // launched although the host could not rule it out
    c->nh_bound = std::min(c->nh_bound + n, cap);
    if (!masked) c->nh_lo = std::min(c->nh_lo + n, cap);
    if (psg_stream_capturing(c)) { c->count_unknown = true; c->overflow_possible = true; }
}

static const int kGroups[12] = {0, 2, 3, 4, 1, 1, 2, 1, 1, 1, 1, 2};

extern "C" {

int psg_create(psg_ctx** out, int device, void* cuda_stream) {
    if (!out) { g_create_err = "psg_create: out is NULL"; return PSG_EINVAL; }
    *out = nullptr;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n == 0) {
        g_create_err = std::string("psg_create: no CUDA device (") + cudaGetErrorString(e) + "); there is no CPU fallback";
        return PSG_ECUDA;
    }
    if (device < 0 || device >= n) { g_create_err = "psg_create: device ordinal out of range"; return PSG_EINVAL; }
    if ((e = cudaSetDevice(device)) != cudaSuccess) { g_create_err = cudaGetErrorString(e); return PSG_ECUDA; }
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) { g_create_err = cudaGetErrorString(e); return PSG_ECUDA; }
    if (prop.major < 10) {
        g_create_err = "psg_create: kernels are built for sm_100a only; this device is older";
        return PSG_ECUDA;
    }
    psg_ctx* c = new (std::nothrow) psg_ctx();
    if (!c) { g_create_err = "psg_create: out of host memory"; return PSG_ENOMEM; }
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    c->sm_count = prop.multiProcessorCount;
    *out = c;
    return PSG_OK;
}

static void free_all(psg_ctx* c) {
    dfree(c->d_slot_atom); dfree(c->d_slot_gid); dfree(c->d_slot_weight); dfree(c->d_atom_weight);
    dfree(c->d_xi); dfree(c->d_V); dfree(c->d_dVdxi); dfree(c->d_bin); dfree(c->d_V64);
    dfree(c->d_jac); dfree(c->d_gdesc); dfree(c->d_rpart); dfree(c->d_rpart2); dfree(c->d_gdesc_m); dfree(c->d_arrive); dfree(c->d_rdesc); dfree(c->d_gbar); dfree(c->d_whist);
    dfree(c->d_kspring); dfree(c->d_centers);
    dfree(c->md.hills); dfree(c->md.heights); dfree(c->md.n_hills); dfree(c->md.part);
    if (c->abf.own) { dfree(c->abf.hist); dfree(c->abf.fsum); }
    c->abf.hist = nullptr; c->abf.fsum = nullptr;
    dfree(c->d_pos_stage); dfree(c->d_frc_stage); dfree(c->d_fs_stage);
    psg_interface_cv_free(c);
    psg_metad_grid_free(c);
}

int psg_destroy(psg_ctx* c) {
    if (!c) return PSG_EINVAL;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    free_all(c);
    delete c;
    return PSG_OK;
}

int psg_set_tuning(psg_ctx* c, int range_step_lag, int disable_range_step) {
    if (!c) return PSG_EINVAL;
    if (range_step_lag < 0 || range_step_lag > 1024) return fail(c, PSG_EINVAL, "psg_set_tuning: 0 <= range_step_lag <= 1024");
    c->range_lag = range_step_lag > 0 ? range_step_lag : 10;
    c->range_step_off = disable_range_step != 0;
    return PSG_OK;
}

int psg_set_stream(psg_ctx* c, void* s) {
    if (!c) return PSG_EINVAL;
    c->stream = (cudaStream_t)s;
    return PSG_OK;
}

const char* psg_last_error(const psg_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

long long psg_launch_count(const psg_ctx* c) { return c ? c->launches : 0; }

int psg_set_layout(psg_ctx* c, int R, long long N, long long rstride, int ps, int fs) {
    if (!c) return PSG_EINVAL;
    if (R <= 0 || N <= 0) return fail(c, PSG_EINVAL, "psg_set_layout: n_replicas and n_atoms must be > 0");
    if (R > 65535) return fail(c, PSG_EINVAL, "psg_set_layout: at most 65535 replicas per ctx");
    if ((ps != 3 && ps != 4) || (fs != 3 && fs != 4)) return fail(c, PSG_EINVAL, "psg_set_layout: strides must be 3 or 4 floats");
    if (rstride != 0 && rstride < N) return fail(c, PSG_EINVAL, "psg_set_layout: replica_stride_atoms must be 0 or >= n_atoms");
    cudaSetDevice(c->device);
    SysParams& P = c->sys;
    memset(&P, 0, sizeof(P));
    P.R = R; P.N = N; P.rstride = rstride; P.ps = ps; P.fs = fs;
    c->have_layout = true; c->have_cvs = false; c->have_jac = false; c->method = PSG_METHOD_NONE;
    // state sized by the old layout must not survive it: the grid-stored bias and the interface CV hold R, strides and
    // per-replica buffers (their *_set calls come after psg_set_layout); the host-engine staging buffers are re-sized on demand
    psg_interface_cv_free(c);
    c->dti_cv = -1;
    psg_metad_grid_free(c);
    return PSG_OK;
}

int psg_set_cvs(psg_ctx* c, int n_cv, const psg_cv_desc* cvs, int n_slots, const int* slot_atom, int per_rep,
                const float* slot_weight, const float* atom_weight) {
    if (!c) return PSG_EINVAL;
    if (!c->have_layout) return fail(c, PSG_ESTATE, "psg_set_cvs: call psg_set_layout first");
    if (n_cv < 1 || n_cv > PSG_MAX_CV || !cvs) return fail(c, PSG_EINVAL, "psg_set_cvs: 1 <= n_cv <= PSG_MAX_CV");
    if (n_slots < 0 || n_slots > PSG_MAX_SLOTS) return fail(c, PSG_EINVAL, "psg_set_cvs: 0 <= n_slots <= PSG_MAX_SLOTS");
    if (n_slots > 0 && !slot_atom) return fail(c, PSG_EINVAL, "psg_set_cvs: slot_atom_idx is NULL");
    cudaSetDevice(c->device);
    SysParams P = c->sys;
    P.n_cv = n_cv; P.n_slots = n_slots; P.per_rep = per_rep ? 1 : 0;
    P.n_groups = 0; P.n_ranges = 0; P.any_rgyr = 0; P.any_shape_range = 0;
    P.has_box = 0; P.box[0] = P.box[1] = P.box[2] = 0.0;   // psg_set_box comes after psg_set_cvs
    P.span_begin = P.N; P.span_end = 0;
    std::vector<int> slot_gid(n_slots > 0 ? n_slots : 1, -1);
    int dti_k = -1;
    for (int k = 0; k < n_cv; ++k) {
        const psg_cv_desc& d = cvs[k];
        if (d.type < PSG_CV_DISTANCE || d.type > PSG_CV_DIST_TO_INTERFACE) return fail(c, PSG_EINVAL, "psg_set_cvs: unknown CV type");
        if (d.n_groups != kGroups[d.type]) return fail(c, PSG_EINVAL, "psg_set_cvs: wrong n_groups for this CV type");
        if ((d.type == PSG_CV_COM_COMPONENT || d.type == PSG_CV_DISPLACEMENT || d.type == PSG_CV_PRINCIPAL_MOMENT || d.type == PSG_CV_DIST_TO_INTERFACE) &&
            (d.axis < 0 || d.axis > 2))
            return fail(c, PSG_EINVAL, "psg_set_cvs: axis must be 0, 1 or 2");
        const bool shape = d.type >= PSG_CV_PRINCIPAL_MOMENT && d.type <= PSG_CV_SHAPE_ANISOTROPY;
        if (!(d.period >= 0.0)) return fail(c, PSG_EINVAL, "psg_set_cvs: period must be >= 0");
        CvDev& C = P.cv[k];
        C.type = d.type; C.n_groups = d.n_groups; C.axis = d.axis; C.period = d.period; C.gid0 = P.n_groups;
        if (d.type == PSG_CV_RGYR || shape) P.any_rgyr = 1;   // per-atom Jacobian depends on r_i - c: the generic kernels
        if (shape && d.group_is_range[0]) P.any_shape_range = 1;
        const bool is_dti = d.type == PSG_CV_DIST_TO_INTERFACE;
        if (is_dti) {
            if (dti_k >= 0) return fail(c, PSG_EINVAL, "psg_set_cvs: at most one DistanceToInterface CV per ctx");
            if (per_rep) return fail(c, PSG_EINVAL, "psg_set_cvs: DistanceToInterface needs a shared index list");
            if (d.group_is_range[0] || !d.group_is_range[1])
                return fail(c, PSG_EINVAL, "psg_set_cvs: DistanceToInterface takes explicit mobile atoms (group 0) and a contiguous interface range (group 1)");
            dti_k = k;
            P.any_rgyr = 1;   // (keeps every fused one-launch step off: this CV has kernels of its own)
        }
        for (int g = 0; g < d.n_groups; ++g) {
            GroupDev& G = P.grp[P.n_groups];
            memset(&G, 0, sizeof(G));
            G.cv = k; G.g = g; G.range_id = -1;
            if (d.group_is_range[g] && is_dti) {
                // the interface atoms: a range that only interface_cv.cu walks (not in the table of the moment kernels)
                if (d.range_size[g] <= 0 || d.range_begin[g] < 0 || d.range_begin[g] + d.range_size[g] > P.N)
                    return fail(c, PSG_EINVAL, "psg_set_cvs: atom range outside [0, n_atoms)");
                G.is_range = 1; G.rbegin = d.range_begin[g]; G.rsize = d.range_size[g];
            } else if (d.group_is_range[g]) {
                if (P.n_ranges >= PSG_MAX_RANGE_GROUPS) return fail(c, PSG_EINVAL, "psg_set_cvs: too many range groups");
                if (d.range_size[g] <= 0 || d.range_begin[g] < 0 || d.range_begin[g] + d.range_size[g] > P.N)
                    return fail(c, PSG_EINVAL, "psg_set_cvs: atom range outside [0, n_atoms)");
                G.is_range = 1; G.rbegin = d.range_begin[g]; G.rsize = d.range_size[g]; G.range_id = P.n_ranges;
                P.range_gid[P.n_ranges++] = P.n_groups;
                if (G.rbegin < P.span_begin) P.span_begin = G.rbegin;
                if (G.rbegin + G.rsize > P.span_end) P.span_end = G.rbegin + G.rsize;
            } else {
                if (d.group_size[g] <= 0 || d.group_begin[g] < 0 || d.group_begin[g] + d.group_size[g] > n_slots)
                    return fail(c, PSG_EINVAL, "psg_set_cvs: group slice outside the slot list");
                G.begin = d.group_begin[g]; G.size = d.group_size[g];
                for (int s = G.begin; s < G.begin + G.size; ++s) {
                    if (slot_gid[s] != -1) return fail(c, PSG_EINVAL, "psg_set_cvs: a slot belongs to two groups");
                    slot_gid[s] = P.n_groups;
                }
            }
            P.n_groups++;
        }
    }
    for (int s = 0; s < n_slots; ++s)
        if (slot_gid[s] < 0) return fail(c, PSG_EINVAL, "psg_set_cvs: a slot belongs to no group");
    size_t n_idx = (size_t)n_slots * (per_rep ? P.R : 1);
    for (size_t i = 0; i < n_idx; ++i)
        if (slot_atom[i] < 0 || slot_atom[i] >= P.N) return fail(c, PSG_EINVAL, "psg_set_cvs: atom index out of range");
    if (slot_weight)
        for (int s = 0; s < n_slots; ++s)
            if (!(slot_weight[s] > 0.f)) return fail(c, PSG_EINVAL, "psg_set_cvs: weights must be > 0");
    if (P.n_ranges > 0) {
        P.range_blocks = (int)((P.span_end - P.span_begin + PSG_RANGE_TILE - 1) / PSG_RANGE_TILE);
    } else {
        P.span_begin = P.span_end = 0; P.range_blocks = 0;
    }
    // device copies
    CK(c, dalloc(c->d_slot_atom, n_idx));
    CK(c, dalloc(c->d_slot_gid, (size_t)n_slots));
    if (n_idx) CK(c, cudaMemcpy(c->d_slot_atom, slot_atom, n_idx * sizeof(int), cudaMemcpyHostToDevice));
    if (n_slots) CK(c, cudaMemcpy(c->d_slot_gid, slot_gid.data(), n_slots * sizeof(int), cudaMemcpyHostToDevice));
    dfree(c->d_slot_weight); dfree(c->d_atom_weight);
    if (slot_weight && n_slots) {
        CK(c, dalloc(c->d_slot_weight, (size_t)n_slots));
        CK(c, cudaMemcpy(c->d_slot_weight, slot_weight, n_slots * sizeof(float), cudaMemcpyHostToDevice));
    }
    if (atom_weight && P.n_ranges) {
        CK(c, dalloc(c->d_atom_weight, (size_t)P.N));
        CK(c, cudaMemcpy(c->d_atom_weight, atom_weight, (size_t)P.N * sizeof(float), cudaMemcpyHostToDevice));
    }
    for (int i = 0; i < PSG_MAX_SLOTS; ++i) P.slot_atom_c[i] = (!per_rep && i < n_slots) ? slot_atom[i] : 0;
    for (int i = 0; i < PSG_MAX_SLOTS; ++i) P.slot_gid_c[i] = (unsigned char)(i < n_slots ? slot_gid[i] : 0);
    P.simple_groups = (P.n_ranges == 0 && !P.any_rgyr) ? 1 : 0;
    for (int k = 0; k < PSG_MAX_CV; ++k)
        for (int g = 0; g < PSG_MAX_GROUPS; ++g) {
            int slot = 0;
            if (k < n_cv) {
                const GroupDev& G = P.grp[P.cv[k].gid0 + (g < P.cv[k].n_groups ? g : 0)];
                if (G.is_range || G.size != 1) P.simple_groups = 0;
                else slot = G.begin;
            }
            P.cv_slot[k * PSG_MAX_GROUPS + g] = slot;
            P.cv_atom[k * PSG_MAX_GROUPS + g] = (!per_rep && n_slots > 0) ? slot_atom[slot] : 0;
        }
    P.slot_atom = c->d_slot_atom; P.slot_gid = c->d_slot_gid; P.slot_weight = c->d_slot_weight; P.atom_weight = c->d_atom_weight;
    // scratch
    size_t R = (size_t)P.R;
    CK(c, dalloc(c->d_xi, R * n_cv)); CK(c, dalloc(c->d_V, R)); CK(c, dalloc(c->d_dVdxi, R * n_cv));
    CK(c, dalloc(c->d_bin, R)); CK(c, dalloc(c->d_V64, R));
    CK(c, dalloc(c->d_jac, R * (size_t)n_slots * 3));
    CK(c, dalloc(c->d_gdesc, R * P.n_groups * PSG_GDESC_DOUBLES));
    CK(c, dalloc(c->d_rpart, R * P.n_ranges * (size_t)P.range_blocks * PSG_MOM));
    CK(c, dalloc(c->d_rpart2, P.any_shape_range ? R * P.n_ranges * (size_t)P.range_blocks * 6 : 0));
    CK(c, dalloc(c->d_gdesc_m, P.any_shape_range ? R * P.n_groups * 6 : 0));
    CK(c, dalloc(c->d_arrive, 2 * R));
    CK(c, cudaMemset(c->d_arrive, 0, 2 * R * sizeof(unsigned)));
    CK(c, dalloc(c->d_whist, R * 2 * n_cv));
    CK(c, cudaMemset(c->d_whist, 0, R * 2 * n_cv * sizeof(double)));
    c->est_first = true;
    CK(c, dalloc(c->d_gbar, 2));
    CK(c, cudaMemset(c->d_gbar, 0, 2 * sizeof(unsigned)));
    CK(c, dalloc(c->d_rdesc, R * P.n_ranges * 4));
    CK(c, cudaMemset(c->d_rdesc, 0, std::max<size_t>(R * P.n_ranges * 4, 1) * sizeof(float4)));
    CK(c, cudaMemset(c->d_V, 0, R * sizeof(float)));
    CK(c, cudaMemset(c->d_bin, 0xff, R * sizeof(int)));
    c->sys = P;
    c->have_cvs = true; c->have_jac = false; c->method = PSG_METHOD_NONE;
    c->dti_cv = -1;
    if (dti_k >= 0) {
        // DistanceToInterface as a CV of the path: the same state psg_interface_cv_set builds, from the descriptor
        const psg_cv_desc& d = cvs[dti_k];
        const GroupDev& G0 = P.grp[P.cv[dti_k].gid0];
        int rc = psg_interface_cv_set(c, G0.size, slot_atom + G0.begin, slot_weight ? slot_weight + G0.begin : nullptr, d.range_begin[1],
                                      d.range_size[1], d.axis, d.dti_sigma, d.dti_scope[0], d.dti_scope[1], d.dti_bins, d.dti_coeff);
        if (rc != PSG_OK) { c->have_cvs = false; return rc; }
        c->dti_cv = dti_k;
    }
    return PSG_OK;
}

int psg_set_box(psg_ctx* c, const double* box) {
    if (!c) return PSG_EINVAL;
    if (!c->have_cvs) return fail(c, PSG_ESTATE, "psg_set_box: call psg_set_cvs first");
    bool on = false;
    if (box)
        for (int x = 0; x < 3; ++x) {
            if (!(box[x] >= 0.0)) return fail(c, PSG_EINVAL, "psg_set_box: box lengths must be >= 0");
            on |= box[x] > 0.0;
        }
    c->sys.has_box = on ? 1 : 0;
    for (int x = 0; x < 3; ++x) c->sys.box[x] = on ? box[x] : 0.0;
    c->have_jac = false;
    return PSG_OK;
}

int psg_set_harmonic(psg_ctx* c, const float* kspring, const float* centers) {
    if (!c) return PSG_EINVAL;
    if (!c->have_cvs) return fail(c, PSG_ESTATE, "psg_set_harmonic: call psg_set_cvs first");
    if (!kspring || !centers) return fail(c, PSG_EINVAL, "psg_set_harmonic: NULL argument");
    cudaSetDevice(c->device);
    int n_cv = c->sys.n_cv;
    size_t R = (size_t)c->sys.R;
    CK(c, dalloc(c->d_kspring, (size_t)n_cv));
    CK(c, dalloc(c->d_centers, R * n_cv));
    CK(c, cudaMemcpy(c->d_kspring, kspring, n_cv * sizeof(float), cudaMemcpyHostToDevice));
    CK(c, cudaMemcpy(c->d_centers, centers, R * n_cv * sizeof(float), cudaMemcpyHostToDevice));
    c->method = PSG_METHOD_HARMONIC;
    return PSG_OK;
}

int psg_set_metad(psg_ctx* c, const float* sigma, float w0, float kB_deltaT, int capacity, int stride) {
    if (!c) return PSG_EINVAL;
    if (!c->have_cvs) return fail(c, PSG_ESTATE, "psg_set_metad: call psg_set_cvs first");
    if (!sigma || capacity < 0 || stride < 0) return fail(c, PSG_EINVAL, "psg_set_metad: bad argument");
    cudaSetDevice(c->device);
    MetadState& M = c->md;
    int n_cv = c->sys.n_cv;
    HillConsts hc;
    memset(&hc, 0, sizeof(hc));
    hc.n_cv = n_cv;
    const double log2e = 1.4426950408889634074;
    for (int k = 0; k < n_cv; ++k) {
        if (!(sigma[k] > 0.f)) return fail(c, PSG_EINVAL, "psg_set_metad: sigma must be > 0");
        double sg = (double)sigma[k], per = c->sys.cv[k].period;
        hc.nc[k] = (float)(-log2e / (2.0 * sg * sg));
        hc.gscale[k] = 1.0 / (sg * sg);
        hc.inv_sigma_d[k] = 1.0 / sg;
        hc.period_d[k] = per > 0 ? per : 1e300;   // non-periodic: rint(d / 1e300) = 0, no wrap
        if (per > 0) {
            hc.pmask |= 1 << k;
            hc.inv_period[k] = (float)(1.0 / per);
            // -P = np_hi + np_lo; |k| <= 1 for CV values inside one period, so k * np_hi is exact
            hc.np_hi[k] = (float)(-per);
            hc.np_lo[k] = (float)(-per - (double)hc.np_hi[k]);
        }
    }
    hc.neq = 1;
    while (hc.neq < n_cv && hc.nc[hc.neq] == hc.nc[0]) hc.neq++;
    M.hc = hc;
    M.w0 = (double)w0; M.kB_deltaT = (double)kB_deltaT; M.capacity = capacity; M.stride = stride;
    M.rec = n_cv <= 3 ? 1 : 2;
    M.precision = PSG_HILLS_F32;
    int n_rt = 0;
    size_t part = psg_hill_part_doubles(c, &M.max_chunks, &n_rt);
    CK(c, dalloc(M.hills, (size_t)capacity * M.rec + 2));
    CK(c, dalloc(M.heights, (size_t)capacity + 2));
    CK(c, dalloc(M.n_hills, 2));
    CK(c, dalloc(M.part, part));
    CK(c, cudaMemset(M.n_hills, 0, 2 * sizeof(int)));
    CK(c, cudaMemset(M.part, 0, part * sizeof(double)));   // a cleared word = "not published yet" (hills.cuh)
    CK(c, psg_launch_null_hills(c, 0, capacity));   // invariant: records beyond the count are null (contribute 0)
    c->nh_bound = c->nh_lo = 0; c->count_unknown = false; c->overflow_possible = false;
    c->method = PSG_METHOD_METAD;
    return PSG_OK;
}

int psg_set_hill_precision(psg_ctx* c, int mode) {
    if (!c) return PSG_EINVAL;
    if (c->method != PSG_METHOD_METAD) return fail(c, PSG_ESTATE, "psg_set_hill_precision: metadynamics is not selected");
    if (mode != PSG_HILLS_F32 && mode != PSG_HILLS_F64) return fail(c, PSG_EINVAL, "psg_set_hill_precision: unknown mode");
    c->md.precision = mode;
    return PSG_OK;
}

int psg_load_hills(psg_ctx* c, int n, const float* d_centers, const float* d_heights) {
    if (!c) return PSG_EINVAL;
    if (c->method != PSG_METHOD_METAD) return fail(c, PSG_ESTATE, "psg_load_hills: metadynamics is not selected");
    if (n < 0 || (n > 0 && (!d_centers || !d_heights))) return fail(c, PSG_EINVAL, "psg_load_hills: bad argument");
    if (n > c->md.capacity) return fail(c, PSG_ECAPACITY, "psg_load_hills: more hills than capacity");
    cudaSetDevice(c->device);
    CK(c, psg_launch_pack_hills(c, n, d_centers, d_heights));
    const long long old_bound = c->count_unknown ? c->md.capacity : c->nh_bound;
    if (old_bound > n) CK(c, psg_launch_null_hills(c, n, (int)old_bound));
    const int cnt[2] = {n, 0};                  // exact count, overflow flag cleared
    CK(c, cudaMemcpyAsync(c->md.n_hills, cnt, 2 * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));   // cnt is a stack variable
    c->nh_bound = c->nh_lo = n; c->count_unknown = false; c->overflow_possible = false;
    return PSG_OK;
}

int psg_get_hills(psg_ctx* c, int* n_out, float* d_centers, float* d_heights, int max_n) {
    if (!c) return PSG_EINVAL;
    if (c->method != PSG_METHOD_METAD) return fail(c, PSG_ESTATE, "psg_get_hills: metadynamics is not selected");
    cudaSetDevice(c->device);
    int cnt[2] = {0, 0};
    CK(c, cudaMemcpyAsync(cnt, c->md.n_hills, 2 * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    const int n = cnt[0];
    if (n_out) *n_out = n;
    c->nh_bound = c->nh_lo = n; c->count_unknown = false;   // exact now
    if (cnt[1]) return fail(c, PSG_ECAPACITY, "psg_get_hills: an earlier deposit overflowed the hill store; hills were dropped");
    if (d_centers && d_heights) {
        if (max_n < n) return fail(c, PSG_ECAPACITY, "psg_get_hills: output arrays too small");
        CK(c, psg_launch_unpack_hills(c, n, d_centers, d_heights));
        CK(c, cudaStreamSynchronize(c->stream));
    }
    return PSG_OK;
}

int psg_set_abf(psg_ctx* c, const float* lower, const float* upper, const int* shape, const int* periodic, int n_threshold,
                int* d_hist, float* d_fsum) {
    if (!c) return PSG_EINVAL;
    if (!c->have_cvs) return fail(c, PSG_ESTATE, "psg_set_abf: call psg_set_cvs first");
    if (!lower || !upper || !shape || !periodic || n_threshold < 1) return fail(c, PSG_EINVAL, "psg_set_abf: bad argument");
    if ((d_hist == nullptr) != (d_fsum == nullptr)) return fail(c, PSG_EINVAL, "psg_set_abf: give both d_hist and d_fsum or neither");
    cudaSetDevice(c->device);
    AbfState& G = c->abf;
    if (G.own) { dfree(G.hist); dfree(G.fsum); }
    memset(&G, 0, sizeof(G));
    int n_cv = c->sys.n_cv;
    long long nb = 1;
    for (int k = 0; k < n_cv; ++k) {
        if (shape[k] < 1 || !(upper[k] > lower[k])) return fail(c, PSG_EINVAL, "psg_set_abf: need shape >= 1 and upper > lower");
        G.lower[k] = lower[k];
        G.invd[k] = (float)((double)shape[k] / ((double)upper[k] - (double)lower[k]));
        G.shape[k] = shape[k];
        G.periodic[k] = periodic[k] ? 1 : 0;
        nb *= shape[k];
        if (nb > 0x7fffffffLL) return fail(c, PSG_EINVAL, "psg_set_abf: grid has more than 2^31 bins");
    }
    G.n_bins = nb; G.n_threshold = n_threshold;
    if (d_hist) {
        G.hist = d_hist; G.fsum = d_fsum; G.own = false;
    } else {
        G.own = true;
        CK(c, dalloc(G.hist, (size_t)nb));
        CK(c, dalloc(G.fsum, (size_t)nb * n_cv));
        CK(c, cudaMemset(G.hist, 0, nb * sizeof(int)));
        CK(c, cudaMemset(G.fsum, 0, nb * n_cv * sizeof(float)));
    }
    c->method = PSG_METHOD_ABF;
    c->abf_delta_pending = false;
    return PSG_OK;
}

int psg_abf_state(psg_ctx* c, int** h, float** f, long long* nb) {
    if (!c) return PSG_EINVAL;
    if (c->method != PSG_METHOD_ABF) return fail(c, PSG_ESTATE, "psg_abf_state: ABF is not selected");
    if (h) *h = c->abf.hist;
    if (f) *f = c->abf.fsum;
    if (nb) *nb = c->abf.n_bins;
    return PSG_OK;
}

// ---------------------------------------------------------------------------- hot path
int psg_cv_eval(psg_ctx* c, const float* d_pos, float* d_xi, float* d_jac) {
    if (!c) return PSG_EINVAL;
    NvtxRange nvtx_("psg_cv_eval");
    if (!c->have_cvs) return fail(c, PSG_ESTATE, "psg_cv_eval: no CVs configured");
    if (!d_pos || !d_xi) return fail(c, PSG_EINVAL, "psg_cv_eval: NULL pointer");
    CK(c, psg_launch_cv_eval(c, d_pos, d_xi, d_jac));
    c->have_jac = true;
    return PSG_OK;
}

int psg_bias_eval(psg_ctx* c, const float* d_xi, float* d_V, float* d_dVdxi) {
    if (!c) return PSG_EINVAL;
    NvtxRange nvtx_("psg_bias_eval");
    if (!d_xi || !d_dVdxi) return fail(c, PSG_EINVAL, "psg_bias_eval: NULL pointer");
    if (c->method == PSG_METHOD_HARMONIC) CK(c, psg_launch_harmonic(c, d_xi, d_V, d_dVdxi));
    else if (c->method == PSG_METHOD_METAD) CK(c, psg_launch_hillsum(c, d_xi, d_V, d_dVdxi));
    else if (c->method == PSG_METHOD_METAD_GRID) return psg_metad_grid_eval(c, d_xi, d_V, d_dVdxi);
    else return fail(c, PSG_ESTATE, "psg_bias_eval: select harmonic or metadynamics first (ABF uses psg_abf_update)");
    return PSG_OK;
}

int psg_deposit_hill(psg_ctx* c, const float* d_xi, const unsigned char* d_mask) {
    if (!c) return PSG_EINVAL;
    NvtxRange nvtx_("psg_deposit_hill");
    if (c->method == PSG_METHOD_METAD_GRID) return psg_metad_grid_deposit(c, d_xi, d_mask);
    if (c->method != PSG_METHOD_METAD) return fail(c, PSG_ESTATE, "psg_deposit_hill: metadynamics is not selected");
    if (!d_xi) return fail(c, PSG_EINVAL, "psg_deposit_hill: NULL pointer");
    int rc = deposit_admit(c, c->sys.R, d_mask != nullptr, "psg_deposit_hill: hill store would overflow (count + R > capacity); nothing launched");
    if (rc != PSG_OK) return rc;
    CK(c, psg_launch_deposit(c, d_xi, d_mask));
    deposit_account(c, c->sys.R, d_mask != nullptr);
    return PSG_OK;
}

int psg_abf_update(psg_ctx* c, const float* d_xi, const float* d_fsample, int* d_bin, float* d_dVdxi) {
    if (!c) return PSG_EINVAL;
    NvtxRange nvtx_("psg_abf_update");
    if (c->method != PSG_METHOD_ABF) return fail(c, PSG_ESTATE, "psg_abf_update: ABF is not selected");
    if (!d_xi || !d_fsample || !d_dVdxi) return fail(c, PSG_EINVAL, "psg_abf_update: NULL pointer");
    CK(c, psg_launch_abf(c, d_xi, d_fsample, d_bin, d_dVdxi));
    return PSG_OK;
}

// Shared-grid ABF with the replicas spread over several GPUs: phase 1 into per-step delta arrays ...
int psg_abf_accumulate_delta(psg_ctx* c, const float* d_pos, const float* d_fsample, int* d_hist_delta, float* d_fsum_delta) {
    if (!c) return PSG_EINVAL;
    if (c->method != PSG_METHOD_ABF) return fail(c, PSG_ESTATE, "psg_abf_accumulate_delta: ABF is not selected");
    if (!d_pos || !d_fsample || !d_hist_delta || !d_fsum_delta) return fail(c, PSG_EINVAL, "psg_abf_accumulate_delta: NULL pointer");
    const size_t nb = (size_t)c->abf.n_bins;
    CK(c, cudaMemsetAsync(d_hist_delta, 0, nb * sizeof(int), c->stream));
    CK(c, cudaMemsetAsync(d_fsum_delta, 0, nb * c->sys.n_cv * sizeof(float), c->stream));
    if (psg_abf_step_supported(c)) {
        CK(c, psg_launch_abf_phase(c, 1, d_pos, d_fsample, nullptr, d_hist_delta, d_fsum_delta));
    } else {
        CK(c, psg_launch_cv_eval(c, d_pos, c->d_xi, nullptr));
        CK(c, psg_launch_abf_accumulate(c, c->d_xi, d_fsample, d_hist_delta, d_fsum_delta));
    }
    c->have_jac = true;
    c->abf_delta_pending = true;
    return PSG_OK;
}

// ... and, after the all-reduce over ranks, grid += delta and phase 2 (mean force from the updated grid, force scatter)
int psg_abf_apply_grid_delta(psg_ctx* c, const int* d_hist_delta, const float* d_fsum_delta, const float* d_pos, float* d_force) {
    if (!c) return PSG_EINVAL;
    if (c->method != PSG_METHOD_ABF) return fail(c, PSG_ESTATE, "psg_abf_apply_grid_delta: ABF is not selected");
    if (!d_hist_delta || !d_fsum_delta || !d_pos || !d_force) return fail(c, PSG_EINVAL, "psg_abf_apply_grid_delta: NULL pointer");
    if (!c->abf_delta_pending)
        return fail(c, PSG_ESTATE, "psg_abf_apply_grid_delta: no pending psg_abf_accumulate_delta on this ctx");
    CK(c, psg_launch_abf_add_delta(c, d_hist_delta, d_fsum_delta));
    if (psg_abf_step_supported(c)) {
        CK(c, psg_launch_abf_phase(c, 2, d_pos, nullptr, d_force, c->abf.hist, c->abf.fsum));
    } else {
        CK(c, psg_launch_abf_mean(c, nullptr, c->d_dVdxi));
        CK(c, psg_launch_apply(c, d_pos, c->d_dVdxi, d_force));
    }
    c->abf_delta_pending = false;
    return PSG_OK;
}

int psg_abf_estimate(psg_ctx* c, const float* d_pos, const float* d_vel, const float* d_mass, double dt, const float* d_fbias_prev,
                     float* d_fsample) {
    if (!c) return PSG_EINVAL;
    if (!c->have_cvs) return fail(c, PSG_ESTATE, "psg_abf_estimate: no CVs configured");
    if (!d_pos || !d_vel || !d_mass || !d_fsample) return fail(c, PSG_EINVAL, "psg_abf_estimate: NULL pointer");
    if (!(dt > 0.0)) return fail(c, PSG_EINVAL, "psg_abf_estimate: dt must be > 0");
    if (c->sys.n_ranges > 0 || c->dti_cv >= 0) return fail(c, PSG_EINVAL, "psg_abf_estimate: explicit groups only (this ctx has range groups)");
    CK(c, psg_launch_abf_estimate(c, d_pos, d_vel, d_mass, dt, d_fbias_prev, d_fsample));
    return PSG_OK;
}

int psg_abf_estimate_reset(psg_ctx* c) {
    if (!c) return PSG_EINVAL;
    c->est_first = true;
    return PSG_OK;
}

int psg_hill_heights(psg_ctx* c, const float* d_xi, const unsigned char* d_mask, float* d_heights) {
    if (!c) return PSG_EINVAL;
    if (c->method != PSG_METHOD_METAD) return fail(c, PSG_ESTATE, "psg_hill_heights: metadynamics is not selected");
    if (!d_xi || !d_heights) return fail(c, PSG_EINVAL, "psg_hill_heights: NULL pointer");
    CK(c, psg_launch_hill_heights(c, d_xi, d_mask, d_heights));
    return PSG_OK;
}

int psg_append_hills(psg_ctx* c, int n, const float* d_centers, const float* d_heights) {
    if (!c) return PSG_EINVAL;
    if (c->method != PSG_METHOD_METAD) return fail(c, PSG_ESTATE, "psg_append_hills: metadynamics is not selected");
    if (n < 0 || (n > 0 && (!d_centers || !d_heights))) return fail(c, PSG_EINVAL, "psg_append_hills: n >= 0 and no NULL pointer");
    // (zero heights are skipped on the device: like a masked deposit, the host only knows bounds)
    int rc = deposit_admit(c, n, true, "psg_append_hills: hill store would overflow (count + n > capacity); nothing launched");
    if (rc != PSG_OK) return rc;
    if (n > 0) CK(c, psg_launch_append_hills(c, n, d_centers, d_heights));
    deposit_account(c, n, true);
    return PSG_OK;
}

int psg_apply_bias_forces(psg_ctx* c, const float* d_pos, const float* d_dVdxi, float* d_force) {
    if (!c) return PSG_EINVAL;
    NvtxRange nvtx_("psg_apply_bias_forces");
    if (!c->have_jac) return fail(c, PSG_ESTATE, "psg_apply_bias_forces: no cached Jacobian; call psg_cv_eval on these positions first");
    if (!d_pos || !d_dVdxi || !d_force) return fail(c, PSG_EINVAL, "psg_apply_bias_forces: NULL pointer");
    CK(c, psg_launch_apply(c, d_pos, d_dVdxi, d_force));
    return PSG_OK;
}

int psg_step(psg_ctx* c, const float* d_pos, float* d_force, const float* d_fsample, long long step) {
    if (!c) return PSG_EINVAL;
    NvtxRange nvtx_("psg_step");
    if (!c->have_cvs || c->method == PSG_METHOD_NONE) return fail(c, PSG_ESTATE, "psg_step: configure CVs and a method first");
    if (!d_pos || !d_force) return fail(c, PSG_EINVAL, "psg_step: NULL pointer");
    if (c->method == PSG_METHOD_ABF && !d_fsample) return fail(c, PSG_EINVAL, "psg_step: ABF needs d_fsample");
    if (c->method == PSG_METHOD_METAD) {
        const MetadState& M = c->md;
        if (M.stride > 0 && step > 0 && step % M.stride == 0) {
            // xi -> deposit (heights from the OLD list) -> bias with the NEW list
            int rc = deposit_admit(c, c->sys.R, false, "psg_step: hill store would overflow; nothing launched");
            if (rc != PSG_OK) return rc;
            CK(c, psg_launch_cv_eval(c, d_pos, c->d_xi, nullptr));
            CK(c, psg_launch_deposit(c, c->d_xi, nullptr));
            deposit_account(c, c->sys.R, false);
        }
        if (psg_metad_step_supported(c)) {
            CK(c, psg_launch_metad_step(c, d_pos, d_force));
            c->have_jac = false;
            return PSG_OK;
        }
        CK(c, psg_launch_cv_eval(c, d_pos, c->d_xi, nullptr));
        CK(c, psg_launch_hillsum(c, c->d_xi, c->d_V, c->d_dVdxi));
    } else if (c->method == PSG_METHOD_METAD_GRID) {
        // xi -> deposit onto the grid (heights from the grid BEFORE the event) -> interpolated bias of the new grid -> forces
        if (c->mgrid_stride > 0 && step > 0 && step % c->mgrid_stride == 0) {
            CK(c, psg_launch_cv_eval(c, d_pos, c->d_xi, nullptr));
            int rc = psg_metad_grid_deposit(c, c->d_xi, nullptr);
            if (rc != PSG_OK) return rc;
        }
        c->have_jac = false;
        return psg_metad_grid_step(c, d_pos, d_force);
    } else if (c->method == PSG_METHOD_HARMONIC) {
        if (psg_range_step_supported(c, d_pos, d_force)) {
            CK(c, psg_launch_range_step(c, d_pos, d_force));   // large contiguous groups: one persistent launch
            c->have_jac = false;
            return PSG_OK;
        }
        CK(c, psg_launch_cv_eval(c, d_pos, c->d_xi, nullptr));
        CK(c, psg_launch_harmonic(c, c->d_xi, c->d_V, c->d_dVdxi));
    } else {
        if (psg_abf_step_supported(c)) {
            CK(c, psg_launch_abf_step(c, d_pos, d_fsample, d_force));   // one launch: CVs, grid update, barrier, forces
            c->have_jac = true;
            return PSG_OK;
        }
        CK(c, psg_launch_cv_eval(c, d_pos, c->d_xi, nullptr));
        CK(c, psg_launch_abf(c, c->d_xi, d_fsample, nullptr, c->d_dVdxi));
    }
    c->have_jac = true;
    CK(c, psg_launch_apply(c, d_pos, c->d_dVdxi, d_force));
    return PSG_OK;
}

int psg_step_outputs(psg_ctx* c, float** xi, float** V, float** dV, int** bin) {
    if (!c) return PSG_EINVAL;
    if (!c->have_cvs) return fail(c, PSG_ESTATE, "psg_step_outputs: no CVs configured");
    if (xi) *xi = c->d_xi;
    if (V) *V = c->d_V;
    if (dV) *dV = c->d_dVdxi;
    if (bin) *bin = c->method == PSG_METHOD_ABF ? c->d_bin : nullptr;
    return PSG_OK;
}

int psg_step_host(psg_ctx* c, const float* h_pos, float* h_force, const float* h_fsample, long long step) {
    if (!c) return PSG_EINVAL;
    NvtxRange nvtx_("psg_step_host");
    if (!c->have_cvs || c->method == PSG_METHOD_NONE) return fail(c, PSG_ESTATE, "psg_step_host: configure CVs and a method first");
    if (!h_pos || !h_force) return fail(c, PSG_EINVAL, "psg_step_host: NULL pointer");
    if (c->method == PSG_METHOD_ABF && !h_fsample) return fail(c, PSG_EINVAL, "psg_step_host: ABF needs h_fsample");
    cudaSetDevice(c->device);
    const SysParams& P = c->sys;
    size_t n_arr = P.rstride == 0 ? 1 : (size_t)P.R;
    size_t atoms = P.rstride == 0 ? (size_t)P.N : (size_t)(P.R - 1) * P.rstride + P.N;
    (void)n_arr;
    size_t pb = atoms * P.ps * sizeof(float), fb = atoms * P.fs * sizeof(float);
    if (c->n_pos_stage < atoms * P.ps) { CK(c, dalloc(c->d_pos_stage, atoms * P.ps)); c->n_pos_stage = atoms * P.ps; }
    if (c->n_frc_stage < atoms * P.fs) { CK(c, dalloc(c->d_frc_stage, atoms * P.fs)); c->n_frc_stage = atoms * P.fs; }
    CK(c, cudaMemcpyAsync(c->d_pos_stage, h_pos, pb, cudaMemcpyHostToDevice, c->stream));
    CK(c, cudaMemcpyAsync(c->d_frc_stage, h_force, fb, cudaMemcpyHostToDevice, c->stream));
    const float* fsd = nullptr;
    if (c->method == PSG_METHOD_ABF) {
        if (c->n_fs_stage < (size_t)P.R * P.n_cv) { CK(c, dalloc(c->d_fs_stage, (size_t)P.R * P.n_cv)); c->n_fs_stage = (size_t)P.R * P.n_cv; }
        CK(c, cudaMemcpyAsync(c->d_fs_stage, h_fsample, (size_t)P.R * P.n_cv * sizeof(float), cudaMemcpyHostToDevice, c->stream));
        fsd = c->d_fs_stage;
    }
    int rc = psg_step(c, c->d_pos_stage, c->d_frc_stage, fsd, step);
    if (rc != PSG_OK) return rc;
    CK(c, cudaMemcpyAsync(h_force, c->d_frc_stage, fb, cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    return PSG_OK;
}

int psg_sync_check(psg_ctx* c) {
    if (!c) return PSG_EINVAL;
    cudaSetDevice(c->device);
    CK(c, cudaStreamSynchronize(c->stream));
    CK(c, cudaGetLastError());
    if (c->method == PSG_METHOD_METAD && c->md.n_hills && c->overflow_possible) {
        // the host could not rule an overflow out (masked or captured deposits): ask the device
        int cnt[2] = {0, 0};
        CK(c, cudaMemcpy(cnt, c->md.n_hills, 2 * sizeof(int), cudaMemcpyDeviceToHost));
        if (cnt[1]) return fail(c, PSG_ECAPACITY, "psg_sync_check: a deposit overflowed the hill store; hills were dropped");
    }
    return PSG_OK;
}

}  // extern "C"
