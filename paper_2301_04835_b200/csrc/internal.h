// internal.h -- shared declarations of libpsg.so (CUDA path). Not part of the ABI.
// Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>

#include "psg.h"

#define PSG_MAX_GROUPS_TOTAL (PSG_MAX_CV * PSG_MAX_GROUPS)
#define PSG_MAX_DEVICES 64        // per-device caches of function attributes / occupancy (device ordinal modulo this)
#define PSG_GDESC_DOUBLES 8      // per (replica, group): vx vy vz | cx cy cz | coef | W
#define PSG_MOM 5                // moments per range group: W, sum w x, sum w y, sum w z, sum w |r|^2
#define PSG_RANGE_TILE 2048      // atoms per block / slice in the range-moment, dense-apply and fused range-step kernels
#define PSG_RANGE_THREADS 256    // threads that reduce one slice's moments (k_range_moments block = A group of k_range_step: same thread -> atom map, same bits)
#define PSG_HILL_RT 8            // replicas per thread in the hill sum
#ifndef PSG_HILL_WARPS
#define PSG_HILL_WARPS 16        // warps per CTA in the hill sum: two halves share the tile's replicas and split its hills
#endif
#define PSG_HILL_HALF (PSG_HILL_WARPS / 2)
#define PSG_HILL_TILE_R (PSG_HILL_RT * PSG_HILL_HALF)   // replicas per CTA tile (64): warp w and warp w + HALF own the same 8 replicas
#define PSG_HILL_SUB 4096        // 16-byte hill records per shared-memory stage (64 KB): 64 hills per lane and pass of the hill loop; with 2,048 the
                                 // loop's peeled entry / exit iterations and the per-stage bookkeeping cost config 1 5 % and config 4 0.5 %

struct CvDev {
    int type, n_groups, axis, gid0;   // gid0: global id of this CV's first group
    double period;
};

struct GroupDev {
    int cv, g;          // owner
    int is_range;
    int begin, size;    // explicit: slot slice
    int range_id;       // range: index into the range table, else -1
    long long rbegin, rsize;
};

// Everything a kernel needs to know about the system; passed by value.
struct SysParams {
    int R;
    long long N, rstride;       // rstride = 0: shared array
    int ps, fs;                 // floats per atom in pos / force
    int n_cv, n_slots, per_rep, n_groups, n_ranges;
    int any_rgyr;
    int any_shape_range;        // a gyration-tensor shape CV over a contiguous range: second moments from k_range_second
    int has_box;                // minimum-image convention on (psg_set_box); explicit groups only
    double box[3];              // orthorhombic box lengths, 0 = open in that direction
    CvDev cv[PSG_MAX_CV];
    GroupDev grp[PSG_MAX_GROUPS_TOTAL];
    int range_gid[PSG_MAX_RANGE_GROUPS];     // range id -> global group id
    long long span_begin, span_end;          // union span of all range groups
    int range_blocks;                        // blocks per replica over the span
    int slot_atom_c[PSG_MAX_SLOTS];          // shared index list (per_rep == 0): read from kernel parameters
    unsigned char slot_gid_c[PSG_MAX_SLOTS]; // global group id of a slot, from kernel parameters too (slot_gid is the device copy)
    // fast gather of the fused metadynamics step: when every group is ONE explicit atom (simple_groups), group g of CV k
    // is slot cv_slot[4 k + g] and, with a shared index list, atom cv_atom[4 k + g]; unused groups repeat group 0
    int simple_groups;
    int cv_slot[PSG_MAX_CV * PSG_MAX_GROUPS];
    int cv_atom[PSG_MAX_CV * PSG_MAX_GROUPS];
    const int* slot_atom;        // device [n_slots] or [R][n_slots]
    const int* slot_gid;         // device [n_slots]: global group id of a slot
    const float* slot_weight;    // device [n_slots] or nullptr
    const float* atom_weight;    // device [N] or nullptr
};

struct HillConsts {
    float inv_period[PSG_MAX_CV];   // 0 if not periodic (then the wrap is the identity)
    float np_hi[PSG_MAX_CV], np_lo[PSG_MAX_CV];   // -P as two binary32 constants (Cody-Waite)
    float nc[PSG_MAX_CV];           // -log2(e) / (2 sigma_k^2): base-2 exponent = log2 W + sum_k nc_k d_k^2
    double gscale[PSG_MAX_CV];      // dV/dxi_k = -gscale_k * sum_h W e d_k,  gscale_k = 1 / sigma_k^2
    double period_d[PSG_MAX_CV];    // binary64 path; 1e300 if not periodic
    double inv_sigma_d[PSG_MAX_CV];
    int n_cv, pmask;
    int neq;                        // number of leading CVs whose nc equals nc[0]
};

struct MetadState {
    float4* hills;          // kernel-side records: n_cv<=3: {s0,s1,s2,log2 W}; n_cv==4: {s0..s3},{log2 W,0,0,0}
    float* heights;         // W as deposited / loaded (exported by psg_get_hills; read by the binary64 path)
    int* n_hills;           // device: [0] the exact count, [1] sticky overflow flag (a deposit was clamped at capacity)
    int capacity;
    double* part;           // [max_chunks][n_rtiles][TILE_R][1+n_cv]: published chunk partials, a cleared word = not there yet
    int max_chunks;
    double w0, kB_deltaT;
    int stride;
    int precision;
    int rec;                // float4s per hill record
    HillConsts hc;
};

struct AbfState {
    float lower[PSG_MAX_CV], invd[PSG_MAX_CV];
    int shape[PSG_MAX_CV], periodic[PSG_MAX_CV];
    int n_threshold;
    long long n_bins;
    int* hist;
    float* fsum;
    bool own;
};

struct psg_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    long long launches = 0;
    bool have_layout = false, have_cvs = false, have_jac = false;
    int method = PSG_METHOD_NONE;
    SysParams sys{};
    // device copies of setup arrays
    int* d_slot_atom = nullptr; int* d_slot_gid = nullptr; float* d_slot_weight = nullptr; float* d_atom_weight = nullptr;
    // per-replica scratch / step outputs
    float* d_xi = nullptr; float* d_V = nullptr; float* d_dVdxi = nullptr; int* d_bin = nullptr;
    double* d_V64 = nullptr;
    float* d_jac = nullptr;          // [R][n_slots][3]
    double* d_gdesc = nullptr;       // [R][n_groups][PSG_GDESC_DOUBLES]
    double* d_rpart = nullptr;       // [R][n_ranges][range_blocks][PSG_MOM]
    double* d_rpart2 = nullptr;      // [R][n_ranges][range_blocks][6]: second moments about the group's first atom (shape CVs over ranges)
    double* d_gdesc_m = nullptr;     // [R][n_groups][6]: the symmetric matrix M of d xi / d r_i = w_i M (r_i - c) of such a group
    unsigned* d_arrive = nullptr;    // [2][R]: arrive / done counters of the fused range step (zero between launches)
    double* d_whist = nullptr;       // [R][2][n_cv]: W(t - dt), W(t - 2 dt) of the ABF force estimator
    bool est_first = true;           // the next psg_abf_estimate initialises the history
    unsigned* d_gbar = nullptr;      // [2]: grid-barrier counters of the fused ABF step (zero between launches)
    float4* d_rdesc = nullptr;       // [R][n_ranges][4]: tagged force descriptors of the fused range step (zero between launches)
    // harmonic
    float* d_kspring = nullptr; float* d_centers = nullptr;
    MetadState md{};
    long long nh_bound = 0;          // host UPPER bound of the hill count (+R per deposit call; exact while no mask was used)
    long long nh_lo = 0;             // host LOWER bound (+0 for a masked call): a deposit is refused only when overflow is certain
    bool overflow_possible = false;  // a deposit was launched that the host could not prove to fit: psg_sync_check asks the device
    bool count_unknown = false;      // a deposit was enqueued under stream capture: replays move the device counter behind the
                                     // host's back, so kernels read the device counter until psg_get_hills / psg_load_hills
    AbfState abf{};
    bool abf_delta_pending = false;  // psg_abf_accumulate_delta has run, psg_abf_apply_grid_delta has not
    // host-engine staging (psg_step_host)
    float* d_pos_stage = nullptr; float* d_frc_stage = nullptr; float* d_fs_stage = nullptr;
    size_t n_pos_stage = 0, n_frc_stage = 0, n_fs_stage = 0;   // their sizes in floats (grown on demand: the layout may change)
    int range_lag = 10;              // items the position producer of k_range_step may run ahead of the force group
    bool range_step_off = false;     // psg_set_tuning: take the separate kernels instead of k_range_step
    int sm_count = 148;
    void* dti = nullptr;             // state of the DistanceToInterface CV (interface_cv.cu)
    void* mgrid = nullptr;           // state of grid-stored metadynamics (metad_grid.cu)
    int dti_cv = -1;                 // index of the PSG_CV_DIST_TO_INTERFACE CV (its value and forces come from interface_cv.cu), else -1
    int mgrid_stride = 0;            // PSG_METHOD_METAD_GRID: psg_step deposits when step % stride == 0
};
void psg_interface_cv_free(psg_ctx* c);
cudaError_t psg_launch_dti_eval(psg_ctx* c, const float* d_pos, float* d_xi, int xi_stride, int xi_col);
cudaError_t psg_launch_dti_apply(psg_ctx* c, const float* d_pos, const float* d_dVdxi, int dv_stride, int dv_col, float* d_force);
void psg_metad_grid_free(psg_ctx* c);

// ---- launchers implemented in the .cu files (all enqueue on ctx->stream) ----
cudaError_t psg_launch_cv_eval(psg_ctx* c, const float* d_pos, float* d_xi, float* d_jac);
cudaError_t psg_launch_apply(psg_ctx* c, const float* d_pos, const float* d_dVdxi, float* d_force);
cudaError_t psg_launch_harmonic(psg_ctx* c, const float* d_xi, float* d_V, float* d_dVdxi);
cudaError_t psg_launch_hillsum(psg_ctx* c, const float* d_xi, float* d_V, float* d_dVdxi);
cudaError_t psg_launch_deposit(psg_ctx* c, const float* d_xi, const unsigned char* d_mask);
cudaError_t psg_launch_hill_heights(psg_ctx* c, const float* d_xi, const unsigned char* d_mask, float* d_heights);
cudaError_t psg_launch_append_hills(psg_ctx* c, int n, const float* d_centers, const float* d_heights);
cudaError_t psg_launch_pack_hills(psg_ctx* c, int n, const float* d_centers, const float* d_heights);
cudaError_t psg_launch_unpack_hills(psg_ctx* c, int n, float* d_centers, float* d_heights);
cudaError_t psg_launch_null_hills(psg_ctx* c, int begin, int end);   // records [begin, end) := null
cudaError_t psg_launch_abf(psg_ctx* c, const float* d_xi, const float* d_fsample, int* d_bin, float* d_dVdxi);
cudaError_t psg_launch_metad_step(psg_ctx* c, const float* d_pos, float* d_force);   // fused; n_ranges == 0
bool psg_metad_step_supported(const psg_ctx* c);
cudaError_t psg_launch_abf_estimate(psg_ctx* c, const float* d_pos, const float* d_vel, const float* d_mass, double dt,
                                    const float* d_fbias_prev, float* d_fsample);
bool psg_abf_step_supported(const psg_ctx* c);
cudaError_t psg_launch_abf_step(psg_ctx* c, const float* d_pos, const float* d_fsample, float* d_force);   // fused ABF step
cudaError_t psg_launch_abf_phase(psg_ctx* c, int phase, const float* d_pos, const float* d_fsample, float* d_force, int* hist,
                                 float* fsum);   // one half of the fused ABF step (phase 1 or 2)
cudaError_t psg_launch_abf_add_delta(psg_ctx* c, const int* d_hist_delta, const float* d_fsum_delta);
cudaError_t psg_launch_abf_accumulate(psg_ctx* c, const float* d_xi, const float* d_fsample, int* hist, float* fsum);   // k_abf_accumulate
cudaError_t psg_launch_abf_mean(psg_ctx* c, int* d_bin, float* d_dVdxi);                                             // k_abf_mean
bool psg_range_step_supported(const psg_ctx* c, const float* d_pos, const float* d_force);
cudaError_t psg_launch_range_step(psg_ctx* c, const float* d_pos, float* d_force);   // fused harmonic step over range groups
bool psg_stream_capturing(const psg_ctx* c);
size_t psg_hill_part_doubles(const psg_ctx* c, int* max_chunks_out, int* n_rtiles_out);
// The layout the thread-per-(replica, CV) kernels cover (k_cv_eval_lean, k_abf_step_lean, k_abf_estimate_lean): explicit groups
// only, no minimum-image box, no DistanceToInterface CV, every CV a point-group CV (no Rg, no shape CV).
inline bool psg_lean_layout(const psg_ctx* c) {
    const SysParams& P = c->sys;
    if (P.n_ranges > 0 || P.any_rgyr || P.has_box || c->dti_cv >= 0 || P.n_cv < 1 || P.n_slots < 1) return false;
    for (int k = 0; k < P.n_cv; ++k) {
        const int t = P.cv[k].type;
        if (!(t == PSG_CV_DISTANCE || t == PSG_CV_ANGLE || t == PSG_CV_DIHEDRAL || t == PSG_CV_DISPLACEMENT || t == PSG_CV_COM_COMPONENT))
            return false;
    }
    return true;
}
