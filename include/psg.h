/*
 * psg.h -- C ABI of libpsg.so: the per-MD-step enhanced-sampling hot path of
 * PySAGES (arXiv 2301.04835; citations are lines of /root/reference/PAPER.md),
 * batched over replicas / walkers / windows, as hand-written sm_100a CUDA.
 *
 *   gather CV atoms in place  ->  collective variables + analytic Jacobians
 *   ->  bias energy and gradient  ->  force[i] += -dV/dxi * dxi/dr_i
 *
 * The paper's hook "gets called as part of the time integration routine ...
 * computes the collective variables ... the computed biasing forces are added to
 * the backend net forces" on engine-owned buffers reached without
 * a copy (DLPack).  Here the engine hands over raw DEVICE pointers.
 *
 * Conventions
 *  - Every function is extern "C", never throws, returns an int status
 *    (PSG_OK = 0, errors < 0).  psg_last_error() gives the message.
 *  - "host" / "device" in a parameter comment says where the pointer must live.
 *  - Setup calls (psg_set_*, psg_load_hills) copy their host arrays, may allocate
 *    and may synchronise the ctx stream; they are not on the hot path.
 *  - Hot-path calls take device pointers only, enqueue work on the ctx stream and
 *    return immediately: no allocation, no host synchronisation, CUDA-graph
 *    capturable.  Arguments are validated on the host BEFORE anything is launched.
 *  - Ownership: the caller owns positions and forces.  Positions are read only.
 *    The force array is modified ONLY at atoms that belong to a CV group, ONLY by
 *    adding to x, y, z; w (stride 4) keeps its bits.  The ctx owns the hill store,
 *    the ABF grid (unless caller-provided), and all scratch.
 *  - Layout: positions / forces are float32, `stride` floats per atom (3 or 4;
 *    4 = float4 x,y,z,w, 16-byte aligned).  Replica r's array starts at
 *    base + r * replica_stride_atoms * stride floats; replica_stride_atoms = 0
 *    means all replicas index ONE shared array.
 *  - Degenerate geometry (coincident points, collinear bonds, Rg = 0) and CVs
 *    outside the ABF grid are NOT errors: the Jacobian / mean force is defined 0.
 *  - One ctx per stream; calls on one ctx are not thread-safe.
 *  - There is no CPU fallback: without a CUDA device psg_create fails.
 */
#ifndef PSG_H
#define PSG_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct psg_ctx psg_ctx;

enum { PSG_OK = 0, PSG_EINVAL = -1, PSG_ENOMEM = -2, PSG_ECUDA = -3, PSG_ECAPACITY = -4, PSG_ESTATE = -5 };

/* Collective variables, PAPER.md:L185-L189 (Sec. 2.2). Every argument is a GROUP of
 * atoms reduced to its weighted barycenter (barycenter(p)). */
enum {
    PSG_CV_DISTANCE = 1,      /* TwoPointCV Distance: |c2 - c1|                         (L185) */
    PSG_CV_ANGLE = 2,         /* ThreePointCV Angle at the 2nd group, in [0, pi]        (L186) */
    PSG_CV_DIHEDRAL = 3,      /* FourPointCV DihedralAngle in (-pi, pi], IUPAC sign     (L187, L81) */
    PSG_CV_COM_COMPONENT = 4, /* AxisCV Component: barycenter coordinate along an axis  (L188) */
    PSG_CV_RGYR = 5,          /* RadiusofGyration: sqrt(sum w|r-c|^2 / sum w)           (L189) */
    PSG_CV_DISPLACEMENT = 6,  /* TwoPointCV Displacement c2 - c1: one CV per component (axis) (L185) */
    /* Gyration-tensor shape CVs of ONE group, explicit atoms or a contiguous range (L188-L189; reading R-SHAPE):
     * S = sum w (r - c)(r - c)^T / sum w, eigenvalues l1 >= l2 >= l3. */
    PSG_CV_PRINCIPAL_MOMENT = 7, /* AxisCV PrincipalMoment: l_axis, axis 0 = the largest               (L188) */
    PSG_CV_ASPHERICITY = 8,      /* l1 - (l2 + l3)/2                                                    (L189) */
    PSG_CV_ACYLINDRICITY = 9,    /* l2 - l3                                                             (L189) */
    PSG_CV_SHAPE_ANISOTROPY = 10, /* ((l1 - (l2+l3)/2)^2 + 3/4 (l2 - l3)^2) / (l1+l2+l3)^2; 0 for a point (L189) */
    /* The paper's worked CV (L203-L290, Eq. 4-8; listing of Appendix A): group 0 = the mobile atoms (explicit,
     * weights = slot_weight), group 1 = the interface atoms (a contiguous range); parameters in psg_cv_desc::dti_*.
     *   xi = barycenter(group 0)[axis] - sum_j softmax(coeff |mass_{j+1} - mass_j|)_j (c_{j+1} + c_j) / 2,
     *   mass_j = sum_{i in group 1} exp(-(x_i - c_j)^2 / (2 sigma^2)),  c = linspace(scope[0], scope[1], bins).
     * At most one per ctx, shared index list; psg_step then runs the separate kernels in sequence (CVs, bias, forces) and
     * every method (harmonic, metadynamics, grid metadynamics, ABF) applies to it like to any other CV. */
    PSG_CV_DIST_TO_INTERFACE = 11
};

enum { PSG_METHOD_NONE = 0, PSG_METHOD_HARMONIC = 1, PSG_METHOD_METAD = 2, PSG_METHOD_ABF = 3, PSG_METHOD_METAD_GRID = 4 };

/* precision of the metadynamics hill sum */
enum {
    PSG_HILLS_F32 = 0, /* binary32 terms on the FP32/SFU pipes, binary64 accumulation (default) */
    PSG_HILLS_F64 = 1  /* binary64 terms: meets 1e-5 rel / 1e-6 abs on ill-conditioned gradients too */
};

#define PSG_MAX_CV 4
#define PSG_MAX_GROUPS 4
#define PSG_MAX_SLOTS 64
#define PSG_MAX_RANGE_GROUPS 8

typedef struct {
    int type;                            /* PSG_CV_* */
    int n_groups;                        /* 2, 3, 4, 1, 1, 2 for the first six types, 1 for the shape CVs, 2 for DistanceToInterface */
    int group_is_range[PSG_MAX_GROUPS];  /* 0: explicit atoms (a slice of the slot list); 1: contiguous atom range */
    int group_begin[PSG_MAX_GROUPS];     /* explicit: slots [begin, begin + size) */
    int group_size[PSG_MAX_GROUPS];
    long long range_begin[PSG_MAX_GROUPS]; /* range: atoms [range_begin, range_begin + range_size) of the replica's array */
    long long range_size[PSG_MAX_GROUPS];
    int axis;                            /* PSG_CV_COM_COMPONENT, PSG_CV_DISPLACEMENT: 0, 1, 2; PSG_CV_PRINCIPAL_MOMENT: which eigenvalue */
    double period;                       /* 0 = not periodic; 2*pi for a dihedral (binary64: the wrap must not lose bits) */
    /* PSG_CV_DIST_TO_INTERFACE only (Eq. 6-8): kernel width, bin-centre range, number of bins (2..1024), softmax sharpness */
    double dti_sigma, dti_scope[2], dti_coeff;
    int dti_bins;
} psg_cv_desc;

/* ------------------------------------------------------------------ lifetime */
/* device: CUDA ordinal.  cuda_stream: a cudaStream_t (borrowed, may be NULL = legacy default stream). */
int psg_create(psg_ctx** out, int device, void* cuda_stream);
int psg_destroy(psg_ctx* ctx);
/* Change the stream later work is enqueued on (e.g. torch's current stream). */
int psg_set_stream(psg_ctx* ctx, void* cuda_stream);
/* Message of the last error on ctx; ctx == NULL: the last psg_create failure of this thread. Never NULL. */
const char* psg_last_error(const psg_ctx* ctx);

/* --------------------------------------------------------------------- setup */
/* Snapshot layout: R replicas of n_atoms atoms.  Must precede psg_set_cvs. */
int psg_set_layout(psg_ctx* ctx, int n_replicas, long long n_atoms, long long replica_stride_atoms,
                   int pos_stride_floats, int frc_stride_floats);

/* CVs over groups of atoms.  All arrays are HOST and copied.
 *  slot_atom_idx : 0-based atom indices, [n_slots] (per_replica_indices = 0, shared by all replicas)
 *                  or [R][n_slots] (per_replica_indices = 1); every index is range-checked here.
 *  slot_weight   : [n_slots] weights of explicit atoms (masses), NULL = 1 (plain barycenter).
 *  atom_weight   : [n_atoms] weights used by RANGE groups, NULL = 1.
 * Each slot belongs to exactly one (cv, group); an atom shared by two CVs is listed twice. */
int psg_set_cvs(psg_ctx* ctx, int n_cv, const psg_cv_desc* cvs, int n_slots, const int* slot_atom_idx,
                int per_replica_indices, const float* slot_weight, const float* atom_weight);

/* Minimum-image convention for periodic POSITIONS (the paper is silent: Fig. 3 and App. A subtract raw coordinates,
 * PAPER.md:L230, L466, reading R-MI).  box [3] (host): orthorhombic box lengths, 0 = open
 * in that direction; NULL or all zeros switches it off (the default after psg_set_layout).  With a box, (i) the atoms of
 * a group are taken as the images nearest to the group's FIRST atom before the barycenter / radius of gyration
 * is formed (a molecule split by wrapping is made whole; the group must be smaller than half the box), and (ii) the
 * displacement vectors between group centres in Distance, Angle and Dihedral are nearest images.  Component reads the
 * centre as is.  Contiguous-range groups follow the same rule, the first atom being the range's first (a chain wrapped
 * atom by atom into the box is made whole; psg_step then takes the separate streaming kernels, not k_range_step).
 * Call after psg_set_cvs. */
int psg_set_box(psg_ctx* ctx, const double* box);

/* Harmonic bias, PAPER.md:L125 (Sec. 2.1.1): V = 1/2 sum_k k_k (xi_k - xi0_k)^2, differences of periodic
 * CVs wrapped to the nearest image.  kspring [n_cv], centers [R][n_cv] (host). Selects the method. */
int psg_set_harmonic(psg_ctx* ctx, const float* kspring, const float* centers);

/* Metadynamics, PAPER.md:L147-L151 (Sec. 2.1.5): V(xi) = sum_h W_h exp(-1/2 sum_k (d_hk/sigma_k)^2).
 *  sigma [n_cv] host; w0 initial height; kB_deltaT > 0: well-tempered, W = w0 exp(-V/(kB dT)) (L149);
 *  <= 0: standard.  capacity: hills the store can hold.  stride: psg_step deposits when step % stride == 0
 *  (L147 "deposited at user-defined intervals"); 0 = psg_step never deposits.  Empties the store. Selects the method. */
int psg_set_metad(psg_ctx* ctx, const float* sigma, float w0, float kB_deltaT, int capacity, int stride);
int psg_set_hill_precision(psg_ctx* ctx, int mode /* PSG_HILLS_* */);
/* Replace the store's contents by n hills: centers [n][n_cv], heights [n], DEVICE pointers (copied). */
int psg_load_hills(psg_ctx* ctx, int n, const float* d_centers, const float* d_heights);
/* Synchronises. *n_out (host) = exact hill count; if d_centers/d_heights are non-NULL (device) and
 * max_n >= count they receive the store's contents as [n][n_cv] / [n].  PSG_ECAPACITY (after filling *n_out) if an
 * earlier deposit was clamped at capacity. */
int psg_get_hills(psg_ctx* ctx, int* n_out, float* d_centers, float* d_heights, int max_n);

/* ABF, PAPER.md:L143 (Sec. 2.1.4), Grid(lower, upper, shape, periodic) of L82, N of L501/L507.
 * lower, upper, shape, periodic: [n_cv] host.  d_hist int32 [prod(shape)], d_fsum float32
 * [prod(shape)][n_cv]: device, caller-owned when non-NULL, else allocated (zeroed) and owned by ctx. */
int psg_set_abf(psg_ctx* ctx, const float* lower, const float* upper, const int* shape, const int* periodic,
                int n_threshold, int* d_hist, float* d_fsum);
/* Device pointers of the grid in use (to read it back / checkpoint it). */
int psg_abf_state(psg_ctx* ctx, int** d_hist_out, float** d_fsum_out, long long* n_bins_out);

/* ------------------------------------------------ hot path (device pointers) */
/* CVs and Jacobians of every replica ("computes the collective variables"; L185-L189).
 *  d_pos : positions, see Layout.   d_xi : out [R][n_cv].
 *  d_jac : out, nullable, [R][n_slots][3] = d(xi_cv(slot))/d(r_slot) for the explicit slots.
 * The Jacobian (explicit slots and the implicit form for range groups) is also cached in ctx
 * for the next psg_apply_bias_forces. */
int psg_cv_eval(psg_ctx* ctx, const float* d_pos, float* d_xi, float* d_jac);

/* Bias energy and gradient at given CV values for the selected method (harmonic or metadynamics).
 *  d_xi [R][n_cv] in;  d_V [R] out, nullable;  d_dVdxi [R][n_cv] out. */
int psg_bias_eval(psg_ctx* ctx, const float* d_xi, float* d_V, float* d_dVdxi);

/* Append one hill per replica at xi: all walkers see the list as it was BEFORE this
 * call and append in replica order.  d_mask [R] nullable (NULL = all deposit).
 * Capacity: the exact count lives on the device; the host tracks a lower and an upper bound of it, equal as long as no
 * mask was used.  PSG_ECAPACITY, nothing launched, when the overflow is certain (exact for d_mask == NULL: count + R >
 * capacity).  A MASKED call whose overflow the host cannot rule out is launched; the kernel never writes beyond
 * capacity, drops the excess hills and raises a sticky flag that the next psg_sync_check / psg_get_hills returns as
 * PSG_ECAPACITY (cleared by psg_load_hills / psg_set_metad).  No padding of `capacity` is needed.
 * CUDA graphs: a deposit (this call, psg_append_hills, or a psg_step on a deposit step) may be captured; replays then
 * append behind the host's back, so from that moment every launch of this ctx takes the hill count from the device
 * counter and capacity is enforced by the device clamp alone, until psg_get_hills or psg_load_hills re-synchronises. */
int psg_deposit_hill(psg_ctx* ctx, const float* d_xi, const unsigned char* d_mask);
/* The same event in two halves, for walkers spread over several GPUs (multiple-walker metadynamics needs
 * ONE exchange per deposit, an all-gather of the new hills; PAPER.md:L404-L406 runs replicas on separate GPUs).
 * psg_hill_heights: d_heights [R] (device, binary32) := the height every walker of THIS ctx would deposit at d_xi now,
 *   w0 or w0 exp(-V/(kB dT)) from the list as it is, 0 where d_mask[r] == 0; appends nothing.
 * psg_append_hills: append n ready-made hills, centres d_centers [n][n_cv] and heights d_heights [n] (device), in order,
 *   skipping zero heights.  After every rank has all-gathered (xi, heights) in rank order and appended them, every rank's
 *   list is IDENTICAL: the centres a single ctx holding all the walkers would have appended with psg_deposit_hill, with
 *   heights equal to that ctx's up to the binary32 rounding of V_old (the hill sum's chunk length depends on the walkers
 *   per ctx).  Capacity as for a masked psg_deposit_hill (zero heights are skipped on the device).  Neither call synchronises. */
int psg_hill_heights(psg_ctx* ctx, const float* d_xi, const unsigned char* d_mask, float* d_heights);
int psg_append_hills(psg_ctx* ctx, int n, const float* d_centers, const float* d_heights);

/* ABF grid update for all replicas, then the mean force from the fully updated grid (two-phase):
 *  bin in binary32: I_k = floor(fl(fl(xi_k - lower_k) * invd_k)); in-grid: hist[bin] += 1, Fsum[bin][k] += f_k;
 *  d_dVdxi[r][k] := Fsum[bin][k] / max(hist[bin], N);  outside: bin = -1, 0.
 *  d_fsample [R][n_cv] in;  d_bin [R] out nullable;  d_dVdxi [R][n_cv] out. */
int psg_abf_update(psg_ctx* ctx, const float* d_xi, const float* d_fsample, int* d_bin, float* d_dVdxi);

/* The same update in two halves, for replicas spread over several GPUs that share ONE grid (shared-grid ABF
 * needs one exchange per step, an all-reduce of the step's histogram and force-sum contributions; the paper runs replicas on
 * separate GPUs).  Reading R-ABF-2 (two-phase) then spans the ranks: ALL replicas of ALL ranks
 * accumulate before anyone reads a mean force.
 * psg_abf_accumulate_delta: gather -> CVs (+ Jacobians, cached) -> bin; the contributions of THIS ctx's replicas go to
 *   d_hist_delta int32 [n_bins] and d_fsum_delta float32 [n_bins][n_cv] (device, caller-owned, overwritten: zeroed first);
 *   the ctx grid is not touched.  Bins stay in the ctx (psg_step_outputs).
 * psg_abf_apply_grid_delta: grid += the (all-reduced) deltas, then every replica reads its mean force from the updated grid
 *   and force[i] += -Fbar_k dxi_k/dr_i, as psg_step does.  PSG_ESTATE without a pending psg_abf_accumulate_delta.
 * With one rank the two calls build the grid psg_step builds (histogram bit for bit; force sums up to the order of the
 * binary32 additions).  Neither call synchronises; both are graph-capturable. */
int psg_abf_accumulate_delta(psg_ctx* ctx, const float* d_pos, const float* d_fsample, int* d_hist_delta, float* d_fsum_delta);
int psg_abf_apply_grid_delta(psg_ctx* ctx, const int* d_hist_delta, const float* d_fsum_delta, const float* d_pos, float* d_force);

/* ABF instantaneous generalized-force estimator.  The paper says only "based on the algorithm
 * described in [43]"; this is DESIGN.md reading R-ABF-EST: with J[k][i] = d xi_k/d r_i and momenta
 * p_i = m_i v_i of the CV atoms, solve (J J^T) W = J p per replica; d_fsample[r][k] := (3/2 W(t) - 2 W(t - dt)
 * + 1/2 W(t - 2 dt)) / dt + d_fbias_prev[r][k], the last term being the mean force dV/dxi applied at the previous step
 * (NULL = 0).  The result is the `d_fsample` input of psg_abf_update / psg_step.  The history W(t - dt), W(t - 2 dt) is
 * ctx-owned; the first call after setup or psg_abf_estimate_reset initialises it to W(t) (so the first sample is
 * d_fbias_prev alone).  d_vel has the layout of d_pos; d_mass [n_atoms] (device) is shared by the replicas.  A singular
 * J J^T gives W = 0 for that replica.  Explicit groups only (PSG_EINVAL with range groups). */
int psg_abf_estimate(psg_ctx* ctx, const float* d_pos, const float* d_vel, const float* d_mass, double dt,
                     const float* d_fbias_prev, float* d_fsample);
int psg_abf_estimate_reset(psg_ctx* ctx);

/* force[i] += -sum_k dVdxi[r][k] * d(xi_k)/d(r_i), using the Jacobian cached by the last
 * psg_cv_eval on these positions (PSG_ESTATE if there was none).  d_force in/out. */
int psg_apply_bias_forces(psg_ctx* ctx, const float* d_pos, const float* d_dVdxi, float* d_force);

/* One whole step of the selected method, fused: gather -> CVs -> (deposit if due) -> bias -> forces.
 *  d_fsample: ABF only, else NULL.  step: 1-based MD step number (deposit phase).
 * Afterwards xi / V / dVdxi / bin of this step can be read with psg_step_outputs.
 * ONE kernel launch per step where a fused kernel covers the configuration, with the same results as the
 * separate calls: metadynamics over explicit groups (k_hills); ABF over explicit groups (k_abf_step);
 * harmonic windows whose groups are all contiguous ranges, float4 positions and forces 16-byte aligned, one
 * array per window, at most (SM count) slices of 2,048 atoms per window (k_range_step).  Anything else runs the
 * kernels of the separate calls in sequence.  k_abf_step and k_range_step contain inter-CTA waits and are
 * launched cooperatively: the launch fails (PSG_ECUDA) rather than hangs if the grid cannot be co-resident.
 * Every hot-path call is wrapped in an NVTX range of its own name. */
int psg_step(psg_ctx* ctx, const float* d_pos, float* d_force, const float* d_fsample, long long step);
/* Device pointers (ctx-owned, valid until destroy/reconfigure) of the last step's per-replica results:
 * xi [R][n_cv], V [R] (0 for ABF), dVdxi [R][n_cv], bin [R] (ABF only, else NULL). Any out may be NULL. */
int psg_step_outputs(psg_ctx* ctx, float** d_xi, float** d_V, float** d_dVdxi, int** d_bin);

/* The same step for an engine whose arrays live on the HOST (pinned memory recommended): copies
 * h_pos (and h_force) to ctx-owned device buffers, runs psg_step, copies the forces back and waits. */
int psg_step_host(psg_ctx* ctx, const float* h_pos, float* h_force, const float* h_fsample, long long step);

/* The only other call that synchronises: waits for the ctx stream and returns sticky CUDA errors, and PSG_ECAPACITY if a
 * masked or graph-captured deposit was clamped at the hill store's capacity. */
int psg_sync_check(psg_ctx* ctx);

/* ------------------------------------------------------------- DistanceToInterface */
/* The paper's own worked collective variable (Eq. 4-8; listing of Appendix A), for all
 * replicas of the ctx layout (psg_set_layout), as calls of its own (PSG_CV_DIST_TO_INTERFACE configures the same kernels
 * through psg_set_cvs and puts the CV on the psg_step path; use one or the other on a ctx):
 *   xi = barycenter(mobile atoms)[axis] - sum_j softmax(coeff |mass_{j+1} - mass_j|)_j (c_{j+1} + c_j) / 2,
 *   mass_j = sum_i exp(-(x_i - c_j)^2 / (2 sigma^2)) over the interface atoms, c = linspace(scope0, scope1, bins).
 * psg_interface_cv_set (host arrays copied; allocates): mobile_idx [n_mobile <= PSG_MAX_SLOTS] 0-based, mobile_w nullable
 *   (= 1); interface atoms = the contiguous range [iface_begin, iface_begin + iface_size) of every replica's array;
 *   2 <= bins <= 1024.
 * psg_interface_cv_eval: d_xi [R] out; also keeps d interface / d mass_j per replica for the apply call.
 * psg_interface_cv_apply: force[i][axis] += -d_dVdxi[r] * d xi / d x_i for interface and mobile atoms of replica r, with
 *   the derivatives written out analytically (the paper obtains them by autodiff); call after psg_interface_cv_eval on
 *   the same positions.  Both enqueue on the ctx stream, no sync.  All arithmetic is binary64 (see interface_cv.cu). */
int psg_interface_cv_set(psg_ctx* ctx, int n_mobile, const int* mobile_idx, const float* mobile_w, long long iface_begin,
                         long long iface_size, int axis, double sigma, double scope0, double scope1, int bins, double coeff);
int psg_interface_cv_eval(psg_ctx* ctx, const float* d_pos, float* d_xi);
int psg_interface_cv_apply(psg_ctx* ctx, const float* d_pos, const float* d_dVdxi, float* d_force);

/* ------------------------------------------------------------- grid-stored metadynamics */
/* "optional support for storing the bias potentials ... on a pre-defined grid".  The paper
 * gives neither layout nor interpolation; reading R-GRID: Grid(lower, upper, shape, periodic) as in L82 with
 * shape[k] NODES per CV (periodic: one period, h = (upper - lower)/shape; open: nodes on both ends, h = (upper - lower)/
 * (shape - 1)); every node holds the hill sum and its gradient, [nodes][1 + n_cv] binary64, row-major, last CV fastest;
 * the bias at xi is the multilinear interpolation of the 2^n_cv surrounding nodes (value and gradient alike; outside an
 * open grid xi is clamped to the nearest face).  First version: calls of their own beside psg_cv_eval (which produces
 * d_xi) and psg_apply_bias_forces (which consumes d_dVdxi); they do not touch the hill list of psg_set_metad.
 * psg_metad_grid_set (host arrays copied; allocates and zeroes the grid; needs psg_set_layout for the walker count R):
 *   lower, upper, sigma [n_cv]; shape >= 2; w0 > 0; kB_deltaT = 0: standard, > 0: well-tempered heights
 *   w0 exp(-V_grid(xi) / kB_deltaT) from the grid BEFORE the event.  At most 2^27 nodes.
 * psg_metad_grid_deposit: one synchronous event -- every walker r with d_mask[r] != 0 (NULL: all) adds its hill, centred on
 *   d_xi[r] (device, [R][n_cv] binary32), to every node, in replica order.  Two launches on the ctx stream, no sync.
 * psg_metad_grid_eval: d_V [R] and d_dVdxi [R][n_cv] (device, binary32; either may be NULL).  One launch, no sync.
 * psg_metad_grid_step: the per-step path with the bias on the grid in ONE launch: CVs and Jacobians of the configured CVs
 *   (psg_set_cvs; n_cv and R must match the grid) -> interpolated bias at the binary32 CV values -> force[i] += -dV/dxi *
 *   dxi/dr_i in place.  xi, V, dV/dxi are left in the buffers psg_step_outputs returns (feed that xi to
 *   psg_metad_grid_deposit every `stride` steps).  CVs over atom ranges take three launches instead.  No sync.
 * psg_metad_grid_state: device pointers of the node array and of the heights [R] (binary64) of the last event; owned by
 *   the ctx, valid until the next psg_metad_grid_set or psg_destroy.
 * All of this state is dropped by psg_set_layout (it is sized by the layout).
 * Errors: PSG_EINVAL (arguments), PSG_ESTATE (call order), PSG_ENOMEM, PSG_ECUDA. */
/* psg_set_metad_grid: the grid-stored bias as the METHOD of the ctx (PAPER.md:L151 with the deposit interval of L147):
 *   psg_metad_grid_set with the same arguments, then psg_step / psg_step_host run CVs -> (one deposit event onto the grid
 *   when step % stride == 0, step >= 1; stride = 0: never) -> interpolated bias -> forces, psg_bias_eval is
 *   psg_metad_grid_eval and psg_deposit_hill is psg_metad_grid_deposit.  Call after psg_set_cvs (n_cv must match).  A
 *   periodic CV needs a periodic grid spanning exactly its period and an open CV an open grid: PSG_EINVAL otherwise (a
 *   dihedral on an open grid would be clamped at +-pi instead of wrapped). */
int psg_set_metad_grid(psg_ctx* ctx, const double* lower, const double* upper, const int* shape, const int* periodic,
                       const double* sigma, double w0, double kB_deltaT, int stride);
int psg_metad_grid_set(psg_ctx* ctx, int n_cv, const double* lower, const double* upper, const int* shape, const int* periodic,
                       const double* sigma, double w0, double kB_deltaT);
int psg_metad_grid_deposit(psg_ctx* ctx, const float* d_xi, const unsigned char* d_mask);
int psg_metad_grid_eval(psg_ctx* ctx, const float* d_xi, float* d_V, float* d_dVdxi);
int psg_metad_grid_step(psg_ctx* ctx, const float* d_pos, float* d_force);
int psg_metad_grid_state(psg_ctx* ctx, double** d_grid_out, long long* n_nodes_out, double** d_heights_out);

#ifdef __cplusplus
}
#endif
#endif /* PSG_H */
