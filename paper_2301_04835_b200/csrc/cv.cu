// cv.cu -- CV evaluation (psg_cv_eval) and bias-force application (psg_apply_bias_forces).
//   k_range_moments : HBM-bound block reduction of the weighted moments of large contiguous groups
//   k_cv_eval       : one warp per replica: gather explicit atoms, combine moments, CVs + Jacobians (fp64 regs)
//   k_apply_sparse  : one thread per (replica, slot): red.global.add of -dV/dxi * J into the force array
//   k_apply_dense   : HBM-bound force read-modify-write over contiguous groups (implicit Jacobian)
#include "geom.cuh"

// --------------------------------------------------------------------------------------------
// Moments of range groups. grid = (range_blocks, R); block b covers atoms [span_begin + b*TILE, +TILE).
// Every atom is loaded once (coalesced float4) and contributes to each range group that contains it.
// Output: rpart[r][q][b][5] in binary64 (products of binary32 inputs are exact in binary64).
template <bool BOX>   // BOX: minimum image on (psg_set_box); a separate instantiation keeps the open-boundary kernel as lean as it was
__global__ void __launch_bounds__(PSG_RANGE_THREADS, 4) k_range_moments(const __grid_constant__ SysParams P, const float* __restrict__ pos,
                                                        double* __restrict__ rpart) {
    constexpr int NT = PSG_RANGE_THREADS, PER = PSG_RANGE_TILE / NT;
    const int r = blockIdx.y, b = blockIdx.x, tid = threadIdx.x;
    const float* p = pos + (long long)r * P.rstride * P.ps;
    const long long t0 = P.span_begin + (long long)b * PSG_RANGE_TILE;
    float x[PER], y[PER], z[PER];
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        long long a = t0 + tid + (long long)i * NT;
        x[i] = y[i] = z[i] = 0.f;
        if (a < P.span_end) {
            if (P.ps == 4) {
                float4 v = __ldg(reinterpret_cast<const float4*>(p) + a);
                x[i] = v.x; y[i] = v.y; z[i] = v.z;
            } else {
                x[i] = __ldg(p + a * 3); y[i] = __ldg(p + a * 3 + 1); z[i] = __ldg(p + a * 3 + 2);
            }
        }
    }
    // per group: skip blocks that do not touch it; a block that lies wholly inside several groups is reduced once and
    // the moments are copied (the same bits); one pair of barriers for all groups. k_range_step's A group does the same.
    __shared__ double red[NT / 32][PSG_MAX_RANGE_GROUPS][PSG_MOM];
    const long long t1 = t0 + PSG_RANGE_TILE < P.span_end ? t0 + PSG_RANGE_TILE : P.span_end;
    bool have_full = false;
    double mf[PSG_MOM] = {0, 0, 0, 0, 0};
    for (int q = 0; q < P.n_ranges; ++q) {
        const GroupDev& G = P.grp[P.range_gid[q]];
        const long long gb = G.rbegin, ge = G.rbegin + G.rsize;
        double m[PSG_MOM] = {0, 0, 0, 0, 0};
        if (t0 < ge && t1 > gb) {   // block-uniform
            // minimum image (psg_set_box, reading R-MI): the group's atoms are the images nearest to its FIRST atom, so
            // the moments depend on the group and a block's sums cannot be shared between groups
            const bool inside = gb <= t0 && t1 <= ge && !BOX;
            D3 first = d3(0, 0, 0);
            if (BOX) first = load_pos(p, gb, P.ps);
            if (inside && have_full) {
#pragma unroll
                for (int i = 0; i < PSG_MOM; ++i) m[i] = mf[i];
            } else {
#pragma unroll
                for (int i = 0; i < PER; ++i) {
                    // branch-free: an atom outside the group enters with w = 0 and r = 0, which adds exactly +0
                    const long long a = t0 + tid + (long long)i * NT;
                    const bool in = a >= gb && a < ge && a < t1;
                    float wf = 0.f;
                    if (in) wf = P.atom_weight ? __ldg(P.atom_weight + a) : 1.f;   // (weights are re-read per group pass: L1/L2 hits)
                    double xd = in ? (double)x[i] : 0.0, yd = in ? (double)y[i] : 0.0, zd = in ? (double)z[i] : 0.0;
                    if (BOX && in) {
                        const D3 d = min_image(d3(xd - first.x, yd - first.y, zd - first.z), P.box);
                        xd = first.x + d.x; yd = first.y + d.y; zd = first.z + d.z;
                    }
                    const double wd = (double)wf;
                    m[0] += wd; m[1] += wd * xd; m[2] += wd * yd; m[3] += wd * zd;
                    m[4] += wd * (xd * xd + yd * yd + zd * zd);
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
        if ((tid & 31) == 0) {
#pragma unroll
            for (int i = 0; i < PSG_MOM; ++i) red[tid >> 5][q][i] = m[i];
        }
    }
    __syncthreads();
    if (tid < P.n_ranges * PSG_MOM) {
        const int q = tid / PSG_MOM, i = tid % PSG_MOM;
        double s = 0;
#pragma unroll
        for (int wq = 0; wq < NT / 32; ++wq) s += red[wq][q][i];
        rpart[(((long long)r * P.n_ranges + q) * P.range_blocks + b) * PSG_MOM + i] = s;
    }
}

// --------------------------------------------------------------------------------------------
// Second moments of the range groups that carry a gyration-tensor shape CV (PAPER.md:L188-L189 over large groups): per block
// and group the six sums of w e e^T, e = r - (the group's first atom; with a box the nearest image), binary64. grid =
// (range_blocks, R) like k_range_moments; only launched when such a CV exists.
template <bool BOX>
__global__ void __launch_bounds__(256) k_range_second(const __grid_constant__ SysParams P, const float* __restrict__ pos,
                                                       double* __restrict__ rpart2) {
    const int r = blockIdx.y, b = blockIdx.x, tid = threadIdx.x;
    const float* p = pos + (long long)r * P.rstride * P.ps;
    const long long t0 = P.span_begin + (long long)b * PSG_RANGE_TILE;
    const long long t1 = t0 + PSG_RANGE_TILE < P.span_end ? t0 + PSG_RANGE_TILE : P.span_end;
    __shared__ double red[8][6];
    for (int q = 0; q < P.n_ranges; ++q) {
        const GroupDev& G = P.grp[P.range_gid[q]];
        if (!is_shape_cv(P.cv[G.cv].type)) continue;   // block-uniform
        const long long gb = G.rbegin, ge = G.rbegin + G.rsize;
        double m[6] = {0, 0, 0, 0, 0, 0};
        if (t0 < ge && t1 > gb) {
            const D3 first = load_pos(p, gb, P.ps);
            for (long long a = t0 + tid; a < t1; a += 256) {
                if (a < gb || a >= ge) continue;
                const D3 x = load_pos(p, a, P.ps);
                D3 e = x - first;
                if (BOX) e = min_image(e, P.box);
                const double w = P.atom_weight ? (double)__ldg(P.atom_weight + a) : 1.0;
                m[0] += w * e.x * e.x; m[1] += w * e.x * e.y; m[2] += w * e.x * e.z;
                m[3] += w * e.y * e.y; m[4] += w * e.y * e.z; m[5] += w * e.z * e.z;
            }
        }
#pragma unroll
        for (int i = 0; i < 6; ++i) m[i] = warp_sum(m[i]);
        __syncthreads();
        if ((tid & 31) == 0)
#pragma unroll
            for (int i = 0; i < 6; ++i) red[tid >> 5][i] = m[i];
        __syncthreads();
        if (tid < 6) {
            double s = 0;
#pragma unroll
            for (int wq = 0; wq < 8; ++wq) s += red[wq][tid];   // fixed order
            rpart2[(((long long)r * P.n_ranges + q) * P.range_blocks + b) * 6 + tid] = s;
        }
    }
}

// --------------------------------------------------------------------------------------------
// One warp per replica. Writes xi (fp32), the compact Jacobian of explicit slots (fp32, to jac_user and/or
// jac_cache) and the per-group descriptors gdesc[r][gid] = {v(3), c(3), coef, W} (fp64) for range groups.
__global__ void __launch_bounds__(256) k_cv_eval(const __grid_constant__ SysParams P, const float* __restrict__ pos,
                                                  const double* __restrict__ rpart, float* __restrict__ xi,
                                                  float* __restrict__ jac_user, float* __restrict__ jac_cache,
                                                  double* __restrict__ gdesc, const double* __restrict__ rpart2,
                                                  double* __restrict__ gdesc_m) {
    __shared__ WarpCvSmem sm[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int r = blockIdx.x * 8 + wid;
    if (r >= P.R) return;
    WarpCvSmem& S = sm[wid];
    warp_cv_eval<true>(P, r, pos, rpart, S, lane, rpart2);
    if (lane < P.n_cv) xi[(long long)r * P.n_cv + lane] = (float)S.xi[lane];
    for (int s = lane; s < P.n_slots; s += 32) {
        D3 j = slot_jacobian(P, r, pos, S, s);
        long long o = ((long long)r * P.n_slots + s) * 3;
        if (jac_user) { jac_user[o] = (float)j.x; jac_user[o + 1] = (float)j.y; jac_user[o + 2] = (float)j.z; }
        jac_cache[o] = (float)j.x; jac_cache[o + 1] = (float)j.y; jac_cache[o + 2] = (float)j.z;
    }
    if (P.n_ranges > 0 && lane < P.n_groups) {
        double* d = gdesc + ((long long)r * P.n_groups + lane) * PSG_GDESC_DOUBLES;
        d[0] = S.v[lane][0]; d[1] = S.v[lane][1]; d[2] = S.v[lane][2];
        d[3] = S.cen[lane][0]; d[4] = S.cen[lane][1]; d[5] = S.cen[lane][2];
        d[6] = S.coef[lane]; d[7] = S.cen[lane][3];
        if (gdesc_m) {   // shape CVs over ranges: the matrix M of d xi / d r_i = w_i M (r_i - c)
            double* m = gdesc_m + ((long long)r * P.n_groups + lane) * 6;
#pragma unroll
            for (int e = 0; e < 6; ++e) m[e] = S.sec[lane][e];
        }
    }
}

// --------------------------------------------------------------------------------------------
// psg_cv_eval for the common layout (psg_lean_layout: explicit groups, no box, point-group CVs): TWO THREADS per (replica, CV),
// in different warps, one for the value (sqrt / atan2 chain), one for the derivative (cv_jacobian_only), each gathering the few
// atoms of its CV's groups itself.  A binary64 warp instruction then carries 32 chains; the warp-per-replica kernel above issues
// each of them for the 1-4 lanes that own a CV.  Same xi bits; the Jacobian agrees to ~1 ulp of binary64 before
// it is rounded to binary32.
#define CVL_RB 32   // replicas per CTA: CVL_RB x n_cv value threads followed by as many derivative threads (whole warps)
__global__ void __launch_bounds__(CVL_RB * PSG_MAX_CV * 2) k_cv_eval_lean(const __grid_constant__ SysParams P, const float* __restrict__ pos,
                                                                        float* __restrict__ xi, float* __restrict__ jac_user,
                                                                        float* __restrict__ jac_cache) {
    const int n_cv = P.n_cv, tid = threadIdx.x;
    const int role = tid >= CVL_RB * n_cv ? 1 : 0;
    const int t = tid - role * CVL_RB * n_cv, rl = t / n_cv, k = t - rl * n_cv;
    const int r = blockIdx.x * CVL_RB + rl;
    if (r >= P.R) return;
    const CvDev& C = P.cv[k];
    D3 c[4], dc[4];
    double Wg[4];
    thread_group_centres(P, r, C, pos + (long long)r * P.rstride * P.ps, c, Wg);
    if (role == 0) {
        xi[(long long)r * n_cv + k] = (float)cv_from_centers<false>(C.type, C.axis, c, dc, nullptr);
        return;
    }
    cv_jacobian_only(C.type, C.axis, c, dc);
#pragma unroll
    for (int g = 0; g < 4; ++g)
        if (g < C.n_groups) {
            const GroupDev& Gd = P.grp[C.gid0 + g];
            const double iw = 1.0 / Wg[g];
            for (int i = 0; i < Gd.size; ++i) {
                const int s = Gd.begin + i;
                const double w = P.slot_weight ? (double)P.slot_weight[s] : 1.0;
                const float jx = (float)(w * (dc[g].x * iw)), jy = (float)(w * (dc[g].y * iw)), jz = (float)(w * (dc[g].z * iw));
                const long long o = ((long long)r * P.n_slots + s) * 3;
                if (jac_user) { jac_user[o] = jx; jac_user[o + 1] = jy; jac_user[o + 2] = jz; }
                jac_cache[o] = jx; jac_cache[o + 1] = jy; jac_cache[o + 2] = jz;
            }
        }
}

// --------------------------------------------------------------------------------------------
// Sparse scatter: thread per (replica, slot). Atoms shared between CVs (6, 8, 14 of phi/psi) or between
// walkers of a shared array collide, hence L2 reductions (force_add: red.global.add.v2.f32 + one scalar per float4 record).
__global__ void __launch_bounds__(256) k_apply_sparse(const __grid_constant__ SysParams P, const float* __restrict__ jac,
                                                       const float* __restrict__ dVdxi, float* __restrict__ force) {
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)P.R * P.n_slots) return;
    int r = (int)(t / P.n_slots), s = (int)(t % P.n_slots);
    int gid = P.slot_gid_c[s];
    float dv = -dVdxi[(long long)r * P.n_cv + P.grp[gid].cv];
    int atom = slot_atom_of(P, r, s);
    float* f = force + ((long long)r * P.rstride + atom) * P.fs;
    const float* j = jac + t * 3;
    force_add(f, dv * j[0], dv * j[1], dv * j[2], P.fs);
}

// --------------------------------------------------------------------------------------------
// Dense application over range groups: grid = (range_blocks, R). Per atom:
//   F_i += sum_{groups containing i} -dV_cv * w_i * ( v_g  +  coef_g * (r_i - c_g) )
// Force is read and written once (float4, w preserved bit for bit); positions are read only when an Rg
// CV needs r_i. Each replica owns its atoms here (no atomics); with a shared array (rstride = 0) several
// replicas would hit the same atoms, so that case uses atomics.
template <bool BOX>
__global__ void __launch_bounds__(256) k_apply_dense(const __grid_constant__ SysParams P, const float* __restrict__ pos,
                                                      const double* __restrict__ gdesc, const float* __restrict__ dVdxi,
                                                      float* __restrict__ force, const double* __restrict__ gdesc_m) {
    constexpr int PER = PSG_RANGE_TILE / 256;
    const int r = blockIdx.y, b = blockIdx.x, tid = threadIdx.x;
    const long long t0 = P.span_begin + (long long)b * PSG_RANGE_TILE;
    __shared__ float s_v[PSG_MAX_RANGE_GROUPS][3], s_chi[PSG_MAX_RANGE_GROUPS][3], s_clo[PSG_MAX_RANGE_GROUPS][3],
        s_k[PSG_MAX_RANGE_GROUPS];
    __shared__ long long s_b[PSG_MAX_RANGE_GROUPS], s_e[PSG_MAX_RANGE_GROUPS];
    __shared__ double s_first[PSG_MAX_RANGE_GROUPS][3], s_cd[PSG_MAX_RANGE_GROUPS][3];   // minimum image: first atom, centre
    __shared__ float s_M[PSG_MAX_RANGE_GROUPS][6];   // shape CVs: -dV/dxi * M (symmetric), s_shape = 1
    __shared__ int s_shape[PSG_MAX_RANGE_GROUPS];
    if (tid < P.n_ranges) {
        int gid = P.range_gid[tid];
        const GroupDev& G = P.grp[gid];
        const double* d = gdesc + ((long long)r * P.n_groups + gid) * PSG_GDESC_DOUBLES;
        double dv = -(double)dVdxi[(long long)r * P.n_cv + G.cv];
#pragma unroll
        for (int x = 0; x < 3; ++x) {
            s_v[tid][x] = (float)(dv * d[x]);
            float hi = (float)d[3 + x];
            s_chi[tid][x] = hi;
            s_clo[tid][x] = (float)(d[3 + x] - (double)hi);   // centre as hi + lo: (r - hi) - lo keeps r - c accurate
        }
        s_k[tid] = (float)(dv * d[6]);
        s_b[tid] = G.rbegin; s_e[tid] = G.rbegin + G.rsize;
        s_shape[tid] = gdesc_m != nullptr && d[6] == PSG_COEF_SHAPE;
        if (s_shape[tid]) {
            const double* m = gdesc_m + ((long long)r * P.n_groups + gid) * 6;
#pragma unroll
            for (int e = 0; e < 6; ++e) s_M[tid][e] = (float)(dv * m[e]);
        }
        if (BOX) {
            const D3 f0 = load_pos(pos + (long long)r * P.rstride * P.ps, G.rbegin, P.ps);
            s_first[tid][0] = f0.x; s_first[tid][1] = f0.y; s_first[tid][2] = f0.z;
            s_cd[tid][0] = d[3]; s_cd[tid][1] = d[4]; s_cd[tid][2] = d[5];
        }
    }
    __syncthreads();
    const float* p = pos + (long long)r * P.rstride * P.ps;
    float* f = force + (long long)r * P.rstride * P.fs;
    const bool shared_arr = P.rstride == 0;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
        long long a = t0 + tid + (long long)i * 256;
        if (a >= P.span_end) continue;
        float ax = 0.f, ay = 0.f, az = 0.f;
        float px = 0.f, py = 0.f, pz = 0.f;
        if (P.any_rgyr) {
            if (P.ps == 4) {
                float4 v = __ldg(reinterpret_cast<const float4*>(p) + a);
                px = v.x; py = v.y; pz = v.z;
            } else {
                px = __ldg(p + a * 3); py = __ldg(p + a * 3 + 1); pz = __ldg(p + a * 3 + 2);
            }
        }
        bool any = false;
        for (int q = 0; q < P.n_ranges; ++q) {
            if (a >= s_b[q] && a < s_e[q]) {
                any = true;
                float k = s_k[q];
                float dx, dy, dz;   // r_i - c_g
                if (BOX) {   // r_i = the image nearest to the group's first atom, as in the moments
                    const D3 d = min_image(d3((double)px - s_first[q][0], (double)py - s_first[q][1], (double)pz - s_first[q][2]), P.box);
                    dx = (float)((s_first[q][0] + d.x) - s_cd[q][0]);
                    dy = (float)((s_first[q][1] + d.y) - s_cd[q][1]);
                    dz = (float)((s_first[q][2] + d.z) - s_cd[q][2]);
                } else {
                    dx = (px - s_chi[q][0]) - s_clo[q][0]; dy = (py - s_chi[q][1]) - s_clo[q][1]; dz = (pz - s_chi[q][2]) - s_clo[q][2];
                }
                if (s_shape[q]) {   // gyration-tensor shape CV: w M (r - c), M symmetric
                    ax += s_M[q][0] * dx + s_M[q][1] * dy + s_M[q][2] * dz;
                    ay += s_M[q][1] * dx + s_M[q][3] * dy + s_M[q][4] * dz;
                    az += s_M[q][2] * dx + s_M[q][4] * dy + s_M[q][5] * dz;
                } else {
                    ax += s_v[q][0] + k * dx;
                    ay += s_v[q][1] + k * dy;
                    az += s_v[q][2] + k * dz;
                }
            }
        }
        if (!any) continue;
        float w = P.atom_weight ? __ldg(P.atom_weight + a) : 1.f;
        ax *= w; ay *= w; az *= w;
        if (shared_arr) {
            force_add(f + a * P.fs, ax, ay, az, P.fs);
        } else if (P.fs == 4) {
            float4* fp = reinterpret_cast<float4*>(f) + a;
            float4 v = *fp;
            v.x += ax; v.y += ay; v.z += az;
            *fp = v;
        } else {
            f[a * 3] += ax; f[a * 3 + 1] += ay; f[a * 3 + 2] += az;
        }
    }
}

cudaError_t psg_launch_cv_eval(psg_ctx* c, const float* d_pos, float* d_xi, float* d_jac) {
    const SysParams& P = c->sys;
    if (P.n_ranges > 0) {
        dim3 g(P.range_blocks, P.R);
        if (P.has_box) k_range_moments<true><<<g, PSG_RANGE_THREADS, 0, c->stream>>>(P, d_pos, c->d_rpart);
        else k_range_moments<false><<<g, PSG_RANGE_THREADS, 0, c->stream>>>(P, d_pos, c->d_rpart);
        c->launches++;
    }
    if (P.any_shape_range) {
        dim3 g(P.range_blocks, P.R);
        if (P.has_box) k_range_second<true><<<g, 256, 0, c->stream>>>(P, d_pos, c->d_rpart2);
        else k_range_second<false><<<g, 256, 0, c->stream>>>(P, d_pos, c->d_rpart2);
        c->launches++;
    }
    if (psg_lean_layout(c)) {
        k_cv_eval_lean<<<(P.R + CVL_RB - 1) / CVL_RB, CVL_RB * P.n_cv * 2, 0, c->stream>>>(P, d_pos, d_xi, d_jac, c->d_jac);
        c->launches++;
        return cudaGetLastError();
    }
    k_cv_eval<<<(P.R + 7) / 8, 256, 0, c->stream>>>(P, d_pos, c->d_rpart, d_xi, d_jac, c->d_jac, c->d_gdesc,
                                                    P.any_shape_range ? c->d_rpart2 : nullptr, P.any_shape_range ? c->d_gdesc_m : nullptr);
    c->launches++;
    cudaError_t e = cudaGetLastError();
    // DistanceToInterface: k_cv_eval left 0 in its column and zero Jacobians for its mobile slots; its own kernels fill the column
    if (e == cudaSuccess && c->dti_cv >= 0) e = psg_launch_dti_eval(c, d_pos, d_xi, P.n_cv, c->dti_cv);
    return e;
}

cudaError_t psg_launch_apply(psg_ctx* c, const float* d_pos, const float* d_dVdxi, float* d_force) {
    const SysParams& P = c->sys;
    if (P.n_slots > 0) {
        long long n = (long long)P.R * P.n_slots;
        k_apply_sparse<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(P, c->d_jac, d_dVdxi, d_force);
        c->launches++;
    }
    if (P.n_ranges > 0) {
        dim3 g(P.range_blocks, P.R);
        if (P.has_box) k_apply_dense<true><<<g, 256, 0, c->stream>>>(P, d_pos, c->d_gdesc, d_dVdxi, d_force, P.any_shape_range ? c->d_gdesc_m : nullptr);
        else k_apply_dense<false><<<g, 256, 0, c->stream>>>(P, d_pos, c->d_gdesc, d_dVdxi, d_force, P.any_shape_range ? c->d_gdesc_m : nullptr);
        c->launches++;
    }
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && c->dti_cv >= 0) e = psg_launch_dti_apply(c, d_pos, d_dVdxi, P.n_cv, c->dti_cv, d_force);
    return e;
}
