// geom.cuh -- device-side collective variables and analytic Jacobians.
// Inputs are binary32 coordinates; the geometry of a handful of group centres is done in
// binary64 registers and rounded once on store: it is ~200 flops per
// CV, invisible next to the hill sum, and removes the near-degenerate fp32 failures.
// CVs: PAPER.md:L185-L189 (Sec. 2.2). Written from the definitions; shares nothing with oracle/.
#pragma once
#include "internal.h"

struct D3 {
    double x, y, z;
};
__device__ __forceinline__ D3 d3(double x, double y, double z) { return D3{x, y, z}; }
__device__ __forceinline__ D3 operator-(D3 a, D3 b) { return D3{a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ D3 operator+(D3 a, D3 b) { return D3{a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ D3 operator*(double s, D3 a) { return D3{s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ double dot(D3 a, D3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
__device__ __forceinline__ D3 cross(D3 a, D3 b) {
    return D3{a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}

// Minimum-image convention (reading R-MI; the paper is silent on periodic positions): box = nullptr or the three
// orthorhombic box lengths, 0 = open in that direction.  d <- d - L rint(d / L).
__device__ __forceinline__ D3 min_image(D3 d, const double* box) {
    if (box) {
        if (box[0] > 0.0) d.x -= box[0] * rint(d.x / box[0]);
        if (box[1] > 0.0) d.y -= box[1] * rint(d.y / box[1]);
        if (box[2] > 0.0) d.z -= box[2] * rint(d.z / box[2]);
    }
    return d;
}
__device__ __forceinline__ const double* sys_box(const SysParams& P) { return P.has_box ? P.box : nullptr; }

// xi = f(c_0..c_3) and, if JAC, dxi/dc_g into dc[0..3] (zero where undefined). Displacements between centres are nearest
// images when a box is given.
template <bool JAC>
__device__ __forceinline__ double cv_from_centers(int type, int axis, const D3* c, D3* dc, const double* box = nullptr) {
    if (JAC) {
#pragma unroll
        for (int g = 0; g < 4; ++g) dc[g] = d3(0, 0, 0);
    }
    if (type == PSG_CV_DISTANCE) {
        D3 d = min_image(c[1] - c[0], box);
        double r = sqrt(dot(d, d));
        if (JAC && r > 0.0) {
            double ir = 1.0 / r;
            dc[1] = ir * d;
            dc[0] = (-ir) * d;
        }
        return r;
    }
    if (type == PSG_CV_ANGLE) {
        // vertex at the second group; theta = atan2(|u x v|, u.v)
        D3 u = min_image(c[0] - c[1], box), v = min_image(c[2] - c[1], box);
        D3 n = cross(u, v);
        double nn = sqrt(dot(n, n));
        double th = atan2(nn, dot(u, v));
        if (JAC && nn > 0.0) {
            // moving c0 inside the plane, perpendicular to u: direction (u x n), length 1/|u|
            dc[0] = (1.0 / (dot(u, u) * nn)) * cross(u, n);
            dc[2] = (-1.0 / (dot(v, v) * nn)) * cross(v, n);
            dc[1] = (-1.0) * (dc[0] + dc[2]);
        }
        return th;
    }
    if (type == PSG_CV_DIHEDRAL) {
        D3 b1 = min_image(c[1] - c[0], box), b2 = min_image(c[2] - c[1], box), b3 = min_image(c[3] - c[2], box);
        D3 m = cross(b1, b2), n = cross(b2, b3);
        double l2 = dot(b2, b2), l = sqrt(l2);
        double phi = atan2(l * dot(b1, n), dot(m, n));
        if (JAC) {
            double mm = dot(m, m), nn = dot(n, n);
            if (mm > 0.0 && nn > 0.0) {
                D3 f0 = (-l / mm) * m;         // end atoms move the angle only through their own plane normal
                D3 f3 = (l / nn) * n;
                double p = dot(b1, b2) / l2, q = dot(b3, b2) / l2;
                dc[0] = f0;
                dc[3] = f3;
                dc[1] = (-(1.0 + p)) * f0 + q * f3;   // torque balance about the b2 axis
                dc[2] = (-(1.0 + q)) * f3 + p * f0;
            }
        }
        return phi;
    }
    if (type == PSG_CV_DISPLACEMENT) {   // PAPER.md:L185 Displacement: component `axis` of c2 - c1
        const D3 d = min_image(c[1] - c[0], box);
        if (JAC) {
            dc[1] = d3(axis == 0 ? 1.0 : 0.0, axis == 1 ? 1.0 : 0.0, axis == 2 ? 1.0 : 0.0);
            dc[0] = (-1.0) * dc[1];
        }
        return axis == 0 ? d.x : (axis == 1 ? d.y : d.z);
    }
    if (type == PSG_CV_COM_COMPONENT) {
        if (JAC) dc[0] = d3(axis == 0 ? 1.0 : 0.0, axis == 1 ? 1.0 : 0.0, axis == 2 ? 1.0 : 0.0);
        return axis == 0 ? c[0].x : (axis == 1 ? c[0].y : c[0].z);
    }
    return 0.0;
}

// force[i] += (fx, fy, fz) where several CVs / walkers may hit the same atom (A8): fire-and-forget L2 atomics.  A float4
// force record is 16-byte aligned, so x and y go as ONE vector reduction (red.global.add.v2.f32) and z as a scalar one; w is
// never touched.  Records of 3 floats are only 4-byte aligned: three scalar reductions.
__device__ __forceinline__ void force_add(float* __restrict__ fa, float fx, float fy, float fz, int fs) {
    if (fs == 4) {
        atomicAdd(reinterpret_cast<float2*>(fa), make_float2(fx, fy));
        atomicAdd(fa + 2, fz);
    } else {
        atomicAdd(fa, fx);
        atomicAdd(fa + 1, fy);
        atomicAdd(fa + 2, fz);
    }
}

// Reciprocal and reciprocal square root in binary64 without the library's subroutine calls: the hardware seed (MUFU.RCP64H /
// RSQ64H, ~20 bits) refined by two Newton steps (~1 ulp).  Several of them overlap in one thread (no call boundary), which is
// what shortens the Jacobian chain of the fused step's prologue.  x must be finite and > 0.
__device__ __forceinline__ double fast_rcp(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(fma(-x, r, 1.0), r, r);
    r = fma(fma(-x, r, 1.0), r, r);
    return r;
}
__device__ __forceinline__ double fast_rsqrt(double x) {
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(0.5 * r, fma(-x * r, r, 1.0), r);
    r = fma(0.5 * r, fma(-x * r, r, 1.0), r);
    return r;
}

// dxi/dc_g alone (no value, no box), same formulas as cv_from_centers<true> with fast_rcp / fast_rsqrt in place of divisions
// and square roots; zero where undefined.  Used by the fused metadynamics step, whose value threads take the atan2 chain.
__device__ __forceinline__ void cv_jacobian_only(int type, int axis, const D3* c, D3* dc) {
#pragma unroll
    for (int g = 0; g < 4; ++g) dc[g] = d3(0, 0, 0);
    if (type == PSG_CV_DISTANCE) {
        const D3 d = c[1] - c[0];
        const double r2 = dot(d, d);
        if (r2 > 0.0) {
            const double ir = fast_rsqrt(r2);
            dc[1] = ir * d;
            dc[0] = (-ir) * d;
        }
    } else if (type == PSG_CV_ANGLE) {
        const D3 u = c[0] - c[1], v = c[2] - c[1];
        const D3 n = cross(u, v);
        const double n2 = dot(n, n);
        if (n2 > 0.0) {
            const double inn = fast_rsqrt(n2);
            dc[0] = (fast_rcp(dot(u, u)) * inn) * cross(u, n);
            dc[2] = (-fast_rcp(dot(v, v)) * inn) * cross(v, n);
            dc[1] = (-1.0) * (dc[0] + dc[2]);
        }
    } else if (type == PSG_CV_DIHEDRAL) {
        const D3 b1 = c[1] - c[0], b2 = c[2] - c[1], b3 = c[3] - c[2];
        const D3 m = cross(b1, b2), n = cross(b2, b3);
        const double l2 = dot(b2, b2), mm = dot(m, m), nn = dot(n, n);
        if (mm > 0.0 && nn > 0.0) {
            const double il2 = fast_rcp(l2), l = l2 * fast_rsqrt(l2);
            const D3 f0 = (-l * fast_rcp(mm)) * m, f3 = (l * fast_rcp(nn)) * n;
            const double p = dot(b1, b2) * il2, q = dot(b3, b2) * il2;
            dc[0] = f0;
            dc[3] = f3;
            dc[1] = (-(1.0 + p)) * f0 + q * f3;
            dc[2] = (-(1.0 + q)) * f3 + p * f0;
        }
    } else if (type == PSG_CV_DISPLACEMENT) {
        dc[1] = d3(axis == 0 ? 1.0 : 0.0, axis == 1 ? 1.0 : 0.0, axis == 2 ? 1.0 : 0.0);
        dc[0] = (-1.0) * dc[1];
    } else if (type == PSG_CV_COM_COMPONENT) {
        dc[0] = d3(axis == 0 ? 1.0 : 0.0, axis == 1 ? 1.0 : 0.0, axis == 2 ? 1.0 : 0.0);
    }
}

// the raw binary32 record of an atom (w of a 3-float record reads as 0): lets a load be issued long before its use
__device__ __forceinline__ float4 load_pos_raw(const float* __restrict__ p, long long atom, int ps) {
    if (ps == 4) return __ldg(reinterpret_cast<const float4*>(p) + atom);
    const float* q = p + atom * 3;
    return make_float4(__ldg(q), __ldg(q + 1), __ldg(q + 2), 0.f);
}
__device__ __forceinline__ D3 load_pos(const float* __restrict__ p, long long atom, int ps) {
    if (ps == 4) {
        float4 v = __ldg(reinterpret_cast<const float4*>(p) + atom);
        return d3((double)v.x, (double)v.y, (double)v.z);
    }
    const float* q = p + atom * 3;
    return d3((double)__ldg(q), (double)__ldg(q + 1), (double)__ldg(q + 2));
}

// ---- gyration-tensor shape CVs (reading R-SHAPE) ---------------------------------------
// A symmetric 3x3 matrix held as six scalars, diagonalised by cyclic Jacobi rotations in registers: each rotation acts on
// the 2x2 block (app, aqq, apq), the two entries (arp, arq) that couple it to the third axis, and columns p, q of the
// eigenvector matrix.  t = tan(theta) is the smaller root, so the iteration converges quadratically (<= 6 sweeps here).
__device__ __forceinline__ void jacobi_rotate(double& app, double& aqq, double& apq, double& arp, double& arq,
                                              D3& vp, D3& vq) {
    if (apq == 0.0) return;
    const double th = (aqq - app) / (2.0 * apq);
    const double t = copysign(1.0, th) / (fabs(th) + sqrt(th * th + 1.0));
    const double c = 1.0 / sqrt(t * t + 1.0), s = t * c;
    app -= t * apq; aqq += t * apq; apq = 0.0;
    const double rp = c * arp - s * arq, rq = s * arp + c * arq;
    arp = rp; arq = rq;
    const D3 np_ = c * vp - s * vq, nq = s * vp + c * vq;
    vp = np_; vq = nq;
}
__device__ __forceinline__ void swap_desc(double& la, double& lb, D3& va, D3& vb) {
    if (la < lb) { double t = la; la = lb; lb = t; D3 v = va; va = vb; vb = v; }
}
// eigenvalues l[0] >= l[1] >= l[2] of {xx, xy, xz, yy, yz, zz} and their unit eigenvectors
__device__ __forceinline__ void sym3_eigen(const double* m, double* l, D3* v) {
    double xx = m[0], xy = m[1], xz = m[2], yy = m[3], yz = m[4], zz = m[5];
    D3 vx = d3(1, 0, 0), vy = d3(0, 1, 0), vz = d3(0, 0, 1);
    for (int sweep = 0; sweep < 16; ++sweep) {
        const double off = xy * xy + xz * xz + yz * yz;
        if (off <= 1e-60 * (xx * xx + yy * yy + zz * zz)) break;
        jacobi_rotate(xx, yy, xy, xz, yz, vx, vy);
        jacobi_rotate(xx, zz, xz, xy, yz, vx, vz);
        jacobi_rotate(yy, zz, yz, xy, xz, vy, vz);
    }
    swap_desc(xx, yy, vx, vy); swap_desc(yy, zz, vy, vz); swap_desc(xx, yy, vx, vy);
    l[0] = xx; l[1] = yy; l[2] = zz; v[0] = vx; v[1] = vy; v[2] = vz;
}
__device__ __forceinline__ bool is_shape_cv(int type) { return type >= PSG_CV_PRINCIPAL_MOMENT && type <= PSG_CV_SHAPE_ANISOTROPY; }
// value of the shape CV and g[k] = d xi / d l_k
__device__ __forceinline__ double shape_from_eigenvalues(int type, int axis, const double* l, double* g) {
    g[0] = g[1] = g[2] = 0.0;
    if (type == PSG_CV_PRINCIPAL_MOMENT) {
        g[0] = axis == 0 ? 1.0 : 0.0; g[1] = axis == 1 ? 1.0 : 0.0; g[2] = axis == 2 ? 1.0 : 0.0;
        return axis == 0 ? l[0] : axis == 1 ? l[1] : l[2];
    }
    const double b = l[0] - 0.5 * (l[1] + l[2]), a = l[1] - l[2];
    if (type == PSG_CV_ASPHERICITY) { g[0] = 1.0; g[1] = -0.5; g[2] = -0.5; return b; }
    if (type == PSG_CV_ACYLINDRICITY) { g[1] = 1.0; g[2] = -1.0; return a; }
    const double tr = l[0] + l[1] + l[2], num = b * b + 0.75 * a * a;   // PSG_CV_SHAPE_ANISOTROPY
    if (!(tr > 0.0)) return 0.0;
    const double i2 = 1.0 / (tr * tr), k = 2.0 * num * i2 / tr;
    g[0] = 2.0 * b * i2 - k; g[1] = (1.5 * a - b) * i2 - k; g[2] = (-1.5 * a - b) * i2 - k;
    return num * i2;
}
#define PSG_COEF_SHAPE (-1.0)   // WarpCvSmem::coef of a shape-CV group: sec[] holds (2/W) sum_k g_k v_k v_k^T

// atom of slot s of replica r: a shared index list is read from the kernel parameters (no global load ahead of the gather:
// with a cold L2 the index load and the position load were two dependent DRAM round trips), a per-replica one from memory
__device__ __forceinline__ int slot_atom_of(const SysParams& P, int r, int s) {
    return P.per_rep ? __ldg(P.slot_atom + (long long)r * P.n_slots + s) : P.slot_atom_c[s];
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Per-warp shared scratch for one replica's CV evaluation.
struct WarpCvSmem {
    double cen[PSG_MAX_GROUPS_TOTAL][4];   // cx cy cz W
    double m2[PSG_MAX_GROUPS_TOTAL];       // sum w |r|^2 (RGYR groups)
    double v[PSG_MAX_GROUPS_TOTAL][3];     // dxi/dc_g / W_g
    double coef[PSG_MAX_GROUPS_TOTAL];     // RGYR: 1/(W Rg); shape CVs: PSG_COEF_SHAPE; else 0
    double sec[PSG_MAX_GROUPS_TOTAL][6];   // shape CVs: sum w x'x'^T (x' = r - first atom), then the matrix M of d xi/d r_i = w_i M (r_i - c)
    double xi[PSG_MAX_CV];
};

// One warp evaluates all CVs of replica r.
//  - group centres: explicit groups gathered from pos by one lane per group; range groups from the
//    partial moments written by k_range_moments (rpart != nullptr when n_ranges > 0)
//  - lane k < n_cv computes CV k (value, and with JAC the per-group derivative)
// On return (after __syncwarp) sm.xi / sm.v / sm.coef / sm.cen are valid for the whole warp.
template <bool JAC>
__device__ __forceinline__ void warp_cv_eval(const SysParams& P, int r, const float* __restrict__ pos,
                                             const double* __restrict__ rpart, WarpCvSmem& sm, int lane,
                                             const double* __restrict__ rpart2 = nullptr) {
    const float* p = pos + (long long)r * P.rstride * P.ps;
    // range groups: all lanes sum the block partials (fixed order => deterministic)
    for (int q = 0; q < P.n_ranges; ++q) {
        const double* src = rpart + ((long long)r * P.n_ranges + q) * P.range_blocks * PSG_MOM;
        double a[PSG_MOM] = {0, 0, 0, 0, 0};
        for (int b = lane; b < P.range_blocks; b += 32) {
#pragma unroll
            for (int i = 0; i < PSG_MOM; ++i) a[i] += __ldcg(src + (long long)b * PSG_MOM + i);
        }
#pragma unroll
        for (int i = 0; i < PSG_MOM; ++i) a[i] = warp_sum(a[i]);
        if (lane == 0) {
            int gid = P.range_gid[q];
            double iw = 1.0 / a[0];
            sm.cen[gid][0] = a[1] * iw; sm.cen[gid][1] = a[2] * iw; sm.cen[gid][2] = a[3] * iw; sm.cen[gid][3] = a[0];
            sm.m2[gid] = a[4];
        }
        // a gyration-tensor shape CV over this range: the six second moments about the range's first atom (k_range_second),
        // S = sum w x'x'^T / W - c'c'^T with c' = c - first, as for explicit groups
        const int gid_q = P.range_gid[q];
        if (rpart2 && is_shape_cv(P.cv[P.grp[gid_q].cv].type)) {
            const double* s2 = rpart2 + ((long long)r * P.n_ranges + q) * P.range_blocks * 6;
            double e[6] = {0, 0, 0, 0, 0, 0};
            for (int b = lane; b < P.range_blocks; b += 32) {
#pragma unroll
                for (int i = 0; i < 6; ++i) e[i] += __ldcg(s2 + (long long)b * 6 + i);
            }
#pragma unroll
            for (int i = 0; i < 6; ++i) e[i] = warp_sum(e[i]);
            if (lane == 0) {
                const D3 first = load_pos(p, P.grp[gid_q].rbegin, P.ps);
                const double iw = 1.0 / a[0];
                const D3 cp = d3(a[1] * iw - first.x, a[2] * iw - first.y, a[3] * iw - first.z);
                sm.sec[gid_q][0] = e[0] * iw - cp.x * cp.x; sm.sec[gid_q][1] = e[1] * iw - cp.x * cp.y; sm.sec[gid_q][2] = e[2] * iw - cp.x * cp.z;
                sm.sec[gid_q][3] = e[3] * iw - cp.y * cp.y; sm.sec[gid_q][4] = e[4] * iw - cp.y * cp.z; sm.sec[gid_q][5] = e[5] * iw - cp.z * cp.z;
            }
        }
    }
    // explicit groups: lane j gathers group j
    if (lane < P.n_groups && !P.grp[lane].is_range) {
        const GroupDev& G = P.grp[lane];
        double sx = 0, sy = 0, sz = 0, sw = 0, s2 = 0;
        double q[6] = {0, 0, 0, 0, 0, 0};
        const bool shape = is_shape_cv(P.cv[G.cv].type);
        const double* box = sys_box(P);
        const D3 first = load_pos(p, slot_atom_of(P, r, G.begin), P.ps);
        for (int i = 0; i < G.size; ++i) {
            int s = G.begin + i;
            D3 x = load_pos(p, slot_atom_of(P, r, s), P.ps);
            if (box) x = first + min_image(x - first, box);   // the image nearest to the group's first atom
            double w = P.slot_weight ? (double)P.slot_weight[s] : 1.0;
            sx += w * x.x; sy += w * x.y; sz += w * x.z; sw += w;
            s2 += w * dot(x, x);
            if (shape) {   // second moments about the first atom: no cancellation against |c|^2 far from the origin
                const D3 e = x - first;
                q[0] += w * e.x * e.x; q[1] += w * e.x * e.y; q[2] += w * e.x * e.z;
                q[3] += w * e.y * e.y; q[4] += w * e.y * e.z; q[5] += w * e.z * e.z;
            }
        }
        double iw = 1.0 / sw;
        sm.cen[lane][0] = sx * iw; sm.cen[lane][1] = sy * iw; sm.cen[lane][2] = sz * iw; sm.cen[lane][3] = sw;
        sm.m2[lane] = s2;
        if (shape) {   // S = sum w x'x'^T / W - c'c'^T, c' = c - first
            const D3 cp = d3(sx * iw - first.x, sy * iw - first.y, sz * iw - first.z);
            sm.sec[lane][0] = q[0] * iw - cp.x * cp.x; sm.sec[lane][1] = q[1] * iw - cp.x * cp.y; sm.sec[lane][2] = q[2] * iw - cp.x * cp.z;
            sm.sec[lane][3] = q[3] * iw - cp.y * cp.y; sm.sec[lane][4] = q[4] * iw - cp.y * cp.z; sm.sec[lane][5] = q[5] * iw - cp.z * cp.z;
        }
    }
    __syncwarp();
    if (lane < P.n_cv) {
        const CvDev& C = P.cv[lane];
        int g0 = C.gid0;
        if (C.type == PSG_CV_RGYR) {
            // Rg^2 = sum w|r|^2 / W - |c|^2 (binary64 moments); dRg/dr_i = w_i (r_i - c) / (W Rg)
            D3 c = d3(sm.cen[g0][0], sm.cen[g0][1], sm.cen[g0][2]);
            double W = sm.cen[g0][3];
            double rg2 = sm.m2[g0] / W - dot(c, c);
            double rg = rg2 > 0.0 ? sqrt(rg2) : 0.0;
            sm.xi[lane] = rg;
            sm.coef[g0] = rg > 0.0 ? 1.0 / (W * rg) : 0.0;
            sm.v[g0][0] = sm.v[g0][1] = sm.v[g0][2] = 0.0;
        } else if (is_shape_cv(C.type)) {
            // eigenvalues of the gyration tensor; d l_k / d r_i = (2 w_i / W)(v_k . (r_i - c)) v_k, chained through g = d xi / d l
            double l[3], g[3];
            D3 v[3];
            sym3_eigen(sm.sec[g0], l, v);
            sm.xi[lane] = shape_from_eigenvalues(C.type, C.axis, l, g);
            const double k = 2.0 / sm.cen[g0][3];
            double M[6] = {0, 0, 0, 0, 0, 0};
#pragma unroll
            for (int e = 0; e < 3; ++e) {
                const double ge = k * g[e];
                M[0] += ge * v[e].x * v[e].x; M[1] += ge * v[e].x * v[e].y; M[2] += ge * v[e].x * v[e].z;
                M[3] += ge * v[e].y * v[e].y; M[4] += ge * v[e].y * v[e].z; M[5] += ge * v[e].z * v[e].z;
            }
#pragma unroll
            for (int e = 0; e < 6; ++e) sm.sec[g0][e] = M[e];
            sm.coef[g0] = PSG_COEF_SHAPE;
            sm.v[g0][0] = sm.v[g0][1] = sm.v[g0][2] = 0.0;
        } else {
            D3 c[4], dc[4];
#pragma unroll
            for (int g = 0; g < 4; ++g)
                c[g] = g < C.n_groups ? d3(sm.cen[g0 + g][0], sm.cen[g0 + g][1], sm.cen[g0 + g][2]) : d3(0, 0, 0);
            sm.xi[lane] = cv_from_centers<JAC>(C.type, C.axis, c, dc, sys_box(P));
            if (JAC) {
#pragma unroll
                for (int g = 0; g < 4; ++g)
                    if (g < C.n_groups) {
                        double iw = 1.0 / sm.cen[g0 + g][3];
                        sm.v[g0 + g][0] = dc[g].x * iw; sm.v[g0 + g][1] = dc[g].y * iw; sm.v[g0 + g][2] = dc[g].z * iw;
                        sm.coef[g0 + g] = 0.0;
                    }
            }
        }
    }
    __syncwarp();
}

// The centres (and total weights) of the groups of CV C of replica r, gathered by ONE thread with the arithmetic of
// warp_cv_eval's gather (same sums, same order, same division: a CV value computed from them keeps its bits).  Explicit groups,
// no box.  Used by the thread-per-(replica, CV) kernels.
__device__ __forceinline__ void thread_group_centres(const SysParams& P, int r, const CvDev& C, const float* __restrict__ p, D3 (&c)[4],
                                                     double (&Wg)[4]) {
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        c[g] = d3(0, 0, 0);
        Wg[g] = 1.0;
        if (g < C.n_groups) {
            const GroupDev& Gd = P.grp[C.gid0 + g];
            double sx = 0, sy = 0, sz = 0, sw = 0;
#pragma unroll 4
            for (int i = 0; i < Gd.size; ++i) {
                const int s = Gd.begin + i;
                const D3 x = load_pos(p, slot_atom_of(P, r, s), P.ps);
                const double w = P.slot_weight ? (double)P.slot_weight[s] : 1.0;
                sx += w * x.x; sy += w * x.y; sz += w * x.z; sw += w;
            }
            const double iw = 1.0 / sw;
            c[g] = d3(sx * iw, sy * iw, sz * iw);
            Wg[g] = sw;
        }
    }
}

// d(xi)/d(r_slot) for an explicit slot s (weight w_s) given the per-group vector
__device__ __forceinline__ D3 slot_jacobian(const SysParams& P, int r, const float* __restrict__ pos,
                                            const WarpCvSmem& sm, int s) {
    int gid = P.slot_gid_c[s];
    double w = P.slot_weight ? (double)P.slot_weight[s] : 1.0;
    D3 j = d3(w * sm.v[gid][0], w * sm.v[gid][1], w * sm.v[gid][2]);
    if (sm.coef[gid] != 0.0) {   // explicit RGYR group: w (r - c) / (W Rg); shape-CV group: w M (r - c)
        D3 x = load_pos(pos + (long long)r * P.rstride * P.ps, slot_atom_of(P, r, s), P.ps);
        if (P.has_box) {
            const D3 first = load_pos(pos + (long long)r * P.rstride * P.ps, slot_atom_of(P, r, P.grp[gid].begin), P.ps);
            x = first + min_image(x - first, P.box);
        }
        const D3 d = d3(x.x - sm.cen[gid][0], x.y - sm.cen[gid][1], x.z - sm.cen[gid][2]);
        if (sm.coef[gid] == PSG_COEF_SHAPE) {   // w M (r - c), M symmetric
            const double* M = sm.sec[gid];
            j = d3(w * (M[0] * d.x + M[1] * d.y + M[2] * d.z), w * (M[1] * d.x + M[3] * d.y + M[4] * d.z),
                   w * (M[2] * d.x + M[4] * d.y + M[5] * d.z));
        } else {
            const double k = w * sm.coef[gid];
            j = d3(k * d.x, k * d.y, k * d.z);
        }
    }
    return j;
}
