// abf_estimate.cu -- ABF instantaneous-force estimator (PAPER.md:L143 only cites its reference [43], so
// this is DESIGN.md reading R-ABF-EST):
//   J[k][i] = d xi_k / d r_i,  p_i = m_i v_i,  G = J J^T,  b = J p,  G W = b,
//   fsample = (3/2 W(t) - 2 W(t - dt) + 1/2 W(t - 2 dt)) / dt + Fbias_prev
// One warp per replica (warps loop): CVs and Jacobians as in k_cv_eval (binary64 registers), slot Jacobians to shared
// memory, b and the n_cv x n_cv Gram matrix by lanes striding the slots (an atom shared by two CVs couples them), a
// <= 4 x 4 solve with partial pivoting by lane 0, history in ctx-owned binary64 buffers.  Latency-bound like every
// per-replica kernel here; explicit groups only.
#include "geom.cuh"

struct AbfEstArgs {
    const float* pos;
    const float* vel;        // layout of pos
    const float* mass;       // [N]
    const float* fbias_prev; // [R][n_cv], nullable
    double* whist;           // [R][2][n_cv]
    float* fsample;          // [R][n_cv]
    double dt;
    int first;
};

struct EstSmem {
    WarpCvSmem cv;
    double j[PSG_MAX_SLOTS][3];
    int atom[PSG_MAX_SLOTS];
    int cvk[PSG_MAX_SLOTS];   // CV that owns the slot (cached: the pair loop must not chase global / parameter loads)
    double M[PSG_MAX_CV][PSG_MAX_CV + 1], W[PSG_MAX_CV];   // lane 0's augmented matrix and solution: run-time indexed, so in
                                                           // shared memory (in registers they would be demoted to local memory)
};

__global__ void __launch_bounds__(128, 8) k_abf_estimate(const __grid_constant__ SysParams P, const __grid_constant__ AbfEstArgs A) {
    __shared__ EstSmem sm[4];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    EstSmem& S = sm[wid];
    const int n_cv = P.n_cv;
    for (int r = blockIdx.x * 4 + wid; r < P.R; r += gridDim.x * 4) {
        warp_cv_eval<true>(P, r, A.pos, nullptr, S.cv, lane);
        const int* sa = P.slot_atom + (P.per_rep ? (long long)r * P.n_slots : 0);
        const float* v = A.vel + (long long)r * P.rstride * P.ps;
        double b[PSG_MAX_CV] = {0, 0, 0, 0};
        for (int s = lane; s < P.n_slots; s += 32) {
            const D3 j = slot_jacobian(P, r, A.pos, S.cv, s);
            const int a = sa[s];
            S.j[s][0] = j.x; S.j[s][1] = j.y; S.j[s][2] = j.z;
            S.atom[s] = a;
            const double m = (double)__ldg(A.mass + a);
            const double px = m * (double)v[(long long)a * P.ps], py = m * (double)v[(long long)a * P.ps + 1],
                         pz = m * (double)v[(long long)a * P.ps + 2];
            const int k = P.grp[P.slot_gid[s]].cv;
            S.cvk[s] = k;
            const double t = j.x * px + j.y * py + j.z * pz;
#pragma unroll
            for (int q = 0; q < PSG_MAX_CV; ++q) b[q] += q == k ? t : 0.0;
        }
        __syncwarp();
        double G[PSG_MAX_CV][PSG_MAX_CV];
#pragma unroll
        for (int k = 0; k < PSG_MAX_CV; ++k)
#pragma unroll
            for (int l = 0; l < PSG_MAX_CV; ++l) G[k][l] = 0.0;
        for (int s = lane; s < P.n_slots; s += 32) {
            const int k = S.cvk[s], a = S.atom[s];
            for (int s2 = 0; s2 < P.n_slots; ++s2) {
                if (S.atom[s2] != a) continue;
                const int l = S.cvk[s2];
                const double t = S.j[s][0] * S.j[s2][0] + S.j[s][1] * S.j[s2][1] + S.j[s][2] * S.j[s2][2];
#pragma unroll
                for (int q = 0; q < PSG_MAX_CV; ++q)
#pragma unroll
                    for (int u = 0; u < PSG_MAX_CV; ++u) G[q][u] += (q == k && u == l) ? t : 0.0;
            }
        }
#pragma unroll
        for (int k = 0; k < PSG_MAX_CV; ++k) {
            b[k] = warp_sum(b[k]);
#pragma unroll
            for (int l = 0; l < PSG_MAX_CV; ++l) G[k][l] = warp_sum(G[k][l]);
        }
        if (lane == 0) {
            double (*M)[PSG_MAX_CV + 1] = S.M;
            double* W = S.W;
            bool ok = true;
#pragma unroll
            for (int k = 0; k < PSG_MAX_CV; ++k) {
#pragma unroll
                for (int l = 0; l < PSG_MAX_CV; ++l) M[k][l] = G[k][l];
                M[k][PSG_MAX_CV] = b[k];
                W[k] = 0.0;
            }
            for (int k = 0; k < n_cv; ++k) M[k][n_cv] = M[k][PSG_MAX_CV];   // the right-hand side next to the n_cv columns
            for (int c = 0; c < n_cv && ok; ++c) {   // Gaussian elimination, partial pivoting
                int piv = c;
                for (int k = c + 1; k < n_cv; ++k)
                    if (fabs(M[k][c]) > fabs(M[piv][c])) piv = k;
                if (!(fabs(M[piv][c]) > 0.0)) { ok = false; break; }
                if (piv != c)
                    for (int l = 0; l <= n_cv; ++l) { double t = M[c][l]; M[c][l] = M[piv][l]; M[piv][l] = t; }
                for (int k = c + 1; k < n_cv; ++k) {
                    const double f = M[k][c] / M[c][c];
                    for (int l = c; l <= n_cv; ++l) M[k][l] -= f * M[c][l];
                }
            }
            if (ok)
                for (int k = n_cv - 1; k >= 0; --k) {
                    double s = M[k][n_cv];
                    for (int l = k + 1; l < n_cv; ++l) s -= M[k][l] * W[l];
                    W[k] = s / M[k][k];
                }
            double* h1 = A.whist + ((long long)r * 2 + 0) * n_cv;
            double* h2 = A.whist + ((long long)r * 2 + 1) * n_cv;
            for (int k = 0; k < n_cv; ++k) {
                if (A.first) { h1[k] = W[k]; h2[k] = W[k]; }
                const double dW = (1.5 * W[k] - 2.0 * h1[k] + 0.5 * h2[k]) / A.dt;
                const double fb = A.fbias_prev ? (double)A.fbias_prev[(long long)r * n_cv + k] : 0.0;
                A.fsample[(long long)r * n_cv + k] = (float)(dW + fb);
                h2[k] = h1[k];
                h1[k] = W[k];
            }
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------------------------
// The same estimator with ONE THREAD per (replica, CV) for explicit groups without a box and point-group CVs (the layout of
// k_abf_step_lean, abf_step.cu): the thread gathers the atoms of its CV's groups, takes the derivative (cv_jacobian_only: the
// estimator needs no CV value), forms its slots' Jacobians, its b_k = J_k . p and, after a barrier, row k of the Gram matrix;
// the thread of CV 0 solves the n_cv x n_cv system.  A warp instruction then carries 32 chains instead of 1-8: the
// warp-per-replica kernel above spends its time issuing binary64 instructions for a few live lanes (23 us for 4,096 replicas).
#define EST_RB 16   // replicas per CTA; block = EST_RB x n_cv threads
struct EstLeanRep {
    double M[PSG_MAX_CV][PSG_MAX_CV + 1], W[PSG_MAX_CV];
};
__global__ void __launch_bounds__(EST_RB * PSG_MAX_CV) k_abf_estimate_lean(const __grid_constant__ SysParams P, const __grid_constant__ AbfEstArgs A) {
    extern __shared__ __align__(16) unsigned char est_smem[];
    const int ns = P.n_slots, n_cv = P.n_cv;
    double* s_j = reinterpret_cast<double*>(est_smem);                       // [EST_RB][ns][3]
    EstLeanRep* s_rep = reinterpret_cast<EstLeanRep*>(s_j + (size_t)EST_RB * ns * 3);
    int* s_atom = reinterpret_cast<int*>(s_rep + EST_RB);                    // [EST_RB][ns]
    int* s_cvk = s_atom + EST_RB * ns;                                       // [EST_RB][ns]
    const int tid = threadIdx.x, rl = tid / n_cv, k = tid - rl * n_cv;
    const int r = blockIdx.x * EST_RB + rl;
    const bool live = r < P.R;
    const CvDev& C = P.cv[k];
    double* jr = s_j + (size_t)rl * ns * 3;
    int* ar = s_atom + rl * ns;
    int* kr = s_cvk + rl * ns;
    EstLeanRep& S = s_rep[rl];
    if (live) {
        const float* p = A.pos + (long long)r * P.rstride * P.ps;
        const float* v = A.vel + (long long)r * P.rstride * P.ps;
        D3 c[4], dc[4];
        double Wg[4];
        thread_group_centres(P, r, C, p, c, Wg);
        cv_jacobian_only(C.type, C.axis, c, dc);
        double b = 0.0;
#pragma unroll
        for (int g = 0; g < 4; ++g)
            if (g < C.n_groups) {
                const GroupDev& Gd = P.grp[C.gid0 + g];
                const double iw = 1.0 / Wg[g];
                for (int i = 0; i < Gd.size; ++i) {
                    const int s = Gd.begin + i, a = slot_atom_of(P, r, s);
                    const double w = P.slot_weight ? (double)P.slot_weight[s] : 1.0;
                    const double jx = w * (dc[g].x * iw), jy = w * (dc[g].y * iw), jz = w * (dc[g].z * iw);
                    jr[s * 3] = jx; jr[s * 3 + 1] = jy; jr[s * 3 + 2] = jz;
                    ar[s] = a; kr[s] = k;
                    const double m = (double)__ldg(A.mass + a);
                    const double px = m * (double)v[(long long)a * P.ps], py = m * (double)v[(long long)a * P.ps + 1],
                                 pz = m * (double)v[(long long)a * P.ps + 2];
                    b += jx * px + jy * py + jz * pz;
                }
            }
#pragma unroll
        for (int l = 0; l <= PSG_MAX_CV; ++l) S.M[k][l] = 0.0;
        S.M[k][n_cv] = b;
    }
    __syncthreads();
    if (live) {
        // row k of G = J J^T: this CV's slots against every slot on the same atom (an atom shared by two CVs couples them)
#pragma unroll
        for (int g = 0; g < 4; ++g)
            if (g < C.n_groups) {
                const GroupDev& Gd = P.grp[C.gid0 + g];
                for (int i = 0; i < Gd.size; ++i) {
                    const int s = Gd.begin + i, a = ar[s];
                    for (int s2 = 0; s2 < ns; ++s2) {
                        if (ar[s2] != a) continue;
                        S.M[k][kr[s2]] += jr[s * 3] * jr[s2 * 3] + jr[s * 3 + 1] * jr[s2 * 3 + 1] + jr[s * 3 + 2] * jr[s2 * 3 + 2];
                    }
                }
            }
    }
    __syncthreads();
    if (live && k == 0) {
        double (*M)[PSG_MAX_CV + 1] = S.M;
        double* W = S.W;
        bool ok = true;
        for (int q = 0; q < PSG_MAX_CV; ++q) W[q] = 0.0;
        for (int c0 = 0; c0 < n_cv && ok; ++c0) {   // Gaussian elimination, partial pivoting (as in k_abf_estimate)
            int piv = c0;
            for (int q = c0 + 1; q < n_cv; ++q)
                if (fabs(M[q][c0]) > fabs(M[piv][c0])) piv = q;
            if (!(fabs(M[piv][c0]) > 0.0)) { ok = false; break; }
            if (piv != c0)
                for (int l = 0; l <= n_cv; ++l) { double t = M[c0][l]; M[c0][l] = M[piv][l]; M[piv][l] = t; }
            for (int q = c0 + 1; q < n_cv; ++q) {
                const double f = M[q][c0] / M[c0][c0];
                for (int l = c0; l <= n_cv; ++l) M[q][l] -= f * M[c0][l];
            }
        }
        if (ok)
            for (int q = n_cv - 1; q >= 0; --q) {
                double t = M[q][n_cv];
                for (int l = q + 1; l < n_cv; ++l) t -= M[q][l] * W[l];
                W[q] = t / M[q][q];
            }
        double* h1 = A.whist + ((long long)r * 2 + 0) * n_cv;
        double* h2 = A.whist + ((long long)r * 2 + 1) * n_cv;
        for (int q = 0; q < n_cv; ++q) {
            if (A.first) { h1[q] = W[q]; h2[q] = W[q]; }
            const double dW = (1.5 * W[q] - 2.0 * h1[q] + 0.5 * h2[q]) / A.dt;
            const double fb = A.fbias_prev ? (double)A.fbias_prev[(long long)r * n_cv + q] : 0.0;
            A.fsample[(long long)r * n_cv + q] = (float)(dW + fb);
            h2[q] = h1[q];
            h1[q] = W[q];
        }
    }
}

cudaError_t psg_launch_abf_estimate(psg_ctx* c, const float* d_pos, const float* d_vel, const float* d_mass, double dt,
                                    const float* d_fbias_prev, float* d_fsample) {
    AbfEstArgs A{};
    A.pos = d_pos; A.vel = d_vel; A.mass = d_mass; A.fbias_prev = d_fbias_prev; A.whist = c->d_whist; A.fsample = d_fsample;
    A.dt = dt; A.first = c->est_first ? 1 : 0;
    if (psg_lean_layout(c)) {
        const int ns = c->sys.n_slots;
        const size_t smem = (size_t)EST_RB * ns * 3 * sizeof(double) + EST_RB * sizeof(EstLeanRep) + (size_t)2 * EST_RB * ns * sizeof(int);
        if (smem <= 48 * 1024) {
            k_abf_estimate_lean<<<(c->sys.R + EST_RB - 1) / EST_RB, EST_RB * c->sys.n_cv, smem, c->stream>>>(c->sys, A);
            c->launches++;
            c->est_first = false;
            return cudaGetLastError();
        }
    }
    int grid = (c->sys.R + 3) / 4;
    const int cap = c->sm_count * 8;
    if (grid > cap) grid = cap;
    k_abf_estimate<<<grid, 128, 0, c->stream>>>(c->sys, A);
    c->launches++;
    c->est_first = false;
    return cudaGetLastError();
}
