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

cudaError_t psg_launch_abf_estimate(psg_ctx* c, const float* d_pos, const float* d_vel, const float* d_mass, double dt,
                                    const float* d_fbias_prev, float* d_fsample) {
    AbfEstArgs A{};
    A.pos = d_pos; A.vel = d_vel; A.mass = d_mass; A.fbias_prev = d_fbias_prev; A.whist = c->d_whist; A.fsample = d_fsample;
    A.dt = dt; A.first = c->est_first ? 1 : 0;
    int grid = (c->sys.R + 3) / 4;
    const int cap = c->sm_count * 8;
    if (grid > cap) grid = cap;
    k_abf_estimate<<<grid, 128, 0, c->stream>>>(c->sys, A);
    c->launches++;
    c->est_first = false;
    return cudaGetLastError();
}
