// metad_grid.cu -- grid-stored metadynamics ("storing the bias potentials ... on a pre-defined grid";
// SURVEY NEXT-2; reading R-GRID).  First version, calls of its own (psg_metad_grid_*):
//   k_grid_eval     thread per walker: multilinear interpolation of the 2^n_cv surrounding nodes, value and gradient alike;
//                   the same kernel produces the well-tempered heights of a deposit event (from the grid BEFORE the event)
//   k_grid_deposit  thread per node: adds the value and gradient of every new hill at its node, walkers in replica order
//                   (a fixed order, so the node sums are deterministic); hills staged through shared memory
// The node array is [nodes][1 + n_cv] binary64, row-major with the last CV fastest; all arithmetic is binary64: a node sums
// thousands of deposits over a run and every later bias value is a difference-free read of it, so the store is where
// precision matters, and the deposit runs once per `stride` steps, not per step.  Shares nothing with oracle/.
#include <math.h>

#include "geom.cuh"

#define GRID_TILE 128

struct GridParams {
    int n_cv, R;
    int shape[PSG_MAX_CV], periodic[PSG_MAX_CV];
    double lower[PSG_MAX_CV], h[PSG_MAX_CV], period[PSG_MAX_CV], inv_period[PSG_MAX_CV], inv_s2[PSG_MAX_CV];   // period = 0: open
    double w0, kB_deltaT;
    long long nodes;
};

struct GridState {
    GridParams G;
    double* grid = nullptr;     // [nodes][1 + n_cv]
    double* height = nullptr;   // [R] heights of the last deposit event (0 where masked out)
};

static GridState* gs(psg_ctx* c) { return reinterpret_cast<GridState*>(c->mgrid); }

// lower node index i0 and fraction f of coordinate x along CV k
__device__ __forceinline__ void grid_cell(const GridParams& G, int k, double x, int& i0, double& f) {
    const int n = G.shape[k];
    double t = (x - G.lower[k]) / G.h[k];
    if (G.periodic[k]) {
        t -= (double)n * floor(t / (double)n);
        if (t >= (double)n) t = 0.0;
        i0 = (int)floor(t);
    } else {
        t = fmin(fmax(t, 0.0), (double)(n - 1));       // outside an open grid: the nearest face
        i0 = max(min((int)floor(t), n - 2), 0);
    }
    f = t - (double)i0;
}

// out[0] = V, out[1 + k] = dV/dxi_k at the binary32 CV values xi[0..n_cv): multilinear interpolation of 2^n_cv nodes
__device__ __forceinline__ void grid_interp(const GridParams& G, const double* __restrict__ grid, const float* xi, double* out) {
    const int n = G.n_cv, rec = 1 + n;
    int i0[PSG_MAX_CV];
    double f[PSG_MAX_CV];
#pragma unroll
    for (int k = 0; k < PSG_MAX_CV; ++k)
        if (k < n) grid_cell(G, k, (double)xi[k], i0[k], f[k]);
#pragma unroll
    for (int c = 0; c < 1 + PSG_MAX_CV; ++c) out[c] = 0.0;
    for (int corner = 0; corner < (1 << n); ++corner) {
        double w = 1.0;
        long long flat = 0;
#pragma unroll
        for (int k = 0; k < PSG_MAX_CV; ++k)
            if (k < n) {
                const int up = (corner >> k) & 1;
                int i = i0[k] + up;
                if (G.periodic[k]) { if (i >= G.shape[k]) i -= G.shape[k]; }
                else i = min(i, G.shape[k] - 1);
                w *= up ? f[k] : 1.0 - f[k];
                flat = flat * G.shape[k] + i;
            }
        const double* node = grid + flat * rec;
#pragma unroll
        for (int c = 0; c < 1 + PSG_MAX_CV; ++c)
            if (c < rec) out[c] += w * node[c];
    }
}

// V and dV/dxi of walker r.  height == nullptr: write V / dVdxi (binary32, the bias arrays of the rest of the path).
// height != nullptr: write the height this walker deposits, w0 exp(-V / kB dT) or w0, 0 if masked.
__global__ void __launch_bounds__(128) k_grid_eval(const __grid_constant__ GridParams G, const double* __restrict__ grid,
                                                    const float* __restrict__ xi, float* __restrict__ V, float* __restrict__ dVdxi,
                                                    double* __restrict__ height, const unsigned char* __restrict__ mask) {
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= G.R) return;
    const int n = G.n_cv;
    float x[PSG_MAX_CV];
#pragma unroll
    for (int k = 0; k < PSG_MAX_CV; ++k) x[k] = k < n ? xi[(long long)r * n + k] : 0.f;
    double out[1 + PSG_MAX_CV];
    grid_interp(G, grid, x, out);
    if (height) {
        double W = 0.0;
        if (!mask || mask[r]) W = G.kB_deltaT > 0.0 ? G.w0 * exp(-out[0] / G.kB_deltaT) : G.w0;
        height[r] = W;
        return;
    }
    if (V) V[r] = (float)out[0];
    if (dVdxi) {
#pragma unroll
        for (int k = 0; k < PSG_MAX_CV; ++k)
            if (k < n) dVdxi[(long long)r * n + k] = (float)out[1 + k];
    }
}

// One deposit event: node += sum over walkers (in replica order) of W_r exp(-1/2 sum_k (d_k / sigma_k)^2) and its gradient
// -g d_k / sigma_k^2, d_k the (periodic) distance from the walker to the node.
__global__ void __launch_bounds__(GRID_TILE) k_grid_deposit(const __grid_constant__ GridParams G, double* __restrict__ grid,
                                                            const float* __restrict__ xi, const double* __restrict__ height) {
    __shared__ double s_x[GRID_TILE][PSG_MAX_CV];
    __shared__ double s_w[GRID_TILE];
    const long long node = (long long)blockIdx.x * GRID_TILE + threadIdx.x;
    const bool live = node < G.nodes;
    const int n = G.n_cv, rec = 1 + n;
    double x[PSG_MAX_CV] = {0, 0, 0, 0};
    if (live) {
        long long rem = node;
        for (int k = n - 1; k >= 0; --k) {
            const int i = (int)(rem % G.shape[k]);
            rem /= G.shape[k];
            x[k] = G.lower[k] + (double)i * G.h[k];
        }
    }
    double acc[1 + PSG_MAX_CV] = {0, 0, 0, 0, 0};
    if (live)
        for (int c = 0; c < rec; ++c) acc[c] = grid[node * rec + c];
    for (int base = 0; base < G.R; base += GRID_TILE) {
        __syncthreads();
        const int r = base + threadIdx.x;
        if (r < G.R) {
            s_w[threadIdx.x] = height[r];
            for (int k = 0; k < n; ++k) s_x[threadIdx.x][k] = (double)xi[(long long)r * n + k];
        }
        __syncthreads();
        const int cnt = min(GRID_TILE, G.R - base);
        if (!live) continue;
        for (int j = 0; j < cnt; ++j) {
            const double W = s_w[j];
            if (W == 0.0) continue;      // masked out
            double d[PSG_MAX_CV], e = 0.0;
#pragma unroll
            for (int k = 0; k < PSG_MAX_CV; ++k)
                if (k < n) {
                    d[k] = x[k] - s_x[j][k];
                    d[k] -= G.period[k] * rint(d[k] * G.inv_period[k]);      // open: period = inv_period = 0, the identity
                    e += d[k] * d[k] * G.inv_s2[k];
                }
            const double g = W * exp(-0.5 * e);
            acc[0] += g;
#pragma unroll
            for (int k = 0; k < PSG_MAX_CV; ++k)
                if (k < n) acc[1 + k] += -g * d[k] * G.inv_s2[k];
        }
    }
    if (live)
        for (int c = 0; c < rec; ++c) grid[node * rec + c] = acc[c];
}

extern "C" int psg_metad_grid_set(psg_ctx* c, int n_cv, const double* lower, const double* upper, const int* shape,
                                  const int* periodic, const double* sigma, double w0, double kB_deltaT) {
    if (!c) return PSG_EINVAL;
    auto bad = [&](const char* m) { c->err = m; return PSG_EINVAL; };
    if (!c->have_layout) { c->err = "psg_metad_grid_set: call psg_set_layout first"; return PSG_ESTATE; }
    if (n_cv < 1 || n_cv > PSG_MAX_CV || !lower || !upper || !shape || !periodic || !sigma)
        return bad("psg_metad_grid_set: 1 <= n_cv <= PSG_MAX_CV and no NULL array");
    if (!(w0 > 0.0) || !(kB_deltaT >= 0.0)) return bad("psg_metad_grid_set: need w0 > 0 and kB_deltaT >= 0");
    GridParams G;
    memset(&G, 0, sizeof(G));
    G.n_cv = n_cv; G.R = c->sys.R; G.w0 = w0; G.kB_deltaT = kB_deltaT; G.nodes = 1;
    for (int k = 0; k < n_cv; ++k) {
        if (shape[k] < 2 || !(upper[k] > lower[k]) || !(sigma[k] > 0.0))
            return bad("psg_metad_grid_set: need shape >= 2, upper > lower, sigma > 0 for every CV");
        G.shape[k] = shape[k]; G.periodic[k] = periodic[k] ? 1 : 0; G.lower[k] = lower[k];
        G.h[k] = (upper[k] - lower[k]) / (double)(periodic[k] ? shape[k] : shape[k] - 1);
        G.period[k] = periodic[k] ? upper[k] - lower[k] : 0.0;
        G.inv_period[k] = periodic[k] ? 1.0 / G.period[k] : 0.0;
        G.inv_s2[k] = 1.0 / (sigma[k] * sigma[k]);
        G.nodes *= shape[k];
        if (G.nodes > (1ll << 27)) return bad("psg_metad_grid_set: more than 2^27 nodes");
    }
    cudaSetDevice(c->device);
    GridState* S = gs(c);
    if (!S) { S = new GridState(); c->mgrid = S; }
    if (S->grid) cudaFree(S->grid);
    if (S->height) cudaFree(S->height);
    S->grid = S->height = nullptr;
    S->G = G;
    const size_t bytes = sizeof(double) * (size_t)G.nodes * (1 + n_cv);
    if (cudaMalloc((void**)&S->grid, bytes) != cudaSuccess || cudaMalloc((void**)&S->height, sizeof(double) * (size_t)G.R) != cudaSuccess) {
        c->err = "psg_metad_grid_set: out of device memory";
        return PSG_ENOMEM;
    }
    cudaMemsetAsync(S->grid, 0, bytes, c->stream);
    cudaMemsetAsync(S->height, 0, sizeof(double) * (size_t)G.R, c->stream);
    return PSG_OK;
}

extern "C" int psg_metad_grid_deposit(psg_ctx* c, const float* d_xi, const unsigned char* d_mask) {
    if (!c) return PSG_EINVAL;
    GridState* S = gs(c);
    if (!S) { c->err = "psg_metad_grid_deposit: call psg_metad_grid_set first"; return PSG_ESTATE; }
    if (!d_xi) { c->err = "psg_metad_grid_deposit: NULL pointer"; return PSG_EINVAL; }
    const GridParams& G = S->G;
    k_grid_eval<<<(G.R + 127) / 128, 128, 0, c->stream>>>(G, S->grid, d_xi, nullptr, nullptr, S->height, d_mask);
    k_grid_deposit<<<(unsigned)((G.nodes + GRID_TILE - 1) / GRID_TILE), GRID_TILE, 0, c->stream>>>(G, S->grid, d_xi, S->height);
    c->launches += 2;
    if (cudaGetLastError() != cudaSuccess) { c->err = "psg_metad_grid_deposit: launch failed"; return PSG_ECUDA; }
    return PSG_OK;
}

extern "C" int psg_metad_grid_eval(psg_ctx* c, const float* d_xi, float* d_V, float* d_dVdxi) {
    if (!c) return PSG_EINVAL;
    GridState* S = gs(c);
    if (!S) { c->err = "psg_metad_grid_eval: call psg_metad_grid_set first"; return PSG_ESTATE; }
    if (!d_xi || (!d_V && !d_dVdxi)) { c->err = "psg_metad_grid_eval: NULL pointer"; return PSG_EINVAL; }
    const GridParams& G = S->G;
    k_grid_eval<<<(G.R + 127) / 128, 128, 0, c->stream>>>(G, S->grid, d_xi, d_V, d_dVdxi, nullptr, nullptr);
    c->launches += 1;
    if (cudaGetLastError() != cudaSuccess) { c->err = "psg_metad_grid_eval: launch failed"; return PSG_ECUDA; }
    return PSG_OK;
}

// The per-step path with the bias on the grid, ONE launch (SURVEY rows A1, A2, A8 with the grid in place of the hill sum):
// warp per walker -- gather the CV atoms in place, CVs and Jacobians in binary64 registers (geom.cuh), xi rounded to
// binary32 (reading R-XI32: the bias is a function of the binary32 CV the caller sees), lane 0 interpolates the grid, every
// lane scatters force[i] += -dV/dxi_k * dxi_k/dr_i for its slots (red.global.add.f32: atoms shared between CVs collide).
// The grid is read-only here, so there is no barrier and the launch is an ordinary one.
__global__ void __launch_bounds__(256) k_grid_step(const __grid_constant__ SysParams P, const __grid_constant__ GridParams G,
                                                    const double* __restrict__ grid, const float* __restrict__ pos,
                                                    float* __restrict__ force, float* __restrict__ xi_out,
                                                    float* __restrict__ V_out, float* __restrict__ dV_out) {
    __shared__ WarpCvSmem sm[8];
    __shared__ float s_dv[8][PSG_MAX_CV];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int r = blockIdx.x * 8 + wid;
    if (r >= P.R) return;
    WarpCvSmem& S = sm[wid];
    warp_cv_eval<true>(P, r, pos, nullptr, S, lane);
    if (lane == 0) {
        float x[PSG_MAX_CV];
#pragma unroll
        for (int k = 0; k < PSG_MAX_CV; ++k) x[k] = k < P.n_cv ? (float)S.xi[k] : 0.f;
        double out[1 + PSG_MAX_CV];
        grid_interp(G, grid, x, out);
        V_out[r] = (float)out[0];
#pragma unroll
        for (int k = 0; k < PSG_MAX_CV; ++k)
            if (k < P.n_cv) {
                xi_out[(long long)r * P.n_cv + k] = x[k];
                dV_out[(long long)r * P.n_cv + k] = s_dv[wid][k] = (float)out[1 + k];
            }
    }
    __syncwarp();
    for (int s = lane; s < P.n_slots; s += 32) {
        const D3 j = slot_jacobian(P, r, pos, S, s);
        const float dv = -s_dv[wid][P.grp[P.slot_gid_c[s]].cv];
        const int atom = slot_atom_of(P, r, s);
        float* f = force + ((long long)r * P.rstride + atom) * P.fs;
        force_add(f, dv * (float)j.x, dv * (float)j.y, dv * (float)j.z, P.fs);
    }
}

extern "C" int psg_metad_grid_step(psg_ctx* c, const float* d_pos, float* d_force) {
    if (!c) return PSG_EINVAL;
    GridState* S = gs(c);
    if (!S) { c->err = "psg_metad_grid_step: call psg_metad_grid_set first"; return PSG_ESTATE; }
    if (!c->have_cvs) { c->err = "psg_metad_grid_step: no CVs configured"; return PSG_ESTATE; }
    if (!d_pos || !d_force) { c->err = "psg_metad_grid_step: NULL pointer"; return PSG_EINVAL; }
    const SysParams& P = c->sys;
    if (P.n_cv != S->G.n_cv || P.R != S->G.R) { c->err = "psg_metad_grid_step: the grid was set for another n_cv or walker count"; return PSG_ESTATE; }
    if (P.n_ranges > 0 || c->dti_cv >= 0) {   // range groups / the interface CV: their values and forces live in kernels of their own
        int e = psg_cv_eval(c, d_pos, c->d_xi, nullptr);
        if (e == PSG_OK) e = psg_metad_grid_eval(c, c->d_xi, c->d_V, c->d_dVdxi);
        if (e == PSG_OK) e = psg_apply_bias_forces(c, d_pos, c->d_dVdxi, d_force);
        return e;
    }
    k_grid_step<<<(P.R + 7) / 8, 256, 0, c->stream>>>(P, S->G, S->grid, d_pos, d_force, c->d_xi, c->d_V, c->d_dVdxi);
    c->launches += 1;
    if (cudaGetLastError() != cudaSuccess) { c->err = "psg_metad_grid_step: launch failed"; return PSG_ECUDA; }
    return PSG_OK;
}

extern "C" int psg_set_metad_grid(psg_ctx* c, const double* lower, const double* upper, const int* shape, const int* periodic,
                                  const double* sigma, double w0, double kB_deltaT, int stride) {
    if (!c) return PSG_EINVAL;
    if (!c->have_cvs) { c->err = "psg_set_metad_grid: call psg_set_cvs first"; return PSG_ESTATE; }
    if (!lower || !upper || !shape || !periodic || !sigma || stride < 0) { c->err = "psg_set_metad_grid: bad argument"; return PSG_EINVAL; }
    for (int k = 0; k < c->sys.n_cv; ++k) {
        const double per = c->sys.cv[k].period;
        if (per > 0.0) {
            if (!periodic[k] || fabs((upper[k] - lower[k]) - per) > 1e-9 * per) {
                c->err = "psg_set_metad_grid: a periodic CV needs a periodic grid spanning exactly its period";
                return PSG_EINVAL;
            }
        } else if (periodic[k]) {
            c->err = "psg_set_metad_grid: a periodic grid on a CV that is not periodic";
            return PSG_EINVAL;
        }
    }
    int rc = psg_metad_grid_set(c, c->sys.n_cv, lower, upper, shape, periodic, sigma, w0, kB_deltaT);
    if (rc != PSG_OK) return rc;
    c->mgrid_stride = stride;
    c->method = PSG_METHOD_METAD_GRID;
    return PSG_OK;
}

extern "C" int psg_metad_grid_state(psg_ctx* c, double** d_grid_out, long long* n_nodes_out, double** d_heights_out) {
    if (!c) return PSG_EINVAL;
    GridState* S = gs(c);
    if (!S) { c->err = "psg_metad_grid_state: call psg_metad_grid_set first"; return PSG_ESTATE; }
    if (d_grid_out) *d_grid_out = S->grid;
    if (n_nodes_out) *n_nodes_out = S->G.nodes;
    if (d_heights_out) *d_heights_out = S->height;
    return PSG_OK;
}

void psg_metad_grid_free(psg_ctx* c) {
    GridState* S = gs(c);
    if (!S) return;
    if (S->grid) cudaFree(S->grid);
    if (S->height) cudaFree(S->height);
    delete S;
    c->mgrid = nullptr;
}
