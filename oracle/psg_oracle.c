/*
 * psg_oracle.c -- ORACLE. Test infrastructure, not the product.
 *
 * A plain, slow, fp64 CPU restatement of the per-MD-step enhanced-sampling hot
 * path that PySAGES (arXiv 2301.04835; /root/reference/PAPER.md) defines:
 *   gather CV atoms -> collective variables + analytic Jacobians -> bias energy
 *   and gradient -> F_i += -dV/dxi * dxi/dr_i.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.  It shares no code, header,
 * table or constant with paper_2301_04835_b200/csrc (the CUDA path) and neither
 * side includes the other.
 *
 * The paper names the quantities but prints no formula for them (the only
 * equations are Eq. 1-3, and the interface CV Eq. 4-8), so
 * each function below is the textbook definition of the quantity the cited
 * passage names, under the readings listed in DESIGN.md ("Readings").
 * Inputs arrive as IEEE binary32 (the engine's arrays) and are widened exactly
 * to binary64; every operation is binary64 except the ABF bin index, which
 * DESIGN.md reading R-ABF-1 defines in binary32 so that "bit-exact" is
 * meaningful.  Compile with -O2 -ffp-contract=off, no fast-math.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): closed-form geometries,
 * central finite differences, translation/rotation invariance of forces,
 * periodicity, single-hill closed forms, hand-computed ABF tables.
 * Parity unpinned (no passage, closed form or invariant fixes them; they follow
 * DESIGN.md readings only): the order of simultaneous deposits by several
 * walkers (orc_deposit_hills), the two-phase mean-force read of a shared ABF
 * grid (orc_abf_update), the stride phase of deposits.  The minimum-image
 * convention (orc_layout.box, reading R-MI) is a reading too -- the paper is
 * silent on periodic positions -- but its arithmetic is pinned
 * (tests/test_oracle_minimum_image.py: geometries across a face, box-vector
 * shift invariance, finite differences).  The ABF force estimator
 * (orc_abf_estimate, reading R-ABF-EST) is a reading as well -- the paper only
 * cites its reference [43] -- with its arithmetic pinned by closed-form
 * trajectories and numpy's least squares (tests/test_oracle_abf_estimator.py).
 * The gyration-tensor shape CVs (shape_cv, reading R-SHAPE) are named by the
 * paper without a formula; their arithmetic is pinned by hand-computed point
 * sets, numpy.linalg.eigvalsh, the trace identity with the pinned Rg, rotation
 * invariance and finite differences (tests/test_oracle_shape_cv.py).
 * Grid-stored metadynamics (orc_grid_*, reading R-GRID): the paper gives no
 * layout or interpolation; pinned by the hill sum at the nodes, multilinear
 * functions, scipy's interpolator and h^2 convergence
 * (tests/test_oracle_grid_metad.py).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { ORC_DISTANCE = 1, ORC_ANGLE = 2, ORC_DIHEDRAL = 3, ORC_COMPONENT = 4, ORC_RGYR = 5, ORC_DISPLACEMENT = 6,
       /* gyration-tensor shape CVs, PAPER.md:L188-L189 (reading R-SHAPE) */
       ORC_PRINCIPAL_MOMENT = 7, ORC_ASPHERICITY = 8, ORC_ACYLINDRICITY = 9, ORC_SHAPE_ANISOTROPY = 10 };

/* One collective variable: a function of 1..4 *groups* of atoms, each group
 * reduced to its (weighted) barycenter -- PAPER.md:L185-L189 (Sec. 2.2:
 * TwoPointCV/ThreePointCV/FourPointCV/AxisCV "groups"), L227-L229 (Fig. 3,
 * barycenter(p1)).  A group is either an explicit slice [begin, begin+size) of
 * the slot list, or a contiguous atom range of the replica's array. */
typedef struct {
    int type;
    int n_groups;
    int is_range[4];
    int slot_begin[4];
    int slot_size[4];
    long long range_begin[4];
    long long range_size[4];
    int axis;       /* ORC_COMPONENT, ORC_DISPLACEMENT: 0, 1 or 2; ORC_PRINCIPAL_MOMENT: which eigenvalue, 0 = largest */
    double period;  /* 0 = not periodic */
} orc_cv;

/* Where the engine's arrays are: PAPER.md:L37 (Snapshot: positions, forces). */
typedef struct {
    int n_replicas;
    long long n_atoms;
    long long replica_stride_atoms; /* 0: every replica indexes ONE shared array */
    int pos_stride;                 /* floats per atom in pos: 3 or 4 */
    int n_cv;
    int n_slots;
    int per_replica_slots;          /* 0: slot_atom[n_slots]; 1: slot_atom[R][n_slots] */
    double box[3];                  /* orthorhombic box lengths for the minimum-image convention; 0 = open in that direction
                                     * (reading R-MI of DESIGN.md; the paper is silent on periodic positions) */
} orc_layout;

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---------- small vector helpers (fp64) ---------- */
static void v_sub(const double *a, const double *b, double *o) { o[0] = a[0] - b[0]; o[1] = a[1] - b[1]; o[2] = a[2] - b[2]; }
static double v_dot(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
static void v_cross(const double *a, const double *b, double *o) {
    o[0] = a[1] * b[2] - a[2] * b[1];
    o[1] = a[2] * b[0] - a[0] * b[2];
    o[2] = a[0] * b[1] - a[1] * b[0];
}

/* Nearest-image difference for a periodic CV: d <- d - P*rint(d/P).
 * DESIGN.md reading R-PER (the paper is silent; Grid(..., periodic=True),
 * PAPER.md:L82). */
static double wrap_period(double d, double period) {
    if (period > 0.0) d -= period * rint(d / period);
    return d;
}

/* number of atoms of group g of a CV and the i-th atom's index and weight */
/* nearest image of a displacement vector in an orthorhombic box: d <- d - L rint(d / L) per periodic direction */
static void min_image(double *d, const double *box) {
    if (!box) return;
    for (int x = 0; x < 3; ++x)
        if (box[x] > 0) d[x] -= box[x] * rint(d[x] / box[x]);
}

/* position of atom a as the image nearest to ref (ref == NULL: as stored) */
static void atom_image(const float *pos, int ps, long long a, const double *ref, const double *box, double *r) {
    for (int x = 0; x < 3; ++x) r[x] = (double)pos[a * ps + x];
    if (ref && box) {
        double d[3] = {r[0] - ref[0], r[1] - ref[1], r[2] - ref[2]};
        min_image(d, box);
        for (int x = 0; x < 3; ++x) r[x] = ref[x] + d[x];
    }
}

static long long group_count(const orc_cv *cv, int g) { return cv->is_range[g] ? cv->range_size[g] : (long long)cv->slot_size[g]; }

static long long group_atom(const orc_cv *cv, int g, long long i, const int *slot_atom) {
    return cv->is_range[g] ? cv->range_begin[g] + i : (long long)slot_atom[cv->slot_begin[g] + i];
}

/* weight of the i-th atom of group g: explicit groups index slot_weight by slot,
 * range groups index atom_weight by atom; NULL => 1 (barycenter, Fig. 3). */
static double group_weight(const orc_cv *cv, int g, long long i, const float *slot_weight, const float *atom_weight) {
    if (cv->is_range[g]) return atom_weight ? (double)atom_weight[cv->range_begin[g] + i] : 1.0;
    return slot_weight ? (double)slot_weight[cv->slot_begin[g] + i] : 1.0;
}

/* c_g = sum_i w_i r_i / sum_i w_i  (PAPER.md:L227-L229 barycenter; with masses
 * as weights the "center of mass" of L332, L408). */
static void group_center(const orc_cv *cv, int g, const float *pos, int ps, const int *slot_atom,
                         const float *slot_weight, const float *atom_weight, const double *box, double *c, double *wsum) {
    double s[3] = {0, 0, 0}, W = 0, first[3];
    long long n = group_count(cv, g);
    atom_image(pos, ps, group_atom(cv, g, 0, slot_atom), NULL, NULL, first);
    for (long long i = 0; i < n; ++i) {
        long long a = group_atom(cv, g, i, slot_atom);
        double w = group_weight(cv, g, i, slot_weight, atom_weight), r[3];
        atom_image(pos, ps, a, first, box, r);   /* with a box: the image nearest to the group's first atom (R-MI) */
        s[0] += w * r[0];
        s[1] += w * r[1];
        s[2] += w * r[2];
        W += w;
    }
    c[0] = s[0] / W; c[1] = s[1] / W; c[2] = s[2] / W;
    *wsum = W;
}

/* xi and d(xi)/d(c_g) for the CVs that are functions of group centers only. */
static double point_cv(const orc_cv *cv, double c[4][3], double dc[4][3], const double *box) {
    memset(dc, 0, sizeof(double) * 12);
    switch (cv->type) {
    case ORC_DISTANCE: { /* PAPER.md:L185 Distance: xi = |c2 - c1| */
        double d[3]; v_sub(c[1], c[0], d); min_image(d, box);
        double r = sqrt(v_dot(d, d));
        if (r > 0) for (int x = 0; x < 3; ++x) { dc[1][x] = d[x] / r; dc[0][x] = -d[x] / r; }
        return r;
    }
    case ORC_ANGLE: { /* PAPER.md:L186 Angle; vertex at the second group (reading R-ANG) */
        double q[3], s[3], n[3], t[3];
        v_sub(c[0], c[1], q); v_sub(c[2], c[1], s); min_image(q, box); min_image(s, box); v_cross(q, s, n);
        double nn = sqrt(v_dot(n, n));
        double th = atan2(nn, v_dot(q, s));
        if (nn > 0) {
            double q2 = v_dot(q, q), s2 = v_dot(s, s);
            v_cross(q, n, t); for (int x = 0; x < 3; ++x) dc[0][x] = t[x] / (q2 * nn);
            v_cross(s, n, t); for (int x = 0; x < 3; ++x) dc[2][x] = -t[x] / (s2 * nn);
            for (int x = 0; x < 3; ++x) dc[1][x] = -(dc[0][x] + dc[2][x]);
        }
        return th;
    }
    case ORC_DIHEDRAL: { /* PAPER.md:L187 DihedralAngle, L81; IUPAC sign (reading R-DIH) */
        double b1[3], b2[3], b3[3], n1[3], n2[3];
        v_sub(c[1], c[0], b1); v_sub(c[2], c[1], b2); v_sub(c[3], c[2], b3);
        min_image(b1, box); min_image(b2, box); min_image(b3, box);
        v_cross(b1, b2, n1); v_cross(b2, b3, n2);
        double lb2 = sqrt(v_dot(b2, b2));
        double phi = atan2(lb2 * v_dot(b1, n2), v_dot(n1, n2));
        double n1s = v_dot(n1, n1), n2s = v_dot(n2, n2);
        if (n1s > 0 && n2s > 0) {
            double a = v_dot(b1, b2) / (lb2 * lb2), e = v_dot(b3, b2) / (lb2 * lb2);
            for (int x = 0; x < 3; ++x) {
                dc[0][x] = -(lb2 / n1s) * n1[x];
                dc[3][x] = (lb2 / n2s) * n2[x];
            }
            for (int x = 0; x < 3; ++x) {
                dc[1][x] = -(1.0 + a) * dc[0][x] + e * dc[3][x];
                dc[2][x] = -(1.0 + e) * dc[3][x] + a * dc[0][x];
            }
        }
        return phi;
    }
    case ORC_DISPLACEMENT: { /* PAPER.md:L185 Displacement (TwoPointCV): the vector c2 - c1; one CV per component (axis) */
        double d[3]; v_sub(c[1], c[0], d); min_image(d, box);
        dc[1][cv->axis] = 1.0; dc[0][cv->axis] = -1.0;
        return d[cv->axis];
    }
    case ORC_COMPONENT: /* PAPER.md:L188 Component: barycenter coordinate along an axis */
        dc[0][cv->axis] = 1.0;
        return c[0][cv->axis];
    }
    return NAN;
}

/* Eigenvalues and eigenvectors of a symmetric 3x3 matrix by cyclic Jacobi rotations (the textbook method: each rotation
 * J zeroes one off-diagonal pair, A <- J^T A J, V <- V J, until the off-diagonal part has vanished).  Every product is
 * written out as a plain triple loop.  On return lam[0] >= lam[1] >= lam[2] and column k of V is the unit eigenvector of
 * lam[k].  Pinned against numpy.linalg.eigvalsh through the CVs below (tests/test_oracle_shape_cv.py). */
static void sym3_eig(double S[3][3], double lam[3], double V[3][3]) {
    double A[3][3], J[3][3], T[3][3];
    static const int pairs[3][2] = {{0, 1}, {0, 2}, {1, 2}};
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { A[i][j] = S[i][j]; V[i][j] = i == j ? 1.0 : 0.0; }
    for (int sweep = 0; sweep < 64; ++sweep) {
        double off = A[0][1] * A[0][1] + A[0][2] * A[0][2] + A[1][2] * A[1][2];
        double dia = A[0][0] * A[0][0] + A[1][1] * A[1][1] + A[2][2] * A[2][2];
        if (off <= 1e-60 * dia || off == 0.0) break;
        for (int e = 0; e < 3; ++e) {
            int p = pairs[e][0], q = pairs[e][1];
            if (A[p][q] == 0.0) continue;
            double theta = (A[q][q] - A[p][p]) / (2.0 * A[p][q]);
            double t = (theta >= 0 ? 1.0 : -1.0) / (fabs(theta) + sqrt(theta * theta + 1.0));
            double c = 1.0 / sqrt(t * t + 1.0), sn = t * c;
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) J[i][j] = i == j ? 1.0 : 0.0;
            J[p][p] = c; J[q][q] = c; J[p][q] = sn; J[q][p] = -sn;
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {         /* T = A J */
                T[i][j] = 0; for (int k = 0; k < 3; ++k) T[i][j] += A[i][k] * J[k][j];
            }
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {         /* A = J^T T */
                A[i][j] = 0; for (int k = 0; k < 3; ++k) A[i][j] += J[k][i] * T[k][j];
            }
            A[p][q] = A[q][p] = 0.0;                                          /* what the rotation is built to do */
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {         /* T = V J */
                T[i][j] = 0; for (int k = 0; k < 3; ++k) T[i][j] += V[i][k] * J[k][j];
            }
            memcpy(V, T, sizeof(T));
        }
    }
    lam[0] = A[0][0]; lam[1] = A[1][1]; lam[2] = A[2][2];
    for (int a = 0; a < 2; ++a) for (int b = 0; b < 2 - a; ++b) if (lam[b] < lam[b + 1]) {   /* bubble sort, descending */
        double x = lam[b]; lam[b] = lam[b + 1]; lam[b + 1] = x;
        for (int i = 0; i < 3; ++i) { x = V[i][b]; V[i][b] = V[i][b + 1]; V[i][b + 1] = x; }
    }
}

/* Gyration-tensor shape CVs of one group, PAPER.md:L188 (PrincipalMoment) and L189 (Asphericity, Acylindricity,
 * ShapeAnisotropy).  The paper only names them; reading R-SHAPE of DESIGN.md takes the polymer-physics definitions:
 *   S = sum_i w_i (r_i - c)(r_i - c)^T / W   (the weights of the barycenter, so that tr S = Rg^2 of reading R-RG),
 *   eigenvalues l1 >= l2 >= l3,
 *   PrincipalMoment(axis k) = l_k,  Asphericity b = l1 - (l2 + l3)/2,  Acylindricity c = l2 - l3,
 *   ShapeAnisotropy kappa^2 = (b^2 + 3/4 c^2) / (l1 + l2 + l3)^2   (0 for a point).
 * First-order perturbation theory gives d l_k / d r_i = (2 w_i / W) (v_k . (r_i - c)) v_k  (the barycenter's own
 * dependence on r_i drops out because sum_i w_i (r_i - c) = 0), and the chain rule through (l1, l2, l3) the rest.
 * At a degenerate pair of eigenvalues the single eigenvalues are not differentiable; the formula then returns the
 * derivative along the eigenvectors the Jacobi iteration happened to produce. */
static double shape_cv(const orc_cv *cv, const float *pos, int ps, const int *slot_atom,
                       const float *slot_weight, const float *atom_weight, const double *box, double *jac) {
    double c[3], W, first[3], r[3], S[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}, lam[3], V[3][3], g[3] = {0, 0, 0}, xi = NAN;
    group_center(cv, 0, pos, ps, slot_atom, slot_weight, atom_weight, box, c, &W);
    long long n = group_count(cv, 0);
    atom_image(pos, ps, group_atom(cv, 0, 0, slot_atom), NULL, NULL, first);
    for (long long i = 0; i < n; ++i) {
        double w = group_weight(cv, 0, i, slot_weight, atom_weight);
        atom_image(pos, ps, group_atom(cv, 0, i, slot_atom), first, box, r);
        double d[3] = {r[0] - c[0], r[1] - c[1], r[2] - c[2]};
        for (int x = 0; x < 3; ++x) for (int y = 0; y < 3; ++y) S[x][y] += w * d[x] * d[y] / W;
    }
    sym3_eig(S, lam, V);
    double tr = lam[0] + lam[1] + lam[2];
    switch (cv->type) {
    case ORC_PRINCIPAL_MOMENT: xi = lam[cv->axis]; g[cv->axis] = 1.0; break;
    case ORC_ASPHERICITY: xi = lam[0] - 0.5 * (lam[1] + lam[2]); g[0] = 1.0; g[1] = -0.5; g[2] = -0.5; break;
    case ORC_ACYLINDRICITY: xi = lam[1] - lam[2]; g[1] = 1.0; g[2] = -1.0; break;
    case ORC_SHAPE_ANISOTROPY: {
        double b = lam[0] - 0.5 * (lam[1] + lam[2]), a = lam[1] - lam[2];
        double num = b * b + 0.75 * a * a;
        xi = tr > 0 ? num / (tr * tr) : 0.0;
        if (tr > 0) {
            /* d num / d l = (2b, -b + 3a/2, -b - 3a/2);  d (num / tr^2) / d l_k = dnum_k / tr^2 - 2 num / tr^3 */
            double dn[3] = {2.0 * b, -b + 1.5 * a, -b - 1.5 * a};
            for (int k = 0; k < 3; ++k) g[k] = dn[k] / (tr * tr) - 2.0 * num / (tr * tr * tr);
        }
        break;
    }
    }
    if (jac) for (long long i = 0; i < n; ++i) {
        double w = group_weight(cv, 0, i, slot_weight, atom_weight);
        atom_image(pos, ps, group_atom(cv, 0, i, slot_atom), first, box, r);
        double d[3] = {r[0] - c[0], r[1] - c[1], r[2] - c[2]};
        for (int x = 0; x < 3; ++x) jac[3 * i + x] = 0.0;
        for (int k = 0; k < 3; ++k) {
            double proj = V[0][k] * d[0] + V[1][k] * d[1] + V[2][k] * d[2];
            for (int x = 0; x < 3; ++x) jac[3 * i + x] += (2.0 * w / W) * g[k] * proj * V[x][k];
        }
    }
    return xi;
}

/* Evaluate one CV of one replica.  jac (nullable) receives d(xi)/d(r_i), three
 * doubles per atom, for the atoms of group 0, then group 1, ... in group order.
 * Returns xi. */
static double cv_one(const orc_cv *cv, const float *pos, int ps, const int *slot_atom,
                     const float *slot_weight, const float *atom_weight, const double *box, double *jac) {
    if (cv->type >= ORC_PRINCIPAL_MOMENT && cv->type <= ORC_SHAPE_ANISOTROPY)
        return shape_cv(cv, pos, ps, slot_atom, slot_weight, atom_weight, box, jac);
    if (cv->type == ORC_RGYR) {
        /* PAPER.md:L189 RadiusofGyration. Reading R-RG: Rg^2 = sum w|r-c|^2 / sum w,
         * same weights as the barycenter; dRg/dr_i = w_i (r_i - c)/(W Rg). */
        double c[3], W, first[3], r[3];
        group_center(cv, 0, pos, ps, slot_atom, slot_weight, atom_weight, box, c, &W);
        long long n = group_count(cv, 0);
        atom_image(pos, ps, group_atom(cv, 0, 0, slot_atom), NULL, NULL, first);
        double s2 = 0;
        for (long long i = 0; i < n; ++i) {
            long long a = group_atom(cv, 0, i, slot_atom);
            double w = group_weight(cv, 0, i, slot_weight, atom_weight);
            atom_image(pos, ps, a, first, box, r);
            double d[3] = {r[0] - c[0], r[1] - c[1], r[2] - c[2]};
            s2 += w * v_dot(d, d);
        }
        double rg = sqrt(s2 / W);
        if (jac) for (long long i = 0; i < n; ++i) {
            long long a = group_atom(cv, 0, i, slot_atom);
            double w = group_weight(cv, 0, i, slot_weight, atom_weight);
            atom_image(pos, ps, a, first, box, r);
            for (int x = 0; x < 3; ++x)
                jac[3 * i + x] = rg > 0 ? w * (r[x] - c[x]) / (W * rg) : 0.0;
        }
        return rg;
    }
    double c[4][3], W[4], dc[4][3];
    for (int g = 0; g < cv->n_groups; ++g) group_center(cv, g, pos, ps, slot_atom, slot_weight, atom_weight, box, c[g], &W[g]);
    double xi = point_cv(cv, c, dc, box);
    if (jac) {
        long long o = 0;
        for (int g = 0; g < cv->n_groups; ++g) {
            long long n = group_count(cv, g);
            for (long long i = 0; i < n; ++i, ++o) {
                /* chain rule through the barycenter: d xi/d r_i = (w_i/W_g) d xi/d c_g */
                double w = group_weight(cv, g, i, slot_weight, atom_weight) / W[g];
                for (int x = 0; x < 3; ++x) jac[3 * o + x] = w * dc[g][x];
            }
        }
    }
    return xi;
}

/* NULL when no direction is periodic */
static const double *orc_box(const orc_layout *L) {
    return (L->box[0] > 0 || L->box[1] > 0 || L->box[2] > 0) ? L->box : NULL;
}

static long long cv_natoms(const orc_cv *cv) {
    long long n = 0;
    for (int g = 0; g < cv->n_groups; ++g) n += group_count(cv, g);
    return n;
}

/* Total Jacobian rows per replica (sum over CVs of atoms in their groups). */
long long orc_jac_rows(const orc_layout *L, const orc_cv *cvs) {
    long long n = 0;
    for (int k = 0; k < L->n_cv; ++k) n += cv_natoms(&cvs[k]);
    return n;
}

/* cv_eval: xi[R][n_cv]; jac (nullable) [R][jac_rows][3], rows ordered CV by CV,
 * group by group, atom by atom.  PAPER.md:L39 ("computes the CVs"), L185-L189. */
void orc_cv_eval(const orc_layout *L, const orc_cv *cvs, const int *slot_atom, const float *slot_weight,
                 const float *atom_weight, const float *pos, double *xi, double *jac) {
    long long rows = orc_jac_rows(L, cvs);
#pragma omp parallel for schedule(static)
    for (int r = 0; r < L->n_replicas; ++r) {
        const float *p = pos + (long long)r * L->replica_stride_atoms * L->pos_stride;
        const int *sa = slot_atom + (L->per_replica_slots ? (long long)r * L->n_slots : 0);
        long long o = 0;
        for (int k = 0; k < L->n_cv; ++k) {
            double *j = jac ? jac + ((long long)r * rows + o) * 3 : NULL;
            xi[(long long)r * L->n_cv + k] = cv_one(&cvs[k], p, L->pos_stride, sa, slot_weight, atom_weight, orc_box(L), j);
            o += cv_natoms(&cvs[k]);
        }
    }
}

/* Harmonic bias, PAPER.md:L125 (Sec. 2.1.1): H_b = H + k/2 (xi - xi0)^2.
 * Multi-CV: V = 1/2 sum_k k_k D_k^2, dV/dxi_k = k_k D_k, D wrapped for periodic CVs. */
void orc_harmonic(int n_replicas, int n_cv, const double *xi, const double *kspring, const double *center,
                  const double *period, double *V, double *dVdxi) {
    for (int r = 0; r < n_replicas; ++r) {
        double v = 0;
        for (int k = 0; k < n_cv; ++k) {
            double d = wrap_period(xi[r * n_cv + k] - center[r * n_cv + k], period[k]);
            v += 0.5 * kspring[k] * d * d;
            dVdxi[r * n_cv + k] = kspring[k] * d;
        }
        V[r] = v;
    }
}

/* Metadynamics bias, PAPER.md:L147 (Sec. 2.1.5): a sum of Gaussians of user
 * height and width.  V(xi) = sum_h W_h exp(-1/2 sum_k (d_hk/sigma_k)^2),
 * dV/dxi_k = -sum_h W_h exp(..) d_hk/sigma_k^2, d_hk = wrap(xi_k - s_hk).
 * Tabs[R][n_cv] (nullable) = sum_h |term| of the gradient sum: its conditioning. */
void orc_metad(int n_replicas, int n_cv, const double *xi, long long n_hills, const float *centers /*[n][n_cv]*/,
               const float *heights, const double *sigma, const double *period, double *V, double *dVdxi, double *Tabs) {
#pragma omp parallel for schedule(static)
    for (int r = 0; r < n_replicas; ++r) {
        double v = 0, g[8] = {0}, t[8] = {0}, d[8];
        for (long long h = 0; h < n_hills; ++h) {
            double e = 0;
            for (int k = 0; k < n_cv; ++k) {
                d[k] = wrap_period(xi[r * n_cv + k] - (double)centers[h * n_cv + k], period[k]);
                e += (d[k] / sigma[k]) * (d[k] / sigma[k]);
            }
            double w = (double)heights[h] * exp(-0.5 * e);
            v += w;
            for (int k = 0; k < n_cv; ++k) {
                double term = -w * d[k] / (sigma[k] * sigma[k]);
                g[k] += term;
                t[k] += fabs(term);
            }
        }
        if (V) V[r] = v;
        for (int k = 0; k < n_cv; ++k) {
            if (dVdxi) dVdxi[r * n_cv + k] = g[k];
            if (Tabs) Tabs[r * n_cv + k] = t[k];
        }
    }
}

/* Hill deposition.  Standard: W = w0.  Well-tempered
 * (kB_deltaT > 0): W = w0 exp(-V_old(xi)/(kB dT)), V_old from the list BEFORE
 * this event (reading R-WT).  Several walkers deposit synchronously and append
 * in replica order (reading R-MW, parity unpinned).  Centres and heights are
 * stored as binary32 (the hill store's type).  Returns the new hill count. */
long long orc_deposit_hills(int n_replicas, int n_cv, const float *xi /*[R][n_cv]*/, const unsigned char *mask,
                            double w0, double kB_deltaT, const double *sigma, const double *period,
                            long long n_hills, float *centers, float *heights) {
    double *xd = (double *)malloc(sizeof(double) * (size_t)n_replicas * n_cv);
    double *V = (double *)malloc(sizeof(double) * (size_t)n_replicas);
    for (long long i = 0; i < (long long)n_replicas * n_cv; ++i) xd[i] = (double)xi[i];
    if (kB_deltaT > 0) orc_metad(n_replicas, n_cv, xd, n_hills, centers, heights, sigma, period, V, NULL, NULL);
    long long n = n_hills;
    for (int r = 0; r < n_replicas; ++r) {
        if (mask && !mask[r]) continue;
        for (int k = 0; k < n_cv; ++k) centers[n * n_cv + k] = xi[r * n_cv + k];
        heights[n] = (float)(kB_deltaT > 0 ? w0 * exp(-V[r] / kB_deltaT) : w0);
        ++n;
    }
    free(xd); free(V);
    return n;
}

/* ABF bin index of one CV value, DEFINED IN BINARY32 (reading R-ABF-1):
 * t = fl32(fl32(xi - lower) * invd), I = (int)floorf(t), two separately rounded
 * operations (this file is compiled with -ffp-contract=off).  invd =
 * (float)((double)shape / ((double)upper - (double)lower)).  Grid(lower, upper,
 * shape, periodic): PAPER.md:L82 (Fig. 2). */
static int abf_bin_1d(float xi, float lower, float upper, int shape, int periodic) {
    volatile float invd = (float)((double)shape / ((double)upper - (double)lower));
    volatile float d = xi - lower;
    volatile float t = d * invd;
    float f = floorf(t);
    if (!(f == f)) return -1; /* NaN is outside */
    if (periodic) {
        double m = fmod((double)f, (double)shape);
        if (m < 0) m += shape;
        return (int)m;
    }
    if (f < 0.0f || f >= (float)shape) return -1;
    return (int)f;
}

/* ABF grid update, PAPER.md:L143 (Sec. 2.1.4), L501/L507 (N = threshold before
 * the full average is used).  For every replica: bin xi; in-grid -> hist[bin]+=1,
 * Fsum[bin][k] += f_k.  After ALL replicas have accumulated (two-phase, reading
 * R-ABF-3, parity unpinned) each reads Fbar_k = Fsum[bin][k]/max(hist[bin], N);
 * outside -> bin = -1 and Fbar = 0.  dVdxi := Fbar (reading R-ABF-4). */
void orc_abf_update(int n_replicas, int n_cv, const float *xi, const float *fsample, const float *lower,
                    const float *upper, const int *shape, const int *periodic, int n_threshold,
                    int *hist, double *fsum /*[nbins][n_cv]*/, int *bin_out, double *dVdxi) {
    int *bins = (int *)malloc(sizeof(int) * (size_t)n_replicas);
    for (int r = 0; r < n_replicas; ++r) {
        long long flat = 0;
        int inside = 1;
        for (int k = 0; k < n_cv; ++k) {
            int i = abf_bin_1d(xi[r * n_cv + k], lower[k], upper[k], shape[k], periodic[k]);
            if (i < 0) { inside = 0; break; }
            flat = flat * shape[k] + i; /* row-major, last CV fastest */
        }
        bins[r] = inside ? (int)flat : -1;
        if (inside) {
            hist[flat] += 1;
            for (int k = 0; k < n_cv; ++k) fsum[flat * n_cv + k] += (double)fsample[r * n_cv + k];
        }
    }
    for (int r = 0; r < n_replicas; ++r) {
        int b = bins[r];
        if (bin_out) bin_out[r] = b;
        for (int k = 0; k < n_cv; ++k) {
            double m = 0;
            if (b >= 0) {
                int cnt = hist[b] > n_threshold ? hist[b] : n_threshold;
                m = fsum[(long long)b * n_cv + k] / (double)cnt;
            }
            dVdxi[r * n_cv + k] = m;
        }
    }
    free(bins);
}

/* Bias forces, PAPER.md:L39 ("computed biasing forces are added to the backend
 * net forces"): force[i] += -sum_k dVdxi_k d(xi_k)/d(r_i), summed over every CV
 * and every replica that references atom i of that array.
 * force: fp64 [n_arrays][N][3], n_arrays = R (own arrays) or 1 (shared). */
void orc_apply_forces(const orc_layout *L, const orc_cv *cvs, const int *slot_atom, const float *slot_weight,
                      const float *atom_weight, const float *pos, const double *dVdxi, double *force) {
    int shared = L->replica_stride_atoms == 0;
    long long maxrows = 0;
    for (int k = 0; k < L->n_cv; ++k) { long long n = cv_natoms(&cvs[k]); if (n > maxrows) maxrows = n; }
#pragma omp parallel if (!shared)
    {
        double *jac = (double *)malloc(sizeof(double) * 3 * (size_t)maxrows);
#pragma omp for schedule(static)
        for (int r = 0; r < L->n_replicas; ++r) {
            const float *p = pos + (long long)r * L->replica_stride_atoms * L->pos_stride;
            double *f = force + (shared ? 0 : (long long)r * L->n_atoms * 3);
            const int *sa = slot_atom + (L->per_replica_slots ? (long long)r * L->n_slots : 0);
            for (int k = 0; k < L->n_cv; ++k) {
                const orc_cv *cv = &cvs[k];
                cv_one(cv, p, L->pos_stride, sa, slot_weight, atom_weight, orc_box(L), jac);
                double dv = dVdxi[(long long)r * L->n_cv + k];
                long long o = 0;
                for (int g = 0; g < cv->n_groups; ++g) {
                    long long n = group_count(cv, g);
                    for (long long i = 0; i < n; ++i, ++o) {
                        long long a = group_atom(cv, g, i, sa);
                        for (int x = 0; x < 3; ++x) f[a * 3 + x] += -dv * jac[3 * o + x];
                    }
                }
            }
        }
        free(jac);
    }
}

/* ABF instantaneous-force estimator.  PAPER.md:L143 says only "based on the algorithm described
 * in [43]" (Darve et al. 2008, not available here), so this follows SURVEY.md 8(f) / DESIGN.md reading R-ABF-EST:
 *   J[k][i] = d xi_k / d r_i over the atoms of the CVs (contributions of one atom to one CV through several slots add),
 *   p_i = m_i v_i,   G = J J^T  (n_cv x n_cv),   b = J p,   solve G W = b,
 *   dW/dt = (3/2 W(t) - 2 W(t - dt) + 1/2 W(t - 2 dt)) / dt      (second-order backward difference),
 *   fsample = dW/dt + Fbias_prev       (Fbias_prev = the mean force dV/dxi applied at the previous step: the atoms felt
 *                                       -Fbias_prev J, which is added back to recover the unbiased generalized force).
 * whist [R][2][n_cv] holds W(t - dt), W(t - 2 dt) and is advanced; first != 0 initialises both to W(t) (dW/dt = 0).
 * vel has the layout of pos; mass [n_atoms] is shared by the replicas.  A singular G gives W = 0 for that replica.
 * Pins: a constant and a linearly growing force on a free particle are recovered exactly (the difference formula is exact
 * for quadratics), W equals the least-squares solution of J^T W = p, momentum orthogonal to every row of J gives 0. */
void orc_abf_estimate(const orc_layout *L, const orc_cv *cvs, const int *slot_atom, const float *slot_weight,
                      const float *atom_weight, const float *pos, const float *vel, const float *mass, double dt,
                      const double *fbias_prev /*[R][n_cv], nullable = 0*/, double *whist /*[R][2][n_cv]*/, int first,
                      double *fsample /*[R][n_cv]*/, double *w_out /*[R][n_cv], nullable*/) {
    const int n_cv = L->n_cv;
    long long maxrows = 0;
    for (int k = 0; k < n_cv; ++k) { long long n = cv_natoms(&cvs[k]); if (n > maxrows) maxrows = n; }
    for (int r = 0; r < L->n_replicas; ++r) {
        const float *p = pos + (long long)r * L->replica_stride_atoms * L->pos_stride;
        const float *v = vel + (long long)r * L->replica_stride_atoms * L->pos_stride;
        const int *sa = slot_atom + (L->per_replica_slots ? (long long)r * L->n_slots : 0);
        /* dense rows of J over the atoms of this replica's array would be huge: keep (atom, vector) lists per CV */
        double *jac[4]; long long *atoms[4]; long long na[4];
        for (int k = 0; k < n_cv; ++k) {
            na[k] = cv_natoms(&cvs[k]);
            jac[k] = (double *)malloc(sizeof(double) * 3 * (size_t)na[k]);
            atoms[k] = (long long *)malloc(sizeof(long long) * (size_t)na[k]);
            cv_one(&cvs[k], p, L->pos_stride, sa, slot_weight, atom_weight, orc_box(L), jac[k]);
            long long o = 0;
            for (int g = 0; g < cvs[k].n_groups; ++g)
                for (long long i = 0; i < group_count(&cvs[k], g); ++i) atoms[k][o++] = group_atom(&cvs[k], g, i, sa);
        }
        double G[4][4] = {{0}}, b[4] = {0}, W[4] = {0};
        for (int k = 0; k < n_cv; ++k) {
            for (long long i = 0; i < na[k]; ++i) {
                long long a = atoms[k][i];
                double m = (double)mass[a];
                for (int x = 0; x < 3; ++x) b[k] += jac[k][3 * i + x] * m * (double)v[a * L->pos_stride + x];
                for (int l = 0; l < n_cv; ++l)
                    for (long long j = 0; j < na[l]; ++j)
                        if (atoms[l][j] == a)
                            for (int x = 0; x < 3; ++x) G[k][l] += jac[k][3 * i + x] * jac[l][3 * j + x];
            }
        }
        /* Gaussian elimination with partial pivoting on the augmented matrix */
        double A[4][5];
        int ok = 1;
        for (int k = 0; k < n_cv; ++k) { for (int l = 0; l < n_cv; ++l) A[k][l] = G[k][l]; A[k][n_cv] = b[k]; }
        for (int c = 0; c < n_cv && ok; ++c) {
            int piv = c;
            for (int k = c + 1; k < n_cv; ++k) if (fabs(A[k][c]) > fabs(A[piv][c])) piv = k;
            if (!(fabs(A[piv][c]) > 0)) { ok = 0; break; }
            if (piv != c) for (int l = 0; l <= n_cv; ++l) { double t = A[c][l]; A[c][l] = A[piv][l]; A[piv][l] = t; }
            for (int k = c + 1; k < n_cv; ++k) {
                double f = A[k][c] / A[c][c];
                for (int l = c; l <= n_cv; ++l) A[k][l] -= f * A[c][l];
            }
        }
        if (ok) for (int k = n_cv - 1; k >= 0; --k) {
            double s = A[k][n_cv];
            for (int l = k + 1; l < n_cv; ++l) s -= A[k][l] * W[l];
            W[k] = s / A[k][k];
        }
        double *h1 = whist + ((long long)r * 2 + 0) * n_cv, *h2 = whist + ((long long)r * 2 + 1) * n_cv;
        for (int k = 0; k < n_cv; ++k) {
            if (first) { h1[k] = W[k]; h2[k] = W[k]; }
            double dW = (1.5 * W[k] - 2.0 * h1[k] + 0.5 * h2[k]) / dt;
            fsample[(long long)r * n_cv + k] = dW + (fbias_prev ? fbias_prev[(long long)r * n_cv + k] : 0.0);
            if (w_out) w_out[(long long)r * n_cv + k] = W[k];
            h2[k] = h1[k]; h1[k] = W[k];
        }
        for (int k = 0; k < n_cv; ++k) { free(jac[k]); free(atoms[k]); }
    }
}

/* DistanceToInterface, the paper's own worked CV: PAPER.md:L203-L290 (Sec. 2.2.1, Eq. 4-8) and the
 * listing of Appendix A (L444-L475), followed line by line, for ONE replica:
 *   mobile_axis   = barycenter(p1)[axis]                                   (weighted by wm, NULL = 1)
 *   positions     = coordinate `axis` of every atom of p2                  (atoms [ibegin, ibegin + n_i) of the array)
 *   centers_j     = linspace(scope0, scope1, bins)
 *   mass_j        = sum_i exp(-1/2 ((x_i - centers_j) / sigma)^2)          (Eq. 6)
 *   mass_diff_j   = |mass_{j+1} - mass_j|,  centers_mean_j = (centers_{j+1} + centers_j) / 2      (Eq. 7 up to 1/delta)
 *   probability   = softmax(mass_diff * coeff);  interface = sum_j probability_j centers_mean_j   (Eq. 8)
 *   xi            = mobile_axis - interface
 * Derivatives (the paper takes them by autodiff; written out here): d xi/d r_m = (w_m / W) e_axis for mobile atoms;
 * for interface atoms d xi/d x_i = -sum_j G_j d mass_j/d x_i with d mass_j/d x_i = -e_ij (x_i - centers_j)/sigma^2 and
 * G_j = d interface/d mass_j = coeff [ s_{j-1} p_{j-1} (cm_{j-1} - I) - s_j p_j (cm_j - I) ], s_j = sign(mass_{j+1} - mass_j).
 * Outputs: *xi; jac_mobile [n_m][3]; dxi_dx [n_i] (nullable); mass_out [bins] (nullable). */
void orc_dist_to_interface(const float *pos, int ps, int n_m, const int *mobile_idx, const float *wm, long long ibegin,
                           long long n_i, int axis, double sigma, double scope0, double scope1, int bins, double coeff,
                           double *xi, double *jac_mobile, double *dxi_dx, double *mass_out) {
    double W = 0, mob = 0;
    for (int m = 0; m < n_m; ++m) {
        double w = wm ? (double)wm[m] : 1.0;
        mob += w * (double)pos[(long long)mobile_idx[m] * ps + axis];
        W += w;
    }
    mob /= W;
    double *c = (double *)malloc(sizeof(double) * (size_t)bins), *mass = (double *)calloc((size_t)bins, sizeof(double));
    for (int j = 0; j < bins; ++j) c[j] = bins > 1 ? scope0 + (scope1 - scope0) * (double)j / (double)(bins - 1) : scope0;
    for (int j = 0; j < bins; ++j)
        for (long long i = 0; i < n_i; ++i) {
            double d = ((double)pos[(ibegin + i) * ps + axis] - c[j]) / sigma;
            mass[j] += exp(-0.5 * d * d);
        }
    int nb = bins - 1;
    double *md = (double *)malloc(sizeof(double) * (size_t)nb), *p = (double *)malloc(sizeof(double) * (size_t)nb);
    double mx = -INFINITY, Z = 0, I = 0;
    for (int j = 0; j < nb; ++j) { md[j] = fabs(mass[j + 1] - mass[j]); if (md[j] * coeff > mx) mx = md[j] * coeff; }
    for (int j = 0; j < nb; ++j) { p[j] = exp(md[j] * coeff - mx); Z += p[j]; }      /* softmax, shifted by its maximum */
    for (int j = 0; j < nb; ++j) { p[j] /= Z; I += p[j] * 0.5 * (c[j + 1] + c[j]); }
    *xi = mob - I;
    if (jac_mobile)
        for (int m = 0; m < n_m; ++m)
            for (int x = 0; x < 3; ++x) jac_mobile[3 * m + x] = x == axis ? (wm ? (double)wm[m] : 1.0) / W : 0.0;
    if (dxi_dx) {
        double *G = (double *)calloc((size_t)bins, sizeof(double));
        for (int j = 0; j < nb; ++j) {
            double diff = mass[j + 1] - mass[j];
            double s = diff > 0 ? 1.0 : (diff < 0 ? -1.0 : 0.0);
            double t = coeff * s * p[j] * (0.5 * (c[j + 1] + c[j]) - I);   /* d I / d md_j times the sign of the difference */
            G[j + 1] += t;
            G[j] -= t;
        }
        for (long long i = 0; i < n_i; ++i) {
            double x = (double)pos[(ibegin + i) * ps + axis], dI = 0;
            for (int j = 0; j < bins; ++j) {
                double d = x - c[j];
                dI += G[j] * (-exp(-0.5 * (d / sigma) * (d / sigma)) * d / (sigma * sigma));
            }
            dxi_dx[i] = -dI;
        }
        free(G);
    }
    if (mass_out) memcpy(mass_out, mass, sizeof(double) * (size_t)bins);
    free(c); free(mass); free(md); free(p);
}

/* ---------------------------------------------------------------------------------------------------------------
 * Grid-stored metadynamics, PAPER.md:L151 ("optional support for storing the bias potentials ... on a pre-defined
 * grid", trading accuracy for speed).  The paper gives neither the layout nor the interpolation, so
 * this follows reading R-GRID of DESIGN.md:
 *   - Grid(lower, upper, shape, periodic) as in PAPER.md:L82.  CV k has shape[k] NODES; a periodic CV spans exactly
 *     one period upper - lower with spacing h = (upper - lower)/shape (node `shape` is node 0 again); an open CV has
 *     its first and last nodes on lower and upper, h = (upper - lower)/(shape - 1).
 *   - every node stores the hill sum of Eq. "sum of Gaussians" and its gradient, 1 + n_cv binary64
 *     numbers, node index row-major with the last CV fastest.
 *   - a deposit adds the new hill's value and gradient AT every node (orc_grid_deposit).
 *   - the bias at xi is the multilinear interpolation of the 2^n_cv surrounding nodes, value and each gradient
 *     component alike (orc_grid_eval); outside an open grid the CV is clamped to the nearest face first.
 *   - well-tempered heights use the interpolated value before the event; several walkers deposit synchronously in
 *     replica order (the readings R-WT and R-MW of the hill list).
 * Pins (tests/test_oracle_grid_metad.py): node values against the separately pinned hill sum (orc_metad), exact
 * reproduction of multilinear functions written straight into the grid, scipy's RegularGridInterpolator, the h^2
 * convergence to the exact hill sum, periodic images, well-tempered heights by hand.
 * --------------------------------------------------------------------------------------------------------------- */
typedef struct {
    int n_cv;
    double lower[4], upper[4];
    int shape[4];
    int periodic[4];
} orc_grid;

long long orc_grid_nodes(const orc_grid *G) {
    long long n = 1;
    for (int k = 0; k < G->n_cv; ++k) n *= G->shape[k];
    return n;
}

static double grid_spacing(const orc_grid *G, int k) {
    return (G->upper[k] - G->lower[k]) / (double)(G->periodic[k] ? G->shape[k] : G->shape[k] - 1);
}

/* V [R] and dVdxi [R][n_cv] by multilinear interpolation of grid [nodes][1 + n_cv] */
void orc_grid_eval(const orc_grid *G, const double *grid, int n_replicas, const double *xi, double *V, double *dVdxi) {
    const int n = G->n_cv, rec = 1 + n;
    for (int r = 0; r < n_replicas; ++r) {
        int i0[4];
        double f[4];
        for (int k = 0; k < n; ++k) {
            double t = (xi[r * n + k] - G->lower[k]) / grid_spacing(G, k);
            if (G->periodic[k]) {
                t -= (double)G->shape[k] * floor(t / (double)G->shape[k]);   /* into [0, shape) */
                if (t >= (double)G->shape[k]) t = 0.0;                      /* rounding at the upper edge */
                i0[k] = (int)floor(t);
            } else {
                if (t < 0.0) t = 0.0;
                if (t > (double)(G->shape[k] - 1)) t = (double)(G->shape[k] - 1);
                i0[k] = (int)floor(t);
                if (i0[k] > G->shape[k] - 2) i0[k] = G->shape[k] - 2;       /* the last cell owns its upper node */
                if (i0[k] < 0) i0[k] = 0;                                   /* a one-node dimension */
            }
            f[k] = t - (double)i0[k];
        }
        double out[5] = {0, 0, 0, 0, 0};
        for (int corner = 0; corner < (1 << n); ++corner) {
            double w = 1.0;
            long long flat = 0;
            for (int k = 0; k < n; ++k) {
                int up = (corner >> k) & 1;
                int i = i0[k] + up;
                if (G->periodic[k]) i %= G->shape[k];
                else if (i > G->shape[k] - 1) i = G->shape[k] - 1;
                w *= up ? f[k] : 1.0 - f[k];
                flat = flat * G->shape[k] + i;
            }
            for (int c = 0; c < rec; ++c) out[c] += w * grid[flat * rec + c];
        }
        if (V) V[r] = out[0];
        if (dVdxi) for (int k = 0; k < n; ++k) dVdxi[r * n + k] = out[1 + k];
    }
}

/* One synchronous deposit event of the walkers with mask[r] != 0 (NULL: all).  heights_out [R] (nullable) receives
 * the height each walker deposited (0 where masked out). */
void orc_grid_deposit(const orc_grid *G, double *grid, int n_replicas, const float *xi /*[R][n_cv]*/,
                      const unsigned char *mask, double w0, double kB_deltaT, const double *sigma, double *heights_out) {
    const int n = G->n_cv, rec = 1 + n;
    const long long nodes = orc_grid_nodes(G);
    double *xd = (double *)malloc(sizeof(double) * (size_t)n_replicas * n);
    double *Vold = (double *)malloc(sizeof(double) * (size_t)n_replicas);
    for (long long i = 0; i < (long long)n_replicas * n; ++i) xd[i] = (double)xi[i];
    orc_grid_eval(G, grid, n_replicas, xd, Vold, NULL);       /* every height from the grid BEFORE this event */
    for (int r = 0; r < n_replicas; ++r) {
        double W = 0.0;
        if (!mask || mask[r]) {
            W = kB_deltaT > 0 ? w0 * exp(-Vold[r] / kB_deltaT) : w0;
            for (long long node = 0; node < nodes; ++node) {
                long long rem = node;
                double d[4], e = 0;
                for (int k = n - 1; k >= 0; --k) {
                    int i = (int)(rem % G->shape[k]);
                    rem /= G->shape[k];
                    double x = G->lower[k] + (double)i * grid_spacing(G, k);
                    d[k] = wrap_period(x - xd[r * n + k], G->periodic[k] ? G->upper[k] - G->lower[k] : 0.0);
                    e += (d[k] / sigma[k]) * (d[k] / sigma[k]);
                }
                double g = W * exp(-0.5 * e);
                grid[node * rec] += g;
                for (int k = 0; k < n; ++k) grid[node * rec + 1 + k] += -g * d[k] / (sigma[k] * sigma[k]);
            }
        }
        if (heights_out) heights_out[r] = W;
    }
    free(xd); free(Vold);
}
