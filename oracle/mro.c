/*
 * oracle/mro.c -- plain, slow, obviously-correct CPU restatement of the relaxation step of
 * Candelaresi, Pontin & Hornig, "Mimetic methods for Lagrangian relaxation of magnetic fields"
 * (arxiv 1405.0942; text in PAPER.md).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header, table or
 * helper with the CUDA path (paper_1405_0942_b200/csrc, include/mr.h) and neither includes the other.
 *
 * Everything is fp64 scalar loops over nodes in the paper's order and notation; nothing is blocked, fused
 * or algebraically shortened.  The mimetic curl is the literal Eqs. 2.3-2.7 (edge-by-edge circulation, four
 * triangles about x_ijk, |nA|, unit normals, 3x3 solve).  Citations are PAPER.md line numbers.
 *
 * Layout: a vector field is double[3][nz][ny][nx], idx = (k*ny + j)*nx + i  (i = x-direction fastest).
 * n[3] = {nx, ny, nz}; reference grid X_a = lo_a + idx_a*h_a, h_a = (hi_a-lo_a)/(n_a-1).
 *
 * Readings of the paper where it is silent:
 *   Q1  loop points I..IV are the four nearest neighbours +a, +b, -a, -b in the index surface (a,b);
 *   Q2  A = |sum_r n_r A_r| (norm of the vector sum, Eqs. 2.4/2.6/2.7);
 *   Q3  dx/dX: 2nd-order central differences inside, 2nd-order one-sided 3-point normal to a face
 *       -- the paper does not state its stencil (:257 says "second-order"); pinned through the whole chain only: the
 *       relaxed states of TABLES 4.1 / 4.2 (tests/test_oracle_next.py) come out to the paper's printed digits;
 *   Q4  the "classical" operator is the analytic product/chain-rule expansion of Eq. 2.1 (:49), formulas
 *       re-derived here because Craig & Sneyd (1986) is not available -- parity UNPINNED against the paper;
 *   Q5  time stepping on this path is forward Euler with all u from the old x;
 *   Q8  line-tied on all six faces: boundary nodes never move, J and u are 0 there;
 *   Q9  xi = max over interior nodes of the pointwise ratio |JxB|/|B|^2.
 *   Q12 periodic axis (Eqs. 2.12-2.14, :147-164): every node of the axis is an inner point, the ghost nodes are
 *       x(f-1) = x(l) - (L + dX) e_a and x(l+1) = x(f) + (L + dX) e_a with L = X_l - X_f, i.e. the period is n_a h_a;
 *       B(X,0) is periodic;
 *   Q22 integrator (section 2.4, :131-143): Cash-Karp RK5(4), the step advances with the fifth-order solution,
 *       Lambda = max over nodes and components of |x5 - x4|; reject if Lambda > Lambda0 and retry with Eq. 2.11;
 *       accept otherwise, and enlarge dt by Eq. 2.11 if Lambda < Lambda0/2 (growth capped at 5x: Lambda may be 0);
 *       the last step is clipped to end at t_end without changing the dt handed on; a recomputation uses at most 0.9 dt;
 *   Q26 a trial in which a stage folds the grid (det <= 0 or non-finite) is rejected and recomputed with dt/2; 40 such
 *       trials in a row stop the run (:333 "a drop of the time step by several orders of magnitude, at which point the
 *       simulation is stopped");
 *   Q23 convexity (Eqs. 3.10-3.11, :231-243): kappa(node) = 1 iff every trihedron of the node whose three
 *       neighbours exist has sgn det = di dj dk, else -1;
 *   Q24 eps* (Eq. 3.7, :214): alpha* = J.B/B^2 at the interior nodes of the grid line through (i_c, j_c), maximum
 *       over ordered pairs of a_r (alpha*_i - alpha*_j)/|X_i - X_j|.
 *
 * Return codes: 0 ok, 1 bad argument, 5 numeric failure (det <= 0, non-finite, or singular normal matrix).
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MRO_OK 0
#define MRO_BADARG 1
#define MRO_NUMERIC 5

static int g_threads = 1; /* OpenMP threads used by the grid loops; 1 unless the timing harness raises it */

void mro_set_threads(int t) { g_threads = t < 1 ? 1 : t; }
int mro_get_threads(void) { return g_threads; }
int mro_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_num_procs();
#else
    return 1;
#endif
}

typedef struct {
    int nx, ny, nz;
    size_t N;
    double h[3];
    double lo[3];
    int per[3];    /* 1 = periodic axis (Eqs. 2.12-2.14), 0 = line-tied faces */
    double P[3];   /* period n_a h_a = L_a + dX_a (reading Q12) */
} grid_t;

/* Boundary type per logical axis for every call that follows: 0 line-tied (default), 1 periodic.  A process-wide
 * setting (the oracle is single-user test infrastructure); the Python wrapper sets it around each call. */
static int g_bc[3] = { 0, 0, 0 };
void mro_set_bc(const int bc[3]) { for (int a = 0; a < 3; ++a) g_bc[a] = bc ? (bc[a] != 0) : 0; }

static int make_grid(const int n[3], const double lo[3], const double hi[3], grid_t* g)
{
    if (!n || n[0] < 3 || n[1] < 3 || n[2] < 3) return MRO_BADARG;
    g->nx = n[0]; g->ny = n[1]; g->nz = n[2];
    g->N = (size_t)n[0] * (size_t)n[1] * (size_t)n[2];
    for (int a = 0; a < 3; ++a) {
        if (lo && hi) {
            if (!(hi[a] > lo[a])) return MRO_BADARG;
            g->h[a] = (hi[a] - lo[a]) / (double)(n[a] - 1);
            g->lo[a] = lo[a];
        } else {
            g->h[a] = 1.0; g->lo[a] = 0.0;
        }
        g->per[a] = g_bc[a];
        g->P[a] = (double)n[a] * g->h[a];
    }
    return MRO_OK;
}

static inline size_t at(const grid_t* g, int i, int j, int k)
{
    return ((size_t)k * (size_t)g->ny + (size_t)j) * (size_t)g->nx + (size_t)i;
}

/* Value of one component f of a nodal field at an index that may lie one or two nodes outside a PERIODIC axis: the
 * index is wrapped (B is periodic, Eq. 2.14); if f is the component `shift` of the positions x, the ghost value is
 * shifted by -/+ (L + dX) along that axis (Eqs. 2.12, 2.13).  shift = -1 for periodic fields. */
static double val(const grid_t* g, const double* f, int shift, int i, int j, int k)
{
    int idx[3] = { i, j, k };
    const int n[3] = { g->nx, g->ny, g->nz };
    double add = 0.0;
    for (int a = 0; a < 3; ++a) {
        if (idx[a] < 0) { idx[a] += n[a]; if (a == shift) add -= g->P[a]; }
        else if (idx[a] >= n[a]) { idx[a] -= n[a]; if (a == shift) add += g->P[a]; }
    }
    return f[at(g, idx[0], idx[1], idx[2])] + add;
}

/* is the node an inner point along every axis (line-tied faces excluded, periodic axes have no faces)? */
static int inner_node(const grid_t* g, int i, int j, int k)
{
    return (g->per[0] || (i > 0 && i < g->nx - 1)) && (g->per[1] || (j > 0 && j < g->ny - 1)) && (g->per[2] || (k > 0 && k < g->nz - 1));
}

/* X_ijk, the fixed reference grid ("x(X,0)=X"; :170 rectangular grid). */
int mro_reference_grid(const int n[3], const double lo[3], const double hi[3], double* X)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                size_t p = at(&g, i, j, k);
                X[0 * g.N + p] = g.lo[0] + (double)i * g.h[0];
                X[1 * g.N + p] = g.lo[1] + (double)j * g.h[1];
                X[2 * g.N + p] = g.lo[2] + (double)k * g.h[2];
            }
    return MRO_OK;
}

/* ---- O1: first derivative of a nodal scalar along logical axis a at node (i,j,k) (reading Q3) ---------- */
static double ddX(const grid_t* g, const double* f, int a, int i, int j, int k, int shift)
{
    int idx[3] = { i, j, k };
    if (g->per[a]) {              /* periodic axis: central everywhere, ghosts by Eqs. 2.12-2.14 */
        int p[3] = { i, j, k }, m[3] = { i, j, k };
        p[a] += 1; m[a] -= 1;
        return (val(g, f, shift, p[0], p[1], p[2]) - val(g, f, shift, m[0], m[1], m[2])) / (2.0 * g->h[a]);
    }
    int na = (a == 0) ? g->nx : (a == 1) ? g->ny : g->nz;
    int c = idx[a];
    int p1[3] = { i, j, k }, p2[3] = { i, j, k };
    double two_h = 2.0 * g->h[a];
    if (c == 0) {                 /* one-sided, nodes 0,1,2 :  (-3 f0 + 4 f1 - f2) / 2h */
        p1[a] = 1; p2[a] = 2;
        return (-3.0 * f[at(g, i, j, k)] + 4.0 * f[at(g, p1[0], p1[1], p1[2])] - f[at(g, p2[0], p2[1], p2[2])]) / two_h;
    } else if (c == na - 1) {     /* one-sided, nodes n-1,n-2,n-3 : (3 f0 - 4 f-1 + f-2) / 2h */
        p1[a] = na - 2; p2[a] = na - 3;
        return (3.0 * f[at(g, i, j, k)] - 4.0 * f[at(g, p1[0], p1[1], p1[2])] + f[at(g, p2[0], p2[1], p2[2])]) / two_h;
    }
    p1[a] = c + 1; p2[a] = c - 1; /* central: (f+ - f-) / 2h */
    return (f[at(g, p1[0], p1[1], p1[2])] - f[at(g, p2[0], p2[1], p2[2])]) / two_h;
}

static double det3(const double F[3][3])
{   /* cofactor expansion along the first row (O2) */
    return F[0][0] * (F[1][1] * F[2][2] - F[1][2] * F[2][1])
         - F[0][1] * (F[1][0] * F[2][2] - F[1][2] * F[2][0])
         + F[0][2] * (F[1][0] * F[2][1] - F[1][1] * F[2][0]);
}

/* F_ia = dx_i/dX_a at one node (Eq. 2.1). */
static void jacobian_at(const grid_t* g, const double* x, int i, int j, int k, double F[3][3])
{
    for (int c = 0; c < 3; ++c)
        for (int a = 0; a < 3; ++a)
            F[c][a] = ddX(g, x + (size_t)c * g->N, a, i, j, k, c);
}

/* O1+O2 on all nodes: F[(c*3+a)*N + p] = dx_c/dX_a, det[p] = Delta.  F or det may be NULL. */
int mro_jacobian(const int n[3], const double lo[3], const double hi[3], const double* x, double* F, double* det)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    int bad = 0;
#pragma omp parallel for num_threads(g_threads) reduction(| : bad)
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                double Fl[3][3];
                jacobian_at(&g, x, i, j, k, Fl);
                double d = det3(Fl);
                size_t p = at(&g, i, j, k);
                if (F) for (int c = 0; c < 3; ++c) for (int a = 0; a < 3; ++a) F[(size_t)(c * 3 + a) * g.N + p] = Fl[c][a];
                if (det) det[p] = d;
                if (!(d > 0.0) || !isfinite(d)) bad = 1;
            }
    return bad ? MRO_NUMERIC : MRO_OK;
}

/* O3: B_i = (1/Delta) sum_a F_ia B0_a on ALL nodes (Eq. 2.1).  det may be NULL. */
int mro_push_forward(const int n[3], const double lo[3], const double hi[3], const double* x, const double* B0,
                     double* B, double* det)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    int bad = 0;
#pragma omp parallel for num_threads(g_threads) reduction(| : bad)
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                double F[3][3];
                jacobian_at(&g, x, i, j, k, F);
                double d = det3(F);
                size_t p = at(&g, i, j, k);
                if (!(d > 0.0) || !isfinite(d)) bad = 1;
                for (int c = 0; c < 3; ++c) {
                    double s = 0.0;
                    for (int a = 0; a < 3; ++a) s += F[c][a] * B0[(size_t)a * g.N + p];
                    B[(size_t)c * g.N + p] = s / d;
                }
                if (det) det[p] = d;
            }
    return bad ? MRO_NUMERIC : MRO_OK;
}

static void cross3(const double a[3], const double b[3], double c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

/* Solve M J = r (3x3) by Gaussian elimination with partial pivoting.  0 ok, 1 singular. */
static int solve3(double M[3][3], double r[3], double J[3])
{
    for (int col = 0; col < 3; ++col) {
        int piv = col; double big = fabs(M[col][col]);
        for (int row = col + 1; row < 3; ++row) if (fabs(M[row][col]) > big) { big = fabs(M[row][col]); piv = row; }
        if (!(big > 0.0) || !isfinite(big)) return 1;
        if (piv != col) {
            for (int c = 0; c < 3; ++c) { double t = M[col][c]; M[col][c] = M[piv][c]; M[piv][c] = t; }
            double t = r[col]; r[col] = r[piv]; r[piv] = t;
        }
        for (int row = col + 1; row < 3; ++row) {
            double f = M[row][col] / M[col][col];
            for (int c = col; c < 3; ++c) M[row][c] -= f * M[col][c];
            r[row] -= f * r[col];
        }
    }
    for (int row = 2; row >= 0; --row) {
        double s = r[row];
        for (int c = row + 1; c < 3; ++c) s -= M[row][c] * J[c];
        J[row] = s / M[row][row];
    }
    return 0;
}

static void load3(const grid_t* g, const double* f, int i, int j, int k, double v[3])
{
    size_t p = at(g, i, j, k);
    v[0] = f[p]; v[1] = f[g->N + p]; v[2] = f[2 * g->N + p];
}
/* neighbour values across a periodic face: positions (shifted ghost, Eqs. 2.12/2.13) and periodic fields (Eq. 2.14) */
static void load3x(const grid_t* g, const double* x, int i, int j, int k, double v[3])
{
    for (int c = 0; c < 3; ++c) v[c] = val(g, x + (size_t)c * g->N, c, i, j, k);
}
static void load3f(const grid_t* g, const double* f, int i, int j, int k, double v[3])
{
    for (int c = 0; c < 3; ++c) v[c] = val(g, f + (size_t)c * g->N, -1, i, j, k);
}

/*
 * O4m at one interior node: the nearest-neighbour mimetic curl, literally.
 * For each of the three index surfaces (a,b) = (j,k), (k,i), (i,j) through x_ijk:
 *   loop points  I = +a, II = +b, III = -a, IV = -b                        (Fig. 2.1, reading Q1)
 *   dx_r = x_{r+1} - x_r,  B_r = (B(X_r) + B(X_{r+1}))/2  (cyclic)          (:80)
 *   circulation  sum_r B_r . dx_r                                          (Eq. 2.3, :74)
 *   n_r A_r = (x_r - x_ijk) x (x_{r+1} - x_ijk)/2, nA = sum_r n_r A_r      (Eqs. 2.5, 2.4; :86-90, :82)
 *   J . n = circulation / A,   A = |nA|, n = nA/A                          (Eq. 2.7, :98; reading Q2)
 * and the three equations are solved for J by inverting the matrix of normals (:101-103).
 */
static int curl_mimetic_at(const grid_t* g, const double* x, const double* B, int i, int j, int k, double J[3])
{
    static const int surf[3][2] = { { 1, 2 }, { 2, 0 }, { 0, 1 } };
    double xc[3]; load3(g, x, i, j, k, xc);
    double M[3][3], rhs[3];
    for (int s = 0; s < 3; ++s) {
        int a = surf[s][0], b = surf[s][1];
        int off[4][3] = { { 0, 0, 0 }, { 0, 0, 0 }, { 0, 0, 0 }, { 0, 0, 0 } };
        off[0][a] = +1; off[1][b] = +1; off[2][a] = -1; off[3][b] = -1;
        double xr[4][3], Br[4][3];
        for (int r = 0; r < 4; ++r) {
            load3x(g, x, i + off[r][0], j + off[r][1], k + off[r][2], xr[r]);
            load3f(g, B, i + off[r][0], j + off[r][1], k + off[r][2], Br[r]);
        }
        double circ = 0.0, nA[3] = { 0.0, 0.0, 0.0 };
        for (int r = 0; r < 4; ++r) {
            int r1 = (r + 1) % 4;
            double dx[3], Bm[3], e0[3], e1[3], tri[3];
            for (int c = 0; c < 3; ++c) {
                dx[c] = xr[r1][c] - xr[r][c];
                Bm[c] = 0.5 * (Br[r][c] + Br[r1][c]);
                e0[c] = xr[r][c] - xc[c];
                e1[c] = xr[r1][c] - xc[c];
            }
            circ += Bm[0] * dx[0] + Bm[1] * dx[1] + Bm[2] * dx[2];
            cross3(e0, e1, tri);
            for (int c = 0; c < 3; ++c) nA[c] += 0.5 * tri[c];
        }
        double A = sqrt(nA[0] * nA[0] + nA[1] * nA[1] + nA[2] * nA[2]);
        if (!(A > 0.0) || !isfinite(A)) return 1;
        for (int c = 0; c < 3; ++c) M[s][c] = nA[c] / A;
        rhs[s] = circ / A;
    }
    return solve3(M, rhs, J);
}

/* O4m on the grid: J at interior nodes from GIVEN nodal x and B; J = 0 on boundary nodes (reading Q8). */
/* (lo/hi may be NULL when no axis is periodic: the operator itself does not use the spacing, only the period does) */
int mro_curl_mimetic_dom(const int n[3], const double lo[3], const double hi[3], const double* x, const double* B, double* J)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    if ((!lo || !hi) && (g.per[0] || g.per[1] || g.per[2])) return MRO_BADARG;
    int bad = 0;
    memset(J, 0, 3 * g.N * sizeof(double));
#pragma omp parallel for num_threads(g_threads) reduction(| : bad)
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                double Jl[3];
                if (!inner_node(&g, i, j, k)) continue;
                if (curl_mimetic_at(&g, x, B, i, j, k, Jl)) { bad = 1; continue; }
                size_t p = at(&g, i, j, k);
                for (int c = 0; c < 3; ++c) J[(size_t)c * g.N + p] = Jl[c];
            }
    return bad ? MRO_NUMERIC : MRO_OK;
}

int mro_curl_mimetic(const int n[3], const double* x, const double* B, double* J)
{
    return mro_curl_mimetic_dom(n, NULL, NULL, x, B, J);
}

/* second derivative d2 f / dX_a dX_b at an interior node (compact central differences, reading Q4) */
static double d2dX(const grid_t* g, const double* f, int a, int b, int i, int j, int k, int shift)
{
    int o[3] = { i, j, k };
    if (a == b) {
        int p[3] = { i, j, k }, m[3] = { i, j, k };
        p[a] += 1; m[a] -= 1;
        return (val(g, f, shift, p[0], p[1], p[2]) - 2.0 * f[at(g, o[0], o[1], o[2])] + val(g, f, shift, m[0], m[1], m[2])) / (g->h[a] * g->h[a]);
    }
    int pp[3] = { i, j, k }, pm[3] = { i, j, k }, mp[3] = { i, j, k }, mm[3] = { i, j, k };
    pp[a] += 1; pp[b] += 1;
    pm[a] += 1; pm[b] -= 1;
    mp[a] -= 1; mp[b] += 1;
    mm[a] -= 1; mm[b] -= 1;
    return (val(g, f, shift, pp[0], pp[1], pp[2]) - val(g, f, shift, pm[0], pm[1], pm[2]) - val(g, f, shift, mp[0], mp[1], mp[2])
            + val(g, f, shift, mm[0], mm[1], mm[2]))
           / (4.0 * g->h[a] * g->h[b]);
}

static void inverse3(const double F[3][3], double d, double Fi[3][3])
{   /* adjugate / determinant */
    Fi[0][0] = (F[1][1] * F[2][2] - F[1][2] * F[2][1]) / d;
    Fi[0][1] = (F[0][2] * F[2][1] - F[0][1] * F[2][2]) / d;
    Fi[0][2] = (F[0][1] * F[1][2] - F[0][2] * F[1][1]) / d;
    Fi[1][0] = (F[1][2] * F[2][0] - F[1][0] * F[2][2]) / d;
    Fi[1][1] = (F[0][0] * F[2][2] - F[0][2] * F[2][0]) / d;
    Fi[1][2] = (F[0][2] * F[1][0] - F[0][0] * F[1][2]) / d;
    Fi[2][0] = (F[1][0] * F[2][1] - F[1][1] * F[2][0]) / d;
    Fi[2][1] = (F[0][1] * F[2][0] - F[0][0] * F[2][1]) / d;
    Fi[2][2] = (F[0][0] * F[1][1] - F[0][1] * F[1][0]) / d;
}

/*
 * O4d at one interior node: the "classical"/direct-derivative curl: J = curl_x B with
 * B = F B0 / Delta (Eq. 2.1) differentiated analytically -- products of first and second derivatives of x.
 *   N_i      = F_ij B0_j
 *   N_{i,a}  = H_ija B0_j + F_ij G_ja,      H_ija = d2 x_i/dX_j dX_a,  G_ja = dB0_j/dX_a
 *   D_{,a}   = Delta (F^-1)_bi H_iba        (Jacobi's formula)
 *   B_{i,a}  = N_{i,a}/Delta - N_i D_{,a}/Delta^2
 *   dB_i/dx_m = B_{i,a} (F^-1)_am ,  J_l = eps_lmi dB_i/dx_m.
 */
static int curl_direct_at(const grid_t* g, const double* x, const double* B0, int i, int j, int k, double J[3])
{
    double F[3][3], Fi[3][3], H[3][3][3], G[3][3], b0[3];
    jacobian_at(g, x, i, j, k, F);
    double d = det3(F);
    if (!(d > 0.0) || !isfinite(d)) return 1;
    inverse3(F, d, Fi);
    for (int c = 0; c < 3; ++c)
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b)
                H[c][a][b] = d2dX(g, x + (size_t)c * g->N, a, b, i, j, k, c);
    for (int c = 0; c < 3; ++c)
        for (int a = 0; a < 3; ++a)
            G[c][a] = ddX(g, B0 + (size_t)c * g->N, a, i, j, k, -1);
    load3(g, B0, i, j, k, b0);

    double Nv[3], dN[3][3], dD[3], dB[3][3], dBdx[3][3];
    for (int c = 0; c < 3; ++c) {
        Nv[c] = 0.0;
        for (int q = 0; q < 3; ++q) Nv[c] += F[c][q] * b0[q];
    }
    for (int c = 0; c < 3; ++c)
        for (int a = 0; a < 3; ++a) {
            double s = 0.0;
            for (int q = 0; q < 3; ++q) s += H[c][q][a] * b0[q] + F[c][q] * G[q][a];
            dN[c][a] = s;
        }
    for (int a = 0; a < 3; ++a) {
        double s = 0.0;
        for (int b = 0; b < 3; ++b)
            for (int c = 0; c < 3; ++c) s += Fi[b][c] * H[c][b][a];
        dD[a] = d * s;
    }
    for (int c = 0; c < 3; ++c)
        for (int a = 0; a < 3; ++a)
            dB[c][a] = dN[c][a] / d - Nv[c] * dD[a] / (d * d);
    for (int c = 0; c < 3; ++c)
        for (int m = 0; m < 3; ++m) {
            double s = 0.0;
            for (int a = 0; a < 3; ++a) s += dB[c][a] * Fi[a][m];
            dBdx[c][m] = s;   /* dB_c/dx_m */
        }
    J[0] = dBdx[2][1] - dBdx[1][2];
    J[1] = dBdx[0][2] - dBdx[2][0];
    J[2] = dBdx[1][0] - dBdx[0][1];
    return 0;
}

/* O4d on the grid: J at interior nodes from x and B0; 0 on boundary nodes. */
int mro_curl_direct(const int n[3], const double lo[3], const double hi[3], const double* x, const double* B0, double* J)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    int bad = 0;
    memset(J, 0, 3 * g.N * sizeof(double));
#pragma omp parallel for num_threads(g_threads) reduction(| : bad)
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                double Jl[3];
                if (!inner_node(&g, i, j, k)) continue;
                if (curl_direct_at(&g, x, B0, i, j, k, Jl)) { bad = 1; continue; }
                size_t p = at(&g, i, j, k);
                for (int c = 0; c < 3; ++c) J[(size_t)c * g.N + p] = Jl[c];
            }
    return bad ? MRO_NUMERIC : MRO_OK;
}

/*
 * Fields of the current state: B on all nodes (O1-O3), J on interior nodes by operator op (0 mimetic O4m,
 * 1 direct O4d), u = gamma J x B on interior nodes and 0 on the boundary (O5; Eq. 1.5 :40, :147).
 * Any of B, J, u, det may be NULL.
 */
int mro_fields(const int n[3], const double lo[3], const double hi[3], const double* x, const double* B0,
               double gamma, int op, double* B, double* J, double* u, double* det)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    if (op != 0 && op != 1) return MRO_BADARG;
    double* Bl = B ? B : (double*)malloc(3 * g.N * sizeof(double));
    double* Jl = J ? J : (double*)malloc(3 * g.N * sizeof(double));
    if (!Bl || !Jl) return MRO_BADARG;
    rc = mro_push_forward(n, lo, hi, x, B0, Bl, det);
    int rc2 = (op == 0) ? mro_curl_mimetic_dom(n, lo, hi, x, Bl, Jl) : mro_curl_direct(n, lo, hi, x, B0, Jl);
    if (u) {
        /* J is 0 on boundary nodes, hence u = 0 there (line-tied, :147) */
#pragma omp parallel for num_threads(g_threads)
        for (long long p = 0; p < (long long)g.N; ++p) {
            double a[3] = { Jl[p], Jl[g.N + p], Jl[2 * g.N + p] };
            double b[3] = { Bl[p], Bl[g.N + p], Bl[2 * g.N + p] };
            double c[3]; cross3(a, b, c);
            for (int q = 0; q < 3; ++q) u[(size_t)q * g.N + p] = gamma * c[q];
        }
    }
    if (!B) free(Bl);
    if (!J) free(Jl);
    return rc ? rc : rc2;
}

/* O6: nsteps forward-Euler steps x <- x + dt*u(x) in place (Eq. 1.2 :17; reading Q5). Stops at the first
 * numeric failure and returns 5 (x then holds the last state whose velocity could not be formed). */
int mro_step(const int n[3], const double lo[3], const double hi[3], double* x, const double* B0,
             double gamma, double dt, long long nsteps, int op)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    if (nsteps < 0 || !(dt > 0.0)) return MRO_BADARG;
    double* u = (double*)malloc(3 * g.N * sizeof(double));
    if (!u) return MRO_BADARG;
    for (long long s = 0; s < nsteps; ++s) {
        rc = mro_fields(n, lo, hi, x, B0, gamma, op, NULL, NULL, u, NULL);
        if (rc) break;
#pragma omp parallel for num_threads(g_threads)
        for (long long p = 0; p < (long long)(3 * g.N); ++p) x[p] += dt * u[p];
    }
    free(u);
    return rc;
}

/*
 * O7: diagnostics of a state.  out[0] = E_M = 1/2 sum zeta |B|^2 Delta dXdYdZ over ALL nodes, zeta = 1/2 per
 * face the node lies on (Eq. 3.13 :251, :249);  out[1] = max over interior nodes of |J x B|;
 * out[2] = xi = max over interior nodes of |J x B|/|B|^2 (Eq. 4.1 :264, reading Q9);  out[3] = min Delta.
 * The energy is summed in long double, plane by plane in index order.
 */
int mro_diagnostics(const int n[3], const double lo[3], const double hi[3], const double* x, const double* B0,
                    int op, double out[4])
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    double* B = (double*)malloc(3 * g.N * sizeof(double));
    double* J = (double*)malloc(3 * g.N * sizeof(double));
    double* det = (double*)malloc(g.N * sizeof(double));
    if (!B || !J || !det) return MRO_BADARG;
    rc = mro_fields(n, lo, hi, x, B0, 1.0, op, B, J, NULL, det);
    long double E = 0.0L;
    double fmax = 0.0, xi = 0.0, dmin = INFINITY;
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                size_t p = at(&g, i, j, k);
                double b[3] = { B[p], B[g.N + p], B[2 * g.N + p] };
                double b2 = b[0] * b[0] + b[1] * b[1] + b[2] * b[2];
                double zeta = 1.0;
                if (!g.per[0] && (i == 0 || i == g.nx - 1)) zeta *= 0.5;
                if (!g.per[1] && (j == 0 || j == g.ny - 1)) zeta *= 0.5;
                if (!g.per[2] && (k == 0 || k == g.nz - 1)) zeta *= 0.5;
                E += (long double)(zeta * b2 * det[p]);
                if (det[p] < dmin || isnan(det[p])) dmin = det[p];
                int interior = inner_node(&g, i, j, k);
                if (interior) {
                    double jv[3] = { J[p], J[g.N + p], J[2 * g.N + p] }, f[3];
                    cross3(jv, b, f);
                    double fm = sqrt(f[0] * f[0] + f[1] * f[1] + f[2] * f[2]);
                    if (fm > fmax) fmax = fm;
                    if (fm / b2 > xi) xi = fm / b2;
                }
            }
    out[0] = (double)(0.5L * E * (long double)g.h[0] * (long double)g.h[1] * (long double)g.h[2]);
    out[1] = fmax; out[2] = xi; out[3] = dmin;
    free(B); free(J); free(det);
    return rc;
}

/* =========================================================================================================
 * Time stepping of section 2.4: the fifth-order adaptive Runge-Kutta formula of Cash & Karp
 * ([4] of the paper) with the embedded fourth-order solution, step control by Eq. 2.11 (reading Q22).
 * ========================================================================================================= */

/* Butcher tableau of the Cash-Karp pair (Cash & Karp 1990; also Press et al., the paper's [21]). */
static const double CK_A[6][5] = {
    { 0.0, 0.0, 0.0, 0.0, 0.0 },
    { 1.0 / 5.0, 0.0, 0.0, 0.0, 0.0 },
    { 3.0 / 40.0, 9.0 / 40.0, 0.0, 0.0, 0.0 },
    { 3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0, 0.0, 0.0 },
    { -11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0, 0.0 },
    { 1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0 } };
static const double CK_B5[6] = { 37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0 };
static const double CK_B4[6] = { 2825.0 / 27648.0, 0.0, 18575.0 / 48384.0, 13525.0 / 55296.0, 277.0 / 14336.0, 1.0 / 4.0 };

/* right-hand side of an autonomous system y' = f(y) with m unknowns; returns 0 or an error code */
typedef int (*mro_rhs_fn)(const double* y, double* dydt, void* user);

/*
 * One trial step of size dt from y (m values): y5 = fifth-order, y4 = embedded fourth-order solution (either may
 * be NULL), *lambda = max_q |y5_q - y4_q| (the "maximum error").  Stage s evaluates f at
 * y + dt sum_{r<s} a_sr k_r; work must hold 7 m doubles.  Plain loops in the order of the tableau.
 */
int mro_cash_karp_trial(long long m, const double* y, double dt, mro_rhs_fn f, void* user, double* y5, double* y4,
                        double* lambda, double* work)
{
    double* k[6];
    for (int s = 0; s < 6; ++s) k[s] = work + (size_t)s * (size_t)m;
    double* ys = work + (size_t)6 * (size_t)m;
    for (int s = 0; s < 6; ++s) {
        for (long long q = 0; q < m; ++q) {
            double acc = 0.0;
            for (int r = 0; r < s; ++r) acc += CK_A[s][r] * k[r][q];
            ys[q] = y[q] + dt * acc;
        }
        int rc = f(ys, k[s], user);
        if (rc) return rc;
    }
    double lam = 0.0;
    for (long long q = 0; q < m; ++q) {
        double s5 = 0.0, s4 = 0.0;
        for (int s = 0; s < 6; ++s) { s5 += CK_B5[s] * k[s][q]; s4 += CK_B4[s] * k[s][q]; }
        double v5 = y[q] + dt * s5, v4 = y[q] + dt * s4;
        double e = fabs(v5 - v4);
        if (e > lam || isnan(e)) lam = e;
        if (y5) y5[q] = v5;
        if (y4) y4[q] = v4;
    }
    *lambda = lam;
    return MRO_OK;
}

/* Eq. 2.11: dt' = dt |Lambda0 / Lambda|^0.2 */
static double eq_2_11(double dt, double Lambda, double Lambda0)
{
    return dt * pow(fabs(Lambda0 / Lambda), 0.2);
}

/*
 * The step control as section 2.4 words it, sentence by sentence.  Returns 1 if the result of the
 * trial is kept, 0 if it "is rejected and recomputed with dt = dt'"; *dt_prime is the step length to go on with.
 * Three guards are not in the paper's text; each is a separate clause below and a reading in DESIGN.md:
 *   Q22a  a recomputation is tried with at most 0.9 dt: just above Lambda0 the factor of Eq. 2.11 rounds to 1 and the very
 *         same trial would be recomputed for ever (met at Lambda = 1.0000000000000002e-8, Lambda0 = 1e-8 on the IsoHelix
 *         run of TABLE 4.1); 0.9 is the safety factor of the stepper the paper cites for its error measure ([21]);
 *   Q22b  an increase is at most 5 dt: Lambda may be 0 (a state at rest), where Eq. 2.11 has no value;
 *   Q26   a trial without an error measure (Lambda is NaN) is treated like one that folded the grid: recomputed with dt/2.
 */
int mro_step_control(double dt, double Lambda, double Lambda0, double* dt_prime)
{
    if (isnan(Lambda)) {                        /* Q26 */
        *dt_prime = 0.5 * dt;
        return 0;
    }
    /* "If the error in x exceeds a prescribed limit the step length is reduced via (2.11) ... If Lambda > Lambda0 the
     * result is rejected and recomputed with dt = dt'." */
    if (Lambda > Lambda0) {
        *dt_prime = eq_2_11(dt, Lambda, Lambda0);
        if (*dt_prime > 0.9 * dt) *dt_prime = 0.9 * dt;          /* Q22a */
        return 0;
    }
    /* the result is kept; the step length stays ... */
    *dt_prime = dt;
    /* ... unless: "Should Lambda fall below Lambda0/2, dt' is increased according to the same equation" */
    if (Lambda < Lambda0 / 2.0) {
        const double most = 5.0 * dt;                             /* Q22b */
        *dt_prime = Lambda > 0.0 ? eq_2_11(dt, Lambda, Lambda0) : most;
        if (*dt_prime > most) *dt_prime = most;
    }
    return 1;
}

typedef struct {
    const int* n; const double* lo; const double* hi; const double* B0; double gamma; int op;
} relax_rhs_t;

static int relax_rhs(const double* x, double* u, void* user)
{
    const relax_rhs_t* r = (const relax_rhs_t*)user;
    return mro_fields(r->n, r->lo, r->hi, x, r->B0, r->gamma, r->op, NULL, NULL, u, NULL);
}

/* how many trials in a row may fold the grid before the run is given up (reading Q26): 2^-40 = 9e-13, "a drop of the
 * time step by several orders of magnitude, at which point the simulation is stopped" */
#define MRO_MAX_FOLDED_TRIALS 40

/*
 * Integrate dx/dt = u(x) = gamma J x B (Eq. 1.5) from *t to t_end with the adaptive Cash-Karp scheme of section 2.4.
 * *dt: first trial step in, step handed on out.  trace (may be NULL, capacity trace_cap rows of 4 doubles) records every
 * trial: {t, dt tried, Lambda, kept}.  counts[0] = results kept, counts[1] = results rejected.
 *
 * A trial in which some stage meets det(dx/dX) <= 0 or a non-finite value has no result at all; the paper does not say
 * what its code does then (reading Q26): it counts as rejected (Lambda = NaN in the trace) and is recomputed with half the
 * step; MRO_MAX_FOLDED_TRIALS of them in a row end the run with return code 5, x being the last kept state (:333).
 * Returns 0, 1 (bad argument), 5 (numeric failure as just described) or 7 (max_trials exhausted).
 */
int mro_step_adaptive(const int n[3], const double lo[3], const double hi[3], double* x, const double* B0, double gamma,
                      int op, double t_end, double lambda0, double* t, double* dt, long long max_trials,
                      long long counts[2], double* trace, long long trace_cap)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    if (!(lambda0 > 0.0) || !(*dt > 0.0) || !t || !dt || !counts) return MRO_BADARG;
    const long long m = (long long)(3 * g.N);
    double* work = (double*)malloc((size_t)8 * (size_t)m * sizeof(double));
    if (!work) return MRO_BADARG;
    double* x_new = work + (size_t)7 * (size_t)m;
    relax_rhs_t r = { n, lo, hi, B0, gamma, op };
    counts[0] = counts[1] = 0;
    long long trials = 0;
    int folded_in_a_row = 0;
    rc = MRO_OK;
    while (*t < t_end && rc == MRO_OK) {
        if (trials >= max_trials) { rc = 7; break; }
        /* the step to try: dt, or what is left to t_end if that is shorter (the run ends exactly there) */
        const double left = t_end - *t;
        const int is_last = *dt >= left;
        const double tried = is_last ? left : *dt;
        double Lambda = NAN, dt_prime = 0.0;
        int kept = 0;
        const int trial_rc = mro_cash_karp_trial(m, x, tried, relax_rhs, &r, x_new, NULL, &Lambda, work);
        if (trial_rc == MRO_NUMERIC) {
            /* Q26: no result; recompute with half the step, give up after MRO_MAX_FOLDED_TRIALS in a row */
            Lambda = NAN;
            dt_prime = 0.5 * tried;
            if (++folded_in_a_row >= MRO_MAX_FOLDED_TRIALS) rc = MRO_NUMERIC;
        } else if (trial_rc != MRO_OK) {
            rc = trial_rc;
            break;
        } else {
            folded_in_a_row = 0;
            kept = mro_step_control(tried, Lambda, lambda0, &dt_prime);
        }
        if (trace && trials < trace_cap) {
            double* row = trace + 4 * trials;
            row[0] = *t; row[1] = tried; row[2] = Lambda; row[3] = (double)kept;
        }
        ++trials;
        counts[kept ? 0 : 1]++;
        if (kept) {
            memcpy(x, x_new, (size_t)m * sizeof(double));
            *t = is_last ? t_end : *t + tried;
            /* the shortened last step says nothing about the step length: hand on the caller's dt unless the control shrank it */
            if (!is_last || dt_prime < *dt) *dt = dt_prime;
        } else {
            *dt = dt_prime;                   /* "recomputed with dt = dt'" */
        }
    }
    free(work);
    return rc;
}

/* =========================================================================================================
 * Diagnostics of section 3.2 beyond E_M and xi: convexity (Eqs. 3.10-3.11), alpha* and eps* (Eqs. 3.5-3.7),
 * sigma_B and sigma_x (Eqs. 3.8-3.9).
 * ========================================================================================================= */

/* kappa per node (int, +1 / -1; reading Q23) and the number of nodes with kappa = -1.  kappa may be NULL. */
int mro_convexity(const int n[3], const double lo[3], const double hi[3], const double* x, int* kappa, long long* n_concave)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    const int nn[3] = { g.nx, g.ny, g.nz };
    long long bad = 0;
    for (int k = 0; k < g.nz; ++k)
        for (int j = 0; j < g.ny; ++j)
            for (int i = 0; i < g.nx; ++i) {
                const int idx[3] = { i, j, k };
                double xc[3]; load3(&g, x, i, j, k, xc);
                int kap = 1;
                for (int di = -1; di <= 1; di += 2)
                    for (int dj = -1; dj <= 1; dj += 2)
                        for (int dk = -1; dk <= 1; dk += 2) {
                            const int d[3] = { di, dj, dk };
                            int exists = 1;
                            for (int a = 0; a < 3; ++a)
                                if (!g.per[a] && (idx[a] + d[a] < 0 || idx[a] + d[a] >= nn[a])) exists = 0;
                            if (!exists) continue;
                            double v[3][3], nb[3];   /* v[0] = dx^lambda, v[1] = dx^mu, v[2] = dx^nu (Eq. 3.10) */
                            load3x(&g, x, i + di, j, k, nb); for (int c = 0; c < 3; ++c) v[0][c] = nb[c] - xc[c];
                            load3x(&g, x, i, j + dj, k, nb); for (int c = 0; c < 3; ++c) v[1][c] = nb[c] - xc[c];
                            load3x(&g, x, i, j, k + dk, nb); for (int c = 0; c < 3; ++c) v[2][c] = nb[c] - xc[c];
                            const double dd = det3(v);    /* det of the matrix with rows dx^lambda, dx^mu, dx^nu */
                            const int sgn = dd > 0.0 ? 1 : (dd < 0.0 ? -1 : 0);
                            if (sgn != di * dj * dk) kap = -1;           /* Eq. 3.11 */
                        }
                if (kappa) kappa[at(&g, i, j, k)] = kap;
                if (kap < 0) ++bad;
            }
    if (n_concave) *n_concave = bad;
    return MRO_OK;
}

/*
 * alpha* = J.B/B^2 (Eq. 3.5) at the inner nodes of the grid line (ic, jc, .) -- s_alpha of Eq. 3.6 when that line is the
 * z axis -- into alpha[nz] (0 at line-tied end nodes), and eps* = max over ordered pairs (k1, k2), k1 != k2, of
 * a_r (alpha*_k1 - alpha*_k2)/|X_k1 - X_k2| (Eq. 3.7; reference positions X).  alpha may be NULL.
 */
int mro_eps_star(const int n[3], const double lo[3], const double hi[3], const double* x, const double* B0, int op,
                 int ic, int jc, double a_r, double* alpha, double* eps)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    if (ic < 0 || ic >= g.nx || jc < 0 || jc >= g.ny || !inner_node(&g, ic, jc, g.nz / 2)) return MRO_BADARG;
    double* B = (double*)malloc(3 * g.N * sizeof(double));
    double* J = (double*)malloc(3 * g.N * sizeof(double));
    double* al = (double*)malloc((size_t)g.nz * sizeof(double));
    if (!B || !J || !al) return MRO_BADARG;
    rc = mro_fields(n, lo, hi, x, B0, 1.0, op, B, J, NULL, NULL);
    const int k_lo = g.per[2] ? 0 : 1, k_hi = g.per[2] ? g.nz - 1 : g.nz - 2;
    for (int k = 0; k < g.nz; ++k) {
        size_t p = at(&g, ic, jc, k);
        double b[3] = { B[p], B[g.N + p], B[2 * g.N + p] }, jv[3] = { J[p], J[g.N + p], J[2 * g.N + p] };
        al[k] = (k >= k_lo && k <= k_hi) ? (jv[0] * b[0] + jv[1] * b[1] + jv[2] * b[2]) / (b[0] * b[0] + b[1] * b[1] + b[2] * b[2]) : 0.0;
        if (alpha) alpha[k] = al[k];
    }
    double e = 0.0;
    for (int k1 = k_lo; k1 <= k_hi; ++k1)
        for (int k2 = k_lo; k2 <= k_hi; ++k2) {
            if (k1 == k2) continue;
            double s = a_r * (al[k1] - al[k2]) / fabs((double)(k1 - k2) * g.h[2]);
            if (s > e) e = s;
        }
    *eps = e;
    free(B); free(J); free(al);
    return rc;
}

/* sigma_B (Eq. 3.8) and sigma_x (Eq. 3.9): root of the mean over ALL N nodes of |B - B_ref|^2 resp. |x - x_ref|^2. */
int mro_sigma(const int n[3], const double lo[3], const double hi[3], const double* x, const double* B0,
              const double* x_ref, const double* B_ref, double* sigma_x, double* sigma_B)
{
    grid_t g; int rc = make_grid(n, lo, hi, &g); if (rc) return rc;
    double* B = (double*)malloc(3 * g.N * sizeof(double));
    if (!B) return MRO_BADARG;
    rc = mro_push_forward(n, lo, hi, x, B0, B, NULL);
    long double sx = 0.0L, sb = 0.0L;
    for (size_t p = 0; p < g.N; ++p)
        for (int c = 0; c < 3; ++c) {
            double dx = x[(size_t)c * g.N + p] - x_ref[(size_t)c * g.N + p];
            double db = B[(size_t)c * g.N + p] - B_ref[(size_t)c * g.N + p];
            sx += (long double)(dx * dx);
            sb += (long double)(db * db);
        }
    *sigma_x = sqrt((double)(sx / (long double)g.N));
    *sigma_B = sqrt((double)(sb / (long double)g.N));
    free(B);
    return rc;
}
