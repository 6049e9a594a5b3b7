// mr_next.cuh -- kernels of the SURVEY 8(f) rows: the stage combinations and the error maximum of the adaptive
// Cash-Karp integrator (section 2.4), convexity (Eqs. 3.10-3.11), alpha* / eps* (Eqs. 3.5-3.7) and
// sigma_B, sigma_x (Eqs. 3.8-3.9).  The right-hand side u = gamma J x B itself is the RHS instantiation of the step
// kernels (mr_sym.cuh, mr_direct.cuh, mr_generic.cuh).
#pragma once
#include "mr_generic.cuh"

namespace mr {

// Butcher tableau of the Cash-Karp pair (Cash & Karp 1990; the paper's [4]): a_sr, the fifth-order weights
// b_s and the differences b_s - b*_s to the embedded fourth-order weights.
struct CashKarp {
    double a[6][5];
    double b5[6];
    double db[6];
};
inline CashKarp cash_karp()
{
    CashKarp t = { { { 0, 0, 0, 0, 0 },
                     { 1.0 / 5.0, 0, 0, 0, 0 },
                     { 3.0 / 40.0, 9.0 / 40.0, 0, 0, 0 },
                     { 3.0 / 10.0, -9.0 / 10.0, 6.0 / 5.0, 0, 0 },
                     { -11.0 / 54.0, 5.0 / 2.0, -70.0 / 27.0, 35.0 / 27.0, 0 },
                     { 1631.0 / 55296.0, 175.0 / 512.0, 575.0 / 13824.0, 44275.0 / 110592.0, 253.0 / 4096.0 } },
                   { 37.0 / 378.0, 0.0, 250.0 / 621.0, 125.0 / 594.0, 0.0, 512.0 / 1771.0 },
                   { 0, 0, 0, 0, 0, 0 } };
    const double b4[6] = { 2825.0 / 27648.0, 0.0, 18575.0 / 48384.0, 13525.0 / 55296.0, 277.0 / 14336.0, 1.0 / 4.0 };
    for (int s = 0; s < 6; ++s) t.db[s] = t.b5[s] - b4[s];
    return t;
}

struct StageArgs {
    const void* k[6];     // stage velocities k_1 .. k_6 (padded layout, like xi)
    double c[6];          // coefficient of each (the kernels multiply by the step length dt, which they read from device memory:
                          // the launches of a trial step do not depend on dt and can be replayed as a CUDA graph)
    int n;                // how many of them enter
};

// xi_s = xi + sum_r (dt a_sr) k_r over the whole padded field (the padding stays zero); elementwise, vectorised by two
template <typename T>
__global__ void __launch_bounds__(256)
k_rk_stage(const T* __restrict__ xi, T* __restrict__ xs, StageArgs a, long long n2, const double* __restrict__ dt)
{
    using V = typename std::conditional<sizeof(T) == 8, double2, float2>::type;
    const double h = *dt;
#pragma unroll
    for (int r = 0; r < 6; ++r) a.c[r] = h * a.c[r];
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n2; q += (long long)gridDim.x * blockDim.x) {
        V v = reinterpret_cast<const V*>(xi)[q];
        double s0 = 0.0, s1 = 0.0;
#pragma unroll
        for (int r = 0; r < 6; ++r)
            if (r < a.n) {
                const V kv = reinterpret_cast<const V*>(a.k[r])[q];
                s0 += a.c[r] * (double)kv.x;
                s1 += a.c[r] * (double)kv.y;
            }
        v.x = (T)((double)v.x + s0);
        v.y = (T)((double)v.y + s1);
        reinterpret_cast<V*>(xs)[q] = v;
    }
}

// xi5 = xi + sum_s (dt b_s) k_s, and (into *partial, zeroed by the caller) the grid's maximum of |x5 - x4| = |sum_s dt (b_s - b*_s) k_s| ("the maximum error in
// x").  A maximum does not depend on the order: the result is deterministic.
template <typename T>
__global__ void __launch_bounds__(256)
k_rk_final(const T* __restrict__ xi, T* __restrict__ x5, StageArgs b5, StageArgs db, long long n2, double* __restrict__ partial,
           const double* __restrict__ dt)
{
    using V = typename std::conditional<sizeof(T) == 8, double2, float2>::type;
    const double h = *dt;
#pragma unroll
    for (int r = 0; r < 6; ++r) { b5.c[r] = h * b5.c[r]; db.c[r] = h * db.c[r]; }
    double lam = 0.0;
    bool nan = false;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n2; q += (long long)gridDim.x * blockDim.x) {
        V v = reinterpret_cast<const V*>(xi)[q];
        double s0 = 0.0, s1 = 0.0, e0 = 0.0, e1 = 0.0;
#pragma unroll
        for (int r = 0; r < 6; ++r) {
            const V kv = reinterpret_cast<const V*>(b5.k[r])[q];
            s0 += b5.c[r] * (double)kv.x;
            s1 += b5.c[r] * (double)kv.y;
            e0 += db.c[r] * (double)kv.x;
            e1 += db.c[r] * (double)kv.y;
        }
        v.x = (T)((double)v.x + s0);
        v.y = (T)((double)v.y + s1);
        reinterpret_cast<V*>(x5)[q] = v;
        nan = nan || e0 != e0 || e1 != e1;
        lam = fmax(lam, fmax(fabs(e0), fabs(e1)));
    }
    if (nan) lam = NAN;
    __shared__ double sh[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double w = __shfl_down_sync(0xffffffffu, lam, o);
        lam = (w > lam || w != w) ? w : lam;
    }
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = lam;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) lam = (sh[w] > lam || sh[w] != sh[w]) ? sh[w] : lam;
        // lam >= 0 or NaN: as 64-bit patterns the non-negative doubles order like unsigned integers and a (positive) NaN lies
        // above +inf, so one atomic maximum per block gives the grid's maximum, NaN winning, whatever the order of the blocks
        atomicMax(reinterpret_cast<unsigned long long*>(partial), (unsigned long long)__double_as_longlong(fabs(lam)));
    }
}

// Convexity (Eqs. 3.10-3.11): kappa(node) = +1 iff every trihedron of the node whose three neighbours
// exist has sgn det(dx^lambda, dx^mu, dx^nu) = di dj dk, else -1; the nodes with kappa = -1 are counted.
template <typename T>
__global__ void __launch_bounds__(256)
k_convexity(const T* __restrict__ xi, GridP<T> g, int* __restrict__ kappa, unsigned long long* __restrict__ count)
{
    int i, j, k;
    if (!node_of_thread(g.nx, g.ny, g.nz, i, j, k)) return;
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    const Nbr nb = neighbours(g, i, j, k);
    const int idx[3] = { i, j, k }, n[3] = { g.nx, g.ny, g.nz };
    // edge vectors to the six neighbours: x(+-a) - x = +-h_a e_a + xi(+-a) - xi  (doubles: the sign decides an integer)
    double e[3][2][3];
    bool have[3][2];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            have[a][s] = g.per[a] || (s == 0 ? idx[a] > 0 : idx[a] < n[a] - 1);
            const long long o = s == 0 ? nb.m[a] : nb.p[a];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                double v = have[a][s] ? (double)xi[c * g.comp + p + o] - (double)xi[c * g.comp + p] : 0.0;
                if (c == a) v += (s == 0 ? -0.5 : 0.5) * (double)g.twoh[a];
                e[a][s][c] = v;
            }
        }
    int kap = 1;
#pragma unroll
    for (int si = 0; si < 2; ++si)
#pragma unroll
        for (int sj = 0; sj < 2; ++sj)
#pragma unroll
            for (int sk = 0; sk < 2; ++sk) {
                if (!(have[0][si] && have[1][sj] && have[2][sk])) continue;
                const double* u = e[0][si];
                const double* v = e[1][sj];
                const double* w = e[2][sk];
                const double d = u[0] * (v[1] * w[2] - v[2] * w[1]) - u[1] * (v[0] * w[2] - v[2] * w[0]) + u[2] * (v[0] * w[1] - v[1] * w[0]);
                const int sgn = d > 0.0 ? 1 : (d < 0.0 ? -1 : 0);
                const int prod = (si ? 1 : -1) * (sj ? 1 : -1) * (sk ? 1 : -1);         // di dj dk (s = 0: -1, s = 1: +1)
                if (sgn != prod) kap = -1;                                               // Eq. 3.11
            }
    if (kappa) kappa[((long long)k * g.ny + j) * g.nx + i] = kap;
    if (kap < 0) atomicAdd(count, 1ULL);
}

// alpha* = J.B/B^2 (Eq. 3.5) on the inner nodes of the grid line (ic, jc, .), 0 at line-tied end nodes
template <typename T, int OP>
__global__ void k_alpha_line(const T* __restrict__ xi, const T* __restrict__ b, GridP<T> g, int ic, int jc, double* __restrict__ alpha,
                             int* __restrict__ flag)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.nz) return;
    double al = 0.0;
    if (inner_node(g, ic, jc, k)) {
        T J[3], B[3], D;
        bool bad = false;
        if (OP == 0) node_J_mimetic(xi, b, g, ic, jc, k, J, B, D, bad);
        else node_J_direct(xi, b, g, ic, jc, k, J, B, D, bad);
        if (bad) atomicOr(flag, FLAG_NUMERIC);
        al = ((double)J[0] * B[0] + (double)J[1] * B[1] + (double)J[2] * B[2]) / ((double)B[0] * B[0] + (double)B[1] * B[1] + (double)B[2] * B[2]);
    }
    alpha[k] = al;
}

// eps* = max over ordered pairs k1 != k2 of inner nodes of a_r (alpha*_k1 - alpha*_k2)/|Z_k1 - Z_k2| (Eq. 3.7); one block
__global__ void k_eps_star(const double* __restrict__ alpha, int k_lo, int k_hi, double a_r, double hz, double* __restrict__ out)
{
    double e = 0.0;
    for (int k1 = k_lo + (int)threadIdx.x; k1 <= k_hi; k1 += blockDim.x)
        for (int k2 = k_lo; k2 <= k_hi; ++k2)
            if (k1 != k2) e = fmax(e, a_r * (alpha[k1] - alpha[k2]) / fabs((double)(k1 - k2) * hz));
    __shared__ double sh[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e = fmax(e, __shfl_down_sync(0xffffffffu, e, o));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) e = fmax(e, sh[w]);
        *out = e;
    }
}

// sums over all nodes of |x - x_ref|^2 and |B - B_ref|^2 (Eqs. 3.8-3.9); refs are dense caller arrays; one partial per
// block, folded in index order (deterministic)
struct SumPair {
    double a, b;
};
template <typename T>
__global__ void __launch_bounds__(256)
k_sigma(const T* __restrict__ xi, const T* __restrict__ b, GridP<T> g, DomainP d, const T* __restrict__ x_ref, const T* __restrict__ B_ref,
        SumPair* __restrict__ partials)
{
    double sx = 0.0, sb = 0.0;
    const long long rows = (long long)g.ny * g.nz, N = (long long)g.nx * g.ny * g.nz;
    for (long long r = blockIdx.x; r < rows; r += gridDim.x) {
        const int j = (int)(r % g.ny), k = (int)(r / g.ny);
        for (int i = threadIdx.x; i < g.nx; i += blockDim.x) {
            const long long p = (long long)k * g.plane + (long long)j * g.pitch + i, q = ((long long)k * g.ny + j) * g.nx + i;
            const int idx[3] = { i, j, k };
            T B[3], D;
            node_B(xi, b, g, i, j, k, B, D);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double x = __dadd_rn(ref_coord(d.lo[c], d.h[c], idx[c]), (double)xi[c * g.comp + p]);
                const double dx = x - (double)x_ref[c * N + q], db = (double)B[c] - (double)B_ref[c * N + q];
                sx += dx * dx;
                sb += db * db;
            }
        }
    }
    __shared__ SumPair sh[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sx += __shfl_down_sync(0xffffffffu, sx, o);
        sb += __shfl_down_sync(0xffffffffu, sb, o);
    }
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = { sx, sb };
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < (int)(blockDim.x >> 5); ++w) { sx += sh[w].a; sb += sh[w].b; }
        partials[blockIdx.x] = { sx, sb };
    }
}
__global__ void k_sum_final(const SumPair* __restrict__ partials, int n, SumPair* __restrict__ out)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double a = 0.0, b = 0.0;
        for (int q = 0; q < n; ++q) { a += partials[q].a; b += partials[q].b; }
        *out = { a, b };
    }
}

}  // namespace mr
