// mr_generic.cuh -- layout conversion, field materialisation, the generic (global-memory) step kernel and the
// diagnostics reduction.  One thread per node; every stencil value is read straight from global memory through
// L1/L2.  These kernels serve mr_set_*, mr_get_fields, mr_diagnostics, the direct operator and any grid the
// streaming TMA kernel (mr_stream.cuh) does not take; they are also its A/B reference in the tests.
#pragma once
#include "mr_common.cuh"

namespace mr {

struct DomainP {
    double lo[3];
    double h[3];
};

// X_a = lo_a + idx*h_a evaluated as a separately rounded product and sum (no FMA contraction), so that the
// reference grid is bit-identical to the host-side definition lo + idx*h.
__device__ __forceinline__ double ref_coord(double lo, double h, int idx) { return __dadd_rn(lo, __dmul_rn((double)idx, h)); }

__device__ __forceinline__ bool node_of_thread(int nx, int ny, int nz, int& i, int& j, int& k)
{
    i = blockIdx.x * blockDim.x + threadIdx.x;
    j = blockIdx.y * blockDim.y + threadIdx.y;
    k = blockIdx.z * blockDim.z + threadIdx.z;
    return i < nx && j < ny && k < nz;
}

// x (dense) -> xi = x - X (padded).  Boundary nodes must sit on X: |xi| <= 1e-6 h, else FLAG_BOUNDARY; they are
// stored as exact zeros so that line-tied faces are exact.
template <typename T>
__global__ void k_import_x(const T* __restrict__ x, T* __restrict__ xi, GridP<T> g, DomainP d, int* __restrict__ flag)
{
    int i, j, k;
    if (!node_of_thread(g.nx, g.ny, g.nz, i, j, k)) return;
    const long long N = (long long)g.nx * g.ny * g.nz;
    const long long q = ((long long)k * g.ny + j) * g.nx + i;
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    const bool bnd = !inner_node(g, i, j, k);
    const int idx[3] = { i, j, k };
    bool off = false;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double X = ref_coord(d.lo[c], d.h[c], idx[c]);
        double v = (double)x[c * N + q] - X;
        if (bnd) {
            // on the reference grid up to 1e-6 h, plus the rounding of X itself when x comes in as fp32
            const double tol = 1e-6 * d.h[c] + (sizeof(T) == 4 ? 2.4e-7 * fabs(X) : 0.0);
            if (!(fabs(v) <= tol)) off = true;
            v = 0.0;
        }
        xi[c * g.comp + p] = (T)v;
    }
    if (off) atomicOr(flag, FLAG_BOUNDARY);
}

// xi (dense) -> xi (padded): the displacement itself crosses the ABI (on an fp32 context x = X + xi would lose
// eps |X| per node, 300 times the rounding of xi).  Nodes on a line-tied face must have xi = 0, else FLAG_BOUNDARY.
template <typename T>
__global__ void k_import_xi(const T* __restrict__ src, T* __restrict__ xi, GridP<T> g, int* __restrict__ flag)
{
    int i, j, k;
    if (!node_of_thread(g.nx, g.ny, g.nz, i, j, k)) return;
    const long long N = (long long)g.nx * g.ny * g.nz;
    const long long q = ((long long)k * g.ny + j) * g.nx + i;
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    const bool bnd = !inner_node(g, i, j, k);
    bool off = false;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        T v = src[c * N + q];
        if (bnd) {
            if (!(fabs((double)v) <= 1e-6 * 0.5 * (double)g.twoh[c])) off = true;
            v = T(0);
        }
        xi[c * g.comp + p] = v;
    }
    if (off) atomicOr(flag, FLAG_BOUNDARY);
}

// padded field (xi, or a velocity) -> dense caller buffer
template <typename T>
__global__ void k_export_padded(const T* __restrict__ src, T* __restrict__ dst, GridP<T> g)
{
    int i, j, k;
    if (!node_of_thread(g.nx, g.ny, g.nz, i, j, k)) return;
    const long long N = (long long)g.nx * g.ny * g.nz;
    const long long q = ((long long)k * g.ny + j) * g.nx + i;
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
#pragma unroll
    for (int c = 0; c < 3; ++c) dst[c * N + q] = src[c * g.comp + p];
}

// Ghost layers of the periodic axes (Eqs. 2.12-2.14; reading Q12): in the displacement xi = x - X, and in b, the
// ghost node of index idx < 0 or idx >= n is the node idx mod n.  `f` points at the node (0, 0, 0) of a padded field whose
// periodic axes carry gx / gy / gz layers either side; every ghost node copies its three components from the node it wraps
// to.  The streaming kernels read their halos out of these layers; one thread per ghost node, x fastest.
template <typename T>
__global__ void __launch_bounds__(256)
k_wrap(T* __restrict__ f, GridP<T> g, int gx, int gy, int gz)
{
    const long long px = g.nx + 2 * gx, py = g.ny + 2 * gy;
    const long long nA = 2LL * gz * py * px;                 // the z slabs (all rows, all columns)
    const long long nB = (long long)g.nz * 2 * gy * px;      // the y slabs of the planes 0 .. nz-1
    const long long nC = (long long)g.nz * g.ny * 2 * gx;    // the x slabs of the rows 0 .. ny-1 of those planes
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < nA + nB + nC; q += (long long)gridDim.x * blockDim.x) {
        long long i, j, k, r = q;
        if (r < nA) {
            i = r % px - gx; r /= px;
            j = r % py - gy; r /= py;
            k = r < gz ? r - gz : g.nz + (r - gz);
        } else if ((r -= nA) < nB) {
            i = r % px - gx; r /= px;
            const long long jj = r % (2 * gy); r /= 2 * gy;
            j = jj < gy ? jj - gy : g.ny + (jj - gy);
            k = r;
        } else {
            r -= nB;
            const long long ii = r % (2 * gx); r /= 2 * gx;
            i = ii < gx ? ii - gx : g.nx + (ii - gx);
            j = r % g.ny;
            k = r / g.ny;
        }
        const long long si = (i % g.nx + g.nx) % g.nx, sj = (j % g.ny + g.ny) % g.ny, sk = (k % g.nz + g.nz) % g.nz;
        const long long dst = k * g.plane + j * g.pitch + i, src = sk * g.plane + sj * g.pitch + si;
#pragma unroll
        for (int c = 0; c < 3; ++c) f[c * g.comp + dst] = f[c * g.comp + src];
    }
}

// B0 (dense) -> b_a = scale_a * B0_a (padded), scale_a = 4 h_b h_c
template <typename T>
__global__ void k_import_B0(const T* __restrict__ B0, T* __restrict__ b, GridP<T> g, double s0, double s1, double s2)
{
    int i, j, k;
    if (!node_of_thread(g.nx, g.ny, g.nz, i, j, k)) return;
    const long long N = (long long)g.nx * g.ny * g.nz;
    const long long q = ((long long)k * g.ny + j) * g.nx + i;
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    b[p] = (T)((double)B0[q] * s0);
    b[g.comp + p] = (T)((double)B0[N + q] * s1);
    b[2 * g.comp + p] = (T)((double)B0[2 * N + q] * s2);
}

// Materialise x = X + xi, B (all nodes) and J (interior, 0 on the boundary) into dense caller buffers.  The fields are
// evaluated in fp64 whatever the storage type T of the state is and rounded to T at the end: on an fp32 context they
// are then as accurate as the fp32 STATE allows (J formed in fp32 arithmetic carries eps |B| / (2h |grad B|), about 1.2e-5
// of max |J| at h = 8/511, reading Q15); the step kernels themselves compute in T.
template <typename T, int OP>
__global__ void k_fields(const T* __restrict__ xi, const T* __restrict__ b, GridP<double> g, DomainP d,
                         T* __restrict__ x_out, T* __restrict__ B_out, T* __restrict__ J_out, int* __restrict__ flag)
{
    int i, j, k;
    if (!node_of_thread(g.nx, g.ny, g.nz, i, j, k)) return;
    const long long N = (long long)g.nx * g.ny * g.nz;
    const long long q = ((long long)k * g.ny + j) * g.nx + i;
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    if (x_out) {
        const int idx[3] = { i, j, k };
#pragma unroll
        for (int c = 0; c < 3; ++c) x_out[c * N + q] = (T)__dadd_rn(ref_coord(d.lo[c], d.h[c], idx[c]), (double)xi[c * g.comp + p]);
    }
    if (!B_out && !J_out) return;
    const bool bnd = !inner_node(g, i, j, k);
    double B[3], J[3] = { 0.0, 0.0, 0.0 }, D;
    bool bad = false;
    if (bnd || !J_out) {
        node_B(xi, b, g, i, j, k, B, D);
        bad = !(D > 0.0);
    } else if (OP == 0) {
        node_J_mimetic(xi, b, g, i, j, k, J, B, D, bad);
    } else {
        node_J_direct(xi, b, g, i, j, k, J, B, D, bad);
    }
    if (bad) atomicOr(flag, FLAG_NUMERIC);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (B_out) B_out[c * N + q] = (T)B[c];
        if (J_out) J_out[c * N + q] = (T)J[c];
    }
}

// Generic fused step: xi_out = xi_in + dtg * J x B on interior nodes, copy on boundary nodes (S1-S5).
// RHS = true: xi_out = dtg * J x B instead (the velocity u = gamma J x B with dtg = gamma; 0 on boundary nodes).
template <typename T, int OP, bool RHS = false>
__global__ void __launch_bounds__(256)
k_step_generic(const T* __restrict__ xi_in, T* __restrict__ xi_out, const T* __restrict__ b, GridP<T> g, T dtg,
               int* __restrict__ flag)
{
    int i, j, k;
    if (!node_of_thread(g.nx, g.ny, g.nz, i, j, k)) return;
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    const bool bnd = !inner_node(g, i, j, k);
    T o[3] = { xi_in[p], xi_in[g.comp + p], xi_in[2 * g.comp + p] };
    if (RHS) o[0] = o[1] = o[2] = T(0);
    if (!bnd) {
        T B[3], J[3], u[3], D;
        bool bad = false;
        if (OP == 0) node_J_mimetic(xi_in, b, g, i, j, k, J, B, D, bad);
        else node_J_direct(xi_in, b, g, i, j, k, J, B, D, bad);
        cross3(J, B, u);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            o[c] += dtg * u[c];
            bad = bad || !(fabs(o[c]) < T(1e30));
        }
        if (bad) atomicOr(flag, FLAG_NUMERIC);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) xi_out[c * g.comp + p] = o[c];
}

// ---------------------------------------------------------------------------------------------------------
// Diagnostics (S6): E = 1/16 sum zeta |B|^2 D  (= 1/2 h1h2h3 sum zeta |B|^2 Delta, Eq. 3.13), max |JxB|,
// max |JxB|/|B|^2 (Eq. 4.1) over interior nodes, min D.  fp64 accumulators whatever T is.  Stage 1: each block
// owns a fixed, contiguous set of rows (j,k) and reduces in a fixed order (warp shuffle tree, then warps in
// order); stage 2: one block folds the per-block partials in index order.  Hence deterministic.
// ---------------------------------------------------------------------------------------------------------
struct DiagPartial {
    double e, fmax, xi, dmin;
};

__device__ __forceinline__ void diag_combine(DiagPartial& a, const DiagPartial& o)
{
    a.e += o.e;
    a.fmax = fmax(a.fmax, o.fmax);
    a.xi = fmax(a.xi, o.xi);
    // NaN-propagating minimum: a NaN determinant must surface in min_det
    a.dmin = (o.dmin < a.dmin || o.dmin != o.dmin) ? o.dmin : a.dmin;
}

__device__ __forceinline__ DiagPartial diag_block_reduce(DiagPartial v)
{
    __shared__ DiagPartial sh[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        DiagPartial w;
        w.e = __shfl_down_sync(0xffffffffu, v.e, o);
        w.fmax = __shfl_down_sync(0xffffffffu, v.fmax, o);
        w.xi = __shfl_down_sync(0xffffffffu, v.xi, o);
        w.dmin = __shfl_down_sync(0xffffffffu, v.dmin, o);
        diag_combine(v, w);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < nw; ++w) diag_combine(v, sh[w]);
    }
    return v;  // valid in thread 0
}

template <typename T, int OP>
__global__ void __launch_bounds__(256)
k_diag(const T* __restrict__ xi, const T* __restrict__ b, GridP<T> g, DiagPartial* __restrict__ partials,
       int* __restrict__ flag)
{
    DiagPartial acc = { 0.0, 0.0, 0.0, INFINITY };
    const long long rows = (long long)g.ny * g.nz;
    bool bad = false;
    for (long long r = blockIdx.x; r < rows; r += gridDim.x) {
        const int j = (int)(r % g.ny), k = (int)(r / g.ny);
        for (int i = threadIdx.x; i < g.nx; i += blockDim.x) {
            const bool bnd = !inner_node(g, i, j, k);
            T B[3], J[3], D;
            if (bnd) {
                node_B(xi, b, g, i, j, k, B, D);
                bad = bad || !(D > T(0));
            } else {
                if (OP == 0) node_J_mimetic(xi, b, g, i, j, k, J, B, D, bad);
                else node_J_direct(xi, b, g, i, j, k, J, B, D, bad);
            }
            const double b2 = (double)B[0] * B[0] + (double)B[1] * B[1] + (double)B[2] * B[2];
            double zeta = 1.0;
            if (!g.per[0] && (i == 0 || i == g.nx - 1)) zeta *= 0.5;
            if (!g.per[1] && (j == 0 || j == g.ny - 1)) zeta *= 0.5;
            if (!g.per[2] && (k == 0 || k == g.nz - 1)) zeta *= 0.5;
            DiagPartial v = { zeta * b2 * (double)D, 0.0, 0.0, (double)D };
            if (!bnd) {
                T f[3];
                cross3(J, B, f);
                const double fm = sqrt((double)f[0] * f[0] + (double)f[1] * f[1] + (double)f[2] * f[2]);
                v.fmax = fm;
                v.xi = fm / b2;
            }
            diag_combine(acc, v);
        }
    }
    if (bad) atomicOr(flag, FLAG_NUMERIC);
    acc = diag_block_reduce(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc;
}

// S6 contributions of the nodes on line-tied faces only (zeta |B|^2 D and min D; they carry no J): the complement of the
// streaming pass of the direct operator, which reduces the inner nodes.  Same row ownership and order as k_diag.
template <typename T>
__global__ void __launch_bounds__(128)
k_diag_faces(const T* __restrict__ xi, const T* __restrict__ b, GridP<T> g, DiagPartial* __restrict__ partials, int* __restrict__ flag)
{
    DiagPartial acc = { 0.0, 0.0, 0.0, INFINITY };
    const long long rows = (long long)g.ny * g.nz;
    bool bad = false;
    for (long long r = blockIdx.x; r < rows; r += gridDim.x) {
        const int j = (int)(r % g.ny), k = (int)(r / g.ny);
        const bool face_row = (!g.per[1] && (j == 0 || j == g.ny - 1)) || (!g.per[2] && (k == 0 || k == g.nz - 1));
        if (!face_row && g.per[0]) continue;
        const int cnt = face_row ? g.nx : 2;                 // the whole row, or its two end nodes
        for (int q = threadIdx.x; q < cnt; q += blockDim.x) {
            const int i = face_row ? q : (q == 0 ? 0 : g.nx - 1);
            if (inner_node(g, i, j, k)) continue;
            T B[3], D;
            node_B(xi, b, g, i, j, k, B, D);
            bad = bad || !(D > T(0));
            const double b2 = (double)B[0] * B[0] + (double)B[1] * B[1] + (double)B[2] * B[2];
            double zeta = 1.0;
            if (!g.per[0] && (i == 0 || i == g.nx - 1)) zeta *= 0.5;
            if (!g.per[1] && (j == 0 || j == g.ny - 1)) zeta *= 0.5;
            if (!g.per[2] && (k == 0 || k == g.nz - 1)) zeta *= 0.5;
            DiagPartial v = { zeta * b2 * (double)D, 0.0, 0.0, (double)D };
            diag_combine(acc, v);
        }
    }
    if (bad) atomicOr(flag, FLAG_NUMERIC);
    acc = diag_block_reduce(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = acc;
}

__global__ void k_diag_final(const DiagPartial* __restrict__ partials, int n, DiagPartial* __restrict__ out)
{
    DiagPartial acc = { 0.0, 0.0, 0.0, INFINITY };
    for (int q = threadIdx.x; q < n; q += blockDim.x) diag_combine(acc, partials[q]);
    acc = diag_block_reduce(acc);
    if (threadIdx.x == 0) *out = acc;
}

}  // namespace mr
