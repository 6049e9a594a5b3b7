// mr_common.cuh -- device-side grid description and the per-node arithmetic shared by all kernels of libmr.so.
//
// Internal state layout:
//   xi[c][k][j][i]  displacement xi = x - X of the node from its reference position, padded rows (pitch),
//   b [c][k][j][i]  B(X,0) pre-scaled per component: b_a = 4 h_b h_c B0_a  ((a,b,c) cyclic),
// so that every stencil below works on UN-NORMALISED differences (no division by h anywhere):
//   dF_ca  = 2 h_a dx_c/dX_a = delta_a xi_c + 2 h_a [c == a]                       (Eq. 2.1)
//   D      = det dF = 8 h1 h2 h3 Delta
//   B_c    = dF_ca b_a / D                                                          (Eq. 2.1)
//   J      = dF chat / D,  chat_p = eps_pqr delta_q B . delta_r x                   (Eqs. 2.3-2.7 in closed form)
// delta_a is the central difference f(+1) - f(-1) inside and the second-order one-sided difference
// -3 f0 + 4 f1 - f2 (resp. 3 f0 - 4 f-1 + f-2) on a face, both equal to 2 h_a d/dX_a up to O(h^2).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace mr {

template <typename T>
struct GridP {
    int nx, ny, nz;
    int pitch;            // padded row length in elements (multiple of 16)
    long long plane;      // pitch * ny
    long long comp;       // plane * nz (stride between components)
    T twoh[3];            // 2 h_a
    int per[3];           // 1 = periodic axis (Eqs. 2.12-2.14): in the displacement xi = x - X the ghost nodes of the paper
                          // are a plain wrap of the index (X itself carries the shift by the period n_a h_a), 0 = line-tied
};

// is (i,j,k) an inner point along every axis (not on a line-tied face)?  Periodic axes have no faces.
template <typename T>
__device__ __forceinline__ bool inner_node(const GridP<T>& g, int i, int j, int k)
{
    return (g.per[0] || (i > 0 && i < g.nx - 1)) && (g.per[1] || (j > 0 && j < g.ny - 1)) && (g.per[2] || (k > 0 && k < g.nz - 1));
}

// element offsets of the +1 / -1 neighbours along the three axes (index wrapped on a periodic axis)
struct Nbr {
    long long p[3], m[3];
};
template <typename T>
__device__ __forceinline__ Nbr neighbours(const GridP<T>& g, int i, int j, int k)
{
    Nbr q;
    const long long s[3] = { 1LL, (long long)g.pitch, g.plane };
    const int idx[3] = { i, j, k }, n[3] = { g.nx, g.ny, g.nz };
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        q.p[a] = (g.per[a] && idx[a] == n[a] - 1) ? -(long long)(n[a] - 1) * s[a] : s[a];
        q.m[a] = (g.per[a] && idx[a] == 0) ? (long long)(n[a] - 1) * s[a] : -s[a];
    }
    return q;
}

enum : int { FLAG_NUMERIC = 1, FLAG_BOUNDARY = 2 };

// un-normalised first difference (2 h_a d/dX_a) of f along an axis with element stride s, at index idx of n
// (S = storage type of the field, T = arithmetic type: mr_get_fields evaluates an fp32 state in fp64)
template <typename T, typename S>
__device__ __forceinline__ T delta_axis(const S* __restrict__ f, long long p, long long s, int idx, int n)
{
    if (idx == 0) return T(4) * (T)f[p + s] - T(3) * (T)f[p] - (T)f[p + 2 * s];
    if (idx == n - 1) return T(3) * (T)f[p] - T(4) * (T)f[p - s] + (T)f[p - 2 * s];
    return (T)f[p + s] - (T)f[p - s];
}

// ... with the neighbour offsets sp / sm of this node (periodic axis: central difference through the wrap)
template <typename T, typename S>
__device__ __forceinline__ T delta_axis(const S* __restrict__ f, long long p, long long sp, long long sm, int idx, int n, bool per)
{
    if (!per && idx == 0) return T(4) * (T)f[p + sp] - T(3) * (T)f[p] - (T)f[p + 2 * sp];
    if (!per && idx == n - 1) return T(3) * (T)f[p] - T(4) * (T)f[p + sm] + (T)f[p + 2 * sm];
    return (T)f[p + sp] - (T)f[p + sm];
}

template <typename T>
__device__ __forceinline__ T det3(const T (&m)[3][3])
{
    T c0 = m[1][1] * m[2][2] - m[1][2] * m[2][1];
    T c1 = m[1][2] * m[2][0] - m[1][0] * m[2][2];
    T c2 = m[1][0] * m[2][1] - m[1][1] * m[2][0];
    return m[0][0] * c0 + m[0][1] * c1 + m[0][2] * c2;
}

// dF[c][a] at node (i,j,k) from global memory (any node, faces included)
template <typename T, typename S>
__device__ __forceinline__ void node_dF(const S* __restrict__ xi, const GridP<T>& g, int i, int j, int k, T (&dF)[3][3])
{
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    const Nbr q = neighbours(g, i, j, k);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const S* f = xi + c * g.comp;
        dF[c][0] = delta_axis<T>(f, p, q.p[0], q.m[0], i, g.nx, g.per[0] != 0);
        dF[c][1] = delta_axis<T>(f, p, q.p[1], q.m[1], j, g.ny, g.per[1] != 0);
        dF[c][2] = delta_axis<T>(f, p, q.p[2], q.m[2], k, g.nz, g.per[2] != 0);
        dF[c][c] += g.twoh[c];
    }
}

// B and D = det dF at node (i,j,k) from global memory
template <typename T, typename S>
__device__ __forceinline__ void node_B(const S* __restrict__ xi, const S* __restrict__ b, const GridP<T>& g,
                                       int i, int j, int k, T (&B)[3], T& D)
{
    T dF[3][3];
    node_dF(xi, g, i, j, k, dF);
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    const T b0 = (T)b[p], b1 = (T)b[g.comp + p], b2 = (T)b[2 * g.comp + p];
    D = det3(dF);
    const T inv = T(1) / D;
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = (dF[c][0] * b0 + dF[c][1] * b1 + dF[c][2] * b2) * inv;
}

// closed form of the nearest-neighbour mimetic curl (identity I1): given the un-normalised central
// differences dB[a][c] = B_c(+a) - B_c(-a) and the centre's dF, D:  J = dF chat / D.
template <typename T>
__device__ __forceinline__ void mimetic_J(const T (&dF)[3][3], const T (&dB)[3][3], T invD, T (&J)[3])
{
    // chat_p = sum_c ( dB[q][c] dF[c][r] - dB[r][c] dF[c][q] ), (p,q,r) cyclic
    T ch[3];
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const int q = (p + 1) % 3, r = (p + 2) % 3;
        ch[p] = dB[q][0] * dF[0][r] + dB[q][1] * dF[1][r] + dB[q][2] * dF[2][r]
              - dB[r][0] * dF[0][q] - dB[r][1] * dF[1][q] - dB[r][2] * dF[2][q];
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) J[c] = (dF[c][0] * ch[0] + dF[c][1] * ch[1] + dF[c][2] * ch[2]) * invD;
}

// Mimetic J at an INTERIOR node, everything from global memory (generic path: B recomputed at the 6 neighbours).
template <typename T, typename S>
__device__ __forceinline__ void node_J_mimetic(const S* __restrict__ xi, const S* __restrict__ b, const GridP<T>& g,
                                               int i, int j, int k, T (&J)[3], T (&B)[3], T& D, bool& bad)
{
    T dF[3][3];
    node_dF(xi, g, i, j, k, dF);
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    D = det3(dF);
    const T inv = T(1) / D;
    {
        const T b0 = (T)b[p], b1 = (T)b[g.comp + p], b2 = (T)b[2 * g.comp + p];
#pragma unroll
        for (int c = 0; c < 3; ++c) B[c] = (dF[c][0] * b0 + dF[c][1] * b1 + dF[c][2] * b2) * inv;
    }
    T dB[3][3];
    const int n[3] = { g.nx, g.ny, g.nz };
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        T Bp[3], Bm[3], Dp, Dm;
        int ip[3] = { i, j, k }, im[3] = { i, j, k };
        ip[a] = ip[a] + 1 == n[a] ? 0 : ip[a] + 1;             // only an inner node comes here: a wrap means a periodic axis
        im[a] = im[a] == 0 ? n[a] - 1 : im[a] - 1;
        node_B(xi, b, g, ip[0], ip[1], ip[2], Bp, Dp);
        node_B(xi, b, g, im[0], im[1], im[2], Bm, Dm);
        bad = bad || !(Dp > T(0)) || !(Dm > T(0));
#pragma unroll
        for (int c = 0; c < 3; ++c) dB[a][c] = Bp[c] - Bm[c];
    }
    bad = bad || !(D > T(0));
    mimetic_J(dF, dB, inv, J);
}

// Direct-derivative ("classical") J at an INTERIOR node: the analytic derivative of B = dF b / D (Eq. 2.1) with
// un-normalised second differences W[c][q][a] = 4 h_q h_a d2x_c/dX_q dX_a and g[q][a] = delta_a b_q:
//   Nt[c][a] = W[c][q][a] b_q + dF[c][q] g[q][a],  t[a] = adj[q][c] W[c][q][a]  (= delta_a D, Jacobi),
//   Q[c][a]  = Nt[c][a] - B_c t[a],   dB_c/dx_m = Q[c][a] adj[a][m] / D^2,   J_l = eps_lmc dB_c/dx_m.
template <typename T, typename S>
__device__ __forceinline__ void node_J_direct(const S* __restrict__ xi, const S* __restrict__ b, const GridP<T>& g,
                                              int i, int j, int k, T (&J)[3], T (&B)[3], T& D, bool& bad)
{
    T dF[3][3];
    node_dF(xi, g, i, j, k, dF);
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    const Nbr nb = neighbours(g, i, j, k);
    T W[3][3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const S* f = xi + c * g.comp;
        const T f0 = (T)f[p];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            W[c][a][a] = T(4) * ((T)f[p + nb.p[a]] - T(2) * f0 + (T)f[p + nb.m[a]]);
#pragma unroll
            for (int q = a + 1; q < 3; ++q) {
                const T m = (T)f[p + nb.p[a] + nb.p[q]] - (T)f[p + nb.p[a] + nb.m[q]] - (T)f[p + nb.m[a] + nb.p[q]] + (T)f[p + nb.m[a] + nb.m[q]];
                W[c][a][q] = m;
                W[c][q][a] = m;
            }
        }
    }
    T bb[3], gq[3][3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const S* f = b + q * g.comp;
        bb[q] = (T)f[p];
#pragma unroll
        for (int a = 0; a < 3; ++a) gq[q][a] = (T)f[p + nb.p[a]] - (T)f[p + nb.m[a]];
    }
    // adjugate: adj[a][m] = D * (dF^-1)[a][m]
    T adj[3][3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int a1 = (a + 1) % 3, a2 = (a + 2) % 3;
#pragma unroll
        for (int m = 0; m < 3; ++m) {
            const int m1 = (m + 1) % 3, m2 = (m + 2) % 3;
            adj[a][m] = dF[m1][a1] * dF[m2][a2] - dF[m1][a2] * dF[m2][a1];
        }
    }
    D = dF[0][0] * adj[0][0] + dF[0][1] * adj[1][0] + dF[0][2] * adj[2][0];
    bad = bad || !(D > T(0));
    const T inv = T(1) / D;
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = (dF[c][0] * bb[0] + dF[c][1] * bb[1] + dF[c][2] * bb[2]) * inv;
    T t[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        T acc = T(0);
#pragma unroll
        for (int q = 0; q < 3; ++q)
#pragma unroll
            for (int c = 0; c < 3; ++c) acc += adj[q][c] * W[c][q][a];
        t[a] = acc;
    }
    T Q[3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            T acc = -B[c] * t[a];
#pragma unroll
            for (int q = 0; q < 3; ++q) acc += W[c][q][a] * bb[q] + dF[c][q] * gq[q][a];
            Q[c][a] = acc;
        }
    // G[c][m] = sum_a Q[c][a] adj[a][m]  (only the off-diagonal entries are needed)
    auto G = [&](int c, int m) { return Q[c][0] * adj[0][m] + Q[c][1] * adj[1][m] + Q[c][2] * adj[2][m]; };
    const T inv2 = inv * inv;
    J[0] = (G(2, 1) - G(1, 2)) * inv2;
    J[1] = (G(0, 2) - G(2, 0)) * inv2;
    J[2] = (G(1, 0) - G(0, 1)) * inv2;
}

template <typename T>
__device__ __forceinline__ void cross3(const T (&a)[3], const T (&b)[3], T (&c)[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

}  // namespace mr
