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
};

enum : int { FLAG_NUMERIC = 1, FLAG_BOUNDARY = 2 };

// un-normalised first difference (2 h_a d/dX_a) of f along an axis with element stride s, at index idx of n
template <typename T>
__device__ __forceinline__ T delta_axis(const T* __restrict__ f, long long p, long long s, int idx, int n)
{
    if (idx == 0) return T(4) * f[p + s] - T(3) * f[p] - f[p + 2 * s];
    if (idx == n - 1) return T(3) * f[p] - T(4) * f[p - s] + f[p - 2 * s];
    return f[p + s] - f[p - s];
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
template <typename T>
__device__ __forceinline__ void node_dF(const T* __restrict__ xi, const GridP<T>& g, int i, int j, int k, T (&dF)[3][3])
{
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T* f = xi + c * g.comp;
        dF[c][0] = delta_axis(f, p, 1LL, i, g.nx);
        dF[c][1] = delta_axis(f, p, (long long)g.pitch, j, g.ny);
        dF[c][2] = delta_axis(f, p, g.plane, k, g.nz);
        dF[c][c] += g.twoh[c];
    }
}

// B and D = det dF at node (i,j,k) from global memory
template <typename T>
__device__ __forceinline__ void node_B(const T* __restrict__ xi, const T* __restrict__ b, const GridP<T>& g,
                                       int i, int j, int k, T (&B)[3], T& D)
{
    T dF[3][3];
    node_dF(xi, g, i, j, k, dF);
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    const T b0 = b[p], b1 = b[g.comp + p], b2 = b[2 * g.comp + p];
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
template <typename T>
__device__ __forceinline__ void node_J_mimetic(const T* __restrict__ xi, const T* __restrict__ b, const GridP<T>& g,
                                               int i, int j, int k, T (&J)[3], T (&B)[3], T& D, bool& bad)
{
    T dF[3][3];
    node_dF(xi, g, i, j, k, dF);
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    D = det3(dF);
    const T inv = T(1) / D;
    {
        const T b0 = b[p], b1 = b[g.comp + p], b2 = b[2 * g.comp + p];
#pragma unroll
        for (int c = 0; c < 3; ++c) B[c] = (dF[c][0] * b0 + dF[c][1] * b1 + dF[c][2] * b2) * inv;
    }
    T dB[3][3];
    const int di[3] = { 1, 0, 0 }, dj[3] = { 0, 1, 0 }, dk[3] = { 0, 0, 1 };
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        T Bp[3], Bm[3], Dp, Dm;
        node_B(xi, b, g, i + di[a], j + dj[a], k + dk[a], Bp, Dp);
        node_B(xi, b, g, i - di[a], j - dj[a], k - dk[a], Bm, Dm);
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
template <typename T>
__device__ __forceinline__ void node_J_direct(const T* __restrict__ xi, const T* __restrict__ b, const GridP<T>& g,
                                              int i, int j, int k, T (&J)[3], T (&B)[3], T& D, bool& bad)
{
    T dF[3][3];
    node_dF(xi, g, i, j, k, dF);
    const long long p = (long long)k * g.plane + (long long)j * g.pitch + i;
    const long long s[3] = { 1LL, (long long)g.pitch, g.plane };
    T W[3][3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T* f = xi + c * g.comp;
        const T f0 = f[p];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            W[c][a][a] = T(4) * (f[p + s[a]] - T(2) * f0 + f[p - s[a]]);
#pragma unroll
            for (int q = a + 1; q < 3; ++q) {
                const T m = f[p + s[a] + s[q]] - f[p + s[a] - s[q]] - f[p - s[a] + s[q]] + f[p - s[a] - s[q]];
                W[c][a][q] = m;
                W[c][q][a] = m;
            }
        }
    }
    T bb[3], gq[3][3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const T* f = b + q * g.comp;
        bb[q] = f[p];
#pragma unroll
        for (int a = 0; a < 3; ++a) gq[q][a] = f[p + s[a]] - f[p - s[a]];
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
