// mr_lean.cuh -- the lean-state streaming step kernel for the mimetic operator (S1-S5 in one pass).
//
// Same data flow as mr_pair.cuh (a CTA marches along k over an xy tile, every tile thread owns the two nodes (i, j)
// and (i, j+1), B is shared through a double-buffered shared plane, B/J/u never touch HBM), re-cut so that TWO CTAs
// fit on an SM (ncu r1c: the 255-register pair kernel ran 2 warps per scheduler and was latency-bound):
//   * the state a node carries from one plane to the next is 13 values instead of ~40.  With n_q the area vectors of
//     the three index surfaces through the node (Eqs. 2.5/2.6) the closed form of Eqs. 2.3-2.7 reads
//         D J = n_0 x delta_i B + n_1 x delta_j B + n_2 x (B(k+1) - B(k-1)),
//     and the in-plane part is folded as soon as the plane's B is in shared memory:
//         P(k) = n_0 x delta_i B + n_1 x delta_j B - n_2 x B(k-1)          (3 values)
//     so that only P, n_2, s = dt gamma / D, the own B and the own xi stay in registers (13 values per node);
//   * b (the pre-scaled B(X,0)) is read straight from global memory one plane ahead (coalesced, read-only path),
//     not through shared memory: the shared-memory footprint is 4 xi planes + 2 B planes = 100 KB;
//   * the own xi(k) is carried in registers, so the slot of plane k is free one iteration earlier and the TMA ring of
//     4 slots runs two planes ahead of the plane being differenced.
// Iteration t of the main loop (one bar.sync):
//   A  stage A of plane t+1 at the pair (and at the ring node of the threads that carry one): dF, n_q, D, 1/D,
//      B(t+1) = dF b / D (Eq. 2.1) -> shared B plane (t+1)&1;
//   F  finish plane t: D J = P(t) + n_2(t) x B(t+1);  u = gamma J x B(t) (Eq. 1.5);  xi+ = xi + dt u -> HBM;
//   -- bar.sync; the slot of plane t+1 is refilled with plane t+1+R --
//   I  in-plane part of plane t+1: P(t+1) from the shared B plane and the own pair.
#pragma once
#include <type_traits>

#include "mr_pair.cuh"

namespace mr {

template <typename T, int TY, int R>
struct LeanLayout {
    static_assert(TY % 2 == 0 && TY >= 8 && TY <= 32 && R >= 4, "tile / ring sizes");
    static constexpr int TX = 32;
    static constexpr int HXL = 16 / (int)sizeof(T), HXR = 2 * HXL;
    static constexpr int BW = TX + HXL + HXR;
    static constexpr int XH = TY + 4;
    static constexpr int CSX = BW * XH;
    static constexpr int round128(int bytes) { return (bytes + 127) / 128 * 128; }
    static constexpr int SLOTX = round128(3 * CSX * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr uint32_t XBOX_BYTES = 3u * CSX * sizeof(T);
    static constexpr int BBW = TX + 2, BBH = TY + 2;
    static constexpr int BCS = BBW * BBH;
    static constexpr int BSLOT = round128(3 * BCS * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr int NWARPS = TY / 2, NTHREADS = NWARPS * 32;
    static constexpr size_t OFF_X = 0;
    static constexpr size_t OFF_BB = OFF_X + (size_t)R * SLOTX * sizeof(T);
    static constexpr size_t OFF_BAR = OFF_BB + (size_t)2 * BSLOT * sizeof(T);
    static constexpr size_t BYTES = OFF_BAR + (size_t)R * 8 + 128;   // +128: base alignment slack
};

// Stage A at one node from its un-normalised differences dF (without the 2h diagonal): area vectors n_q, D = det dF,
// inv = 1/D and B = dF b / D (Eq. 2.1).
template <typename T>
__device__ __forceinline__ void lean_push(T (&dF)[3][3], const T (&b)[3], const T (&twoh)[3], T (&n)[3][3], T (&B)[3], T& inv,
                                          bool& ok, bool in_dom)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) dF[c][c] += twoh[c];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const int q1 = (q + 1) % 3, q2 = (q + 2) % 3;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
            n[q][c] = dF[c1][q1] * dF[c2][q2] - dF[c2][q1] * dF[c1][q2];
        }
    }
    const T D = dF[0][0] * n[0][0] + dF[1][0] * n[0][1] + dF[2][0] * n[0][2];
    ok = ok && (positive_finite(D) || !in_dom);
    inv = fast_rcp(D);
    const T b0 = b[0] * inv, b1 = b[1] * inv, b2 = b[2] * inv;
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = dF[c][0] * b0 + dF[c][1] * b1 + dF[c][2] * b2;
}

#ifndef MR_LEAN_UNROLL
#define MR_LEAN_UNROLL 2
#endif
constexpr int kLeanUnroll = MR_LEAN_UNROLL;

template <typename T, int TY, int R>
#ifndef MR_LEAN_MINB
#define MR_LEAN_MINB 2
#endif
__global__ void __launch_bounds__(TY * 16, MR_LEAN_MINB)
k_step_lean(const __grid_constant__ CUtensorMap map_in, const T* __restrict__ bsrc, T* __restrict__ out, const StreamArgs<T> a)
{
    using L = LeanLayout<T, TY, R>;
    constexpr int TX = L::TX, NT = L::NWARPS, BW = L::BW, CSX = L::CSX, BBW = L::BBW, BCS = L::BCS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((128u - (ptx::smem_u32(smem_raw) & 127u)) & 127u);
    const T* sx = reinterpret_cast<const T*>(smem + L::OFF_X);
    T* sB = reinterpret_cast<T*>(smem + L::OFF_BB);
    const uint32_t sx_u32 = ptx::smem_u32(sx);
    const uint32_t bar_x = ptx::smem_u32(smem + L::OFF_BAR);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x % a.ntiles, chunk = blockIdx.x / a.ntiles;
    const int i0 = (tile % a.tiles_x) * TX, j0 = (tile / a.tiles_x) * TY;
    const int nz = a.nz;
    const int k0 = chunk * a.chunk_len, k1 = min(k0 + a.chunk_len, nz);
    const int kend = min(k1, nz - 1);                                   // the loop forms B of the planes k0 .. kend
    const int pfirst = max(k0 - 2, 0), plast = min(k1 + 1, nz - 1);     // xi planes this item touches
    const T twoh[3] = { a.twoh[0], a.twoh[1], a.twoh[2] };

    // ---- TMA producer: lane 0 of the last warp (it carries no ring node) ----
    const bool producer = tid == (NT - 1) * 32;
    int next_load = pfirst;                                             // next xi plane to request (producer only)
    auto refill = [&](int upto) {                                       // request every plane <= upto not yet requested
        for (const int last = min(upto, plast); next_load <= last; ++next_load) {
            const uint32_t s = (uint32_t)((next_load - pfirst) % R);
            ptx::mbar_expect_tx(bar_x + 8u * s, L::XBOX_BYTES);
            ptx::tma_load_4d(sx_u32 + s * (uint32_t)(L::SLOTX * sizeof(T)), &map_in, i0 - L::HXL, j0 - 2, next_load, 0, bar_x + 8u * s);
        }
    };
    if (producer) {
        for (int s = 0; s < R; ++s) ptx::mbar_init(bar_x + 8u * s, 1);
        ptx::fence_mbar_init();
    }
    __syncthreads();
    if (producer) refill(pfirst + R - 1);

    auto wait_x = [&](int p) { const int q = p - pfirst; ptx::mbar_wait(bar_x + 8u * (uint32_t)(q % R), (uint32_t)((q / R) & 1)); };
    auto xplane = [&](int p) -> const T* { return sx + ((p - pfirst) % R) * L::SLOTX; };

    // nodes of this thread in tile coordinates: 0, 1 = the pair (lane, 2 warp), (lane, 2 warp + 1); 2 = a node of the
    // halo-1 ring for the threads of the first warps (only its push-forward B is formed).  Column ring: 8 rows of the left
    // and 8 rows of the right column per half-warp, so that at the row strides BW / BBW the 16 lanes of a
    // shared-memory wavefront fall into distinct banks.
    int ti2, tj2;
    constexpr int NRINGW = 2 + (TY + 15) / 16;      // ring warps: two rows, then 16 rows of both columns per warp
    static_assert(NRINGW < NT, "the last warp (TMA producer) carries no ring node");
    bool ring = warp < NRINGW;
    if (warp == 0) { ti2 = lane; tj2 = -1; }
    else if (warp == 1) { ti2 = lane; tj2 = TY; }
    else {
        ti2 = (lane >> 3) & 1 ? TX : -1;
        tj2 = (lane & 7) + 8 * (lane >> 4) + 16 * (warp - 2);
        if (tj2 >= TY) { ring = false; tj2 = 0; }
    }
    const int ti[3] = { lane, lane, ti2 }, tj[3] = { 2 * warp, 2 * warp + 1, tj2 };
    int ox[3], oB[3], gb[3];
    unsigned edge[3];
    bool dom[3];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        const int gi = i0 + ti[n], gj = j0 + tj[n];
        ox[n] = (tj[n] + 2) * BW + (ti[n] + L::HXL);
        oB[n] = (tj[n] + 1) * BBW + (ti[n] + 1);
        dom[n] = gi >= 0 && gi < a.nx && gj >= 0 && gj < a.ny && (n < 2 || ring);
        gb[n] = dom[n] ? gj * a.pitch + gi : 0;
        edge[n] = !dom[n] ? 0u
            : (gi == 0 ? 1u : 0u) | (gi == a.nx - 1 ? 2u : 0u) | (gj == 0 ? 4u : 0u) | (gj == a.ny - 1 ? 8u : 0u);
    }
    auto load_b = [&](int p, int n, T(&b)[3]) {     // pre-scaled B(X,0) of node n on plane p, straight from HBM / L2
        const T* g = bsrc + (long long)p * a.plane + gb[n];
#pragma unroll
        for (int c = 0; c < 3; ++c) b[c] = dom[n] ? __ldg(g + c * a.comp) : T(0);
    };
    auto store_B = [&](int p, int n, const T(&B)[3]) {
        T* d = sB + (p & 1) * L::BSLOT + oB[n];
        d[0] = B[0];
        d[BCS] = B[1];
        d[2 * BCS] = B[2];
    };

    const int gi = i0 + lane, gja = j0 + tj[0];
    const bool in_x = gi > 0 && gi < a.nx - 1;
    const bool in_xy[2] = { in_x && gja > 0 && gja < a.ny - 1, in_x && gja + 1 < a.ny - 1 };
    const bool st[2] = { gi < a.nx && gja < a.ny, gi < a.nx && gja + 1 < a.ny };


    // every plane requested so far is needed by the prologue or the first iteration
    for (int p = pfirst; p <= min(pfirst + R - 1, plast); ++p) wait_x(p);

    bool ok = true;
    // State carried over the barrier, per node of the pair (plane t = the plane the next iteration finishes):
    //   nA   area vectors n_0, n_1 of plane t          n2   area vector n_2 of plane t
    //   W    n_2(t) x B(t-1)                           s    dt gamma / D of plane t (0 where the node does not move)
    //   B0   own B(t)                                  xc   own xi(t)
    //   bq   own b(t+1), prefetched                    xr, bqr   own xi(t), b(t+1) of the ring node
    T nA[2][2][3], n2[2][3], W[2][3], s[2], B0[2][3], xc[2][3], bq[2][3], xr[3], bqr[3];
#pragma unroll
    for (int n = 0; n < 2; ++n) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            nA[n][0][c] = T(0); nA[n][1][c] = T(0); n2[n][c] = T(0); W[n][c] = T(0); B0[n][c] = T(0); xc[n][c] = T(0);
        }
        s[n] = T(0);
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) { xr[c] = T(0); bqr[c] = T(0); }
    if (k0 > 0) {
        // own B(k0-1) and own xi(k0-1) of the pair, every operand from shared memory / HBM
        const int p = k0 - 1;
        const T* pc = xplane(p);
        const T* pa = xplane(p + 1);
#pragma unroll
        for (int n = 0; n < 2; ++n) {
            T dF[3][3], nv[3][3], b[3], inv;
            const T* f = pc + ox[n];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                xc[n][c] = f[c * CSX];
                dF[c][0] = f[c * CSX + 1] - f[c * CSX - 1];
                dF[c][1] = f[c * CSX + BW] - f[c * CSX - BW];
            }
            if (p == 0) {
                const T* pb = xplane(2);
#pragma unroll
                for (int c = 0; c < 3; ++c) dF[c][2] = T(4) * pa[ox[n] + c * CSX] - T(3) * xc[n][c] - pb[ox[n] + c * CSX];
            } else {
                const T* pb = xplane(p - 1);
#pragma unroll
                for (int c = 0; c < 3; ++c) dF[c][2] = pa[ox[n] + c * CSX] - pb[ox[n] + c * CSX];
            }
            if (edge[n]) face_fix<T, BW, CSX>(f, edge[n], dF);
            load_b(p, n, b);
            lean_push(dF, b, twoh, nv, B0[n], inv, ok, dom[n]);
        }
        if (ring) {
            const T* f = pc + ox[2];
#pragma unroll
            for (int c = 0; c < 3; ++c) xr[c] = f[c * CSX];
        }
    }
#pragma unroll
    for (int n = 0; n < 2; ++n) load_b(k0, n, bq[n]);
    if (ring) load_b(k0, 2, bqr);

    T* po = out + (long long)k0 * a.plane + (long long)gja * a.pitch + gi;
    // a tile is "plain" when neither it nor its halo-1 ring touches a face of the domain: no one-sided in-plane
    // differences, no masks; the two instantiations of the main loop differ only in that
    const bool plain = i0 > 0 && i0 + TX <= a.nx - 2 && j0 > 0 && j0 + TY <= a.ny - 2;
    auto run = [&](auto plain_c) {
        constexpr bool PLAIN = decltype(plain_c)::value;
#pragma unroll kLeanUnroll
        for (int t = k0 - 1; t < kend; ++t) {
            const int q1 = t + 1 - pfirst;
            const T* f1 = sx + (q1 % R) * L::SLOTX + ox[0];       // xi plane t+1, node 0 of the pair
            const T* f2 = sx + ((q1 + 1) % R) * L::SLOTX + ox[0]; // xi plane t+2
            const bool fin = t >= k0;                              // plane t is finished (written) by this item
            // ---------------- I: in-plane part of D J of plane t ----------------
            T P[2][3];
            if (fin) {
                const T* g = sB + (t & 1) * L::BSLOT + oB[0];
#pragma unroll
                for (int n = 0; n < 2; ++n) {
                    T dBi[3], dBj[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const T* gc = g + c * BCS + n * BBW;
                        dBi[c] = gc[1] - gc[-1];
                        dBj[c] = n == 0 ? B0[1][c] - gc[-BBW] : gc[BBW] - B0[0][c];
                    }
                    cross_set(nA[n][0], dBi, P[n]);
                    cross_acc(nA[n][1], dBj, P[n]);
#pragma unroll
                    for (int c = 0; c < 3; ++c) P[n][c] -= W[n][c];
                }
            } else {
#pragma unroll
                for (int n = 0; n < 2; ++n)
#pragma unroll
                    for (int c = 0; c < 3; ++c) P[n][c] = T(0);
            }
            // ---------------- A: stage A of plane t+1;  F: finish plane t ----------------
            T x1[2][3];           // own xi(t+1)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                x1[0][c] = f1[c * CSX];
                x1[1][c] = f1[c * CSX + BW];
            }
            const bool inner_k = t + 1 > 0 && t + 1 < nz - 1;
#pragma unroll
            for (int n = 0; n < 2; ++n) {
                T dF[3][3];
                const T* fn = f1 + n * BW;
                if (t + 1 == 0) {          // bottom face: -3 x(0) + 4 x(1) - x(2)
                    const T* f3 = sx + ((q1 + 2) % R) * L::SLOTX + ox[0] + n * BW;
#pragma unroll
                    for (int c = 0; c < 3; ++c) dF[c][2] = T(4) * f2[c * CSX + n * BW] - T(3) * x1[n][c] - f3[c * CSX];
                } else if (t + 2 <= nz - 1) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) dF[c][2] = f2[c * CSX + n * BW] - xc[n][c];
                } else {                   // top face: 3 x(nz-1) - 4 x(nz-2) + x(nz-3); plane nz-3 is still in its slot
                    const T* fm = sx + ((q1 - 2) % R) * L::SLOTX + ox[0] + n * BW;
#pragma unroll
                    for (int c = 0; c < 3; ++c) dF[c][2] = T(3) * x1[n][c] - T(4) * xc[n][c] + fm[c * CSX];
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    dF[c][0] = fn[c * CSX + 1] - fn[c * CSX - 1];
                    dF[c][1] = n == 0 ? x1[1][c] - fn[c * CSX - BW] : fn[c * CSX + BW] - x1[0][c];
                }
                if (!PLAIN && edge[n]) face_fix<T, BW, CSX>(fn, edge[n], dF);
                T nv[3][3], Bn[3], inv;
                lean_push(dF, bq[n], twoh, nv, Bn, inv, ok, PLAIN || dom[n]);
                store_B(t + 1, n, Bn);
                if (t + 2 <= kend) load_b(t + 2, n, bq[n]);     // b of the plane the next iteration pushes forward
                if (fin) {
                    // D J = P + n_2 x B(t+1);  u = gamma J x B(t);  xi+ = xi + dt u
                    T uu[3];
                    cross_acc(n2[n], Bn, P[n]);
                    cross_set(P[n], B0[n], uu);
#pragma unroll
                    for (int c = 0; c < 3; ++c) xc[n][c] = fma(s[n], uu[c], xc[n][c]);
                    ok = ok && is_finite(xc[n][0] + xc[n][1] + xc[n][2]);
                    if (PLAIN || st[n]) {
                        T* pn = po + n * a.pitch;
                        pn[0] = xc[n][0];
                        pn[a.comp] = xc[n][1];
                        pn[2 * a.comp] = xc[n][2];
                    }
                }
                // the node's state moves on to plane t+1
                cross_set(nv[2], B0[n], W[n]);
                s[n] = (inner_k && (PLAIN || in_xy[n])) ? a.dtg * inv : T(0);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    nA[n][0][c] = nv[0][c];
                    nA[n][1][c] = nv[1][c];
                    n2[n][c] = nv[2][c];
                    B0[n][c] = Bn[c];
                    xc[n][c] = x1[n][c];
                }
            }
            if (fin) po += a.plane;
            if (ring && t + 1 < kend) {
                // stage A of plane t+1 at the ring node
                T dFr[3][3], nr[3][3], B[3], inv, xr1[3];
                const T* fr = sx + (q1 % R) * L::SLOTX + ox[2];
                const T* fr2 = sx + ((q1 + 1) % R) * L::SLOTX + ox[2];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    xr1[c] = fr[c * CSX];
                    dFr[c][0] = fr[c * CSX + 1] - fr[c * CSX - 1];
                    dFr[c][1] = fr[c * CSX + BW] - fr[c * CSX - BW];
                }
                if (t + 1 == 0) {
                    const T* f3 = sx + ((q1 + 2) % R) * L::SLOTX + ox[2];
#pragma unroll
                    for (int c = 0; c < 3; ++c) dFr[c][2] = T(4) * fr2[c * CSX] - T(3) * xr1[c] - f3[c * CSX];
                } else if (t + 2 <= nz - 1) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) dFr[c][2] = fr2[c * CSX] - xr[c];
                } else {
                    const T* fm = sx + ((q1 - 2) % R) * L::SLOTX + ox[2];
#pragma unroll
                    for (int c = 0; c < 3; ++c) dFr[c][2] = T(3) * xr1[c] - T(4) * xr[c] + fm[c * CSX];
                }
                if (!PLAIN && edge[2]) face_fix<T, BW, CSX>(fr, edge[2], dFr);
                lean_push(dFr, bqr, twoh, nr, B, inv, ok, PLAIN || dom[2]);
                store_B(t + 1, 2, B);
#pragma unroll
                for (int c = 0; c < 3; ++c) xr[c] = xr1[c];
                if (t + 2 < kend) load_b(t + 2, 2, bqr);
            }
            ptx::cta_sync();
            // every read of the xi plane t+1 is done: its slot takes the plane t+1+R
            if (producer) refill(t + 1 + R);
            if (t + 3 <= plast) { const int q = t + 3 - pfirst; ptx::mbar_wait(bar_x + 8u * (uint32_t)(q % R), (uint32_t)((q / R) & 1)); }
        }
    };
    if (plain) run(std::true_type{});
    else run(std::false_type{});
    if (k1 == nz) {   // the top plane (line-tied) is carried through
#pragma unroll
        for (int n = 0; n < 2; ++n)
            if (st[n]) {
                T* pl = out + (long long)(nz - 1) * a.plane + (long long)(gja + n) * a.pitch + gi;
                pl[0] = xc[n][0];
                pl[a.comp] = xc[n][1];
                pl[2 * a.comp] = xc[n][2];
            }
    }
    if (!ok) atomicOr(a.flag, FLAG_NUMERIC);
}

// ----------------------------------------------------------------------------------------------- host side

#ifndef MR_LTY
#define MR_LTY 16
#define MR_LR 4
#endif
constexpr int kLTY = MR_LTY, kLR = MR_LR;

template <typename T>
inline cudaError_t lean_set_smem(size_t bytes)
{
    cudaError_t e = cudaFuncSetAttribute(k_step_lean<T, kLTY, kLR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_step_lean<T, kLTY, kLR>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
}

inline bool build_lean_plan(StreamPlan* p, const StreamGeom& g, bool f64, void* xi0, void* xi1, void* b, int sm_count,
                            std::string* why)
{
    using Ld = LeanLayout<double, kLTY, kLR>;
    using Lf = LeanLayout<float, kLTY, kLR>;
    p->usable = false;
    p->f64 = f64;
    p->g = g;
    p->xi[0] = xi0;
    p->xi[1] = xi1;
    p->b = b;
    p->name = f64 ? "lean_tma_f64" : "lean_tma_f32";
    const int bw = f64 ? Ld::BW : Lf::BW;
    if (!encode_map(&p->map_xi[0], f64, xi0, g, bw, kLTY + 4) || !encode_map(&p->map_xi[1], f64, xi1, g, bw, kLTY + 4)) {
        *why = "cuTensorMapEncodeTiled failed";
        return false;
    }
    p->tiles_x = (g.nx + Ld::TX - 1) / Ld::TX;
    p->tiles_y = (g.ny + kLTY - 1) / kLTY;
    p->smem_bytes = f64 ? Ld::BYTES : Lf::BYTES;
    cudaError_t e = f64 ? lean_set_smem<double>(p->smem_bytes) : lean_set_smem<float>(p->smem_bytes);
    if (e != cudaSuccess) {
        *why = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e);
        return false;
    }
    int per_sm = 1;
    e = f64 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_step_lean<double, kLTY, kLR>, Ld::NTHREADS, p->smem_bytes)
            : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_step_lean<float, kLTY, kLR>, Lf::NTHREADS, p->smem_bytes);
    if (e != cudaSuccess || per_sm < 1) per_sm = 1;
    choose_chunks(p->tiles_x * p->tiles_y, g.nz, sm_count * per_sm, &p->nchunks, &p->chunk_len);
    p->usable = true;
    return true;
}

template <typename T>
inline cudaError_t launch_lean_step(const StreamPlan& p, int cur, T dtg, int* flag, cudaStream_t stream)
{
    using L = LeanLayout<T, kLTY, kLR>;
    StreamArgs<T> a;
    a.nx = p.g.nx; a.ny = p.g.ny; a.nz = p.g.nz;
    a.pitch = p.g.pitch; a.plane = p.g.plane; a.comp = p.g.comp;
    for (int c = 0; c < 3; ++c) a.twoh[c] = (T)p.g.twoh[c];
    a.dtg = dtg;
    a.tiles_x = p.tiles_x;
    a.ntiles = p.tiles_x * p.tiles_y;
    a.chunk_len = p.chunk_len;
    a.flag = flag;
    const int grid = a.ntiles * p.nchunks;
    k_step_lean<T, kLTY, kLR><<<grid, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], static_cast<const T*>(p.b),
                                                                            static_cast<T*>(p.xi[1 - cur]), a);
    return cudaGetLastError();
}

}  // namespace mr
