// mr_pair.cuh -- the register-paired streaming step kernel for the mimetic operator (S1-S5 in one pass).
//
// Same data flow as mr_stream.cuh (TMA rings of xi and b planes, CTA marching along k, B shared through a
// double-buffered shared plane, B/J/u never in HBM), with the shared-memory traffic per node cut down: the
// first streaming kernel was bound by the shared-memory data pipe (60 % busy at 0.67 ms/step on C4, ncu r1b),
// not by HBM.  Here every tile thread owns TWO nodes, (i, j) and (i, j+1), so that
//   * the j-differences of xi and of B inside the pair come from registers (own values), only the rows j-1 and
//     j+2 are read from shared memory: 4 instead of 5 xi reads and 3 instead of 4 B reads per node and component;
//   * the own column xi(k), xi(k+1), xi(k+2) stays in registers (no re-read of the centre value);
//   * address arithmetic, barrier and mbarrier waits are paid once per pair.
// Warp roles (TX = 32, TY rows per tile, TY/2 tile warps):
//   tile warps 0..TY/2-1   lane = i, warp w owns rows 2w and 2w+1;
//   ring warp  TY/2        the halo-1 rows j = -1 and j = TY (two nodes per thread, push-forward B only);
//   ring warp  TY/2+1      the halo-1 columns i = -1 and i = TX, lanes interleaved (8 rows left, 8 rows right per
//                          half-warp) so that with the row stride BW = 38 doubles the 16 lanes of a shared-memory
//                          wavefront fall into distinct banks; its lane 0 is the TMA producer.
// The xi / b boxes are TX + HXL + HXR wide: the left halo is widened to 16 bytes because the TMA unit wants the
// innermost start coordinate 16-byte aligned, the right one is padded so that the row stride is 2 (mod 4)
// doubles -- conflict-free column access.
#pragma once
#include <type_traits>

#include "mr_stream.cuh"

namespace mr {

template <typename T, int TY, int R, int RB>
struct PairLayout {
    static_assert(TY % 2 == 0 && TY >= 8 && TY <= 32 && R >= 4 && RB >= 2, "tile / ring sizes");
    static constexpr int TX = 32;
    static constexpr int HXL = 16 / (int)sizeof(T), HXR = 2 * HXL;
    static constexpr int BW = TX + HXL + HXR;
    static constexpr int XH = TY + 4, BH = TY + 2;
    static constexpr int CSX = BW * XH, CSB = BW * BH;
    static constexpr int round128(int bytes) { return (bytes + 127) / 128 * 128; }
    static constexpr int SLOTX = round128(3 * CSX * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr int SLOTB = round128(3 * CSB * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr uint32_t XBOX_BYTES = 3u * CSX * sizeof(T), BBOX_BYTES = 3u * CSB * sizeof(T);
    static constexpr int BBW = TX + 2, BBH = TY + 2;
    static constexpr int BCS = BBW * BBH;
    static constexpr int BSLOT = round128(3 * BCS * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr int NTILEW = TY / 2, NWARPS = NTILEW, NTHREADS = NWARPS * 32;
    static constexpr size_t OFF_X = 0;
    static constexpr size_t OFF_B0 = OFF_X + (size_t)R * SLOTX * sizeof(T);
    static constexpr size_t OFF_BB = OFF_B0 + (size_t)RB * SLOTB * sizeof(T);
    static constexpr size_t OFF_BAR = OFF_BB + (size_t)2 * BSLOT * sizeof(T);
    static constexpr size_t BYTES = OFF_BAR + (size_t)(R + RB) * 8 + 128;
};

// one-sided in-plane corrections of dF at a face node (reading Q3); f = the node in component 0 of its xi plane
template <typename T, int BW, int CSX>
__device__ __forceinline__ void face_fix(const T* __restrict__ f, unsigned edge, T (&dF)[3][3])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T xc = f[c * CSX];
        if (edge & 1u) dF[c][0] = T(4) * f[c * CSX + 1] - T(3) * xc - f[c * CSX + 2];
        if (edge & 2u) dF[c][0] = T(3) * xc - T(4) * f[c * CSX - 1] + f[c * CSX - 2];
        if (edge & 4u) dF[c][1] = T(4) * f[c * CSX + BW] - T(3) * xc - f[c * CSX + 2 * BW];
        if (edge & 8u) dF[c][1] = T(3) * xc - T(4) * f[c * CSX - BW] + f[c * CSX - 2 * BW];
    }
}

// Area vectors of the three index surfaces through a node, n_q = dF_{q+1} x dF_{q+2} (columns of dF; un-normalised
// Eq. 2.5/2.6 -- the vector sum of the four triangles), D = det dF = dF_0 . n_0, 1/D and B = dF b / D (Eq. 2.1).
// dF comes in without the 2h diagonal.
template <typename T, int CSB>
__device__ __forceinline__ void push_forward_n(T (&dF)[3][3], const T* __restrict__ bs, const T (&twoh)[3], T (&n)[3][3], T (&B)[3],
                                               T& inv, bool& ok, bool in_dom)
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
    const T b0 = bs[0] * inv, b1 = bs[CSB] * inv, b2 = bs[2 * CSB] * inv;
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = dF[c][0] * b0 + dF[c][1] * b1 + dF[c][2] * b2;
}

// acc = n x v  /  acc += n x v, as chains of fused multiply-adds
template <typename T>
__device__ __forceinline__ void cross_set(const T (&n)[3], const T (&v)[3], T (&acc)[3])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        acc[c] = fma(n[c1], v[c2], -(n[c2] * v[c1]));
    }
}
template <typename T>
__device__ __forceinline__ void cross_acc(const T (&n)[3], const T (&v)[3], T (&acc)[3])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        acc[c] = fma(-n[c2], v[c1], fma(n[c1], v[c2], acc[c]));
    }
}

template <typename T, int TY, int R, int RB>
__global__ void __launch_bounds__(TY * 16, 1)
k_step_pair(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_b, T* __restrict__ out,
            const StreamArgs<T> a)
{
    using L = PairLayout<T, TY, R, RB>;
    constexpr int TX = L::TX, NT = L::NTILEW, BW = L::BW, CSX = L::CSX, CSB = L::CSB, BBW = L::BBW, BCS = L::BCS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((128u - (ptx::smem_u32(smem_raw) & 127u)) & 127u);
    const T* sx = reinterpret_cast<const T*>(smem + L::OFF_X);
    const T* sb = reinterpret_cast<const T*>(smem + L::OFF_B0);
    T* sB = reinterpret_cast<T*>(smem + L::OFF_BB);
    const uint32_t sx_u32 = ptx::smem_u32(sx), sb_u32 = ptx::smem_u32(sb);
    const uint32_t bar_x = ptx::smem_u32(smem + L::OFF_BAR), bar_b = bar_x + 8u * R;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x % a.ntiles, chunk = blockIdx.x / a.ntiles;
    const int i0 = (tile % a.tiles_x) * TX, j0 = (tile / a.tiles_x) * TY;
    const int nz = a.nz;
    const int k0 = chunk * a.chunk_len, k1 = min(k0 + a.chunk_len, nz);
    const int pfirst = max(k0 - 2, 0), plast = min(k1 + 1, nz - 1);     // xi planes this item touches
    const int bfirst = max(k0 - 1, 0), blast = min(k1, nz - 1);         // planes whose B is formed
    const T twoh[3] = { a.twoh[0], a.twoh[1], a.twoh[2] };

    // ---- TMA producer: lane 0 of the last warp (one without a ring node); a slot is refilled once its plane is dead ----
    const bool producer = tid == (NT - 1) * 32;
    auto load_x = [&](int p, uint32_t s) {
        ptx::mbar_expect_tx(bar_x + 8u * s, L::XBOX_BYTES);
        ptx::tma_load_4d(sx_u32 + s * (uint32_t)(L::SLOTX * sizeof(T)), &map_in, i0 - L::HXL, j0 - 2, p, 0, bar_x + 8u * s);
    };
    auto load_b = [&](int p, uint32_t s) {
        ptx::mbar_expect_tx(bar_b + 8u * s, L::BBOX_BYTES);
        ptx::tma_load_4d(sb_u32 + s * (uint32_t)(L::SLOTB * sizeof(T)), &map_b, i0 - L::HXL, j0 - 1, p, 0, bar_b + 8u * s);
    };
    if (producer) {
        for (int s = 0; s < R + RB; ++s) ptx::mbar_init(bar_x + 8u * s, 1);
        ptx::fence_mbar_init();
    }
    __syncthreads();
    if (producer) {   // the first R xi planes and RB b planes
        for (int p = pfirst; p <= min(plast, pfirst + R - 1); ++p) load_x(p, (uint32_t)(p - pfirst));
        for (int p = bfirst; p <= min(blast, bfirst + RB - 1); ++p) load_b(p, (uint32_t)(p - bfirst));
    }

    auto wait_x = [&](int p) { const int q = p - pfirst; ptx::mbar_wait(bar_x + 8u * (uint32_t)(q % R), (uint32_t)((q / R) & 1)); };
    auto wait_b = [&](int p) { const int q = p - bfirst; ptx::mbar_wait(bar_b + 8u * (uint32_t)(q % RB), (uint32_t)((q / RB) & 1)); };
    auto xplane = [&](int p) -> const T* { return sx + ((p - pfirst) % R) * L::SLOTX; };
    auto bplane = [&](int p) -> const T* { return sb + ((p - bfirst) % RB) * L::SLOTB; };

    // every plane the prologue reads: xi pfirst..min(k0+1, plast), b bfirst..k0
    for (int p = pfirst; p <= min(k0 + 1, plast); ++p) wait_x(p);
    for (int p = bfirst; p <= k0; ++p) wait_b(p);

    // nodes of this thread in tile coordinates: 0, 1 = the pair (lane, 2 warp), (lane, 2 warp + 1); 2 = a node of the
    // halo-1 ring for the threads that carry one (only its push-forward B is formed)
    int ti[3], tj[3];
    ti[0] = ti[1] = lane;
    tj[0] = 2 * warp;
    tj[1] = 2 * warp + 1;
    bool ring = false;
#ifdef MR_NO_RING
    if (true) { ti[2] = 0; tj[2] = 0; }
    else
#endif
    if (warp == 0) { ring = true; ti[2] = lane; tj[2] = -1; }
    else if (warp == 1) { ring = true; ti[2] = lane; tj[2] = TY; }
    else if (warp < 4) {
        // columns: half of the rows per warp, left and right side in the same half-warp (distinct banks at stride BW)
        constexpr int HALF = TY / 2;
        ring = lane < 2 * HALF;
        ti[2] = (lane / HALF) & 1 ? TX : -1;
        tj[2] = (lane % HALF) + HALF * (warp - 2);
    } else { ti[2] = 0; tj[2] = 0; }
    int ox[3], ob[3], oB[3];
    unsigned edge[3];
    bool dom[3];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        const int gi = i0 + ti[n], gj = j0 + tj[n];
        ox[n] = (tj[n] + 2) * BW + (ti[n] + L::HXL);
        ob[n] = (tj[n] + 1) * BW + (ti[n] + L::HXL);
        oB[n] = (tj[n] + 1) * BBW + (ti[n] + 1);
        dom[n] = gi >= 0 && gi < a.nx && gj >= 0 && gj < a.ny;
        edge[n] = !dom[n] ? 0u
            : (gi == 0 ? 1u : 0u) | (gi == a.nx - 1 ? 2u : 0u) | (gj == 0 ? 4u : 0u) | (gj == a.ny - 1 ? 8u : 0u);
    }

    // stage A of plane p at one node with every operand from shared memory (prologue only)
    auto A_from_smem = [&](int p, int n, T(&nv)[3][3], T(&B)[3], T& inv, bool& ok) {
        const T* pc = xplane(p) + ox[n];
        const T *pa, *pb;
        T ca, cb, cc;     // on a k face: dk = ca * pa + cb * pb + cc * pc
        if (p == 0) { pa = xplane(1) + ox[n]; pb = xplane(2) + ox[n]; ca = T(4); cb = T(-1); cc = T(-3); }
        else if (p == nz - 1) { pa = xplane(p - 1) + ox[n]; pb = xplane(p - 2) + ox[n]; ca = T(-4); cb = T(1); cc = T(3); }
        else { pa = xplane(p + 1) + ox[n]; pb = xplane(p - 1) + ox[n]; ca = T(1); cb = T(-1); cc = T(0); }
        T dF[3][3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            dF[c][0] = pc[c * CSX + 1] - pc[c * CSX - 1];
            dF[c][1] = pc[c * CSX + BW] - pc[c * CSX - BW];
            dF[c][2] = (p == 0 || p == nz - 1) ? ca * pa[c * CSX] + cc * pc[c * CSX] + cb * pb[c * CSX] : pa[c * CSX] - pb[c * CSX];
        }
        if (edge[n]) face_fix<T, BW, CSX>(pc, edge[n], dF);
        push_forward_n<T, CSB>(dF, bplane(p) + ob[n], twoh, nv, B, inv, ok, dom[n]);
    };
    auto store_B = [&](int p, int n, const T(&B)[3]) {
        T* d = sB + (p & 1) * L::BSLOT + oB[n];
        d[0] = B[0];
        d[BCS] = B[1];
        d[2 * BCS] = B[2];
    };

    bool ok = true;
    // running ring positions of the xi planes k+1, k+2 and the b plane k+1 of the main loop
    int sl0 = (k0 - pfirst) % R, sl1 = (k0 + 1 - pfirst) % R, sl2 = (k0 + 2 - pfirst) % R;
    uint32_t par2 = (uint32_t)(((k0 + 2 - pfirst) / R) & 1);
    int slb = (k0 + 1 - bfirst) % RB;
    uint32_t parb = (uint32_t)(((k0 + 1 - bfirst) / RB) & 1);
    auto advance = [&]() {
        sl0 = sl1;
        sl1 = sl2;
        if (++sl2 == R) { sl2 = 0; par2 ^= 1u; }
        if (++slb == RB) { slb = 0; parb ^= 1u; }
    };
    // own-column k-difference of plane k+1 (k+1 <= nz-1): central x2 - x0 with x2 = xi(k+2) read here, or on the top
    // face 3 x1 - 4 x0 + xi(k-1) (plane nz-3 is still in its slot: nothing is loaded beyond plane nz-1)
    auto column_dk = [&](int k, int n, const T(&x0)[3], const T(&x1)[3], T(&x2)[3], T(&dk)[3]) {
        if (k + 2 <= nz - 1) {
            const T* p2 = sx + sl2 * L::SLOTX + ox[n];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                x2[c] = p2[c * CSX];
                dk[c] = x2[c] - x0[c];
            }
        } else {
            const T* pm = xplane(k - 1) + ox[n];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                x2[c] = T(0);
                dk[c] = T(3) * x1[c] - T(4) * x0[c] + pm[c * CSX];
            }
        }
    };

    const int gi = i0 + lane, gja = j0 + tj[0];
    const bool in_x = gi > 0 && gi < a.nx - 1;
    const bool in_xy0 = in_x && gja > 0 && gja < a.ny - 1, in_xy1 = in_x && gja + 1 < a.ny - 1;
    // Per-plane state of the pair, two sets used in turn (the loop is unrolled twice, so no register moves):
    //   nq    area vectors n_0, n_1, n_2 of the plane      invq  1 / det dF
    //   Bq    own B of the plane                            Wq    n_2(plane) x B(plane - 1), the lower half of the
    //   Xq    own xi of the planes k+1, k+2                       k-loop term n_2 x (B(k+1) - B(k-1))
    T nq[2][2][3][3], invq[2][2], Bq[2][2][3], Wq[2][2][3], Xq[2][2][3];
#pragma unroll
    for (int n = 0; n < 2; ++n) {
        const T* pb = xplane(min(k0 + 1, nz - 1)) + ox[n];
        T Bl[3] = { T(0), T(0), T(0) };
        if (k0 > 0) {
            T nt[3][3], it;
            A_from_smem(k0 - 1, n, nt, Bl, it, ok);
        }
        A_from_smem(k0, n, nq[0][n], Bq[0][n], invq[0][n], ok);
        store_B(k0, n, Bq[0][n]);
        cross_set(nq[0][n][2], Bl, Wq[0][n]);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Xq[0][n][c] = pb[c * CSX];
            Xq[1][n][c] = T(0);
        }
    }
    if (ring) {
        T nt[3][3], B[3], inv;
        A_from_smem(k0, 2, nt, B, inv, ok);
        store_B(k0, 2, B);
    }
    ptx::cta_sync();
    if (producer) {   // planes < k0 of xi and <= k0 of b are dead: top the rings up to k0-1+R resp. k0+RB
        for (int p = pfirst + R; p <= min(plast, k0 - 1 + R); ++p) load_x(p, (uint32_t)((p - pfirst) % R));
        for (int p = bfirst + RB; p <= min(blast, k0 + RB); ++p) load_b(p, (uint32_t)((p - bfirst) % RB));
    }
    T* po = out + (long long)k0 * a.plane + (long long)gja * a.pitch + gi;
    const bool st0 = gi < a.nx && gja < a.ny, st1 = gi < a.nx && gja + 1 < a.ny;
    // a tile is "plain" when neither it nor its halo-1 ring touches a face of the domain: no one-sided differences,
    // no masks; the two instantiations of the main loop differ only in that
    const bool plain = i0 > 0 && i0 + TX <= a.nx - 2 && j0 > 0 && j0 + TY <= a.ny - 2;
    // the main loop takes the planes k0 .. kend-1, each with a stage A of plane k+1; the top plane nz-1 (line-tied,
    // nothing above it) is copied through from its slot afterwards
    const int kend = min(k1, nz - 1);
    auto run = [&](auto plain_c) {
        constexpr bool PLAIN = decltype(plain_c)::value;
        for (int kb = k0; kb < kend; kb += 2) {
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int k = kb + u;
                if (k >= kend) break;
                T(&ncur)[2][3][3] = nq[u];
                T(&nnew)[2][3][3] = nq[u ^ 1];
                T(&Bc)[2][3] = Bq[u];
                T(&Bn)[2][3] = Bq[u ^ 1];
                T(&x1)[2][3] = Xq[u];
                T(&x2)[2][3] = Xq[u ^ 1];
#ifdef MR_NO_STAGEB
                const bool inner_k = false;
#else
                const bool inner_k = k > 0;          // (k <= nz-2 inside this loop)
#endif
                const T* f0 = sx + sl0 * L::SLOTX + ox[0];
                T x0[2][3];                           // own xi of plane k (re-read: plane k stays in its slot)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    x0[0][c] = f0[c * CSX];
                    x0[1][c] = f0[c * CSX + BW];
                }
#ifdef MR_COPY_ONLY   /* experiment: the data movement alone (TMA ring, barrier per plane, coalesced store), no arithmetic */
                {
                    if (k + 2 <= nz - 1) ptx::mbar_wait(bar_x + 8u * (uint32_t)sl2, par2);
                    ptx::mbar_wait(bar_b + 8u * (uint32_t)slb, parb);
                    const T* bs = sb + slb * L::SLOTB + ob[0];
                    if (PLAIN || st0) { po[0] = x0[0][0] + T(1e-30) * bs[0]; po[a.comp] = x0[0][1] + T(1e-30) * bs[CSB]; po[2 * a.comp] = x0[0][2] + T(1e-30) * bs[2 * CSB]; }
                    if (PLAIN || st1) { po[a.pitch] = x0[1][0] + T(1e-30) * bs[BW]; po[a.comp + a.pitch] = x0[1][1] + T(1e-30) * bs[CSB + BW]; po[2 * a.comp + a.pitch] = x0[1][2] + T(1e-30) * bs[2 * CSB + BW]; }
                    po += a.plane;
                    ptx::cta_sync();
                    if (producer) {
                        if (k + R <= plast) load_x(k + R, (uint32_t)sl0);
                        if (k + 1 + RB <= blast) load_b(k + 1 + RB, (uint32_t)slb);
                    }
                    advance();
                    continue;
                }
#endif
                T DJ[2][3];     // D J = sum_q n_q x delta_q B (closed form of Eqs. 2.3-2.7), built up in two parts
                if (inner_k) {
                    // ---- in-plane part of D J of plane k: n_0 x delta_i B + n_1 x delta_j B ----
                    const T* g = sB + (k & 1) * L::BSLOT + oB[0];
                    T dBi[2][3], dBj[2][3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const T* gc = g + c * BCS;
                        dBi[0][c] = gc[1] - gc[-1];
                        dBi[1][c] = gc[BBW + 1] - gc[BBW - 1];
                        dBj[0][c] = Bc[1][c] - gc[-BBW];
                        dBj[1][c] = gc[2 * BBW] - Bc[0][c];
                    }
#pragma unroll
                    for (int n = 0; n < 2; ++n) {
                        cross_set(ncur[n][0], dBi[n], DJ[n]);
                        cross_acc(ncur[n][1], dBj[n], DJ[n]);
                    }
                }
                {
                    // ---- stage A of plane k+1 at the pair ----
                    T dF[2][3][3];
                    const T* f = sx + sl1 * L::SLOTX + ox[0];
                    if (k + 2 <= nz - 1) {
#ifndef MR_NO_REFILL
                        ptx::mbar_wait(bar_x + 8u * (uint32_t)sl2, par2);
#endif
                        const T* f2 = sx + sl2 * L::SLOTX + ox[0];
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            x2[0][c] = f2[c * CSX];
                            x2[1][c] = f2[c * CSX + BW];
                            dF[0][c][2] = x2[0][c] - x0[0][c];
                            dF[1][c][2] = x2[1][c] - x0[1][c];
                        }
                    } else {   // top face: 3 x(nz-1) - 4 x(nz-2) + x(nz-3); plane nz-3 is still in its slot
                        const T* fm = xplane(k - 1) + ox[0];
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            dF[0][c][2] = T(3) * x1[0][c] - T(4) * x0[0][c] + fm[c * CSX];
                            dF[1][c][2] = T(3) * x1[1][c] - T(4) * x0[1][c] + fm[c * CSX + BW];
                        }
                    }
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const T* fc = f + c * CSX;
                        dF[0][c][0] = fc[1] - fc[-1];
                        dF[1][c][0] = fc[BW + 1] - fc[BW - 1];
                        dF[0][c][1] = x1[1][c] - fc[-BW];
                        dF[1][c][1] = fc[2 * BW] - x1[0][c];
                    }
                    if (!PLAIN) {
                        if (edge[0]) face_fix<T, BW, CSX>(f, edge[0], dF[0]);
                        if (edge[1]) face_fix<T, BW, CSX>(f + BW, edge[1], dF[1]);
                    }
#ifndef MR_NO_REFILL
                    ptx::mbar_wait(bar_b + 8u * (uint32_t)slb, parb);
#endif
                    const T* bs = sb + slb * L::SLOTB + ob[0];
                    push_forward_n<T, CSB>(dF[0], bs, twoh, nnew[0], Bn[0], invq[u ^ 1][0], ok, PLAIN || dom[0]);
                    push_forward_n<T, CSB>(dF[1], bs + BW, twoh, nnew[1], Bn[1], invq[u ^ 1][1], ok, PLAIN || dom[1]);
                    store_B(k + 1, 0, Bn[0]);
                    store_B(k + 1, 1, Bn[1]);
                    cross_set(nnew[0][2], Bc[0], Wq[u ^ 1][0]);
                    cross_set(nnew[1][2], Bc[1], Wq[u ^ 1][1]);
                    if (ring) {
                        // ---- stage A of plane k+1 at the ring node (every operand from shared memory) ----
                        T dFr[3][3], nr[3][3], B[3], inv;
                        const T* fr = sx + sl1 * L::SLOTX + ox[2];
                        const T* fr0 = sx + sl0 * L::SLOTX + ox[2];
                        if (k + 2 <= nz - 1) {
                            const T* fr2 = sx + sl2 * L::SLOTX + ox[2];
#pragma unroll
                            for (int c = 0; c < 3; ++c) dFr[c][2] = fr2[c * CSX] - fr0[c * CSX];
                        } else {
                            const T* fm = xplane(k - 1) + ox[2];
#pragma unroll
                            for (int c = 0; c < 3; ++c) dFr[c][2] = T(3) * fr[c * CSX] - T(4) * fr0[c * CSX] + fm[c * CSX];
                        }
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            dFr[c][0] = fr[c * CSX + 1] - fr[c * CSX - 1];
                            dFr[c][1] = fr[c * CSX + BW] - fr[c * CSX - BW];
                        }
                        if (!PLAIN && edge[2]) face_fix<T, BW, CSX>(fr, edge[2], dFr);
                        push_forward_n<T, CSB>(dFr, sb + slb * L::SLOTB + ob[2], twoh, nr, B, inv, ok, PLAIN || dom[2]);
                        store_B(k + 1, 2, B);
                    }
                }
                if (inner_k) {
                    // ---- k part of D J: n_2 x (B(k+1) - B(k-1)); u = gamma J x B (Eq. 1.5); xi += dt u inside ----
#pragma unroll
                    for (int n = 0; n < 2; ++n) {
                        T uu[3];
                        cross_acc(ncur[n][2], Bn[n], DJ[n]);
#pragma unroll
                        for (int c = 0; c < 3; ++c) DJ[n][c] -= Wq[u][n][c];
                        cross_set(DJ[n], Bc[n], uu);
                        const bool doit = PLAIN || (n == 0 ? in_xy0 : in_xy1);
                        const T sc = doit ? a.dtg * invq[u][n] : T(0);
#pragma unroll
                        for (int c = 0; c < 3; ++c) x0[n][c] = fma(sc, uu[c], x0[n][c]);
                        ok = ok && (is_finite(x0[n][0] + x0[n][1] + x0[n][2]) || !doit);
                    }
                }
                if (PLAIN || st0) {
                    po[0] = x0[0][0];
                    po[a.comp] = x0[0][1];
                    po[2 * a.comp] = x0[0][2];
                }
                if (PLAIN || st1) {
                    po[a.pitch] = x0[1][0];
                    po[a.comp + a.pitch] = x0[1][1];
                    po[2 * a.comp + a.pitch] = x0[1][2];
                }
                po += a.plane;
#ifndef MR_NO_BAR
                ptx::cta_sync();
#endif
                // the xi plane k and the b plane k+1 are dead now: their slots take the planes k+R and k+1+RB
#ifdef MR_NO_REFILL
                if (false) {
#else
                if (producer) {
#endif
                    if (k + R <= plast) load_x(k + R, (uint32_t)sl0);
                    if (k + 1 + RB <= blast) load_b(k + 1 + RB, (uint32_t)slb);
                }
                advance();
            }
        }
    };
    if (plain) run(std::true_type{});
    else run(std::false_type{});
    if (k1 == nz) {
        const T* pt = xplane(nz - 1) + ox[0];
        T* pl = out + (long long)(nz - 1) * a.plane + (long long)gja * a.pitch + gi;
        if (st0) { pl[0] = pt[0]; pl[a.comp] = pt[CSX]; pl[2 * a.comp] = pt[2 * CSX]; }
        if (st1) { pl[a.pitch] = pt[BW]; pl[a.comp + a.pitch] = pt[CSX + BW]; pl[2 * a.comp + a.pitch] = pt[2 * CSX + BW]; }
    }
#ifndef MR_NO_FLAG
    if (!ok) atomicOr(a.flag, FLAG_NUMERIC);
#endif
}

// ----------------------------------------------------------------------------------------------- host side

#ifndef MR_PTY
#define MR_PTY 16
#define MR_PR 6
#define MR_PRB 3
#endif
constexpr int kPTY = MR_PTY, kPR = MR_PR, kPRB = MR_PRB;

template <typename T>
inline cudaError_t pair_set_smem(size_t bytes)
{
    return cudaFuncSetAttribute(k_step_pair<T, kPTY, kPR, kPRB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

inline bool build_pair_plan(StreamPlan* p, const StreamGeom& g, bool f64, void* xi0, void* xi1, void* b, int sm_count,
                            std::string* why)
{
    using Ld = PairLayout<double, kPTY, kPR, kPRB>;
    using Lf = PairLayout<float, kPTY, kPR, kPRB>;
    p->usable = false;
    p->f64 = f64;
    p->g = g;
    p->xi[0] = xi0;
    p->xi[1] = xi1;
    p->name = f64 ? "pair_tma_f64_32x16" : "pair_tma_f32_32x16";
    const int bw = f64 ? Ld::BW : Lf::BW;
    if (!encode_map(&p->map_xi[0], f64, xi0, g, bw, kPTY + 4) || !encode_map(&p->map_xi[1], f64, xi1, g, bw, kPTY + 4) ||
        !encode_map(&p->map_b, f64, b, g, bw, kPTY + 2)) {
        *why = "cuTensorMapEncodeTiled failed";
        return false;
    }
    p->tiles_x = (g.nx + Ld::TX - 1) / Ld::TX;
    p->tiles_y = (g.ny + kPTY - 1) / kPTY;
    p->smem_bytes = f64 ? Ld::BYTES : Lf::BYTES;
    cudaError_t e = f64 ? pair_set_smem<double>(p->smem_bytes) : pair_set_smem<float>(p->smem_bytes);
    if (e != cudaSuccess) {
        *why = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e);
        return false;
    }
    choose_chunks(p->tiles_x * p->tiles_y, g.nz, sm_count, &p->nchunks, &p->chunk_len);
    p->usable = true;
    return true;
}

template <typename T>
inline cudaError_t launch_pair_step(const StreamPlan& p, int cur, T dtg, int* flag, cudaStream_t stream)
{
    using L = PairLayout<T, kPTY, kPR, kPRB>;
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
    k_step_pair<T, kPTY, kPR, kPRB><<<grid, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], p.map_b,
                                                                                 static_cast<T*>(p.xi[1 - cur]), a);
    return cudaGetLastError();
}

}  // namespace mr
