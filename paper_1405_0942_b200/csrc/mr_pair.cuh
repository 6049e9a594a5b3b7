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

// D = det dF, 1/D, B = dF b / D (Eq. 2.1) from a finished dF (diagonal 2h not yet added)
template <typename T, int CSB>
__device__ __forceinline__ void push_forward(T (&dF)[3][3], const T* __restrict__ bs, const T (&twoh)[3], T (&B)[3], T& inv,
                                             bool& ok, bool in_dom)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) dF[c][c] += twoh[c];
    const T D = det3(dF);
    ok = ok && (positive_finite(D) || !in_dom);
    inv = fast_rcp(D);
    const T b0 = bs[0] * inv, b1 = bs[CSB] * inv, b2 = bs[2 * CSB] * inv;
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = dF[c][0] * b0 + dF[c][1] * b1 + dF[c][2] * b2;
}

// xi += s (dF chat) x B, chat_p = eps_pqr dB_q . dF_r (closed form of Eqs. 2.3-2.7, Eq. 1.5); dB[a][c] = delta_a B_c
template <typename T>
__device__ __forceinline__ void relax_node(const T (&dB)[3][3], const T (&dF)[3][3], const T (&Bc)[3], T s, bool doit, T (&x)[3],
                                           bool& ok)
{
    T ch[3];
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const int q = (p + 1) % 3, r = (p + 2) % 3;
        ch[p] = dB[q][0] * dF[0][r] + dB[q][1] * dF[1][r] + dB[q][2] * dF[2][r]
              - dB[r][0] * dF[0][q] - dB[r][1] * dF[1][q] - dB[r][2] * dF[2][q];
    }
    T J[3], u[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) J[c] = dF[c][0] * ch[0] + dF[c][1] * ch[1] + dF[c][2] * ch[2];
    cross3(J, Bc, u);
    const T n0 = x[0] + s * u[0], n1 = x[1] + s * u[1], n2 = x[2] + s * u[2];
    ok = ok && (is_finite(n0 + n1 + n2) || !doit);
    x[0] = doit ? n0 : x[0];
    x[1] = doit ? n1 : x[1];
    x[2] = doit ? n2 : x[2];
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
    int next_x = pfirst, next_b = bfirst;
    auto refill = [&](int dead_x, int dead_b) {
        for (; next_x <= plast && next_x - R <= dead_x; ++next_x) {
            const uint32_t s = (uint32_t)((next_x - pfirst) % R);
            ptx::mbar_expect_tx(bar_x + 8u * s, L::XBOX_BYTES);
            ptx::tma_load_4d(sx_u32 + s * (uint32_t)(L::SLOTX * sizeof(T)), &map_in, i0 - L::HXL, j0 - 2, next_x, 0, bar_x + 8u * s);
        }
        for (; next_b <= blast && next_b - RB <= dead_b; ++next_b) {
            const uint32_t s = (uint32_t)((next_b - bfirst) % RB);
            ptx::mbar_expect_tx(bar_b + 8u * s, L::BBOX_BYTES);
            ptx::tma_load_4d(sb_u32 + s * (uint32_t)(L::SLOTB * sizeof(T)), &map_b, i0 - L::HXL, j0 - 1, next_b, 0, bar_b + 8u * s);
        }
    };
    if (producer) {
        for (int s = 0; s < R + RB; ++s) ptx::mbar_init(bar_x + 8u * s, 1);
        ptx::fence_mbar_init();
    }
    __syncthreads();
    if (producer) refill(pfirst - 1, bfirst - 1);

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
    auto A_from_smem = [&](int p, int n, T(&dF)[3][3], T(&B)[3], T& inv, bool& ok) {
        const T* pc = xplane(p) + ox[n];
        const T *pa, *pb;
        T ca, cb, cc;     // on a k face: dk = ca * pa + cb * pb + cc * pc
        if (p == 0) { pa = xplane(1) + ox[n]; pb = xplane(2) + ox[n]; ca = T(4); cb = T(-1); cc = T(-3); }
        else if (p == nz - 1) { pa = xplane(p - 1) + ox[n]; pb = xplane(p - 2) + ox[n]; ca = T(-4); cb = T(1); cc = T(3); }
        else { pa = xplane(p + 1) + ox[n]; pb = xplane(p - 1) + ox[n]; ca = T(1); cb = T(-1); cc = T(0); }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            dF[c][0] = pc[c * CSX + 1] - pc[c * CSX - 1];
            dF[c][1] = pc[c * CSX + BW] - pc[c * CSX - BW];
            dF[c][2] = (p == 0 || p == nz - 1) ? ca * pa[c * CSX] + cc * pc[c * CSX] + cb * pb[c * CSX] : pa[c * CSX] - pb[c * CSX];
        }
        if (edge[n]) face_fix<T, BW, CSX>(pc, edge[n], dF);
        push_forward<T, CSB>(dF, bplane(p) + ob[n], twoh, B, inv, ok, dom[n]);
    };
    auto store_B = [&](int p, int n, const T(&B)[3]) {
        T* d = sB + (p & 1) * L::BSLOT + oB[n];
        d[0] = B[0];
        d[BCS] = B[1];
        d[2 * BCS] = B[2];
    };

    bool ok = true;
    // running ring positions of the xi planes k+1, k+2 and the b plane k+1 of the main loop
    int sl1 = (k0 + 1 - pfirst) % R, sl2 = (k0 + 2 - pfirst) % R;
    uint32_t par2 = (uint32_t)(((k0 + 2 - pfirst) / R) & 1);
    int slb = (k0 + 1 - bfirst) % RB;
    uint32_t parb = (uint32_t)(((k0 + 1 - bfirst) / RB) & 1);
    auto advance = [&]() {
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
    const unsigned edges = edge[0] | edge[1];
    T X[3][3][3];        // own xi at planes k, k+1, k+2 (rotating), per node (pair + ring node)
    T Bq[3][2][3];       // own B at planes k-1, k, k+1 (rotating)
    T dFq[2][2][3][3];   // dF at planes k, k+1 (rotating)
    T invq[2][2];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        const T* pa = xplane(k0) + ox[n];
        const T* pb = xplane(min(k0 + 1, nz - 1)) + ox[n];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            X[0][n][c] = pa[c * CSX];
            X[1][n][c] = pb[c * CSX];
            X[2][n][c] = T(0);
        }
    }
#pragma unroll
    for (int n = 0; n < 2; ++n) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Bq[0][n][c] = T(0);
            Bq[2][n][c] = T(0);
        }
        if (k0 > 0) {
            T dFt[3][3], it;
            A_from_smem(k0 - 1, n, dFt, Bq[0][n], it, ok);
        }
        A_from_smem(k0, n, dFq[0][n], Bq[1][n], invq[0][n], ok);
        store_B(k0, n, Bq[1][n]);
        invq[1][n] = T(0);
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int q = 0; q < 3; ++q) dFq[1][n][c][q] = T(0);
    }
    if (ring) {
        T dF[3][3], B[3], inv;
        A_from_smem(k0, 2, dF, B, inv, ok);
        store_B(k0, 2, B);
    }
    ptx::cta_sync();
    if (producer) refill(k0, k0);
    T* po = out + (long long)k0 * a.plane + (long long)gja * a.pitch + gi;
    const bool st0 = gi < a.nx && gja < a.ny, st1 = gi < a.nx && gja + 1 < a.ny;

    for (int kb = k0; kb < k1; kb += 6) {
#pragma unroll
        for (int u = 0; u < 6; ++u) {
            const int k = kb + u;
            if (k >= k1) break;
            T(&x0)[3][3] = X[u % 3];
            T(&x1)[3][3] = X[(u + 1) % 3];
            T(&x2)[3][3] = X[(u + 2) % 3];
            T(&Bm)[2][3] = Bq[u % 3];
            T(&Bc)[2][3] = Bq[(u + 1) % 3];
            T(&Bp)[2][3] = Bq[(u + 2) % 3];
            T(&dFc)[2][3][3] = dFq[u % 2];
            T(&dFn)[2][3][3] = dFq[(u + 1) % 2];
            if (k + 1 <= nz - 1) {
                // ---- stage A of plane k+1 at the pair ----
                T dk[2][3];
                if (k + 2 <= nz - 1) ptx::mbar_wait(bar_x + 8u * (uint32_t)sl2, par2);
                column_dk(k, 0, x0[0], x1[0], x2[0], dk[0]);
                column_dk(k, 1, x0[1], x1[1], x2[1], dk[1]);
                const T* f = sx + sl1 * L::SLOTX + ox[0];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const T* fc = f + c * CSX;
                    dFn[0][c][0] = fc[1] - fc[-1];
                    dFn[1][c][0] = fc[BW + 1] - fc[BW - 1];
                    dFn[0][c][1] = x1[1][c] - fc[-BW];
                    dFn[1][c][1] = fc[2 * BW] - x1[0][c];
                    dFn[0][c][2] = dk[0][c];
                    dFn[1][c][2] = dk[1][c];
                }
                if (edges) {
                    if (edge[0]) face_fix<T, BW, CSX>(f, edge[0], dFn[0]);
                    if (edge[1]) face_fix<T, BW, CSX>(f + BW, edge[1], dFn[1]);
                }
                ptx::mbar_wait(bar_b + 8u * (uint32_t)slb, parb);
                const T* bs = sb + slb * L::SLOTB + ob[0];
                push_forward<T, CSB>(dFn[0], bs, twoh, Bp[0], invq[(u + 1) % 2][0], ok, dom[0]);
                push_forward<T, CSB>(dFn[1], bs + BW, twoh, Bp[1], invq[(u + 1) % 2][1], ok, dom[1]);
                store_B(k + 1, 0, Bp[0]);
                store_B(k + 1, 1, Bp[1]);
                if (ring) {
                    // ---- stage A of plane k+1 at the ring node ----
                    T dkr[3], dF[3][3], B[3], inv;
                    column_dk(k, 2, x0[2], x1[2], x2[2], dkr);
                    const T* fr = sx + sl1 * L::SLOTX + ox[2];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        dF[c][0] = fr[c * CSX + 1] - fr[c * CSX - 1];
                        dF[c][1] = fr[c * CSX + BW] - fr[c * CSX - BW];
                        dF[c][2] = dkr[c];
                    }
                    if (edge[2]) face_fix<T, BW, CSX>(fr, edge[2], dF);
                    push_forward<T, CSB>(dF, sb + slb * L::SLOTB + ob[2], twoh, B, inv, ok, dom[2]);
                    store_B(k + 1, 2, B);
                }
            }
            if (k > 0 && k < nz - 1) {
                // ---- stage B of plane k at the pair ----
                const T* g = sB + (k & 1) * L::BSLOT + oB[0];
                T dB[2][3][3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const T* gc = g + c * BCS;
                    dB[0][0][c] = gc[1] - gc[-1];
                    dB[1][0][c] = gc[BBW + 1] - gc[BBW - 1];
                    dB[0][1][c] = Bc[1][c] - gc[-BBW];
                    dB[1][1][c] = gc[2 * BBW] - Bc[0][c];
                    dB[0][2][c] = Bp[0][c] - Bm[0][c];
                    dB[1][2][c] = Bp[1][c] - Bm[1][c];
                }
                relax_node(dB[0], dFc[0], Bc[0], a.dtg * invq[u % 2][0], in_xy0, x0[0], ok);
                relax_node(dB[1], dFc[1], Bc[1], a.dtg * invq[u % 2][1], in_xy1, x0[1], ok);
            }
            if (st0) {
                po[0] = x0[0][0];
                po[a.comp] = x0[0][1];
                po[2 * a.comp] = x0[0][2];
            }
            if (st1) {
                po[a.pitch] = x0[1][0];
                po[a.comp + a.pitch] = x0[1][1];
                po[2 * a.comp + a.pitch] = x0[1][2];
            }
            po += a.plane;
            ptx::cta_sync();
            // xi planes <= k+1 and b planes <= k+1 are dead now (own columns live in registers): refill their slots
            if (producer) refill(k + 1, k + 1);
            advance();
        }
    }
    if (!ok) atomicOr(a.flag, FLAG_NUMERIC);
}

// ----------------------------------------------------------------------------------------------- host side

constexpr int kPTY = 16, kPR = 6, kPRB = 3;

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
