// mr_sym.cuh -- the streaming step kernel of the mimetic operator (S1-S5 in one pass) and, as its DIAG
// instantiation, the grid-wide reduction S6 by the same pass.
//
// Work item = (32 x 16 xy tile, chunk of z-planes); a CTA marches along k.  Per plane the TMA unit streams the box of
// xi (halo 2 in j, 16 bytes in i) and of b (halo 1) into one of four shared-memory ring positions.  Each of the 16
// tile warps owns one row of the tile (one node per thread); four more warps own the halo-1 ring of the tile (row
// below, row above, both columns; only B is formed there) and the TMA producer.  Iteration p of a tile warp:
//     A(p):    dF, n_0 = dF_1 x dF_2, D = dF_0 . n_0, 1/D, B(p) = dF b / D (Eq. 2.1) -> shared B plane p % 4;
//              record(p) = (dF, n_0) -> Tensor Memory (own columns);
//     arrive READY[p] (one lane), bar.arrive SLOT[p];  wait READY[p-1]
//     F(p-1):  record(p-1) <- Tensor Memory;  D J = n_0 x delta_i B + n_1 x delta_j B + n_2 x (B(p) - B(p-2))  (closed
//              form of Eqs. 2.3-2.7), u = gamma J x B (Eq. 1.5), xi+ = xi + dt u -> HBM   (DIAG: the reduction of S6).
// One mbarrier phase READY[t] = "every warp has published B(t)" AND "the plane t+3 has landed": the TMA of the plane
// t+3 completes its bytes on that barrier, so a warp polls ONE barrier per plane, half an iteration after the phase
// it waits for began to fill (the wait is a poll, not a stall), and A(p+1) starts without any wait.  A(p) and F(p-1)
// belong to different planes and are independent: every warp carries the same load and nobody waits for the slowest
// warp of the current plane.  A warp that starts A(p) has seen READY[p-2] complete, i.e. every warp has finished
// F(p-4): four B planes suffice.  The producer's warp collects the bar.arrive of SLOT[p] (every warp is done with the
// xi / b planes p) and requests the plane p+4 into that ring position.
//
// The k loop is unrolled by four with the phase q = (p - first_p) % 4 a compile-time constant: every ring position,
// B plane, barrier, TMEM record and the rotating register sets (own B of the last planes: period 4, own xi: period 2)
// are named at compile time, so the loop carries no register moves and no address arithmetic (ncu of the rolled loop:
// 82 of its 356 instructions per node were moves, profiles/r1f_full.md).
#pragma once
#include <climits>
#include <type_traits>

#include "mr_generic.cuh"
#include "mr_lanes.cuh"
#include "mr_stream_common.cuh"
#include "mr_tmem.cuh"

namespace mr {

template <typename T>
struct SymLayout {
    static constexpr int NV = Lanes<T>::NV;                         // nodes per thread along i (fp64: 1, fp32: 2)
    static constexpr int TX = 32 * NV, TY = 16, R = 4, NB = 4;
    static constexpr int HXL = 16 / (int)sizeof(T), HXR = 2 * HXL;  // x halo: 16 / 32 bytes (TMA alignment), >= NV + 1 nodes
    static constexpr int BW = TX + HXL + HXR;
    static constexpr int XH = TY + 4, BH = TY + 2;
    static constexpr int CSX = BW * XH, CSB = BW * BH;
    static constexpr int round128(int bytes) { return (bytes + 127) / 128 * 128; }
    static constexpr int SLOTX = round128(3 * CSX * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr int SLOTB = round128(3 * CSB * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr uint32_t XBOX_BYTES = 3u * CSX * sizeof(T), BBOX_BYTES = 3u * CSB * sizeof(T);
    static constexpr int BBW = TX + 2 * NV, BBH = TY + 2;           // B plane: the tile and one (aligned) thread column either side
    static constexpr int BCS = BBW * BBH;
    static constexpr int BSLOT = round128(3 * BCS * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr int NTW = TY, NWARPS = TY + 4, NTHREADS = NWARPS * 32;     // tile warps + 4 ring warps
    static constexpr size_t OFF_X = 0;
    static constexpr size_t OFF_B0 = OFF_X + (size_t)R * SLOTX * sizeof(T);
    static constexpr size_t OFF_BB = OFF_B0 + (size_t)R * SLOTB * sizeof(T);
    static constexpr size_t OFF_BAR = OFF_BB + (size_t)NB * BSLOT * sizeof(T);
    static constexpr size_t BYTES = OFF_BAR + (size_t)NB * 8 + 128;
    // TMEM record of a node: chunk 0 = columns 0, 1 of dF, n_0[0], n_0[1] (8 values), chunk 1 = column 2 of dF, n_0[2]
    static constexpr int WN = (int)sizeof(typename Lanes<T>::V) / 4;     // 32-bit words per value (a double or a pair of floats)
    static constexpr int C0W = 8 * WN, C1W = 4 * WN, REC = 16 * WN; // record stride (12 values, padded to 16)
    static constexpr int TMEM_COLS = (NTW / 4) * 2 * REC;           // warps of a lane quarter x two records (plane parity)
};

template <int Q> using Phase = std::integral_constant<int, Q>;

namespace tmem {
template <> struct Words<f2> {
    static constexpr int N = 2;
    static __device__ __forceinline__ void put(uint32_t* w, f2 v) { w[0] = __float_as_uint(v.x); w[1] = __float_as_uint(v.y); }
    static __device__ __forceinline__ f2 get(const uint32_t* w) { return f2{ __uint_as_float(w[0]), __uint_as_float(w[1]) }; }
};
}  // namespace tmem
inline __device__ double Lanes<double>::rcp(double d) { return fast_rcp(d); }

// xi+ = xi + dt u  |  the reduction S6  |  out = u = gamma J x B  |  the step AND S6 of the state it starts from, in one pass
// (S6 fused into the step costs no extra HBM traffic)
enum : int { MODE_STEP = 0, MODE_DIAG = 1, MODE_RHS = 2, MODE_STEPDIAG = 3 };

// PER = false: all six faces line-tied (the hot path: no periodic logic is compiled in);  PER = true: at least one periodic axis
template <typename T, int MODE, bool PER>
__global__ void __maxnreg__(96)
k_step_sym(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_b, const T* __restrict__ in,
           T* __restrict__ out, const StreamArgs<T> a)
{
    using L = SymLayout<T>;
    using LN = Lanes<T>;
    using V = typename LN::V;                      // what a thread owns along i: one double, or a packed pair of floats
    using W32 = tmem::Words<V>;
    constexpr bool DIAG = MODE == MODE_DIAG || MODE == MODE_STEPDIAG, RHS = MODE == MODE_RHS, STORE = MODE != MODE_DIAG;
    constexpr int NV = L::NV;
    constexpr int TX = L::TX, TY = L::TY, NTW = L::NTW, BW = L::BW, CSX = L::CSX, CSB = L::CSB, BBW = L::BBW, BCS = L::BCS;
    constexpr int NW = L::NWARPS, WN = L::WN, C0W = L::C0W, C1W = L::C1W, REC = L::REC;
    static_assert(L::TMEM_COLS == 256 || L::TMEM_COLS == 128, "TMEM columns: a power of two");
    constexpr uint32_t PLANE_BYTES = L::XBOX_BYTES + L::BBOX_BYTES;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t tm_base_s;
    unsigned char* smem = smem_raw + ((128u - (ptx::smem_u32(smem_raw) & 127u)) & 127u);
    const T* sx = reinterpret_cast<const T*>(smem + L::OFF_X);
    const T* sb = reinterpret_cast<const T*>(smem + L::OFF_B0);
    T* sB = reinterpret_cast<T*>(smem + L::OFF_BB);
    const uint32_t sx_u32 = ptx::smem_u32(sx), sb_u32 = ptx::smem_u32(sb);
    const uint32_t bar = ptx::smem_u32(smem + L::OFF_BAR);          // READY[0..3]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool tilew = warp < NTW;
    const int tile = blockIdx.x % a.ntiles, chunk = blockIdx.x / a.ntiles;
    const int i0 = (tile % a.tiles_x) * TX, j0 = (tile / a.tiles_x) * TY + a.jorg;
    const int nz = a.nz;
    // a periodic axis (Eqs. 2.12-2.14) has no face: its ghost layers (two planes / rows, 16 bytes of columns either side) sit
    // in the padded arrays, B is formed on the first ghost layer like on any halo node, and every node is an inner point
    const bool perx = PER && (a.per & 1) != 0, pery = PER && (a.per & 2) != 0, perz = PER && (a.per & 4) != 0;
    const int ox = PER ? a.ox : 0, oy = PER ? a.oy : 0, oz = PER ? a.oz : 0;
    const int zface_lo = perz ? INT_MIN : 0, zface_hi = perz ? INT_MIN : nz - 1;    // the planes of the line-tied z faces
    const int zx_lo = perz ? -2 : 0, zx_hi = perz ? nz + 1 : nz - 1;               // the xi / b planes that exist
    const int k0 = chunk * a.chunk_len, k1 = min(k0 + a.chunk_len, nz);
    const int kend = PER ? min(k1, zx_hi - (perz ? 1 : 0)) : min(k1, nz - 1);   // planes k0 .. kend-1 are finished here (line-tied: nz-1 carried through)
    const int first_p = PER ? max(k0 - 1, zx_lo + (perz ? 1 : 0)) : max(k0 - 1, 0);   // B is formed on the planes first_p .. kend
    const int plast = PER ? min(kend + 1, zx_hi) : min(kend + 1, nz - 1);           // last xi / b plane this item touches
    const V twoh[3] = { LN::bc(a.twoh[0]), LN::bc(a.twoh[1]), LN::bc(a.twoh[2]) };

    const bool pwarp = warp == NW - 1, producer = pwarp && lane == 0;
    if (producer) {
        for (int s = 0; s < 4; ++s) ptx::mbar_init(bar + 8u * s, NW);           // one arrival per working warp + the producer's
        ptx::fence_mbar_init();
    }
    if (warp == 0) tmem::alloc<L::TMEM_COLS>(&tm_base_s);
    tmem::fence_before_sync();
    __syncthreads();
    tmem::fence_after_sync();
    const uint32_t tm0 = tm_base_s + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * 2 * REC);

    // The plane P = first_p + r lives in the ring position (r + 1) % 4 and completes its bytes on READY[(r + 1) % 4] in
    // the phase of the plane t = P - 3.  A plane beyond the item's last one is "delivered" empty: the producer's arrival alone.
    constexpr int BAR_SLOT = 1;                       // named barriers BAR_SLOT .. BAR_SLOT + 3
    auto request = [&](int r) {                       // producer: the plane first_p + r
        const uint32_t s = (uint32_t)(r + 1) & 3u, b = bar + 8u * s;
        const int P = first_p + r;
        if (P <= plast) {
            ptx::mbar_expect_tx(b, PLANE_BYTES);
            ptx::tma_load_4d(sx_u32 + s * (uint32_t)(L::SLOTX * sizeof(T)), &map_in, i0 - L::HXL + ox, j0 - 2 + oy, P + oz, 0, b);
            ptx::tma_load_4d(sb_u32 + s * (uint32_t)(L::SLOTB * sizeof(T)), &map_b, i0 - L::HXL + ox, j0 - 1 + oy, P + oz, 0, b);
        } else {
            ptx::mbar_arrive(b);
        }
    };
    if (pwarp) {
        if (producer)
            for (int r = 0; r < 4; ++r) request(r);
        // the producer's warp: SLOT[p] complete = every warp is done with the xi / b planes p -> the plane p + 4
        for (int u = 0; first_p + u <= kend; ++u) {
            ptx::named_sync(BAR_SLOT + (u & 3), NW * 32);
            if (producer) request(u + 4);
        }
    } else {
        // the phases of the planes first_p - 3 .. first_p - 1 publish no B: the working warps arrive right away
        __syncwarp();
        if (lane == 0) { ptx::mbar_arrive(bar + 8u); ptx::mbar_arrive(bar + 16u); ptx::mbar_arrive(bar + 24u); }
    }

    // the node of this thread: tile warps own the row `warp` of the tile; ring warps a node of the halo-1 ring (row below,
    // row above, both columns) or none (the producer's warp)
    int ti, tj;
    bool has_node = true;
    if (tilew) { ti = NV * lane; tj = warp; }
    else if (warp == NTW) { ti = NV * lane; tj = -1; }
    else if (warp == NTW + 1) { ti = NV * lane; tj = TY; }
    else if (warp == NTW + 2) { ti = (lane >> 3) & 1 ? TX : -NV; tj = (lane & 7) + 8 * (lane >> 4); }
    else { ti = 0; tj = 0; has_node = false; }
    const int gi = i0 + ti, gj = j0 + tj;                   // (first) node of this thread; the second one is gi + 1
    const T* px = sx + (tj + 2) * BW + (ti + L::HXL);       // this thread in component 0 of the ring position 0 (xi, b, B)
    const T* pb = sb + (tj + 1) * BW + (ti + L::HXL);
    T* pB = sB + (tj + 1) * BBW + (ti + NV);
    // per node e of the thread: a node or a periodic ghost (dom) / on which line-tied faces (1: i = 0, 2: i = nx-1, 4: j = 0,
    // 8: j = ny-1) / an inner point in xy / a node this thread stores (st)
    bool dom[NV], in_xy[NV], st[NV];
    unsigned edge = 0u;                                     // bits of the node e shifted by 8 e (bits 16, 32 of `special`: the k faces)
    bool any_st = false;
    const bool row_real = gj >= 0 && gj < a.ny;
    const bool row_in = row_real || (gj >= -oy && gj < a.ny + oy);
#pragma unroll
    for (int e = 0; e < NV; ++e) {
        const int g = gi + e;
        if constexpr (PER) {
            const bool real = has_node && row_real && g >= 0 && g < a.nx;
            dom[e] = has_node && row_in && g >= -ox && g < a.nx + ox;
            in_xy[e] = real && (perx || (g > 0 && g < a.nx - 1)) && (pery || (gj > 0 && gj < a.ny - 1));
            st[e] = tilew && real;
            if (real) edge |= ((g == 0 && !perx ? 1u : 0u) | (g == a.nx - 1 && !perx ? 2u : 0u) | (gj == 0 && !pery ? 4u : 0u) |
                               (gj == a.ny - 1 && !pery ? 8u : 0u)) << (8 * e);
        } else {
            dom[e] = has_node && row_real && g >= 0 && g < a.nx;
            in_xy[e] = g > 0 && g < a.nx - 1 && gj > 0 && gj < a.ny - 1;
            st[e] = tilew && dom[e];
            if (dom[e]) edge |= ((g == 0 ? 1u : 0u) | (g == a.nx - 1 ? 2u : 0u) | (gj == 0 ? 4u : 0u) | (gj == a.ny - 1 ? 8u : 0u)) << (8 * e);
        }
        any_st = any_st || st[e];
    }

    bool ok = true;
    V xh[2][3], Bh[4][3], sh[2];                             // own xi(p), xi(p-1); own B(p) .. B(p-3); dt gamma / D of p, p-1
    // a value of this thread's node(s) straight from global memory (0 outside the grid)
    auto from_global = [&](const T* f, long long o) {
        V v = LN::bc(T(0));
#pragma unroll
        for (int e = 0; e < NV; ++e)
            if (dom[e]) LN::set(v, e, f[o + e]);
        return v;
    };
    {
        // own xi of the plane below the first one (for the first k-difference) straight from global memory
        const long long o = (long long)(first_p - 1) * a.plane + (long long)gj * a.pitch + gi;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            xh[0][c] = LN::bc(T(0));
            xh[1][c] = (PER ? first_p > zx_lo : first_p > 0) ? from_global(in + c * a.comp, o) : LN::bc(T(0)); // phase 0 reads xi(first_p - 1) from xh[1]
#pragma unroll
            for (int q = 0; q < 4; ++q) Bh[q][c] = LN::bc(T(0));
        }
    }
    sh[0] = sh[1] = LN::bc(T(0));
    if (tilew) {         // the first F reads the own B of the plane first_p - 1 (never formed) from the B plane 3: a finite stand-in
#pragma unroll
        for (int c = 0; c < 3; ++c) LN::st(pB + 3 * L::BSLOT + c * BCS, LN::bc(T(0)));
    }
    T* po = out + (long long)first_p * a.plane + (long long)gj * a.pitch + gi;     // plane t = p-1 of the first F
    // store the thread's node(s) that lie inside the grid
    auto store_nodes = [&](T* q, V v) {
        if (NV == 2 && st[0] && st[NV - 1]) { LN::st(q, v); return; }
#pragma unroll
        for (int e = 0; e < NV; ++e)
            if (st[e]) q[e] = LN::get(v, e);
    };
    DiagPartial acc = { 0.0, 0.0, 0.0, INFINITY };          // DIAG: this thread's partial
    auto diag_node = [&](int k, const V(&c0)[3], const V(&n0)[3], const V(&B)[3], const V(&uu)[3]) {
#pragma unroll
        for (int e = 0; e < NV; ++e) {
            if (!st[e]) continue;
            const double zxy = ((edge >> (8 * e)) & 3u ? 0.5 : 1.0) * ((edge >> (8 * e)) & 12u ? 0.5 : 1.0);          // Eq. 3.13
            double D = 0.0, b2 = 0.0, u2 = 0.0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                D += (double)LN::get(c0[c], e) * (double)LN::get(n0[c], e);
                b2 += (double)LN::get(B[c], e) * (double)LN::get(B[c], e);
                u2 += (double)LN::get(uu[c], e) * (double)LN::get(uu[c], e);
            }
            const bool kface = k == zface_lo || k == zface_hi;
            DiagPartial v = { zxy * (kface ? 0.5 : 1.0) * b2 * D, 0.0, 0.0, D };
            if (in_xy[e] && !kface) {
                const double fm = sqrt(u2) / D;
                v.fmax = fm;
                v.xi = fm / b2;
            }
            diag_combine(acc, v);
        }
    };

    if (!pwarp) {        // the planes first_p, first_p + 1 and, for the one-sided difference on the bottom face, 2
        ptx::mbar_wait(bar + 8u, 0u);
        ptx::mbar_wait(bar + 16u, 0u);
        if (PER ? first_p == zface_lo : first_p == 0) ptx::mbar_wait(bar + 24u, 0u);
    }
    int p = first_p;
    uint32_t gpar = 0u;                                      // parity of the group of four planes
    auto body = [&](auto phase, auto tile_c) {
        constexpr int Q = decltype(phase)::value;
        constexpr bool TILE = decltype(tile_c)::value;
        constexpr int S0 = (Q + 1) & 3, S1 = (Q + 2) & 3, S2 = (Q + 3) & 3;      // ring positions of the planes p, p+1, p+2 (= p-2)
        constexpr int QM1 = (Q + 3) & 3, QM2 = (Q + 2) & 3;                      // B planes / own B of p-1, p-2
        V(&x1)[3] = xh[Q & 1];
        const V(&xp)[3] = xh[(Q + 1) & 1];
        V(&Bp)[3] = Bh[Q];
        const bool fin = TILE && p > first_p;
        // ---------------- A(p): push-forward of the plane p at the own node(s) ----------------
        const bool work = TILE || (has_node && p < kend);
        const T* fr = px + S0 * L::SLOTX;
        if (work) {
            const T* f2p = px + S1 * L::SLOTX;
            V dF[3][3], bq[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                x1[c] = LN::ld(fr + c * CSX);
                dF[c][0] = LN::di(fr + c * CSX, x1[c]);
                dF[c][1] = LN::ld(fr + c * CSX + BW) - LN::ld(fr + c * CSX - BW);
                dF[c][2] = LN::ld(f2p + c * CSX) - xp[c];
                bq[c] = LN::ld(pb + S0 * L::SLOTB + c * CSB);
            }
            const unsigned special = PER ? (edge | (p == zface_lo ? 16u : 0u) | (p == zface_hi ? 32u : 0u))
                                         : (edge | (p == 0 ? 16u : 0u) | (p == nz - 1 ? 32u : 0u));
            if (special) {
                if (special & 16u) {            // bottom face: -3 x(0) + 4 x(1) - x(2)
                    const T* f3 = px + S2 * L::SLOTX;
#pragma unroll
                    for (int c = 0; c < 3; ++c) dF[c][2] = LN::bc(T(4)) * LN::ld(f2p + c * CSX) - LN::bc(T(3)) * x1[c] - LN::ld(f3 + c * CSX);
                }
                if (special & 32u) {            // top face: 3 x(nz-1) - 4 x(nz-2) + x(nz-3); the own xi of the plane nz-3 comes from
                                                // global memory (once per column; a last chunk of one plane never loads that plane)
                    const long long o3 = (long long)(nz - 3) * a.plane + (long long)gj * a.pitch + gi;
#pragma unroll
                    for (int c = 0; c < 3; ++c) dF[c][2] = LN::bc(T(3)) * x1[c] - LN::bc(T(4)) * xp[c] + from_global(in + c * a.comp, o3);
                }
                // one-sided in-plane differences of a node on an x / y face (reading Q3), node by node
#pragma unroll
                for (int e = 0; e < NV; ++e) {
                    const unsigned eb = (edge >> (8 * e)) & 15u;
                    if (!eb) continue;
                    T d1[3][3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) { d1[c][0] = LN::get(dF[c][0], e); d1[c][1] = LN::get(dF[c][1], e); d1[c][2] = T(0); }
                    face_fix<T, BW, CSX>(fr + e, eb, d1);
#pragma unroll
                    for (int c = 0; c < 3; ++c) { LN::set(dF[c][0], e, d1[c][0]); LN::set(dF[c][1], e, d1[c][1]); }
                }
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) dF[c][c] += twoh[c];
            V n0[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
                n0[c] = fma(dF[c1][1], dF[c2][2], -(dF[c2][1] * dF[c1][2]));
            }
            const V D = fma(dF[0][0], n0[0], fma(dF[1][0], n0[1], dF[2][0] * n0[2]));
#pragma unroll
            for (int e = 0; e < NV; ++e) ok = ok && (positive_finite(LN::get(D, e)) || !dom[e]);
            const V inv = LN::rcp(D);
            // dF b first, the division last: the nine products do not wait for the reciprocal's Newton chain
#pragma unroll
            for (int c = 0; c < 3; ++c) Bp[c] = fma(dF[c][0], bq[0], fma(dF[c][1], bq[1], dF[c][2] * bq[2])) * inv;
            T* d = pB + Q * L::BSLOT;
            LN::st(d, Bp[0]);
            LN::st(d + BCS, Bp[1]);
            LN::st(d + 2 * BCS, Bp[2]);
            if constexpr (TILE) {
                V sn = LN::bc(a.dtg) * inv;
                const bool kin = PER ? (p != zface_lo && p != zface_hi) : (p > 0 && p < nz - 1);
#pragma unroll
                for (int e = 0; e < NV; ++e)
                    if (!(kin && in_xy[e])) LN::set(sn, e, T(0));
                sh[Q & 1] = sn;
                uint32_t v0[C0W], v1[C1W];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    W32::put(v0 + c * WN, dF[c][0]);
                    W32::put(v0 + (3 + c) * WN, dF[c][1]);
                    W32::put(v1 + c * WN, dF[c][2]);
                }
                W32::put(v0 + 6 * WN, n0[0]);
                W32::put(v0 + 7 * WN, n0[1]);
                W32::put(v1 + 3 * WN, n0[2]);
                tmem::st<C0W>(tm0 + (Q & 1) * REC, v0);
                tmem::st<C1W>(tm0 + (Q & 1) * REC + C0W, v1);
            }
        } else if (!TILE && has_node) {
#pragma unroll
            for (int c = 0; c < 3; ++c) x1[c] = LN::ld(fr + c * CSX);
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar + 8u * Q);                   // this warp's part of B(p) is in shared memory
        ptx::named_arrive(BAR_SLOT + Q, NW * 32);                        // ... and it is done with the xi / b planes p
        ptx::mbar_wait(bar + 8u * QM1, Q >= 2 ? gpar ^ 1u : gpar);      // B(p-1) is published, the plane p+2 has landed
        // ---------------- F(p-1): finish the plane t = p-1 ----------------
        // (a chunk that starts inside the grid runs F(k0 - 1) once without storing it: the plane belongs to the chunk below)
        if (fin) {
            uint32_t w0[C0W], w1[C1W];
            tmem::wait_st();                                 // record(p-1) was stored an iteration ago
            tmem::ld<C0W>(tm0 + ((Q + 1) & 1) * REC, w0);
            tmem::ld<C1W>(tm0 + ((Q + 1) & 1) * REC + C0W, w1);
            const T* g = pB + QM1 * L::BSLOT;
            const V(&Bc)[3] = Bh[QM1];
            // own B(p-2) back from its shared plane (intact until A(p+2)): cheaper than six more registers carried
            const T* gm = pB + QM2 * L::BSLOT;
            V dBi[3], dBj[3], dBk[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const T* gc = g + c * BCS;
                dBi[c] = LN::di(gc, Bc[c]);
                dBj[c] = LN::ld(gc + BBW) - LN::ld(gc - BBW);
                dBk[c] = Bp[c] - LN::ld(gm + c * BCS);
            }
            tmem::wait_ld(w0);
            tmem::wait_ld(w1);
            V c0[3], c1[3], c2[3], n0[3], n1[3], n2[3], DJ[3], uu[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                c0[c] = W32::get(w0 + c * WN);
                c1[c] = W32::get(w0 + (3 + c) * WN);
                c2[c] = W32::get(w1 + c * WN);
            }
            n0[0] = W32::get(w0 + 6 * WN);
            n0[1] = W32::get(w0 + 7 * WN);
            n0[2] = W32::get(w1 + 3 * WN);
            cross_set(c2, c0, n1);                  // n_1 = dF_2 x dF_0,  n_2 = dF_0 x dF_1  (Eqs. 2.5/2.6)
            cross_set(c0, c1, n2);
            cross_set(n0, dBi, DJ);
            cross_acc(n1, dBj, DJ);
            cross_acc(n2, dBk, DJ);
            cross_set(DJ, Bc, uu);
            if constexpr (DIAG) {
                if (p > k0) diag_node(p - 1, c0, n0, Bc, uu);
            }
            if constexpr (STORE) {
                const V s = sh[(Q + 1) & 1];
                V x[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) x[c] = RHS ? s * uu[c] : fma(s, uu[c], xp[c]);
                const V xs = x[0] + x[1] + x[2];
#pragma unroll
                for (int e = 0; e < NV; ++e) ok = ok && is_finite(LN::get(xs, e));
                if (any_st && p > k0) {
                    store_nodes(po, x[0]);
                    store_nodes(po + a.comp, x[1]);
                    store_nodes(po + 2 * a.comp, x[2]);
                }
                po += a.plane;
            }
        }
    };
    auto run = [&](auto tile_c) {
#pragma unroll 1
        for (;;) {
            body(Phase<0>{}, tile_c);
            if (++p > kend) break;
            body(Phase<1>{}, tile_c);
            if (++p > kend) break;
            body(Phase<2>{}, tile_c);
            if (++p > kend) break;
            body(Phase<3>{}, tile_c);
            if (++p > kend) break;
            gpar ^= 1u;
        }
    };
    if (tilew) run(std::true_type{});
    else if (!pwarp) run(std::false_type{});

    if (k1 == nz && tilew && !perz) {   // the top plane (line-tied) is carried through / enters the energy sum
        const int ql = (nz - 1 - first_p) & 3;
        if constexpr (DIAG) {
            uint32_t w0[C0W], w1[C1W];
            tmem::wait_st();                                // (tcgen05 operations are warp-wide: no per-thread predicate here)
            tmem::ld<C0W>(tm0 + (ql & 1) * REC, w0);
            tmem::ld<C1W>(tm0 + (ql & 1) * REC + C0W, w1);
            tmem::wait_ld(w0);
            tmem::wait_ld(w1);
            V c0[3], n0[3], Bt[3];
            const V zero[3] = { LN::bc(T(0)), LN::bc(T(0)), LN::bc(T(0)) };
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                c0[c] = W32::get(w0 + c * WN);
                Bt[c] = ql == 0 ? Bh[0][c] : ql == 1 ? Bh[1][c] : ql == 2 ? Bh[2][c] : Bh[3][c];
            }
            n0[0] = W32::get(w0 + 6 * WN);
            n0[1] = W32::get(w0 + 7 * WN);
            n0[2] = W32::get(w1 + 3 * WN);
            diag_node(nz - 1, c0, n0, Bt, zero);
        }
        if (STORE && any_st) {
            T* pl = out + (long long)(nz - 1) * a.plane + (long long)gj * a.pitch + gi;
#pragma unroll
            for (int c = 0; c < 3; ++c) store_nodes(pl + c * a.comp, RHS ? LN::bc(T(0)) : (ql & 1) ? xh[1][c] : xh[0][c]);
        }
    }
    if (!ok) atomicOr(a.flag, FLAG_NUMERIC);
    tmem::fence_before_sync();
    __syncthreads();                                        // the pipeline is drained: shared memory is free
    if constexpr (DIAG) {
        // fixed-order reduction: lanes by a shuffle tree, then the tile warps in index order; one partial per CTA
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            DiagPartial w;
            w.e = __shfl_down_sync(0xffffffffu, acc.e, o);
            w.fmax = __shfl_down_sync(0xffffffffu, acc.fmax, o);
            w.xi = __shfl_down_sync(0xffffffffu, acc.xi, o);
            w.dmin = __shfl_down_sync(0xffffffffu, acc.dmin, o);
            diag_combine(acc, w);
        }
        DiagPartial* shp = reinterpret_cast<DiagPartial*>(smem);
        if (tilew && lane == 0) shp[warp] = acc;
        __syncthreads();
        if (tid == 0) {
            DiagPartial v = shp[0];
            for (int w = 1; w < NTW; ++w) diag_combine(v, shp[w]);
            (STORE ? static_cast<DiagPartial*>(a.partials) : reinterpret_cast<DiagPartial*>(out))[blockIdx.x] = v;
        }
    }
    if (warp == 0) tmem::dealloc<L::TMEM_COLS>(tm_base_s);
}

// ----------------------------------------------------------------------------------------------- host side

template <typename T>
using SymKernel = void (*)(const CUtensorMap, const CUtensorMap, const T*, T*, const StreamArgs<T>);

// the instantiation for a mode and for "some axis is periodic"
template <typename T>
inline SymKernel<T> sym_kernel(int mode, bool per)
{
    if (per)
        return mode == MODE_STEP ? k_step_sym<T, MODE_STEP, true> : mode == MODE_DIAG ? k_step_sym<T, MODE_DIAG, true>
             : mode == MODE_RHS ? k_step_sym<T, MODE_RHS, true> : k_step_sym<T, MODE_STEPDIAG, true>;
    return mode == MODE_STEP ? k_step_sym<T, MODE_STEP, false> : mode == MODE_DIAG ? k_step_sym<T, MODE_DIAG, false>
         : mode == MODE_RHS ? k_step_sym<T, MODE_RHS, false> : k_step_sym<T, MODE_STEPDIAG, false>;
}

inline bool build_sym_plan(StreamPlan* p, const StreamGeom& g, bool f64, void* xi0, void* xi1, void* b, int sm_count,
                           std::string* why)
{
    using Ld = SymLayout<double>;
    using Lf = SymLayout<float>;
    p->usable = false;
    p->f64 = f64;
    p->g = g;
    p->xi[0] = node_base(xi0, g, f64);      // xi0, xi1, b: the starts of the padded arrays (what the tensor maps span)
    p->xi[1] = node_base(xi1, g, f64);
    p->b = node_base(b, g, f64);
    p->name = f64 ? "sym_tmem_f64" : "sym_tmem_f32";
    const int bw = f64 ? Ld::BW : Lf::BW;
    if (!encode_map(&p->map_xi[0], f64, xi0, g, bw, Ld::TY + 4) || !encode_map(&p->map_xi[1], f64, xi1, g, bw, Ld::TY + 4) ||
        !encode_map(&p->map_b, f64, b, g, bw, Ld::TY + 2)) {
        *why = "cuTensorMapEncodeTiled failed";
        return false;
    }
    p->smem_bytes = f64 ? Ld::BYTES : Lf::BYTES;
    cudaError_t e = cudaSuccess;
    const int sb = (int)p->smem_bytes;
    const bool per = g.per[0] || g.per[1] || g.per[2];
    const void* fn[4];
    for (int m = 0; m < 4; ++m) fn[m] = f64 ? (const void*)sym_kernel<double>(m, per) : (const void*)sym_kernel<float>(m, per);
    for (int m = 0; m < 4 && e == cudaSuccess; ++m) e = cudaFuncSetAttribute(fn[m], cudaFuncAttributeMaxDynamicSharedMemorySize, sb);
    if (e != cudaSuccess) {
        *why = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e);
        return false;
    }
    choose_tilings(p, f64 ? Ld::TX : Lf::TX, Ld::TY, true, sm_count);
    p->usable = true;
    return true;
}

// tensor map of the adaptive integrator's stage buffer (same box as the state buffers)
inline bool sym_bind_stage(StreamPlan* p, void* xs)
{
    const int bw = p->f64 ? SymLayout<double>::BW : SymLayout<float>::BW;
    if (!encode_map(&p->map_xi[2], p->f64, xs, p->g, bw, SymLayout<double>::TY + 4)) return false;
    p->xi[2] = node_base(xs, p->g, p->f64);
    return true;
}

// One step (rhs = false: out = xi + dtg J x B) or one right-hand side (rhs = true: out = dtg J x B, dtg = gamma) of the
// state in the plan's buffer `cur` (0, 1: the state buffers; 2: the stage buffer) into the padded field `out`.
template <typename T>
inline cudaError_t launch_sym_step(const StreamPlan& p, int cur, T dtg, int* flag, cudaStream_t stream, bool rhs = false, void* out = nullptr)
{
    const StreamArgs<T> a = stream_args<T>(p, p.step, dtg, flag);
    T* o = static_cast<T*>(out ? out : p.xi[1 - cur]);
    sym_kernel<T>(rhs ? MODE_RHS : MODE_STEP, a.per != 0)<<<a.ntiles * p.step.nchunks, SymLayout<T>::NTHREADS, p.smem_bytes, stream>>>(
        p.map_xi[cur], p.map_b, static_cast<const T*>(p.xi[cur]), o, a);
    return cudaGetLastError();
}

// One step of the state in buffer `cur` into the other state buffer AND S6 of the state it starts from: one DiagPartial per CTA
// into `partials` (the tiling in which every node is a tile node, like launch_sym_diag: same partials, same order, same sums)
template <typename T>
inline cudaError_t launch_sym_stepdiag(const StreamPlan& p, int cur, T dtg, DiagPartial* partials, int* nblocks, int* flag, cudaStream_t stream)
{
    StreamArgs<T> a = stream_args<T>(p, p.all, dtg, flag);
    a.partials = partials;
    *nblocks = a.ntiles * p.all.nchunks;
    sym_kernel<T>(MODE_STEPDIAG, a.per != 0)<<<*nblocks, SymLayout<T>::NTHREADS, p.smem_bytes, stream>>>(
        p.map_xi[cur], p.map_b, static_cast<const T*>(p.xi[cur]), static_cast<T*>(p.xi[1 - cur]), a);
    return cudaGetLastError();
}

// S6 of the state in buffer `cur` by the same pass (no update, no store): one DiagPartial per CTA into `partials`
template <typename T>
inline cudaError_t launch_sym_diag(const StreamPlan& p, int cur, DiagPartial* partials, int* nblocks, int* flag, cudaStream_t stream)
{
    const StreamArgs<T> a = stream_args<T>(p, p.all, (T)0, flag);
    *nblocks = a.ntiles * p.all.nchunks;
    sym_kernel<T>(MODE_DIAG, a.per != 0)<<<*nblocks, SymLayout<T>::NTHREADS, p.smem_bytes, stream>>>(
        p.map_xi[cur], p.map_b, static_cast<const T*>(p.xi[cur]), reinterpret_cast<T*>(partials), a);
    return cudaGetLastError();
}

}  // namespace mr
