// mr_duo.cuh -- the warp-specialised streaming step kernel for the mimetic operator (S1-S5 in one pass).
//
// ncu of the register-paired kernel (profiles/r1c_full.md): one CTA of 8 warps per SM, 255 registers, every pipe
// below 45 % and the warps waiting on each other's latencies -- the kernel is bound by the number of nodes the
// register file can keep in flight, not by HBM (the same TMA ring with the arithmetic stubbed out runs at 96 % of the
// measured copy bandwidth; the halo-1 ring alone cost 0.14 of its 0.64 ms because it sat on the critical path of half
// the warps).  This kernel splits the work of a node between warps that hand the node's state over through Tensor
// Memory (mr_tmem.cuh), so that 20 warps of 96 registers share the SM and the roles run out of step:
//
//   A-warps (0..TY/2-1, lane = i, rows 2a and 2a+1)
//       plane p:  dF from the xi ring in shared memory (TMA; the j-differences inside the pair and the k-differences
//                 from registers), n_0 = dF_1 x dF_2 (area vector, Eqs. 2.5/2.6), D = dF_0 . n_0, 1/D,
//                 B(p) = dF b / D (Eq. 2.1) -> shared B plane p % NB;   record(p) = dF, n_0, s = dt gamma / D, own xi(p)
//                 (16 values) -> TMEM buffer p % NB (tcgen05.st);   bar.arrive FULL[p % NB]
//   R-warps (TY..TY+3: ring row below, ring row above, both ring columns, TMA producer)
//       plane p:  B(p) of the tile's halo-1 ring, one node per thread -> shared B plane;  bar.arrive FULL[p % NB];
//                 the producer's warp collects the slot-release arrivals of the A- and R-warps and refills the rings
//   F-warps (TY/2..TY-1, same lanes and rows as the A-warps: the partner warp sits in the same TMEM lane quarter)
//       plane t:  record(t) (tcgen05.ld), n_1 = dF_2 x dF_0, n_2 = dF_0 x dF_1;  bar.sync FULL[(t+1) % NB];
//                 D J = n_0 x delta_i B + n_1 x delta_j B + n_2 x (B(t+1) - B(t-1))  (closed form of Eqs. 2.3-2.7) from
//                 the shared B plane t and the own B(t-1), B(t), B(t+1);  u = gamma J x B (Eq. 1.5);
//                 xi+ = xi + dt u -> HBM   (DIAG: the reduction of S6 instead);   bar.arrive FREE[t % NB]
// The A- and R-warps wait on FREE[p % NB] before they overwrite a buffer, so they run up to NB-1 planes ahead of the
// F-warps; the xi / b rings are touched by the A- and R-warps only and recycled behind barriers of their own.
// B, J, u never touch HBM: the algorithmic traffic is read xi + read b + write xi+ = 9 elements per node.
#pragma once
#include <type_traits>

#include "mr_generic.cuh"
#include "mr_stream_common.cuh"
#include "mr_tmem.cuh"

namespace mr {

template <typename T, int TY, int R, int RB, int NB>
struct DuoLayout {
    static_assert(TY % 2 == 0 && TY >= 8 && TY <= 16 && R >= 4 && RB >= 2 && NB >= 3, "tile / ring sizes");
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
    static constexpr int NAW = TY / 2, NWARPS = 2 * NAW + 4, NTHREADS = NWARPS * 32;   // A-, F- and four R-warps
    static constexpr size_t OFF_X = 0;
    static constexpr size_t OFF_B0 = OFF_X + (size_t)R * SLOTX * sizeof(T);
    static constexpr size_t OFF_BB = OFF_B0 + (size_t)RB * SLOTB * sizeof(T);
    static constexpr size_t OFF_BAR = OFF_BB + (size_t)NB * BSLOT * sizeof(T);
    static constexpr size_t BYTES = OFF_BAR + (size_t)(R + RB) * 8 + 128;   // +128: base alignment slack
};

template <typename T, int TY, int R, int RB, int NB, bool DIAG>
#ifndef MR_DUO_MAXREG
#define MR_DUO_MAXREG 96
#endif
// 20 warps x 32 x 96 registers = 60 K of the SM's 64 K
__global__ void __maxnreg__(MR_DUO_MAXREG)
k_step_duo(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_b, T* __restrict__ out,
           const StreamArgs<T> a)
{
    using L = DuoLayout<T, TY, R, RB, NB>;
    using W32 = tmem::Words<T>;
    constexpr int TX = L::TX, NAW = L::NAW, BW = L::BW, CSX = L::CSX, CSB = L::CSB, BBW = L::BBW, BCS = L::BCS;
    constexpr int NTH = L::NTHREADS;
    constexpr int CW = 8 * W32::N;                  // words per TMEM chunk (8 values)
    constexpr int REC = 2 * CW;                     // words per node record: {n0, n1, x0, x1 | n2, s, x2, -, -, -}
    constexpr int PAIRCOLS = 2 * REC * NB;          // columns of one A/F warp pair
    static_assert(((NAW + 3) / 4) * PAIRCOLS <= 512, "TMEM columns");
    // named barriers, one of each kind per buffer: an A-warp may run NB-1 planes ahead of the slowest one
    constexpr int BAR_FULL = 1, BAR_FREE = 1 + NB, BAR_A = 1 + 2 * NB;
    static_assert(1 + 3 * NB <= 16, "named barriers");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t tm_base_s;
    unsigned char* smem = smem_raw + ((128u - (ptx::smem_u32(smem_raw) & 127u)) & 127u);
    const T* sx = reinterpret_cast<const T*>(smem + L::OFF_X);
    const T* sb = reinterpret_cast<const T*>(smem + L::OFF_B0);
    T* sB = reinterpret_cast<T*>(smem + L::OFF_BB);
    const uint32_t sx_u32 = ptx::smem_u32(sx), sb_u32 = ptx::smem_u32(sb);
    const uint32_t bar_x = ptx::smem_u32(smem + L::OFF_BAR), bar_b = bar_x + 8u * R;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NAG = NAW + 4;                    // warps of the stage-A group (A-warps and R-warps)
    const bool isA = warp < NAW, isF = warp >= NAW && warp < 2 * NAW;
    const int widx = isA ? warp : isF ? warp - NAW : 0;       // the A-warp and the F-warp of the same rows share widx
    const int tile = blockIdx.x % a.ntiles, chunk = blockIdx.x / a.ntiles;
    const int i0 = (tile % a.tiles_x) * TX, j0 = (tile / a.tiles_x) * TY;
    const int nz = a.nz;
    const int k0 = chunk * a.chunk_len, k1 = min(k0 + a.chunk_len, nz);
    const int kend = min(k1, nz - 1);               // planes k0 .. kend-1 are finished here (and nz-1 carried through)
    const int first_p = max(k0 - 1, 0);             // the A-warps form B of the planes first_p .. kend
    const int pfirst = max(first_p - 1, 0), plast = min(kend + 1, nz - 1);   // xi planes this item touches
    const int bfirst = first_p, blast = kend;                                // b planes

    const bool producer = tid == (2 * NAW + 3) * 32;
    if (producer) {
        for (int s = 0; s < R + RB; ++s) ptx::mbar_init(bar_x + 8u * s, 1);
        ptx::fence_mbar_init();
    }
    if (warp == 0) tmem::alloc<512>(&tm_base_s);
    tmem::fence_before_sync();
    __syncthreads();
    tmem::fence_after_sync();
    const uint32_t tm0 = tm_base_s + ((uint32_t)(32 * (widx & 3)) << 16) + (uint32_t)((widx >> 2) * PAIRCOLS);
    auto rec_addr = [&](int buf, int n, int c) -> uint32_t { return tm0 + (uint32_t)((buf * 2 + n) * REC + c * CW); };

    const int gi = i0 + lane, gja = j0 + 2 * widx;
    const bool st[2] = { gi < a.nx && gja < a.ny, gi < a.nx && gja + 1 < a.ny };
    const int oB0 = (2 * widx + 1) * BBW + (lane + 1);      // the pair's node 0 inside a shared B plane
    bool ok = true;
    DiagPartial diag_acc = { 0.0, 0.0, 0.0, INFINITY };   // DIAG: the F-warp's partial (valid in lane 0)

    if (!isF) {
        // ======================== A-warps (tile pairs) and R-warps (halo-1 ring): stage A ========================
        const T twoh[3] = { a.twoh[0], a.twoh[1], a.twoh[2] };
        auto load_x = [&](int p) {
            const uint32_t s = (uint32_t)((p - pfirst) % R);
            ptx::mbar_expect_tx(bar_x + 8u * s, L::XBOX_BYTES);
            ptx::tma_load_4d(sx_u32 + s * (uint32_t)(L::SLOTX * sizeof(T)), &map_in, i0 - L::HXL, j0 - 2, p, 0, bar_x + 8u * s);
        };
        auto load_b = [&](int p) {
            const uint32_t s = (uint32_t)((p - bfirst) % RB);
            ptx::mbar_expect_tx(bar_b + 8u * s, L::BBOX_BYTES);
            ptx::tma_load_4d(sb_u32 + s * (uint32_t)(L::SLOTB * sizeof(T)), &map_b, i0 - L::HXL, j0 - 1, p, 0, bar_b + 8u * s);
        };
        int next_x = pfirst, next_b = bfirst;                      // next planes to request (producer only)
        auto refill = [&](int upto_x, int upto_b) {
            for (const int last = min(upto_x, plast); next_x <= last; ++next_x) load_x(next_x);
            for (const int last = min(upto_b, blast); next_b <= last; ++next_b) load_b(next_b);
        };
        if (producer) refill(pfirst + R - 1, bfirst + RB - 1);
        auto wait_x = [&](int p) { const int q = p - pfirst; ptx::mbar_wait(bar_x + 8u * (uint32_t)(q % R), (uint32_t)((q / R) & 1)); };
        auto xplane = [&](int p) -> const T* { return sx + ((p - pfirst) % R) * L::SLOTX; };
        const bool plain = i0 > 0 && i0 + TX <= a.nx - 2 && j0 > 0 && j0 + TY <= a.ny - 2;
        for (int p = pfirst; p <= min(first_p + 1, plast); ++p) wait_x(p);
        if (first_p == 0 && plast >= 2) wait_x(2);          // the one-sided difference on the bottom face

      if (isA) {
        const int ox0 = (2 * warp + 2) * BW + (lane + L::HXL), ob0 = (2 * warp + 1) * BW + (lane + L::HXL);
        unsigned edge[2];
        bool dom[2];
#pragma unroll
        for (int n = 0; n < 2; ++n) {
            const int gj = gja + n;
            dom[n] = gi < a.nx && gj < a.ny;
            edge[n] = !dom[n] ? 0u : (gi == 0 ? 1u : 0u) | (gi == a.nx - 1 ? 2u : 0u) | (gj == 0 ? 4u : 0u) | (gj == a.ny - 1 ? 8u : 0u);
        }
        const bool in_x = gi > 0 && gi < a.nx - 1;
        const bool in_xy[2] = { in_x && gja > 0 && gja < a.ny - 1, in_x && gja + 1 < a.ny - 1 };
        T xc[2][3];                                         // own xi(p-1) of the pair
#pragma unroll
        for (int c = 0; c < 3; ++c) { xc[0][c] = T(0); xc[1][c] = T(0); }
        if (first_p > 0) {
            const T* f = xplane(first_p - 1);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                xc[0][c] = f[ox0 + c * CSX];
                xc[1][c] = f[ox0 + c * CSX + BW];
            }
        }
        auto runA = [&](auto plain_c) {
            constexpr bool PLAIN = decltype(plain_c)::value;
            int buf = first_p % NB;
            // running ring positions: xi planes p-2 .. p+2 (slots sm2, sm1, s0, s1, s2), parity of the plane p+1, b plane p
            int s0 = (first_p - pfirst) % R, s1 = (s0 + 1) % R, s2 = (s0 + 2) % R, sm1 = (s0 + R - 1) % R, sm2 = (s0 + R - 2) % R;
            uint32_t par1 = (uint32_t)(((first_p + 1 - pfirst) / R) & 1);
            int sb0 = 0;
            uint32_t parb = 0u;
#pragma unroll 1
            for (int p = first_p; p <= kend; ++p) {
                const T* f1 = sx + s0 * L::SLOTX;                     // xi plane p
                const T* f2 = sx + s1 * L::SLOTX;                     // xi plane p+1
                if (p + 1 <= plast) ptx::mbar_wait(bar_x + 8u * (uint32_t)s1, par1);
                ptx::mbar_wait(bar_b + 8u * (uint32_t)sb0, parb);
                const T* bs = sb + sb0 * L::SLOTB;
                const bool inner_k = p > 0 && p < nz - 1;
                T x1[2][3], dF[2][3][3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    x1[0][c] = f1[ox0 + c * CSX];
                    x1[1][c] = f1[ox0 + c * CSX + BW];
                }
                if (p == 0) {                   // bottom face: -3 x(0) + 4 x(1) - x(2)
                    const T* f3 = sx + s2 * L::SLOTX;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        dF[0][c][2] = T(4) * f2[ox0 + c * CSX] - T(3) * x1[0][c] - f3[ox0 + c * CSX];
                        dF[1][c][2] = T(4) * f2[ox0 + c * CSX + BW] - T(3) * x1[1][c] - f3[ox0 + c * CSX + BW];
                    }
                } else if (p + 1 <= nz - 1) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        dF[0][c][2] = f2[ox0 + c * CSX] - xc[0][c];
                        dF[1][c][2] = f2[ox0 + c * CSX + BW] - xc[1][c];
                    }
                } else {                        // top face: 3 x(nz-1) - 4 x(nz-2) + x(nz-3); plane nz-3 is still in its slot
                    const T* fm = sx + sm2 * L::SLOTX;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        dF[0][c][2] = T(3) * x1[0][c] - T(4) * xc[0][c] + fm[ox0 + c * CSX];
                        dF[1][c][2] = T(3) * x1[1][c] - T(4) * xc[1][c] + fm[ox0 + c * CSX + BW];
                    }
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const T* fc = f1 + ox0 + c * CSX;
                    dF[0][c][0] = fc[1] - fc[-1];
                    dF[1][c][0] = fc[BW + 1] - fc[BW - 1];
                    dF[0][c][1] = x1[1][c] - fc[-BW];
                    dF[1][c][1] = fc[2 * BW] - x1[0][c];
                }
                if (!PLAIN) {
                    if (edge[0]) face_fix<T, BW, CSX>(f1 + ox0, edge[0], dF[0]);
                    if (edge[1]) face_fix<T, BW, CSX>(f1 + ox0 + BW, edge[1], dF[1]);
                }
                // the buffer p % NB (shared B plane and TMEM records) must have been read by the F-warps
                if (p >= first_p + NB) {
                    ptx::named_sync(BAR_FREE + buf, NTH);
                    tmem::fence_after_sync();
                }
                T* Bd = sB + buf * L::BSLOT;
#pragma unroll
                for (int n = 0; n < 2; ++n) {
                    T n0[3], Bn[3], inv;
                    duo_push<T, CSB>(dF[n], bs + ob0 + n * BW, twoh, n0, Bn, inv, ok, PLAIN || dom[n]);
                    T* d = Bd + oB0 + n * BBW;
                    d[0] = Bn[0];
                    d[BCS] = Bn[1];
                    d[2 * BCS] = Bn[2];
                    const T sn = (inner_k && (PLAIN || in_xy[n])) ? a.dtg * inv : T(0);
                    // record(p) = columns 0, 1 of dF, xi_0, xi_1 | column 2 of dF, n_0, s, xi_2
                    uint32_t w0[CW], w1[CW];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        W32::put(w0 + c * W32::N, dF[n][c][0]);
                        W32::put(w0 + (3 + c) * W32::N, dF[n][c][1]);
                        W32::put(w1 + c * W32::N, dF[n][c][2]);
                        W32::put(w1 + (3 + c) * W32::N, n0[c]);
                    }
                    W32::put(w0 + 6 * W32::N, x1[n][0]);
                    W32::put(w0 + 7 * W32::N, x1[n][1]);
                    W32::put(w1 + 6 * W32::N, sn);
                    W32::put(w1 + 7 * W32::N, x1[n][2]);
                    if constexpr (CW == 16) { tmem::st16(rec_addr(buf, n, 0), w0); tmem::st16(rec_addr(buf, n, 1), w1); }
                    else { tmem::st8(rec_addr(buf, n, 0), w0); tmem::st8(rec_addr(buf, n, 1), w1); }
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) { xc[0][c] = x1[0][c]; xc[1][c] = x1[1][c]; }
                tmem::wait_st();
                tmem::fence_before_sync();
                ptx::named_arrive(BAR_FULL + buf, NTH);           // B(p) and record(p) are published
                // this warp is done with the xi / b planes p (the producer's warp collects the arrivals)
                ptx::named_arrive(BAR_A + buf, NAG * 32);
                if (++buf == NB) buf = 0;
                sm2 = sm1; sm1 = s0; s0 = s1; s1 = s2;
                if (s1 == 0) par1 ^= 1u;                          // the slot of the plane p+1 wrapped around
                if (++s2 == R) s2 = 0;
                if (++sb0 == RB) { sb0 = 0; parb ^= 1u; }
            }
        };
        if (plain) runA(std::true_type{});
        else runA(std::false_type{});
      } else {
        // ---- R-warps: warp 2 NAW owns the ring rows j = -1 and j = TY (two nodes per thread), warp 2 NAW + 1 the ring
        // columns i = -1 and i = TX (8 rows left and 8 rows right per half-warp: distinct banks) and the TMA producer
        // R-warps: 2 NAW -> ring row j = -1, 2 NAW + 1 -> ring row j = TY, 2 NAW + 2 -> both ring columns,
        // 2 NAW + 3 -> no node: its lane 0 is the TMA producer and its warp collects the slot-release arrivals
        const int rw = warp - 2 * NAW;
        const bool rows = rw < 3;                            // "this warp only arrives on the slot-release barrier"
        const int nr = rw < 3 ? 1 : 0;
        int ti[2], tj[2], oxr[2], obr[2], oBr[2];
        unsigned edge[2];
        bool dom[2];
        if (rw == 0) { ti[0] = lane; tj[0] = -1; }
        else if (rw == 1) { ti[0] = lane; tj[0] = TY; }
        else { ti[0] = (lane >> 3) & 1 ? TX : -1; tj[0] = (lane & 7) + 8 * (lane >> 4); }
        ti[1] = ti[0]; tj[1] = tj[0];
#pragma unroll
        for (int m = 0; m < 2; ++m) {
            const int gi2 = i0 + ti[m], gj2 = j0 + tj[m];
            oxr[m] = (tj[m] + 2) * BW + (ti[m] + L::HXL);
            obr[m] = (tj[m] + 1) * BW + (ti[m] + L::HXL);
            oBr[m] = (tj[m] + 1) * BBW + (ti[m] + 1);
            dom[m] = gi2 >= 0 && gi2 < a.nx && gj2 >= 0 && gj2 < a.ny && tj[m] < TY + 1 && m < nr;
            edge[m] = !dom[m] ? 0u : (gi2 == 0 ? 1u : 0u) | (gi2 == a.nx - 1 ? 2u : 0u) | (gj2 == 0 ? 4u : 0u) | (gj2 == a.ny - 1 ? 8u : 0u);
        }
        T xr[2][3];                                         // own xi(p-1) of the ring nodes
#pragma unroll
        for (int c = 0; c < 3; ++c) { xr[0][c] = T(0); xr[1][c] = T(0); }
        if (first_p > 0) {
            const T* f = xplane(first_p - 1);
#pragma unroll
            for (int c = 0; c < 3; ++c) { xr[0][c] = f[oxr[0] + c * CSX]; xr[1][c] = f[oxr[1] + c * CSX]; }
        }
        int buf = first_p % NB;
        int s0 = (first_p - pfirst) % R, s1 = (s0 + 1) % R, s2 = (s0 + 2) % R, sm1 = (s0 + R - 1) % R, sm2 = (s0 + R - 2) % R;
        uint32_t par1 = (uint32_t)(((first_p + 1 - pfirst) / R) & 1);
        int sb0 = 0;
        uint32_t parb = 0u;
#pragma unroll 1
        for (int p = first_p; p <= kend; ++p) {
            const T* f1 = sx + s0 * L::SLOTX;
            const T* f2 = sx + s1 * L::SLOTX;
            if (p + 1 <= plast) ptx::mbar_wait(bar_x + 8u * (uint32_t)s1, par1);
            ptx::mbar_wait(bar_b + 8u * (uint32_t)sb0, parb);
            const T* bs = sb + sb0 * L::SLOTB;
            const bool work = p >= k0 && p < kend;              // the planes whose in-plane differences are taken
            T dFr[2][3][3], x1[2][3];
#pragma unroll
            for (int m = 0; m < 1; ++m) {
                const T* fr = f1 + oxr[m];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    x1[m][c] = fr[c * CSX];
                    dFr[m][c][0] = fr[c * CSX + 1] - fr[c * CSX - 1];
                    dFr[m][c][1] = fr[c * CSX + BW] - fr[c * CSX - BW];
                }
                if (p == 0) {
                    const T* f3 = sx + s2 * L::SLOTX;
#pragma unroll
                    for (int c = 0; c < 3; ++c) dFr[m][c][2] = T(4) * f2[oxr[m] + c * CSX] - T(3) * x1[m][c] - f3[oxr[m] + c * CSX];
                } else if (p + 1 <= nz - 1) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) dFr[m][c][2] = f2[oxr[m] + c * CSX] - xr[m][c];
                } else {
                    const T* fm = sx + sm2 * L::SLOTX;
#pragma unroll
                    for (int c = 0; c < 3; ++c) dFr[m][c][2] = T(3) * x1[m][c] - T(4) * xr[m][c] + fm[oxr[m] + c * CSX];
                }
                if (edge[m]) face_fix<T, BW, CSX>(fr, edge[m], dFr[m]);
            }
            if (p >= first_p + NB) ptx::named_sync(BAR_FREE + buf, NTH);
            if (work) {
                T* Bd = sB + buf * L::BSLOT;
#pragma unroll
                for (int m = 0; m < 1; ++m) {
                    if (m < nr) {
                        T n0[3], B[3], inv;
                        duo_push<T, CSB>(dFr[m], bs + obr[m], twoh, n0, B, inv, ok, dom[m]);
                        T* d = Bd + oBr[m];
                        d[0] = B[0];
                        d[BCS] = B[1];
                        d[2 * BCS] = B[2];
                    }
                }
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) xr[0][c] = x1[0][c];
            ptx::named_arrive(BAR_FULL + buf, NTH);
            if (rows) {
                ptx::named_arrive(BAR_A + buf, NAG * 32);
            } else {
                ptx::named_sync(BAR_A + buf, NAG * 32);         // every A- and R-warp is done with the xi / b planes p
                if (producer) refill(p + R, p + RB);            // the slots of the planes <= p take the planes up to p+R / p+RB
            }
            if (++buf == NB) buf = 0;
            sm2 = sm1; sm1 = s0; s0 = s1; s1 = s2;
            if (s1 == 0) par1 ^= 1u;
            if (++s2 == R) s2 = 0;
            if (++sb0 == RB) { sb0 = 0; parb ^= 1u; }
        }
      }
    } else {
        // =============================================== F-warps ===============================================
        auto ownB = [&](int buf, T(&B)[2][3]) {
            const T* g = sB + buf * L::BSLOT + oB0;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                B[0][c] = g[c * BCS];
                B[1][c] = g[c * BCS + BBW];
            }
        };
        auto fetch = [&](int buf, int n, uint32_t(&w0)[CW], uint32_t(&w1)[CW]) {
            if constexpr (CW == 16) { tmem::ld16(rec_addr(buf, n, 0), w0); tmem::ld16(rec_addr(buf, n, 1), w1); }
            else { tmem::ld8(rec_addr(buf, n, 0), w0); tmem::ld8(rec_addr(buf, n, 1), w1); }
        };
        T Bm[2][3], Bc[2][3];                           // own B(t-1), B(t) of the pair
        // DIAG: the same pass with the update replaced by the reduction of S6 (E, max |JxB|, max |JxB|/B^2, min D)
        DiagPartial acc = { 0.0, 0.0, 0.0, INFINITY };
        const bool f_in_x = gi > 0 && gi < a.nx - 1;
        const bool f_in_xy[2] = { f_in_x && gja > 0 && gja < a.ny - 1, f_in_x && gja + 1 < a.ny - 1 };
        double zxy[2];                                  // trapezoid weights of the node's column (Eq. 3.13)
#pragma unroll
        for (int n = 0; n < 2; ++n)
            zxy[n] = ((gi == 0 || gi == a.nx - 1) ? 0.5 : 1.0) * ((gja + n == 0 || gja + n == a.ny - 1) ? 0.5 : 1.0);
        auto diag_node = [&](int n, int k, const T(&c0)[3], const T(&n0)[3], const T(&B)[3], const T(&uu)[3]) {
            if (!st[n]) return;
            const double D = (double)c0[0] * n0[0] + (double)c0[1] * n0[1] + (double)c0[2] * n0[2];
            const double b2 = (double)B[0] * B[0] + (double)B[1] * B[1] + (double)B[2] * B[2];
            const bool kface = k == 0 || k == nz - 1;
            DiagPartial v = { zxy[n] * (kface ? 0.5 : 1.0) * b2 * D, 0.0, 0.0, D };
            if (f_in_xy[n] && !kface) {
                const double fm = sqrt((double)uu[0] * uu[0] + (double)uu[1] * uu[1] + (double)uu[2] * uu[2]) / D;
                v.fmax = fm;
                v.xi = fm / b2;
            }
            diag_combine(acc, v);
        };
#pragma unroll
        for (int c = 0; c < 3; ++c) { Bm[0][c] = T(0); Bm[1][c] = T(0); }
        int buf = first_p % NB;                         // buffer of the plane t
        if (k0 > 0) {
            ptx::named_sync(BAR_FULL + buf, NTH);       // plane k0-1: only the own B is needed
            ownB(buf, Bm);
            ptx::named_arrive(BAR_FREE + buf, NTH);
            if (++buf == NB) buf = 0;
        }
        ptx::named_sync(BAR_FULL + buf, NTH);           // plane k0
        tmem::fence_after_sync();
        ownB(buf, Bc);
        T* po = out + (long long)k0 * a.plane + (long long)gja * a.pitch + gi;
#pragma unroll 1
        for (int t = k0; t < kend; ++t) {
            const int bufn = buf + 1 == NB ? 0 : buf + 1;
            uint32_t w0[CW], w1[CW];
            fetch(buf, 0, w0, w1);                      // record(t) of node 0 (published with plane t)
            ptx::named_sync(BAR_FULL + bufn, NTH);      // plane t+1
            tmem::fence_after_sync();
            T Bp[2][3];
            ownB(bufn, Bp);
            const T* g = sB + buf * L::BSLOT + oB0;
#pragma unroll
            for (int n = 0; n < 2; ++n) {
                T dBi[3], dBj[3], dBk[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const T* gc = g + c * BCS + n * BBW;
                    dBi[c] = gc[1] - gc[-1];
                    dBj[c] = n == 0 ? Bc[1][c] - gc[-BBW] : gc[BBW] - Bc[0][c];
                    dBk[c] = Bp[n][c] - Bm[n][c];
                }
                tmem::wait_ld(w0);
                tmem::wait_ld(w1);
                T c0[3], c1[3], c2[3], n0[3], n1[3], n2[3], x[3], DJ[3], uu[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    c0[c] = W32::get(w0 + c * W32::N);
                    c1[c] = W32::get(w0 + (3 + c) * W32::N);
                    c2[c] = W32::get(w1 + c * W32::N);
                    n0[c] = W32::get(w1 + (3 + c) * W32::N);
                }
                x[0] = W32::get(w0 + 6 * W32::N);
                x[1] = W32::get(w0 + 7 * W32::N);
                x[2] = W32::get(w1 + 7 * W32::N);
                const T s = W32::get(w1 + 6 * W32::N);
                cross_set(c2, c0, n1);                  // n_1 = dF_2 x dF_0,  n_2 = dF_0 x dF_1  (Eqs. 2.5/2.6)
                cross_set(c0, c1, n2);
                if (n == 0) fetch(buf, 1, w0, w1);      // record(t) of node 1, under the arithmetic of node 0
                // D J = n_0 x delta_i B + n_1 x delta_j B + n_2 x delta_k B;  u = gamma J x B;  xi+ = xi + dt u
                cross_set(n0, dBi, DJ);
                cross_acc(n1, dBj, DJ);
                cross_acc(n2, dBk, DJ);
                cross_set(DJ, Bc[n], uu);
                if constexpr (DIAG) {
                    diag_node(n, t, c0, n0, Bc[n], uu);
                } else {
#pragma unroll
                    for (int c = 0; c < 3; ++c) x[c] = fma(s, uu[c], x[c]);
                    ok = ok && is_finite(x[0] + x[1] + x[2]);
                    if (st[n]) {
                        T* pn = po + n * a.pitch;
                        pn[0] = x[0];
                        pn[a.comp] = x[1];
                        pn[2 * a.comp] = x[2];
                    }
                }
            }
            po += a.plane;
            tmem::fence_before_sync();
            ptx::named_arrive(BAR_FREE + buf, NTH);     // the B plane t and record(t) may be overwritten
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                Bm[0][c] = Bc[0][c]; Bm[1][c] = Bc[1][c];
                Bc[0][c] = Bp[0][c]; Bc[1][c] = Bp[1][c];
            }
            buf = bufn;
        }
        if (k1 == nz) {   // the top plane (line-tied) is carried through: its xi sits in record(nz-1)
#pragma unroll
            for (int n = 0; n < 2; ++n) {
                uint32_t w0[CW], w1[CW];
                fetch(buf, n, w0, w1);
                tmem::wait_ld(w0);
                tmem::wait_ld(w1);
                if constexpr (DIAG) {
                    T c0[3], n0[3];
                    const T zero[3] = { T(0), T(0), T(0) };
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        c0[c] = W32::get(w0 + c * W32::N);
                        n0[c] = W32::get(w1 + (3 + c) * W32::N);
                    }
                    diag_node(n, nz - 1, c0, n0, Bc[n], zero);
                } else if (st[n]) {
                    T* pl = out + (long long)(nz - 1) * a.plane + (long long)(gja + n) * a.pitch + gi;
                    pl[0] = W32::get(w0 + 6 * W32::N);
                    pl[a.comp] = W32::get(w0 + 7 * W32::N);
                    pl[2 * a.comp] = W32::get(w1 + 7 * W32::N);
                }
            }
        }
        if constexpr (DIAG) {
            // fixed-order reduction: lanes by a shuffle tree, then the F-warps in index order (below)
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                DiagPartial w;
                w.e = __shfl_down_sync(0xffffffffu, acc.e, o);
                w.fmax = __shfl_down_sync(0xffffffffu, acc.fmax, o);
                w.xi = __shfl_down_sync(0xffffffffu, acc.xi, o);
                w.dmin = __shfl_down_sync(0xffffffffu, acc.dmin, o);
                diag_combine(acc, w);
            }
            diag_acc = acc;
        }
    }
    if (!ok) atomicOr(a.flag, FLAG_NUMERIC);
    tmem::fence_before_sync();
    __syncthreads();                                    // the pipeline is drained: shared memory is free
    if constexpr (DIAG) {
        DiagPartial* sh = reinterpret_cast<DiagPartial*>(smem);
        if (isF && lane == 0) sh[widx] = diag_acc;
        __syncthreads();
        if (tid == 0) {
            DiagPartial v = sh[0];
            for (int w = 1; w < NAW; ++w) diag_combine(v, sh[w]);
            reinterpret_cast<DiagPartial*>(out)[blockIdx.x] = v;
        }
    }
    if (warp == 0) tmem::dealloc<512>(tm_base_s);
}

// ----------------------------------------------------------------------------------------------- host side

#ifndef MR_DTY
#define MR_DTY 16
#define MR_DR 5
#define MR_DRB 3
#define MR_DNB 3
#endif
constexpr int kDTY = MR_DTY, kDR = MR_DR, kDRB = MR_DRB, kDNB = MR_DNB;

template <typename T>
inline cudaError_t duo_set_smem(size_t bytes)
{
    cudaError_t e = cudaFuncSetAttribute(k_step_duo<T, kDTY, kDR, kDRB, kDNB, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_step_duo<T, kDTY, kDR, kDRB, kDNB, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

inline bool build_duo_plan(StreamPlan* p, const StreamGeom& g, bool f64, void* xi0, void* xi1, void* b, int sm_count,
                           std::string* why)
{
    using Ld = DuoLayout<double, kDTY, kDR, kDRB, kDNB>;
    using Lf = DuoLayout<float, kDTY, kDR, kDRB, kDNB>;
    p->usable = false;
    p->f64 = f64;
    p->g = g;
    p->xi[0] = xi0;
    p->xi[1] = xi1;
    p->b = b;
    p->name = f64 ? "duo_tmem_f64" : "duo_tmem_f32";
    const int bw = f64 ? Ld::BW : Lf::BW;
    if (!encode_map(&p->map_xi[0], f64, xi0, g, bw, kDTY + 4) || !encode_map(&p->map_xi[1], f64, xi1, g, bw, kDTY + 4) ||
        !encode_map(&p->map_b, f64, b, g, bw, kDTY + 2)) {
        *why = "cuTensorMapEncodeTiled failed";
        return false;
    }
    p->tiles_x = (g.nx + Ld::TX - 1) / Ld::TX;
    p->tiles_y = (g.ny + kDTY - 1) / kDTY;
    p->smem_bytes = f64 ? Ld::BYTES : Lf::BYTES;
    cudaError_t e = f64 ? duo_set_smem<double>(p->smem_bytes) : duo_set_smem<float>(p->smem_bytes);
    if (e != cudaSuccess) {
        *why = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e);
        return false;
    }
    choose_chunks(p->tiles_x * p->tiles_y, g.nz, sm_count, &p->nchunks, &p->chunk_len);
    p->usable = true;
    return true;
}

template <typename T>
inline cudaError_t launch_duo_step(const StreamPlan& p, int cur, T dtg, int* flag, cudaStream_t stream)
{
    using L = DuoLayout<T, kDTY, kDR, kDRB, kDNB>;
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
    k_step_duo<T, kDTY, kDR, kDRB, kDNB, false><<<grid, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], p.map_b,
                                                                                              static_cast<T*>(p.xi[1 - cur]), a);
    return cudaGetLastError();
}

// S6 of the state in buffer `cur` by the same pass (no update, no store): one DiagPartial per CTA into `partials`
template <typename T>
inline cudaError_t launch_duo_diag(const StreamPlan& p, int cur, DiagPartial* partials, int* nblocks, int* flag, cudaStream_t stream)
{
    using L = DuoLayout<T, kDTY, kDR, kDRB, kDNB>;
    StreamArgs<T> a;
    a.nx = p.g.nx; a.ny = p.g.ny; a.nz = p.g.nz;
    a.pitch = p.g.pitch; a.plane = p.g.plane; a.comp = p.g.comp;
    for (int c = 0; c < 3; ++c) a.twoh[c] = (T)p.g.twoh[c];
    a.dtg = (T)0;
    a.tiles_x = p.tiles_x;
    a.ntiles = p.tiles_x * p.tiles_y;
    a.chunk_len = p.chunk_len;
    a.flag = flag;
    const int grid = a.ntiles * p.nchunks;
    *nblocks = grid;
    k_step_duo<T, kDTY, kDR, kDRB, kDNB, true><<<grid, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], p.map_b,
                                                                                             reinterpret_cast<T*>(partials), a);
    return cudaGetLastError();
}

}  // namespace mr
