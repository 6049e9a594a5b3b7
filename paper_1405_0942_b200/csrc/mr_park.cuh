// mr_park.cuh -- the streaming step kernel for the mimetic operator with the per-node state parked in Tensor Memory
// (S1-S5 in one pass).
//
// Data flow and arithmetic are those of mr_lean.cuh (xy tile, CTA marching along k, every tile thread owns the nodes
// (i, j) and (i, j+1), xi planes by TMA into a shared ring, b straight from HBM one plane ahead, B shared through a
// double-buffered shared plane; D J = n_0 x delta_i B + n_1 x delta_j B + n_2 x (B(k+1) - B(k-1)), the closed form
// of Eqs. 2.3-2.7).  What is new: of the 19 values a node carries from one plane to the next (area vectors n_0, n_1,
// n_2, W = n_2 x B(k-1), s = dt gamma / D, own B, own xi) only the own B and xi stay in registers; the other 13 are
// parked in TMEM (mr_tmem.cuh) at the end of an iteration and fetched just before their use:
//   chunk I(n)  n_0, n_1          fetched at the top of the next iteration (in-plane part of D J)
//   chunk F(n)  n_2, W, s         fetched when the plane is finished (k part of D J, u = gamma J x B, update)
// With the state out of the way the kernel fits into 128 registers without spills, so that two CTAs (16 warps)
// share an SM: twice the warps of the register-resident pair kernel, with the two CTAs out of step so that one's
// shared-memory phase overlaps the other's FP64 phase.  The TMEM traffic (2 x 128 B per node and plane in fp64)
// runs on the tensor-memory data path, not on the shared-memory crossbar the stencil exchange is bound by.
#pragma once
#include "mr_lean.cuh"
#include "mr_tmem.cuh"

namespace mr {

#ifndef MR_PARK_MINB
#define MR_PARK_MINB 2
#endif

// shared memory of k_step_park: the LeanLayout (xi ring, two B planes, mbarriers) followed by the scratch of the ring
// threads: own xi(t) [3][128] and own b of two planes [2][3][128] (filled by cp.async, no registers held)
template <typename T, int TY, int R>
struct ParkLayout {
    using L = LeanLayout<T, TY, R>;
    static constexpr int NRT = 128;                                                   // ring threads (<= 4 warps)
    static constexpr size_t OFF_RX = (L::OFF_BAR + (size_t)R * 8 + 127) / 128 * 128;
    static constexpr size_t OFF_RB = OFF_RX + (size_t)3 * NRT * sizeof(T);
    static constexpr size_t BYTES = OFF_RB + (size_t)6 * NRT * sizeof(T) + 128;       // +128: base alignment slack
};

template <typename T, int TY, int R>
__global__ void __launch_bounds__(TY * 16, MR_PARK_MINB)
k_step_park(const __grid_constant__ CUtensorMap map_in, const T* __restrict__ bsrc, T* __restrict__ out, const StreamArgs<T> a)
{
    using L = LeanLayout<T, TY, R>;
    using W32 = tmem::Words<T>;
    constexpr int TX = L::TX, NT = L::NWARPS, BW = L::BW, CSX = L::CSX, BBW = L::BBW, BCS = L::BCS;
    constexpr int NCOLS = 512 / MR_PARK_MINB;                 // TMEM columns of this CTA
    constexpr int CW = 8 * W32::N;                            // words per chunk (8 values)
    constexpr int CPW = NCOLS / ((NT + 3) / 4);               // columns of one warp
    static_assert(CPW >= 8 * CW, "a thread parks two buffers of two chunks per node");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t tm_base_s;
    unsigned char* smem = smem_raw + ((128u - (ptx::smem_u32(smem_raw) & 127u)) & 127u);
    const T* sx = reinterpret_cast<const T*>(smem + L::OFF_X);
    T* sB = reinterpret_cast<T*>(smem + L::OFF_BB);
    const uint32_t sx_u32 = ptx::smem_u32(sx);
    const uint32_t bar_x = ptx::smem_u32(smem + L::OFF_BAR);
    using PL = ParkLayout<T, TY, R>;
    constexpr int NRT = PL::NRT;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    T* srx = reinterpret_cast<T*>(smem + PL::OFF_RX) + (tid & (NRT - 1));      // [c * NRT]: own xi(t) of the ring node
    T* srb = reinterpret_cast<T*>(smem + PL::OFF_RB) + (tid & (NRT - 1));      // [(buf * 3 + c) * NRT]: own b of the ring node
    const int tile = blockIdx.x % a.ntiles, chunk = blockIdx.x / a.ntiles;
    const int i0 = (tile % a.tiles_x) * TX, j0 = (tile / a.tiles_x) * TY;
    const int nz = a.nz;
    const int k0 = chunk * a.chunk_len, k1 = min(k0 + a.chunk_len, nz);
    const int kend = min(k1, nz - 1);                                   // the loop forms B of the planes k0 .. kend
    const int pfirst = max(k0 - 2, 0), plast = min(k1 + 1, nz - 1);     // xi planes this item touches
    const T twoh[3] = { a.twoh[0], a.twoh[1], a.twoh[2] };

    // ---- TMA producer: lane 0 of the last warp (it carries no ring node); warp 0 owns the TMEM allocation ----
    const bool producer = tid == (NT - 1) * 32;
    int next_load = pfirst;
    auto refill = [&](int upto) {
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
    if (warp == 0) tmem::alloc<NCOLS>(&tm_base_s);
    tmem::fence_before_sync();
    __syncthreads();
    tmem::fence_after_sync();
    if (producer) refill(pfirst + R - 1);
    const uint32_t tm_base = tm_base_s;
    const uint32_t tm0 = tm_base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * CPW);
    const uint32_t tI[2] = { tm0, tm0 + 2 * CW }, tF[2] = { tm0 + CW, tm0 + 3 * CW };

    auto wait_x = [&](int p) { const int q = p - pfirst; ptx::mbar_wait(bar_x + 8u * (uint32_t)(q % R), (uint32_t)((q / R) & 1)); };
    auto xplane = [&](int p) -> const T* { return sx + ((p - pfirst) % R) * L::SLOTX; };

    // nodes of this thread (mr_lean.cuh): 0, 1 = the pair (lane, 2 warp), (lane, 2 warp + 1); 2 = a halo-1 ring node
    int ti2, tj2;
    constexpr int NRINGW = 2 + (TY + 15) / 16;
    static_assert(NRINGW < NT && NRINGW * 32 <= NRT, "the last warp (TMA producer) carries no ring node");
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
    auto load_b = [&](int p, int n, T(&b)[3]) {
        const T* g = bsrc + (long long)p * a.plane + gb[n];
#pragma unroll
        for (int c = 0; c < 3; ++c) b[c] = dom[n] ? __ldg(g + c * a.comp) : T(0);
    };
    auto ring_b_async = [&](int p) {                 // b of the ring node on plane p -> scratch buffer p & 1
        if (dom[2]) {
            const T* g = bsrc + (long long)p * a.plane + gb[2];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const uint32_t dst = ptx::smem_u32(srb + ((p & 1) * 3 + c) * NRT);
                asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst), "l"(g + c * a.comp), "n"((int)sizeof(T)) : "memory");
            }
        }
    };
    auto store_B = [&](int p, int n, const T(&B)[3]) {
        T* d = sB + (p & 1) * L::BSLOT + oB[n];
        d[0] = B[0];
        d[BCS] = B[1];
        d[2 * BCS] = B[2];
    };
    // chunk <-> values
    auto park = [&](uint32_t taddr, const T(&v)[8]) {
        uint32_t w[CW];
#pragma unroll
        for (int i = 0; i < 8; ++i) W32::put(w + i * W32::N, v[i]);
        if constexpr (CW == 16) tmem::st16(taddr, w); else tmem::st8(taddr, w);
    };
    auto fetch = [&](uint32_t taddr, uint32_t(&w)[CW]) {
        if constexpr (CW == 16) tmem::ld16(taddr, w); else tmem::ld8(taddr, w);
    };

    const int gi = i0 + lane, gja = j0 + tj[0];
    const bool in_x = gi > 0 && gi < a.nx - 1;
    const bool in_xy[2] = { in_x && gja > 0 && gja < a.ny - 1, in_x && gja + 1 < a.ny - 1 };
    const bool st[2] = { gi < a.nx && gja < a.ny, gi < a.nx && gja + 1 < a.ny };

    for (int p = pfirst; p <= min(pfirst + R - 1, plast); ++p) wait_x(p);

    bool ok = true;
    // Register state carried over the barrier: own B(t), own xi(t), own b(t+1) of the pair (and of the ring node)
    T xc[2][3], bq[2][3];
#pragma unroll
    for (int n = 0; n < 2; ++n)
#pragma unroll
        for (int c = 0; c < 3; ++c) xc[n][c] = T(0);
    {
        const T zero[8] = { T(0), T(0), T(0), T(0), T(0), T(0), T(0), T(0) };
        const uint32_t off = (uint32_t)((k0 - 1) & 1) * (4 * CW);
        park(tI[0] + off, zero); park(tI[1] + off, zero); park(tF[0] + off, zero); park(tF[1] + off, zero);
    }
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
            T Bp[3];
            lean_push(dF, b, twoh, nv, Bp, inv, ok, dom[n]);
            store_B(p, n, Bp);      // only the own position is read back (W of plane k0)
        }
        if (ring) {
            const T* f = pc + ox[2];
#pragma unroll
            for (int c = 0; c < 3; ++c) srx[c * NRT] = f[c * CSX];
        }
    }
    if (k0 == 0) {   // "own B(-1)" is read back (times n_2 of the line-tied plane 0, which never moves): keep it finite
        const T zero3[3] = { T(0), T(0), T(0) };
        store_B(-1, 0, zero3);
        store_B(-1, 1, zero3);
    }
#pragma unroll
    for (int n = 0; n < 2; ++n) load_b(k0, n, bq[n]);
    if (ring) ring_b_async(k0);
    tmem::wait_st();

    T* po = out + (long long)k0 * a.plane + (long long)gja * a.pitch + gi;
    const bool plain = i0 > 0 && i0 + TX <= a.nx - 2 && j0 > 0 && j0 + TY <= a.ny - 2;
    auto run = [&](auto plain_c) {
        constexpr bool PLAIN = decltype(plain_c)::value;
#pragma unroll 1
        for (int t = k0 - 1; t < kend; ++t) {
            const int q1 = t + 1 - pfirst;
            const T* f1 = sx + (q1 % R) * L::SLOTX + ox[0];       // xi plane t+1, node 0 of the pair
            const T* f2 = sx + ((q1 + 1) % R) * L::SLOTX + ox[0]; // xi plane t+2
            const bool fin = t >= k0;                              // plane t is finished (written) by this item
            const uint32_t cur = (uint32_t)(t & 1) * (4 * CW), nxt = (4 * CW) - cur;   // TMEM buffers of plane t / t+1
            const bool inner_k = t + 1 > 0 && t + 1 < nz - 1;
            const T* g = sB + (t & 1) * L::BSLOT + oB[0];
#pragma unroll
            for (int n = 0; n < 2; ++n) {
                // ---------------- A: stage A of plane t+1 ----------------
                T Bn[3], x1[3], B0[3];   // own B(t+1), own xi(t+1), own B(t) (re-read from the shared plane)
                {
                    T dF[3][3];
                    const T* fn = f1 + n * BW;
#pragma unroll
                    for (int c = 0; c < 3; ++c) x1[c] = fn[c * CSX];
                    if (t + 1 == 0) {          // bottom face: -3 x(0) + 4 x(1) - x(2)
                        const T* f3 = sx + ((q1 + 2) % R) * L::SLOTX + ox[0] + n * BW;
#pragma unroll
                        for (int c = 0; c < 3; ++c) dF[c][2] = T(4) * f2[c * CSX + n * BW] - T(3) * x1[c] - f3[c * CSX];
                    } else if (t + 2 <= nz - 1) {
#pragma unroll
                        for (int c = 0; c < 3; ++c) dF[c][2] = f2[c * CSX + n * BW] - xc[n][c];
                    } else {                   // top face: 3 x(nz-1) - 4 x(nz-2) + x(nz-3); plane nz-3 is still in its slot
                        const T* fm = sx + ((q1 - 2) % R) * L::SLOTX + ox[0] + n * BW;
#pragma unroll
                        for (int c = 0; c < 3; ++c) dF[c][2] = T(3) * x1[c] - T(4) * xc[n][c] + fm[c * CSX];
                    }
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        dF[c][0] = fn[c * CSX + 1] - fn[c * CSX - 1];
                        dF[c][1] = fn[c * CSX + BW] - fn[c * CSX - BW];
                    }
                    if (!PLAIN && edge[n]) face_fix<T, BW, CSX>(fn, edge[n], dF);
                    T nv[3][3], inv;
                    lean_push(dF, bq[n], twoh, nv, Bn, inv, ok, PLAIN || dom[n]);
                    store_B(t + 1, n, Bn);
                    if (t + 2 <= kend) load_b(t + 2, n, bq[n]);     // b of the plane the next iteration pushes forward
                    // the state of plane t+1 goes to the other TMEM buffer: n_0, n_1 | n_2, W = n_2 x B(t), s
                    T Wn[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) B0[c] = g[c * BCS + n * BBW];
                    cross_set(nv[2], B0, Wn);
                    const T sn = (inner_k && (PLAIN || in_xy[n])) ? a.dtg * inv : T(0);
                    const T vI[8] = { nv[0][0], nv[0][1], nv[0][2], nv[1][0], nv[1][1], nv[1][2], T(0), T(0) };
                    const T vF[8] = { nv[2][0], nv[2][1], nv[2][2], Wn[0], Wn[1], Wn[2], sn, T(0) };
                    park(tI[n] + nxt, vI);
                    park(tF[n] + nxt, vF);
                }
                // ---------------- I + F: D J of plane t, u = gamma J x B, xi+ = xi + dt u ----------------
                {
                    uint32_t wI[CW], wF[CW];
                    fetch(tI[n] + cur, wI);
                    fetch(tF[n] + cur, wF);
                    T dBi[3], dBj[3], DJ[3], uu[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const T* gc = g + c * BCS + n * BBW;
                        dBi[c] = gc[1] - gc[-1];
                        dBj[c] = gc[BBW] - gc[-BBW];
                    }
                    tmem::wait_ld(wI);
                    tmem::wait_ld(wF);
                    if (fin) {
                        T n0[3], n1[3], n2[3];
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            n0[c] = W32::get(wI + c * W32::N);
                            n1[c] = W32::get(wI + (3 + c) * W32::N);
                            n2[c] = W32::get(wF + c * W32::N);
                            DJ[c] = -W32::get(wF + (3 + c) * W32::N);
                        }
                        const T s = W32::get(wF + 6 * W32::N);
                        cross_acc(n0, dBi, DJ);
                        cross_acc(n1, dBj, DJ);
                        cross_acc(n2, Bn, DJ);
                        cross_set(DJ, B0, uu);
#pragma unroll
                        for (int c = 0; c < 3; ++c) xc[n][c] = fma(s, uu[c], xc[n][c]);
                        ok = ok && is_finite(xc[n][0] + xc[n][1] + xc[n][2]);
                        if (PLAIN || st[n]) {
                            T* pn = po + n * a.pitch;
                            pn[0] = xc[n][0];
                            pn[a.comp] = xc[n][1];
                            pn[2 * a.comp] = xc[n][2];
                        }
                    }
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) xc[n][c] = x1[c];
                asm volatile("" ::: "memory");     // keep the two nodes apart: registers, not overlap, are the limit
            }
            if (fin) po += a.plane;
            if (ring && t + 1 < kend) {
                // stage A of plane t+1 at the ring node (own xi(t) and b(t+1) wait in the shared scratch)
                T dFr[3][3], nr[3][3], B[3], inv, xr[3], xr1[3], bqr[3];
                const T* fr = sx + (q1 % R) * L::SLOTX + ox[2];
                const T* fr2 = sx + ((q1 + 1) % R) * L::SLOTX + ox[2];
                asm volatile("cp.async.wait_all;" ::: "memory");
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    xr[c] = srx[c * NRT];
                    bqr[c] = dom[2] ? srb[(((t + 1) & 1) * 3 + c) * NRT] : T(0);
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
                for (int c = 0; c < 3; ++c) srx[c * NRT] = xr1[c];
                if (t + 2 < kend) ring_b_async(t + 2);
            }
            tmem::wait_st();
            ptx::cta_sync();
            // every read of the xi plane t+1 is done: its slot takes the plane t+1+R
            if (producer) refill(t + 1 + R);
            if (t + 3 <= plast) { const int q = t + 3 - pfirst; ptx::mbar_wait(bar_x + 8u * (uint32_t)(q % R), (uint32_t)((q / R) & 1)); }
        }
    };
#ifdef MR_ONLY_PLAIN
    run(std::true_type{});
#elif defined(MR_ONLY_EDGE)
    run(std::false_type{});
#else
    if (plain) run(std::true_type{});
    else run(std::false_type{});
#endif
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
    tmem::fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem::dealloc<NCOLS>(tm_base);
}

// ----------------------------------------------------------------------------------------------- host side

#ifndef MR_KTY
#define MR_KTY 16
#define MR_KR 4
#endif
constexpr int kKTY = MR_KTY, kKR = MR_KR;

template <typename T>
inline cudaError_t park_set_smem(size_t bytes)
{
    cudaError_t e = cudaFuncSetAttribute(k_step_park<T, kKTY, kKR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_step_park<T, kKTY, kKR>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
}

inline bool build_park_plan(StreamPlan* p, const StreamGeom& g, bool f64, void* xi0, void* xi1, void* b, int sm_count,
                            std::string* why)
{
    using Ld = LeanLayout<double, kKTY, kKR>;
    using Lf = LeanLayout<float, kKTY, kKR>;
    p->usable = false;
    p->f64 = f64;
    p->g = g;
    p->xi[0] = xi0;
    p->xi[1] = xi1;
    p->b = b;
    p->name = f64 ? "park_tmem_f64" : "park_tmem_f32";
    const int bw = f64 ? Ld::BW : Lf::BW;
    if (!encode_map(&p->map_xi[0], f64, xi0, g, bw, kKTY + 4) || !encode_map(&p->map_xi[1], f64, xi1, g, bw, kKTY + 4)) {
        *why = "cuTensorMapEncodeTiled failed";
        return false;
    }
    p->tiles_x = (g.nx + Ld::TX - 1) / Ld::TX;
    p->tiles_y = (g.ny + kKTY - 1) / kKTY;
    p->smem_bytes = f64 ? ParkLayout<double, kKTY, kKR>::BYTES : ParkLayout<float, kKTY, kKR>::BYTES;
    cudaError_t e = f64 ? park_set_smem<double>(p->smem_bytes) : park_set_smem<float>(p->smem_bytes);
    if (e != cudaSuccess) {
        *why = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e);
        return false;
    }
    int per_sm = 1;
    e = f64 ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_step_park<double, kKTY, kKR>, Ld::NTHREADS, p->smem_bytes)
            : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_step_park<float, kKTY, kKR>, Lf::NTHREADS, p->smem_bytes);
    if (e != cudaSuccess || per_sm < 1) per_sm = 1;
    if (per_sm > MR_PARK_MINB) per_sm = MR_PARK_MINB;      // TMEM: 512 / MR_PARK_MINB columns per CTA
    choose_chunks(p->tiles_x * p->tiles_y, g.nz, sm_count * per_sm, &p->nchunks, &p->chunk_len);
    p->usable = true;
    return true;
}

template <typename T>
inline cudaError_t launch_park_step(const StreamPlan& p, int cur, T dtg, int* flag, cudaStream_t stream)
{
    using L = LeanLayout<T, kKTY, kKR>;
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
    k_step_park<T, kKTY, kKR><<<grid, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], static_cast<const T*>(p.b),
                                                                            static_cast<T*>(p.xi[1 - cur]), a);
    return cudaGetLastError();
}

}  // namespace mr
