// mr_sym2.cuh -- the symmetric split-phase streaming step kernel with TWO rows per tile warp (experiment).
// Same scheme as mr_sym.cuh; 8 tile warps x 2 nodes per thread + 4 ring warps = 12 warps of up to 160 registers:
// the per-iteration overhead (polls, ring positions, addresses) is paid per pair, the j-differences inside the pair
// come from registers.
//
// Same ingredients as mr_duo.cuh (TMA rings of xi and b, B shared through shared-memory planes, the node's record
// parked in Tensor Memory, dedicated warps for the halo-1 ring), but without roles: each of the 16 tile warps owns one
// row of the 32 x 16 tile (one node per thread) and in iteration p does
//     A(p):    dF, n_0, D, 1/D, B(p) = dF b / D (Eq. 2.1) -> shared B plane p % NB;  record(p) -> TMEM (own columns);
//              mbarrier.arrive FULL[p % NB]
//     F(p-1):  mbarrier wait FULL[(p-1) % NB] -- a phase that completed about one iteration ago, so the wait is a
//              poll, not a stall --, D J = n_0 x delta_i B + n_1 x delta_j B + n_2 x (B(p) - B(p-2)) (closed form of
//              Eqs. 2.3-2.7), u = gamma J x B (Eq. 1.5), xi+ = xi + dt u -> HBM.
// The two halves of an iteration belong to different planes and are independent: every warp carries the same load
// (no A/F imbalance), and nobody waits for the slowest warp of the current plane.  A buffer p % NB is overwritten
// NB planes later; a warp that starts A(p) has seen FULL[p-2] complete, i.e. every warp has finished F(p-4): NB = 4.
#pragma once
#include <type_traits>

#include "mr_sym.cuh"

namespace mr {

template <typename T, int TY, int R, int RB, int NB>
struct Sym2Layout {
    static_assert(TY == 16 && R >= 4 && RB == R && NB >= 4, "tile / ring sizes (xi and b share the ring positions)");
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
    static constexpr int NTW = TY / 2, NWARPS = TY / 2 + 4, NTHREADS = NWARPS * 32;     // tile warps + 4 R-warps
    static constexpr size_t OFF_X = 0;
    static constexpr size_t OFF_B0 = OFF_X + (size_t)R * SLOTX * sizeof(T);
    static constexpr size_t OFF_BB = OFF_B0 + (size_t)RB * SLOTB * sizeof(T);
    static constexpr size_t OFF_BAR = OFF_BB + (size_t)NB * BSLOT * sizeof(T);
    static constexpr size_t BYTES = OFF_BAR + (size_t)(R + NB) * 8 + 128;
};

template <typename T, int TY, int R, int RB, int NB>
__global__ void __maxnreg__(160)
k_step_sym2(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_b, T* __restrict__ out,
           const StreamArgs<T> a)
{
    using L = Sym2Layout<T, TY, R, RB, NB>;
    using W32 = tmem::Words<T>;
    constexpr int TX = L::TX, NTW = L::NTW, BW = L::BW, CSX = L::CSX, CSB = L::CSB, BBW = L::BBW, BCS = L::BCS;
    constexpr int NW = L::NWARPS;
    constexpr int CW = 8 * W32::N, REC = 2 * CW;                   // record: 16 values in two chunks
    constexpr int WCOLS = 4 * REC;                                  // two record buffers (plane parity) x two nodes per tile warp
    static_assert(((NTW + 3) / 4) * WCOLS <= 512, "TMEM columns");
    constexpr int BAR_A = 1;                                        // named barriers BAR_A .. BAR_A + NB - 1
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t tm_base_s;
    unsigned char* smem = smem_raw + ((128u - (ptx::smem_u32(smem_raw) & 127u)) & 127u);
    const T* sx = reinterpret_cast<const T*>(smem + L::OFF_X);
    const T* sb = reinterpret_cast<const T*>(smem + L::OFF_B0);
    T* sB = reinterpret_cast<T*>(smem + L::OFF_BB);
    const uint32_t sx_u32 = ptx::smem_u32(sx), sb_u32 = ptx::smem_u32(sb);
    const uint32_t bar_x = ptx::smem_u32(smem + L::OFF_BAR), bar_full = bar_x + 8u * R;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const bool tilew = warp < NTW;
    const int tile = blockIdx.x % a.ntiles, chunk = blockIdx.x / a.ntiles;
    const int i0 = (tile % a.tiles_x) * TX, j0 = (tile / a.tiles_x) * TY;
    const int nz = a.nz;
    const int k0 = chunk * a.chunk_len, k1 = min(k0 + a.chunk_len, nz);
    const int kend = min(k1, nz - 1);
    const int first_p = max(k0 - 1, 0);
    const int pfirst = max(first_p - 1, 0), plast = min(kend + 1, nz - 1);
    const T twoh[3] = { a.twoh[0], a.twoh[1], a.twoh[2] };

    const bool pwarp = warp == NW - 1, producer = pwarp && lane == 0;
    if (producer) {
        for (int s = 0; s < R; ++s) ptx::mbar_init(bar_x + 8u * s, 1);
        for (int s = 0; s < NB; ++s) ptx::mbar_init(bar_full + 8u * s, NW);      // one arrival per warp
        ptx::fence_mbar_init();
    }
    if (warp == 0) tmem::alloc<512>(&tm_base_s);
    tmem::fence_before_sync();
    __syncthreads();
    tmem::fence_after_sync();
    const uint32_t tm0 = tm_base_s + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * WCOLS);

    // one ring position and one mbarrier per plane for the xi box and the b box (they are born and die together)
    int next_x = pfirst;
    auto refill = [&](int upto) {
        for (const int last = min(upto, plast); next_x <= last; ++next_x) {
            const uint32_t s = (uint32_t)((next_x - pfirst) % R);
            ptx::mbar_expect_tx(bar_x + 8u * s, L::XBOX_BYTES + L::BBOX_BYTES);
            ptx::tma_load_4d(sx_u32 + s * (uint32_t)(L::SLOTX * sizeof(T)), &map_in, i0 - L::HXL, j0 - 2, next_x, 0, bar_x + 8u * s);
            ptx::tma_load_4d(sb_u32 + s * (uint32_t)(L::SLOTB * sizeof(T)), &map_b, i0 - L::HXL, j0 - 1, next_x, 0, bar_x + 8u * s);
        }
    };
    if (producer) refill(pfirst + R - 1);

    // the node of this thread: tile warps own the row `warp` of the tile; R-warps a node of the halo-1 ring (row below,
    // row above, both columns) or none (the producer's warp)
    int ti, tj;
    bool has_node = true;
    if (tilew) { ti = lane; tj = 2 * warp; }
    else if (warp == NTW) { ti = lane; tj = -1; }
    else if (warp == NTW + 1) { ti = lane; tj = TY; }
    else if (warp == NTW + 2) { ti = (lane >> 3) & 1 ? TX : -1; tj = (lane & 7) + 8 * (lane >> 4); }
    else { ti = 0; tj = 0; has_node = false; }
    // node 0 = (ti, tj); tile warps also own node 1 = (ti, tj + 1): its offsets are +BW / +BBW / +pitch
    const int gi = i0 + ti, gj0 = j0 + tj;
    const int ox = (tj + 2) * BW + (ti + L::HXL), ob = (tj + 1) * BW + (ti + L::HXL), oB = (tj + 1) * BBW + (ti + 1);
    bool dom[2], in_xy[2], st[2];
    unsigned edge[2];
#pragma unroll
    for (int n = 0; n < 2; ++n) {
        const int gj = gj0 + n;
        dom[n] = has_node && (n == 0 || tilew) && gi >= 0 && gi < a.nx && gj >= 0 && gj < a.ny;
        edge[n] = !dom[n] ? 0u : (gi == 0 ? 1u : 0u) | (gi == a.nx - 1 ? 2u : 0u) | (gj == 0 ? 4u : 0u) | (gj == a.ny - 1 ? 8u : 0u);
        in_xy[n] = gi > 0 && gi < a.nx - 1 && gj > 0 && gj < a.ny - 1;
        st[n] = tilew && dom[n];
    }

    auto wait_x = [&](int p) { const int q = p - pfirst; ptx::mbar_wait(bar_x + 8u * (uint32_t)(q % R), (uint32_t)((q / R) & 1)); };
    for (int p = pfirst; p <= min(first_p + 1, plast); ++p) wait_x(p);
    if (first_p == 0 && plast >= 2) wait_x(2);

    bool ok = true;
    T xc[2][3], Bm[2][3], Bc[2][3], x1[2][3];          // own xi(p-1), B(p-2), B(p-1), xi(p) of the node(s)
#pragma unroll
    for (int n = 0; n < 2; ++n)
#pragma unroll
        for (int c = 0; c < 3; ++c) { xc[n][c] = T(0); Bm[n][c] = T(0); Bc[n][c] = T(0); x1[n][c] = T(0); }
    if (first_p > 0) {
        const T* f = sx + ((first_p - 1 - pfirst) % R) * L::SLOTX + ox;
#pragma unroll
        for (int c = 0; c < 3; ++c) { xc[0][c] = f[c * CSX]; xc[1][c] = f[c * CSX + BW]; }
    }
    T* po = out + (long long)k0 * a.plane + (long long)gj0 * a.pitch + gi;     // plane t = p-1 of the first F
    int buf = 0, pb = 0;
    uint32_t cpar = 0u, ppar = 0u;
    uint32_t rp = 0u;
    int s0 = (first_p - pfirst) % R, s1 = (s0 + 1) % R, s2 = (s0 + 2) % R, sm1 = (s0 + R - 1) % R, sm2 = (s0 + R - 2) % R;
    uint32_t par1 = (uint32_t)(((first_p + 1 - pfirst) / R) & 1);
  auto run = [&](auto tile_c) {
    constexpr bool TILE = decltype(tile_c)::value;
    constexpr int NN = TILE ? 2 : 1;
#pragma unroll 1
    for (int p = first_p; p <= kend; ++p) {
        const T* f1 = sx + s0 * L::SLOTX;                     // xi plane p
        const T* f2 = sx + s1 * L::SLOTX;                     // xi plane p+1
        if (p + 1 <= plast) ptx::mbar_wait(bar_x + 8u * (uint32_t)s1, par1);
        const T* bs = sb + s0 * L::SLOTB;
        // ---------------- A(p): push-forward of the plane p at the own node(s) ----------------
        T Bp[2][3];
#pragma unroll
        for (int c = 0; c < 3; ++c) { Bp[0][c] = T(0); Bp[1][c] = T(0); }
        if (TILE || (has_node && p >= k0 && p < kend)) {
            T dF[NN][3][3];
#pragma unroll
            for (int n = 0; n < NN; ++n) {
                const T* fr = f1 + ox + n * BW;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    x1[n][c] = fr[c * CSX];
                    dF[n][c][0] = fr[c * CSX + 1] - fr[c * CSX - 1];
                }
            }
#pragma unroll
            for (int n = 0; n < NN; ++n) {
                const T* fr = f1 + ox + n * BW;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    if (TILE) dF[n][c][1] = n == 0 ? x1[1][c] - fr[c * CSX - BW] : fr[c * CSX + BW] - x1[0][c];
                    else dF[n][c][1] = fr[c * CSX + BW] - fr[c * CSX - BW];
                }
                if (p == 0) {                   // bottom face: -3 x(0) + 4 x(1) - x(2)
                    const T* f3 = sx + s2 * L::SLOTX;
#pragma unroll
                    for (int c = 0; c < 3; ++c) dF[n][c][2] = T(4) * f2[ox + n * BW + c * CSX] - T(3) * x1[n][c] - f3[ox + n * BW + c * CSX];
                } else if (p + 1 <= nz - 1) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) dF[n][c][2] = f2[ox + n * BW + c * CSX] - xc[n][c];
                } else {                        // top face: 3 x(nz-1) - 4 x(nz-2) + x(nz-3); plane nz-3 is still in its slot
                    const T* fm = sx + sm2 * L::SLOTX;
#pragma unroll
                    for (int c = 0; c < 3; ++c) dF[n][c][2] = T(3) * x1[n][c] - T(4) * xc[n][c] + fm[ox + n * BW + c * CSX];
                }
                if (edge[n]) face_fix<T, BW, CSX>(fr, edge[n], dF[n]);
            }
#pragma unroll
            for (int n = 0; n < NN; ++n) {
                T n0[3], inv;
                duo_push<T, CSB>(dF[n], bs + ob + n * BW, twoh, n0, Bp[n], inv, ok, dom[n]);
                T* d = sB + buf * L::BSLOT + oB + n * BBW;
                d[0] = Bp[n][0];
                d[BCS] = Bp[n][1];
                d[2 * BCS] = Bp[n][2];
                if constexpr (TILE) {
                    const T sn = (p > 0 && p < nz - 1 && in_xy[n]) ? a.dtg * inv : T(0);
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
                    const uint32_t ra = tm0 + (rp * 2 + n) * REC;
                    if constexpr (CW == 16) { tmem::st16(ra, w0); tmem::st16(ra + CW, w1); }
                    else { tmem::st8(ra, w0); tmem::st8(ra + CW, w1); }
                }
            }
        } else if (!TILE && has_node) {
            const T* fr = f1 + ox;
#pragma unroll
            for (int c = 0; c < 3; ++c) x1[0][c] = fr[c * CSX];
        }
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(bar_full + 8u * (uint32_t)buf);      // this warp's part of B(p) is in shared memory
        if (!TILE && pwarp) {
            ptx::named_sync(BAR_A + buf, NW * 32);            // every warp is done with the xi / b planes p
            if (producer) refill(p + R);
        } else {
            ptx::named_arrive(BAR_A + buf, NW * 32);
        }
        // ---------------- F(p-1): finish the plane t = p-1 ----------------
        if (p > first_p) {
            ptx::mbar_wait(bar_full + 8u * (uint32_t)pb, ppar);   // every warp has published B(p-1) (about an iteration ago)
            const int t = p - 1;
            if (TILE && t >= k0) {
                tmem::wait_st();
#pragma unroll
                for (int n = 0; n < NN; ++n) {
                    uint32_t w0[CW], w1[CW];
                    const uint32_t ra = tm0 + ((rp ^ 1u) * 2 + n) * REC;
                    if constexpr (CW == 16) { tmem::ld16(ra, w0); tmem::ld16(ra + CW, w1); }
                    else { tmem::ld8(ra, w0); tmem::ld8(ra + CW, w1); }
                    const T* g = sB + pb * L::BSLOT + oB + n * BBW;
                    T dBi[3], dBj[3], dBk[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const T* gc = g + c * BCS;
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
                    cross_set(c2, c0, n1);
                    cross_set(c0, c1, n2);
                    cross_set(n0, dBi, DJ);
                    cross_acc(n1, dBj, DJ);
                    cross_acc(n2, dBk, DJ);
                    cross_set(DJ, Bc[n], uu);
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
                po += a.plane;
            }
        }
#pragma unroll
        for (int n = 0; n < NN; ++n)
#pragma unroll
            for (int c = 0; c < 3; ++c) { Bm[n][c] = Bc[n][c]; Bc[n][c] = Bp[n][c]; xc[n][c] = x1[n][c]; }
        pb = buf; ppar = cpar;
        if (++buf == NB) { buf = 0; cpar ^= 1u; }
        rp ^= 1u;
        sm2 = sm1; sm1 = s0; s0 = s1; s1 = s2;
        if (s1 == 0) par1 ^= 1u;
        if (++s2 == R) s2 = 0;
    }
  };
  if (tilew) run(std::true_type{});
  else run(std::false_type{});
    if (k1 == nz) {   // the top plane (line-tied) is carried through
#pragma unroll
        for (int n = 0; n < 2; ++n)
            if (st[n]) {
                T* pl = out + (long long)(nz - 1) * a.plane + (long long)(gj0 + n) * a.pitch + gi;
                pl[0] = x1[n][0];
                pl[a.comp] = x1[n][1];
                pl[2 * a.comp] = x1[n][2];
            }
    }
    if (!ok) atomicOr(a.flag, FLAG_NUMERIC);
    tmem::fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem::dealloc<512>(tm_base_s);
}

// ----------------------------------------------------------------------------------------------- host side

constexpr int kS2TY = 16, kS2R = 4, kS2RB = 4, kS2NB = 4;

inline bool build_sym2_plan(StreamPlan* p, const StreamGeom& g, bool f64, void* xi0, void* xi1, void* b, int sm_count,
                           std::string* why)
{
    using Ld = Sym2Layout<double, kS2TY, kS2R, kS2RB, kS2NB>;
    using Lf = Sym2Layout<float, kS2TY, kS2R, kS2RB, kS2NB>;
    p->usable = false;
    p->f64 = f64;
    p->g = g;
    p->xi[0] = xi0;
    p->xi[1] = xi1;
    p->b = b;
    p->name = f64 ? "sym2_tmem_f64" : "sym2_tmem_f32";
    const int bw = f64 ? Ld::BW : Lf::BW;
    if (!encode_map(&p->map_xi[0], f64, xi0, g, bw, kS2TY + 4) || !encode_map(&p->map_xi[1], f64, xi1, g, bw, kS2TY + 4) ||
        !encode_map(&p->map_b, f64, b, g, bw, kS2TY + 2)) {
        *why = "cuTensorMapEncodeTiled failed";
        return false;
    }
    p->tiles_x = (g.nx + Ld::TX - 1) / Ld::TX;
    p->tiles_y = (g.ny + kS2TY - 1) / kS2TY;
    p->smem_bytes = f64 ? Ld::BYTES : Lf::BYTES;
    cudaError_t e = f64 ? cudaFuncSetAttribute(k_step_sym2<double, kS2TY, kS2R, kS2RB, kS2NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem_bytes)
                        : cudaFuncSetAttribute(k_step_sym2<float, kS2TY, kS2R, kS2RB, kS2NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->smem_bytes);
    if (e != cudaSuccess) {
        *why = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e);
        return false;
    }
    choose_chunks(p->tiles_x * p->tiles_y, g.nz, sm_count, &p->nchunks, &p->chunk_len);
    p->usable = true;
    return true;
}

template <typename T>
inline cudaError_t launch_sym2_step(const StreamPlan& p, int cur, T dtg, int* flag, cudaStream_t stream)
{
    using L = Sym2Layout<T, kS2TY, kS2R, kS2RB, kS2NB>;
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
    k_step_sym2<T, kS2TY, kS2R, kS2RB, kS2NB><<<grid, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], p.map_b, static_cast<T*>(p.xi[1 - cur]), a);
    return cudaGetLastError();
}

}  // namespace mr
