// mr_stream.cuh -- the fused streaming step kernel for the mimetic operator (S1-S5 in one pass).
//
// Work item = (xy tile of TX x TY nodes, chunk of z-planes).  A CTA marches along k.  TMA (cp.async.bulk.tensor,
// 4-D tiled maps over [c][k][j][i]) streams, per plane, the box (TX+2HX) x (TY+4) x 1 x 3 of the displacement xi
// and the box (TX+2HX) x (TY+2) x 1 x 3 of the pre-scaled b into shared-memory rings several planes ahead;
// out-of-domain parts of a box are zero-filled by the TMA unit, so domain edges need no address logic.
//
// Warp roles (TX = 32, one warp = one row of the tile):
//   tile warps 0..TY-1   one node per thread; the thread keeps its own column's xi(k), xi(k+1), xi(k+2), B(k-1), B(k),
//                        B(k+1), dF(k), 1/D(k) in registers (the k-neighbours never come from shared memory);
//   ring warps TY..TY+3  the halo-1 ring of the tile (row below, row above, left column, right column): only the
//                        push-forward B of those nodes is formed, so that the tile warps all carry the same load;
//                        warp counts are kept a multiple of 4 (registers are per SM sub-partition).
// Per iteration k (one bar.sync):
//   A. B(k+1) = dF b / det dF (Eq. 2.1) at every tile and ring node from the xi plane k+1 in shared memory and the
//      own column registers; one-sided second-order differences on faces sit in rarely taken branches.  B(k+1) goes
//      to a double-buffered shared plane.
//   B. tile warps: J(k) = dF chat / D with chat_p = eps_pqr delta_qB . delta_rx (closed form of Eqs. 2.3-2.7): the
//      k-difference of B from registers, the i/j-differences from the shared B(k) plane; u = J x B,
//      xi+ = xi + dt*gamma*u on interior nodes (copy on line-tied boundary nodes), coalesced store.
// B, J and u never touch HBM: the algorithmic traffic is read xi + read b + write xi+ = 9 elements per node.
// The k loop is unrolled six times so that the rotating register sets (period 3 and 2) need no moves.
#pragma once
#include <cuda.h>

#include <algorithm>
#include <cstring>
#include <string>

#include "mr_common.cuh"

namespace mr {

struct StreamGeom {
    int nx, ny, nz, pitch;
    long long plane, comp;
    double twoh[3];
};

template <typename T>
struct StreamArgs {
    int nx, ny, nz;
    int pitch;
    long long plane, comp;
    T twoh[3];
    T dtg;
    int tiles_x, ntiles, chunk_len;
    int* flag;
};

struct StreamPlan {
    bool usable = false;
    bool f64 = true;
    const char* name = "stream";
    std::string why;
    StreamGeom g{};
    CUtensorMap map_xi[2];
    CUtensorMap map_b;
    void* xi[2] = { nullptr, nullptr };
    const void* b = nullptr;
    int tiles_x = 0, tiles_y = 0, nchunks = 0, chunk_len = 0;
    size_t smem_bytes = 0;
};

// ----------------------------------------------------------------------------------------------- PTX wrappers
namespace ptx {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra WAIT_DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
// 4-D tiled TMA load global -> shared, completion on an mbarrier
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(dst),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0;" ::: "memory"); }

}  // namespace ptx

// ----------------------------------------------------------------------------------------------- per-type helpers

// 1/d to about one ulp: hardware seed (2^-23) and two Newton steps (double), rounded reciprocal (float)
__device__ __forceinline__ double fast_rcp(double d)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    double e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    e = fma(-d, r, 1.0);
    return fma(r, e, r);
}
__device__ __forceinline__ float fast_rcp(float d) { return __frcp_rn(d); }

// d > 0 and finite, decided on the bit pattern (integer pipe, keeps the FP64 pipe free)
__device__ __forceinline__ bool positive_finite(double d) { return (unsigned)(__double2hiint(d) - 1) < 0x7fefffffu; }
__device__ __forceinline__ bool positive_finite(float d) { return (__float_as_uint(d) - 1u) < 0x7f7fffffu; }
__device__ __forceinline__ bool is_finite(double d) { return ((unsigned)__double2hiint(d) & 0x7fffffffu) < 0x7ff00000u; }
__device__ __forceinline__ bool is_finite(float d) { return (__float_as_uint(d) & 0x7fffffffu) < 0x7f800000u; }

// ----------------------------------------------------------------------------------------------- the kernel

template <typename T, int TX, int TY, int R, int RB>
struct StreamLayout {
    static_assert(TX == 32, "one warp owns one tile row");
    static_assert(TY >= 8 && TY <= 32 && R >= 4 && RB >= 2, "tile / ring sizes");
    // halo 2 in y for xi, halo 1 for b; in x the halo is widened to 16 bytes (2 doubles / 4 floats) because the
    // TMA unit faults when the innermost start coordinate is not 16-byte aligned in global memory.
    static constexpr int HX = 16 / (int)sizeof(T);
    static constexpr int BW = TX + 2 * HX;
    static constexpr int XH = TY + 4, BH = TY + 2;
    static constexpr int CSX = BW * XH, CSB = BW * BH;      // component strides inside the boxes
    static constexpr int round128(int bytes) { return (bytes + 127) / 128 * 128; }
    static constexpr int SLOTX = round128(3 * CSX * (int)sizeof(T)) / (int)sizeof(T);   // slot strides (elements)
    static constexpr int SLOTB = round128(3 * CSB * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr uint32_t XBOX_BYTES = 3u * CSX * sizeof(T), BBOX_BYTES = 3u * CSB * sizeof(T);
    static constexpr int BBW = TX + 2, BBH = TY + 2;        // shared B plane (halo 1)
    static constexpr int BCS = BBW * BBH;
    static constexpr int BSLOT = round128(3 * BCS * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr int NWARPS = TY + 4, NTHREADS = NWARPS * 32;
    static constexpr size_t OFF_X = 0;
    static constexpr size_t OFF_B0 = OFF_X + (size_t)R * SLOTX * sizeof(T);
    static constexpr size_t OFF_BB = OFF_B0 + (size_t)RB * SLOTB * sizeof(T);
    static constexpr size_t OFF_BAR = OFF_BB + (size_t)2 * BSLOT * sizeof(T);
    static constexpr size_t BYTES = OFF_BAR + (size_t)(R + RB) * 8 + 128;   // +128: base alignment slack
};

// Stage A at one node: dF (un-normalised Jacobian), 1/D and B = dF b / D (Eq. 2.1).
//   f    : the node's position in component 0 of the xi plane it lives on (shared memory),
//   dk   : the k-direction differences, formed by the caller (central or one-sided),
//   edge : bit 0/1 node on the low/high x face, bit 2/3 low/high y face,
//   bs   : the node's position in component 0 of the b plane.
template <typename T, int BW, int CSX, int CSB>
__device__ __forceinline__ void stage_A(const T* __restrict__ f, const T (&dk)[3], unsigned edge,
                                        const T* __restrict__ bs, const T (&twoh)[3], T (&dF)[3][3], T (&B)[3], T& inv,
                                        bool& ok)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        dF[c][0] = f[c * CSX + 1] - f[c * CSX - 1];
        dF[c][1] = f[c * CSX + BW] - f[c * CSX - BW];
        dF[c][2] = dk[c];
    }
    if (edge) {   // a face node: second-order one-sided difference normal to the face (reading Q3)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const T xc = f[c * CSX];
            if (edge & 1u) dF[c][0] = T(4) * f[c * CSX + 1] - T(3) * xc - f[c * CSX + 2];
            if (edge & 2u) dF[c][0] = T(3) * xc - T(4) * f[c * CSX - 1] + f[c * CSX - 2];
            if (edge & 4u) dF[c][1] = T(4) * f[c * CSX + BW] - T(3) * xc - f[c * CSX + 2 * BW];
            if (edge & 8u) dF[c][1] = T(3) * xc - T(4) * f[c * CSX - BW] + f[c * CSX - 2 * BW];
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) dF[c][c] += twoh[c];
    const T D = det3(dF);
    ok = ok && positive_finite(D);
    inv = fast_rcp(D);
    const T b0 = bs[0] * inv, b1 = bs[CSB] * inv, b2 = bs[2 * CSB] * inv;
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = dF[c][0] * b0 + dF[c][1] * b1 + dF[c][2] * b2;
}

// Stage B at one interior node: xi += s * (dF chat) x B with s = dt*gamma/D (closed form of Eqs. 2.3-2.7, Eq. 1.5).
template <typename T, int BBW, int BCS>
__device__ __forceinline__ void stage_B(const T* __restrict__ Bs, const T (&Bm)[3], const T (&Bc)[3], const T (&Bp)[3],
                                        const T (&dF)[3][3], T s, T (&x)[3])
{
    T dB[3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        dB[0][c] = Bs[c * BCS + 1] - Bs[c * BCS - 1];
        dB[1][c] = Bs[c * BCS + BBW] - Bs[c * BCS - BBW];
        dB[2][c] = Bp[c] - Bm[c];
    }
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
#pragma unroll
    for (int c = 0; c < 3; ++c) x[c] += s * u[c];
}

template <typename T, int TX, int TY, int R, int RB, bool KEEPX>
__global__ void __launch_bounds__((TY + 4) * 32, 1)
k_step_stream(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_b, T* __restrict__ out,
              const StreamArgs<T> a)
{
    using L = StreamLayout<T, TX, TY, R, RB>;
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

    // ---- TMA producer: lane 0 of the last ring warp; a slot is refilled once its plane is dead ----
    const bool producer = tid == (TY + 3) * 32;
    int next_x = pfirst, next_b = bfirst;
    auto refill = [&](int dead_x, int dead_b) {
        for (; next_x <= plast && next_x - R <= dead_x; ++next_x) {
            const uint32_t s = (uint32_t)((next_x - pfirst) % R);
            ptx::mbar_expect_tx(bar_x + 8u * s, L::XBOX_BYTES);
            ptx::tma_load_4d(sx_u32 + s * (uint32_t)(L::SLOTX * sizeof(T)), &map_in, i0 - L::HX, j0 - 2, next_x, 0, bar_x + 8u * s);
        }
        for (; next_b <= blast && next_b - RB <= dead_b; ++next_b) {
            const uint32_t s = (uint32_t)((next_b - bfirst) % RB);
            ptx::mbar_expect_tx(bar_b + 8u * s, L::BBOX_BYTES);
            ptx::tma_load_4d(sb_u32 + s * (uint32_t)(L::SLOTB * sizeof(T)), &map_b, i0 - L::HX, j0 - 1, next_b, 0, bar_b + 8u * s);
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

    // node of this thread: tile warps own one tile node, the four ring warps the halo-1 ring (row below, row above,
    // left column, right column; the upper lanes of the column warps repeat the lower ones)
    int ti, tj;
    if (warp < TY) { ti = lane; tj = warp; }
    else if (warp == TY) { ti = lane; tj = -1; }
    else if (warp == TY + 1) { ti = lane; tj = TY; }
    else if (warp == TY + 2) { ti = -1; tj = lane % TY; }
    else { ti = TX; tj = lane % TY; }
    const int gi = i0 + ti, gj = j0 + tj;
    const int ox = (tj + 2) * L::BW + (ti + L::HX);       // offsets inside the xi box, the b box, the shared B plane
    const int ob = (tj + 1) * L::BW + (ti + L::HX);
    const int oB = (tj + 1) * L::BBW + (ti + 1);
    const bool in_dom = gi >= 0 && gi < a.nx && gj >= 0 && gj < a.ny;
    const unsigned edge = !in_dom ? 0u
        : (gi == 0 ? 1u : 0u) | (gi == a.nx - 1 ? 2u : 0u) | (gj == 0 ? 4u : 0u) | (gj == a.ny - 1 ? 8u : 0u);

    // stage A of plane p with every operand from shared memory (prologue only; handles the one-sided k faces)
    auto A_from_smem = [&](int p, T(&dF)[3][3], T(&B)[3], T& inv, bool& ok) {
        const T* pc = xplane(p) + ox;
        T dk[3];
        if (p == 0) {
            const T* p1 = xplane(1) + ox;
            const T* p2 = xplane(2) + ox;
#pragma unroll
            for (int c = 0; c < 3; ++c) dk[c] = T(4) * p1[c * L::CSX] - T(3) * pc[c * L::CSX] - p2[c * L::CSX];
        } else if (p == nz - 1) {
            const T* p1 = xplane(p - 1) + ox;
            const T* p2 = xplane(p - 2) + ox;
#pragma unroll
            for (int c = 0; c < 3; ++c) dk[c] = T(3) * pc[c * L::CSX] - T(4) * p1[c * L::CSX] + p2[c * L::CSX];
        } else {
            const T* p1 = xplane(p + 1) + ox;
            const T* p2 = xplane(p - 1) + ox;
#pragma unroll
            for (int c = 0; c < 3; ++c) dk[c] = p1[c * L::CSX] - p2[c * L::CSX];
        }
        stage_A<T, L::BW, L::CSX, L::CSB>(pc, dk, edge, bplane(p) + ob, twoh, dF, B, inv, ok);
    };
    auto store_B = [&](int p, const T(&B)[3]) {
        T* d = sB + (p & 1) * L::BSLOT + oB;
        d[0] = B[0];
        d[L::BCS] = B[1];
        d[2 * L::BCS] = B[2];
    };

    bool ok = true;
    // running ring positions of the xi planes k, k+1, k+2 and the b plane k+1 of the main loop
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
    // k-differences of plane k+1 (k+1 <= nz-1): central x2 - x0, or one-sided on the top face
    // 3 f(nz-1) - 4 f(nz-2) + f(nz-3) (plane nz-3 is still in its slot: nothing is loaded beyond plane nz-1).
    // With KEEPX the own column values x0 = xi(k), x1 = xi(k+1) live in registers and x2 = xi(k+2) is read here;
    // without it x0 is (re)read from shared memory too.
    auto column_dk = [&](int k, T(&x0)[3], const T(&x1)[3], T(&x2)[3], T(&dk)[3]) {
        if (!KEEPX) {
            const T* p0 = sx + sl0 * L::SLOTX + ox;
#pragma unroll
            for (int c = 0; c < 3; ++c) x0[c] = p0[c * L::CSX];
        }
        if (k + 2 <= nz - 1) {
            ptx::mbar_wait(bar_x + 8u * (uint32_t)sl2, par2);
            const T* p2 = sx + sl2 * L::SLOTX + ox;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                x2[c] = p2[c * L::CSX];
                dk[c] = x2[c] - x0[c];
            }
        } else {
            const T* pm = xplane(k - 1) + ox;
            const T* p1 = sx + sl1 * L::SLOTX + ox;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                x2[c] = T(0);
                dk[c] = T(3) * (KEEPX ? x1[c] : p1[c * L::CSX]) - T(4) * x0[c] + pm[c * L::CSX];
            }
        }
    };
    constexpr int DEADLAG = KEEPX ? 1 : 0;    // after iteration k the xi planes <= k + DEADLAG are dead

    if (warp < TY) {
        // =========================================== tile warps ===========================================
        const bool in_xy = gi > 0 && gi < a.nx - 1 && gj > 0 && gj < a.ny - 1;
        T X[3][3];       // own xi at planes k, k+1, k+2 (rotating; only X[0] is used without KEEPX)
        T Bq[3][3];      // own B at planes k-1, k, k+1 (rotating)
        T dFq[2][3][3];  // dF at planes k, k+1 (rotating)
        T invq[2];
        {
            const T* pa = xplane(k0) + ox;
            const T* pb = xplane(min(k0 + 1, nz - 1)) + ox;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                X[0][c] = pa[c * L::CSX];
                X[1][c] = pb[c * L::CSX];
                X[2][c] = T(0);
                Bq[0][c] = T(0);
                Bq[2][c] = T(0);
            }
            if (k0 > 0) {
                T dFt[3][3], it;
                A_from_smem(k0 - 1, dFt, Bq[0], it, ok);
            }
            A_from_smem(k0, dFq[0], Bq[1], invq[0], ok);
            store_B(k0, Bq[1]);
            invq[1] = T(0);
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int q = 0; q < 3; ++q) dFq[1][c][q] = T(0);
        }
        ptx::cta_sync();
        T* po = out + (long long)k0 * a.plane + (long long)gj * a.pitch + gi;
        const bool in_store = gi < a.nx && gj < a.ny;

        for (int kb = k0; kb < k1; kb += 6) {
#pragma unroll
            for (int u = 0; u < 6; ++u) {
                const int k = kb + u;
                if (k >= k1) break;
                T(&x0)[3] = X[KEEPX ? u % 3 : 0];
                T(&x1)[3] = X[KEEPX ? (u + 1) % 3 : 1];
                T(&x2)[3] = X[KEEPX ? (u + 2) % 3 : 2];
                T(&Bm)[3] = Bq[u % 3];
                T(&Bc)[3] = Bq[(u + 1) % 3];
                T(&Bp)[3] = Bq[(u + 2) % 3];
                if (k + 1 <= nz - 1) {
                    T dk[3];
                    column_dk(k, x0, x1, x2, dk);
                    ptx::mbar_wait(bar_b + 8u * (uint32_t)slb, parb);
                    stage_A<T, L::BW, L::CSX, L::CSB>(sx + sl1 * L::SLOTX + ox, dk, edge, sb + slb * L::SLOTB + ob, twoh,
                                                      dFq[(u + 1) % 2], Bp, invq[(u + 1) % 2], ok);
                    store_B(k + 1, Bp);
                } else if (!KEEPX) {
                    const T* p0 = sx + sl0 * L::SLOTX + ox;
#pragma unroll
                    for (int c = 0; c < 3; ++c) x0[c] = p0[c * L::CSX];
                }
                if (in_xy && k > 0 && k < nz - 1) {
                    stage_B<T, L::BBW, L::BCS>(sB + (k & 1) * L::BSLOT + oB, Bm, Bc, Bp, dFq[u % 2], a.dtg * invq[u % 2], x0);
                    ok = ok && is_finite(x0[0]) && is_finite(x0[1]) && is_finite(x0[2]);
                }
                if (in_store) {
                    po[0] = x0[0];
                    po[a.comp] = x0[1];
                    po[2 * a.comp] = x0[2];
                }
                po += a.plane;
                ptx::cta_sync();
                advance();
            }
        }
    } else {
        // =========================================== ring warps ===========================================
        T X[3][3];   // own xi at planes k, k+1, k+2 (rotated by moves)
        {
            const T* pa = xplane(k0) + ox;
            const T* pb = xplane(min(k0 + 1, nz - 1)) + ox;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                X[0][c] = pa[c * L::CSX];
                X[1][c] = pb[c * L::CSX];
                X[2][c] = T(0);
            }
            T dF[3][3], B[3], inv;
            A_from_smem(k0, dF, B, inv, ok);
            store_B(k0, B);
        }
        ptx::cta_sync();
        if (producer) refill(k0 - 1 + DEADLAG, k0);
        for (int k = k0; k < k1; ++k) {
            if (k + 1 <= nz - 1) {
                T dk[3], dF[3][3], B[3], inv;
                column_dk(k, X[0], X[1], X[2], dk);
                ptx::mbar_wait(bar_b + 8u * (uint32_t)slb, parb);
                stage_A<T, L::BW, L::CSX, L::CSB>(sx + sl1 * L::SLOTX + ox, dk, edge, sb + slb * L::SLOTB + ob, twoh, dF, B, inv, ok);
                store_B(k + 1, B);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    X[0][c] = X[1][c];
                    X[1][c] = X[2][c];
                }
            }
            ptx::cta_sync();
            // xi planes <= k + DEADLAG and b planes <= k+1 are dead now: refill their slots
            if (producer) refill(k + DEADLAG, k + 1);
            advance();
        }
    }
    if (!ok) atomicOr(a.flag, FLAG_NUMERIC);
}

// ----------------------------------------------------------------------------------------------- host side

typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline PFN_encodeTiled get_encode_fn()
{
    static PFN_encodeTiled fn = nullptr;
    if (fn) return fn;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess || !p) return nullptr;
    fn = reinterpret_cast<PFN_encodeTiled>(p);
    return fn;
}

constexpr int kTX = 32, kTY = 16, kR = 6, kRB = 3;
constexpr bool kKEEPX = false;

#ifndef MR_L2_PROMOTION
#define MR_L2_PROMOTION CU_TENSOR_MAP_L2_PROMOTION_L2_256B
#endif
inline bool encode_map(CUtensorMap* m, bool f64, void* base, const StreamGeom& g, int bw, int bh)
{
    PFN_encodeTiled enc = get_encode_fn();
    if (!enc) return false;
    const cuuint64_t es = f64 ? 8 : 4;
    cuuint64_t dims[4] = { (cuuint64_t)g.nx, (cuuint64_t)g.ny, (cuuint64_t)g.nz, 3 };
    cuuint64_t strides[3] = { (cuuint64_t)g.pitch * es, (cuuint64_t)g.plane * es, (cuuint64_t)g.comp * es };
    cuuint32_t box[4] = { (cuuint32_t)bw, (cuuint32_t)bh, 1, 3 };
    cuuint32_t estr[4] = { 1, 1, 1, 1 };
    CUresult r = enc(m, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, MR_L2_PROMOTION,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// choose the number of z-chunks: minimise waves * (chunk_len + restart overhead) over the concurrent CTA slots
inline void choose_chunks(int ntiles, int nz, int slots, int* nchunks, int* chunk_len)
{
    double best = 1e300;
    int bc = 1;
    const int maxc = std::max(1, nz / 4);
    for (int c = 1; c <= maxc; ++c) {
        const int len = (nz + c - 1) / c;
        const int cc = (nz + len - 1) / len;              // chunks actually produced by this length
        const long long items = (long long)ntiles * cc;
        const long long waves = (items + slots - 1) / slots;
        const double cost = (double)waves * (len + 3.0);
        if (cost < best - 1e-9) { best = cost; bc = cc; }
    }
    *nchunks = bc;
    *chunk_len = (nz + bc - 1) / bc;
    *nchunks = (nz + *chunk_len - 1) / *chunk_len;
}

template <typename T>
inline cudaError_t stream_set_smem(size_t bytes)
{
    return cudaFuncSetAttribute(k_step_stream<T, kTX, kTY, kR, kRB, kKEEPX>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

inline bool build_stream_plan(StreamPlan* p, const StreamGeom& g, bool f64, void* xi0, void* xi1, void* b, int sm_count,
                              std::string* why)
{
    using Ld = StreamLayout<double, kTX, kTY, kR, kRB>;
    using Lf = StreamLayout<float, kTX, kTY, kR, kRB>;
    p->usable = false;
    p->f64 = f64;
    p->g = g;
    p->xi[0] = xi0;
    p->xi[1] = xi1;
    p->name = f64 ? "stream_tma_f64_32x16" : "stream_tma_f32_32x16";
    const int bw = f64 ? Ld::BW : Lf::BW;
    if (!encode_map(&p->map_xi[0], f64, xi0, g, bw, kTY + 4) || !encode_map(&p->map_xi[1], f64, xi1, g, bw, kTY + 4) ||
        !encode_map(&p->map_b, f64, b, g, bw, kTY + 2)) {
        *why = "cuTensorMapEncodeTiled failed";
        return false;
    }
    p->tiles_x = (g.nx + kTX - 1) / kTX;
    p->tiles_y = (g.ny + kTY - 1) / kTY;
    p->smem_bytes = f64 ? Ld::BYTES : Lf::BYTES;
    cudaError_t e = f64 ? stream_set_smem<double>(p->smem_bytes) : stream_set_smem<float>(p->smem_bytes);
    if (e != cudaSuccess) {
        *why = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e);
        return false;
    }
    choose_chunks(p->tiles_x * p->tiles_y, g.nz, sm_count, &p->nchunks, &p->chunk_len);
    p->usable = true;
    return true;
}

template <typename T>
inline cudaError_t launch_stream_step(const StreamPlan& p, int cur, T dtg, int* flag, cudaStream_t stream)
{
    using L = StreamLayout<T, kTX, kTY, kR, kRB>;
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
    k_step_stream<T, kTX, kTY, kR, kRB, kKEEPX><<<grid, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], p.map_b,
                                                                                   static_cast<T*>(p.xi[1 - cur]), a);
    return cudaGetLastError();
}

}  // namespace mr
