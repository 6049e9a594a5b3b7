// mr_stream.cuh -- the fused streaming step kernel for the mimetic operator (S1-S5 in one pass).
//
// Work item = (xy tile of TX x TY nodes, chunk of z-planes).  A CTA of TX*TY threads (one per node of the tile)
// marches along k.  TMA (cp.async.bulk.tensor, 4-D tiled map over [c][k][j][i]) streams, per plane, the box
// (TX+4) x (TY+4) x 1 x 3 of the displacement xi and of the pre-scaled b into shared-memory rings several planes
// ahead; out-of-domain parts of a box are zero-filled by the TMA unit, so domain edges need no address logic.
//
// Per iteration k (one __syncthreads each):
//   1. B(k+1) = dF b / det dF for the tile AND its halo-1 cross, from the xi planes k, k+1, k+2 in shared memory
//      (one-sided second-order differences on faces); stored in a double-buffered shared B plane.  Each thread keeps
//      its own B(k-1), B(k), B(k+1), dF(k), 1/D(k) in registers.
//   2. J(k) = dF chat / D with chat_p = eps_pqr delta_qB . delta_rx (closed form of Eqs. 2.3-2.7): the k-difference
//      of B comes from registers, the i/j-differences from the shared B(k) plane written one iteration earlier.
//   3. u = J x B, xi+ = xi + dt*gamma*u on interior nodes (copy on line-tied boundary nodes), coalesced store.
// B, J and u never touch HBM: the algorithmic traffic is read xi + read b + write xi+ = 9 elements per node.
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
    int tiles_x = 0, tiles_y = 0, nchunks = 0, chunk_len = 0;
    size_t smem_bytes = 0;
};

// ----------------------------------------------------------------------------------------------- PTX wrappers
namespace ptx {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra WAIT_DONE;\n\t"
        "bra WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// 4-D tiled TMA load global -> shared, completion on an mbarrier
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
        : "memory");
}

}  // namespace ptx

// ----------------------------------------------------------------------------------------------- the kernel

template <typename T, int TX, int TY, int R, int RB>
struct StreamLayout {
    // xi / b box: halo 2 in y; in x the halo is widened to 16 bytes (2 doubles / 4 floats) because the TMA unit
    // faults ("illegal instruction") when the innermost start coordinate is not 16-byte aligned in global memory.
    static constexpr int HX = 16 / (int)sizeof(T);
    static constexpr int BW = TX + 2 * HX, BH = TY + 4;
    static constexpr int CS = BW * BH;                  // component stride inside a box
    static constexpr int SLOT = 3 * CS;                 // elements per box
    static constexpr int SLOT_STRIDE = (SLOT * (int)sizeof(T) + 127) / 128 * 128 / (int)sizeof(T);
    static constexpr int BBW = TX + 2, BBH = TY + 2;    // B plane (halo 1)
    static constexpr int BCS = BBW * BBH;
    static constexpr int BSLOT = (3 * BCS * (int)sizeof(T) + 127) / 128 * 128 / (int)sizeof(T);
    static constexpr uint32_t BOX_BYTES = SLOT * sizeof(T);
    static constexpr size_t OFF_X = 0;
    static constexpr size_t OFF_B0 = OFF_X + (size_t)R * SLOT_STRIDE * sizeof(T);
    static constexpr size_t OFF_BB = OFF_B0 + (size_t)RB * SLOT_STRIDE * sizeof(T);
    static constexpr size_t OFF_BAR = OFF_BB + (size_t)2 * BSLOT * sizeof(T);
    static constexpr size_t BYTES = OFF_BAR + (size_t)(R + RB) * 8 + 128;   // +128: manual base alignment
    static constexpr int HALO = 2 * TX + 2 * TY;
};

// un-normalised first difference along an in-plane axis with element stride s at smem offset o
template <typename T>
__device__ __forceinline__ T sdelta(const T* __restrict__ f, int o, int s, int idx, int n)
{
    if (idx == 0) return T(4) * f[o + s] - T(3) * f[o] - f[o + 2 * s];
    if (idx == n - 1) return T(3) * f[o] - T(4) * f[o - s] + f[o - 2 * s];
    return f[o + s] - f[o - s];
}

// B, dF, D, 1/D of one node from the shared xi planes.  kmode: 0 interior (pa = k+1, pb = k-1), 1 low face
// (pa = 1, pb = 2), 2 high face (pa = nz-2, pb = nz-3); pc is the node's own plane.
template <typename T, int BW, int CS>
__device__ __forceinline__ void stream_node(const T* __restrict__ pc, const T* __restrict__ pa, const T* __restrict__ pb,
                                            int kmode, const T* __restrict__ bs, int o, int gi, int gj, int nx, int ny,
                                            const T (&twoh)[3], T (&dF)[3][3], T (&B)[3], T& D, T& inv)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T* f = pc + c * CS;
        dF[c][0] = sdelta(f, o, 1, gi, nx);
        dF[c][1] = sdelta(f, o, BW, gj, ny);
        const T fa = pa[c * CS + o], fb = pb[c * CS + o];
        T dk;
        if (kmode == 0) dk = fa - fb;
        else if (kmode == 1) dk = T(4) * fa - T(3) * f[o] - fb;
        else dk = T(3) * f[o] - T(4) * fa + fb;
        dF[c][2] = dk;
        dF[c][c] += twoh[c];
    }
    D = det3(dF);
    inv = T(1) / D;
    const T b0 = bs[o], b1 = bs[CS + o], b2 = bs[2 * CS + o];
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = (dF[c][0] * b0 + dF[c][1] * b1 + dF[c][2] * b2) * inv;
}

template <typename T, int TX, int TY, int R, int RB>
__global__ void __launch_bounds__(TX* TY, 1)
k_step_stream(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_b, T* __restrict__ out,
              const StreamArgs<T> a)
{
    using L = StreamLayout<T, TX, TY, R, RB>;
    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~(uintptr_t)127);
    T* sx = reinterpret_cast<T*>(smem + L::OFF_X);
    T* sb = reinterpret_cast<T*>(smem + L::OFF_B0);
    T* sB = reinterpret_cast<T*>(smem + L::OFF_BB);
    uint64_t* bar_x = reinterpret_cast<uint64_t*>(smem + L::OFF_BAR);
    uint64_t* bar_b = bar_x + R;

    const int tid = threadIdx.x;
    const int ti = tid % TX, tj = tid / TX;
    const int tile = blockIdx.x % a.ntiles, chunk = blockIdx.x / a.ntiles;
    const int i0 = (tile % a.tiles_x) * TX, j0 = (tile / a.tiles_x) * TY;
    const int k0 = chunk * a.chunk_len, k1 = min(k0 + a.chunk_len, a.nz);
    const int pfirst = max(k0 - 2, 0), plast = min(k1 + 1, a.nz - 1);     // xi planes this item touches
    const int bfirst = max(k0 - 1, 0), blast = min(k1, a.nz - 1);         // planes whose B is formed
    const int gi = i0 + ti, gj = j0 + tj;
    const bool in_dom = gi < a.nx && gj < a.ny;
    const bool in_xy = gi > 0 && gi < a.nx - 1 && gj > 0 && gj < a.ny - 1;
    const T twoh[3] = { a.twoh[0], a.twoh[1], a.twoh[2] };

    // halo node served by this thread (tid < HALO): bottom row, top row, left column, right column
    int hbi = 0, hbj = 0;
    const bool has_halo = tid < L::HALO;
    if (tid < TX) { hbi = tid + 2; hbj = 1; }
    else if (tid < 2 * TX) { hbi = tid - TX + 2; hbj = TY + 2; }
    else if (tid < 2 * TX + TY) { hbi = 1; hbj = tid - 2 * TX + 2; }
    else { hbi = TX + 2; hbj = tid - 2 * TX - TY + 2; }
    const int hgi = i0 + hbi - 2, hgj = j0 + hbj - 2;
    const int own_o = (tj + 2) * L::BW + (ti + L::HX);
    const int halo_o = hbj * L::BW + (hbi - 2 + L::HX);

    int next_x = pfirst, next_b = bfirst;   // next planes to request (thread 0 only)
    if (tid == 0) {
        for (int s = 0; s < R + RB; ++s) ptx::mbar_init(&bar_x[s], 1);
        ptx::fence_mbar_init();
    }
    __syncthreads();
    if (tid == 0) {
        for (; next_x <= plast && next_x - pfirst < R; ++next_x) {
            const int s = (next_x - pfirst) % R;
            ptx::mbar_expect_tx(&bar_x[s], L::BOX_BYTES);
            ptx::tma_load_4d(sx + (size_t)s * L::SLOT_STRIDE, &map_in, i0 - L::HX, j0 - 2, next_x, 0, &bar_x[s]);
        }
        for (; next_b <= blast && next_b - bfirst < RB; ++next_b) {
            const int s = (next_b - bfirst) % RB;
            ptx::mbar_expect_tx(&bar_b[s], L::BOX_BYTES);
            ptx::tma_load_4d(sb + (size_t)s * L::SLOT_STRIDE, &map_b, i0 - L::HX, j0 - 2, next_b, 0, &bar_b[s]);
        }
    }

    int waited_x = pfirst - 1;
    auto ensure_x = [&](int p) {
        while (waited_x < p) {
            ++waited_x;
            const int q = waited_x - pfirst;
            ptx::mbar_wait(&bar_x[q % R], (uint32_t)((q / R) & 1));
        }
    };
    auto xplane = [&](int p) -> const T* { return sx + (size_t)((p - pfirst) % R) * L::SLOT_STRIDE; };

    bool bad = false;
    // forms B(p) for the thread's own node (returned) and, if with_halo, its halo node; writes both to the shared
    // B plane p&1.
    auto form_B = [&](int p, bool with_halo, T(&dF)[3][3], T(&B)[3], T& inv) {
        int kmode = 0, qa = p + 1, qb = p - 1;
        if (p == 0) { kmode = 1; qa = 1; qb = 2; }
        else if (p == a.nz - 1) { kmode = 2; qa = p - 1; qb = p - 2; }
        ensure_x(kmode == 0 ? p + 1 : (kmode == 1 ? 2 : p));
        {
            const int q = p - bfirst;
            ptx::mbar_wait(&bar_b[q % RB], (uint32_t)((q / RB) & 1));
        }
        const T* pc = xplane(p);
        const T* pa = xplane(qa);
        const T* pb = xplane(qb);
        const T* bs = sb + (size_t)((p - bfirst) % RB) * L::SLOT_STRIDE;
        T* Bdst = sB + (size_t)(p & 1) * L::BSLOT;
        T D;
        stream_node<T, L::BW, L::CS>(pc, pa, pb, kmode, bs, own_o, gi, gj, a.nx, a.ny, twoh, dF, B, D, inv);
        if (in_dom && !(D > T(0))) bad = true;
        {
            const int o = (tj + 1) * L::BBW + (ti + 1);
            Bdst[o] = B[0];
            Bdst[L::BCS + o] = B[1];
            Bdst[2 * L::BCS + o] = B[2];
        }
        if (with_halo && has_halo) {
            T hdF[3][3], hB[3], hD, hinv;
            stream_node<T, L::BW, L::CS>(pc, pa, pb, kmode, bs, halo_o, hgi, hgj, a.nx, a.ny, twoh, hdF, hB, hD, hinv);
            const int o = (hbj - 1) * L::BBW + (hbi - 1);
            Bdst[o] = hB[0];
            Bdst[L::BCS + o] = hB[1];
            Bdst[2 * L::BCS + o] = hB[2];
        }
    };

    T Bm[3] = { T(0), T(0), T(0) }, Bc[3], Bp[3] = { T(0), T(0), T(0) };
    T dFc[3][3], dFp[3][3], invc, invp = T(0);
    if (k0 > 0) {
        T dFt[3][3], it;
        form_B(k0 - 1, false, dFt, Bm, it);
    }
    form_B(k0, true, dFc, Bc, invc);
    __syncthreads();

    for (int k = k0; k < k1; ++k) {
        if (k + 1 <= a.nz - 1) form_B(k + 1, true, dFp, Bp, invp);

        // ---- J(k), u, update of the own node ----
        const T* pc = xplane(k);
        T o3[3] = { pc[own_o], pc[L::CS + own_o], pc[2 * L::CS + own_o] };
        if (in_xy && k > 0 && k < a.nz - 1) {
            const T* Bs = sB + (size_t)(k & 1) * L::BSLOT;
            const int o = (tj + 1) * L::BBW + (ti + 1);
            T dB[3][3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                dB[0][c] = Bs[c * L::BCS + o + 1] - Bs[c * L::BCS + o - 1];
                dB[1][c] = Bs[c * L::BCS + o + L::BBW] - Bs[c * L::BCS + o - L::BBW];
                dB[2][c] = Bp[c] - Bm[c];
            }
            T J[3], u[3];
            mimetic_J(dFc, dB, invc, J);
            cross3(J, Bc, u);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                o3[c] += a.dtg * u[c];
                bad = bad || !(fabs(o3[c]) < T(1e30));
            }
        }
        if (in_dom) {
            const long long p = (long long)k * a.plane + (long long)gj * a.pitch + gi;
            out[p] = o3[0];
            out[a.comp + p] = o3[1];
            out[2 * a.comp + p] = o3[2];
        }
        __syncthreads();
        // xi plane k-1 and b plane k+1 are dead now: refill their slots
        if (tid == 0) {
            for (; next_x <= plast && next_x - R <= k - 1; ++next_x) {
                const int s = (next_x - pfirst) % R;
                ptx::mbar_expect_tx(&bar_x[s], L::BOX_BYTES);
                ptx::tma_load_4d(sx + (size_t)s * L::SLOT_STRIDE, &map_in, i0 - L::HX, j0 - 2, next_x, 0, &bar_x[s]);
            }
            for (; next_b <= blast && next_b - RB <= k + 1; ++next_b) {
                const int s = (next_b - bfirst) % RB;
                ptx::mbar_expect_tx(&bar_b[s], L::BOX_BYTES);
                ptx::tma_load_4d(sb + (size_t)s * L::SLOT_STRIDE, &map_b, i0 - L::HX, j0 - 2, next_b, 0, &bar_b[s]);
            }
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Bm[c] = Bc[c];
            Bc[c] = Bp[c];
#pragma unroll
            for (int q = 0; q < 3; ++q) dFc[c][q] = dFp[c][q];
        }
        invc = invp;
    }
    if (bad) atomicOr(a.flag, FLAG_NUMERIC);
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

constexpr int kTX = 32, kTY = 16, kR = 6, kRB = 4;

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
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
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
    return cudaFuncSetAttribute(k_step_stream<T, kTX, kTY, kR, kRB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

inline bool build_stream_plan(StreamPlan* p, const StreamGeom& g, bool f64, void* xi0, void* xi1, void* b, int sm_count,
                              std::string* why)
{
    p->usable = false;
    p->f64 = f64;
    p->g = g;
    p->xi[0] = xi0;
    p->xi[1] = xi1;
    p->name = f64 ? "stream_tma_f64_32x16" : "stream_tma_f32_32x16";
    const int bw = f64 ? StreamLayout<double, kTX, kTY, kR, kRB>::BW : StreamLayout<float, kTX, kTY, kR, kRB>::BW;
    if (!encode_map(&p->map_xi[0], f64, xi0, g, bw, kTY + 4) || !encode_map(&p->map_xi[1], f64, xi1, g, bw, kTY + 4) ||
        !encode_map(&p->map_b, f64, b, g, bw, kTY + 4)) {
        *why = "cuTensorMapEncodeTiled failed";
        return false;
    }
    p->tiles_x = (g.nx + kTX - 1) / kTX;
    p->tiles_y = (g.ny + kTY - 1) / kTY;
    p->smem_bytes = f64 ? StreamLayout<double, kTX, kTY, kR, kRB>::BYTES : StreamLayout<float, kTX, kTY, kR, kRB>::BYTES;
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
    k_step_stream<T, kTX, kTY, kR, kRB><<<grid, kTX * kTY, p.smem_bytes, stream>>>(p.map_xi[cur], p.map_b,
                                                                                 static_cast<T*>(p.xi[1 - cur]), a);
    return cudaGetLastError();
}

}  // namespace mr
