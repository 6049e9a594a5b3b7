// mr_stream_common.cuh -- what the streaming (TMA-fed) step kernels of libmr.so share: the launch-plan structs, the PTX
// wrappers (mbarrier, cp.async.bulk.tensor, named barriers), the per-type scalar helpers, the per-node pieces of the
// arithmetic (one-sided face differences, area vector + push-forward, cross products) and the host-side tensor-map
// encoding and z-chunking.  Work item of every streaming kernel = (xy tile of 32 x 16 nodes, chunk of z-planes): a CTA
// marches along k while the TMA unit streams, per plane, the box of the displacement xi and of the pre-scaled b (4-D
// tiled maps over [c][k][j][i]) into shared-memory rings; out-of-domain parts of a box are zero-filled by the TMA
// unit, so line-tied domain edges need no address logic.  A periodic axis (Eqs. 2.12-2.14) carries ghost layers in the
// padded array itself (mr_api.cu keeps them equal to the wrapped nodes, k_wrap): the maps span the padded extent, the box
// coordinates are shifted by the ghost width, and a box over the edge reads the neighbours through the wrap.
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
    int ghost[3];         // ghost layers in front of (and behind) the nodes of a periodic axis, 0 on a line-tied one
    int per[3];
    long long shift() const { return (long long)ghost[2] * plane + (long long)ghost[1] * pitch + ghost[0]; }   // node (0,0,0)
};

template <typename T>
struct StreamArgs {
    int nx, ny, nz;
    int pitch;
    long long plane, comp;
    T twoh[3];
    T dtg;
    int tiles_x, ntiles, chunk_len;
    int jorg;             // row of the first tile: 1 when the line-tied face row j = 0 is left to the halo ring (see Tiling)
    int ox, oy, oz;       // box coordinate of the node (0, 0, 0) in the tensor maps (= the ghost widths)
    int per;              // bit a: axis a is periodic (no face, no one-sided difference, every node an inner point)
    int* flag;
    void* partials;       // MODE_STEPDIAG: where the per-CTA partials of S6 go (the step's output is `out`)
};

// How the xy plane is cut into tiles.  `all`: every node is a tile node (what S6 needs: it sums over all of them).  `step`:
// the nodes on LINE-TIED faces never move and both state buffers hold their zero displacement for good, so a step (or a
// right-hand side) need not own them: the tiles start at row 1, and a face that falls exactly one node past the last tile is
// served by that tile's halo ring (mimetic) or by nobody (direct).  On the paper's grids of 2^m + 1 nodes that is 4 x 8 tiles
// instead of 5 x 9 (129^2), 2 x 4 instead of 3 x 5 (65^2), 1 x 2 instead of 2 x 3 (33^2).
struct Tiling {
    int tiles_x = 0, tiles_y = 0, nchunks = 0, chunk_len = 0, jorg = 0;
};

struct StreamPlan {
    bool usable = false;
    bool f64 = true;
    const char* name = "stream";
    std::string why;
    StreamGeom g{};
    CUtensorMap map_xi[3];      // the two state buffers and, once bound, the stage buffer of the adaptive integrator
    CUtensorMap map_b;
    void* xi[3] = { nullptr, nullptr, nullptr };
    const void* b = nullptr;
    Tiling all, step;
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

// ----------------------------------------------------------------------------------------------- more PTX wrappers
namespace ptx {
__device__ __forceinline__ void named_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void mbar_arrive(uint32_t bar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory"); }
__device__ __forceinline__ void named_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }
}  // namespace ptx

// ----------------------------------------------------------------------------------------------- per-node arithmetic

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

// The A-warp's share of stage A at one node: dF comes in without the 2h diagonal and leaves with it; n_0 = dF_1 x dF_2
// (area vector of the jk index surface, Eqs. 2.5/2.6), D = det dF = dF_0 . n_0, inv = 1/D, B = dF b / D (Eq. 2.1).
// n_1 and n_2 are formed by the F-warp from the columns of dF.
template <typename T, int CSB>
__device__ __forceinline__ void duo_push(T (&dF)[3][3], const T* __restrict__ bs, const T (&twoh)[3], T (&n0)[3], T (&B)[3], T& inv,
                                         bool& ok, bool in_dom)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) dF[c][c] += twoh[c];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        n0[c] = dF[c1][1] * dF[c2][2] - dF[c2][1] * dF[c1][2];
    }
    const T D = dF[0][0] * n0[0] + dF[1][0] * n0[1] + dF[2][0] * n0[2];
    ok = ok && (positive_finite(D) || !in_dom);
    inv = fast_rcp(D);
    // dF b first, the division last: the nine products do not wait for the reciprocal's Newton chain
    const T b0 = bs[0], b1 = bs[CSB], b2 = bs[2 * CSB];
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = (dF[c][0] * b0 + dF[c][1] * b1 + dF[c][2] * b2) * inv;
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


#ifndef MR_L2_PROMOTION
#define MR_L2_PROMOTION CU_TENSOR_MAP_L2_PROMOTION_L2_256B
#endif
inline bool encode_map(CUtensorMap* m, bool f64, void* base, const StreamGeom& g, int bw, int bh)
{
    PFN_encodeTiled enc = get_encode_fn();
    if (!enc) return false;
    const cuuint64_t es = f64 ? 8 : 4;
    // `base` is the start of the padded array (the ghost layers of a periodic axis included)
    cuuint64_t dims[4] = { (cuuint64_t)(g.nx + 2 * g.ghost[0]), (cuuint64_t)(g.ny + 2 * g.ghost[1]), (cuuint64_t)(g.nz + 2 * g.ghost[2]), 3 };
    cuuint64_t strides[3] = { (cuuint64_t)g.pitch * es, (cuuint64_t)g.plane * es, (cuuint64_t)g.comp * es };
    cuuint32_t box[4] = { (cuuint32_t)bw, (cuuint32_t)bh, 1, 3 };
    cuuint32_t estr[4] = { 1, 1, 1, 1 };
    CUresult r = enc(m, f64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base, dims, strides, box, estr,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, MR_L2_PROMOTION,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// the real-node base of a padded array whose storage starts at `raw`
inline void* node_base(void* raw, const StreamGeom& g, bool f64)
{
    return static_cast<char*>(raw) + (size_t)g.shift() * (f64 ? 8 : 4);
}

// choose the number of z-chunks: minimise waves * (chunk_len + restart overhead) over the concurrent CTA slots
inline void choose_chunks(int ntiles, int nz, int slots, int* nchunks, int* chunk_len)
{
    double best = 1e300;
    int bc = 1;
    const int maxc = nz;      // down to one plane per chunk: a grid of a few tiles is bound by the latency of a CTA's march, and
                              // the three planes of restart overhead cost nothing while SMs are idle (C1: 11.4 -> 8.4 us per step)
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


// the two tilings of a plan: tx / ty = tile size, ring = the kernel forms B on the halo-1 ring of a tile (mimetic)
inline void choose_tilings(StreamPlan* p, int tx, int ty, bool ring, int sm_count)
{
    const StreamGeom& g = p->g;
    p->all.tiles_x = (g.nx + tx - 1) / tx;
    p->all.tiles_y = (g.ny + ty - 1) / ty;
    p->all.jorg = 0;
    p->step = p->all;
    if (!g.per[0]) {
        if (ring) { if ((g.nx - 1) % tx == 0) p->step.tiles_x = (g.nx - 1) / tx; }
        else p->step.tiles_x = (g.nx - 1 + tx - 1) / tx;
    }
    if (!g.per[1] && (g.ny - 2 + ty - 1) / ty < p->all.tiles_y) {
        p->step.tiles_y = (g.ny - 2 + ty - 1) / ty;
        p->step.jorg = 1;
    }
    choose_chunks(p->all.tiles_x * p->all.tiles_y, g.nz, sm_count, &p->all.nchunks, &p->all.chunk_len);
    choose_chunks(p->step.tiles_x * p->step.tiles_y, g.nz, sm_count, &p->step.nchunks, &p->step.chunk_len);
}

template <typename T>
inline StreamArgs<T> stream_args(const StreamPlan& p, const Tiling& t, T dtg, int* flag)
{
    StreamArgs<T> a;
    a.nx = p.g.nx; a.ny = p.g.ny; a.nz = p.g.nz;
    a.pitch = p.g.pitch; a.plane = p.g.plane; a.comp = p.g.comp;
    for (int c = 0; c < 3; ++c) a.twoh[c] = (T)p.g.twoh[c];
    a.dtg = dtg;
    a.tiles_x = t.tiles_x;
    a.ntiles = t.tiles_x * t.tiles_y;
    a.chunk_len = t.chunk_len;
    a.jorg = t.jorg;
    a.ox = p.g.ghost[0]; a.oy = p.g.ghost[1]; a.oz = p.g.ghost[2];
    a.per = (p.g.per[0] ? 1 : 0) | (p.g.per[1] ? 2 : 0) | (p.g.per[2] ? 4 : 0);
    a.flag = flag;
    a.partials = nullptr;
    return a;
}

}  // namespace mr
