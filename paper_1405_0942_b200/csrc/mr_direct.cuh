// mr_direct.cuh -- the streaming step kernel for the direct-derivative ("classical") operator (S1, S2, S3d, S4, S5 in
// one pass; reading Q4 of DESIGN.md: the analytic derivative of Eq. 2.1).
//
// The direct operator needs no neighbour's B: J at a node follows from the 19-point stencil of xi (first and second
// differences) and the 7-point stencil of b around it.  The global-memory kernel (mr_generic.cuh) issues 123 loads
// per node and is bound by them (2.23 ms per step on C4, 19 % of the FP64 roof).  Here a CTA marches along k over a
// 32 x TY tile; the TMA unit streams the halo-1 boxes of xi and b of every plane into shared-memory rings (the same
// 4-D tiled tensor maps as the mimetic kernels) and every operand of a node comes from the planes k-1, k, k+1 in
// shared memory.  One node per thread, one warp per tile row.  No data is exchanged between threads, so the only
// synchronisation is the recycling of the ring slots: every warp arrives on a named barrier when it is done with
// the plane k-1, only the producer's warp waits on it.
#pragma once
#include "mr_generic.cuh"
#include "mr_stream_common.cuh"

namespace mr {

template <typename T, int TY, int R>
struct DirectLayout {
    static_assert(TY >= 4 && TY <= 16 && R >= 4 && R <= 7, "tile / ring sizes");
    static constexpr int TX = 32;
    static constexpr int HX = 16 / (int)sizeof(T);            // x halo widened to 16 bytes (TMA start alignment)
    static constexpr int BW = TX + 3 * HX;                     // 38 doubles / 44 floats: a multiple of 16 bytes
    static constexpr int BH = TY + 2;
    static constexpr int CS = BW * BH;                         // component stride inside a box
    static constexpr int round128(int bytes) { return (bytes + 127) / 128 * 128; }
    static constexpr int SLOT = round128(3 * CS * (int)sizeof(T)) / (int)sizeof(T);
    static constexpr uint32_t BOX_BYTES = 3u * CS * sizeof(T);
    static constexpr int NWARPS = TY, NTHREADS = NWARPS * 32;
    static constexpr size_t OFF_X = 0;
    static constexpr size_t OFF_B = OFF_X + (size_t)R * SLOT * sizeof(T);
    static constexpr size_t OFF_BAR = OFF_B + (size_t)R * SLOT * sizeof(T);
    static constexpr size_t BYTES = OFF_BAR + (size_t)R * 8 + 128;
};

// J, B, D at an interior node from the three shared-memory planes around it.  xm/xc/xp and bm/bc/bp point at the
// node in component 0 of the planes k-1, k, k+1; S = row stride, CS = component stride.  Same arithmetic as
// node_J_direct (mr_common.cuh): W[c][q][a] = 4 h_q h_a d2x_c/dX_q dX_a, g[q][a] = delta_a b_q,
//   Nt = W b + dF g,  t = adj : W,  Q = Nt - B t,  dB_c/dx_m = Q adj / D^2,  J = curl.
template <typename T, int S, int CS>
__device__ __forceinline__ void direct_J_smem(const T* __restrict__ xm, const T* __restrict__ xc, const T* __restrict__ xp,
                                              const T* __restrict__ bm, const T* __restrict__ bc, const T* __restrict__ bp,
                                              const T (&twoh)[3], T (&J)[3], T (&B)[3], T& D, bool& bad)
{
    T dF[3][3], W[3][3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T* m = xm + c * CS;
        const T* z = xc + c * CS;
        const T* p = xp + c * CS;
        const T f0 = z[0], fe = z[1], fw = z[-1], fn = z[S], fs = z[-S], fu = p[0], fd = m[0];
        dF[c][0] = fe - fw;
        dF[c][1] = fn - fs;
        dF[c][2] = fu - fd;
        dF[c][c] += twoh[c];
        W[c][0][0] = T(4) * (fe - T(2) * f0 + fw);
        W[c][1][1] = T(4) * (fn - T(2) * f0 + fs);
        W[c][2][2] = T(4) * (fu - T(2) * f0 + fd);
        const T w01 = z[S + 1] - z[-S + 1] - z[S - 1] + z[-S - 1];
        const T w02 = p[1] - m[1] - p[-1] + m[-1];
        const T w12 = p[S] - m[S] - p[-S] + m[-S];
        W[c][0][1] = w01; W[c][1][0] = w01;
        W[c][0][2] = w02; W[c][2][0] = w02;
        W[c][1][2] = w12; W[c][2][1] = w12;
    }
    T bb[3], gq[3][3];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const T* z = bc + q * CS;
        bb[q] = z[0];
        gq[q][0] = z[1] - z[-1];
        gq[q][1] = z[S] - z[-S];
        gq[q][2] = bp[q * CS] - bm[q * CS];
    }
    T adj[3][3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int a1 = (a + 1) % 3, a2 = (a + 2) % 3;
#pragma unroll
        for (int m = 0; m < 3; ++m) {
            const int m1 = (m + 1) % 3, m2 = (m + 2) % 3;
            adj[a][m] = dF[m1][a1] * dF[m2][a2] - dF[m1][a2] * dF[m2][a1];
        }
    }
    D = dF[0][0] * adj[0][0] + dF[0][1] * adj[1][0] + dF[0][2] * adj[2][0];
    bad = bad || !(D > T(0));
    const T inv = T(1) / D;
#pragma unroll
    for (int c = 0; c < 3; ++c) B[c] = (dF[c][0] * bb[0] + dF[c][1] * bb[1] + dF[c][2] * bb[2]) * inv;
    T t[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        T acc = T(0);
#pragma unroll
        for (int q = 0; q < 3; ++q)
#pragma unroll
            for (int c = 0; c < 3; ++c) acc += adj[q][c] * W[c][q][a];
        t[a] = acc;
    }
    T Q[3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            T acc = -B[c] * t[a];
#pragma unroll
            for (int q = 0; q < 3; ++q) acc += W[c][q][a] * bb[q] + dF[c][q] * gq[q][a];
            Q[c][a] = acc;
        }
    auto G = [&](int c, int m) { return Q[c][0] * adj[0][m] + Q[c][1] * adj[1][m] + Q[c][2] * adj[2][m]; };
    const T inv2 = inv * inv;
    J[0] = (G(2, 1) - G(1, 2)) * inv2;
    J[1] = (G(0, 2) - G(2, 0)) * inv2;
    J[2] = (G(1, 0) - G(0, 1)) * inv2;
}

// MODE (mr_sym.cuh): MODE_STEP xi+ = xi + dtg J x B;  MODE_RHS out = dtg J x B;  MODE_DIAG the reduction S6 (one
// DiagPartial per CTA into `out`)
template <typename T, int TY, int R, int MODE>
__global__ void __launch_bounds__(TY * 32, 1)
k_step_direct(const __grid_constant__ CUtensorMap map_in, const __grid_constant__ CUtensorMap map_b, T* __restrict__ out,
              const StreamArgs<T> a)
{
    using L = DirectLayout<T, TY, R>;
    constexpr bool DIAG = MODE == 1, RHS = MODE == 2;
    constexpr int TX = L::TX, BW = L::BW, CS = L::CS, NTH = L::NTHREADS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((128u - (ptx::smem_u32(smem_raw) & 127u)) & 127u);
    const T* sx = reinterpret_cast<const T*>(smem + L::OFF_X);
    const T* sb = reinterpret_cast<const T*>(smem + L::OFF_B);
    const uint32_t sx_u32 = ptx::smem_u32(sx), sb_u32 = ptx::smem_u32(sb);
    const uint32_t bar = ptx::smem_u32(smem + L::OFF_BAR);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tile = blockIdx.x % a.ntiles, chunk = blockIdx.x / a.ntiles;
    const int i0 = (tile % a.tiles_x) * TX, j0 = (tile / a.tiles_x) * TY + a.jorg;
    const int nz = a.nz;
    const int k0 = chunk * a.chunk_len, k1 = min(k0 + a.chunk_len, nz);
    // a periodic axis (Eqs. 2.12-2.14) has no face: its ghost layers sit in the padded arrays, every node is an inner point
    const bool perx = (a.per & 1) != 0, pery = (a.per & 2) != 0, perz = (a.per & 4) != 0;
    const int pfirst = max(k0 - 1, perz ? -1 : 0), plast = min(k1, perz ? nz : nz - 1);        // planes this item touches
    const T twoh[3] = { a.twoh[0], a.twoh[1], a.twoh[2] };

    // ---- TMA producer: lane 0 of the last warp; one mbarrier per slot covers the xi box and the b box ----
    const bool pwarp = warp == TY - 1, producer = pwarp && lane == 0;
    int next = pfirst;
    auto refill = [&](int upto) {
        for (const int last = min(upto, plast); next <= last; ++next) {
            const uint32_t s = (uint32_t)((next - pfirst) % R);
            ptx::mbar_expect_tx(bar + 8u * s, 2u * L::BOX_BYTES);
            ptx::tma_load_4d(sx_u32 + s * (uint32_t)(L::SLOT * sizeof(T)), &map_in, i0 - L::HX + a.ox, j0 - 1 + a.oy, next + a.oz, 0, bar + 8u * s);
            ptx::tma_load_4d(sb_u32 + s * (uint32_t)(L::SLOT * sizeof(T)), &map_b, i0 - L::HX + a.ox, j0 - 1 + a.oy, next + a.oz, 0, bar + 8u * s);
        }
    };
    if (producer) {
        for (int s = 0; s < R; ++s) ptx::mbar_init(bar + 8u * s, 1);
        ptx::fence_mbar_init();
    }
    __syncthreads();
    if (producer) refill(pfirst + R - 1);

    const int gi = i0 + lane, gj = j0 + warp;
    const bool in_dom = gi < a.nx && gj < a.ny;
    const bool in_xy = in_dom && (perx || (gi > 0 && gi < a.nx - 1)) && (pery || (gj > 0 && gj < a.ny - 1));
    const int o = (warp + 1) * BW + lane + L::HX;                      // this node inside a box
    auto wait_plane = [&](int p) { const int q = p - pfirst; ptx::mbar_wait(bar + 8u * (uint32_t)(q % R), (uint32_t)((q / R) & 1)); };
    for (int p = pfirst; p <= min(k0, plast); ++p) wait_plane(p);

    bool bad = false;
    T* po = out + (long long)k0 * a.plane + (long long)gj * a.pitch + gi;
    DiagPartial acc = { 0.0, 0.0, 0.0, INFINITY };          // DIAG: this thread's partial over its INNER nodes (zeta = 1); the
                                                            // nodes on the line-tied faces are left to k_diag_faces
    int sm = (k0 - 1 - pfirst + R) % R, sc = (k0 - pfirst) % R, sp = (k0 + 1 - pfirst) % R;   // slots of k-1, k, k+1
    uint32_t parp = (uint32_t)(((k0 + 1 - pfirst) / R) & 1);
    int gen = 0;                                                       // named barrier of this iteration (k - k0) % R
#pragma unroll 1
    for (int k = k0; k < k1; ++k) {
        if (k + 1 <= plast) ptx::mbar_wait(bar + 8u * (uint32_t)sp, parp);
        const T* xc = sx + sc * L::SLOT + o;
        T x[3] = { xc[0], xc[CS], xc[2 * CS] };
        if (RHS) x[0] = x[1] = x[2] = T(0);
        const bool inner = in_xy && (perz || (k > 0 && k < nz - 1));
        if (inner) {
            T J[3], B[3], u[3], D;
            direct_J_smem<T, BW, CS>(sx + sm * L::SLOT + o, xc, sx + sp * L::SLOT + o, sb + sm * L::SLOT + o, sb + sc * L::SLOT + o,
                                     sb + sp * L::SLOT + o, twoh, J, B, D, bad);
            cross3(J, B, u);
            if constexpr (DIAG) {
                const double b2 = (double)B[0] * B[0] + (double)B[1] * B[1] + (double)B[2] * B[2];
                const double fm = sqrt((double)u[0] * u[0] + (double)u[1] * u[1] + (double)u[2] * u[2]);
                DiagPartial v = { b2 * (double)D, fm, fm / b2, (double)D };
                diag_combine(acc, v);
            } else {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    x[c] += a.dtg * u[c];
                    bad = bad || !(fabs(x[c]) < T(1e30));
                }
            }
        }
        if (!DIAG && in_dom) {
            po[0] = x[0];
            po[a.comp] = x[1];
            po[2 * a.comp] = x[2];
        }
        po += a.plane;
        // this warp is done with the plane k-1: the producer's warp collects the arrivals and recycles the slot
        if (pwarp) {
            ptx::named_sync(1 + gen, NTH);
            if (producer) refill(k - 1 + R);
        } else {
            ptx::named_arrive(1 + gen, NTH);
        }
        if (++gen == R) gen = 0;
        sm = sc; sc = sp;
        if (++sp == R) { sp = 0; parp ^= 1u; }
    }
    if constexpr (DIAG) {
        __syncthreads();                                    // the ring is drained: shared memory is free
#pragma unroll
        for (int o2 = 16; o2 > 0; o2 >>= 1) {
            DiagPartial w;
            w.e = __shfl_down_sync(0xffffffffu, acc.e, o2);
            w.fmax = __shfl_down_sync(0xffffffffu, acc.fmax, o2);
            w.xi = __shfl_down_sync(0xffffffffu, acc.xi, o2);
            w.dmin = __shfl_down_sync(0xffffffffu, acc.dmin, o2);
            diag_combine(acc, w);
        }
        DiagPartial* shp = reinterpret_cast<DiagPartial*>(smem);
        if (lane == 0) shp[warp] = acc;
        __syncthreads();
        if (tid == 0) {
            DiagPartial v = shp[0];
            for (int w = 1; w < TY; ++w) diag_combine(v, shp[w]);
            reinterpret_cast<DiagPartial*>(out)[blockIdx.x] = v;
        }
    }
    if (bad) atomicOr(a.flag, FLAG_NUMERIC);
}

// ----------------------------------------------------------------------------------------------- host side

constexpr int kXTY = 16, kXR = 5;

inline bool build_direct_plan(StreamPlan* p, const StreamGeom& g, bool f64, void* xi0, void* xi1, void* b, int sm_count,
                              std::string* why)
{
    using Ld = DirectLayout<double, kXTY, kXR>;
    using Lf = DirectLayout<float, kXTY, kXR>;
    p->usable = false;
    p->f64 = f64;
    p->g = g;
    p->xi[0] = node_base(xi0, g, f64);      // xi0, xi1, b: the starts of the padded arrays (what the tensor maps span)
    p->xi[1] = node_base(xi1, g, f64);
    p->b = node_base(b, g, f64);
    p->name = f64 ? "direct_tma_f64" : "direct_tma_f32";
    const int bw = f64 ? Ld::BW : Lf::BW;
    if (!encode_map(&p->map_xi[0], f64, xi0, g, bw, kXTY + 2) || !encode_map(&p->map_xi[1], f64, xi1, g, bw, kXTY + 2) ||
        !encode_map(&p->map_b, f64, b, g, bw, kXTY + 2)) {
        *why = "cuTensorMapEncodeTiled failed";
        return false;
    }
    p->smem_bytes = f64 ? Ld::BYTES : Lf::BYTES;
    cudaError_t e = cudaSuccess;
    const int sb = (int)p->smem_bytes;
    if (f64) {
        e = cudaFuncSetAttribute(k_step_direct<double, kXTY, kXR, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, sb);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_step_direct<double, kXTY, kXR, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, sb);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_step_direct<double, kXTY, kXR, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, sb);
    } else {
        e = cudaFuncSetAttribute(k_step_direct<float, kXTY, kXR, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, sb);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_step_direct<float, kXTY, kXR, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, sb);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_step_direct<float, kXTY, kXR, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, sb);
    }
    if (e != cudaSuccess) {
        *why = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e);
        return false;
    }
    choose_tilings(p, Ld::TX, kXTY, false, sm_count);
    p->usable = true;
    return true;
}

inline bool direct_bind_stage(StreamPlan* p, void* xs)
{
    const int bw = p->f64 ? DirectLayout<double, kXTY, kXR>::BW : DirectLayout<float, kXTY, kXR>::BW;
    if (!encode_map(&p->map_xi[2], p->f64, xs, p->g, bw, kXTY + 2)) return false;
    p->xi[2] = node_base(xs, p->g, p->f64);
    return true;
}

// one step / one right-hand side of the state in the plan's buffer `cur` (see launch_sym_step)
template <typename T>
inline cudaError_t launch_direct_step(const StreamPlan& p, int cur, T dtg, int* flag, cudaStream_t stream, bool rhs = false, void* out = nullptr)
{
    using L = DirectLayout<T, kXTY, kXR>;
    const StreamArgs<T> a = stream_args<T>(p, p.step, dtg, flag);
    T* o = static_cast<T*>(out ? out : p.xi[1 - cur]);
    const int grid = a.ntiles * p.step.nchunks;
    if (rhs) k_step_direct<T, kXTY, kXR, 2><<<grid, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], p.map_b, o, a);
    else k_step_direct<T, kXTY, kXR, 0><<<grid, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], p.map_b, o, a);
    return cudaGetLastError();
}

// S6 over the INNER nodes by the same pass: one DiagPartial per CTA into partials[0 .. *nblocks)
template <typename T>
inline cudaError_t launch_direct_diag(const StreamPlan& p, int cur, DiagPartial* partials, int* nblocks, int* flag, cudaStream_t stream)
{
    using L = DirectLayout<T, kXTY, kXR>;
    const StreamArgs<T> a = stream_args<T>(p, p.step, (T)0, flag);       // (the nodes on the faces are k_diag_faces' anyway)
    *nblocks = a.ntiles * p.step.nchunks;
    k_step_direct<T, kXTY, kXR, 1><<<*nblocks, L::NTHREADS, p.smem_bytes, stream>>>(p.map_xi[cur], p.map_b, reinterpret_cast<T*>(partials), a);
    return cudaGetLastError();
}

}  // namespace mr
