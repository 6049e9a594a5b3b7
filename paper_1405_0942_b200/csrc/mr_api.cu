// mr_api.cu -- the C-ABI of include/mr.h: argument validation, workspace carving, kernel launches.
#include "../../include/mr.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "mr_common.cuh"
#include "mr_generic.cuh"
#include "mr_stream_common.cuh"
#include "mr_direct.cuh"
#include "mr_sym.cuh"

using namespace mr;

namespace {

constexpr int kMaxPartialBlocks = 4096;
constexpr size_t kAlign = 256;

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
    int pitch;
    long long plane, comp;
    size_t field_bytes;   // one padded 3-component field
    size_t stage_bytes;   // one dense 3-component field
    size_t off_xi[2], off_b, off_stage, off_partials, off_diag, off_flag, total;
};

bool make_layout(const mr_grid* g, mr_dtype dt, Layout* L)
{
    if (!g) return false;
    if (g->nx < 5 || g->ny < 5 || g->nz < 5 || g->nx > 4096 || g->ny > 4096 || g->nz > 4096) return false;
    if (dt != MR_F64 && dt != MR_F32) return false;
    const size_t es = dt == MR_F64 ? 8 : 4;
    L->pitch = (g->nx + 15) / 16 * 16;
    L->plane = (long long)L->pitch * g->ny;
    L->comp = L->plane * g->nz;
    L->field_bytes = align_up((size_t)(3 * L->comp) * es, kAlign);
    L->stage_bytes = align_up((size_t)3 * g->nx * g->ny * g->nz * es, kAlign);
    size_t o = 0;
    L->off_xi[0] = o; o += L->field_bytes;
    L->off_xi[1] = o; o += L->field_bytes;
    L->off_b = o; o += L->field_bytes;
    L->off_stage = o; o += L->stage_bytes;
    L->off_partials = o; o += align_up(sizeof(DiagPartial) * kMaxPartialBlocks, kAlign);
    L->off_diag = o; o += kAlign;
    L->off_flag = o; o += kAlign;
    L->total = o;
    return true;
}

thread_local std::string g_create_error;

}  // namespace

struct mr_ctx {
    mr_grid grid;
    mr_domain dom;
    mr_dtype dtype;
    double gamma;
    double h[3];
    Layout L;
    char* ws;
    cudaStream_t stream;
    int cur;            // which xi buffer holds the current state
    bool have_B0;
    bool failed;
    double time;
    int64_t steps;
    int64_t launches;
    int sm_count;
    int force_variant;  // 0 auto (streaming kernels), 1 generic (global-memory kernels, the A/B reference)
    const char* variant;
    StreamPlan plan6;   // the streaming kernel of the direct-derivative operator (mr_direct.cuh)
    StreamPlan plan7;   // the symmetric split-phase streaming kernel of the mimetic operator (mr_sym.cuh)
    std::string err;

    void* xi(int w) const { return ws + L.off_xi[w]; }
    void* b() const { return ws + L.off_b; }
    void* stage() const { return ws + L.off_stage; }
    DiagPartial* partials() const { return reinterpret_cast<DiagPartial*>(ws + L.off_partials); }
    DiagPartial* diag_out() const { return reinterpret_cast<DiagPartial*>(ws + L.off_diag); }
    int* flag() const { return reinterpret_cast<int*>(ws + L.off_flag); }
    size_t esize() const { return dtype == MR_F64 ? 8 : 4; }
    size_t dense_bytes() const { return (size_t)3 * grid.nx * grid.ny * grid.nz * esize(); }
};

namespace {

mr_status fail(mr_ctx* c, mr_status s, const std::string& msg)
{
    if (c) c->err = msg; else g_create_error = msg;
    return s;
}

mr_status cuda_fail(mr_ctx* c, const char* what, cudaError_t e)
{
    return fail(c, MR_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define MR_CUDA(c, call)                                             \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) return cuda_fail((c), #call, e_);     \
    } while (0)

template <typename T>
GridP<T> grid_params(const mr_ctx* c)
{
    GridP<T> g;
    g.nx = c->grid.nx; g.ny = c->grid.ny; g.nz = c->grid.nz;
    g.pitch = c->L.pitch; g.plane = c->L.plane; g.comp = c->L.comp;
    for (int a = 0; a < 3; ++a) g.twoh[a] = (T)(2.0 * c->h[a]);
    return g;
}

DomainP domain_params(const mr_ctx* c)
{
    DomainP d;
    for (int a = 0; a < 3; ++a) { d.lo[a] = c->dom.lo[a]; d.h[a] = c->h[a]; }
    return d;
}

void node_launch_dims(const mr_ctx* c, dim3& grid, dim3& block)
{
    block = dim3(32, 8, 1);
    grid = dim3((c->grid.nx + 31) / 32, (c->grid.ny + 7) / 8, c->grid.nz);
}

mr_status read_flag(mr_ctx* c, int* out)
{
    MR_CUDA(c, cudaMemcpyAsync(out, c->flag(), sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    return MR_OK;
}

template <typename T>
mr_status do_set_B0(mr_ctx* c, const void* B0_dev)
{
    dim3 grid, block;
    node_launch_dims(c, grid, block);
    const double s0 = 4.0 * c->h[1] * c->h[2], s1 = 4.0 * c->h[2] * c->h[0], s2 = 4.0 * c->h[0] * c->h[1];
    k_import_B0<T><<<grid, block, 0, c->stream>>>(static_cast<const T*>(B0_dev), static_cast<T*>(c->b()),
                                                  grid_params<T>(c), s0, s1, s2);
    c->launches++;
    MR_CUDA(c, cudaGetLastError());
    c->have_B0 = true;
    return MR_OK;
}

template <typename T>
mr_status do_set_x(mr_ctx* c, const void* x_dev)
{
    dim3 grid, block;
    node_launch_dims(c, grid, block);
    const int other = 1 - c->cur;
    MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, sizeof(int), c->stream));
    k_import_x<T><<<grid, block, 0, c->stream>>>(static_cast<const T*>(x_dev), static_cast<T*>(c->xi(other)),
                                                 grid_params<T>(c), domain_params(c), c->flag());
    c->launches++;
    MR_CUDA(c, cudaGetLastError());
    int f = 0;
    mr_status s = read_flag(c, &f);
    if (s != MR_OK) return s;
    if (f & FLAG_BOUNDARY)
        return fail(c, MR_ERR_INVALID_ARG, "mr_set_x: a line-tied boundary node is not on the reference grid X");
    c->cur = other;
    c->failed = false;
    c->time = 0.0;
    c->steps = 0;
    return MR_OK;
}

template <typename T>
mr_status do_fields(mr_ctx* c, mr_operator op, void* x_out, void* B_out, void* J_out)
{
    dim3 grid, block;
    node_launch_dims(c, grid, block);
    const T* xi = static_cast<const T*>(c->xi(c->cur));
    const T* b = static_cast<const T*>(c->b());
    if (op == MR_OP_MIMETIC)
        k_fields<T, 0><<<grid, block, 0, c->stream>>>(xi, b, grid_params<T>(c), domain_params(c), static_cast<T*>(x_out),
                                                      static_cast<T*>(B_out), static_cast<T*>(J_out), c->flag());
    else
        k_fields<T, 1><<<grid, block, 0, c->stream>>>(xi, b, grid_params<T>(c), domain_params(c), static_cast<T*>(x_out),
                                                      static_cast<T*>(B_out), static_cast<T*>(J_out), c->flag());
    c->launches++;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

template <typename T>
mr_status launch_generic_step(mr_ctx* c, double dt, mr_operator op)
{
    dim3 grid, block;
    node_launch_dims(c, grid, block);
    const T* in = static_cast<const T*>(c->xi(c->cur));
    T* out = static_cast<T*>(c->xi(1 - c->cur));
    const T* b = static_cast<const T*>(c->b());
    const T dtg = (T)(dt * c->gamma);
    if (op == MR_OP_MIMETIC)
        k_step_generic<T, 0><<<grid, block, 0, c->stream>>>(in, out, b, grid_params<T>(c), dtg, c->flag());
    else
        k_step_generic<T, 1><<<grid, block, 0, c->stream>>>(in, out, b, grid_params<T>(c), dtg, c->flag());
    c->launches++;
    return MR_OK;
}

template <typename T>
mr_status do_step(mr_ctx* c, int64_t n, double dt, mr_operator op)
{
    const bool mim = op == MR_OP_MIMETIC;
    const bool use_sym = mim && c->force_variant == 0 && c->plan7.usable;
    const bool use_dstream = !mim && c->force_variant == 0 && c->plan6.usable;
    c->variant = use_dstream ? c->plan6.name : use_sym ? c->plan7.name : (mim ? "generic_mimetic" : "generic_direct");
    MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, sizeof(int), c->stream));
    for (int64_t s = 0; s < n; ++s) {
        if (use_dstream || use_sym) {
            const T dtg = (T)(dt * c->gamma);
            cudaError_t e = use_dstream ? launch_direct_step<T>(c->plan6, c->cur, dtg, c->flag(), c->stream)
                                        : launch_sym_step<T>(c->plan7, c->cur, dtg, c->flag(), c->stream);
            if (e != cudaSuccess) return cuda_fail(c, "streaming step launch", e);
            c->launches++;
        } else {
            launch_generic_step<T>(c, dt, op);
        }
        c->cur = 1 - c->cur;
    }
    MR_CUDA(c, cudaGetLastError());
    c->time += dt * (double)n;
    c->steps += n;
    int f = 0;
    mr_status st = read_flag(c, &f);
    if (st != MR_OK) return st;
    if (f & FLAG_NUMERIC) {
        c->failed = true;
        return fail(c, MR_ERR_NUMERIC, "mr_step: det(dx/dX) <= 0 or a non-finite value was met");
    }
    return MR_OK;
}

template <typename T>
mr_status do_diag(mr_ctx* c, mr_operator op, mr_diag* out)
{
    const long long rows = (long long)c->grid.ny * c->grid.nz;
    int blocks = c->sm_count * 8;
    if (blocks > kMaxPartialBlocks) blocks = kMaxPartialBlocks;
    if (blocks > rows) blocks = (int)rows;
    const T* xi = static_cast<const T*>(c->xi(c->cur));
    const T* b = static_cast<const T*>(c->b());
    MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, sizeof(int), c->stream));
    const int threads = c->grid.nx >= 256 ? 256 : (c->grid.nx >= 128 ? 128 : (c->grid.nx >= 64 ? 64 : 32));
    const bool fused = op == MR_OP_MIMETIC && c->plan7.usable && c->force_variant == 0 &&
                       c->plan7.tiles_x * c->plan7.tiles_y * c->plan7.nchunks <= kMaxPartialBlocks;
    if (fused) {
        // the streaming pass of the step kernel with the update replaced by the reduction (mr_sym.cuh, DIAG)
        cudaError_t e = launch_sym_diag<T>(c->plan7, c->cur, c->partials(), &blocks, c->flag(), c->stream);
        if (e != cudaSuccess) return cuda_fail(c, "streaming diagnostics launch", e);
    } else if (op == MR_OP_MIMETIC)
        k_diag<T, 0><<<blocks, threads, 0, c->stream>>>(xi, b, grid_params<T>(c), c->partials(), c->flag());
    else
        k_diag<T, 1><<<blocks, threads, 0, c->stream>>>(xi, b, grid_params<T>(c), c->partials(), c->flag());
    k_diag_final<<<1, 256, 0, c->stream>>>(c->partials(), blocks, c->diag_out());
    c->launches += 2;
    MR_CUDA(c, cudaGetLastError());
    DiagPartial r;
    MR_CUDA(c, cudaMemcpyAsync(&r, c->diag_out(), sizeof(r), cudaMemcpyDeviceToHost, c->stream));
    int f = 0;
    mr_status st = read_flag(c, &f);
    if (st != MR_OK) return st;
    const double vol8 = 8.0 * c->h[0] * c->h[1] * c->h[2];
    out->time = c->time;
    out->steps = c->steps;
    out->energy = r.e / 16.0;
    out->max_jxb = r.fmax;
    out->xi = r.xi;
    out->min_det = r.dmin / vol8;
    if (f & FLAG_NUMERIC) return fail(c, MR_ERR_NUMERIC, "mr_diagnostics: det(dx/dX) <= 0 or a non-finite value was met");
    return MR_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------- C ABI

extern "C" size_t mr_workspace_bytes(const mr_grid* grid, mr_dtype dtype)
{
    Layout L;
    return make_layout(grid, dtype, &L) ? L.total : 0;
}

extern "C" mr_status mr_create(const mr_grid* grid, const mr_domain* domain, const mr_boundary* boundary, mr_ctx** out)
{
    if (out) *out = nullptr;
    if (!grid || !domain || !boundary || !out) return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: null argument");
    Layout L;
    if (!make_layout(grid, boundary->dtype, &L))
        return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: each of nx, ny, nz must be in [5, 4096] and dtype MR_F64 or MR_F32");
    for (int a = 0; a < 3; ++a) {
        if (!std::isfinite(domain->lo[a]) || !std::isfinite(domain->hi[a]) || !(domain->hi[a] > domain->lo[a]))
            return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: domain needs finite hi > lo on every axis");
        if (boundary->bc[a] == MR_BC_PERIODIC)
            return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: periodic boundaries (Eqs. 2.12-2.14) are not implemented");
        if (boundary->bc[a] != MR_BC_LINE_TIED) return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: unknown boundary type");
    }
    if (!(boundary->gamma > 0.0) || !std::isfinite(boundary->gamma))
        return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: gamma must be finite and > 0");
    if (!boundary->workspace || (reinterpret_cast<uintptr_t>(boundary->workspace) % kAlign) != 0)
        return fail(nullptr, MR_ERR_WORKSPACE, "mr_create: workspace is null or not 256-byte aligned");
    if (boundary->workspace_bytes < L.total)
        return fail(nullptr, MR_ERR_WORKSPACE, "mr_create: workspace smaller than mr_workspace_bytes()");

    int dev = 0;
    MR_CUDA(nullptr, cudaGetDevice(&dev));
    cudaDeviceProp prop;
    MR_CUDA(nullptr, cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10)
        return fail(nullptr, MR_ERR_CUDA, "mr_create: this library is built for sm_100a (B200) only");

    mr_ctx* c = new (std::nothrow) mr_ctx();
    if (!c) return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: out of host memory");
    c->grid = *grid;
    c->dom = *domain;
    c->dtype = boundary->dtype;
    c->gamma = boundary->gamma;
    const int n[3] = { grid->nx, grid->ny, grid->nz };
    for (int a = 0; a < 3; ++a) c->h[a] = (domain->hi[a] - domain->lo[a]) / (double)(n[a] - 1);
    c->L = L;
    c->ws = static_cast<char*>(boundary->workspace);
    c->stream = static_cast<cudaStream_t>(boundary->stream);
    c->cur = 0;
    c->have_B0 = false;
    c->failed = false;
    c->time = 0.0;
    c->steps = 0;
    c->launches = 0;
    c->sm_count = prop.multiProcessorCount;
    c->force_variant = 0;
    c->variant = "";

    cudaError_t e = cudaMemsetAsync(c->ws, 0, L.off_stage, c->stream);   // xi = 0 (x = X), b = 0, incl. padding
    if (e == cudaSuccess) e = cudaMemsetAsync(c->ws + L.off_partials, 0, L.total - L.off_partials, c->stream);
    if (e != cudaSuccess) { delete c; return cuda_fail(nullptr, "mr_create: cudaMemsetAsync", e); }

    StreamGeom sg;
    sg.nx = grid->nx; sg.ny = grid->ny; sg.nz = grid->nz;
    sg.pitch = L.pitch; sg.plane = L.plane; sg.comp = L.comp;
    for (int a = 0; a < 3; ++a) sg.twoh[a] = 2.0 * c->h[a];
    std::string why;
    if (!build_direct_plan(&c->plan6, sg, c->dtype == MR_F64, c->xi(0), c->xi(1), c->b(), c->sm_count, &why)) {
        c->plan6.usable = false;
        c->plan6.why = why;
    }
    if (!build_sym_plan(&c->plan7, sg, c->dtype == MR_F64, c->xi(0), c->xi(1), c->b(), c->sm_count, &why)) {
        c->plan7.usable = false;
        c->plan7.why = why;
    }
    *out = c;
    return MR_OK;
}

extern "C" mr_status mr_destroy(mr_ctx* ctx)
{
    delete ctx;
    return MR_OK;
}

extern "C" mr_status mr_set_B0(mr_ctx* ctx, const void* B0_dev)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!B0_dev) return fail(ctx, MR_ERR_INVALID_ARG, "mr_set_B0: null pointer");
    return ctx->dtype == MR_F64 ? do_set_B0<double>(ctx, B0_dev) : do_set_B0<float>(ctx, B0_dev);
}

extern "C" mr_status mr_set_B0_host(mr_ctx* ctx, const void* B0_host)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!B0_host) return fail(ctx, MR_ERR_INVALID_ARG, "mr_set_B0_host: null pointer");
    MR_CUDA(ctx, cudaMemcpyAsync(ctx->stage(), B0_host, ctx->dense_bytes(), cudaMemcpyHostToDevice, ctx->stream));
    mr_status s = mr_set_B0(ctx, ctx->stage());
    if (s != MR_OK) return s;
    MR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return MR_OK;
}

extern "C" mr_status mr_set_x(mr_ctx* ctx, const void* x_dev)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!x_dev) return fail(ctx, MR_ERR_INVALID_ARG, "mr_set_x: null pointer");
    return ctx->dtype == MR_F64 ? do_set_x<double>(ctx, x_dev) : do_set_x<float>(ctx, x_dev);
}

extern "C" mr_status mr_set_x_host(mr_ctx* ctx, const void* x_host)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!x_host) return fail(ctx, MR_ERR_INVALID_ARG, "mr_set_x_host: null pointer");
    MR_CUDA(ctx, cudaMemcpyAsync(ctx->stage(), x_host, ctx->dense_bytes(), cudaMemcpyHostToDevice, ctx->stream));
    return mr_set_x(ctx, ctx->stage());
}

extern "C" mr_status mr_step(mr_ctx* ctx, int64_t n, double dt, mr_operator op)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (n < 0 || !(dt > 0.0) || !std::isfinite(dt)) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step: need n >= 0 and finite dt > 0");
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step: unknown operator");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_step: B0 has not been set");
    if (ctx->failed) return fail(ctx, MR_ERR_NUMERIC, "mr_step: context is in the failed state (call mr_set_x)");
    return ctx->dtype == MR_F64 ? do_step<double>(ctx, n, dt, op) : do_step<float>(ctx, n, dt, op);
}

extern "C" mr_status mr_diagnostics(mr_ctx* ctx, mr_operator op, mr_diag* out)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!out) return fail(ctx, MR_ERR_INVALID_ARG, "mr_diagnostics: null output");
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_diagnostics: unknown operator");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_diagnostics: B0 has not been set");
    return ctx->dtype == MR_F64 ? do_diag<double>(ctx, op, out) : do_diag<float>(ctx, op, out);
}

extern "C" mr_status mr_get_fields(mr_ctx* ctx, mr_operator op, void* x_dev, void* B_dev, void* J_dev)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_get_fields: unknown operator");
    if (!x_dev && !B_dev && !J_dev) return MR_OK;
    if ((B_dev || J_dev) && !ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_get_fields: B0 has not been set");
    return ctx->dtype == MR_F64 ? do_fields<double>(ctx, op, x_dev, B_dev, J_dev) : do_fields<float>(ctx, op, x_dev, B_dev, J_dev);
}

extern "C" mr_status mr_get_fields_host(mr_ctx* ctx, mr_operator op, void* x_host, void* B_host, void* J_host)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    void* outs[3] = { x_host, B_host, J_host };
    for (int w = 0; w < 3; ++w) {
        if (!outs[w]) continue;
        mr_status s = mr_get_fields(ctx, op, w == 0 ? ctx->stage() : nullptr, w == 1 ? ctx->stage() : nullptr,
                                    w == 2 ? ctx->stage() : nullptr);
        if (s != MR_OK) return s;
        MR_CUDA(ctx, cudaMemcpyAsync(outs[w], ctx->stage(), ctx->dense_bytes(), cudaMemcpyDeviceToHost, ctx->stream));
    }
    MR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return MR_OK;
}

extern "C" const char* mr_last_error(const mr_ctx* ctx)
{
    return ctx ? ctx->err.c_str() : g_create_error.c_str();
}

extern "C" int64_t mr_launch_count(const mr_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" const char* mr_step_variant(const mr_ctx* ctx) { return ctx ? ctx->variant : ""; }

extern "C" mr_status mr_set_variant(mr_ctx* ctx, const char* name)
{
    if (!ctx || !name) return MR_ERR_INVALID_ARG;
    if (!std::strcmp(name, "auto")) ctx->force_variant = 0;
    else if (!std::strcmp(name, "generic")) ctx->force_variant = 1;
    else return fail(ctx, MR_ERR_INVALID_ARG, "mr_set_variant: expected auto or generic");
    return MR_OK;
}
