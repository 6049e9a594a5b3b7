// mr_api.cu -- the C-ABI of include/mr.h: argument validation, workspace carving, kernel launches, and the host side of
// the adaptive integrator (accept / reject, Eq. 2.11).
#include "../../include/mr.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include "mr_common.cuh"
#include "mr_generic.cuh"
#include "mr_stream_common.cuh"
#include "mr_direct.cuh"
#include "mr_sym.cuh"
#include "mr_next.cuh"

using namespace mr;

namespace {

constexpr int kMaxPartialBlocks = 4096;
constexpr int kHistoryBatch = 1024;       // records of mr_step_monitored kept on the device between two copies to the host
constexpr size_t kAlign = 256;

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
    int pitch;
    long long plane, comp;
    int ghost[3];         // ghost layers either side of a periodic axis (0 on a line-tied one), DESIGN.md "Data layout"
    long long shift;      // element offset of the node (0, 0, 0) inside a padded field
    size_t field_bytes;   // one padded 3-component field
    size_t stage_bytes;   // one dense 3-component field
    size_t off_xi[2], off_b, off_stage, off_partials, off_history, off_diag, off_flag, total;
    size_t adaptive_total;   // the second workspace: 7 padded fields
};

// per = which axes are periodic (null = none)
bool make_layout(const mr_grid* g, mr_dtype dt, const int* per, Layout* L)
{
    if (!g) return false;
    if (g->nx < 5 || g->ny < 5 || g->nz < 5 || g->nx > 4096 || g->ny > 4096 || g->nz > 4096) return false;
    if (dt != MR_F64 && dt != MR_F32) return false;
    const size_t es = dt == MR_F64 ? 8 : 4;
    // a periodic axis carries its ghost nodes in the array: 2 planes / rows, 16 bytes of columns (the x halo of the TMA boxes)
    L->ghost[0] = (per && per[0]) ? (int)(16 / es) : 0;
    L->ghost[1] = (per && per[1]) ? 2 : 0;
    L->ghost[2] = (per && per[2]) ? 2 : 0;
    L->pitch = (g->nx + 2 * L->ghost[0] + 15) / 16 * 16;
    L->plane = (long long)L->pitch * (g->ny + 2 * L->ghost[1]);
    L->comp = L->plane * (g->nz + 2 * L->ghost[2]);
    L->shift = (long long)L->ghost[2] * L->plane + (long long)L->ghost[1] * L->pitch + L->ghost[0];
    L->field_bytes = align_up((size_t)(3 * L->comp) * es, kAlign);
    L->stage_bytes = align_up((size_t)3 * g->nx * g->ny * g->nz * es, kAlign);
    size_t o = 0;
    L->off_xi[0] = o; o += L->field_bytes;
    L->off_xi[1] = o; o += L->field_bytes;
    L->off_b = o; o += L->field_bytes;
    L->off_stage = o; o += L->stage_bytes;
    L->off_partials = o; o += align_up(sizeof(DiagPartial) * (2 * kMaxPartialBlocks), kAlign);
    L->off_history = o; o += align_up(sizeof(DiagPartial) * kHistoryBatch, kAlign);
    L->off_diag = o; o += kAlign;
    L->off_flag = o; o += kAlign;
    L->total = o;
    L->adaptive_total = 7 * L->field_bytes;
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
    int per[3];
    bool any_periodic;
    Layout L;
    char* ws;
    char* aws;          // adaptive workspace (k_1 .. k_6, stage state) or null
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
    bool plans_built;
    StreamPlan plan_dir;   // the streaming kernel of the direct-derivative operator (mr_direct.cuh)
    StreamPlan plan_mim;   // the streaming kernel of the mimetic operator (mr_sym.cuh)
    // mr_step on a grid that lives in the L2: kStepsPerGraph steps captured once as a CUDA graph and replayed (the step is
    // bound by launch latency there); the key is everything a captured launch depends on
    cudaGraphExec_t step_graph = nullptr;
    cudaStream_t cap_stream = nullptr;     // the capture is recorded on a stream of the library's own (the caller's may be the
                                           // legacy default stream, which cannot be captured); the graph runs on the caller's
    int sg_op = -1, sg_cur = -1, sg_variant = -1;
    double sg_dtg = 0.0;
    bool graphs_enabled = true;
    // mr_step_adaptive: the launches of one Cash-Karp trial step (they read dt from device memory) captured once per
    // (operator, state buffer) and replayed; dt goes in and Lambda and the flag come back through three pinned host words
    cudaGraphExec_t trial_graph[2][2] = { { nullptr, nullptr }, { nullptr, nullptr } };
    int tg_variant[2][2] = { { -1, -1 }, { -1, -1 } };
    int64_t tg_launches[2][2] = { { 0, 0 }, { 0, 0 } };
    double* pinned = nullptr;              // [0] dt of the trial, [1] the flag word (as an int), [2] Lambda
    // mr_step_host_async: a second dense staging field (caller-owned), a stream of the library's own for the device -> host copies
    char* sws = nullptr;
    cudaStream_t d2h_stream = nullptr;
    cudaEvent_t ev_fields = nullptr, ev_d2h = nullptr;
    bool d2h_pending = false, pipeline_open = false;
    std::string err;

    ~mr_ctx()
    {
        if (step_graph) cudaGraphExecDestroy(step_graph);
        for (int o = 0; o < 2; ++o)
            for (int w = 0; w < 2; ++w)
                if (trial_graph[o][w]) cudaGraphExecDestroy(trial_graph[o][w]);
        if (cap_stream) cudaStreamDestroy(cap_stream);
        if (d2h_stream) cudaStreamDestroy(d2h_stream);
        if (ev_fields) cudaEventDestroy(ev_fields);
        if (ev_d2h) cudaEventDestroy(ev_d2h);
        if (pinned) cudaFreeHost(pinned);
    }

    // a padded field starts at *_raw (what the tensor maps and the elementwise kernels span); the kernels that index by
    // node get the address of the node (0, 0, 0)
    size_t node0() const { return (size_t)L.shift * esize(); }
    void* xi_raw(int w) const { return ws + L.off_xi[w]; }
    void* b_raw() const { return ws + L.off_b; }
    void* xi(int w) const { return ws + L.off_xi[w] + node0(); }
    void* b() const { return ws + L.off_b + node0(); }
    void* stage() const { return ws + L.off_stage; }
    DiagPartial* partials() const { return reinterpret_cast<DiagPartial*>(ws + L.off_partials); }
    DiagPartial* diag_out() const { return reinterpret_cast<DiagPartial*>(ws + L.off_diag); }
    DiagPartial* history() const { return reinterpret_cast<DiagPartial*>(ws + L.off_history); }
    int* flag() const { return reinterpret_cast<int*>(ws + L.off_flag); }
    double* lambda_dev() const { return reinterpret_cast<double*>(ws + L.off_flag + 8); }   // next to the flag: one memset, one copy
    double* dt_dev() const { return reinterpret_cast<double*>(ws + L.off_diag + 128); }   // the trial step length (kernels read it)
    void* kbuf_raw(int s) const { return aws + (size_t)s * L.field_bytes; }  // s = 0..5: k_1..k_6, 6: the stage state
    void* kbuf(int s) const { return aws + (size_t)s * L.field_bytes + node0(); }
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
    for (int a = 0; a < 3; ++a) { g.twoh[a] = (T)(2.0 * c->h[a]); g.per[a] = c->per[a]; }
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

// the TMA descriptors and launch geometry of the streaming kernels, on first use
void ensure_plans(mr_ctx* c)
{
    if (c->plans_built) return;
    c->plans_built = true;
    StreamGeom sg;
    sg.nx = c->grid.nx; sg.ny = c->grid.ny; sg.nz = c->grid.nz;
    sg.pitch = c->L.pitch; sg.plane = c->L.plane; sg.comp = c->L.comp;
    for (int a = 0; a < 3; ++a) sg.twoh[a] = 2.0 * c->h[a];
    for (int a = 0; a < 3; ++a) { sg.ghost[a] = c->L.ghost[a]; sg.per[a] = c->per[a]; }
    std::string why;
    if (!build_direct_plan(&c->plan_dir, sg, c->dtype == MR_F64, c->xi_raw(0), c->xi_raw(1), c->b_raw(), c->sm_count, &why)) {
        c->plan_dir.usable = false;
        c->plan_dir.why = why;
    }
    if (!build_sym_plan(&c->plan_mim, sg, c->dtype == MR_F64, c->xi_raw(0), c->xi_raw(1), c->b_raw(), c->sm_count, &why)) {
        c->plan_mim.usable = false;
        c->plan_mim.why = why;
    }
    if (c->aws) {
        if (c->plan_mim.usable && !sym_bind_stage(&c->plan_mim, c->kbuf_raw(6))) c->plan_mim.usable = false;
        if (c->plan_dir.usable && !direct_bind_stage(&c->plan_dir, c->kbuf_raw(6))) c->plan_dir.usable = false;
    }
}

// keep the ghost layers of the periodic axes of a padded field equal to the nodes they wrap to (`field` = its node (0,0,0))
template <typename T>
void wrap_ghosts(mr_ctx* c, void* field)
{
    if (!c->any_periodic) return;
    const int* gh = c->L.ghost;
    const long long px = c->grid.nx + 2 * gh[0], py = c->grid.ny + 2 * gh[1];
    const long long n = 2LL * gh[2] * py * px + (long long)c->grid.nz * 2 * gh[1] * px + (long long)c->grid.nz * c->grid.ny * 2 * gh[0];
    long long blocks = (n + 255) / 256;
    if (blocks > (long long)c->sm_count * 16) blocks = (long long)c->sm_count * 16;
    k_wrap<T><<<(unsigned)blocks, 256, 0, c->stream>>>(static_cast<T*>(field), grid_params<T>(c), gh[0], gh[1], gh[2]);
    c->launches++;
}

bool streaming(mr_ctx* c, mr_operator op)
{
    ensure_plans(c);
    if (c->force_variant != 0) return false;
    return op == MR_OP_MIMETIC ? c->plan_mim.usable : c->plan_dir.usable;
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
    wrap_ghosts<T>(c, c->b());
    MR_CUDA(c, cudaGetLastError());
    c->have_B0 = true;
    return MR_OK;
}

// x (as_xi = false) or xi (as_xi = true), dense -> the other state buffer; adopted if the line-tied faces are on X
template <typename T>
mr_status do_set_x(mr_ctx* c, const void* src, bool as_xi)
{
    dim3 grid, block;
    node_launch_dims(c, grid, block);
    const int other = 1 - c->cur;
    MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, sizeof(int), c->stream));
    if (as_xi)
        k_import_xi<T><<<grid, block, 0, c->stream>>>(static_cast<const T*>(src), static_cast<T*>(c->xi(other)), grid_params<T>(c), c->flag());
    else
        k_import_x<T><<<grid, block, 0, c->stream>>>(static_cast<const T*>(src), static_cast<T*>(c->xi(other)), grid_params<T>(c),
                                                     domain_params(c), c->flag());
    c->launches++;
    wrap_ghosts<T>(c, c->xi(other));
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
        k_fields<T, 0><<<grid, block, 0, c->stream>>>(xi, b, grid_params<double>(c), domain_params(c), static_cast<T*>(x_out),
                                                      static_cast<T*>(B_out), static_cast<T*>(J_out), c->flag());
    else
        k_fields<T, 1><<<grid, block, 0, c->stream>>>(xi, b, grid_params<double>(c), domain_params(c), static_cast<T*>(x_out),
                                                      static_cast<T*>(B_out), static_cast<T*>(J_out), c->flag());
    c->launches++;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

// One pass of the hot path over the state in buffer `in` (0, 1: the state buffers, 2: the adaptive stage buffer):
// rhs = false: out = xi + dtg J x B (a step), rhs = true: out = dtg J x B (the velocity for dtg = gamma).
template <typename T>
mr_status launch_pass(mr_ctx* c, mr_operator op, int in, void* out, double dtg_d, bool rhs)
{
    const T dtg = (T)dtg_d;
    if (streaming(c, op)) {
        cudaError_t e = op == MR_OP_MIMETIC ? launch_sym_step<T>(c->plan_mim, in, dtg, c->flag(), c->stream, rhs, out)
                                            : launch_direct_step<T>(c->plan_dir, in, dtg, c->flag(), c->stream, rhs, out);
        if (e != cudaSuccess) return cuda_fail(c, "streaming step launch", e);
        c->variant = op == MR_OP_MIMETIC ? c->plan_mim.name : c->plan_dir.name;
    } else {
        dim3 grid, block;
        node_launch_dims(c, grid, block);
        const T* src = static_cast<const T*>(in == 2 ? c->kbuf(6) : c->xi(in));
        const T* b = static_cast<const T*>(c->b());
        T* o = static_cast<T*>(out);
        const GridP<T> g = grid_params<T>(c);
        if (op == MR_OP_MIMETIC) {
            if (rhs) k_step_generic<T, 0, true><<<grid, block, 0, c->stream>>>(src, o, b, g, dtg, c->flag());
            else k_step_generic<T, 0, false><<<grid, block, 0, c->stream>>>(src, o, b, g, dtg, c->flag());
        } else {
            if (rhs) k_step_generic<T, 1, true><<<grid, block, 0, c->stream>>>(src, o, b, g, dtg, c->flag());
            else k_step_generic<T, 1, false><<<grid, block, 0, c->stream>>>(src, o, b, g, dtg, c->flag());
        }
        c->variant = op == MR_OP_MIMETIC ? "generic_mimetic" : "generic_direct";
    }
    c->launches++;
    return MR_OK;
}

constexpr int kStepsPerGraph = 16;          // even: the state is back in the buffer it started from

template <typename T>
mr_status launch_steps(mr_ctx* c, int64_t n, double dtg, mr_operator op)
{
    for (int64_t s = 0; s < n; ++s) {
        mr_status st = launch_pass<T>(c, op, c->cur, c->xi(1 - c->cur), dtg, false);
        if (st != MR_OK) return st;
        wrap_ghosts<T>(c, c->xi(1 - c->cur));
        c->cur = 1 - c->cur;
    }
    return MR_OK;
}

// the graph of kStepsPerGraph steps from the buffer c->cur with this operator, dt and kernel choice (captured on first use,
// re-captured when any of them changes); null if the stream cannot be captured right now (e.g. the caller is capturing)
template <typename T>
cudaGraphExec_t step_graph_for(mr_ctx* c, double dtg, mr_operator op)
{
    if (c->step_graph && c->sg_op == (int)op && c->sg_cur == c->cur && c->sg_variant == c->force_variant && c->sg_dtg == dtg)
        return c->step_graph;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(c->stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); return nullptr; }
    if (c->step_graph) { cudaGraphExecDestroy(c->step_graph); c->step_graph = nullptr; }
    ensure_plans(c);                                   // (tensor maps and function attributes: not inside a capture)
    if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
        c->cap_stream = nullptr;
        cudaGetLastError();
        return nullptr;
    }
    if (cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    const int64_t launches0 = c->launches;
    const int cur0 = c->cur;
    cudaStream_t user = c->stream;
    c->stream = c->cap_stream;
    const mr_status st = launch_steps<T>(c, kStepsPerGraph, dtg, op);
    c->stream = user;
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
    c->launches = launches0;                            // nothing ran
    c->cur = cur0;
    if (st != MR_OK || e != cudaSuccess || !g) { if (g) cudaGraphDestroy(g); cudaGetLastError(); return nullptr; }
    cudaGraphExec_t ex = nullptr;
    if (cudaGraphInstantiate(&ex, g, 0) != cudaSuccess) { ex = nullptr; cudaGetLastError(); }
    cudaGraphDestroy(g);
    c->step_graph = ex;
    c->sg_op = (int)op; c->sg_cur = c->cur; c->sg_variant = c->force_variant; c->sg_dtg = dtg;
    return ex;
}

template <typename T>
mr_status do_step(mr_ctx* c, int64_t n, double dt, mr_operator op)
{
    MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, sizeof(int), c->stream));
    const double dtg = dt * c->gamma;
    int64_t left = n;
    // a grid whose three fields fit the L2 is bound by launch latency: replay kStepsPerGraph steps per graph launch
    if (c->graphs_enabled && n >= 2 * kStepsPerGraph && 3 * c->L.field_bytes <= ((size_t)96 << 20)) {
        if (cudaGraphExec_t ex = step_graph_for<T>(c, dtg, op)) {
            const int64_t per_graph = (c->any_periodic ? 2 : 1) * kStepsPerGraph;
            for (; left >= kStepsPerGraph; left -= kStepsPerGraph) {
                MR_CUDA(c, cudaGraphLaunch(ex, c->stream));
                c->launches += per_graph;
            }
            c->variant = streaming(c, op) ? (op == MR_OP_MIMETIC ? c->plan_mim.name : c->plan_dir.name)
                                          : (op == MR_OP_MIMETIC ? "generic_mimetic" : "generic_direct");
        }
    }
    {
        mr_status st = launch_steps<T>(c, left, dtg, op);
        if (st != MR_OK) return st;
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

// S6 of the current state, enqueued: the four raw sums / extrema into *dst (device)
template <typename T>
mr_status enqueue_diag(mr_ctx* c, mr_operator op, DiagPartial* dst)
{
    const long long rows = (long long)c->grid.ny * c->grid.nz;
    int blocks = c->sm_count * 8;
    if (blocks > kMaxPartialBlocks) blocks = kMaxPartialBlocks;
    if (blocks > rows) blocks = (int)rows;
    const T* xi = static_cast<const T*>(c->xi(c->cur));
    const T* b = static_cast<const T*>(c->b());
    const int threads = c->grid.nx >= 256 ? 256 : (c->grid.nx >= 128 ? 128 : (c->grid.nx >= 64 ? 64 : 32));
    const bool stream_ok = streaming(c, op);
    const StreamPlan& pl = op == MR_OP_MIMETIC ? c->plan_mim : c->plan_dir;
    const Tiling& tl = op == MR_OP_MIMETIC ? pl.all : pl.step;
    const bool fused = stream_ok && tl.tiles_x * tl.tiles_y * tl.nchunks <= kMaxPartialBlocks;
    int total = blocks;
    if (fused && op == MR_OP_MIMETIC) {
        // the streaming pass of the step kernel with the update replaced by the reduction (mr_sym.cuh, MODE_DIAG)
        cudaError_t e = launch_sym_diag<T>(c->plan_mim, c->cur, c->partials(), &total, c->flag(), c->stream);
        if (e != cudaSuccess) return cuda_fail(c, "streaming diagnostics launch", e);
        c->launches++;
    } else if (fused) {
        // direct operator: the inner nodes by the streaming pass, the nodes on the faces by a pass of their own
        int inner_blocks = 0;
        cudaError_t e = launch_direct_diag<T>(c->plan_dir, c->cur, c->partials(), &inner_blocks, c->flag(), c->stream);
        if (e != cudaSuccess) return cuda_fail(c, "streaming diagnostics launch", e);
        k_diag_faces<T><<<blocks, 128, 0, c->stream>>>(xi, b, grid_params<T>(c), c->partials() + inner_blocks, c->flag());
        total = inner_blocks + blocks;
        c->launches += 2;
    } else {
        if (op == MR_OP_MIMETIC) k_diag<T, 0><<<blocks, threads, 0, c->stream>>>(xi, b, grid_params<T>(c), c->partials(), c->flag());
        else k_diag<T, 1><<<blocks, threads, 0, c->stream>>>(xi, b, grid_params<T>(c), c->partials(), c->flag());
        c->launches++;
    }
    k_diag_final<<<1, 256, 0, c->stream>>>(c->partials(), total, dst);
    c->launches++;
    MR_CUDA(c, cudaGetLastError());
    return MR_OK;
}

void fill_diag(const mr_ctx* c, const DiagPartial& r, double time, int64_t steps, mr_diag* out)
{
    out->time = time;
    out->steps = steps;
    out->energy = r.e / 16.0;
    out->max_jxb = r.fmax;
    out->xi = r.xi;
    out->min_det = r.dmin / (8.0 * c->h[0] * c->h[1] * c->h[2]);
}

template <typename T>
mr_status do_diag(mr_ctx* c, mr_operator op, mr_diag* out)
{
    MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, sizeof(int), c->stream));
    mr_status st = enqueue_diag<T>(c, op, c->diag_out());
    if (st != MR_OK) return st;
    DiagPartial r;
    MR_CUDA(c, cudaMemcpyAsync(&r, c->diag_out(), sizeof(r), cudaMemcpyDeviceToHost, c->stream));
    int f = 0;
    st = read_flag(c, &f);
    if (st != MR_OK) return st;
    fill_diag(c, r, c->time, c->steps, out);
    if (f & FLAG_NUMERIC) return fail(c, MR_ERR_NUMERIC, "mr_diagnostics: det(dx/dX) <= 0 or a non-finite value was met");
    return MR_OK;
}

// n steps; every `every`-th of them (the first included) also reduces S6 of the state it STARTS from.  The mimetic streaming
// kernel does both in one pass (MODE_STEPDIAG: the diagnosis costs no memory traffic); otherwise S6 is a pass of its own.  The
// records stay on the device, kHistoryBatch at a time.
template <typename T>
mr_status do_step_monitored(mr_ctx* c, int64_t n, double dt, mr_operator op, int64_t every, mr_diag* hist, int64_t cap, int64_t* written)
{
    MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, sizeof(int), c->stream));
    const double dtg = dt * c->gamma;
    const bool fused = op == MR_OP_MIMETIC && streaming(c, op) &&
                       c->plan_mim.all.tiles_x * c->plan_mim.all.tiles_y * c->plan_mim.all.nchunks <= kMaxPartialBlocks;
    static thread_local DiagPartial host[kHistoryBatch];
    double times[kHistoryBatch];
    int64_t stepno[kHistoryBatch];
    int64_t total = 0;
    int pending = 0;
    auto flush = [&]() -> mr_status {
        if (!pending) return MR_OK;
        MR_CUDA(c, cudaMemcpyAsync(host, c->history(), sizeof(DiagPartial) * pending, cudaMemcpyDeviceToHost, c->stream));
        MR_CUDA(c, cudaStreamSynchronize(c->stream));
        for (int q = 0; q < pending; ++q) fill_diag(c, host[q], times[q], stepno[q], hist + total + q);
        total += pending;
        pending = 0;
        return MR_OK;
    };
    const double t0 = c->time;
    const int64_t s0 = c->steps;
    for (int64_t s = 0; s < n; ++s) {
        // (the clock follows the state: an early return below leaves time / steps at the step the state has reached)
        c->time = t0 + dt * (double)s;
        c->steps = s0 + s;
        const bool rec = every > 0 && s % every == 0 && total + pending < cap;
        if (rec) {
            times[pending] = t0 + dt * (double)s;
            stepno[pending] = s0 + s;
        }
        if (rec && fused) {
            int nb = 0;
            cudaError_t e = launch_sym_stepdiag<T>(c->plan_mim, c->cur, (T)dtg, c->partials(), &nb, c->flag(), c->stream);
            if (e != cudaSuccess) return cuda_fail(c, "streaming step + diagnostics launch", e);
            k_diag_final<<<1, 256, 0, c->stream>>>(c->partials(), nb, c->history() + pending);
            c->launches += 2;
            c->variant = c->plan_mim.name;
            wrap_ghosts<T>(c, c->xi(1 - c->cur));
            c->cur = 1 - c->cur;
        } else {
            if (rec) {
                mr_status st = enqueue_diag<T>(c, op, c->history() + pending);
                if (st != MR_OK) return st;
            }
            mr_status st = launch_steps<T>(c, 1, dtg, op);
            if (st != MR_OK) return st;
        }
        if (rec && ++pending == kHistoryBatch) {
            mr_status st = flush();
            if (st != MR_OK) return st;
        }
    }
    c->time = t0 + dt * (double)n;
    c->steps = s0 + n;
    MR_CUDA(c, cudaGetLastError());
    mr_status st = flush();
    if (st != MR_OK) return st;
    if (written) *written = total;
    int f = 0;
    st = read_flag(c, &f);
    if (st != MR_OK) return st;
    if (f & FLAG_NUMERIC) {
        c->failed = true;
        return fail(c, MR_ERR_NUMERIC, "mr_step_monitored: det(dx/dX) <= 0 or a non-finite value was met");
    }
    return MR_OK;
}

// ---- section 2.4: one Cash-Karp trial step from the state buffer `cur`; the fifth-order solution goes to the other
// state buffer.  Everything is enqueued on c->stream and nothing depends on the step length, which the kernels read from
// dt_dev(): pinned[0] -> dt_dev() goes in first, the flag -> pinned[1] and Lambda = max |x5 - x4| -> pinned[2] come out last.
template <typename T>
mr_status enqueue_trial(mr_ctx* c, mr_operator op)
{
    static const CashKarp ck = cash_karp();
    const long long n2 = 3 * c->L.comp / 2;             // element pairs of a padded field (pitch is a multiple of 16)
    const int blocks = c->sm_count * 8 < kMaxPartialBlocks ? c->sm_count * 8 : kMaxPartialBlocks;
    const T* x = static_cast<const T*>(c->xi_raw(c->cur));      // the elementwise kernels run over the whole padded fields
    T* xs = static_cast<T*>(c->kbuf_raw(6));
    MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, 16, c->stream));                  // the flag and Lambda (an atomic maximum from 0)
    MR_CUDA(c, cudaMemcpyAsync(c->dt_dev(), c->pinned, sizeof(double), cudaMemcpyHostToDevice, c->stream));
    for (int s = 0; s < 6; ++s) {
        if (s > 0) {
            StageArgs a;
            a.n = s;
            for (int r = 0; r < 6; ++r) { a.k[r] = c->kbuf_raw(r < s ? r : 0); a.c[r] = r < s ? ck.a[s][r] : 0.0; }
            k_rk_stage<T><<<blocks, 256, 0, c->stream>>>(x, xs, a, n2, c->dt_dev());
            c->launches++;
            wrap_ghosts<T>(c, c->kbuf(6));                        // (the ghosts of the k_r are not kept)
        }
        mr_status st = launch_pass<T>(c, op, s == 0 ? c->cur : 2, c->kbuf(s), c->gamma, true);
        if (st != MR_OK) return st;
    }
    StageArgs b5, db;
    b5.n = db.n = 6;
    for (int r = 0; r < 6; ++r) { b5.k[r] = db.k[r] = c->kbuf_raw(r); b5.c[r] = ck.b5[r]; db.c[r] = ck.db[r]; }
    k_rk_final<T><<<blocks, 256, 0, c->stream>>>(x, static_cast<T*>(c->xi_raw(1 - c->cur)), b5, db, n2, c->lambda_dev(), c->dt_dev());
    c->launches++;
    wrap_ghosts<T>(c, c->xi(1 - c->cur));
    MR_CUDA(c, cudaGetLastError());
    MR_CUDA(c, cudaMemcpyAsync(c->pinned + 1, c->flag(), 16, cudaMemcpyDeviceToHost, c->stream));    // the flag, Lambda
    return MR_OK;
}

// the captured trial step for this operator and state buffer (null: not available, enqueue the launches instead)
template <typename T>
cudaGraphExec_t trial_graph_for(mr_ctx* c, mr_operator op)
{
    const int o = op == MR_OP_MIMETIC ? 0 : 1, w = c->cur;
    if (c->trial_graph[o][w] && c->tg_variant[o][w] == c->force_variant) return c->trial_graph[o][w];
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(c->stream, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); return nullptr; }
    if (c->trial_graph[o][w]) { cudaGraphExecDestroy(c->trial_graph[o][w]); c->trial_graph[o][w] = nullptr; }
    ensure_plans(c);
    if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
        c->cap_stream = nullptr;
        cudaGetLastError();
        return nullptr;
    }
    if (cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    const int64_t launches0 = c->launches;
    cudaStream_t user = c->stream;
    c->stream = c->cap_stream;
    const mr_status st = enqueue_trial<T>(c, op);
    c->stream = user;
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
    c->tg_launches[o][w] = c->launches - launches0;
    c->launches = launches0;                            // nothing ran
    if (st != MR_OK || e != cudaSuccess || !g) { if (g) cudaGraphDestroy(g); cudaGetLastError(); return nullptr; }
    cudaGraphExec_t ex = nullptr;
    if (cudaGraphInstantiate(&ex, g, 0) != cudaSuccess) { ex = nullptr; cudaGetLastError(); }
    cudaGraphDestroy(g);
    c->trial_graph[o][w] = ex;
    c->tg_variant[o][w] = c->force_variant;
    return ex;
}

// one trial step of length h: Lambda comes back (the one device -> host exchange of the step)
template <typename T>
mr_status rk_trial(mr_ctx* c, mr_operator op, double h, double* lambda, int* numeric)
{
    if (!c->pinned) MR_CUDA(c, cudaHostAlloc(reinterpret_cast<void**>(&c->pinned), 4 * sizeof(double), cudaHostAllocDefault));
    c->pinned[0] = h;
    cudaGraphExec_t ex = c->graphs_enabled ? trial_graph_for<T>(c, op) : nullptr;
    if (ex) {
        MR_CUDA(c, cudaGraphLaunch(ex, c->stream));
        c->launches += c->tg_launches[op == MR_OP_MIMETIC ? 0 : 1][c->cur];
        c->variant = streaming(c, op) ? (op == MR_OP_MIMETIC ? c->plan_mim.name : c->plan_dir.name)
                                      : (op == MR_OP_MIMETIC ? "generic_mimetic" : "generic_direct");
    } else {
        mr_status st = enqueue_trial<T>(c, op);
        if (st != MR_OK) return st;
    }
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    *numeric = *reinterpret_cast<const int*>(c->pinned + 1);
    *lambda = c->pinned[2];
    return MR_OK;
}

constexpr int kMaxFoldedTrials = 40;     // trials in a row that may fold the grid (each retried at dt/2) before the run is given up

// Eq. 2.11 and the accept / reject rule of PAPER.md:139-143 (reading Q22)
bool step_control(double dt, double lambda, double lambda0, double* dt_next)
{
    if (lambda > lambda0 || lambda != lambda) {
        // (a retry is at most 0.9 dt: just above lambda0 the factor of Eq. 2.11 rounds to 1 and the trial would repeat for ever)
        const double f = lambda != lambda ? 0.5 : std::pow(std::fabs(lambda0 / lambda), 0.2);
        *dt_next = dt * (f < 0.9 ? f : 0.9);
        return false;
    }
    if (lambda < 0.5 * lambda0) {
        const double f = lambda > 0.0 ? std::pow(std::fabs(lambda0 / lambda), 0.2) : 5.0;
        *dt_next = dt * (f > 5.0 ? 5.0 : f);
    } else {
        *dt_next = dt;
    }
    return true;
}

template <typename T>
mr_status do_adaptive(mr_ctx* c, double t_end, double lambda0, double* dt, mr_operator op, int64_t max_trials, mr_adapt_stats* stats,
                      double* trace, int64_t trace_cap)
{
    mr_adapt_stats s = { 0, 0, 0, c->time, *dt, 0.0 };
    int64_t trials = 0;
    int folded_in_a_row = 0;            // DESIGN.md reading Q26
    mr_status rc = MR_OK;
    while (c->time < t_end) {
        if (trials >= max_trials) { rc = fail(c, MR_ERR_INVALID_ARG, "mr_step_adaptive: max_trials exhausted before t_end"); break; }
        const double rest = t_end - c->time;
        const bool clipped = *dt >= rest;
        const double h = clipped ? rest : *dt;
        double lam = 0.0, dt_next = 0.0;
        int numeric = 0;
        rc = rk_trial<T>(c, op, h, &lam, &numeric);
        if (rc != MR_OK) break;
        s.rhs_evals += 6;
        if (numeric & FLAG_NUMERIC) { lam = NAN; ++folded_in_a_row; }   // a stage folded the grid: the trial counts as failed
        else folded_in_a_row = 0;
        s.last_lambda = lam;
        const bool ok = step_control(h, lam, lambda0, &dt_next);
        if (trace && trials < trace_cap) {
            trace[4 * trials + 0] = c->time; trace[4 * trials + 1] = h; trace[4 * trials + 2] = lam; trace[4 * trials + 3] = ok ? 1.0 : 0.0;
        }
        ++trials;
        if (ok) {
            c->cur = 1 - c->cur;
            c->time = clipped ? t_end : c->time + h;
            c->steps++;
            s.accepted++;
            if (!clipped || dt_next < *dt) *dt = dt_next;     // a clipped last step does not change the dt handed on
        } else {
            s.rejected++;
            *dt = dt_next;
            if (folded_in_a_row >= kMaxFoldedTrials || !(dt_next > 1e-300)) {
                rc = fail(c, MR_ERR_NUMERIC, "mr_step_adaptive: the step length collapsed (cf. PAPER.md:333)");
                break;
            }
        }
    }
    s.time = c->time;
    s.dt_next = *dt;
    if (stats) *stats = s;
    return rc;
}

template <typename T>
mr_status do_eps_star(mr_ctx* c, mr_operator op, int ic, int jc, double a_r, double* alpha_host, double* eps)
{
    double* alpha = reinterpret_cast<double*>(c->partials());          // nz <= 4096 doubles fit the partials area
    const T* xi = static_cast<const T*>(c->xi(c->cur));
    const T* b = static_cast<const T*>(c->b());
    MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, sizeof(int), c->stream));
    const int nz = c->grid.nz;
    if (op == MR_OP_MIMETIC) k_alpha_line<T, 0><<<(nz + 63) / 64, 64, 0, c->stream>>>(xi, b, grid_params<T>(c), ic, jc, alpha, c->flag());
    else k_alpha_line<T, 1><<<(nz + 63) / 64, 64, 0, c->stream>>>(xi, b, grid_params<T>(c), ic, jc, alpha, c->flag());
    const int k_lo = c->per[2] ? 0 : 1, k_hi = c->per[2] ? nz - 1 : nz - 2;
    k_eps_star<<<1, 256, 0, c->stream>>>(alpha, k_lo, k_hi, a_r, c->h[2], reinterpret_cast<double*>(c->diag_out()));
    c->launches += 2;
    MR_CUDA(c, cudaGetLastError());
    if (alpha_host) MR_CUDA(c, cudaMemcpyAsync(alpha_host, alpha, sizeof(double) * nz, cudaMemcpyDeviceToHost, c->stream));
    MR_CUDA(c, cudaMemcpyAsync(eps, c->diag_out(), sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    int f = 0;
    mr_status st = read_flag(c, &f);
    if (st != MR_OK) return st;
    if (f & FLAG_NUMERIC) return fail(c, MR_ERR_NUMERIC, "mr_eps_star: det(dx/dX) <= 0 on the line");
    return MR_OK;
}

template <typename T>
mr_status do_sigma(mr_ctx* c, const void* x_ref, const void* B_ref, double* sx, double* sb)
{
    const long long rows = (long long)c->grid.ny * c->grid.nz;
    int blocks = c->sm_count * 8 < kMaxPartialBlocks ? c->sm_count * 8 : kMaxPartialBlocks;
    if (blocks > rows) blocks = (int)rows;
    SumPair* partials = reinterpret_cast<SumPair*>(c->partials());
    k_sigma<T><<<blocks, 256, 0, c->stream>>>(static_cast<const T*>(c->xi(c->cur)), static_cast<const T*>(c->b()), grid_params<T>(c),
                                              domain_params(c), static_cast<const T*>(x_ref), static_cast<const T*>(B_ref), partials);
    k_sum_final<<<1, 32, 0, c->stream>>>(partials, blocks, reinterpret_cast<SumPair*>(c->diag_out()));
    c->launches += 2;
    MR_CUDA(c, cudaGetLastError());
    SumPair r;
    MR_CUDA(c, cudaMemcpyAsync(&r, c->diag_out(), sizeof(r), cudaMemcpyDeviceToHost, c->stream));
    MR_CUDA(c, cudaStreamSynchronize(c->stream));
    const double N = (double)c->grid.nx * c->grid.ny * c->grid.nz;
    *sx = std::sqrt(r.a / N);
    *sb = std::sqrt(r.b / N);
    return MR_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------- C ABI

extern "C" size_t mr_workspace_bytes(const mr_grid* grid, mr_dtype dtype)
{
    Layout L;
    return make_layout(grid, dtype, nullptr, &L) ? L.total : 0;
}

namespace {
bool periodic_axes(const int32_t* bc, int (&per)[3])
{
    for (int a = 0; a < 3; ++a) {
        if (!bc || (bc[a] != MR_BC_LINE_TIED && bc[a] != MR_BC_PERIODIC)) return false;
        per[a] = bc[a] == MR_BC_PERIODIC ? 1 : 0;
    }
    return true;
}
}  // namespace

extern "C" size_t mr_workspace_bytes_bc(const mr_grid* grid, mr_dtype dtype, const int32_t* bc)
{
    Layout L;
    int per[3];
    return periodic_axes(bc, per) && make_layout(grid, dtype, per, &L) ? L.total : 0;
}

extern "C" size_t mr_adaptive_workspace_bytes_bc(const mr_grid* grid, mr_dtype dtype, const int32_t* bc)
{
    Layout L;
    int per[3];
    return periodic_axes(bc, per) && make_layout(grid, dtype, per, &L) ? L.adaptive_total : 0;
}

extern "C" size_t mr_adaptive_workspace_bytes(const mr_grid* grid, mr_dtype dtype)
{
    Layout L;
    return make_layout(grid, dtype, nullptr, &L) ? L.adaptive_total : 0;
}

extern "C" mr_status mr_create(const mr_grid* grid, const mr_domain* domain, const mr_boundary* boundary, mr_ctx** out)
{
    if (out) *out = nullptr;
    if (!grid || !domain || !boundary || !out) return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: null argument");
    Layout L;
    if (!make_layout(grid, boundary->dtype, nullptr, &L))
        return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: each of nx, ny, nz must be in [5, 4096] and dtype MR_F64 or MR_F32");
    int per[3] = { 0, 0, 0 };
    for (int a = 0; a < 3; ++a) {
        per[a] = boundary->bc[a] == MR_BC_PERIODIC ? 1 : 0;
        if (!std::isfinite(domain->lo[a]) || !std::isfinite(domain->hi[a]) || !(domain->hi[a] > domain->lo[a]))
            return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: domain needs finite hi > lo on every axis");
        if (boundary->bc[a] != MR_BC_LINE_TIED && boundary->bc[a] != MR_BC_PERIODIC)
            return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: unknown boundary type");
    }
    if (!(boundary->gamma > 0.0) || !std::isfinite(boundary->gamma))
        return fail(nullptr, MR_ERR_INVALID_ARG, "mr_create: gamma must be finite and > 0");
    if (!boundary->workspace || (reinterpret_cast<uintptr_t>(boundary->workspace) % kAlign) != 0)
        return fail(nullptr, MR_ERR_WORKSPACE, "mr_create: workspace is null or not 256-byte aligned");
    make_layout(grid, boundary->dtype, per, &L);      // (ghost layers on the periodic axes)
    if (boundary->workspace_bytes < L.total)
        return fail(nullptr, MR_ERR_WORKSPACE, "mr_create: workspace smaller than mr_workspace_bytes_bc()");

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
    c->any_periodic = false;
    for (int a = 0; a < 3; ++a) {
        c->h[a] = (domain->hi[a] - domain->lo[a]) / (double)(n[a] - 1);
        c->per[a] = boundary->bc[a] == MR_BC_PERIODIC ? 1 : 0;
        c->any_periodic = c->any_periodic || c->per[a];
    }
    c->L = L;
    c->ws = static_cast<char*>(boundary->workspace);
    c->aws = nullptr;
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
    c->plans_built = false;

    cudaError_t e = cudaMemsetAsync(c->ws, 0, L.off_stage, c->stream);   // xi = 0 (x = X), b = 0, incl. padding
    if (e == cudaSuccess) e = cudaMemsetAsync(c->ws + L.off_partials, 0, L.total - L.off_partials, c->stream);
    if (e != cudaSuccess) { delete c; return cuda_fail(nullptr, "mr_create: cudaMemsetAsync", e); }
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
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_set_x: mr_step_host_async calls are in flight (mr_host_sync first)");
    if (!x_dev) return fail(ctx, MR_ERR_INVALID_ARG, "mr_set_x: null pointer");
    return ctx->dtype == MR_F64 ? do_set_x<double>(ctx, x_dev, false) : do_set_x<float>(ctx, x_dev, false);
}

extern "C" mr_status mr_set_x_host(mr_ctx* ctx, const void* x_host)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!x_host) return fail(ctx, MR_ERR_INVALID_ARG, "mr_set_x_host: null pointer");
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_set_x_host: mr_step_host_async calls are in flight (mr_host_sync first)");
    MR_CUDA(ctx, cudaMemcpyAsync(ctx->stage(), x_host, ctx->dense_bytes(), cudaMemcpyHostToDevice, ctx->stream));
    return mr_set_x(ctx, ctx->stage());
}

extern "C" mr_status mr_set_xi(mr_ctx* ctx, const void* xi_dev)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_set_xi: mr_step_host_async calls are in flight (mr_host_sync first)");
    if (!xi_dev) return fail(ctx, MR_ERR_INVALID_ARG, "mr_set_xi: null pointer");
    return ctx->dtype == MR_F64 ? do_set_x<double>(ctx, xi_dev, true) : do_set_x<float>(ctx, xi_dev, true);
}

extern "C" mr_status mr_get_xi(mr_ctx* ctx, void* xi_dev)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!xi_dev) return fail(ctx, MR_ERR_INVALID_ARG, "mr_get_xi: null pointer");
    dim3 grid, block;
    node_launch_dims(ctx, grid, block);
    if (ctx->dtype == MR_F64)
        k_export_padded<double><<<grid, block, 0, ctx->stream>>>(static_cast<const double*>(ctx->xi(ctx->cur)), static_cast<double*>(xi_dev), grid_params<double>(ctx));
    else
        k_export_padded<float><<<grid, block, 0, ctx->stream>>>(static_cast<const float*>(ctx->xi(ctx->cur)), static_cast<float*>(xi_dev), grid_params<float>(ctx));
    ctx->launches++;
    MR_CUDA(ctx, cudaGetLastError());
    return MR_OK;
}

extern "C" mr_status mr_step(mr_ctx* ctx, int64_t n, double dt, mr_operator op)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_step: mr_step_host_async calls are in flight (mr_host_sync first)");
    if (n < 0 || !(dt > 0.0) || !std::isfinite(dt)) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step: need n >= 0 and finite dt > 0");
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step: unknown operator");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_step: B0 has not been set");
    if (ctx->failed) return fail(ctx, MR_ERR_NUMERIC, "mr_step: context is in the failed state (call mr_set_x)");
    return ctx->dtype == MR_F64 ? do_step<double>(ctx, n, dt, op) : do_step<float>(ctx, n, dt, op);
}

extern "C" mr_status mr_step_monitored(mr_ctx* ctx, int64_t n, double dt, mr_operator op, int64_t every, mr_diag* history_host,
                                       int64_t capacity, int64_t* written)
{
    if (written) *written = 0;
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_step_monitored: mr_step_host_async calls are in flight (mr_host_sync first)");
    if (n < 0 || !(dt > 0.0) || !std::isfinite(dt)) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step_monitored: need n >= 0 and finite dt > 0");
    if (every < 0 || capacity < 0 || (every > 0 && capacity > 0 && !history_host))
        return fail(ctx, MR_ERR_INVALID_ARG, "mr_step_monitored: need every >= 0, capacity >= 0 and a history array");
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step_monitored: unknown operator");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_step_monitored: B0 has not been set");
    if (ctx->failed) return fail(ctx, MR_ERR_NUMERIC, "mr_step_monitored: context is in the failed state (call mr_set_x)");
    return ctx->dtype == MR_F64 ? do_step_monitored<double>(ctx, n, dt, op, every, history_host, capacity, written)
                                : do_step_monitored<float>(ctx, n, dt, op, every, history_host, capacity, written);
}

extern "C" mr_status mr_rhs(mr_ctx* ctx, mr_operator op, void* u_dev)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!u_dev) return fail(ctx, MR_ERR_INVALID_ARG, "mr_rhs: null pointer");
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_rhs: unknown operator");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_rhs: B0 has not been set");
    // the velocity in the padded layout into the spare state buffer, then dense into the caller's array
    void* tmp = ctx->xi(1 - ctx->cur);
    mr_status st = ctx->dtype == MR_F64 ? launch_pass<double>(ctx, op, ctx->cur, tmp, ctx->gamma, true)
                                        : launch_pass<float>(ctx, op, ctx->cur, tmp, ctx->gamma, true);
    if (st != MR_OK) return st;
    dim3 grid, block;
    node_launch_dims(ctx, grid, block);
    if (ctx->dtype == MR_F64)
        k_export_padded<double><<<grid, block, 0, ctx->stream>>>(static_cast<const double*>(tmp), static_cast<double*>(u_dev), grid_params<double>(ctx));
    else
        k_export_padded<float><<<grid, block, 0, ctx->stream>>>(static_cast<const float*>(tmp), static_cast<float*>(u_dev), grid_params<float>(ctx));
    ctx->launches++;
    MR_CUDA(ctx, cudaGetLastError());
    return MR_OK;
}

extern "C" mr_status mr_bind_adaptive_workspace(mr_ctx* ctx, void* workspace_dev, size_t bytes)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!workspace_dev || (reinterpret_cast<uintptr_t>(workspace_dev) % kAlign) != 0)
        return fail(ctx, MR_ERR_WORKSPACE, "mr_bind_adaptive_workspace: workspace is null or not 256-byte aligned");
    if (bytes < ctx->L.adaptive_total)
        return fail(ctx, MR_ERR_WORKSPACE, "mr_bind_adaptive_workspace: smaller than mr_adaptive_workspace_bytes_bc()");
    ctx->aws = static_cast<char*>(workspace_dev);
    for (int o = 0; o < 2; ++o)                   // captured trial steps point into the previous buffer
        for (int w = 0; w < 2; ++w)
            if (ctx->trial_graph[o][w]) { cudaGraphExecDestroy(ctx->trial_graph[o][w]); ctx->trial_graph[o][w] = nullptr; }
    MR_CUDA(ctx, cudaMemsetAsync(ctx->aws, 0, ctx->L.adaptive_total, ctx->stream));       // the padding must stay finite
    if (ctx->plans_built) {
        if (ctx->plan_mim.usable && !sym_bind_stage(&ctx->plan_mim, ctx->kbuf_raw(6))) ctx->plan_mim.usable = false;
        if (ctx->plan_dir.usable && !direct_bind_stage(&ctx->plan_dir, ctx->kbuf_raw(6))) ctx->plan_dir.usable = false;
    }
    return MR_OK;
}

extern "C" mr_status mr_step_adaptive(mr_ctx* ctx, double t_end, double lambda0, double* dt, mr_operator op, int64_t max_trials,
                                      mr_adapt_stats* stats, double* trace_host, int64_t trace_cap)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_step_adaptive: mr_step_host_async calls are in flight (mr_host_sync first)");
    if (!dt || !(*dt > 0.0) || !std::isfinite(*dt) || !(lambda0 > 0.0) || !std::isfinite(t_end) || max_trials < 0)
        return fail(ctx, MR_ERR_INVALID_ARG, "mr_step_adaptive: need finite t_end, lambda0 > 0, *dt > 0, max_trials >= 0");
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step_adaptive: unknown operator");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_step_adaptive: B0 has not been set");
    if (!ctx->aws) return fail(ctx, MR_ERR_STATE, "mr_step_adaptive: no adaptive workspace bound (mr_bind_adaptive_workspace)");
    if (ctx->failed) return fail(ctx, MR_ERR_NUMERIC, "mr_step_adaptive: context is in the failed state (call mr_set_x)");
    return ctx->dtype == MR_F64 ? do_adaptive<double>(ctx, t_end, lambda0, dt, op, max_trials, stats, trace_host, trace_cap)
                                : do_adaptive<float>(ctx, t_end, lambda0, dt, op, max_trials, stats, trace_host, trace_cap);
}

extern "C" mr_status mr_diagnostics(mr_ctx* ctx, mr_operator op, mr_diag* out)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_diagnostics: mr_step_host_async calls are in flight (mr_host_sync first)");
    if (!out) return fail(ctx, MR_ERR_INVALID_ARG, "mr_diagnostics: null output");
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_diagnostics: unknown operator");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_diagnostics: B0 has not been set");
    return ctx->dtype == MR_F64 ? do_diag<double>(ctx, op, out) : do_diag<float>(ctx, op, out);
}

extern "C" mr_status mr_convexity(mr_ctx* ctx, int32_t* kappa_dev, int64_t* n_concave)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!n_concave) return fail(ctx, MR_ERR_INVALID_ARG, "mr_convexity: null output");
    dim3 grid, block;
    node_launch_dims(ctx, grid, block);
    unsigned long long* cnt = reinterpret_cast<unsigned long long*>(ctx->diag_out());
    MR_CUDA(ctx, cudaMemsetAsync(cnt, 0, sizeof(unsigned long long), ctx->stream));
    if (ctx->dtype == MR_F64)
        k_convexity<double><<<grid, block, 0, ctx->stream>>>(static_cast<const double*>(ctx->xi(ctx->cur)), grid_params<double>(ctx), kappa_dev, cnt);
    else
        k_convexity<float><<<grid, block, 0, ctx->stream>>>(static_cast<const float*>(ctx->xi(ctx->cur)), grid_params<float>(ctx), kappa_dev, cnt);
    ctx->launches++;
    MR_CUDA(ctx, cudaGetLastError());
    unsigned long long r = 0;
    MR_CUDA(ctx, cudaMemcpyAsync(&r, cnt, sizeof(r), cudaMemcpyDeviceToHost, ctx->stream));
    MR_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    *n_concave = (int64_t)r;
    return MR_OK;
}

extern "C" mr_status mr_eps_star(mr_ctx* ctx, mr_operator op, int32_t ic, int32_t jc, double a_r, double* alpha_host, double* eps_star)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_eps_star: mr_step_host_async calls are in flight (mr_host_sync first)");
    if (!eps_star) return fail(ctx, MR_ERR_INVALID_ARG, "mr_eps_star: null output");
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_eps_star: unknown operator");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_eps_star: B0 has not been set");
    const bool in_x = ctx->per[0] ? (ic >= 0 && ic < ctx->grid.nx) : (ic > 0 && ic < ctx->grid.nx - 1);
    const bool in_y = ctx->per[1] ? (jc >= 0 && jc < ctx->grid.ny) : (jc > 0 && jc < ctx->grid.ny - 1);
    if (!in_x || !in_y) return fail(ctx, MR_ERR_INVALID_ARG, "mr_eps_star: the line (ic, jc, .) must consist of inner nodes");
    return ctx->dtype == MR_F64 ? do_eps_star<double>(ctx, op, ic, jc, a_r, alpha_host, eps_star)
                                : do_eps_star<float>(ctx, op, ic, jc, a_r, alpha_host, eps_star);
}

extern "C" mr_status mr_sigma(mr_ctx* ctx, const void* x_ref_dev, const void* B_ref_dev, double* sigma_x, double* sigma_B)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!x_ref_dev || !B_ref_dev || !sigma_x || !sigma_B) return fail(ctx, MR_ERR_INVALID_ARG, "mr_sigma: null pointer");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_sigma: B0 has not been set");
    return ctx->dtype == MR_F64 ? do_sigma<double>(ctx, x_ref_dev, B_ref_dev, sigma_x, sigma_B)
                                : do_sigma<float>(ctx, x_ref_dev, B_ref_dev, sigma_x, sigma_B);
}

extern "C" mr_status mr_get_fields(mr_ctx* ctx, mr_operator op, void* x_dev, void* B_dev, void* J_dev)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_get_fields: unknown operator");
    if (!x_dev && !B_dev && !J_dev) return MR_OK;
    if ((B_dev || J_dev) && !ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_get_fields: B0 has not been set");
    return ctx->dtype == MR_F64 ? do_fields<double>(ctx, op, x_dev, B_dev, J_dev) : do_fields<float>(ctx, op, x_dev, B_dev, J_dev);
}

/* the host variant synchronises anyway, so it also reports a folded grid (the device variant is asynchronous and does not) */
extern "C" mr_status mr_get_fields_host(mr_ctx* ctx, mr_operator op, void* x_host, void* B_host, void* J_host)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_get_fields_host: mr_step_host_async calls are in flight (mr_host_sync first)");
    void* outs[3] = { x_host, B_host, J_host };
    MR_CUDA(ctx, cudaMemsetAsync(ctx->flag(), 0, sizeof(int), ctx->stream));
    for (int w = 0; w < 3; ++w) {
        if (!outs[w]) continue;
        mr_status s = mr_get_fields(ctx, op, w == 0 ? ctx->stage() : nullptr, w == 1 ? ctx->stage() : nullptr,
                                    w == 2 ? ctx->stage() : nullptr);
        if (s != MR_OK) return s;
        MR_CUDA(ctx, cudaMemcpyAsync(outs[w], ctx->stage(), ctx->dense_bytes(), cudaMemcpyDeviceToHost, ctx->stream));
    }
    int f = 0;
    mr_status st = read_flag(ctx, &f);
    if (st != MR_OK) return st;
    if (f & FLAG_NUMERIC) return fail(ctx, MR_ERR_NUMERIC, "mr_get_fields_host: det(dx/dX) <= 0 or a non-finite value was met");
    return MR_OK;
}

extern "C" size_t mr_stream_workspace_bytes(const mr_grid* grid, mr_dtype dtype)
{
    Layout L;
    return make_layout(grid, dtype, nullptr, &L) ? L.stage_bytes : 0;
}

extern "C" mr_status mr_bind_stream_workspace(mr_ctx* ctx, void* workspace_dev, size_t bytes)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!workspace_dev || (reinterpret_cast<uintptr_t>(workspace_dev) % kAlign) != 0)
        return fail(ctx, MR_ERR_WORKSPACE, "mr_bind_stream_workspace: workspace is null or not 256-byte aligned");
    if (bytes < ctx->L.stage_bytes)
        return fail(ctx, MR_ERR_WORKSPACE, "mr_bind_stream_workspace: smaller than mr_stream_workspace_bytes()");
    if (ctx->pipeline_open) return fail(ctx, MR_ERR_STATE, "mr_bind_stream_workspace: calls are in flight (mr_host_sync first)");
    ctx->sws = static_cast<char*>(workspace_dev);
    return MR_OK;
}

namespace {
template <typename T>
mr_status do_step_host_async(mr_ctx* c, const void* x_in, void* x_out, int64_t n, double dt, mr_operator op)
{
    if (!c->d2h_stream) {
        MR_CUDA(c, cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking));
        MR_CUDA(c, cudaEventCreateWithFlags(&c->ev_fields, cudaEventDisableTiming));
        MR_CUDA(c, cudaEventCreateWithFlags(&c->ev_d2h, cudaEventDisableTiming));
    }
    if (!c->pipeline_open) {             // the flag word collects the faults of every call until mr_host_sync reads it
        MR_CUDA(c, cudaMemsetAsync(c->flag(), 0, sizeof(int), c->stream));
        c->pipeline_open = true;
    }
    dim3 grid, block;
    node_launch_dims(c, grid, block);
    // host -> device into the staging field of the context, import into the spare state buffer, adopt it
    MR_CUDA(c, cudaMemcpyAsync(c->stage(), x_in, c->dense_bytes(), cudaMemcpyHostToDevice, c->stream));
    const int other = 1 - c->cur;
    k_import_x<T><<<grid, block, 0, c->stream>>>(static_cast<const T*>(c->stage()), static_cast<T*>(c->xi(other)), grid_params<T>(c),
                                                 domain_params(c), c->flag());
    c->launches++;
    wrap_ghosts<T>(c, c->xi(other));
    c->cur = other;
    c->time = 0.0;
    c->steps = 0;
    mr_status st = launch_steps<T>(c, n, dt * c->gamma, op);
    if (st != MR_OK) return st;
    c->time += dt * (double)n;
    c->steps += n;
    // the new positions, dense, into the second staging field once the previous call's copy has left it ...
    if (c->d2h_pending) MR_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_d2h, 0));
    k_fields<T, 0><<<grid, block, 0, c->stream>>>(static_cast<const T*>(c->xi(c->cur)), static_cast<const T*>(c->b()), grid_params<double>(c),
                                                  domain_params(c), reinterpret_cast<T*>(c->sws), nullptr, nullptr, c->flag());
    c->launches++;
    MR_CUDA(c, cudaGetLastError());
    MR_CUDA(c, cudaEventRecord(c->ev_fields, c->stream));
    // ... and device -> host on the library's stream, while the caller's stream goes on with the next call
    MR_CUDA(c, cudaStreamWaitEvent(c->d2h_stream, c->ev_fields, 0));
    MR_CUDA(c, cudaMemcpyAsync(x_out, c->sws, c->dense_bytes(), cudaMemcpyDeviceToHost, c->d2h_stream));
    MR_CUDA(c, cudaEventRecord(c->ev_d2h, c->d2h_stream));
    c->d2h_pending = true;
    return MR_OK;
}
}  // namespace

extern "C" mr_status mr_step_host_async(mr_ctx* ctx, const void* x_in_host, void* x_out_host, int64_t n, double dt, mr_operator op)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!x_in_host || !x_out_host) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step_host_async: null pointer");
    if (n < 0 || !(dt > 0.0) || !std::isfinite(dt)) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step_host_async: need n >= 0 and finite dt > 0");
    if (op != MR_OP_MIMETIC && op != MR_OP_DIRECT) return fail(ctx, MR_ERR_INVALID_ARG, "mr_step_host_async: unknown operator");
    if (!ctx->have_B0) return fail(ctx, MR_ERR_STATE, "mr_step_host_async: B0 has not been set");
    if (!ctx->sws) return fail(ctx, MR_ERR_STATE, "mr_step_host_async: no stream workspace bound (mr_bind_stream_workspace)");
    return ctx->dtype == MR_F64 ? do_step_host_async<double>(ctx, x_in_host, x_out_host, n, dt, op)
                                : do_step_host_async<float>(ctx, x_in_host, x_out_host, n, dt, op);
}

extern "C" mr_status mr_host_sync(mr_ctx* ctx)
{
    if (!ctx) return MR_ERR_INVALID_ARG;
    if (!ctx->pipeline_open) return MR_OK;
    int f = 0;
    mr_status st = read_flag(ctx, &f);                          // (synchronises the caller's stream)
    if (st != MR_OK) return st;
    if (ctx->d2h_stream) MR_CUDA(ctx, cudaStreamSynchronize(ctx->d2h_stream));
    ctx->pipeline_open = false;
    ctx->d2h_pending = false;
    if (f & FLAG_BOUNDARY) {
        ctx->failed = true;
        return fail(ctx, MR_ERR_INVALID_ARG, "mr_host_sync: a line-tied boundary node of some x_in was not on the reference grid X");
    }
    if (f & FLAG_NUMERIC) {
        ctx->failed = true;
        return fail(ctx, MR_ERR_NUMERIC, "mr_host_sync: det(dx/dX) <= 0 or a non-finite value was met");
    }
    ctx->failed = false;
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
    else if (!std::strcmp(name, "graph")) ctx->graphs_enabled = true;        // (the default) mr_step replays CUDA graphs on small grids
    else if (!std::strcmp(name, "nograph")) ctx->graphs_enabled = false;
    else return fail(ctx, MR_ERR_INVALID_ARG, "mr_set_variant: expected auto, generic, graph or nograph");
    return MR_OK;
}

// ------------------------------------------------------------------------------- mr_convexity_noalloc (include/mr.h)
// Convexity of a dense array of node positions for callers that have no way to hand the library device memory beyond their
// own input and output: the per-plane counters the kernel needs live in this file-scope array, which is part of the loaded
// module (MR_NOALLOC_MAX_PLANES * 8 bytes = 8 KiB on every GPU that loads libmr.so, until the process exits).
//
// In host code `g_noalloc_counts` is only a handle for the runtime, not a device address, so it is never passed to a kernel:
// noalloc_scratch() asks the runtime once per device (with that device current) where the array lives there and the launch
// gets that pointer.

static __device__ __align__(256) unsigned long long g_noalloc_counts[MR_NOALLOC_MAX_PLANES];

namespace {

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mutex;
unsigned long long* g_noalloc_ptr[kNoallocMaxDevices];      // device address of g_noalloc_counts per device ordinal, null = not asked yet

// the array's address on the current device (first use on a device: cudaGetSymbolAddress, which also loads the module there)
cudaError_t noalloc_scratch(unsigned long long** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kNoallocMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_noalloc_counts);
        if (e != cudaSuccess) return e;
        g_noalloc_ptr[dev] = static_cast<unsigned long long*>(p);
    }
    *out = g_noalloc_ptr[dev];
    return cudaSuccess;
}

// k_convexity (mr_next.cuh) on dense positions x[3][nz][ny][nx], every face an open end of the grid: kappa = +1 iff each
// trihedron of the node whose three neighbours exist has sgn det = di dj dk (Eqs. 3.10-3.11).  The nodes
// with kappa = -1 are counted per z-plane into plane_count[k] (zeroed by the caller): one atomic per block that found any.
template <typename T>
__global__ void __launch_bounds__(256)
k_convexity_dense(const T* __restrict__ x, int nx, int ny, int nz, int* __restrict__ kappa, unsigned long long* __restrict__ plane_count)
{
    const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y, k = blockIdx.z;
    const bool in = i < nx && j < ny;
    const long long N = (long long)nx * ny * nz, p = ((long long)k * ny + j) * nx + i;
    int kap = 1;
    if (in) {
        const int idx[3] = { i, j, k }, n[3] = { nx, ny, nz };
        const long long stride[3] = { 1, nx, (long long)nx * ny };
        double e[3][2][3];      // edge vectors to the six neighbours (doubles: their sign decides an integer)
        bool have[3][2];
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                have[a][s] = s == 0 ? idx[a] > 0 : idx[a] < n[a] - 1;
                const long long o = s == 0 ? -stride[a] : stride[a];
#pragma unroll
                for (int c = 0; c < 3; ++c) e[a][s][c] = have[a][s] ? (double)x[c * N + p + o] - (double)x[c * N + p] : 0.0;
            }
#pragma unroll
        for (int si = 0; si < 2; ++si)
#pragma unroll
            for (int sj = 0; sj < 2; ++sj)
#pragma unroll
                for (int sk = 0; sk < 2; ++sk) {
                    if (!(have[0][si] && have[1][sj] && have[2][sk])) continue;
                    const double* u = e[0][si];
                    const double* v = e[1][sj];
                    const double* w = e[2][sk];
                    const double d = u[0] * (v[1] * w[2] - v[2] * w[1]) - u[1] * (v[0] * w[2] - v[2] * w[0]) + u[2] * (v[0] * w[1] - v[1] * w[0]);
                    const int sgn = d > 0.0 ? 1 : (d < 0.0 ? -1 : 0);
                    const int prod = (si ? 1 : -1) * (sj ? 1 : -1) * (sk ? 1 : -1);
                    if (sgn != prod) kap = -1;
                }
        if (kappa) kappa[p] = kap;
    }
    __shared__ int sh[8];
    const unsigned concave = __ballot_sync(0xffffffffu, in && kap < 0);
    if (threadIdx.x == 0) sh[threadIdx.y] = __popc(concave);
    __syncthreads();
    if (threadIdx.x == 0 && threadIdx.y == 0) {
        int total = 0;
        for (int w = 0; w < 8; ++w) total += sh[w];
        if (total) atomicAdd(plane_count + k, (unsigned long long)total);
    }
}

}  // namespace

extern "C" mr_status mr_convexity_noalloc(const void* x_dev, const mr_grid* grid, mr_dtype dtype, int32_t* kappa_dev, int64_t* n_concave,
                                          void* stream)
{
    if (!x_dev || !grid || !n_concave) return fail(nullptr, MR_ERR_INVALID_ARG, "mr_convexity_noalloc: null argument");
    if (dtype != MR_F64 && dtype != MR_F32) return fail(nullptr, MR_ERR_INVALID_ARG, "mr_convexity_noalloc: dtype must be MR_F64 or MR_F32");
    if (grid->nx < 2 || grid->ny < 2 || grid->nz < 2 || grid->nx > 4096 || grid->ny > 4096)
        return fail(nullptr, MR_ERR_INVALID_ARG, "mr_convexity_noalloc: need 2 <= nx, ny <= 4096 and nz >= 2");
    if (grid->nz > MR_NOALLOC_MAX_PLANES)
        return fail(nullptr, MR_ERR_INVALID_ARG,
                    "mr_convexity_noalloc: nz = " + std::to_string(grid->nz) + " is more than the " + std::to_string(MR_NOALLOC_MAX_PLANES) +
                        " z-planes the library's static scratch has counters for (MR_NOALLOC_MAX_PLANES); use mr_convexity on a context instead");
    unsigned long long* counts = nullptr;
    MR_CUDA(nullptr, noalloc_scratch(&counts));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int nz = grid->nz;
    // the array still holds whatever the previous call (of any thread, on this device) counted
    MR_CUDA(nullptr, cudaMemsetAsync(counts, 0, sizeof(unsigned long long) * nz, s));
    const dim3 block(32, 8, 1), blocks((grid->nx + 31) / 32, (grid->ny + 7) / 8, nz);
    if (dtype == MR_F64) k_convexity_dense<double><<<blocks, block, 0, s>>>(static_cast<const double*>(x_dev), grid->nx, grid->ny, nz, kappa_dev, counts);
    else k_convexity_dense<float><<<blocks, block, 0, s>>>(static_cast<const float*>(x_dev), grid->nx, grid->ny, nz, kappa_dev, counts);
    MR_CUDA(nullptr, cudaGetLastError());
    unsigned long long host[MR_NOALLOC_MAX_PLANES];
    MR_CUDA(nullptr, cudaMemcpyAsync(host, counts, sizeof(unsigned long long) * nz, cudaMemcpyDeviceToHost, s));
    MR_CUDA(nullptr, cudaStreamSynchronize(s));
    unsigned long long total = 0;
    for (int k = 0; k < nz; ++k) total += host[k];
    *n_concave = (int64_t)total;
    return MR_OK;
}

// ------------------------------------------------------------------------------- mr_measure_fp64_peak (include/mr.h)
// The roof of the direct operator is plain FP64 arithmetic: a kernel of independent DFMA chains, no memory
// traffic, timed with CUDA events, gives the rate the FP64 pipes of this board deliver in the regime asked for.
static __device__ double g_fp64_sink;

namespace {
constexpr int kPeakChains = 8, kPeakIters = 4096;

__global__ void __launch_bounds__(256) k_fp64_chains(double seed)
{
    double a[kPeakChains];
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) a[c] = seed + (double)(threadIdx.x + c);
    const double m = 1.0 - 1e-9 * seed, b = 1e-9;
#pragma unroll 4
    for (int it = 0; it < kPeakIters; ++it)
#pragma unroll
        for (int c = 0; c < kPeakChains; ++c) a[c] = fma(a[c], m, b);
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < kPeakChains; ++c) s += a[c];
    if (s == -1.0) g_fp64_sink = s;          // never true: keeps the chains alive
}
}  // namespace

extern "C" mr_status mr_measure_fp64_peak(double seconds, void* stream, double* tflops)
{
    if (!tflops || !(seconds > 0.0) || !(seconds <= 60.0)) return fail(nullptr, MR_ERR_INVALID_ARG, "mr_measure_fp64_peak: need 0 < seconds <= 60 and an output");
    int dev = 0, sms = 0;
    MR_CUDA(nullptr, cudaGetDevice(&dev));
    MR_CUDA(nullptr, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int blocks = sms * 8, threads = 256;
    const double flop_per_launch = 2.0 * kPeakChains * kPeakIters * (double)blocks * threads;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    MR_CUDA(nullptr, cudaEventCreate(&e0));
    cudaError_t e = cudaEventCreate(&e1);
    float ms = 0.f;
    long long launches = 0;
    if (e == cudaSuccess) {
        // calibrate on three launches, then run as many as fill the time asked for between the two events
        for (int q = 0; q < 3; ++q) k_fp64_chains<<<blocks, threads, 0, s>>>(1.0);
        e = cudaEventRecord(e0, s);
        k_fp64_chains<<<blocks, threads, 0, s>>>(1.0);
        if (e == cudaSuccess) e = cudaEventRecord(e1, s);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess) {
            launches = (long long)(seconds * 1e3 / (ms > 1e-3f ? ms : 1e-3f)) + 1;
            e = cudaEventRecord(e0, s);
            for (long long q = 0; q < launches; ++q) k_fp64_chains<<<blocks, threads, 0, s>>>(1.0);
            if (e == cudaSuccess) e = cudaEventRecord(e1, s);
            if (e == cudaSuccess) e = cudaEventSynchronize(e1);
            if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
            if (e == cudaSuccess) e = cudaGetLastError();
        }
    }
    cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (e != cudaSuccess) return cuda_fail(nullptr, "mr_measure_fp64_peak", e);
    *tflops = flop_per_launch * (double)launches / ((double)ms * 1e-3) / 1e12;
    return MR_OK;
}
