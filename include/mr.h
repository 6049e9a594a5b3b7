/*
 * mr.h -- C-ABI boundary of the B200-native Lagrangian magneto-frictional relaxation step
 * (Candelaresi, Pontin & Hornig, arxiv 1405.0942; citations are PAPER.md line numbers).
 *
 * The library advances the Lagrangian map x(X,t) of a structured 3-D grid under u = gamma J x B (Eq. 1.5,
 * PAPER.md:40) with the frozen-in field B = (dx/dX) B(X,0) / det(dx/dX) (Eq. 2.1, :59), J = curl B by the
 * nearest-neighbour mimetic operator (Eqs. 2.2-2.7, :68-105) or by the direct-derivative ("classical") variant
 * (:49, :257), line-tied boundaries (:147), and the grid-wide diagnostics E_M (Eq. 3.13, :251) and
 * xi = max |J x B|/B^2 (Eq. 4.1, :264).  Every step of that path runs in hand-written sm_100a CUDA kernels;
 * there is no CPU fallback.
 *
 * Conventions
 *   - A vector field on the grid is a dense array T[3][nz][ny][nx] (component-major, i fastest:
 *     idx = (k*ny + j)*nx + i), T = double (MR_F64) or float (MR_F32).
 *   - Reference grid X_ijk = lo + idx*h, h_a = (hi_a - lo_a)/(n_a - 1); nodes include the boundary (:170).
 *   - "_dev" pointers are CUDA device pointers on the context's device; "_host" pointers are host pointers
 *     (pinned memory makes the copies asynchronous and fast, pageable memory also works).
 *   - Ownership: the CALLER owns every device and host buffer and the stream.  The library never allocates
 *     device memory: mr_create binds a caller-provided workspace of at least mr_workspace_bytes_bc() bytes
 *     (256-byte aligned) that must outlive the context.  mr_ctx itself is host memory owned by the library, and so are
 *     the CUDA graphs it replays (mr_set_variant), the stream it records them on (they RUN on the caller's stream) and
 *     32 bytes of pinned host memory through which mr_step_adaptive exchanges dt, Lambda and the error flag.
 *   - All work is enqueued on the caller's stream.  mr_set_B0, mr_get_fields, mr_get_xi and mr_rhs are asynchronous
 *     (the buffers may be reused once the stream has passed the call); every other call synchronises that stream
 *     before it returns (mr_set_x / mr_set_xi for the check of the line-tied faces, mr_step* for the error flag, the
 *     diagnostics for their scalars, the *_host calls for the copies).
 *   - Errors are return codes; nothing throws or aborts.  mr_last_error(ctx) gives a message for the last
 *     failing call on that context.  After MR_ERR_NUMERIC the context stays failed until mr_set_x succeeds.
 */
#ifndef MR_H_
#define MR_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mr_ctx mr_ctx; /* opaque */

typedef enum {
    MR_OK = 0,
    MR_ERR_INVALID_ARG = 1, /* null pointer, bad size, unsupported option */
    MR_ERR_WORKSPACE = 2,   /* workspace null, misaligned or too small */
    MR_ERR_CUDA = 3,        /* a CUDA runtime/driver call failed (no device, launch failure, ...) */
    MR_ERR_STATE = 4,       /* B0 has not been set, a workspace is not bound, or mr_step_host_async calls are in flight */
    MR_ERR_NUMERIC = 5      /* det(dx/dX) <= 0 or a non-finite value was met (grid folded, cf. :333) */
} mr_status;

typedef enum {
    MR_OP_MIMETIC = 0, /* Eqs. 2.3-2.7 (:68-105): three Stokes loops through the 4 nearest neighbours */
    MR_OP_DIRECT = 1   /* analytic derivative of Eq. 2.1: products of 1st and 2nd differences of x (:49) */
} mr_operator;

typedef enum {
    MR_BC_LINE_TIED = 0, /* u = 0 and B.n fixed on the face (:147) */
    MR_BC_PERIODIC = 1   /* Eqs. 2.12-2.14 (:147-164): every node of the axis is an inner point, nodes at lo + idx*h,
                            period n*h = (hi - lo) + h; the ghost nodes are x(-1) = x(n-1) - n*h e_a, x(n) = x(0) + n*h e_a
                            and B(X,0) must be periodic.  The ghost nodes live in the padded arrays of the workspace (two
                            planes / rows, 16 bytes of columns either side of a periodic axis), refreshed after every pass. */
} mr_bc;

typedef enum { MR_F64 = 0, MR_F32 = 1 } mr_dtype;

typedef struct { int32_t nx, ny, nz; } mr_grid;      /* nodes per logical axis, each 5 <= n <= 4096 */
typedef struct { double lo[3], hi[3]; } mr_domain;   /* hi > lo componentwise */

/* "boundary" + options of mr_create */
typedef struct {
    mr_bc bc[3];            /* per logical axis (both faces) */
    double gamma;           /* > 0; Eq. 1.5, the paper uses 1 (:55) */
    mr_dtype dtype;         /* storage and arithmetic type of the state; reductions always accumulate in fp64 */
    void* workspace;        /* device pointer, >= mr_workspace_bytes_bc(grid, dtype, bc), 256-byte aligned, caller-owned */
    size_t workspace_bytes;
    void* stream;           /* cudaStream_t (0 = legacy default stream), caller-owned */
} mr_boundary;

typedef struct {
    double time;     /* sum of dt over all steps taken since the last mr_set_x / mr_create */
    int64_t steps;   /* number of steps taken since then */
    double energy;   /* E_M = 1/2 sum zeta |B|^2 Delta dXdYdZ over all nodes, zeta = 1/2 per face (Eq. 3.13) */
    double max_jxb;  /* max over interior nodes of |J x B| */
    double xi;       /* max over interior nodes of |J x B| / |B|^2 (Eq. 4.1) */
    double min_det;  /* min over all nodes of Delta = det(dx/dX) */
} mr_diag;

/* Bytes of device workspace mr_create needs for this grid and dtype (0 if the arguments are invalid).
 * Holds the double-buffered state, the pre-scaled B(X,0), a staging buffer for the *_host calls and the
 * reduction partials; about 4 fields = 12*nx*ny*nz elements.  Pure host arithmetic, needs no GPU.
 * mr_workspace_bytes: all six faces line-tied.  mr_workspace_bytes_bc: bc[3] = the mr_bc of the x, y, z axes; a periodic
 * axis adds its ghost layers (two planes / rows, 16 bytes of columns either side) to every field. */
size_t mr_workspace_bytes(const mr_grid* grid, mr_dtype dtype);
size_t mr_workspace_bytes_bc(const mr_grid* grid, mr_dtype dtype, const int32_t* bc);

/* Create a context on the current CUDA device; the state is initialised to x = X, so a run that starts on
 * the reference grid needs no mr_set_x.
 * Returns MR_ERR_INVALID_ARG for bad sizes/options (checked before any CUDA call), MR_ERR_WORKSPACE,
 * MR_ERR_CUDA (e.g. no sm_100 device).  On failure *out is NULL. */
mr_status mr_create(const mr_grid* grid, const mr_domain* domain, const mr_boundary* boundary, mr_ctx** out);

/* Free the host-side context (the workspace stays with the caller).  NULL is allowed. */
mr_status mr_destroy(mr_ctx* ctx);

/* Set the initial field B(X,0) at the nodes (Eq. 2.1): dense T[3][nz][ny][nx] in the context dtype; copied
 * (and pre-scaled) into the workspace, the source may be reused once the stream has passed this call. */
mr_status mr_set_B0(mr_ctx* ctx, const void* B0_dev);
mr_status mr_set_B0_host(mr_ctx* ctx, const void* B0_host);

/* Set the node positions x (dense, context dtype), e.g. a displaced initial grid or a checkpoint; resets
 * time/steps and clears a numeric failure.  Line-tied boundary nodes must equal X (|x - X| <= 1e-6*h, plus 2.4e-7*|X| of input rounding when the context is fp32),
 * otherwise MR_ERR_INVALID_ARG is returned and the state is unchanged.  (Synchronises for that check.) */
mr_status mr_set_x(mr_ctx* ctx, const void* x_dev);
mr_status mr_set_x_host(mr_ctx* ctx, const void* x_host);

/* The same through the DISPLACEMENT xi = x - X (dense, context dtype): on an fp32 context positions lose eps*|X| per
 * node at the ABI, 300 times the rounding of xi itself (reading Q15), so fp32 callers exchange xi.  Nodes on
 * line-tied faces must have |xi| <= 1e-6*h.  mr_get_xi is asynchronous. */
mr_status mr_set_xi(mr_ctx* ctx, const void* xi_dev);
mr_status mr_get_xi(mr_ctx* ctx, void* xi_dev);

/* Take n >= 0 explicit steps x <- x + dt * gamma * J x B on interior nodes, boundary nodes fixed (Eq. 1.2,
 * :17; :147), all velocities from the old x.  dt > 0.  Synchronises the stream at the end and returns
 * MR_ERR_NUMERIC if any node had det <= 0 or a non-finite value during these steps, MR_ERR_STATE without B0. */
mr_status mr_step(mr_ctx* ctx, int64_t n, double dt, mr_operator op);

/* Grid-wide reduction of the CURRENT state (no update): fills *out.  Deterministic (fixed-order two-stage
 * reduction).  Synchronises the stream. */
mr_status mr_diagnostics(mr_ctx* ctx, mr_operator op, mr_diag* out);

/* Materialise fields of the current state into caller buffers (dense, context dtype); any pointer may be
 * NULL.  x = node positions; B = pushed-forward field on ALL nodes; J = current on interior nodes by `op`,
 * 0 on boundary nodes. */
mr_status mr_get_fields(mr_ctx* ctx, mr_operator op, void* x_dev, void* B_dev, void* J_dev);
mr_status mr_get_fields_host(mr_ctx* ctx, mr_operator op, void* x_host, void* B_host, void* J_host);

/* ---- streaming through host buffers: one step of the whole path per call, positions in, positions out ------------------
 * mr_step_host_async = mr_set_x_host(x_in_host) + mr_step(n, dt, op) + mr_get_fields_host(x = x_out_host), but ASYNCHRONOUS:
 * it returns once the work is enqueued.  The device->host copy of a call runs on a stream of the library's own and overlaps
 * the host->device copy of the next call (PCIe is full duplex), so a sequence of calls moves 2 x 24 nx ny nz bytes per call at
 * the rate of ONE direction.  Needs a second dense staging field, bound once (caller-owned device memory, 256-byte aligned,
 * mr_stream_workspace_bytes = 3 nx ny nz elements).  x_in_host / x_out_host: [3][nz][ny][nx] in the context dtype, pinned host
 * memory (pageable memory works but serialises the copies); both must stay valid and x_out_host unread until mr_host_sync.
 * mr_host_sync waits for everything enqueued and reports what mr_set_x / mr_step would have: MR_ERR_INVALID_ARG if some
 * x_in had a line-tied boundary node off the reference grid, MR_ERR_NUMERIC if some state folded (the context is then failed).
 * Between the first mr_step_host_async and mr_host_sync the error word of the context belongs to the calls in flight: the
 * calls that use it themselves (mr_set_x, mr_set_x_host, mr_set_xi, mr_step, mr_step_monitored, mr_step_adaptive,
 * mr_diagnostics, mr_eps_star, mr_get_fields_host) return MR_ERR_STATE until mr_host_sync has been called. */
size_t mr_stream_workspace_bytes(const mr_grid* grid, mr_dtype dtype);
mr_status mr_bind_stream_workspace(mr_ctx* ctx, void* workspace_dev, size_t bytes);
mr_status mr_step_host_async(mr_ctx* ctx, const void* x_in_host, void* x_out_host, int64_t n, double dt, mr_operator op);
mr_status mr_host_sync(mr_ctx* ctx);

/* mr_step that also watches the run (the time series of Fig. 4.1, :245-264): n steps, and for every `every`-th of them (the
 * first included; every = 0: none) the diagnostics of the state that step STARTS from, appended to history_host[0 .. capacity)
 * (host memory; *written = how many).  With the mimetic operator the step kernel reduces S6 in the same pass (the diagnosis
 * costs no memory traffic); a record equals what mr_diagnostics would return at that point, bit for bit.
 * Synchronises like mr_step. */
mr_status mr_step_monitored(mr_ctx* ctx, int64_t n, double dt, mr_operator op, int64_t every, mr_diag* history_host,
                            int64_t capacity, int64_t* written);

/* The velocity u = gamma J x B (Eq. 1.5, :40) of the current state, dense, context dtype, 0 on line-tied boundary
 * nodes: the right-hand side of dx/dt = u that mr_step and mr_step_adaptive integrate.  Asynchronous. */
mr_status mr_rhs(mr_ctx* ctx, mr_operator op, void* u_dev);

/* ---- section 2.4 (:131-143): adaptive Cash-Karp RK5(4) with the step control of Eq. 2.11 -------------------------
 * Needs a second caller-owned device buffer for the six stage velocities and the stage state (7 fields), bound once. */
size_t mr_adaptive_workspace_bytes(const mr_grid* grid, mr_dtype dtype);                 /* all faces line-tied */
size_t mr_adaptive_workspace_bytes_bc(const mr_grid* grid, mr_dtype dtype, const int32_t* bc);
mr_status mr_bind_adaptive_workspace(mr_ctx* ctx, void* workspace_dev, size_t bytes);

typedef struct {
    int64_t accepted, rejected; /* trial steps of this call */
    int64_t rhs_evals;          /* 6 per trial */
    double time;                /* reached (== t_end unless max_trials ran out or the run failed) */
    double dt_next;             /* step length handed on (also written to *dt) */
    double last_lambda;         /* Lambda = max |x5 - x4| of the last trial */
} mr_adapt_stats;

/* Integrate from the context's time to t_end.  Each trial step evaluates u six times (the RHS instantiation of the
 * step kernels), forms the fifth-order solution and Lambda = max over nodes and components of |x5 - x4| on the device
 * and brings ONE scalar back; the host rejects the trial if Lambda > lambda0 and retries with dt' = dt |lambda0/Lambda|^0.2
 * (Eq. 2.11), accepts it otherwise and enlarges dt by the same formula if Lambda < lambda0/2 (growth capped at 5x).
 * The last step is clipped to end at t_end.  *dt: first trial step in, step handed on out.  trace_host (may be NULL):
 * trace_cap rows {t, dt tried, Lambda, accepted} of the trials.  A trial in which a stage met det <= 0 or a non-finite value
 * has no result: it counts as rejected (Lambda = NaN in the trace) and is retried with dt/2 (reading Q26; the
 * paper reports "a drop of the time step by several orders of magnitude, at which point the simulation is stopped", :333).
 * Returns MR_ERR_STATE without B0 or without the adaptive workspace; MR_ERR_NUMERIC after 40 such trials in a row (2^-40
 * of the step first tried), or if the step length underflows: the state is then the last accepted one, *dt the collapsed
 * step; MR_ERR_INVALID_ARG if max_trials ran out before t_end. */
mr_status mr_step_adaptive(mr_ctx* ctx, double t_end, double lambda0, double* dt, mr_operator op, int64_t max_trials,
                           mr_adapt_stats* stats, double* trace_host, int64_t trace_cap);

/* ---- section 3.2 diagnostics beyond E_M and xi ------------------------------------------------------------------
 * Convexity (Eqs. 3.10-3.11, :231-243): kappa = +1 where every trihedron of the node (three nearest neighbours, one per
 * axis, all that exist) has sgn det = di dj dk, else -1, into kappa_dev (dense int32[nz][ny][nx], may be NULL); the
 * number of nodes with kappa = -1 into *n_concave (the early warning of :333). */
mr_status mr_convexity(mr_ctx* ctx, int32_t* kappa_dev, int64_t* n_concave);

/* alpha* = J.B/B^2 (Eq. 3.5, :206) at the inner nodes of the grid line (ic, jc, .) -- s_alpha of Eq. 3.6 when the line
 * is the z axis -- into alpha_host[nz] (may be NULL; 0 at line-tied end nodes), and
 * eps* = max over pairs of a_r (alpha*_i - alpha*_j)/|X_i - X_j| (Eq. 3.7, :214) into *eps_star. */
mr_status mr_eps_star(mr_ctx* ctx, mr_operator op, int32_t ic, int32_t jc, double a_r, double* alpha_host, double* eps_star);

/* sigma_x and sigma_B (Eqs. 3.9, 3.8, :221-229): root mean square over ALL nodes of |x - x_ref| and |B - B_ref|;
 * the references are dense device arrays in the context dtype (for the IsoHelix field Eqs. 3.3 and 3.2). */
mr_status mr_sigma(mr_ctx* ctx, const void* x_ref_dev, const void* B_ref_dev, double* sigma_x, double* sigma_B);

/* ---- the one entry point that needs no device memory beyond its input and output ------------------------------------
 * Everything above works in a workspace the caller allocates.  Some callers cannot allocate at all: a plug-in that runs
 * inside a host application whose own memory manager has taken the whole card (a raw cudaMalloc there fails, or fights the
 * pool), a monitoring hook in a time-critical loop (cudaMalloc and cudaFree stall every stream of the device while they
 * run), or code that is simply handed two pointers and a stream and nothing else.  For them: the convexity check of
 * Eqs. 3.10-3.11 (:231-243, the early warning of :333) on a dense array of node POSITIONS, without a context.  The call
 * issues no cudaMalloc, cudaFree, or library routine that allocates; its only scratch memory is a fixed array of
 * MR_NOALLOC_MAX_PLANES 64-bit counters (8 KiB) built into libmr.so, which every GPU that loads the library carries until
 * the process ends.
 *
 *   x_dev      in   T[3][nz][ny][nx] positions (dense, i fastest), T by `dtype`; device memory of the current device
 *   grid       in   2 <= nx, ny <= 4096, 2 <= nz <= MR_NOALLOC_MAX_PLANES.  A grid with more z-planes than the scratch has
 *                   counters for is refused with MR_ERR_INVALID_ARG before anything is launched (mr_last_error(NULL) says so);
 *                   such a grid needs mr_convexity on a context.
 *   kappa_dev  out  int32[nz][ny][nx], +1 / -1 per node as mr_convexity writes it; may be NULL
 *   n_concave  out  host: how many nodes have kappa = -1
 *   stream          cudaStream_t of the caller (0 = legacy default stream); the call waits for it before it returns
 *
 * All six faces are treated as ends of the grid (a node there has only the trihedra whose neighbours exist), which is what
 * mr_convexity does on a context without periodic axes; the two then agree node for node -- up to trihedra whose determinant
 * is within rounding of zero, because this call differences the positions while a context differences the displacements it
 * stores (in fp64 a 1e-14 effect).
 *
 * Set-up: the FIRST call on each device looks up where the built-in array lives on that device (and thereby loads the
 * library's kernels there); make that first call outside any stream capture.  Later calls on the device reuse the address.
 * Sharing: there is ONE array per device, used by every call from every thread, and it keeps what the last call counted.
 * Each call zeroes the counters it is going to use (on `stream`) before its kernel runs, so calls that follow one another
 * on the GPU are independent; two calls that can overlap on the GPU (different streams, or different threads without
 * ordering between their streams) race on the counters and return garbage counts -- serialise them.
 * Errors go to mr_last_error(NULL), like those of mr_create. */
#define MR_NOALLOC_MAX_PLANES 1024
mr_status mr_convexity_noalloc(const void* x_dev, const mr_grid* grid, mr_dtype dtype, int32_t* kappa_dev, int64_t* n_concave,
                               void* stream);

/* Message for the last error on this context ("" if none); ctx == NULL gives the last mr_create failure.
 * The pointer stays valid until the next failing call on the same context (or mr_destroy). */
const char* mr_last_error(const mr_ctx* ctx);

/* Introspection for benchmarks and tests: number of kernel launches issued by this context so far, and the
 * name of the step-kernel variant the last mr_step used ("" before the first step). */
int64_t mr_launch_count(const mr_ctx* ctx);
const char* mr_step_variant(const mr_ctx* ctx);

/* Measurement aid for the roofline of the direct operator, which is bound by plain FP64 arithmetic (bench.py --operator
 * direct): runs a kernel of independent DFMA chains (8 per thread, no memory traffic; 8 CTAs of 256 threads per SM) back to
 * back on `stream` for about `seconds` (0 < seconds <= 60), times it with CUDA events and writes the rate in TFLOP/s (2 FLOP
 * per DFMA) to *tflops: a short run gives the burst figure at full clocks, a run of seconds the one under the board's power
 * cap.  Needs no context; allocates no device memory; waits for the stream.  Errors go to mr_last_error(NULL). */
mr_status mr_measure_fp64_peak(double seconds, void* stream, double* tflops);

/* Choose the step kernel.  "auto" (default): the streaming TMA kernels (mimetic: csrc/mr_sym.cuh, direct:
 * csrc/mr_direct.cuh).  "generic": the global-memory kernels of csrc/mr_generic.cuh for both operators (one thread per
 * node, every stencil value straight from global memory): the A/B reference of the tests.  Both agree to rounding.
 * "graph" (default) / "nograph": whether mr_step, on a grid whose fields fit the L2 (launch-latency bound), replays its
 * launches sixteen steps at a time as a CUDA graph; the kernels and the results are the same either way. */
mr_status mr_set_variant(mr_ctx* ctx, const char* name);

#ifdef __cplusplus
}
#endif
#endif /* MR_H_ */
