"""Thin ctypes binding of the C-ABI library ``libmr.so`` (include/mr.h): argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels.  PyTorch supplies device memory (the
workspace and the field tensors) and the CUDA stream; nothing here computes.  Importing this module fails loudly
if ``libmr.so`` has not been built (``python -m paper_1405_0942_b200.build``); there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmr.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "paper_1405_0942_b200: %s is missing -- build it with `python -m paper_1405_0942_b200.build` "
        "(nvcc, sm_100a).  There is no CPU fallback for the relaxation step." % LIB_PATH)

lib = C.CDLL(LIB_PATH)

# ---- enums (include/mr.h) ---------------------------------------------------------------------------------
MR_OK, MR_ERR_INVALID_ARG, MR_ERR_WORKSPACE, MR_ERR_CUDA, MR_ERR_STATE, MR_ERR_NUMERIC = range(6)
MR_OP_MIMETIC, MR_OP_DIRECT = 0, 1
MR_BC_LINE_TIED, MR_BC_PERIODIC = 0, 1
MR_F64, MR_F32 = 0, 1

STATUS_NAMES = {0: "MR_OK", 1: "MR_ERR_INVALID_ARG", 2: "MR_ERR_WORKSPACE", 3: "MR_ERR_CUDA", 4: "MR_ERR_STATE",
                5: "MR_ERR_NUMERIC"}
OPERATORS = {"mimetic": MR_OP_MIMETIC, "direct": MR_OP_DIRECT}
BOUNDARIES = {"line_tied": MR_BC_LINE_TIED, "periodic": MR_BC_PERIODIC}


class mr_grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32)]


class mr_domain(C.Structure):
    _fields_ = [("lo", C.c_double * 3), ("hi", C.c_double * 3)]


class mr_boundary(C.Structure):
    _fields_ = [("bc", C.c_int * 3), ("gamma", C.c_double), ("dtype", C.c_int), ("workspace", C.c_void_p),
                ("workspace_bytes", C.c_size_t), ("stream", C.c_void_p)]


class mr_adapt_stats(C.Structure):
    _fields_ = [("accepted", C.c_int64), ("rejected", C.c_int64), ("rhs_evals", C.c_int64), ("time", C.c_double),
                ("dt_next", C.c_double), ("last_lambda", C.c_double)]


class mr_diag(C.Structure):
    _fields_ = [("time", C.c_double), ("steps", C.c_int64), ("energy", C.c_double), ("max_jxb", C.c_double),
                ("xi", C.c_double), ("min_det", C.c_double)]


_ctx_p = C.c_void_p
lib.mr_workspace_bytes.argtypes = [C.POINTER(mr_grid), C.c_int]
lib.mr_workspace_bytes.restype = C.c_size_t
lib.mr_create.argtypes = [C.POINTER(mr_grid), C.POINTER(mr_domain), C.POINTER(mr_boundary), C.POINTER(_ctx_p)]
lib.mr_create.restype = C.c_int
lib.mr_destroy.argtypes = [_ctx_p]
lib.mr_destroy.restype = C.c_int
lib.mr_adaptive_workspace_bytes.argtypes = [C.POINTER(mr_grid), C.c_int]
lib.mr_adaptive_workspace_bytes.restype = C.c_size_t
lib.mr_workspace_bytes_bc.argtypes = [C.POINTER(mr_grid), C.c_int, C.POINTER(C.c_int32)]
lib.mr_workspace_bytes_bc.restype = C.c_size_t
lib.mr_adaptive_workspace_bytes_bc.argtypes = [C.POINTER(mr_grid), C.c_int, C.POINTER(C.c_int32)]
lib.mr_adaptive_workspace_bytes_bc.restype = C.c_size_t
lib.mr_bind_adaptive_workspace.argtypes = [_ctx_p, C.c_void_p, C.c_size_t]
lib.mr_bind_adaptive_workspace.restype = C.c_int
lib.mr_step_adaptive.argtypes = [_ctx_p, C.c_double, C.c_double, C.POINTER(C.c_double), C.c_int, C.c_int64, C.POINTER(mr_adapt_stats),
                                 C.c_void_p, C.c_int64]
lib.mr_step_adaptive.restype = C.c_int
lib.mr_rhs.argtypes = [_ctx_p, C.c_int, C.c_void_p]
lib.mr_rhs.restype = C.c_int
lib.mr_convexity.argtypes = [_ctx_p, C.c_void_p, C.POINTER(C.c_int64)]
lib.mr_convexity.restype = C.c_int
lib.mr_eps_star.argtypes = [_ctx_p, C.c_int, C.c_int32, C.c_int32, C.c_double, C.c_void_p, C.POINTER(C.c_double)]
lib.mr_eps_star.restype = C.c_int
lib.mr_sigma.argtypes = [_ctx_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
lib.mr_sigma.restype = C.c_int
for _n in ("mr_set_B0", "mr_set_B0_host", "mr_set_x", "mr_set_x_host", "mr_set_xi", "mr_get_xi"):
    getattr(lib, _n).argtypes = [_ctx_p, C.c_void_p]
    getattr(lib, _n).restype = C.c_int
lib.mr_step.argtypes = [_ctx_p, C.c_int64, C.c_double, C.c_int]
lib.mr_step.restype = C.c_int
lib.mr_diagnostics.argtypes = [_ctx_p, C.c_int, C.POINTER(mr_diag)]
lib.mr_diagnostics.restype = C.c_int
for _n in ("mr_get_fields", "mr_get_fields_host"):
    getattr(lib, _n).argtypes = [_ctx_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
    getattr(lib, _n).restype = C.c_int
lib.mr_last_error.argtypes = [_ctx_p]
lib.mr_last_error.restype = C.c_char_p
lib.mr_launch_count.argtypes = [_ctx_p]
lib.mr_launch_count.restype = C.c_int64
lib.mr_step_variant.argtypes = [_ctx_p]
lib.mr_step_variant.restype = C.c_char_p
lib.mr_set_variant.argtypes = [_ctx_p, C.c_char_p]
lib.mr_step_monitored.argtypes = [_ctx_p, C.c_int64, C.c_double, C.c_int, C.c_int64, C.POINTER(mr_diag), C.c_int64, C.POINTER(C.c_int64)]
lib.mr_stream_workspace_bytes.argtypes = [C.POINTER(mr_grid), C.c_int]
lib.mr_stream_workspace_bytes.restype = C.c_size_t
lib.mr_bind_stream_workspace.argtypes = [_ctx_p, C.c_void_p, C.c_size_t]
lib.mr_step_host_async.argtypes = [_ctx_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_int]
lib.mr_host_sync.argtypes = [_ctx_p]
lib.mr_set_variant.restype = C.c_int
lib.mr_convexity_noalloc.argtypes = [C.c_void_p, C.POINTER(mr_grid), C.c_int, C.c_void_p, C.POINTER(C.c_int64), C.c_void_p]
lib.mr_convexity_noalloc.restype = C.c_int
NOALLOC_MAX_PLANES = 1024      # MR_NOALLOC_MAX_PLANES of include/mr.h
lib.mr_measure_fp64_peak.argtypes = [C.c_double, C.c_void_p, C.POINTER(C.c_double)]
lib.mr_measure_fp64_peak.restype = C.c_int


class MrError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, status), message))
        self.status = status


class NumericError(MrError):
    """MR_ERR_NUMERIC: det(dx/dX) <= 0 or a non-finite value (the grid folded)."""


def _raise(status, ctx):
    msg = (lib.mr_last_error(ctx) or b"").decode()
    raise (NumericError if status == MR_ERR_NUMERIC else MrError)(status, msg)


def workspace_bytes(n, dtype="f64", bc=("line_tied",) * 3) -> int:
    g = mr_grid(*[int(v) for v in n])
    bcs = (C.c_int32 * 3)(*[BOUNDARIES[b] for b in bc])
    return int(lib.mr_workspace_bytes_bc(C.byref(g), MR_F64 if dtype == "f64" else MR_F32, bcs))


def _op(op):
    return OPERATORS[op] if isinstance(op, str) else int(op)


def measure_fp64_peak(seconds, device=None):
    """mr_measure_fp64_peak: TFLOP/s of a DFMA-chain kernel run for about ``seconds`` on the current stream of ``device``."""
    import torch

    out = C.c_double()
    with torch.cuda.device(device):
        st = lib.mr_measure_fp64_peak(float(seconds), torch.cuda.current_stream().cuda_stream, C.byref(out))
    if st != MR_OK:
        _raise(st, None)
    return out.value


def convexity_noalloc(x, kappa=None):
    """mr_convexity_noalloc: how many nodes of the position field ``x`` are concave (Eq. 3.11), with no context and no
    workspace.  It is the call for code that may not allocate on the GPU (a plug-in inside an application that owns all
    device memory, a check inside a loop that cannot afford the device-wide stall of cudaMalloc): the library allocates
    nothing, and neither does this wrapper -- the only scratch is a small array built into ``libmr.so``.

    ``x``: contiguous CUDA tensor (3, nz, ny, nx), float64 or float32, with nz <= ``NOALLOC_MAX_PLANES`` (more planes raise
    ``MrError``; use ``Relaxation.convexity``).  ``kappa``: optional int32 CUDA tensor (nz, ny, nx) OF THE CALLER'S that
    receives +1 / -1 per node.  Runs on the current stream of ``x``'s device and waits for it.  All calls on a device share
    that one scratch array: do not issue calls that can overlap on the GPU (other streams, other threads)."""
    import torch

    if x.device.type != "cuda" or x.dtype not in (torch.float64, torch.float32) or x.dim() != 4 or x.shape[0] != 3 or not x.is_contiguous():
        raise MrError(MR_ERR_INVALID_ARG, "x must be a contiguous float64/float32 CUDA tensor of shape (3, nz, ny, nx)")
    nz, ny, nx = (int(v) for v in x.shape[1:])
    if kappa is not None and (kappa.device != x.device or kappa.dtype != torch.int32 or tuple(kappa.shape) != (nz, ny, nx)
                              or not kappa.is_contiguous()):
        raise MrError(MR_ERR_INVALID_ARG, "kappa must be a contiguous int32 tensor of shape (nz, ny, nx) on x's device")
    n = C.c_int64()
    with torch.cuda.device(x.device):
        st = lib.mr_convexity_noalloc(x.data_ptr(), C.byref(mr_grid(nx, ny, nz)), MR_F64 if x.dtype == torch.float64 else MR_F32,
                                      kappa.data_ptr() if kappa is not None else None, C.byref(n),
                                      torch.cuda.current_stream(x.device).cuda_stream)
    if st != MR_OK:
        _raise(st, None)
    return int(n.value)


class Relaxation:
    """mr_create / mr_set_B0 / mr_set_x / mr_step / mr_diagnostics / mr_get_fields on one CUDA device.

    ``n=(nx,ny,nz)``, ``lo``/``hi`` the domain corners; ``dtype`` "f64" or "f32"; fields are torch CUDA tensors
    (or pinned/pageable host tensors for the ``*_host`` calls) of shape ``(3, nz, ny, nx)`` in that dtype.
    """

    def __init__(self, n, lo, hi, dtype="f64", gamma=1.0, bc=("line_tied",) * 3, device="cuda", stream=None, workspace=None,
                 adaptive_workspace=None):
        """``workspace`` / ``adaptive_workspace``: uint8 CUDA tensors of the caller's own (256-byte aligned, at least
        ``workspace_bytes(...)`` / ``mr_adaptive_workspace_bytes_bc`` bytes); allocated here when not given."""
        import torch

        for b in bc:
            if b not in BOUNDARIES:
                raise MrError(MR_ERR_INVALID_ARG, "unknown boundary type %r (expected one of %s)" % (b, sorted(BOUNDARIES)))
        self._torch = torch
        self.n = tuple(int(v) for v in n)
        self.shape = (3, self.n[2], self.n[1], self.n[0])
        self.dtype = dtype
        self.tdtype = torch.float64 if dtype == "f64" else torch.float32
        self.device = torch.device(device)
        if self.device.type != "cuda":
            raise MrError(MR_ERR_INVALID_ARG, "the relaxation step runs on a CUDA device only")
        if self.device.index is None:
            self.device = torch.device("cuda", torch.cuda.current_device())
        self._ctx = _ctx_p()
        self.bc = tuple(bc)
        nbytes = workspace_bytes(self.n, dtype, self.bc)
        if nbytes == 0:
            raise MrError(MR_ERR_INVALID_ARG, "invalid grid %r / dtype %r" % (self.n, dtype))
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            if workspace is not None:
                self.workspace = workspace
                nbytes = int(workspace.numel())
            else:
                with torch.cuda.stream(self.stream):        # the workspace belongs to the stream the library works on
                    self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            self._aworkspace = None
            self._aworkspace_given = adaptive_workspace
            g = mr_grid(*self.n)
            d = mr_domain((C.c_double * 3)(*[float(v) for v in lo]), (C.c_double * 3)(*[float(v) for v in hi]))
            bcs = (C.c_int * 3)(*[BOUNDARIES[b] for b in bc])
            b = mr_boundary(bcs, float(gamma), MR_F64 if dtype == "f64" else MR_F32, self.workspace.data_ptr(),
                            nbytes, self.stream.cuda_stream)
            st = lib.mr_create(C.byref(g), C.byref(d), C.byref(b), C.byref(self._ctx))
        if st != MR_OK:
            self._ctx = _ctx_p()
            _raise(st, None)

    # -- helpers ----------------------------------------------------------------------------------------
    def _check(self, st):
        if st != MR_OK:
            _raise(st, self._ctx)

    def _dev(self, t, name):
        if t is None:
            return None
        if t.device != self.device or t.dtype != self.tdtype or tuple(t.shape) != self.shape or not t.is_contiguous():
            raise MrError(MR_ERR_INVALID_ARG, "%s must be a contiguous %s tensor of shape %r on %s"
                          % (name, self.tdtype, self.shape, self.device))
        self._order(t)
        return t.data_ptr()

    def _order(self, t):
        """The library enqueues on its own stream: if the caller's current stream is another one, make ours wait for the
        work already queued there (the tensor's producer) and tell the allocator that ours uses the tensor."""
        cur = self._torch.cuda.current_stream(self.device)
        if cur != self.stream:
            self.stream.wait_stream(cur)
            t.record_stream(self.stream)

    def _publish(self):
        """The other direction of _order, after an asynchronous call that writes (or still reads) a caller tensor on the library's
        stream: the caller's current stream waits for it, so the caller may use the tensor there without synchronising."""
        cur = self._torch.cuda.current_stream(self.device)
        if cur != self.stream:
            cur.wait_stream(self.stream)

    def _host(self, t, name):
        if t is None:
            return None
        if t.device.type != "cpu" or t.dtype != self.tdtype or tuple(t.shape) != self.shape or not t.is_contiguous():
            raise MrError(MR_ERR_INVALID_ARG, "%s must be a contiguous CPU %s tensor of shape %r" % (name, self.tdtype, self.shape))
        return t.data_ptr()

    def empty_field(self):
        return self._torch.empty(self.shape, dtype=self.tdtype, device=self.device)

    # -- the C-ABI calls ----------------------------------------------------------------------------------
    def set_B0(self, B0):
        with self._torch.cuda.device(self.device):
            if B0.device.type == "cpu":
                self._check(lib.mr_set_B0_host(self._ctx, self._host(B0, "B0")))
            else:
                self._check(lib.mr_set_B0(self._ctx, self._dev(B0, "B0")))
                self._publish()

    def set_x(self, x):
        with self._torch.cuda.device(self.device):
            if x.device.type == "cpu":
                self._check(lib.mr_set_x_host(self._ctx, self._host(x, "x")))
            else:
                self._check(lib.mr_set_x(self._ctx, self._dev(x, "x")))

    def step(self, n, dt, op="mimetic"):
        with self._torch.cuda.device(self.device):
            self._check(lib.mr_step(self._ctx, int(n), float(dt), _op(op)))

    def step_monitored(self, n, dt, op="mimetic", every=1):
        """mr_step_monitored: n steps; returns the diagnostics (list of dicts) of the states the steps 0, every, 2 every, ... start from."""
        cap = 0 if every <= 0 else (int(n) + int(every) - 1) // int(every)
        hist = (mr_diag * max(cap, 1))()
        w = C.c_int64()
        with self._torch.cuda.device(self.device):
            rc = lib.mr_step_monitored(self._ctx, int(n), float(dt), _op(op), int(every), hist, cap, C.byref(w))
        out = [{"time": h.time, "steps": h.steps, "energy": h.energy, "max_jxb": h.max_jxb, "xi": h.xi, "min_det": h.min_det}
               for h in hist[: w.value]]
        self._check(rc)
        return out

    def diagnostics(self, op="mimetic"):
        out = mr_diag()
        with self._torch.cuda.device(self.device):
            self._check(lib.mr_diagnostics(self._ctx, _op(op), C.byref(out)))
        return {"time": out.time, "steps": out.steps, "energy": out.energy, "max_jxb": out.max_jxb, "xi": out.xi,
                "min_det": out.min_det}

    def get_fields(self, op="mimetic", x=False, B=False, J=False, host=False):
        """Returns the requested fields as new tensors (device, or pinned host with ``host=True``) in a dict."""
        torch = self._torch
        out = {}
        for name, want in (("x", x), ("B", B), ("J", J)):
            if want:
                out[name] = (torch.empty(self.shape, dtype=self.tdtype, pin_memory=True) if host else self.empty_field())
        self.get_fields_into(op, out.get("x"), out.get("B"), out.get("J"))
        return out

    def get_fields_into(self, op="mimetic", x=None, B=None, J=None):
        host = any(t is not None and t.device.type == "cpu" for t in (x, B, J))
        with self._torch.cuda.device(self.device):
            if host:
                self._check(lib.mr_get_fields_host(self._ctx, _op(op), self._host(x, "x"), self._host(B, "B"), self._host(J, "J")))
            else:
                self._check(lib.mr_get_fields(self._ctx, _op(op), self._dev(x, "x"), self._dev(B, "B"), self._dev(J, "J")))
                self._publish()

    def set_xi(self, xi):
        """mr_set_xi: the displacement x - X (what fp32 contexts should exchange instead of positions)."""
        with self._torch.cuda.device(self.device):
            self._check(lib.mr_set_xi(self._ctx, self._dev(xi, "xi")))

    def get_xi(self):
        out = self.empty_field()
        with self._torch.cuda.device(self.device):
            self._check(lib.mr_get_xi(self._ctx, self._dev(out, "xi")))
            self._publish()
        return out

    def rhs(self, op="mimetic"):
        """mr_rhs: the velocity u = gamma J x B of the current state (0 on line-tied boundary nodes)."""
        out = self.empty_field()
        with self._torch.cuda.device(self.device):
            self._check(lib.mr_rhs(self._ctx, _op(op), self._dev(out, "u")))
            self._publish()
        return out

    def step_adaptive(self, t_end, lambda0, dt, op="mimetic", max_trials=1000000, trace=False):
        """mr_step_adaptive: returns a dict (accepted, rejected, rhs_evals, time, dt_next, last_lambda[, trace])."""
        torch = self._torch
        with torch.cuda.device(self.device):
            if self._aworkspace is None:
                g = mr_grid(*self.n)
                bcs = (C.c_int32 * 3)(*[BOUNDARIES[b] for b in self.bc])
                nb = int(lib.mr_adaptive_workspace_bytes_bc(C.byref(g), MR_F64 if self.dtype == "f64" else MR_F32, bcs))
                if self._aworkspace_given is not None:
                    self._aworkspace = self._aworkspace_given
                    nb = int(self._aworkspace.numel())
                else:
                    with torch.cuda.stream(self.stream):
                        self._aworkspace = torch.empty(nb, dtype=torch.uint8, device=self.device)
                self._check(lib.mr_bind_adaptive_workspace(self._ctx, self._aworkspace.data_ptr(), nb))
            st, d = mr_adapt_stats(), C.c_double(float(dt))
            cap = int(min(max_trials, 100000)) if trace else 0
            buf = (C.c_double * (4 * cap))() if cap else None
            rc = lib.mr_step_adaptive(self._ctx, float(t_end), float(lambda0), C.byref(d), _op(op), int(max_trials), C.byref(st),
                                      C.cast(buf, C.c_void_p) if cap else None, cap)
        out = {"accepted": st.accepted, "rejected": st.rejected, "rhs_evals": st.rhs_evals, "time": st.time, "dt_next": st.dt_next,
               "last_lambda": st.last_lambda}
        if trace:
            n = st.accepted + st.rejected
            out["trace"] = [tuple(buf[4 * q:4 * q + 4]) for q in range(min(n, cap))]
        self.last_adaptive = out
        self._check(rc)
        return out

    def convexity(self, want_field=False):
        """mr_convexity: (number of nodes with kappa = -1, kappa as an int32 tensor (nz, ny, nx) or None)."""
        torch = self._torch
        n = C.c_int64()
        kap = torch.empty(self.shape[1:], dtype=torch.int32, device=self.device) if want_field else None
        with torch.cuda.device(self.device):
            if kap is not None:
                self._order(kap)
            self._check(lib.mr_convexity(self._ctx, kap.data_ptr() if kap is not None else None, C.byref(n)))
        return int(n.value), kap

    def eps_star(self, ic, jc, a_r, op="mimetic"):
        """mr_eps_star: (alpha* along the grid line (ic, jc, .) as a list of nz floats, eps*)."""
        al = (C.c_double * self.n[2])()
        e = C.c_double()
        with self._torch.cuda.device(self.device):
            self._check(lib.mr_eps_star(self._ctx, _op(op), int(ic), int(jc), float(a_r), C.cast(al, C.c_void_p), C.byref(e)))
        return list(al), e.value

    def sigma(self, x_ref, B_ref):
        """mr_sigma: (sigma_x, sigma_B) against dense device references."""
        sx, sb = C.c_double(), C.c_double()
        with self._torch.cuda.device(self.device):
            self._check(lib.mr_sigma(self._ctx, self._dev(x_ref, "x_ref"), self._dev(B_ref, "B_ref"), C.byref(sx), C.byref(sb)))
        return sx.value, sb.value

    def set_variant(self, name):
        self._check(lib.mr_set_variant(self._ctx, name.encode()))

    @property
    def launch_count(self):
        return int(lib.mr_launch_count(self._ctx))

    @property
    def step_variant(self):
        return (lib.mr_step_variant(self._ctx) or b"").decode()

    def step_host_async(self, x_in, x_out, n, dt, op="mimetic"):
        """mr_step_host_async: positions in (host tensor), n steps, positions out (host tensor), enqueued without waiting; the
        copy out overlaps the next call's copy in.  Keep both tensors alive and x_out unread until host_sync()."""
        torch = self._torch
        with torch.cuda.device(self.device):
            if getattr(self, "_sworkspace", None) is None:
                g = mr_grid(*self.n)
                nb = int(lib.mr_stream_workspace_bytes(C.byref(g), MR_F64 if self.dtype == "f64" else MR_F32))
                with torch.cuda.stream(self.stream):
                    self._sworkspace = torch.empty(nb, dtype=torch.uint8, device=self.device)
                self._check(lib.mr_bind_stream_workspace(self._ctx, self._sworkspace.data_ptr(), nb))
            self._check(lib.mr_step_host_async(self._ctx, self._host(x_in, "x_in"), self._host(x_out, "x_out"), int(n), float(dt), _op(op)))
            # the copies are queued, not done: hold both host tensors until host_sync() (a pinned block dropped by the caller
            # could be handed out again by the host allocator while a copy still uses it)
            self.__dict__.setdefault("_in_flight", []).append((x_in, x_out))

    def host_sync(self):
        """mr_host_sync: wait for every step_host_async enqueued; raises what mr_set_x / mr_step would have raised."""
        try:
            with self._torch.cuda.device(self.device):
                self._check(lib.mr_host_sync(self._ctx))
        finally:
            self.__dict__.get("_in_flight", []).clear()

    def close(self):
        if getattr(self, "_ctx", None):
            lib.mr_destroy(self._ctx)
            self._ctx = _ctx_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
