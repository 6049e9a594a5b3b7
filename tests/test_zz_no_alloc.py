"""mr_convexity_noalloc: the one call of the library for code that cannot allocate device memory.

A plug-in inside an application that owns every byte of the card, or a check inside a loop that cannot take the device-wide
stall of cudaMalloc, can give the library its input and output arrays and a stream, and nothing more.  This call therefore
keeps its scratch (one counter per z-plane) in an array built into libmr.so instead of a caller workspace.  Checked here
against the existing path, mr_convexity on a context (which counts in the caller-allocated workspace): same count, same
kappa node for node -- integers, so the bar is equality, as in test_convexity_matches_oracle.

Collected last on purpose (pytest -x stops at the first failure; a problem here must not hide the parity tests), and
written to pass both alone in a fresh process and after every other test: the built-in array is shared by all calls and
keeps the previous call's counts, which is exactly what the back-to-back calls on different grids below would expose.
"""
import ctypes as C

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_1405_0942_b200 import inputs as I  # noqa: E402

from gpu_common import dev, make_sim  # noqa: E402


@pytest.fixture(scope="module")
def mr():
    from paper_1405_0942_b200 import build
    build.build()
    from paper_1405_0942_b200 import mr as m
    return m


def _context_answer(mr, g, x, dtype):
    """the existing path: a context holding x, mr_convexity with its counter in the caller's workspace"""
    B0 = np.zeros(g.shape)
    B0[2] = 1.0
    sim = make_sim(mr, g, x, B0, dtype=dtype)
    n, kap = sim.convexity(want_field=True)
    # the positions as the context holds them, in its dtype: what a caller of the context-free call would have in hand
    return n, kap, sim.get_fields(x=True)["x"]


def _dyadic_case(n, seed):
    """Positions whose every coordinate is a multiple of 2^-10 below 8 in magnitude (h = 1/4, kicks of up to 0.9 h rounded
    to 2^-10): exact in fp32, and so are the displacements, the edge vectors and -- in the kernels' double arithmetic -- the
    determinants.  Differencing positions (this call) and differencing displacements (the context) then decide every sign
    from the same exact number, so even an fp32 comparison is an equality."""
    g = I.Grid(n, tuple(-0.125 * (v - 1) for v in n), tuple(0.125 * (v - 1) for v in n))
    rng = np.random.default_rng(seed)
    xi = np.round(rng.uniform(-0.9, 0.9, size=g.shape) * 0.25 * 1024.0) / 1024.0
    for a in range(3):                                   # line-tied faces stay on X
        sl = [slice(None)] * 4
        for end in (0, -1):
            sl[3 - a] = end
            xi[tuple(sl)] = 0.0
    return g, I.reference_grid(g) + xi


@pytest.mark.gpu
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_noalloc_convexity_equals_the_context_path_on_two_calls_in_a_row(mr, dtype):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    if dtype == "f64":
        # 0.9 h random kicks: a good share of concave nodes (the case of test_convexity_matches_oracle), then a second,
        # smaller grid with fewer planes and another seed
        ga = I.Grid((37, 21, 13), (-4.0, -4.0, -8.0), (4.0, 4.0, 8.0))
        gb = I.Grid((70, 9, 6), (-4.0, -1.0, -1.0), (4.0, 1.0, 1.0))
        cases = [(ga, I.rough_displacement(ga, 0.9, seed=21)), (gb, I.rough_displacement(gb, 0.7, seed=22))]
    else:
        cases = [_dyadic_case((33, 17, 9), 31), _dyadic_case((17, 41, 5), 32)]
    want = [_context_answer(mr, g, x, dtype) for g, x in cases]
    assert all(0 < w[0] < g.nodes for w, (g, _) in zip(want, cases))
    # the two calls back to back (the second starts from the counters the first one left behind), then the first again
    for q in (0, 1, 0):
        n_ref, kap_ref, x_dev = want[q]
        kap = torch.full_like(kap_ref, 7)
        n = mr.convexity_noalloc(x_dev, kap)
        assert n == n_ref, (q, n, n_ref)
        assert torch.equal(kap, kap_ref), q
        assert mr.convexity_noalloc(x_dev) == n_ref          # kappa is optional
    # an undistorted grid has no concave node, whatever was counted before
    g = cases[0][0]
    td = torch.float64 if dtype == "f64" else torch.float32
    assert mr.convexity_noalloc(dev(I.reference_grid(g), td)) == 0


def test_noalloc_refuses_what_its_scratch_cannot_hold(mr):
    """Argument checks come before any CUDA call, so they run without a GPU: more z-planes than the built-in array has
    counters for is an error with a message that names the limit, not a silent overrun."""
    n = C.c_int64(-1)
    fake = C.c_void_p(256)
    def call(nx, ny, nz, dtype=0, x=fake):
        return mr.lib.mr_convexity_noalloc(x, C.byref(mr.mr_grid(nx, ny, nz)), dtype, None, C.byref(n), None)
    assert mr.NOALLOC_MAX_PLANES == 1024
    assert call(8, 8, mr.NOALLOC_MAX_PLANES + 1) == mr.MR_ERR_INVALID_ARG
    msg = mr.lib.mr_last_error(None).decode()
    assert "1025" in msg and "1024" in msg and "mr_convexity" in msg
    assert call(8, 8, 1) == mr.MR_ERR_INVALID_ARG
    assert call(5000, 8, 8) == mr.MR_ERR_INVALID_ARG
    assert call(8, 8, 8, dtype=3) == mr.MR_ERR_INVALID_ARG
    assert call(8, 8, 8, x=None) == mr.MR_ERR_INVALID_ARG
    assert n.value == -1
    if not torch.cuda.is_available():
        assert call(8, 8, 8) == mr.MR_ERR_CUDA           # no device: fails loudly, no fallback
