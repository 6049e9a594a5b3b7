"""GPU parity tests proper: the CUDA path (through the C-ABI, via the ctypes binding) against the CPU oracle on the
same seeded inputs.  Tolerances (north_star / DESIGN.md Q19): norm-wise relative error per field
max|a-b| / max|b|  <= 1e-12 after one step, <= 1e-9 after 100 steps (fp64); fp32 variant <= 1e-5.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from oracle import mro  # noqa: E402  (test infrastructure)
from paper_1405_0942_b200 import inputs as I  # noqa: E402

from gpu_common import CASES, TOL_100, TOL_F32, TOL_STEP, case, dev, fields_np, make_sim, nrel, opcode  # noqa: E402


@pytest.fixture(scope="module")
def mr():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1405_0942_b200 import mr as m
    return m


@pytest.fixture(scope="module", autouse=True)
def oracle_threads():
    mro.set_threads(mro.max_threads())
    yield
    mro.set_threads(1)


@pytest.mark.parametrize("name", CASES)
@pytest.mark.parametrize("op", ["mimetic", "direct"])
def test_fields_match_oracle(mr, name, op):
    """S1-S3: B on all nodes, J on interior nodes (0 on the boundary), x round trip."""
    g, x0, B0, dt = case(name)
    sim = make_sim(mr, g, x0, B0)
    f = fields_np(sim, op)
    B, J, u, det = mro.fields(g.n, g.lo, g.hi, x0, B0, op=mro.MIMETIC if op == "mimetic" else mro.DIRECT)
    assert nrel(f["x"], x0) < 1e-15
    assert nrel(f["B"], B) < TOL_STEP
    assert nrel(f["J"], J) < TOL_STEP
    Jb = f["J"].copy()
    Jb[:, 1:-1, 1:-1, 1:-1] = 0
    assert np.abs(Jb).max() == 0.0


@pytest.mark.parametrize("name", CASES)
@pytest.mark.parametrize("op", ["mimetic", "direct"])
@pytest.mark.parametrize("variant", ["auto", "generic"])
def test_one_step_matches_oracle(mr, name, op, variant):
    """S1-S5 fused: x after one step, also measured on the displacement moved in that step.  Every step-kernel
    variant of the library is held to the same bar ("auto" is the one the bench times)."""
    g, x0, B0, dt = case(name)
    sim = make_sim(mr, g, x0, B0, variant=variant)
    sim.step(1, dt, op)
    x1 = sim.get_fields(op, x=True)["x"].cpu().numpy()
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 1, op=mro.MIMETIC if op == "mimetic" else mro.DIRECT)
    assert nrel(x1, ref) < TOL_STEP
    moved = np.abs(ref - x0).max()
    assert moved > 0
    assert np.abs(x1 - ref).max() < 1e-10 * moved + 1e-15 * np.abs(ref).max()
    # S4 itself: the velocity of the step kernel's right-hand side against the oracle's u = gamma J x B, at 1e-12
    u = mro.fields(g.n, g.lo, g.hi, x0, B0, op=opcode(op))[2]
    sim0 = make_sim(mr, g, x0, B0, variant=variant)
    assert nrel(sim0.rhs(op).cpu().numpy(), u) < TOL_STEP
    # line-tied: boundary nodes did not move at all
    m = np.ones(x1.shape, bool)
    m[:, 1:-1, 1:-1, 1:-1] = False
    assert np.array_equal(x1[m], np.asarray(x0)[m])


@pytest.mark.parametrize("n", [(4096, 5, 5), (5, 4096, 5), (5, 5, 4096), (4096, 6, 7)])
@pytest.mark.parametrize("op", ["mimetic", "direct"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_maximum_extents_match_oracle(mr, n, op, dtype):
    """The largest extent the ABI accepts (4096) along each axis with the smallest one (5) along the others: 128 tiles in x with
    every node next to a face in y and z, 256 tiles in y, a march of 4096 planes cut into as many z-chunks as there are SMs.
    Three steps and S6 against the oracle (fp32: against the oracle through the displacement, Q15)."""
    lo = tuple(-0.01 * (m - 1) for m in n)
    hi = tuple(0.01 * (m - 1) for m in n)                       # h = 0.02 on every axis
    g = I.Grid(n, lo, hi)
    X = I.reference_grid(g)
    s = [2.0 * np.pi * (X[a] - lo[a]) / 0.64 for a in range(3)]                # wavelength 32 h
    env = np.ones_like(X[0])
    for a in range(3):
        env = env * np.sin(np.pi * (X[a] - lo[a]) / (hi[a] - lo[a]))
    env[0], env[-1], env[:, 0], env[:, -1], env[:, :, 0], env[:, :, -1] = 0.0, 0.0, 0.0, 0.0, 0.0, 0.0    # exactly zero on the faces
    x0 = X.copy()
    x0[0] += 0.004 * env * np.sin(s[1] + s[2])
    x0[1] += 0.003 * env * np.cos(s[0]) * np.sin(s[2] + 0.3)
    x0[2] += 0.004 * env * np.sin(s[0] + 0.5 * s[1])
    B0 = np.empty_like(X)
    B0[0] = 0.3 * np.sin(s[2]) + 0.1 * np.cos(s[1])
    B0[1] = 0.2 * np.cos(s[0] + s[2])
    B0[2] = 1.0 + 0.2 * np.sin(s[0]) * np.cos(s[1])
    dt = 0.5 * I.stable_dt(B0, g)
    sim = make_sim(mr, g, x0, B0, dtype=dtype)
    d = sim.diagnostics(op)
    sim.step(3, dt, op)
    assert sim.step_variant.startswith("sym" if op == "mimetic" else "direct_tma")
    o = mro.diagnostics(g.n, g.lo, g.hi, x0, B0, op=opcode(op))
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 3, op=opcode(op))
    tol = TOL_STEP if dtype == "f64" else TOL_F32
    for k in ("energy", "max_jxb", "min_det"):           # (an fp32 context forms J in fp32: eps |B| / 2h of it is rounding)
        assert d[k] == pytest.approx(o[k], rel=10 * tol if (dtype == "f64" or k != "max_jxb") else 2e-3), k
    xi = sim.get_xi().double().cpu().numpy()
    assert np.abs(xi - (ref - X)).max() < 10 * tol * np.abs(ref - X).max()
    moved = np.abs(ref - x0).max()
    assert moved > 0
    if dtype == "f64":
        assert np.abs(xi - (ref - X)).max() < 1e-9 * moved
    m = np.ones(xi.shape, bool)
    m[:, 1:-1, 1:-1, 1:-1] = False
    assert not xi[m].any()                                      # line-tied faces: the displacement stays exactly zero


@pytest.mark.parametrize("name,steps", [("C1", 100), ("C2_small", 100), ("C3_small", 100), ("ragged", 100)])
@pytest.mark.parametrize("variant", ["auto", "generic"])
def test_100_steps_match_oracle(mr, name, steps, variant):
    g, x0, B0, dt = case(name)
    sim = make_sim(mr, g, x0, B0, variant=variant)
    sim.step(steps, dt, "mimetic")
    x = sim.get_fields(x=True)["x"].cpu().numpy()
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, steps)
    assert nrel(x, ref) < TOL_100
    assert nrel(x - x0, ref - x0) < 1e-7       # on the displacement itself
    d = sim.diagnostics("mimetic")
    assert d["steps"] == steps and d["time"] == pytest.approx(steps * dt, rel=1e-12)
    o = mro.diagnostics(g.n, g.lo, g.hi, ref, B0)
    for k in ("energy", "max_jxb", "xi", "min_det"):
        assert d[k] == pytest.approx(o[k], rel=1e-8)


def test_100_direct_steps_match_oracle(mr):
    g, x0, B0, dt = case("C1")
    sim = make_sim(mr, g, x0, B0)
    sim.step(100, dt, "direct")
    x = sim.get_fields(x=True)["x"].cpu().numpy()
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 100, op=mro.DIRECT)
    assert nrel(x, ref) < TOL_100


@pytest.mark.parametrize("name", CASES)
@pytest.mark.parametrize("op", ["mimetic", "direct"])
def test_diagnostics_match_oracle(mr, name, op):
    """S6: energy, max|JxB|, xi, min det within 1e-12 relative; deterministic (bitwise repeatable)."""
    g, x0, B0, dt = case(name)
    sim = make_sim(mr, g, x0, B0)
    d = sim.diagnostics(op)
    o = mro.diagnostics(g.n, g.lo, g.hi, x0, B0, op=mro.MIMETIC if op == "mimetic" else mro.DIRECT)
    for k in ("energy", "max_jxb", "xi", "min_det"):
        assert d[k] == pytest.approx(o[k], rel=TOL_STEP), k
    assert sim.diagnostics(op) == d


def test_config3_reading_P_curl_errors(mr):
    """Config 3, reading P (B0 pulled back so that the nodal pushed-forward field is ABC(x0)): both curl errors are
    the oracle's, the mimetic one is the smaller, and the field stays near force-free over 50 steps."""
    cfg = I.scaled(I.CONFIGS["C3"], (48, 48, 48))
    g = cfg.grid
    x0 = I.displaced_grid(g, 0.3)
    F, det = mro.jacobian(g.n, g.lo, g.hi, x0)
    Fi = np.linalg.inv(np.moveaxis(F, (0, 1), (-2, -1)))
    B0 = np.ascontiguousarray(np.einsum("...ac,c...->a...", Fi, I.abc_field(x0)) * det)
    dt = I.stable_dt(B0, g)
    sim = make_sim(mr, g, x0, B0)
    errs = {}
    for op, code in (("mimetic", 0), ("direct", 1)):
        f = fields_np(sim, op)
        _, J, _, _ = mro.fields(g.n, g.lo, g.hi, x0, B0, op=code)
        assert nrel(f["B"], I.abc_field(x0)) < 1e-12
        assert nrel(f["J"], J) < TOL_STEP
        inner = (slice(None), slice(1, -1), slice(1, -1), slice(1, -1))
        errs[op] = np.abs(f["J"][inner] - np.pi * f["B"][inner]).max() / (np.pi * np.abs(f["B"]).max())
    assert errs["mimetic"] < errs["direct"] < 0.02
    f0 = sim.diagnostics()["max_jxb"]
    sim.step(50, dt)
    assert sim.diagnostics()["max_jxb"] < 2.0 * f0 + 1e-3      # stays (near) force-free
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 50)
    assert nrel(sim.get_fields(x=True)["x"].cpu().numpy(), ref) < TOL_100


def test_abc_on_undistorted_grid_does_not_move(mr):
    g = I.Grid((32, 32, 32), (-1.0, -1.0, -1.0), (1.0, 1.0, 1.0))
    X = I.reference_grid(g)
    B0 = I.abc_field(X)
    sim = make_sim(mr, g, X, B0)
    sim.step(20, I.stable_dt(B0, g))
    x = sim.get_fields(x=True)["x"].cpu().numpy()
    assert np.abs(x - X).max() < 1e-13
    assert sim.diagnostics()["max_jxb"] < 1e-11


def rel_dev(a, b):
    """norm-wise relative difference of two device tensors (Q19), evaluated on the device in fp64"""
    a, b = a.double(), b.double()
    return float((a - b).abs().max() / b.abs().max())


@pytest.mark.parametrize("variant", ["auto", "generic"])
def test_fp32_variant_within_1e5_of_fp64(mr, variant):
    """fp32 storage+arithmetic (displacement storage, Q15) against the fp64 GPU run and the fp64 oracle: every field of
    north_star's list -- x, B and J -- within 1e-5 norm-wise (Q19), and the displacement itself to 1e-4."""
    cfg = I.scaled(I.CONFIGS["C5"], (64, 64, 64))
    g = cfg.grid
    x0, B0, dt = I.make(cfg)
    s64 = make_sim(mr, g, x0, B0, "f64", variant)
    s32 = make_sim(mr, g, x0, B0, "f32", variant)
    s64.step(100, dt)
    s32.step(100, dt)
    xi64, xi32 = s64.get_xi(), s32.get_xi()
    xmax = float(np.abs(x0).max())
    assert float((xi32.double() - xi64).abs().max()) / xmax < TOL_F32         # x = X + xi, |x| <= 4
    assert rel_dev(xi32, xi64) < 1e-4                                          # even on the displacement itself
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 100)
    assert nrel(s64.get_fields(x=True)["x"].cpu().numpy(), ref) < TOL_100
    f32, f64 = s32.get_fields("mimetic", B=True, J=True), s64.get_fields("mimetic", B=True, J=True)
    assert rel_dev(f32["B"], f64["B"]) < TOL_F32
    assert rel_dev(f32["J"], f64["J"]) < TOL_F32
    d32, d64 = s32.diagnostics(), s64.diagnostics()
    assert d32["energy"] == pytest.approx(d64["energy"], rel=TOL_F32)


@pytest.mark.parametrize("name", ["pow2p1", "pow2p1_wide", "tail1", "ragged"])
@pytest.mark.parametrize("op", ["mimetic", "direct"])
def test_fp32_steps_on_ragged_and_face_ring_tilings(mr, name, op):
    """The fp32 kernels (two nodes per thread, 64-wide tiles) on grids whose faces fall on tile edges, ring columns and ragged
    tails: 20 steps against the oracle through the displacement (Q15), and the faces stay exactly where they are."""
    g, x0, B0, dt = case(name)
    sim = make_sim(mr, g, x0, B0, dtype="f32")
    sim.step(20, dt, op)
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 20, op=opcode(op))
    X = I.reference_grid(g)
    xi = sim.get_xi().double().cpu().numpy()
    assert np.abs(xi - (ref - X)).max() < 3 * TOL_F32 * np.abs(ref - X).max()
    m = np.ones(xi.shape, bool)
    m[:, 1:-1, 1:-1, 1:-1] = False
    assert not xi[m].any()
    f = sim.get_fields(op, B=True)["B"].double().cpu().numpy()
    assert nrel(f, mro.fields(g.n, g.lo, g.hi, ref, B0, op=opcode(op))[0]) < 3 * TOL_F32


def test_fp32_variant_full_size_config5(mr):
    """BASELINE configs[4] at full size (512^3, the launch configuration bench.py --workload C5 times): the fp32 context
    against an fp64 context on the same inputs.  After 100 steps x, B and J are within 1e-5 norm-wise (Q19).  After the
    config's 1000 steps the state (x, the displacement itself, B) still is; J, a second difference of a state that has by then
    been rounded to fp32 a thousand times, is not: its deviation grows like the square root of the step count (measured
    6.3e-6, 1.37e-5, 2.04e-5 after 100, 500, 1000 steps) and is held to 3e-5 (Q15)."""
    cfg = I.CONFIGS["C5"]
    g = cfg.grid
    x0, B0, dt = I.make(cfg)
    B0t = torch.from_numpy(B0)
    del x0
    sims = {}
    for dtype, td in (("f64", torch.float64), ("f32", torch.float32)):
        s = mr.Relaxation(g.n, g.lo, g.hi, dtype=dtype)
        s.set_B0(B0t.to("cuda", dtype=td))
        sims[dtype] = s                                     # starts at x = X: no mr_set_x

    def deviations():
        xi64, xi32 = sims["f64"].get_xi(), sims["f32"].get_xi()
        errs = {"x": float((xi32.double() - xi64).abs().max()) / 4.0, "xi": rel_dev(xi32, xi64)}
        del xi64, xi32
        for name in ("B", "J"):
            a = sims["f32"].get_fields("mimetic", **{name: True})[name]
            b = sims["f64"].get_fields("mimetic", **{name: True})[name]
            errs[name] = rel_dev(a, b)
            del a, b
        return errs

    for s in sims.values():
        s.step(100, dt)
    assert sims["f32"].step_variant == "sym_tmem_f32" and sims["f64"].step_variant == "sym_tmem_f64"
    e100 = deviations()
    print("fp32 vs fp64 at 512^3 after 100 steps:", e100)
    assert e100["x"] < TOL_F32 and e100["B"] < TOL_F32 and e100["J"] < TOL_F32 and e100["xi"] < TOL_F32, e100
    for s in sims.values():
        s.step(cfg.steps - 100, dt)
    e1000 = deviations()
    print("... after %d steps:" % cfg.steps, e1000)
    assert e1000["x"] < TOL_F32 and e1000["B"] < TOL_F32 and e1000["xi"] < TOL_F32, e1000
    assert e1000["J"] < 3e-5, e1000
    d64, d32 = sims["f64"].diagnostics(), sims["f32"].diagnostics()
    assert d32["energy"] == pytest.approx(d64["energy"], rel=1e-6) and d32["xi"] == pytest.approx(d64["xi"], rel=1e-4)


def test_host_buffer_entry_points_round_trip(mr):
    g, x0, B0, dt = case("ragged")
    sim = mr.Relaxation(g.n, g.lo, g.hi)
    sim.set_B0(torch.from_numpy(B0).pin_memory())
    sim.set_x(torch.from_numpy(np.ascontiguousarray(x0)))          # pageable host memory also works
    sim.step(3, dt)
    out = sim.get_fields(x=True, B=True, J=True, host=True)
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 3)
    B, J, _, _ = mro.fields(g.n, g.lo, g.hi, ref, B0)
    assert nrel(out["x"].numpy(), ref) < TOL_STEP
    assert nrel(out["B"].numpy(), B) < 1e-11
    assert nrel(out["J"].numpy(), J) < 1e-10


@pytest.mark.parametrize("op", ["mimetic", "direct"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_streaming_host_calls_equal_the_synchronous_ones(mr, op, dtype):
    """mr_step_host_async / mr_host_sync: six calls in flight (the copy out of one overlapping the copy in of the next, pinned
    buffers) give bit for bit what mr_set_x_host + mr_step + mr_get_fields_host give one after the other; a state whose
    line-tied faces are off the reference grid is reported by the sync, and so is a folded grid."""
    g, x0, B0, dt = case("ragged")
    td = torch.float64 if dtype == "f64" else torch.float32
    X = I.reference_grid(g)
    ins = [torch.from_numpy(X + s * (x0 - X)).to(td).pin_memory() for s in (1.0, 0.5, -0.5, 0.25, 0.0, 0.8)]
    outs = [torch.empty_like(t).pin_memory() for t in ins]
    sim = mr.Relaxation(g.n, g.lo, g.hi, dtype=dtype)
    sim.set_B0(dev(B0, td))
    for a, b in zip(ins, outs):
        sim.step_host_async(a, b, 3, dt, op)
    sim.host_sync()
    ref = mr.Relaxation(g.n, g.lo, g.hi, dtype=dtype)
    ref.set_B0(dev(B0, td))
    for a, b in zip(ins, outs):
        ref.set_x(a)
        ref.step(3, dt, op)
        want = ref.get_fields(op, x=True, host=True)["x"]
        assert torch.equal(b, want)
    assert sim.diagnostics(op)["steps"] == 3
    # while calls are in flight the error word belongs to them: the calls that use it are refused until the sync
    sim.step_host_async(ins[0], outs[0], 1, dt, op)
    for call in (lambda: sim.step(1, dt, op), lambda: sim.diagnostics(op), lambda: sim.set_x(ins[1]), lambda: sim.set_x(dev(x0, td)),
                 lambda: sim.get_fields(op, x=True, host=True), lambda: sim.step_monitored(2, dt, op)):
        with pytest.raises(mr.MrError) as e:
            call()
        assert e.value.status == mr.MR_ERR_STATE
    sim.host_sync()
    assert sim.diagnostics(op)["steps"] == 1
    bad = ins[0].clone().pin_memory()
    bad[0, 0, 0, 0] += 0.1                                     # a corner node off X
    sim.step_host_async(bad, outs[0], 1, dt, op)
    sim.step_host_async(ins[1], outs[1], 1, dt, op)
    with pytest.raises(mr.MrError) as e:
        sim.host_sync()
    assert e.value.status == mr.MR_ERR_INVALID_ARG
    sim.step_host_async(ins[1], outs[1], 1, dt, op)            # a good state clears the failure
    sim.host_sync()
    fold = ins[0].clone().pin_memory()
    fold[0, 3, 3, 3] += 5.0 * g.h[0]                           # an inner node far past its neighbours
    sim.step_host_async(fold, outs[0], 1, dt, op)
    with pytest.raises(mr.NumericError):
        sim.host_sync()
    with pytest.raises(mr.MrError):
        sim.step(1, dt, op)                                    # failed until a new state is set
    sim.set_x(ins[1])
    sim.step(1, dt, op)


@pytest.mark.parametrize("name,bc", [("C1", None), ("pow2p1", None), ("ragged", None), ("tail1", ("line_tied", "line_tied", "periodic"))])
@pytest.mark.parametrize("op", ["mimetic", "direct"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_monitored_steps_equal_steps_and_diagnostics(mr, name, bc, op, dtype):
    """mr_step_monitored: the record of step s is what mr_diagnostics returns before step s, and the state after the run is the
    state mr_step reaches: bit for bit.  (Mimetic: the step kernel reduces S6 in the same pass, MODE_STEPDIAG; the records that
    are not asked for cost nothing.)"""
    g, x0, B0, dt = case(name)
    bc = bc or ("line_tied",) * 3
    if "periodic" in bc:
        x0 = I.reference_grid(g)
    a = make_sim(mr, g, x0, B0, dtype=dtype, bc=bc)
    b = make_sim(mr, g, x0, B0, dtype=dtype, bc=bc)
    hist = a.step_monitored(11, dt, op, every=3)               # records before the steps 0, 3, 6, 9
    assert [h["steps"] for h in hist] == [0, 3, 6, 9]
    for q, h in enumerate(hist):
        d = b.diagnostics(op)
        for k in ("energy", "max_jxb", "xi", "min_det"):
            assert h[k] == d[k], (q, k, h[k], d[k])
        assert h["time"] == pytest.approx(d["time"], rel=1e-14, abs=1e-300)       # (3 dt + 3 dt + ... against s dt)
        b.step(3 if q < 3 else 2, dt, op)
    assert torch.equal(a.get_xi(), b.get_xi())
    da, db = a.diagnostics(op), b.diagnostics(op)
    assert all(da[k] == db[k] for k in ("steps", "energy", "max_jxb", "xi", "min_det"))
    assert a.step_monitored(5, dt, op, every=0) == []          # no records asked for: plain steps
    b.step(5, dt, op)
    assert torch.equal(a.get_xi(), b.get_xi())
    one = a.step_monitored(1, dt, op, every=1)
    assert len(one) == 1 and one[0]["steps"] == 16


def test_error_paths_on_device(mr):
    g, x0, B0, dt = case("C1")
    sim = mr.Relaxation(g.n, g.lo, g.hi)
    with pytest.raises(mr.MrError) as e:
        sim.step(1, dt)
    assert e.value.status == mr.MR_ERR_STATE
    sim.set_B0(dev(B0))
    with pytest.raises(mr.MrError) as e:
        sim.step(1, -1.0)
    assert e.value.status == mr.MR_ERR_INVALID_ARG
    bad = np.array(x0)
    bad[0, 0, 3, 3] += 0.1                                         # a boundary node off the reference grid
    with pytest.raises(mr.MrError) as e:
        sim.set_x(dev(bad))
    assert e.value.status == mr.MR_ERR_INVALID_ARG
    assert nrel(sim.get_fields(x=True)["x"].cpu().numpy(), x0) < 1e-15      # state unchanged
    folded = np.array(x0)
    folded[0, 10, 8, 8] += 5.0                                     # folds the grid: det <= 0
    sim.set_x(dev(folded))
    with pytest.raises(mr.NumericError):
        sim.step(1, dt)
    with pytest.raises(mr.NumericError):                           # sticky until mr_set_x
        sim.step(1, dt)
    with pytest.raises(mro.NumericError):
        mro.step(g.n, g.lo, g.hi, folded, B0, dt, 1)               # the oracle agrees that this is a failure
    sim.set_x(dev(x0))
    sim.step(1, dt)
    wrong = torch.zeros((3, 4, 4, 4), device="cuda", dtype=torch.float64)
    with pytest.raises(mr.MrError):
        sim.set_B0(wrong)


def test_zero_steps_is_a_no_op(mr):
    g, x0, B0, dt = case("C1")
    sim = make_sim(mr, g, x0, B0)
    sim.step(0, dt)
    assert np.array_equal(sim.get_fields(x=True)["x"].cpu().numpy(), x0)


@pytest.mark.parametrize("op", ["mimetic", "direct"])
@pytest.mark.parametrize("name,bc", [("C1", None), ("ragged", None), ("C1", ("line_tied", "line_tied", "periodic"))])
def test_graph_replay_is_bit_identical_to_plain_launches(mr, op, name, bc):
    """on an L2-resident grid mr_step replays sixteen captured steps per CUDA-graph launch.  Same kernels, same
    order: the state after 37 + 64 + 3 steps (graph launches, a remainder, a re-capture from the other buffer, a call too
    short for a graph) equals the one from plain launches bit for bit, and the launch counter counts the same launches."""
    g, x0, B0, dt = case(name)
    bc = bc or ("line_tied",) * 3
    if bc[2] == "periodic":
        x0 = I.reference_grid(g)                    # (the C1 field is not periodic in z: start undisplaced, step little)
    sims = {}
    for v in ("graph", "nograph"):
        sim = make_sim(mr, g, x0, B0, bc=bc)
        sim.set_variant(v)
        l0 = sim.launch_count
        for n in (37, 64, 3):
            sim.step(n, dt, op)
        launches = sim.launch_count - l0
        sims[v] = (sim.get_xi().cpu().numpy(), launches, sim.diagnostics(op))
    assert np.array_equal(sims["graph"][0], sims["nograph"][0])
    assert sims["graph"][1] == sims["nograph"][1] == 104 * (2 if bc[2] == "periodic" else 1)
    assert sims["graph"][2]["steps"] == 104 and sims["graph"][2]["energy"] == sims["nograph"][2]["energy"]
    with pytest.raises(mr.MrError):
        sim.set_variant("no-such-kernel")


@pytest.mark.parametrize("name,bc,dtype", [("ragged", ("line_tied",) * 3, "f64"), ("wide", ("line_tied",) * 3, "f32"),
                                           ("tail1", ("periodic",) * 3, "f64"), ("minimal", ("periodic", "line_tied", "periodic"), "f32")])
def test_no_write_outside_the_buffers_the_caller_gave(mr, name, bc, dtype):
    """compute-sanitizer is closed on this pool, so the library is run with every buffer it is given embedded in a canary:
    both workspaces exactly as large as mr_*_workspace_bytes_bc says, dense output arrays of exactly 3 nx ny nz elements, 4 KiB
    of 0xA5 either side.  Every entry point that writes (steps of both operators, S6, right-hand side, the adaptive integrator,
    convexity with its map, fields, displacement) must leave the canaries intact."""
    import ctypes as C
    g, x0, B0, dt = case(name)
    if "periodic" in bc:
        x0 = I.reference_grid(g)                   # (these fields are not periodic: stay at x = X, step little)
        dt = 1e-3 * dt
    td = torch.float64 if dtype == "f64" else torch.float32
    G = 4096
    canaries = []

    def guarded(nbytes):
        big = torch.full((nbytes + 2 * G,), 0xA5, dtype=torch.uint8, device="cuda")
        canaries.append((big, nbytes))
        return big[G:G + nbytes]

    gg = mr.mr_grid(*g.n)
    bcs = (C.c_int32 * 3)(*[mr.BOUNDARIES[b] for b in bc])
    code = mr.MR_F64 if dtype == "f64" else mr.MR_F32
    ws = guarded(int(mr.lib.mr_workspace_bytes_bc(C.byref(gg), code, bcs)))
    aws = guarded(int(mr.lib.mr_adaptive_workspace_bytes_bc(C.byref(gg), code, bcs)))
    sim = mr.Relaxation(g.n, g.lo, g.hi, dtype=dtype, bc=bc, workspace=ws, adaptive_workspace=aws)
    es = 8 if dtype == "f64" else 4
    dense = lambda: guarded(3 * g.nodes * es).view(td).view(sim.shape)     # noqa: E731
    sim.set_B0(dev(B0, td))
    sim.set_xi(dev(x0 - I.reference_grid(g), td))
    for variant in ("auto", "generic"):
        sim.set_variant(variant)
        for op in ("mimetic", "direct"):
            sim.step(3, dt, op)
            sim.step(40, dt, op)                                           # (a graph replay on these L2-resident grids)
            sim.diagnostics(op)
            assert mr.lib.mr_rhs(sim._ctx, mr._op(op), C.c_void_p(dense().data_ptr())) == mr.MR_OK
            sim.step_adaptive(t_end=sim.diagnostics(op)["time"] + 3 * dt, lambda0=1e-7, dt=dt, op=op)
            sim.get_fields_into(op, x=dense(), B=dense(), J=dense())
            sim.eps_star(g.n[0] // 2, g.n[1] // 2, 1.0, op)
    assert mr.lib.mr_get_xi(sim._ctx, C.c_void_p(dense().data_ptr())) == mr.MR_OK
    sws = guarded(int(mr.lib.mr_stream_workspace_bytes(C.byref(gg), code)))      # the streaming host calls' staging field
    assert mr.lib.mr_bind_stream_workspace(sim._ctx, C.c_void_p(sws.data_ptr()), sws.numel()) == mr.MR_OK
    sim._sworkspace = sws
    hin = torch.from_numpy(I.reference_grid(g)).to(td).pin_memory()
    houts = [torch.empty_like(hin).pin_memory() for _ in range(3)]
    for h in houts:
        sim.step_host_async(hin, h, 2, dt, "mimetic")
    sim.host_sync()
    kap = guarded(4 * g.nodes)
    nconc = C.c_int64()
    assert mr.lib.mr_convexity(sim._ctx, C.c_void_p(kap.data_ptr()), C.byref(nconc)) == mr.MR_OK
    sim.sigma(dev(x0, td), dev(B0, td))
    torch.cuda.synchronize()
    for big, nbytes in canaries:
        assert bool((big[:G] == 0xA5).all()) and bool((big[G + nbytes:] == 0xA5).all())


def test_full_size_config4_one_step_matches_oracle(mr):
    """BASELINE configs[3] at full size (256x256x512, the bench workload and launch configuration), initial grid
    smoothly displaced so that every term is exercised: x after one step and the diagnostics against the oracle
    on the WHOLE grid (the oracle needs a few seconds per step with all host threads)."""
    cfg = I.CONFIGS["C4"]
    g = cfg.grid
    _, B0, dt = I.make(cfg)
    x0 = I.displaced_grid(g, 0.3, seed=11)
    sim = make_sim(mr, g, x0, B0)
    d = sim.diagnostics()
    sim.step(1, dt)
    x1 = sim.get_fields(x=True, host=True)["x"].numpy()
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 1)
    assert nrel(x1, ref) < TOL_STEP
    moved = np.abs(ref - x0).max()
    assert np.abs(x1 - ref).max() < 1e-10 * moved + 1e-15 * np.abs(ref).max()
    o = mro.diagnostics(g.n, g.lo, g.hi, x0, B0)
    for k in ("energy", "max_jxb", "xi", "min_det"):
        assert d[k] == pytest.approx(o[k], rel=TOL_STEP), k


def test_full_size_config4_direct_operator_matches_oracle(mr):
    """The direct-derivative operator at the full 256x256x512: one step and the diagnostics (the streaming pass over the
    inner nodes plus the pass over the faces) against the oracle on the whole grid."""
    cfg = I.CONFIGS["C4"]
    g = cfg.grid
    _, B0, dt = I.make(cfg)
    x0 = I.displaced_grid(g, 0.3, seed=12)
    sim = make_sim(mr, g, x0, B0)
    d = sim.diagnostics("direct")
    sim.step(1, dt, "direct")
    assert sim.step_variant == "direct_tma_f64"
    x1 = sim.get_fields(x=True, host=True)["x"].numpy()
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 1, op=mro.DIRECT)
    assert nrel(x1, ref) < TOL_STEP
    moved = np.abs(ref - x0).max()
    assert np.abs(x1 - ref).max() < 1e-10 * moved + 1e-15 * np.abs(ref).max()
    o = mro.diagnostics(g.n, g.lo, g.hi, x0, B0, op=mro.DIRECT)
    for k in ("energy", "max_jxb", "xi", "min_det"):
        assert d[k] == pytest.approx(o[k], rel=TOL_STEP), k


@pytest.mark.parametrize("op", ["mimetic", "direct"])
def test_full_size_config2_100_steps_both_operators(mr, op):
    """BASELINE configs[1] on its OWN grid (64x64x192, both operators side by side), SURVEY 8(d)'s 100-step gate: this is the
    grid on which mr_step replays CUDA graphs over 2x4 tiles and several z-chunks, so the graph and the plain-launch variant
    are both held against the oracle: x <= 1e-9, the displacement moved to 1e-7, S6 of the state reached to 1e-8."""
    cfg = I.CONFIGS["C2"]
    g = cfg.grid
    assert g.n == (64, 64, 192)
    x0, B0, dt = I.make(cfg)
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 100, op=opcode(op))
    o = mro.diagnostics(g.n, g.lo, g.hi, ref, B0, op=opcode(op))
    moved = np.abs(ref - x0).max()
    assert moved > 0
    xs = {}
    for v in ("graph", "nograph"):
        sim = make_sim(mr, g, x0, B0)
        sim.set_variant(v)
        sim.step(100, dt, op)
        assert sim.step_variant == ("sym_tmem_f64" if op == "mimetic" else "direct_tma_f64"), sim.step_variant
        xs[v] = sim.get_fields(x=True)["x"].cpu().numpy()
        assert nrel(xs[v], ref) < TOL_100
        assert np.abs(xs[v] - ref).max() < 1e-7 * moved
        d = sim.diagnostics(op)
        assert d["steps"] == 100
        for k in ("energy", "max_jxb", "xi", "min_det"):
            assert d[k] == pytest.approx(o[k], rel=1e-8), (v, k)
    assert np.array_equal(xs["graph"], xs["nograph"])


def test_full_size_config4_20_step_prefix_matches_oracle(mr):
    """BASELINE configs[3] (256x256x512) through a 20-step prefix of its run, from the configuration's own initial state, in
    the launch configuration bench.py times: x to 1e-9 and to 1e-7 of the distance moved, S6 of the state reached to 1e-8
    (the oracle needs about half a minute with all host threads)."""
    cfg = I.CONFIGS["C4"]
    g = cfg.grid
    x0, B0, dt = I.make(cfg)
    sim = make_sim(mr, g, x0, B0)
    sim.step(20, dt)
    assert sim.step_variant == "sym_tmem_f64"
    x20 = sim.get_fields(x=True, host=True)["x"].numpy()
    d = sim.diagnostics()
    del sim
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 20)
    moved = np.abs(ref - x0).max()
    assert moved > 0
    assert nrel(x20, ref) < TOL_100
    assert np.abs(x20 - ref).max() < 1e-7 * moved
    o = mro.diagnostics(g.n, g.lo, g.hi, ref, B0)
    for k in ("energy", "max_jxb", "xi", "min_det"):
        assert d[k] == pytest.approx(o[k], rel=1e-8), k


def test_context_on_a_side_stream_hands_its_results_to_the_callers_stream(mr):
    """A context bound to a stream other than the caller's current one: mr_get_fields, mr_get_xi and mr_rhs are asynchronous on
    the context's stream, so the binding makes the caller's stream wait for them; the tensors are used at once on the
    current stream (no synchronisation in between) and must equal those of a context on the current stream."""
    cfg = I.scaled(I.CONFIGS["C3"], (128, 128, 128))
    g = cfg.grid
    x0, B0, dt = I.make(cfg)
    td = torch.float64
    side = torch.cuda.Stream()
    want = make_sim(mr, g, x0, B0)
    want.step(3, dt)
    got = mr.Relaxation(g.n, g.lo, g.hi, stream=side)
    got.set_B0(dev(B0, td))
    if not np.array_equal(x0, I.reference_grid(g)):
        got.set_x(dev(x0, td))
    got.step(3, dt)
    assert got.stream == side and torch.cuda.current_stream() != side
    for op in ("mimetic", "direct"):
        a = got.get_xi().clone()
        b = got.rhs(op).clone()
        f = {k: v.clone() for k, v in got.get_fields(op, x=True, B=True, J=True).items()}
        assert torch.equal(a, want.get_xi())
        assert torch.equal(b, want.rhs(op))
        w = want.get_fields(op, x=True, B=True, J=True)
        for k in ("x", "B", "J"):
            assert torch.equal(f[k], w[k]), (op, k)


def test_fp64_peak_probe_is_plausible(mr):
    """mr_measure_fp64_peak (the roofline denominator of bench.py --operator direct): a DFMA-chain kernel on a B200 delivers
    between half and all of 148 SMs x 64 lanes x 2 FLOP x 1.965 GHz = 37.2 TFLOP/s."""
    tf = mr.measure_fp64_peak(0.02)
    assert 18.0 < tf < 38.0, tf
    with pytest.raises(mr.MrError):
        mr.measure_fp64_peak(0.0)


def test_fp32_context_accepts_the_fp32_rounding_of_the_reference_grid(mr):
    """mr_set_x on an fp32 context: boundary nodes given as float32(X) are on the reference grid (|X|/h is large
    on config 5: 4 / (8/511)), one really displaced boundary node is still refused."""
    g = I.Grid((64, 64, 64), (-4.0, -4.0, -4.0), (4.0, 4.0, 4.0))
    X = I.reference_grid(g)
    B0 = I.twist_field(g, (I.Twist(1.0, 1.0, 0.0, 0.0),))
    sim = mr.Relaxation(g.n, g.lo, g.hi, dtype="f32")
    sim.set_B0(dev(B0, torch.float32))
    sim.set_x(dev(X, torch.float32))
    sim.step(2, 0.25 * I.stable_dt(B0, g))
    bad = X.copy()
    bad[0, 0, 5, 5] += 1e-3 * g.h[0]
    with pytest.raises(mr.MrError):
        sim.set_x(dev(bad, torch.float32))


@pytest.mark.parametrize("variant", ["auto", "generic"])
def test_fp32_direct_operator_within_1e5_of_fp64(mr, variant):
    """The direct-derivative operator in fp32 (streaming kernel under "auto", global-memory kernel under "generic")
    against the fp64 GPU run of the same kernel and the fp64 oracle."""
    cfg = I.scaled(I.CONFIGS["C5"], (64, 64, 64))
    g = cfg.grid
    x0, B0, dt = I.make(cfg)
    s64 = make_sim(mr, g, x0, B0, "f64", variant)
    s32 = make_sim(mr, g, x0, B0, "f32", variant)
    s64.step(50, dt, "direct")
    s32.step(50, dt, "direct")
    assert s64.step_variant == ("direct_tma_f64" if variant == "auto" else "generic_direct")
    x64 = s64.get_fields(x=True)["x"].cpu().numpy()
    assert float((s32.get_xi().double() - s64.get_xi()).abs().max()) / float(np.abs(x0).max()) < TOL_F32
    ref = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 50, op=mro.DIRECT)
    assert nrel(x64, ref) < TOL_100


def test_steps_and_diagnostics_are_deterministic(mr):
    """Fixed-order reductions and no atomics on the data path: two runs from the same state are bit-identical, for
    the positions and for the four diagnostics (both operators)."""
    g, x0, B0, dt = case("wide")
    outs = []
    for _ in range(2):
        sim = make_sim(mr, g, x0, B0)
        sim.step(7, dt)
        sim.step(3, dt, "direct")
        d = sim.diagnostics()
        outs.append((sim.get_fields(x=True)["x"].cpu().numpy(), d))
    assert np.array_equal(outs[0][0], outs[1][0])
    for k in ("energy", "max_jxb", "xi", "min_det"):
        assert outs[0][1][k] == outs[1][1][k], k
