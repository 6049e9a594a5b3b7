"""Helpers shared by the GPU parity tests: tolerances, the seeded parity cases, context construction."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import mro  # noqa: E402  (test infrastructure)
from paper_1405_0942_b200 import inputs as I  # noqa: E402

TOL_STEP = 1e-12
TOL_100 = 1e-9
TOL_F32 = 1e-5


def nrel(a, b):
    """norm-wise relative error of a field (Q19)"""
    return float(np.abs(np.asarray(a) - np.asarray(b)).max() / max(np.abs(b).max(), 1e-300))


def dev(a, dtype=torch.float64):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda", dtype=dtype)


def make_sim(mr, g, x0, B0, dtype="f64", variant=None, bc=("line_tied",) * 3):
    """A context holding (x0, B0).  A context starts at x = X, so an undisplaced start needs no mr_set_x; an fp32 context
    takes the DISPLACEMENT (formed in fp64, then rounded): positions would lose eps |X| per node at the ABI (Q15)."""
    td = torch.float64 if dtype == "f64" else torch.float32
    sim = mr.Relaxation(g.n, g.lo, g.hi, dtype=dtype, bc=bc)
    if variant:
        sim.set_variant(variant)
    sim.set_B0(dev(B0, td))
    X = I.reference_grid(g)
    if not np.array_equal(x0, X):
        if dtype == "f64":
            sim.set_x(dev(x0, td))
        else:
            sim.set_xi(dev(np.asarray(x0) - X, td))
    return sim


def fields_np(sim, op):
    f = sim.get_fields(op, x=True, B=True, J=True)
    return {k: v.double().cpu().numpy() for k, v in f.items()}


def case(name):
    """(grid, x0, B0, dt) for the parity cases: sizes the oracle finishes in seconds that still span several
    tiles with a ragged tail."""
    if name == "C1":
        cfg = I.CONFIGS["C1"]
        x0, B0, dt = I.make(cfg)
        return cfg.grid, x0, B0, dt
    if name == "C1_rough":      # C1 field on a non-smoothly distorted grid
        cfg = I.CONFIGS["C1"]
        _, B0, dt = I.make(cfg)
        return cfg.grid, I.rough_displacement(cfg.grid, 0.2, seed=5), B0, dt
    if name == "ragged":        # odd sizes: row padding, partial tiles in every direction
        g = I.Grid((37, 21, 13), (-4.0, -4.0, -8.0), (4.0, 4.0, 8.0))
        B0 = I.twist_field(g, (I.Twist(1.0, 0.3, -0.2, 0.4), I.Twist(-0.7, -1.0, 0.5, -3.0)))
        return g, I.displaced_grid(g, 0.3, seed=7), B0, 0.5 * I.stable_dt(B0, g)
    if name == "minimal":       # the smallest legal grid
        g = I.Grid((5, 5, 5), (-1.0, -1.0, -1.0), (1.0, 1.0, 1.0))
        B0 = I.twist_field(g, (I.Twist(0.5, 0.0, 0.0, 0.0, a=1.0, l=1.0),))
        return g, I.displaced_grid(g, 0.2, seed=3), B0, 0.25 * I.stable_dt(B0, g)
    if name == "wide":          # several tiles in x and y, few planes
        g = I.Grid((130, 70, 9), (-4.0, -4.0, -2.0), (4.0, 4.0, 2.0))
        B0 = I.twist_field(g, (I.Twist(1.0, 1.0, 0.0, 0.0), I.Twist(-1.0, -1.0, 0.0, 0.5)))
        return g, I.displaced_grid(g, 0.3, seed=9), B0, 0.5 * I.stable_dt(B0, g)
    if name == "tail1":         # nz = 21: the z-chunking leaves a last chunk of ONE plane; one row in the last y tile
        g = I.Grid((17, 17, 21), (-4.0, -4.0, -10.0), (4.0, 4.0, 10.0))
        B0 = I.isohelix_B0(g, np.pi / 4)
        return g, I.displaced_grid(g, 0.25, seed=13), B0, 0.5 * I.stable_dt(B0, g)
    if name == "pow2p1":        # 2^m + 1 nodes in x and y (the paper's grids): the step tiling leaves the line-tied faces i = nx-1
                                # and j = 0 to the halo ring of the tiles (Tiling, mr_stream_common.cuh)
        g = I.Grid((33, 33, 11), (-4.0, -4.0, -5.0), (4.0, 4.0, 5.0))
        B0 = I.isohelix_B0(g, np.pi / 2)
        return g, I.displaced_grid(g, 0.25, seed=21), B0, 0.5 * I.stable_dt(B0, g)
    if name == "pow2p1_wide":   # ... with nx - 1 = 64 (the fp32 kernel's tile width) and several tiles in x
        g = I.Grid((129, 17, 9), (-8.0, -2.0, -2.0), (8.0, 2.0, 2.0))
        B0 = I.twist_field(g, (I.Twist(1.0, 2.0, 0.0, 0.0), I.Twist(-1.0, -3.0, 0.5, 0.5)))
        return g, I.displaced_grid(g, 0.3, seed=23), B0, 0.5 * I.stable_dt(B0, g)
    if name == "C2_small":      # config 2 field at a quarter of the resolution
        cfg = I.scaled(I.CONFIGS["C2"], (32, 32, 96))
        x0, B0, dt = I.make(cfg)
        return cfg.grid, x0, B0, dt
    if name == "C3_small":      # config 3 (reading D) at 48^3
        cfg = I.scaled(I.CONFIGS["C3"], (48, 48, 48))
        x0, B0, dt = I.make(cfg)
        return cfg.grid, x0, B0, dt
    raise KeyError(name)


CASES = ["C1", "C1_rough", "ragged", "minimal", "wide", "tail1", "pow2p1", "pow2p1_wide", "C2_small", "C3_small"]


def opcode(op):
    return mro.MIMETIC if op == "mimetic" else mro.DIRECT
