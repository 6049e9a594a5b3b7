"""Pins of the CPU oracle (oracle/mro.c) against what the paper and the mathematics fix (CPU only).

Each test names the oracle part (O1..O7) it pins and the passage behind it.  None of the
expected values comes from the oracle itself or from the CUDA path: they are closed forms, library
routines (numpy.gradient, numpy.linalg, sympy), independent numpy re-codings written here, or the values
in tests/golden/ (each with its citation).
"""
import os

import numpy as np
import pytest

from oracle import mro
from paper_1405_0942_b200 import inputs as I
from conftest import read_golden

AX = {0: 3, 1: 2, 2: 1}  # logical axis a -> numpy axis of a (3,nz,ny,nx) array


def grid(n, lo=(-1.0, -1.0, -1.0), hi=(1.0, 1.0, 1.0)):
    return I.Grid(tuple(n), tuple(lo), tuple(hi))


def interior(a):
    return a[..., 1:-1, 1:-1, 1:-1]


def relerr(a, b):
    return np.abs(a - b).max() / max(np.abs(b).max(), 1e-300)


def quad_map(g, amp=0.05, seed=1):
    """x_c = X_c + amp * (quadratic polynomial in X); returns x and the analytic Jacobian F[c,a]."""
    rng = np.random.default_rng(seed)
    X = I.reference_grid(g)
    lin = rng.normal(size=(3, 3)) * amp
    quad = rng.normal(size=(3, 3, 3)) * amp
    quad = 0.5 * (quad + quad.transpose(0, 2, 1))
    x = X.copy()
    F = np.zeros((3, 3) + X.shape[1:])
    for c in range(3):
        F[c, c] += 1.0
        for a in range(3):
            x[c] += lin[c, a] * X[a]
            F[c, a] += lin[c, a]
            for b in range(3):
                x[c] += quad[c, a, b] * X[a] * X[b]
                F[c, a] += 2.0 * quad[c, a, b] * X[b]
    return x, F, (lin, quad)


# ------------------------------------------------------------------ O1-O3: Jacobian, determinant, push-forward

def test_identity_map_gives_B0():
    """x = X  =>  F = I, Delta = 1, B = B0 (north_star pin "B = B0 when x = X"; Eq. 2.1)."""
    g = grid((9, 8, 11), (-4, -4, -8), (4, 4, 8))
    X = I.reference_grid(g)
    B0 = I.twist_field(g, (I.Twist(1.0, 0.3, -0.2, 0.5),))
    B, det = mro.push_forward(g.n, g.lo, g.hi, X, B0)
    assert np.abs(det - 1.0).max() < 1e-13
    assert np.abs(B - B0).max() < 1e-13


def test_reference_grid_matches_inputs():
    g = grid((7, 6, 5), (-4, -3, -2), (1, 2, 3))
    assert np.array_equal(mro.reference_grid(g.n, g.lo, g.hi), I.reference_grid(g))


def test_jacobian_equals_numpy_gradient_edge_order_2():
    """O1 (reading Q3) is exactly numpy.gradient(..., edge_order=2): central inside, 3-point one-sided at faces."""
    g = grid((7, 9, 8), (-1, -2, -3), (1.5, 2, 4))
    rng = np.random.default_rng(3)
    x = rng.normal(size=g.shape)
    F, det = mro.jacobian(g.n, g.lo, g.hi, x, strict=False)
    for c in range(3):
        for a in range(3):
            ref = np.gradient(x[c], g.h[a], axis=AX[a] - 1, edge_order=2)
            assert np.abs(F[c, a] - ref).max() < 1e-12 * max(1.0, np.abs(ref).max())
    Fm = np.moveaxis(F, (0, 1), (-2, -1))
    assert relerr(det, np.linalg.det(Fm)) < 1e-12


def test_affine_map_exact():
    """x = A X + b  =>  F = A and B = A B0 / det A on ALL nodes (central and one-sided differences are exact)."""
    g = grid((6, 7, 8))
    A = np.array([[1.1, 0.2, -0.1], [0.05, 0.9, 0.3], [-0.2, 0.1, 1.2]])
    b = np.array([0.3, -0.4, 0.5])
    X = I.reference_grid(g)
    x = np.einsum("ca,a...->c...", A, X) + b[:, None, None, None]
    rng = np.random.default_rng(5)
    B0 = rng.normal(size=g.shape)
    F, det = mro.jacobian(g.n, g.lo, g.hi, x)
    assert np.abs(F - A[:, :, None, None, None]).max() < 1e-13
    assert np.abs(det - np.linalg.det(A)).max() < 1e-13
    B, _ = mro.push_forward(g.n, g.lo, g.hi, x, B0)
    assert np.abs(B - np.einsum("ca,a...->c...", A, B0) / np.linalg.det(A)).max() < 1e-12


def test_quadratic_map_exact_on_all_nodes_including_faces():
    """Second-order differences (central AND the one-sided face stencil) are exact for quadratic maps."""
    g = grid((7, 8, 9), (-1, -1, -1), (1, 1.5, 2))
    x, Fa, _ = quad_map(g)
    rng = np.random.default_rng(7)
    B0 = rng.normal(size=g.shape)
    F, det = mro.jacobian(g.n, g.lo, g.hi, x)
    assert np.abs(F - Fa).max() < 5e-14
    deta = np.linalg.det(np.moveaxis(Fa, (0, 1), (-2, -1)))
    assert np.abs(det - deta).max() < 1e-13
    B, _ = mro.push_forward(g.n, g.lo, g.hi, x, B0)
    assert np.abs(B - np.einsum("ca...,a...->c...", Fa, B0) / deta).max() < 1e-12


def test_flux_through_each_cell_face_is_conserved():
    """B . (F_a x F_b) = B0_c at every node (flux through the image of each surface element)."""
    g = grid((8, 9, 10), (-4, -4, -8), (4, 4, 8))
    x = I.rough_displacement(g, 0.3, seed=11)
    B0 = I.twist_field(g, (I.Twist(1.0, 0.0, 0.0, 0.0),))
    F, det = mro.jacobian(g.n, g.lo, g.hi, x)
    B, _ = mro.push_forward(g.n, g.lo, g.hi, x, B0)
    for c, (a, b) in enumerate([(1, 2), (2, 0), (0, 1)]):
        area = np.cross(F[:, a], F[:, b], axis=0)
        flux = (B * area).sum(axis=0)
        assert np.abs(flux - B0[c]).max() < 1e-12


def test_line_tied_faces_keep_normal_field():
    """Boundary nodes fixed => B.n = B0.n on every face node, however distorted the interior."""
    g = grid((8, 9, 10), (-4, -4, -8), (4, 4, 8))
    x = I.rough_displacement(g, 0.3, seed=12)
    B0 = I.twist_field(g, (I.Twist(1.0, 0.5, 0.0, 1.0),))
    B, _ = mro.push_forward(g.n, g.lo, g.hi, x, B0)
    for a in range(3):
        for side in (0, -1):
            sl = [slice(None)] * 4
            sl[AX[a]] = side
            sl[0] = a
            assert np.abs(B[tuple(sl)] - B0[tuple(sl)]).max() < 1e-12


def test_isohelix_closed_form_pair_second_order():
    """Eq. 3.1 is the pull-back of B0 z^ under Eq. 3.3: with x = x_relax the pushed-forward
    field is z^ and Delta = 1 up to the O(h^2) error of the differences."""
    phi = np.pi / 4
    errs, derr = [], []
    for n in (17, 33):
        g = grid((n, n, n), (-4, -4, -10), (4, 4, 10))
        B, det = mro.push_forward(g.n, g.lo, g.hi, I.isohelix_x_relax(g, phi), I.isohelix_B0(g, phi))
        ez = np.zeros_like(B)
        ez[2] = 1.0
        errs.append(np.abs(B - ez).max())
        derr.append(np.abs(det - 1.0).max())
    assert errs[0] < 0.08 and errs[1] < 0.025
    assert 3.0 < errs[0] / errs[1] < 5.0          # second order
    assert derr[1] < derr[0] / 2.5


def test_isohelix_side_boundary_normal_component(golden_dir):
    """the normal component at the side boundaries is 'of the order of 4.1e-5' (input generator)."""
    gold = read_golden(os.path.join(golden_dir, "paper_values.txt"))["isohelix_side_normal"]
    g = grid((65, 65, 161), (-4, -4, -10), (4, 4, 10))
    vals = []
    for phi in (np.pi / 4, np.pi / 2, np.pi):
        B0 = I.isohelix_B0(g, phi)
        vals.append(max(np.abs(B0[0, :, :, 0]).max(), np.abs(B0[0, :, :, -1]).max()))
    assert vals[0] / 3 < gold < vals[-1] * 3
    assert vals[0] == pytest.approx(8.73e-5 * np.pi / 4, rel=0.02)   # analytic maximum (Q20)


# ------------------------------------------------------------------ O4m: nearest-neighbour mimetic curl

def shift(f, a, s):
    """value at index+s along logical axis a, restricted to interior nodes"""
    sl = [slice(None), slice(1, -1), slice(1, -1), slice(1, -1)]
    n = f.shape[AX[a]]
    sl[AX[a]] = slice(1 + s, n - 1 + s)
    return f[tuple(sl)]


def curl_short_form(x, B):
    """Identity I1: J = dF c / det(dF), c_p = eps_pqr d_qB . d_rx with un-normalised differences."""
    dx = [shift(x, a, 1) - shift(x, a, -1) for a in range(3)]
    dB = [shift(B, a, 1) - shift(B, a, -1) for a in range(3)]
    c = [(dB[q] * dx[r]).sum(0) - (dB[r] * dx[q]).sum(0) for (q, r) in [(1, 2), (2, 0), (0, 1)]]
    dF = np.stack(dx, 1)
    det = np.linalg.det(np.moveaxis(dF, (0, 1), (-2, -1)))
    return np.einsum("ca...,a...->c...", dF, np.stack(c, 0)) / det


def curl_chain_rule(x, B, h):
    """Identity I2: central differences of nodal B in X, chain rule with F^-1 (numpy.linalg.inv)."""
    F = np.stack([(shift(x, a, 1) - shift(x, a, -1)) / (2 * h[a]) for a in range(3)], 1)
    G = np.stack([(shift(B, a, 1) - shift(B, a, -1)) / (2 * h[a]) for a in range(3)], 1)
    Fi = np.linalg.inv(np.moveaxis(F, (0, 1), (-2, -1)))
    dBdx = np.einsum("ca...,...am->cm...", G, Fi)
    return np.stack([dBdx[2, 1] - dBdx[1, 2], dBdx[0, 2] - dBdx[2, 0], dBdx[1, 0] - dBdx[0, 1]], 0)


def test_uniform_field_has_zero_curl_on_rough_grid():
    """north_star pin: zero curl for a uniform field on arbitrarily distorted grids."""
    g = grid((11, 12, 13))
    x = I.rough_displacement(g, 0.3, seed=21)
    B = np.empty(g.shape)
    B[0], B[1], B[2] = 0.3, -1.2, 0.7
    J = mro.curl_mimetic(g.n, x, B)
    assert np.abs(J).max() < 1e-12


def test_linear_field_curl_exact_on_rough_grid():
    """B = G x + c sampled at the distorted nodes => J = axial vector of G - G^T exactly (Stokes on flat loops
    plus the vector area; distinguishes reading Q2 'vector sum' from the scalar sum of triangle areas)."""
    g = grid((10, 11, 12))
    x = I.rough_displacement(g, 0.3, seed=22)
    rng = np.random.default_rng(23)
    G = rng.normal(size=(3, 3))
    c = rng.normal(size=3)
    B = np.einsum("cm,m...->c...", G, x) + c[:, None, None, None]
    J = mro.curl_mimetic(g.n, x, B)
    want = np.array([G[2, 1] - G[1, 2], G[0, 2] - G[2, 0], G[1, 0] - G[0, 1]])
    assert np.abs(interior(J) - want[:, None, None, None]).max() < 2e-12
    # boundary nodes carry J = 0 (reading Q8)
    Jb = J.copy()
    interior(Jb)[...] = 0.0
    assert np.abs(Jb).max() == 0.0


def test_abc_on_undistorted_grid_is_discretely_beltrami():
    """ABC field, x = X, equal spacings: J = (sin(k h)/h) B exactly (central differences of single Fourier modes)
    hence J x B = 0 -- the discrete statement of 'a Beltrami/ABC field stays force-free' (north_star)."""
    g = grid((16, 16, 16))
    X = I.reference_grid(g)
    B = I.abc_field(X)
    J = mro.curl_mimetic(g.n, X, B)
    h = g.h[0]
    assert np.abs(interior(J) - np.sin(np.pi * h) / h * interior(B)).max() < 1e-12
    # and the full pipeline: velocity is zero, the grid does not move
    _, _, u, _ = mro.fields(g.n, g.lo, g.hi, X, B)
    assert np.abs(u).max() < 1e-12
    x1 = mro.step(g.n, g.lo, g.hi, X, B, 1e-3, 5)
    assert np.abs(x1 - X).max() < 1e-13


def test_literal_equals_short_form_equals_chain_rule():
    """Three independent codings of the mimetic curl agree: Eqs. 2.3-2.7 literally (C), I1 and I2 (numpy here)."""
    g = grid((9, 10, 11), (-1, -1, -1), (1, 1.2, 1.5))
    x = I.rough_displacement(g, 0.25, seed=31)
    rng = np.random.default_rng(32)
    B = rng.normal(size=g.shape)
    J = interior(mro.curl_mimetic(g.n, x, B))
    scale = np.abs(J).max()
    assert np.abs(J - curl_short_form(x, B)).max() < 1e-12 * scale
    assert np.abs(J - curl_chain_rule(x, B, g.h)).max() < 1e-12 * scale


def test_mimetic_second_order_on_smoothly_distorted_grid():
    """Nodal B = ABC(x0) on the config-3 displaced grid: J -> pi B at second order."""
    errs = []
    for n in (16, 32):
        g = grid((n, n, n))
        x0 = I.displaced_grid(g, 0.3)
        B = I.abc_field(x0)
        J = mro.curl_mimetic(g.n, x0, B)
        errs.append(np.abs(interior(J) - np.pi * interior(B)).max() / (np.pi * np.abs(B).max()))
    assert errs[0] < 0.05
    assert 3.0 < errs[0] / errs[1] < 5.0


# ------------------------------------------------------------------ O4d: direct-derivative ("classical") curl

def test_direct_equals_mimetic_on_undistorted_grid():
    """north_star pin: mimetic and direct operators agree on undistorted grids (any nodal B0)."""
    g = grid((9, 8, 10), (-1, -2, -1), (1, 2, 2))
    X = I.reference_grid(g)
    rng = np.random.default_rng(41)
    B0 = rng.normal(size=g.shape)
    Jm = mro.curl_mimetic(g.n, X, B0)
    Jd = mro.curl_direct(g.n, g.lo, g.hi, X, B0)
    assert np.abs(Jm - Jd).max() < 1e-12 * np.abs(Jm).max()


def test_direct_exact_for_quadratic_map_and_field_sympy():
    """Quadratic map and quadratic B0: all differences in O4d are exact, so J equals the analytic curl of
    F B0 / Delta (computed symbolically with sympy).  The mimetic operator is only O(h^2) here."""
    import sympy as sp          # a hard requirement: without it O4d would silently lose its only analytic pin
    g = grid((7, 8, 9), (-1, -1, -1), (1, 1.5, 2))
    x, _, (lin, quad) = quad_map(g, amp=0.05, seed=43)
    rng = np.random.default_rng(44)
    b_c = rng.normal(size=3)
    b_l = rng.normal(size=(3, 3))
    b_q = rng.normal(size=(3, 3, 3))
    Xs = sp.symbols("X0 X1 X2")
    xs = [Xs[c] + sum(float(lin[c, a]) * Xs[a] for a in range(3))
          + sum(float(quad[c, a, b]) * Xs[a] * Xs[b] for a in range(3) for b in range(3)) for c in range(3)]
    B0s = [float(b_c[c]) + sum(float(b_l[c, a]) * Xs[a] for a in range(3))
           + sum(float(b_q[c, a, b]) * Xs[a] * Xs[b] for a in range(3) for b in range(3)) for c in range(3)]
    Fs = sp.Matrix(3, 3, lambda c, a: sp.diff(xs[c], Xs[a]))
    Bs = (Fs * sp.Matrix(B0s)) / Fs.det()
    Fi = Fs.inv()
    dBdx = sp.Matrix(3, 3, lambda c, m: sum(sp.diff(Bs[c], Xs[a]) * Fi[a, m] for a in range(3)))
    Js = [dBdx[2, 1] - dBdx[1, 2], dBdx[0, 2] - dBdx[2, 0], dBdx[1, 0] - dBdx[0, 1]]
    f = sp.lambdify(Xs, Js, "numpy")
    X = I.reference_grid(g)
    B0 = np.stack([np.broadcast_to(v, X[0].shape) for v in sp.lambdify(Xs, B0s, "numpy")(X[0], X[1], X[2])])
    want = np.stack([np.broadcast_to(v, X[0].shape) for v in f(X[0], X[1], X[2])])
    Jd = mro.curl_direct(g.n, g.lo, g.hi, x, np.ascontiguousarray(B0))
    assert np.abs(interior(Jd) - interior(want)).max() < 1e-11 * np.abs(want).max()
    # the mimetic result differs at O(h^2): the two operators are genuinely different codes
    B, _ = mro.push_forward(g.n, g.lo, g.hi, x, np.ascontiguousarray(B0))
    Jm = mro.curl_mimetic(g.n, x, B)
    assert np.abs(interior(Jm) - interior(want)).max() > 1e-5 * np.abs(want).max()


def _reading_P_B0(g, x0):
    """Config 3, reading P: B0 := Delta_h F_h^-1 ABC(x0) per node, so that the pushed-forward nodal field is ABC(x0)."""
    F, det = mro.jacobian(g.n, g.lo, g.hi, x0)
    Fi = np.linalg.inv(np.moveaxis(F, (0, 1), (-2, -1)))           # [..., a, c]
    Bt = I.abc_field(x0)
    return np.ascontiguousarray(np.einsum("...ac,c...->a...", Fi, Bt) * det)


def test_both_operators_second_order_on_config3_reading_P():
    errs = {0: [], 1: []}
    for n in (32, 64):
        g = grid((n, n, n))
        x0 = I.displaced_grid(g, 0.3)
        B0 = _reading_P_B0(g, x0)
        for op in (0, 1):
            B, J, _, _ = mro.fields(g.n, g.lo, g.hi, x0, B0, op=op)
            assert np.abs(B - I.abc_field(x0)).max() < 1e-12
            errs[op].append(np.abs(interior(J) - np.pi * interior(B)).max() / (np.pi * np.abs(B).max()))
    for op in (0, 1):
        assert errs[op][0] < 0.03
        assert 3.0 < errs[op][0] / errs[op][1] < 5.0
    assert errs[0][1] < errs[1][1]           # the mimetic operator is the more accurate one (paper's claim, :260)


# ------------------------------------------------------------------ O5-O6: velocity and update

def test_velocity_is_gamma_J_cross_B_and_zero_on_boundary():
    cfg = I.CONFIGS["C1"]
    g = cfg.grid
    x = I.rough_displacement(g, 0.1, seed=51)
    _, B0, _ = I.make(cfg)
    B, J, u, _ = mro.fields(g.n, g.lo, g.hi, x, B0, gamma=1.7)
    assert np.abs(u - 1.7 * np.cross(J, B, axis=0)).max() < 1e-13
    ub = u.copy()
    interior(ub)[...] = 0
    assert np.abs(ub).max() == 0.0
    x1 = mro.step(g.n, g.lo, g.hi, x, B0, 0.01, 1, gamma=1.7)
    assert np.abs(x1 - (x + 0.01 * u)).max() < 1e-14


def test_c1_fourfold_rotation_symmetry_is_preserved():
    """C1 is invariant under (x,y) -> (-y,x) (nx = ny, square domain): a wrong sign or a swapped index in any
    of O1-O6 breaks this after a few steps."""
    cfg = I.CONFIGS["C1"]
    g = cfg.grid
    x0, B0, dt = I.make(cfg)
    x = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 30)
    assert np.abs(x - x0).max() > 1e-3       # it did move
    # rotate by +90 degrees about z: node (i,j) -> (n-1-j, i); vector (vx,vy) -> (-vy, vx)
    xr = np.empty_like(x)
    rot = lambda f: np.flip(np.swapaxes(f, -1, -2), axis=-1)   # f'(j', i') with i' = n-1-j, j' = i
    xr[0] = -rot(x[1])
    xr[1] = rot(x[0])
    xr[2] = rot(x[2])
    assert np.abs(xr - x).max() < 1e-13


# ------------------------------------------------------------------ O7: diagnostics

def test_energy_closed_forms():
    """x = X, B0 = z^  =>  E = Lx Ly Lz / 2 exactly (zeta are trapezoid weights; Eq. 3.13);
    affine map x = A X  =>  E = |A z^|^2 V / (2 det A); uniform field => xi = 0."""
    g = grid((6, 7, 9), (-4, -4, -8), (4, 4, 8))
    X = I.reference_grid(g)
    B0 = np.zeros(g.shape)
    B0[2] = 1.0
    d = mro.diagnostics(g.n, g.lo, g.hi, X, B0)
    assert d["energy"] == pytest.approx(0.5 * 8 * 8 * 16, rel=1e-14)
    assert d["min_det"] == pytest.approx(1.0, abs=1e-13)
    A = np.array([[1.1, 0.2, -0.1], [0.05, 0.9, 0.3], [-0.2, 0.1, 1.2]])
    x = np.einsum("ca,a...->c...", A, X)
    d = mro.diagnostics(g.n, g.lo, g.hi, x, B0)
    assert d["energy"] == pytest.approx(0.5 * (A[:, 2] ** 2).sum() * 8 * 8 * 16 / np.linalg.det(A), rel=1e-13)
    assert d["min_det"] == pytest.approx(np.linalg.det(A), rel=1e-13)
    assert d["xi"] < 1e-12 and d["max_jxb"] < 1e-12


def test_diagnostics_match_numpy_recomputation_from_fields():
    cfg = I.CONFIGS["C1"]
    g = cfg.grid
    x0, B0, dt = I.make(cfg)
    x = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 3)
    B, J, u, det = mro.fields(g.n, g.lo, g.hi, x, B0)
    w = [np.ones(g.n[a]) for a in range(3)]
    for a in range(3):
        w[a][0] = w[a][-1] = 0.5
    zeta = w[2][:, None, None] * w[1][None, :, None] * w[0][None, None, :]
    E = 0.5 * np.prod(g.h) * (zeta * (B ** 2).sum(0) * det).sum()
    f = np.sqrt((interior(u) ** 2).sum(0))
    d = mro.diagnostics(g.n, g.lo, g.hi, x, B0)
    assert d["energy"] == pytest.approx(E, rel=1e-13)
    assert d["max_jxb"] == pytest.approx(f.max(), rel=1e-13)
    assert d["xi"] == pytest.approx((f / (interior(B) ** 2).sum(0)).max(), rel=1e-13)
    assert d["min_det"] == det.min()


# ------------------------------------------------------------------ whole run

def test_c1_energy_decays_monotonically_and_matches_survey_probe(golden_dir):
    """Monotone energy decay under Eq. 1.5 on config C1, and the independent numpy
    prototype values quoted in SURVEY.md section 8(c)."""
    gold = read_golden(os.path.join(golden_dir, "c1_survey_probe.txt"))
    cfg = I.CONFIGS["C1"]
    g = cfg.grid
    x, B0, dt = I.make(cfg)
    d0 = mro.diagnostics(g.n, g.lo, g.hi, x, B0)
    assert d0["energy"] == pytest.approx(gold["E_0"], rel=2e-12)
    assert d0["max_jxb"] == pytest.approx(gold["max_jxb_0"], rel=2e-6)
    assert d0["xi"] == pytest.approx(gold["xi_0"], rel=2e-6)
    E = [d0["energy"]]
    for _ in range(10):
        x = mro.step(g.n, g.lo, g.hi, x, B0, dt, 10)
        E.append(mro.diagnostics(g.n, g.lo, g.hi, x, B0)["energy"])
    assert all(b < a for a, b in zip(E[:-1], E[1:]))
    d = mro.diagnostics(g.n, g.lo, g.hi, x, B0)
    assert d["energy"] == pytest.approx(gold["E_100"], rel=2e-12)
    assert d["xi"] == pytest.approx(gold["xi_100"], rel=5e-6)
    assert d["min_det"] == pytest.approx(gold["min_det_100"], abs=1e-4)
    assert d["energy"] > gold["E_background"]


def test_energy_decay_rate_is_minus_integral_of_lorentz_force_squared():
    """dE/dt = -gamma * int |J x B|^2 dV for u = gamma J x B (refs [6,27]): pins the sign AND the
    magnitude of u and of dt against the energy of Eq. 3.13 (discretisation error ~ a few per cent on C1@24x24x48)."""
    cfg = I.scaled(I.CONFIGS["C1"], (24, 24, 48))
    g = cfg.grid
    x0, B0, _ = I.make(cfg)
    dt = 1e-4
    for gamma in (1.0, 2.5):
        B, J, u, det = mro.fields(g.n, g.lo, g.hi, x0, B0, gamma=gamma)
        rate = -(np.prod(g.h)) * ((interior(u) ** 2).sum(0) * interior(det)).sum() / gamma
        E0 = mro.diagnostics(g.n, g.lo, g.hi, x0, B0)["energy"]
        E1 = mro.diagnostics(g.n, g.lo, g.hi, mro.step(g.n, g.lo, g.hi, x0, B0, dt, 1, gamma=gamma), B0)["energy"]
        assert (E1 - E0) / dt == pytest.approx(rate, rel=0.08)


def test_c2_initial_diagnostics_match_survey_probe(golden_dir):
    gold = read_golden(os.path.join(golden_dir, "c2_survey_probe.txt"))
    cfg = I.CONFIGS["C2"]
    g = cfg.grid
    x0, B0, dt = I.make(cfg)
    mro.set_threads(mro.max_threads())
    try:
        d = mro.diagnostics(g.n, g.lo, g.hi, x0, B0)
    finally:
        mro.set_threads(1)
    assert d["energy"] == pytest.approx(gold["E_0"], rel=2e-12)
    assert d["max_jxb"] == pytest.approx(gold["max_jxb_0"], rel=2e-6)
    assert dt == pytest.approx(2.61e-3, rel=5e-3)


def test_numeric_failure_is_reported():
    g = grid((6, 6, 6))
    x = I.reference_grid(g)
    x[0, 3, 3, 3] += 10.0            # folds the grid: det <= 0 somewhere
    B0 = np.ones(g.shape)
    with pytest.raises(mro.NumericError):
        mro.push_forward(g.n, g.lo, g.hi, x, B0)
