"""Pins of the oracle's SURVEY 8(f) parts (CPU only): the adaptive Cash-Karp integrator of section 2.4, periodic
boundaries (Eqs. 2.12-2.14), convexity (Eqs. 3.10-3.11), alpha*/eps* (Eqs. 3.5-3.7) and sigma_B, sigma_x (Eqs. 3.8-3.9).

Each pin is something other than the oracle's own formula: order conditions and exact quadrature of the Runge-Kutta
pair, the controller's stated rules on hand-made numbers, the paper's ghost-node equations fed to the (already pinned)
line-tied code on an extended grid, closed forms, hand-constructed concave cells, and independent numpy codings.
"""
import numpy as np
import pytest

from oracle import mro
from paper_1405_0942_b200 import inputs as I


# ---------------------------------------------------------------------------------------------- section 2.4: RK5(4)

def test_cash_karp_quadrature_is_exact_to_its_order():
    """y' = t^p as the autonomous system (t, y)' = (1, t^p): the fifth-order weights integrate t^p exactly for p <= 4,
    the embedded fourth-order ones for p <= 3 (and not beyond): pins both weight rows and the nodes c_s = sum_r a_sr."""
    dt = 0.7
    for p in range(0, 7):
        y5, y4, lam = mro.cash_karp_trial([0.0, 0.0], dt, lambda y, p=p: np.array([1.0, y[0] ** p]))
        exact = dt ** (p + 1) / (p + 1)
        assert y5[0] == pytest.approx(dt, rel=1e-15) and y4[0] == pytest.approx(dt, rel=1e-15)
        e5, e4 = abs(y5[1] - exact) / exact, abs(y4[1] - exact) / exact
        assert (e5 < 1e-14) == (p <= 4), (p, e5)
        assert (e4 < 1e-14) == (p <= 3), (p, e4)
        assert lam == pytest.approx(abs(y5[1] - y4[1]), rel=1e-12, abs=1e-17)


@pytest.mark.parametrize("name", ["riccati", "pendulum"])
def test_cash_karp_local_error_orders(name):
    """Nonlinear systems with closed-form / conserved solutions: halving dt divides the one-step error of the fifth-order
    solution by 2^6 and that of the embedded one by 2^5 (pins the coupling coefficients a_sr: a wrong one breaks the
    order conditions)."""
    if name == "riccati":          # y' = -y^2, y(0) = 1  ->  y = 1/(1+t)
        f = lambda y: -y * y
        y0 = np.array([1.0])
        exact = lambda t: np.array([1.0 / (1.0 + t)])
    else:                          # y'' = -sin y as a system, reference by a much finer integration with the same pair
        f = lambda y: np.array([y[1], -np.sin(y[0])])
        y0 = np.array([1.0, 0.3])

        def exact(t, n=200):
            y = y0.copy()
            for _ in range(n):
                y, _, _ = mro.cash_karp_trial(y, t / n, f)
            return y
    errs5, errs4 = [], []
    for dt in (0.1, 0.05, 0.025):
        y5, y4, _ = mro.cash_karp_trial(y0, dt, f)
        ex = exact(dt)
        errs5.append(np.abs(y5 - ex).max())
        errs4.append(np.abs(y4 - ex).max())
    assert 5.3 < np.log2(errs5[1] / errs5[2]) < 6.4, errs5         # local error O(dt^6)
    assert 4.1 < np.log2(errs4[1] / errs4[2]) < 5.4, errs4         # local error O(dt^5)
    assert errs5[2] < 0.2 * errs4[2]


def test_step_control_follows_the_paper():
    """reject iff Lambda > Lambda0 and retry with dt' = dt |Lambda0/Lambda|^0.2 (Eq. 2.11); accept
    otherwise; below Lambda0/2 the step grows by the same formula; in between it stays."""
    lam0 = 1e-6
    ok, dtn = mro.step_control(0.1, 32e-6, lam0)
    assert not ok and dtn == pytest.approx(0.1 * (1.0 / 32.0) ** 0.2, rel=1e-14) and dtn == pytest.approx(0.05, rel=1e-14)
    ok, dtn = mro.step_control(0.1, 0.75e-6, lam0)
    assert ok and dtn == 0.1
    ok, dtn = mro.step_control(0.1, lam0 / 32.0, lam0)
    assert ok and dtn == pytest.approx(0.2, rel=1e-14)
    ok, dtn = mro.step_control(0.1, lam0, lam0)                   # Lambda = Lambda0 is not "exceeds"
    assert ok and dtn == 0.1
    ok, dtn = mro.step_control(0.1, 0.0, lam0)                    # reading Q22: growth capped at 5x
    assert ok and dtn == pytest.approx(0.5)
    ok, dtn = mro.step_control(0.1, 1e-30, lam0)
    assert ok and dtn == pytest.approx(0.5)
    # reading Q22: just above Lambda0 the factor of Eq. 2.11 rounds to 1 (the value met on the IsoHelix run: the same trial
    # would repeat for ever); a retry is at most 0.9 dt
    ok, dtn = mro.step_control(0.3667726365104183, 1.0000000000000002e-08, 1e-8)
    assert not ok and dtn == 0.9 * 0.3667726365104183
    ok, dtn = mro.step_control(0.1, 1.2e-6, lam0)
    assert not ok and dtn == pytest.approx(0.09, rel=1e-14)          # 1.2^-0.2 = 0.964 > 0.9
    ok, dtn = mro.step_control(0.1, 2e-6, lam0)
    assert not ok and dtn == pytest.approx(0.1 * 0.5 ** 0.2, rel=1e-14)   # 0.871 < 0.9: Eq. 2.11 as printed


def test_a_trial_that_folds_the_grid_is_recomputed_with_half_the_step():
    """Reading Q26 (the paper only says the run "is stopped" after "a drop of the time step by several orders of magnitude",
    PAPER.md:333): a step far beyond the stability limit turns cells inside out in a stage; such a trial has no result, is
    rejected with Lambda = NaN and recomputed with dt/2 until a stage survives.  It leaves no trace in x: the run equals, bit
    for bit, one that starts with the first step length that did not fold."""
    cfg = I.CONFIGS["C1"]
    g = cfg.grid
    x0, B0, _ = I.make(cfg)
    x, t, dt_next, (acc, rej), trace = mro.step_adaptive(g.n, g.lo, g.hi, x0, B0, t_end=1.0, lam0=1e-7, dt=4.0)
    folded = np.isnan(trace[:, 2])
    nf = int(folded.sum())
    assert nf >= 2 and folded[:nf].all() and not folded[nf:].any()            # they come first, in a row
    assert np.array_equal(trace[:nf, 1], 1.0 * 0.5 ** np.arange(nf))          # 4.0 is clipped to t_end = 1, then halved
    assert not trace[:nf, 3].any() and np.all(trace[:nf, 0] == 0.0)
    assert trace[nf, 1] == 0.5 ** nf and t == 1.0 and acc + rej == len(trace) and rej >= nf
    x2, t2, dt2, (acc2, rej2), trace2 = mro.step_adaptive(g.n, g.lo, g.hi, x0, B0, t_end=1.0, lam0=1e-7, dt=0.5 ** nf)
    assert np.array_equal(x, x2) and dt2 == dt_next and acc2 == acc and rej2 == rej - nf
    assert np.array_equal(trace2, trace[nf:])


def test_forty_folded_trials_in_a_row_stop_the_run():
    """Reading Q26, the other half: a state that is folded already (one node pushed past its third neighbour) fails in the first
    stage whatever the step; after 40 halvings (2^-40 = 9e-13 of the first step: "several orders of magnitude") the run
    stops with the numeric return code, the state untouched."""
    cfg = I.CONFIGS["C1"]
    g = cfg.grid
    x0, B0, _ = I.make(cfg)
    xf = x0.copy()
    xf[0, 9, 5, 5] = x0[0, 9, 5, 8]                 # x_6 - x_4 ... fine, but x_7 - x_5 < 0: det(dx/dX) < 0 at node 6
    assert mro.diagnostics(g.n, g.lo, g.hi, xf, B0, strict=False)["min_det"] < 0
    with pytest.raises(mro.NumericError):
        mro.step_adaptive(g.n, g.lo, g.hi, xf, B0, t_end=1.0, lam0=1e-7, dt=0.125)
    x, t, dt_next, (acc, rej), trace = mro.step_adaptive(g.n, g.lo, g.hi, xf, B0, t_end=1.0, lam0=1e-7, dt=0.125, strict=False)
    assert (acc, rej) == (0, 40) and t == 0.0 and np.array_equal(x, xf)
    assert dt_next == 0.125 * 0.5 ** 40 and np.isnan(trace[:, 2]).all()
    assert np.array_equal(trace[:, 1], 0.125 * 0.5 ** np.arange(40))


def test_adaptive_relaxation_on_config1():
    """C1 with the adaptive integrator: the run ends exactly at t_end, rejected trials leave no trace in x, every
    accepted Lambda is within tolerance, the energy decays monotonically over the accepted steps,
    and the result agrees with forward Euler at a much smaller step."""
    cfg = I.CONFIGS["C1"]
    g = cfg.grid
    x0, B0, _ = I.make(cfg)
    lam0 = 1e-7
    x, t, dt_next, (acc, rej), trace = mro.step_adaptive(g.n, g.lo, g.hi, x0, B0, t_end=0.3, lam0=lam0, dt=0.2)
    assert t == 0.3 and acc >= 2 and rej >= 1 and len(trace) == acc + rej
    assert trace[0][3] == 0.0                                      # dt = 0.2 is beyond the stability limit: first trial rejected
    for (tt, h, lam, ok) in trace:
        assert (lam <= lam0) == bool(ok)
    assert np.sum(trace[trace[:, 3] == 1.0, 1]) == pytest.approx(0.3, rel=1e-13)
    # replay of the accepted steps only: identical state (a rejected trial changes nothing but dt)
    y = np.array(x0)
    E = [mro.diagnostics(g.n, g.lo, g.hi, y, B0)["energy"]]
    for (tt, h, lam, ok) in trace:
        if ok:
            y5, _, _ = mro.cash_karp_trial(y.ravel(), h, lambda v: mro.fields(g.n, g.lo, g.hi, v.reshape(g.shape), B0)[2].ravel())
            y = y5.reshape(g.shape)
            E.append(mro.diagnostics(g.n, g.lo, g.hi, y, B0)["energy"])
    assert np.abs(y - x).max() < 1e-13
    assert all(b < a for a, b in zip(E[:-1], E[1:]))
    xe = mro.step(g.n, g.lo, g.hi, x0, B0, 1e-4, 3000)
    assert np.abs(x - xe).max() < 2e-4 * np.abs(xe - x0).max()


# ---------------------------------------------------------------------------------------------- Eqs. 2.12-2.14

def _periodic_case(n=(9, 8, 10)):
    """x/y line-tied, z periodic; displacement and field periodic in z with the period n_z h_z."""
    g = I.Grid(n, (-1.0, -1.0, -1.0), (1.0, 1.0, 0.8))             # h_z = 0.2, period 2
    X = I.reference_grid(g)
    Pz = n[2] * g.h[2]
    ph = 2.0 * np.pi * (X[2] - g.lo[2]) / Pz
    bump = np.sin(0.5 * np.pi * (X[0] + 1.0)) * np.sin(0.5 * np.pi * (X[1] + 1.0))     # zero on the x/y faces
    x = X.copy()
    x[0] += 0.04 * bump * np.sin(ph)
    x[1] += 0.03 * bump * np.cos(2 * ph)
    x[2] += 0.05 * bump * np.sin(ph + 0.3)
    B0 = np.empty_like(X)
    B0[0] = 0.3 * np.sin(ph) + 0.1 * X[1]
    B0[1] = 0.2 * np.cos(ph) * (1.0 + 0.5 * X[0])
    B0[2] = 1.0 + 0.1 * np.sin(2 * ph) * X[0]
    return g, x, B0, Pz


@pytest.mark.parametrize("op", [mro.MIMETIC, mro.DIRECT])
def test_periodic_axis_equals_the_papers_ghost_nodes(op):
    """Eqs. 2.12-2.14 verbatim: extend the grid by two ghost planes on either side of z (positions copied from the other
    end and shifted by -/+ (L_z + dZ) in z, B(X,0) copied), hand the extended grid to the LINE-TIED code, and compare its
    B and J on the original planes with the periodic code."""
    g, x, B0, Pz = _periodic_case()
    nz = g.n[2]
    idx = np.arange(-2, nz + 2)
    wrap = idx % nz
    shift = np.where(idx < 0, -Pz, np.where(idx >= nz, Pz, 0.0))
    xe = x[:, wrap].copy()
    xe[2] += shift[:, None, None]
    Be = B0[:, wrap].copy()
    ge = I.Grid((g.n[0], g.n[1], nz + 4), (g.lo[0], g.lo[1], g.lo[2] - 2 * g.h[2]), (g.hi[0], g.hi[1], g.hi[2] + 2 * g.h[2]))
    Bx, Jx, ux, detx = mro.fields(ge.n, ge.lo, ge.hi, xe, Be, op=op)
    Bp, Jp, up, detp = mro.fields(g.n, g.lo, g.hi, x, B0, op=op, bc=(0, 0, 1))
    inner = slice(2, nz + 2)
    assert np.abs(Bp - Bx[:, inner]).max() < 1e-14
    assert np.abs(detp - detx[inner]).max() < 1e-14
    assert np.abs(Jp - Jx[:, inner]).max() < 1e-12
    assert np.abs(up - ux[:, inner]).max() < 1e-12
    assert np.abs(Jp[:, 0, 1:-1, 1:-1]).max() > 1e-3                # the end planes of a periodic axis are inner planes
    # Eq. 2.14: with these ghosts the field is periodic
    assert np.abs(Bx[:, 1] - Bx[:, nz + 1]).max() < 1e-14


def test_fully_periodic_abc_field_is_discretely_beltrami_everywhere():
    """ABC field of wavenumber pi on the periodic cube [-1, 1)^3: J = (sin(pi h)/h) B at EVERY node (closed form of
    central differences on Fourier modes) -- there is no boundary left -- and the energy is the plain sum."""
    n = 16
    h = 2.0 / n
    g = I.Grid((n, n, n), (-1.0,) * 3, (1.0 - h,) * 3)
    X = I.reference_grid(g)
    B0 = I.abc_field(X)
    bc = (1, 1, 1)
    for op in (mro.MIMETIC, mro.DIRECT):
        B, J, u, det = mro.fields(g.n, g.lo, g.hi, X, B0, op=op, bc=bc)
        assert np.abs(J - np.sin(np.pi * h) / h * B).max() < 1e-13
        assert np.abs(u).max() < 1e-13
    d = mro.diagnostics(g.n, g.lo, g.hi, X, B0, bc=bc)
    assert d["energy"] == pytest.approx(0.5 * (B0 ** 2).sum() * h ** 3, rel=1e-14)       # zeta = 1 everywhere
    assert d["energy"] == pytest.approx(0.5 * 3.0 * 8.0, rel=1e-12)                        # <|B|^2> = 3 over the period
    # a rigid shift of the whole periodic grid changes nothing
    x = X + np.array([0.3, -0.2, 0.1])[:, None, None, None]
    B2, J2, _, _ = mro.fields(g.n, g.lo, g.hi, x, B0, bc=bc)
    assert np.abs(B2 - B0).max() < 1e-14 and np.abs(J2 - np.sin(np.pi * h) / h * B0).max() < 1e-12


def test_periodic_steps_keep_a_uniform_field_at_rest_and_relax_a_twist():
    g, x, B0, Pz = _periodic_case()
    bc = (0, 0, 1)
    Bu = np.zeros_like(B0)
    Bu[2] = 1.0
    X = I.reference_grid(g)
    assert np.abs(mro.step(g.n, g.lo, g.hi, X, Bu, 1e-3, 5, bc=bc) - X).max() == 0.0
    E = [mro.diagnostics(g.n, g.lo, g.hi, x, B0, bc=bc)["energy"]]
    y = x
    for _ in range(5):
        y = mro.step(g.n, g.lo, g.hi, y, B0, 2e-3, 4, bc=bc)
        E.append(mro.diagnostics(g.n, g.lo, g.hi, y, B0, bc=bc)["energy"])
    assert all(b < a for a, b in zip(E[:-1], E[1:]))
    assert np.abs(y[:, 0] - x[:, 0]).max() > 0                      # the end plane of the periodic axis moves


# ---------------------------------------------------------------------------------------------- Eqs. 3.10-3.11

def test_convexity_of_hand_made_grids():
    g = I.Grid((7, 6, 5), (0.0, 0.0, 0.0), (6.0, 5.0, 4.0))        # h = 1
    X = I.reference_grid(g)
    kap, bad = mro.convexity(g.n, g.lo, g.hi, X)
    assert bad == 0 and (kap == 1).all()
    # a positive affine map keeps every trihedron's orientation, a reflection flips all of them
    A = np.array([[1.0, 0.3, 0.1], [-0.2, 0.9, 0.2], [0.1, 0.0, 1.1]])
    xa = np.einsum("ab,b...->a...", A, X)
    assert mro.convexity(g.n, g.lo, g.hi, xa)[1] == 0
    xr = X.copy()
    xr[0] *= -1.0
    kap, bad = mro.convexity(g.n, g.lo, g.hi, xr)
    assert bad == g.nodes and (kap == -1).all()
    # one interior node pushed 1.5 h past its +x neighbour: exactly that node and that neighbour see a flipped trihedron
    x = X.copy()
    i, j, k = 3, 2, 2
    x[0, k, j, i] += 1.5
    kap, bad = mro.convexity(g.n, g.lo, g.hi, x)
    want = np.ones_like(kap)
    want[k, j, i] = -1
    want[k, j, i + 1] = -1
    assert bad == 2 and np.array_equal(kap, want)
    # a node pushed diagonally out of the plane of its neighbours but inside its cell stays convex
    x = X.copy()
    x[:, k, j, i] += np.array([0.4, -0.3, 0.2])
    assert mro.convexity(g.n, g.lo, g.hi, x)[1] == 0


def test_convexity_with_a_periodic_axis_uses_the_shifted_ghosts():
    g, x, B0, Pz = _periodic_case()
    assert mro.convexity(g.n, g.lo, g.hi, x, bc=(0, 0, 1))[1] == 0
    # without the shift of Eqs. 2.12/2.13 the wrap-around trihedra would all be flipped; with it they are not
    X = I.reference_grid(g)
    kap, bad = mro.convexity(g.n, g.lo, g.hi, X, bc=(0, 0, 1))
    assert bad == 0


# ---------------------------------------------------------------------------------------------- Eqs. 3.5-3.9

def test_eps_star_closed_form_linear_twist():
    """B = z^ + tau(Z) (-Y, X, 0) with tau = c Z: curl B on the axis is 2 tau z^, so alpha* = 2 c Z there (central
    differences are exact on these bilinear components) and eps* = 2 c a_r (Eq. 3.7)."""
    g = I.Grid((9, 9, 13), (-2.0, -2.0, -3.0), (2.0, 2.0, 3.0))
    X = I.reference_grid(g)
    c, a_r = 0.07, np.sqrt(2.0)
    B0 = np.empty_like(X)
    B0[0] = -c * X[2] * X[1]
    B0[1] = c * X[2] * X[0]
    B0[2] = 1.0
    for op in (mro.MIMETIC, mro.DIRECT):
        al, eps = mro.eps_star(g.n, g.lo, g.hi, X, B0, 4, 4, a_r, op=op)
        Z = g.axes()[2]
        assert np.abs(al[1:-1] - 2 * c * Z[1:-1]).max() < 1e-14 and al[0] == 0.0 and al[-1] == 0.0
        assert eps == pytest.approx(2 * c * a_r, rel=1e-12)


def test_eps_star_equals_a_numpy_coding_and_vanishes_for_a_beltrami_field():
    cfg = I.CONFIGS["C1"]
    g = cfg.grid
    x0, B0, dt = I.make(cfg)
    x = mro.step(g.n, g.lo, g.hi, x0, B0, dt, 5)
    ic, jc, a_r = 7, 8, 1.3
    al, eps = mro.eps_star(g.n, g.lo, g.hi, x, B0, ic, jc, a_r)
    B, J, _, _ = mro.fields(g.n, g.lo, g.hi, x, B0)
    a2 = (J[:, :, jc, ic] * B[:, :, jc, ic]).sum(0) / (B[:, :, jc, ic] ** 2).sum(0)
    assert np.abs(al[1:-1] - a2[1:-1]).max() < 1e-15
    Z = g.axes()[2][1:-1]
    d = a2[1:-1, None] - a2[None, 1:-1]
    dist = np.abs(Z[:, None] - Z[None, :])
    np.fill_diagonal(dist, np.inf)
    assert eps == pytest.approx(a_r * (d / dist).max(), rel=1e-13)
    gb = I.Grid((17, 17, 17), (-1.0,) * 3, (1.0,) * 3)
    Xb = I.reference_grid(gb)
    al, eps = mro.eps_star(gb.n, gb.lo, gb.hi, Xb, I.abc_field(Xb), 8, 8, 1.0)
    h = gb.h[0]
    assert np.abs(al[1:-1] - np.sin(np.pi * h) / h).max() < 1e-12 and eps < 1e-11


def test_sigma_closed_forms_and_isohelix_pair():
    g = I.Grid((9, 9, 11), (-4.0, -4.0, -10.0), (4.0, 4.0, 10.0))
    X = I.reference_grid(g)
    B0 = I.isohelix_B0(g, np.pi / 4)
    off_x, off_B = np.array([0.3, -0.4, 1.2]), np.array([0.1, 0.2, -0.2])
    sx, sb = mro.sigma(g.n, g.lo, g.hi, X, B0, X - off_x[:, None, None, None], B0 + off_B[:, None, None, None])
    assert sx == pytest.approx(np.sqrt((off_x ** 2).sum()), rel=1e-13)            # Eq. 3.9 with a constant offset
    assert sb == pytest.approx(np.sqrt((off_B ** 2).sum()), rel=1e-13)            # Eq. 3.8 (B = B0 at x = X)
    # the exact relaxed state (Eqs. 3.2, 3.3): sigma_x = 0 and sigma_B = O(h^2)
    Bz = np.zeros_like(X)
    Bz[2] = 1.0
    vals = []
    for n in (17, 33):
        gg = I.Grid((n, n, n), (-4.0, -4.0, -10.0), (4.0, 4.0, 10.0))
        xr = I.isohelix_x_relax(gg, np.pi / 4)
        Bref = np.zeros(gg.shape)
        Bref[2] = 1.0
        sx, sb = mro.sigma(gg.n, gg.lo, gg.hi, xr, I.isohelix_B0(gg, np.pi / 4), xr, Bref, strict=False)
        assert sx == 0.0
        vals.append(sb)
    assert 3.0 < vals[0] / vals[1] < 5.0
    assert vals[0] < 2e-2


# ---------------------------------------------------------------------------------------------- Table 4.1 of the paper

def read_table_4_1(golden_dir):
    """rows of tests/golden/paper_table_4_1.txt: {(phi/pi, method, n): (xi, eps*, sigma_B, sigma_x)} as printed in the paper"""
    import os
    rows = {}
    with open(os.path.join(golden_dir, "paper_table_4_1.txt")) as f:
        for line in f:
            line = line.split("#", 1)[0].split()
            if line:
                rows[(float(line[0]), line[1], int(line[2]))] = tuple(float(v) for v in line[3:7])
    return rows


def isohelix_setup(n, phi):
    """IsoHelix configuration of section 3.1: n^3 nodes on the 8 x 8 x 20 cuboid, x(0) = X"""
    g = I.Grid((n, n, n), (-4.0, -4.0, -10.0), (4.0, 4.0, 10.0))
    Bref = np.zeros(g.shape)
    Bref[2] = 1.0                                                          # Eq. 3.2
    return g, I.isohelix_B0(g, phi), I.isohelix_x_relax(g, phi), Bref


def test_isohelix_relaxation_reproduces_table_4_1_mimetic_n17(golden_dir):
    """The paper's own numbers for this path (TABLE 4.1): the IsoHelix field with phi = pi/4 on 17^3 nodes,
    relaxed by the mimetic operator and the adaptive Cash-Karp integrator (section 2.4) until the independent measures have
    stabilised, ends at eps* = 1.0e-2, sigma_B = 1.3e-3, sigma_x = 9.6e-3 (two digits printed).  The whole chain enters:
    Jacobian, push-forward, the Stokes-loop curl, u = J x B, the line-tied faces, the integrator, and Eqs. 3.7-3.9.  A wrong
    sign, stencil or loop point does not converge to these values (the direct operator on the same grid ends at
    eps* = 0.3, sigma_B = 1.1e-2, sigma_x = 2.4e-2)."""
    xi_p, eps_p, sB_p, sx_p = read_table_4_1(golden_dir)[(0.25, "mimetic", 17)]
    g, B0, xr, Bref = isohelix_setup(17, np.pi / 4)
    x, t, dt, (acc, rej), _ = mro.step_adaptive(g.n, g.lo, g.hi, I.reference_grid(g), B0, t_end=256.0, lam0=1e-8, dt=1e-3,
                                               max_trials=20000)
    assert t == 256.0
    sx, sb = mro.sigma(g.n, g.lo, g.hi, x, B0, xr, Bref)
    _, eps = mro.eps_star(g.n, g.lo, g.hi, x, B0, 8, 8, np.sqrt(2.0))
    d = mro.diagnostics(g.n, g.lo, g.hi, x, B0)
    # two printed digits: half a unit of the last digit is 5 % at 1.0e-2; measured here 1.026e-2, 1.274e-3, 9.497e-3
    assert eps == pytest.approx(eps_p, rel=0.06), eps
    assert sb == pytest.approx(sB_p, rel=0.06), sb
    assert sx == pytest.approx(sx_p, rel=0.03), sx
    assert d["xi"] < 1e-4 and d["energy"] < 640.0005          # xi keeps falling; the free energy is gone
    assert mro.convexity(g.n, g.lo, g.hi, x)[1] == 0


def test_pontin09_relaxation_reproduces_table_4_2_mimetic_n17(golden_dir):
    """TABLE 4.2: the Pontin09 field (Eq. 3.4, phi_1,2 = +-pi/2) on 17^3 nodes relaxed by the mimetic operator
    ends at eps* = 1.1e-1.  The positions of its two twist regions are not printed; L_i = -+4 is the reading (Q25) under
    which the oracle (here, 1.146e-1 at t = 256) and the CUDA path (1.143e-1 at t = 512; 1.77e-2 against 1.8e-2 on 33^3) reproduce
    the table."""
    import os
    eps_p = None
    with open(os.path.join(golden_dir, "paper_table_4_2.txt")) as f:
        for line in f:
            line = line.split("#", 1)[0].split()
            if line and line[0] == "mimetic" and int(line[1]) == 17:
                eps_p = float(line[3])
    g = I.Grid((17, 17, 17), (-4.0, -4.0, -10.0), (4.0, 4.0, 10.0))
    B0 = I.pontin09_B0(g, (np.pi / 2, -np.pi / 2), (-4.0, 4.0))
    assert np.abs(B0[2] - 1.0).max() == 0.0 and B0[0, 8, 8, 8] == 0.0          # Eq. 3.4: B_z = B0, no twist field on the axis
    x, t, dt, counts, _ = mro.step_adaptive(g.n, g.lo, g.hi, I.reference_grid(g), B0, t_end=256.0, lam0=1e-8, dt=1e-3, max_trials=20000)
    _, eps = mro.eps_star(g.n, g.lo, g.hi, x, B0, 8, 8, np.sqrt(2.0))
    assert eps == pytest.approx(eps_p, rel=0.06), eps
    assert mro.diagnostics(g.n, g.lo, g.hi, x, B0)["xi"] < 1e-3
