"""Seeded synthetic workloads for the relaxation step: closed forms only, numpy only.

This module serves BOTH the CPU oracle tests and the CUDA path (tests, bench.py) and therefore holds
none of the method's arithmetic (no Jacobian, push-forward, curl, update or reduction): it only evaluates
the closed-form initial fields and grids named by BASELINE.json ``configs`` and by PAPER.md section 3.1.
The recipe for every configuration is restated in DESIGN.md ("Input recipe").

Array convention (everywhere in this repository): a vector field on the grid is a C-contiguous array of
shape ``(3, nz, ny, nx)``; component 0/1/2 is the Cartesian x/y/z component; the logical index ``i``
(x-direction) is the fastest one, ``idx = (k*ny + j)*nx + i``.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Sequence, Tuple

import numpy as np

SEED = 14050942  # arxiv id of the paper, reading Q17


@dataclass(frozen=True)
class Grid:
    """Logically rectangular grid: ``n = (nx, ny, nz)`` nodes (boundary included) on ``[lo, hi]``."""

    n: Tuple[int, int, int]
    lo: Tuple[float, float, float]
    hi: Tuple[float, float, float]

    @property
    def h(self) -> Tuple[float, float, float]:
        return tuple((self.hi[a] - self.lo[a]) / (self.n[a] - 1) for a in range(3))

    @property
    def shape(self) -> Tuple[int, int, int, int]:
        return (3, self.n[2], self.n[1], self.n[0])

    @property
    def nodes(self) -> int:
        return self.n[0] * self.n[1] * self.n[2]

    def axes(self):
        """1-D node coordinates per logical axis: ``lo_a + idx*h_a`` (uniform reference grid)."""
        return tuple(self.lo[a] + np.arange(self.n[a], dtype=np.float64) * self.h[a] for a in range(3))


def reference_grid(g: Grid) -> np.ndarray:
    """The undistorted grid ``X_ijk`` (x(X,0)=X) as a ``(3,nz,ny,nx)`` float64 array."""
    ax, ay, az = g.axes()
    X = np.empty(g.shape, dtype=np.float64)
    X[0] = ax[None, None, :]
    X[1] = ay[None, :, None]
    X[2] = az[:, None, None]
    return X


# ----------------------------------------------------------------------------------------------------------
# Gaussian twist regions (BASELINE.json configs 1, 2, 4, 5; same family as PAPER.md Eq. 3.4, :190)
# ----------------------------------------------------------------------------------------------------------

@dataclass(frozen=True)
class Twist:
    k: float
    xc: float
    yc: float
    zc: float
    a: float = float(np.sqrt(2.0))
    l: float = 2.0


def twist_field(g: Grid, twists: Sequence[Twist], Bz: float = 1.0) -> np.ndarray:
    """``B0 = Bz*z^ + sum_m k_m exp(-((X-x_m)^2+(Y-y_m)^2)/a^2 - (Z-z_m)^2/l^2) * (-(Y-y_m), X-x_m, 0)``.

    Every term is analytically divergence free. DESIGN.md readings Q13/Q14 fix the centres and signs.
    """
    ax, ay, az = g.axes()
    B0 = np.zeros(g.shape, dtype=np.float64)
    B0[2] = Bz
    for t in twists:
        gx = np.exp(-((ax - t.xc) ** 2) / t.a ** 2)
        gy = np.exp(-((ay - t.yc) ** 2) / t.a ** 2)
        gz = np.exp(-((az - t.zc) ** 2) / t.l ** 2)
        amp = t.k * gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
        B0[0] += amp * (-(ay - t.yc))[None, :, None]
        B0[1] += amp * (ax - t.xc)[None, None, :]
    return B0


def braid_twists(z_scale: float = 1.0) -> Tuple[Twist, ...]:
    """Six twists, centres (+-1, 0, z_m), z_m = -20 + 8m, sign k_m = x_m = +1 (m even) / -1 (m odd) (Q13).

    ``z_scale`` compresses the z-structure (centres and length l) for config 5 (Q14: z_scale = 1/6).
    """
    out = []
    for m in range(6):
        s = 1.0 if m % 2 == 0 else -1.0
        out.append(Twist(k=s, xc=s, yc=0.0, zc=(-20.0 + 8.0 * m) * z_scale, l=2.0 * z_scale))
    return tuple(out)


# ----------------------------------------------------------------------------------------------------------
# ABC Beltrami field and the smooth seeded displacement (BASELINE.json config 3)
# ----------------------------------------------------------------------------------------------------------

def abc_field(P: np.ndarray, A: float = 1.0, B: float = 1.0, C: float = 1.0, k: float = np.pi) -> np.ndarray:
    """ABC field at the points ``P`` (shape (3,...)): curl = k * field (a Beltrami field, Eq. 1.4)."""
    x, y, z = P[0], P[1], P[2]
    out = np.empty_like(P, dtype=np.float64)
    out[0] = A * np.sin(k * z) + C * np.cos(k * y)
    out[1] = B * np.sin(k * x) + A * np.cos(k * z)
    out[2] = C * np.sin(k * y) + B * np.cos(k * x)
    return out


def smooth_displacement(g: Grid, seed: int = SEED, modes: int = 8, max_wavenumber: int = 4) -> np.ndarray:
    """Per component a sum of ``modes`` products of sines that vanish on all six faces (reading Q17).

    d_c = sum_m a_cm sin(p pi s_x) sin(q pi s_y) sin(r pi s_z),  s_a = (X_a - lo_a)/(hi_a - lo_a),
    a_cm ~ N(0,1), p,q,r uniform integers in 1..max_wavenumber, all from one ``default_rng(seed)`` stream in
    the order (component, mode) -> (a, p, q, r).  Each component is scaled to max|d_c| = 1.
    """
    rng = np.random.default_rng(seed)
    s = [np.arange(g.n[a], dtype=np.float64) / (g.n[a] - 1) for a in range(3)]
    d = np.zeros(g.shape, dtype=np.float64)
    for c in range(3):
        for _ in range(modes):
            a = rng.normal()
            p, q, r = (int(v) for v in rng.integers(1, max_wavenumber + 1, size=3))
            sx = np.sin(p * np.pi * s[0])
            sy = np.sin(q * np.pi * s[1])
            sz = np.sin(r * np.pi * s[2])
            # exact zeros on the faces (sin(p*pi) is only ~1e-16 in floating point)
            sx[0] = sx[-1] = 0.0
            sy[0] = sy[-1] = 0.0
            sz[0] = sz[-1] = 0.0
            d[c] += a * sz[:, None, None] * sy[None, :, None] * sx[None, None, :]
        d[c] /= np.abs(d[c]).max()
    return d


def displaced_grid(g: Grid, amplitude: float = 0.3, seed: int = SEED) -> np.ndarray:
    """``x0 = X + amplitude * h_c * d_c`` (config 3: amplitude 0.3); boundary nodes stay on X exactly."""
    X = reference_grid(g)
    d = smooth_displacement(g, seed)
    h = g.h
    for c in range(3):
        X[c] += amplitude * h[c] * d[c]
    return X


def rough_displacement(g: Grid, amplitude: float = 0.3, seed: int = SEED) -> np.ndarray:
    """Non-smooth distortion: independent uniform(-1,1)*amplitude*h_c per interior node; zero on the boundary.

    Used for the "arbitrarily distorted grid" pins of the mimetic curl."""
    rng = np.random.default_rng(seed)
    X = reference_grid(g)
    d = rng.uniform(-1.0, 1.0, size=g.shape)
    d[:, 0] = d[:, -1] = 0.0
    d[:, :, 0] = d[:, :, -1] = 0.0
    d[:, :, :, 0] = d[:, :, :, -1] = 0.0
    h = g.h
    for c in range(3):
        X[c] += amplitude * h[c] * d[c]
    return X


# ----------------------------------------------------------------------------------------------------------
# IsoHelix closed-form pair (Eqs. 3.1 and 3.3, :172, :182-186)
# ----------------------------------------------------------------------------------------------------------

def isohelix_B0(g: Grid, phi: float, B0: float = 1.0, a_r: float = float(np.sqrt(2.0)), a_z: float = 2.0) -> np.ndarray:
    """Eq. 3.1: ``B = (2 B0 Z/a_z^2) exp(-(X^2+Y^2)/a_r^2 - Z^2/a_z^2) phi (Y, -X, 0) + B0 z^``."""
    X = reference_grid(g)
    e = np.exp(-(X[0] ** 2 + X[1] ** 2) / a_r ** 2 - X[2] ** 2 / a_z ** 2)
    c = 2.0 * B0 * X[2] / a_z ** 2 * e * phi
    out = np.empty_like(X)
    out[0] = c * X[1]
    out[1] = -c * X[0]
    out[2] = B0
    return out


def isohelix_x_relax(g: Grid, phi: float, a_r: float = float(np.sqrt(2.0)), a_z: float = 2.0) -> np.ndarray:
    """Eq. 3.3: rotation of (X,Y) by the angle ``-exp(...)*phi`` about the z axis; Z unchanged."""
    X = reference_grid(g)
    ang = np.exp(-(X[0] ** 2 + X[1] ** 2) / a_r ** 2 - X[2] ** 2 / a_z ** 2) * phi
    out = np.empty_like(X)
    out[0] = np.cos(ang) * X[0] + np.sin(ang) * X[1]
    out[1] = np.cos(ang) * X[1] - np.sin(ang) * X[0]
    out[2] = X[2]
    return out


def pontin09_B0(g: Grid, phi: Sequence[float], L: Sequence[float], B0: float = 1.0, a_r: float = float(np.sqrt(2.0)),
                a_z: float = 2.0) -> np.ndarray:
    """Eq. 3.4: ``B = B0 z^ + sum_i (2 B0 phi_i / (pi a_r)) exp(-(X^2+Y^2)/a_r^2 - (Z-L_i)^2/a_z^2) (-Y, X, 0)``;
    ``L_i`` = positions of the twist regions along z (the paper does not print them: DESIGN.md reading Q25)."""
    X = reference_grid(g)
    out = np.zeros_like(X)
    out[2] = B0
    for ph, Li in zip(phi, L):
        c = 2.0 * B0 * ph / (np.pi * a_r) * np.exp(-(X[0] ** 2 + X[1] ** 2) / a_r ** 2 - (X[2] - Li) ** 2 / a_z ** 2)
        out[0] += -c * X[1]
        out[1] += c * X[0]
    return out


# ----------------------------------------------------------------------------------------------------------
# The five BASELINE.json configurations
# ----------------------------------------------------------------------------------------------------------

def stable_dt(B0: np.ndarray, g: Grid) -> float:
    """Fixed step for the configs that do not state one (reading Q6): ``0.5 / (max|B0|^2 * sum_a h_a^-2)``."""
    b2 = float((np.asarray(B0, dtype=np.float64) ** 2).sum(axis=0).max())
    return 0.5 / (b2 * sum(1.0 / ha ** 2 for ha in g.h))


@dataclass(frozen=True)
class Config:
    name: str
    grid: Grid
    dtype: str            # "f64" | "f32"
    steps: int
    dt: float | None      # None -> stable_dt(B0, grid)
    kind: str             # "twist1" | "braid" | "braid_z6" | "abc"
    note: str = ""
    twists: Tuple[Twist, ...] = field(default_factory=tuple)


CONFIGS = {
    "C1": Config("C1", Grid((16, 16, 32), (-4.0, -4.0, -8.0), (4.0, 4.0, 8.0)), "f64", 100, 0.01, "twist1",
                 "tiny relaxation, one twist k=1 at the origin", (Twist(1.0, 0.0, 0.0, 0.0),)),
    "C2": Config("C2", Grid((64, 64, 192), (-4.0, -4.0, -24.0), (4.0, 4.0, 24.0)), "f64", 2000, None, "braid",
                 "braided field, six twists", braid_twists()),
    "C3": Config("C3", Grid((128, 128, 128), (-1.0, -1.0, -1.0), (1.0, 1.0, 1.0)), "f64", 200, None, "abc",
                 "ABC field on a smoothly displaced grid"),
    "C4": Config("C4", Grid((256, 256, 512), (-4.0, -4.0, -24.0), (4.0, 4.0, 24.0)), "f64", 10000, None, "braid",
                 "large braided relaxation (the roofline case)", braid_twists()),
    "C5": Config("C5", Grid((512, 512, 512), (-4.0, -4.0, -4.0), (4.0, 4.0, 4.0)), "f32", 1000, None, "braid_z6",
                 "fp32 variant, braid compressed 6x in z", braid_twists(1.0 / 6.0)),
}


def scaled(cfg: Config, n: Tuple[int, int, int]) -> Config:
    """Same domain and field as ``cfg`` on a different node count (for parity tests the oracle finishes fast)."""
    return Config(cfg.name + "@%dx%dx%d" % n, Grid(tuple(n), cfg.grid.lo, cfg.grid.hi), cfg.dtype, cfg.steps,
                  cfg.dt if tuple(n) == cfg.grid.n else None, cfg.kind, cfg.note, cfg.twists)


def make(cfg: Config, seed: int = SEED):
    """Return ``(x0, B0, dt)`` (float64 arrays of shape ``cfg.grid.shape``) for a configuration.

    For "abc" (config 3) this is the literal reading D: ``B0 = ABC(X)``, ``x0 = X + 0.3 h d``. Reading P (B0 pulled
    back so that the pushed-forward nodal field is ABC(x0)) needs the discrete Jacobian and is therefore assembled
    in the tests from oracle output, not here.
    """
    g = cfg.grid
    if cfg.kind in ("twist1", "braid", "braid_z6"):
        B0 = twist_field(g, cfg.twists)
        x0 = reference_grid(g)
    elif cfg.kind == "abc":
        x0 = displaced_grid(g, 0.3, seed)
        B0 = abc_field(reference_grid(g))
    else:
        raise ValueError(cfg.kind)
    dt = cfg.dt if cfg.dt is not None else stable_dt(B0, g)
    return x0, B0, dt
