"""Seeded synthetic workloads for the ship-wave residual F(u).

This module serves BOTH the oracle tests and the CUDA path with bit-identical
inputs.  It holds none of the method's arithmetic (no reconstruction, no
kernels, no residual rows): only mesh parameters and the analytic
Gaussian-sum state the five BASELINE.json configs describe.

Recipe (BASELINE.json `configs`, reading Q11 of DESIGN.md):
  zeta(x,y) = sum_{i=1..8} a_i exp(-((x-c_i)^2 + (y-d_i)^2) / w_i^2)
  a_i ~ U(-amp, amp), c_i ~ U(0,16), d_i ~ U(0,8), w_i ~ U(1,3)
  rng = numpy.random.default_rng(seed); draw order a[8], c[8], d[8], w[8]
  phi = x + 0.1 * d(zeta)/dx
  u (eq. (18)) per y-line l:  [phi_{1,l}, (phi_x)_{1..N,l}],
  all l; then [zeta_{1,l}, (zeta_x)_{1..N,l}], all l.   zeta_x, phi_x analytic.
  V = default_rng(seed_V).standard_normal((b, n)).

These states stand in for the paper's converged eps=1, F=0.7 solutions
(Table 1), which are not available.
"""
from __future__ import annotations

from dataclasses import dataclass, asdict

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    N: int          # nodes in x
    M: int          # nodes in y
    h: float        # dx = dy
    x1: float       # upstream truncation (paper's x_0 / x_1, L162, L227)
    y1: float
    froude: float   # F, eq. (9)
    eps: float      # source strength, eq. (6)
    n_rad: float    # radiation exponent n = 0.05, L189
    amp: float      # Gaussian amplitude bound
    seed: int
    b: int          # Jv batch size (0 = none)
    seed_V: int

    @property
    def n(self) -> int:
        """Number of unknowns 2(N+1)M."""
        return 2 * (self.N + 1) * self.M

    @property
    def targets(self) -> int:
        """Half-mesh midpoints (N-1)M."""
        return (self.N - 1) * self.M

    @property
    def sources(self) -> int:
        return self.N * self.M

    @property
    def pairs(self) -> int:
        return self.targets * self.sources

    def params(self, dy_scheme: int = 0) -> dict:
        return dict(N=self.N, M=self.M, x1=self.x1, y1=self.y1, dx=self.h,
                    dy=self.h, froude=self.froude, eps=self.eps,
                    n_rad=self.n_rad, dy_scheme=dy_scheme)

    def asdict(self) -> dict:
        return asdict(self)


# The five BASELINE.json configs, in order (CONFIGS[4] is the headline 721x241).
CONFIGS = (
    Config("cfg1_31x11",   31,  11, 0.8,    -8.0, 0.0, 0.7, 0.1, 0.05, 0.02, 0,  0,   0),
    Config("cfg2_61x21",   61,  21, 0.4,    -8.0, 0.0, 0.7, 0.2, 0.05, 0.02, 1,  8,   2),
    Config("cfg3_181x61",  181, 61, 0.3,   -16.0, 0.0, 0.7, 0.5, 0.05, 0.05, 3, 16, 103),
    Config("cfg4_361x121", 361, 121, 0.15, -16.0, 0.0, 0.7, 0.5, 0.05, 0.05, 4, 32, 104),
    Config("cfg5_721x241", 721, 241, 0.075, -16.0, 0.0, 0.7, 1.0, 0.05, 0.1,  5, 16, 105),
)
BY_NAME = {c.name: c for c in CONFIGS}

# The meshes the paper itself solves on, eps = 1: 91x31 "contemporary" and
# 361x121, 721x241 (L275), all F = 0.7; Fig. 2/3's 45x13 (L247); Fig. 7's
# F = 1.4 mesh (L336: 721x241, dx = dy = 0.3, x0 = -56).  The solver tests and bench.py's `solve`
# section start these from the flat state (L227); the seeded Gaussian state is also defined.
PAPER_MESHES = (
    Config("paper_45x13",    45,  13, 0.4,    -9.0, 0.0, 0.7, 1.0, 0.05, 0.05, 11, 0, 111),
    Config("paper_91x31",    91,  31, 0.3,    -9.0, 0.0, 0.7, 1.0, 0.05, 0.05, 12, 0, 112),
    Config("paper_361x121", 361, 121, 0.15,  -14.0, 0.0, 0.7, 1.0, 0.05, 0.05, 13, 0, 113),
    Config("paper_721x241", 721, 241, 0.075, -14.0, 0.0, 0.7, 1.0, 0.05, 0.05, 14, 0, 114),
    Config("paper_fig7_721x241", 721, 241, 0.3, -56.0, 0.0, 1.4, 1.0, 0.05, 0.05, 15, 0, 115),
)
PAPER_BY_NAME = {c.name: c for c in PAPER_MESHES}


def custom(N, M, h, x1, *, y1=0.0, froude=0.7, eps=0.1, n_rad=0.05, amp=0.02,
           seed=0, b=0, seed_V=None, name=None) -> Config:
    """A config of the same family at another shape (ragged/edge-case tests)."""
    return Config(name or f"custom_{N}x{M}", N, M, h, x1, y1, froude, eps,
                  n_rad, amp, seed, b, seed + 100 if seed_V is None else seed_V)


def mesh(cfg: Config):
    """Node coordinates x_k = x1 + (k-1) h, y_l = y1 + (l-1) h (0-based arrays)."""
    x = cfg.x1 + np.arange(cfg.N, dtype=np.float64) * cfg.h
    y = cfg.y1 + np.arange(cfg.M, dtype=np.float64) * cfg.h
    return x, y


def gaussians(cfg: Config):
    rng = np.random.default_rng(cfg.seed)
    a = rng.uniform(-cfg.amp, cfg.amp, 8)
    c = rng.uniform(0.0, 16.0, 8)
    d = rng.uniform(0.0, 8.0, 8)
    w = rng.uniform(1.0, 3.0, 8)
    return a, c, d, w


def surface(cfg: Config, X, Y):
    """Analytic zeta, zeta_x, zeta_xx of the Gaussian sum at points (X, Y)."""
    a, c, d, w = gaussians(cfg)
    X = np.asarray(X, dtype=np.float64)[..., None]
    Y = np.asarray(Y, dtype=np.float64)[..., None]
    g = a * np.exp(-((X - c) ** 2 + (Y - d) ** 2) / w ** 2)
    gx = g * (-2.0 * (X - c) / w ** 2)
    gxx = g * (4.0 * (X - c) ** 2 / w ** 4 - 2.0 / w ** 2)
    return g.sum(-1), gx.sum(-1), gxx.sum(-1)


def pack(cfg: Config, phi1, phi_x, zeta1, zeta_x):
    """Pack per-line upstream values [M] and slopes [M, N] into u, eq. (18) L149."""
    N, M = cfg.N, cfg.M
    u = np.empty(cfg.n, dtype=np.float64)
    top = u[: (N + 1) * M].reshape(M, N + 1)
    bot = u[(N + 1) * M:].reshape(M, N + 1)
    top[:, 0] = phi1
    top[:, 1:] = phi_x
    bot[:, 0] = zeta1
    bot[:, 1:] = zeta_x
    return u


def state(cfg: Config) -> np.ndarray:
    """The seeded state vector u (length 2(N+1)M, float64)."""
    x, y = mesh(cfg)
    X, Y = np.meshgrid(x, y)                      # [M, N]
    z, zx, zxx = surface(cfg, X, Y)
    phi1 = x[0] + 0.1 * zx[:, 0]
    return pack(cfg, phi1, 1.0 + 0.1 * zxx, z[:, 0], zx)


def flat_state(cfg: Config) -> np.ndarray:
    """The flat-surface initial guess u_0: phi_1 = x_1, phi_x = 1,
    zeta_1 = 0, zeta_x = 0."""
    M, N = cfg.M, cfg.N
    return pack(cfg, np.full(M, cfg.x1), np.ones((M, N)), np.zeros(M), np.zeros((M, N)))


def directions(cfg: Config, b: int | None = None) -> np.ndarray:
    """The Jv batch V [b, n], entries ~ N(0,1) (BASELINE.json configs)."""
    b = cfg.b if b is None else b
    return np.random.default_rng(cfg.seed_V).standard_normal((b, cfg.n))
