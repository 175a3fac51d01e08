"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no projector, no gradient, no prox, no CP
step): it only produces *inputs* -- the five problem shapes of BASELINE.json `configs`, the
temporal basis tables Phi[j,k] = phi_j(t_k) (an input of the method, Eq. 8),
random test vectors, and synthetic measured data g = exact analytic line integrals of a seeded,
moving ellipsoid phantom sampled at the bin centres (stand-in for the paper's moving-circles
validation, and for the foam scan, which are not available).

Recipe: RNG numpy.random.default_rng([0, cfg, stream]) with
stream 0 = phantom, 1 = noise, 2 = operator test vectors, 3 = power-iteration start.
Geometry conventions are the ones DESIGN.md fixes (R1/R2): unit voxel and bin spacing,
s_b = b-(Nd-1)/2, theta_k = k*pi/N_theta0, t_k = k/N_theta.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, replace

import numpy as np


@dataclass(frozen=True)
class Config:
    """One problem shape.  m = number of temporal basis functions (the paper's M)."""
    cfg: int
    n: int            # grid side N (nx == ny)
    nz: int           # slices
    nd: int           # detector bins
    n_angles: int     # N_theta
    n_half_rot: int   # N_pi
    m: int
    basis: str        # "fourier" | "bspline"
    iters: int
    lambda1: float = 1e-3
    lambda2: float = 1.0
    n_objects: int = 3
    noise: str = "gauss"   # "gauss" | "poisson"

    @property
    def n_theta0(self) -> int:
        return self.n_angles // self.n_half_rot

    @property
    def V(self) -> int:
        return self.n * self.n * self.nz * self.m

    @property
    def S(self) -> int:
        return self.n_angles * self.nd * self.nz

    @property
    def nominal_updates(self) -> int:
        """voxel*angle*basis count of one operator call (BASELINE.json metric unit)."""
        return self.n * self.n * self.nz * self.n_angles * self.m

    def scaled(self, **kw) -> "Config":
        return replace(self, **kw)


# BASELINE.json `configs` 1..5 (index 0 unused so CONFIGS[c].cfg == c)
CONFIGS = {
    1: Config(1, 32, 1, 32, 128, 4, 4, "fourier", 20, n_objects=3),
    2: Config(2, 128, 8, 128, 720, 4, 8, "fourier", 50, n_objects=12, noise="poisson"),
    3: Config(3, 512, 32, 512, 1440, 8, 16, "fourier", 100, n_objects=40),
    4: Config(4, 1024, 64, 1024, 3000, 10, 16, "bspline", 100, n_objects=200),
    5: Config(5, 2048, 32, 2048, 3600, 12, 16, "fourier", 50, n_objects=500),
}


# ----------------------------------------------------------------------------------------------
# temporal basis tables (inputs of the method; readings R10/R11 in DESIGN.md)
# ----------------------------------------------------------------------------------------------
def basis_table(kind: str, m: int, n_angles: int) -> np.ndarray:
    """Phi[j,k] = phi_j(t_k), t_k = k/n_angles, float64, shape (m, n_angles)."""
    t = np.arange(n_angles, dtype=np.float64) / n_angles
    phi = np.zeros((m, n_angles), dtype=np.float64)
    if kind == "fourier":
        # real Fourier: 1, cos 2pi t, sin 2pi t, cos 4pi t, ...  (config 1 lists the first four)
        phi[0] = 1.0
        for j in range(1, m):
            r = (j + 1) // 2
            phi[j] = np.cos(2 * np.pi * r * t) if j % 2 == 1 else np.sin(2 * np.pi * r * t)
    elif kind == "bspline":
        # uniform cubic B-splines, knot spacing 1/(m-3): phi_j(t) = B3(t(m-3) - (j-1))
        if m < 4:
            raise ValueError("cubic B-spline table needs m >= 4")
        u = t[None, :] * (m - 3) - (np.arange(m, dtype=np.float64)[:, None] - 1.0)
        au = np.abs(u)
        phi = np.where(au < 1.0, 2.0 / 3.0 - au ** 2 + 0.5 * au ** 3,
                       np.where(au < 2.0, (2.0 - au) ** 3 / 6.0, 0.0))
    elif kind == "box":
        # cardinal box basis (phi_j(t) = 1 on [j/m,(j+1)/m)); used by tests only
        idx = np.minimum((t * m).astype(np.int64), m - 1)
        phi[idx, np.arange(n_angles)] = 1.0
    else:
        raise ValueError(f"unknown basis {kind!r}")
    return np.ascontiguousarray(phi)


def rng(cfg: int, stream: int) -> np.random.Generator:
    return np.random.default_rng([0, cfg, stream])


def test_vectors(c: Config, stream: int = 2):
    """Seeded N(0,1) operator-parity vectors: primal-shaped f[z][y][x][j] and sinogram g[z][k][b]."""
    r = rng(c.cfg, stream)
    f = r.standard_normal((c.nz, c.n, c.n, c.m))
    g = r.standard_normal((c.nz, c.n_angles, c.nd))
    return f, g


# ----------------------------------------------------------------------------------------------
# phantoms: ellipsoids  (A, B, C semi-axes; psi in-plane rotation; centre; density), all moving
# ----------------------------------------------------------------------------------------------
def phantom_params(c: Config) -> dict:
    """Seeded phantom description in voxel units (field of view radius 0.5*N)."""
    r = rng(c.cfg, 0)
    k, N, Nz = c.n_objects, c.n, c.nz
    p = {}
    if c.cfg == 1:
        rad = r.uniform(0.05, 0.2, k) * N
        p["A0"], p["B0"] = rad, rad.copy()
    else:
        p["A0"] = r.uniform(0.04, 0.15, k) * N
        p["B0"] = r.uniform(0.04, 0.15, k) * N
    p["C"] = r.uniform(0.5, 1.5, k) * max(Nz, 1)
    p["psi"] = r.uniform(0.0, np.pi, k) if c.cfg != 1 else np.zeros(k)
    p["rho"] = r.uniform(0.2, 1.0, k)
    p["c0"] = r.uniform(-0.15, 0.15, (k, 2)) * N
    p["cz"] = r.uniform(0.0, max(Nz - 1, 0), k)
    p["vel"] = r.uniform(-0.05, 0.05, (k, 2)) * N          # cfg 1: linear drift
    p["amp"] = r.uniform(0.0, 0.05, k) * N                  # cfg 2/3/5: sinusoidal centre
    p["freq"] = r.integers(1, 3, k).astype(np.float64)
    p["ph_c"] = r.uniform(0, 2 * np.pi, k)
    p["ph_r"] = r.uniform(0, 2 * np.pi, k)
    p["way"] = np.cumsum(r.uniform(-0.03, 0.03, (k, 5, 2)) * N, axis=1)  # cfg 4 waypoints
    return p


def _state_at(c: Config, p: dict, t):
    """Ellipse parameters at times t (array, shape (K,)) -> arrays of shape (n_obj, K)."""
    t = np.asarray(t, dtype=np.float64)[None, :]
    A = np.repeat(p["A0"][:, None], t.shape[1], 1)
    B = np.repeat(p["B0"][:, None], t.shape[1], 1)
    cx = np.repeat(p["c0"][:, 0:1], t.shape[1], 1)
    cy = np.repeat(p["c0"][:, 1:2], t.shape[1], 1)
    if c.cfg == 1:
        cx = cx + p["vel"][:, 0:1] * t
        cy = cy + p["vel"][:, 1:2] * t
    elif c.cfg == 4:
        # piecewise-linear path through 5 waypoints at t = 0, 1/4, 1/2, 3/4, 1
        u = np.clip(t * 4.0, 0.0, 4.0 - 1e-12)
        i0 = np.floor(u).astype(np.int64)[0]
        w = (u - np.floor(u))[0]
        cx = cx + (1 - w) * p["way"][:, i0, 0] + w * p["way"][:, np.minimum(i0 + 1, 4), 0]
        cy = cy + (1 - w) * p["way"][:, i0, 1] + w * p["way"][:, np.minimum(i0 + 1, 4), 1]
    elif c.cfg == 5:
        A = A * (1 + 0.15 * np.sin(2 * np.pi * t + p["ph_r"][:, None]))
        B = p["A0"][:, None] * p["B0"][:, None] / A            # area preserving
    else:
        s = np.sin(2 * np.pi * p["freq"][:, None] * t + p["ph_c"][:, None])
        cx = cx + p["amp"][:, None] * s
        cy = cy + p["amp"][:, None] * s * 0.5
        sc = 1 + 0.2 * np.sin(2 * np.pi * t + p["ph_r"][:, None])
        A, B = A * sc, B * sc
    return A, B, cx, cy


def sinogram(c: Config, noise: bool = True, device: str = "cpu"):
    """Synthetic measured data g[z][k][b] (float64 torch tensor on `device`).

    Exact line integral of each moving ellipsoid at time t_k, sampled at bin centres:
    2 rho A B sqrt(max(0, d^2 - s'^2)) / d^2 with d^2 = A^2 cos^2(th-psi) + B^2 sin^2(th-psi),
    s' = s - cx cos th - cy sin th, scaled by sqrt(max(0, 1-((z-cz)/C)^2)) for slice z.
    """
    import torch

    p = phantom_params(c)
    k = np.arange(c.n_angles)
    th = k * (np.pi / c.n_theta0)
    t = k / c.n_angles
    A, B, cx, cy = _state_at(c, p, t)
    d2 = (A * np.cos(th[None] - p["psi"][:, None])) ** 2 + (B * np.sin(th[None] - p["psi"][:, None])) ** 2
    sc = cx * np.cos(th)[None] + cy * np.sin(th)[None]
    amp = 2 * p["rho"][:, None] * A * B / d2

    dev = torch.device(device)
    T = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64, device=dev)
    s = torch.arange(c.nd, dtype=torch.float64, device=dev) - (c.nd - 1) / 2.0
    g = torch.zeros((c.nz, c.n_angles, c.nd), dtype=torch.float64, device=dev)
    d2_t, sc_t, amp_t = T(d2), T(sc), T(amp)
    zz = np.arange(c.nz, dtype=np.float64)
    for o in range(c.n_objects):
        prof = amp_t[o][:, None] * torch.sqrt(torch.clamp(d2_t[o][:, None] - (s[None, :] - sc_t[o][:, None]) ** 2, min=0.0))
        hz = np.sqrt(np.maximum(0.0, 1.0 - ((zz - p["cz"][o]) / p["C"][o]) ** 2)) if c.nz > 1 else np.ones(1)
        nzs = np.nonzero(hz)[0]
        if len(nzs):
            g[nzs] += T(hz[nzs])[:, None, None] * prof[None]
    if not noise:
        return g
    r = rng(c.cfg, 1)
    gmax = float(g.max())
    if c.noise == "poisson":
        g = g * (2.0 / max(gmax, 1e-30))
        counts = r.poisson(1e4 * np.exp(-g.cpu().numpy()))
        g = T(-np.log(np.maximum(counts, 1) / 1e4))
    else:
        # chunked over z to bound host memory at the large configs
        for z in range(c.nz):
            g[z] += T(r.standard_normal((c.n_angles, c.nd)) * (0.01 * gmax))
    return g


def small(cfg_like: int = 1, **kw) -> Config:
    """A shrunken variant of a config (same structure) for tests that need odd/ragged sizes."""
    return CONFIGS[cfg_like].scaled(**kw)


def describe(c: Config) -> str:
    return (f"cfg{c.cfg}_{c.n}x{c.n}x{c.nz}_nd{c.nd}_ang{c.n_angles}x{c.n_half_rot}pi_m{c.m}_{c.basis}")


__all__ = ["Config", "CONFIGS", "basis_table", "rng", "test_vectors", "phantom_params", "sinogram",
           "small", "describe", "math"]
