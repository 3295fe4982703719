"""Seeded synthetic workloads shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no interpolation weights, no FFT,
no field solve): only the grids, initial conditions, drive field and random arrays
that define BASELINE.json's five configs.  It imports neither the
CUDA binding nor the oracle.  The paper used no dataset -- all its runs start from
analytic initial conditions -- so these generators ARE the
workload; the config-4 uniform grids stand in for "phase-space grids shaped like the
paper's runs".  Everything is produced in float64 and rounded once to float32; the
same float32 bytes go to the oracle (promoted to double) and to the GPU.
"""
from dataclasses import dataclass, field as _field
import math

import numpy as np

SEED = 13015892

LAGRANGE = 0
BSPLINE = 1
SPLIT_XVX = 0
SPLIT_VXV = 1

_ISQ2PI = 1.0 / math.sqrt(2.0 * math.pi)


@dataclass
class Config:
    name: str
    Nx: int
    Nv: int
    L: float
    vmin: float
    vmax: float
    kind: int = LAGRANGE
    order: int = 17
    dt: float = 0.1
    steps: int = 100
    split: int = SPLIT_XVX
    # f_eq(v) = sum_g amp*exp(-c (v-mu)^2) as (amp, mu, c) triples; empty => full-f storage
    feq: list = _field(default_factory=list)
    # perturbation: f0 = (1 + alpha cos(k x)) * profile(v)
    alpha: float = 0.0
    k: float = 0.0
    # profile(v), same Gaussian-sum format (what f0 is built from)
    profile: list = _field(default_factory=list)
    keen: bool = False

    @property
    def dx(self):
        return self.L / self.Nx

    @property
    def dv(self):
        return (self.vmax - self.vmin) / self.Nv

    def x(self):
        return np.arange(self.Nx, dtype=np.float64) * self.dx

    def v(self):
        return self.vmin + np.arange(self.Nv, dtype=np.float64) * self.dv


_MAXW = [(_ISQ2PI, 0.0, 0.5)]
_BUMP = [(0.9 * _ISQ2PI, 0.0, 0.5), (0.2 * _ISQ2PI, 4.5, 4.0)]


def config(idx, **over):
    """BASELINE.json configs 0-3 (config 4 is `sweep_case`)."""
    if idx == 0:   # linear Landau, full-f
        c = Config("landau_linear_64", 64, 64, 4 * math.pi, -6.0, 6.0, LAGRANGE, 17, 0.1, 100,
                   feq=[], alpha=1e-3, k=0.5, profile=_MAXW)
    elif idx == 1:  # nonlinear Landau, delta-f
        c = Config("landau_nonlinear_256", 256, 256, 4 * math.pi, -6.0, 6.0, LAGRANGE, 17, 0.1, 600,
                   feq=list(_MAXW), alpha=0.5, k=0.5, profile=_MAXW)
    elif idx == 2:  # bump on tail, delta-f vs the unperturbed two-Gaussian profile
        c = Config("bump_on_tail_1024", 1024, 1024, 20 * math.pi, -9.0, 9.0, LAGRANGE, 17, 0.05, 2000,
                   feq=list(_BUMP), alpha=0.04, k=0.3, profile=_BUMP)
    elif idx == 3:  # KEEN wave, delta-f vs Maxwellian, external drive
        c = Config("keen_2048x4096", 2048, 4096, 2 * math.pi / 0.26, -6.0, 6.0, LAGRANGE, 17, 0.05, 4000,
                   feq=list(_MAXW), alpha=0.0, k=0.26, profile=_MAXW, keen=True)
    else:
        raise ValueError(idx)
    for key, val in over.items():
        setattr(c, key, val)
    return c


def metric_config():
    """The grid BASELINE.json's metric is quoted on: fp32 delta-f, 2048 x 2048, LAG17.
    Physics = config 1's nonlinear Landau set-up on the larger grid."""
    return config(1, name="landau_nonlinear_2048_deltaf", Nx=2048, Nv=2048)


def gaussians(v, gs):
    out = np.zeros_like(v, dtype=np.float64)
    for amp, mu, c in gs:
        out += amp * np.exp(-c * (v - mu) ** 2)
    return out


def initial_f(cfg):
    """Stored array at t=0, float32 [Nv][Nx]: f0 in full-f mode, f0 - f_eq(v) in delta-f mode."""
    x = cfg.x()[None, :]
    v = cfg.v()[:, None]
    f0 = (1.0 + cfg.alpha * np.cos(cfg.k * x)) * gaussians(v, cfg.profile)
    if cfg.feq:
        f0 = f0 - gaussians(v, cfg.feq)
    return np.ascontiguousarray(f0, dtype=np.float32)


def keen_amplitude(t):
    """a(t) of P:273 with t0=0, tL=69, tR=307, twL=twR=20."""
    tL, tR, tw, t0 = 69.0, 307.0, 20.0, 0.0
    eps = 0.5 * (math.tanh((t0 - tL) / tw) - math.tanh((t0 - tR) / tw))
    return (0.5 * (math.tanh((t - tL) / tw) - math.tanh((t - tR) / tw)) - eps) / (1.0 - eps)


def keen_E_ext(cfg, t):
    """E_ext = -E_app(t, x), E_app = E_max k a(t) sin(kx - w t), E_max=0.2, k=0.26, w=0.37
    (the advecting field is E - E_app).  float32 [Nx]."""
    Emax, k, w = 0.2, 0.26, 0.37
    e = -Emax * k * keen_amplitude(t) * np.sin(k * cfg.x() - w * t)
    return e.astype(np.float32)


def uniform_grid(Nx, Nv, seed=SEED):
    """Config 4: f ~ U[0,1) float32."""
    rng = np.random.default_rng(seed)
    return rng.random((Nv, Nx), dtype=np.float32)


def uniform_shifts(n, seed=SEED + 1, lo=-8.0, hi=8.0):
    """Config 4: per-line shifts uniform in [-8, 8] cells, float64."""
    rng = np.random.default_rng(seed)
    return rng.uniform(lo, hi, size=n)


def smooth_grid(Nx, Nv, seed=SEED + 2, modes=6):
    """A band-limited random periodic field (delta-f-like, zero mean-ish), float32 [Nv][Nx]."""
    rng = np.random.default_rng(seed)
    x = np.arange(Nx) / Nx
    v = np.arange(Nv) / Nv
    f = np.zeros((Nv, Nx))
    for _ in range(modes):
        kx, kv = rng.integers(0, 5, size=2)
        ph1, ph2 = rng.uniform(0, 2 * math.pi, size=2)
        f += rng.normal() * np.cos(2 * math.pi * kx * x[None, :] + ph1) * np.cos(2 * math.pi * kv * v[:, None] + ph2)
    return np.ascontiguousarray(f / max(1e-30, np.abs(f).max()), dtype=np.float32)


SWEEP_N = (512, 2048, 8192, 16384)
SWEEP_KINDS = ((LAGRANGE, 3), (LAGRANGE, 9), (LAGRANGE, 17), (BSPLINE, 3))
