"""Seeded, synthetic input generators shared by the CUDA path and the oracle.

This module holds NONE of the method's arithmetic (no lattice, no collision,
no interpolation, no boundary rule): it only produces the inputs both sides
consume — mesh coordinates, the five BASELINE.json workloads, and random test
states.  It imports neither the CUDA binding nor oracle/.

Mesh recipes
  tanh_mesh    : BASELINE.json configs, x_j = 0.5*(1 + tanh(b*(2j/(N-1) - 1))/tanh(b)),
                 j = 0..N-1; every node is a fluid node; delta = x_1 - x_0
                 (reading A1).
  uniform_mesh : Eq. 24-25, x_j = (j + 0.5)/N, delta = 1/N.
  erf_mesh     : Eq. 26, N_y + 2 points j = 0..N_y+1; the fluid
                 nodes are j = 1..N_y and delta = y_1.
  wallgap_mesh : hand-made; first / last spacing 2.5 / 1.75 lattice units, so that
                 q of Eq. 28 is far from 1 and differs between the walls.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SQRT3 = math.sqrt(3.0)


def tanh_mesh(n: int, b: float):
    j = np.arange(n, dtype=np.float64)
    x = 0.5 * (1.0 + np.tanh(b * (2.0 * j / (n - 1) - 1.0)) / math.tanh(b))
    return x, float(x[1] - x[0])


def uniform_mesh(n: int):
    j = np.arange(n, dtype=np.float64)
    return (j + 0.5) / n, 1.0 / n


def erf_points(npts: int, a: float):
    """All N_y + 2 points of Eq. 26 (npts = N_y + 2), walls' ghost points included."""
    return np.array([0.5 * (math.erf(a * (j / (npts - 1) - 0.5)) / math.erf(a / 2.0) + 1.0) for j in range(npts)])


def erf_mesh(npts: int, a: float):
    """Fluid nodes 1..N_y of Eq. 26 and delta = y_1."""
    y = erf_points(npts, a)
    return y[1:-1].copy(), float(y[1])


def wallgap_mesh(n: int, q_lo: float = 2.5, q_hi: float = 1.75):
    """Hand-made mesh for the q != 1 cases of Eq. 28: the first / last spacing is q_lo / q_hi
    lattice units (different at the two walls, so a swapped pair shows), the interior spacings ramp between 1 and
    1.5 l.u. with two of them exactly 1; walls at 0 and 1, i.e. x_0 = delta/2.  Returns (x, delta)."""
    k = np.arange(n - 1, dtype=np.float64)
    s = 1.0 + 0.5 * np.sin(math.pi * k / (n - 2)) ** 2
    s[0], s[-1] = q_lo, q_hi
    s[1], s[-2] = 1.0, 1.0
    delta = 1.0 / (float(s.sum()) + 1.0)
    x = delta * (0.5 + np.concatenate(([0.0], np.cumsum(s))))
    return x, delta


@dataclass
class Workload:
    name: str
    dim: int
    n: int
    mesh: str            # "tanh" | "uniform" | "erf" | "wallgap"
    stretch: float
    Ra: float
    Pr: float = 0.71
    Ma: float = 0.1 * SQRT3   # BASELINE.json: U = 0.1 l.u.  =>  Ma = U / c_s
    seed: int = 0
    noise_amp: float = 1e-3
    steps: int = 1000
    coords: list = field(default_factory=list)
    delta: float = 0.0

    def __post_init__(self):
        if self.mesh == "tanh":
            x, d = tanh_mesh(self.n, self.stretch)
        elif self.mesh == "uniform":
            x, d = uniform_mesh(self.n)
        elif self.mesh == "erf":
            x, d = erf_mesh(self.n, self.stretch)
        elif self.mesh == "wallgap":
            x, d = wallgap_mesh(self.n)
        else:
            raise ValueError(self.mesh)
        self.coords = [x.copy() for _ in range(self.dim)]
        self.delta = d

    @property
    def nodes(self) -> int:
        return len(self.coords[0]) ** self.dim

    @property
    def shape(self):
        m = len(self.coords[0])
        return (1, m, m) if self.dim == 2 else (m, m, m)


# BASELINE.json "configs", in order; uniform counterparts share the name + "_uniform".
_CONFIGS = {
    "c1_64sq": dict(dim=2, n=64, mesh="tanh", stretch=1.2, Ra=1e5, steps=1000),
    "c2_512sq": dict(dim=2, n=512, mesh="tanh", stretch=1.5, Ra=1e7, steps=20000),
    "c3_1024sq": dict(dim=2, n=1024, mesh="tanh", stretch=2.0, Ra=1e8, steps=50000),
    "c4_128cu": dict(dim=3, n=128, mesh="tanh", stretch=1.5, Ra=1e6, steps=5000),
    "c5_256cu": dict(dim=3, n=256, mesh="tanh", stretch=1.8, Ra=1e7, steps=10000),
}


def workload(name: str) -> Workload:
    uniform = name.endswith("_uniform")
    key = name[: -len("_uniform")] if uniform else name
    cfg = dict(_CONFIGS[key])
    if uniform:
        cfg.update(mesh="uniform", stretch=0.0)
    return Workload(name=name, **cfg)


def workload_names():
    return list(_CONFIGS)


def custom_workload(name, dim, n, mesh="tanh", stretch=1.5, Ra=1e6, **kw) -> Workload:
    return Workload(name=name, dim=dim, n=n, mesh=mesh, stretch=stretch, Ra=Ra, **kw)


def random_state(shape_zyx, qf: int, qg: int, seed: int, amp: float = 0.02):
    """A seeded, smooth-plus-noise positive population state for parity tests.

    Values are only *inputs*: f_i ~ 1/qf * (1 + amp * noise), g_i ~ amp * noise;
    no lattice weights or equilibria are used, so the state is far from
    equilibrium and exercises every relaxation rate.
    """
    rng = np.random.default_rng(seed)
    nz, ny, nx = shape_zyx
    zz, yy, xx = np.meshgrid(np.linspace(0, 1, nz) if nz > 1 else np.zeros(1),
                             np.linspace(0, 1, ny), np.linspace(0, 1, nx), indexing="ij")
    f = np.empty((qf, nz, ny, nx))
    g = np.empty((qg, nz, ny, nx))
    for i in range(qf):
        smooth = np.sin(2 * math.pi * (xx * (1 + i % 3) + yy * (1 + i % 2) + zz * (1 + i % 4)) + i)
        f[i] = (1.0 / qf) * (1.0 + amp * smooth + amp * rng.uniform(-1, 1, size=(nz, ny, nx)))
    for i in range(qg):
        smooth = np.cos(2 * math.pi * (xx * (1 + i % 2) - yy * (1 + i % 3) + zz) + 0.5 * i)
        g[i] = amp * (smooth + rng.uniform(-1, 1, size=(nz, ny, nx)))
    return f, g
