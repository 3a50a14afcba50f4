"""Seeded synthetic inputs shaped like the paper's workloads ("Input recipe").

The five BASELINE.json configs stand in for the paper's collapsing-water-column
(Tables 2/4) and rising-bubble cases: a
sharp two-phase volume-fraction field, a 1000:1 density ratio
and a box with walls on the sides/bottom and an open top.  The paper's own
field snapshots are not available; these generators reproduce their structure.

This module contains input generation ONLY (analytic profiles and random
numbers).  None of the method's arithmetic (stencils, density law, residuals)
lives here; both the oracle and the CUDA path consume these arrays as data.

All arrays are float64, C-contiguous, shape (nz, ny, nx) -- x fastest -- with
cell centres at ((i+1/2)hx, (j+1/2)hy, (k+1/2)hz).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import rng

# boundary-condition codes; same integer values as include/mg.h
BC_NEUMANN, BC_DIRICHLET, BC_DIRICHLET_HALO = 0, 1, 2


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    h: float
    levels: int
    bc: tuple                       # x-, x+, y-, y+, z-, z+
    nu_pre: int = 2
    nu_post: int = 2
    coarse_sweeps: int = 50
    omega: float = 2.0 / 3.0
    tol: float = 1e-8
    rho_l: float = 1000.0
    rho_g: float = 1.0
    mu_l: float = 1e-3
    mu_g: float = 1e-5
    dt: float = 1.0
    fields: dict = field(default_factory=dict)

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def n(self):
        return self.nx * self.ny * self.nz


def centres(nx, ny, nz, h):
    """Open-mesh cell-centre coordinates, broadcastable to (nz, ny, nx)."""
    x = ((np.arange(nx) + 0.5) * h).reshape(1, 1, nx)
    y = ((np.arange(ny) + 0.5) * h).reshape(1, ny, 1)
    z = ((np.arange(nz) + 0.5) * h).reshape(nz, 1, 1)
    return x, y, z


def water_column_alpha(nx, ny, nz, h, smooth_cells=2.0):
    """alpha=1 where x<0.25 and z<0.5 (unit box), tanh-smoothed (config 2, 5)."""
    x, y, z = centres(nx, ny, nz, h)
    d = np.minimum(0.25 - x, 0.5 - z) + 0.0 * y
    return np.ascontiguousarray(0.5 * (1.0 + np.tanh(d / (smooth_cells * h))))


def bubble_alpha(nx, ny, nz, h, centres_xyz, radius, smooth_cells=1.5):
    """alpha=0 inside each sphere, 1 outside; product of tanh profiles (configs 3, 4)."""
    x, y, z = centres(nx, ny, nz, h)
    a = np.ones((nz, ny, nx))
    for (cx, cy, cz) in centres_xyz:
        d = np.sqrt((x - cx) ** 2 + (y - cy) ** 2 + (z - cz) ** 2) - radius
        a *= 0.5 * (1.0 + np.tanh(d / (smooth_cells * h)))
    return np.ascontiguousarray(a)


def random_velocity(seeds, shape):
    """Three i.i.d. N(0,1) component fields (RHS source of configs 2-4)."""
    n = int(np.prod(shape))
    return tuple(rng.normal(s, n).reshape(shape) for s in seeds)


def bubble_centres(seed, count=4, radius=0.06, gap=0.02,
                   lo=(0.1, 0.1, 0.1), hi=(0.9, 0.9, 0.4)):
    """Rejection-sampled non-overlapping sphere centres (config 4)."""
    u = rng.uniform01(seed, 3 * 4096).reshape(-1, 3)
    out = []
    for row in u:
        c = tuple(lo[d] + (hi[d] - lo[d]) * row[d] for d in range(3))
        if all(np.linalg.norm(np.subtract(c, o)) >= 2 * radius + gap for o in out):
            out.append(c)
            if len(out) == count:
                return out
    raise RuntimeError("could not place bubbles")


def solenoidal_velocity(seeds, nx, ny, nz, h, modes=8):
    """q = curl(psi); each psi component is a sum of `modes` Fourier modes with
    integer wave-vectors in [1,4]^3, amplitudes N(0,1)/|kappa|^2 and random
    phases, evaluated analytically at the cell centres and scaled to
    max|q|_inf = 1 (config 5)."""
    x, y, z = centres(nx, ny, nz, h)
    # d(psi_c)/d(axis) for every component c and axis
    grad = [[np.zeros((nz, ny, nx)) for _ in range(3)] for _ in range(3)]
    for c, seed in enumerate(seeds):
        kap = 1 + np.floor(4.0 * rng.uniform01(seed, 3 * modes)).astype(np.int64).reshape(modes, 3)
        kap = np.minimum(kap, 4)
        amp = rng.normal(seed + 100, modes) / np.sum(kap.astype(np.float64) ** 2, axis=1)
        pha = 2.0 * np.pi * rng.uniform01(seed + 200, modes)
        for m in range(modes):
            kx, ky, kz = (2.0 * np.pi * kap[m]).tolist()
            cosarg = np.cos(kx * x + ky * y + kz * z + pha[m])
            for ax, kk in enumerate((kx, ky, kz)):
                grad[c][ax] += amp[m] * kk * cosarg
    u = grad[2][1] - grad[1][2]
    v = grad[0][2] - grad[2][0]
    w = grad[1][0] - grad[0][1]
    s = 1.0 / max(np.abs(u).max(), np.abs(v).max(), np.abs(w).max())
    return (np.ascontiguousarray(u * s), np.ascontiguousarray(v * s), np.ascontiguousarray(w * s))


_NNNNND = (BC_NEUMANN,) * 5 + (BC_DIRICHLET,)   # p_nh: walls on sides/bottom, open top


def config1(n=32, levels=4):
    """32^3, constant coefficient, zero Dirichlet, b ~ U[-1,1] mean-free, seed 1001."""
    w = Workload("config1_const_dirichlet", n, n, n, 1.0 / n, levels, (BC_DIRICHLET,) * 6, tol=1e-8)
    b = rng.uniform(1001, w.n).reshape(w.shape)
    w.fields["b"] = np.ascontiguousarray(b - b.mean())
    return w


def config2(n=128, levels=6):
    """128^3 water column, variable coefficient, RHS source velocity seeds 2001-2003."""
    w = Workload("config2_water_column", n, n, n, 1.0 / n, levels, _NNNNND, tol=1e-7)
    w.fields["alpha"] = water_column_alpha(n, n, n, w.h, 2.0)
    w.fields["u"], w.fields["v"], w.fields["w"] = random_velocity((2001, 2002, 2003), w.shape)
    return w


def config3(n=256, levels=7):
    """256^3 rising bubble, radius 0.125 at (0.5,0.5,0.25), seeds 3001-3003."""
    w = Workload("config3_rising_bubble", n, n, n, 1.0 / n, levels, _NNNNND, tol=1e-7)
    w.fields["alpha"] = bubble_alpha(n, n, n, w.h, [(0.5, 0.5, 0.25)], 0.125, 1.5)
    w.fields["u"], w.fields["v"], w.fields["w"] = random_velocity((3001, 3002, 3003), w.shape)
    return w


def config4(nx=512, ny=512, nz=256, levels=7):
    """512x512x256, four bubbles of radius 0.06 (centres seed 4000), seeds 4001-4003."""
    h = 1.0 / nx
    w = Workload("config4_four_bubbles", nx, ny, nz, h, levels, _NNNNND, tol=1e-7)
    zs = nz * h
    cs = bubble_centres(4000, 4, 0.06, 0.02, (0.1, 0.1, 0.2 * zs), (0.9, 0.9, 0.8 * zs))
    w.fields["alpha"] = bubble_alpha(nx, ny, nz, h, cs, 0.06, 1.5)
    w.fields["u"], w.fields["v"], w.fields["w"] = random_velocity((4001, 4002, 4003), w.shape)
    return w


def config5(n=256, levels=7):
    """Full time step on 256^3: water-column alpha, solenoidal q (seeds 5001-5003), dt = 0.1 h."""
    w = Workload("config5_time_step", n, n, n, 1.0 / n, levels, _NNNNND, tol=1e-6)
    w.dt = 0.1 * w.h
    w.fields["alpha"] = water_column_alpha(n, n, n, w.h, 2.0)
    w.fields["u"], w.fields["v"], w.fields["w"] = solenoidal_velocity((5001, 5002, 5003), n, n, n, w.h)
    return w


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
