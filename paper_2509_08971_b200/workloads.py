"""Seeded synthetic inputs for the five BASELINE.json configs (C0..C4).

This module serves BOTH the CUDA path and the oracle (tests, bench).  It holds none of the method's
arithmetic: it only builds initial conserved fields (rho, mx, my, mz, E) of PAPER.md P:93 eq.2 from
primitive initial data, as float64 arrays of shape (nz, ny, nx), x fastest.  Recipe: DESIGN.md
"Input recipe" (readings G12-G14).  It imports neither the CUDA binding nor oracle/.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

BC_PERIODIC = 0
BC_OUTFLOW = 1
BC_REFLECT = 2
_M64 = (1 << 64) - 1


@dataclass
class Workload:
    name: str
    n: tuple            # (nx, ny, nz)
    gamma: float
    bc: int
    spacing: tuple      # (dx, dy, dz)
    cfl: float
    t_end: float | None = None      # "run to t" configs
    nsteps: int | None = None       # fixed-step configs
    state: list | None = None       # [rho, mx, my, mz, E], numpy (nz,ny,nx) or torch device tensors
    meta: dict = field(default_factory=dict)


def _cons(rho, u, v, w, p, gamma):
    E = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)
    return [rho, rho * u, rho * v, rho * w, E]


def shock_tube(name, n, x_lo, x_hi, x0, left, right, gamma, cfl, t_end):
    """1-D Riemann problem; left/right = (rho, u, p); cells with centre < x0 take the left state
    (G12).  Sod: eq.20."""
    dx = (x_hi - x_lo) / n
    xc = x_lo + (np.arange(n) + 0.5) * dx
    m = xc < x0
    rho = np.where(m, left[0], right[0]).astype(np.float64)
    u = np.where(m, left[1], right[1]).astype(np.float64)
    p = np.where(m, left[2], right[2]).astype(np.float64)
    z = np.zeros(n)
    st = [a.reshape(1, 1, n) for a in _cons(rho, u, z, z, p, gamma)]
    return Workload(name, (n, 1, 1), gamma, BC_OUTFLOW, (dx, 1.0, 1.0), cfl, t_end=t_end, state=st,
                    meta={"x_lo": x_lo, "x0": x0, "left": left, "right": right})


def sod(n=1000, t_end=0.2, cfl=0.4):
    """C0 (BASELINE.json configs[0])."""
    return shock_tube("sod", n, 0.0, 1.0, 0.5, (1.0, 0.0, 1.0), (0.125, 0.0, 0.1), 1.4, cfl, t_end)


def leblanc(n=4096, t_end=6.0, cfl=0.3):
    """C1 (configs[1]): specific internal energies 0.1 / 1e-7, p = (gamma-1) rho e."""
    g = 5.0 / 3.0
    return shock_tube("leblanc", n, 0.0, 9.0, 3.0, (1.0, 0.0, (g - 1.0) * 1.0 * 0.1),
                      (1e-3, 0.0, (g - 1.0) * 1e-3 * 1e-7), g, cfl, t_end)


def sedov(n=128, t_end=0.05, cfl=0.3, E0=1.0):
    """C2 (configs[2]): [-1,1]^3, rho=1, p=1e-5, E0 spread as internal energy over the cells whose
    centre radius is < 2 dx (G13: 32 cells for even n)."""
    g = 1.4
    dx = 2.0 / n
    xc = -1.0 + (np.arange(n) + 0.5) * dx
    Z, Y, X = np.meshgrid(xc, xc, xc, indexing="ij")
    hot = (X * X + Y * Y + Z * Z) < (2.0 * dx) ** 2
    nhot = int(hot.sum())
    rho = np.ones((n, n, n))
    E = np.full((n, n, n), 1e-5 / (g - 1.0))
    E[hot] = E0 / (nhot * dx ** 3)
    z = np.zeros((n, n, n))
    return Workload("sedov", (n, n, n), g, BC_OUTFLOW, (dx, dx, dx), cfl, t_end=t_end,
                    state=[rho, z.copy(), z.copy(), z.copy(), E], meta={"nhot": nhot, "E0": E0})


class SplitMix64:
    def __init__(self, seed):
        self.s = seed & _M64

    def next(self):
        self.s = (self.s + 0x9E3779B97F4A7C15) & _M64
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
        return z ^ (z >> 31)


def sine_modes(seed=12345):
    """4 fields x 8 modes of (kx,ky,kz,phase): integer wavevectors, k != 0, |k|^2 <= 16."""
    rng = SplitMix64(seed)
    modes = []
    for _f in range(4):
        fm = []
        for _m in range(8):
            while True:
                k = [int(rng.next() % 9) - 4 for _ in range(3)]
                k2 = k[0] ** 2 + k[1] ** 2 + k[2] ** 2
                if 0 < k2 <= 16:
                    break
            phi = 2.0 * np.pi * ((rng.next() >> 11) * 2.0 ** -53)
            fm.append((k[0], k[1], k[2], phi))
        modes.append(fm)
    return modes


def _mode_sum(xp, modes, X, Y, Z):
    acc = None
    for (kx, ky, kz, phi) in modes:
        t = xp.sin(2.0 * np.pi * (kx * X + ky * Y + kz * Z) + phi)
        acc = t if acc is None else acc + t
    return acc


def turbulence(n=512, nsteps=20, cfl=0.4, seed=12345, device=None, slab=64):
    """C3 / C4 (configs[3], [4]): periodic [0,1)^3, gamma=1.4, rho = 1 + 0.1 sum_8 sin, velocity =
    s * sum_8 sin per component with RMS speed = 0.1 sqrt(gamma) (RMS Mach 0.1 at rho=1, p=1), p=1.
    device=None -> numpy; otherwise torch tensors built slab by slab on that device."""
    g = 1.4
    modes = sine_modes(seed)
    d = 1.0 / n
    if device is None:
        xc = (np.arange(n) + 0.5) * d
        Z, Y, X = np.meshgrid(xc, xc, xc, indexing="ij")
        rho = 1.0 + 0.1 * _mode_sum(np, modes[0], X, Y, Z)
        vel = [_mode_sum(np, modes[1 + c], X, Y, Z) for c in range(3)]
        rms = np.sqrt(np.mean(vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2))
        s = 0.1 * np.sqrt(g) / rms
        st = _cons(rho, s * vel[0], s * vel[1], s * vel[2], np.ones_like(rho), g)
    else:
        import torch
        xc = (torch.arange(n, device=device, dtype=torch.float64) + 0.5) * d
        st = [torch.empty((n, n, n), device=device, dtype=torch.float64) for _ in range(5)]
        ssq = torch.zeros((), device=device, dtype=torch.float64)
        # pass 1: unscaled velocities into st[1..3], rho into st[0]; pass 2: scale, build m and E
        for k0 in range(0, n, slab):
            k1 = min(n, k0 + slab)
            Z, Y, X = torch.meshgrid(xc[k0:k1], xc, xc, indexing="ij")
            st[0][k0:k1] = 1.0 + 0.1 * _mode_sum(torch, modes[0], X, Y, Z)
            for c in range(3):
                v = _mode_sum(torch, modes[1 + c], X, Y, Z)
                st[1 + c][k0:k1] = v
                ssq += (v * v).sum()
            del X, Y, Z, v
        s = 0.1 * np.sqrt(g) / float(torch.sqrt(ssq / float(n) ** 3))
        for k0 in range(0, n, slab):
            k1 = min(n, k0 + slab)
            rho = st[0][k0:k1]
            ke = torch.zeros_like(rho)
            for c in range(3):
                v = st[1 + c][k0:k1] * s
                ke += v * v
                st[1 + c][k0:k1] = rho * v
            st[4][k0:k1] = 1.0 / (g - 1.0) + 0.5 * rho * ke
            del ke, v
    return Workload("turb%d" % n, (n, n, n), g, BC_PERIODIC, (d, d, d), cfl, nsteps=nsteps, state=st,
                    meta={"seed": seed, "modes": modes})


def kelvin_helmholtz(n=256, t_end=None, nsteps=100, cfl=0.4, gamma=1.4, p0=2.5, amp=0.01):
    """NEXT-2: non-radiative panel of the paper's 2-D Kelvin-Helmholtz run:
    [-0.5,0.5]^2, rho_low = 1, rho_high = 2.5 in the layer |y| <= 0.25, v_x = -0.5 in the layer and +0.5
    elsewhere.  The paper gives neither pressure, gamma, grid, boundaries nor the seed perturbation
    (G18): p = 2.5, gamma = 1.4, periodic, n x n x 1, v_y = amp sin(4 pi x) (exp(-(y-1/4)^2/s^2)
    + exp(-(y+1/4)^2/s^2)), s = 0.05."""
    d = 1.0 / n
    xc = -0.5 + (np.arange(n) + 0.5) * d
    Y, X = np.meshgrid(xc, xc, indexing="ij")
    layer = np.abs(Y) <= 0.25
    rho = np.where(layer, 2.5, 1.0)
    u = np.where(layer, -0.5, 0.5)
    s2 = 0.05 ** 2
    v = amp * np.sin(4.0 * np.pi * X) * (np.exp(-(Y - 0.25) ** 2 / s2) + np.exp(-(Y + 0.25) ** 2 / s2))
    p = np.full_like(rho, p0)
    z = np.zeros_like(rho)
    st = [a.reshape(1, n, n) for a in _cons(rho, u, v, z, p, gamma)]
    return Workload("kh%d" % n, (n, n, 1), gamma, BC_PERIODIC, (d, d, 1.0), cfl, t_end=t_end, nsteps=nsteps, state=st)


def random_state(n, seed, gamma=1.4, amp=0.3):
    """Generic positive random state on an (nx,ny,nz) grid for invariant / parity tests."""
    nx, ny, nz = n
    rng = np.random.default_rng(seed)
    rho = 1.0 + amp * (rng.random((nz, ny, nx)) - 0.5)
    p = 1.0 + amp * (rng.random((nz, ny, nx)) - 0.5)
    vel = [amp * (rng.random((nz, ny, nx)) - 0.5) for _ in range(3)]
    return _cons(rho, vel[0], vel[1], vel[2], p, gamma)
