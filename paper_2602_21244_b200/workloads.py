"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 1-5).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: no Philox, no pairing, no operator, no moments -- only numpy's own
seeded generator, Maxwellian sampling and cell layouts.  It imports neither ``oracle`` nor
the CUDA binding.  Recipes are stated in DESIGN.md ("Input recipe"); the populations are
stand-ins for the paper's Couette, cavity and Mach-10 cylinder
 flows, whose particle data are not available.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

KB = 1.380649e-23
MASS_AR = 6.63e-26  # kg
ACT_TANH, ACT_RELU, ACT_SILU = 0, 1, 2


@dataclass
class Population:
    name: str
    n_cells: int
    cell: np.ndarray  # int32 [n], UNSORTED order (binning has real work to do)
    vx: np.ndarray    # float32 [n]
    vy: np.ndarray
    vz: np.ndarray
    counts: np.ndarray  # int64 [n_cells]

    @property
    def n(self):
        return int(self.cell.shape[0])

    def pairs_per_step(self, pairs_per_cell: int) -> int:
        half = self.counts // 2
        if pairs_per_cell < 0:
            return int(half.sum())
        return int(np.minimum(half, pairs_per_cell).sum())


def _scatter_index(n: int) -> np.ndarray:
    """Bijection p -> (p*1000003 + 12345) mod n used to un-sort the cell-sorted layout."""
    a = 1000003
    while np.gcd(a, n) != 1:
        a += 2
    return ((np.arange(n, dtype=np.int64) * a + 12345) % n).astype(np.int64)


def _populate(name, counts, T_cell, ux_cell, uy_cell, seed, shuffle=True) -> Population:
    counts = np.asarray(counts, np.int64)
    K = counts.shape[0]
    n = int(counts.sum())
    cell_sorted = np.repeat(np.arange(K, dtype=np.int32), counts)
    rng = np.random.default_rng(seed)
    sig = np.sqrt(KB * np.asarray(T_cell, np.float64) / MASS_AR)[cell_sorted]
    vx = (np.asarray(ux_cell, np.float64)[cell_sorted] + sig * rng.standard_normal(n)).astype(np.float32)
    vy = (np.asarray(uy_cell, np.float64)[cell_sorted] + sig * rng.standard_normal(n)).astype(np.float32)
    vz = (sig * rng.standard_normal(n)).astype(np.float32)
    if shuffle and n > 0:
        dst = _scatter_index(n)
        cell = np.empty_like(cell_sorted)
        cell[dst] = cell_sorted
        out = []
        for v in (vx, vy, vz):
            w = np.empty_like(v)
            w[dst] = v
            out.append(w)
        vx, vy, vz = out
    else:
        cell = cell_sorted
    return Population(name, K, cell, vx, vy, vz, counts)


def tiny_box(seed=0, n_cells=64, per_cell=100, T=273.0) -> Population:
    """cfg 1: 64 cells x 100 argon particles, Maxwellian 273 K, zero drift."""
    K = n_cells
    return _populate("tiny_vhs_box", np.full(K, per_cell), np.full(K, T), np.zeros(K), np.zeros(K), seed)


def couette(seed=1, n_cells=200, per_cell=1000, T=273.0, U=250.0) -> Population:
    """cfg 2: linear drift u_x from -U to +U across cells."""
    K = n_cells
    ux = -U + 2.0 * U * (np.arange(K) + 0.5) / K
    return _populate("couette_1d", np.full(K, per_cell), np.full(K, T), ux, np.zeros(K), seed)


def cavity(seed=2, nx=100, ny=100, per_cell=100, T=273.0, U0=50.0) -> Population:
    """cfg 3: single-vortex drift u=U0 sin(pi x)cos(pi y), v=-U0 cos(pi x)sin(pi y); cell id = ix*ny+iy."""
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    X, Y = np.meshgrid(x, y, indexing="ij")
    ux = (U0 * np.sin(np.pi * X) * np.cos(np.pi * Y)).ravel()
    uy = (-U0 * np.cos(np.pi * X) * np.sin(np.pi * Y)).ravel()
    K = nx * ny
    return _populate("cavity_2d", np.full(K, per_cell), np.full(K, T), ux, uy, seed)


def mach10_cylinder(seed=4, nx=400, ny=200, n_total=20_000_000) -> Population:
    """cfg 5: freestream 200 K / 2640 m/s, shocked band 7000 K at 4x density, wake 1000 K at
    0.25x density, empty body disc.  Geometry scales with (nx, ny) so reduced sizes keep the
    same cell-size mix; n_total is met exactly."""
    sx, sy = nx / 400.0, ny / 200.0
    ix = np.arange(nx)[:, None] + 0.5
    iy = np.arange(ny)[None, :] + 0.5
    cx, cy = 160.0 * sx, 100.0 * sy
    r = np.sqrt(((ix - cx) / sx) ** 2 + ((iy - cy) / sy) ** 2)
    body = r < 30.0
    shock = (r >= 30.0) & (r < 70.0) & (ix < cx)
    wake = (~body) & (~shock) & (ix >= cx) & (np.abs(iy - cy) / sy < 30.0)
    weight = np.full((nx, ny), 4, np.int64)  # freestream
    T = np.full((nx, ny), 200.0)
    ux = np.full((nx, ny), 2640.0)
    weight[shock], T[shock], ux[shock] = 16, 7000.0, 660.0
    weight[wake], T[wake], ux[wake] = 1, 1000.0, 0.0
    weight[body], T[body], ux[body] = 0, 200.0, 0.0
    w = weight.ravel()
    counts = (n_total * w) // int(w.sum())
    rem = n_total - int(counts.sum())
    nonempty = np.flatnonzero(w > 0)
    counts[nonempty[:rem]] += 1
    return _populate("mach10_cylinder", counts, T.ravel(), ux.ravel(), np.zeros(nx * ny), seed)


def abinitio_pair_batch(seed=3, n=10_000_000, T=7000.0, b_max=1e-9):
    """cfg 4: E_r/k_B [K] from a 7000 K Maxwellian relative-speed distribution, b = b_max sqrt(U)."""
    rng = np.random.default_rng(seed)
    z2 = (rng.standard_normal((n, 3)) ** 2).sum(axis=1)
    # g_a ~ N(0, 2 kB T/m) per component => E_r/kB = m g^2/(4 kB) = T |z|^2 / 2  (mu = m/2)
    E_over_k = (0.5 * T * z2).astype(np.float32)
    b = (b_max * np.sqrt(rng.random(n))).astype(np.float32)
    return E_over_k, b


def random_mlp(seed, dims, scale=1.0):
    """Random-init MLP: W, b ~ U(-1,1)/sqrt(fan_in), float32 (BASELINE.json 'random-init')."""
    rng = np.random.default_rng(1000 + seed)
    Ws, bs = [], []
    for l in range(len(dims) - 1):
        fan_in = dims[l]
        Ws.append(((2.0 * rng.random((dims[l + 1], dims[l])) - 1.0) * scale / np.sqrt(fan_in)).astype(np.float32))
        bs.append(((2.0 * rng.random(dims[l + 1]) - 1.0) / np.sqrt(fan_in)).astype(np.float32))
    return Ws, bs


SIGMA_V = float(np.sqrt(2.0 * KB * 273.0 / MASS_AR))  # global velocity scale
