"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no kernel G_k, no treecode,
no convolution): it only makes quadrature meshes, weights, fields f = V*psi and
parameters shaped like the paper's workloads.  Both `oracle/` (through the
tests) and the CUDA library consume its output; neither imports the other.

What stands in for what ("Input recipe"):
  * Chebyshev points of the first kind, Eq. (15), with Fejer's
    first rule for the weights (formula from refs [50,51], which
    the paper does not print -- reading R14 in DESIGN.md).
  * The paper's adaptive meshes come from Eq. (16)-(17) refinement on radial
    atomic data that is not available; BASELINE.json's
    geometric rule "refine a cell of edge h while h > 0.35*max(d, 0.05)" stands
    in for it.  (p+1)^3 points per cell, N_m = (p+1)^3 N_c.
  * Atom positions for CO: PAPER.md:522 (C on the negative z axis).

Everything is numpy float64, deterministic, seed = 20030183 + config index.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 20030183


# --------------------------------------------------------------------------
# quadrature: Chebyshev-1 points + Fejer-1 weights on [-1, 1]
# --------------------------------------------------------------------------
def fejer1(npts: int):
    """Nodes x_i = cos((2i+1)pi/(2n)), i=0..n-1 (Eq. (15), n=p+1) and
    Fejer first-rule weights w_i = (2/n)[1 - 2 sum_{m=1..floor(n/2)} cos(2 m th_i)/(4m^2-1)]."""
    n = int(npts)
    i = np.arange(n, dtype=np.float64)
    th = (2.0 * i + 1.0) * math.pi / (2.0 * n)
    x = np.cos(th)
    w = np.ones(n, dtype=np.float64)
    for m in range(1, n // 2 + 1):
        w -= 2.0 * np.cos(2.0 * m * th) / (4.0 * m * m - 1.0)
    w *= 2.0 / n
    return x, w


def _points_in_cells(cx, cy, cz, h, npts):
    """Tensor (npts)^3 Fejer grid in every cubic cell (centre c, edge h).  Returns x,y,z,w."""
    t, wt = fejer1(npts)
    half = 0.5 * h[:, None]
    # per-axis coordinates [ncell, npts]
    ax = cx[:, None] + half * t[None, :]
    ay = cy[:, None] + half * t[None, :]
    az = cz[:, None] + half * t[None, :]
    aw = half * wt[None, :]
    nc = cx.shape[0]
    x = np.broadcast_to(ax[:, :, None, None], (nc, npts, npts, npts)).reshape(-1)
    y = np.broadcast_to(ay[:, None, :, None], (nc, npts, npts, npts)).reshape(-1)
    z = np.broadcast_to(az[:, None, None, :], (nc, npts, npts, npts)).reshape(-1)
    w = (aw[:, :, None, None] * aw[:, None, :, None] * aw[:, None, None, :]).reshape(-1)
    return (np.ascontiguousarray(x), np.ascontiguousarray(y),
            np.ascontiguousarray(z), np.ascontiguousarray(w))


def uniform_cells(L: float, cells_per_axis: int):
    """Cell centres/edges of a uniform cells_per_axis^3 tiling of [-L, L]^3."""
    m = int(cells_per_axis)
    h = 2.0 * L / m
    c = -L + h * (np.arange(m, dtype=np.float64) + 0.5)
    cx, cy, cz = np.meshgrid(c, c, c, indexing="ij")
    cx, cy, cz = cx.reshape(-1), cy.reshape(-1), cz.reshape(-1)
    return cx, cy, cz, np.full(cx.shape, h)


def adaptive_cells(L: float, nuclei, c_ref: float = 0.35, d_min: float = 0.05,
                   max_level: int = 40):
    """Octree cells over [-L, L]^3: a cell of edge h is bisected in all three directions
    while h > c_ref * max(d, d_min), d = distance from the cell centre to the nearest nucleus
    (BASELINE.json configs 1-3; stands in for PAPER.md:167-181 Eq. (16)-(17))."""
    nuc = np.asarray(nuclei, dtype=np.float64).reshape(-1, 3)
    cx = np.array([0.0]); cy = np.array([0.0]); cz = np.array([0.0])
    h = 2.0 * L
    out = []
    off = np.array([-0.25, 0.25])
    ox, oy, oz = np.meshgrid(off, off, off, indexing="ij")
    ox, oy, oz = ox.reshape(-1), oy.reshape(-1), oz.reshape(-1)
    for _ in range(max_level):
        if cx.size == 0:
            break
        d = np.full(cx.shape, np.inf)
        for a in range(nuc.shape[0]):
            d = np.minimum(d, np.sqrt((cx - nuc[a, 0]) ** 2 + (cy - nuc[a, 1]) ** 2
                                      + (cz - nuc[a, 2]) ** 2))
        refine = h > c_ref * np.maximum(d, d_min)
        keep = ~refine
        if keep.any():
            out.append((cx[keep], cy[keep], cz[keep], np.full(int(keep.sum()), h)))
        px, py, pz = cx[refine], cy[refine], cz[refine]
        cx = (px[:, None] + h * ox[None, :]).reshape(-1)
        cy = (py[:, None] + h * oy[None, :]).reshape(-1)
        cz = (pz[:, None] + h * oz[None, :]).reshape(-1)
        h *= 0.5
    if cx.size:
        raise RuntimeError("adaptive_cells: max_level reached")
    return tuple(np.concatenate([o[i] for o in out]) for i in range(4))


def mesh_from_cells(cells, npts: int = 4):
    cx, cy, cz, h = cells
    return _points_in_cells(cx, cy, cz, h, npts)


# --------------------------------------------------------------------------
# fields
# --------------------------------------------------------------------------
def _erf(a):
    # vectorised erf without scipy dependency at import time
    from scipy.special import erf
    return erf(a)


def _dist(x, y, z, c):
    return np.sqrt((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2)


def screened_potential(x, y, z, nuclei, charges):
    """V = sum_a [ -Z_a/r_a + (Z_a - 1) erf(r_a)/r_a ]  (reading R17: "smooth Gaussian screening")."""
    v = np.zeros_like(x)
    for c, Z in zip(nuclei, charges):
        r = _dist(x, y, z, c)
        v += -Z / r + (Z - 1.0) * _erf(r) / r
    return v


def random_orbitals(rng, x, y, z, nuclei, charges, n_orb):
    """Seeded sums over nuclei of c e^{-alpha r_a} + d e^{-beta r_a^2},
    c,d ~ U(-1,1), alpha ~ U(0.8, Z_a), beta ~ U(0.2, 2)."""
    psi = np.zeros((n_orb, x.shape[0]))
    rs = [_dist(x, y, z, c) for c in nuclei]
    for o in range(n_orb):
        for r, Z in zip(rs, charges):
            c_, d_ = rng.uniform(-1.0, 1.0, size=2)
            alpha = rng.uniform(0.8, max(Z, 0.8 + 1e-9))
            beta = rng.uniform(0.2, 2.0)
            psi[o] += c_ * np.exp(-alpha * r) + d_ * np.exp(-beta * r * r)
    return psi


# --------------------------------------------------------------------------
# configs
# --------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    w: np.ndarray
    f: np.ndarray            # [n_orb, N]
    k: np.ndarray            # [n_orb]
    theta: float
    degree: int
    leaf_size: int
    batch_size: int
    subtract: bool = True
    meta: dict = field(default_factory=dict)

    @property
    def N(self):
        return int(self.x.shape[0])

    @property
    def n_orb(self):
        return int(self.f.shape[0])

    def coords(self):
        """SoA double[3][N] as the C ABI wants it."""
        return np.ascontiguousarray(np.stack([self.x, self.y, self.z]))


def hydrogen_fields(x, y, z):
    """psi = e^{-r}/sqrt(pi), V = -1/r, f = V*psi (BASELINE.json config 0)."""
    r = np.sqrt(x * x + y * y + z * z)
    psi = np.exp(-r) / math.sqrt(math.pi)
    return psi, (-1.0 / r) * psi


def config0(leaf_size=2000, batch_size=2000, theta=0.7, degree=8, cells_per_axis=8, L=8.0):
    x, y, z, w = mesh_from_cells(uniform_cells(L, cells_per_axis), 4)
    psi, f = hydrogen_fields(x, y, z)
    return Workload("cfg0_hydrogen_uniform", x, y, z, w, f[None, :].copy(), np.array([1.0]),
                    theta, degree, leaf_size, batch_size, True,
                    {"psi": psi, "L": L, "cells": cells_per_axis ** 3})


def hydrogen_adaptive(L=20.0):
    """Config-1 geometry with Z=1: the mesh on which the hydrogen <=1e-3 pin is attainable
    (reading R19)."""
    cells = adaptive_cells(L, [(0.0, 0.0, 0.0)])
    x, y, z, w = mesh_from_cells(cells, 4)
    psi, f = hydrogen_fields(x, y, z)
    return Workload("hydrogen_adaptive", x, y, z, w, f[None, :].copy(), np.array([1.0]),
                    0.7, 8, 2000, 2000, True, {"psi": psi, "L": L, "cells": cells[0].shape[0]})


def config1(leaf_size=2000, batch_size=2000, theta=0.7, degree=8):
    nuclei = [(0.0, 0.0, 0.0)]
    cells = adaptive_cells(20.0, nuclei)
    x, y, z, w = mesh_from_cells(cells, 4)
    r = np.sqrt(x * x + y * y + z * z)
    V = -4.0 / r + 3.0 * _erf(r) / r
    psi = np.stack([np.exp(-3.7 * r), np.exp(-1.0 * r)])
    eps = np.array([-3.86, -0.21])
    return Workload("cfg1_be_like", x, y, z, w, V[None, :] * psi, np.sqrt(-2.0 * eps),
                    theta, degree, leaf_size, batch_size, True,
                    {"cells": cells[0].shape[0], "eps": eps, "psi": psi})


def config2(leaf_size=2000, batch_size=2000, theta=0.7, degree=8):
    nuclei = [(0.0, 0.0, -1.066), (0.0, 0.0, 1.066)]
    charges = [6.0, 8.0]
    rng = np.random.default_rng(SEED_BASE + 2)
    cells = adaptive_cells(20.0, nuclei)
    x, y, z, w = mesh_from_cells(cells, 4)
    V = screened_potential(x, y, z, nuclei, charges)
    psi = random_orbitals(rng, x, y, z, nuclei, charges, 7)
    eps = np.sort(rng.uniform(-19.0, -0.3, size=7))
    return Workload("cfg2_co_like", x, y, z, w, V[None, :] * psi, np.sqrt(-2.0 * eps),
                    theta, degree, leaf_size, batch_size, True,
                    {"cells": cells[0].shape[0], "eps": eps, "psi": psi})


def config3(leaf_size=2000, batch_size=2000, theta=0.7, degree=8, n_orb=21):
    nuclei, charges = [], []
    for m in range(6):
        a = math.pi / 3.0 * m
        nuclei.append((2.64 * math.cos(a), 2.64 * math.sin(a), 0.0)); charges.append(6.0)
    for m in range(6):
        a = math.pi / 3.0 * m
        nuclei.append((4.69 * math.cos(a), 4.69 * math.sin(a), 0.0)); charges.append(1.0)
    rng = np.random.default_rng(SEED_BASE + 3)
    cells = adaptive_cells(24.0, nuclei)
    x, y, z, w = mesh_from_cells(cells, 4)
    V = screened_potential(x, y, z, nuclei, charges)
    psi = random_orbitals(rng, x, y, z, nuclei, charges, n_orb)
    eps = np.sort(rng.uniform(-10.0, -0.2, size=n_orb))
    return Workload("cfg3_c6h6_like", x, y, z, w, V[None, :] * psi, np.sqrt(-2.0 * eps),
                    theta, degree, leaf_size, batch_size, True,
                    {"cells": cells[0].shape[0], "eps": eps, "psi": psi})


def config4(N=1_000_000, k=1.0, theta=0.7, degree=8, leaf_size=2000, batch_size=2000,
            subtract=False, seed_offset=4):
    """Uniform random points in the unit cube, w ~ U(0,1)/N, f ~ U(-1,1)  (BASELINE.json config 4;
    the single-GPU Yukawa analogue of PAPER.md:494-500 Fig. 11)."""
    rng = np.random.default_rng(SEED_BASE + seed_offset)
    x, y, z = rng.random(N), rng.random(N), rng.random(N)
    w = rng.random(N) / N
    f = rng.uniform(-1.0, 1.0, size=(1, N))
    return Workload(f"cfg4_random_N{N}", x, y, z, w, f, np.array([float(k)]),
                    theta, degree, leaf_size, batch_size, subtract, {})


def random_cloud(N, n_orb=1, seed=0, k=None, clustered=False, **kw):
    """Small seeded test clouds (parity cases spanning several tiles and a ragged tail)."""
    rng = np.random.default_rng(SEED_BASE + 1000 + seed)
    if clustered:
        c = rng.random((max(1, N // 200), 3))
        idx = rng.integers(0, c.shape[0], size=N)
        p = c[idx] + 0.03 * rng.standard_normal((N, 3))
        x, y, z = p[:, 0].copy(), p[:, 1].copy(), p[:, 2].copy()
    else:
        x, y, z = rng.random(N), rng.random(N), rng.random(N)
    w = rng.random(N) / max(N, 1)
    f = rng.uniform(-1.0, 1.0, size=(n_orb, N))
    kk = np.asarray(k, dtype=np.float64) if k is not None else rng.uniform(0.5, 5.0, size=n_orb)
    return Workload(f"cloud_N{N}_s{seed}", x, y, z, w, f, kk,
                    kw.get("theta", 0.7), kw.get("degree", 8), kw.get("leaf_size", 2000),
                    kw.get("batch_size", 2000), kw.get("subtract", True), {})


def density_workload(c):
    """The same mesh with ONE field: the electron density rho = 2 sum_o psi_o^2 / int psi_o^2 of the config's
    orbitals (doubly occupied, quadrature-normalised) -- the input of the Hartree-potential convolution
    (Eq. (19); the workload shape of PAPER.md:482-490 Table 4).  k is unused by that kernel."""
    psi = np.atleast_2d(c.meta["psi"])
    rho = np.zeros(c.N)
    for o in range(psi.shape[0]):
        rho += 2.0 * psi[o] ** 2 / float((c.w * psi[o] ** 2).sum())
    return Workload(c.name + "_density", c.x, c.y, c.z, c.w, rho[None, :].copy(), c.k[:1].copy(),
                    c.theta, c.degree, c.leaf_size, c.batch_size, True, dict(c.meta))


def sample_targets(N, n, seed=0):
    """Seeded sorted sample of target indices (for sampled parity at full sizes)."""
    rng = np.random.default_rng(SEED_BASE + 2000 + seed)
    n = min(n, N)
    return np.sort(rng.choice(N, size=n, replace=False)).astype(np.int64)


CONFIGS = {0: config0, 1: config1, 2: config2, 3: config3, 4: config4}
