"""Seeded synthetic inputs for the lens-map hot path (BASELINE.json configs 0-4).

This module is the ONLY thing the CPU oracle (`oracle/`) and the CUDA path
(`paper_2004_06352_b200/`) have in common.  It holds none of the method's
arithmetic: it draws lens parameters and grid geometry with
``numpy.random.default_rng(seed)`` in a fixed order (recipe: SURVEY.md §8(d),
restated in DESIGN.md §4) and hands out plain numpy arrays.  The only formula in
here is the unit conversion sigma -> b0 that BASELINE.json's configs state
(b0 = (D_ls/D_s) * 6*pi*(sigma/c)^2 in arcsec, reading §8c-4) -- it builds an
INPUT of the method, not part of it.

The paper's workloads (M1149: 217 potentials on 5000x5000 px, §5;
Abell 2744: 258 potentials, 6000x6000 px, 10014 maps, §2.4) are not
available; these configs take their shape (a few cluster-scale halos + hundreds
of galaxy-scale potentials, 1e6-1e7 pixels, many maps) and stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

# Lens types at the boundary (include/lh.h)
DPIE, NSIE, SIS = 0, 1, 2

# 64-byte AoS record == `lh_lens` in include/lh.h (and the oracle's own declaration)
LENS_DTYPE = np.dtype(
    [
        ("type", "<i4"),
        ("_pad", "<i4"),
        ("x", "<f8"),
        ("y", "<f8"),
        ("ellipticity", "<f8"),
        ("theta", "<f8"),
        ("rcore", "<f8"),
        ("rcut", "<f8"),
        ("b0", "<f8"),
    ],
    align=False,
)
assert LENS_DTYPE.itemsize == 64

C_KMS = 299792.458
ARCSEC_PER_RAD = 648000.0 / np.pi


def b0_from_sigma(sigma_kms, dls_over_ds=0.5):
    """b0 [arcsec] = (D_ls/D_s) * 6*pi*(sigma/c)^2 (radians -> arcsec)."""
    return dls_over_ds * 6.0 * np.pi * (np.asarray(sigma_kms, dtype=np.float64) / C_KMS) ** 2 * ARCSEC_PER_RAD


@dataclass(frozen=True)
class Grid:
    """Pixel (i, j) sits at (x0 + i*dx, y0 + j*dx); plane index = j*nx + i."""

    x0: float
    y0: float
    dx: float
    nx: int
    ny: int

    @property
    def npix(self) -> int:
        return self.nx * self.ny

    def xs(self):
        return self.x0 + np.arange(self.nx, dtype=np.float64) * self.dx

    def ys(self):
        return self.y0 + np.arange(self.ny, dtype=np.float64) * self.dx


def centred_grid(half_width: float, n: int) -> Grid:
    """n x n pixels spanning +/-half_width, pixel-centre sampling (reading §8c-10)."""
    dx = 2.0 * half_width / n
    x0 = -half_width + 0.5 * dx
    return Grid(x0=x0, y0=x0, dx=dx, nx=n, ny=n)


def make_lenses(n: int) -> np.ndarray:
    return np.zeros(n, dtype=LENS_DTYPE)


def lens(type_=DPIE, x=0.0, y=0.0, ellipticity=0.0, theta=0.0, rcore=0.0, rcut=0.0, b0=0.0) -> np.ndarray:
    """One-element lens array (convenience for tests)."""
    a = make_lenses(1)
    a[0] = (type_, 0, x, y, ellipticity, theta, rcore, rcut, b0)
    return a


def _draw_halos(rng, nh: int, out: np.ndarray, off: int):
    for h in range(nh):
        r = 20.0 * np.sqrt(rng.random())
        phi = 2.0 * np.pi * rng.random()
        e = rng.uniform(0.2, 0.6)
        th = rng.uniform(0.0, np.pi)
        rc = rng.uniform(5.0, 20.0)
        rt = 1000.0
        sig = rng.uniform(800.0, 1200.0)
        out[off + h] = (DPIE, 0, r * np.cos(phi), r * np.sin(phi), e, th, rc, rt, b0_from_sigma(sig))


def _draw_galaxies(rng, ng: int, hc: float, out: np.ndarray, off: int, types=None):
    for g in range(ng):
        x = rng.uniform(-hc, hc)
        y = rng.uniform(-hc, hc)
        e = rng.uniform(0.0, 0.6)
        th = rng.uniform(0.0, np.pi)
        rc = rng.uniform(0.01, 0.1)
        rt = rng.uniform(5.0, 50.0)
        sig = rng.uniform(50.0, 300.0)
        t = DPIE if types is None else types(g)
        out[off + g] = (t, 0, x, y, e, th, rc, rt, b0_from_sigma(sig))


def cluster(seed: int, nhalo: int, ngal: int, hc: float, types=None, return_rng=False):
    """`nhalo` cluster-scale dPIE halos first, then `ngal` galaxy-scale potentials."""
    rng = np.random.default_rng(seed)
    out = make_lenses(nhalo + ngal)
    _draw_halos(rng, nhalo, out, 0)
    _draw_galaxies(rng, ngal, hc, out, nhalo, types)
    return (out, rng) if return_rng else out


def _cfg2_type(g: int) -> int:
    m = g % 10
    return NSIE if m == 8 else (SIS if m == 9 else DPIE)


@dataclass(frozen=True)
class Config:
    name: str
    lenses: np.ndarray  # [nmodel*nlens] model-major
    nmodel: int
    nlens: int
    grid: Grid
    outputs: tuple  # names of the planes the config asks for

    @property
    def evals(self) -> int:
        return self.grid.npix * self.nlens * self.nmodel


ALL_PLANES = ("ax", "ay", "a11", "a12", "a22", "kappa", "gamma1", "gamma2", "mu")


def config(idx: int, scale: int = 1) -> Config:
    """BASELINE.json config `idx` (0-4).  `scale` > 1 divides the grid side (same
    extent, coarser pixels) for parity tests the oracle can finish in seconds."""
    if idx == 0:
        g = centred_grid(50.0, 64 // scale)
        L = cluster(0, 0, 10, 40.0)
        return Config("cfg0_tiny_all_outputs", L, 1, 10, g, ALL_PLANES)
    if idx == 1:
        g = centred_grid(100.0, 1024 // scale)
        L = cluster(1, 2, 98, 100.0)
        return Config("cfg1_cluster_gradient", L, 1, 100, g, ("ax", "ay"))
    if idx == 2:
        g = centred_grid(100.0, 2048 // scale)
        L = cluster(2, 3, 497, 100.0, _cfg2_type)
        return Config("cfg2_cluster_maps_mixed", L, 1, 500, g, ("kappa", "gamma1", "gamma2", "mu"))
    if idx == 3:
        g = centred_grid(150.0, 4096 // scale)
        L = cluster(3, 4, 996, 150.0)
        return Config("cfg3_large_grad_maps", L, 1, 1000, g, ("ax", "ay", "kappa", "gamma1", "gamma2", "mu"))
    if idx == 4:
        g = centred_grid(100.0, 1024 // scale)
        base, rng = cluster(4, 2, 298, 100.0, return_rng=True)  # perturbations continue the same stream
        nmodel = 64
        out = make_lenses(nmodel * 300)
        sig_of = lambda b0: C_KMS * np.sqrt(b0 / (0.5 * 6.0 * np.pi * ARCSEC_PER_RAD))
        for m in range(nmodel):
            mod = base.copy()
            for h in range(2):
                z = rng.standard_normal(7)
                sig = max(sig_of(base["b0"][h]) + 0.02 * 400.0 * z[0], 1.0)
                rc = max(base["rcore"][h] + 0.02 * 15.0 * z[1], 0.1)
                rt = base["rcut"][h] + 0.02 * 0.0 * z[2]
                e = min(max(base["ellipticity"][h] + 0.02 * 0.4 * z[3], 0.0), 0.95)
                th = base["theta"][h] + 0.02 * np.pi * z[4]
                x = base["x"][h] + 0.02 * 40.0 * z[5]
                y = base["y"][h] + 0.02 * 40.0 * z[6]
                mod[h] = (DPIE, 0, x, y, e, th, rc, rt, b0_from_sigma(sig))
            out[m * 300 : (m + 1) * 300] = mod
        return Config("cfg4_mcmc_batch_gradient", out, nmodel, 300, g, ("ax", "ay"))
    raise ValueError(f"no config {idx}")


def random_points(seed: int, grid: Grid, n: int):
    """`n` distinct pixel indices (i, j) of `grid`, seeded -- for sampled parity at full size."""
    rng = np.random.default_rng(seed)
    flat = rng.choice(grid.npix, size=min(n, grid.npix), replace=False)
    flat.sort()
    return (flat % grid.nx).astype(np.int64), (flat // grid.nx).astype(np.int64)


# ---------------------------------------------------------------- sharding
def row_slab(grid: Grid, rank: int, world: int):
    """Contiguous row slab of `grid` owned by `rank` of `world` (pixels are independent):
    returns (j0, nrows) -- rows [j0, j0 + nrows) of the SAME grid.  Rows are split as evenly as possible, earlier
    ranks take the extra rows; a rank may own zero rows when world > grid.ny.  There is deliberately no
    "sub-grid" with an origin of its own: a slab is addressed as (grid, j0, nrows) everywhere (lh_grid_eval_rows,
    lh_grid_eval_rows_host, oracle.grid(rows=...)), so that row j0 + j always has the coordinate of the full
    grid's definition, y0 + (j0 + j)*dx, and the slabs stacked are the full map bit for bit on any grid."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    base, extra = divmod(grid.ny, world)
    rows = base + (1 if rank < extra else 0)
    j0 = rank * base + min(rank, extra)
    return j0, rows


def model_slab(nmodel: int, rank: int, world: int):
    """Models [m0, m1) of a batch owned by `rank` (batch path shards by model, no exchange)."""
    if not (0 <= rank < world):
        raise ValueError("rank outside [0, world)")
    base, extra = divmod(nmodel, world)
    m0 = rank * base + min(rank, extra)
    return m0, m0 + base + (1 if rank < extra else 0)


# ---------------------------------------------------------------- constraints (NEXT row f3)
# 32-byte record == `lh_constraint` in include/lh.h (and the oracle's own declaration)
CONSTRAINT_DTYPE = np.dtype([("source", "<i4"), ("_pad", "<i4"), ("x", "<f8"), ("y", "<f8"), ("sigma", "<f8")])


def make_constraints(rows) -> np.ndarray:
    """rows: iterable of (source, x, y, sigma)."""
    rows = list(rows)
    c = np.zeros(len(rows), dtype=CONSTRAINT_DTYPE)
    for k, (s, x, y, sg) in enumerate(rows):
        c[k] = (s, 0, x, y, sg)
    return c
