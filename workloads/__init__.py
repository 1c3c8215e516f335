"""Seeded synthetic inputs for the PIC hot path (serves the oracle AND the CUDA path).

This module holds input data only: grids, time steps, particle clouds and initial fields for
the five configurations of BASELINE.json (C1..C5, recipe in SURVEY.md §8(d) and DESIGN.md
"Input recipe"). It contains none of the method's arithmetic (no shape factor, push, deposit,
curl or sort) and is imported by neither `oracle/` nor the package `paper_2101_12149_b200`.

The inputs stand in for the paper's uniform-plasma weak-scaling runs (§4.1.1) and
its laser-wakefield stage (§4.2), whose input decks are not available here.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

# CODATA 2018, as input data (each library carries its own c and eps0)
C_LIGHT = 299792458.0
Q_E = 1.602176634e-19
EPS0 = 8.8541878128e-12
M_E = 9.1093837015e-31
M_P = 1.67262192369e-27


@dataclass
class SpeciesSpec:
    name: str
    charge: float
    mass: float
    ppc: int
    density: float          # m^-3 (peak)
    sigma: float            # u/c per component ~ Normal(0, sigma)


@dataclass
class Config:
    name: str
    seed: int
    n_cells: tuple
    dx: tuple
    order: int
    dtype: str              # "f64" | "f32"
    steps: int
    species: list
    periodic: tuple = (1, 1, 1)
    sort_interval: int = 4
    tile: tuple = (8, 8, 8)
    cfl: float = 0.99
    z_first: int = 0        # first z-cell holding particles (C4)
    ramp_cells: int = 0     # linear density ramp length in z-cells (C4, reading Q8)
    laser: bool = False     # load the reading-Q9 laser pulse into E/B
    extra: dict = field(default_factory=dict)

    @property
    def dt(self) -> float:
        return self.cfl / (C_LIGHT * math.sqrt(sum(1.0 / (d * d) for d in self.dx)))

    @property
    def np_dtype(self):
        return np.float64 if self.dtype == "f64" else np.float32

    @property
    def n_particles(self) -> int:
        nz = self.n_cells[2] - self.z_first
        return sum(s.ppc for s in self.species) * self.n_cells[0] * self.n_cells[1] * nz


def _e(ppc, n, sigma):
    return SpeciesSpec("electrons", -Q_E, M_E, ppc, n, sigma)


CONFIGS = {
    "C1": Config("C1", 1001, (16, 16, 16), (1e-6,) * 3, 1, "f64", 20, [_e(2, 1e24, 0.01)]),
    "C2": Config("C2", 1002, (128, 128, 128), (1e-6,) * 3, 3, "f64", 100, [_e(8, 1e25, 0.01)]),
    "C3": Config("C3", 1003, (128, 128, 128), (1e-6,) * 3, 1, "f32", 100, [_e(8, 1e25, 0.01)]),
    "C4": Config("C4", 1004, (128, 128, 1024), (0.1e-6, 0.1e-6, 0.8e-6 / 32), 3, "f64", 200,
                 [_e(2, 5e24, 0.0)], periodic=(1, 1, 0), z_first=128, ramp_cells=64, laser=True),
    "C5": Config("C5", 1005, (256, 256, 256), (1e-6,) * 3, 3, "f64", 50,
                 [_e(4, 1e25, 0.1), SpeciesSpec("protons", Q_E, M_P, 4, 1e25, 0.002)]),
}


def scaled(cfg: Config, n_cells, name=None, **kw) -> Config:
    """The same recipe on a smaller grid (parity-test sizes the oracle finishes in seconds)."""
    import copy
    c = copy.deepcopy(cfg)
    c.n_cells = tuple(n_cells)
    c.name = name or (cfg.name + "@" + "x".join(str(v) for v in n_cells))
    for k, v in kw.items():
        setattr(c, k, v)
    return c


def make_species(cfg: Config, spec: SpeciesSpec, rng: np.random.Generator, shuffle=True):
    """Particles of one species: per cell (x fastest) `ppc` particles, position uniform in the
    cell, u = sigma*c*Normal(0,1) per component, weight = n(z)*dV/ppc. Generated in fp64, rounded
    once for fp32; one seeded permutation so that the first sort does real work."""
    nx, ny, nz = cfg.n_cells
    z0 = cfg.z_first
    ncell = nx * ny * (nz - z0)
    n = ncell * spec.ppc
    cell = np.repeat(np.arange(ncell, dtype=np.int64), spec.ppc)
    ci = cell % nx
    cj = (cell // nx) % ny
    ck = cell // (nx * ny) + z0
    pos = rng.random((3, n))
    x = (ci + pos[0]) * cfg.dx[0]
    y = (cj + pos[1]) * cfg.dx[1]
    z = (ck + pos[2]) * cfg.dx[2]
    if spec.sigma > 0:
        u = rng.standard_normal((3, n)) * (spec.sigma * C_LIGHT)
    else:
        u = np.zeros((3, n))
    dv = cfg.dx[0] * cfg.dx[1] * cfg.dx[2]
    if cfg.ramp_cells > 0:
        dens = spec.density * np.clip((z / cfg.dx[2] - z0) / cfg.ramp_cells, 0.0, 1.0)
    else:
        dens = np.full(n, spec.density)
    w = dens * dv / spec.ppc
    arrs = [x, y, z, u[0], u[1], u[2], w]
    if shuffle:
        p = rng.permutation(n)
        arrs = [a[p] for a in arrs]
    dt = cfg.np_dtype
    out = [np.ascontiguousarray(a.astype(dt)) for a in arrs]
    # rounding to fp32 may land a position exactly on the upper domain edge: pull it back inside
    for a, d in zip(out[:3], range(3)):
        L = dt(cfg.n_cells[d] * cfg.dx[d])
        a[a >= L] = np.nextafter(L, dt(0))
    return dict(zip(("x", "y", "z", "ux", "uy", "uz", "w"), out))


def laser_fields(cfg: Config):
    """Reading Q9: linearly polarised Gaussian pulse loaded into Ex and By (each sampled at its
    own Yee location), z-cells 16..112 with an 8-cell cos^2 taper, as input DATA."""
    nx, ny, nz = cfg.n_cells
    dx, dy, dz = cfg.dx
    lam, a0, w0, fwhm = 0.8e-6, 2.0, 5e-6, 15e-15
    om = 2 * math.pi * C_LIGHT / lam
    k = 2 * math.pi / lam
    E0 = a0 * M_E * C_LIGHT * om / Q_E
    tau = fwhm / math.sqrt(2 * math.log(2))
    zc = (64 + 0.5) * dz
    xc, yc = 0.5 * nx * dx, 0.5 * ny * dy

    def win(zcell):
        lo, hi, tp = 16.0, 112.0, 8.0
        wv = np.zeros_like(zcell)
        inside = (zcell >= lo) & (zcell <= hi)
        wv[inside] = 1.0
        up = inside & (zcell < lo + tp)
        wv[up] = np.sin(0.5 * math.pi * (zcell[up] - lo) / tp) ** 2
        dn = inside & (zcell > hi - tp)
        wv[dn] = np.sin(0.5 * math.pi * (hi - zcell[dn]) / tp) ** 2
        return wv

    def pulse(sx, sy, sz):
        xs = (np.arange(nx) + sx) * dx
        ys = (np.arange(ny) + sy) * dy
        zs = (np.arange(nz) + sz) * dz
        r2 = (xs[None, None, :] - xc) ** 2 + (ys[None, :, None] - yc) ** 2
        zz = zs - zc
        lon = np.exp(-(zz / (C_LIGHT * tau)) ** 2) * np.cos(k * zz) * win(zs / dz)
        return E0 * np.exp(-r2 / w0 ** 2) * lon[:, None, None]

    dt = cfg.np_dtype
    zero = lambda: np.zeros((nz, ny, nx), dtype=dt)
    Ex = pulse(0.5, 0.0, 0.0).astype(dt)
    By = (pulse(0.5, 0.0, 0.5) / C_LIGHT).astype(dt)
    return [Ex, zero(), zero()], [zero(), By, zero()]


def random_fields(cfg: Config, rng: np.random.Generator, e_scale=1e9, b_scale=3.0, modes=3):
    """Smooth random periodic E and B (a few low Fourier modes per component) — input data for
    the one-step parity tests, so that gather and push see non-trivial fields."""
    nx, ny, nz = cfg.n_cells
    ii = np.arange(nx)[None, None, :] / nx
    jj = np.arange(ny)[None, :, None] / ny
    kk = np.arange(nz)[:, None, None] / nz
    out = []
    for scale in (e_scale,) * 3 + (b_scale,) * 3:
        f = np.zeros((nz, ny, nx))
        for _ in range(modes):
            m = rng.integers(0, 3, size=3)
            ph = rng.random(3) * 2 * math.pi
            f += rng.standard_normal() * np.cos(2 * math.pi * m[0] * ii + ph[0]) * \
                np.cos(2 * math.pi * m[1] * jj + ph[1]) * np.cos(2 * math.pi * m[2] * kk + ph[2])
        out.append(np.ascontiguousarray((scale * f).astype(cfg.np_dtype)))
    return out[:3], out[3:]


def generate(cfg: Config, shuffle=True):
    """(list of (SpeciesSpec, arrays dict), E or None, B or None) for a configuration."""
    rng = np.random.default_rng(cfg.seed)
    species = [(s, make_species(cfg, s, rng, shuffle=shuffle)) for s in cfg.species]
    E = B = None
    if cfg.laser:
        E, B = laser_fields(cfg)
    return species, E, B
