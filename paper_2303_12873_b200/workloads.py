"""Seeded synthetic inputs shaped like BASELINE.json's configs (SURVEY.md
section 8(d) table).  This module serves BOTH the
oracle and the CUDA path and therefore holds none of the method's arithmetic:
it only draws positions, momenta and weights from ``numpy.random.default_rng``
and evaluates analytic initial laser fields on the Yee locations.

No public dataset is involved: the paper's own runs (ref [13])
are not in the container; these inputs stand in for the *shapes* of its
workloads (uniform plasma, laser-wakefield box, plasma mirror).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

C_LIGHT = 299792458.0
Q_E = 1.602176634e-19
M_E = 9.1093837015e-31
M_P = 1.67262192369e-27
EPS0 = 8.8541878128e-12
SEED0 = 12873


@dataclass
class Species:
    name: str
    q: float
    m: float
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    ux: np.ndarray
    uy: np.ndarray
    uz: np.ndarray
    w: np.ndarray

    @property
    def n(self) -> int:
        return int(self.x.size)

    def arrays(self):
        return (self.x, self.y, self.z, self.ux, self.uy, self.uz, self.w)


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    dt: float
    order: int
    nsteps: int
    sort_every: int
    species: list = field(default_factory=list)
    fields: dict | None = None          # {"Ex": flat array, ...} or None (= zeros)
    xmin: float = 0.0
    ymin: float = 0.0
    zmin: float = 0.0

    @property
    def ncell(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def nparticles(self) -> int:
        return sum(s.n for s in self.species)

    def grid_args(self):
        return (self.nx, self.ny, self.nz, self.dx, self.dy, self.dz, self.xmin, self.ymin, self.zmin)


def courant_dt(dx, dy, dz, cfl=0.99):
    """dt = cfl x the 3-D Courant limit (reading R17)."""
    return cfl / (C_LIGHT * np.sqrt(1.0 / dx ** 2 + 1.0 / dy ** 2 + 1.0 / dz ** 2))


def _positions_in_cells(rng, nx, ny, nz, ppc, dx, dy, dz, xmin, ymin, zmin, cell_mask=None):
    """ppc uniform positions in every (selected) cell, cell-major order
    (k, j, i fastest, then particle in cell) -> arrives cell-sorted (R28)."""
    if cell_mask is None:
        k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
        i = i.reshape(-1); j = j.reshape(-1); k = k.reshape(-1)
    else:
        k, j, i = np.nonzero(cell_mask)                     # C order of a (nz,ny,nx) mask
    i = np.repeat(i, ppc); j = np.repeat(j, ppc); k = np.repeat(k, ppc)
    n = i.size
    r = rng.random((3, n))
    x = xmin + (i + r[0]) * dx
    y = ymin + (j + r[1]) * dy
    z = zmin + (k + r[2]) * dz
    # strictly inside [min, max): (i + r) may round up to the next integer
    x = np.minimum(x, np.nextafter(xmin + nx * dx, -np.inf))
    y = np.minimum(y, np.nextafter(ymin + ny * dy, -np.inf))
    z = np.minimum(z, np.nextafter(zmin + nz * dz, -np.inf))
    return x, y, z


def _maxwellian(rng, n, u_th):
    """Gaussian u = gamma v per Cartesian component, sigma = u_th * c (R26)."""
    if u_th == 0.0:
        return np.zeros(n), np.zeros(n), np.zeros(n)
    u = rng.normal(size=(3, n)) * (u_th * C_LIGHT)
    return u[0].copy(), u[1].copy(), u[2].copy()


def _shuffle(rng, sp: Species):
    perm = rng.permutation(sp.n)
    for name in ("x", "y", "z", "ux", "uy", "uz", "w"):
        setattr(sp, name, np.ascontiguousarray(getattr(sp, name)[perm]))


def uniform_plasma(nx, ny, nz, ppc=8, u_th=0.01, order=1, seed=SEED0, nsteps=10, sort_every=0,
                   protons=False, dx=0.5e-6, dy=None, dz=None, n0=1e25, shuffle=False,
                   name="uniform") -> Workload:
    """Configs 0-2: periodic uniform plasma.  Electrons: Maxwellian u_th; with
    ``protons`` a cold proton species co-located with the electrons (R19) so
    that Gauss's law holds with E(0) = 0."""
    dy = dx if dy is None else dy
    dz = dx if dz is None else dz
    rng = np.random.default_rng(seed)
    x, y, z = _positions_in_cells(rng, nx, ny, nz, ppc, dx, dy, dz, 0.0, 0.0, 0.0)
    n = x.size
    ux, uy, uz = _maxwellian(rng, n, u_th)
    w = np.full(n, n0 * dx * dy * dz / ppc)                      # R27
    sp = [Species("electrons", -Q_E, M_E, x, y, z, ux, uy, uz, w)]
    if protons:
        zero = np.zeros(n)
        sp.append(Species("protons", +Q_E, M_P, x.copy(), y.copy(), z.copy(), zero.copy(), zero.copy(),
                          zero.copy(), w.copy()))
    if shuffle:
        for s_i, s in enumerate(sp):
            _shuffle(np.random.default_rng(seed + 1000 * (s_i + 1) + 7), s)
    return Workload(name, nx, ny, nz, dx, dy, dz, courant_dt(dx, dy, dz), order, nsteps, sort_every, sp)


def _yee_coords(nx, ny, nz, dx, dy, dz, ox, oy, oz):
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    return (i + ox) * dx, (j + oy) * dy, (k + oz) * dz


def _laser_fields(nx, ny, nz, dx, dy, dz, a0, lam, w0, ctau, z0):
    """Linearly polarised (x), +z-propagating Gaussian pulse at t = 0 with a
    flat phase (R32): Ex = E0 exp(-r^2/w0^2) exp(-(z-z0)^2/ctau^2) cos(k0 (z-z0)),
    By = Ex/c, each sampled at its own Yee location.  w0 = inf -> plane wave (R35)."""
    k0 = 2 * np.pi / lam
    E0 = a0 * M_E * C_LIGHT * (k0 * C_LIGHT) / Q_E
    out = {}
    for comp, (ox, oy, oz), scale in (("Ex", (0.5, 0.0, 0.0), 1.0), ("By", (0.5, 0.0, 0.5), 1.0 / C_LIGHT)):
        X, Y, Z = _yee_coords(nx, ny, nz, dx, dy, dz, ox, oy, oz)
        env = np.exp(-((Z - z0) / ctau) ** 2)
        if np.isfinite(w0):
            xc, yc = 0.5 * nx * dx, 0.5 * ny * dy
            env = env * np.exp(-((X - xc) ** 2 + (Y - yc) ** 2) / w0 ** 2)
        out[comp] = (scale * E0 * env * np.cos(k0 * (Z - z0))).reshape(-1)
    return out


def lwfa_box(nx=128, ny=128, nz=1024, seed=SEED0 + 3, nsteps=500, order=3, sort_every=1, shuffle=False):
    """Config 3 (readings R31-R34): 128x128x1024, dz = lambda/32, dx = dy = 4 dz,
    2 ppc cold electrons, linear ramp over cells 600-700, flat to cell 1000;
    Gaussian pulse a0 = 2, w0 = 8 um, 30 fs FWHM centred at cell 400.  ``nx, ny``
    may be cropped (same z profile, w0 unchanged) for parity runs; nz may be
    cropped proportionally (profile positions scale with nz/1024)."""
    lam = 0.8e-6
    dz = lam / 32; dx = dy = 4 * dz
    ppc, n0 = 2, 5e24
    s = nz / 1024.0
    ramp0, ramp1, flat1 = 600 * s, 700 * s, 1000 * s
    rng = np.random.default_rng(seed)
    kk = np.arange(nz)
    mask = np.zeros((nz, ny, nx), dtype=bool)
    mask[(kk + 1 > ramp0) & (kk < flat1)] = True
    x, y, z = _positions_in_cells(rng, nx, ny, nz, ppc, dx, dy, dz, 0.0, 0.0, 0.0, mask)
    zc = z / dz
    dens = n0 * np.clip((zc - ramp0) / (ramp1 - ramp0), 0.0, 1.0) * (zc < flat1)
    keep = dens > 0
    x, y, z, dens = x[keep], y[keep], z[keep], dens[keep]
    n = x.size
    zero = np.zeros(n)
    w = dens * dx * dy * dz / ppc                                 # R27: n at the particle's own position
    sp = Species("electrons", -Q_E, M_E, x, y, z, zero.copy(), zero.copy(), zero.copy(), w)
    if shuffle:
        _shuffle(np.random.default_rng(seed + 1007), sp)
    ctau = C_LIGHT * 30e-15 / np.sqrt(2 * np.log(2))
    fields = _laser_fields(nx, ny, nz, dx, dy, dz, a0=2.0, lam=lam, w0=8e-6, ctau=ctau * s, z0=400 * s * dz)
    return Workload("lwfa", nx, ny, nz, dx, dy, dz, courant_dt(dx, dy, dz), order, nsteps, sort_every, [sp],
                    fields)


def plasma_mirror(nx=256, ny=256, nz=512, seed=SEED0 + 4, nsteps=200, order=3, sort_every=1, shuffle=False):
    """Config 4 (reading R35): dx = lambda/64, slab of 30 n_c over cells 400-464,
    exponential pre-plasma (L = lambda/10 = 6.4 cells) over cells 368-400,
    electrons 16 ppc (u_th = 0.005 c), protons 4 ppc (cold); plane-wave pulse
    a0 = 10, 2 cycles FWHM, centred at cell 176.  nx, ny may be cropped."""
    lam = 0.8e-6
    dx = dy = dz = lam / 64
    n_c = EPS0 * M_E * (2 * np.pi * C_LIGHT / lam) ** 2 / Q_E ** 2
    n_slab = 30.0 * n_c
    L = 6.4
    s = nz / 512.0
    pre0, front, rear = 368 * s, 400 * s, 464 * s
    kk = np.arange(nz)
    mask = np.zeros((nz, ny, nx), dtype=bool)
    mask[(kk + 1 > pre0) & (kk < rear)] = True

    def make(name, q, m, ppc, u_th, sd):
        rng = np.random.default_rng(sd)
        x, y, z = _positions_in_cells(rng, nx, ny, nz, ppc, dx, dy, dz, 0.0, 0.0, 0.0, mask)
        zc = z / dz
        dens = np.where(zc >= front, n_slab, n_slab * np.exp((zc - front) / (L * s)))
        dens = dens * ((zc >= pre0) & (zc < rear))
        keep = dens > 0
        x, y, z, dens = x[keep], y[keep], z[keep], dens[keep]
        ux, uy, uz = _maxwellian(rng, x.size, u_th)
        sp = Species(name, q, m, x, y, z, ux, uy, uz, dens * dx * dy * dz / ppc)
        if shuffle:
            _shuffle(np.random.default_rng(sd + 7), sp)
        return sp

    sp = [make("electrons", -Q_E, M_E, 16, 0.005, seed), make("protons", +Q_E, M_P, 4, 0.0, seed + 1000)]
    ctau = 2 * lam / np.sqrt(2 * np.log(2))
    fields = _laser_fields(nx, ny, nz, dx, dy, dz, a0=10.0, lam=lam, w0=np.inf, ctau=ctau * s, z0=176 * s * dz)
    return Workload("plasma_mirror", nx, ny, nz, dx, dy, dz, courant_dt(dx, dy, dz), order, nsteps, sort_every,
                    sp, fields)


def config(index: int, parity: bool = False, **kw) -> Workload:
    """BASELINE.json configs[index] at full size, or (parity=True) at the size
    the oracle finishes in seconds (last column)."""
    seed = SEED0 + index
    ppc = kw.pop("ppc", 8) if index <= 2 else None      # configs 0-2 name 8 particles per cell; experiments may override
    if index == 0:
        n = kw.pop("n", 32)
        return uniform_plasma(n, n, n, ppc, 0.01, 1, seed, nsteps=10, sort_every=0, name="config0", **kw)
    if index == 1:
        n = kw.pop("n", 32 if parity else 128)
        return uniform_plasma(n, n, n, ppc, 0.01, 3, seed, nsteps=100, sort_every=4, protons=True,
                              name="config1", **kw)
    if index == 2:
        n = kw.pop("n", 32 if parity else 256)
        # the config names no sort cadence; at u_th = 0.05 c about 7 % of the particles change cell per
        # step, so sorting every step keeps the fused kernel's per-cell fast path at ~93 % (R25)
        return uniform_plasma(n, n, n, ppc, 0.05, 3, seed, nsteps=10 if parity else 50, sort_every=1,
                              name="config2", **kw)
    if index == 3:
        if parity:
            kw.setdefault("nx", 16); kw.setdefault("ny", 16); kw.setdefault("nsteps", 20)
        return lwfa_box(seed=seed, **kw)
    if index == 4:
        if parity:
            kw.setdefault("nx", 8); kw.setdefault("ny", 8); kw.setdefault("nsteps", 20)
        return plasma_mirror(seed=seed, **kw)
    raise ValueError("config index must be 0..4")
