"""ORACLE (test infrastructure, NOT the product): ctypes binding of
``pic_oracle.c`` plus ``OracleSim``, the explicit EM-PIC cycle composed stage
by stage in the order of SURVEY.md section 8(c.1) (section II:
"explicit algorithms, which iterate forward in time").

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline``
/ ``--impl reference`` legs may import this module.  It imports nothing from
``paper_2303_12873_b200`` and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pic_oracle.c")
_HDR = os.path.join(_HERE, "pic_oracle.h")
_LIB = os.path.join(_HERE, "libpic_oracle.so")

_dp = C.POINTER(C.c_double)
_lp = C.POINTER(C.c_longlong)


class OraGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("xmin", C.c_double), ("ymin", C.c_double), ("zmin", C.c_double)]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction).  Returns the .so path."""
    stale = (not os.path.exists(_LIB)
             or os.path.getmtime(_LIB) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-std=c11", "-Wall", "-shared",
                               "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        G = C.POINTER(OraGrid)
        L.ora_const_c.restype = C.c_double
        L.ora_const_eps0.restype = C.c_double
        L.ora_shape.restype = C.c_double
        L.ora_shape.argtypes = [C.c_int, C.c_double]
        L.ora_courant_dt.restype = C.c_double
        L.ora_courant_dt.argtypes = [G]
        L.ora_gather.argtypes = [G, C.c_int, C.c_longlong] + [_dp] * 15
        L.ora_shape0.restype = C.c_double
        L.ora_shape0.argtypes = [C.c_double]
        L.ora_gather_variant.argtypes = [G, C.c_int, C.c_int, C.c_longlong] + [_dp] * 15
        L.ora_smooth_binomial.argtypes = [G, C.c_int, _dp]
        L.ora_gather_f32.argtypes = [G, C.c_int, C.c_int, C.c_longlong] + [_dp] * 15
        L.ora_boris_f32.argtypes = [C.c_longlong, C.c_double, C.c_double, C.c_double] + [_dp] * 9
        L.ora_boris.argtypes = [C.c_longlong, C.c_double, C.c_double, C.c_double] + [_dp] * 9
        L.ora_move.argtypes = [C.c_longlong, C.c_double] + [_dp] * 9
        L.ora_deposit_esirkepov.argtypes = [G, C.c_int, C.c_longlong, C.c_double, C.c_double] + [_dp] * 10
        L.ora_deposit_direct.argtypes = [G, C.c_int, C.c_longlong, C.c_double, C.c_double] + [_dp] * 10
        L.ora_wrap.argtypes = [G, C.c_longlong] + [_dp] * 3
        L.ora_yee_push_B.argtypes = [G, C.c_double] + [_dp] * 6
        L.ora_yee_push_E.argtypes = [G, C.c_double] + [_dp] * 9
        L.ora_deposit_rho.argtypes = [G, C.c_int, C.c_longlong, C.c_double] + [_dp] * 5
        L.ora_cell_keys.argtypes = [G, C.c_longlong] + [_dp] * 3 + [_lp]
        L.ora_counting_sort.argtypes = [C.c_longlong, C.c_longlong, _lp, _lp, _lp]
        _lib = L
    return _lib


def _d(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"], "need contiguous float64"
    return a.ctypes.data_as(_dp)


def _l(a: np.ndarray):
    assert a.dtype == np.int64 and a.flags["C_CONTIGUOUS"], "need contiguous int64"
    return a.ctypes.data_as(_lp)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError("oracle %s failed with code %d" % (what, rc))


C_LIGHT = 299792458.0
EPS0 = 8.8541878128e-12


def make_grid(nx, ny, nz, dx, dy, dz, xmin=0.0, ymin=0.0, zmin=0.0) -> OraGrid:
    return OraGrid(int(nx), int(ny), int(nz), float(dx), float(dy), float(dz),
                   float(xmin), float(ymin), float(zmin))


def shape(n: int, r: float) -> float:
    return lib().ora_shape(int(n), float(r))


def courant_dt(g: OraGrid) -> float:
    return lib().ora_courant_dt(C.byref(g))


def gather(g: OraGrid, order: int, x, y, z, E, B):
    """E, B: 3-tuples of flat nx*ny*nz arrays.  Returns (Exp,Eyp,Ezp,Bxp,Byp,Bzp)."""
    x, y, z = _f64(x), _f64(y), _f64(z)
    n = x.size
    F = [_f64(a) for a in (*E, *B)]
    out = [np.empty(n) for _ in range(6)]
    _check(lib().ora_gather(C.byref(g), order, n, _d(x), _d(y), _d(z), *[_d(a) for a in F],
                            *[_d(a) for a in out]), "gather")
    return tuple(out)


def shape0(r: float) -> float:
    return lib().ora_shape0(float(r))


def gather_variant(g: OraGrid, order: int, variant: int, x, y, z, E, B):
    """NEXT-3: variant 0 = gather(); 1 = order n-1 along each component's staggered directions."""
    x, y, z = _f64(x), _f64(y), _f64(z)
    n = x.size
    F = [_f64(a) for a in (*E, *B)]
    out = [np.empty(n) for _ in range(6)]
    _check(lib().ora_gather_variant(C.byref(g), order, variant, n, _d(x), _d(y), _d(z), *[_d(a) for a in F],
                                    *[_d(a) for a in out]), "gather_variant")
    return tuple(out)


def gather_f32(g: OraGrid, order: int, variant: int, x, y, z, E, B):
    """NEXT-4: the gather in single precision (shape and field values rounded to float); returns doubles."""
    x, y, z = _f64(x), _f64(y), _f64(z)
    n = x.size
    F = [_f64(a) for a in (*E, *B)]
    out = [np.empty(n) for _ in range(6)]
    _check(lib().ora_gather_f32(C.byref(g), order, variant, n, _d(x), _d(y), _d(z), *[_d(a) for a in F],
                                *[_d(a) for a in out]), "gather_f32")
    return tuple(out)


def boris_f32(q, m, dt, ux, uy, uz, Ep, Bp):
    """NEXT-4: the Boris push in single precision, in place on doubles that hold float values."""
    n = ux.size
    _check(lib().ora_boris_f32(n, q, m, dt, _d(ux), _d(uy), _d(uz), *[_d(_f64(a)) for a in (*Ep, *Bp)]),
           "boris_f32")


def smooth_binomial(g: OraGrid, npass: int, F: np.ndarray):
    """NEXT-3: in-place periodic 1-2-1 smoothing, `npass` passes of x, y, z."""
    _check(lib().ora_smooth_binomial(C.byref(g), int(npass), _d(F)), "smooth_binomial")


def boris(q, m, dt, ux, uy, uz, Ep, Bp):
    """In place on ux,uy,uz (contiguous float64)."""
    n = ux.size
    _check(lib().ora_boris(n, q, m, dt, _d(ux), _d(uy), _d(uz), *[_d(_f64(a)) for a in (*Ep, *Bp)]),
           "boris")


def move(dt, x, y, z, ux, uy, uz):
    n = x.size
    out = [np.empty(n) for _ in range(3)]
    _check(lib().ora_move(n, dt, _d(x), _d(y), _d(z), _d(ux), _d(uy), _d(uz), *[_d(a) for a in out]),
           "move")
    return tuple(out)


def deposit_esirkepov(g, order, q, dt, w, p0, p1, J):
    """Accumulates into J = (Jx,Jy,Jz), flat contiguous float64 arrays."""
    n = p0[0].size
    rc = lib().ora_deposit_esirkepov(C.byref(g), order, n, q, dt, _d(_f64(w)),
                                     *[_d(_f64(a)) for a in p0], *[_d(_f64(a)) for a in p1],
                                     *[_d(a) for a in J])
    _check(rc, "deposit_esirkepov")


def deposit_direct(g, order, q, dt, w, p0, p1, J):
    """NEXT-3: direct deposition; accumulates into J = (Jx,Jy,Jz)."""
    n = p0[0].size
    rc = lib().ora_deposit_direct(C.byref(g), order, n, q, dt, _d(_f64(w)),
                                  *[_d(_f64(a)) for a in p0], *[_d(_f64(a)) for a in p1],
                                  *[_d(a) for a in J])
    _check(rc, "deposit_direct")


def wrap(g, x, y, z):
    _check(lib().ora_wrap(C.byref(g), x.size, _d(x), _d(y), _d(z)), "wrap")


def yee_push_B(g, dth, E, B):
    _check(lib().ora_yee_push_B(C.byref(g), dth, *[_d(a) for a in E], *[_d(a) for a in B]), "yee_push_B")


def yee_push_E(g, dt, E, B, J):
    _check(lib().ora_yee_push_E(C.byref(g), dt, *[_d(a) for a in E], *[_d(a) for a in B],
                                *[_d(a) for a in J]), "yee_push_E")


def deposit_rho(g, order, q, w, x, y, z, rho):
    _check(lib().ora_deposit_rho(C.byref(g), order, x.size, q, _d(_f64(w)), _d(_f64(x)), _d(_f64(y)),
                                 _d(_f64(z)), _d(rho)), "deposit_rho")


def cell_keys(g, x, y, z) -> np.ndarray:
    key = np.empty(x.size, dtype=np.int64)
    _check(lib().ora_cell_keys(C.byref(g), x.size, _d(_f64(x)), _d(_f64(y)), _d(_f64(z)), _l(key)),
           "cell_keys")
    return key


def counting_sort(ncell: int, key: np.ndarray):
    perm = np.empty(key.size, dtype=np.int64)
    off = np.empty(ncell + 1, dtype=np.int64)
    _check(lib().ora_counting_sort(ncell, key.size, _l(key), _l(perm), _l(off)), "counting_sort")
    return perm, off


class _Species:
    __slots__ = ("q", "m", "x", "y", "z", "ux", "uy", "uz", "w", "id")


class OracleSim:
    """The PIC cycle of SURVEY.md 8(c.1), steps 1-8, on host arrays.  Mirrors
    the method names of the CUDA binding so one test can drive both.

    ``open_z`` (NEXT-2: non-periodic longitudinal boundary, moving window, antenna): the box ends at
    z = zmin and z = zmin + nz dz; every field value with a z index outside 0 .. nz-1 IS ZERO at all times, current
    deposited there is dropped, and a particle that leaves through a z face is deleted after it has deposited.
    It is written with the periodic functions above, unchanged, on arrays that carry ``ZPAD`` extra planes at either
    end: the extra planes are forced back to zero after every operation that writes them, and they are wide enough
    (4 >= the reach of every stencil) that the periodic seam between them is never felt."""

    ZPAD = 4

    def __init__(self, nx, ny, nz, dx, dy, dz, xmin, ymin, zmin, dt, order, nspecies, gather_variant=0,
                 smooth_passes=0, open_z=False, deposit_variant=0, precision=0):
        if deposit_variant not in (0, 1):
            raise ValueError("deposit_variant must be 0 (Esirkepov) or 1 (direct)")
        if precision not in (0, 1):
            raise ValueError("precision must be 0 (fp64) or 1 (fp32 fields and momenta, fp64 positions)")
        self.deposit_variant, self.precision = int(deposit_variant), int(precision)
        self.open_z = bool(open_z)
        self.nz_phys = int(nz)
        self.pad = self.ZPAD if self.open_z else 0
        self.g = make_grid(nx, ny, nz + 2 * self.pad, dx, dy, dz, xmin, ymin, zmin - self.pad * dz)
        if gather_variant not in (0, 1) or smooth_passes < 0:
            raise ValueError("gather_variant must be 0 or 1, smooth_passes >= 0")
        if self.open_z and smooth_passes:
            raise ValueError("smoothing is periodic: not with open_z")
        self.gather_variant, self.smooth_passes = int(gather_variant), int(smooth_passes)   # NEXT-3 options
        if order not in (1, 2, 3):
            raise ValueError("order must be 1, 2 or 3")
        if not (0.0 < dt <= courant_dt(self.g)):
            raise ValueError("dt outside (0, Courant limit]")
        self.dt, self.order = float(dt), int(order)
        self.nx, self.ny = int(nx), int(ny)
        self.ncell = nx * ny * nz                          # physical cells
        self.ncell_all = nx * ny * (nz + 2 * self.pad)
        self.E = [np.zeros(self.ncell_all) for _ in range(3)]
        self.B = [np.zeros(self.ncell_all) for _ in range(3)]
        self.J = [np.zeros(self.ncell_all) for _ in range(3)]
        self.species: list[_Species | None] = [None] * nspecies
        self.cell_offset: list[np.ndarray | None] = [None] * nspecies
        self.plane_sources = []                            # (component index 0..2 of J, plane k, values) for the next step
        self.deleted = 0
        self.damp = None                                   # NEXT-2: damping factors of the layers next to the open ends

    # ---- open-z helpers ------------------------------------------------------------------------------------
    def _phys(self, a):
        """View of the physical planes of a padded flat array."""
        nz_all = self.nz_phys + 2 * self.pad
        return a.reshape(nz_all, self.ny, self.nx)[self.pad:self.pad + self.nz_phys]

    def _zero_pads(self, arrays):
        if not self.open_z:
            return
        nz_all = self.nz_phys + 2 * self.pad
        for a in arrays:
            v = a.reshape(nz_all, self.ny, self.nx)
            v[:self.pad] = 0.0
            v[self.pad + self.nz_phys:] = 0.0

    @property
    def zmin(self):
        return self.g.zmin + self.pad * self.g.dz

    def _delete_outside_z(self):
        lo, hi = self.zmin, self.zmin + self.nz_phys * self.g.dz
        for sp in self.species:
            if sp is None or sp.x.size == 0:
                continue
            keep = (sp.z >= lo) & (sp.z < hi)
            if not keep.all():
                self.deleted += int((~keep).sum())
                for name in ("x", "y", "z", "ux", "uy", "uz", "w", "id"):
                    setattr(sp, name, np.ascontiguousarray(getattr(sp, name)[keep]))

    def set_fields(self, Ex=None, Ey=None, Ez=None, Bx=None, By=None, Bz=None):
        for dst, src in zip(self.E + self.B, (Ex, Ey, Ez, Bx, By, Bz)):
            dst[:] = 0.0
            if src is not None:
                self._phys(dst)[...] = np.asarray(src, dtype=np.float64).reshape(self.nz_phys, self.ny, self.nx)

    def load_particles(self, s, q, m, x, y, z, ux, uy, uz, w, id_base=0):
        sp = _Species()
        sp.q, sp.m = float(q), float(m)
        for name, a in zip(("x", "y", "z", "ux", "uy", "uz", "w"), (x, y, z, ux, uy, uz, w)):
            setattr(sp, name, np.array(a, dtype=np.float64, copy=True).reshape(-1))
        sp.id = np.arange(sp.x.size, dtype=np.uint64) + np.uint64(id_base)
        self.species[s] = sp
        self.cell_offset[s] = None

    def append_particles(self, s, x, y, z, ux, uy, uz, w, ids):
        """NEXT-2: fresh plasma entering a moving window (the caller draws it)."""
        sp = self.species[s]
        for name, a in zip(("x", "y", "z", "ux", "uy", "uz", "w"), (x, y, z, ux, uy, uz, w)):
            setattr(sp, name, np.concatenate([getattr(sp, name), np.asarray(a, dtype=np.float64).reshape(-1)]))
        sp.id = np.concatenate([sp.id, np.asarray(ids, dtype=np.uint64).reshape(-1)])
        self.cell_offset[s] = None

    def add_plane_source(self, comp, k, values):
        """NEXT-2 antenna: J_comp[:, :, k] += values in the NEXT step, after deposition and before the E push
        (comp = 0, 1, 2 for Jx, Jy, Jz; values = ny x nx array, x fastest)."""
        self.plane_sources.append((int(comp), int(k), np.asarray(values, dtype=np.float64).reshape(self.ny, self.nx).copy()))

    def set_damping(self, factors):
        """NEXT-2: an absorbing layer in front of each open z end.  factors[m], m = 0 .. len-1, multiplies every value
        of B (after each B half push) and of E (after the E push) on the plane m cells away from the face (m = 0: the
        plane next to it), at both ends.  The caller supplies the profile (e.g. exp(-a ((n - m)/n)^2))."""
        if not self.open_z:
            raise ValueError("damping layers sit in front of open ends: needs open_z")
        f = np.asarray(factors, dtype=np.float64).reshape(-1)
        if 2 * f.size > self.nz_phys:
            raise ValueError("the two layers overlap")
        self.damp = f.copy() if f.size else None

    def _apply_damping(self, arrays):
        if self.damp is None:
            return
        for a in arrays:
            v = self._phys(a)
            for m, fm in enumerate(self.damp):
                v[m] *= fm
                v[self.nz_phys - 1 - m] *= fm

    def shift_window(self, ncells=1):
        """NEXT-2 moving window: the box moves up by ncells cells along z.  Field index k now names what was
        k + ncells, the top ncells planes are new (zero), particles below the new zmin are deleted."""
        if not self.open_z:
            raise ValueError("a moving window needs open_z")
        n = int(ncells)
        for a in self.E + self.B + self.J:
            v = self._phys(a)
            v[:self.nz_phys - n] = v[n:].copy()
            v[self.nz_phys - n:] = 0.0
        self.g.zmin = self.g.zmin + n * self.g.dz
        self._delete_outside_z()
        self.cell_offset = [None] * len(self.species)

    def step(self, nsteps=1):
        g, dt, n = self.g, self.dt, self.order
        for _ in range(nsteps):
            for a in self.J:                       # reading R13: J overwritten each step
                a[:] = 0.0
            for sp in self.species:
                if sp is None or sp.x.size == 0:
                    continue
                if self.precision:                 # NEXT-4: gather and push in fp32, the rest in fp64
                    F = gather_f32(g, n, self.gather_variant, sp.x, sp.y, sp.z, self.E, self.B)
                    boris_f32(sp.q, sp.m, dt, sp.ux, sp.uy, sp.uz, F[:3], F[3:])
                else:
                    if self.gather_variant:
                        F = gather_variant(g, n, self.gather_variant, sp.x, sp.y, sp.z, self.E, self.B)
                    else:
                        F = gather(g, n, sp.x, sp.y, sp.z, self.E, self.B)         # step 1
                    boris(sp.q, sp.m, dt, sp.ux, sp.uy, sp.uz, F[:3], F[3:])      # step 2
                x1, y1, z1 = move(dt, sp.x, sp.y, sp.z, sp.ux, sp.uy, sp.uz)      # step 3
                if self.deposit_variant:
                    deposit_direct(g, n, sp.q, dt, sp.w, (sp.x, sp.y, sp.z), (x1, y1, z1), self.J)
                else:
                    deposit_esirkepov(g, n, sp.q, dt, sp.w, (sp.x, sp.y, sp.z), (x1, y1, z1), self.J)  # 4
                if self.open_z:                    # no wrap along z: leavers are deleted below
                    zkeep = z1.copy()
                    wrap(g, x1, y1, z1)
                    z1 = zkeep
                else:
                    wrap(g, x1, y1, z1)                                           # step 5
                sp.x, sp.y, sp.z = x1, y1, z1
            if self.open_z:
                self._zero_pads(self.J)            # current deposited outside the box is dropped
                self._delete_outside_z()
            for comp, k, vals in self.plane_sources:                              # NEXT-2 antenna
                self._phys(self.J[comp])[k] += vals
            self.plane_sources = []
            for a in self.J:                       # NEXT-3: optional binomial smoothing of J
                if self.smooth_passes:
                    smooth_binomial(g, self.smooth_passes, a)
            yee_push_B(g, 0.5 * dt, self.E, self.B)                               # step 6
            self._zero_pads(self.B)
            self._apply_damping(self.B)
            yee_push_E(g, dt, self.E, self.B, self.J)                             # step 7
            self._zero_pads(self.E)
            self._apply_damping(self.E)
            yee_push_B(g, 0.5 * dt, self.E, self.B)                               # step 8
            self._zero_pads(self.B)
            self._apply_damping(self.B)

    def sort(self):
        for s, sp in enumerate(self.species):
            if sp is None:
                continue
            key = cell_keys(self.g, sp.x, sp.y, sp.z)
            perm, off = counting_sort(self.ncell_all, key)
            for name in ("x", "y", "z", "ux", "uy", "uz", "w", "id"):
                setattr(sp, name, np.ascontiguousarray(getattr(sp, name)[perm]))
            self.cell_offset[s] = off

    def get_fields(self):
        return {k: np.ascontiguousarray(self._phys(v)).reshape(-1).copy()
                for k, v in zip(("Ex", "Ey", "Ez", "Bx", "By", "Bz", "Jx", "Jy", "Jz"), self.E + self.B + self.J)}

    def get_particles(self, s):
        sp = self.species[s]
        return {k: getattr(sp, k).copy() for k in ("x", "y", "z", "ux", "uy", "uz", "w", "id")}

    def deposit_rho(self, s=-1):
        rho = np.zeros(self.ncell_all)
        for i, sp in enumerate(self.species):
            if sp is None or (s >= 0 and i != s):
                continue
            deposit_rho(self.g, self.order, sp.q, sp.w, sp.x, sp.y, sp.z, rho)
        return np.ascontiguousarray(self._phys(rho)).reshape(-1).copy()
