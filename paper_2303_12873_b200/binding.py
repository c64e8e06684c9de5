"""Thin ctypes binding of ``libpic_b200.so`` (include/pic.h).  Argument
marshalling only: every step of the PIC cycle runs in the CUDA kernels behind
the C ABI.  PyTorch supplies the device arena (one uint8 tensor) and the CUDA
stream; nothing else.  There is no CPU fallback: a missing library raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpic_b200.so")

PIC_OK, PIC_EINVAL, PIC_ENOMEM, PIC_ECUDA, PIC_ESTATE, PIC_EPHYS = 0, -1, -2, -3, -4, -5
PIC_NCOUNTERS = 9
PIC_NSTAGES = 8
_CODE_NAMES = {0: "PIC_OK", -1: "PIC_EINVAL", -2: "PIC_ENOMEM", -3: "PIC_ECUDA", -4: "PIC_ESTATE",
               -5: "PIC_EPHYS"}

# every symbol include/pic.h declares (tests check the library exports each one)
SYMBOLS = ("pic_query_arena", "pic_init_grid", "pic_set_fields", "pic_load_particles", "pic_step",
           "pic_sort", "pic_get_fields", "pic_get_particles", "pic_deposit_rho", "pic_get_cell_offsets",
           "pic_get_counters", "pic_get_stage_ms", "pic_set_option", "pic_sync", "pic_last_error",
           "pic_destroy", "pic_version", "pic_step_stage", "pic_halo_doubles", "pic_export_halo",
           "pic_import_halo", "pic_export_leavers", "pic_import_arrivals", "pic_shift_window", "pic_add_plane",
           "pic_set_damping")
# include/pic_noalloc.h
NOALLOC_SYMBOLS = ("pic_cell_offsets_noalloc", "pic_noalloc_last_error")
NOALLOC_MAX_CELLS = 2048 * 16384 - 1


class PicError(RuntimeError):
    def __init__(self, code: int, where: str, text: str = ""):
        self.code = code
        super().__init__("%s returned %s (%d)%s" % (where, _CODE_NAMES.get(code, "?"), code,
                                                    (": " + text) if text else ""))


_lib = None


def load_library(path: str | None = None):
    """dlopen the CUDA library and declare its prototypes.  Raises if missing."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise FileNotFoundError(
            "%s is missing: build it with `python -m paper_2303_12873_b200.build` "
            "(there is no CPU fallback)" % p)
    L = C.CDLL(p)
    vp, i, d, ll = C.c_void_p, C.c_int, C.c_double, C.c_longlong
    L.pic_version.restype = C.c_char_p
    L.pic_last_error.restype = C.c_char_p
    L.pic_last_error.argtypes = [vp]
    L.pic_query_arena.argtypes = [i, i, i, i, i, C.POINTER(ll), C.POINTER(C.c_size_t)]
    L.pic_init_grid.argtypes = [C.POINTER(vp), i, i, i, d, d, d, d, d, d, d, i, i, C.POINTER(ll), vp,
                                C.c_size_t, vp]
    L.pic_set_fields.argtypes = [vp] + [vp] * 6 + [i]
    L.pic_load_particles.argtypes = [vp, i, d, d, ll] + [vp] * 7 + [i]
    L.pic_step.argtypes = [vp, i]
    L.pic_sort.argtypes = [vp]
    L.pic_get_fields.argtypes = [vp] + [vp] * 9 + [i]
    L.pic_get_particles.argtypes = [vp, i, C.POINTER(ll)] + [vp] * 8 + [i]
    L.pic_deposit_rho.argtypes = [vp, i, vp, i]
    L.pic_get_cell_offsets.argtypes = [vp, i, vp, i]
    L.pic_get_counters.argtypes = [vp, C.POINTER(C.c_ulonglong)]
    L.pic_get_stage_ms.argtypes = [vp, C.POINTER(C.c_float)]
    L.pic_set_option.argtypes = [vp, C.c_char_p, ll]
    L.pic_sync.argtypes = [vp]
    L.pic_destroy.argtypes = [vp]
    L.pic_step_stage.argtypes = [vp, i]
    L.pic_halo_doubles.argtypes = [vp, i]
    L.pic_halo_doubles.restype = ll
    L.pic_export_halo.argtypes = [vp, i, i, i, vp]
    L.pic_import_halo.argtypes = [vp, i, i, i, vp]
    L.pic_export_leavers.argtypes = [vp, i, i, i, vp, ll, C.POINTER(ll)]
    L.pic_import_arrivals.argtypes = [vp, i, vp, ll, d, d, d]
    L.pic_shift_window.argtypes = [vp, i, C.POINTER(ll)]
    L.pic_add_plane.argtypes = [vp, i, i, vp, i]
    L.pic_set_damping.argtypes = [vp, i, C.POINTER(d)]
    L.pic_cell_offsets_noalloc.argtypes = [i, i, i, d, d, d, d, d, d, ll, vp, vp, vp, vp, vp]
    L.pic_cell_offsets_noalloc.restype = i
    L.pic_noalloc_last_error.argtypes = []
    L.pic_noalloc_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        if name not in ("pic_version", "pic_last_error"):
            getattr(L, name).restype = i
    if path is None:
        _lib = L
    return L


def query_arena(nx, ny, nz, order, np_max) -> int:
    L = load_library()
    arr = (C.c_longlong * len(np_max))(*[int(v) for v in np_max])
    out = C.c_size_t(0)
    rc = L.pic_query_arena(nx, ny, nz, order, len(np_max), arr, C.byref(out))
    if rc != PIC_OK:
        raise PicError(rc, "pic_query_arena")
    return int(out.value)


def cell_offsets_noalloc(nx, ny, nz, dx, dy, dz, xmin, ymin, zmin, x, y, z, offsets, stream=None):
    """pic_cell_offsets_noalloc (include/pic_noalloc.h): for callers that may not allocate device memory (a
    hook inside another code's loop whose pool owns the GPU, a latency-critical step, an out-of-memory
    path), the counting sort's cell-offset table from caller buffers only.  x, y, z: torch.cuda float64
    tensors of n entries; offsets: a torch.cuda int32/uint32 tensor of nx*ny*nz + 1 entries that the caller
    owns and this call overwrites.  Queued on `stream` (default: torch's current stream of that device);
    the library's 64 KiB built-in scratch is shared, so do not overlap two calls on one GPU."""
    import torch
    L = load_library()
    n = int(x.numel())
    for a in (x, y, z):
        assert a.is_cuda and a.is_contiguous() and a.dtype == torch.float64 and a.numel() == n
    assert offsets.is_cuda and offsets.is_contiguous() and offsets.element_size() == 4
    assert offsets.numel() >= nx * ny * nz + 1
    with torch.cuda.device(offsets.device):
        st = stream if stream is not None else torch.cuda.current_stream(offsets.device)
        rc = L.pic_cell_offsets_noalloc(nx, ny, nz, dx, dy, dz, xmin, ymin, zmin, n,
                                        C.c_void_p(x.data_ptr()) if n else None,
                                        C.c_void_p(y.data_ptr()) if n else None,
                                        C.c_void_p(z.data_ptr()) if n else None,
                                        C.c_void_p(offsets.data_ptr()), C.c_void_p(st.cuda_stream))
    if rc != PIC_OK:
        raise PicError(rc, "pic_cell_offsets_noalloc", (L.pic_noalloc_last_error() or b"").decode())


def _is_torch(a) -> bool:
    return hasattr(a, "data_ptr") and hasattr(a, "is_cuda")


def _ptr(a, dtype_np, want_device: bool):
    """Address of a contiguous float64/uint64 buffer (numpy = host, torch.cuda = device)."""
    if a is None:
        return None
    if _is_torch(a):
        assert a.is_contiguous(), "need a contiguous tensor"
        assert a.is_cuda == want_device, "mixing host and device buffers in one call"
        assert a.element_size() == np.dtype(dtype_np).itemsize
        return C.c_void_p(a.data_ptr())
    assert not want_device, "mixing host and device buffers in one call"
    assert a.dtype == dtype_np and a.flags["C_CONTIGUOUS"], "need contiguous %s" % dtype_np
    return C.c_void_p(a.ctypes.data)


def _on_device(arrs) -> bool:
    return any(_is_torch(a) and a.is_cuda for a in arrs if a is not None)


def _prep(a, dtype=np.float64):
    """Host inputs become contiguous numpy arrays of the right dtype; device tensors pass through."""
    if a is None or _is_torch(a):
        return a
    return np.ascontiguousarray(a, dtype=dtype).reshape(-1)


class Sim:
    """One simulation on one GPU: mirrors the C ABI call for call."""

    FIELD_NAMES = ("Ex", "Ey", "Ez", "Bx", "By", "Bz", "Jx", "Jy", "Jz")

    def __init__(self, nx, ny, nz, dx, dy, dz, xmin, ymin, zmin, dt, order, np_max, device="cuda:0",
                 stream=None):
        import torch  # device memory and streams only
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: libpic_b200 has no CPU fallback")
        self._L = load_library()
        self._torch = torch
        self.device = torch.device(device)
        self.nx, self.ny, self.nz, self.order = int(nx), int(ny), int(nz), int(order)
        self.ncell = self.nx * self.ny * self.nz
        self.np_max = [int(v) for v in np_max]
        self.nspecies = len(self.np_max)
        nbytes = query_arena(nx, ny, nz, order, self.np_max)
        self.arena_bytes = nbytes
        with torch.cuda.device(self.device):
            self.arena = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.arena.data_ptr()
            self._arena_ptr = (base + 255) // 256 * 256
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            arr = (C.c_longlong * self.nspecies)(*self.np_max)
            ctx = C.c_void_p()
            rc = self._L.pic_init_grid(C.byref(ctx), nx, ny, nz, dx, dy, dz, xmin, ymin, zmin, dt, order,
                                       self.nspecies, arr, C.c_void_p(self._arena_ptr), nbytes,
                                       C.c_void_p(self.stream.cuda_stream))
        if rc != PIC_OK:
            raise PicError(rc, "pic_init_grid")
        self._ctx = ctx

    @classmethod
    def from_workload(cls, wl, device="cuda:0", load=True, np_max=None):
        sim = cls(*wl.grid_args(), wl.dt, wl.order, np_max or [max(s.n, 1) for s in wl.species], device=device)
        if load:
            if wl.fields:
                sim.set_fields(**wl.fields)
            for s, sp in enumerate(wl.species):
                sim.load_particles(s, sp.q, sp.m, *sp.arrays())
        return sim

    # -- helpers ---------------------------------------------------------------
    def _check(self, rc, where):
        if rc != PIC_OK:
            raise PicError(rc, where, (self._L.pic_last_error(self._ctx) or b"").decode())

    def close(self):
        if getattr(self, "_ctx", None):
            self._L.pic_destroy(self._ctx)
            self._ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C ABI, call for call ------------------------------------------------
    def set_fields(self, Ex=None, Ey=None, Ez=None, Bx=None, By=None, Bz=None):
        arrs = [_prep(a) for a in (Ex, Ey, Ez, Bx, By, Bz)]
        dev = _on_device(arrs)
        for a in arrs:
            assert a is None or (a.numel() if _is_torch(a) else a.size) == self.ncell
        self._check(self._L.pic_set_fields(self._ctx, *[_ptr(a, np.float64, dev) for a in arrs], int(dev)),
                    "pic_set_fields")

    def load_particles(self, species, q, m, x, y, z, ux, uy, uz, w):
        arrs = [_prep(a) for a in (x, y, z, ux, uy, uz, w)]
        dev = _on_device(arrs)
        n = arrs[0].numel() if _is_torch(arrs[0]) else arrs[0].size
        for a in arrs:
            assert (a.numel() if _is_torch(a) else a.size) == n
        self._check(self._L.pic_load_particles(self._ctx, species, q, m, n,
                                               *[_ptr(a, np.float64, dev) for a in arrs], int(dev)),
                    "pic_load_particles")

    def step(self, nsteps=1):
        self._check(self._L.pic_step(self._ctx, int(nsteps)), "pic_step")

    def sort(self):
        self._check(self._L.pic_sort(self._ctx), "pic_sort")

    def sync(self):
        self._check(self._L.pic_sync(self._ctx), "pic_sync")

    def get_fields(self, names=FIELD_NAMES, device=False):
        """dict name -> flat array (numpy on host, or torch on the device)."""
        out = {}
        ptrs = []
        for nm in self.FIELD_NAMES:
            if nm in names:
                out[nm] = (self._torch.empty(self.ncell, dtype=self._torch.float64, device=self.device)
                           if device else np.empty(self.ncell))
                ptrs.append(_ptr(out[nm], np.float64, device))
            else:
                ptrs.append(None)
        self._check(self._L.pic_get_fields(self._ctx, *ptrs, int(device)), "pic_get_fields")
        return out

    def num_particles(self, species) -> int:
        n = C.c_longlong(0)
        self._check(self._L.pic_get_particles(self._ctx, species, C.byref(n), *([None] * 8), 0),
                    "pic_get_particles")
        return int(n.value)

    def get_particles(self, species, device=False):
        n = self.num_particles(species)
        out = {}
        t = self._torch
        for nm in ("x", "y", "z", "ux", "uy", "uz", "w"):
            out[nm] = t.empty(n, dtype=t.float64, device=self.device) if device else np.empty(n)
        out["id"] = (t.empty(n, dtype=t.int64, device=self.device) if device
                     else np.empty(n, dtype=np.uint64))
        nn = C.c_longlong(0)
        ptrs = [_ptr(out[nm], np.float64, device) for nm in ("x", "y", "z", "ux", "uy", "uz", "w")]
        ptrs.append(_ptr(out["id"], np.uint64, device))
        self._check(self._L.pic_get_particles(self._ctx, species, C.byref(nn), *ptrs, int(device)),
                    "pic_get_particles")
        return out

    def get_fields_into(self, out):
        """pic_get_fields into caller buffers: dict name -> contiguous float64 buffer of ncell entries
        (numpy / pinned torch CPU tensors = host, torch.cuda tensors = device); missing names are skipped."""
        dev = _on_device(out.values())
        ptrs = [_ptr(out.get(nm), np.float64, dev) for nm in self.FIELD_NAMES]
        self._check(self._L.pic_get_fields(self._ctx, *ptrs, int(dev)), "pic_get_fields")

    def get_particles_into(self, species, out):
        """pic_get_particles into caller buffers: dict with any of x,y,z,ux,uy,uz,w (float64) and id (uint64/int64)."""
        dev = _on_device(out.values())
        nn = C.c_longlong(0)
        ptrs = [_ptr(out.get(nm), np.float64, dev) for nm in ("x", "y", "z", "ux", "uy", "uz", "w")]
        ptrs.append(_ptr(out.get("id"), np.uint64, dev))
        self._check(self._L.pic_get_particles(self._ctx, species, C.byref(nn), *ptrs, int(dev)),
                    "pic_get_particles")
        return int(nn.value)

    def deposit_rho(self, species=-1, device=False):
        t = self._torch
        rho = t.empty(self.ncell, dtype=t.float64, device=self.device) if device else np.empty(self.ncell)
        self._check(self._L.pic_deposit_rho(self._ctx, species, _ptr(rho, np.float64, device), int(device)),
                    "pic_deposit_rho")
        return rho

    def get_cell_offsets(self, species):
        off = np.empty(self.ncell + 1, dtype=np.uint32)
        self._check(self._L.pic_get_cell_offsets(self._ctx, species, C.c_void_p(off.ctypes.data), 0),
                    "pic_get_cell_offsets")
        return off

    def counters(self):
        arr = (C.c_ulonglong * PIC_NCOUNTERS)()
        self._check(self._L.pic_get_counters(self._ctx, arr), "pic_get_counters")
        v = list(arr)
        return {"fast": v[0], "slow": v[1], "global": v[2], "launches": v[3], "steps": v[4], "sorts": v[5],
                "yee_tma": v[6], "fallbacks": v[7], "deleted": v[8]}

    # -- NEXT-1: brick calls (device buffers = torch.cuda float64 tensors) -------------------------
    def step_stage(self, stage):
        self._check(self._L.pic_step_stage(self._ctx, int(stage)), "pic_step_stage")

    def halo_doubles(self, dim):
        n = self._L.pic_halo_doubles(self._ctx, int(dim))
        if n < 0:
            raise PicError(PIC_EINVAL, "pic_halo_doubles")
        return int(n)

    def export_halo(self, group, dim, side, buf):
        assert buf.is_cuda and buf.dtype == self._torch.float64 and buf.numel() >= self.halo_doubles(dim)
        self._check(self._L.pic_export_halo(self._ctx, group, dim, side, C.c_void_p(buf.data_ptr())), "pic_export_halo")

    def import_halo(self, group, dim, side, buf):
        assert buf.is_cuda and buf.dtype == self._torch.float64 and buf.numel() >= self.halo_doubles(dim)
        self._check(self._L.pic_import_halo(self._ctx, group, dim, side, C.c_void_p(buf.data_ptr())), "pic_import_halo")

    def export_leavers(self, species, dim, side, buf):
        """buf: torch.cuda float64 tensor of 8 * capacity entries.  Returns the number of records written."""
        assert buf.is_cuda and buf.dtype == self._torch.float64
        cnt = C.c_longlong(0)
        self._check(self._L.pic_export_leavers(self._ctx, species, dim, side, C.c_void_p(buf.data_ptr()),
                                               buf.numel() // 8, C.byref(cnt)), "pic_export_leavers")
        return int(cnt.value)

    def import_arrivals(self, species, buf, count, shift=(0.0, 0.0, 0.0)):
        assert count == 0 or (buf.is_cuda and buf.dtype == self._torch.float64 and buf.numel() >= 8 * count)
        self._check(self._L.pic_import_arrivals(self._ctx, species, C.c_void_p(buf.data_ptr()) if count else None,
                                                int(count), float(shift[0]), float(shift[1]), float(shift[2])),
                    "pic_import_arrivals")

    # -- NEXT-2: moving window, plane source, fresh plasma ---------------------------------------
    def shift_window(self, ncells=1):
        """Returns the number of particles the window left behind (deleted)."""
        n = C.c_longlong(0)
        self._check(self._L.pic_shift_window(self._ctx, int(ncells), C.byref(n)), "pic_shift_window")
        return int(n.value)

    def add_plane(self, name, k, values):
        """F[:, :, k] += values (ny x nx, x fastest; numpy on the host or a torch.cuda tensor)."""
        dev = _on_device([values])
        self._check(self._L.pic_add_plane(self._ctx, self.FIELD_NAMES.index(name), int(k),
                                          _ptr(values, np.float64, dev), int(dev)), "pic_add_plane")

    def set_damping(self, factors):
        """Absorbing layers in front of the open z ends: factors[m] scales E and B on the plane m cells from a face."""
        f = np.ascontiguousarray(factors, dtype=np.float64).reshape(-1)
        self._check(self._L.pic_set_damping(self._ctx, int(f.size), f.ctypes.data_as(C.POINTER(C.c_double))),
                    "pic_set_damping")

    def append_particles(self, species, x, y, z, ux, uy, uz, w, ids):
        """Appends particles given as host arrays (marshalled into the 8-double records of pic_import_arrivals)."""
        t = self._torch
        n = len(x)
        if n == 0:
            return
        rec = np.empty((n, 8))
        for k, a in enumerate((x, y, z, ux, uy, uz, w)):
            rec[:, k] = a
        rec[:, 7] = np.asarray(ids, dtype=np.uint64).view(np.float64)
        buf = t.from_numpy(rec.reshape(-1)).to(self.device)
        self.import_arrivals(species, buf, n)
        self.sync()

    def set_option(self, name, value):
        self._check(self._L.pic_set_option(self._ctx, name.encode(), int(value)), "pic_set_option")

    def stage_ms(self):
        arr = (C.c_float * PIC_NSTAGES)()
        self._check(self._L.pic_get_stage_ms(self._ctx, arr), "pic_get_stage_ms")
        return dict(zip(("zero_J", "particles", "fold_J", "yee_B", "yee_E", "sort", "steps", "sorts"), list(arr)))

    def last_error(self) -> str:
        return (self._L.pic_last_error(self._ctx) or b"").decode()
