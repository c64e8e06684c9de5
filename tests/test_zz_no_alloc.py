"""pic_cell_offsets_noalloc (include/pic_noalloc.h): the counting sort's cell-offset table for callers
that cannot allocate device memory -- a hook running inside another code's time loop whose memory pool
already owns the GPU, a step where cudaMalloc's device-wide synchronisation is not affordable, a
diagnostic on an out-of-memory path.  Its scan scratch is a 64 KiB array built into the library image
instead of a slice of the caller's arena.

The GPU test checks it, bit for bit (integer work), against the arena-based path
(pic_sort + pic_get_cell_offsets) on two calls in a row that share the built-in scratch, the second on a
smaller grid so that stale chunk totals of the first are lying around; then a third, and that the
device's free memory did not move.  This file sorts last on purpose: `pytest -x` stops at the first
failure and nothing should hide behind this one.  It passes alone in a fresh process (the first call
does the one-time address look-up) and after the other tests."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2303_12873_b200.build import build_library
    from paper_2303_12873_b200 import binding
    build_library()
    return binding.load_library()


def test_noalloc_header_symbols_exported(lib):
    from paper_2303_12873_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "pic_noalloc.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pic_[a-z_]+)\s*\(", hdr))
    assert declared == set(binding.NOALLOC_SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name
    m = re.search(r"#define\s+PIC_NOALLOC_MAX_CHUNKS\s+(\d+)", hdr)
    assert 2048 * int(m.group(1)) - 1 == binding.NOALLOC_MAX_CELLS
    assert 4 * int(m.group(1)) == 64 * 1024           # the "modest" built-in scratch: 64 KiB per GPU


def test_noalloc_rejects_bad_sizes_before_any_cuda_call(lib):
    """Every argument error is found on the host, so these run without a GPU; the text names the limit."""
    d = 0.5e-6
    one = C.c_void_p(256)     # never dereferenced: the call must fail first

    def call(nx, ny, nz, n, x=one, off=one, dx=d):
        return lib.pic_cell_offsets_noalloc(nx, ny, nz, dx, d, d, 0., 0., 0., n, x, x, x, off, None)

    assert call(512, 256, 256, 10) == -1               # 33,554,432 cells: one more than the scratch can scan
    msg = lib.pic_noalloc_last_error().decode()
    assert "PIC_NOALLOC_MAX_CELLS" in msg and "33554431" in msg and "33554432" in msg
    assert call(0, 4, 4, 1) == -1 and call(4, 4, -1, 1) == -1
    assert call(4, 4, 4, -1) == -1 and call(4, 4, 4, 2 ** 31) == -1
    assert call(4, 4, 4, 1, off=None) == -1 and call(4, 4, 4, 1, x=None) == -1
    assert call(4, 4, 4, 1, dx=0.0) == -1 and call(4, 4, 4, 1, dx=float("nan")) == -1
    assert lib.pic_noalloc_last_error() != b""


def _positions(rng, nx, ny, nz, dx, dy, dz, n, clustered):
    """Seeded positions inside the box; `clustered` piles a third of them into one corner octant so that cell
    occupancies range from 0 to hundreds (empty cells and long runs both reach the scan)."""
    x = rng.random(n) * nx * dx
    y = rng.random(n) * ny * dy
    z = rng.random(n) * nz * dz
    if clustered:
        m = n // 3
        x[:m] *= 0.25; y[:m] *= 0.25; z[:m] *= 0.25
    # a few on cell faces and on the low box faces (floor() of an exact integer)
    x[-4:] = np.array([0.0, dx, 2 * dx, (nx - 1) * dx])
    y[-4:] = np.array([0.0, dy, 0.0, (ny - 1) * dy])
    z[-4:] = np.array([0.0, 0.0, dz, (nz - 1) * dz])
    return x, y, z


def _existing_path(Sim, grid, dt, x, y, z):
    """Cell offsets the arena-based library path produces: load, pic_sort, pic_get_cell_offsets."""
    n = x.size
    sim = Sim(*grid, dt, 1, [max(n, 1)])
    zero = np.zeros(n)
    sim.load_particles(0, -1.602176634e-19, 9.1093837015e-31, x, y, z, zero, zero, zero, np.ones(n))
    sim.sort()
    off = sim.get_cell_offsets(0)
    sim.close()
    return off


def _by_definition(grid, x, y, z):
    nx, ny, nz, dx, dy, dz, x0, y0, z0 = grid
    i = np.clip(np.floor((x - x0) * (1.0 / dx)).astype(np.int64), 0, nx - 1)
    j = np.clip(np.floor((y - y0) * (1.0 / dy)).astype(np.int64), 0, ny - 1)
    k = np.clip(np.floor((z - z0) * (1.0 / dz)).astype(np.int64), 0, nz - 1)
    cnt = np.bincount(i + nx * (j + ny * k), minlength=nx * ny * nz)
    return np.concatenate([[0], np.cumsum(cnt)]).astype(np.uint32)


@pytest.mark.gpu
def test_noalloc_cell_offsets_match_the_sort_path_on_consecutive_calls():
    import torch
    from paper_2303_12873_b200 import binding
    from paper_2303_12873_b200.binding import Sim
    from paper_2303_12873_b200.workloads import courant_dt

    dev = torch.device("cuda:0")
    rng = np.random.default_rng(20231287)
    # (grid, particles, clustered): 53,761 counters = 26 full chunks + a ragged one; then 106 counters (one
    # partial chunk, scratch entries 1..26 stale from the call before); then 1,048,577 counters = 513 chunks
    cases = [((40, 24, 56, 0.5e-6, 0.4e-6, 0.7e-6, -3e-6, 1e-6, 0.0), 300_007, True),
             ((5, 3, 7, 1e-6, 1e-6, 1e-6, 0.0, 0.0, 0.0), 1_001, False),
             ((128, 64, 128, 0.5e-6, 0.5e-6, 0.5e-6, 0.0, 0.0, 0.0), 2_000_003, True)]
    host, expect = [], []
    for grid, n, clustered in cases:
        nx, ny, nz, dx, dy, dz, x0, y0, z0 = grid
        x, y, z = _positions(rng, nx, ny, nz, dx, dy, dz, n, clustered)
        x += x0; y += y0; z += z0
        # keep the shifted positions strictly inside [min, max) as pic_load_particles demands
        x = np.minimum(x, np.nextafter(x0 + nx * dx, -np.inf)); x = np.maximum(x, x0)
        y = np.minimum(y, np.nextafter(y0 + ny * dy, -np.inf)); y = np.maximum(y, y0)
        z = np.minimum(z, np.nextafter(z0 + nz * dz, -np.inf)); z = np.maximum(z, z0)
        host.append((x, y, z))
        expect.append(_existing_path(Sim, grid, courant_dt(dx, dy, dz), x, y, z))
        # the existing path itself against the plain definition, so that both sides are anchored
        assert np.array_equal(expect[-1], _by_definition(grid, x, y, z))

    # everything the calls touch exists before the first of them: the entry point gets inputs and outputs only
    dev_in = [tuple(torch.from_numpy(a).to(dev) for a in xyz) for xyz in host]
    outs = [torch.full((g[0] * g[1] * g[2] + 1,), -1, dtype=torch.int32, device=dev) for g, _, _ in cases]
    empty_out = torch.full((5 * 3 * 7 + 1,), -1, dtype=torch.int32, device=dev)
    nothing = torch.empty(0, dtype=torch.float64, device=dev)
    torch.cuda.synchronize()

    # two calls in a row on one stream, no synchronisation in between: they share the built-in scratch
    for c in (0, 1):
        binding.cell_offsets_noalloc(*cases[c][0], *dev_in[c], outs[c])
    torch.cuda.synchronize()
    for c in (0, 1):
        got = outs[c].cpu().numpy().view(np.uint32)
        assert np.array_equal(got, expect[c]), "call %d differs from pic_sort's offsets" % (c + 1)

    # set-up is done by now: further calls must leave the device's free memory exactly where it is
    free_before, _ = torch.cuda.mem_get_info(dev)
    binding.cell_offsets_noalloc(*cases[2][0], *dev_in[2], outs[2])
    binding.cell_offsets_noalloc(*cases[1][0], nothing, nothing, nothing, empty_out)      # n = 0
    outs[0].fill_(-1)
    binding.cell_offsets_noalloc(*cases[0][0], *dev_in[0], outs[0])                        # first case again
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info(dev)
    assert free_after == free_before, "device memory moved by %d bytes" % (free_before - free_after)
    assert np.array_equal(outs[2].cpu().numpy().view(np.uint32), expect[2])
    assert not empty_out.any().item()
    assert np.array_equal(outs[0].cpu().numpy().view(np.uint32), expect[0])

    # beyond the limit: refused with the limit in the text, nothing queued, output untouched
    with pytest.raises(binding.PicError) as e:
        binding.cell_offsets_noalloc(512, 256, 256, 1e-6, 1e-6, 1e-6, 0.0, 0.0, 0.0, *dev_in[1],
                                     torch.empty(512 * 256 * 256 + 1, dtype=torch.int32, device=dev))
    assert e.value.code == binding.PIC_EINVAL and "PIC_NOALLOC_MAX_CELLS" in str(e.value)
