"""CPU-side checks of the boundary (no compute calls without a GPU): the C-ABI
library builds for sm_100a, loads, exports every symbol include/pic.h declares,
and its pure host functions behave as the header states."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2303_12873_b200.build import build_library
    from paper_2303_12873_b200 import binding
    build_library()
    return binding.load_library()


def test_header_symbols_all_exported(lib):
    from paper_2303_12873_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "pic.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pic_[a-z_]+)\s*\(", hdr))
    assert declared == set(binding.SYMBOLS)
    for name in declared:
        assert hasattr(lib, name), name


def test_probe_library_is_separate_and_the_product_library_never_allocates(lib):
    """include/pic_probes.h: the machine-rate probes (the only code that calls cudaMalloc) live in libpic_probes.so;
    libpic_b200.so exports none of them and does not even import cudaMalloc / cudaFree."""
    import subprocess
    from paper_2303_12873_b200 import binding, peaks
    hdr = open(os.path.join(ROOT, "include", "pic_probes.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    assert set(re.findall(r"\b(pic_[a-z_]+)\s*\(", hdr)) == set(peaks.PROBE_SYMBOLS)
    P = peaks.load_library()
    for name in peaks.PROBE_SYMBOLS:
        assert hasattr(P, name) and not hasattr(lib, name), name
    undefined = subprocess.run(["nm", "-D", "--undefined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    for sym in ("cudaMalloc", "cudaFree", "cudaMallocAsync", "cudaMallocManaged"):
        assert not re.search(r"\b%s\b" % sym, undefined), sym


def test_version_and_null_ctx_behaviour(lib):
    assert b"sm_100a" in lib.pic_version()
    assert lib.pic_last_error(None) == b"NULL context"
    assert lib.pic_step(None, 1) == -1
    assert lib.pic_sort(None) == -1
    assert lib.pic_sync(None) == -1
    assert lib.pic_destroy(None) == -1


def test_query_arena_is_pure_and_accounts_for_double_buffer():
    from paper_2303_12873_b200 import binding
    small = binding.query_arena(32, 32, 32, 1, [262144])
    # two SoA copies of 8 arrays of 8 bytes per particle, nine padded field components + one scratch
    assert small >= 2 * 8 * 8 * 262144 + 10 * 8 * 40 * 40 * 40
    assert small == binding.query_arena(32, 32, 32, 1, [262144])
    big = binding.query_arena(256, 256, 256, 3, [134217728])
    assert 2 * 64 * 134217728 < big < 24 * 2 ** 30          # config 2 fits one B200 several times over
    for bad in ((0, 4, 4, 1, [1]), (4, 4, 4, 0, [1]), (4, 4, 4, 4, [1]), (4, 4, 4, 1, [-1]), (4, 4, 4, 1, [2 ** 31])):
        with pytest.raises(binding.PicError) as e:
            binding.query_arena(*bad)
        assert e.value.code == binding.PIC_EINVAL


def test_init_rejects_bad_arguments_before_touching_the_gpu(lib):
    ctx = C.c_void_p()
    npm = (C.c_longlong * 1)(8)
    d = 0.5e-6
    # NULL arena, misaligned arena, dt too large: all PIC_EINVAL without a CUDA call
    assert lib.pic_init_grid(C.byref(ctx), 4, 4, 4, d, d, d, 0., 0., 0., 1e-16, 1, 1, npm, None, 1 << 30, None) == -1
    assert lib.pic_init_grid(C.byref(ctx), 4, 4, 4, d, d, d, 0., 0., 0., 1e-16, 1, 1, npm, C.c_void_p(264), 1 << 30,
                             None) == -1
    assert lib.pic_init_grid(C.byref(ctx), 4, 4, 4, d, d, d, 0., 0., 0., 1e-14, 1, 1, npm, C.c_void_p(256), 1 << 30,
                             None) == -1
    # arena too small: PIC_ENOMEM
    assert lib.pic_init_grid(C.byref(ctx), 4, 4, 4, d, d, d, 0., 0., 0., 1e-16, 1, 1, npm, C.c_void_p(256), 1024,
                             None) == -2
    assert not ctx.value


def test_binding_refuses_to_run_without_a_gpu():
    import torch
    from paper_2303_12873_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.Sim(4, 4, 4, 1e-6, 1e-6, 1e-6, 0, 0, 0, 1e-16, 1, [8])


def test_missing_library_fails_loudly(tmp_path):
    from paper_2303_12873_b200 import binding
    with pytest.raises(FileNotFoundError, match="no CPU fallback"):
        binding.load_library(str(tmp_path / "nope.so"))
