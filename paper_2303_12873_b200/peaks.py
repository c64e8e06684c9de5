"""Measured machine rates behind the rooflines ("Builder must
measure first"): fp64 DFMA issue rate, the shared-memory return path for
LDS.64 / LDS.128 with 1 .. 32 distinct addresses per warp in the fused
kernel's [x][z][y] stencil strides, and the global ``red.add.f64`` rate.

    python -m paper_2303_12873_b200.peaks            # markdown tables + one JSON line
    python -m paper_2303_12873_b200.peaks --lds      # only the LDS table (one launch per row: for ncu)

Argument marshalling only; the probes are CUDA kernels behind the C ABI
(``pic_probe_*`` in include/pic_probes.h, csrc/peaks.cu, built into libpic_probes.so).
"""
from __future__ import annotations

import ctypes as C
import json
import sys

import os

from .binding import PIC_OK, PicError

PROBE_SYMBOLS = ("pic_probe_dfma", "pic_probe_dmma", "pic_probe_lds", "pic_probe_red")
_PROBE_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libpic_probes.so")
_probe_lib = None


def load_library():
    """dlopen libpic_probes.so (include/pic_probes.h): the probes allocate device memory themselves, so they
    are kept out of libpic_b200.so.  Raises if it has not been built."""
    global _probe_lib
    if _probe_lib is None:
        if not os.path.exists(_PROBE_LIB_PATH):
            raise FileNotFoundError("%s is missing: build it with `python -m paper_2303_12873_b200.build`" % _PROBE_LIB_PATH)
        L = C.CDLL(_PROBE_LIB_PATH)
        i, d, ll = C.c_int, C.c_double, C.c_longlong
        L.pic_probe_dfma.argtypes = [i, i, C.POINTER(d)]
        L.pic_probe_dmma.argtypes = [i, i, C.POINTER(d)]
        L.pic_probe_lds.argtypes = [i, C.POINTER(i), C.c_uint, i, i, i, C.POINTER(d)]
        L.pic_probe_red.argtypes = [i, ll, ll, i, C.POINTER(d)]
        for name in PROBE_SYMBOLS:
            getattr(L, name).restype = i
        _probe_lib = L
    return _probe_lib

# the fresh-sort tile kernel's stencil strides: word(x, y, z) = y + SZ z + SX x
SZ, SX = 8, 66
PLANE = 8 * SX          # displacement between a probe's eight loads: same banks, other words


def _word(x, y, z):
    return y + SZ * z + SX * x


def lds_patterns(vec_bytes):
    """(name, number of distinct addresses, lane -> word map) in the gather's address patterns."""
    ys = 1 if vec_bytes == 8 else 2          # LDS.128 needs even words
    out = []
    for d in (1, 2, 4, 5, 8):
        out.append(("%d cell%s along x" % (d, "" if d == 1 else "s"), d,
                    [_word(1 + (l * d) // 32, 0, 1) for l in range(32)]))
    out.append(("4 cells x stagger shift in y and z", 16,
                [_word(1 + l // 8, ys * (1 - (l & 1)), 1 - ((l >> 1) & 1)) for l in range(32)]))
    step = 1 if vec_bytes == 8 else 2
    out.append(("32 consecutive %d-byte words" % vec_bytes, 32, [64 + step * l for l in range(32)]))
    return out


def _cells(sizes):
    """lane -> word map from a list of run lengths: run r reads the stencil word of cell r (distinct banks)."""
    words = []
    for r, n in enumerate(sizes):
        words += [_word(1 + r % 8, r // 8, 1)] * n        # r < 8: even 8-byte banks, r >= 8: the odd ones
    assert len(words) == 32
    return words


def rule_patterns():
    """Lane patterns that tell apart the possible rules for when an LDS.64 is served in ONE wavefront
    (all words used here sit in different 8-byte banks, so none of the patterns has a bank conflict)."""
    return [
        ("16 cells, 2 lanes each (pairs equal)", _cells([2] * 16)),
        ("2 cells alternating by lane (l & 1)", [_word(1 + (l & 1), 0, 1) for l in range(32)]),
        ("2 cells alternating by pair ((l >> 1) & 1)", [_word(1 + ((l >> 1) & 1), 0, 1) for l in range(32)]),
        ("runs 6,6,4,6,6,4 (even boundaries, mixed quads)", _cells([6, 6, 4, 6, 6, 4])),
        ("runs 2,4,4,4,2,2,4,4,4,2 (pairs equal, quads mixed)", _cells([2, 4, 4, 4, 2, 2, 4, 4, 4, 2])),
        ("runs 7,25 (one odd boundary)", _cells([7, 25])),
        ("runs 8,24", _cells([8, 24])),
        ("runs 9,23", _cells([9, 23])),
        ("runs 7,9,7,9 (odd boundaries inside both half-warps)", _cells([7, 9, 7, 9])),
        ("runs of 3 (11 cells)", _cells([3] * 10 + [2])),
        ("lane l reads word l % 16 (half-warps read the same 16 consecutive words)", [64 + (l % 16) for l in range(32)]),
        ("lane l reads word l % 8", [64 + (l % 8) for l in range(32)]),
        ("lane l reads word l // 2 (16 consecutive words, pairs equal)", [64 + l // 2 for l in range(32)]),
        ("lane l reads word l // 4 (8 consecutive words)", [64 + l // 4 for l in range(32)]),
        ("lanes l and l ^ 16 equal, 16 cells", [_word(1 + (l % 16) % 8, (l % 16) // 8, 1) for l in range(32)]),
    ]


def rule_table(warps=32):
    rows = []
    for k, (name, words) in enumerate(rule_patterns()):
        clk = probe_lds(8, words, 0xFFFFFFFF, warps)
        rows.append({"launch": k, "pattern": name, "distinct": len(set(words)), "clk_per_warp_instr_per_sm": clk})
    return rows


def probe_dfma(warps, iters=4000):
    L = load_library()
    out = C.c_double(0.0)
    rc = L.pic_probe_dfma(warps, iters, C.byref(out))
    if rc != PIC_OK:
        raise PicError(rc, "pic_probe_dfma")
    return out.value


def probe_dmma(warps, iters=2000):
    L = load_library()
    out = C.c_double(0.0)
    rc = L.pic_probe_dmma(warps, iters, C.byref(out))
    if rc != PIC_OK:
        raise PicError(rc, "pic_probe_dmma")
    return out.value


def probe_lds(vec_bytes, lane_word, active_mask, warps, iters=4000, plane=PLANE):
    L = load_library()
    arr = (C.c_int * 32)(*lane_word)
    out = C.c_double(0.0)
    rc = L.pic_probe_lds(vec_bytes, arr, active_mask, plane, warps, iters, C.byref(out))
    if rc != PIC_OK:
        raise PicError(rc, "pic_probe_lds")
    return out.value


def probe_red(pattern, footprint, plane=264 * 264, n=64):
    L = load_library()
    out = C.c_double(0.0)
    rc = L.pic_probe_red(pattern, footprint, plane, n, C.byref(out))
    if rc != PIC_OK:
        raise PicError(rc, "pic_probe_red")
    return out.value


ACTIVE = ((32, 0xFFFFFFFF), (26, 0x03FFFFFF), (16, 0x0000FFFF))
RED_PATTERNS = ("32 consecutive doubles per warp (8 sectors)", "one 32-byte sector per lane",
                "one 128-byte line per lane", "all lanes one double",
                "flush-like: 8 places x 4 planes", "8 places x 4 consecutive doubles")


def lds_table(warps_list=(8, 16, 32)):
    rows = []
    k = 0
    for vec in (8, 16):
        for name, d, words in lds_patterns(vec):
            for nact, mask in ACTIVE:
                for w in warps_list:
                    clk = probe_lds(vec, words, mask, w)
                    rows.append({"launch": k, "op": "LDS.%d" % (8 * vec), "pattern": name, "distinct": d,
                                 "active_lanes": nact, "warps_per_sm": w, "clk_per_warp_instr_per_sm": clk,
                                 "bytes_per_clk_per_sm": nact * vec / clk})
                    k += 1
    return rows


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    import torch          # only to make a CUDA context current on device 0
    torch.cuda.set_device(0)
    torch.cuda.synchronize()
    res = {}
    if "--rule" in argv:      # only the rule finder (one launch per row: for ncu)
        print("| # | LDS.64 lane pattern (32 active lanes, 32 warps/SM) | distinct addr | clk per warp instr per SM |\n|---|---|---|---|")
        for r in rule_table():
            print("| %d | %s | %d | %.2f |" % (r["launch"], r["pattern"], r["distinct"], r["clk_per_warp_instr_per_sm"]))
        return res
    if "--lds" not in argv:
        print("## DFMA (one block per SM, 8 independent chains per thread)\n")
        print("| warps/SM | clk per warp DFMA per SM | fp64 lanes/clk/SM |\n|---|---|---|")
        res["dfma"] = []
        for w in (4, 8, 16, 32):
            clk = probe_dfma(w)
            res["dfma"].append({"warps_per_sm": w, "clk_per_warp_instr_per_sm": clk, "lanes_per_clk": 32.0 / clk})
            print("| %d | %.3f | %.1f |" % (w, clk, 32.0 / clk))
    if "--lds" not in argv:
        print("\n## DMMA m8n8k4 (256 FMA per warp instruction, 8 independent accumulator fragments per warp)\n")
        print("| warps/SM | clk per warp DMMA per SM | fp64 FMA/clk/SM |\n|---|---|---|")
        res["dmma"] = []
        for w in (4, 8, 16):
            clk = probe_dmma(w)
            res["dmma"].append({"warps_per_sm": w, "clk_per_warp_instr_per_sm": clk, "fma_per_clk": 256.0 / clk})
            print("| %d | %.3f | %.1f |" % (w, clk, 256.0 / clk))
    print("\n## Shared-memory loads, word(x,y,z) = y + %d z + %d x (fresh tile stencil)\n" % (SZ, SX))
    print("| # | op | lane pattern | distinct addr | active lanes | warps/SM | clk per warp instr per SM |"
          " lane bytes/clk/SM |\n|---|---|---|---|---|---|---|---|")
    res["lds"] = lds_table()
    for r in res["lds"]:
        print("| %d | %s | %s | %d | %d | %d | %.2f | %.0f |" % (
            r["launch"], r["op"], r["pattern"], r["distinct"], r["active_lanes"], r["warps_per_sm"],
            r["clk_per_warp_instr_per_sm"], r["bytes_per_clk_per_sm"]))
    if "--lds" not in argv:
        print("\n## red.global.add.f64 (whole GPU, 8 x 256 threads per SM, 64 REDs per thread)\n")
        print("| pattern | footprint | G lane-REDs/s |\n|---|---|---|")
        res["red"] = []
        for fp, label in ((5 << 20, "40 MB (L2-resident)"), (65 << 20, "520 MB (three 256^3 J components are 430 MB)")):
            for p, name in enumerate(RED_PATTERNS):
                v = probe_red(p, fp)
                res["red"].append({"pattern": name, "footprint_doubles": fp, "lane_reds_per_s": v})
                print("| %s | %s | %.1f |" % (name, label, v / 1e9))
    print("\nJSON " + json.dumps(res))
    return res


if __name__ == "__main__":
    main()
