"""Measured machine rates behind the rooflines ("Builder must
measure first"): fp64 DFMA issue rate, the shared-memory return path for
LDS.64 / LDS.128 with 1 .. 32 distinct addresses per warp in the fused
kernel's [x][z][y] stencil strides, and the global ``red.add.f64`` rate.

    python -m paper_2303_12873_b200.peaks            # markdown tables + one JSON line
    python -m paper_2303_12873_b200.peaks --lds      # only the LDS table (one launch per row: for ncu)

Argument marshalling only; the probes are CUDA kernels behind the C ABI
(``pic_probe_*`` in include/pic.h, csrc/peaks.cu).
"""
from __future__ import annotations

import ctypes as C
import json
import sys

from .binding import PIC_OK, PicError, load_library

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


def probe_dfma(warps, iters=4000):
    L = load_library()
    out = C.c_double(0.0)
    rc = L.pic_probe_dfma(warps, iters, C.byref(out))
    if rc != PIC_OK:
        raise PicError(rc, "pic_probe_dfma")
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


def lds_table(warps_list=(8, 16)):
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
    if "--lds" not in argv:
        print("## DFMA (one block per SM, 8 independent chains per thread)\n")
        print("| warps/SM | clk per warp DFMA per SM | fp64 lanes/clk/SM |\n|---|---|---|")
        res["dfma"] = []
        for w in (4, 8, 16, 32):
            clk = probe_dfma(w)
            res["dfma"].append({"warps_per_sm": w, "clk_per_warp_instr_per_sm": clk, "lanes_per_clk": 32.0 / clk})
            print("| %d | %.3f | %.1f |" % (w, clk, 32.0 / clk))
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
