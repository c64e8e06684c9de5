#!/usr/bin/env python
"""bench.py -- throughput of the whole PIC hot path on B200 (driver contract).

A "step" is one pass of every row of SURVEY.md 8(a): zero J, fused
gather + Boris push + Esirkepov deposition (all species), J guard fold, Yee
B half / E / B half, with the per-cell counting sort run every
``sort_every`` steps INSIDE the timed region (so its cost is amortised into
the step time).  N = 1 workload: BASELINE.json configs[2] (256^3 cells, 8 ppc
electrons = 134,217,728 particles, order 3, u_th = 0.05 c) -- the
configuration BASELINE.json:north_star quotes its target on; it fits one GPU
(about 19 GB of arena).  N > 1: independent replicas of that workload, one per
GPU (replicas only, no data-path collective).

  value     particle-updates/s of the whole step, inputs resident in HBM
  e2e       the same metric through the C ABI with HOST buffers: every step
            pic_load_particles (H2D) + pic_sort + pic_step + pic_get_particles
            and pic_get_fields (D2H) from/to pinned host memory
  roofline  the dominant kernel (fused per-tile particle kernel).  It is bound by
            on-chip arithmetic and shared-memory issue, not by HBM,
            so the headline roofline is the fp64 pipe ("bound": "alu": algorithmic
            fp64 instructions per launch / average launch duration against
            148 SMs x 64 lanes x 1965 MHz); roofline_hbm (algorithmic bytes against
            the measured HBM peak) and roofline_smem stand beside it.  Launch
            durations come from CUDA events on the library's stream over the
            timed region
  cpu_baseline   the oracle (oracle/, as it stands) timed on the host cores on
            a bounded sample of the same workload

``--impl reference`` times the oracle alone (this tier's reference arm).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle-updates/sec (gather+push+deposit, fp64) and Yee cell-updates/sec on 1 B200"
UNIT = "particle-updates/s"

# Algorithmic HBM bytes of the fused particle kernel:
# per particle read x,y,z,ux,uy,uz,w (56 B) + write x,y,z,ux,uy,uz (48 B); per cell read the
# six E,B values (48 B) and read-modify-write the three J values (48 B).
BYTES_PER_PARTICLE = 104.0
BYTES_PER_CELL = 96.0
# Yee: B half (72 B/cell) + E (96 B/cell) + B half (72 B/cell)
YEE_BYTES_PER_CELL = 240.0
# fp64-pipe roofline of the fused kernel.  ALGORITHMIC fp64-pipe instructions per particle
# (an FMA counts once): order 3 = gather 6 x (64 + 16 + 4) = 504 FMA + nine shape-weight sets ~108
# + push and move ~130 + Esirkepov ~465 + ~20; orders 1 and 2 likewise.  What the committed kernel EXECUTES
# (ncu, thread level: DFMA + DADD + DMUL) is reported beside it, parsed from the committed ncu export of that order
# (profiles/r03_ncu_order<N>.raw.csv): 288 / 883 / 1,204 at orders 1 / 2 / 3 (profiles/r03_orders.md).
FP64_INSTR_PER_PARTICLE = {1: 380.0, 2: 710.0, 3: 1230.0}
FP64_LANES_PER_SM = 64
N_SM = 148
SM_MAX_MHZ = 1965.0


def _measured_counters(config_index, order):
    """ncu counters of ONE launch of the dominant kernel, parsed from the committed `ncu --page raw --csv` export of a
    `ncu --set full` capture (profiles/r03_ncu_order<N>.raw.csv; the command that made it is in profiles/r03_orders.md).
    Only configs[2] at full size has captures, one per shape order.  Nothing is copied by hand: the numbers are read
    from the export, whose name and sha256 go into the bench line.  None when there is no capture of this workload:
    the bench then reports traffic = null."""
    if config_index != 2:
        return None
    path = os.path.join(ROOT, "profiles", "r03_ncu_order%d.raw.csv" % order)
    try:
        import csv
        import hashlib
        with open(path, "rb") as fh:
            sha = hashlib.sha256(fh.read()).hexdigest()
        with open(path, newline="") as fh:
            rows = list(csv.reader(fh))
        d = dict(zip(rows[0], rows[2]))

        def num(k):
            return float(d[k].replace(",", ""))
        units = dict(zip(rows[0], rows[1]))
        scale = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}
        dram = sum(num(k) * scale[units[k]] for k in ("dram__bytes_read.sum", "dram__bytes_write.sum"))
        npart = 134217728.0
        cycles = num("sm__cycles_elapsed.max")
        fp64 = sum(num("smsp__sass_thread_inst_executed_op_%s_pred_on.sum.per_cycle_elapsed" % op)
                   for op in ("dfma", "dadd", "dmul")) * cycles / npart
        lsu = num("SM_A.TriageCompute.l1tex__data_pipe_lsu_wavefronts.avg") * N_SM / npart
        return {"source": "profiles/%s (ncu --set full, one launch, 256^3 x 8 ppc; profiles/r03_orders.md)" % os.path.basename(path),
                "sha256": sha, "kernel": d.get("Kernel Name"), "dram_bytes_per_launch": dram,
                "executed_fp64_instr_per_particle": round(fp64, 1), "lsu_wavefronts_per_particle": round(lsu, 2),
                "gpu_time_ms_under_ncu": num("gpu__time_duration.sum")}
    except Exception:
        return None


def _host_info():
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except Exception:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model}


def _pin_to_one_core(which=-1):
    """taskset-style pinning of this process to one core: the which-th of the cores it may run
    on; returns (core, previous affinity) or (None, None)."""
    try:
        cores = sorted(os.sched_getaffinity(0))
        core = cores[which % len(cores)]
        os.sched_setaffinity(0, {core})
        return core, set(cores)
    except Exception:
        return None, None


def _peaks():
    """(HBM GB/s, 'measured'|'fallback') from MEASURED_PEAKS.json, else the guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured"
    except Exception:
        return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=self.fh, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.fh.close()
        sm, mx, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        with open(self.path) as fh:
            for line in fh:
                p = [t.strip() for t in line.split(",")]
                if len(p) < 7:
                    continue
                try:
                    sm.append(float(p[0])); mx.append(float(p[1])); power.append(float(p[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, p[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
        os.unlink(self.path)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), power_w_max=max(power),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# --------------------------------------------------------------------------- oracle legs
def _oracle_sample(index: int, crop: bool = True):
    """The bounded sample of configs[index] the oracle is timed on (last column).  crop = False: the
    size the slow parity tests run (32^3 of config 1, the crops of configs 3 and 4)."""
    from paper_2303_12873_b200 import workloads as W
    # configs 1-2: a 16^3 crop (same ppc, u_th, order, dx, dt) keeps one oracle step under a second
    wl = W.config(index, parity=True, **({"n": 16} if (crop and index in (1, 2)) else {}))
    desc = "%s: %dx%dx%d cells, %d particles, order %d (%s of configs[%d], same ppc/u_th/order/dx/dt)" % (
        wl.name, wl.nx, wl.ny, wl.nz, wl.nparticles, wl.order, "crop" if crop else "parity size", index)
    return wl, desc


def _oracle_sim(wl):
    from oracle import ora
    o = ora.OracleSim(*wl.grid_args(), wl.dt, wl.order, len(wl.species))
    if wl.fields:
        o.set_fields(**wl.fields)
    for s, sp in enumerate(wl.species):
        o.load_particles(s, sp.q, sp.m, *sp.arrays())
    return o


def time_oracle(index: int, budget_s: float = 12.0, max_steps: int = 40, core_index: int = -1, crop: bool = True,
                min_steps: int = 2, warm: bool = True):
    """particle-updates/s of the oracle as it stands, single-threaded, pinned to one host core."""
    wl, desc = _oracle_sample(index, crop)
    o = _oracle_sim(wl)
    core, before = _pin_to_one_core(core_index)
    try:
        if warm:
            o.step(1)                               # warm-up (page in, build tables)
        t0 = time.perf_counter()
        n = 0
        while n < max_steps and (n < min_steps or time.perf_counter() - t0 < budget_s):
            o.step(1)
            n += 1
        dt = time.perf_counter() - t0
    finally:
        if before:
            os.sched_setaffinity(0, before)
    return {"value": wl.nparticles * n / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "pinned_to_core": core,
            "sample": "%s, %d steps in %.1f s" % (desc, n, dt),
            "cell_updates_per_s": wl.ncell * n / dt}


def time_oracle_all_cores(index: int, budget_s: float = 8.0):
    """Upper bound of a zero-communication CPU decomposition: one independent oracle replica per
    host core, run concurrently as separate processes, rates summed."""
    ncores = os.cpu_count() or 1
    cmd = [sys.executable, os.path.abspath(__file__), "--oracle-worker", "--config", str(index),
           "--oracle-budget", str(budget_s)]
    procs = [subprocess.Popen(cmd + ["--oracle-core", str(k)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
             for k in range(ncores)]          # replica k pinned to core k
    total, ok = 0.0, 0
    for pr in procs:
        try:
            out, _ = pr.communicate(timeout=20 * budget_s + 120)
            total += float(json.loads(out.strip().splitlines()[-1])["value"])
            ok += 1
        except Exception:
            pr.kill()
    return {"value": total, "unit": UNIT, "cores": ok,
            "how": "%d independent oracle replicas run concurrently (one process per host core), rates summed" % ok}


def run_reference(args):
    """--impl reference: the oracle on the host cores, K steps of a bounded sample after W warm-ups."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl, desc = _oracle_sample(args.config)
    o = _oracle_sim(wl)
    for _ in range(args.warmup):
        o.step(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(1)
    dt = time.perf_counter() - t0
    val = wl.nparticles * args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": "configs[%d]" % args.config, "sample": desc},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# --------------------------------------------------------------------------- GPU leg
def _pinned_copy(torch, a):
    t = torch.empty(a.shape, dtype=torch.float64, pin_memory=True)
    t.numpy()[...] = a
    return t


def run_ours(args):
    import numpy as np
    import torch
    from paper_2303_12873_b200 import workloads as W
    from paper_2303_12873_b200.binding import Sim      # raises if libpic_b200.so is missing: no fallback

    from paper_2303_12873_b200 import replicas as R
    rank, local, world = R.rank_env(os.environ)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # ---- workload: configs[index], one replica per rank (seed offset by rank) ----
    t_gen = time.perf_counter()
    kw = {}
    if args.n is not None:
        kw["n"] = args.n
    if args.ppc is not None:
        kw["ppc"] = args.ppc
    wl = W.config(args.config, parity=False, **kw)
    if args.order is not None:
        wl.order = args.order       # same geometry, particles and dt; only the shape order of every stage changes
    wl = R.make_replica(wl, rank)   # replicas differ only by a cyclic shift of the particle momenta
    sort_every = wl.sort_every if wl.sort_every > 0 else 0
    if args.sort_every is not None:
        sort_every = max(0, args.sort_every)
    t_gen = time.perf_counter() - t_gen
    npart, ncell = wl.nparticles, wl.ncell

    sim = Sim.from_workload(wl, device="cuda:%d" % local)
    options = {}
    for kv in args.option:
        name, _, val = kv.partition("=")
        options[name] = int(val)
        sim.set_option(name, int(val))
    sim.sort()
    sim.sync()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def run_steps(k, first_index):
        for it in range(k):
            if sort_every and (first_index + it) % sort_every == 0 and (first_index + it) > 0:
                sim.sort()
            sim.step(1)

    # ---- untimed set-up: the generator starts configs 0-2 from exactly ppc particles in every cell (reading R28);
    # the occupancy relaxes to Poisson within ~16 steps and the fused kernel slows by a fifth over them
    # (DESIGN.md section 6).  These steps are part of bringing the plasma to the state that is timed, so the
    # number does not depend on how many --warmup steps the caller asks for.
    relax = max(0, args.relax)
    run_steps(relax, 0)
    # ---- device-resident timing: W warm-ups, then exactly K steps ----
    run_steps(args.warmup, relax)
    sim.sync()
    sim.set_option("stage_timing", 1)
    c0 = sim.counters()
    clocks = ClockSampler(local)
    clocks.start()
    barrier()
    ev0 = torch.cuda.Event(enable_timing=True)
    ev1 = torch.cuda.Event(enable_timing=True)
    ev0.record(sim.stream)
    run_steps(args.steps, relax + args.warmup)
    ev1.record(sim.stream)
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    clk = clocks.stop()
    st = sim.stage_ms()
    sim.set_option("stage_timing", 0)
    c1 = sim.counters()
    ms_total = R.max_over_ranks(ms_total, dist, device="cuda")
    value = R.job_rate(npart, args.steps, ms_total * 1e-3, world)

    # ---- rooflines of the dominant kernel (fused particle kernel, one launch per species per step) ----
    nspec = sum(1 for s in wl.species if s.n > 0)
    n_launch = max(1, int(round(st["steps"])) * nspec)
    ms_launch = st["particles"] / n_launch
    np_launch = npart / nspec
    alg_bytes = BYTES_PER_PARTICLE * np_launch + BYTES_PER_CELL * ncell
    hbm_peak, peak_kind = _peaks()
    hbm_kind = "measured (MEASURED_PEAKS.json hbm_gbs)" if peak_kind == "measured" else "fallback (B200_PROFILING.md)"
    kname = "particles_tile_kernel<%d>" % wl.order
    # The kernel is bound by on-chip arithmetic/LSU issue, not by HBM: the headline
    # roofline is the fp64 pipe; the HBM and shared-memory figures are reported beside it.
    fp64_peak = FP64_LANES_PER_SM * N_SM * SM_MAX_MHZ * 1e6 / 1e12          # T fp64 instructions/s
    fp64_per_particle = FP64_INSTR_PER_PARTICLE.get(wl.order, FP64_INSTR_PER_PARTICLE[3])
    fp64_alg = fp64_per_particle * np_launch
    fp64_ach = fp64_alg / (ms_launch * 1e-3) / 1e12
    full_size = args.n is None and args.ppc is None
    mc = _measured_counters(args.config, wl.order) if full_size else None
    roofline = {"bound": "alu", "kernel": kname, "achieved": fp64_ach, "peak": fp64_peak,
                "peak_kind": "derived: 148 SMs x 64 fp64 lanes/clk x 1965 MHz (DESIGN.md 5.1; DFMA probe: 62.5 lanes/clk/SM)",
                "unit": "T fp64-instr/s", "frac": fp64_ach / fp64_peak,
                "traffic": mc.get("dram_bytes_per_launch") if mc else None,
                "traffic_source": mc.get("source") if mc else None,
                "traffic_sha256": mc.get("sha256") if mc else None,
                "ms_per_launch": ms_launch, "algorithmic_fp64_instr_per_particle": fp64_per_particle,
                "algorithmic_fp64_instr_per_launch": fp64_alg,
                "executed_fp64_instr_per_particle": mc.get("executed_fp64_instr_per_particle") if mc else None,
                "particle_updates_per_s_kernel_only": np_launch / (ms_launch * 1e-3)}
    hbm_ach = alg_bytes / (ms_launch * 1e-3) / 1e9
    roofline_hbm = {"bound": "hbm", "kernel": kname, "achieved": hbm_ach, "peak": hbm_peak, "peak_kind": hbm_kind,
                    "unit": "GB/s", "frac": hbm_ach / hbm_peak, "algorithmic_bytes_per_launch": alg_bytes}
    roofline_smem = None
    if mc and mc.get("lsu_wavefronts_per_particle"):
        # LSU data pipe: one wavefront per clock per SM; wavefronts per particle from the committed ncu capture
        wf_peak = N_SM * SM_MAX_MHZ * 1e6                                    # wavefronts/s
        wf_ach = mc["lsu_wavefronts_per_particle"] * np_launch / (ms_launch * 1e-3)
        roofline_smem = {"bound": "lsu", "kernel": kname, "achieved": wf_ach / 1e9, "peak": wf_peak / 1e9,
                         "peak_kind": "derived: 148 SMs x 1 wavefront/clk x 1965 MHz (profiles/r02_lsu.md)",
                         "unit": "G wavefronts/s", "frac": wf_ach / wf_peak,
                         "lsu_wavefronts_per_particle": mc["lsu_wavefronts_per_particle"]}
    nsteps_t = max(1.0, st["steps"])
    yee_ms = (st["yee_B"] + st["yee_E"]) / nsteps_t
    stages = {"per_step_ms": {k: st[k] / nsteps_t for k in ("zero_J", "particles", "fold_J", "yee_B", "yee_E")},
              "sort_ms_each": (st["sort"] / st["sorts"]) if st["sorts"] else None,
              "sorts_in_timed_region": int(st["sorts"]),
              "yee_cell_updates_per_s": ncell / (yee_ms * 1e-3) if yee_ms > 0 else None,
              "yee_gbs": YEE_BYTES_PER_CELL * ncell / (yee_ms * 1e-3) / 1e9 if yee_ms > 0 else None}
    roofline_yee = None
    if yee_ms > 0:
        yee_gbs = YEE_BYTES_PER_CELL * ncell / (yee_ms * 1e-3) / 1e9
        yee_kernels = {1: "push_B_tma_kernel x2 + push_E_tma_kernel (one tile per block)"}.get(
                           c1.get("yee_tma"), "push_B_kernel x2 + push_E_kernel (plain: the TMA tensor maps could not be built)")
        roofline_yee = {"bound": "hbm", "kernel": yee_kernels, "achieved": yee_gbs,
                        "peak": hbm_peak, "peak_kind": hbm_kind, "unit": "GB/s", "frac": yee_gbs / hbm_peak,
                        "algorithmic_bytes_per_step": YEE_BYTES_PER_CELL * ncell,
                        "cell_updates_per_s": ncell / (yee_ms * 1e-3)}
    paths = {k: c1[k] - c0[k] for k in ("fast", "slow", "global")}

    # ---- end to end through the C ABI with pinned HOST buffers (rank-local; max over ranks) ----
    e2e = None
    if args.e2e_steps > 0:
        host_in = [[_pinned_copy(torch, a) for a in sp.arrays()] for sp in wl.species]
        host_out = [{nm: torch.empty(sp.n, dtype=torch.float64, pin_memory=True)
                     for nm in ("x", "y", "z", "ux", "uy", "uz")} for sp in wl.species]
        fld_out = {nm: torch.empty(ncell, dtype=torch.float64, pin_memory=True) for nm in Sim.FIELD_NAMES}
        h2d = sum(7 * 8 * sp.n for sp in wl.species)
        d2h = sum(6 * 8 * sp.n for sp in wl.species) + 9 * 8 * ncell
        del sim
        torch.cuda.empty_cache()
        sim = Sim.from_workload(wl, device="cuda:%d" % local, load=False)
        for name, val in options.items():
            sim.set_option(name, val)
        if wl.fields:
            sim.set_fields(**wl.fields)

        def e2e_step():
            for s, sp in enumerate(wl.species):
                sim.load_particles(s, sp.q, sp.m, *host_in[s])
            sim.sort()
            sim.step(1)
            for s in range(len(wl.species)):
                sim.get_particles_into(s, host_out[s])
            sim.get_fields_into(fld_out)

        e2e_step()                                   # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            e2e_step()
        barrier()
        dt_e = time.perf_counter() - t0
        dt_e = R.max_over_ranks(dt_e, dist, device="cuda")
        e2e = {"value": R.job_rate(npart, args.e2e_steps, dt_e, world), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": args.e2e_steps, "ms_per_step": 1e3 * dt_e / args.e2e_steps,
               "what": "pic_load_particles(host) + pic_sort + pic_step(1) + pic_get_particles(host) + "
                       "pic_get_fields(host), pinned buffers, wall clock around synchronising calls"}

    # ---- the oracle beside it (rank 0, N = 1 only) ----
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = time_oracle(args.config)
        cpu["host"] = _host_info()
        if args.config != 0:       # config 0 at full size as well (262,144 particles, order 1)
            try:
                cpu["config0_full_size"] = time_oracle(0, budget_s=6.0, max_steps=10)
            except Exception as exc:
                cpu["config0_full_size"] = {"error": str(exc)}
        # ... and the sizes the slow parity tests step configs 1, 3 and 4 at: one cold step each (a 32^3 order-3 step
        # takes the oracle several seconds)
        cpu["parity_sizes"] = {}
        for k in (1, 3, 4):
            try:
                r = time_oracle(k, budget_s=0.0, max_steps=1, crop=False, min_steps=1, warm=False)
                cpu["parity_sizes"]["configs[%d]" % k] = {"value": r["value"], "unit": UNIT, "sample": r["sample"]}
            except Exception as exc:
                cpu["parity_sizes"]["configs[%d]" % k] = {"error": str(exc)}
        try:
            cpu["all_cores"] = time_oracle_all_cores(args.config)
        except Exception as exc:      # a reported baseline, never a reason to lose the bench line
            cpu["all_cores"] = {"error": str(exc)}

    if dist is not None:
        dist.destroy_process_group()
    if rank != 0:
        return 0
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[%d]" % args.config, "name": wl.name,
                       "grid": [wl.nx, wl.ny, wl.nz], "particles": npart, "species": len(wl.species),
                       "order": wl.order, "sort_every": sort_every, "replicas": world, "options": options,
                       **({"ppc_override": args.ppc} if args.ppc is not None else {}),
                       **({"order_override": args.order} if args.order is not None else {}),
                       "relaxation_steps": relax,
                       "l2": "inputs larger than L2 (%.1f GB of particles + fields per step)" % (
                           (BYTES_PER_PARTICLE * npart + 9 * 8 * ncell) / 1e9),
                       "generation_s": round(t_gen, 1)},
            "cell_updates_per_s": world * ncell * args.steps / (ms_total * 1e-3),
            "roofline": roofline, "roofline_hbm": roofline_hbm, "roofline_smem": roofline_smem,
            "roofline_yee": roofline_yee, "stages": stages, "particle_paths": paths,
            "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(c1["launches"] - c0["launches"]),
            "clocks": clk}
    print(json.dumps(line))
    return 0


def run_bricks(args):
    """--bricks PX,PY,PZ: the same workload cut into PX x PY x PZ bricks that all live on THIS GPU and exchange halos and
    particles through the C-ABI brick calls (NEXT-1).  It measures what the decomposition costs on
    one GPU (pack / unpack / migration kernels, the per-face synchronisations, smaller launches); it is NOT a scaling
    number.  Prints one JSON line of its own kind ("kind": "bricks_on_one_gpu")."""
    import torch
    from paper_2303_12873_b200 import bricks as B
    from paper_2303_12873_b200 import workloads as W
    from paper_2303_12873_b200.binding import Sim
    torch.cuda.set_device(0)
    procs = tuple(int(v) for v in args.bricks.split(","))
    kw = {"n": args.n} if args.n is not None else {}
    wl = W.config(args.config, parity=False, **kw)
    lay = B.BrickLayout(wl.nx, wl.ny, wl.nz, wl.dx, wl.dy, wl.dz, 0.0, 0.0, 0.0, procs)
    sims, _ = B.make_local_bricks(Sim, lay, wl, slack=1.15)
    st = B.BrickStepper(lay, sims, B.LocalTransport(range(lay.size)), len(wl.species), leaver_capacity=1 << 21)
    st.start()
    for s in sims.values():
        s.sort()
    for _ in range(args.warmup):
        st.step()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        st.step()
    ev1.record()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    ms = ev0.elapsed_time(ev1) / args.steps
    n_now = sum(s.get_particles(0)["x"].size for s in sims.values()) if lay.size <= 2 else None
    print(json.dumps({"kind": "bricks_on_one_gpu", "metric": METRIC, "value": wl.nparticles / (ms * 1e-3), "unit": UNIT,
                      "ms_per_step": ms, "wall_ms_per_step": 1e3 * wall / args.steps, "steps": args.steps,
                      "warmup": args.warmup, "n_gpus": 1, "scaling": "none: every brick runs on the same GPU",
                      "config": {"workload": "configs[%d]" % args.config, "grid": [wl.nx, wl.ny, wl.nz],
                                 "particles": wl.nparticles, "bricks": list(procs), "brick_cells": list(lay.nl),
                                 "sort": "every step, per brick"},
                      "particles_after": n_now}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=16)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs index (default 2: 256^3 x 8 ppc)")
    ap.add_argument("--n", "--cube", dest="n", type=int, default=None,
                    help="override the cube edge of configs 0-2 (debugging; under torchrun use --cube: --n is ambiguous there)")
    ap.add_argument("--ppc", type=int, default=None,
                    help="particles per cell of configs 0-2 (default: the 8 the configs name; experiments only)")
    ap.add_argument("--order", type=int, default=None, choices=(1, 2, 3),
                    help="run the chosen config's geometry and particles at another shape order (experiments)")
    ap.add_argument("--relax", type=int, default=16,
                    help="untimed set-up steps before the warm-up that relax the lattice start to Poisson occupancy")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--sort-every", type=int, default=None, help="override the workload's sort cadence (steps)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--option", action="append", default=[], metavar="NAME=VALUE",
                    help="pic_set_option(NAME, VALUE) before the run (experiments: force_path=1, gather_variant=1, ...)")
    ap.add_argument("--bricks", default=None, metavar="PX,PY,PZ",
                    help="cost of the brick decomposition on ONE GPU (NEXT-1): every brick a context on this GPU")
    ap.add_argument("--oracle-worker", action="store_true", help=argparse.SUPPRESS)
    ap.add_argument("--oracle-budget", type=float, default=8.0, help=argparse.SUPPRESS)
    ap.add_argument("--oracle-core", type=int, default=-1, help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.oracle_worker:      # one replica of the all-cores oracle baseline (no CUDA, no torch)
        print(json.dumps(time_oracle(args.config, budget_s=args.oracle_budget, core_index=args.oracle_core)))
        return 0
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    if args.bricks:
        return run_bricks(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
