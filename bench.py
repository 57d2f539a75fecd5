#!/usr/bin/env python
"""bench.py — throughput of the whole SPH hot path on B200.

Contract (driver): `python bench.py --gpus N --steps K --warmup W` prints ONE JSON line on rank 0.

  step      one sph_step(1): dt reduction, reinit, kick, drift, cell hash, radix sort, reorder,
            wall extrapolation x2, neighbour-list build, pair pass A, pair pass B (+ second kick)
            on one synthetic config (replayed as a CUDA graph of the same kernels)
  workload  BASELINE.json configs[4] at N_fluid = 16.8 M (cfg4_256: the size the target's ">= 50 % of the
            roofline at >= 16 M particles" is quoted at; the other sizes of the sweep and configs 0-3 via
            --config); inputs are seeded/synthetic (paper_2110_02621_b200.inputs)
  value     fluid particle-steps/s with the state resident in HBM (CUDA events on the launching
            stream; L2 flushed between timed steps; max over ranks)
  e2e       same metric through the HOST-pointer C-ABI calls: sph_set_particles_host + K x
            (sph_step(1) + sph_get_stats) + sph_get_fields_host, all inside the timed region
  roofline  the dominant kernel (largest stage time) against the FP32 ALU peak
  cpu_baseline  the CPU oracle (oracle/, as it stands) on the host cores, on a bounded sample of the same
            workload: for the cfg4 sweep its 1 M size (cfg4_100), else the config itself

N > 1: replicas only: every rank runs the same configuration independently, no
data-path collective; value = particle-steps of all ranks / max-over-ranks time; scaling "weak".

`--impl reference` times the CPU oracle instead (rank 0 only) and prints the same line shape.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "particle-steps/s"
UNIT = "fluid particle-steps/s"

# Algorithmic FP32 operation counts per neighbour hit (fma = 2), DESIGN.md §7.  They are the
# paper's equations counted once, independent of the cell scheme; candidate tests are reported
# separately (CAND_FLOPS each) because they are overhead of the 27-cell walk, not of the method.
FLOPS_HIT = {"pass_a": 40.0, "pass_b": 50.0, "wall": 30.0}
CAND_FLOPS = 8.0
# ncu counters of the dominant kernels (dram bytes per launch, L1 data-pipe wavefronts and issue-active as
# fractions of peak) are looked up in a committed table of `ncu --set full` captures, profiles/ncu_kernels.csv,
# keyed by workload, kernel AND the hash of the kernel sources they were captured from (csrc_hash() below):
# a capture of other sources is stale and yields null, never a number.
NCU_TABLE = os.path.join(ROOT, "profiles", "ncu_kernels.csv")


def csrc_hash():
    """sha256 (first 16 hex digits) over include/sph.h and paper_2110_02621_b200/csrc/*, sorted by name."""
    import glob
    import hashlib
    h = hashlib.sha256()
    files = [os.path.join(ROOT, "include", "sph.h")] + sorted(glob.glob(os.path.join(ROOT, "paper_2110_02621_b200", "csrc", "*")))
    for f in files:
        h.update(os.path.basename(f).encode())
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_lookup(workload, kernel):
    """Row of profiles/ncu_kernels.csv for (workload, kernel, csrc_hash()) or None."""
    import csv
    try:
        with open(NCU_TABLE) as fh:
            rows = [r for r in csv.DictReader(l for l in fh if not l.startswith("#"))]
    except OSError:
        return None
    hsh = csrc_hash()
    for r in rows:
        if r["workload"] == workload and r["kernel"] == kernel and r["csrc_hash"] == hsh:
            return r
    return None


FP32_LANES_PER_SM = 128
N_SM = 148


def make_config_name(name):
    return {"cfg0": "cfg0_dam_break_2d", "cfg1": "cfg1_dam_break_3d_box", "cfg1_small": "cfg1_dam_break_3d_box",
            "cfg2a": "cfg2a_two_phase_2d", "cfg2b": "cfg2b_two_phase_2d", "cfg3": "cfg3_sloshing_spheres_3d",
            "cfg3_4m": "cfg3_sloshing_spheres_3d"}.get(name, name)


def make_config(name):
    from paper_2110_02621_b200 import inputs
    if name == "cfg0":
        return inputs.dam_break_2d()
    if name == "cfg1":
        return inputs.dam_break_3d_box()
    if name == "cfg1_small":
        return inputs.dam_break_3d_box(dp=0.02)
    if name == "cfg2a":
        return inputs.two_phase_2d(equal_c=True)
    if name == "cfg2b":
        return inputs.two_phase_2d(equal_c=False)
    if name == "cfg3":
        return inputs.sloshing_spheres_3d()
    if name == "cfg3_4m":
        return inputs.sloshing_spheres_3d(dp=0.00585)
    if name == "cfg3_small":
        return inputs.sloshing_spheres_3d(dp=0.0125)
    if name.startswith("cfg4_"):
        return inputs.box_sweep_3d(n=int(name.split("_")[1]))
    if name.startswith("x1_"):   # NEXT-2: the paper's two-phase hydrostatic tank, e.g. x1_0.005
        return inputs.hydrostatic_tank_x1(dp=float(name.split("_")[1]))
    raise SystemExit("unknown --config %r" % name)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs
    (the recipe's clocks line, /opt/skills/guides/B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, gpu_index):
        self.rows = []
        self.proc = None
        self.idx = gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, pw, reasons = [], [], [], set()
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for k, name in enumerate(self.NAMES):
                if f[4 + k].lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(smax)),
                    power_w_max=float(max(pw)), reasons=sorted(reasons), samples=len(sm))


def stencil_candidates(cfg, g):
    """Number of (fluid i, candidate j) distance tests the 27/9-cell walk performs at the current
    positions, from the library's own cell ranges (host-side integer bookkeeping for the report:
    sum over cells of n_f(c) * sum_{c' in stencil(c)} (n_f(c') + n_w(c')))."""
    _, _, cs, ce = g.debug_cells()
    nc = g.num_cells()
    cnt = (ce - cs).astype(np.int64)
    nf, nw = cnt[:nc], cnt[nc:]
    edge = 2.0 * cfg["h"] * (1.0 + 1.0 / 1024.0)
    dims = [max(1, int(np.ceil((cfg["domain_max"][k] - cfg["domain_min"][k]) / edge)))
            for k in range(cfg["dim"])]
    while len(dims) < 3:
        dims.append(1)
    nx, ny, nz = dims
    assert nx * ny * nz == nc, (dims, nc)
    tot = (nf + nw).reshape(nz, ny, nx)
    wallc = nw.reshape(nz, ny, nx)

    def box(a):
        for ax in range(3):
            if a.shape[ax] == 1:
                continue
            p = np.zeros_like(a)
            sl = [slice(None)] * 3
            p += a
            s1, s2 = list(sl), list(sl)
            s1[ax] = slice(1, None); s2[ax] = slice(None, -1)
            p[tuple(s1)] += a[tuple(s2)]
            p[tuple(s2)] += a[tuple(s1)]
            a = p
        return a

    f3 = nf.reshape(nz, ny, nx)
    cand_fluid_rows = int((f3 * box(tot)).sum())          # tests issued by the fluid pair passes
    cand_wall_rows = int((wallc * box(f3)).sum())         # tests issued by the wall extrapolation
    return cand_fluid_rows, cand_wall_rows


def oracle_rate(cfg, steps, warmup=0):
    """Time `steps` oracle steps (after `warmup`) on the host cores; returns
    (fluid particle-steps/s, seconds, threads)."""
    from oracle import orc
    o = orc.Oracle(cfg)
    o.set_particles(cfg["pos"], cfg["vel"], cfg["rho"], cfg["tag"])
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    return cfg["n_fluid"] * steps / dt, dt, os.cpu_count() or 1


def cpu_sample_config(name):
    """Bounded sample of workload `name` for the oracle legs (about 10-30 s of CPU work for 10-25 steps):
    the cfg4 sweep is sampled at its 1 M size (same recipe), cfg3 at dp = 0.0125,
    cfg1 at full size when few steps are asked for, everything else as is."""
    if name.startswith("cfg4_") and int(name.split("_")[1]) > 100:
        return "cfg4_100", "cfg4 sweep at its N_fluid = 1 M size"
    if name in ("cfg3", "cfg3_4m"):
        return "cfg3_small", "cfg3 geometry at dp = 0.0125"
    return name, "full size"


def run_reference(args):
    """--impl reference: the CPU oracle as it stands (this tier's reference arm), rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    name, what = cpu_sample_config(args.config)
    if name == "cfg1" and (args.steps + args.warmup) > 30:
        name, what = "cfg1_small", "cfg1 at dp = 0.02"
    cfg = make_config(name)
    rate, secs, cores = oracle_rate(cfg, args.steps, args.warmup)
    sample = "%s: %s (%d fluid + %d wall particles), %d steps after %d warm-up" % (
        what, cfg["name"], cfg["n_fluid"], cfg["n_wall"], args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": make_config_name(args.config), "sample": sample},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2110_02621_b200 import sph

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libsph has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = make_config(args.config)
    if args.wall_osc:
        # NEXT-1: rigid wall motion x_w(t) = x_w(0) + A0 sin(2 pi f0 t) along x;
        # not the headline workload: the line's config.workload says so.
        a0, f0 = (float(x) for x in args.wall_osc.split(","))
        cfg["wall_osc_amp"], cfg["wall_osc_freq"] = (a0, 0.0, 0.0), f0
    if args.no_graph:
        cfg["flags"] = cfg["flags"] | sph.FLAG_NO_GRAPH
    nfl, nwl = cfg["n_fluid"], cfg["n_wall"]
    K, W = args.steps, max(args.warmup, 0)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    # ---- device-resident run ------------------------------------------------------------------
    dev = {k: torch.from_numpy(cfg[k]).cuda() for k in ("pos", "vel", "rho", "tag")}
    g = sph.Sph(cfg)
    g.set_particles(dev["pos"], dev["vel"], dev["rho"], dev["tag"])
    for _ in range(W):
        flush.zero_()
        g.step(1)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    r0 = g.get_stats(with_pairs=False)["rebuilds"]
    l0 = g.launch_count()
    for k in range(K):
        flush.zero_()              # L2 flush between timed iterations (outside the event pair)
        ev[k][0].record()
        g.step(1)
        ev[k][1].record()
    barrier()
    clocks = sampler.stop()
    ms = float(sum(a.elapsed_time(b) for a, b in ev))
    ms = max_over_ranks(ms, "cuda")
    st = g.get_stats()
    st_timed = st
    launches = g.launch_count() - l0        # after the stats read: it adds the rebuild branches the graph replays took
    rebuilds = st["rebuilds"] - r0          # steps of the timed region that rebuilt the cell list and the neighbour lists
    if st["escaped"] or st["nonfinite"]:
        raise SystemExit("bench run went bad: %r" % (st,))
    value = whole_job_rate(nfl * K, world, ms * 1e-3)
    pairs_s = world * st["npairs"] * K / (ms * 1e-3)

    # ---- per-stage times (CUDA events recorded by the library on the same stream) ---------------
    # (a) the default step as timed above (lists kept over several steps): averages per step;
    # (b) "each kernel timed separately" (BASELINE.json config 4): a context with list_skin = 0, in which
    #     every step runs every kernel (sort, reorder, both list builds) once: per-launch times for the roofline.
    g.set_profiling(True)
    KP = min(K, 32)
    for _ in range(KP):
        flush.zero_()
        g.step(1)
    stage_def, ns = g.get_timings()
    g.set_profiling(False)
    stage_def = {k: v / max(ns, 1) for k, v in stage_def.items()}
    stage_def["rebuilds_per_step"] = g.last_timing_rebuilds / max(ns, 1)
    st = g.get_stats()
    # measured roofline of the gather form: the passes' list walk with an empty pair body, on the lists of this state
    gather = g.gather_floor()
    gather32 = g.gather_floor(body_fma=32)   # the same walks under a synthetic pair body of 32 FFMAs (about 70 instructions per pair in all)
    skin = sph.DEFAULT_LIST_SKIN if cfg.get("list_skin", -1.0) < 0 else cfg["list_skin"]
    if skin > 0:
        g.close()
        g = sph.Sph(dict(cfg, list_skin=0.0))
        g.set_particles(dev["pos"], dev["vel"], dev["rho"], dev["tag"])
        for _ in range(max(W, 1)):
            g.step(1)
    g.set_profiling(True)
    for _ in range(KP):
        flush.zero_()
        g.step(1)
    stage_ms, ns = g.get_timings()
    g.set_profiling(False)
    stage_ms = {k: v / max(ns, 1) for k, v in stage_ms.items()}
    pointwise = g.time_pointwise()
    cand_f, cand_w = stencil_candidates(cfg, g)
    off, _ = _neighbour_counts(g)
    tag = cfg["tag"]
    wall_pairs = int((off[1:] - off[:-1])[tag < 0].sum())
    fluid_pairs = int(st["npairs"])
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak_derived = N_SM * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12       # TFLOP/s at max SM clock
    # measured non-tensor FP32 peak (SURVEY.md section 8(d) "Peaks"): register-resident FMA loop, this device, now
    fma_sampler = ClockSampler(local)
    fma_sampler.start()
    if args.derived_peak:
        peak = peak_derived
    else:
        peak = sph.fma_peak_tflops()
        for _ in range(20):             # keep the loop running long enough for nvidia-smi to sample its clocks
            peak = max(peak, sph.fma_peak_tflops())
    fma_clocks = fma_sampler.stop()
    l1_patterns = sph.gather_pattern_cycles()
    kern = {}
    # Pair stages.  The 27-cell candidate walk runs once per step in k_build (fluid-fluid) and inside
    # k_wall / the wall part of the passes (fluid-wall); the fluid pair passes read the neighbour lists.
    # hits: flops of the paper's equations; candidates: CAND_FLOPS each, charged to the stage that tests them.
    # pass A, pass B and the two wall passes: as they run in the default (timed) step; the list builds (fluid rows
    # + wall rows, one "build" stage), sort and reorder: per launch, from the list_skin = 0 context.
    cand_b = (cand_f + cand_w) * (1.0 + skin) ** cfg["dim"]     # the builds walk cells of edge 2h(1 + skin)
    for name, src, hits, cands, per_step in (("pass_a", stage_def, fluid_pairs, 0, 1), ("pass_b", stage_def, fluid_pairs, 0, 1),
                                             ("build", stage_ms, 0, cand_f + cand_w, 1), ("wall", stage_def, wall_pairs, 0, 2)):
        t = src.get(name, 0.0) * 1e-3 / per_step
        if t <= 0:
            continue
        fl = FLOPS_HIT.get(name, 0.0) * hits
        kern[name] = {"ms": 1e3 * t, "hits": hits, "candidates": cands,
                      "tflops_hit_only": fl / t / 1e12, "frac_hit_only": fl / t / 1e12 / peak,
                      "tflops_with_candidates": (fl + CAND_FLOPS * cands) / t / 1e12,
                      "frac_with_candidates": (fl + CAND_FLOPS * cands) / t / 1e12 / peak}
    # list builds + pass A + pass B together, per step of the default configuration (builds amortised over the
    # steps that keep their lists)
    t_pair = (stage_def["pass_a"] + stage_def["pass_b"] + stage_def.get("build", 0.0)) * 1e-3
    fl_pair = (FLOPS_HIT["pass_a"] + FLOPS_HIT["pass_b"]) * fluid_pairs
    pair_stages = {"ms": 1e3 * t_pair, "frac_hit_only": fl_pair / t_pair / 1e12 / peak,
                   "frac_with_candidates": (fl_pair + CAND_FLOPS * cand_b * stage_def["rebuilds_per_step"]) / t_pair / 1e12 / peak}
    # HBM-bound stages: algorithmic bytes per fluid particle
    hbm = _peaks().get("hbm_gbs", 6650.0)
    bytes_pp = {"predict": 140.0, "sort": (16.0 + 4.0) * g_sort_passes(g), "reorder": 100.0}
    for name, b in bytes_pp.items():
        t = stage_ms[name] * 1e-3
        if t > 0:
            kern[name] = {"ms": 1e3 * t, "gbs": b * nfl / t / 1e9, "frac_hbm": b * nfl / t / 1e9 / hbm}
    dom = max(("pass_a", "pass_b"), key=lambda k: stage_def[k])   # the list build is reported under "kernels"
    ncu = ncu_lookup(cfg["name"], "k_" + dom)
    roofline = {"bound": "alu", "kernel": "k_" + dom, "achieved": kern[dom]["tflops_hit_only"],
                "peak": peak, "unit": "TFLOP/s", "frac": kern[dom]["frac_hit_only"],
                "traffic": float(ncu["dram_bytes"]) if ncu else None,
                "l1_data_pipe_frac_ncu": float(ncu["l1_data_pipe_frac"]) if ncu else None,
                "issue_active_frac_ncu": float(ncu["issue_active_frac"]) if ncu else None,
                "ncu_capture": (ncu["capture"] if ncu else None), "csrc_hash": csrc_hash(),
                "peak_source": ("derived from unit counts (--derived-peak: profiler capture, not a bench line)" if args.derived_peak else
                                "measured: sph_debug_fma_peak (register-resident FMA loop, 8 chains x 2048 threads per SM) on this device in this run"),
                "peak_derived": peak_derived, "peak_clocks": {"sm_mhz": fma_clocks.get("sm_mhz"), "sm_max_mhz": fma_clocks.get("sm_max_mhz")},
                "flops_per_hit": FLOPS_HIT[dom], "flops_per_candidate": CAND_FLOPS,
                # sph_debug_gather_floor: what the memory requests of a pass alone take (same lists, same records, same
                # launch configuration, empty pair body), and what merged lists / coalesced records / an SM-affine
                # block order would make of them; sph_debug_gather_patterns: the L1's cost per request by address pattern
                "gather_floor": {"own_entries_ms": gather["own_entries"], "lane_pair_shared_ms": gather["lane_pair_shared"],
                                 "quad_shared_ms": gather["quad_shared"], "coalesced_ms": gather["coalesced"],
                                 "own_entries_sm_affine_ms": gather["own_entries_sm_affine"], "requests": gather["requests"],
                                 "cycles_per_request": gather["own_entries"] * 1e-3 * sm_max * 1e6 * N_SM / max(gather["requests"], 1),
                                 "pass_a_over_floor": stage_def["pass_a"] / gather["own_entries"] if gather["own_entries"] > 0 else None,
                                 "pass_b_over_floor": stage_def["pass_b"] / gather["own_entries"] if gather["own_entries"] > 0 else None,
                                 "with_synthetic_body_of_32_fma_per_pair_ms": {k: gather32[k] for k in ("own_entries", "lane_pair_shared", "quad_shared", "coalesced", "own_entries_sm_affine")},
                                 "l1_cycles_per_request_by_pattern": l1_patterns},
                # list build + pass A + pass B together (the candidate walk is k_build's):
                "pair_stages": pair_stages}
    g.close()

    # ---- end to end through the HOST-pointer entry points ----------------------------------------
    n = len(cfg["tag"])
    pin = {k: torch.from_numpy(cfg[k]).pin_memory() for k in ("pos", "vel", "rho", "tag")}
    out = {k: torch.empty(s, dtype=torch.float32).pin_memory() for k, s in
           (("pos", (n, 3)), ("vel", (n, 3)), ("rho", (n,)))}
    g2 = sph.Sph(cfg)
    KE = K
    g2.set_particles(pin["pos"].numpy(), pin["vel"].numpy(), pin["rho"].numpy(), pin["tag"].numpy())
    g2.step(1)  # warm the allocator / module load outside the timed region
    # host-side wall clock: the region is repeated and the median repetition kept (the box's host
    # cores are shared; every repetition does the full region: upload + set-up, KE steps, read-back)
    reps = []
    for _rep in range(3):
        barrier()
        t0 = time.perf_counter()
        g2.set_particles(pin["pos"].numpy(), pin["vel"].numpy(), pin["rho"].numpy(), pin["tag"].numpy())
        for _ in range(KE):
            g2.step(1)
            s2 = g2.get_stats(with_pairs=False)   # device -> host read of the step's result (t, dt, E_k, mass, x_front)
        g2.get_fields_into_host(pos=out["pos"].numpy(), vel=out["vel"].numpy(), rho=out["rho"].numpy())
        torch.cuda.synchronize()
        reps.append(time.perf_counter() - t0)
    e2e_s = sorted(reps)[1]
    e2e_s = max_over_ranks(e2e_s, "cuda")
    h2d = (n * (12 + 12 + 4 + 4)) / KE
    d2h = (n * 4 + n * (12 + 12 + 4)) / KE + 88      # tag read-back + fields, + sph_stats per step
    e2e = {"value": world * nfl * KE / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d,
           "d2h_bytes_per_step": d2h,
           "region": "sph_set_particles_host + %d x (sph_step(1) + sph_get_stats_ex(no pair count)) + sph_get_fields_host; median of 3 repetitions" % KE}
    g2.close()

    # ---- CPU oracle on the host cores (rank 0, N = 1 only) -----------------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        osteps = args.cpu_steps
        cname, what = cpu_sample_config(args.config)
        ccfg = cfg if cname == args.config else make_config(cname)
        rate, secs, cores = oracle_rate(ccfg, osteps)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "%s: %s (%d fluid + %d wall), %d steps, %.1f s" % (what, ccfg["name"], ccfg["n_fluid"], ccfg["n_wall"], osteps, secs)}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg["name"] + ("+wall_osc(%s)" % args.wall_osc if args.wall_osc else ""),
                       "n_fluid": nfl, "n_wall": nwl, "dim": cfg["dim"],
                       "dp": cfg["dp"], "l2": "flushed between timed steps (256 MiB write)",
                       "list_skin": skin,
                       "parallelism": "replicas only" if world > 1 else "1 gpu"},
            "pair_interactions_per_s": pairs_s, "pairs_per_step": fluid_pairs,
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
            "list_skin_max": skin, "list_skin_at_end": st_timed["list_skin"], "rebuilds_in_timed_steps": int(rebuilds),
            "roofline": roofline, "kernels": kern, "stage_ms_per_step": stage_def,
            "stage_ms_per_launch_skin0": stage_ms, "pointwise_standalone_ms": pointwise,
            "cpu_baseline": cpu,
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def max_over_ranks(value, device=None):
    """Replicas-only multi-GPU timing rule: every rank times its own replica, the job time is the
    max over ranks (torch.distributed all_reduce MAX; backend nccl on GPUs, gloo in the CPU test)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank, world, seconds):
    """value of the JSON line: units processed by all replicas / max-over-ranks time."""
    return world * units_per_rank / seconds


def _neighbour_counts(g):
    import ctypes as C
    off = np.zeros(g.n + 1, np.int64)
    tot = C.c_int64(0)
    g._ck(g.L.sph_debug_neighbours(g.ctx, off.ctypes.data_as(C.c_void_p), None, 0, C.byref(tot), g._st()))
    return off, tot.value


def g_sort_passes(g):
    bits = 1
    while (1 << bits) < g.num_cells():
        bits += 1
    p8, p9 = (bits + 7) // 8, (bits + 8) // 9   # 9-bit digits when that saves a pass (sph_sort.cuh)
    return min(p8, p9)


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg4_256",
                    help="cfg0 cfg1 cfg2a cfg2b cfg3 cfg3_4m cfg4_<n> (n^3 fluid particles) x1_<dp>; default cfg4_256 (16.8 M)")
    ap.add_argument("--cpu-steps", type=int, default=20,
                    help="oracle steps of the cpu_baseline leg (1 M particles: about 0.6 s per step on 16 cores)")
    ap.add_argument("--csrc-hash", action="store_true", help="print the hash profiles/ncu_kernels.csv is keyed by and exit")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--derived-peak", action="store_true",
                    help="skip the FMA-loop peak measurement (126 launches) and use the derived peak: for profiler launch lists only")
    ap.add_argument("--no-graph", action="store_true",
                    help="SPH_FLAG_NO_GRAPH: plain launches instead of the step graph (same kernels; for profiler captures)")
    ap.add_argument("--wall-osc", default="", metavar="A0,F0",
                    help="move the walls along x as A0 sin(2 pi F0 t) (metres, Hz); implies a non-headline line")
    args = ap.parse_args()
    if args.csrc_hash:
        print(csrc_hash())
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
