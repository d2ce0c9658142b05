#!/usr/bin/env python
"""bench.py — electron-collisions/s (real + null) of the avalanche hot path on B200, with its roofline.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload all|config1|config2|config3s|config3|config4|config4x16|config5|...]
  python bench.py --impl reference ...     # the oracle on the host cores

A "step" is one pass of the whole hot path (avm_run: primary injection, persistent transport kernel with secondary
append and lane refill, tallies) over one batch of primaries of a workload.  The default run (`--workload all`) times
ALL FIVE BASELINE.json configs: the headline (`value`, `config.workload`, `roofline`, `e2e`, `cpu_baseline`) is config 3
with its time cut — the largest one by collisions per step that fits the bench budget — timed for
exactly K steps after W warm-ups; the other four are in `per_config`, each with its own steps / warm-ups stated there.
Prints ONE JSON line.  Nothing here reads /root/reference.
"""
from __future__ import annotations

import argparse
import glob
import hashlib
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "electron-collisions/s (real+null)"
UNIT = "collisions/s"
HEADLINE = "config3s"
# workload -> (multiplier of --steps, oracle sample = first n primaries; 0 = all).  Oracle samples follow SURVEY.md §8(d)
# "Oracle timing" (config 3: first primaries only, config 5: first 8), sized for ~1-10 s each on the box's cores.
ALL = {"config1": (4, 0), "config2": (2, 0), "config3s": (1, 2048), "config4": (1, 0), "config5": (0.5, 8),
       "config5hg": (0.2, -1),      # not a BASELINE config (D4): config 5's stack at dV = 500 V, 1e4-1e5 electrons per avalanche;
                                    # -1: no oracle leg (one such avalanche is ~4e9 collisions on one core)
       # HEAVY entries (multiplier 0): ONE timed run each, un-banded and banded, no warm-up of their own (the kernels are warm
       # from the entries before them and one run lasts seconds), no e2e leg — stated in the entry's `timing`.
       "config3": (0, 8),           # BASELINE config 3 AS STATED: 1 cm gap, no time cut, ~1.3e12 steps (~28 s; ~13 s banded)
       "config4x16": (0, -1),       # replicated variants that show the map path's throughput asymptote
       "config4x64": (0, -1)}
HEAVY = {k for k, (m, _) in ALL.items() if m == 0}
# Algorithmic FP64 thread-instructions per unit: what the method must do — NOT what
# the kernel executes (the executed count and the FP64 pipe's busy share come from the ncu capture, when it is current).
FP64_PER_NULL = {False: 90.0, True: 170.0}       # free flight + energy + bin + decision; key = B != 0
FP64_PER_REAL_EXTRA = 110.0                      # deflection angles, basis, rotation, renormalise, speed
FP64_PER_ION_EXTRA = 80.0                        # Opal-Beaty atan/tan, child direction
FP64_PER_GRID_EXTRA = 45.0                       # fold + 7 lerps x 4 channels per step in a grid slab
GATHER_BYTES_PER_GRID_STEP = 128.0               # 8 nodes x 16 B of the fp32 map; the widened copy moves 256
FP64_LANES_PER_SM = 64                           # one warp-wide FP64 instruction / 2 clk / scheduler
NCU_CAPTURE_FILE = os.path.join(ROOT, "profiles", "ncu_capture.json.txt")


def kernel_source_hash() -> str:
    """sha256 over the kernel sources: an ncu capture describes the kernels only while this is unchanged."""
    h = hashlib.sha256()
    for p in sorted(glob.glob(os.path.join(ROOT, "paper_2509_15377_b200", "csrc", "*"))):
        if p.endswith((".cu", ".cuh", ".inc")):
            h.update(os.path.basename(p).encode())
            h.update(open(p, "rb").read())
    return h.hexdigest()[:16]


def ncu_capture(workload: str) -> dict:
    """Figures of the committed `ncu --set full` capture of the transport kernel on this workload (profiles/), or nulls
    when there is none or the kernels have changed since (never a stale number)."""
    out = {"traffic": None, "sass_fp64_per_collision_ncu": None, "fp64_pipe_active_pct_ncu": None, "ncu_source": None}
    try:
        d = json.load(open(NCU_CAPTURE_FILE))
    except Exception:
        return out
    e = d.get("workloads", {}).get(workload)
    if e is None:
        return out
    if d.get("kernel_source_hash") != kernel_source_hash():
        out["ncu_source"] = f"{e.get('profile')}: stale (kernels changed since the capture), figures withheld"
        return out
    out.update(traffic=e.get("dram_bytes_per_launch"), sass_fp64_per_collision_ncu=e.get("sass_fp64_per_collision"),
               fp64_pipe_active_pct_ncu=e.get("fp64_pipe_active_pct"),
               ncu_source=f"{e.get('profile')} (ncu --set full, one launch; dram__bytes_read.sum + dram__bytes_write.sum)")
    return out


def make_workload(name: str, rank: int = 0):
    from paper_2509_15377_b200.gen import configs
    if name == "config1":
        w = configs.config1(id_offset=rank * 1000)
    elif name == "config2":
        w = configs.config2(id_offset=rank * 100)
    elif name.startswith("config2x"):
        w = configs.replicate(configs.config2(), int(name[len("config2x"):]))
    elif name == "config3s":                      # config 3 with a time cut (the full run is ~1e12 steps)
        w = configs.config3(n_primaries=100000, t_max=20.0, id_offset=rank * 100000)
        w.name = "config3s"
        w.note += "; time cut t_max=20 ns"
    elif name == "config3":                       # as BASELINE states it: no time cut
        w = configs.config3(n_primaries=100000, id_offset=rank * 100000)
    elif name == "config4":
        w = configs.config4(id_offset=rank * 1000)
    elif name.startswith("config4x"):
        w = configs.replicate(configs.config4(), int(name[len("config4x"):]))
    elif name == "config5":
        w = configs.config5(id_offset=rank * 200)
    elif name == "config5hg":
        w = configs.config5hg(id_offset=rank * 8)
    else:
        raise SystemExit(f"unknown workload {name}")
    return w


def config_dict(w, world: int) -> dict:
    """What defines the workload — identical in both arms (`--impl ours` / `--impl reference`)."""
    return {"workload": w.name, "note": w.note, "n_primaries_per_gpu": w.n_primaries, "seed": "workload seed + step index",
            "t_max_ns": None if not np.isfinite(w.t_max) else w.t_max,
            "l2": "GPU arm: 256 MiB buffer written between timed iterations",
            "parallelism": f"replicas over primaries x{world}, no collective"}


def grid_fraction(field) -> float:
    """Share of the steps taken inside grid slabs.  Not tallied by the path; estimated as the grid slabs' share of the
    drift length (exact for one slab: configs 1-4; DESIGN.md §6 for config 5)."""
    tot = sum(s.z_hi - s.z_lo for s in field.slabs)
    return sum(s.z_hi - s.z_lo for s in field.slabs if s.kind == 1) / tot


def alg_fp64(tallies_u64: np.ndarray, L: int, level_type: np.ndarray, has_b: bool, grid_frac: float = 0.0) -> float:
    n_null, n_real = float(tallies_u64[L]), float(tallies_u64[L + 1])
    n_ion = float(sum(int(tallies_u64[l]) for l in range(L) if level_type[l] == 2))
    return ((n_null + n_real) * (FP64_PER_NULL[has_b] + grid_frac * FP64_PER_GRID_EXTRA) + n_real * FP64_PER_REAL_EXTRA
            + n_ion * FP64_PER_ION_EXTRA)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if not self.proc:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        try:
            for line in open(self.path):
                c = [x.strip() for x in line.split(",")]
                if len(c) < 9:
                    continue
                try:
                    sm.append(float(c[1])); mx.append(float(c[2]))
                except ValueError:
                    continue
                for nm, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm),
                       sm_mhz_peak_seen=float(max(sm)))
        out["reasons"] = sorted(reasons)
        return out


def measured_peaks(avm, ctx) -> dict:
    """The roofline denominators, measured on this GPU in this run: FP64 thread-instructions per second (the
    library's DFMA probe; nominal = SMs x 64 FP64 lanes x max SM clock), random 32-byte-sector gather bandwidth with the
    working set in L2 (2.7 MB = the gas table, 64 MB) and in HBM (1 GiB), shared-memory random 8-byte loads per second."""
    sm_max_mhz, hbm = 1965.0, None
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            mp = json.load(f)
            sm_max_mhz = float(mp.get("sm_max_mhz", sm_max_mhz)); hbm = mp.get("hbm_gbs")
    except Exception:
        pass
    nominal = ctx.sm_count * FP64_LANES_PER_SM * sm_max_mhz * 1e6
    best = max(avm.fp64_probe(ctx, iters=1 << 15)["dfma_per_s"] for _ in range(3))
    g = {}
    for label, nbytes, iters in (("l2_2p7MB", 2_700_000 // 32 * 32, 4096), ("l2_64MB", 64 << 20, 4096), ("hbm_1GiB", 1 << 30, 1024)):
        g[label] = max(avm.gather_probe(ctx, nbytes, iters=iters)["GBps"] for _ in range(2))
    sm = max(avm.smem_probe(ctx)["loads_per_s"] for _ in range(2))
    return {"fp64_nominal": nominal, "fp64_measured": best, "sm_max_mhz": sm_max_mhz, "gather_GBps": g,
            "smem_random_8B_loads_per_s": sm, "hbm_copy_GBps_MEASURED_PEAKS": hbm}


def oracle_leg(w, n_prim: int, threads: int) -> dict:
    """The oracle, as it stands, on the first n_prim primaries of the workload (identical Philox streams)."""
    from oracle import avmo
    avmo.build()
    t0 = time.perf_counter()
    r = avmo.run(w.gas, w.field, w.primaries[:n_prim], seed=w.seed, t_max=w.t_max, capacity=w.capacity, n_threads=threads)
    dt = time.perf_counter() - t0
    L = w.gas.n_levels
    coll = int(r.tallies_u64[L]) + int(r.tallies_u64[L + 1])
    return {"seconds": dt, "collisions": coll, "null": int(r.tallies_u64[L]), "real": int(r.tallies_u64[L + 1]),
            "electrons": int(r.n), "primaries": int(n_prim)}


def cpu_baseline_entry(w, sample: int, cores: int, one_core: bool = False) -> dict:
    n_prim = min(w.n_primaries, sample) if sample > 0 else w.n_primaries
    o = oracle_leg(w, n_prim, cores)
    out = {"value": o["collisions"] / o["seconds"], "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"first {n_prim} of {w.n_primaries} primaries of {w.name}, seed {w.seed}, {cores} threads over disjoint "
                     f"primary ranges, {o['collisions']} collisions in {o['seconds']:.2f} s",
           "avalanches_per_s": n_prim / o["seconds"], "null_per_s": o["null"] / o["seconds"], "real_per_s": o["real"] / o["seconds"]}
    if one_core:
        # SURVEY §8(d) "Oracle timing": the serial figure in the same harness — one thread on a sample sized to ~the same
        # seconds (1/cores of the primaries, at least one)
        n1 = max(1, n_prim // max(cores, 1))
        o1 = oracle_leg(w, n1, 1)
        out["one_core"] = {"value": o1["collisions"] / o1["seconds"], "unit": UNIT, "cores": 1,
                           "sample": f"first {n1} primaries, 1 thread, {o1['collisions']} collisions in {o1['seconds']:.2f} s",
                           "ns_per_collision": 1e9 * o1["seconds"] / max(o1["collisions"], 1)}
    return out


def workload_list(args):
    if args.workload == "all":
        return [(nm, max(1, int(round(args.steps * mult))), smp) for nm, (mult, smp) in ALL.items()
                if not (args.skip_heavy and nm in HEAVY)]
    smp = args.ref_primaries if args.ref_primaries > 0 else ALL.get(args.workload, (1, 0))[1]
    return [(args.workload, args.steps, smp)]


def run_reference(args) -> None:
    """--impl reference: the oracle on the host cores (rank 0 only), same metric/unit/config as our arm.  The headline is
    timed for K steps after W warm-ups on a bounded sample; the other configs get one bounded run each in per_config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    wl = workload_list(args)
    head = HEADLINE if args.workload == "all" else args.workload
    per, line = [], None
    for name, _, sample in wl:
        w = make_workload(name)
        if args.ref_primaries > 0:
            sample = args.ref_primaries
        if name == head:
            n_prim = min(w.n_primaries, sample) if sample > 0 else w.n_primaries
            for _ in range(args.warmup):
                oracle_leg(w, n_prim, cores)
            tot_c = tot_s = tot_n = tot_r = 0.0
            for _ in range(args.steps):
                o = oracle_leg(w, n_prim, cores)
                tot_c += o["collisions"]; tot_s += o["seconds"]; tot_n += o["null"]; tot_r += o["real"]
            v = tot_c / tot_s
            smp = f"first {n_prim} of {w.n_primaries} primaries of {w.name} per step, {cores} threads over disjoint primary ranges"
            cb = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": smp}
            line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                    "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / max(args.steps, 1), "higher_is_better": True,
                    "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                    "config": config_dict(w, args.gpus), "null_per_s": tot_n / tot_s, "real_per_s": tot_r / tot_s,
                    "avalanches_per_s": n_prim * args.steps / tot_s, "cpu_baseline": cb,
                    "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
            per.append({"workload": name, "value": v, "unit": UNIT, "ms_per_step": line["ms_per_step"], "steps": args.steps,
                        "null_per_s": line["null_per_s"], "real_per_s": line["real_per_s"],
                        "avalanches_per_s": line["avalanches_per_s"], "cpu_baseline": cb})
        elif sample < 0:
            continue                                                  # no oracle leg for this workload (see ALL)
        else:
            cb = cpu_baseline_entry(w, sample, cores)
            per.append({"workload": name, "value": cb["value"], "unit": UNIT, "steps": 1, "null_per_s": cb["null_per_s"],
                        "real_per_s": cb["real_per_s"], "avalanches_per_s": cb["avalanches_per_s"], "cpu_baseline": cb})
    line["per_config"] = per
    print(json.dumps(line), flush=True)


def bench_workload(avm, ctx, torch, dist, name, steps, warmup, sample, rank, world, peaks, flush, with_cpu, cores, head_name=None):
    """W warm-ups + exactly `steps` timed steps of one workload (device-timed, inputs resident) and the same through the
    user's call with host buffers (e2e); returns its per_config entry (rank 0) and the clock samples of the timed region."""
    w = make_workload(name, rank)
    id_offset = rank * w.n_primaries
    gg, fg = avm.gas_create(ctx, w.gas), avm.field_create(ctx, w.field)
    L = w.gas.n_levels
    has_b = any(v != 0.0 for v in w.field.B)
    bufs = avm.RunBuffers(ctx, w.capacity, w.n_primaries, L)
    prim_host = torch.from_numpy(w.primaries.copy()).pin_memory()
    prim_dev = prim_host.to(ctx.device)
    host = avm.HostBuffers(w.capacity, w.n_primaries, L, pinned=True)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def device_step(seed, flags=0):
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _, n = avm.run(ctx, gg, fg, prim_dev, bufs, seed=seed, t_max=w.t_max, id_offset=id_offset, flags=flags)
        e1.record()
        e1.synchronize()
        t = bufs.tallies_u64.cpu().numpy().view(np.uint64)
        k, kt = avm.run_stats(ctx)
        return {"ms": e0.elapsed_time(e1), "n": n, "tallies": t, "launches": k, "transport_launches": kt,
                "transport_ms": avm.run_transport_ms(ctx)}

    def e2e_step(seed):
        """The user's call: host primaries in (H2D inside avm_run), endpoints and tallies back to pinned host."""
        flush.zero_()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        _, n = avm.run(ctx, gg, fg, prim_host, bufs, seed=seed, t_max=w.t_max, id_offset=id_offset)
        res = avm.fetch(ctx, bufs, n, host)
        dt = time.perf_counter() - t0
        per_el = sum(getattr(host, a).element_size() * (getattr(host, a).numel() // host.capacity) for a in ("id", "avalanche", "status", "n_steps", "birth", "end"))
        d2h = n * per_el + host.per_avalanche.numel() * 8 + host.tallies_u64.numel() * 8 + host.tallies_f64.numel() * 8
        return {"s": dt, "n": n, "tallies": res.tallies_u64.copy(), "d2h": d2h}

    heavy = name in HEAVY
    if heavy:
        warmup = 0
    for i in range(warmup):
        device_step(w.seed + 1000 + i)
    sampler = ClockSampler(ctx.device.index or 0)
    barrier()
    sampler.start()
    st = [device_step(w.seed + i) for i in range(steps)]
    barrier()
    clocks = sampler.stop()
    for i in range(min(warmup, 2)):
        e2e_step(w.seed + 2000 + i)
    barrier()
    e2e = [] if heavy else [e2e_step(w.seed + i) for i in range(steps)]
    barrier()
    # the same workload under the energy-banded null-collision rate (AVM_RUN_BANDED): same collision physics (boundary losses differ: DESIGN.md §3.5 N7) in
    # fewer null steps, so collisions/s falls while avalanches/s rises — reported beside the headline, never as it
    for i in range(min(warmup, 2)):
        device_step(w.seed + 3000 + i, avm.RUN_BANDED)
    barrier()
    bd = [device_step(w.seed + i, avm.RUN_BANDED) for i in range(steps)]
    barrier()

    gfrac = grid_fraction(w.field)
    tot_ms = sum(s["ms"] for s in st)
    t_ms = sum(s["transport_ms"] for s in st)
    sums = [sum(int(s["tallies"][L]) for s in st), sum(int(s["tallies"][L + 1]) for s in st), sum(int(s["n"]) for s in st),
            sum(s["launches"] for s in st), sum(int(s["tallies"][L]) + int(s["tallies"][L + 1]) for s in e2e),
            sum(alg_fp64(s["tallies"], L, w.gas.level_type, has_b, gfrac) for s in st), sum(s["transport_launches"] for s in st)]
    e2e_s = sum(s["s"] for s in e2e) if e2e else 1.0
    bd_ms = sum(s["ms"] for s in bd)
    bd_sums = [sum(int(s["tallies"][L]) for s in bd), sum(int(s["tallies"][L + 1]) for s in bd), sum(int(s["n"]) for s in bd)]
    vals = torch.tensor([tot_ms, e2e_s, t_ms, bd_ms], dtype=torch.float64, device=ctx.device)
    sums_t = torch.tensor(sums + bd_sums, dtype=torch.float64, device=ctx.device)
    if dist is not None:
        dist.all_reduce(vals, op=dist.ReduceOp.MAX)          # reporting only: max time over ranks, job totals
        dist.all_reduce(sums_t, op=dist.ReduceOp.SUM)
    tot_ms_max, e2e_s_max, _, bd_ms_max = (float(x) for x in vals.cpu())
    null, real, electrons, launches, e2e_coll, _, _, bd_null, bd_real, bd_el = (float(x) for x in sums_t.cpu())
    if rank != 0:
        return None, clocks
    # roofline of the dominant kernel (transport_kernel), this rank: algorithmic units per launch / its average launch
    # duration (CUDA events recorded inside avm_run around each launch, on the ctx stream)
    n_launch = max(sums[6], 1)
    achieved = (sums[5] / n_launch) / ((t_ms / n_launch) * 1e-3)
    cap = ncu_capture(w.name)
    roofline = {"bound": "alu", "kernel": "transport_kernel", "achieved": achieved / 1e12, "peak": peaks["fp64_measured"] / 1e12,
                "unit": "T FP64 thread-instr/s", "frac": achieved / peaks["fp64_measured"],
                "frac_kind": "ALGORITHMIC FP64 thread-instructions of SURVEY §8(d) (null 90/170, real +110, ionisation +80, grid +45), "
                             "held fixed, / DFMA rate measured in this run; the kernel executes fewer (sass_fp64_per_collision_ncu)",
                "traffic": cap["traffic"], "sass_fp64_per_collision_ncu": cap["sass_fp64_per_collision_ncu"],
                "fp64_pipe_active_pct_ncu": cap["fp64_pipe_active_pct_ncu"], "ncu_source": cap["ncu_source"],
                "peak_source": "measured: avm_fp64_probe DFMA rate on this GPU in this run", "peak_nominal": peaks["fp64_nominal"] / 1e12,
                "alg_fp64_per_collision": sums[5] / max(sums[0] + sums[1], 1.0),
                # the three readings of "how busy is the FP64 pipe", side by side: algorithmic work / peak (frac, above), the
                # FP64 thread-instructions the kernel EXECUTES (ncu, per collision) x this run's collisions / time / peak, and
                # the share of cycles the FP64 pipe is busy (ncu).  The last two are null when the capture is stale.
                "frac_algorithmic": achieved / peaks["fp64_measured"],
                "frac_executed_lanes": (None if cap["sass_fp64_per_collision_ncu"] is None else
                                        cap["sass_fp64_per_collision_ncu"] * (sums[0] + sums[1]) / (t_ms * 1e-3) / peaks["fp64_measured"]),
                "frac_pipe_busy": None if cap["fp64_pipe_active_pct_ncu"] is None else cap["fp64_pipe_active_pct_ncu"] / 100.0,
                "launch_ms": t_ms / n_launch, "transport_share_of_step": t_ms / max(tot_ms, 1e-9)}
    if gfrac > 0.0:      # maps: the field gather against the MEASURED random-sector bandwidth; report the lower fraction's bound
        gb = gfrac * (sums[0] + sums[1]) * GATHER_BYTES_PER_GRID_STEP
        # the touched region (the holes' neighbourhood, a few MB per map) stays in L2 / L1 (DRAM traffic is ~3 B per step,
        # profiles/): the L2-resident random-sector rate is the binding denominator; the HBM one is printed beside it
        ach = gb / (t_ms * 1e-3) / 1e9
        roofline["gather"] = {"achieved_GBps": ach, "peak_GBps": peaks["gather_GBps"]["l2_64MB"],
                              "peak_kind": "measured random 32-byte-sector gather, 64 MB working set (L2-resident), this run",
                              "frac": ach / peaks["gather_GBps"]["l2_64MB"], "frac_vs_hbm_random_gather": ach / peaks["gather_GBps"]["hbm_1GiB"],
                              "bytes_per_grid_step": GATHER_BYTES_PER_GRID_STEP, "grid_step_fraction": gfrac}
    wall = tot_ms_max * 1e-3
    entry = {"workload": w.name, "value": (null + real) / wall, "unit": UNIT, "steps": steps, "warmup": warmup,
             "ms_per_step": tot_ms_max / max(steps, 1), "null_per_s": null / wall, "real_per_s": real / wall,
             "avalanches_per_s": world * w.n_primaries * steps / wall, "electrons_per_step": electrons / max(steps, 1) / world,
             "collisions_per_step": (null + real) / max(steps, 1) / world, "roofline": roofline,
             "e2e": (None if heavy else
                     {"value": e2e_coll / e2e_s_max, "unit": UNIT, "h2d_bytes_per_step": int(w.n_primaries * 64),
                      "d2h_bytes_per_step": int(sum(s["d2h"] for s in e2e) / max(len(e2e), 1)), "ms_per_step": 1e3 * e2e_s_max / max(steps, 1)}),
             "gpu_launches": int(launches), "config": config_dict(w, world), "capacity": w.capacity, "clocks": clocks,
             "banded": {"what": "same workload with AVM_RUN_BANDED (energy-banded null-collision rate, DESIGN.md §3.5): other random streams; the same collision "
                                "physics, but termination is tested at sampled points only (R13), so longer flights lose fewer electrons at absorbing "
                                "planes (config 1, oracle alone: gain +1.1 %, cathode share -2.1 points; DESIGN.md §3.5 N7) — not a like-for-like speed-up there",
                        "value": (bd_null + bd_real) / (bd_ms_max * 1e-3), "unit": UNIT, "ms_per_step": bd_ms_max / max(steps, 1),
                        "null_per_s": bd_null / (bd_ms_max * 1e-3), "real_per_s": bd_real / (bd_ms_max * 1e-3),
                        "avalanches_per_s": world * w.n_primaries * steps / (bd_ms_max * 1e-3),
                        "electrons_per_step": bd_el / max(steps, 1) / world,
                        "speedup_avalanches_per_s": tot_ms_max / max(bd_ms_max, 1e-9)}}
    if heavy:
        entry["timing"] = ("heavy entry: ONE timed run un-banded and ONE banded, device-timed like the others (CUDA events, inputs resident, "
                           "L2 flushed before), no warm-up runs of its own (kernels and clocks are warm from the preceding entries; one run "
                           "lasts seconds) and no e2e leg (host copies are < 0.1 % of such a run: see config3s / config4)")
    if with_cpu and sample >= 0:
        entry["cpu_baseline"] = cpu_baseline_entry(w, sample, cores, one_core=(name == head_name))
    return entry, clocks


def run_ours(args) -> None:
    import torch
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}: launch with torch.distributed.run --nproc-per-node {args.gpus}")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libavm has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    from paper_2509_15377_b200 import build as _build
    if rank == 0:
        _build.build()                               # no-op when libavm.so is newer than its sources
    if dist is not None:
        dist.barrier()
    from paper_2509_15377_b200 import avm            # raises when libavm.so is missing

    # weak scaling: every rank runs the whole workload on its own id range — avalanches are
    # independent, gas table and field are replicated, no data-path collective.
    ctx = avm.ctx_create(local_rank)
    peaks = measured_peaks(avm, ctx)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=ctx.device)       # > 126 MB L2
    cores = os.cpu_count() or 1
    with_cpu = world == 1 and not args.no_cpu_baseline
    head = HEADLINE if args.workload == "all" else args.workload
    per = []
    for name, steps, sample in workload_list(args):
        e, _ = bench_workload(avm, ctx, torch, dist, name, steps, args.warmup, sample, rank, world, peaks, flush, with_cpu, cores, head_name=head)
        if e is not None:
            per.append(e)
        torch.cuda.empty_cache()
    if rank == 0:
        h = next(e for e in per if e["workload"] == head)
        line = {"metric": METRIC, "value": h["value"], "unit": UNIT, "n_gpus": world, "steps": h["steps"], "warmup": args.warmup,
                "ms_per_step": h["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic", "config": h["config"],
                "null_per_s": h["null_per_s"], "real_per_s": h["real_per_s"], "avalanches_per_s": h["avalanches_per_s"],
                "electrons_per_step": h["electrons_per_step"], "collisions_per_step": h["collisions_per_step"],
                "e2e": h["e2e"], "gpu_launches": h["gpu_launches"], "roofline": h["roofline"], "clocks": h["clocks"],
                "headline": f"{head}: the largest BASELINE config by collisions per step that fits the bench budget (DESIGN.md §6); "
                            "all five configs are in per_config",
                "measured_peaks": {"fp64_T_thread_instr_per_s": peaks["fp64_measured"] / 1e12, "gather_GBps": peaks["gather_GBps"],
                                   "smem_random_8B_loads_per_s": peaks["smem_random_8B_loads_per_s"],
                                   "hbm_copy_GBps_MEASURED_PEAKS": peaks["hbm_copy_GBps_MEASURED_PEAKS"]},
                "kernel_source_hash": kernel_source_hash()}
        if "cpu_baseline" in h:
            line["cpu_baseline"] = h["cpu_baseline"]
        line["per_config"] = [{k: v for k, v in e.items() if k not in ("config",)} | {"note": e["config"]["note"]} for e in per]
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="all")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-primaries", type=int, default=0, help="oracle legs: first n primaries only (0 = the workload's default sample)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--skip-heavy", action="store_true", help="--workload all without the single-run heavy entries (config3 in full, config4x16/x64)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
