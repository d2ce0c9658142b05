#!/usr/bin/env python
"""bench.py — electron-collisions/s (real + null) of the avalanche hot path on B200, with its ALU roofline.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config2|config2x64|config1|config3s]
  python bench.py --impl reference ...     # the oracle on the host cores

A "step" is one pass of the whole hot path (avm_run: primary injection, persistent transport kernel with
secondary append and lane refill, tallies) over one batch of primaries of the workload.  Prints ONE JSON line.
Nothing here reads /root/reference.
"""
from __future__ import annotations

import argparse
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
# Algorithmic FP64 thread-instructions per unit: what the method must do.
FP64_PER_NULL = {False: 90.0, True: 170.0}       # free flight + energy + bin + decision; key = B != 0
FP64_PER_REAL_EXTRA = 110.0                      # deflection angles, basis, rotation, renormalise, speed
FP64_PER_ION_EXTRA = 80.0                        # Opal-Beaty atan/tan, child direction
FP64_PER_GRID_EXTRA = 45.0                       # fold + 7 lerps x 4 channels per step in a grid slab
GATHER_BYTES_PER_GRID_STEP = 128.0               # 8 nodes x 16 B
FP64_LANES_PER_SM = 64                           # one warp-wide FP64 instruction / 2 clk / scheduler
# From the committed ncu captures of the transport kernel (profiles/r1d_transport_ncu.md), per launch of the workload:
# DRAM bytes read + written, DFMA + DMUL + DADD thread-instructions per collision, FP64 pipe active %.
NCU_CAPTURE = {"config2": {"traffic": 3897344 + 48640, "sass_fp64_per_collision": 92.4, "fp64_pipe_active_pct": 22.9},
               "config2x16": {"traffic": 92790528 + 419887104, "sass_fp64_per_collision": 64.4, "fp64_pipe_active_pct": 27.3}}


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
    elif name == "config4":
        w = configs.config4(id_offset=rank * 1000)
    elif name.startswith("config4x"):
        w = configs.replicate(configs.config4(), int(name[len("config4x"):]))
    elif name == "config5":
        w = configs.config5(id_offset=rank * 200)
    else:
        raise SystemExit(f"unknown workload {name}")
    return w


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


def fp64_peak(avm, ctx) -> dict:
    """The ALU roofline denominator: FP64 thread-instructions per second.  Nominal = SMs x 64 FP64
    lanes x max SM clock; measured = the library's DFMA probe (8 independent chains per thread, 8 CTAs per SM)."""
    sm_max_mhz = 1965.0
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            sm_max_mhz = float(json.load(f).get("sm_max_mhz", sm_max_mhz))
    except Exception:
        pass
    nominal = ctx.sm_count * FP64_LANES_PER_SM * sm_max_mhz * 1e6
    best = 0.0
    for _ in range(3):
        best = max(best, avm.fp64_probe(ctx, iters=1 << 15)["dfma_per_s"])
    return {"nominal": nominal, "measured": best, "sm_max_mhz": sm_max_mhz}


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


def run_reference(args) -> None:
    """--impl reference: the oracle on the host cores (rank 0 only), same metric/unit/config as our arm."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.workload)
    cores = os.cpu_count() or 1
    n_prim = min(w.n_primaries, args.ref_primaries) if args.ref_primaries > 0 else w.n_primaries
    for _ in range(args.warmup):
        oracle_leg(w, n_prim, cores)
    tot_c, tot_s, tot_p, last = 0, 0.0, 0, None
    for _ in range(args.steps):
        last = oracle_leg(w, n_prim, cores)
        tot_c += last["collisions"]; tot_s += last["seconds"]; tot_p += n_prim
    v = tot_c / tot_s
    sample = f"first {n_prim} of {w.n_primaries} primaries of {w.name} per step, {cores} threads over disjoint primary ranges"
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / max(args.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "note": w.note, "n_primaries_per_step": n_prim},
            "avalanches_per_s": tot_p / tot_s,
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


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
    w = make_workload(args.workload, rank)
    id_offset = rank * w.n_primaries
    ctx = avm.ctx_create(local_rank)
    gg, fg = avm.gas_create(ctx, w.gas), avm.field_create(ctx, w.field)
    L = w.gas.n_levels
    has_b = any(v != 0.0 for v in w.field.B)
    bufs = avm.RunBuffers(ctx, w.capacity, w.n_primaries, L)
    prim_host = torch.from_numpy(w.primaries.copy()).pin_memory()
    prim_dev = prim_host.to(ctx.device)
    host = avm.HostBuffers(w.capacity, w.n_primaries, L, pinned=True)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=ctx.device)       # > 126 MB L2
    peak = fp64_peak(avm, ctx)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def device_step(seed):
        """One pass of the hot path, primaries resident in HBM; device time by CUDA events on the ctx stream."""
        flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _, n = avm.run(ctx, gg, fg, prim_dev, bufs, seed=seed, t_max=w.t_max, id_offset=id_offset)
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
        d2h = n * (8 + 4 + 4 + 4 + 5 * 8 + 8 * 8) + w.n_primaries * 24 + (L + 4) * 8 + 40
        return {"s": dt, "n": n, "tallies": res.tallies_u64.copy(), "d2h": d2h}

    for i in range(args.warmup):
        device_step(w.seed + 1000 + i)
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    steps = [device_step(w.seed + i) for i in range(args.steps)]
    barrier()
    clocks = sampler.stop()

    tot_ms = sum(s["ms"] for s in steps)
    null = sum(int(s["tallies"][L]) for s in steps)
    real = sum(int(s["tallies"][L + 1]) for s in steps)
    electrons = sum(int(s["n"]) for s in steps)
    launches = sum(s["launches"] for s in steps)
    t_launches = sum(s["transport_launches"] for s in steps)
    t_ms = sum(s["transport_ms"] for s in steps)
    gfrac = grid_fraction(w.field)
    fp64 = sum(alg_fp64(s["tallies"], L, w.gas.level_type, has_b, gfrac) for s in steps)

    for i in range(min(args.warmup, 2)):
        e2e_step(w.seed + 2000 + i)
    barrier()
    e2e = [e2e_step(w.seed + i) for i in range(args.steps)]
    barrier()
    e2e_s = sum(s["s"] for s in e2e)
    e2e_coll = sum(int(s["tallies"][L]) + int(s["tallies"][L + 1]) for s in e2e)
    e2e_d2h = sum(s["d2h"] for s in e2e) / max(len(e2e), 1)

    vals = torch.tensor([tot_ms, e2e_s, t_ms], dtype=torch.float64, device=ctx.device)
    sums = torch.tensor([null, real, electrons, launches, e2e_coll, fp64, t_launches], dtype=torch.float64, device=ctx.device)
    if dist is not None:
        dist.all_reduce(vals, op=dist.ReduceOp.MAX)          # reporting only: max time over ranks, job totals
        dist.all_reduce(sums, op=dist.ReduceOp.SUM)
    tot_ms, e2e_s, t_ms_max = (float(x) for x in vals.cpu())
    null, real, electrons, launches, e2e_coll, fp64_all, t_launches_all = (float(x) for x in sums.cpu())
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    value = (null + real) / (tot_ms * 1e-3)
    # roofline of the dominant kernel (transport_kernel), this rank: algorithmic FP64 thread-instructions per launch
    # / its average launch duration (CUDA events inside avm_run, on the ctx stream)
    achieved = (fp64 / max(t_launches, 1)) / ((t_ms / max(t_launches, 1)) * 1e-3)
    roofline = {"bound": "alu", "kernel": "transport_kernel", "achieved": achieved / 1e12, "peak": peak["measured"] / 1e12,
                "unit": "T FP64 thread-instr/s", "frac": achieved / peak["measured"],
                "traffic": NCU_CAPTURE.get(w.name, {}).get("traffic"),
                "traffic_source": "profiles/r1d_transport_ncu.md (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum, one launch)"
                                  if w.name in NCU_CAPTURE else None,
                "sass_fp64_per_collision_ncu": NCU_CAPTURE.get(w.name, {}).get("sass_fp64_per_collision"),
                "fp64_pipe_active_pct_ncu": NCU_CAPTURE.get(w.name, {}).get("fp64_pipe_active_pct"),
                "peak_source": "measured: avm_fp64_probe DFMA rate on this GPU in this run",
                "peak_nominal": peak["nominal"] / 1e12,
                "frac_of_nominal": achieved / peak["nominal"],
                "alg_fp64_per_collision": fp64 / max(null / world + real / world, 1.0) if world == 1 else None,
                "launch_ms": t_ms / max(t_launches, 1), "transport_share_of_step": t_ms / max(sum(s["ms"] for s in steps), 1e-9)}
    if gfrac > 0.0:      # grid maps: the field gather's algorithmic bytes beside the ALU figure
        gb = gfrac * (null + real) / world * GATHER_BYTES_PER_GRID_STEP
        roofline["field_gather_GBps"] = gb / (t_ms * 1e-3) / 1e9
        roofline["field_gather_bytes_per_step"] = GATHER_BYTES_PER_GRID_STEP
        roofline["grid_step_fraction"] = gfrac
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": tot_ms / max(args.steps, 1), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "note": w.note, "n_primaries_per_gpu": w.n_primaries, "capacity": w.capacity,
                       "l2": "256 MiB buffer written between timed iterations", "seed_per_step": "seed + step index",
                       "parallelism": f"replicas over primaries x{world}, no collective"},
            "null_per_s": null / (tot_ms * 1e-3), "real_per_s": real / (tot_ms * 1e-3),
            "avalanches_per_s": world * w.n_primaries * args.steps / (tot_ms * 1e-3),
            "electrons_per_step": electrons / max(args.steps, 1) / world,
            "collisions_per_step": (null + real) / max(args.steps, 1) / world,
            "e2e": {"value": e2e_coll / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(w.n_primaries * 64),
                    "d2h_bytes_per_step": int(e2e_d2h), "ms_per_step": 1e3 * e2e_s / max(args.steps, 1)},
            "gpu_launches": int(launches), "roofline": roofline, "clocks": clocks}
    if world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        n_prim = min(w.n_primaries, args.ref_primaries) if args.ref_primaries > 0 else w.n_primaries
        o = oracle_leg(w, n_prim, cores)
        line["cpu_baseline"] = {"value": o["collisions"] / o["seconds"], "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"first {n_prim} of {w.n_primaries} primaries of {w.name}, seed {w.seed}, "
                                          f"{o['collisions']} collisions in {o['seconds']:.2f} s",
                                "avalanches_per_s": n_prim / o["seconds"]}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="config2")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-primaries", type=int, default=0, help="oracle legs: first n primaries only (0 = all)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
