"""Thresholds of the same-seed comparisons = the observed values (gpurun_out/parity_margins.txt, copied into BASELINE.md §4)
with a stated margin: round 2 observed 100 % identical histories on configs 1-4 in full and on config 5's first 4
avalanches (99.8 % on its first 6: one electron of 444), endpoint errors of identical histories <= 3.4e-7 (config 4) and
<= 1.8e-5 (config 5, histories of 2e6 steps); required here: >= 99.5 % / 98 % identical, errors <= 3e-6 / 1e-4.

GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (primaries resident on the
device, the workload's capacity, default launch shape).

Configs 1, 2 and 4 are small enough for the oracle in full: the whole run is compared electron by electron.  Configs 3
(with bench's time cut) and 5 are not: the GPU runs them in full, properties that hold at any size are checked on every
electron (charge conservation, the step bookkeeping of the tallies, status validity, per-avalanche counts), and the
first avalanches — identical Philox streams to the oracle's run of the same primaries — are compared one by one.
"""
import os

import numpy as np
import pytest
import torch

from paper_2509_15377_b200.gen import configs
from test_gpu_parity import assert_run_same_seed

pytestmark = pytest.mark.gpu
CORES = os.cpu_count() or 1


@pytest.fixture(scope="module")
def ctx(avm):
    return avm.ctx_create(0)


def run_as_bench(avm, ctx, w, t_max=None):
    """avm_run the way bench.py's device_step does, then fetch."""
    gg, fg = avm.gas_create(ctx, w.gas), avm.field_create(ctx, w.field)
    bufs = avm.RunBuffers(ctx, w.capacity, w.n_primaries, w.gas.n_levels)
    prim_dev = torch.from_numpy(w.primaries.copy()).to(ctx.device)
    _, n = avm.run(ctx, gg, fg, prim_dev, bufs, seed=w.seed, t_max=w.t_max if t_max is None else t_max)
    return avm.fetch(ctx, bufs, n)


def check_invariants(r, w):
    """Properties of any correct run, whatever its size (D3)."""
    L = w.gas.n_levels
    t = r.tallies_u64
    ion = sum(int(t[l]) for l in range(L) if w.gas.level_type[l] == 2)
    att = sum(int(t[l]) for l in range(L) if w.gas.level_type[l] == 3)
    assert r.n == w.n_primaries + ion                                  # electrons = primaries + ionisations
    assert int((r.status == 5).sum()) == att                           # attached electrons = attachment collisions
    assert np.all((r.status >= 1) & (r.status <= 7))                   # every electron has a non-zero status
    assert sum(int(t[l]) for l in range(L)) == int(t[L + 1])           # level counts sum to the real collisions
    assert int(r.n_steps.astype(np.int64).sum()) == int(t[L + 3])      # steps
    ended_before_decision = int(((r.status != 5) & (r.n_steps > 0)).sum())
    assert int(t[L]) + int(t[L + 1]) + ended_before_decision == int(t[L + 3])   # null + real + last flights = steps
    pa = r.per_avalanche
    assert int(pa[:, 0].sum()) == r.n and np.array_equal(pa[:, 1], pa[:, 0] - 1) and int(pa[:, 2].sum()) == att
    assert np.array_equal(np.bincount(r.avalanche.astype(np.int64), minlength=w.n_primaries), pa[:, 0].astype(np.int64))
    assert len(np.unique(r.id)) == r.n                                 # hashed child ids do not collide (R16)
    assert np.all(r.end[3] >= r.birth[3])


def first_avalanches(r, m):
    """The electrons of avalanches 0 .. m-1 as a run result of their own."""
    sel = r.avalanche < m
    return type(r)(int(sel.sum()), r.id[sel], r.avalanche[sel], r.status[sel], r.n_steps[sel], r.birth[:, sel],
                   r.end[:, sel], r.per_avalanche[:m], r.tallies_u64, r.tallies_f64)


def test_config2_full_size(avm, ctx, oracle):
    w = configs.config2()
    gpu = run_as_bench(avm, ctx, w)
    check_invariants(gpu, w)
    cpu = oracle.run(w.gas, w.field, w.primaries, seed=w.seed, capacity=w.capacity, n_threads=CORES)
    assert cpu.n > 100000
    assert_run_same_seed(cpu, gpu, w.gas.n_levels, min_identical=0.999, label='config2 full size')
    L = w.gas.n_levels
    assert abs(int(gpu.tallies_u64[L + 3]) / int(cpu.tallies_u64[L + 3]) - 1) < 1e-3
    assert abs(gpu.n / cpu.n - 1) < 1e-3
    Wc = cpu.tallies_f64[2] / cpu.tallies_f64[3]; Wg = gpu.tallies_f64[2] / gpu.tallies_f64[3]
    assert abs(Wg / Wc - 1) < 1e-3


def test_config3_time_cut_full_size(avm, ctx, oracle):
    """bench's config3s: 1e5 primaries with B, t_max = 20 ns (the wide launch shape is chosen from the primary count)."""
    w = configs.config3(n_primaries=100000, t_max=20.0)
    gpu = run_as_bench(avm, ctx, w)
    check_invariants(gpu, w)
    assert (gpu.status == 6).sum() > 0.9 * w.n_primaries               # almost all reach the time cut
    m = 96
    cpu = oracle.run(w.gas, w.field, w.primaries[:m], seed=w.seed, t_max=20.0, n_threads=CORES)
    assert_run_same_seed(cpu, first_avalanches(gpu, m), w.gas.n_levels, min_identical=0.99, end_rtol=1e-9, label='config3 time cut, first 96 avalanches of the full-size run')


@pytest.mark.parametrize("flags", [0, 16], ids=["global", "banded"])
def test_config3_in_full(avm, ctx, oracle, flags):
    """BASELINE config 3 as stated — 1 cm gap, 1e5 primaries, NO time cut: ~1.3e12 steps un-banded (~3e11 banded), 1.4e7 per
    electron, several relaunches of the persistent kernel.  Every electron either reaches the far plane (status 2) or is
    attached on the way (status 5).  Any-size invariants on all of them; the first 32 avalanches electron by electron
    against the oracle's run of the same primaries (identical Philox streams); and what the config is for — drift
    velocity, Lorentz angle, diffusion, attachment over the FULL gap — of the other 99 968 electrons against those 32
    oracle electrons as a sample of the same population (3 standard errors of a 32-electron sample)."""
    w = configs.config3()
    assert w.n_primaries == 100000 and not np.isfinite(w.t_max)
    gg, fg = avm.gas_create(ctx, w.gas), avm.field_create(ctx, w.field)
    bufs = avm.RunBuffers(ctx, w.capacity, w.n_primaries, w.gas.n_levels)
    prim_dev = torch.from_numpy(w.primaries.copy()).to(ctx.device)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    _, n = avm.run(ctx, gg, fg, prim_dev, bufs, seed=w.seed, flags=flags)
    e1.record(); e1.synchronize()
    gpu = avm.fetch(ctx, bufs, n)
    check_invariants(gpu, w)
    L = w.gas.n_levels
    steps = int(gpu.tallies_u64[L + 3])
    _, n_transport = avm.run_stats(ctx)
    assert n == 100000 and steps > (1e12 if flags == 0 else 2e11)
    assert set(np.unique(gpu.status)) == {2, 5}                          # far plane or attached, nothing else
    assert int(gpu.n_steps.max()) > (1e7 if flags == 0 else 2e6)
    m = 32
    cpu = oracle.run(w.gas, w.field, w.primaries[:m], seed=w.seed, capacity=64, n_threads=CORES, flags=1 if flags else 0)
    from conftest import record_margin
    record_margin(f"config3 in full (flags {flags}): {steps:.4g} steps in {e0.elapsed_time(e1) / 1e3:.2f} s, {n_transport} transport launches, "
                  f"attached share {float((gpu.status == 5).mean()):.4f} (oracle's 32: {float((cpu.status == 5).mean()):.3f}), "
                  f"longest history {int(gpu.n_steps.max())} steps")
    # 1.4e7-step histories: accumulated rounding stays far below a decision's width in a uniform field (observed on B200: 32 of 32
    # identical, worst endpoint error 4.1e-12; 1.09e12 steps in 31.2 s un-banded, 2.3e11 in 12.1 s banded)
    assert_run_same_seed(cpu, first_avalanches(gpu, m), L, min_identical=0.93, end_rtol=1e-9, label=f"config3 in full (flags {flags}), first 32 avalanches")
    # the rest of the population against the oracle's 32 as a sample of it
    rest = gpu.avalanche >= m
    p_att = float((gpu.status[rest] == 5).mean())
    assert 0.05 < p_att < 0.7
    assert abs(float((cpu.status == 5).mean()) - p_att) <= 3.0 * np.sqrt(p_att * (1.0 - p_att) / m) + 1e-9
    g2, c2 = rest & (gpu.status == 2), cpu.status == 2
    nc = int(c2.sum())
    assert nc >= 10
    for name, fg_, fc_ in (("drift time", gpu.end[3] - gpu.birth[3], cpu.end[3] - cpu.birth[3]),
                           ("E x B displacement x", gpu.end[0] - gpu.birth[0], cpu.end[0] - cpu.birth[0]),
                           ("displacement y", gpu.end[1] - gpu.birth[1], cpu.end[1] - cpu.birth[1])):
        mu, sd = float(fg_[g2].mean()), float(fg_[g2].std(ddof=1))
        assert abs(float(fc_[c2].mean()) - mu) <= 3.0 * sd / np.sqrt(nc), (name, mu, sd, float(fc_[c2].mean()))
        ratio = float(fc_[c2].var(ddof=1)) / sd ** 2                      # diffusion: sample variance of nc against the population's
        assert abs(ratio - 1.0) <= 3.5 * np.sqrt(2.0 / (nc - 1)), (name, ratio)
    # transport coefficients of the full gap from the GPU's own endpoints: W = 0.98 cm / <T>, Lorentz angle, in the range the
    # 20 ns slice gives (test_config3_drift_lorentz_angle_and_diffusion) — the slice and the full gap must tell the same story
    d = gpu.end[0:3, g2] - gpu.birth[0:3, g2]
    T = (gpu.end[3, g2] - gpu.birth[3, g2])
    ang = float(np.degrees(np.arctan2(np.hypot(d[0].mean(), d[1].mean()), d[2].mean())))
    assert 1.0 < ang < 6.0 and 4e-4 < float(d[2].mean() / T.mean()) < 1.2e-3, (ang, float(d[2].mean() / T.mean()))


def test_config4_full_size(avm, ctx, oracle):
    w = configs.config4()
    gpu = run_as_bench(avm, ctx, w)
    check_invariants(gpu, w)
    cpu = oracle.run(w.gas, w.field, w.primaries, seed=w.seed, capacity=w.capacity, n_threads=CORES)
    assert cpu.n > 5000
    assert_run_same_seed(cpu, gpu, w.gas.n_levels, min_identical=0.995, end_rtol=3e-6, label='config4 full size')
    L = w.gas.n_levels
    assert abs(int(gpu.tallies_u64[L + 3]) / int(cpu.tallies_u64[L + 3]) - 1) < 2e-3


def test_config5_full_size(avm, ctx, oracle):
    w = configs.config5()
    gpu = run_as_bench(avm, ctx, w)
    check_invariants(gpu, w)
    m = 4
    cpu = oracle.run(w.gas, w.field, w.primaries[:m], seed=w.seed, capacity=1 << 16, n_threads=m)
    assert_run_same_seed(cpu, first_avalanches(gpu, m), w.gas.n_levels, min_identical=0.98, end_rtol=1e-4, label='config5 full size, first 4 avalanches')


def test_config3_drift_lorentz_angle_and_diffusion(avm, ctx, oracle):
    """What config 3 is for (BASELINE.json): drift velocity vector, Lorentz angle and diffusion in E = 1 kV/cm with
    B = 1 T at 30 degrees, from the endpoints of the full-size GPU run (time cut 20 ns, 1e5 electrons) against the oracle's
    run of 6000 other primaries (independent streams: seed 1): components within 3 combined standard errors and 1.5 %."""
    w = configs.config3(n_primaries=100000, t_max=20.0)
    gpu = run_as_bench(avm, ctx, w)
    wo = configs.config3(n_primaries=6000, seed=1, t_max=20.0)
    cpu = oracle.run(wo.gas, wo.field, wo.primaries, seed=1, t_max=20.0, n_threads=CORES)

    def transport(r):
        sel = r.status == 6                                            # reached the time cut: same flight time for all
        d = r.end[0:3, sel] - r.birth[0:3, sel]
        T = (r.end[3, sel] - r.birth[3, sel]).mean()
        n = sel.sum()
        W = d.mean(axis=1) / T
        W_se = d.std(axis=1, ddof=1) / np.sqrt(n) / T
        D = d.var(axis=1, ddof=1) / (2 * T)                            # diffusion coefficients along x, y, z
        D_se = D * np.sqrt(2.0 / (n - 1))
        return W, W_se, D, D_se, n

    Wg, Wg_se, Dg, Dg_se, ng = transport(gpu)
    Wc, Wc_se, Dc, Dc_se, nc = transport(cpu)
    assert ng > 90000 and nc > 5400
    for a in range(3):
        se = np.hypot(Wg_se[a], Wc_se[a])
        assert abs(Wg[a] - Wc[a]) <= 3 * se + 0.015 * np.linalg.norm(Wc), (a, Wg, Wc, se)
        assert abs(Dg[a] - Dc[a]) <= 3 * np.hypot(Dg_se[a], Dc_se[a]) + 0.015 * Dc[a], (a, Dg, Dc)
    # Lorentz angle: between the drift velocity and the force direction (+z, reading R1); its standard error from the
    # transverse components' (the oracle's 6000 electrons dominate it)
    ang = lambda W: np.degrees(np.arccos(W[2] / np.linalg.norm(W)))
    ang_se = lambda W, se: np.degrees(np.hypot(se[0], se[1]) / W[2])
    assert Wg[2] > 0 and abs(Wg[0]) > 3 * Wg_se[0]                     # E x B drift along x is resolved
    assert abs(ang(Wg) - ang(Wc)) <= 3 * np.hypot(ang_se(Wg, Wg_se), ang_se(Wc, Wc_se)) + 0.1, (ang(Wg), ang(Wc))
    assert 1.0 < ang(Wg) < 6.0


def test_config5hg_high_gain_stack(avm, ctx, oracle):
    """The high-gain variant of config 5 (D4: the three maps at dV = 500 V; NOT a BASELINE config): avalanches of
    10^4-10^5 electrons through the three-map stack — the append / refill / occupancy stress BASELINE's config 5 text asks
    for and the synthetic gas does not deliver at 400 V.  The oracle cannot run it in test time (one avalanche is ~4e9
    collisions on one core), so: the any-size invariants on every electron of the full run, un-banded and banded, and
    electron-by-electron parity with the oracle on ONE such GEM (config 4's cell at 500 V, 32 primaries, ~40 electrons each,
    both rate modes)."""
    w = configs.config5hg()
    gpu = run_as_bench(avm, ctx, w)
    check_invariants(gpu, w)
    size = gpu.per_avalanche[:, 0].astype(float)
    assert 5e3 < size.mean() < 3e5 and size.max() > 1e4, size
    gg, fg = avm.gas_create(ctx, w.gas), avm.field_create(ctx, w.field)
    bufs = avm.RunBuffers(ctx, w.capacity, w.n_primaries, w.gas.n_levels)
    _, n = avm.run(ctx, gg, fg, torch.from_numpy(w.primaries.copy()).to(ctx.device), bufs, seed=w.seed, flags=avm.RUN_BANDED)
    banded = avm.fetch(ctx, bufs, n)
    check_invariants(banded, w)
    sb = banded.per_avalanche[:, 0].astype(float)
    assert 5e3 < sb.mean() < 3e5
    from conftest import record_margin
    L = w.gas.n_levels
    record_margin(f"config5hg (8 primaries, dV 500 V): electrons per avalanche un-banded {sorted(size.astype(int))}, banded {sorted(sb.astype(int))}; "
                  f"collisions {int(gpu.tallies_u64[L] + gpu.tallies_u64[L + 1])} / {int(banded.tallies_u64[L] + banded.tallies_u64[L + 1])}")
    del bufs, fg
    torch.cuda.empty_cache()
    w4 = configs.config4(n_primaries=32, dv=configs.HG_DV)
    for flags, oflags in ((0, 0), (avm.RUN_BANDED, 1)):
        cpu = oracle.run(w4.gas, w4.field, w4.primaries, seed=0, capacity=1 << 18, n_threads=CORES, flags=oflags)
        g4, f4 = avm.gas_create(ctx, w4.gas), avm.field_create(ctx, w4.field)
        b4 = avm.RunBuffers(ctx, 1 << 18, 32, L)
        _, n4 = avm.run(ctx, g4, f4, torch.from_numpy(w4.primaries.copy()).to(ctx.device), b4, seed=0, flags=flags)
        assert cpu.n > 600
        assert_run_same_seed(cpu, avm.fetch(ctx, b4, n4), L, min_identical=0.99, end_rtol=3e-6, label=f'single GEM at 500 V, 32 primaries, flags {flags}')


def test_config5_as_worded_200_high_gain_avalanches(avm, ctx, oracle):
    """BASELINE config 5 as it is WORDED — "200 primaries with avalanches of 1e4-1e5 electrons each, stressing secondary
    append, compaction and occupancy" (triple GEM, gain 1e4 and up) — needs the 500 V maps with the
    synthetic gas (D4): config5hg with 200 primaries, ~4e6 electrons through the three-map stack, under the
    banded rate (un-banded is the same run in 3x the steps).  Any-size invariants on every electron (observed on B200:
    5.07e6 electrons, 8.3e10 collisions in 8.0 s, 133 of 200 avalanches above 1e4 electrons, largest 1.07e5).

    NOT asserted here, and open: the first 2 avalanches of this stack against the banded oracle,
    electron by electron.  Measured once in round 3: 3089 (oracle) vs 3127 electrons, 94.5 % of the ids in common, 95.3 % of
    those with identical histories, median endpoint error 1.3e-9 but one history 2.2e-2 off — one avalanche grown from one
    primary through three GEMs, where an early rounding flip replaces a whole sub-tree.  Per-step parity on the same maps
    holds at 1e-12 and the single-GEM test above is 100 % identical, so this reads as amplification, but it has not been
    traced to its first diverging step and is therefore not claimed as parity."""
    w = configs.config5hg(n_primaries=200)
    w.capacity = 200 * 120000
    gg, fg = avm.gas_create(ctx, w.gas), avm.field_create(ctx, w.field)
    L = w.gas.n_levels
    bufs = avm.RunBuffers(ctx, w.capacity, w.n_primaries, L)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    _, n = avm.run(ctx, gg, fg, torch.from_numpy(w.primaries.copy()).to(ctx.device), bufs, seed=w.seed, flags=avm.RUN_BANDED)
    e1.record(); e1.synchronize()
    gpu = avm.fetch(ctx, bufs, n)
    check_invariants(gpu, w)
    size = gpu.per_avalanche[:, 0].astype(float)
    assert n > 1.5e6 and (size >= 1e4).sum() >= 60, (n, np.sort(size)[-5:])
    from conftest import record_margin
    record_margin(f"config5 as worded (config5hg, 200 primaries, banded): {n} electrons, {int(gpu.tallies_u64[L] + gpu.tallies_u64[L + 1])} collisions in "
                  f"{e0.elapsed_time(e1) / 1e3:.2f} s; avalanche size median {int(np.median(size))}, max {int(size.max())}, {(size >= 1e4).sum()} of 200 above 1e4")
