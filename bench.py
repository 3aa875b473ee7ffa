#!/usr/bin/env python
"""bench.py -- CRKSPH pair-interactions/s on one (or N independent) B200(s).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cosmo] [--n-side 256] [--impl ours|reference]

A "step" is one pass of the whole hot path (crk_step_derivs: sort + leaves + interaction list, volumes, RK moments +
3x3 solve, grad v, momentum/energy) over one synthetic particle set (BASELINE.json configs[3]: 256^3 = 16.8 M
Zel'dovich-displaced particles, recipe in DESIGN.md).  Prints ONE JSON line (contract in the task statement):
  value     pair-interactions/s = ALGORITHMIC pair terms per step / step time, inputs resident in HBM: accepted ordered
            pairs of the four pair sums the method defines (volumes + RK moments + grad v over the gather set, forces over
            the symmetric set: 3 x gather + sym).  The library evaluates the moments and grad v sums in ONE merged sweep,
            so the pair evaluations it actually executes per step are 2 x gather + sym; that rate is reported beside the
            headline as executed_pair_evals_per_s.  The CPU baseline counts with the same 3 x gather + sym formula.
  e2e       the same through crk_step_derivs_host (pinned HOST buffers, H2D + D2H inside the timed region)
  roofline  dominant kernel (k_forces, Eqs. 17-18) algorithmic FP32 flop rate against the FP32 FMA-pipe peak
  cpu_baseline  the FP64 oracle, as it stands, on the FULL workload of the line (grid neighbour build; the O(n^2)
                brute-force build on a bounded window is kept as a second key)
With --impl reference the oracle itself is the timed arm.  N > 1: one process per GPU, each with its own seeded box
(weak scaling, no data-path collective); rank 0 prints the aggregate.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import crk_workloads as wl  # noqa: E402

METRIC = "CRKSPH pair-interactions/sec"
UNIT = "pair-interactions/s"
# canonical algorithmic FP32 flops per accepted ordered pair (restated in DESIGN.md)
FLOPS_PER_PAIR = {"volumes": 16.0, "moments": 100.0, "gradv": 90.0, "forces": 250.0}
FP32_PEAK_THEORETICAL = 148 * 128 * 2 * 1.965e9     # SMs x FP32 lanes x 2 (FMA) x max SM clock
# ncu-derived, per-launch numbers of the dominant kernel (dram bytes, FMA-pipe %) are NOT hard-coded here: they are read from
# the text summary that `python -m paper_2202_02840_b200.ncu_summary` wrote from the kept ncu capture (file named below),
# and only for the workload that capture was taken on; otherwise `traffic` is null.
NCU_SUMMARY = os.path.join(ROOT, "profiles", "r02_ncu_kernels.json")


BASE_SEEDS = {"tiny_uniform": 1001, "blast_wave": 1002, "clustered": 1003, "cosmo": 1004, "cosmo_large": 1005,
              "clustered_large": 1006}


def rank_seed(config: str, rank: int) -> int:
    """N > 1 shards by independent boxes: rank r evaluates its own seeded box of the same recipe (rank 0 = the
    BASELINE seed), so there is no data-path collective."""
    return BASE_SEEDS[config] + 7919 * rank


def aggregate_over_ranks(ms, e2e_ms, pairs, particles, world, device):
    """whole-job numbers: times are the MAX over ranks, work is the SUM over ranks (one all-reduce each; the only
    collectives of the run, outside the timed region).  Works with nccl (cuda device) and gloo (cpu device)."""
    import torch
    import torch.distributed as dist
    tot = torch.tensor([ms, e2e_ms], device=device, dtype=torch.float64)
    work = torch.tensor([pairs, particles], device=device, dtype=torch.float64)
    if world > 1:
        dist.all_reduce(tot, op=dist.ReduceOp.MAX)
        dist.all_reduce(work, op=dist.ReduceOp.SUM)
    return float(tot[0]), float(tot[1]), float(work[0]), float(work[1])


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region"""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], None, set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [t.strip() for t in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax = float(f[1])
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_sample(ps, target_particles=30000):
    """bounded window of the workload for the CPU oracle: a cube around the box centre holding ~target particles"""
    half = 0.5 * (target_particles / ps.n) ** (1.0 / 3.0)
    idx, _ = wl.select_window(ps, (0.5, 0.5, 0.5), half, 0.0)
    return ps.subset(idx), half


def time_oracle(sub, grid=False):
    """one full derivative evaluation by the oracle as it stands (FP64; grid=True: neighbours through the uniform-grid build,
    bit-identical structure to the O(n^2) scan).  Returns (pairs, seconds, threads, kind)."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import crk_oracle
    o = crk_oracle.Oracle(sub.box, sub.gamma, sub.n_h)
    t0 = time.perf_counter()
    try:
        d = o.step_derivs(sub, grid=grid)
    except RuntimeError:                       # fewer than 3 grid cells per side: the brute-force build is the only one
        grid = False
        t0 = time.perf_counter()
        d = o.step_derivs(sub)
    dt = time.perf_counter() - t0
    pairs = 3.0 * float(d["nbr_count"].astype(np.int64).sum()) + float(d["pair_count"].astype(np.int64).sum())
    kind = "oracle (FP64, uniform-grid neighbour build)" if grid else "oracle (FP64, brute-force O(n^2) neighbour build)"
    return pairs, dt, crk_oracle.get_threads(), kind


def grid_oracle_feasible(ps, full_limit):
    """the uniform-grid build bins at the largest h: fine for the lattice-like workloads, quadratic in the densest cell of a
    clustered one -- those, and workloads beyond `full_limit` particles, are timed on a bounded window instead"""
    return ps.n <= full_limit and float(ps.h.max()) / float(ps.h.min()) < 4.0


def workload_stats(ps, gather_cnt=None, sym_cnt=None, seg=None):
    """what BASELINE.json says about a config, measured: h range, neighbour numbers, leaves that need more than one list segment"""
    st = {"h_min": float(ps.h.min()), "h_max": float(ps.h.max()), "h_max_over_min": float(ps.h.max() / ps.h.min()),
          "h_p99_over_p1": float(np.percentile(ps.h, 99) / np.percentile(ps.h, 1))}
    if gather_cnt is not None:
        st.update(nbr_mean=float(gather_cnt.mean()), nbr_min=int(gather_cnt.min()), nbr_max=int(gather_cnt.max()))
    if sym_cnt is not None:
        st.update(pairs_mean=float(sym_cnt.mean()), pairs_max=int(sym_cnt.max()))
    if seg is not None:
        st.update(multi_segment_leaf_frac=float((seg[:, 0] != 0).mean()), candidates_first_segment_mean=float((seg[:, 1] & 0x7fff).mean()),
                  rows_first_segment_mean=float((seg[:, 1] >> 16).mean()))
    return st


def run_reference(args, rank, world):
    """--impl reference: the oracle (oracle/crk_oracle.cpp) timed as it stands on the host cores; each step is one full
    derivative evaluation of a bounded window of the same workload (sized so that K + W steps end within minutes)."""
    if rank != 0:
        return
    ps = wl.make_config(args.config, args.n_side)
    grid = float(ps.h.max()) / float(ps.h.min()) < 4.0
    sub, half = oracle_sample(ps, args.reference_particles if grid else args.oracle_particles)
    for _ in range(1 if args.warmup > 0 else 0):
        time_oracle(sub, grid)
    tot_pairs, tot_t, cores, kind = 0.0, 0.0, 0, ""
    for _ in range(args.steps):
        pairs, dt, cores, kind = time_oracle(sub, grid)
        tot_pairs += pairs; tot_t += dt
    value = tot_pairs / tot_t
    sample = f"cube of half-width {half:.4f} at the box centre of {ps.name} n_side={ps.meta['n_side']}: {sub.n} of {ps.n} particles"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": 1 if args.warmup > 0 else 0, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{ps.name} n_side={ps.meta['n_side']} (bounded sample)", "particles": sub.n},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": kind, "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2202_02840_b200 import Crk, crk_measure_fp32_peak

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # each rank owns an independent seeded box of the same recipe (weak scaling; the path has no exchange step on one box)
    ps = wl.make_config(args.config, args.n_side, seed=rank_seed(args.config, rank))
    if args.n_h is not None:
        ps.h[:] = (ps.h * (args.n_h / ps.n_h)).astype(np.float32)
        ps.n_h = float(args.n_h)
    names = ("x", "y", "z", "h", "vx", "vy", "vz", "m", "u")
    host = [torch.from_numpy(np.ascontiguousarray(getattr(ps, k))).pin_memory() for k in names]
    t = [h.to(dev, non_blocking=True) for h in host]
    out = [torch.empty(ps.n, device=dev) for _ in range(4)]
    ctx = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h)

    # accepted ordered pairs per sweep (exact counts from the staged API, outside the timed region)
    ctx.build_cells(*t[:4])
    _, _, cnt = ctx.volumes(t[7])
    ctx.rk_coefficients(want=False)
    res = ctx.hydro_derivs(t[4], t[5], t[6], t[8])
    gather_pairs = float(cnt.to(torch.int64).sum().item())
    sym_pairs = float(res[4].to(torch.int64).sum().item())
    pairs_per_step = 3.0 * gather_pairs + sym_pairs
    wstats = workload_stats(ps, cnt.cpu().numpy(), res[4].cpu().numpy(), ctx.leaf_segments().cpu().numpy().astype(np.uint32))
    wstats["s14_fallback_particles"] = int(ctx.stats()["n_fallback"])     # particles with a singular m2 (S14)
    del cnt, res
    big = ps.n > 40_000_000 or args.no_next_rows        # 512^3: skip the next-row extras (they need copies of the state)

    ctx.set_timing(True)
    for _ in range(max(args.warmup, 3)):
        ctx.step_derivs(*t, out=out)
    torch.cuda.synchronize()
    ctx.reset_stats()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        ctx.step_derivs(*t, out=out)
    e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = e0.elapsed_time(e1)
    st = ctx.stats()
    clocks = sampler.stop() if rank == 0 else None
    launches = st["launches"]

    next_rows = None
    if not big:
        # NEXT row 1 (compatible energy sweep, Eqs. 19-23) on the resident state: reported beside the step, not part of it
        du = torch.empty(ps.n, device=dev)
        ctx.compatible_energy(1e-3, out=du)
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record()
        for _ in range(3):
            ctx.compatible_energy(1e-3, out=du)
        c1.record()
        torch.cuda.synchronize()
        compat_ms = c0.elapsed_time(c1) / 3
        # NEXT row 3 (evolved h, Eqs. 51-53): a 40 B/particle stream pass (posh 16 + posV 16 + perm 4 read, h 4 written)
        ctx.evolve_h(out=du)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(5):
            ctx.evolve_h(out=du)
        c1.record()
        torch.cuda.synchronize()
        evolve_ms = c0.elapsed_time(c1) / 5
        # NEXT row 2a (time-step criteria, Eqs. 46-50): the momentum sweep with the two extra maxima, and the stream pass
        ctx_ts = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, timestep=True)
        ctx_ts.set_timing(True)
        for _ in range(2):
            ctx_ts.step_derivs(*t, out=out)
        torch.cuda.synchronize()
        ctx_ts.reset_stats()
        for _ in range(3):
            ctx_ts.step_derivs(*t, out=out)
        torch.cuda.synchronize()
        forces_ts_ms = ctx_ts.stats()["ms_forces"]
        ctx_ts.timestep(0.25, out=du)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(5):
            ctx_ts.timestep(0.25, out=du)
        c1.record()
        torch.cuda.synchronize()
        timestep_ms = c0.elapsed_time(c1) / 5
        dt_global = float(du.min().item())
        # NEXT row 2b (velocity-Verlet step, Eq. 43 = two derivative evaluations + two stream passes) on a copy of the state
        tk = [q.clone() for q in t]
        ctx_ts.kdk_step(*tk, 0.1 * dt_global)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(3):
            ctx_ts.kdk_step(*tk, 0.1 * dt_global)
        c1.record()
        torch.cuda.synchronize()
        kdk_ms = c0.elapsed_time(c1) / 3
        ctx_r = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, kdk_reuse=True)
        ctx_r.kdk_step(*tk, 0.1 * dt_global)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(3):
            ctx_r.kdk_step(*tk, 0.1 * dt_global)
        c1.record()
        torch.cuda.synchronize()
        kdk_reuse_ms = c0.elapsed_time(c1) / 3
        del ctx_r
        ctx_c = Crk(box=ps.box, gamma=ps.gamma, n_h=ps.n_h, kdk_reuse=True, kdk_compatible=True)
        ctx_c.kdk_step(*tk, 0.1 * dt_global)
        torch.cuda.synchronize()
        c0.record()
        for _ in range(3):
            ctx_c.kdk_step(*tk, 0.1 * dt_global)
        c1.record()
        torch.cuda.synchronize()
        kdk_compat_ms = c0.elapsed_time(c1) / 3
        # NEXT row 4b (active / passive particles): the hydro sweeps for the 10 % of the particles with the
        # smallest h (the deepest time bins of a hierarchical scheme), against the same call with every particle active
        order = torch.argsort(t[3])
        act = torch.zeros(ps.n, device=dev, dtype=torch.uint8)
        act[order[: ps.n // 10]] = 1
        allon = torch.ones(ps.n, device=dev, dtype=torch.uint8)
        ctx.hydro_derivs_active(act, t[4], t[5], t[6], t[8], out=out)
        torch.cuda.synchronize()
        active_ms = {}
        slab = (t[0] < 0.1 * ps.box).to(torch.uint8)           # a spatially compact active set (a slab holding ~10 % of the particles)
        for key, mask in (("active_10pct_ms", act), ("active_slab10pct_ms", slab), ("active_100pct_ms", allon)):
            c0.record()
            for _ in range(3):
                ctx.hydro_derivs_active(mask, t[4], t[5], t[6], t[8], out=out)
            c1.record()
            torch.cuda.synchronize()
            active_ms[key] = c0.elapsed_time(c1) / 3
            sa = ctx.stats()
            active_ms[key.replace("_ms", "_leaves")] = [int(sa["n_active_leaves"]), int(sa["n_halo_leaves"]), int(sa["n_leaves"])]
        del order, act, allon, slab
        del du, ctx_ts, ctx_c, tk
        next_rows = {"forces_with_timestep_maxima_ms": forces_ts_ms, "timestep_pass_ms": timestep_ms,
                     "timestep_global_min": dt_global, "kdk_step_ms": kdk_ms, "kdk_step_reuse_ms": kdk_reuse_ms,
                     "kdk_step_compatible_reuse_ms": kdk_compat_ms, "evolve_h_ms": evolve_ms,
                     "evolve_h_gbs_moved": 40.0 * ps.n / (evolve_ms * 1e-3) / 1e9,
                     "compatible_energy_ms": compat_ms,
                     "compatible_energy_fp32_frac": (FLOPS_PER_PAIR["forces"] + 20.0) * sym_pairs / (compat_ms * 1e-3) / FP32_PEAK_THEORETICAL,
                     "hydro_active": active_ms}

    # end to end through the host-pointer C ABI entry (pinned host inputs -> device -> compute -> host outputs)
    oh = [torch.empty(ps.n).pin_memory() for _ in range(4)]
    ctx.set_timing(False)
    ctx.step_derivs_host(*host, oh)
    torch.cuda.synchronize()
    k2 = max(1, min(args.steps, 5))
    t0 = time.perf_counter()
    for _ in range(k2):
        ctx.step_derivs_host(*host, oh)
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t0) / k2

    ms_all, e2e_all, pairs_all, n_all = aggregate_over_ranks(ms, e2e_ms, pairs_per_step, float(ps.n), world, dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_per_step = ms_all / args.steps
    value = pairs_all / (ms_per_step * 1e-3)
    peaks, peak_kind = load_peaks()
    fp32_meas, _ = crk_measure_fp32_peak(5)
    fp32_3reg, _ = crk_measure_fp32_peak(5, three_reg=True)
    forces_ms = st["ms_forces"]
    forces_flops = FLOPS_PER_PAIR["forces"] * sym_pairs
    achieved = forces_flops / (forces_ms * 1e-3) / 1e12 if forces_ms > 0 else None
    ncu = None
    if os.path.exists(NCU_SUMMARY):
        with open(NCU_SUMMARY) as f:
            ncu = json.load(f)
        if ncu.get("workload") != f"{ps.name} n_side={ps.meta['n_side']}" or args.n_h is not None:
            ncu = None
    kf = (ncu or {}).get("kernels", {}).get("k_forces")
    roofline = {"bound": "alu", "kernel": "k_forces (Eqs. 17-18 + limited viscosity)",
                "achieved": achieved, "peak": FP32_PEAK_THEORETICAL / 1e12, "unit": "TFLOP/s",
                "frac": (achieved / (FP32_PEAK_THEORETICAL / 1e12)) if achieved else None,
                "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md section 5.4; MEASURED_PEAKS.json has no FP32 figure)",
                "peak_measured": fp32_meas / 1e12,
                "frac_vs_peak_measured": (achieved / (fp32_meas / 1e12)) if achieved and fp32_meas > 0 else None,
                "peak_measured_source": "crk_measure_fp32_peak: register-resident FFMA chains on every SM, this run",
                "peak_measured_3reg": fp32_3reg / 1e12,
                "frac_vs_peak_measured_3reg": (achieved / (fp32_3reg / 1e12)) if achieved and fp32_3reg > 0 else None,
                "peak_measured_3reg_source": "crk_measure_fp32_peak_3reg: the same loop with three register operands per FFMA "
                                             "(a = b*c + a, the form of every accumulated pair sum): the register file feeds it at "
                                             "~61 % of the nominal rate (DESIGN.md section 5.4)",
                "flops_per_pair": FLOPS_PER_PAIR["forces"], "pairs_per_launch": sym_pairs, "kernel_ms": forces_ms,
                "traffic": (kf["dram_bytes_read"] + kf["dram_bytes_write"]) if kf else None,
                "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum; algorithmic minimum 144 B j-state + 16 B outputs per particle)",
                "traffic_source": (os.path.relpath(NCU_SUMMARY, ROOT) + " <- " + ncu.get("source", "?")) if kf else None,
                "ncu_fma_pipe_pct": {k: v.get("fma_pipe_pct") for k, v in ncu["kernels"].items()} if ncu else None}
    passes = {k: st[k] for k in ("ms_sort", "ms_tree", "ms_lists", "ms_volumes", "ms_rk", "ms_gradv", "ms_forces")}
    passes["ms_hydro_prep"] = max(st["ms_hydro"] - st["ms_forces"] - st["ms_gradv"], 0.0)   # pack + permute v, u into the state rows
    alg_flops = (FLOPS_PER_PAIR["volumes"] + FLOPS_PER_PAIR["moments"] + FLOPS_PER_PAIR["gradv"]) * gather_pairs + forces_flops
    sweeps_ms = st["ms_volumes"] + st["ms_rk"] + st["ms_gradv"] + st["ms_forces"]
    sort_bytes = ps.n * (st["sort_passes"] * 32.0 + 16 + 12 + 32 + 16)    # radix passes + pack + gather
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": f"{ps.name} n_side={ps.meta['n_side']} ({ps.n} particles per GPU, ~{gather_pairs / ps.n:.1f} neighbours"
                               + (f", n_h rescaled to {args.n_h}" if args.n_h is not None else "") + ")",
                   "particles": int(n_all), "pairs_per_step": pairs_all,
                   "l2": "inputs and per-step state exceed the 126 MB L2 (no flush needed)" if ps.n * 200 > 126e6
                         else "state fits in L2 (small config; not the headline)",
                   "stats": wstats},
        "value_counts": "algorithmic pair terms: 3 x gather pairs (volumes, RK moments, grad v) + symmetric pairs (forces)",
        # what the kernels execute: moments and grad v share one sweep (ratio of rank 0's counts applied to the whole job)
        "executed_pair_evals_per_s": value * (2.0 * gather_pairs + sym_pairs) / pairs_per_step,
        "particle_updates_per_s": n_all / (ms_per_step * 1e-3),
        "passes_ms": passes, "timed_steps": st["timed_steps"],
        "fp32_frac_pair_passes": alg_flops / (sweeps_ms * 1e-3) / FP32_PEAK_THEORETICAL if sweeps_ms > 0 else None,
        "sort_gbs": sort_bytes / (st["ms_sort"] * 1e-3) / 1e9 if st["ms_sort"] > 0 else None,
        "hbm_peak_gbs": peaks.get("hbm_gbs"), "peaks": peak_kind,
        "e2e": {"value": pairs_all / (e2e_all * 1e-3), "unit": UNIT, "ms_per_step": e2e_all,
                "h2d_bytes_per_step": int(9 * 4 * n_all), "d2h_bytes_per_step": int(4 * 4 * n_all)},
        "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
        "passes_note": "ms_rk = RK moments + FP64 solve + the Eq. 26 velocity-gradient sums in one sweep (ms_gradv is 0 in crk_step_derivs)",
        "next_rows": next_rows,
    }
    if world == 1 and not args.no_cpu_baseline:
        # the oracle as it stands on the FULL workload of this line where its grid build can take it (same config as `value`);
        # clustered / very large workloads: a bounded window.  The O(n^2) brute-force build on a window stays as a second key.
        if grid_oracle_feasible(ps, args.cpu_full_limit):
            pairs, dt, cores, kind = time_oracle(ps, grid=True)
            sample = f"the full workload: all {ps.n} particles, one derivative evaluation"
            same = True
        else:
            sub, half = oracle_sample(ps, args.oracle_particles)
            pairs, dt, cores, kind = time_oracle(sub, grid=False)
            sample = f"cube of half-width {half:.4f} at the box centre: {sub.n} of {ps.n} particles (the uniform-grid build is quadratic in the densest cell of this workload)"
            same = False
        line["cpu_baseline"] = {"value": pairs / dt, "unit": UNIT, "cores": cores, "kind": kind, "seconds": dt,
                                "same_config": same, "sample": sample}
        if same and not args.no_bruteforce:
            sub, half = oracle_sample(ps, args.oracle_particles)
            pairs, dt, cores, kind = time_oracle(sub, grid=False)
            line["cpu_baseline_bruteforce"] = {"value": pairs / dt, "unit": UNIT, "cores": cores, "kind": kind, "seconds": dt,
                                               "sample": f"cube of half-width {half:.4f} at the box centre: {sub.n} of {ps.n} particles"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cosmo", choices=list(wl.CONFIG_NAMES))
    ap.add_argument("--n-side", type=int, default=None)
    ap.add_argument("--oracle-particles", type=int, default=262144,
                    help="size of the bounded sample handed to the O(n^2) oracle (262144 particles ~ 10-20 s of CPU work)")
    ap.add_argument("--reference-particles", type=int, default=2097152,
                    help="--impl reference on a lattice-like workload: particles of the window each step evaluates (grid build)")
    ap.add_argument("--cpu-full-limit", type=int, default=20_000_000,
                    help="cpu_baseline runs the oracle on the full workload up to this many particles")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-bruteforce", action="store_true", help="skip the secondary O(n^2) cpu baseline")
    ap.add_argument("--no-next-rows", action="store_true", help="skip the timings of the NEXT rows (they run beside the step)")
    ap.add_argument("--n-h", type=float, default=None,
                    help="NEXT row 4: rescale every support radius to this many particle spacings (paper default 4 = 268 "
                         "neighbours, PAPER.md:336); not the BASELINE workload")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
