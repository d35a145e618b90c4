#!/usr/bin/env python
"""bench.py - AMH sampling rate (MH proposals/s summed over all chains) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

A step = one pass of the whole hot path over one batch: amh_run on a full config of BASELINE.json
(default config 1: L = 128, 1,024 chains, 10,000 sweeps, local:global 10:1, window 8, T = 1) from
the seeded random start.  Inputs are synthetic (amh_inputs) and resident
in HBM when the timed region starts; the e2e leg goes through amh_run_host with pinned host
buffers.  Multi-GPU = chain sharding, no data-path collective: rank r
runs chains [r*B, (r+1)*B), weak scaling.  Rank 0 prints ONE JSON line.

--impl reference times the fp64 CPU oracle (oracle/) as it stands on the host cores, on a bounded
sample of the same workload; it is the only place besides the cpu_baseline leg where this file
executes anything under oracle/.
"""
from __future__ import annotations

import argparse
import json
import os
import re
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import amh_inputs as gi  # noqa: E402

METRIC = "mh_proposals_per_sec"
UNIT = "proposals/s"
LANE_OPS_PER_PAIR = 20          # fp32 lane-ops of one pair evaluation
FP32_LANES_PER_SM = 128


# ------------------------------------------------------------------------------------------------
def pair_counts(L: int, w: int, min_sep: int = 3):
    """Algorithmic pair evaluations per sweep: sum over k of the pairs that straddle
    the flipped bond, for a global and for a local sweep, and the all-pairs count of the sweep-end energy."""
    i = np.arange(L)[:, None]; j = np.arange(L)[None, :]
    sep_ok = (j - i) >= min_sep
    g = l = 0
    for k in range(2 * L):
        c = k // 2
        split = c + (k & 1)
        if k == 0 or k == 2 * L - 1:
            continue
        cross = sep_ok & (i < split) & (j >= split)
        g += int(cross.sum())
        lo, hi = max(0, c - w), min(L - 1, c + w)
        l += int((cross & (i >= lo) & (j <= hi)).sum())
    return g, l, int(sep_ok.sum())


def algorithmic_pair_evals(cfg: gi.Config) -> int:
    g, l, allp = pair_counts(cfg.L, cfg.window)
    cyc = cfg.n_global + cfg.n_local
    full, rem = divmod(cfg.n_sweeps, cyc)
    n_g = full * cfg.n_global + min(rem, cfg.n_global)
    n_l = cfg.n_sweeps - n_g
    return cfg.B * (n_g * g + n_l * l + cfg.n_sweeps * allp)


def run_kwargs(cfg: gi.Config, B: int, chain_offset: int):
    kw = dict(n_global=cfg.n_global, n_local=cfg.n_local, window=cfg.window, seed=1, chain_offset=chain_offset)
    if cfg.replicas:
        kw["per_chain_T"] = gi.per_chain_temperature(B, cfg.replicas, cfg.t_start, cfg.t_end, chain_offset)
    else:
        kw.update(t_start=cfg.t_start, t_end=cfg.t_end, ramp_sweeps=cfg.n_sweeps)
    return kw


def shard(cfg: gi.Config, rank: int, world: int):
    """Chain sharding: rank r runs chains [r B, (r+1) B) of a world*B batch - weak scaling,
    no data-path collective.  Returns (chain_offset, start states, run kwargs) of this rank."""
    off = rank * cfg.B
    return off, gi.initial_states(cfg.B, cfg.n, seed=1, chain_offset=off), run_kwargs(cfg, cfg.B, off)


def job_rate(world: int, proposals_per_rank: int, steps: int, max_total_ms: float) -> float:
    """Whole-job proposals/s: the units all ranks processed / the slowest rank's device time."""
    return world * proposals_per_rank * steps / (max_total_ms * 1e-3)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); power.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return {}


def profiled_traffic(cfg_name: str):
    """dram bytes per launch of the sweep kernel from the committed ncu --set full summary, or None."""
    path = os.path.join(ROOT, "profiles", "traffic.txt")
    try:
        for line in open(path):
            m = re.match(r"\s*%s\s+sweep_kernel\s+dram_bytes_per_launch\s*=\s*([0-9.eE+]+)" % re.escape(cfg_name), line)
            if m:
                return float(m.group(1))
    except OSError:
        pass
    return None


# ------------------------------------------------------------------------------------------------
def oracle_leg(cfg: gi.Config, steps: int = 1, warmup: int = 0, target_s: float = 15.0):
    """The fp64 oracle, as it stands, on the host cores, on a bounded sample of the workload: the first 64 chains
    of the batch for as many whole cycles of the schedule as fit in about `target_s` seconds of wall time per step
    (sized from a two-cycle calibration run; at least two cycles, at most the config's sweep count)."""
    import oracle
    oracle.build()
    ref = gi.reference_torsions(cfg.L, cfg.cfg_seed)
    CB = oracle.coords(ref)[3]
    D = np.linalg.norm(CB[:, None] - CB[None], axis=-1)
    m = oracle.Model(gi.distogram_from_distances(D, n_bins=cfg.n_bins, lo=cfg.d_lo, hi=cfg.d_hi), gi.bin_edges(cfg.n_bins, cfg.d_lo, cfg.d_hi))
    chains = min(cfg.B, 64)
    s0 = gi.initial_states(chains, cfg.n, seed=1)
    kw = run_kwargs(cfg, chains, 0)
    cyc = cfg.n_global + cfg.n_local
    t0 = time.perf_counter()
    m.run(s0, min(cfg.n_sweeps, 2 * cyc), **kw)
    t_cal = (time.perf_counter() - t0) / 2.0
    sweeps = int(min(cfg.n_sweeps, cyc * max(2, int(target_s / max(t_cal, 1e-6)))))
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        m.run(s0, sweeps, **kw)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    props = chains * sweeps * cfg.n
    t = float(np.mean(times))
    return dict(value=props / t, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                sample="%d chains x %d sweeps of %s (%d proposals, %.1f s per step, fp64, full rebuild + full re-sum per proposal)"
                       % (chains, sweeps, cfg.name, props, t)), t


def oracle_threshold(cfg: gi.Config, runs: int = 10, proposals: int = 100000):
    """Energy threshold of the time-to-threshold metric (protocol of PAPER.md:184-188): the oracle
    runs `runs` single chains of `proposals` proposals each under the config's schedule, one core per chain; E* = mean
    of their minimum sweep-end energies, cpu_s = wall time of those runs."""
    import oracle
    oracle.build()
    ref = gi.reference_torsions(cfg.L, cfg.cfg_seed)
    CB = oracle.coords(ref)[3]
    D = np.linalg.norm(CB[:, None] - CB[None], axis=-1)
    m = oracle.Model(gi.distogram_from_distances(D, n_bins=cfg.n_bins, lo=cfg.d_lo, hi=cfg.d_hi), gi.bin_edges(cfg.n_bins, cfg.d_lo, cfg.d_hi))
    sweeps = max(1, -(-proposals // cfg.n))
    s0 = gi.initial_states(runs, cfg.n, seed=1)
    t0 = time.perf_counter()
    r = m.run(s0, sweeps, **run_kwargs(cfg, runs, 0))
    dt = time.perf_counter() - t0
    return dict(threshold=float(np.mean(r["best_energy"])), cpu_s=dt, cpu_runs=runs, cpu_sweeps_per_run=sweeps,
                cpu_cores=min(runs, oracle.num_threads()))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, choices=sorted(gi.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--sweeps", type=int, default=0, help="override the config's sweep count (experiments only; the line says so)")
    ap.add_argument("--chains", type=int, default=0, help="override the config's chain count (experiments only)")
    ap.add_argument("--warps-per-chain", type=int, default=0)
    ap.add_argument("--chains-per-cta", type=int, default=0)
    ap.add_argument("--spec-local", type=int, default=0)
    ap.add_argument("--ring-cols", type=int, default=0)
    ap.add_argument("--lanes-per-step", type=int, default=0)
    ap.add_argument("--spec-global", type=int, default=-1)
    ap.add_argument("--exchange", action="store_true", help="configs with temperature replicas: amh_run_pt (replica exchange after every cycle, NEXT-3) instead of amh_run; the line says so")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = gi.CONFIGS[args.config]
    overridden = bool(args.sweeps or args.chains)
    if overridden:
        import dataclasses
        cfg = dataclasses.replace(cfg, n_sweeps=args.sweeps or cfg.n_sweeps, B=args.chains or cfg.B)
    workload = dict(workload=cfg.name + ("-override" if overridden else ""), L=cfg.L, chains_per_gpu=cfg.B, sweeps=cfg.n_sweeps,
                    schedule="%d global : %d local" % (cfg.n_global, cfg.n_local), window=cfg.window,
                    temperature=("per-chain %g..%g x%d" % (cfg.t_start, cfg.t_end, cfg.replicas)) if cfg.replicas
                    else ("%g -> %g geometric" % (cfg.t_start, cfg.t_end) if cfg.t_start != cfg.t_end else "%g" % cfg.t_start),
                    n_bins=cfg.n_bins, proposal="uniform", parallelism="chains sharded x%d" % world)

    # ---------------- reference arm: the oracle on the host cores --------------------------------
    if args.impl == "reference":
        if rank != 0:
            return
        cb, t = oracle_leg(cfg, steps=max(1, args.steps), warmup=min(args.warmup, 1))
        line = dict(impl="reference", metric=METRIC, value=cb["value"], unit=UNIT, n_gpus=0, steps=args.steps,
                    warmup=args.warmup, ms_per_step=t * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="f64", data="synthetic", config=workload, cpu_baseline=cb,
                    e2e=dict(value=cb["value"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0))
        print(json.dumps(line))
        return

    # ---------------- our arm --------------------------------------------------------------------
    import torch
    import paper_2211_03193_b200 as pkg
    pkg.lib()                                   # fails loudly without the CUDA extension
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    L, B, n = cfg.L, cfg.B, cfg.n
    edges = gi.bin_edges(cfg.n_bins, cfg.d_lo, cfg.d_hi)
    # reference geometry from the CUDA path itself (a throw-away context with a flat table)
    g0 = pkg.AMH(np.full((L, L, cfg.n_bins), 1.0 / cfg.n_bins, np.float32), edges)
    ref = gi.reference_torsions(L, cfg.cfg_seed)
    cb = g0.coords(torch.from_numpy(ref[None]).cuda())[0].double().cpu().numpy()
    g0.close()
    D = np.linalg.norm(cb[:, None] - cb[None], axis=-1)
    p = gi.distogram_from_distances(D, n_bins=cfg.n_bins, lo=cfg.d_lo, hi=cfg.d_hi)
    g = pkg.AMH(p, edges, pkg.default_options(warps_per_chain=args.warps_per_chain, chains_per_cta=args.chains_per_cta,
                                               spec_local=args.spec_local, ring_cols=args.ring_cols,
                                               lanes_per_step=args.lanes_per_step, spec_global=args.spec_global))
    del p
    chain_offset, s0_np, kw = shard(cfg, rank, world)
    s0_host = torch.from_numpy(s0_np).pin_memory()
    s0_dev = s0_host.cuda()
    states = torch.empty_like(s0_dev)
    if "per_chain_T" in kw:
        kw["per_chain_T"] = torch.from_numpy(kw["per_chain_T"]).cuda()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2
    stream = torch.cuda.current_stream()
    info = g.launch_info(B, cfg.window)

    exchange = bool(args.exchange and cfg.replicas)
    tts = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not exchange:
        tts = oracle_threshold(cfg)
        kw["energy_threshold"] = tts["threshold"]

    if exchange:
        args.no_e2e = True                                   # the exchange run is an experiment line: device-timed rate only
        # replica exchange: one amh_run per cycle + amh_exchange, enqueued by amh_run_pt; temperatures reset every step
        T0 = kw.pop("per_chain_T")
        Tcur = T0.clone()
        ptkw = dict(n_global=cfg.n_global, n_local=cfg.n_local, window=cfg.window, seed=kw["seed"], chain_offset=chain_offset)
        n_cycles = cfg.n_sweeps // (cfg.n_global + cfg.n_local)
        workload["exchange"] = "amh_run_pt: %d cycles, exchange after each, groups of %d" % (n_cycles, cfg.replicas)

    def run_step():
        if exchange:
            Tcur.copy_(T0)
            return g.run_pt(states, n_cycles, Tcur, cfg.replicas, **ptkw)
        return g.run(states, cfg.n_sweeps, want=("energy", "best_energy"), **kw)

    def one_step():
        states.copy_(s0_dev)
        return run_step()

    for _ in range(args.warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    launches = 0
    res = None
    for a, b in ev:
        flush.fill_(1)                                  # L2 flush between timed iterations (outside the events)
        states.copy_(s0_dev)
        a.record(stream)
        res = run_step()
        b.record(stream)
        launches += (2 * n_cycles) if exchange else 1
    barrier()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    clocks = sampler.stop() if sampler else None
    tmax = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
    total_ms = float(tmax.item())
    ms_per_step = total_ms / args.steps
    props_per_step = world * cfg.proposals
    value = job_rate(world, cfg.proposals, args.steps, total_ms)
    best = float(res["best_energy"].min().item()) if res is not None else None
    if tts is not None:
        hit = int(res["first_hit_sweep"].item())
        tts.update(first_hit_sweep=hit, gpu_s=(ms_per_step * 1e-3 * (hit + 1) / cfg.n_sweeps) if hit >= 0 else None,
                   protocol="E* = mean over 10 oracle chains (100,000 proposals each, this config's schedule) of the minimum "
                            "sweep-end energy; gpu_s = step time x (first sweep at whose end some chain of the batch has V <= E*, "
                            "+ 1) / sweeps; cpu_s = wall time of the oracle runs, one core per chain")
        # nine more seeds (PAPER.md:184-188 takes means over repeated runs; median over 10 seeds),
        # each run only long enough to see its hit
        hits = [hit]
        if hit >= 0:
            short = int(min(cfg.n_sweeps, 8 * (hit + 1) + 4 * (cfg.n_global + cfg.n_local)))
            for seed in range(2, 11):
                states.copy_(torch.from_numpy(gi.initial_states(B, n, seed=seed, chain_offset=chain_offset)).cuda())
                rr = g.run(states, short, want=("energy",), **dict(kw, seed=seed))
                hits.append(int(rr["first_hit_sweep"].item()))
            ok = sorted(h for h in hits if h >= 0)
            med = ok[len(ok) // 2] if len(ok) == len(hits) else None
            tts.update(first_hit_sweeps_10_seeds=hits, gpu_s_median=(ms_per_step * 1e-3 * (med + 1) / cfg.n_sweeps) if med is not None else None)
        tts["speedup_vs_oracle"] = (tts["cpu_s"] / tts["gpu_s"]) if tts["gpu_s"] else None
        kw.pop("energy_threshold")

    # ---------------- global-only and local-only rates, short runs from the final states ----------
    phase_rates = None
    if rank == 0 and world == 1 and not exchange:
        phase_rates = {}
        cyc = cfg.n_global + cfg.n_local
        for name, (ng, nl, sw) in (("global_only", (1, 0, max(2, 2 * cfg.n_global))), ("local_only", (0, 1, max(10, 2 * cfg.n_local)))):
            pk = dict(kw, n_global=ng, n_local=nl, sweep_offset=cfg.n_sweeps)
            tmp = states.clone()
            g.run(tmp, 1, want=("energy",), **pk)
            a2, b2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a2.record(stream); g.run(tmp, sw, want=("energy",), **pk); b2.record(stream)
            torch.cuda.synchronize()
            phase_rates[name] = dict(value=B * sw * n / (a2.elapsed_time(b2) * 1e-3), unit=UNIT, sweeps=sw,
                                     ms_per_sweep=a2.elapsed_time(b2) / sw)

    # ---------------- e2e: the same step through amh_run_host, pinned host buffers ----------------
    e2e = None
    if not args.no_e2e:
        hs = torch.empty_like(s0_host).pin_memory()
        hkw = dict(kw)
        if "per_chain_T" in hkw:
            hkw["per_chain_T"] = hkw["per_chain_T"].cpu().numpy()
        hs.copy_(s0_host); g.run_host(hs.numpy(), cfg.n_sweeps, **hkw)         # warm-up (staging arena)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            hs.copy_(s0_host)
            rh = g.run_host(hs.numpy(), cfg.n_sweeps, **hkw)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        te = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if dist is not None:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        h2d = B * n * 4 + (B * 4 if cfg.replicas else 0)
        d2h = B * n * 4 + 2 * B * 4
        e2e = dict(value=props_per_step * args.steps / float(te.item()), unit=UNIT, h2d_bytes_per_step=h2d,
                   d2h_bytes_per_step=d2h, api="amh_run_host (pinned host buffers; copies inside the timed region)",
                   best_energy=float(rh["best_energy"].min()))

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---------------- roofline of the dominant kernel (sweep_kernel, one launch per step) ---------
    peaks = measured_peaks()
    sm_max_mhz = (clocks or {}).get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
    peak = info["n_sm"] * FP32_LANES_PER_SM * sm_max_mhz * 1e6 / 1e9          # Glane-op/s
    pair_evals = algorithmic_pair_evals(cfg)
    achieved = pair_evals * LANE_OPS_PER_PAIR / (ms_per_step * 1e-3) / 1e9
    roofline = dict(bound="alu", achieved=achieved, peak=peak, unit="Glane-op/s", frac=achieved / peak,
                    traffic=profiled_traffic(cfg.name), kernel="amh::sweep_kernel<SG, RING> (one of four variants, chosen per launch)",
                    pair_evals_per_launch=pair_evals, lane_ops_per_pair_eval=LANE_OPS_PER_PAIR,
                    pair_evals_per_s=pair_evals / (ms_per_step * 1e-3),
                    peak_source="derived: %d SMs x 128 fp32 lanes x %.0f MHz (clocks.max.sm)" % (info["n_sm"], sm_max_mhz),
                    hbm_gbs_measured=peaks.get("hbm_gbs"))
    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline, _ = oracle_leg(cfg)

    workload.update(l2="flushed between timed steps (256 MiB write)", threads_per_chain=info["threads_per_chain"],
                    chains_per_cta=info["chains_per_cta"], ring_cols=info["ring_cols"], ring_rows=info["ring_rows"],
                    smem_bytes_per_cta=info["smem_bytes"], ctas_resident_per_sm=info["ctas_per_sm"],
                    step="amh_run over the full config from the seeded random start", best_energy=best)
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32",
                data="synthetic", config=workload, clocks=clocks, e2e=e2e, gpu_launches=launches,
                roofline=roofline, cpu_baseline=cpu_baseline, time_to_threshold=tts, phase_rates=phase_rates)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
