#!/usr/bin/env python
"""bench.py - AMH sampling rate (MH proposals/s summed over all chains) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference] [--per-config full|slice|off]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 \
        --master-port P bench.py --gpus N --steps K --warmup W

A step = one pass of the whole hot path over one batch: amh_run on a full config of BASELINE.json
(default config 1: L = 128, 1,024 chains, 10,000 sweeps, local:global 10:1, window 8, T = 1) from
the seeded random start.  Inputs are synthetic (amh_inputs) and resident
in HBM when the timed region starts; the e2e leg goes through amh_run_host with pinned host
buffers.  Multi-GPU = chain sharding, no data-path collective: rank r
runs chains [r*B, (r+1)*B), weak scaling; `--gpus N` without a launcher environment starts the N
ranks itself (torch.distributed.run on 127.0.0.1).  Rank 0 prints ONE JSON line.  At N = 1 the line
also carries `per_config`: every other config of BASELINE.json, one timed step each.

--impl reference times the fp64 CPU oracle (oracle/) as it stands on the host cores, on a bounded
sample of the same workload; it is the only place besides the cpu_baseline legs where this file
executes anything under oracle/.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import re
import socket
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
# Thread instructions of ONE pair evaluation in the built kernel (cuobjdump -sass of sweep_kernel<1,1,1>, the body of
# local_new_sum; profiles/r2_sass_pair_eval.md): 9 FADD + 3 FMNMX + 2 FSEL + 1 FMUL + 4 FFMA + 1 MUFU.SQRT + 4 integer
# (SHL, LOP3, IADD3, IADD) + 4 shared-memory loads (2 LDS.128 points, 2 LDS table entries) = 28.  (SURVEY.md 8(d) estimated 20.)
LANE_OPS_PER_PAIR = 28
LANE_OPS_BY_PIPE = {"fadd_fmnmx_fsel": 14, "ffma_fmul": 5, "mufu": 1, "int": 4, "lds": 4}
LANE_OPS_DISTANCE = 8           # of those, what a pair beyond the last bin centre needs: 1 load, 3 FADD, 1 FMUL, 2 FFMA, 1 compare
# config 3 (fp64): arithmetic of one six-term pair counted from the formulas of R25, one op per add / multiply / fma, a root at 9
# (reciprocal-root seed + Newton steps), atan2 at 45 (one division at 10, a degree-19 odd polynomial, octant fix-ups), an
# interpolation at 8: distance 15 + 8; three dihedrals 3 x (9 + 12 + 9 + 9 + 1 + 45); two angles 2 x (6 + 6 + 6 + 9 + 45);
# five more interpolations 40  = 462 -> 460.  (ncu counts 414 executed DADD + DMUL + DFMA per algorithmic pair:
# profiles/r2_ncu_per_config.md.)
LANE_OPS_PER_PAIR_TR5 = 460
FP32_LANES_PER_SM = 128
FP64_LANES_PER_SM = 64


# ------------------------------------------------------------------------------------------------
def pair_counts(L: int, w: int, min_sep: int = 3, slots: int = 2):
    """Algorithmic pair evaluations per sweep: sum over k of the pairs that straddle
    the flipped bond, for a global and for a local sweep, and the all-pairs count of the sweep-end energy."""
    i = np.arange(L)[:, None]; j = np.arange(L)[None, :]
    sep_ok = (j - i) >= min_sep
    g = l = 0
    for k in range(slots * L):
        c, slot = divmod(k, slots)
        if slots == 2:
            split = c + slot
            if k == 0 or k == 2 * L - 1:
                continue
        else:
            if slot >= 3:
                continue
            split = c + (1 if slot > 0 else 0)
            if split <= 0 or split >= L:
                continue
        cross = sep_ok & (i < split) & (j >= split)
        g += int(cross.sum())
        lo, hi = max(0, c - w), min(L - 1, c + w)
        l += int((cross & (i >= lo) & (j <= hi)).sum())
    return g, l, int(sep_ok.sum())


def algorithmic_pair_evals(cfg: gi.Config) -> int:
    g, l, allp = pair_counts(cfg.L, cfg.window, slots=cfg.slots)
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


def start_states(cfg: gi.Config, B: int, seed: int, chain_offset: int = 0) -> np.ndarray:
    if cfg.slots == 5:
        return gi.initial_states_tr5(B, cfg.L, seed, chain_offset)
    return gi.initial_states(B, cfg.n, seed=seed, chain_offset=chain_offset)


def shard(cfg: gi.Config, rank: int, world: int):
    """Chain sharding: rank r runs chains [r B, (r+1) B) of a world*B batch - weak scaling,
    no data-path collective.  Returns (chain_offset, start states, run kwargs) of this rank."""
    off = rank * cfg.B
    return off, start_states(cfg, cfg.B, 1, off), run_kwargs(cfg, cfg.B, off)


def job_rate(world: int, proposals_per_rank: int, steps: int, max_total_ms: float) -> float:
    """Whole-job proposals/s: the units all ranks processed / the slowest rank's device time."""
    return world * proposals_per_rank * steps / (max_total_ms * 1e-3)


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def spawn_ranks(n: int, argv) -> int:
    """`bench.py --gpus N` without a launcher environment: start the N ranks on this node (one per GPU) with
    torch.distributed.run on 127.0.0.1 and return its exit code."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n),
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + list(argv)
    env = dict(os.environ, NCCL_DEBUG=os.environ.get("NCCL_DEBUG", "INFO"), NCCL_DEBUG_SUBSYS=os.environ.get("NCCL_DEBUG_SUBSYS", "INIT"))
    return subprocess.call(cmd, env=env)


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


def profiled_per_proposal(cfg_name: str, key: str):
    """a figure of the sweep kernel from the committed ncu --set full summaries (profiles/r2_traffic.txt:
    `<cfg> <key> = <value>`), or None.  key = dram_bytes_fixed | dram_bytes_per_proposal | l2_bytes_per_proposal |
    thread_inst_per_proposal."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.txt")
    try:
        for line in open(path):
            m = re.match(r"\s*%s\s+%s\s*=\s*([0-9.eE+-]+)" % (re.escape(cfg_name), re.escape(key)), line)
            if m:
                return float(m.group(1))
    except OSError:
        pass
    return None


# ------------------------------------------------------------------------------------------------
def oracle_model(cfg: gi.Config):
    """The config's energy model in the oracle, from the oracle's own reference geometry."""
    import oracle
    oracle.build()
    edges = gi.bin_edges(cfg.n_bins, cfg.d_lo, cfg.d_hi)
    if cfg.slots == 5:
        ref = gi.reference_torsions_tr5(cfg.L, cfg.cfg_seed)
        D, OM, TH, PH = oracle.tr5_pair_geometry(ref)
        return oracle.TR5Model(gi.distogram_from_distances(D, n_bins=cfg.n_bins, lo=cfg.d_lo, hi=cfg.d_hi), edges,
                               gi.periodic_map_from_values(OM, 24, -math.pi, math.pi, True),
                               gi.periodic_map_from_values(TH, 24, -math.pi, math.pi, True),
                               gi.periodic_map_from_values(PH, 12, 0.0, math.pi, False))
    ref = gi.reference_torsions(cfg.L, cfg.cfg_seed)
    CB = oracle.coords(ref)[3]
    D = np.linalg.norm(CB[:, None] - CB[None], axis=-1)
    return oracle.Model(gi.distogram_from_distances(D, n_bins=cfg.n_bins, lo=cfg.d_lo, hi=cfg.d_hi), edges)


def oracle_leg(cfg: gi.Config, steps: int = 1, warmup: int = 0, target_s: float = 15.0, max_chains: int = 64):
    """The fp64 oracle, as it stands, on the host cores, on a bounded sample of the workload: the first chains
    of the batch for as many whole cycles of the schedule as fit in about `target_s` seconds of wall time per step
    (sized from a calibration run; at least one cycle, at most the config's sweep count)."""
    import oracle
    m = oracle_model(cfg)
    chains = min(cfg.B, max_chains)
    s0 = start_states(cfg, chains, 1)
    kw = run_kwargs(cfg, chains, 0)
    cyc = cfg.n_global + cfg.n_local
    ncal = 1 if cfg.L > 256 or cfg.slots == 5 else 2
    if cfg.L > 256 or cfg.slots == 5:
        chains = min(chains, max(oracle.num_threads(), 1)); s0 = s0[:chains]; kw = run_kwargs(cfg, chains, 0)
    t0 = time.perf_counter()
    m.run(s0, min(cfg.n_sweeps, ncal * cyc), **kw)
    t_cal = (time.perf_counter() - t0) / ncal
    sweeps = int(min(cfg.n_sweeps, cyc * max(1, int(target_s / max(t_cal, 1e-6)))))
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
    m = oracle_model(cfg)
    sweeps = max(1, -(-proposals // cfg.n))
    s0 = start_states(cfg, runs, 1)
    t0 = time.perf_counter()
    r = m.run(s0, sweeps, **run_kwargs(cfg, runs, 0))
    dt = time.perf_counter() - t0
    return dict(threshold=float(np.mean(r["best_energy"])), cpu_s=dt, cpu_runs=runs, cpu_sweeps_per_run=sweeps,
                cpu_cores=min(runs, oracle.num_threads()))


# ------------------------------------------------------------------------------------------------
class Workload:
    """One config on the CUDA path: context (tables built from the CUDA path's own reference geometry), start states."""

    def __init__(self, pkg, torch, cfg: gi.Config, rank: int, world: int, launch_over=None):
        self.pkg, self.torch, self.cfg = pkg, torch, cfg
        L = cfg.L
        edges = gi.bin_edges(cfg.n_bins, cfg.d_lo, cfg.d_hi)
        opts = pkg.default_options(**launch_over) if launch_over else None
        if cfg.slots == 5:
            ref = gi.reference_torsions_tr5(L, cfg.cfg_seed)
            flat = [np.full((L, L, nb), 1.0 / nb, np.float32) for nb in (cfg.n_bins, 24, 24, 12)]
            g0 = pkg.AMH(flat[0], edges, orientation=flat[1:])
            D, OM, TH, PH = [x[0].cpu().numpy() for x in g0.pair_geometry(torch.from_numpy(ref[None]).cuda())]
            g0.close()
            self.g = pkg.AMH(gi.distogram_from_distances(D, n_bins=cfg.n_bins, lo=cfg.d_lo, hi=cfg.d_hi), edges, opts,
                             orientation=(gi.periodic_map_from_values(OM, 24, -math.pi, math.pi, True),
                                          gi.periodic_map_from_values(TH, 24, -math.pi, math.pi, True),
                                          gi.periodic_map_from_values(PH, 12, 0.0, math.pi, False)))
        else:
            # reference geometry from the CUDA path itself (a throw-away context with a flat table)
            g0 = pkg.AMH(np.full((L, L, cfg.n_bins), 1.0 / cfg.n_bins, np.float32), edges)
            ref = gi.reference_torsions(L, cfg.cfg_seed)
            cb = g0.coords(torch.from_numpy(ref[None]).cuda())[0].double().cpu().numpy()
            g0.close()
            D = np.linalg.norm(cb[:, None] - cb[None], axis=-1)
            self.g = pkg.AMH(gi.distogram_from_distances(D, n_bins=cfg.n_bins, lo=cfg.d_lo, hi=cfg.d_hi), edges, opts)
        self.chain_offset, s0_np, self.kw = shard(cfg, rank, world)
        self.s0_host = torch.from_numpy(s0_np).pin_memory()
        self.s0_dev = self.s0_host.cuda()
        self.states = torch.empty_like(self.s0_dev)
        if "per_chain_T" in self.kw:
            self.kw["per_chain_T"] = torch.from_numpy(self.kw["per_chain_T"]).cuda()
        self.info = self.g.launch_info(cfg.B, cfg.window)

    def kernel_label(self) -> str:
        i = self.info
        if self.cfg.slots == 5:
            return "amh::tr5_sweep_kernel (fp64, one CTA of %d threads per chain)" % i["threads_per_chain"]
        return ("amh::sweep_kernel<SG=%d, RING=%d, CB64=%d>: %d chains x %d warps per CTA, %d local proposals per pass, %d lanes each"
                % (i["spec_global"], i["ring"], i["cb64"], i["chains_per_cta"], i["warps_per_chain"], i["nspec"], i["lanes_per_step"]))

    def launch_dict(self) -> dict:
        i = self.info
        return dict(kernel=self.kernel_label(), threads_per_chain=i["threads_per_chain"], chains_per_cta=i["chains_per_cta"],
                    ring_cols=i["ring_cols"], ring_rows=i["ring_rows"], smem_bytes_per_cta=i["smem_bytes"],
                    ctas_resident_per_sm=i["ctas_per_sm"])

    def run(self, sweeps=None, want=("energy", "best_energy"), **over):
        return self.g.run(self.states, self.cfg.n_sweeps if sweeps is None else sweeps, want=want, **dict(self.kw, **over))

    def reset(self):
        self.states.copy_(self.s0_dev)

    def near_fraction(self, states) -> float:
        """fraction of the pairs j - i >= 3 of (a sample of) these states that lie below the last bin centre, i.e. that need
        more than their distance (measured with torch on the C-betas amh_coords returns; reporting only)"""
        torch, cfg = self.torch, self.cfg
        pick = states[:: max(1, states.shape[0] // 64)][:64]
        cb = self.g.coords(pick).double()
        d = torch.cdist(cb, cb)
        i = torch.arange(cfg.L, device=d.device)
        mask = (i[None, :] - i[:, None]) >= 3
        c_last = cfg.d_hi - 0.5 * (cfg.d_hi - cfg.d_lo) / cfg.n_bins
        return float(((d < c_last) & mask[None]).sum().item()) / float(mask.sum().item() * d.shape[0])

    def roofline(self, ms_per_step: float, n_sm: int, sm_max_mhz: float, peaks: dict, l2_peak_gbs, gather_peak) -> dict:
        cfg = self.cfg
        pair_evals = algorithmic_pair_evals(cfg)
        fp64 = cfg.slots == 5
        ops = LANE_OPS_PER_PAIR_TR5 if fp64 else LANE_OPS_PER_PAIR
        lanes = FP64_LANES_PER_SM if fp64 else FP32_LANES_PER_SM
        peak = n_sm * lanes * sm_max_mhz * 1e6 / 1e9          # Glane-op/s
        achieved = pair_evals * ops / (ms_per_step * 1e-3) / 1e9
        dram_f = profiled_per_proposal(cfg.name, "dram_bytes_fixed")
        dram_p = profiled_per_proposal(cfg.name, "dram_bytes_per_proposal")
        dram = None if dram_f is None else dram_f + (dram_p or 0.0) * cfg.proposals
        l2b = profiled_per_proposal(cfg.name, "l2_bytes_per_proposal")
        r = dict(bound="alu", achieved=achieved, peak=peak, unit="Glane-op/s", frac=achieved / peak,
                 traffic=dram,
                 traffic_source="dram__bytes_read + dram__bytes_write of the ncu --set full capture of this config's kernel (profiles/r2_traffic.txt): "
                                "a fixed first touch of the tables where they stay in L2, bytes per proposal x proposals where they do not (configs 3, 4)",
                 kernel=self.kernel_label(), pair_evals_per_launch=pair_evals, lane_ops_per_pair_eval=ops,
                 lane_ops_by_pipe=None if fp64 else LANE_OPS_BY_PIPE, pair_evals_per_s=pair_evals / (ms_per_step * 1e-3),
                 peak_source="derived: %d SMs x %d %s lanes x %.0f MHz (clocks.max.sm)" % (n_sm, lanes, "fp64" if fp64 else "fp32", sm_max_mhz),
                 hbm_gbs_measured=peaks.get("hbm_gbs"))
        if not fp64:
            # `frac` charges a pair the arithmetic it needs: every pair its distance (8 lane-ops); only a near pair - and every
            # in-window pair of a local proposal, where no far test is made - the other 20.  near fraction = the smaller of the
            # start and the final states' (the states in between are at least as compact as the random start).  The all-pairs
            # count of SURVEY.md 8(d) (every straddling pair at the full 28) is kept beside it: it charges the kernel work it
            # skips exactly, and passes 1 where most pairs are far (config 4).
            f = min(self.near_fraction(self.s0_dev), self.near_fraction(self.states))
            gsum, lsum, allp = pair_counts(cfg.L, cfg.window, slots=cfg.slots)
            cyc = cfg.n_global + cfg.n_local
            full, rem = divmod(cfg.n_sweeps, cyc)
            n_g = full * cfg.n_global + min(rem, cfg.n_global)
            n_l = cfg.n_sweeps - n_g
            per_global_pair = LANE_OPS_DISTANCE + f * (LANE_OPS_PER_PAIR - LANE_OPS_DISTANCE)
            ops_w = cfg.B * (n_l * lsum * LANE_OPS_PER_PAIR + (n_g * gsum + cfg.n_sweeps * allp) * per_global_pair)
            per_s = 1.0 / (ms_per_step * 1e-3) / 1e9
            r["achieved_all_pairs"], r["frac_all_pairs"] = r["achieved"], r["frac"]
            r["frac_all_pairs_without_sweep_end_energy"] = cfg.B * (n_g * gsum + n_l * lsum) * LANE_OPS_PER_PAIR * per_s / peak
            r["achieved"] = ops_w * per_s
            r["frac"] = r["achieved"] / peak
            r["frac_without_sweep_end_energy"] = cfg.B * (n_l * lsum * LANE_OPS_PER_PAIR + n_g * gsum * per_global_pair) * per_s / peak
            r["near_fraction"] = f
            r["note"] = ("achieved / frac charge a pair beyond the last bin centre only its distance test (%d lane-ops; its term is exactly 0 and "
                         "the kernel skips it) and every other pair the %d lane-ops of a full evaluation; *_all_pairs charge EVERY straddling "
                         "pair the full %d (SURVEY.md 8(d)'s unit) and can exceed 1 where most pairs are far (config 4); "
                         "*_without_sweep_end_energy leave out the all-pairs energy of every sweep end (a9), which 8(d)'s pairs/proposal "
                         "column does not contain." % (LANE_OPS_DISTANCE, LANE_OPS_PER_PAIR, LANE_OPS_PER_PAIR))
            # a batch with fewer CTAs than SMs (config 0: 32 chains) cannot occupy the chip: the same figure against the SMs it can
            ctas = -(-cfg.B // max(1, self.info["chains_per_cta"]))
            if ctas < n_sm:
                r["occupied_sms"] = ctas
                r["frac_of_occupied_sms"] = r["frac"] * n_sm / ctas
                r["frac_all_pairs_of_occupied_sms"] = r["frac_all_pairs"] * n_sm / ctas
        if r["frac"] is not None and r["frac"] > 1.0:          # a fraction above 1 is a counting error, not a result
            r["frac_rejected"], r["frac"] = r["frac"], None
        ipp = profiled_per_proposal(cfg.name, "thread_inst_per_proposal")
        if ipp is not None:
            r["executed_thread_inst_per_algorithmic_pair"] = ipp * cfg.proposals / pair_evals
        if l2_peak_gbs:
            a = (l2b * cfg.proposals / (ms_per_step * 1e-3) / 1e9) if l2b is not None else None
            r["l2"] = dict(achieved=a, peak=l2_peak_gbs, unit="GB/s", frac=(a / l2_peak_gbs) if a is not None else None,
                           peak_source="amh_probe_l2_read measured in this run: read-only sweep of a %d MB buffer by every SM, L1 bypassed"
                                       % (48 if cfg.L < 512 else 92),
                           achieved_source="lts__t_bytes per proposal of the ncu capture (profiles/r2_traffic.txt) x proposals / this run's time")
        if gather_peak:
            r["gather_ceiling"] = dict(peak=gather_peak, unit="8-byte gathers/s",
                                       note="amh_probe_gather measured in this run: the near-pair look-ups of the global phase cannot exceed it")
        return r


def time_steps(torch, wl: Workload, steps: int, warmup: int, flush, stream, barrier, run_step):
    for _ in range(warmup):
        wl.reset(); run_step()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    res = None
    for a, b in ev:
        flush.fill_(1)                                  # L2 flush between timed iterations (outside the events)
        wl.reset()
        a.record(stream)
        res = run_step()
        b.record(stream)
    barrier()
    return sum(a.elapsed_time(b) for a, b in ev), res


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, choices=sorted(gi.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--per-config", default="full", choices=["full", "slice", "off"],
                    help="N = 1 only: after the headline, one timed step of every other config (full = the whole config; slice = a few cycles)")
    ap.add_argument("--sweeps", type=int, default=0, help="override the config's sweep count (experiments only; the line says so)")
    ap.add_argument("--chains", type=int, default=0, help="override the config's chain count (experiments only)")
    ap.add_argument("--warps-per-chain", type=int, default=0)
    ap.add_argument("--chains-per-cta", type=int, default=0)
    ap.add_argument("--spec-local", type=int, default=0)
    ap.add_argument("--ring-cols", type=int, default=0)
    ap.add_argument("--lanes-per-step", type=int, default=0)
    ap.add_argument("--spec-global", type=int, default=-1)
    ap.add_argument("--local-stride", type=int, default=0, help="NEXT-4 variant: strided order of the local sweeps (experiments only; the line says so; not Alg. 1's trajectories)")
    ap.add_argument("--exchange", action="store_true", help="configs with temperature replicas: amh_run_pt (replica exchange after every cycle, NEXT-3) instead of amh_run; the line says so")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--dry-run", action="store_true", help="launcher / sharding check without a GPU: gloo, no kernels, the line reports the shards")
    args = ap.parse_args()

    # `--gpus N` without a launcher environment: start the N ranks ourselves
    if "WORLD_SIZE" not in os.environ and args.gpus > 1 and args.impl == "ours":
        sys.exit(spawn_ranks(args.gpus, sys.argv[1:]))

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = gi.CONFIGS[args.config]
    overridden = bool(args.sweeps or args.chains or args.local_stride)
    if overridden:
        import dataclasses
        cfg = dataclasses.replace(cfg, n_sweeps=args.sweeps or cfg.n_sweeps, B=args.chains or cfg.B)

    def workload_dict(c: gi.Config, over=False):
        return dict(workload=c.name + ("-override" if over else ""), L=c.L, chains_per_gpu=c.B, sweeps=c.n_sweeps,
                    variables_per_chain=c.n, schedule="%d global : %d local" % (c.n_global, c.n_local), window=c.window,
                    temperature=("per-chain %g..%g x%d" % (c.t_start, c.t_end, c.replicas)) if c.replicas
                    else ("%g -> %g geometric" % (c.t_start, c.t_end) if c.t_start != c.t_end else "%g" % c.t_start),
                    n_bins=c.n_bins, proposal="uniform", parallelism="chains sharded x%d" % world,
                    l2="flushed between timed steps (256 MiB write)",
                    step="amh_run over the full config from the seeded random start")
    workload = workload_dict(cfg, overridden)

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

    # ---------------- launcher / sharding check without a GPU ------------------------------------
    if args.dry_run:
        import torch
        import torch.distributed as dist
        if world > 1:
            dist.init_process_group("gloo")
        off, s0, kw = shard(cfg, rank, world)
        mine = torch.tensor([rank, off, off + cfg.B, int(np.float64(s0.sum()) * 1000) % 1000003], dtype=torch.int64)
        allr = [torch.zeros_like(mine) for _ in range(world)]
        if world > 1:
            dist.all_gather(allr, mine)
        else:
            allr = [mine]
        tmax = torch.tensor([1.0 + rank], dtype=torch.float64)
        if world > 1:
            dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        if rank == 0:
            print(json.dumps(dict(metric=METRIC, dry_run=True, n_gpus=len(allr), value=job_rate(world, cfg.proposals, 1, float(tmax.item())),
                                  shards=[[int(x) for x in r] for r in allr], config=workload)))
        if world > 1:
            dist.destroy_process_group()
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

    launch_over = dict(warps_per_chain=args.warps_per_chain, chains_per_cta=args.chains_per_cta, spec_local=args.spec_local,
                       ring_cols=args.ring_cols, lanes_per_step=args.lanes_per_step, spec_global=args.spec_global)
    wl = Workload(pkg, torch, cfg, rank, world, launch_over)
    if args.local_stride:
        wl.kw["local_stride"] = args.local_stride
        workload["order"] = "NEXT-4 variant: strided local sweeps, stride %d (not Alg. 1's order)" % args.local_stride
    g, kw, states, B, n = wl.g, wl.kw, wl.states, cfg.B, cfg.n
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2
    stream = torch.cuda.current_stream()
    info = wl.info

    exchange = bool(args.exchange and cfg.replicas)
    tts = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not exchange:
        tts = oracle_threshold(cfg) if cfg.slots == 2 and cfg.L <= 256 else None
        if tts is not None:
            kw["energy_threshold"] = tts["threshold"]

    if exchange:
        args.no_e2e = True                                   # the exchange run is an experiment line: device-timed rate only
        # replica exchange: one amh_run per cycle + amh_exchange, enqueued by amh_run_pt; temperatures reset every step
        T0 = kw.pop("per_chain_T")
        Tcur = T0.clone()
        ptkw = dict(n_global=cfg.n_global, n_local=cfg.n_local, window=cfg.window, seed=kw["seed"], chain_offset=wl.chain_offset)
        n_cycles = cfg.n_sweeps // (cfg.n_global + cfg.n_local)
        workload["exchange"] = "amh_run_pt: %d cycles, exchange after each, groups of %d" % (n_cycles, cfg.replicas)

    def run_step():
        if exchange:
            Tcur.copy_(T0)
            return g.run_pt(states, n_cycles, Tcur, cfg.replicas, **ptkw)
        return wl.run()

    sampler = ClockSampler(local_rank) if rank == 0 else None
    total_ms, res = time_steps(torch, wl, args.steps, args.warmup, flush, stream, barrier, run_step)
    launches = args.steps * ((2 * n_cycles) if exchange else 1)
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
        kw.pop("energy_threshold")

        def timed_to(sweeps, seed):
            """device time of an amh_run of `sweeps` sweeps from the seeded start (the time to reach the threshold, measured)"""
            s = wl.s0_dev if seed == 1 else torch.from_numpy(start_states(cfg, B, seed, wl.chain_offset)).cuda()
            states.copy_(s)
            a2, b2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a2.record(stream)
            rr = g.run(states, sweeps, want=("energy",), **dict(kw, seed=seed, energy_threshold=tts["threshold"]))
            b2.record(stream)
            torch.cuda.synchronize()
            return a2.elapsed_time(b2) * 1e-3, int(rr["first_hit_sweep"].item())
        gpu_s = None
        if hit >= 0:
            timed_to(hit + 1, 1)
            gpu_s, h2 = timed_to(hit + 1, 1)
            assert h2 == hit
        tts.update(first_hit_sweep=hit, gpu_s=gpu_s,
                   protocol="E* = mean over 10 oracle chains (100,000 proposals each, this config's schedule) of the minimum "
                            "sweep-end energy; gpu_s = MEASURED device time (CUDA events) of an amh_run of exactly first_hit_sweep + 1 sweeps "
                            "from the same start, first_hit_sweep = first sweep at whose end some chain of the batch has V <= E*; "
                            "cpu_s = wall time of the oracle runs, one core per chain")
        # nine more seeds (PAPER.md:184-188 takes means over repeated runs; median over 10 seeds)
        hits, times = [hit], [gpu_s]
        if hit >= 0:
            short = int(min(cfg.n_sweeps, 8 * (hit + 1) + 4 * (cfg.n_global + cfg.n_local)))
            for seed in range(2, 11):
                _, h = timed_to(short, seed)
                hits.append(h)
                times.append(timed_to(h + 1, seed)[0] if h >= 0 else None)
            ok = sorted(x for x in times if x is not None)
            tts.update(first_hit_sweeps_10_seeds=hits, gpu_s_10_seeds=times, gpu_s_median=ok[len(ok) // 2] if len(ok) == len(times) else None)
        tts["speedup_vs_oracle_chain"] = (tts["cpu_s"] / tts["gpu_s"]) if tts["gpu_s"] else None
        tts["note"] = "speedup is over the deliberately slow fp64 oracle (full rebuild + full re-sum per proposal), not over a tuned CPU implementation"

    # ---------------- global-only and local-only rates, short runs from the final states ----------
    phase_rates = None
    if rank == 0 and world == 1 and not exchange:
        phase_rates = {}
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
        e2e_steps = min(args.steps, 5)
        hs = torch.empty_like(wl.s0_host).pin_memory()
        hkw = dict(kw)
        if "per_chain_T" in hkw:
            hkw["per_chain_T"] = hkw["per_chain_T"].cpu().numpy()
        hs.copy_(wl.s0_host); g.run_host(hs.numpy(), cfg.n_sweeps, **hkw)         # warm-up (staging arena)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            hs.copy_(wl.s0_host)
            rh = g.run_host(hs.numpy(), cfg.n_sweeps, **hkw)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        te = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if dist is not None:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        h2d = B * n * 4 + (B * 4 if cfg.replicas else 0)
        d2h = B * n * 4 + 2 * B * 4
        e2e = dict(value=props_per_step * e2e_steps / float(te.item()), unit=UNIT, h2d_bytes_per_step=h2d,
                   d2h_bytes_per_step=d2h, steps=e2e_steps, api="amh_run_host (pinned host buffers; copies inside the timed region)",
                   best_energy=float(rh["best_energy"].min()))

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---------------- ceilings measured in this run, roofline of the dominant kernel (one launch per step) ---------
    peaks = measured_peaks()
    sm_max_mhz = (clocks or {}).get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
    l2_48 = pkg.probe_l2_read(48 << 20, 20)
    l2_92 = pkg.probe_l2_read(92 << 20, 12)
    gather = pkg.probe_gather(64 << 20, 5)
    ceilings = dict(l2_read_gbs_48mb=l2_48, l2_read_gbs_92mb=l2_92, gathers_per_s_64mb=gather, hbm_gbs_measured=peaks.get("hbm_gbs"),
                    source="amh_probe_l2_read / amh_probe_gather in this run; hbm from MEASURED_PEAKS.json")
    roofline = wl.roofline(ms_per_step, info["n_sm"], sm_max_mhz, peaks, l2_92 if cfg.L >= 512 else l2_48, gather)
    launch_headline = dict(wl.launch_dict(), best_energy=best)
    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline, _ = oracle_leg(cfg)

    # ---------------- every other config, one timed step each (N = 1) -------------------------------------------------
    per_config = None
    if world == 1 and args.per_config != "off" and not overridden and not exchange:
        per_config = {}
        for cid in sorted(gi.CONFIGS):
            if cid == args.config:
                continue
            c2 = gi.CONFIGS[cid]
            sliced = args.per_config == "slice" and c2.proposals > 2e9
            if sliced:
                import dataclasses
                c2 = dataclasses.replace(c2, n_sweeps=4 * (c2.n_global + c2.n_local))
            del wl.g
            torch.cuda.empty_cache()
            wl = Workload(pkg, torch, c2, 0, 1)
            smp = ClockSampler(local_rank)
            wl.reset(); wl.run(sweeps=min(c2.n_sweeps, 2 * (c2.n_global + c2.n_local)))      # warm-up: tables into L2, code loaded
            ms, r2 = time_steps(torch, wl, 1, 0, flush, stream, barrier, wl.run)
            ck = smp.stop()
            entry = dict(value=c2.proposals / (ms * 1e-3), unit=UNIT, ms_per_step=ms, steps=1, warmup="2 cycles",
                         dtype="f64" if c2.slots == 5 else "f32",
                         config=workload_dict(c2, sliced), launch=wl.launch_dict(), clocks=ck,
                         best_energy=float(r2["best_energy"].min().item()),
                         roofline=wl.roofline(ms, info["n_sm"], sm_max_mhz, peaks, l2_92 if c2.L >= 512 else l2_48, gather))
            if not args.no_cpu_baseline:
                entry["cpu_baseline"] = oracle_leg(c2, target_s=4.0, max_chains=16)[0]
            per_config[c2.name] = entry

    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=args.warmup,
                ms_per_step=ms_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64" if cfg.slots == 5 else "f32",
                data="synthetic", config=workload, launch=launch_headline, clocks=clocks, e2e=e2e, gpu_launches=launches,
                roofline=roofline, ceilings=ceilings, cpu_baseline=cpu_baseline, time_to_threshold=tts, phase_rates=phase_rates,
                per_config=per_config)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
