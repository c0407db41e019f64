#!/usr/bin/env python
"""bench.py -- states integrated per second over one global step (BASELINE.json metric).

`python bench.py --gpus N --steps K --warmup W` : one "step" = one pass of the whole hot path
(chem_integrate over the config's batch of synthetic states).  The top-level line is BASELINE.json
configs[1] (h2co-shaped 13 species / 27 reactions, 1,048,576 states, dt = 1e-6 s); at N = 1 the same line
carries `"configs"`: the other four BASELINE.json configs, each timed the same way (device-resident and end to end)
with its roofline fraction, failed-state count and the divergence measure D of PAPER.md Eq. 3.
N > 1: every rank integrates its own batch of that size (weak scaling, no collective on the data path).
`--impl reference` times the CPU oracle as it stands on a bounded sample of the same workload.
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

from paper_1607_03884_b200 import diagnostics, shard, synth  # noqa: E402

METRIC = "states integrated/sec per global step (fp64)"
UNIT = "states/s"
# ALU roofline: 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz = 37.2 TFLOP/s; the library's DFMA
# probe measures 34.8 TFLOP/s (profiles/r2_fp64_peak.md) and is rerun and printed by every bench run
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the integration kernel from the committed
# `ncu --set full` captures, keyed by (config index, kernel id); None where no capture of that pair is on file.
NCU_TRAFFIC = {
    (0, 2): (1.842944e6 + 0.225536e6, "profiles/r3_metrics_all_configs.md (ncu --metrics pass)"),
    (1, 2): (115.299840e6 + 109.461760e6, "profiles/r1_final_config1.md (ncu --set full)"),
    (1, 3): (44.098521e9 + 23.691889e9, "profiles/r3_tps_config1.md, r3_tps_metrics_config1.csv (ncu --metrics pass): lane-private LU factors stream through L2 / HBM"),
    (2, 2): (0.331e9, "profiles/r2_mapping_config2.md (ncu --metrics pass)"),
    (2, 3): (208.304123e9 + 113.344515e9, "profiles/r3_metrics_all_configs.md (ncu --metrics pass)"),
    (3, 1): (253.852416e6 + 234.944512e6, "profiles/r3_metrics_all_configs.md (ncu --metrics pass)"),
    (4, 1): (259.344640e6 + 239.524864e6, "profiles/r3_metrics_all_configs.md (ncu --metrics pass)"),
}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 7 and r[3 + i] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


FLOP_CONVENTION = "+,-,*,/ = 1, fma = 2, exp/log/pow/sqrt = 20 flop each (chem_flop_model; frac_transcendental_1: 1 each)"


def algorithmic_flops(stats, fm):
    """DESIGN.md flop model: per-state counters x per-operation algorithmic flops."""
    s = {k: float(stats[k].astype(np.float64).sum()) for k in ("nfcn", "njac", "ndec", "nsol", "nstep")}
    return s["nfcn"] * fm["rhs"] + s["njac"] * fm["jac"] + s["ndec"] * fm["lu"] + s["nsol"] * fm["newton"] + s["nstep"] * fm["err"]


def config_dict(cfg, N, NR, world):
    """the `config` object of a bench line: the same for the GPU arm and the reference arm"""
    return {"workload": cfg["name"], "mechanism": f"{cfg['kind']}-shaped synthetic, {N} species / {NR} reactions",
            "states_per_gpu": cfg["n_states"], "t_end": cfg["t_end"], "rtol": synth.RTOL, "atol": synth.ATOL, "P": synth.P_ATM,
            "parallelism": f"batch sharded over {world} GPU(s), no collective",
            "l2": f"inputs+outputs {2 * cfg['n_states'] * N * 8 / 1e6:.0f} MB per step"
                  + (" exceed the 126 MB L2 (no flush)" if 2 * cfg["n_states"] * N * 8 > 126e6 else
                     ": smaller than the 126 MB L2, a 256 MB buffer is written between timed steps (flush)")}


def cpu_baseline(mech, cfg, y0, seconds_target=12.0):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload."""
    from oracle import oracle as orc
    M = orc.Mechanism(mech)
    probe = min(4096, y0.shape[0])
    t0 = time.perf_counter()
    _, _, cores = M.integrate(y0[:probe], synth.P_ATM, cfg["t_end"], synth.RTOL, synth.ATOL)
    rate = probe / max(time.perf_counter() - t0, 1e-6)
    n = int(min(y0.shape[0], max(probe, rate * seconds_target)))
    t0 = time.perf_counter()
    M.integrate(y0[:n], synth.P_ATM, cfg["t_end"], synth.RTOL, synth.ATOL)
    dt = time.perf_counter() - t0
    return {"value": n / dt, "unit": UNIT, "cores": int(cores), "kind": "oracle",
            "sample": f"first {n} states of the {y0.shape[0]}-state batch, one global step, {dt:.2f} s"}


def run_reference(args, cfg, mech):
    """--impl reference: the CPU oracle, bounded sample per step, rank 0 only."""
    rank, _, world = shard.env_world()
    if rank != 0:
        return
    from oracle import oracle as orc
    M = orc.Mechanism(mech)
    n = min(cfg["n_states"], 65536)
    y0 = synth.make_states(mech, n, cfg["dist"], synth.STATE_SEED)
    cores = 0
    for _ in range(args.warmup):
        _, _, cores = M.integrate(y0[: max(n // 16, 1)], synth.P_ATM, cfg["t_end"], synth.RTOL, synth.ATOL)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, _, cores = M.integrate(y0, synth.P_ATM, cfg["t_end"], synth.RTOL, synth.ATOL)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt
    sample = (f"each step integrates the first {n} states of the {cfg['n_states']}-state batch of the workload "
              f"(the metric is intensive: states/s)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(cfg, int(mech["n_species"]), int(mech["n_reactions"]), max(args.gpus, 1)),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(cores), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


class Flusher:
    """writes a buffer larger than the 126 MB L2 (timing rule for inputs smaller than L2)"""

    def __init__(self, torch):
        self.buf = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")

    def __call__(self):
        self.buf.fill_(1)


def time_config(torch, binding, gm, mech, cfg, steps, warmup, kernel, rank, world, e2e_steps, sampler=None):
    """Device-resident and end-to-end timing of one config; returns the measured numbers (rank-local reductions done)."""
    n = cfg["n_states"]
    N = gm.n_species
    y0 = synth.make_states(mech, n, cfg["dist"], synth.STATE_SEED + rank)
    y_dev = torch.from_numpy(y0).cuda()
    y_out = torch.empty_like(y_dev)
    y_pin = torch.from_numpy(y0).pin_memory()
    y_out_pin = torch.empty(y_pin.shape, dtype=torch.float64, pin_memory=True)     # empty_like would not be pinned
    flush = Flusher(torch) if 2 * n * N * 8 <= 126e6 else None
    if kernel == 0:
        run = lambda: binding.chem_integrate(gm, synth.P_ATM, cfg["t_end"], synth.RTOL, synth.ATOL, y_dev, y_out)
    else:
        run = lambda: binding.chem_integrate_ex(gm, synth.P_ATM, cfg["t_end"], synth.RTOL, synth.ATOL, y_dev, y_out,
                                                want_stats=False, kernel=kernel)
    # per-state counters for the flop model and the divergence measure (outside the timed region)
    _, st = binding.chem_integrate_ex(gm, synth.P_ATM, cfg["t_end"], synth.RTOL, synth.ATOL, y_dev, y_out, kernel=kernel)
    torch.cuda.synchronize()
    used_kernel = binding.chem_last_kernel(gm)
    stats = binding.stats_to_numpy(st)
    failed = int((stats["status"] != 0).sum())
    flops_per_launch = algorithmic_flops(stats, gm.flop_model())
    flops_per_launch_t1 = algorithmic_flops(stats, gm.flop_model(transcendental_1=True))
    D = diagnostics.divergence_summary(stats["nstep"])

    for _ in range(warmup):
        run()
    torch.cuda.synchronize()
    if sampler is not None and rank == 0:
        sampler.start()
    shard.barrier()
    torch.cuda.synchronize()
    l0 = binding.chem_launch_count()
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(steps)]
    for i in range(steps):
        if flush is not None:
            flush()
        ev0[i].record()
        run()
        ev1[i].record()
    torch.cuda.synchronize()
    shard.barrier()
    launches = binding.chem_launch_count() - l0
    clocks = sampler.stop() if (sampler is not None and rank == 0) else None
    step_ms = np.array([ev0[i].elapsed_time(ev1[i]) for i in range(steps)])
    total_s = float(step_ms.sum()) * 1e-3
    total_s, units = shard.reduce_max_sum(total_s, float(n * steps), device="cuda")

    # end to end through the C ABI with HOST (pinned) buffers: H2D + kernel + D2H inside the call
    host = lambda: binding.chem_integrate_host(gm, synth.P_ATM, cfg["t_end"], synth.RTOL, synth.ATOL, y_pin.numpy(),
                                               y_out_pin.numpy(), kernel=kernel)
    host()
    shard.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        host()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s, e2e_units = shard.reduce_max_sum(e2e_s, float(n * e2e_steps), device="cuda")
    assert np.array_equal(y_out_pin.numpy(), y_out.cpu().numpy()), "host-buffer path disagrees with device path"
    del y_dev, y_out, flush
    torch.cuda.empty_cache()
    return dict(n=n, N=N, total_s=total_s, units=units, kernel_s=float(step_ms.mean()) * 1e-3, launches=int(launches),
                clocks=clocks, e2e_s=e2e_s, e2e_units=e2e_units, e2e_steps=e2e_steps, failed=failed,
                flops_per_launch=flops_per_launch, flops_per_launch_t1=flops_per_launch_t1, D=D, used_kernel=used_kernel, y0=y0,
                mean_steps=float(stats["nstep"].mean()), max_steps=int(stats["nstep"].max()))


_probe = {}


def roofline(binding, ci, r, peaks, which):
    """The roofline record of one config.  `bound` is the roof the ALGORITHM is nearer to (algorithmic flops against the
    fp64 peak, algorithmic bytes against the HBM peak), and achieved / peak / frac follow it.  Beside it: `hbm_frac`, the
    share of the HBM bandwidth the kernel actually used (DRAM bytes of the committed ncu capture of this config and kernel
    over the live kernel time; the algorithmic figure when no capture is on file), `hbm_frac_algorithmic`, and `limiter`,
    which says "latency" when the kernel is near neither roof."""
    if "tf" not in _probe:
        _probe["tf"] = binding.chem_fp64_probe()          # outside every timed region
    achieved = r["flops_per_launch"] / r["kernel_s"] / 1e12
    alu_frac = achieved / FP64_PEAK_TFLOPS
    traffic = NCU_TRAFFIC.get((ci, r["used_kernel"]))
    alg_bytes = 2 * r["n"] * r["N"] * 8
    alg_gbs = alg_bytes / r["kernel_s"] / 1e9
    hbm_frac_alg = alg_gbs / peaks["hbm_gbs"]
    hbm_frac = (traffic[0] / r["kernel_s"] / 1e9) / peaks["hbm_gbs"] if traffic else hbm_frac_alg
    if alu_frac >= hbm_frac_alg:
        head = {"bound": "alu", "achieved": achieved, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": alu_frac}
    else:
        head = {"bound": "hbm", "achieved": alg_gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": hbm_frac_alg}
    nearest = max(alu_frac, hbm_frac)
    limiter = ("latency: %.0f %% of the fp64 peak and %.0f %% of the HBM bandwidth in use, neither roof is near (DESIGN.md 7)"
               % (100 * alu_frac, 100 * hbm_frac)) if nearest < 0.5 else ("hbm" if hbm_frac > alu_frac else "alu")
    head.update({
        "traffic": traffic[0] if traffic else None, "traffic_source": traffic[1] if traffic else None,
        "traffic_over_algorithmic": traffic[0] / alg_bytes if traffic else None,
        "kernel": binding.KERNEL_NAMES.get(r["used_kernel"], "?"), "kernel_ms": 1e3 * r["kernel_s"],
        "flops_per_launch": r["flops_per_launch"], "flop_convention": FLOP_CONVENTION,
        "alu_frac": alu_frac, "frac_transcendental_1": r["flops_per_launch_t1"] / r["kernel_s"] / 1e12 / FP64_PEAK_TFLOPS,
        "peak_source": "derived: 148 SM x 64 FP64 FMA/clk x 2 x 1.965 GHz (DESIGN.md 7, profiles/r2_fp64_peak.md)",
        "peak_measured_dfma_probe": _probe["tf"],
        "hbm_frac": hbm_frac, "hbm_frac_source": "ncu dram bytes / live kernel time" if traffic else "algorithmic bytes (no ncu capture on file)",
        "hbm_frac_algorithmic": hbm_frac_alg, "hbm_peak_source": which, "limiter": limiter})
    return head


def summary_row(ci, name, r, roof, total_s, units, steps):
    """compact per-config record for the `summary` array, the LAST key of the line (it survives a truncated tail)"""
    return {"i": ci, "workload": name, "kernel": r["used_kernel"], "ms_per_step": round(1e3 * total_s / steps, 3),
            "value": round(units / total_s, 1), "frac": round(roof["frac"], 4), "frac_t1": round(roof["frac_transcendental_1"], 4),
            "hbm_frac": round(roof["hbm_frac"], 4), "e2e_over_device": round((r["e2e_units"] / r["e2e_s"]) / (units / total_s), 3),
            "failed": r["failed"], "D_mean": round(r["D"]["mean"], 3) if r["D"].get("mean") is not None else None}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="index into BASELINE.json configs of the top-level line (default 1)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--only", action="store_true", help="time the top-level config only (no `configs` array)")
    ap.add_argument("--kernel", type=int, default=0, help="0 auto, 1 group kernel, 2 warp per state, 3 thread per state")
    ap.add_argument("--states", type=int, default=0, help="profiling aid: use only the first N states of the config (not a bench line)")
    args = ap.parse_args()
    cfg = dict(synth.CONFIGS[args.config])
    if args.states > 0:
        cfg["n_states"] = min(args.states, cfg["n_states"])
        cfg["name"] += f"[first {cfg['n_states']} states: profiling subset]"
    mech = synth.make_mechanism(cfg["kind"], synth.MECH_SEED)
    if args.impl == "reference":
        run_reference(args, cfg, mech)
        return

    import torch
    from paper_1607_03884_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    rank, local_rank, world = shard.env_world()
    torch.cuda.set_device(local_rank)
    shard.init_process_group("nccl")
    warmup = max(args.warmup, 3)
    peaks, which = load_peaks()

    mechs, gms = {cfg["kind"]: mech}, {}

    def gm_of(kind):
        if kind not in mechs:
            mechs[kind] = synth.make_mechanism(kind, synth.MECH_SEED)
        if kind not in gms:
            gms[kind] = binding.chem_mech_load(mechs[kind])
        return gms[kind], mechs[kind]

    gm, _ = gm_of(cfg["kind"])
    r = time_config(torch, binding, gm, mech, cfg, args.steps, warmup, args.kernel, rank, world,
                    max(3, min(args.steps, 5)), sampler=ClockSampler(local_rank))
    others, summary = [], []
    roof = roofline(binding, args.config, r, peaks, which)
    summary.append(summary_row(args.config, cfg["name"], r, roof, r["total_s"], r["units"], args.steps))
    if world == 1 and not args.only and args.states == 0:
        for ci, c in enumerate(synth.CONFIGS):
            if ci == args.config:
                continue
            g2, m2 = gm_of(c["kind"])
            steps2 = 20 if c["n_states"] <= 65536 else 3
            r2 = time_config(torch, binding, g2, m2, c, steps2, 3, args.kernel, rank, world, 3)
            roof2 = roofline(binding, ci, r2, peaks, which)
            summary.append(summary_row(ci, c["name"], r2, roof2, r2["total_s"], r2["units"], steps2))
            others.append({
                "index": ci, "workload": c["name"], "config": config_dict(c, r2["N"], g2.n_reactions, world),
                "value": r2["units"] / r2["total_s"], "unit": UNIT, "steps": steps2, "warmup": 3,
                "ms_per_step": 1e3 * r2["total_s"] / steps2, "us_per_state": 1e6 * r2["total_s"] / r2["units"],
                "roofline": roof2,
                "e2e": {"value": r2["e2e_units"] / r2["e2e_s"], "unit": UNIT, "h2d_bytes_per_step": r2["n"] * r2["N"] * 8,
                        "d2h_bytes_per_step": r2["n"] * r2["N"] * 8, "steps": r2["e2e_steps"], "host_memory": "pinned"},
                "gpu_launches": r2["launches"], "failed_states": r2["failed"],
                "internal_steps": {"mean": r2["mean_steps"], "max": r2["max_steps"]}, "D": r2["D"]})
            del r2
    if rank != 0:
        return
    n, N = r["n"], r["N"]
    cdict = config_dict(cfg, N, gm.n_reactions, world)
    out = {
        "metric": METRIC, "value": r["units"] / r["total_s"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warmup,
        "ms_per_step": 1e3 * r["total_s"] / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": cdict, "clocks": r["clocks"],
        "failed_states": r["failed"], "us_per_state": 1e6 * r["total_s"] / r["units"] * world,
        "e2e": {"value": r["e2e_units"] / r["e2e_s"], "unit": UNIT, "h2d_bytes_per_step": n * N * 8, "d2h_bytes_per_step": n * N * 8,
                "steps": r["e2e_steps"], "host_memory": "pinned"},
        "gpu_launches": r["launches"],
        "roofline": roof,
        "internal_steps": {"mean": r["mean_steps"], "max": r["max_steps"]}, "D": r["D"],
    }
    if others:
        out["configs"] = others
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(mech, cfg, r["y0"])
    out["summary"] = sorted(summary, key=lambda x: x["i"])       # last key on purpose: one short row per config
    print(json.dumps(out))


if __name__ == "__main__":
    main()
