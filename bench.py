#!/usr/bin/env python
"""bench.py -- the FourPhonon scattering-rate hot path on B200 (contract: see DESIGN.md §8).

One "step" = one pass of the whole hot path over the workload (BASELINE.json config 3 by default: diamond 16x16x16,
3ph rates of all 24,576 modes + 4ph rates of 96 target modes + RTA kappa): fp_rates3 -> fp_rates4 -> fp_kappa_rta
through the C ABI with device-resident inputs (`value`), and fp_setup(host arrays) -> fp_rates3 -> fp_rates4 ->
fp_kappa_rta with HOST buffers, copies inside the timed region (`e2e`).  metric = allowed 4ph processes per second
of whole-step time.  N > 1: independent replicas (the path does not shard per north_star).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

METRIC = "4ph processes/s (FP64)"      # (3ph-only workloads count 3ph processes; config.processes_counted_in_value says which)
UNIT = "processes/s"
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12     # 148 SMs x 64 FP64 FMA/clk/SM x 2 flop x 1965 MHz
NCU_TRAFFIC = ROOT / "profiles" / "ncu_traffic.json"     # dram bytes of one launch per (config, kernel), each naming its ncu capture


def ncu_traffic(cfg: int, kernel: str):
    """-> the tracked entry of profiles/ncu_traffic.json for this configuration's dominant kernel, or None."""
    try:
        return json.loads(NCU_TRAFFIC.read_text()).get(f"{cfg}:{kernel}")
    except (OSError, ValueError):
        return None


def workload(cfg: int):
    """-> list of (Inputs, targets3 or None, targets4 or None, (qp_begin, qp_end))"""
    import fp_inputs
    jobs = fp_inputs.make_config(cfg)
    return [(inp, inp.targets3 if inp.ifc3 is not None else None, inp.targets4 if inp.ifc4 is not None else None)
            for inp in jobs.values()]


def workload_name(cfg: int) -> str:
    import fp_inputs
    if cfg in fp_inputs.PAPER_MESHES:                                       # not a BASELINE.json config
        return f"{fp_inputs.CONFIG_NAMES[cfg]} (fp_inputs config {cfg}; synthetic IFCs of configs 0-3)"
    return f"BASELINE.json configs[{cfg}]: {fp_inputs.CONFIG_NAMES[cfg]}"


class ClockSampler(threading.Thread):
    """nvidia-smi-equivalent clock / throttle-reason samples (NVML) during the timed region."""

    def __init__(self, index: int, period: float = 0.1):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.sm, self.reasons, self.max_sm = [], set(), None
        self._stop_evt = threading.Event()

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_sm = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {
                getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
                getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
                getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
            }
            while not self._stop_evt.is_set():
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(self.period)
        except Exception as e:                                              # no NVML: report that, do not fake clocks
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        sm = sorted(self.sm)
        return {"sm_mhz": (sm[len(sm) // 2] if sm else None), "sm_max_mhz": self.max_sm, "reasons": sorted(self.reasons),
                "samples": len(sm)}


def reduce_over_ranks(ms_local: float, units_local: float, dist) -> tuple[float, float]:
    """max step time over ranks, sum of units over ranks (replicas: every rank processes its own copy)."""
    import torch
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return ms_local, units_local
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    u = torch.tensor([units_local], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ---------------------------------------------------------------------------------------------------------------------------
def cpu_oracle_sample(cfg: int, budget_s: float = 15.0):
    """Time the oracle, as it stands, on a bounded sample of the workload's 4ph job: the first target modes over a q'
    range sized from a calibration call so that the timed call is ~budget_s of host work."""
    from oracle.oracle import Oracle
    jobs = workload(cfg)
    job4 = next((j for j in jobs if j[2] is not None), None)
    if job4 is None:                                                        # 3ph-only workloads: a sample of the target modes
        inp, t3, _ = jobs[0]
        orc = Oracle(inp)
        probe = np.ascontiguousarray(t3[:: max(1, len(t3) // 8)][:8])
        t0 = time.perf_counter()
        orc.rates3(probe)
        dt = max(time.perf_counter() - t0, 1e-3)
        n = int(max(8, min(len(t3), 8 * budget_s / dt)))
        t = np.ascontiguousarray(t3[:: max(1, len(t3) // n)][:n])
        t0 = time.perf_counter()
        _, _, c = orc.rates3(t)
        dt = time.perf_counter() - t0
        procs = int(c.sum())
        return {"value": procs / dt, "unit": UNIT, "cores": Oracle.num_threads(), "kind": "oracle",
                "note": "the oracle is a deliberately plain correctness checker, not a tuned CPU implementation",
                "sample": f"oracle rates3 on {len(t)} of the {len(t3)} target modes (evenly spaced): {procs} allowed "
                          f"processes in {dt:.2f} s"}, dt, procs
    inp, _, t4 = job4
    orc = Oracle(inp)
    t = np.ascontiguousarray(t4[:6])
    N = inp.nq
    t0 = time.perf_counter()
    _, _, c = orc.rates4(t, 0, 1)
    dt = max(time.perf_counter() - t0, 1e-3)
    q0 = 1 if N > 1 else 0                                                  # sample range [q0, q0 + nq) stays inside the mesh
    nq = int(max(1, min(N - q0, budget_s / dt)))
    t0 = time.perf_counter()
    _, _, c = orc.rates4(t, q0, q0 + nq)
    dt = time.perf_counter() - t0
    procs = int(c.sum())
    return {"value": procs / dt, "unit": UNIT, "cores": Oracle.num_threads(), "kind": "oracle",
            "note": "the oracle is a deliberately plain correctness checker (full rectangular domain, V from the raw IFC list per process), not a tuned CPU implementation: the GPU/CPU ratio says nothing about kernel quality",
            "sample": f"oracle rates4 on the first {len(t)} target modes, q' in [{q0},{q0 + nq}) of {N}: {procs} allowed "
                      f"processes in {dt:.2f} s"}, dt, procs


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals, secs = [], []
    per_step = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for i in range(args.warmup + args.steps):
        cb, dt, procs = cpu_oracle_sample(args.config, per_step)
        if i >= args.warmup:
            vals.append(procs); secs.append(dt)
    value = sum(vals) / sum(secs)
    cb["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / len(secs), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(args.config), "note": "CPU oracle on a bounded sample per step"},
            "cpu_baseline": cb,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--scratch-gb", type=float, default=48.0,
                    help="per-context scratch: half of it holds the process lists of the split path (DESIGN.md §5.2)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--path", choices=["auto", "fused", "split", "split-serial"], default="auto",
                    help="execution path of fp_rates3/4 (fp_set_path); auto = split when the scratch holds the lists")
    ap.add_argument("--precision", choices=["fp64", "mixed"], default="fp64",
                    help="mixed = fp_set_precision(FP_PREC_MIXED): level-2 contraction in FP32 (not the headline: fails the 1e-9 bar)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2510_00518_b200 as fp

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    fp.build_library(force=False)          # no-op when the in-tree .so is newer than its sources (nvcc, sm_100a)
    fp.load_library()

    jobs = workload(args.config)
    scratch = int(args.scratch_gb * (1 << 30))
    path_id = {"auto": fp.FP_PATH_AUTO, "fused": fp.FP_PATH_FUSED, "split": fp.FP_PATH_SPLIT,
               "split-serial": fp.FP_PATH_SPLIT_SERIAL}[args.path]
    ctxs, dev_targets = [], []
    for inp, t3, t4 in jobs:
        ctx = fp.Context.from_inputs(inp, scratch_bytes=scratch, device=dev)
        ctx.set_path(path_id)
        if args.precision == "mixed":
            ctx.set_precision(fp.FP_PREC_MIXED)
        ctxs.append(ctx)
        dev_targets.append((None if t3 is None else torch.from_numpy(np.ascontiguousarray(t3)).to(dev),
                            None if t4 is None else torch.from_numpy(np.ascontiguousarray(t4)).to(dev)))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)          # > 126 MB L2

    def step_device():
        """fp_rates3 -> fp_rates4 -> fp_kappa_rta with device-resident inputs and outputs."""
        res = {}
        for ctx, (inp, t3, t4), (d3, d4) in zip(ctxs, jobs, dev_targets):
            if d3 is not None:
                g3, w3, c3 = ctx.rates3(d3)
                res["c3"] = c3
                if len(t3) == ctx.nmodes:
                    res["kappa"] = ctx.kappa_rta(g3.sum(dim=1))
            if d4 is not None:
                g4, w4, c4 = ctx.rates4(d4)
                res["c4"] = c4
        return res

    def step_host():
        """the same pass from HOST buffers: fp_setup(host) + rates with host targets/outputs (copies inside)."""
        h2d = d2h = 0
        res = {}
        for inp, t3, t4 in jobs:
            with fp.Context.from_inputs(inp, scratch_bytes=scratch, device=dev) as ctx:
                ctx.set_path(path_id)
                if args.precision == "mixed":
                    ctx.set_precision(fp.FP_PREC_MIXED)
                h2d += inp.omega.nbytes + inp.eig.nbytes + inp.vg.nbytes
                for ifc in (inp.ifc3, inp.ifc4):
                    if ifc is not None:
                        h2d += sum(np.asarray(a).nbytes for a in ifc)
                if t3 is not None:
                    g3, w3, c3 = ctx.rates3(t3)
                    h2d += t3.nbytes; d2h += g3.nbytes + w3.nbytes + c3.nbytes
                    if len(t3) == ctx.nmodes:
                        gt = g3.sum(axis=1)
                        res["kappa"] = ctx.kappa_rta(gt)
                        h2d += gt.nbytes; d2h += 72
                if t4 is not None:
                    g4, w4, c4 = ctx.rates4(t4)
                    h2d += t4.nbytes; d2h += g4.nbytes + w4.nbytes + c4.nbytes
                    res["c4"] = c4
        return res, h2d, d2h

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ------------------------------------------------------------------------------------------
    for _ in range(max(args.warmup, 1)):                                   # at least one untimed pass: it also yields the counts
        flush.fill_(1)
        res = step_device()
    n4 = int(res["c4"].sum().item()) if "c4" in res else 0
    n3 = int(res["c3"].sum().item()) if "c3" in res else 0
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        flush.fill_(1)                                                     # L2 flush between timed iterations
        res = step_device()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop()
    counted = "4ph" if n4 > 0 else "3ph"                                  # configs 0 and 1 have no 4ph work: count 3ph processes
    ms_step, procs_all = reduce_over_ranks(ms_total / args.steps, float(n4 if n4 > 0 else n3), dist if world > 1 else None)
    value = procs_all / (ms_step * 1e-3)

    # ---- end to end from host buffers ------------------------------------------------------------------------------------
    for _ in range(min(args.warmup, 1)):
        step_host()
    barrier()
    e0.record()
    for _ in range(args.steps):
        flush.fill_(1)
        rh, h2d, d2h = step_host()
    e1.record()
    barrier()
    ms_e2e, _ = reduce_over_ranks(e0.elapsed_time(e1) / args.steps, 0.0, dist if world > 1 else None)
    e2e = {"value": procs_all / (ms_e2e * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
           "d2h_bytes_per_step": int(d2h), "ms_per_step": ms_e2e,
           "what": "fp_setup(host arrays) + fp_rates3 + fp_rates4 + fp_kappa_rta with host targets and outputs"}

    # ---- per-kernel profile of one more step (CUDA events on the launch stream, inside the library) ------------------------
    for ctx in ctxs:
        ctx.profile_enable(True); ctx.profile_reset()
    step_device()
    torch.cuda.synchronize()
    kern = {}
    flops = procs = cands = pref = launches = rows = overflows = evaluated = 0
    symmetry = False
    for ctx in ctxs:
        p = ctx.profile_get()
        for k in ("precontract", "enum", "rates", "reduce"):
            kern.setdefault(k, [0.0, 0])
            kern[k][0] += getattr(p, "ms_" + k); kern[k][1] += getattr(p, "n_" + k)
        flops += p.rates_flops; procs += p.processes; cands += p.candidates; pref += p.prefiltered
        launches += p.launches; rows += p.rows; overflows += p.list_overflows; evaluated += p.evaluated
        symmetry = symmetry or ctx.get_symmetry()
        ctx.profile_enable(False)
    dom = max(kern, key=lambda k: kern[k][0])
    ms_c, n_c = kern["rates"]
    ms_en, n_en = kern["enum"]
    split = n_en > 0
    achieved = flops / (ms_c * 1e-3) / 1e12 if ms_c > 0 else 0.0
    probe = fp.fp_probe_fp64_tflops()
    kname = ("k_eval_g (V3/V4 level-2 contraction + row sums over the process lists; the enumerator k_enum_g is timed "
             "separately, see kernel_ms_per_step)") if split else "k_rates (fused enumerate + V3/V4 contraction + weights)"
    tr = ncu_traffic(args.config, "k_eval_g" if split else "k_rates")
    dmma = fp.fp_probe_dmma_tflops()
    step_flops_rate = flops / (ms_step * 1e-3) / 1e12
    mixed = args.precision == "mixed"                                       # FP32 FFMA pipe: 128 lanes/clk/SM, twice the FP64 rate
    peak = FP64_PEAK_TFLOPS * (2.0 if mixed else 1.0)
    roofline = {"bound": "alu", "kernel": kname, "achieved": achieved,
                "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": tr["bytes"] if tr else None,
                "traffic_source": ({"file": "profiles/ncu_traffic.json", "capture": tr["capture"], "launch": tr["launch"],
                                    "launch_ms": tr["duration_ms"], "list_bytes_of_that_launch": tr["list_bytes"]}
                                   if tr else None),
                "algorithmic_bytes_per_launch_avg": 16.0 * evaluated / max(n_c, 1) if split else 20.0 * rows / max(n_c, 1),
                "whole_step": {"achieved": step_flops_rate, "frac": step_flops_rate / peak,
                               "what": "the same executed-flop model over the whole device-timed step (enumerator, "
                                       "pre-contraction and reduction included in the time, not in the flops)"},
                "probes_tflops": {"dfma": probe, "dmma_m8n8k4": dmma["dmma"], "dfma_same_shape": dmma["dfma"],
                                  "dmma_and_dfma_interleaved": dmma["dmma_and_dfma"]},
                "peak_source": ("FP32 (mixed mode): 148 SM x 128 FFMA/clk x 2 x 1.965 GHz; " if mixed else "") +
                               "derived: 148 SM x 64 FP64 FMA/clk x 2 x 1.965 GHz (MEASURED_PEAKS.json has no FP64 "
                               f"entry); DFMA probe on this GPU measured {probe:.2f} TFLOP/s",
                "flops_model": "matrix elements evaluated x executed flops of the level-2 contraction (nat <= 2: nblk x 13 complex "
                               "MAC x 8 flop; generic atom count: (12 nblk + 3 atoms) x 8; DESIGN.md §6); enumeration, decision "
                               "and weights not counted",
                "matrix_elements_per_step": evaluated,
                "pair_symmetry": ("on: the IFC4 list is symmetric in its last two legs, so each unordered {lambda'', lambda'''} "
                                  "pair of the +- and -- channels is evaluated once (both orderings counted as processes, "
                                  "each with its own pinned window decision)") if symmetry else "off",
                "flops_per_launch": flops / max(n_c, 1), "avg_launch_ms": ms_c / max(n_c, 1),
                "dominant_by_time": dom,
                "kernel_ms_per_step": {k: round(v[0], 3) for k, v in kern.items()},
                "rows_per_step": rows, "candidates_per_step": cands, "prefiltered_per_step": pref,
                "processes_per_step": procs,
                "candidates_per_s_in_enumerator": cands / ((ms_en if split else ms_c) * 1e-3) if ms_c > 0 else 0.0,
                "path": "split" if split else "fused", "list_slot_overflows_per_step": overflows}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if args.precision == "fp64" else "f32 level-2 contraction, f64 decision/weights/sums (NOT the headline)",
            "data": "synthetic",
            "config": {"workload": workload_name(args.config), "step": "fp_rates3 + fp_rates4 + fp_kappa_rta",
                       "processes_4ph_per_step": n4, "processes_3ph_per_step": n3, "processes_counted_in_value": counted, "parallelism": f"replicas x{world}",
                       "l2": "flushed between steps (256 MB write)"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches * args.steps), "roofline": roofline}
    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_oracle_sample(args.config)[0]
        print(json.dumps(line))
    for ctx in ctxs:
        ctx.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
