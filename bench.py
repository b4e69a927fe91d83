#!/usr/bin/env python
"""Benchmark of the SFFT hot path (build_system -> solve -> subtract) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]

One step = one pass of the whole hot path over one seeded
synthetic image pair per GPU.  Default workload: BASELINE.json config 4 (4096x4096 FP64 pair,
17x17 delta-basis kernel, DK=DB=2, 1740 unknowns).  Prints ONE JSON line (contract in the task
statement): whole-job pairs/s with inputs resident in HBM (`value`), the same through the C ABI's
host-buffer entry point with the copies inside the timed region (`e2e`), the roofline of the
dominant kernel, and the CPU oracle timed on a bounded sample (`cpu_baseline`).
For N > 1 (torchrun) every rank processes its own independent pair (weak scaling, no collective
in the data path).
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2109_09334_b200 import synth  # noqa: E402

METRIC = "difference-image pairs/s at 4096^2 FP64 (build+solve+subtract, L=17, DK=DB=2)"
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 FP64 FMA/clk x 2 flop x 1.965 GHz
# dram__bytes_read.sum + dram__bytes_write.sum per launch of each stage's dominant kernel at config 4, from the
# `ncu --set full` capture summarised in profiles/r01_f_final.md (bytes)
NCU_TRAFFIC_CFG4 = {"corr": 545.4e6 + 53.5e6, "rowfft": 268.5e6 + 478.8e6, "subtract": 467.5e6 + 112.4e6}


def shard_units(nunits, rank, world):
    """Contiguous slice [lo, hi) of `nunits` independent pairs owned by `rank` (no data-path collective)."""
    base, rem = divmod(nunits, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def workload_name(cfg_index):
    c = synth.CONFIGS[cfg_index]
    return (f"config{cfg_index}: {c['H']}x{c['W']} FP64 pair, {c['L']}x{c['L']} delta-basis, "
            f"{c['basis']} DK={c['DK']} DB={c['DB']}" + (f", batch {c['batch']}" if c["batch"] > 1 else ""))


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index=0, period=0.02):
        super().__init__(daemon=True)
        self.index, self.period, self.stop_flag = index, period, False
        self.sm, self.reasons, self.sm_max, self.ok = [], set(), None, False
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self.stop_flag:
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        self.stop_flag = True
        if self.is_alive():
            self.join(timeout=1.0)
        if not self.ok or not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["nvml_unavailable"]}
        return {"sm_mhz": float(np.median(self.sm)), "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons),
                "samples": len(self.sm)}


def oracle_sample(cfg_index, pair, crop=1024):
    """The oracle as it stands on a bounded sample of the workload: lag tables + difference on a
    crop x crop corner (cost is linear in pixels -> scaled to the full frame) plus the full-size solve
    of that crop's system (n is the full n).  Returns (seconds per full pair, description, cores)."""
    import oracle
    c = synth.CONFIGS[cfg_index]
    bid = oracle.POLY if c["basis"] == "poly" else oracle.BSPLINE
    R = pair.R if pair.R.ndim == 2 else pair.R[0]
    S = pair.S if pair.S.ndim == 2 else pair.S[0]
    ch, cw = min(crop, c["H"]), min(crop, c["W"])
    Rc, Sc = np.ascontiguousarray(R[:ch, :cw]), np.ascontiguousarray(S[:ch, :cw])
    scale = (c["H"] * c["W"]) / float(ch * cw)
    t0 = time.perf_counter()
    M, rhs = oracle.normal_from_lags(Rc, Sc, c["L"], bid, c["DK"], c["DB"])
    t1 = time.perf_counter()
    coef = oracle.solve(M, rhs)
    t2 = time.perf_counter()
    oracle.difference(Rc, Sc, coef, c["L"], bid, c["DK"], c["DB"])
    t3 = time.perf_counter()
    per_pair = (t1 - t0) * scale + (t2 - t1) + (t3 - t2) * scale
    desc = (f"oracle (direct pixel sums, no FFT) on a {ch}x{cw} crop of the pair: normal system {t1 - t0:.2f}s and "
            f"difference {t3 - t2:.2f}s scaled x{scale:.0f} to the full frame, plus the full n={M.shape[0]} solve {t2 - t1:.2f}s")
    return per_pair * c["batch"], desc, oracle.num_threads()


def run_reference(args):
    """--impl reference: the CPU oracle (this tier has no reference implementation) on the same config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    pair = synth.make_pair(cfg) if synth.CONFIGS[cfg]["batch"] == 1 else synth.make_pair(cfg, subfield=0)
    times, desc, cores = [], "", 1
    for i in range(args.warmup + args.steps):
        sec, desc, cores = oracle_sample(cfg, pair, crop=args.ref_crop)
        if i >= args.warmup:
            times.append(sec)
    sec = float(np.mean(times))
    val = 1.0 / sec
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "pairs/s", "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": workload_name(cfg)},
        "cpu_baseline": {"value": val, "unit": "pairs/s", "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--ref-crop", type=int, default=1024)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-pipelined", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    from paper_2109_09334_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the library has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    cfg = args.config
    c = synth.CONFIGS[cfg]
    nb = c["batch"]
    # every rank owns one independent unit (pair, or batch of sub-fields) per step: weak scaling
    lo, hi = shard_units(world, rank, world)
    assert hi - lo == 1
    pair = synth.make_pair(cfg) if nb == 1 else synth.make_batch(cfg)
    plan = B.Plan(c["H"], c["W"], c["L"], c["DK"], c["DB"], c["basis"], nbatch=nb, device=dev)
    dR = torch.from_numpy(np.ascontiguousarray(pair.R)).to(dev)
    dS = torch.from_numpy(np.ascontiguousarray(pair.S)).to(dev)
    dD = torch.empty_like(dS)
    coef = torch.empty((nb, plan.n), dtype=torch.float64, device=dev)

    def step():
        plan.build_system(dR, dS)
        plan.solve(coef)
        plan.subtract(coef, dR, dS, dD)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        step()
    plan.status()
    # ---- timed region: device-resident inputs, CUDA events on the launching stream ----
    sampler = ClockSampler(index=local)
    barrier()
    sampler.start()
    launches0 = plan.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    clocks = sampler.result()
    ms_total = ev0.elapsed_time(ev1)
    launches = plan.launch_count() - launches0
    plan.status()
    # per-stage times from a second, untimed pass with the library's event marks on (stages then run serialised:
    # the moment stage is not forked beside the lag correlation, so the stage sum exceeds ms_per_step slightly)
    psteps = max(3, min(args.steps, 10))
    plan.profile(psteps)
    for _ in range(psteps):
        step()
    stage_ms = plan.profile_read(psteps).mean(axis=0)
    plan.profile(0)
    plan.status()
    t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item()) / args.steps
    value = world * nb / (ms_step * 1e-3)

    # ---- two pairs in flight (informational, not the headline): a second plan on a second stream, so that one
    # pair's latency-bound solve overlaps the other's tensor-bound lag correlation ----
    pipelined = None
    if nb == 1 and not args.no_pipelined:
        s2 = torch.cuda.Stream(device=dev)
        with torch.cuda.stream(s2):
            plan2 = B.Plan(c["H"], c["W"], c["L"], c["DK"], c["DB"], c["basis"], nbatch=nb, device=dev)
            dR2, dS2, dD2, coef2 = dR.clone(), dS.clone(), torch.empty_like(dS), torch.empty_like(coef)

        def step2():
            step()
            with torch.cuda.stream(s2):
                plan2.build_system(dR2, dS2)
                plan2.solve(coef2)
                plan2.subtract(coef2, dR2, dS2, dD2)

        for _ in range(3):
            step2()
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            step2()
        barrier()
        tp = torch.tensor([(time.perf_counter() - t0) / args.steps], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(tp, op=dist.ReduceOp.MAX)
        plan2.status()
        plan2.close()
        pipelined = {"pairs_in_flight": 2, "value": world * 2 * nb / float(tp.item()), "unit": "pairs/s",
                     "note": "two plans on two streams, wall clock around K double steps; not the headline value"}

    # ---- end to end through sfft_run_host: pinned host buffers, H2D + D2H inside the timed region ----
    hR = torch.from_numpy(np.ascontiguousarray(pair.R)).pin_memory()
    hS = torch.from_numpy(np.ascontiguousarray(pair.S)).pin_memory()
    hD = torch.empty_like(hR).pin_memory()
    hC = torch.empty((nb, plan.n), dtype=torch.float64).pin_memory()
    e2e_steps = max(3, min(args.steps, 20))

    def e2e_submit():
        st = B.sfft_run_host_async(plan.h, hR.data_ptr(), hS.data_ptr(), hD.data_ptr(), hC.data_ptr())
        if st != B.SFFT_OK:
            raise B.SfftError(st, "sfft_run_host_async")

    def e2e_wait():
        st = B.sfft_run_host_wait(plan.h)
        if st != B.SFFT_OK:
            raise B.SfftError(st, "sfft_run_host_wait")

    e2e_submit()
    e2e_wait()
    barrier()
    # every step copies its inputs from pinned host memory and its result back; consecutive steps are submitted
    # back to back (sfft_run_host_async), so the copies of one pair overlap the compute of the previous one;
    # the clock stops after the last result has arrived (sfft_run_host_wait)
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_submit()
    e2e_wait()
    barrier()
    e2e_s = torch.tensor([(time.perf_counter() - t0) / e2e_steps], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
    # the same with one call at a time (sfft_run_host: copy in, compute, copy out, synchronise)
    t0 = time.perf_counter()
    for _ in range(3):
        st = B.sfft_run_host(plan.h, hR.data_ptr(), hS.data_ptr(), hD.data_ptr(), hC.data_ptr())
        if st != B.SFFT_OK:
            raise B.SfftError(st, "sfft_run_host")
    e2e_sync_val = world * nb / ((time.perf_counter() - t0) / 3)
    e2e_val = world * nb / float(e2e_s.item())
    img_bytes = nb * c["H"] * c["W"] * 8

    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        names = B.STAGE_NAMES
        stages = {names[i]: round(float(stage_ms[i]), 4) for i in range(len(names))}
        top = int(np.argmax(stage_ms))
        # algorithmic work of each stage per pair; P pixels, FP64
        P = c["H"] * c["W"]
        nKa = (c["DK"] + 1) if c["basis"] == "poly" else (c["DK"] + 4)
        FK = (c["DK"] + 1) * (c["DK"] + 2) // 2 if c["basis"] == "poly" else nKa * nKa
        L = c["L"]
        hbm_peak = peaks.get("hbm_gbs", 6650.0)
        peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback"
        alg = {
            # row FFT: read R (nKa times, L2-served after the first) + S, write nKa+1 half spectra
            "rowfft": ("hbm", (2 * P * 8 + (nKa + 1) * P * 8) * nb / 1e9, hbm_peak, "GB/s"),
            # lag correlation: SURVEY 8(d) pruned-FFT figure ~ (FK(FK+1)/2 + FK) maps x columns x 5 N log2 N x 0.6
            "corr": ("alu", (FK * (FK + 1) // 2 + FK) * (c["W"] // 2 + 1) * 5.0 * c["H"] * np.log2(c["H"]) * 0.6 * nb / 1e12,
                     FP64_PEAK_TFLOPS, "TFLOP/s"),
            # subtract: SURVEY 8(d) Fourier-route figure, L*FK complex MACs per spectrum point (8 flop each)
            "subtract": ("alu", 8.0 * L * FK * c["H"] * (c["W"] // 2) * nb / 1e12, FP64_PEAK_TFLOPS, "TFLOP/s"),
            "solve": ("alu", (plan.n ** 3 / 3.0) * nb / 1e12, FP64_PEAK_TFLOPS, "TFLOP/s"),
        }
        tname = names[top]
        bound, work, peak, unit = alg.get(tname, ("hbm", 0.0, hbm_peak, "GB/s"))
        achieved = work / (stage_ms[top] * 1e-3)
        roofline = {"kernel": tname, "bound": bound, "achieved": achieved, "peak": peak, "unit": unit,
                    "frac": achieved / peak, "traffic": NCU_TRAFFIC_CFG4.get(tname) if cfg == 4 else None,
                    "ms": float(stage_ms[top]),
                    "peak_source": peak_src if bound == "hbm" else "derived: 148 SM x 64 FP64 FMA/clk x 1.965 GHz"}
        if tname == "corr":
            # the x-direction is executed as direct lag sums on the FP64 tensor cores: DMMA flops actually issued
            ex = plan.corr_executed_flops() * nb
            st_dm, dmma = B.sfft_measure_fp64_peak(1)
            roofline["executed_tflops"] = ex / 1e12 / (stage_ms[top] * 1e-3)
            roofline["dmma_peak_measured_tflops"] = dmma if st_dm == B.SFFT_OK else None
        rf_all = {}
        for nm, (bd, wk, pk, un) in alg.items():
            t_ms = stage_ms[names.index(nm)]
            if t_ms > 0:
                rf_all[nm] = {"bound": bd, "achieved": round(wk / (t_ms * 1e-3), 3), "peak": round(pk, 1), "unit": un,
                              "frac": round(wk / (t_ms * 1e-3) / pk, 4)}
        line = {
            "metric": METRIC, "value": value, "unit": "pairs/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "l2": "inputs and intermediates (>= 0.8 GB per step) exceed the 126 MB L2",
                       "unknowns": plan.n, "pairs_per_step_per_gpu": nb},
            "e2e": {"value": e2e_val, "unit": "pairs/s", "h2d_bytes_per_step": 2 * img_bytes,
                    "d2h_bytes_per_step": img_bytes + nb * plan.n * 8, "steps": e2e_steps,
                    "api": "sfft_run_host_async x steps + sfft_run_host_wait (two staging slots, copy streams)",
                    "one_call_at_a_time": e2e_sync_val},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": roofline,
            "stage_roofline": rf_all,
            "pipelined": pipelined,
            "stage_ms": stages,
        }
        if not args.no_cpu_baseline and world == 1:
            sec, desc, cores = oracle_sample(cfg, pair, crop=args.ref_crop)
            line["cpu_baseline"] = {"value": 1.0 / sec, "unit": "pairs/s", "cores": cores, "kind": "oracle", "sample": desc}
        print(json.dumps(line))
    plan.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
