#!/usr/bin/env python
"""Benchmark of the SFFT hot path (build_system -> solve -> subtract) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C] [--no-compare]

One step = one pass of the whole hot path over one seeded
synthetic image pair per GPU.  Default workload: BASELINE.json config 4 (4096x4096 FP64 pair,
17x17 delta-basis kernel, DK=DB=2, 1740 unknowns).  Prints ONE JSON line (contract in the task
statement): whole-job pairs/s with inputs resident in HBM (`value`), the same through the C ABI's
host-buffer entry point with the copies inside the timed region (`e2e`), the roofline of the
dominant kernel, the CPU oracle timed on the full pair (`cpu_baseline`), and library comparison
points (cuFFT / cuSOLVER through torch, never linked into libsfft_b200.so) under `comparison`.
For N > 1 (torchrun): configs 1-4, every rank processes its own independent pair (weak scaling);
config 5, the 64 sub-fields of the batch are cut into contiguous slices, one per rank (strong
scaling).  No collective in the data path either way.
"""
import argparse
import ctypes
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import synth  # noqa: E402

FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 FP64 FMA/clk x 2 flop x 1.965 GHz
# dram__bytes_read.sum + dram__bytes_write.sum per launch of each stage's dominant kernel at config 4, from the
# committed `ncu --set full` capture named in NCU_TRAFFIC_SOURCE (bytes).  Not measured by this run: the line
# carries the source beside the number.
NCU_TRAFFIC_CFG4 = {"rowfft": 268.5e6 + 480.8e6, "subtract": 468.1e6 + 114.5e6, "corr": 539.5e6 + 27.5e6,
                    "subtract_inverse": 268.6e6 + 104.5e6}
_R03 = "profiles/r03_final.md (ncu --set full capture at commit c0f72b4)"
NCU_TRAFFIC_SOURCE = {"rowfft": _R03, "subtract": _R03 + " (k_fir_x)", "corr": _R03 + " (k_corr_os)",
                      "subtract_inverse": _R03 + " (k_rowfft_inverse_sub)"}
REFERENCE_BUDGET_S = 200.0      # wall-clock cap of the --impl reference arm (the oracle is slow by construction)


# BASELINE.json's five configs plus the paper's own CCD frame (DECam, 2046 x 4094 pixels, neither a
# power of two), rendered with the config-3 recipe and fitted with the config-3 model: `--config decam` (or 6).
DECAM = 6
CONFIGS = dict(synth.CONFIGS)
CONFIGS[DECAM] = dict(synth.CONFIGS[3], H=2046, W=4094, recipe=3)


def make_bench_pair(cfg_index, **kw):
    c = CONFIGS[cfg_index]
    if "recipe" in c:
        return synth.make_pair(c["recipe"], H=c["H"], W=c["W"], **kw)
    return synth.make_pair(cfg_index, **kw)


def parse_config(text):
    return DECAM if str(text).lower() == "decam" else int(text)


def metric_name(cfg_index):
    c = CONFIGS[cfg_index]
    size = f"{c['H']}x{c['W']}" if c["H"] != c["W"] else f"{c['H']}^2"
    what = "difference-image pairs/s" if c["batch"] == 1 else f"sub-field pairs/s (batch of {c['batch']} per call)"
    return f"{what} at {size} FP64 (build+solve+subtract, L={c['L']}, {c['basis']} DK={c['DK']} DB={c['DB']})"


def shard_units(nunits, rank, world):
    """Contiguous slice [lo, hi) of `nunits` independent pairs owned by `rank` (no data-path collective)."""
    base, rem = divmod(nunits, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def rank_units(cfg_index, rank, world):
    """Units (pairs / sub-fields) rank `rank` of `world` processes per step, as (first, count, scaling):
    a single-pair config gives every rank its own pair (weak); the config-5 batch is sliced (strong)."""
    nb = CONFIGS[cfg_index]["batch"]
    if nb == 1:
        return rank, 1, "weak"
    lo, hi = shard_units(nb, rank, world)
    return lo, hi - lo, "strong"


L2_BYTES = 126e6


def step_footprint_bytes(cfg_index, nb=None):
    """Bytes one step touches at least: the images R, S, D and the row-spectrum stack (nKa + 1 half spectra)."""
    c = CONFIGS[cfg_index]
    nb = c["batch"] if nb is None else nb
    nKa = c["DK"] + 1 if c["basis"] == "poly" else c["DK"] + 4
    return nb * c["H"] * c["W"] * 8.0 * (3 + nKa + 1)


def needs_l2_flush(cfg_index, nb=None):
    return step_footprint_bytes(cfg_index, nb) < 2 * L2_BYTES


def config_dict(cfg_index):
    """The `config` object of the JSON line: the same for both arms (it names the workload and the timing protocol)."""
    c = CONFIGS[cfg_index]
    fp = step_footprint_bytes(cfg_index)
    l2 = ("L2 flushed between timed steps (a 256 MB device buffer is overwritten; each step is timed by its own pair of "
          "CUDA events)" if needs_l2_flush(cfg_index)
          else f"inputs and intermediates (>= {fp / 1e9:.2f} GB per step) exceed the 126 MB L2: no flush")
    nterm = lambda D: (D + 1) * (D + 2) // 2 if c["basis"] == "poly" else (D + 4) ** 2
    return {"workload": workload_name(cfg_index), "l2": l2, "unknowns": nterm(c["DK"]) * c["L"] ** 2 + nterm(c["DB"]),
            "pair": "fit and apply on the same pair (GPU arm: the subtract reuses the row spectra of the build, "
                    "sfft_plan_set_reuse_spectra)"}


def workload_name(cfg_index):
    c = CONFIGS[cfg_index]
    name = "DECam CCD frame (PAPER.md:393), config-3 recipe and model" if cfg_index == DECAM else f"config{cfg_index}"
    return (f"{name}: {c['H']}x{c['W']} FP64 pair, {c['L']}x{c['L']} delta-basis, "
            f"{c['basis']} DK={c['DK']} DB={c['DB']}" + (f", batch {c['batch']}" if c["batch"] > 1 else ""))


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index=0, period=0.005):
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


def oracle_pass(cfg_index, pair, crop=None):
    """One pass of the oracle as it stands (direct pixel sums, no FFT: normal system, solve, full difference image).
    crop = None: the FULL pair (single-pair configs) -- a measurement, not an extrapolation.  crop = c: a c x c corner,
    its pixel-proportional parts scaled to the full frame plus the full-n solve (labelled fallback for the
    batch-of-64 config, whose full oracle pass takes hours).  Returns (seconds per unit of the workload,
    description, cores)."""
    import oracle
    c = CONFIGS[cfg_index]
    bid = oracle.POLY if c["basis"] == "poly" else oracle.BSPLINE
    R = pair.R if pair.R.ndim == 2 else pair.R[0]
    S = pair.S if pair.S.ndim == 2 else pair.S[0]
    if crop is None:
        t0 = time.perf_counter()
        M, rhs = oracle.normal_from_lags(R, S, c["L"], bid, c["DK"], c["DB"])
        t1 = time.perf_counter()
        coef = oracle.solve(M, rhs)
        t2 = time.perf_counter()
        oracle.difference(R, S, coef, c["L"], bid, c["DK"], c["DB"])
        t3 = time.perf_counter()
        desc = (f"oracle (direct pixel sums, no FFT) on the FULL {c['H']}x{c['W']} pair: normal system {t1 - t0:.2f}s, "
                f"n={M.shape[0]} solve {t2 - t1:.2f}s, difference image {t3 - t2:.2f}s")
        return t3 - t0, desc, oracle.num_threads()
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
    per_unit = (t1 - t0) * scale + (t2 - t1) + (t3 - t2) * scale
    desc = (f"EXTRAPOLATED: oracle on a {ch}x{cw} crop of one sub-field: normal system {t1 - t0:.2f}s and difference "
            f"{t3 - t2:.2f}s scaled x{scale:.0f} to the full frame, plus the full n={M.shape[0]} solve {t2 - t1:.2f}s")
    return per_unit, desc, oracle.num_threads()


def oracle_crop_for(cfg_index):
    return None if CONFIGS[cfg_index]["batch"] == 1 else 256


def run_reference(args):
    """--impl reference: the CPU oracle (this tier has no reference implementation) on the same config.
    A step is one full oracle pass over the pair; the oracle is slow by construction, so the arm stops after
    REFERENCE_BUDGET_S of wall clock and prints the number of steps and warm-ups it ACTUALLY ran."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    single = CONFIGS[cfg]["batch"] == 1
    pair = make_bench_pair(cfg) if single else synth.make_pair(cfg, subfield=0)
    crop = args.ref_crop if args.ref_crop > 0 else oracle_crop_for(cfg)
    t_begin = time.perf_counter()
    times, warm_done = [], 0
    t0 = time.perf_counter()
    sec, desc, cores = oracle_pass(cfg, pair, crop)
    wall = time.perf_counter() - t0           # wall clock of one pass (what the budget is counted in)
    if args.warmup > 0 and 3.0 * wall < REFERENCE_BUDGET_S:
        warm_done = 1                          # the first pass was a warm-up: more passes still fit
        while warm_done < args.warmup and wall < 10.0 and (time.perf_counter() - t_begin) + 2.0 * wall < REFERENCE_BUDGET_S:
            oracle_pass(cfg, pair, crop)       # further warm-ups only while passes are short
            warm_done += 1
    else:
        times.append(sec)                      # a pass is so long that the first one is the measurement
    while len(times) < args.steps and (not times or (time.perf_counter() - t_begin) + wall < REFERENCE_BUDGET_S):
        sec, desc, cores = oracle_pass(cfg, pair, crop)
        times.append(sec)
    sec = float(np.mean(times))
    val = 1.0 / sec
    line = {
        "impl": "reference", "metric": metric_name(cfg), "value": val, "unit": "pairs/s", "n_gpus": args.gpus,
        "steps": len(times), "warmup": warm_done, "steps_requested": args.steps, "warmup_requested": args.warmup,
        "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak" if single else "strong",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_dict(cfg),
        "cpu_baseline": {"value": val, "unit": "pairs/s", "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def load_bench_lib():
    """libsfft_bench.so: FP64 peak probes and flop counters (csrc/bench/, measurement support only)."""
    from paper_2109_09334_b200 import build as libbuild
    L = ctypes.CDLL(libbuild.build_bench_library())
    L.sfft_bench_fp64_peak.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
    L.sfft_bench_corr_flops.argtypes = [ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    return L


def time_cuda(torch, fn, reps=5, warm=2):
    """Median device time (ms) of fn() by CUDA events on the current stream."""
    for _ in range(warm):
        fn()
    ts = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1))
    return float(np.median(ts))


def library_comparison(torch, dev, c, nb, n, stage_ms):
    """Vendor-library comparison points in the same run, same clocks (SURVEY.md 8(d) "Timing protocol"):
    cuFFT batched D2Z / Z2D of the row-transform shape and cuSOLVER potrf + potrs at the solve's size,
    both through torch (comparison only; nothing here is linked into or called by libsfft_b200.so)."""
    out = {"note": "cuFFT / cuSOLVER via torch.fft / torch.linalg, timed with CUDA events; comparison points only"}
    nKa = (c["DK"] + 1) if c["basis"] == "poly" else (c["DK"] + 4)
    try:
        nimg = min(nKa + 1, 8) * min(nb, 8)
        x = torch.randn((nimg, c["H"], c["W"]), dtype=torch.float64, device=dev)
        t_f = time_cuda(torch, lambda: torch.fft.rfft(x, dim=-1))
        X = torch.fft.rfft(x, dim=-1)
        t_i = time_cuda(torch, lambda: torch.fft.irfft(X[:1], n=c["W"], dim=-1))
        byts = nimg * c["H"] * c["W"] * 8 * 2.0
        out["cufft_d2z_rows"] = {"shape": [nimg, c["H"], c["W"]], "ms": t_f, "gbs": byts / (t_f * 1e-3) / 1e9,
                                 "ours_ms_same_transform_count": float(stage_ms[0]) * nimg / ((nKa + 1) * nb),
                                 "note": "unweighted batched 1-D D2Z; ours also applies the y-weights and writes "
                                         "nKa+1 spectra from 2 images"}
        out["cufft_z2d_rows"] = {"shape": [1, c["H"], c["W"]], "ms": t_i,
                                 "note": "one image; ours fuses D = S - model - background into this transform"}
        del x, X
    except Exception as e:   # a comparison point must never take the benchmark down
        out["cufft_error"] = repr(e)[:200]
    try:
        try:
            torch.backends.cuda.preferred_linalg_library("cusolver")
        except Exception:
            pass
        k = nb if nb * n * n * 8.0 * 3 < 60e9 else 1
        g = torch.Generator(device=dev).manual_seed(7)
        A = torch.randn((k, n, n + 16), dtype=torch.float64, device=dev, generator=g)
        Msp = A @ A.transpose(-1, -2)
        b = torch.randn((k, n, 1), dtype=torch.float64, device=dev, generator=g)
        del A

        def potrf_potrs():
            Lc = torch.linalg.cholesky(Msp)
            return torch.cholesky_solve(b, Lc)

        t_s = time_cuda(torch, potrf_potrs, reps=3, warm=1)
        out["cusolver_potrf_potrs"] = {"n": n, "systems": k, "ms": t_s, "ms_per_system": t_s / k,
                                       "ours_ms_per_system": float(stage_ms[5]) / nb}
        del Msp, b
    except Exception as e:
        out["cusolver_error"] = repr(e)[:200]
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=parse_config, default=4, help="1..5 (BASELINE.json configs), or decam (2046x4094)")
    ap.add_argument("--ref-crop", type=int, default=0, help="time the oracle on a crop (0: full pair; config 5: 256)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-pipelined", action="store_true")
    ap.add_argument("--no-compare", action="store_true")
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
    c = CONFIGS[cfg]
    first, nb, scaling = rank_units(cfg, rank, world)
    total_units = world if c["batch"] == 1 else c["batch"]
    if nb < 1:
        raise SystemExit(f"bench.py: rank {rank} of {world} has no unit of config {cfg}")
    if c["batch"] == 1:
        pair = make_bench_pair(cfg)
    else:
        pair = synth.make_batch(cfg, nbatch=nb, first=first, workers=min(16, os.cpu_count() or 1))
    # fit and apply on the same pair: the subtract may reuse the build's row spectra (explicit opt-in)
    plan = B.Plan(c["H"], c["W"], c["L"], c["DK"], c["DB"], c["basis"], nbatch=nb, device=dev, reuse_spectra=True)
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
    if needs_l2_flush(cfg, nb):
        # small configs fit the 126 MB L2: a 256 MB buffer is overwritten between the timed steps, and every step
        # lies between its own pair of events (the flush is outside them)
        flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for ea, eb in evs:
            flush.fill_(1)
            ea.record()
            step()
            eb.record()
        barrier()
        clocks = sampler.result()
        ms_total = sum(ea.elapsed_time(eb) for ea, eb in evs)
        del flush
    else:
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
    value = total_units / (ms_step * 1e-3)

    # ---- the same step captured once in a CUDA graph and replayed (informational, not the headline): the 46 launches
    # of a step, the side-stream fork / join and the programmatic dependent launches of the panel chain are all
    # capturable; replay removes most of the inter-kernel gaps ----
    graph_info = None
    if world == 1 and not args.no_pipelined:
        try:
            gs = torch.cuda.Stream(device=dev)
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.stream(gs):
                B.sfft_plan_set_stream(plan.h, gs.cuda_stream)
                step()
                torch.cuda.synchronize(dev)
                graph.capture_begin()
                step()
                graph.capture_end()
            torch.cuda.synchronize(dev)
            for _ in range(3):
                graph.replay()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(dev)
            g0.record()
            for _ in range(args.steps):
                graph.replay()
            g1.record()
            torch.cuda.synchronize(dev)
            gms = g0.elapsed_time(g1) / args.steps
            graph_info = {"ms_per_step": gms, "value": nb / (gms * 1e-3), "unit": "pairs/s",
                          "note": "one captured step replayed with cudaGraphLaunch; not the headline value"}
            del graph
        except Exception as ex:          # capture is informational: report, do not fail the run
            graph_info = {"error": repr(ex)[:200]}
        finally:
            B.sfft_plan_set_stream(plan.h, plan.stream.cuda_stream)
            torch.cuda.synchronize(dev)
        plan.status()

    # ---- two pairs in flight (informational, not the headline): a second plan on a second stream, so that one
    # pair's latency-bound solve overlaps the other's FP64-bound lag correlation ----
    pipelined = None
    if c["batch"] == 1 and not args.no_pipelined:
        s2 = torch.cuda.Stream(device=dev)
        with torch.cuda.stream(s2):
            plan2 = B.Plan(c["H"], c["W"], c["L"], c["DK"], c["DB"], c["basis"], nbatch=nb, device=dev,
                           reuse_spectra=True)
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
        del dR2, dS2, dD2
        pipelined = {"pairs_in_flight": 2, "value": world * 2 * nb / float(tp.item()), "unit": "pairs/s",
                     "note": "two plans on two streams, wall clock around K double steps; not the headline value"}

    def time_steps(fn, steps, warm=3):
        """ms per call of fn over `steps` back-to-back calls, CUDA events on the current stream, after `warm` calls."""
        for _ in range(warm):
            fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(dev)
        a.record()
        for _ in range(steps):
            fn()
        b.record()
        torch.cuda.synchronize(dev)
        return a.elapsed_time(b) / steps

    # ---- the paper's two-step flow, beside the headline and never instead of it: mask the
    # saturated sources and fill them with the local background, fit on the masked pair, apply to the ORIGINAL pair.
    # The subtract cannot reuse the build's spectra here (they are the masked reference's): reuse_spectra = False ----
    masked_flow = None
    if world == 1 and c["batch"] == 1 and not args.no_pipelined:
        sat = 3000.0
        planm = B.Plan(c["H"], c["W"], c["L"], c["DK"], c["DB"], c["basis"], nbatch=1, device=dev, reuse_spectra=False)
        dRm, dSm = torch.empty_like(dR), torch.empty_like(dS)
        dmask = torch.empty(dR.shape, dtype=torch.uint8, device=dev)

        def masked_step():
            st = B.sfft_mask_fill(planm.h, dR.data_ptr(), dS.data_ptr(), sat, sat, 2, 6, dRm.data_ptr(), dSm.data_ptr(),
                                  dmask.data_ptr())
            if st != B.SFFT_OK:
                raise B.SfftError(st, "sfft_mask_fill")
            planm.build_system(dRm, dSm)
            planm.solve(coef)
            planm.subtract(coef, dR, dS, dD)

        mms = time_steps(masked_step, args.steps)
        planm.status()
        masked_flow = {"ms_per_step": mms, "value": 1.0 / (mms * 1e-3), "unit": "pairs/s",
                       "masked_pixels": int(dmask.sum().item()), "saturation_adu": sat, "grow_px": 2, "fill_half_window_px": 6,
                       "api": "sfft_mask_fill -> sfft_build_system(masked pair) -> sfft_solve -> sfft_subtract(original "
                              "pair), reuse_spectra = 0 (the reference is transformed again)"}
        planm.close()
        del dRm, dSm, dmask

    # ---- several pairs per call through the batch axis (single-pair configs): the dependent panel chain of the
    # solve is shared by the batch.  Entries are circular shifts of the pair (the model is circular: same fit) ----
    batched = None
    if world == 1 and c["batch"] == 1 and not args.no_pipelined:
        batched = {}
        for nbat in (2, 4):
            planb = B.Plan(c["H"], c["W"], c["L"], c["DK"], c["DB"], c["basis"], nbatch=nbat, device=dev, reuse_spectra=True)
            bR = torch.stack([torch.roll(dR, shifts=(17 * e, 29 * e), dims=(0, 1)) for e in range(nbat)]).contiguous()
            bS = torch.stack([torch.roll(dS, shifts=(17 * e, 29 * e), dims=(0, 1)) for e in range(nbat)]).contiguous()
            bD, bC = torch.empty_like(bS), torch.empty((nbat, planb.n), dtype=torch.float64, device=dev)

            def batch_step():
                planb.build_system(bR, bS)
                planb.solve(bC)
                planb.subtract(bC, bR, bS, bD)

            bms = time_steps(batch_step, max(3, args.steps // 2))
            planb.status()
            batched[f"nbatch{nbat}"] = {"ms_per_call": bms, "value": nbat / (bms * 1e-3), "unit": "pairs/s"}
            planb.close()
            del bR, bS, bD, bC
        batched["note"] = "one plan, nbatch pairs per build/solve/subtract call; not the headline value"

    # ---- end to end through sfft_run_host: pinned host buffers, H2D + D2H inside the timed region ----
    hR = torch.from_numpy(np.ascontiguousarray(pair.R)).pin_memory()
    hS = torch.from_numpy(np.ascontiguousarray(pair.S)).pin_memory()
    hD = torch.empty_like(hR).pin_memory()
    hC = torch.empty((nb, plan.n), dtype=torch.float64).pin_memory()
    e2e_steps = max(3, min(args.steps, 20))
    plan.ensure_host_staging()

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
    e2e_sync_val = total_units / ((time.perf_counter() - t0) / 3)
    e2e_val = total_units / float(e2e_s.item())
    img_bytes = nb * c["H"] * c["W"] * 8
    # ---- the same with FP32 storage on the host (FP64 arithmetic unchanged): half the bytes over PCIe.  A second
    # figure beside the FP64 one, never instead of it ----
    hR32, hS32 = hR.to(torch.float32).pin_memory(), hS.to(torch.float32).pin_memory()
    hD32 = torch.empty_like(hR32).pin_memory()

    def e2e32_submit():
        st = B.sfft_run_host_async_f32(plan.h, hR32.data_ptr(), hS32.data_ptr(), hD32.data_ptr(), hC.data_ptr())
        if st != B.SFFT_OK:
            raise B.SfftError(st, "sfft_run_host_async_f32")

    e2e32_submit()
    e2e_wait()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e32_submit()
    e2e_wait()
    barrier()
    e2e32_s = torch.tensor([(time.perf_counter() - t0) / e2e_steps], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(e2e32_s, op=dist.ReduceOp.MAX)
    e2e32_val = total_units / float(e2e32_s.item())
    del hR32, hS32, hD32

    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        names = B.STAGE_NAMES
        stages = {names[i]: round(float(stage_ms[i]), 4) for i in range(len(names))}
        top = int(np.argmax(stage_ms[:8]))          # (entries 8, 9 are the two halves of stage 7)
        # algorithmic work of each stage per pair; P pixels, FP64
        P = c["H"] * c["W"]
        nKa = (c["DK"] + 1) if c["basis"] == "poly" else (c["DK"] + 4)
        FK = (c["DK"] + 1) * (c["DK"] + 2) // 2 if c["basis"] == "poly" else nKa * nKa
        L = c["L"]
        hbm_peak = peaks.get("hbm_gbs", 6650.0)
        peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback"
        alg = {
            # row FFT: read R and S once, write nKa+1 half spectra
            "rowfft": ("hbm", (2 * P * 8 + (nKa + 1) * P * 8) * nb / 1e9, hbm_peak, "GB/s"),
            # lag correlation: SURVEY 8(d) pruned-FFT figure ~ (FK(FK+1)/2 + FK) maps x columns x 5 N log2 N x 0.6
            "corr": ("alu", (FK * (FK + 1) // 2 + FK) * (c["W"] // 2 + 1) * 5.0 * c["H"] * np.log2(c["H"]) * 0.6 * nb / 1e12,
                     FP64_PEAK_TFLOPS, "TFLOP/s"),
            # gather: one write of the n x n matrix
            "gather": ("hbm", plan.ns * plan.ns * 8.0 * nb / 1e9, hbm_peak, "GB/s"),
            # subtract: SURVEY 8(d) Fourier-route figure, L*FK complex MACs per spectrum point (8 flop each)
            "subtract": ("alu", 8.0 * L * FK * c["H"] * (c["W"] // 2) * nb / 1e12, FP64_PEAK_TFLOPS, "TFLOP/s"),
            "solve": ("alu", (plan.ns ** 3 / 3.0) * nb / 1e12, FP64_PEAK_TFLOPS, "TFLOP/s"),
            # inverse row transforms fused with the difference: read the filtered half spectrum and S, write D
            "subtract_inverse": ("hbm", 3 * P * 8.0 * nb / 1e9, hbm_peak, "GB/s"),
        }
        tname = names[top]
        bound, work, peak, unit = alg.get(tname, ("hbm", 0.0, hbm_peak, "GB/s"))
        achieved = work / (stage_ms[top] * 1e-3)
        roofline = {"kernel": tname, "bound": bound, "achieved": achieved, "peak": peak, "unit": unit,
                    "frac": achieved / peak, "traffic": NCU_TRAFFIC_CFG4.get(tname) if cfg == 4 else None,
                    "traffic_source": NCU_TRAFFIC_SOURCE.get(tname) if cfg == 4 else None,
                    "ms": float(stage_ms[top]),
                    "peak_source": peak_src if bound == "hbm" else "derived: 148 SM x 64 FP64 FMA/clk x 1.965 GHz"}
        blib = None
        try:
            blib = load_bench_lib()
        except Exception as e:
            roofline["bench_lib_error"] = repr(e)[:200]
        if blib is not None:
            ex, tc = ctypes.c_double(0.0), ctypes.c_double(0.0)
            if blib.sfft_bench_corr_flops(plan.h, ctypes.byref(ex), ctypes.byref(tc)) == 0:
                t_corr = stage_ms[names.index("corr")] * 1e-3
                roofline["corr_executed_tflops"] = ex.value * nb / 1e12 / t_corr
                roofline["corr_executed_gflop"] = ex.value * nb / 1e9
            pk = ctypes.c_double(0.0)
            for kind, key in ((0, "dfma_peak_measured_tflops"), (1, "dmma_peak_measured_tflops")):
                roofline[key] = pk.value if blib.sfft_bench_fp64_peak(kind, ctypes.byref(pk)) == 0 else None
        rf_all = {}
        for nm, (bd, wk, pk, un) in alg.items():
            t_ms = stage_ms[names.index(nm)]
            if t_ms > 0:
                rf_all[nm] = {"bound": bd, "achieved": round(wk / (t_ms * 1e-3), 3), "peak": round(pk, 1), "unit": un,
                              "frac": round(wk / (t_ms * 1e-3) / pk, 4)}
        line = {
            "metric": metric_name(cfg), "value": value, "unit": "pairs/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": scaling,
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(cfg), "pairs_per_step_per_gpu": nb,
            "e2e": {"value": e2e_val, "unit": "pairs/s", "h2d_bytes_per_step": 2 * img_bytes,
                    "d2h_bytes_per_step": img_bytes + nb * plan.n * 8, "steps": e2e_steps,
                    "api": "sfft_run_host_async x steps + sfft_run_host_wait (two staging slots, copy streams)",
                    "one_call_at_a_time": e2e_sync_val,
                    "f32_storage": {"value": e2e32_val, "unit": "pairs/s", "h2d_bytes_per_step": img_bytes,
                                    "d2h_bytes_per_step": img_bytes // 2 + nb * plan.n * 8,
                                    "api": "sfft_run_host_async_f32: float images on the host, FP64 arithmetic on the device"}},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": roofline,
            "stage_roofline": rf_all,
            "pipelined": pipelined, "cuda_graph": graph_info, "masked_flow": masked_flow, "batched": batched,
            "stage_ms": stages,
        }
        if not args.no_compare and world == 1:
            del hR, hS, hD
            line["comparison"] = library_comparison(torch, dev, c, nb, plan.ns, stage_ms)
        if not args.no_cpu_baseline and world == 1:
            crop = args.ref_crop if args.ref_crop > 0 else oracle_crop_for(cfg)
            sec, desc, cores = oracle_pass(cfg, pair, crop)
            line["cpu_baseline"] = {"value": 1.0 / sec, "unit": "pairs/s", "cores": cores, "kind": "oracle", "sample": desc}
        print(json.dumps(line))
    plan.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
