#!/usr/bin/env python
"""bench.py -- one JSON line for the qsGW Sigma^c build on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload xl|large|medium|small|tiny] [--shard replicas|poles]
  python bench.py --impl reference ...      # the CPU oracle timed on the host cores (bounded sample per step)

A "step" is one pass of the whole hot path -- pack, stage 1, stage 2, stage 3 for every pole chunk, and
the epilogue -- i.e. one Sigma^c build through the C ABI on seeded synthetic inputs of the named BASELINE.json config.
The default workload is `xl`, the largest single-GPU configuration (BASELINE.json's metric names no config); its Z
(130 GB) is produced range by range on the device and fed through qsgw_sigma_begin / _add_poles / _finish.
`value` = F_min / t in TFLOP/s (F_min = F1 + F2sym + F3, the least dense FP64 work the method needs,
so the figure cannot be inflated by redundant work); `ms_per_step` = ms per build.  Inputs are resident in HBM for
`value`; `e2e` repeats the build through qsgw_sigma_build_host with pinned HOST buffers, H2D/D2H copies inside the timed
region.  Every number in the line is measured in this run (the FP64 roofline is cross-checked by an in-run probe); the
one exception, `roofline.traffic`, is the DRAM byte count of a committed ncu capture and names the file it comes from.

N > 1: `--shard replicas` (default): every rank builds its own Sigma (seed + rank), the only collectives
are the timing barrier and the max-over-ranks of the time, "scaling": "weak".  `--shard poles`: ONE
Sigma, rank r builds the pole slice qsgw_sigma_pole_slice gives it and one all-reduce of the N x N matrix finishes the
build, "scaling": "strong".
"""
from __future__ import annotations

import argparse
import ctypes
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "sigma_c_build_fp64_tflops"
UNIT = "TFLOP/s"
# FP64 pipe of sm_100a: DMMA.8x8x4 and DFMA both retire 64 FMA/clk/SM (checked in every run by the probe below)
FP64_FMA_PER_CLK_PER_SM = 64
# dram__bytes_read.sum + dram__bytes_write.sum of ONE stage-2 launch over a full s-block, from committed `ncu --set full`
# summaries (recorded numbers, not measurements of this run; the JSON line names the file)
NCU_STAGE2_DRAM_BYTES_PER_LAUNCH = {
    "xl": (196.99e9, "profiles/r02_full_xl.md"),          # 164.22 GB read + 32.77 GB written
    "large": (29.95e9, "profiles/r02_full_large.md"),    # 18.17 GB read + 11.78 GB written
}


def pole_range(cfg) -> int:
    """Poles per qsgw_sigma_add_poles call when Z is streamed: two s-blocks, so every call crosses a w-chunk boundary."""
    return 2 * (cfg.s_block or 2048)


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


def fp64_peak_tflops(n_sms: int = 148):
    """Roofline denominator for the FP64 contractions: SMs x 64 FMA/clk x 2 x max SM clock."""
    pk, src = _peaks()
    mhz = float(pk.get("sm_max_mhz", 1965.0))
    return n_sms * FP64_FMA_PER_CLK_PER_SM * 2 * mhz * 1e6 / 1e12, src, pk


def measure_fp64_rates(torch, stream_ptr: int, with_dgemm: bool = True):
    """In-run cross-check of the derived FP64 peak: the register-resident DMMA loop and the LDS-fed DMMA loop of
    libqsgw_fp64_probe.so (a bench-only library; best of 3, ~10 ms each) and, as an outside reference that is never on
    the product path, a cuBLAS DGEMM 8192^3 through torch.matmul."""
    from paper_2210_17093_b200 import build
    out = {}
    try:
        lib = ctypes.CDLL(build.build_probe())
        lib.qsgw_fp64_probe.argtypes = [ctypes.c_int] * 4 + [ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        for name, mode in (("dmma_microbench", 0), ("lds_fed_dmma_microbench", 3)):
            best = 0.0
            for _ in range(3):
                tf = ctypes.c_double()
                if lib.qsgw_fp64_probe(mode, 20000, 0, 1, ctypes.c_void_p(stream_ptr), ctypes.byref(tf), None) == 0:
                    best = max(best, tf.value)
            out[name] = best or None
    except Exception as e:      # the probe is a cross-check, not a dependency of the measurement
        out["probe_error"] = str(e)
    if with_dgemm:
        try:
            a = torch.randn((8192, 8192), dtype=torch.float64, device="cuda")
            b = torch.randn((8192, 8192), dtype=torch.float64, device="cuda")
            c = a @ b
            best = 0.0
            for _ in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); c = a @ b; e1.record(); torch.cuda.synchronize()
                best = max(best, 2 * 8192.0 ** 3 / (e0.elapsed_time(e1) * 1e-3) / 1e12)
            out["cublas_dgemm_8192"] = best
            del a, b, c
            torch.cuda.empty_cache()
        except Exception as e:
            out["dgemm_error"] = str(e)
    out["how"] = "measured in this run (best of 3 each); reference figures, the roofline denominator is `value`"
    return out


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
            self.thread.join(timeout=5)

    def summary(self):
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "reasons": sorted(reasons), "samples": len(sm)}


def _cpu_oracle_sample(cfg, B_host, eps, occ, Omega, Z_cols, n_sample):
    """Times the oracle as it stands on `n_sample` poles of the workload (all states, full B); returns (s, F_min)."""
    import oracle
    import qsgw_inputs as qi
    t0 = time.perf_counter()
    oracle.sigma(B_host, eps, occ, Omega[:n_sample], Z_cols[:, :n_sample], cfg.eta, cfg.n_occ)
    dt = time.perf_counter() - t0
    return dt, qi.flop_model(cfg, n_sample)["F_min"]


def _sample_poles(cfg, target_s=20.0, gflops_guess=12.0):
    import qsgw_inputs as qi
    per_pole = qi.flop_model(cfg, 1)["F_full"] * 1.3           # the oracle does the full (non-symmetric) work + D
    n = int(target_s * gflops_guess * 1e9 / per_pole)
    return max(4, min(cfg.n_pole, n))


def _host_inputs_for_reference(cfg, n_sample):
    """B, eps, occ, Omega and the first n_sample columns of Z as numpy arrays.  Drawn on the GPU when the box has one
    (the CPU generator needs minutes for the 32 GB of xl's B); only the oracle runs in the timed steps either way."""
    import torch
    import qsgw_inputs as qi
    dev = "cuda" if torch.cuda.is_available() else "cpu"
    B = qi.make_B(cfg, dev).cpu().numpy()
    Z = qi.make_Z(cfg, 0, n_sample, device=dev).cpu().numpy()
    return B, qi.make_eps(cfg).numpy(), qi.make_occ(cfg).numpy(), qi.make_omega(cfg).numpy(), Z


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores; each step a bounded pole sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    import qsgw_inputs as qi
    cfg = qi.CONFIGS[args.workload]
    n_sample = args.ref_poles or _sample_poles(cfg, target_s=6.0)
    B, eps, occ, Om, Z = _host_inputs_for_reference(cfg, n_sample)
    times = []
    for it in range(args.warmup + args.steps):
        dt, flops = _cpu_oracle_sample(cfg, B, eps, occ, Om, Z, n_sample)
        if it >= args.warmup:
            times.append(dt)
    t = sum(times) / len(times)
    val = flops / t / 1e12
    sample = f"{n_sample} of {cfg.n_pole} poles of '{cfg.name}', all {cfg.n_mo} states, full B; per-step time scales linearly in poles"
    cores = oracle.num_threads()
    out = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": t * 1e3, "ms_per_build_extrapolated": t * 1e3 * cfg.n_pole / n_sample,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_dict(cfg, args, extra={"sample": sample}),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)
    return 0


def _config_dict(cfg, args, extra=None):
    par = "single" if args.gpus <= 1 else ("pole-sharded" if getattr(args, "shard", "replicas") == "poles" else "replicas")
    d = {"workload": cfg.name, "n_mo": cfg.n_mo, "n_occ": cfg.n_occ, "n_aux": cfg.n_aux, "n_pole": cfg.n_pole,
         "s_block": cfg.s_block, "eta": cfg.eta, "seed": cfg.seed, "parallelism": par,
         "l2": "inputs larger than L2 (B + Z >> 126 MB); no explicit flush"}
    if extra:
        d.update(extra)
    return d


def max_over_ranks(ms: float, world: int, device="cpu") -> float:
    """The one data-free collective of the bench: the max over ranks of a rank-local time."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(flops_per_rank: float, world: int, ms_per_step: float) -> float:
    """Weak scaling (replicas): every rank builds its own Sigma, so the job's TFLOP/s is world x flops over the slowest
    rank's time.  Pole-sharded runs pass world = 1 and the flops of the ONE Sigma all ranks build together."""
    return world * flops_per_rank / (ms_per_step * 1e-3) / 1e12


def run_gpu(args):
    import torch
    import torch.distributed as dist
    import qsgw_inputs as qi
    import paper_2210_17093_b200 as pkg

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the qsGW Sigma build has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    sharded = args.shard == "poles" and world > 1
    # everything below runs on one non-default stream (inputs, the plan, the events): the legacy default stream cannot
    # be captured into a CUDA graph
    torch.cuda.set_stream(torch.cuda.Stream(dev))

    base = qi.CONFIGS[args.workload]
    # replicas: every rank its own problem (seed + rank); pole-sharded: ONE problem, the same B on every rank
    cfg = base if sharded else qi.Config(base.name, base.n_mo, base.n_occ, base.n_aux, base.n_pole, base.s_block, base.eta,
                                         base.seed + rank)
    s_lo, n_local = pkg.qsgw_sigma_pole_slice(cfg.n_pole, world, rank) if sharded else (0, cfg.n_pole)
    rng = pole_range(cfg)
    # Z resident when this rank's columns fit beside B and the workspace (<= 48 GB), else produced range by range
    streaming = args.stream_poles or (8.0 * cfg.n_ov * n_local > 48e9)
    fl = qi.flop_model(cfg)
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    peak, peak_src, pk = fp64_peak_tflops(nsm)
    rates = measure_fp64_rates(torch, torch.cuda.current_stream().cuda_stream) if rank == 0 else None

    # ---- inputs, resident in HBM before the timed region
    B = qi.make_B(cfg, dev)
    eps, occ, Om = qi.make_eps(cfg).to(dev), qi.make_occ(cfg).to(dev), qi.make_omega(cfg).to(dev)
    if streaming:
        Zbuf = [torch.empty((cfg.n_ov, rng), dtype=torch.float64, device=dev) for _ in range(2)]
        Z = None
        plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, rng, cfg.s_block)
    else:
        Z = qi.make_Z(cfg, s_lo, s_lo + n_local, device=dev)
        plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, max(n_local, 1), cfg.s_block)
    pkg.qsgw_sigma_set_profiling(plan, True)
    Sigma = torch.empty((cfg.n_mo, cfg.n_mo), dtype=torch.float64, device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); fn(); e1.record()
        return (e0, e1)

    def one_build():
        """One Sigma^c build; returns the CUDA event pairs (on the launch stream) that bracket every kernel of the path."""
        if not streaming and not sharded:
            return [timed(lambda: pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta, Sigma))]
        evs = [timed(lambda: pkg.qsgw_sigma_begin(plan, B, eps, occ, cfg.eta))]
        if streaming:
            # Z (130 GB at xl) is produced range by range on the device just before each add_poles call;
            # the generation is outside the event pairs, every kernel of the path is inside one.
            for k, s0 in enumerate(range(s_lo, s_lo + n_local, rng)):
                s1 = min(s_lo + n_local, s0 + rng)
                zb = Zbuf[k % 2][:, : s1 - s0]
                qi.make_Z(cfg, s0, s1, device=dev, out=zb)
                evs.append(timed(lambda: pkg.qsgw_sigma_add_poles(plan, Om[s0:s1], zb)))
        elif n_local > 0:
            evs.append(timed(lambda: pkg.qsgw_sigma_add_poles(plan, Om[s_lo:s_lo + n_local], Z)))
        evs.append(timed(lambda: pkg.qsgw_sigma_finish(plan, Sigma)))
        if sharded:   # the exchange step of the sharded path: one all-reduce of the N x N matrix, inside the timed region
            evs.append(timed(lambda: pkg.allreduce_sigma(Sigma)))
        return evs

    for _ in range(args.warmup):
        one_build()
    barrier()
    pkg.qsgw_sigma_get_stats(plan, reset=True)
    all_events = []
    with ClockSampler(local) as clocks:
        barrier()
        t_wall0 = time.perf_counter()
        for _ in range(args.steps):
            all_events.append(one_build())
        barrier()
        t_wall = time.perf_counter() - t_wall0
    step_ms = [sum(a.elapsed_time(b) for a, b in evs) for evs in all_events]
    total_ms = max_over_ranks(sum(step_ms), world, dev)
    stats = pkg.qsgw_sigma_get_stats(plan, reset=True)
    ms_per_step = total_ms / args.steps
    value = whole_job_value(fl["F_min"], 1 if sharded else world, ms_per_step)
    assert torch.isfinite(Sigma).all()

    # ---- the same one-shot build without per-launch event timing: identical arguments every step, so the library
    # replays it as ONE CUDA graph (qsgw_sigma_build, include/qsgw_sigma.h).  Reported beside `value`, not instead of it.
    graph_replay = None
    if not streaming and not sharded and plan.stream is not None and plan.stream.cuda_stream != 0:
        pkg.qsgw_sigma_set_profiling(plan, False)
        for _ in range(3):
            pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta, Sigma)
        torch.cuda.synchronize()
        evs = [timed(lambda: pkg.qsgw_sigma_build(plan, B, eps, occ, Om, Z, cfg.eta, Sigma)) for _ in range(args.steps)]
        torch.cuda.synchronize()
        g_ms = sum(a.elapsed_time(b) for a, b in evs) / args.steps
        graph_replay = {"ms_per_build": g_ms, "value": fl["F_min"] / (g_ms * 1e-3) / 1e12, "unit": UNIT, "steps": args.steps,
                        "how": "profiling off: the build is one CUDA graph launch per step"}
        pkg.qsgw_sigma_set_profiling(plan, True)

    out = None
    if rank == 0:
        # dominant kernel: the stage-2 DMMA GEMM (w producer), 57 % of F_min; its launches and flops on THIS rank
        n2 = max(1, stats["launches_stage2"])
        s2_ms = stats["ms_stage2"] / n2
        fl_local = qi.flop_model(cfg, n_local)
        flops_per_launch = fl_local["F2sym"] * args.steps / n2
        achieved = flops_per_launch / (s2_ms * 1e-3) / 1e12
        traffic = NCU_STAGE2_DRAM_BYTES_PER_LAUNCH.get(cfg.name)
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "ms_per_build": ms_per_step, "ms_per_build_best": min(step_ms),
            "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": _config_dict(cfg, args, extra={"z_resident": not streaming, "poles_per_add_poles_call": rng if streaming else n_local,
                                                     "flops_F_min": fl["F_min"], "flops_F_full": fl["F_full"]}),
            "tflops_model_full": (1 if sharded else world) * fl["F_full"] / (ms_per_step * 1e-3) / 1e12,
            "frac_of_fp64_peak": value / (world * peak),
            "fp64_peak_tflops": {"value": peak, "how": f"{nsm} SMs x {FP64_FMA_PER_CLK_PER_SM} FMA/clk x 2 x sm_max_mhz of MEASURED_PEAKS.json ({peak_src})",
                                 "in_run_checks": rates},
            "stage_ms_per_build": {k[3:]: stats[k] / args.steps for k in ("ms_pack", "ms_stage1", "ms_stage2", "ms_stage3", "ms_epilogue")},
            "stage_tflops": {"stage1": fl_local["F1"] * args.steps / max(stats["ms_stage1"], 1e-9) / 1e9,
                             "stage2": fl_local["F2sym"] * args.steps / max(stats["ms_stage2"], 1e-9) / 1e9,
                             "stage3": fl_local["F3"] * args.steps / max(stats["ms_stage3"], 1e-9) / 1e9},
            "roofline": {"bound": "tensor", "kernel": "gemm_tn_dmma_kernel<2,2,EpiPairScatter> (stage 2, w producer)",
                         "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         "launches": stats["launches_stage2"], "avg_launch_ms": s2_ms,
                         "traffic": traffic[0] if traffic else None,
                         "traffic_source": (f"recorded: dram read + write bytes of one launch over a full s-block, ncu, {traffic[1]}"
                                            if traffic else "no committed ncu capture for this workload"),
                         "peak_source": f"FP64 pipe rate at max SM clock ({peak_src} MEASURED_PEAKS.json sm_max_mhz; no FP64 entry is "
                                        "measured there); cross-checked in this run, see fp64_peak_tflops.in_run_checks"},
            "gpu_launches": stats["kernel_launches"],
            "graph_replay": graph_replay,
            "wall_s_timed_region": t_wall,
            "clocks": clocks.summary(),
        }

    # ---- e2e: the same build through the host-buffer entry point (rank-local, max over ranks)
    held = {"B": B, "Z": Z}          # handed over so that the device copies can be freed as soon as the host has them
    del B, Z
    if streaming:
        del Zbuf
    if args.no_e2e or sharded:
        e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
               "how": "skipped (--no-e2e, or pole-sharded run)"}
        hB = hZ = None
    else:
        e2e, hB, hZ = _run_e2e(args, torch, pkg, qi, cfg, plan, held, eps, occ, Om, dev, world, fl, barrier)
    held.clear()
    torch.cuda.empty_cache()

    # ---- cpu_baseline: the oracle as it stands, on rank 0's host cores, bounded sample of the same workload
    if rank == 0:
        out["e2e"] = e2e
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = _cpu_baseline(args, torch, qi, cfg, hB, hZ, eps, occ, Om, dev)
        else:
            out["cpu_baseline"] = None
        print(json.dumps(out), flush=True)
    pkg.qsgw_sigma_destroy(plan)
    if world > 1:
        dist.destroy_process_group()
    return 0


def _pinned_empty(torch, shape):
    """A host tensor of exactly this size, page-locked in place (torch's pinned allocator rounds big requests up to a
    power of two: 130 GB would become 256 GB)."""
    t = torch.empty(shape, dtype=torch.float64)
    rc = torch.cuda.cudart().cudaHostRegister(t.data_ptr(), t.numel() * 8, 0)
    if int(rc) != 0:
        raise RuntimeError(f"cudaHostRegister failed with {rc}")
    return t


def _unpin(torch, t):
    if t is not None:
        torch.cuda.cudart().cudaHostUnregister(t.data_ptr())


def _run_e2e(args, torch, pkg, qi, cfg, plan, held, eps, occ, Om, dev, world, fl, barrier):
    """The build through qsgw_sigma_build_host: B, eps, occ, Omega, Z in page-locked HOST memory, Sigma back to the host,
    all copies inside the timed region.  Returns (e2e dict, host B, host Z) -- the host arrays also serve cpu_baseline."""
    import psutil
    need = 8.0 * (cfg.n_aux * cfg.n_mo ** 2 + cfg.n_ov * cfg.n_pole)
    avail = psutil.virtual_memory().available
    if need + 20e9 > avail:
        return ({"value": None, "unit": UNIT, "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                 "how": f"skipped: the host copy of B and Z needs {need / 1e9:.0f} GB of page-locked memory, {avail / 1e9:.0f} GB available"},
                None, None)
    hB = _pinned_empty(torch, (cfg.n_aux, cfg.n_mo, cfg.n_mo))
    hB.copy_(held.pop("B"))
    hZ = _pinned_empty(torch, (cfg.n_ov, cfg.n_pole))
    Z = held.pop("Z")
    if Z is not None:
        hZ.copy_(Z)
        del Z
    else:       # xl: Z never exists whole on the device; draw it range by range and move it to the host once, untimed
        step = pole_range(cfg)
        zb = torch.empty((cfg.n_ov, step), dtype=torch.float64, device=dev)
        for s0 in range(0, cfg.n_pole, step):
            s1 = min(cfg.n_pole, s0 + step)
            qi.make_Z(cfg, s0, s1, device=dev, out=zb[:, : s1 - s0])
            hZ[:, s0:s1].copy_(zb[:, : s1 - s0])
        del zb
    hE, hO, hOm = eps.cpu().pin_memory(), occ.cpu().pin_memory(), Om.cpu().pin_memory()
    hS = torch.empty((cfg.n_mo, cfg.n_mo), dtype=torch.float64).pin_memory()
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    for _ in range(args.e2e_warmup):
        pkg.qsgw_sigma_build_host(plan, hB, hE, hO, hOm, hZ, cfg.eta, hS)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.e2e_steps):
        pkg.qsgw_sigma_build_host(plan, hB, hE, hO, hOm, hZ, cfg.eta, hS)
    e1.record()
    barrier()
    ms = max_over_ranks(e0.elapsed_time(e1), world, dev) / args.e2e_steps
    h2d = sum(t.numel() * 8 for t in (hB, hE, hO, hOm, hZ))
    assert torch.isfinite(hS).all()
    return ({"value": whole_job_value(fl["F_min"], world, ms), "unit": UNIT, "ms_per_build": ms, "steps": args.e2e_steps,
             "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": hS.numel() * 8,
             "how": "qsgw_sigma_build_host from page-locked host tensors; uploads overlap the kernels; h2d_bytes_per_step counts "
                    "the host tensors handed to the call -- of B the library uploads only the blocks with p <= q (54 % of it)"}, hB, hZ)


def _cpu_baseline(args, torch, qi, cfg, hB, hZ, eps, occ, Om, dev):
    import oracle
    n_sample = args.ref_poles or _sample_poles(cfg)
    if hB is None:
        hB = qi.make_B(cfg, dev).cpu()
        torch.cuda.empty_cache()
    Zs = (hZ[:, :n_sample] if hZ is not None else qi.make_Z(cfg, 0, n_sample, device=dev).cpu()).numpy()
    Bn, en, on, omn = hB.numpy(), eps.cpu().numpy(), occ.cpu().numpy(), Om.cpu().numpy()
    dt, flops = _cpu_oracle_sample(cfg, Bn, en, on, omn, Zs, n_sample)
    cores = oracle.num_threads()
    res = {"value": flops / dt / 1e12, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"{n_sample} of {cfg.n_pole} poles of '{cfg.name}', all {cfg.n_mo} states, full B ({dt:.1f} s); "
                     f"whole build extrapolated linearly in poles: {dt * cfg.n_pole / n_sample:.0f} s",
           "ms_per_build_extrapolated": dt * 1e3 * cfg.n_pole / n_sample}
    if cfg.name in ("tiny", "small"):       # a one-core figure for the two smallest configs
        oracle.set_num_threads(1)
        dt1, _ = _cpu_oracle_sample(cfg, Bn, en, on, omn, Zs, n_sample)
        oracle.set_num_threads(cores)
        res["one_thread"] = {"value": flops / dt1 / 1e12, "unit": UNIT, "cores": 1, "seconds": dt1}
    return res


def run_gpu_diag(args):
    """--path diag: the next row of the scope table, measured to the same bar -- one step is one
    qsgw_sigma_diag_build (pack, stage 1, stage 2 per s-block, the G0W0 diagonal kernel per s-block) for all N
    states on an n_omega-point grid.  value = 1e9 complex Lehmann terms evaluated per second,
    N^2 * n_s * n_omega / t; the kernel is bound by the FP64 ALU rate (8 FP64-pipe instructions per term)."""
    import torch
    import qsgw_inputs as qi
    import paper_2210_17093_b200 as pkg

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("--path diag is a single-GPU measurement")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cfg = qi.CONFIGS[args.workload]
    if cfg.name == "xl":
        raise SystemExit("--path diag needs Z resident on the device: use tiny..large")
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    pk, peak_src = _peaks()
    lane_peak = nsm * FP64_FMA_PER_CLK_PER_SM * float(pk.get("sm_max_mhz", 1965.0)) * 1e6     # FP64 lane-instr / s
    B = qi.make_B(cfg, dev)
    eps, occ, Om = qi.make_eps(cfg).to(dev), qi.make_occ(cfg).to(dev), qi.make_omega(cfg).to(dev)
    Z = qi.make_Z(cfg, device=dev)
    lo, hi = float(eps.min()) - 1.0, float(eps.max()) + 1.0
    grid = torch.linspace(lo, hi, args.n_omega, dtype=torch.float64, device=dev)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_pole, cfg.s_block)
    pkg.qsgw_sigma_set_profiling(plan, True)
    Re = torch.empty((cfg.n_mo, args.n_omega), dtype=torch.float64, device=dev)
    Im = torch.empty_like(Re)
    for _ in range(args.warmup):
        pkg.qsgw_sigma_diag_build(plan, B, eps, occ, Om, Z, cfg.eta, grid, Re, Im)
    torch.cuda.synchronize()
    pkg.qsgw_sigma_get_stats(plan, reset=True)
    evs = []
    with ClockSampler(0) as clocks:
        torch.cuda.synchronize()
        for _ in range(args.steps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); pkg.qsgw_sigma_diag_build(plan, B, eps, occ, Om, Z, cfg.eta, grid, Re, Im); e1.record()
            evs.append((e0, e1))
        torch.cuda.synchronize()
    step_ms = [a.elapsed_time(b) for a, b in evs]
    ms = sum(step_ms) / args.steps
    stats = pkg.qsgw_sigma_get_stats(plan, reset=True)
    assert torch.isfinite(Re).all() and torch.isfinite(Im).all()
    terms = float(cfg.n_mo) ** 2 * cfg.n_pole * args.n_omega
    nd = max(1, stats["launches_diag"])
    d_ms = stats["ms_diag"] / nd
    lane_instr = 8.0 * terms * args.steps / nd                      # FP64-pipe lane-instructions per diag launch
    achieved = lane_instr / (d_ms * 1e-3)
    out = {
        "metric": "g0w0_diag_lehmann_terms_per_s", "value": terms / (ms * 1e-3) / 1e9, "unit": "Gterm/s", "n_gpus": 1,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "path": "diag (SURVEY.md 8(f).1, next row)",
        "config": _config_dict(cfg, args, extra={"n_omega": args.n_omega, "grid": [lo, hi]}),
        "stage_ms_per_build": {"pack": stats["ms_pack"] / args.steps, "stage1": stats["ms_stage1"] / args.steps,
                               "stage2": stats["ms_stage2"] / args.steps, "diag": stats["ms_diag"] / args.steps},
        "roofline": {"bound": "alu", "kernel": "sigma_diag_kernel", "achieved": achieved / 1e12, "peak": lane_peak / 1e12,
                     "unit": "T FP64 lane-instr/s", "frac": achieved / lane_peak, "launches": stats["launches_diag"],
                     "avg_launch_ms": d_ms, "traffic": None,
                     "peak_source": f"{nsm} SMs x 64 FP64 lanes/clk x sm_max_mhz ({peak_src} MEASURED_PEAKS.json); a DFMA-only "
                                    "loop reaches 80 % of it (profiles/r01_fp64_peaks.md); 8 FP64-pipe instructions per term"},
        "gpu_launches": stats["kernel_launches"], "clocks": clocks.summary(),
        "e2e": {"value": None, "unit": "Gterm/s", "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                "how": "B and Z stay on the device between the qsGW build and the diagonal: no host-buffer entry point for this row"},
    }
    if not args.no_cpu_baseline:
        import oracle
        n_sample, states = max(4, min(cfg.n_pole, 64)), list(range(0, cfg.n_mo, max(1, cfg.n_mo // 16)))[:16]
        t0 = time.perf_counter()
        oracle.sigma_diag(B.cpu().numpy(), eps.cpu().numpy(), occ.cpu().numpy(), Om.cpu().numpy()[:n_sample],
                          Z[:, :n_sample].cpu().numpy(), cfg.eta, cfg.n_occ, grid.cpu().numpy(), states=states)
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": len(states) * cfg.n_mo * n_sample * args.n_omega / dt / 1e9, "unit": "Gterm/s",
                               "cores": oracle.num_threads(), "kind": "oracle",
                               "sample": f"{len(states)} states x {n_sample} of {cfg.n_pole} poles x {args.n_omega} grid points "
                                         f"of '{cfg.name}' ({dt:.1f} s, its steps 1-2 included)"}
    print(json.dumps(out), flush=True)
    pkg.qsgw_sigma_destroy(plan)
    return 0


def run_gpu_aomo(args):
    """--path aomo: row 8(f).2, B_mo[P] = C^T B_ao[P] C for all naux auxiliary functions of the workload
    (two batched DMMA GEMMs, 4 N^3 naux flops); value in FP64 TFLOP/s against the same tensor roofline."""
    import torch
    import qsgw_inputs as qi
    import paper_2210_17093_b200 as pkg

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("--path aomo is a single-GPU measurement")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cfg = qi.CONFIGS[args.workload]
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    peak, peak_src, _ = fp64_peak_tflops(nsm)
    B_ao = qi.make_B(cfg, dev)                                   # the config's B stands in for the AO-basis factors
    g = torch.Generator(device=dev); g.manual_seed(cfg.seed)
    C, _ = torch.linalg.qr(torch.randn((cfg.n_mo, cfg.n_mo), generator=g, dtype=torch.float64, device=dev))
    C = C.contiguous()
    work = torch.empty(pkg.qsgw_ri_ao_to_mo_work_doubles(cfg.n_aux, cfg.n_mo, cfg.n_mo), dtype=torch.float64, device=dev)
    B_mo = torch.empty_like(B_ao)
    for _ in range(args.warmup):
        pkg.qsgw_ri_ao_to_mo(B_ao, C, B_mo, work)
    torch.cuda.synchronize()
    evs = []
    with ClockSampler(0) as clocks:
        for _ in range(args.steps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); pkg.qsgw_ri_ao_to_mo(B_ao, C, B_mo, work); e1.record()
            evs.append((e0, e1))
        torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in evs) / args.steps
    flops = 4.0 * float(cfg.n_mo) ** 3 * cfg.n_aux
    val = flops / (ms * 1e-3) / 1e12
    assert torch.isfinite(B_mo).all()
    out = {"metric": "ri_ao_to_mo_fp64_tflops", "value": val, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "path": "aomo (SURVEY.md 8(f).2, next row)",
           "config": _config_dict(cfg, args, extra={"n_ao": cfg.n_mo, "flops": flops}),
           "roofline": {"bound": "tensor", "kernel": "gemm_tn_dmma_kernel<*,*,EpiStore> (two batched launches)",
                        "achieved": val, "peak": peak, "unit": UNIT, "frac": val / peak, "launches": 2 * args.steps,
                        "avg_launch_ms": ms / 2, "traffic": None, "peak_source": f"FP64 pipe rate at max SM clock ({peak_src})"},
           "gpu_launches": 2 * args.steps, "clocks": clocks.summary(),
           "e2e": {"value": None, "unit": UNIT, "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                   "how": "B stays on the device between the transform and the Sigma build: no host-buffer entry point for this row"}}
    if not args.no_cpu_baseline:
        import oracle
        n_s = max(1, min(cfg.n_aux, int(4e11 / (2.0 * float(cfg.n_mo) ** 4))))     # the oracle is the O(N^4) double sum per P
        t0 = time.perf_counter()
        oracle.ao_to_mo(B_ao[:n_s].cpu().numpy(), C.cpu().numpy())
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": 4.0 * float(cfg.n_mo) ** 3 * n_s / dt / 1e12, "unit": UNIT + " (GPU flop model / oracle time)",
                               "cores": oracle.num_threads(), "kind": "oracle",
                               "sample": f"{n_s} of {cfg.n_aux} auxiliary functions of '{cfg.name}' ({dt:.2f} s; the literal double sum, 2 N^4 flops per P)"}
    print(json.dumps(out), flush=True)
    return 0


def run_gpu_mp2(args):
    """--path mp2: row 8(f).3, one qsgw_mp2_build (direct + second-order exchange sums of Eq. (20) in Eq. (21)) on the
    workload's B, eps, occ.  Flop model (2 per FMA): direct = F2sym + F3 with n_s = o*v; exchange, per occupied i:
    2 N^2 v naux (exchange integrals) + 2 [N(N+1)/2] v naux (stage 2) + 2 N^3 v (stage 3)."""
    import torch
    import qsgw_inputs as qi
    import paper_2210_17093_b200 as pkg

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("--path mp2 is a single-GPU measurement")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cfg = qi.CONFIGS[args.workload]
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    peak, peak_src, _ = fp64_peak_tflops(nsm)
    B = qi.make_B(cfg, dev)
    eps, occ = qi.make_eps(cfg).to(dev), qi.make_occ(cfg).to(dev)
    plan = pkg.qsgw_sigma_create(cfg.n_mo, cfg.n_occ, cfg.n_aux, cfg.n_ov, cfg.s_block)
    pkg.qsgw_sigma_set_profiling(plan, True)
    S = torch.empty((cfg.n_mo, cfg.n_mo), dtype=torch.float64, device=dev)
    for _ in range(args.warmup):
        pkg.qsgw_mp2_build(plan, B, eps, occ, cfg.eta, S)
    torch.cuda.synchronize()
    pkg.qsgw_sigma_get_stats(plan, reset=True)
    evs = []
    with ClockSampler(0) as clocks:
        for _ in range(args.steps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); pkg.qsgw_mp2_build(plan, B, eps, occ, cfg.eta, S); e1.record()
            evs.append((e0, e1))
        torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in evs) / args.steps
    stats = pkg.qsgw_sigma_get_stats(plan, reset=True)
    assert torch.isfinite(S).all()
    N, o, v, naux = float(cfg.n_mo), float(cfg.n_occ), float(cfg.n_virt), float(cfg.n_aux)
    npair = N * (N + 1) / 2
    f_direct = 2 * npair * naux * o * v + 2 * N ** 3 * o * v
    f_sox = o * (2 * N * N * v * naux + 2 * npair * v * naux + 2 * N ** 3 * v)
    val = (f_direct + f_sox) / (ms * 1e-3) / 1e12
    out = {"metric": "qsmp2_sigma_c_build_fp64_tflops", "value": val, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "path": "mp2 (SURVEY.md 8(f).3)",
           "config": _config_dict(cfg, args, extra={"flops_direct": f_direct, "flops_exchange": f_sox}),
           "stage_ms_per_build": {"pack": stats["ms_pack"] / args.steps, "gemms": stats["ms_stage2"] / args.steps,
                                  "stage3": stats["ms_stage3"] / args.steps, "epilogue": stats["ms_epilogue"] / args.steps},
           "roofline": {"bound": "tensor", "kernel": "whole build (GEMMs + sigma_accumulate_kernel)", "achieved": val, "peak": peak,
                        "unit": UNIT, "frac": val / peak, "launches": stats["kernel_launches"], "avg_launch_ms": None, "traffic": None,
                        "peak_source": f"FP64 pipe rate at max SM clock ({peak_src})"},
           "gpu_launches": stats["kernel_launches"], "clocks": clocks.summary(),
           "e2e": {"value": None, "unit": UNIT, "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                   "how": "B, eps, occ stay on the device between the AO->MO transform and the build: no host-buffer entry point for this row"}}
    if not args.no_cpu_baseline:
        import oracle
        states = [0, cfg.n_occ - 1, cfg.n_occ, cfg.n_mo - 1] if cfg.n_mo > 120 else None
        t0 = time.perf_counter()
        oracle.mp2(B.cpu().numpy(), eps.cpu().numpy(), occ.cpu().numpy(), cfg.eta, cfg.n_occ, states=states)
        dt = time.perf_counter() - t0
        what = f"whole '{cfg.name}' build" if states is None else f"{len(states)} of {cfg.n_mo} output states of '{cfg.name}', all internal sums"
        out["cpu_baseline"] = {"value": (f_direct + f_sox) * (1.0 if states is None else len(states) / N) / dt / 1e12,
                               "unit": UNIT + " (GPU flop model, scaled by the share of output rows / oracle time)",
                               "cores": oracle.num_threads(), "kind": "oracle", "sample": f"{what} ({dt:.1f} s)"}
    print(json.dumps(out), flush=True)
    pkg.qsgw_sigma_destroy(plan)
    return 0


def run_gpu_casida(args):
    """--path casida: row 8(f).4, the two library steps of the Casida / RPA solve around the eigensolve.
    value = FP64 TFLOP/s of qsgw_casida_matrix on the algorithmic minimum 2 * [n_ov (n_ov + 1) / 2] * naux flops (the
    symmetric half of K = Bov^T Bov); the back-transformation qsgw_casida_z is reported against the HBM roofline
    (16 bytes per element of Z: xi read once, Z written once).  The eigensolve between them is a library call (cuSOLVER
    through torch.linalg.eigh), timed for context only up to `medium`."""
    import torch
    import qsgw_inputs as qi
    import paper_2210_17093_b200 as pkg

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("--path casida is a single-GPU measurement")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    cfg = qi.CONFIGS[args.workload]
    if cfg.name == "xl":
        raise SystemExit("--path casida: C of xl is 130 GB; use tiny..large")
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    peak, peak_src, pk = fp64_peak_tflops(nsm)
    B = qi.make_B(cfg, dev)
    eps = qi.make_eps(cfg).to(dev)
    n_ov = cfg.n_ov
    work = torch.empty(pkg.qsgw_casida_work_doubles(cfg.n_mo, cfg.n_occ, cfg.n_aux), dtype=torch.float64, device=dev)
    C = torch.empty((n_ov, n_ov), dtype=torch.float64, device=dev)

    def timed_loop(fn):
        for _ in range(args.warmup):
            fn()
        torch.cuda.synchronize()
        evs = []
        for _ in range(args.steps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            evs.append((e0, e1))
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in evs) / args.steps

    with ClockSampler(0) as clocks:
        ms_c = timed_loop(lambda: pkg.qsgw_casida_matrix(B, eps, cfg.n_occ, C, work))
    flops = 2.0 * (n_ov * (n_ov + 1) / 2) * cfg.n_aux
    val = flops / (ms_c * 1e-3) / 1e12
    assert torch.isfinite(C).all() and torch.equal(C, C.T)
    eigh_ms = None
    if n_ov <= 10400:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); lam, xi = torch.linalg.eigh(C); e1.record(); torch.cuda.synchronize()
        eigh_ms = e0.elapsed_time(e1)
        xi = xi.contiguous()
    else:       # a stand-in with the right shapes for the back-transformation's timing (values do not matter for it)
        lam = torch.rand(n_ov, dtype=torch.float64, device=dev) + 0.5
        xi = C
    Om = torch.empty(n_ov, dtype=torch.float64, device=dev)
    Z = torch.empty((n_ov, n_ov), dtype=torch.float64, device=dev) if n_ov <= 10400 else work.new_empty((n_ov, n_ov))
    ms_z = timed_loop(lambda: pkg.qsgw_casida_z(eps, cfg.n_occ, lam, xi, Om, Z))
    hbm = float(pk.get("hbm_gbs", 6650.0))
    z_gbs = 16.0 * n_ov * n_ov / (ms_z * 1e-3) / 1e9
    out = {"metric": "casida_matrix_fp64_tflops", "value": val, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_c, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "path": "casida (SURVEY.md 8(f).4)", "config": _config_dict(cfg, args, extra={"n_ov": n_ov, "flops_symmetric_half": flops}),
           "roofline": {"bound": "tensor", "kernel": "gemm_tn_dmma_kernel<2,2,EpiCasida> (upper-triangle tiles)", "achieved": val, "peak": peak,
                        "unit": UNIT, "frac": val / peak, "launches": args.steps, "avg_launch_ms": ms_c, "traffic": None,
                        "peak_source": f"FP64 pipe rate at max SM clock ({peak_src})"},
           "casida_z": {"ms": ms_z, "achieved_gbs": z_gbs, "peak_gbs": hbm, "frac": z_gbs / hbm, "bound": "hbm",
                        "bytes_per_element": 16, "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_src})"},
           "eigensolve_library_ms": eigh_ms, "gpu_launches": 3 * args.steps, "clocks": clocks.summary(),
           "e2e": {"value": None, "unit": UNIT, "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                   "how": "B and C stay on the device between the AO->MO transform, the eigensolve and the Sigma build"}}
    if not args.no_cpu_baseline and n_ov <= 2000:
        import oracle
        t0 = time.perf_counter()
        oracle.casida_matrix(B.cpu().numpy(), eps.cpu().numpy(), cfg.n_occ)
        dt = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": flops / dt / 1e12, "unit": UNIT + " (GPU flop model / oracle time)", "cores": oracle.num_threads(),
                               "kind": "oracle", "sample": f"whole C of '{cfg.name}' ({dt:.1f} s)"}
    print(json.dumps(out), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="xl", choices=["tiny", "small", "medium", "large", "xl"])
    ap.add_argument("--shard", default="replicas", choices=["replicas", "poles"],
                    help="N > 1: independent replicas (weak scaling, the default) or ONE Sigma sharded over the poles + all-reduce")
    ap.add_argument("--stream-poles", action="store_true", help="produce Z range by range (always on when Z does not fit)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--e2e-warmup", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-poles", type=int, default=0, help="poles in the oracle's timed sample (0 = auto, ~20 s)")
    ap.add_argument("--path", default="sigma", choices=["sigma", "diag", "aomo", "mp2", "casida"],
                    help="sigma: the qsGW Sigma^c build (the bench contract); diag: the G0W0 diagonal on a frequency grid")
    ap.add_argument("--n-omega", type=int, default=64, help="grid points of --path diag")
    args = ap.parse_args()
    if args.steps < 1 or args.warmup < 0:
        raise SystemExit("need --steps >= 1 and --warmup >= 0")
    if args.impl == "reference":
        return run_reference(args)
    if args.path == "diag":
        return run_gpu_diag(args)
    if args.path == "aomo":
        return run_gpu_aomo(args)
    if args.path == "mp2":
        return run_gpu_mp2(args)
    if args.path == "casida":
        return run_gpu_casida(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
