#!/usr/bin/env python
"""bench.py -- order-n configurations/s and FP64 FLOP/s of the CoS hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3]
    torchrun --nnodes=1 --nproc-per-node N ... bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path (rows a1..a5 of SURVEY.md §8(a): G assembly, layer
propagation, combine, connected reduction, output) over one batch of seeded synthetic vertex
configurations, through the C-ABI call cos_eval_connected_xt.  Rank 0 prints ONE JSON line.

  value        whole-job configurations/s, inputs resident in HBM, device-timed (CUDA events on the
               launch stream, one event pair per step so that the L2 flush between steps is excluded)
  e2e          the same metric through cos_eval_connected_xt_host (pinned HOST buffers; H2D and D2H
               copies inside the timed region)
  roofline     the dominant kernel (the evaluation kernel) against the FP64 FMA peak measured in the
               same run by cos_probe_dfma (MEASURED_PEAKS.json has no FP64 figure): bound "alu"
  cpu_baseline the oracle (oracle/, as it stands) on the host cores, on a bounded sample
  sweep        (N = 1, ours) per-order results for n = 8..16 (SURVEY.md §8(d) sweep)

--impl reference times the oracle itself (there is no reference implementation to install: the paper
ships no code).  Multi-GPU: configurations are independent, so every rank evaluates its
own batch (weak scaling), no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2501_00675_b200 import sharding
from harness import workloads as wl  # noqa: E402

METRIC = "order-n configurations/sec"
UNIT = "configurations/s"
HEADLINE_CFG = 3          # BASELINE.json configs[2]: n=10, batch 16384 (largest batch at n >= 10)


def config_dict(w):
    """The `config` object of the JSON line: the same for both arms (the reference arm times a bounded sample of this
    workload and says so in `cpu_baseline.sample`)."""
    return {"workload": w.name, "n": w.n, "batch_per_gpu": w.batch, "species_propagations": 1, "g_diag": w.g_diag,
            "l2": "256 MiB device buffer rewritten between steps, outside the per-step event pairs",
            "entry": "cos_eval_connected_xt" if w.kind == "hubbard" else "cos_eval_connected"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=f"cfg{HEADLINE_CFG}")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def get_workload(name: str, rank: int = 0):
    if name.startswith("cfg"):
        w = wl.baseline_config(int(name[3:]))
    elif name.startswith("sweep_dense_n"):
        w = wl.sweep_workload(int(name[len("sweep_dense_n"):]), "dense")
    elif name.startswith("sweep_hubbard_n"):
        w = wl.sweep_workload(int(name[len("sweep_hubbard_n"):]), "hubbard")
    else:
        raise SystemExit(f"unknown workload {name}")
    if rank > 0:          # weak scaling: every rank draws its own batch of the same recipe
        if w.kind == "hubbard":
            w = wl.hubbard_workload(w.name, w.n, w.batch, w.L, w.beta, w.U, w.mu, w.ntau, w.seed + 1000 * rank,
                                    clustered=(name == "cfg4"))
        else:
            w = wl.dense_workload(w.name, w.n, w.batch, w.U, w.seed + 1000 * rank)
    return w


# ----------------------------------------------------------------------------------------------
def ncu_traffic(workload_name: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, parsed from the committed ncu
    summary profiles/r2_traffic.json.txt (written from one `ncu --set full` capture per workload; the file names the
    command).  None when the workload was not captured -- nothing is measured under a profiler in this run."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.json.txt")
    try:
        with open(path) as f:
            rec = json.load(f).get(workload_name)
        return None if rec is None else {"bytes": rec["dram_bytes"], "source": "profiles/r2_traffic.json.txt: " + rec["capture"],
                                         "executed_over_algorithmic": rec.get("executed_over_algorithmic")}
    except (OSError, ValueError, KeyError):
        return None


class ClockSampler:
    """Samples SM clocks and throttle reasons DURING the timed region.

    NVML (pynvml, ~1 ms period) is used when importable: the timed region of the default run lasts only a few
    milliseconds, far below the 100 ms period of an `nvidia-smi -lms` loop, which is the fallback."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None
        self.stop_flag = False
        self.nvml = None
        self.sm, self.mx, self.reasons = [], [], set()

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.nvml = pynvml
            self.mx.append(float(pynvml.nvmlDeviceGetMaxClockInfo(self.handle, pynvml.NVML_CLOCK_SM)))
            self.thread = threading.Thread(target=self._poll_nvml, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _poll_nvml(self):
        n = self.nvml
        bits = {"hw_slowdown": getattr(n, "nvmlClocksEventReasonHwSlowdown", 0x8),
                "hw_thermal_slowdown": getattr(n, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                "sw_thermal_slowdown": getattr(n, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                "sw_power_cap": getattr(n, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        get_reasons = getattr(n, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
            getattr(n, "nvmlDeviceGetCurrentClocksThrottleReasons", None)
        while not self.stop_flag:
            try:
                self.sm.append(float(n.nvmlDeviceGetClockInfo(self.handle, n.NVML_CLOCK_SM)))
                if get_reasons is not None:
                    r = int(get_reasons(self.handle))
                    for nm, bit in bits.items():
                        if r & bit:
                            self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.001)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.nvml is not None:
            self.stop_flag = True
            self.thread.join(timeout=1)
            return {"sm_mhz": float(np.median(self.sm)) if self.sm else None,
                    "sm_max_mhz": max(self.mx) if self.mx else None, "samples": len(self.sm),
                    "reasons": sorted(self.reasons), "source": "nvml"}
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons), "source": "nvidia-smi"}


def cpu_baseline(w, target_seconds: float = 12.0):
    """The oracle as it stands, on the host cores, on a bounded sample of the same workload."""
    import oracle
    oracle.build()
    n = w.n

    def mats(lo, hi):
        if w.kind == "hubbard":
            g, _ = oracle.build_G(w.xy[lo:hi], w.tau[lo:hi], w.table, None, w.beta, w.g_diag)
            return g, None
        return w.G[lo:hi], w.u[lo:hi]

    probe = min(w.batch, max(8, 64 >> max(0, n - 10)))
    g, u = mats(0, probe)
    t0 = time.perf_counter()
    _, _, cores = oracle.eval_all_connected_timed(g, None, U=w.U, u=u, threads=0)
    dt = max(time.perf_counter() - t0, 1e-6)
    sample = int(min(w.batch, max(probe, probe * target_seconds / dt)))
    t0 = time.perf_counter()
    g, u = mats(0, sample)          # G assembly is part of the step (row a1)
    oracle.eval_all_connected_timed(g, None, U=w.U, u=u, threads=0)
    dt = time.perf_counter() - t0
    return {"value": sample / dt, "unit": UNIT, "cores": int(cores), "kind": "oracle",
            "sample": f"first {sample} of {w.batch} configurations of {w.name} (G assembly + all/connected evaluation, "
                      f"OpenMP over configurations, {dt:.2f} s)"}, sample


def parity_on_sample(w, gpu_out, sample):
    """The timed GPU outputs of the first `sample` configurations against the oracle (strict 1e-10 count; the
    conditioning exceptions of DESIGN.md §4 are judged by tests/parity_util.py, here they are only counted)."""
    import oracle
    if w.kind == "hubbard":
        g, _ = oracle.build_G(w.xy[:sample], w.tau[:sample], w.table, None, w.beta, w.g_diag)
        u = None
    else:
        g, u = w.G[:sample], w.u[:sample]
    _, ref = oracle.eval_all_connected(g, None, U=w.U, u=u)
    rel = np.abs(gpu_out[:sample] - ref) / np.abs(ref)
    return {"configurations": int(sample), "max_rel_err": float(rel.max()), "median_rel_err": float(np.median(rel)),
            "over_1e-10": int((rel > 1e-10).sum())}


# ----------------------------------------------------------------------------------------------
def run_reference(args):
    rank, _, world = sharding.env_rank_world()
    if rank != 0:
        return 0
    w = get_workload(args.workload)
    import oracle
    oracle.build()
    # bounded sample per step so that steps+warmup finish within minutes
    sample = min(w.batch, {4: 64, 8: 4096, 10: 2048, 12: 256}.get(w.n, 16 if w.n < 15 else 4))

    def step():
        if w.kind == "hubbard":
            g, _ = oracle.build_G(w.xy[:sample], w.tau[:sample], w.table, None, w.beta, w.g_diag)
            u = None
        else:
            g, u = w.G[:sample], w.u[:sample]
        return oracle.eval_all_connected_timed(g, None, U=w.U, u=u, threads=0)

    cores = 1
    for _ in range(args.warmup):
        cores = step()[2]
    t0 = time.perf_counter()
    for _ in range(args.steps):
        cores = step()[2]
    dt = time.perf_counter() - t0
    value = sample * args.steps / dt
    desc = f"first {sample} of {w.batch} configurations of {w.name} per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": config_dict(w),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(cores), "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------
class GpuRunner:
    """Device buffers + ctx for one workload; every call goes through the C-ABI binding."""

    def __init__(self, torch, api, w, device):
        self.torch, self.w = torch, w
        self.ctx = api.Context(device=device)
        self.n_species = 1                      # BASELINE configs: G_up == G_down (no field) / spinless
        if w.kind == "hubbard":
            self.table = torch.from_numpy(w.table).cuda()
            self.ctx.set_g0_table(self.table, w.beta)
            self.xy = torch.from_numpy(w.xy).cuda()
            self.tau = torch.from_numpy(w.tau).cuda()
            self.h_xy = torch.from_numpy(w.xy).pin_memory()
            self.h_tau = torch.from_numpy(w.tau).pin_memory()
        else:
            self.G = torch.from_numpy(w.G).cuda()
            self.u = torch.from_numpy(w.u).cuda()
            self.h_G = torch.from_numpy(w.G).pin_memory()
            self.h_u = torch.from_numpy(w.u).pin_memory()
        self.out = torch.empty(w.batch, dtype=torch.float64, device="cuda")
        self.h_out = torch.empty(w.batch, dtype=torch.float64).pin_memory()

    def step(self):
        w = self.w
        if w.kind == "hubbard":
            self.ctx.eval_connected_xt(self.xy, self.tau, self.out, U=w.U, g_diag=w.g_diag)
        else:                                   # dense entry: matrices are the input (no a1 row)
            self.ctx.eval_connected(self.G, self.G, self.out, U=w.U, d_u=self.u)
        return self.ctx.last_launch_count()

    def step_e2e(self):
        w, torch = self.w, self.torch
        if w.kind == "hubbard":
            self.ctx.eval_connected_xt_host(self.h_xy, self.h_tau, self.h_out, U=w.U, g_diag=w.g_diag)
            return self.h_xy.numel() * 4 + self.h_tau.numel() * 8, self.h_out.numel() * 8
        self.G.copy_(self.h_G, non_blocking=True)
        self.u.copy_(self.h_u, non_blocking=True)
        self.ctx.eval_connected(self.G, self.G, self.out, U=w.U, d_u=self.u)
        self.h_out.copy_(self.out, non_blocking=True)
        torch.cuda.current_stream().synchronize()
        return self.h_G.numel() * 8 + self.h_u.numel() * 8, self.h_out.numel() * 8

    def flops_per_config(self, api):
        return api.flop_count(self.w.n, self.n_species, True)


def time_steps(torch, runner, steps, warmup, flush):
    """Per-step CUDA-event pairs on the current stream; the L2 flush sits between the pairs."""
    for _ in range(warmup):
        runner.step()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    launches = 0
    for a, b in ev:
        flush.zero_()
        a.record()
        launches += runner.step()
        b.record()
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, b in ev]
    return float(sum(ms)), launches, ms


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2501_00675_b200 import api, build

    rank, local_rank, world = sharding.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (the CUDA path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    build.build()
    w = get_workload(args.workload, rank)
    runner = GpuRunner(torch, api, w, local_rank)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    # roofline denominators measured in the same run
    dfma_tflops = runner.ctx.probe_dfma_tflops()
    smem_gbs = runner.ctx.probe_smem_gbs()

    sampler = ClockSampler(local_rank)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    runner.ctx.enable_kernel_timer(True)
    runner.ctx.reset_kernel_timer()
    # warm-up runs inside time_steps; the kernel timer is reset after warm-up below
    for _ in range(args.warmup):
        runner.step()
    torch.cuda.synchronize()
    runner.ctx.reset_kernel_timer()
    total_ms, launches, per_step = time_steps(torch, runner, args.steps, 0, flush)
    kern_ms, kern_launches = runner.ctx.kernel_time_ms()
    runner.ctx.enable_kernel_timer(False)
    clocks = sampler.stop()
    if world > 1:
        dist.barrier()
    total_ms = sharding.max_over_ranks(total_ms, dist if world > 1 else None, "cuda")
    units = sharding.sum_over_ranks(float(w.batch * args.steps), dist if world > 1 else None, "cuda")
    value = units / (total_ms * 1e-3)

    # end to end through the host-buffer entry point
    for _ in range(3):
        runner.step_e2e()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    h2d = d2h = 0
    for _ in range(args.steps):
        h2d, d2h = runner.step_e2e()
    e2e_s = time.perf_counter() - t0
    e2e_s = sharding.max_over_ranks(e2e_s, dist if world > 1 else None, "cuda")
    e2e_value = units / e2e_s

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    flop_cfg = runner.flops_per_config(api)
    achieved = flop_cfg * w.batch / (kern_ms * 1e-3) * 1e-12
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(w),
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "gpu_launches": launches,
        "clocks": clocks,
        "flop_per_config": flop_cfg,
        "tflops": flop_cfg * value * 1e-12,
        "roofline": {"bound": "alu", "kernel": runner.ctx.last_kernel_name(), "achieved": achieved,
                     "peak": dfma_tflops, "unit": "TFLOP/s", "frac": achieved / dfma_tflops,
                     "peak_source": "cos_probe_dfma: register-only FP64 FMA kernel measured in this run "
                                    "(MEASURED_PEAKS.json has no FP64 figure); nominal 148 SM x 64 FMA/clk x 1.965 GHz = 37.2",
                     "kernel_ms": kern_ms, "kernel_launches_timed": kern_launches,
                     "smem_probe_gbs": smem_gbs, "traffic": None},
    }
    tr = ncu_traffic(w.name)
    if tr is not None:
        line["roofline"]["traffic"] = tr["bytes"]
        line["roofline"]["traffic_source"] = tr["source"]
        # FP64 thread instructions executed (DFMA + DMUL + DADD, predicated on) / algorithmic FMAs, same ncu capture
        line["roofline"]["fp64_executed_over_algorithmic"] = tr["executed_over_algorithmic"]
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"], sample = cpu_baseline(w)
        line["parity_sample"] = parity_on_sample(w, runner.out.cpu().numpy(), sample)
    if not args.no_sweep and world == 1:
        line["two_species"] = two_species_line(torch, api, runner, flush, dfma_tflops)
        line["f32"] = f32_line(torch, api, runner, flush)
        line["mc"] = mc_line(torch, runner, flush, kern_ms)
        line["sweep"] = sweep(torch, api, local_rank, flush, dfma_tflops)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def sweep(torch, api, device, flush, dfma_tflops):
    """n = 8..16, both input styles; 5 timed steps each after 3 warm-up steps."""
    rows = []
    for kind in ("hubbard", "dense"):
        for n in range(8, 17):
            w = wl.sweep_workload(n, kind)
            r = GpuRunner(torch, api, w, device)
            r.ctx.enable_kernel_timer(True)
            for _ in range(3):
                r.step()
            torch.cuda.synchronize()
            r.ctx.reset_kernel_timer()
            total_ms, _, _ = time_steps(torch, r, 5, 0, flush)
            kern_ms, _ = r.ctx.kernel_time_ms()
            flop = r.flops_per_config(api)
            rows.append({"workload": w.name, "n": n, "batch": w.batch, "configs_per_s": w.batch * 5 / (total_ms * 1e-3),
                         "tflops": flop * w.batch * 5 / (total_ms * 1e-3) * 1e-12,
                         "kernel_tflops": flop * w.batch / (kern_ms * 1e-3) * 1e-12,
                         "frac_of_dfma_peak": flop * w.batch / (kern_ms * 1e-3) * 1e-12 / dfma_tflops,
                         "kernel": r.ctx.last_kernel_name()})
            r.ctx.close()
            del r
    return rows


def two_species_line(torch, api, runner, flush, dfma_tflops):
    """The headline workload evaluated with a separate copy of G_down: two propagation instances per configuration
    ("run every Hubbard config twice ... and say which is reported").  Hubbard workloads only."""
    w = runner.w
    if w.kind != "hubbard":
        return None
    ctx = runner.ctx
    Gup = torch.empty((w.batch, w.n, w.n), dtype=torch.float64, device="cuda")
    ctx.build_G(runner.xy, runner.tau, Gup, None, g_diag=w.g_diag)
    Gdn = Gup.clone()
    out = torch.empty(w.batch, dtype=torch.float64, device="cuda")
    ctx.enable_kernel_timer(True)
    for _ in range(3):
        ctx.eval_connected(Gup, Gdn, out, U=w.U)
    torch.cuda.synchronize()
    ctx.reset_kernel_timer()
    steps = 5
    for _ in range(steps):
        flush.fill_(1)
        ctx.eval_connected(Gup, Gdn, out, U=w.U)
    torch.cuda.synchronize()
    kern_ms, _ = ctx.kernel_time_ms()
    ctx.enable_kernel_timer(False)
    flop = api.flop_count(w.n, 2, True)
    same = bool(torch.allclose(out, runner.out, rtol=1e-9, atol=0.0))
    return {"workload": w.name, "species_propagations": 2, "configs_per_s": w.batch / (kern_ms * 1e-3),
            "flop_per_config": flop, "kernel_tflops": flop * w.batch / (kern_ms * 1e-3) * 1e-12,
            "frac_of_dfma_peak": flop * w.batch / (kern_ms * 1e-3) * 1e-12 / dfma_tflops,
            "kernel": ctx.last_kernel_name(), "kernel_ms": kern_ms, "matches_one_species_result": same}


def f32_line(torch, api, runner, flush):
    """FP32 variant ("uplift of up to 80 %") on the headline workload: kernel time against
    the FP64 kernel on the same matrices, and the FP32-vs-FP64 error of the results."""
    w = runner.w
    if w.kind != "hubbard" or w.n > 10:
        return None
    ctx = runner.ctx
    G = torch.empty((w.batch, w.n, w.n), dtype=torch.float64, device="cuda")
    ctx.build_G(runner.xy, runner.tau, G, None, g_diag=w.g_diag)
    o64 = torch.empty(w.batch, dtype=torch.float64, device="cuda")
    o32 = torch.empty_like(o64)
    ms = {}
    ctx.enable_kernel_timer(True)
    for name, fn, out in (("f64", ctx.eval_connected, o64), ("f32", ctx.eval_connected_f32, o32)):
        for _ in range(3):
            fn(G, G, out, U=w.U)
        torch.cuda.synchronize()
        ctx.reset_kernel_timer()
        for _ in range(5):
            flush.fill_(1)
            fn(G, G, out, U=w.U)
        torch.cuda.synchronize()
        ms[name] = ctx.kernel_time_ms()[0]
    ctx.enable_kernel_timer(False)
    rel = ((o32 - o64).abs() / o64.abs()).cpu().numpy()
    return {"workload": w.name, "kernel_ms_f64": ms["f64"], "kernel_ms_f32": ms["f32"], "uplift": ms["f64"] / ms["f32"],
            "configs_per_s_f32": w.batch / (ms["f32"] * 1e-3), "rel_err_vs_f64_median": float(np.median(rel)),
            "rel_err_vs_f64_p90": float(np.quantile(rel, 0.9)), "kernel": "eval_team_kernel<float>"}


def mc_line(torch, runner, flush, eval_kernel_ms):
    """On-device Metropolis driver: walker updates per second on the headline workload and the cost
    of a Monte Carlo step against one plain pass of the hot path ("very little overhead")."""
    w = runner.w
    if w.kind != "hubbard":
        return None
    ctx = runner.ctx
    xy, tau = runner.xy.clone(), runner.tau.clone()
    weight = torch.empty(w.batch, dtype=torch.float64, device="cuda")
    accepted = torch.empty(w.batch, dtype=torch.int64, device="cuda")
    steps = 10
    ctx.mc_run(xy, tau, weight, 2, 1, U=w.U, g_diag=w.g_diag)              # warm-up
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    flush.fill_(1)
    e0.record()
    ctx.mc_run(xy, tau, weight, steps, 2, U=w.U, g_diag=w.g_diag, d_accepted=accepted)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    # one step = 1/(steps+1) of the call (the call also evaluates the initial configurations once)
    per_step = ms / (steps + 1)
    e0.record()
    for _ in range(steps + 1):
        runner.step()
    e1.record()
    torch.cuda.synchronize()
    plain = e0.elapsed_time(e1) / (steps + 1)
    return {"workload": w.name, "walkers": w.batch, "steps": steps, "ms_per_step": per_step,
            "walker_updates_per_s": w.batch / (per_step * 1e-3), "plain_hot_path_ms": plain,
            "overhead_vs_plain_pass": per_step / plain - 1.0,
            "acceptance": float(accepted.double().mean().item() / steps)}


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
