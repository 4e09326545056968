#!/usr/bin/env python
"""bench.py -- CN time steps/s (and BiCGSTAB iterations/s, operator applies/s) of the TDDE propagator on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config hbm|large|medium|...] [--impl ours|reference]

One "step" is one Crank-Nicolson step = one pass of the whole hot path (two start-of-step applies, the BiCGSTAB
iterations with their preconditioner solves, fused vector kernels and on-device scalar updates).
The default workload is BASELINE.json's HBM-scale synthetic config, the largest single-GPU configuration
(vectors of 512 MB: every pass is larger than the 126 MB L2, so no L2 flush is needed between steps).
Prints ONE JSON line (see DESIGN.md "Measurement" for every field).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import tdde_inputs  # noqa: E402

METRIC = "cn_time_steps_per_s"
UNIT = "steps/s"
FP64_FMA_PER_CLK_PER_SM = 64          # B200: 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz = 37.2 TFLOP/s nominal
WORKLOADS = sorted(tdde_inputs.CONFIGS) + ["hydrogen", "nondipole"]
# dram__bytes_read.sum + dram__bytes_write.sum of one in-iteration operator-apply launch per workload, from `ncu --set full`
# captures; bench.py cannot run ncu itself, so it reads the table kept beside the captures (profiles/r02_apply_traffic.md
# names the command).  A workload without a row reports null.
TRAFFIC_TABLE = os.path.join(ROOT, "profiles", "r02_apply_traffic.csv")


def load_problem(name: str, phase: float = 0.0, e0=None, **kw):
    """BASELINE.json configs by name; "hydrogen" = configs[1] with the 1s1/2 state as c0 and the pulse shifted to its maximum."""
    if name == "hydrogen":
        import scipy.linalg as sla
        p = tdde_inputs.make_hydrogen(**({} if e0 is None else {"e0": e0}))
        S, H = p.meta["dense"][-1]
        E, V = sla.eigh(H, S)
        j = int(np.nonzero(E > -p.meta["c"] ** 2)[0][0])
        a = p.meta["chans"].index((-1, 0.5))
        p.c0[a * p.n_rad:(a + 1) * p.n_rad] = V[:, j]
        return p
    if name == "nondipole":       # x-polarised non-dipole operator set, kappa_max = 15, l_max = 2 (24 terms)
        from tdde_inputs import nondipole as nd
        return nd.set_ground_state(nd.make_nondipole(kappa_max=15, l_max=2, n_r=100, r_max=60.0, t_offset=6.0,
                                                     **({} if e0 is None else {"e0": e0})))
    if e0 is not None:
        kw["e0"] = e0
    return tdde_inputs.make_config(name, phase=phase, **kw)


def measured_traffic(workload: str):
    if not os.path.exists(TRAFFIC_TABLE):
        return None
    with open(TRAFFIC_TABLE) as f:
        for line in f:
            cells = [c.strip() for c in line.split(",")]
            if len(cells) >= 2 and cells[0] == workload:
                try:
                    return float(cells[1])
                except ValueError:
                    return None
    return None


def f_apply(p) -> int:
    """Complex FMAs per vector element of one operator apply: n_d + sum_L (n_d + nnz_row(A_L))."""
    nd = 2 * p.w0 + 1
    tot = nd
    for t in p.terms:
        nnz_row = int(np.max(np.diff(t.A_rowptr)))       # interior rows
        tot += (2 * t.w + 1) + nnz_row
    return tot


def num_sms() -> int:
    import torch
    return int(torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.05)

    def result(self):
        self.stop_flag = True
        if self.nv is None or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}


# ----------------------------------------------------------------------------------------------- reference arm
FULL_CSR_MAX_N = 600_000        # the oracle's explicit CSR fits comfortably (Medium: 0.2 G non-zeros)
FULL_PANELS_MAX_N = 8_000_000   # the oracle's matrix-free form on the WHOLE config stays near 20 s per step (Large)


def oracle_sample_problem(cfg_name: str, sample_ang: int, phase: float, e0):
    """The same workload recipe restricted to `sample_ang` angular channels (all radial sizes, bandwidth, terms kept)."""
    args = dict(tdde_inputs.CONFIGS[cfg_name])
    full_n = args["n_ang"] * 2 * args["n_r"]
    args["n_ang"] = min(sample_ang, args["n_ang"])
    if e0 is not None:
        args["e0"] = e0
    p = tdde_inputs.make_synthetic(name=cfg_name + "-sample", phase=phase, **args)
    return p, full_n


def run_oracle(cfg_name: str, steps: int, warmup: int, sample_ang: int, phase: float = 0.0, e0=None, allow_panels: bool = True):
    """Times the CPU oracle as it stands (SciPy CSR / NumPy + textbook BiCGSTAB, one thread).
    Small workloads (Tiny, Hydrogen, Medium) run WHOLE: a measured number.  Large runs whole through the oracle's
    matrix-free form (also measured).  HBM-scale would need minutes per step: there the recipe is cut to `sample_ang`
    channels and the rate is scaled by n_sample / n_full -- labelled "extrapolated"."""
    from oracle import tdde_oracle as orc
    special = cfg_name in ("hydrogen", "nondipole")
    n_full = None if special else tdde_inputs.CONFIGS[cfg_name]["n_ang"] * 2 * tdde_inputs.CONFIGS[cfg_name]["n_r"]
    extrapolated, mode = False, "whole workload, explicit CSR"
    if cfg_name == "nondipole":
        p = load_problem(cfg_name, phase, e0)
        full_n = p.n
        fact = orc.factor_precond(p)
        mode = "whole workload, matrix-free panels"
        step = lambda c, s: orc.cn_step_panels(p, fact, c, p.g_mid(s), p.dt, p.rtol, p.max_iter)
    elif cfg_name == "hydrogen" or n_full <= FULL_CSR_MAX_N:
        p = load_problem(cfg_name, phase, e0)
        full_n = p.n
        ops = orc.assemble(p)
        fact = orc.factor_precond(p)
        step = lambda c, s: orc.cn_step(ops, fact, c, p.g_mid(s), p.dt, p.rtol, p.max_iter, assembled=False)
    elif n_full <= FULL_PANELS_MAX_N and allow_panels:
        p = load_problem(cfg_name, phase, e0)
        full_n = p.n
        fact = orc.factor_precond(p)
        mode = "whole workload, matrix-free panels (CSR would need ~25 GB)"
        step = lambda c, s: orc.cn_step_panels(p, fact, c, p.g_mid(s), p.dt, p.rtol, p.max_iter)
    else:
        p, full_n = oracle_sample_problem(cfg_name, sample_ang, phase, e0)
        ops = orc.assemble(p)
        fact = orc.factor_precond(p)
        extrapolated = True
        mode = (f"recipe cut to {p.n_ang} of {tdde_inputs.CONFIGS[cfg_name]['n_ang']} angular channels (n={p.n}); "
                "value = sample steps/s x n_sample/n_full")
        step = lambda c, s: orc.cn_step(ops, fact, c, p.g_mid(s), p.dt, p.rtol, p.max_iter)
    c = p.c0.copy()
    for s_ in range(warmup):
        c, _ = step(c, s_)
    half = 0
    t0 = time.perf_counter()
    for s_ in range(steps):
        c, info = step(c, warmup + s_)
        half += info.half_iters
    dt = time.perf_counter() - t0
    value = steps / dt * (p.n / full_n)
    return dict(value=value, unit=UNIT, cores=1, kind="oracle", extrapolated=extrapolated, steps=steps, seconds=dt, half_iters=half,
                sample=f"{cfg_name}: {mode}; {steps} CN steps in {dt:.2f} s on 1 core"), p


def reference_main(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # every timed step is a bounded sample of the workload (whole for the small configs, a channel cut for Large / HBM-scale)
    cb, p = run_oracle(args.config, args.steps, args.warmup, args.sample_ang, args.phase, args.e0, allow_panels=False)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": cb["steps"], "warmup": args.warmup, "ms_per_step": 1e3 / cb["value"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.config, "phase": args.phase, "note": "CPU oracle: " + cb["sample"]},
            "cpu_baseline": {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample", "extrapolated")},
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def max_over_ranks(values, device="cpu"):
    """Element-wise MAX of a list of floats over all ranks of the default process group (any backend)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_rate(world: int, steps: int, max_ms: float) -> float:
    """Replicas only: every rank advances its own copy K steps; the job rate is N*K over the slowest rank."""
    return world * steps / (max_ms * 1e-3)


# ------------------------------------------------------------------------------ NEXT-3: channel-slab shards on one GPU
def sharded_main(args):
    """--shards N: the lock-step sharded driver (tdde_group_*) with all N shards in this process on ONE GPU, next to the
    unsharded propagation of the same problem.  It measures the overhead of the sharded driver (halo copies, split reductions, one
    host read per step, halo recomputation), NOT scaling: the pool has one-GPU boxes."""
    import torch
    from paper_2512_21697_b200 import Tdde, TddeGroup, sharding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device")
    K, W, N = args.steps, max(args.warmup, 3), args.shards
    p = load_problem(args.config, args.phase, args.e0)
    g_all = p.g_table(W + K)
    prop = Tdde(p)
    c = prop.to_device(p.c0)
    prop.propagate(c, g_all[:W])
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); st1 = prop.propagate(c, g_all[W:W + K]); e1.record(); torch.cuda.synchronize()
    ms1 = e0.elapsed_time(e1)
    c_ref = c.cpu().numpy().reshape(p.n_ang, p.n_rad)
    prop.close(); del c
    parts = sharding.shard_specs(p, N)
    shards = [Tdde(pl) for _, pl, _ in parts]
    grp = TddeGroup(shards, [sp for _, _, sp in parts])
    c0 = p.c0.reshape(p.n_ang, p.n_rad)
    cs = [sh.to_device(np.ascontiguousarray(c0[pl.halo_lo:pl.halo_hi]).reshape(-1)) for (pl, _, _), sh in zip(parts, shards)]
    grp.propagate(cs, g_all[:W])
    e0.record(); st = grp.propagate(cs, g_all[W:W + K]); e1.record(); torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    err2 = ref2 = 0.0
    for (pl, _, _), cd in zip(parts, cs):
        own = cd.cpu().numpy().reshape(pl.n_local, p.n_rad)[pl.own_slice]
        err2 += float(np.sum(np.abs(own - c_ref[pl.lo:pl.hi]) ** 2)); ref2 += float(np.sum(np.abs(c_ref[pl.lo:pl.hi]) ** 2))
    print(json.dumps({"metric": METRIC, "value": K / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms / K,
                      "higher_is_better": True, "impl": "ours-sharded", "dtype": "f64", "data": "synthetic",
                      "config": {"workload": args.config, "n_ang": p.n_ang, "n_rad": p.n_rad, "n_terms": p.n_terms,
                                 "parallelism": "%d channel-slab shards in ONE process on 1 GPU (lock-step driver: overhead, not scaling)" % N,
                                 "halo_channels_per_side": parts[0][0].reach},
                      "half_iters_per_step": st["half_iters"] / K, "unsharded_ms_per_step": ms1 / K,
                      "unsharded_half_iters_per_step": st1["half_iters"] / K, "overhead": ms / ms1 - 1.0,
                      "rel_diff_vs_unsharded": (err2 / ref2) ** 0.5}))
    grp.close()
    for sh in shards:
        sh.close()


# ----------------------------------------------------------------------------------------------------- our arm
def ours_main(args):
    import torch
    import torch.distributed as dist
    from paper_2512_21697_b200 import Tdde

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    K, W = args.steps, max(args.warmup, 3)
    p = load_problem(args.config, args.phase, args.e0)
    prop = Tdde(p, device=f"cuda:{local}")
    g_all = p.g_table(W + K)
    c = prop.to_device(p.c0)
    n, T = p.n, p.n_terms

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K steps ----
    prop.propagate(c, g_all[:W])
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    launches0 = prop.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    st = prop.propagate(c, g_all[W:W + K])
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = prop.launch_count - launches0
    norm_end = prop.norm(c)

    # ---- per-kernel timings, live, CUDA events on the handle's stream (same process, right after) ----
    g_mid = np.where(g_all[W] == 0.0, 1e-3, g_all[W])          # per-kernel timings: never a field that is exactly zero
    reps = args.kernel_reps
    kt = {name: prop.time_kernel(which, reps, g_mid) for which, name in
          [(0, "apply"), (1, "precond"), (2, "vec_p"), (3, "vec_s"), (4, "vec_xr"), (5, "transpose"), (6, "apply_S")]}
    fp64_peak_meas = prop.fp64_peak()
    dmma_peak_meas, mixed_peak_meas = prop.fp64_pipe_probe(1), prop.fp64_pipe_probe(2)
    pv = None
    if args.paper_variant and prop.apply_path == "banded":
        xv = prop.to_device(p.c0)
        _, ta, ts, nnz = prop.paper_variant(g_mid, xv, reps=3)
        pv = {"nnz": nnz, "assemble_ms": ta, "spmv_ms": ts, "spmv_GBps": 20.0 * nnz / (ts * 1e-3) / 1e9,
              "note": "paper's formulation on this GPU (PAPER.md:301-305): one CSR assembly per step, one SpMV per apply"}
        del xv
    clocks = sampler.result()

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    c_host_t = torch.empty(n, dtype=torch.complex128).pin_memory()
    c_host = c_host_t.numpy()
    c_host[:] = p.c0
    prop.propagate_host(c_host, g_all[:W], W)              # warm-up (allocates the staging buffer)
    barrier()
    t0 = time.perf_counter()
    prop.propagate_host(c_host, g_all[W:W + K], K)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    # the same K steps as K calls of one step each: the state crosses PCIe both ways on EVERY step
    c_host[:] = p.c0
    prop.propagate_host(c_host, g_all[:W], W)
    barrier()
    t0 = time.perf_counter()
    for s_ in range(K):
        prop.propagate_host(c_host, g_all[W + s_:W + s_ + 1], 1)
    torch.cuda.synchronize()
    e2e1_s = time.perf_counter() - t0

    ms, e2e_ms, e2e1_ms = max_over_ranks([ms, e2e_s * 1e3, e2e1_s * 1e3], device="cuda")

    if rank == 0:
        peaks, peak_kind = load_peaks()
        # the timed kernel is the in-iteration apply v = p + i tau (coupling terms) y: the block part (n_d cFMA) is replaced
        # by adding the known vector p, so it is not counted
        subst = prop.apply_path == "banded" and T > 0
        F = f_apply(p) - (2 * p.w0 + 1) if subst else f_apply(p)
        nint = n                                            # algorithmic element count (pads excluded)
        flops_apply = 8.0 * F * nint
        sm_max = float(peaks.get("sm_max_mhz", 1965.0))
        n_sm = num_sms()
        fp64_peak_nominal = n_sm * FP64_FMA_PER_CLK_PER_SM * 2 * sm_max * 1e6
        traffic = measured_traffic(args.config)
        t_apply = kt["apply"] * 1e-3
        ach = flops_apply / t_apply / 1e12
        hbm = float(peaks["hbm_gbs"])
        bytes_per = {"apply": 64 if subst else 48, "precond": 32, "vec_p": 64, "vec_s": 48, "vec_xr": 128, "transpose": 32, "apply_S": 32}
        kernels = {k: {"ms": v, "alg_GBps": bytes_per[k] * nint / (v * 1e-3) / 1e9,
                       "hbm_frac": bytes_per[k] * nint / (v * 1e-3) / 1e9 / hbm} for k, v in kt.items()}
        steps_per_s = whole_job_rate(world, K, ms)
        line = {
            "metric": METRIC, "value": steps_per_s, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.config, "n_ang": p.n_ang, "n_rad": p.n_rad, "n": n, "bandwidth": 2 * p.w0 + 1,
                       "n_terms": T, "dt": p.dt, "rtol": p.rtol, "seed": p.seed, "phase": args.phase, "e0": p.meta.get("e0"),
                       "apply_path": prop.apply_path, "parallelism": "replicas only" if world > 1 else "1 GPU",
                       "l2": "vectors (%.0f MB each) exceed the 126 MB L2; no flush" % (n * 16 / 1e6)},
            "bicgstab_iters_per_s": world * 0.5 * st["half_iters"] / (ms * 1e-3),
            "applies_per_s": world * st["applies"] / (ms * 1e-3),
            "half_iters_per_step": st["half_iters"] / K, "rel_res": st["rel_res"], "s_norm_end": norm_end,
            "gpu_launches": launches,
            "clocks": clocks,
            "e2e": {"value": whole_job_rate(world, K, e2e_ms), "unit": UNIT,
                    "h2d_bytes_per_step": (n * 16 + K * T * 8) / K, "d2h_bytes_per_step": n * 16 / K,
                    "note": "one tdde_propagate_host call of K steps: state vector H2D + g table H2D + K steps + state D2H",
                    "per_step_copies": {"value": whole_job_rate(world, K, e2e1_ms), "unit": UNIT,
                                        "h2d_bytes_per_step": n * 16 + T * 8, "d2h_bytes_per_step": n * 16,
                                        "note": "K tdde_propagate_host calls of one step each"}},
            "roofline": {"bound": "alu",
                         "kernel": (prop.iter_apply_kernel + " (v = A y = p + i tau (sum_L g_L A_L (x) R_L) y with fused <rhat,v>)" if subst else
                                    prop.iter_apply_kernel + " (v = A y with fused <rhat,v>)"),
                         "achieved": ach, "peak": fp64_peak_nominal / 1e12, "unit": "TFLOP/s",
                         "frac": ach / (fp64_peak_nominal / 1e12), "traffic": traffic,
                         "algorithmic_bytes_per_launch": bytes_per["apply"] * nint,
                         "peak_kind": "derived: %d SMs x 64 DFMA/clk x 2 x %.0f MHz" % (n_sm, sm_max),
                         "fp64_peak_measured_tflops": fp64_peak_meas / 1e12,
                         "fp64_pipe_probe_tflops": {"dfma": fp64_peak_meas / 1e12, "dmma": dmma_peak_meas / 1e12,
                                                    "dmma_dfma_mixed": mixed_peak_meas / 1e12,
                                                    "note": "DMMA (mma.sync.m8n8k4.f64) and DFMA share one pipe on B200: one peak for both"},
                         "frac_of_measured_dfma": ach / (fp64_peak_meas / 1e12),
                         "cfma_per_element": F, "flops_per_launch": flops_apply,
                         "alg_hbm_GBps": kernels["apply"]["alg_GBps"], "hbm_peak_GBps": hbm, "hbm_peak_kind": peak_kind},
            "kernels": kernels,
            "paper_variant": pv,
        }
        if world == 1 and not args.no_cpu_baseline:
            n_o = 1 if p.n > FULL_CSR_MAX_N and p.n <= FULL_PANELS_MAX_N else 4
            cb, _ = run_oracle(args.config, n_o, 0, args.sample_ang, args.phase, args.e0)
            line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample", "extrapolated")}
        print(json.dumps(line))
    prop.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="hbm", choices=WORKLOADS)
    ap.add_argument("--phase", type=float, default=0.0, help="phase of g(t) = E0 sin(w t + phase); 0 = BASELINE config")
    ap.add_argument("--e0", type=float, default=None, help="field amplitude E0 (default: the BASELINE value 0.05); the supplementary "
                    "stress run of SURVEY 8(d) D2 uses --phase 1.5708 with a larger E0 so that a step needs several full iterations")
    ap.add_argument("--kernel-reps", type=int, default=10)
    ap.add_argument("--sample-ang", type=int, default=24, help="angular channels of the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--shards", type=int, default=0, help="N >= 2: run the channel-slab sharded driver with N shards in this process on one "
                    "GPU next to the unsharded run (DESIGN.md 7: driver overhead, not scaling)")
    ap.add_argument("--paper-variant", action="store_true",
                    help="also time the paper's formulation (CSR assembly + SpMV) on this GPU; needs 20 B per non-zero")
    args = ap.parse_args()
    if args.impl == "reference":
        reference_main(args)
    elif args.shards >= 2:
        sharded_main(args)
    else:
        ours_main(args)


if __name__ == "__main__":
    main()
