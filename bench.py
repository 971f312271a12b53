#!/usr/bin/env python
"""bench.py -- cell-updates/s of the QUOKKA cell update on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--size n]

One "step" = one pass of the hot path over the box: qk_cfl_dt (eq 21) + qk_hydro_step for the
headline hydro workload (BASELINE.json configs[1], 256^3 Mach-2 turbulence), and qk_cfl_dt +
qk_rhd_step (hydro, N_sub x (radiation transport, exchange)) for the RHD workload
(configs[3], 256^3), reported in the same JSON line under "rhd".  Inputs are the seeded
synthetic generators of paper_2110_01792_b200.inputs.

`value` is timed with CUDA events on the launching stream with the state resident in HBM;
`e2e` is the same step through the C ABI with HOST buffers: every step copies the five
conserved fields host->device from pinned memory (qk_set_state), advances, and copies them
back (qk_get_state), all inside the timed region.  Working set per step (5 x 147 MB read,
plus stage buffers) is several times the 126 MB L2, so no explicit flush is needed.

--impl reference times the CPU oracle (oracle/, plain C, single thread) on a bounded sample of
the same workload; it is a deliberately slow baseline.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "hydro_cell_updates_per_s"
UNIT = "cell-updates/s"
# algorithmic fp64 operations per cell per RK stage (counted from the
# formulas of section 3: one evaluation of every quantity per cell / face, typical branches)
# SURVEY.md section 8(d) / 8(a) figures (branch-free worst-case paths, div and sqrt counted as one op each):
OPS_HYDRO_STAGE = 1240.0    # S3 12 + S4 62 + S5 810 + S6 318 + S7 38
OPS_HYDRO_SWEEP = 388.0     # one direction of one stage: S5 270 + S6 106 + its share of S7 12
OPS_RAD_STAGE = 1080.0      # S8 640 + S9 402 + S10 38
OPS_RAD_SWEEP = 357.0       # one direction: S8 214 + S9 134 + its share of S10 9
HYDRO_WORKLOAD = "config2"  # --workload sedov: the paper's own hydro benchmark problem, context only
CHAT_RATIO = 0.01           # --chat-ratio: c_hat/c of the RHD workload (0.01 = BASELINE configs[3]; 0.5 gives N_sub = 10)
SCHEME_FLAGS = 0            # --plm / --eddington: scheme variants; the headline run uses PPM + Levermore
BYTES_EXCHANGE = 224.0      # 11 reads + 8 writes (eq 26-43) + the 9 reconstruction variables it leaves for the next stage
# dram__bytes_read.sum + dram__bytes_write.sum per launch at 256^3 from the ncu --set full capture summarised in
# profiles/r1_kernels.md (GB); not measured live, null at any other size
NCU_TRAFFIC_GB_256 = {"hydro_sweep_x": 1.465, "hydro_sweep_y": 2.177, "hydro_sweep_z": 3.666,
                      "rad_sweep_x": 1.337, "rad_sweep_y": 1.912, "rad_sweep_z": 3.101, "exchange": 3.750}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ---------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md recipe)
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock, power and clock-event reasons of one GPU through NVML from a thread, every
    ~5 ms, between start() and stop() -- i.e. during the timed region only."""

    def __init__(self, gpu_index):
        self.idx = gpu_index
        self.samples = []
        self.thread = None
        self.stop_flag = False
        self.nv = None

    def _visible_index(self):
        vis = os.environ.get("CUDA_VISIBLE_DEVICES")
        if vis:
            try:
                return int(vis.split(",")[self.idx])
            except Exception:
                return self.idx
        return self.idx

    def _loop(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                self.samples.append((sm, rs, pw))
            except Exception:
                pass
            time.sleep(0.005)

    def start(self):
        try:
            import threading
            import pynvml as nv
            nv.nvmlInit()
            self.nv = nv
            self.h = nv.nvmlDeviceGetHandleByIndex(self._visible_index())
            self.max_sm = nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM)
            self.stop_flag = False
            self.thread = threading.Thread(target=self._loop, daemon=True)
            self.thread.start()
        except Exception as e:      # no NVML: report that instead of inventing a number
            log("clock sampler unavailable: %r" % (e,))
            self.thread = None

    def stop(self):
        if self.thread is None:
            return None
        self.stop_flag = True
        self.thread.join(timeout=2)
        nv = self.nv
        if not self.samples:
            return None
        bits = {"hw_slowdown": nv.nvmlClocksEventReasonHwSlowdown,
                "hw_thermal_slowdown": nv.nvmlClocksEventReasonHwThermalSlowdown,
                "sw_thermal_slowdown": nv.nvmlClocksEventReasonSwThermalSlowdown,
                "sw_power_cap": nv.nvmlClocksEventReasonSwPowerCap,
                "hw_power_brake": nv.nvmlClocksEventReasonHwPowerBrakeSlowdown}
        reasons = sorted(n for n, b in bits.items() if any(r & b for _, r, _ in self.samples))
        return {"sm_mhz": float(np.median([s[0] for s in self.samples])), "sm_max_mhz": float(self.max_sm),
                "reasons": reasons, "samples": len(self.samples),
                "power_w_max": float(max(s[2] for s in self.samples))}


# ---------------------------------------------------------------------------------------------
# the CPU oracle on a bounded sample (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------
def oracle_sample(kind, n, steps, seed_shift=0):
    """Time `steps` oracle steps of the workload generator at n^3.  Returns (updates/s, seconds)."""
    import oracle as O
    from paper_2110_01792_b200 import inputs as I
    params, fields = (I.config2(n=n, seed=1002 + seed_shift) if kind == "hydro"
                      else I.config4(n=n, seed=1004 + seed_shift))
    g = O.Grid(params["nx"], params["ny"], params["nz"], params["dx"], params["gamma"],
               c_hat=params.get("c_hat", 0.0), c=params.get("c", 0.0), bc=params["bc"])
    if "a_rad" in params:
        g.set_constants(params["a_rad"], params["kB_mu"])
    g.set_params(cfl=params["cfl"], flags=params["flags"])
    g.set_all(fields)
    t0 = time.perf_counter()
    for _ in range(steps):
        dt = g.cfl_dt()
        rc = g.hydro_step(dt) if kind == "hydro" else g.rhd_step(dt)
        assert rc == 0, rc
    sec = time.perf_counter() - t0
    g.close()
    return n ** 3 * steps / sec, sec


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = args.ref_size
    # W warm-up "steps" and K timed ones, each one oracle step on the n^3 sample
    import oracle as O
    from paper_2110_01792_b200 import inputs as I
    params, fields = I.config2(n=n)
    g = O.Grid(n, n, n, params["dx"], params["gamma"], bc=params["bc"])
    g.set_params(cfl=params["cfl"], flags=params["flags"])
    g.set_all(fields)
    for _ in range(args.warmup):
        g.hydro_step(g.cfl_dt())
    t0 = time.perf_counter()
    for _ in range(args.steps):
        assert g.hydro_step(g.cfl_dt()) == 0
    sec = time.perf_counter() - t0
    g.close()
    value = n ** 3 * args.steps / sec
    sample = "oracle (plain C, -O2 -ffp-contract=off, 1 thread) on a %d^3 box of the config2 generator, %d steps" % (
        n, args.steps)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[1] generator (hydro, Mach-2 turbulence, periodic, "
                                   "gamma=5/3, CFL 0.3), bounded sample %d^3" % n},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
# the CUDA path
# ---------------------------------------------------------------------------------------------
def one_step(ctx, kind, ex):
    """qk_cfl_dt (min over ranks when the box is decomposed) + one step of the hot path."""
    dt = ctx.qk_cfl_dt()
    if ex is not None:
        dt = ex.global_dt(dt)
    if kind == "hydro":
        ctx.qk_hydro_step(dt)
    else:
        ctx.qk_rhd_step(dt)
    if ex is not None:
        ex.check()


def time_steps(torch, ctx, kind, nsteps, barrier, ex=None, fixed_dt=None):
    """nsteps x (qk_cfl_dt + step) bracketed by barrier + synchronize, timed with CUDA events on the
    stream the kernels are launched on.  Returns milliseconds.  With fixed_dt the per-step qk_cfl_dt (one
    host read of 16 bytes) is left out: the launch queue never drains."""
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(nsteps):
        if fixed_dt is not None:
            ctx.qk_hydro_step(fixed_dt) if kind == "hydro" else ctx.qk_rhd_step(fixed_dt)
            continue
        one_step(ctx, kind, ex)
    e1.record(stream)
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1)


def time_steps_e2e(torch, ctx, kind, nsteps, host_in, host_out, barrier, ex=None):
    """Same step through the C ABI with HOST (pinned) buffers: H2D of the evolving fields, step,
    D2H of the result, every step, inside the timed region."""
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    nf = len(host_in)
    barrier()
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(nsteps):
        for f in range(nf):
            ctx.qk_set_state(f, host_in[f])
        one_step(ctx, kind, ex)
        for f in range(nf):
            ctx.qk_get_state(f, host_out[f])
        host_in, host_out = host_out, host_in      # next step starts from this step's result
    e1.record(stream)
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1)


def run_workload(torch, B, I, kind, n, steps, warmup, rank, world, barrier, allmax, sampler=None, path=None,
                 decompose=False):
    t0 = time.time()
    if kind == "hydro":
        params, fields = I.sedov(n=n) if HYDRO_WORKLOAD == "sedov" else I.config2(n=n, seed=1002 + rank)
    else:
        params, fields = I.config4(n=n, seed=1004 + rank, chat_ratio=CHAT_RATIO)
    params["flags"] |= SCHEME_FLAGS
    log("[rank %d] %s %d^3 inputs generated in %.1f s" % (rank, kind, n, time.time() - t0))
    nf = 5 if kind == "hydro" else 9
    cells = n ** 3
    out = {}
    with B.from_params(params, fields) as ctx:
        if path is not None:
            ctx.qk_set_path(path)
        ex = None
        if decompose and world > 1:
            # one global box of n x n x (world n) cells, rank r owns the z slab r: ghost planes cross ranks by
            # NCCL send/recv before every stage fill, dt is the minimum over ranks
            from paper_2110_01792_b200 import decomp as D
            ex = D.SlabExchange(ctx, rank, world, True, D.TorchTransport())
        out["parallelism"] = ("z-slab decomposition of one %dx%dx%d box, halo exchange per RK stage (NCCL p2p), "
                              "global min dt" % (n, n, n * world)) if ex else "1 box per GPU"
        for _ in range(warmup):
            one_step(ctx, kind, ex)
        ctx.set_all(fields)                        # timed steps are steps 1..K of the config
        torch.cuda.synchronize()
        l0 = ctx.qk_launch_count()
        ctx.qk_set_profiling(True)
        if sampler:
            sampler.start()
        ms = time_steps(torch, ctx, kind, steps, barrier, ex)
        clocks = sampler.stop() if sampler else None
        ktimes = ctx.qk_kernel_times()
        ctx.qk_set_profiling(False)
        launches = ctx.qk_launch_count() - l0
        info = ctx.qk_last_info()
        ms = allmax(ms)
        out.update(ms=ms, value=world * cells * steps / (ms * 1e-3), launches=launches, kernel_ms=ktimes,
                   clocks=clocks, info=info)
        if ex is None:      # same steps at a fixed dt (half the current CFL step), no host round trip per step
            dt_fixed = 0.5 * ctx.qk_cfl_dt()
            ms_f = allmax(time_steps(torch, ctx, kind, steps, barrier, None, dt_fixed))
            out["fixed_dt"] = {"value": world * cells * steps / (ms_f * 1e-3), "unit": UNIT, "ms_per_step": ms_f / steps}
        # end to end with host buffers
        host_a = [torch.from_numpy(np.ascontiguousarray(fields[I.FIELDS[f]])).pin_memory() for f in range(nf)]
        host_b = [torch.empty_like(t).pin_memory() for t in host_a]
        e2e_steps = max(1, min(steps, 5))
        time_steps_e2e(torch, ctx, kind, 1, [t.clone().pin_memory() for t in host_a], host_b, barrier, ex)  # warm
        ms_e = allmax(time_steps_e2e(torch, ctx, kind, e2e_steps, host_a, host_b, barrier, ex))
        out["e2e"] = {"value": world * cells * e2e_steps / (ms_e * 1e-3), "unit": UNIT,
                      "h2d_bytes_per_step": nf * cells * 8, "d2h_bytes_per_step": nf * cells * 8,
                      "ms_per_step": ms_e / e2e_steps, "steps": e2e_steps}
        if ex is not None:
            out["halo"] = {"exchanges": ex.calls, "bytes_sent_per_rank": ex.bytes_sent}
            ex.detach()
    return out


def roofline_alu(kernel_ms, names, ops_per_cell_per_launch, cells, peak_ops, peak_note):
    """Dominant ALU-bound kernel: algorithmic fp64 ops per launch / mean launch duration."""
    present = [nm for nm in names if nm in kernel_ms]
    if present:          # the slowest class of the family is the dominant kernel
        nm = max(present, key=lambda k: kernel_ms[k][0] / kernel_ms[k][1])
        if True:
            tot, cnt = kernel_ms[nm]
            mean_ms = tot / cnt
            achieved = ops_per_cell_per_launch * cells / (mean_ms * 1e-3) / 1e12
            traffic = NCU_TRAFFIC_GB_256.get(nm) if cells == 256 ** 3 else None
            return {"bound": "alu", "kernel": nm, "achieved": achieved, "peak": peak_ops / 1e12,
                    "unit": "TFLOP/s", "frac": achieved / (peak_ops / 1e12),
                    "traffic": None if traffic is None else traffic * 1e9,
                    "launch_ms": mean_ms, "launches": cnt, "peak_source": peak_note,
                    "ops_per_cell_per_launch": ops_per_cell_per_launch}
    return None


def run_ours(args):
    import torch
    from paper_2110_01792_b200 import binding as B
    from paper_2110_01792_b200 import inputs as I

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the library has no CPU path)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()

    def allmax(x):
        if dist is None:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    B.lib()     # fails loudly if libqk.so is absent
    n = args.size
    cells = n ** 3
    # roofline denominators: measured fp64 pipe rate (DMUL+DADD mix, -fmad=false) and HBM copy
    peak_ops = B.qk_fp64_probe(0, 4000)
    peak_fma = B.qk_fp64_probe(1, 4000)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    hbm_note = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"

    sampler = ClockSampler(local) if rank == 0 else None
    path = {"fused": B.QK_PATH_FUSED, "unfused": B.QK_PATH_UNFUSED, "sweep": B.QK_PATH_SWEEP}[args.path]
    hyd = None
    if not args.no_hydro:
        hyd = run_workload(torch, B, I, "hydro", n, args.steps, args.warmup, rank, world, barrier, allmax, sampler, path,
                           decompose=not args.replicas)
    rhd = None
    if not args.no_rhd or hyd is None:
        rhd_steps = max(1, min(args.steps, args.rhd_steps))
        rhd = run_workload(torch, B, I, "rhd", n, rhd_steps, min(args.warmup, 3), rank, world, barrier, allmax,
                           sampler if hyd is None else None, path, decompose=not args.replicas)
        rhd["steps"] = rhd_steps

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    peak_note = "qk_fp64_probe: measured DMUL+DADD lane-ops/s on this GPU (DFMA probe: %.2f T/s)" % (peak_fma / 1e12)
    def family(kms, stage, sweeps, ops_stage, ops_sweep):
        if stage in kms:
            return [stage], ops_stage
        return sweeps, ops_sweep

    roof = None
    if hyd is not None:
        names, ops = family(hyd["kernel_ms"], "hydro_stage", ["hydro_sweep_x", "hydro_sweep_y", "hydro_sweep_z",
                                                              "hydro_flux"], OPS_HYDRO_STAGE, OPS_HYDRO_SWEEP)
        roof = roofline_alu(hyd["kernel_ms"], names, ops, cells, peak_ops, peak_note)
    if hyd is None:      # --no-hydro (profiling aid): the RHD workload alone fills the line
        hyd = rhd
        args.steps = rhd["steps"]
    line = {
        "metric": METRIC if hyd is not rhd else "rhd_cell_updates_per_s", "value": hyd["value"], "unit": UNIT,
        "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": hyd["ms"] / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": ("BASELINE.json configs[1]: pure hydro %d^3, periodic, gamma=5/3, log-normal density, "
                                "k^-2 velocity field at rms Mach 2, CFL 0.3, qk_cfl_dt + qk_hydro_step per step" % n)
                               if HYDRO_WORKLOAD == "config2" else
                               ("Sedov blast %d^3 on [-1,1]^3, periodic, gamma=5/3, CFL 0.25 (PAPER.md:572), "
                                "qk_cfl_dt + qk_hydro_step per step" % n),
                   "scheme": ("PLM" if SCHEME_FLAGS & 8 else "PPM") + (" + Eddington closure" if SCHEME_FLAGS & 16 else " + Levermore closure"),
                   "cells": cells, "l2": "inputs larger than L2 (5 x %.0f MB per stage)" % (cells * 8 / 1e6),
                   "parallelism": hyd.get("parallelism", "1 box on 1 GPU") if world > 1 else "1 box on 1 GPU"},
        "e2e": hyd["e2e"], "gpu_launches": hyd["launches"], "clocks": hyd["clocks"],
        "roofline": roof,
        "kernel_ms": {k: {"total_ms": v[0], "groups": v[1]} for k, v in hyd["kernel_ms"].items()},
        "peaks": {"fp64_dmul_dadd_lane_ops_per_s": peak_ops, "fp64_dfma_lane_ops_per_s": peak_fma,
                  "hbm_gbs": hbm, "hbm_source": hbm_note},
    }
    if hyd.get("halo"):
        line["halo"] = hyd["halo"]
    if hyd.get("fixed_dt"):
        line["fixed_dt"] = hyd["fixed_dt"]
    if rhd is not None:
        ex = rhd["kernel_ms"].get("exchange")
        names, ops = family(rhd["kernel_ms"], "rad_stage", ["rad_sweep_x", "rad_sweep_y", "rad_sweep_z", "rad_flux"],
                            OPS_RAD_STAGE, OPS_RAD_SWEEP)
        rroof = roofline_alu(rhd["kernel_ms"], names, ops, cells, peak_ops, peak_note)
        exroof = None
        if ex:
            ach = BYTES_EXCHANGE * cells / (ex[0] / ex[1] * 1e-3) / 1e9
            exroof = {"bound": "hbm", "kernel": "exchange", "achieved": ach, "peak": hbm, "unit": "GB/s",
                      "frac": ach / hbm, "traffic": NCU_TRAFFIC_GB_256["exchange"] * 1e9 if cells == 256 ** 3 else None,
                      "launch_ms": ex[0] / ex[1], "peak_source": hbm_note}
        line["rhd"] = {
            "metric": "rhd_cell_updates_per_s", "value": rhd["value"], "unit": UNIT, "steps": rhd["steps"],
            "ms_per_step": rhd["ms"] / rhd["steps"], "nsub": rhd["info"]["nsub"],
            "config": {"workload": "BASELINE.json configs[3]: coupled RHD %d^3, periodic, c_hat/c=%g, "
                                   "qk_cfl_dt + qk_rhd_step per step" % (n, CHAT_RATIO)},
            "e2e": rhd["e2e"], "gpu_launches": rhd["launches"],
            "roofline_rad": rroof, "roofline_exchange": exroof, "fixed_dt": rhd.get("fixed_dt"),
            "kernel_ms": {k: {"total_ms": v[0], "groups": v[1]} for k, v in rhd["kernel_ms"].items()},
            "newton_mean_iters": rhd["info"]["newton_total_iters"] / max(1, cells * rhd["info"]["nsub"]),
        }
    if world == 1 and not args.no_cpu_baseline:
        v, sec = oracle_sample("hydro", args.ref_size, 2)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": "oracle (plain C, 1 thread) on a %d^3 box of the config2 generator, 2 steps, "
                                          "%.1f s" % (args.ref_size, sec)}
        if rhd is not None:
            v2, sec2 = oracle_sample("rhd", max(16, args.ref_size * 3 // 4), 2)
            line["rhd"]["cpu_baseline"] = {"value": v2, "unit": UNIT, "cores": 1, "kind": "oracle",
                                           "sample": "oracle on a %d^3 box of the config4 generator, 2 steps, %.1f s"
                                                     % (max(16, args.ref_size * 3 // 4), sec2)}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size", type=int, default=256, help="box edge (BASELINE metric: 256)")
    ap.add_argument("--rhd-steps", type=int, default=10)
    ap.add_argument("--ref-size", type=int, default=128, help="edge of the oracle's bounded sample")
    ap.add_argument("--path", default="sweep", choices=["fused", "unfused", "sweep"], help="stage kernel family")
    ap.add_argument("--replicas", action="store_true",
                    help="N>1: independent boxes per GPU instead of one z-slab-decomposed global box")
    ap.add_argument("--workload", default="config2", choices=["config2", "sedov"],
                    help="hydro workload: BASELINE configs[1] (default, the metric) or the paper's Sedov blast (CFL 0.25)")
    ap.add_argument("--chat-ratio", type=float, default=0.01,
                    help="c_hat/c of the RHD workload; 0.5 makes every step take N_sub = N_sub,max = 10 radiation "
                         "substeps like the paper's RHD benchmark (PAPER.md:604)")
    ap.add_argument("--plm", action="store_true", help="PLM + MC limiter instead of PPM (PAPER.md:164)")
    ap.add_argument("--eddington", action="store_true", help="Eddington approximation instead of the Levermore closure")
    ap.add_argument("--no-rhd", action="store_true")
    ap.add_argument("--no-hydro", action="store_true", help="profiling aid: run only the RHD workload")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    global SCHEME_FLAGS, HYDRO_WORKLOAD, CHAT_RATIO
    CHAT_RATIO = args.chat_ratio
    HYDRO_WORKLOAD = args.workload
    SCHEME_FLAGS = (8 if args.plm else 0) | (16 if args.eddington else 0)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
