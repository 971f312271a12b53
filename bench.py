#!/usr/bin/env python
"""bench.py -- cell-updates/s of the QUOKKA cell update on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--size n]

One "step" = one pass of the hot path over the box: qk_cfl_dt (eq 21) + qk_hydro_step for the
headline hydro workload (BASELINE.json configs[1], 256^3 Mach-2 turbulence), and qk_cfl_dt +
qk_rhd_step (hydro, N_sub x (radiation transport, exchange)) for the RHD workload
(configs[3], 256^3), reported in the same JSON line under "rhd".  Inputs are the seeded
synthetic generators of paper_2110_01792_b200.inputs.

`value` is timed with CUDA events on the launching stream with the state resident in HBM (kernel-class
timing off; the per-kernel times come from a separate pass).  `e2e` is the same step through the C ABI with
HOST buffers: every step uploads the evolving fields from pinned memory (qk_set_state_all), advances
(qk_hydro_step_cfl / qk_rhd_step_cfl: the timestep never visits the host) and downloads the result
(qk_get_state_all), all inside the timed region, with three boxes in flight so that upload, step and download
overlap.  Working set per step (5 x 147 MB read, plus stage buffers) is several times the 126 MB L2, so no
explicit flush is needed.  The same JSON line carries sub-records for the other BASELINE configs: "rhd"
(configs[3]), "rad" (configs[2], 128^3), "size512" (configs[4]), "rhd_nsub10" (the paper's N_sub = 10 shape) and
"small_boxes" (launch-bound sizes: ordinary step, device-resident timestep, replayed CUDA graph).

--impl reference times the CPU oracle (oracle/, plain C, its loops dealt out to the host's cores) on a bounded
sample of the same workload; it is a deliberately slow baseline.
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
# SURVEY.md section 8(a)/(d) figures: algorithmic fp64 operations (one evaluation of every quantity per cell / face,
# branch-free worst-case paths, division and square root counted as one operation each) and compulsory HBM bytes
OPS_HYDRO_STAGE = 1240.0    # S3 12 + S4 62 + S5 810 + S6 318 + S7 38
OPS_HYDRO_SWEEP = 388.0     # one direction of one stage: S5 270 + S6 106 + its share of S7 12
OPS_RAD_STAGE = 1080.0      # S8 640 + S9 402 + S10 38
OPS_RAD_SWEEP = 357.0       # one direction: S8 214 + S9 134 + its share of S10 9
OPS_EXCHANGE = 240.0        # S11 + S12 at the measured mean of 3.3 Newton iterations (160-320)
BYTES_HYDRO_STEP = 200.0    # S7: stage 1 reads 5 writes 5, stage 2 reads 10 writes 5
BYTES_RAD_SUBSTEP = 190.0   # S10
BYTES_EXCHANGE = 152.0      # S12: 11 reads + 8 writes
HYDRO_WORKLOAD = "config2"  # --workload sedov: the paper's own hydro benchmark problem, context only
SCHEME_FLAGS = 0            # --plm / --eddington: scheme variants; the headline run uses PPM + Levermore
# dram__bytes_read.sum + dram__bytes_write.sum per launch at 256^3 from the ncu --set full capture summarised in
# profiles/r2_kernels.md, valid for the library version named in the csv; bench.py checks qk_version() against it
# and reports null otherwise (the field is labelled "traffic_source": a static capture, not a live counter)
NCU_TRAFFIC_GB_256 = {}     # kernel class -> GB per launch, read from profiles/r2_traffic.csv
HBM_GBS = 6650.0            # set from MEASURED_PEAKS.json in run_ours


def load_ncu_traffic(version):
    """profiles/r2_traffic.csv: first line '# qk_version=<...>;size=256', then kernel,dram_read_gb,dram_write_gb."""
    try:
        lines = open(os.path.join(ROOT, "profiles", "r2_traffic.csv")).read().splitlines()
        meta = dict(kv.split("=", 1) for kv in lines[0].lstrip("# ").split(";"))
        if meta.get("qk_version") != version or int(meta.get("size", 0)) != 256:
            return
        for ln in lines[2:]:
            k, r, w = ln.split(",")
            NCU_TRAFFIC_GB_256[k] = float(r) + float(w)
    except Exception:
        pass


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
def oracle_grid(kind, n, seed_shift=0):
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
    return g


def oracle_sample(kind, n, steps, threads):
    """Time `steps` oracle steps of the workload generator at n^3 on `threads` host threads.
    Returns (updates/s, seconds, threads actually used)."""
    import oracle as O
    n0 = O.get_threads()
    O.set_threads(threads)
    used = O.get_threads()
    try:
        g = oracle_grid(kind, n)
        t0 = time.perf_counter()
        for _ in range(steps):
            dt = g.cfl_dt()
            rc = g.hydro_step(dt) if kind == "hydro" else g.rhd_step(dt)
            assert rc == 0, rc
        sec = time.perf_counter() - t0
        g.close()
    finally:
        O.set_threads(n0)
    return n ** 3 * steps / sec, sec, used


def host_cores():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle as O
    n = args.ref_size
    cores = host_cores()
    O.set_threads(cores)
    used = O.get_threads()
    g = oracle_grid("hydro", n)
    for _ in range(args.warmup):
        g.hydro_step(g.cfl_dt())
    t0 = time.perf_counter()
    for _ in range(args.steps):
        assert g.hydro_step(g.cfl_dt()) == 0
    sec = time.perf_counter() - t0
    g.close()
    value = n ** 3 * args.steps / sec
    sample = ("oracle (plain C, gcc -O2 -ffp-contract=off, loops over cells dealt out to %d OpenMP threads) on a %d^3 "
              "box of the config2 generator, %d steps" % (used, n, args.steps))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[1] generator (hydro, Mach-2 turbulence, periodic, "
                                   "gamma=5/3, CFL 0.3), bounded sample %d^3" % n},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------
# the CUDA path
# ---------------------------------------------------------------------------------------------
def one_step(ctx, kind, ex):
    """qk_cfl_dt (min over ranks when the box is decomposed) + one step of the hot path."""
    if kind == "rad":                    # BASELINE configs[2]: static matter, fixed radiation substep 0.3 dx / c_hat
        ctx.qk_rad_step(ctx.rad_dt)
        return
    dt = ctx.qk_cfl_dt()
    if ex is not None:
        dt = ex.global_dt(dt)
    if kind == "hydro":
        ctx.qk_hydro_step(dt)
    else:
        ctx.qk_rhd_step(dt)
    if ex is not None:
        ex.check()


def time_loop(torch, fn, nsteps, barrier):
    """nsteps x fn() bracketed by barrier + synchronize, timed with CUDA events on the stream the kernels are
    launched on.  Returns milliseconds."""
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(nsteps):
        fn()
    e1.record(stream)
    torch.cuda.synchronize()
    barrier()
    return e0.elapsed_time(e1)


NBOX = 3    # boxes in flight in the end-to-end loop: upload of one, step of another, download of a third


def time_e2e(torch, B, I, params, fields, kind, nf, nsteps, barrier, nsub):
    """End to end through the C ABI with HOST (pinned) buffers, three boxes in flight: per step the evolving fields go
    host -> device (qk_set_state_all), the step runs with the device-resident timestep, and the result comes back
    (qk_get_state_all); a box's next step starts from the result it downloaded.  No host synchronisation inside the
    loop: each box has its own compute and copy stream, so uploads, steps and downloads of the two boxes overlap (PCIe is
    full duplex).  Returns ms."""
    ids = list(range(nf))
    boxes = []
    for b in range(NBOX):
        with torch.cuda.stream(torch.cuda.Stream()):      # a compute stream of its own: the two boxes never wait on each other
            ctx = B.from_params(params, fields)
        host_in = [torch.from_numpy(np.ascontiguousarray(fields[I.FIELDS[f]])).clone().pin_memory() for f in range(nf)]
        host_out = [torch.empty_like(t).pin_memory() for t in host_in]
        boxes.append([ctx, host_in, host_out])

    def step(box):
        ctx, hin, hout = box
        ctx.qk_set_state_all(ids, hin)
        if kind == "hydro":
            ctx.qk_hydro_step_cfl()
        else:
            ctx.qk_rhd_step_cfl(nsub)
        ctx.qk_get_state_all(ids, hout)
        box[1], box[2] = hout, hin          # same copy stream: the next upload starts after this download

    for box in boxes:                        # warm-up: one step each
        step(box)
    for box in boxes:
        box[0].qk_wait_copies()
    stream = torch.cuda.current_stream()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    e0.record(stream)
    for s in range(nsteps):
        step(boxes[s % NBOX])
    for box in boxes:
        box[0].qk_wait_copies()
    e1.record(stream)
    torch.cuda.synchronize()
    barrier()
    ms = e0.elapsed_time(e1)
    for box in boxes:
        box[0].close()
    return ms


def kernel_pass(ctx, kind, nsteps, ex):
    """per-kernel-class device times (CUDA events around every launch group) in a pass of its own, so that the headline
    loop runs without the event records"""
    ctx.qk_set_profiling(True)
    for _ in range(nsteps):
        one_step(ctx, kind, ex)
    kt = ctx.qk_kernel_times()
    ctx.qk_set_profiling(False)
    return kt


def run_workload(torch, B, I, kind, params, fields, steps, warmup, rank, world, barrier, allmax, sampler=None,
                 decompose=False, e2e=True, extras=True):
    """Times `steps` steps of one workload; returns a dict of results."""
    n = params["nx"]
    nf = {"hydro": 5, "rhd": 9, "rad": 9}[kind]
    cells = params["nx"] * params["ny"] * params["nz"]
    out = {}
    # a decomposed box owns its storage (cudaMalloc): an allocation of its own can be exported to the neighbours
    with B.from_params(params, fields, torch_storage=not (decompose and world > 1)) as ctx:
        ctx.rad_dt = 0.3 * params["dx"] / params["c_hat"] if params.get("c_hat", 0.0) > 0.0 else None
        ex = None
        how = ""
        if decompose and world > 1:
            # one global box of n x n x (world n) cells, rank r owns the z slab r: boundary planes go
            # straight into the neighbours' peer-mapped ghost planes, overlapped with the interior work of the stage; if a
            # rank cannot attach its peers every rank falls back to the callback exchange (pack, NCCL send/recv, unpack)
            from paper_2110_01792_b200 import decomp as D
            ex = D.PeerExchange(ctx, rank, world, True)
            how = "peer-mapped ghost planes over NVLink, pushes overlapped with the interior sweeps"
            if not ex.ok:
                log("[rank %d] peer-mapped exchange unavailable (%r): callback exchange" % (rank, ex.error))
                ex = D.SlabExchange(ctx, rank, world, True, D.TorchTransport())
                how = "pack / NCCL send-recv / unpack per ghost fill (callback)"
        out["parallelism"] = ("z-slab decomposition of one %dx%dx%d box, halo exchange per RK stage (%s), global min dt"
                              % (n, n, n * world, how)) if ex else "1 box per GPU"
        for _ in range(warmup):
            one_step(ctx, kind, ex)
        ctx.set_all(fields)                        # timed steps are steps 1..K of the config
        torch.cuda.synchronize()
        l0 = ctx.qk_launch_count()
        if sampler:
            sampler.start()
        ms = time_loop(torch, lambda: one_step(ctx, kind, ex), steps, barrier)
        clocks = sampler.stop() if sampler else None
        launches = ctx.qk_launch_count() - l0
        info = ctx.qk_last_info()
        ms = allmax(ms)
        out.update(ms=ms, value=world * cells * steps / (ms * 1e-3), launches=launches, clocks=clocks, info=info)
        out["kernel_ms"] = kernel_pass(ctx, kind, max(2, min(steps, 5)), ex)
        if ex is None and extras and kind != "rad":
            # the same steps with the timestep of eq 21 evaluated on the device: no host read per step
            nsub = max(1, info["nsub"])
            fn = ctx.qk_hydro_step_cfl if kind == "hydro" else (lambda: ctx.qk_rhd_step_cfl(nsub))
            for _ in range(2):
                fn()
            ctx.set_all(fields)                    # the same steps 1..K of the config as the headline loop
            torch.cuda.synchronize()
            ms_d = allmax(time_loop(torch, fn, steps, barrier))
            out["device_dt"] = {"value": world * cells * steps / (ms_d * 1e-3), "unit": UNIT, "ms_per_step": ms_d / steps,
                                "call": "qk_hydro_step_cfl" if kind == "hydro" else "qk_rhd_step_cfl(%d)" % nsub}
        if ex is not None:
            out["halo"] = {"exchange": how, "exchanges": getattr(ex, "calls", None),
                           "bytes_sent_per_rank": getattr(ex, "bytes_sent", None)}
            ex.detach()
    if e2e and kind != "rad":
        e2e_steps = max(3, min(steps, 12))
        nsub = max(1, out["info"]["nsub"])
        ms_e = allmax(time_e2e(torch, B, I, params, fields, kind, nf, e2e_steps, barrier, nsub))
        out["e2e"] = {"value": world * cells * e2e_steps / (ms_e * 1e-3), "unit": UNIT,
                      "h2d_bytes_per_step": nf * cells * 8, "d2h_bytes_per_step": nf * cells * 8,
                      "ms_per_step": ms_e / e2e_steps, "steps": e2e_steps,
                      "how": "qk_set_state_all + %s + qk_get_state_all per step, pinned host buffers, three boxes in flight"
                             % ("qk_hydro_step_cfl" if kind == "hydro" else "qk_rhd_step_cfl(%d)" % nsub)
                             + ("" if world == 1 else "; every rank streams periodic boxes of its own (no halo exchange on this leg)")}
    return out


def small_box_record(torch, B, I, sizes, steps=200):
    """Boxes whose step is bound by launch overhead (BASELINE configs[0] is 32^3): the hydro step with the host
    timestep, with the device-resident timestep, and as a replayed CUDA graph (qk_graph_capture / qk_graph_launch),
    all on a side stream (the legacy default stream cannot be captured)."""
    out = {}
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        for n in sizes:
            p, f = I.config1(n=n)
            cells = n ** 3
            rec = {}
            with B.from_params(p, f) as ctx:
                def host_dt():
                    ctx.qk_hydro_step(ctx.qk_cfl_dt())
                ctx.qk_graph_capture(B.QK_GRAPH_HYDRO)
                for label, fn in (("host_dt", host_dt), ("device_dt", ctx.qk_hydro_step_cfl),
                                  ("graph", lambda: ctx.qk_graph_launch(1))):
                    ctx.set_all({k: f[k] for k in I.FIELDS[:5]})
                    for _ in range(5):
                        fn()
                    ms = time_loop(torch, fn, steps, lambda: None)
                    assert ctx.qk_last_info()["status"] == 0
                    rec[label] = {"value": cells * steps / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms / steps}
            out["%d^3" % n] = rec
    return out


def roofline_alu(kernel_ms, names, ops_per_cell_per_launch, cells, peak_ops, peak_note):
    """Dominant ALU-bound kernel: algorithmic fp64 ops per launch / mean launch duration."""
    present = [nm for nm in names if nm in kernel_ms]
    if not present:
        return None
    nm = max(present, key=lambda k: kernel_ms[k][0] / kernel_ms[k][1])    # the slowest class of the family
    tot, cnt = kernel_ms[nm]
    mean_ms = tot / cnt
    achieved = ops_per_cell_per_launch * cells / (mean_ms * 1e-3) / 1e12
    traffic = NCU_TRAFFIC_GB_256.get(nm) if cells == 256 ** 3 else None
    return {"bound": "alu", "kernel": nm, "achieved": achieved, "peak": peak_ops / 1e12,
            "unit": "TFLOP/s", "frac": achieved / (peak_ops / 1e12),
            "traffic": None if traffic is None else traffic * 1e9,
            "traffic_source": "profiles/r2_traffic.csv (ncu --set full capture of this library version; static, not live)"
                              if traffic is not None else None,
            # the same launch against the HBM roof, on the bytes it really moves (informative: `frac` is the headline)
            "frac_hbm_on_traffic": None if traffic is None else traffic * 1e9 / (mean_ms * 1e-3) / (HBM_GBS * 1e9),
            "launch_ms": mean_ms, "launches": cnt, "peak_source": peak_note,
            "ops_per_cell_per_launch": ops_per_cell_per_launch}


def roofline_step(ms_per_step, cells, ops, nbytes, peak_ops, hbm):
    """Whole step against both roofs: SURVEY 8(d) algorithmic operations and compulsory bytes per cell-update."""
    t = ms_per_step * 1e-3
    a_ops, a_bw = ops * cells / t / 1e12, nbytes * cells / t / 1e9
    return {"ops_per_cell": ops, "bytes_per_cell": nbytes, "achieved_tflops": a_ops, "frac_alu": a_ops / (peak_ops / 1e12),
            "achieved_gbs": a_bw, "frac_hbm": a_bw / hbm, "bound": "alu" if a_ops / (peak_ops / 1e12) > a_bw / hbm else "hbm"}


def run_ours(args):
    import torch
    from paper_2110_01792_b200 import binding as B
    from paper_2110_01792_b200 import inputs as I

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the library has no CPU path)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.backend == "gloo":          # functional check of the decomposed path on a box with fewer GPUs than ranks
        local %= torch.cuda.device_count()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        if args.backend == "gloo":
            dist.init_process_group("gloo")
        else:
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

    L = B.lib()     # fails loudly if libqk.so is absent
    version = L.qk_version().decode()
    load_ncu_traffic(version)
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
    global HBM_GBS
    hbm = HBM_GBS = float(peaks.get("hbm_gbs", 6650.0))
    hbm_note = "MEASURED_PEAKS.json hbm_gbs" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    peak_note = "qk_fp64_probe: measured DMUL+DADD lane-ops/s on this GPU (DFMA probe: %.2f T/s)" % (peak_fma / 1e12)
    single = world == 1
    sampler = ClockSampler(local) if rank == 0 else None
    t_all = time.time()

    def gen(kind, size, **kw):
        t0 = time.time()
        if kind == "hydro":
            p, f = I.sedov(n=size) if HYDRO_WORKLOAD == "sedov" else I.config2(n=size, seed=1002 + rank)
        elif kind == "rad":
            p, f = I.config3(n=size, **kw)
        else:
            p, f = I.config4(n=size, seed=(1004 if size != 512 else 1005) + rank, **kw)
        p["flags"] |= SCHEME_FLAGS
        log("[rank %d] %s %d^3 inputs generated in %.1f s" % (rank, kind, size, time.time() - t0))
        return p, f

    def go(kind, p, f, steps, warmup, **kw):
        return run_workload(torch, B, I, kind, p, f, steps, warmup, rank, world, barrier, allmax,
                            decompose=not args.replicas, **kw)

    # ---- headline: hydro, BASELINE configs[1] ----------------------------------------------------------
    hyd = None
    if not args.no_hydro:
        p, f = gen("hydro", n)
        hyd = go("hydro", p, f, args.steps, args.warmup, sampler=sampler)
        del p, f
    # ---- coupled RHD, BASELINE configs[3] ---------------------------------------------------------------
    rhd = rhd_tau = None
    if not args.no_rhd or hyd is None:
        rhd_steps = max(1, min(args.steps, args.rhd_steps))
        p, f = gen("rhd", n, chat_ratio=args.chat_ratio)
        rhd = go("rhd", p, f, rhd_steps, min(args.warmup, 3), sampler=sampler if hyd is None else None)
        rhd["steps"] = rhd_steps
        if single and not args.quick:     # the same workload with the opt-in optical-depth correction (R6)
            p2 = dict(p, flags=p["flags"] | I.FLAG_TAU_CORR)
            rhd_tau = go("rhd", p2, f, max(2, rhd_steps // 2), 2, e2e=False, extras=False)
        del p, f
    extra = {}
    if single and not args.quick and not args.no_rhd and n == 256 and args.chat_ratio == 0.01:
        # ---- the paper's RHD shape: N_sub = 10 radiation substeps per hydro step, PPM and PLM ----
        p, f = gen("rhd", n, chat_ratio=0.5)
        r10 = {}
        for label, fl in (("ppm", 0), ("plm", I.FLAG_PLM)):
            r = go("rhd", dict(p, flags=p["flags"] | fl), f, 3, 1, e2e=False, extras=False)
            r10[label] = {"value": r["value"], "unit": UNIT, "ms_per_step": r["ms"] / 3, "nsub": r["info"]["nsub"]}
        extra["rhd_nsub10"] = {"config": {"workload": "configs[3] generator with c_hat/c = 0.5: every step takes N_sub = 10 "
                                                      "radiation substeps (the paper's RHD benchmark shape, PAPER.md:604)"},
                               **r10}
        del p, f
        # ---- radiation only, BASELINE configs[2] at its stated size ----------------------------------------
        p, f = gen("rad", 128)
        r = go("rad", p, f, 50, 3, e2e=False, extras=False)
        extra["rad"] = {"metric": "radiation_cell_substeps_per_s", "value": r["value"], "unit": "cell-substeps/s",
                        "steps": 50, "ms_per_step": r["ms"] / 50, "gpu_launches": r["launches"],
                        "config": {"workload": "BASELINE.json configs[2]: radiation only 128^3, outflow, static matter, "
                                               "c_hat = 0.1 c, 50 x qk_rad_step(0.3 dx / c_hat)"},
                        "kernel_ms": {k: {"total_ms": v[0], "groups": v[1]} for k, v in r["kernel_ms"].items()},
                        "status": r["info"]["status"]}
        del p, f
        # ---- launch-bound boxes: ordinary step, device-resident timestep, replayed CUDA graph -------------------
        extra["small_boxes"] = {"config": {"workload": "BASELINE.json configs[0] (32^3) and its generator at 64^3, 128^3: qk_cfl_dt + qk_hydro_step, "
                                                       "qk_hydro_step_cfl, and qk_graph_launch(1) per step (200 steps each)"},
                                **small_box_record(torch, B, I, (32, 64, 128))}
        # ---- BASELINE configs[4]: 512^3 ---------------------------------------------------------------------
        if not args.no_512:
            p, f = gen("rhd", 512)
            r = go("rhd", p, f, 5, 2, e2e=False, extras=False)
            ph = dict(p, c_hat=0.0, c=0.0)
            h = go("hydro", ph, {k: f[k] for k in I.FIELDS}, 5, 2, e2e=False, extras=False)
            extra["size512"] = {"config": {"workload": "BASELINE.json configs[4]: coupled RHD 512^3 (configs[3] generator, "
                                                       "seed 1005), qk_cfl_dt + qk_rhd_step per step; hydro = the same state, "
                                                       "qk_cfl_dt + qk_hydro_step"},
                                "rhd": {"value": r["value"], "unit": UNIT, "ms_per_step": r["ms"] / 5, "steps": 5,
                                        "nsub": r["info"]["nsub"], "gpu_launches": r["launches"],
                                        "kernel_ms": {k: {"total_ms": v[0], "groups": v[1]} for k, v in r["kernel_ms"].items()}},
                                "hydro": {"value": h["value"], "unit": UNIT, "ms_per_step": h["ms"] / 5, "steps": 5},
                                "device_bytes": int(L.qk_state_bytes(512, 512, 512))}
            del p, f
    log("[rank %d] GPU part done in %.1f s" % (rank, time.time() - t_all))

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    def kms(d):
        return {k: {"total_ms": v[0], "groups": v[1], "ms_per_launch_group": v[0] / v[1]} for k, v in d.items()}

    roof = None
    if hyd is not None:
        roof = roofline_alu(hyd["kernel_ms"], ["hydro_sweep_x", "hydro_sweep_y", "hydro_sweep_z"], OPS_HYDRO_SWEEP, cells,
                            peak_ops, peak_note)
    if hyd is None:      # --no-hydro (profiling aid): the RHD workload alone fills the line
        hyd = rhd
        args.steps = rhd["steps"]
    ms_step = hyd["ms"] / args.steps
    line = {
        "metric": METRIC if hyd is not rhd else "rhd_cell_updates_per_s", "value": hyd["value"], "unit": UNIT,
        "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": ("BASELINE.json configs[1]: pure hydro %d^3, periodic, gamma=5/3, log-normal density, "
                                "k^-2 velocity field at rms Mach 2, CFL 0.3, qk_cfl_dt + qk_hydro_step per step" % n)
                               if HYDRO_WORKLOAD == "config2" else
                               ("Sedov blast %d^3 on [-1,1]^3, periodic, gamma=5/3, CFL 0.25 (PAPER.md:572), "
                                "qk_cfl_dt + qk_hydro_step per step" % n),
                   "scheme": ("PLM" if SCHEME_FLAGS & 8 else "PPM") + (" + Eddington closure" if SCHEME_FLAGS & 16 else " + Levermore closure"),
                   "cells": cells, "l2": "inputs larger than L2 (5 x %.0f MB per stage)" % (cells * 8 / 1e6),
                   "parallelism": hyd.get("parallelism", "1 box on 1 GPU") if world > 1 else "1 box on 1 GPU",
                   "library": version},
        "e2e": hyd.get("e2e"), "gpu_launches": hyd["launches"], "clocks": hyd["clocks"],
        "roofline": roof,
        "kernel_ms": kms(hyd["kernel_ms"]),
        "peaks": {"fp64_dmul_dadd_lane_ops_per_s": peak_ops, "fp64_dfma_lane_ops_per_s": peak_fma,
                  "hbm_gbs": hbm, "hbm_source": hbm_note},
    }
    if hyd is not rhd:
        line["roofline_step"] = roofline_step(ms_step, world * cells, 2 * OPS_HYDRO_STAGE, BYTES_HYDRO_STEP, peak_ops, hbm)
    if hyd.get("halo"):
        line["halo"] = hyd["halo"]
    if hyd.get("device_dt"):
        line["device_dt"] = hyd["device_dt"]
    if rhd is not None:
        ex = rhd["kernel_ms"].get("exchange")
        rroof = roofline_alu(rhd["kernel_ms"], ["rad_sweep_x", "rad_sweep_y", "rad_sweep_z"], OPS_RAD_SWEEP, cells, peak_ops,
                             peak_note)
        exroof = None
        nsub = max(1, rhd["info"]["nsub"])
        if ex:
            ach = BYTES_EXCHANGE * cells / (ex[0] / ex[1] * 1e-3) / 1e9
            tr = NCU_TRAFFIC_GB_256.get("exchange") if cells == 256 ** 3 else None
            exroof = {"bound": "hbm", "kernel": "exchange", "achieved": ach, "peak": hbm, "unit": "GB/s",
                      "frac": ach / hbm, "traffic": None if tr is None else tr * 1e9,
                      "traffic_source": "profiles/r2_traffic.csv (static ncu capture)" if tr is not None else None,
                      "bytes_per_cell": BYTES_EXCHANGE, "launch_ms": ex[0] / ex[1], "peak_source": hbm_note}
        rms = rhd["ms"] / rhd["steps"]
        line["rhd"] = {
            "metric": "rhd_cell_updates_per_s", "value": rhd["value"], "unit": UNIT, "steps": rhd["steps"],
            "ms_per_step": rms, "nsub": rhd["info"]["nsub"],
            "config": {"workload": "BASELINE.json configs[3]: coupled RHD %d^3, periodic, c_hat/c=%g, "
                                   "qk_cfl_dt + qk_rhd_step per step; plain HLL radiation flux (the optical-depth "
                                   "correction of reading R6 is opt-in, DESIGN.md section 3)" % (n, args.chat_ratio)},
            "e2e": rhd.get("e2e"), "gpu_launches": rhd["launches"],
            "roofline_rad": rroof, "roofline_exchange": exroof, "device_dt": rhd.get("device_dt"),
            "roofline_step": roofline_step(rms, world * cells,
                                           2 * OPS_HYDRO_STAGE + nsub * (2 * OPS_RAD_STAGE + OPS_EXCHANGE),
                                           BYTES_HYDRO_STEP + nsub * (BYTES_RAD_SUBSTEP + BYTES_EXCHANGE), peak_ops, hbm),
            "kernel_ms": kms(rhd["kernel_ms"]),
            "newton_mean_iters": rhd["info"]["newton_total_iters"] / max(1, cells * nsub),
        }
        if rhd_tau is not None:
            line["rhd"]["with_tau_corr"] = {"value": rhd_tau["value"], "unit": UNIT,
                                            "ms_per_step": rhd_tau["ms"] / max(2, rhd["steps"] // 2),
                                            "guard_faces_last_step": rhd_tau["info"]["guard_faces"]}
    line.update(extra)
    if single and not args.no_cpu_baseline:
        cores = host_cores()
        v1, s1, u1 = oracle_sample("hydro", args.ref_size, 2, 1)
        vN, sN, uN = oracle_sample("hydro", args.ref_size, 2 if cores < 8 else 6, cores)
        line["cpu_baseline"] = {"value": vN, "unit": UNIT, "cores": uN, "kind": "oracle",
                                "sample": "oracle (plain C, OpenMP over cells) on a %d^3 box of the config2 generator, "
                                          "%.1f s on %d threads" % (args.ref_size, sN, uN),
                                "one_core": {"value": v1, "unit": UNIT, "cores": u1, "seconds": s1}}
        if rhd is not None:
            m = max(16, args.ref_size * 3 // 4)
            v2, s2, u2 = oracle_sample("rhd", m, 2, cores)
            v3, s3, u3 = oracle_sample("rhd", m, 1, 1)
            line["rhd"]["cpu_baseline"] = {"value": v2, "unit": UNIT, "cores": u2, "kind": "oracle",
                                           "sample": "oracle on a %d^3 box of the config4 generator, 2 steps, %.1f s on %d "
                                                     "threads" % (m, s2, u2),
                                           "one_core": {"value": v3, "unit": UNIT, "cores": u3, "seconds": s3}}
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
    ap.add_argument("--no-512", action="store_true", help="leave out the 512^3 sub-record (its inputs take ~2 min to generate)")
    ap.add_argument("--quick", action="store_true", help="only the hydro and RHD workloads at --size (no sub-records)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="torch.distributed backend for N > 1; gloo lets ranks share a GPU (rank r uses cuda:r mod #GPUs): "
                         "a functional check of the decomposed path only -- ranks time-slice, the numbers mean nothing")
    args = ap.parse_args()
    global SCHEME_FLAGS, HYDRO_WORKLOAD
    HYDRO_WORKLOAD = args.workload
    SCHEME_FLAGS = (8 if args.plm else 0) | (16 if args.eddington else 0)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
