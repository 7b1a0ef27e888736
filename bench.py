#!/usr/bin/env python
"""bench.py - throughput of the MHD hot path (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype f64|f32] [--n 512] [--impl ours|reference]

A "step" is one full 2N-RK3 time step (3 fused substep kernels + the forcing-table kernel) of the
whole hot path over one synthetic box.  Default workload: BASELINE config 4 (512^3, nu = eta = 5e-4,
helical forcing k_f = 3, f0 = 0.02, seeded solenoidal u of rms 0.1, weak Gaussian A, fixed CFL dt).
Prints ONE JSON line (see DESIGN.md "Measurement" for every key).

N > 1 (torchrun, or `--gpus N` alone: the script then starts its N ranks itself): the ranks share ONE box as z slabs
with a halo exchange per substep overlapped with the inner-domain update:
strong scaling at the workload's size; `--weak` gives every rank a full n^2 x n slab (the paper's two protocols,
PAPER.md:533); `--replicas` runs N independent boxes instead.
"""
import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "MHD cell-updates/s per RK3 step"
UNIT = "cell-updates/s"
WORDS_PER_CELL_STEP = 56           # 14 (substep 0) + 21 + 21, DESIGN.md "algorithmic bytes"
TWO_PI3 = (2 * math.pi,) * 3
CONFIGS = {                        # BASELINE.json configs 3-5 (index = position in configs[])
    256: dict(seed=1003, nu=1e-3, sigma=0.0, name="config3_256^3"),
    512: dict(seed=1004, nu=5e-4, sigma=1.0, name="config4_512^3"),
    1024: dict(seed=1005, nu=2.5e-4, sigma=0.0, name="config5_1024^3"),
}


def workload(n):
    return CONFIGS.get(n, dict(seed=1000 + n, nu=5e-4 * 512 / n, sigma=1.0, name="box_%d^3" % n))


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def committed_traffic(dtype):
    """DRAM bytes per substep launch from the committed ncu --set full summary, or None."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)).get(dtype)
        except Exception:
            return None
    return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self._stop_evt = threading.Event()

    def run(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM)
            names = {
                pynvml.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                pynvml.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                pynvml.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                pynvml.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                pynvml.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
            }
            while not self._stop_evt.is_set():
                self.samples.append(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                r = pynvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                self._stop_evt.wait(0.02)
        except Exception as e:                      # never let the sampler kill the bench
            self.reasons.add("sampler_error:%s" % type(e).__name__)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def time_oracle(n_sample, cfg, steps, warmup=0):
    """The oracle as it stands, timed on the host cores on a bounded sample of the workload."""
    from oracle import forcing as of, mhd_c
    from paper_2012_08758_b200 import inputs
    state = inputs.solenoidal_state(n_sample, cfg["seed"])
    nu = cfg["nu"]
    st = mhd_c.Stepper(state, TWO_PI3, nu, nu, 1.0)
    h = 2 * math.pi / n_sample
    umax = float(np.sqrt((state[1:4] ** 2).sum(axis=0).max()))
    dt = min(0.4 * h / (umax + 1.0), 0.25 * h * h / nu)
    times = []
    for s in range(warmup + steps):
        f = of.forcing_from_draws(*inputs.counter_uniforms(cfg["seed"] + 7, s), 3, cfg["sigma"], dt, 0.02, 1.0)
        t0 = time.perf_counter()
        st.step(dt, f)
        if s >= warmup:
            times.append(time.perf_counter() - t0)
    return n_sample ** 3 / float(np.median(times)), float(np.median(times)), mhd_c.max_threads()


def max_over_ranks(ms, dist, device):
    """The slowest rank's time (the contract's max-over-ranks), identical on every rank."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(n, world, ms_per_step):
    """Replicas only: every rank advances its own n^3 box, value = all ranks' cell updates / slowest rank's time."""
    return world * n ** 3 / (ms_per_step * 1e-3)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = workload(args.n)
    n_sample = min(args.n, args.ref_sample)
    value, sec, cores = time_oracle(n_sample, cfg, args.steps, args.warmup)
    sample = "each step = one RK3 step of the C oracle on a %d^3 box of the %s recipe" % (n_sample, cfg["name"])
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "grid": [args.n] * 3, "sample_grid": [n_sample] * 3},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_ours(args):
    import torch
    from paper_2012_08758_b200 import binding, inputs

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    n = args.n
    cfg = workload(n)
    nu = cfg["nu"]

    def bench_dtype(dtype_name, do_e2e):
        dtype = binding.AC_F64 if dtype_name == "f64" else binding.AC_F32
        es = 8 if dtype_name == "f64" else 4
        ctx = binding.Context((n, n, n), TWO_PI3, dtype, nu=nu, eta=nu, cs=1.0, k_f=3.0, helicity=cfg["sigma"],
                              device="cuda:%d" % local_rank)
        ctx.ac_set_variant(args.variant)
        ctx.ac_set_mixed(args.mixed)
        # pinned host copy of the state, filled field by field (1024^3 fp64: 60 GB, 8.6 GB per field)
        host = torch.empty((7, n, n, n), dtype=torch.float64 if dtype_name == "f64" else torch.float32, pin_memory=True)
        hview = host.numpy()
        if args.paper_protocol:
            # the paper's own benchmark inputs: every field uniform in [0, 1), forcing off
            rng = np.random.default_rng(cfg["seed"] + rank)
            for q in range(7):
                hview[q] = rng.random((n, n, n))
        else:
            for q, field in enumerate(inputs.solenoidal_state_fields(n, cfg["seed"] + rank)):
                hview[q] = field
            del field
        ctx.ac_load_state(host)
        dt = ctx.ac_reduce()["dt_cfl"]
        forcings = [ctx.ac_make_forcing(cfg["seed"] + 7, s, dt, 0.02) for s in range(args.warmup + args.steps)]
        if args.paper_protocol:
            dt = 1.19209e-7                      # constant dt = FLT_EPSILON, forcing disabled
            forcings = [None] * (args.warmup + args.steps)
        for s in range(args.warmup):
            ctx.ac_step(dt, forcings[s])
        ctx.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        sampler = ClockSampler(local_rank)
        sampler.start()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
        l0 = ctx.ac_launch_count()
        ev[0].record(ctx.stream)
        for s in range(args.steps):
            ctx.ac_step(dt, forcings[args.warmup + s])
            ev[s + 1].record(ctx.stream)
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        clocks = sampler.stop()
        launches = ctx.ac_launch_count() - l0
        total_ms = ev[0].elapsed_time(ev[-1])
        per = np.array([ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)])
        total_ms = max_over_ranks(total_ms, dist, "cuda")
        diag = ctx.ac_reduce()
        # S9 (not part of the step): the reductions over the resident state, timed the same way
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        red_ms = []
        for _ in range(5):
            r0.record(ctx.stream)
            ctx.ac_reduce()
            r1.record(ctx.stream)
            torch.cuda.synchronize()
            red_ms.append(r0.elapsed_time(r1))
        red_ms = float(np.median(red_ms))
        ms_per_step = total_ms / args.steps
        value = whole_job_value(n, world, ms_per_step)
        peak, peak_src = measured_peak()
        alg_bytes_launch = WORDS_PER_CELL_STEP / 3.0 * es * n ** 3         # average over the 3 substep launches
        launch_ms = ms_per_step / 3.0
        achieved = alg_bytes_launch / (launch_ms * 1e-3) / 1e9
        res = {
            "value": value, "ms_per_step": ms_per_step, "ms_median": float(np.median(per)),
            "ms_p90": float(np.percentile(per, 90)), "dt": dt, "launches": launches, "clocks": clocks,
            "diag": {k: diag[k] for k in ("urms", "brms", "nonfinite")},
            "s9_reduce": {"ms": red_ms, "algorithmic_bytes": 7 * es * n ** 3,
                          "achieved": 7 * es * n ** 3 / (red_ms * 1e-3) / 1e9, "unit": "GB/s",
                          "frac": 7 * es * n ** 3 / (red_ms * 1e-3) / 1e9 / measured_peak()[0],
                          "words_per_cell": 7,
                          "what": "ac_reduce (stage-1 + stage-2 kernels + 48-byte D2H), median of 5; algorithmic bytes "
                                  "count 7 words per cell (u, A and ln rho: the kernel also reduces min / max ln rho and "
                                  "checks it for non-finite values); SURVEY.md 8(d)'s 6-word count gives 6/7 of frac"},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": committed_traffic(dtype_name), "peak_source": peak_src,
                         "kernel": "substep (avg of the 3 launches of a step)",
                         "note": "reported against HBM as BASELINE.json's metric asks; the kernel itself is limited by "
                                 "issue slots and the FP64 (fp32: packed FMA) pipe at two worker warps per scheduler "
                                 "(61 % / 67 % busy, LSU pipe 80 %: profiles/r02_pair.md) and by the 1000 W power cap; "
                                 "the ghost-zone kernel's time (3.9 %) is charged to the substep kernel",
                         "algorithmic_bytes_per_launch": alg_bytes_launch},
        }
        if do_e2e:
            # end to end through the C ABI with HOST buffers: H2D of the whole state, one step, D2H of the state
            # the 1024^3 state is stored back over its own pinned buffer (a second 60 GB is not needed:
            # the next timed step then simply continues the run)
            out = torch.empty_like(host, pin_memory=True) if n <= 512 else host
            k_e2e = max(1, min(args.steps, args.e2e_steps))
            ctx.ac_load_state(host)
            ctx.ac_step(dt, forcings[0])
            ctx.ac_store_state(out)                        # untimed warm-up of the copy path
            torch.cuda.synchronize()
            if dist is not None:
                dist.barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(ctx.stream)
            for s in range(k_e2e):
                ctx.ac_load_state(host)
                ctx.ac_step(dt, forcings[s])
                ctx.ac_store_state(out)
            e1.record(ctx.stream)
            torch.cuda.synchronize()
            e2e_ms = e0.elapsed_time(e1) / k_e2e
            e2e_ms = max_over_ranks(e2e_ms, dist, "cuda")
            nbytes = 7 * n ** 3 * es
            res["e2e"] = {"value": whole_job_value(n, world, e2e_ms), "unit": UNIT, "h2d_bytes_per_step": nbytes,
                          "d2h_bytes_per_step": nbytes, "ms_per_step": e2e_ms, "steps": k_e2e,
                          "what": "ac_load_state(pinned host) + ac_step + ac_store_state(pinned host) per step"}
            del out
        ctx.ac_free()
        del ctx, host
        torch.cuda.empty_cache()
        return res

    main = bench_dtype(args.dtype, True)
    other_name = "f32" if args.dtype == "f64" else "f64"
    other = bench_dtype(other_name, False) if not args.single_dtype else None

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # the oracle as it stands on 128^3 and 256^3 boxes of the same recipe, all host cores, one
        # untimed warm-up step (thread start-up, first-touch page faults) and the median of the timed ones; and on one
        # thread (64^3 to keep the run short)
        from oracle import mhd_c
        n_s = min(n, args.ref_sample)
        v, sec, cores = time_oracle(n_s, cfg, 3, 1)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "ns_per_cell_step": 1e9 / v,
               "sample": "C oracle (fp64, OpenMP) on a %d^3 box of the same recipe: 1 warm-up + 3 timed RK3 steps, "
                         "median %.2f s per step" % (n_s, sec)}
        if n >= 256 and not args.quick_cpu:
            v2, sec2, _ = time_oracle(256, cfg, 2, 1)
            cpu["box_256"] = {"value": v2, "unit": UNIT, "ns_per_cell_step": 1e9 / v2,
                              "sample": "256^3 box: 1 warm-up + 2 timed steps, median %.2f s per step" % sec2}
        nthreads = mhd_c.max_threads()
        mhd_c.set_threads(1)
        try:
            v1, sec1, _ = time_oracle(min(n_s, 64), cfg, 3, 1)
        finally:
            mhd_c.set_threads(nthreads)
        cpu["one_thread"] = {"value": v1, "unit": UNIT, "ns_per_cell_step": 1e9 / v1,
                             "sample": "%d^3 box, 1 thread: 1 warm-up + 3 timed steps, median %.2f s per step"
                                       % (min(n_s, 64), sec1)}

    if rank == 0:
        line = {
            "metric": METRIC, "value": main["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": main["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": cfg["name"], "grid": [n, n, n], "nu": nu, "eta": nu, "helicity": cfg["sigma"],
                       "k_f": 3, "f0": 0.02, "dt": main["dt"], "l2": "state (14 arrays) far larger than L2; no flush needed",
                       "parallelism": "replicas only" if world > 1 else "single GPU", "variant": args.variant,
                       "mixed": args.mixed,
                       "protocol": "paper (PAPER.md:533)" if args.paper_protocol else "baseline"},
            "ms_median": main["ms_median"], "ms_p90": main["ms_p90"],
            "roofline": main["roofline"], "cpu_baseline": cpu, "e2e": main.get("e2e"),
            "gpu_launches": main["launches"], "clocks": main["clocks"], "diag": main["diag"],
            "s9_reduce": main["s9_reduce"],
            "paper_context": {"astaroth_4xV100_fp64_cell_updates_per_s": 1.0 / 0.65e-9,
                              "pencil_40cores_cell_updates_per_s": 1.0 / 23.17e-9, "source": "PAPER.md:535"},
        }
        if other is not None:
            line["also"] = {"dtype": other_name, "value": other["value"], "ms_per_step": other["ms_per_step"],
                            "ms_median": other["ms_median"], "roofline": other["roofline"], "clocks": other["clocks"],
                            "s9_reduce": other["s9_reduce"],
                            "gpu_launches": other["launches"]}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def run_slab(args):
    """N ranks share ONE box as z slabs: the halo of the current state
    travels on a second stream while the inner planes are updated, the boundary planes follow (slab.SlabRank).
    Strong scaling (one n^3 box over N ranks) or, with --weak, n^2 x n per rank."""
    import torch
    import torch.distributed as dist
    from paper_2012_08758_b200 import binding, inputs, slab

    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    else:
        # one rank: NCCL still carries the halo (the rank sends to itself), so the transport path is the real one
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:29561", rank=0, world_size=1,
                                device_id=torch.device("cuda", local_rank))
    rank = dist.get_rank()
    n = args.n
    cfg = workload(n)
    nu = cfg["nu"]
    nz_global = n * world if args.weak else n
    lengths = (2 * math.pi, 2 * math.pi, 2 * math.pi * nz_global / n)
    peak, peak_src = measured_peak()

    def bench_dtype(dtype_name):
        dtype = binding.AC_F64 if dtype_name == "f64" else binding.AC_F32
        npdt = np.float64 if dtype_name == "f64" else np.float32
        es = 8 if dtype_name == "f64" else 4
        rk = slab.SlabRank((nz_global, n, n), lengths, dist, dtype, device="cuda:%d" % local_rank, variant=args.variant,
                           overlap=not args.no_overlap, transport="pull" if args.transport == "pull" else "buffers",
                           nu=nu, eta=nu, cs=1.0, k_f=3.0, helicity=cfg["sigma"])
        nzl = rk.slab.nzl
        local = np.empty((7, nzl, n, n), dtype=npdt)
        for q, field in enumerate(inputs.solenoidal_state_fields(n, cfg["seed"])):
            # strong: this rank's planes of the one box; weak: every rank holds planes of the same seeded n^3 box
            local[q] = field[(rank * nzl) % n:(rank * nzl) % n + nzl]
        del field
        rk.load_state(local)
        dt = rk.reduce()["dt_cfl"]
        draws = [inputs.counter_uniforms(cfg["seed"] + 7, s) for s in range(args.warmup + args.steps)]
        forcings = [rk.forcing_from_draws(*u, dt, 0.02) for u in draws]
        for s in range(args.warmup):
            rk.step(dt, forcings[s])
        torch.cuda.synchronize()
        dist.barrier()
        sampler = ClockSampler(local_rank)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = rk.slab.ctx.ac_launch_count()
        e0.record(rk.slab.ctx.stream)
        for s in range(args.steps):
            rk.step(dt, forcings[args.warmup + s])
        e1.record(rk.slab.ctx.stream)
        torch.cuda.synchronize()
        dist.barrier()
        clocks = sampler.stop()
        total_ms = max_over_ranks(e0.elapsed_time(e1), dist if world > 1 else None, "cuda")
        launches = rk.slab.ctx.ac_launch_count() - l0
        diag = rk.reduce()
        ms_per_step = total_ms / args.steps
        cells = n * n * nz_global
        alg = WORDS_PER_CELL_STEP / 3.0 * es * cells / world        # per rank and launch
        achieved = alg / (ms_per_step / 3.0 * 1e-3) / 1e9
        res = {"value": cells / (ms_per_step * 1e-3), "ms_per_step": ms_per_step, "dt": dt, "launches": launches,
               "clocks": clocks, "diag": {k: diag[k] for k in ("urms", "brms", "nonfinite")},
               "halo_bytes": 2 * rk.slab.ctx.ac_halo_bytes(),
               "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                            "traffic": committed_traffic(dtype_name), "peak_source": peak_src,
                            "kernel": "substep (per rank; inner + outer launches, halo pack / unpack and ghost kernels "
                                      "charged to it)",
                            "algorithmic_bytes_per_launch": alg}}
        rk.free()
        del rk, local
        torch.cuda.empty_cache()
        return res

    main_res = bench_dtype(args.dtype)
    other_name = "f32" if args.dtype == "f64" else "f64"
    other = bench_dtype(other_name) if not args.single_dtype else None
    if rank == 0:
        line = {
            "metric": METRIC, "value": main_res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": main_res["ms_per_step"], "higher_is_better": True,
            "scaling": "weak" if args.weak else "strong", "vs_baseline": None, "dtype": args.dtype, "data": "synthetic",
            "config": {"workload": cfg["name"] + (" x%d along z (weak)" % world if args.weak else ""),
                       "grid": [n, n, nz_global], "nu": nu, "eta": nu, "helicity": cfg["sigma"], "k_f": 3, "f0": 0.02,
                       "dt": main_res["dt"], "variant": args.variant,
                       "parallelism": "z slabs x%d; halo of 3 planes per side and field per substep, %s, %s" % (
                           world, "pulled from the neighbours' memory by one kernel (CUDA IPC / peer memory)"
                           if args.transport == "pull" else "packed, sent through NCCL, unpacked",
                           "on a second stream beside the inner-domain update (PAPER.md:141-158)"
                           if not args.no_overlap else "before the substep (no overlap)"),
                       "l2": "state far larger than L2; no flush needed",
                       "halo_bytes_per_rank_per_substep": main_res["halo_bytes"]},
            "roofline": main_res["roofline"], "cpu_baseline": None, "e2e": None, "gpu_launches": main_res["launches"],
            "clocks": main_res["clocks"], "diag": main_res["diag"]}
        if other is not None:
            line["also"] = {"dtype": other_name, "value": other["value"], "ms_per_step": other["ms_per_step"],
                            "roofline": other["roofline"], "clocks": other["clocks"], "gpu_launches": other["launches"]}
        print(json.dumps(line))
    dist.destroy_process_group()


def spawn_ranks(args):
    """`python bench.py --gpus N` without torchrun: start the N ranks (one per GPU) the way the driver would."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--n", type=int, default=512)
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--mixed", default="bidiagonal", choices=["bidiagonal", "tensor"],
                    help="reading of the mixed-derivative scheme (G2); every BASELINE number uses bidiagonal")
    ap.add_argument("--single-dtype", action="store_true", help="skip the second precision")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--quick-cpu", action="store_true", help="cpu_baseline without the 256^3 box")
    ap.add_argument("--ref-sample", type=int, default=128, help="box size of the bounded oracle sample")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--slab", action="store_true",
                    help="run through slab.SlabRank even on one GPU (N > 1 always does unless --replicas)")
    ap.add_argument("--replicas", action="store_true", help="N > 1: N independent boxes instead of one box in z slabs")
    ap.add_argument("--weak", action="store_true", help="slab run with n^2 x n cells per rank (weak scaling, PAPER.md:533)")
    ap.add_argument("--no-overlap", action="store_true", help="slab run: exchange before the substep instead of beside it")
    ap.add_argument("--transport", default="nccl", choices=["nccl", "pull"],
                    help="slab run: halo through NCCL send / receive of packed buffers, or pulled from the neighbours' "
                         "memory by one kernel (CUDA IPC mappings: peer memory over NVLink)")
    ap.add_argument("--paper-protocol", action="store_true",
                    help="the paper's benchmark set-up (PAPER.md:533): all fields U[0,1), no forcing, dt = 1.19209e-7")
    args = ap.parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    elif args.slab or args.weak or (world > 1 and not args.replicas):
        run_slab(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
