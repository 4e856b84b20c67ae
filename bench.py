#!/usr/bin/env python
"""bench.py -- RANLUX++ p = 2048 doubles/s on B200 through the C ABI (include/rlxpp.h).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg2|cfg4|cfg5] [--impl reference]

One step = one pass of the whole hot path (load state, multiply9x9 by a^2048, mod_m, to_ranlux,
12 doubles per advance, store) over one batch: BASELINE.json configs[2] ("bulk generation to
HBM": 2^20 streams x 1,536 doubles, stream-interleaved, 12.9 GB written per step per GPU), the
configuration the metric "doubles/sec" is quoted on.  Output (12.9 GB) is far larger than the
126 MB L2, so no flush is needed between steps.  For N > 1 every rank owns its own 2^20 streams
(seeds offset by rank * 2^20): weak scaling, no data-path collective (streams are independent,
PAPER.md line 172).

Prints ONE JSON line (rank 0).  DESIGN.md "Measurement" explains every key.
"""
import argparse
import json
import os
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "RANLUX++ p=2048 doubles/sec"
UNIT = "doubles/s"
IMAD_PER_ADVANCE = 324  # 18 x 18 products 32x32->64 (81 products 64x64->128)
IMAD_PER_DOUBLE = 27    # 324 / 12 (one LCG operation per 12 numbers)
# Warp instructions the dominant kernel executes per advance of one warp's 32 streams (ncu smsp__inst_executed.sum /
# (advances / 32) of the committed --set full captures; profiles/ncu_r02_umma.md).  The issue-slot roofline of the
# kernels that neither HBM nor the tensor pipe binds: one warp instruction per scheduler and clock.
WARP_INST_PER_ADVANCE = {"normal": 813, "cfg5": 216, "cfg2": 158}
TRAFFIC_FILE = "profiles/traffic_r03.json"
SM_COUNT = 148
IMAD_LANES_PER_CLK_SM = 64  # fma-heavy pipe: one warp instruction per 2 cycles per SMSP, 4 SMSPs

WORKLOADS = {
    # name: (streams, doubles per stream, p, description)
    "cfg1": (1024, 384, 2048, "BASELINE configs[0]: 1,024 streams x 384 doubles, p=2048, stream-major (launch-latency bound: 8 CTAs)"),
    "cfg3": (1 << 20, 1536, 2048, "BASELINE configs[2]: 2^20 streams x 1536 doubles, p=2048, interleaved, 12.9 GB/step"),
    "cfg4": (1 << 18, 6144, 2048, "BASELINE configs[3] at p=2048: 2^18 streams x 6144 doubles, interleaved, 12.9 GB/step"),
    "cfg5": (1 << 18, 49152, 2048, "BASELINE configs[4]: 2^18 streams, random 64-bit skips, 49152 doubles fused to sum/sumsq"),
    "devapi": (1 << 18, 1200, 2048, "SURVEY 8f-1: device-side draw API (include/rlxpp_tile.cuh TileStream), 2^18 streams with random "
                                    "cursors, 1200 draws each summed per stream (rlxpp_generate_ragged_reduce, cooperative = 3)"),
    "cfg2": ((1 << 20) + 64, 16, 2048, "BASELINE configs[1]: 2^20+64 raw states x 16 advances in place (AoS)"),
}


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return d.get("hbm_gbs", 6650.0), d.get("sm_max_mhz", 1965.0), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


def job_layout(rank, world, n_streams_per_gpu, seed=1):
    """Weak scaling: the job has world x n_streams_per_gpu streams, rank g owns the contiguous range g and
    seeds its first stream with seed + first (mod 2^64).  -> (first stream, streams of this rank, seed argument)."""
    from paper_2106_02504_b200 import shard
    first, count = shard.stream_range(rank, world, world * n_streams_per_gpu)
    return first, count, shard.rank_seed(seed, first)


def whole_job_rate(units_per_rank, world, ms):
    """`value`: the units ALL ranks processed divided by the slowest rank's time."""
    return units_per_rank * world / (ms * 1e-3)


def spread(xs):
    xs = sorted(xs)
    return {"min": xs[0], "median": xs[len(xs) // 2] if len(xs) % 2 else 0.5 * (xs[len(xs) // 2 - 1] + xs[len(xs) // 2]),
            "max": xs[-1], "mean": sum(xs) / len(xs), "n": len(xs)}


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region (B200_PROFILING.md clocks
    line) through NVML in a background thread (every ~2 ms: the timed region of cfg3 is tens of ms,
    too short for an `nvidia-smi -lms` child to start and report)."""

    def __init__(self, cuda_index):
        import threading
        self.samples = []  # (time, sm_mhz, power_w, reasons bitmask)
        self.max_mhz = None
        self.err = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                self.dev = pynvml.nvmlDeviceGetHandleByUUID("GPU-" + str(torch.cuda.get_device_properties(cuda_index).uuid))
            except Exception:
                self.dev = pynvml.nvmlDeviceGetHandleByIndex(cuda_index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.dev, pynvml.NVML_CLOCK_SM))
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        except Exception as e:  # NVML missing: the clocks object says so instead of inventing numbers
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.dev, nv.NVML_CLOCK_SM)
                try:
                    reasons = nv.nvmlDeviceGetCurrentClocksEventReasons(self.dev)
                except Exception:
                    reasons = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.dev)
                try:
                    power = nv.nvmlDeviceGetPowerUsage(self.dev) / 1e3
                except Exception:
                    power = 0.0
                self.samples.append((time.perf_counter(), float(mhz), power, int(reasons)))
            except Exception as e:
                self.err = repr(e)
                return
            time.sleep(0.002)

    def stop(self, t0=None, t1=None):
        """Ends the sampling; the summary covers the samples taken in [t0, t1] (perf_counter times; default: all).  The
        thread is started before the warm-up (the first NVML queries of a process take tens of ms), so a 40 ms timed
        region still gets its ~20 samples."""
        res = {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0, "source": "nvml"}
        if self._thread is not None:
            self._stop.set()
            self._thread.join(timeout=2)
        if self.err:
            res["error"] = self.err
        if t0 is not None and self.samples:
            inside = [x for x in self.samples if t0 <= x[0] <= t1]
            if not inside:  # region shorter than a sampling period: the sample nearest to it
                mid = 0.5 * (t0 + t1)
                inside = [min(self.samples, key=lambda x: abs(x[0] - mid))]
            self.samples = inside
        if self.samples:
            nv = self.nv
            names = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                     "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                     "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                     "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
            mask = 0
            for x in self.samples:
                mask |= x[3]
            sm = sorted(x[1] for x in self.samples)
            res.update(sm_mhz=sm[len(sm) // 2], sm_min_mhz=sm[0], samples=len(sm),
                       reasons=sorted(k for k, bit in names.items() if mask & bit),
                       power_w_max=max(x[2] for x in self.samples))
        return res


def oracle_sample_rate(n_per, p, target_cpu_seconds=15.0):
    """Times the oracle as it stands on a bounded sample of the same workload."""
    import numpy as np
    import oracle
    from paper_2106_02504_b200 import inputs
    cores = max(1, oracle.hardware_threads())
    probe = 16 * cores
    t0 = time.perf_counter()
    oracle.streams(inputs.seeds(probe), p, n_per, want=("doubles",), nthreads=cores)
    dt = max(time.perf_counter() - t0, 1e-6)
    per_stream_cpu = dt * cores / probe  # includes seeding (one powmod per stream)
    for _ in range(2):  # the small probe overestimates the cost per stream (thread start-up): refine once
        n = int(min(max(target_cpu_seconds / per_stream_cpu, probe), 1 << 20))
        n = max(cores, n // cores * cores)
        t0 = time.perf_counter()
        out = oracle.streams(inputs.seeds(n), p, n_per, want=("doubles",), nthreads=cores)["doubles"]
        dt = time.perf_counter() - t0
        assert out.shape == (n, n_per) and float(np.max(out)) < 1.0
        if dt * cores >= 0.6 * target_cpu_seconds or n >= 1 << 20:
            break
        per_stream_cpu = dt * cores / n
    return n * n_per / dt, cores, n, dt


def oracle_one_core_rate(n_per, p, target_seconds=2.0):
    """The same on ONE host thread ('at 1 core and at all cores'), a short sample."""
    import oracle
    from paper_2106_02504_b200 import inputs
    n = 8
    while True:
        t0 = time.perf_counter()
        oracle.streams(inputs.seeds(n), p, n_per, want=("doubles",), nthreads=1)
        dt = time.perf_counter() - t0
        if dt >= 0.5 * target_seconds or n >= 1 << 16:
            return n * n_per / dt, n, dt
        n = int(min(max(2 * n, n * target_seconds / max(dt, 1e-4)), 1 << 16))


def run_reference(args):
    """--impl reference: the CPU oracle (oracle/), unmodified, on the host cores; each step is a
    bounded sample of the workload (same p, same doubles per stream, fewer streams)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from paper_2106_02504_b200 import inputs
    n_streams, n_per, p, desc = WORKLOADS[args.workload]
    if args.workload == "cfg2":
        n_per = 12 * 16
    cores = max(1, oracle.hardware_threads())
    # size a step for ~3 s of wall clock
    probe = 8 * cores
    t0 = time.perf_counter()
    oracle.streams(inputs.seeds(probe), p, n_per, want=("doubles",), nthreads=cores)
    dt = max(time.perf_counter() - t0, 1e-6)
    budget = min(3.0, 150.0 / max(1, args.steps + args.warmup))
    n = int(max(cores, min(n_streams, probe * budget / dt)))
    n = max(cores, n // cores * cores)
    for _ in range(args.warmup):
        oracle.streams(inputs.seeds(n), p, n_per, want=("doubles",), nthreads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.streams(inputs.seeds(n), p, n_per, want=("doubles",), nthreads=cores)
    dt = time.perf_counter() - t0
    value = n * n_per * args.steps / dt
    sample = f"{n} of {n_streams} streams x {n_per} doubles per step (seeding included), {cores} threads"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u64 integer limbs (unsigned __int128 products) -> f64", "data": "synthetic",
        "config": {"workload": args.workload, "description": desc, "sampled": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--engine", default="umma", choices=["umma", "imad"],
                    help="engine of the LCG advance (include/rlxpp.h): tensor-core GEMM (default) or IMAD.WIDE")
    ap.add_argument("--p", type=int, default=None,
                    help="luxury level (default: the workload's, 2048); BASELINE configs[3] sweeps 24, 389, 1024, 2048")
    ap.add_argument("--layout", default="interleaved", choices=["interleaved", "stream_major"],
                    help="cfg3 / cfg4 output layout (BASELINE cfg3 names the interleaved one; stream_major is context)")
    ap.add_argument("--output", default="f64", choices=["f64", "u48", "f32", "normal"],
                    help="cfg3 / cfg4: what a 48-bit draw is stored as (SURVEY 8f-2): the double (BASELINE), the integer, "
                         "its two 24-bit floats, or a standard normal deviate (Box-Muller, fused); `value` stays in "
                         "48-bit draws per second")
    ap.add_argument("--chunks", type=int, default=0,
                    help="UMMA engine: force the number of chunks per tile (rlxpp_set_chunks; 0 = the library decides)")
    ap.add_argument("--streams", type=int, default=0,
                    help="streams per GPU instead of the workload's (A/B runs and small multi-process dry runs; the line's "
                         "config.workload then carries the shape)")
    ap.add_argument("--per-stream", type=int, default=0, help="doubles per stream instead of the workload's")
    ap.add_argument("--no-compare", action="store_true", help="skip the short run of the other engine")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle cpu_baseline leg")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--sustained-s", type=float, default=3.0,
                    help="after the timed region, repeat the step back to back for at least this many seconds with the clock "
                         "sampler running and report it as `sustained` (0 = skip)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import paper_2106_02504_b200 as rlx
    from paper_2106_02504_b200 import inputs, shard

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    rlx.load()
    engines = {"umma": rlx.RLXPP_ENGINE_UMMA, "imad": rlx.RLXPP_ENGINE_IMAD}
    rlx.rlxpp_set_engine(engines[args.engine])
    rlx.rlxpp_set_chunks(args.chunks)
    umma = args.engine == "umma" and args.workload != "devapi"  # the device API advances with IMADs per thread

    n_streams, n_per, p, desc = WORKLOADS[args.workload]
    if args.p:
        p = args.p
    if args.streams or args.per_stream:  # not a BASELINE configuration any more: say so where the workload is named
        n_streams, n_per = args.streams or n_streams, args.per_stream or n_per
        desc = f"{args.workload} kernels on another shape: {n_streams} streams x {n_per} doubles (--streams / --per-stream)"
        args.no_cpu = True  # the oracle leg and its sample sizes are defined for the BASELINE shapes only
    # weak scaling: the job has world x n_streams streams, rank g owns the contiguous range g
    first_stream, my_streams, first_seed = job_layout(rank, world, n_streams)
    assert my_streams == n_streams
    stream = torch.cuda.current_stream()

    # ---------------------------------------------------------------- set up the step
    if args.workload == "cfg1":
        args.layout = "stream_major"
    if args.workload in ("cfg1", "cfg3", "cfg4"):
        h = rlx.rlxpp_create(n_streams, first_seed, p)
        out = torch.empty((n_per, n_streams), dtype=torch.float64, device="cuda")
        units = n_streams * n_per
        alg_bytes = units * 8 + 2 * 80 * n_streams  # doubles written + state read and written back
        lay = rlx.RLXPP_INTERLEAVED if args.layout == "interleaved" else rlx.RLXPP_STREAM_MAJOR
        if not umma:
            kernel = f"generate_kernel<Fixed<{p}>, {args.layout}, aligned>"
        elif args.workload == "cfg1":
            kernel = f"tc_generate_lanes_kernel<{args.layout}>"   # short call: time-parallel lanes
        elif args.layout == "interleaved" and args.output != "f32":
            kernel = "tc_pair_kernel<aligned, interleaved>"        # two tiles per CTA on one accumulator
        else:
            kernel = f"tc_generate_kernel<{args.layout}, aligned>"

        if args.output == "u48":
            out = out.view(torch.int64)
        elif args.output == "f32":
            out = out.view(torch.float32)

        def step():
            if args.output == "u48":
                rlx.rlxpp_generate_u48(h, out, n_per, lay)
            elif args.output == "f32":
                rlx.rlxpp_generate_floats(h, out, 2 * n_per, lay)
            elif args.output == "normal":
                rlx.rlxpp_generate_normal(h, out, n_per, lay)
            else:
                rlx.rlxpp_generate_doubles(h, out, n_per, lay)
    elif args.workload == "cfg5":
        h = rlx.rlxpp_create(n_streams, first_seed, p)
        sk = torch.from_numpy(inputs.cfg5_skip_distances(n_streams).view(np.int64)).cuda()
        rlx.rlxpp_skip_each(h, sk)
        S = torch.empty(n_streams, dtype=torch.float64, device="cuda")
        Q = torch.empty(n_streams, dtype=torch.float64, device="cuda")
        units = n_streams * n_per
        alg_bytes = (2 * 80 + 16) * n_streams
        kernel = "tc_pair_kernel<unaligned, reduce>" if umma else f"generate_kernel<Fixed<{p}>, reduce, unaligned>"

        def step():
            rlx.rlxpp_generate_reduce(h, S, Q, n_per)
    elif args.workload == "devapi":
        h = rlx.rlxpp_create(n_streams, first_seed, p)
        sk = torch.from_numpy(inputs.cfg5_skip_distances(n_streams).view(np.int64)).cuda()
        rlx.rlxpp_skip_each(h, sk)
        S = torch.empty(n_streams, dtype=torch.float64, device="cuda")
        Q = torch.empty(n_streams, dtype=torch.float64, device="cuda")
        cnt = torch.full((n_streams,), n_per, dtype=torch.int32, device="cuda")
        units = n_streams * n_per
        alg_bytes = (2 * 80 + 16 + 4) * n_streams
        kernel = "ragged_tile_kernel<reduce>"  # rlxpp_dev::TileStream (include/rlxpp_tile.cuh): tensor-core advance per CTA

        def step():
            rlx.rlxpp_generate_ragged_reduce(h, cnt, S, Q, 3)
    else:  # cfg2: raw advances; "doubles" = 12 per advance for the common unit
        h = None
        states = torch.from_numpy(inputs.cfg2_states(1 << 20).view(np.int64)).cuda()
        reps = n_per
        units = n_streams * reps * 12
        alg_bytes = 144 * n_streams
        kernel = "tc_advance_states_group_kernel<AoS>" if umma else f"advance_states_kernel<Fixed<{p}>, AoS>"

        def step():
            rlx.rlxpp_advance_states(states, n_streams, p, reps, rlx.RLXPP_AOS)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------------------------------------------------------- warm-up + timed region
    sampler = ClockSampler(local) if rank == 0 else None  # started before the warm-up, summarised over the timed region
    for _ in range(args.warmup):
        step()
    barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    launches0 = rlx.rlxpp_launch_count()
    barrier()
    t_region0 = time.perf_counter()
    ev[0].record(stream)
    for k in range(args.steps):
        step()
        ev[k + 1].record(stream)
    barrier()
    t_region1 = time.perf_counter()
    launches = rlx.rlxpp_launch_count() - launches0
    clocks = sampler.stop(t_region0, t_region1) if sampler else {}
    total_ms = ev[0].elapsed_time(ev[-1])
    per_launch_ms = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    total_ms = shard.max_over_ranks(total_ms, dist, "cuda")
    ms_per_step = total_ms / args.steps
    value = whole_job_rate(units, world, ms_per_step)

    # ---------------------------------------------------------------- roofline of the dominant kernel
    hbm_gbs, sm_max_mhz, peak_src = peaks()
    kernel_ms = sum(per_launch_ms) / len(per_launch_ms)  # one launch per step: event pairs bracket single launches
    launch_spread = spread(per_launch_ms)
    launch_spread["first"] = per_launch_ms[0]
    imad_nominal = SM_COUNT * IMAD_LANES_PER_CLK_SM * sm_max_mhz * 1e6  # IMAD/s at max clock
    imad_achieved = units * IMAD_PER_DOUBLE / (kernel_ms * 1e-3)
    hbm_achieved = alg_bytes / (kernel_ms * 1e-3) / 1e9
    roof_alu = imad_nominal / IMAD_PER_DOUBLE
    roof_hbm = hbm_gbs * 1e9 / 8 if args.workload in ("cfg1", "cfg3", "cfg4") else float("inf")
    doubles_rate = units / (kernel_ms * 1e-3)
    alu = {"achieved": imad_achieved / 1e9, "peak": imad_nominal / 1e9, "unit": "GIMAD/s", "frac": imad_achieved / imad_nominal,
           "model": "324 products 32x32->64 per advance (27 per double) whatever the engine; peak = "
                    f"{SM_COUNT} SMs x {IMAD_LANES_PER_CLK_SM} IMAD lanes/clk x {sm_max_mhz:.0f} MHz"}
    hbm = {"achieved": hbm_achieved, "peak": hbm_gbs, "unit": "GB/s", "frac": hbm_achieved / hbm_gbs,
           "algorithmic_bytes_per_launch": alg_bytes}
    stores = args.workload in ("cfg1", "cfg3", "cfg4")
    # The bound that binds: with the UMMA engine the products run on the tensor pipe, so a workload
    # that stores its doubles is bound by HBM writes; the IMAD engine and the store-free workloads
    # are bound by integer issue (reported against the 324-product model, north_star).
    if stores and umma:
        roofline = {"bound": "hbm", "kernel": kernel, "achieved": hbm_achieved, "peak": hbm_gbs, "unit": "GB/s",
                    "frac": hbm_achieved / hbm_gbs, "traffic": None, "peak_source": f"HBM copy {peak_src}",
                    "kernel_ms": kernel_ms, "alu": alu, "hbm": hbm}
    else:
        roofline = {"bound": "alu", "kernel": kernel, "achieved": alu["achieved"], "peak": alu["peak"], "unit": "GIMAD/s",
                    "frac": alu["frac"], "traffic": None, "peak_source": alu["model"] + f" (DESIGN.md); HBM {peak_src}",
                    "kernel_ms": kernel_ms, "alu": alu, "hbm": hbm}
    if args.output == "normal":
        # Box-Muller fused into the emission: 818 warp instructions per advance (ncu, profiles/ncu_r02_umma.md), 342 of
        # them fp64: the kernel is bound by instruction issue and the fp64 pipe, not by HBM.  Peak = one warp instruction per scheduler and clock.
        winst = units / 12.0 / 32.0 * WARP_INST_PER_ADVANCE["normal"] / (kernel_ms * 1e-3) / 1e9
        wpeak = SM_COUNT * 4 * sm_max_mhz * 1e6 / 1e9
        roofline = {"bound": "alu", "kernel": kernel.replace("aligned>", "aligned, normal>"), "achieved": winst, "peak": wpeak,
                    "unit": "G warp instructions/s", "frac": winst / wpeak, "traffic": None,
                    "peak_source": f"{WARP_INST_PER_ADVANCE['normal']} warp instructions per advance of 32 streams (ncu, "
                                   f"smsp__inst_executed) x advances; peak = {SM_COUNT} SMs x 4 schedulers x {sm_max_mhz:.0f} MHz",
                    "kernel_ms": kernel_ms, "alu": alu, "hbm": hbm}
    roofline["engine"] = args.engine
    if umma:
        # the products as the tensor core sees them: per 128 advances one M128 x N80 x K96 u8 GEMM tile
        # (2 x 80 x 96 = 15,360 integer ops per advance); int8 dense peak = measured bf16 x 2 (nominal ratio)
        bf16 = 1636.6  # fallback only: MEASURED_PEAKS.json (read below) is the authority
        if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")):
            with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
                bf16 = json.load(f).get("bf16_tflops", bf16)
        tops = units / 12.0 * 15360 / (kernel_ms * 1e-3) / 1e12
        roofline["tensor"] = {"achieved": tops, "peak": 2.0 * bf16, "unit": "TOP/s (u8 x u8 -> s32)", "frac": tops / (2.0 * bf16),
                              "what": "tcgen05.mma kind::i8 work incl. the K 72->96 and N 72->80 padding; peak = measured "
                                      "bf16 x 2 (the guide's nominal int8 : bf16 ratio)"}
        if not stores and args.workload in WARP_INST_PER_ADVANCE:
            # No stores, products on the tensor pipe (far from its peak: see `tensor`): what binds is warp-instruction
            # issue -- the carry chains of the normalisation, to_ranlux and the fused sums.  Peak = one warp instruction
            # per scheduler and clock; achieved = measured instructions per advance (ncu) x advances per second.
            wpa = WARP_INST_PER_ADVANCE[args.workload]
            winst = units / 12.0 / 32.0 * wpa / (kernel_ms * 1e-3) / 1e9
            wpeak = SM_COUNT * 4 * sm_max_mhz * 1e6 / 1e9
            roofline.update(bound="alu", achieved=winst, peak=wpeak, unit="G warp instructions/s", frac=winst / wpeak,
                            peak_source=f"{wpa} warp instructions per advance of 32 streams (ncu smsp__inst_executed, "
                                        f"profiles/ncu_r02_umma.md) x advances/s; peak = {SM_COUNT} SMs x 4 schedulers x "
                                        f"{sm_max_mhz:.0f} MHz (DESIGN.md 6); the tensor pipe's share is in `tensor`")
    roofline["doubles_roofline"] = {"alu": roof_alu, "hbm": (None if roof_hbm == float("inf") else roof_hbm),
                                    "min": min(roof_alu, roof_hbm), "frac": doubles_rate / min(roof_alu, roof_hbm),
                                    "what": "north_star's roofline: the slower of nominal IMAD peak / 27 and HBM peak / 8 B"}
    if clocks.get("sm_mhz"):
        at_clock = SM_COUNT * IMAD_LANES_PER_CLK_SM * clocks["sm_mhz"] * 1e6
        roofline["frac_at_observed_clock"] = imad_achieved / at_clock
    if rank == 0:
        try:
            roofline["imad_microbench_peak"] = rlx.rlxpp_measure_imad_peak(3) / 1e9
            roofline["frac_of_imad_microbench"] = imad_achieved / 1e9 / roofline["imad_microbench_peak"]
            roofline["hbm_write_microbench_peak"] = rlx.rlxpp_measure_hbm_write_peak(8 << 30, 3) / 1e9
            # the write-only denominator next to the driver's copy figure (a copy reads as much as it writes; a kernel
            # that only writes can exceed it): the kernel's own store pattern without its arithmetic
            roofline["frac_of_hbm_write_microbench"] = hbm_achieved / roofline["hbm_write_microbench_peak"]
        except rlx.RlxppError as e:  # the probes are context, the headline does not depend on them
            roofline["probe_error"] = str(e)
    traffic_file = os.path.join(ROOT, TRAFFIC_FILE)
    if os.path.exists(traffic_file):
        with open(traffic_file) as f:
            key = f"{args.workload}:{args.engine}" + ("" if args.layout == "interleaved" else ":" + args.layout)
            roofline["traffic"] = json.load(f).get(key)
    # NOT measured by this run: ncu cannot run inside a timed bench; the figure is the committed capture's
    roofline["traffic_source"] = (f"{TRAFFIC_FILE}: dram__bytes_read.sum + dram__bytes_write.sum of one launch from the committed "
                                  "ncu --set full capture of this kernel (another run of the same build), not this run")
    roofline["per_launch_ms"] = launch_spread

    # ---------------------------------------------------------------- the other engine, same workload (context; before the
    # sustained leg, which leaves the chip at its power-capped clocks)
    compare = None
    if not args.no_compare and args.workload != "devapi" and args.output == "f64":
        other = "imad" if umma else "umma"
        rlx.rlxpp_set_engine(engines[other])
        step()
        torch.cuda.synchronize()
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(stream)
        for _ in range(3):
            step()
        c1.record(stream)
        torch.cuda.synchronize()
        compare = {"engine": other, "value": units / (c0.elapsed_time(c1) / 3 * 1e-3), "unit": UNIT, "steps": 3,
                   "n_gpus": 1, "what": "same workload and launch configuration with the other engine, this rank only"}
        rlx.rlxpp_set_engine(engines[args.engine])

    # ---------------------------------------------------------------- cfg5 with its skip-ahead inside the timed region
    # BASELINE.json configs[4] is "skip-ahead PLUS fused consumption".  `value` above times the fused generation alone (the
    # skip is one call before the first step, as in the paper's use: seed / skip once, then draw); this leg times
    # rlxpp_skip_each (random 64-bit distances: ~32 generic modular products per stream) + rlxpp_generate_reduce per step.
    with_skip = None
    if args.workload == "cfg5" and rank == 0:
        def skip_step():
            rlx.rlxpp_skip_each(h, sk)
            step()
        skip_step()
        torch.cuda.synchronize()
        k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k0.record(stream)
        for _ in range(args.steps):
            skip_step()
        k1.record(stream)
        torch.cuda.synchronize()
        ws_ms = k0.elapsed_time(k1) / args.steps
        with_skip = {"value": units / (ws_ms * 1e-3), "unit": UNIT, "ms_per_step": ws_ms, "steps": args.steps, "n_gpus": 1,
                     "skip_share_of_step": 1.0 - kernel_ms / ws_ms,
                     "what": "rlxpp_skip_each (seeded random 64-bit distance per stream) + rlxpp_generate_reduce per step, this rank"}

    # ---------------------------------------------------------------- sustained: the same step for >= 3 s
    sustained = None
    if args.sustained_s > 0 and rank == 0:
        torch.cuda.synchronize()
        est = max(launch_spread["median"], 1e-3)
        block = max(1, int(100.0 / est))          # ~0.1 s of launches between events
        n_blocks = max(3, int(args.sustained_s * 1e3 / (block * est)) + 1)
        s_sampler = ClockSampler(local)
        sev = [torch.cuda.Event(enable_timing=True) for _ in range(n_blocks + 1)]
        t0 = time.perf_counter()
        sev[0].record(stream)
        for b in range(n_blocks):
            for _ in range(block):
                step()
            sev[b + 1].record(stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        s_clocks = s_sampler.stop()
        blocks_ms = [sev[b].elapsed_time(sev[b + 1]) / block for b in range(n_blocks)]
        s_ms = sev[0].elapsed_time(sev[-1]) / (n_blocks * block)
        sustained = {"value": units / (s_ms * 1e-3), "unit": UNIT, "launches": n_blocks * block, "wall_s": wall,
                     "ms_per_launch": s_ms, "ms_per_launch_by_block": spread(blocks_ms),
                     "first_block_ms": blocks_ms[0], "last_block_ms": blocks_ms[-1],
                     "frac_of_burst_value": units / (s_ms * 1e-3) / (units / (kernel_ms * 1e-3)),
                     "roofline_frac": roofline["frac"] * kernel_ms / s_ms, "clocks": s_clocks,
                     "what": f"the timed step repeated back to back for >= {args.sustained_s:g} s on this rank, CUDA events every "
                             f"{block} launches; NVML clocks / power / reasons sampled throughout"}

    devapi = None
    if args.workload == "devapi":
        def timed(fn, reps=3):
            fn()
            torch.cuda.synchronize()
            c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            c0.record(stream)
            for _ in range(reps):
                fn()
            c1.record(stream)
            torch.cuda.synchronize()
            return units / (c0.elapsed_time(c1) / reps * 1e-3)
        per_thread = timed(lambda: rlx.rlxpp_generate_ragged_reduce(h, cnt, S, Q, False))
        warp_coop = timed(lambda: rlx.rlxpp_generate_ragged_reduce(h, cnt, S, Q, True))
        h2 = rlx.rlxpp_create(n_streams, first_seed, p)  # fresh handle: every cursor 12 (the paper's aligned case)
        aligned_pt = timed(lambda: rlx.rlxpp_generate_ragged_reduce(h2, cnt, S, Q, False))
        aligned_coop = timed(lambda: rlx.rlxpp_generate_ragged_reduce(h2, cnt, S, Q, True))
        aligned_tile = timed(lambda: rlx.rlxpp_generate_ragged_reduce(h2, cnt, S, Q, 3))
        rlx.rlxpp_destroy(h2)
        devapi = {"unit": UNIT, "random_cursors_tile": None, "random_cursors_draw_coop": warp_coop,
                  "random_cursors_draw": per_thread, "aligned_cursors_tile": aligned_tile,
                  "aligned_cursors_draw": aligned_pt, "aligned_cursors_draw_coop": aligned_coop,
                  "what": "PAPER.md lines 174-176: per-thread skipping made the paper's GPU run 7x slower.  draw / draw_coop: "
                          "rlxpp_dev::Stream, the paper's 324 products per thread (draw_coop: one advance pass per warp and 12 "
                          "draws whatever the cursors); tile: rlxpp_dev::TileStream, one tensor-core pass per CTA of 128 streams"}

    # ---------------------------------------------------------------- end to end (host buffers)
    e2e = None
    if not args.no_e2e and args.workload in ("cfg3", "cfg4", "cfg5") and args.output == "f64":
        if h is not None:
            rlx.rlxpp_destroy(h)
            h = None
        if args.workload != "cfg5":
            del out
            torch.cuda.empty_cache()
            host = torch.empty((n_per, n_streams), dtype=torch.float64, pin_memory=True)
            d2h = n_streams * n_per * 8
            h2d = 2 * 64 * 18 * 4  # the two power tables of the seeding / skip kernels

            def e2e_step():
                hh = rlx.rlxpp_create(n_streams, first_seed, p)
                rlx.rlxpp_generate_doubles_host(hh, host, n_per, rlx.RLXPP_INTERLEAVED)
                rlx.rlxpp_destroy(hh)
        else:
            hostS = torch.empty(n_streams, dtype=torch.float64, pin_memory=True)
            hostQ = torch.empty(n_streams, dtype=torch.float64, pin_memory=True)
            hsk = torch.from_numpy(inputs.cfg5_skip_distances(n_streams).view(np.int64)).pin_memory()
            d2h = 16 * n_streams
            h2d = 8 * n_streams + 2 * 64 * 18 * 4

            def e2e_step():
                hh = rlx.rlxpp_create(n_streams, first_seed, p)
                dsk = hsk.cuda(non_blocking=True)
                rlx.rlxpp_skip_each(hh, dsk)
                rlx.rlxpp_generate_reduce_host(hh, hostS, hostQ, n_per)
                rlx.rlxpp_destroy(hh)
        e2e_step()  # warm-up (also pins / allocates the staging buffers' pages)
        barrier()
        t0 = time.perf_counter()
        e2e_each = []
        for _ in range(args.e2e_steps):
            t1 = time.perf_counter()
            e2e_step()  # returns when the host buffer is complete
            e2e_each.append(time.perf_counter() - t1)
        barrier()
        dt = time.perf_counter() - t0
        dt = shard.max_over_ranks(dt, dist, "cuda")
        each = spread([units / t for t in e2e_each])
        e2e = {"value": units * world * args.e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": args.e2e_steps,
               "per_step_this_rank": {"min": each["min"], "median": each["median"], "max": each["max"], "unit": UNIT},
               "d2h_gb_per_s_median_step": d2h * each["median"] / units / 1e9,  # what binds it: the PCIe copy of the result
               "what": "rlxpp_create (seed kernel) + rlxpp_generate_*_host into pinned host memory + rlxpp_destroy, wall clock"}

    # ---------------------------------------------------------------- oracle on the host cores
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        per = n_per if args.workload != "cfg2" else 12 * 16
        v, cores, ns, dt = oracle_sample_rate(per, p)
        v1, n1, dt1 = oracle_one_core_rate(per, p)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{ns} of {n_streams} streams x {per} doubles (seeding included), {dt:.2f} s wall on {cores} threads",
               "one_core": {"value": v1, "unit": UNIT, "ns_per_double": 1e9 / v1,
                            "sample": f"{n1} streams x {per} doubles, {dt1:.2f} s on 1 thread"}}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": ("u8 x u8 -> s32 (tcgen05.mma kind::i8) + u32 limbs -> f64" if umma
                      else "u32 limbs (IMAD.WIDE.U32, 64-bit accumulate) -> f64"), "data": "synthetic",
            "config": {"workload": args.workload if not (args.streams or args.per_stream) else f"{args.workload}-shape {n_streams} x {n_per}", "engine": args.engine, "layout": args.layout, "output": args.output, "description": desc, "n_streams_per_gpu": n_streams,
                       "doubles_per_stream": n_per, "p": p, "l2": "output per step (12.9 GB) exceeds L2; no flush needed"
                       if args.workload in ("cfg3", "cfg4") else ("3 MB of output: L2-resident, launch-latency bound"
                                                                  if args.workload == "cfg1" else
                                                                  "compute-bound; working set is registers"),
                       "parallelism": f"streams sharded over {world} GPU(s), no collective"},
            "lcg_advances_per_s": value / 12.0,
            "value_from_median_launch": units * world / (launch_spread["median"] * 1e-3),
            "roofline": roofline, "sustained": sustained, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
            "clocks": clocks,
            "other_engine": compare,
        }
        if with_skip is not None:
            line["with_skip"] = with_skip
            line["config"]["timed_step"] = ("rlxpp_generate_reduce only; the per-stream skip runs once before the first step "
                                            "(`with_skip` has both inside the timed region)")
        if args.workload == "cfg2":
            line["config"]["deferred_fold"] = True
            line["config"]["timed_step"] = (f"{n_per} products + 1 fold per state: between repetitions the state stays an "
                                            "unreduced product (< 2^591), mod_m runs once at the end; same canonical result")
        if devapi is not None:
            devapi["random_cursors_tile"] = value
            line["device_api"] = devapi
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
