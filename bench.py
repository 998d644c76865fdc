#!/usr/bin/env python
"""bench.py -- throughput of the real-space spherical convolution hot path (one JSON line).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path (sc_convolve: every kernel it launches) over one batch of
seeded synthetic maps of the chosen BASELINE.json configuration (default: config 4, Nside 2048,
theta_max = 20', the configuration the metric is quoted on).

N = 1: `value` = included pixel pairs of the batch / device time; `roofline` for the dominant kernel
(executed FP32 FMA-pipe operations against the FFMA rate measured in this run, next to the
6-FMA-per-pair model figure); `e2e` through the HOST-buffer entry sc_convolve_host; `cpu_baseline` = the
fp64 oracle on the host cores on a bounded pixel sample, whose values are also compared with the GPU
output of this run (`parity`).

N > 1 (torchrun): ONE batch of maps split into latitude bands over the ranks (SURVEY.md
8e): per step a halo exchange of the overlap rows (NCCL point to point) + sc_convolve_band on every
rank, "scaling": "strong"; value = pairs of the whole maps / max time over ranks.  `--replicas` gives
the other way to use N GPUs (independent maps per rank, no data-path collective, "scaling": "weak").

`--impl reference` times the fp64 CPU oracle (oracle/), as it stands, on a bounded pixel sample of the
same workload on the host cores.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from workloads import gen  # noqa: E402

METRIC = "pixel-pair interactions/s"
UNIT = "pairs/s"
# nominal FP32 FMA peak: 148 SMs x 128 FP32 lanes x sm_max_mhz (B200_PROFILING.md unit counts,
# MEASURED_PEAKS.json clock); the roofline's denominator is the rate MEASURED in this run (sc_debug_fma_peak)
N_SM, LANES = 148, 128
EXEC_COUNTS = os.path.join(ROOT, "profiles", "exec_counts.csv")


def _pair_totals():
    rows = {}
    with open(os.path.join(ROOT, "tests", "golden", "pair_totals.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                a = line.split()
                rows[(int(a[0]), int(a[1]))] = int(a[2])
    return rows


def _workload_name(cfg):
    return (f"{cfg.name}: HEALPix Nside={cfg.nside} RING, theta_max={cfg.theta_max / gen.ARCMIN:.0f}', "
            f"B={cfg.batch} fp32 N(0,1) map(s), {cfg.kernel} kernel, {cfg.n_table}-sample cos(theta) table")


def _exec_counts(cfg_name):
    """Per-launch counters of this config's kernels from the committed ncu capture (profiles/exec_counts.csv):
    {kernel: dict(fp32_ops, fma_pipe_pct, smem_pipe_pct, dram_bytes, capture)}.  Instruction counts and DRAM
    bytes per launch are properties of the kernel build + workload, not of a particular run; they go stale
    when the kernels change, which is why the capture is named in the JSON line."""
    out = {}
    try:
        with open(EXEC_COUNTS) as f:
            for line in f:
                if line.startswith("#") or not line.strip():
                    continue
                a = [x.strip() for x in line.split(",")]
                if len(a) >= 9 and a[0] == cfg_name:
                    num = lambda x: float(x) if x not in ("", "null", "None") else None
                    out[a[1]] = dict(fp32_ops=num(a[2]), fma_pipe_pct=num(a[3]), smem_pipe_pct=num(a[4]),
                                     issue_pct=num(a[5]), dram_bytes=num(a[6]), ncu_ms=num(a[7]), capture=a[8])
    except OSError:
        pass
    return out


def _sm_max_mhz():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["sm_max_mhz"]), "MEASURED_PEAKS.json sm_max_mhz"
    except Exception:
        return 1965.0, "fallback 1965 MHz (B200_PROFILING.md)"


def _env_overrides():
    """SC_* environment knobs the library reads at plan creation: echoed so that a stray
    variable cannot silently change the timed path."""
    return {k: v for k, v in sorted(os.environ.items()) if k.startswith("SC_")}


def _ring_start(N, i):
    """First RING pixel of ring i (1-based); i = 4N gives N_pix.  Index arithmetic only."""
    if i < N:
        return 2 * i * (i - 1)
    if i <= 3 * N:
        return 2 * N * (N - 1) + (i - N) * 4 * N
    m = 4 * N - i
    return 12 * N * N - 2 * m * (m + 1)


def _pairs_per_kernel(plan, N):
    """Included pairs of the pixels each kernel writes (from the plan's per-pixel neighbour counts)."""
    import torch
    cnt, _ = plan.neighbour_counts(want_sig=False)
    cs = torch.zeros(cnt.numel() + 1, dtype=torch.int64, device=cnt.device)
    cs[1:] = torch.cumsum(cnt.to(torch.int64), 0)
    part = plan.partition()
    pr, fb = part["polar_rings"], part["first_belt_ring"]
    rng = lambda a, b: int(cs[_ring_start(N, b)] - cs[_ring_start(N, a)]) if b > a else 0   # rings a .. b-1
    polar = rng(1, pr + 1) + rng(4 * N - pr, 4 * N)
    belt = rng(fb, 4 * N - fb + 1) if fb <= 2 * N else 0
    total = int(cs[-1])
    return {"generic_warp_kernel": polar, "sym_kernel": total - polar - belt, "belt_kernel": belt}, part, cnt


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.samples, self.reasons, self.max_mhz = index, False, [], set(), None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                     nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                     nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                     nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                     nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
            while not self.stop_flag:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
                time.sleep(0.02)
        except Exception as e:  # pragma: no cover
            self.reasons.add(f"nvml_unavailable:{type(e).__name__}")

    def result(self):
        self.stop_flag = True
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def oracle_sample(cfg, target_seconds, nthreads=0, maps=None):
    """Time the oracle on a bounded, seeded pixel sample of `cfg`; -> (pairs/s, info).  info carries the
    sample (`sel`), the oracle's values and counts on it (`ref`, `cnt`) for the parity block."""
    import oracle as O
    T = gen.table_for(cfg)
    maps = gen.maps_for(cfg) if maps is None else maps
    O.load()
    probe = gen.sample_pixels(cfg.nside, 4000, seed=7)
    t0 = time.perf_counter()
    O.convolve(cfg.nside, T, cfg.theta_max, maps, sel=probe, nthreads=nthreads)
    dt = time.perf_counter() - t0
    rate_pix = probe.size / max(dt, 1e-6)
    n = int(min(cfg.npix // 2, max(4000, rate_pix * target_seconds)))
    sel = gen.sample_pixels(cfg.nside, n, seed=8)
    t0 = time.perf_counter()
    ref, cnt, _ = O.convolve(cfg.nside, T, cfg.theta_max, maps, sel=sel, nthreads=nthreads)
    dt = time.perf_counter() - t0
    pairs = int(cnt.astype(np.int64).sum()) * len(maps)
    return pairs / dt, {"pixels": int(sel.size), "pairs": pairs, "seconds": dt, "cores": O.last_threads(),
                        "sel": sel, "ref": ref, "cnt": cnt}


def run_reference(args, cfg, rank, world):
    if rank != 0:
        return
    times, pairs = [], 0
    per_step = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    info = None
    for i in range(args.warmup + args.steps):
        v, info = oracle_sample(cfg, per_step)
        if i >= args.warmup:
            times.append(info["seconds"]); pairs += info["pairs"]
    value = pairs / sum(times)
    sample = (f"{info['pixels']} seeded output pixels per step (gen.sample_pixels: poles, cap/belt "
              f"boundaries, equator + random) of {cfg.npix}, all their pairs, B={cfg.batch}")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": _workload_name(cfg)},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": info["cores"], "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def _init(world, local_rank):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        if os.environ.get("RANK", "0") == "0":
            os.environ.setdefault("NCCL_DEBUG", "VERSION")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))


def _barrier(world):
    import torch
    import torch.distributed as dist
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
        torch.cuda.synchronize()


def _fma_peaks(sc):
    """FP32 FMA/s: nominal (unit counts x clock) and measured in this process (scalar FFMA, packed FFMA2)."""
    sm_max, peak_src = _sm_max_mhz()
    nominal = N_SM * LANES * sm_max * 1e6
    m1, m2, m3 = sc.sc_debug_fma_peak(packed=False), sc.sc_debug_fma_peak(packed=True), sc.sc_debug_fma_peak(packed=2)
    measured = max(m1["fma_per_s"], m2["fma_per_s"])
    return nominal, measured, {
        "nominal_gfma": nominal / 1e9,
        "nominal_source": f"{N_SM} SMs x {LANES} FP32 lanes x {sm_max:.0f} MHz ({peak_src})",
        "measured_ffma_gfma": m1["fma_per_s"] / 1e9, "measured_ffma2_gfma": m2["fma_per_s"] / 1e9,
        "measured_ffma2_kernel_operands_gfma": m3["fma_per_s"] / 1e9,
        "kernel_operands": "FFMA2 with the accumulation's operand pattern (accumulator pair += tap pair x map value, a fresh "
                           "64-bit accumulator and 32-bit map value every instruction, the tap pair shared by 4): what the "
                           "register file sustains for it; the fractions of this line are against the constant-operand peak",
        "measured_source": "sc_debug_fma_peak in this run: register-only FFMA / FFMA2 loops, 2 x 1024 threads per SM, "
                           f"best of 3 launches of {m1['elapsed_ms']:.1f} / {m2['elapsed_ms']:.1f} ms (CUDA events)"}


def _roofline(cfg, B, total_pairs, kern_ms, kern_pairs, step_ms, step_min_ms, nominal, measured, peak_info):
    """The roofline object of the JSON line.  Two numerators, both over the FFMA rate measured in this run:
    * executed: thread-level FFMA + FADD + FMUL operations per launch (ncu, committed capture) / the launch time
      measured here with CUDA events -- the hardware utilisation; <= 1 by construction;
    * model: (5 + B) algorithmic FMAs per pair geometry (6 per pair at B = 1) x the pairs of the
      pixels the kernel writes / the same time -- a throughput in model units; it exceeds 1 because the kernels
      share one geometry + table lookup among 8-16 symmetric images (caps) or evaluate it once per tile (belt)."""
    counts = _exec_counts(cfg.name)
    per_kernel = {}
    for k, ms in kern_ms.items():
        c = counts.get(k, {})
        ops = c.get("fp32_ops")
        per_kernel[k] = {
            "ms": ms, "pairs": kern_pairs.get(k),
            "frac_model_6fma": (kern_pairs.get(k, 0) * (5 + B) / (ms * 1e-3) / measured) if ms > 0 else None,
            "executed_fp32_ops": ops,
            "frac_executed": (ops / (ms * 1e-3) / measured) if (ops and ms > 0) else None,
            "fma_pipe_active_pct_ncu": c.get("fma_pipe_pct"), "smem_pipe_pct_ncu": c.get("smem_pipe_pct"),
            "issue_active_pct_ncu": c.get("issue_pct"), "dram_bytes": c.get("dram_bytes"), "capture": c.get("capture")}
    dom = max(kern_ms, key=kern_ms.get) if kern_ms else "generic_kernel"
    d = per_kernel.get(dom, {"ms": step_ms, "pairs": total_pairs, "frac_model_6fma": total_pairs * (5 + B) / (step_ms * 1e-3) / measured,
                             "executed_fp32_ops": None, "frac_executed": None, "fma_pipe_active_pct_ncu": None,
                             "smem_pipe_pct_ncu": None, "dram_bytes": None, "capture": None})
    have_exec = d["frac_executed"] is not None
    achieved = (d["executed_fp32_ops"] if have_exec else d["pairs"] * (5 + B)) / (d["ms"] * 1e-3)
    # whole step: kernels without committed counts (the warp-per-pixel kernel next to the poles, ~1 % of the step) count as 0
    counted = [k for k, v in per_kernel.items() if v["executed_fp32_ops"]]
    covered_ms = sum(per_kernel[k]["ms"] for k in counted)
    all_exec = bool(counted) and covered_ms >= 0.95 * sum(v["ms"] for v in per_kernel.values())
    step_ops = sum(per_kernel[k]["executed_fp32_ops"] for k in counted) if all_exec else None
    lim = None
    if d.get("smem_pipe_pct_ncu") is not None and d.get("fma_pipe_active_pct_ncu") is not None:
        busiest = max(d["smem_pipe_pct_ncu"], d["fma_pipe_active_pct_ncu"])
        # below ~70 % of every pipe the kernel waits on dependent-issue latency (few warps per scheduler), not on a pipe
        lim = ("latency (no pipe saturated)" if busiest < 70.0 else
               "shared-memory pipe" if d["smem_pipe_pct_ncu"] > d["fma_pipe_active_pct_ncu"] else "FMA pipe") + \
              f" (ncu: shared-memory wavefronts {d['smem_pipe_pct_ncu']:.0f} %, FMA pipe {d['fma_pipe_active_pct_ncu']:.0f} %" + \
              (f", issue slots {d['issue_active_pct_ncu']:.0f} %" if d.get("issue_active_pct_ncu") is not None else "") + " of peak)"
    return {
        "bound": "alu", "kernel": dom, "achieved": achieved / 1e9, "peak": measured / 1e9, "unit": "GFMA/s",
        "frac": achieved / measured,
        "frac_is": "executed FP32 FMA-pipe operations / measured FFMA peak" if have_exec else
                   "MODEL units (no committed ncu counts for this config): see frac_model_6fma",
        "traffic": d["dram_bytes"],
        "traffic_source": (f"ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, committed capture {d['capture']} "
                           f"(profiles/exec_counts.csv); algorithmic bytes of the step: {8 * cfg.npix * B}") if d["dram_bytes"] else None,
        "kernel_ms": d["ms"], "kernel_pairs": d["pairs"],
        "executed": {"fp32_ops_per_launch": d["executed_fp32_ops"], "frac": d["frac_executed"],
                     "fma_pipe_active_pct_ncu": d["fma_pipe_active_pct_ncu"],
                     "source": (f"predicated-on thread instructions of the ncu SASS page, FFMA2/FMUL2/FADD2 x 2 + FFMA/FMUL/FADD "
                                f"(smsp__sass_thread_inst_executed_op_ffma_pred_on leaves the packed opcodes out), committed capture "
                                f"{d['capture']} (profiles/exec_counts.csv)") if have_exec else None},
        "frac_model_6fma": d["frac_model_6fma"],
        "model": f"{5 + B} algorithmic FMA per pair geometry (5 + B; 6 per pair at B = 1) x the pairs of the pixels this "
                 f"kernel writes / its mean launch time (CUDA events on the launching stream)",
        "limiter": lim, "peak_measured": peak_info, "peak_nominal": nominal / 1e9,
        "kernels": per_kernel,
        "step": {"ms": step_ms, "min_ms": step_min_ms,
                 "frac_model_6fma": total_pairs * (5 + B) / (step_ms * 1e-3) / measured,
                 "frac_executed": (step_ops / (step_ms * 1e-3) / measured) if step_ops else None,
                 "frac_executed_kernels": counted if step_ops else None}}


def run_ours(args, cfg, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    _init(world, local_rank)
    import paper_1409_4441_b200 as sc
    from paper_1409_4441_b200 import dist as scdist

    T = gen.table_for(cfg)
    # every rank gets its own maps (seed offset): independent problems, weak scaling
    seeds = scdist.rank_seeds(cfg.seeds, rank)
    host_maps = [gen.noise_map(cfg.npix, s) for s in seeds]
    if cfg.ylm_map:
        host_maps.append(gen.ylm_map(cfg.nside, seed=1000 + cfg.seeds[0]).astype(np.float32))
    B = len(host_maps)
    t0 = time.perf_counter()
    plan = sc.Plan(cfg.nside, T, cfg.theta_max, B)
    torch.cuda.synchronize()
    plan_s = time.perf_counter() - t0
    info = plan.info()
    total_pairs = info["total_pairs"]
    key = (cfg.nside, int(round(cfg.theta_max / gen.ARCMIN)))
    golden = _pair_totals().get(key)
    if golden is not None and golden != total_pairs:
        raise SystemExit(f"pair total {total_pairs} != golden {golden}: refusing to report")
    if args.path == "generic":
        plan.set_path(sc.SC_PATH_GENERIC)

    dev_in = [torch.from_numpy(m).cuda() for m in host_maps]
    dev_out = [torch.empty_like(m) for m in dev_in]
    stream = torch.cuda.current_stream()

    for _ in range(args.warmup):
        plan.convolve(dev_in, dev_out)
    _barrier(world)
    sampler = ClockSampler(local_rank); sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(stream)
    launches = 0
    for i in range(args.steps):
        plan.convolve(dev_in, dev_out)
        launches += sc.sc_last_launch_count(plan.handle)
        ev[i + 1].record(stream)
    _barrier(world)
    clocks = sampler.result()
    step_ms = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    total_ms = ev[0].elapsed_time(ev[-1])

    # per-kernel device times (events on the launching stream around every kernel; separate pass)
    kern_ms, kern_pairs, cnt_dev = {}, {}, None
    nprof = max(3, min(args.steps, 10))
    if args.path == "auto":
        for _ in range(nprof):
            for k, v in plan.convolve_profile(dev_in, dev_out).items():
                kern_ms[k] = kern_ms.get(k, 0.0) + v / nprof
        kern_pairs, part, cnt_dev = _pairs_per_kernel(plan, cfg.nside)
    _barrier(world)

    # end to end through the HOST-buffer entry point (pinned host memory, copies inside the timing)
    pin_in = [torch.from_numpy(m).pin_memory() for m in host_maps]
    pin_out = [torch.empty(cfg.npix, dtype=torch.float32).pin_memory() for _ in range(B)]
    e2e_steps = max(1, min(args.steps, 5))
    plan.convolve_host(pin_in, pin_out)
    _barrier(world)
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        plan.convolve_host(pin_in, pin_out)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_launches = sc.sc_last_launch_count(plan.handle)
    checksum = float(np.abs(pin_out[0].numpy()[::4097]).sum())
    if not np.isfinite(checksum) or checksum == 0.0:
        raise SystemExit("non-finite or zero output")

    # max over ranks of the times, sum over ranks of the work
    (total_ms, e2e_s), pairs_step_all = scdist.combine_timing([total_ms, e2e_s], total_pairs * B)
    value = pairs_step_all * args.steps / (total_ms * 1e-3)
    e2e_value = pairs_step_all * e2e_steps / e2e_s

    if rank == 0:
        nominal, measured, peak_info = _fma_peaks(sc)
        step_mean_ms = float(np.mean(step_ms))
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": _workload_name(cfg), "path": args.path,
                           "mode": "one batch per GPU" + (" (independent maps per rank, --replicas)" if world > 1 else ""),
                           "l2": "inputs+outputs (%.0f MB) larger than L2" % (8e-6 * cfg.npix * B),
                           "pairs_per_map": total_pairs, "plan_create_s": plan_s,
                           "n_knife_edge": info["n_knife_edge"], "env_overrides": _env_overrides()},
                "map_convs_per_s": B * world * args.steps / (total_ms * 1e-3),
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 4 * cfg.npix * B,
                        "d2h_bytes_per_step": 4 * cfg.npix * B, "ms_per_step": 1e3 * e2e_s / e2e_steps,
                        "launches_per_step": e2e_launches},
                "gpu_launches": launches,
                "roofline": _roofline(cfg, B, total_pairs, kern_ms, kern_pairs, step_mean_ms, float(np.min(step_ms)),
                                      nominal, measured, peak_info)}
        if not args.no_cpu and world == 1:
            v, oi = oracle_sample(cfg, args.cpu_seconds, maps=host_maps)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": oi["cores"], "kind": "oracle",
                                    "sample": f"{oi['pixels']} seeded output pixels of {cfg.npix} "
                                              f"(all their pairs, B={B}), {oi['seconds']:.1f} s"}
            # the values the oracle just computed are the reference of this run's GPU output on the same pixels
            sel = torch.from_numpy(oi["sel"]).cuda()
            rel, mx = [], []
            for b in range(B):
                got = dev_out[b][sel].cpu().numpy().astype(np.float64)
                err = got - oi["ref"][b]
                rel.append(float(np.sqrt(np.mean(err ** 2) / np.mean(oi["ref"][b] ** 2))))
                mx.append(float(np.max(np.abs(err)) / np.max(np.abs(oi["ref"][b]))))
            counts_equal = None
            if cnt_dev is not None:
                counts_equal = bool(np.array_equal(cnt_dev[sel].cpu().numpy(), oi["cnt"]))
            line["parity"] = {"pixels": oi["pixels"], "maps": B, "rel_rms": max(rel), "max_abs_over_max": max(mx),
                              "counts_equal": counts_equal, "pair_total_equals_golden": golden is not None,
                              "bars": {"rel_rms": 1e-6, "max_abs_over_max": 1e-5},
                              "against": "fp64 oracle values of the cpu_baseline sample, same seeded inputs, this run"}
            if max(rel) > 1e-6 or max(mx) > 1e-5 or counts_equal is False:
                raise SystemExit(f"parity violated: {line['parity']}")
        print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def run_bands(args, cfg, rank, world, local_rank):
    """Strong scaling (the N > 1 default): the SAME maps for the whole job, each rank owns the rows of its latitude
    band, per step a halo exchange of the overlap rows and the band convolution.  One JSON line with
    "scaling": "strong"; value = pairs of the whole map(s) / max time over ranks."""
    import torch
    import torch.distributed as dist
    _init(world, local_rank)
    import paper_1409_4441_b200 as sc
    from paper_1409_4441_b200 import dist as scdist
    T = gen.table_for(cfg)
    host_maps = gen.maps_for(cfg)
    B = len(host_maps)
    t0 = time.perf_counter()
    plan = sc.Plan(cfg.nside, T, cfg.theta_max, B)
    torch.cuda.synchronize()
    plan_s = time.perf_counter() - t0
    total_pairs = plan.info()["total_pairs"]
    bands = [plan.band(world, r) for r in range(world)]
    mine = bands[rank]
    own = scdist._ranges(mine["out_rows"])
    # this rank owns the rows of its band only; the overlap arrives by the halo exchange in every step
    dev_in = [torch.zeros(cfg.npix, dtype=torch.float32, device="cuda") for _ in range(B)]
    for m, h in zip(dev_in, host_maps):
        for lo, hi in own:
            m[lo:hi] = torch.from_numpy(h[lo:hi]).cuda()
    dev_out = [torch.zeros_like(m) for m in dev_in]
    halo_elems = sum(hi - lo for _, lo, hi in scdist.halo_plan(bands, rank)[1])

    def step():
        if world > 1:
            scdist.exchange_halos(dev_in, bands, rank)
        plan.convolve_band(mine["ring_lo"], mine["ring_hi"], dev_in, dev_out)

    for _ in range(args.warmup):
        step()
    _barrier(world)
    sampler = ClockSampler(local_rank); sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    _barrier(world)
    clocks = sampler.result()
    launches = args.steps * sc.sc_last_launch_count(plan.handle)

    # end to end with HOST buffers: own band rows host -> device, halo exchange, band convolution, band rows back
    pin_in = [torch.from_numpy(m).pin_memory() for m in host_maps]
    pin_out = [torch.zeros(cfg.npix, dtype=torch.float32).pin_memory() for _ in range(B)]
    own_elems = sum(hi - lo for lo, hi in own)

    def e2e_step():
        for b in range(B):
            for lo, hi in own:
                dev_in[b][lo:hi].copy_(pin_in[b][lo:hi], non_blocking=True)
        step()
        for b in range(B):
            for lo, hi in own:
                pin_out[b][lo:hi].copy_(dev_out[b][lo:hi], non_blocking=True)
        torch.cuda.synchronize()

    e2e_steps = max(1, min(args.steps, 5))
    e2e_step()
    _barrier(world)
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    e2e_s = time.perf_counter() - t0
    (total_ms, e2e_s), _ = scdist.combine_timing([e0.elapsed_time(e1), e2e_s], 0)
    if rank == 0:
        nominal, measured, peak_info = _fma_peaks(sc)
        value = total_pairs * B * args.steps / (total_ms * 1e-3)
        step_ms = total_ms / args.steps
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": _workload_name(cfg),
                           "mode": "latitude bands + halo exchange (PAPER.md:192): one batch of maps over all GPUs",
                           "l2": "inputs+outputs (%.0f MB) larger than L2" % (8e-6 * cfg.npix * B),
                           "pairs_per_map": total_pairs, "plan_create_s": plan_s,
                           "bands": [[b["ring_lo"], b["ring_hi"]] for b in bands],
                           "halo_bytes_per_step_rank0": 4 * halo_elems * B,
                           "collective": ("NCCL batch_isend_irecv, one packed buffer per peer" if world > 1 else "none (1 GPU)"),
                           "env_overrides": _env_overrides()},
                "map_convs_per_s": B * args.steps / (total_ms * 1e-3), "clocks": clocks,
                "e2e": {"value": total_pairs * B * e2e_steps / e2e_s, "unit": UNIT,
                        "h2d_bytes_per_step": 4 * own_elems * B, "d2h_bytes_per_step": 4 * own_elems * B,
                        "ms_per_step": 1e3 * e2e_s / e2e_steps, "note": "bytes of rank 0; every rank moves its own band rows"},
                "gpu_launches": launches,
                "roofline": {"bound": "alu", "kernel": "band step (all kernels of the band)", "achieved": None, "peak": measured / 1e9,
                             "unit": "GFMA/s", "frac": None, "traffic": None,
                             "frac_model_6fma": total_pairs * (5 + B) / (step_ms * 1e-3) / (measured * world),
                             "model": f"{5 + B} algorithmic FMA per pair geometry x all pairs / step time / (N x measured FFMA peak); "
                                      f"the executed-operation roofline is reported by the N = 1 run",
                             "peak_measured": peak_info, "peak_nominal": nominal / 1e9}}
        print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number (1-5); 6 = paper-scale theta_cut 240' (context)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", default="auto", choices=["auto", "generic"])
    ap.add_argument("--bands", action="store_true",
                    help="strong scaling: ONE batch of maps split into latitude bands over the ranks "
                         "(halo exchange + sc_convolve_band); the default when N > 1")
    ap.add_argument("--replicas", action="store_true",
                    help="N > 1: independent maps per rank (weak scaling, no data-path collective) instead of bands")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline + parity leg")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = gen.config(args.config)
    if args.impl == "reference":
        run_reference(args, cfg, rank, world)
    elif args.bands or (world > 1 and not args.replicas):
        run_bands(args, cfg, rank, world, local_rank)
    else:
        run_ours(args, cfg, rank, world, local_rank)


if __name__ == "__main__":
    main()
