#!/usr/bin/env python
"""bench.py -- throughput of the real-space spherical convolution hot path (one JSON line).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path (sc_convolve: every kernel it launches) over one batch of
seeded synthetic maps of the chosen BASELINE.json configuration (default: config 4, Nside 2048,
theta_max = 20', the configuration the metric is quoted on).  N > 1 (torchrun): every rank convolves
its own independent maps (weak scaling, no data-path collective); value = pairs of all ranks / max
time over ranks.

`--impl reference` times the fp64 CPU oracle (oracle/), as it stands, on a bounded pixel sample of
the same workload on the host cores.
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
# FP32 FMA peak used for the roofline: 148 SMs x 128 FP32 lanes x 1.965 GHz (B200_PROFILING.md unit
# counts, MEASURED_PEAKS.json sm_max_mhz); DESIGN.md "Roofline".
N_SM, LANES = 148, 128


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


def _traffic(cfg_name, kernel):
    """DRAM bytes per launch of `kernel` from the committed ncu --set full capture (profiles/), or None."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    try:
        with open(path) as f:
            for line in f:
                a = [x.strip() for x in line.split(",")]
                if len(a) >= 3 and a[0] == cfg_name and a[1] == kernel:
                    return float(a[2])
    except Exception:
        pass
    return None


def _sm_max_mhz():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["sm_max_mhz"]), "MEASURED_PEAKS.json sm_max_mhz"
    except Exception:
        return 1965.0, "fallback 1965 MHz (B200_PROFILING.md)"


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
    return {"generic_warp_kernel": polar, "sym_kernel": total - polar - belt, "belt_kernel": belt}, part


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


def oracle_sample(cfg, target_seconds, nthreads=0):
    """Time the oracle on a bounded, seeded pixel sample of `cfg`; -> (pairs/s, info)."""
    import oracle as O
    T, maps = gen.table_for(cfg), gen.maps_for(cfg)
    O.load()
    probe = gen.sample_pixels(cfg.nside, 4000, seed=7)
    t0 = time.perf_counter()
    _, cnt, _ = O.convolve(cfg.nside, T, cfg.theta_max, maps, sel=probe, nthreads=nthreads)
    dt = time.perf_counter() - t0
    rate_pix = probe.size / max(dt, 1e-6)
    n = int(min(cfg.npix // 2, max(4000, rate_pix * target_seconds)))
    sel = gen.sample_pixels(cfg.nside, n, seed=8)
    t0 = time.perf_counter()
    _, cnt, _ = O.convolve(cfg.nside, T, cfg.theta_max, maps, sel=sel, nthreads=nthreads)
    dt = time.perf_counter() - t0
    pairs = int(cnt.astype(np.int64).sum()) * cfg.batch
    return pairs / dt, {"pixels": int(sel.size), "pairs": pairs, "seconds": dt, "cores": O.last_threads()}


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


def run_ours(args, cfg, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
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

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        plan.convolve(dev_in, dev_out)
    barrier()
    sampler = ClockSampler(local_rank); sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(stream)
    launches = 0
    for i in range(args.steps):
        plan.convolve(dev_in, dev_out)
        launches += sc.sc_last_launch_count(plan.handle)
        ev[i + 1].record(stream)
    barrier()
    clocks = sampler.result()
    step_ms = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    total_ms = ev[0].elapsed_time(ev[-1])

    # per-kernel device times (events on the launching stream around every kernel; separate pass)
    kern_ms = {}
    nprof = max(3, min(args.steps, 10))
    if args.path == "auto":
        for _ in range(nprof):
            for k, v in plan.convolve_profile(dev_in, dev_out).items():
                kern_ms[k] = kern_ms.get(k, 0.0) + v / nprof
        kern_pairs, part = _pairs_per_kernel(plan, cfg.nside)
    barrier()

    # end to end through the HOST-buffer entry point (pinned host memory, copies inside the timing)
    pin_in = [torch.from_numpy(m).pin_memory() for m in host_maps]
    pin_out = [torch.empty(cfg.npix, dtype=torch.float32).pin_memory() for _ in range(B)]
    e2e_steps = max(1, min(args.steps, 5))
    plan.convolve_host(pin_in, pin_out)
    barrier()
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
        sm_max, peak_src = _sm_max_mhz()
        peak_fma = N_SM * LANES * sm_max * 1e6                      # FMA/s
        # algorithmic FMAs: 6 per pair at B = 1 (3 geometry + table coordinate + lerp + accumulate),
        # 5 + B per pair geometry with a batch
        fma_per_step = total_pairs * (5 + B)
        step_mean_ms = float(np.mean(step_ms))
        if kern_ms:
            dom = max(kern_ms, key=kern_ms.get)                       # the dominant kernel of the step
            dom_ms, dom_pairs = kern_ms[dom], kern_pairs[dom]
        else:
            dom, dom_ms, dom_pairs = "generic_kernel", step_mean_ms, total_pairs
        achieved = dom_pairs * (5 + B) / (dom_ms * 1e-3)
        traffic = _traffic(cfg.name, dom)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": _workload_name(cfg), "path": args.path,
                           "l2": "inputs+outputs (%.0f MB) larger than L2" % (8e-6 * cfg.npix * B),
                           "pairs_per_map": total_pairs, "plan_create_s": plan_s,
                           "n_knife_edge": info["n_knife_edge"]},
                "map_convs_per_s": B * world * args.steps / (total_ms * 1e-3),
                "clocks": clocks,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 4 * cfg.npix * B,
                        "d2h_bytes_per_step": 4 * cfg.npix * B, "ms_per_step": 1e3 * e2e_s / e2e_steps,
                        "launches_per_step": e2e_launches},
                "gpu_launches": launches,
                "roofline": {"bound": "alu", "kernel": dom, "achieved": achieved / 1e9, "peak": peak_fma / 1e9,
                             "unit": "GFMA/s", "frac": achieved / peak_fma, "traffic": traffic,
                             "kernel_ms": dom_ms, "kernel_pairs": dom_pairs,
                             "peak_source": f"{N_SM} SMs x {LANES} FP32 lanes x {sm_max:.0f} MHz ({peak_src})",
                             "model": f"{5 + B} algorithmic FMA per pair geometry (5 + B) x the pairs of the "
                                      f"pixels this kernel writes / its mean launch time (CUDA events)",
                             "kernels_ms": kern_ms, "kernels_pairs": kern_pairs if kern_ms else None,
                             "step": {"achieved": fma_per_step / (step_mean_ms * 1e-3) / 1e9,
                                      "frac": fma_per_step / (step_mean_ms * 1e-3) / peak_fma,
                                      "ms": step_mean_ms, "min_ms": float(np.min(step_ms))}}}
        if not args.no_cpu and world == 1:
            v, oi = oracle_sample(cfg, args.cpu_seconds)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": oi["cores"], "kind": "oracle",
                                    "sample": f"{oi['pixels']} seeded output pixels of {cfg.npix} "
                                              f"(all their pairs, B={B}), {oi['seconds']:.1f} s"}
        print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def run_bands(args, cfg, rank, world, local_rank):
    """Strong scaling (optional mode, not the driver's default): the SAME maps on every rank, each rank
    convolves its latitude band after a halo exchange of the overlap rows.  One JSON line
    with "scaling": "strong"; value = pairs of the whole map(s) / max time over ranks."""
    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    import paper_1409_4441_b200 as sc
    from paper_1409_4441_b200 import dist as scdist
    T = gen.table_for(cfg)
    host_maps = gen.maps_for(cfg)
    B = len(host_maps)
    plan = sc.Plan(cfg.nside, T, cfg.theta_max, B)
    total_pairs = plan.info()["total_pairs"]
    bands = [plan.band(world, r) for r in range(world)]
    mine = bands[rank]
    # this rank owns the rows of its band only; the overlap arrives by the halo exchange in every step
    dev_in = [torch.zeros(cfg.npix, dtype=torch.float32, device="cuda") for _ in range(B)]
    for m, h in zip(dev_in, host_maps):
        for lo, hi in scdist._ranges(mine["out_rows"]):
            m[lo:hi] = torch.from_numpy(h[lo:hi]).cuda()
    dev_out = [torch.zeros_like(m) for m in dev_in]

    def step():
        if world > 1:
            scdist.exchange_halos(dev_in, bands, rank)
        plan.convolve_band(mine["ring_lo"], mine["ring_hi"], dev_in, dev_out)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank); sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    clocks = sampler.result()
    (total_ms,), _ = scdist.combine_timing([e0.elapsed_time(e1)], 0)
    if rank == 0:
        value = total_pairs * B * args.steps / (total_ms * 1e-3)
        halo = sum(hi - lo for lo, hi in scdist._subtract(scdist._ranges(mine["in_rows"]), scdist._ranges(mine["out_rows"])))
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
                          "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": {"workload": _workload_name(cfg), "mode": "latitude bands + halo exchange",
                                     "band_of_rank0": mine, "halo_bytes_per_step_rank0": 4 * halo * B},
                          "map_convs_per_s": B * args.steps / (total_ms * 1e-3), "clocks": clocks,
                          "gpu_launches": args.steps * sc.sc_last_launch_count(plan.handle)}), flush=True)
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
                         "(halo exchange + sc_convolve_band) instead of independent maps per rank")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = gen.config(args.config)
    if args.impl == "reference":
        run_reference(args, cfg, rank, world)
    elif args.bands:
        run_bands(args, cfg, rank, world, local_rank)
    else:
        run_ours(args, cfg, rank, world, local_rank)


if __name__ == "__main__":
    main()
