"""Small runs of every kernel family of libsc for compute-sanitizer:

    compute-sanitizer --tool memcheck  python tests/sanitize_cases.py
    compute-sanitizer --tool racecheck python tests/sanitize_cases.py
    compute-sanitizer --tool initcheck python tests/sanitize_cases.py        (one tool per GPU session)

Cases: BASELINE.json configs 1 and 2 (sym kernel 16-image and batch instances, warp-per-pixel kernel, generic kernel,
audit), Nside 512 / 1 deg (belt kernel with TMA staging, 384-consumer sym instance), a NESTED plan, a latitude band, the
north-cap entry, a two-zone table and the host-buffer entry.  Each result is compared with the generic kernel's
(SC_PATH_GENERIC) on the same plan, so that a sanitizer-clean run is also a run with the right answer.  Not a pytest
file (the name does not start with test_): it is run by hand under the sanitizer; summaries go to profiles/.
"""
import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import paper_1409_4441_b200 as sc  # noqa: E402
from workloads import gen  # noqa: E402


def _both_paths(plan, maps):
    dev = [torch.from_numpy(m).cuda() for m in maps]
    fast = [o.clone() for o in plan.convolve(dev)]
    plan.set_path(sc.SC_PATH_GENERIC)
    ref = [o.clone() for o in plan.convolve(dev)]
    plan.set_path(sc.SC_PATH_AUTO)
    torch.cuda.synchronize()
    worst = 0.0
    for a, b in zip(fast, ref):
        worst = max(worst, float((a - b).abs().max() / b.abs().max()))
    assert worst < 5e-6, worst
    return dev, fast, worst


def main():
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    done = []
    for ci in (1, 2):
        cfg = gen.config(ci)
        T, maps = gen.table_for(cfg), gen.maps_for(cfg)
        with sc.Plan(cfg.nside, T, cfg.theta_max, len(maps)) as plan:
            dev, fast, w = _both_paths(plan, maps)
            done.append((cfg.name, w))
            if ci == 2:
                band = plan.band(3, 1)
                out = [torch.zeros_like(d) for d in dev]
                plan.convolve_band(band["ring_lo"], band["ring_hi"], dev, out)
                pin_in = [torch.from_numpy(m).pin_memory() for m in maps]
                pin_out = [torch.empty_like(p).pin_memory() for p in pin_in]
                plan.convolve_host(pin_in, pin_out)
                torch.cuda.synchronize()
                assert float((pin_out[0].cuda() - fast[0]).abs().max()) == 0.0
                done.append(("band + host entry", 0.0))
    # belt kernel (needs Nside % 512 == 0), 384-consumer sym instance, north cap entry
    nside, theta, n = 512, np.deg2rad(1.0), 4096
    x, th = gen.table_nodes(theta, n)
    T = np.exp(-0.5 * (th / (theta / 3.0)) ** 2)
    m = gen.noise_map(12 * nside * nside, 11)
    with sc.Plan(nside, T, theta, 1) as plan:
        dev, fast, w = _both_paths(plan, [m])
        done.append(("nside512 belt", w))
        rows = plan.cap_rows(nside // 2)
        out = torch.zeros_like(dev[0])
        plan.convolve_cap(nside // 2, [dev[0]], [out])
        torch.cuda.synchronize()
        hi = rows["out_rows"][1]
        assert float((out[:hi] - fast[0][:hi]).abs().max() / fast[0].abs().max()) < 5e-6
        done.append(("north cap", 0.0))
    # two-zone table and NESTED ordering at Nside 64
    nside, theta, n = 64, np.deg2rad(3.4), 1024
    xz, thz = gen.zoned_table_nodes(theta, n, 1.0 / 16.0)
    Tz = np.exp(-0.5 * (thz / (theta / 3.0)) ** 2)
    m = gen.noise_map(12 * nside * nside, 12)
    with sc.Plan(nside, Tz, theta, 1, zone_frac=1.0 / 16.0) as plan:
        done.append(("two-zone", _both_paths(plan, [m])[2]))
    x, th = gen.table_nodes(theta, n)
    with sc.Plan(nside, np.exp(-0.5 * (th / (theta / 3.0)) ** 2), theta, 1, ordering=sc.SC_ORDER_NESTED) as plan:
        done.append(("nested", _both_paths(plan, [m])[2]))
    for name, w in done:
        print(f"ok {name}: fast vs generic max-abs / max {w:.2e}")


if __name__ == "__main__":
    main()
