"""GPU parity: the CUDA path (through the C ABI of include/sc.h) against the fp64 oracle, element by
element, on the seeded inputs of workloads/gen.py.

Bars (BASELINE.json north_star): neighbour enumeration bit-exact (per-pixel counts and index-sum
signatures identical); fp32 outputs within relative-rms <= 1e-6 and max-abs <= 1e-5 * max|out|.
"""
import os

import numpy as np
import pytest

import oracle as O
from workloads import gen

pytestmark = pytest.mark.gpu

REL_RMS_TOL = 1e-6          # BASELINE.json north_star
MAX_ABS_TOL = 1e-5          # times max|out|
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _totals():
    rows = {}
    with open(os.path.join(GOLD, "pair_totals.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                a = line.split()
                rows[(int(a[0]), int(a[1]))] = int(a[2])
    return rows


@pytest.fixture(scope="module")
def sc():
    import torch
    assert torch.cuda.is_available()
    import paper_1409_4441_b200 as sc
    return sc


def _gpu_convolve(sc, plan, maps):
    import torch
    dm = [torch.from_numpy(np.ascontiguousarray(m, np.float32)).cuda() for m in maps]
    out = plan.convolve(dm)
    torch.cuda.synchronize()
    return [o.cpu().numpy() for o in out]


def _check_values(got, want, what):
    """got fp32, want fp64 on the same pixels."""
    want = np.asarray(want, np.float64)
    err = got.astype(np.float64) - want
    relrms = np.sqrt(np.mean(err ** 2) / np.mean(want ** 2))
    maxabs = np.max(np.abs(err)) / np.max(np.abs(want))
    print(f"{what}: rel-rms {relrms:.3e}  max-abs/max|out| {maxabs:.3e}")
    assert relrms <= REL_RMS_TOL, (what, relrms)
    assert maxabs <= MAX_ABS_TOL, (what, maxabs)


def _check_counts(sc, plan, cnt_ref, sig_ref, sel=None):
    cnt, sig = plan.neighbour_counts()
    cnt, sig = cnt.cpu().numpy(), sig.cpu().numpy().view(np.uint64)
    if sel is not None:
        cnt, sig = cnt[sel], sig[sel]
    np.testing.assert_array_equal(cnt, cnt_ref)
    np.testing.assert_array_equal(sig, sig_ref)


PATHS = ["auto", "generic"]


def _set_path(sc, plan, path):
    plan.set_path(sc.SC_PATH_GENERIC if path == "generic" else sc.SC_PATH_AUTO)


@pytest.mark.parametrize("path", PATHS)
def test_config1_full(sc, path):
    """Nside 64, theta_max 3.4 deg: every pixel, values + counts + signatures + exact pair total."""
    cfg = gen.config(1)
    T, maps = gen.table_for(cfg), gen.maps_for(cfg)
    ref, cnt, sig = O.convolve(cfg.nside, T, cfg.theta_max, maps)
    with sc.Plan(cfg.nside, T, cfg.theta_max, cfg.batch) as plan:
        _set_path(sc, plan, path)
        info = plan.info()
        assert info["total_pairs"] == _totals()[(64, 204)] == int(cnt.sum())
        _check_counts(sc, plan, cnt, sig)
        out = _gpu_convolve(sc, plan, maps)
        _check_values(out[0], ref[0], f"cfg1/{path}")
        assert sc.sc_last_launch_count(plan.handle) >= 1
        print("audit:", info)
        assert info["max_t_err"] < info["guard_band"]


@pytest.mark.parametrize("path", PATHS)
def test_config2_full_batch2(sc, path):
    """Nside 256, theta_max 1.5 deg, B = 2 (noise map + band-limited map): every pixel."""
    cfg = gen.config(2)
    T, maps = gen.table_for(cfg), gen.maps_for(cfg)
    ref, cnt, sig = O.convolve(cfg.nside, T, cfg.theta_max, maps)
    with sc.Plan(cfg.nside, T, cfg.theta_max, cfg.batch) as plan:
        _set_path(sc, plan, path)
        assert plan.info()["total_pairs"] == _totals()[(256, 90)] == int(cnt.sum())
        _check_counts(sc, plan, cnt, sig)
        out = _gpu_convolve(sc, plan, maps)
        for b in range(2):
            _check_values(out[b], ref[b], f"cfg2/{path}/map{b}")


def _ring_pixels(tb, rings):
    return np.concatenate([np.arange(tb["start"][r - 1], tb["start"][r - 1] + tb["npr"][r - 1]) for r in rings])


def _structured_subset(nside, theta_max):
    """SURVEY.md 8d's deterministic subset for maps too large for a full oracle pass: every 16th ring plus all rings
    within theta_max of the poles and of the cap/belt boundary rings N and 3N (whole rings, so tile boundaries and
    ragged tails are inside), plus the equator ring."""
    tb = O.ring_table(nside)
    th = np.arccos(np.clip(tb["z"], -1.0, 1.0))
    N = nside
    near = lambda t0: np.abs(th - t0) <= theta_max * 1.02
    keep = near(0.0) | near(np.pi) | near(th[N - 1]) | near(th[3 * N - 1])
    keep[15::16] = True
    keep[2 * N - 1] = True
    rings = np.nonzero(keep)[0] + 1
    return _ring_pixels(tb, rings), rings


def _config_parity(sc, ci, key, sel=None, n_cnt=200000):
    """Values (all maps of the batch) and neighbour sets against the oracle: on every pixel (sel None) or on `sel`;
    the exact pair total over the sphere and counts + signatures on n_cnt further sampled pixels in both cases."""
    cfg = gen.config(ci)
    T, maps = gen.table_for(cfg), gen.maps_for(cfg)
    ref, cnt_v, sig_v = O.convolve(cfg.nside, T, cfg.theta_max, maps, sel=sel)
    pix = np.arange(cfg.npix) if sel is None else sel
    print(f"cfg{ci}: oracle on {pix.size} of {cfg.npix} pixels ({100.0 * pix.size / cfg.npix:.1f} %), {O.last_threads()} threads")
    sel_c = gen.sample_pixels(cfg.nside, n_cnt, seed=200 + ci)
    cnt_c, sig_c = O.count(cfg.nside, cfg.theta_max, sel=sel_c)
    with sc.Plan(cfg.nside, T, cfg.theta_max, cfg.batch) as plan:
        info = plan.info()
        print("audit:", info, plan.partition())
        assert info["total_pairs"] == _totals()[key]
        assert info["max_t_err"] < info["guard_band"]
        cnt, sig = plan.neighbour_counts()
        cnt, sig = cnt.cpu().numpy(), sig.cpu().numpy().view(np.uint64)
        assert int(cnt.astype(np.int64).sum()) == _totals()[key]
        np.testing.assert_array_equal(cnt[sel_c], cnt_c)
        np.testing.assert_array_equal(sig[sel_c], sig_c)
        np.testing.assert_array_equal(cnt[pix], cnt_v)
        np.testing.assert_array_equal(sig[pix], sig_v)
        out = _gpu_convolve(sc, plan, maps)
        for b in range(cfg.batch):
            _check_values(out[b][pix], ref[b], f"cfg{ci}/map{b}")
            assert np.all(np.isfinite(out[b]))
        return out, ref, pix


def test_config3_full_map(sc):
    """Nside 1024, theta_max 30': EVERY pixel against the oracle (values, counts, signatures), exact pair total."""
    _config_parity(sc, 3, (1024, 30))


def test_config4_full_map(sc):
    """Nside 2048, theta_max 20', split-like oscillating kernel (the metric's configuration): EVERY pixel of the
    50,331,648 against the oracle (the full oracle pass takes well under 10 min on the box)."""
    out, ref, _ = _config_parity(sc, 4, (2048, 20))
    # per ring as well, so that one broken short ring or tile cannot hide in the all-sky average
    tb = O.ring_table(2048)
    err2 = np.add.reduceat((out[0].astype(np.float64) - ref[0]) ** 2, tb["start"]) / tb["npr"]
    assert np.sqrt(err2.max() / np.mean(ref[0] ** 2)) <= 2 * REL_RMS_TOL, int(np.argmax(err2)) + 1


def test_config5_structured_subset_batch3(sc):
    """Nside 2048, theta_max 60', B = 3: SURVEY.md 8d's structured subset (every 16th ring + all rings within theta_max
    of the poles and of rings N, 3N + the equator, whole rings: >= 5 % of the pixels), all three maps."""
    cfg = gen.config(5)
    sel, rings = _structured_subset(cfg.nside, cfg.theta_max)
    assert sel.size >= 0.05 * cfg.npix
    _config_parity(sc, 5, (2048, 60), sel=sel, n_cnt=50000)


def test_config6_paper_scale_sampled(sc):
    """The paper's own operating point (theta_cut 240', ~61,000 neighbours per pixel): counts
    and values on 300 sampled pixels.  The belt kernel streams its taps in ring groups at this disc size."""
    cfg = gen.config(6)
    T, maps = gen.table_for(cfg), gen.maps_for(cfg)
    sel = gen.sample_pixels(cfg.nside, 300, seed=66)
    ref, cnt, sig = O.convolve(cfg.nside, T, cfg.theta_max, maps, sel=sel)
    with sc.Plan(cfg.nside, T, cfg.theta_max, 1) as plan:
        info = plan.info()
        assert info["max_t_err"] < info["guard_band"]
        c, s = plan.neighbour_counts()
        c, s = c.cpu().numpy(), s.cpu().numpy().view(np.uint64)
        assert int(c.astype(np.int64).sum()) == info["total_pairs"]
        np.testing.assert_array_equal(c[sel], cnt)
        np.testing.assert_array_equal(s[sel], sig)
        out = _gpu_convolve(sc, plan, maps)
        _check_values(out[0][sel], ref[0], "cfg6 paper scale")
        assert np.all(np.isfinite(out[0]))


@pytest.mark.parametrize("path", PATHS)
def test_paths_agree_config3_rings(sc, path):
    """Whole rings at Nside 1024 (several tiles + ragged tails): pole rings, a mid-cap ring, the
    cap/belt boundary, a belt ring, the equator and their southern mirrors."""
    cfg = gen.config(3)
    T, maps = gen.table_for(cfg), gen.maps_for(cfg)
    t = O.ring_table(cfg.nside)
    N = cfg.nside
    rings = [1, 2, 3, 7, 33, 100, 517, N - 1, N, N + 1, N + 40, 2 * N - 1, 2 * N, 2 * N + 1, 3 * N - 1, 3 * N,
             3 * N + 1, 4 * N - 100, 4 * N - 2, 4 * N - 1]
    sel = np.concatenate([np.arange(t["start"][r - 1], t["start"][r - 1] + t["npr"][r - 1]) for r in rings])
    ref, cnt, sig = O.convolve(cfg.nside, T, cfg.theta_max, maps, sel=sel)
    with sc.Plan(cfg.nside, T, cfg.theta_max, 1) as plan:
        _set_path(sc, plan, path)
        out = _gpu_convolve(sc, plan, maps)
        _check_values(out[0][sel], ref[0], f"cfg3 rings/{path}")
        # per ring too, so that a broken short ring cannot hide in the average
        off = 0
        scale = np.sqrt(np.mean(ref[0] ** 2))
        for r in rings:
            n = int(t["npr"][r - 1])
            e = out[0][sel[off:off + n]].astype(np.float64) - ref[0][off:off + n]
            assert np.sqrt(np.mean(e ** 2)) / scale <= REL_RMS_TOL, r
            off += n


@pytest.mark.parametrize("path", PATHS)
def test_exact_integer_sums(sc, path):
    """K == 1 table and small-integer maps: every product and sum is exact in fp32, so the output
    equals fl32(fl32(sum) * fl32(Omega)) bit for bit iff the neighbour SET used by the convolution
    kernels themselves is the oracle's (counts alone could not see a swapped pixel)."""
    for nside, theta in ((64, 3.4 * gen.DEG), (128, 1.0 * gen.DEG), (37, 5.0 * gen.DEG)):
        npix = 12 * nside * nside
        rng = np.random.default_rng(nside)
        m = rng.integers(-8, 9, size=npix).astype(np.float32)
        T = np.ones(64)
        ref, cnt, _ = O.convolve(nside, T, theta, [m])
        omega = np.float32(4 * np.pi / npix)
        s = np.rint(ref[0] / (4 * np.pi / npix))
        assert np.max(np.abs(s)) < 2 ** 24
        want = s.astype(np.float32) * omega
        with sc.Plan(nside, T, theta, 1) as plan:
            _set_path(sc, plan, path)
            out = _gpu_convolve(sc, plan, [m])
        np.testing.assert_array_equal(out[0], want)


def _handover_rings(N, pr, fb):
    """Whole rings at every kernel hand-over of the AUTO path (polar | sym | belt) and at the cap/belt boundary and the
    equator, with their southern mirrors."""
    fbm = min(fb, 2 * N)
    base = {1, 2, pr, pr + 1, fbm - 1, fbm, N - 1, N, N + 1, 2 * N - 1, 2 * N}
    base = {r for r in base if 1 <= r <= 2 * N}
    return sorted(base | {4 * N - r for r in base} | {2 * N + 1})


@pytest.mark.parametrize("nside,theta_am,ntab,B", [
    (512, 60, 4096, 1),        # belt_kernel<128>, sym 384-consumer variant
    (1024, 30, 8192, 1),       # config 3's launch configuration: belt_kernel<256>
    (1024, 72, 8192, 1),       # discs of ~1500 pixels: running totals in tensor memory (sym), two sets (belt<256>)
    (2048, 20, 16384, 1),      # config 4's launch configuration: belt_kernel<512, 64>, single accumulator set
    (2048, 60, 16384, 1),      # belt_kernel<512, 256, TM>, sym TMEM variant
    (2048, 60, 16384, 3)])     # config 5's launch configuration (B = 3)
def test_exact_integer_sums_fast_kernels(sc, nside, theta_am, ntab, B):
    """north_star: "GPU neighbour enumeration must be bit-exact" -- measured on the kernels that do the work.  K == 1
    table of the config's size and small-integer maps through SC_PATH_AUTO at the sizes that select every variant of
    sym_kernel / belt_kernel / generic_warp_kernel: every product and sum is exact in fp32, so out == fl32(sum) * fl32(Omega)
    bit for bit iff the neighbour SET those kernels used is the oracle's.  Oracle on whole rings at every kernel hand-over
    plus 20,000 random pixels."""
    theta = theta_am * gen.ARCMIN
    npix = 12 * nside * nside
    T = np.ones(ntab)
    maps = [np.random.default_rng(100 * nside + theta_am + b).integers(-8, 9, size=npix).astype(np.float32) for b in range(B)]
    tb = O.ring_table(nside)
    with sc.Plan(nside, T, theta, B) as plan:
        part = plan.partition()
        assert part["polar_rings"] < part["first_belt_ring"] <= 2 * nside, part      # all three kernels are in use
        rings = _handover_rings(nside, part["polar_rings"], part["first_belt_ring"])
        sel = np.unique(np.concatenate([_ring_pixels(tb, rings), gen.sample_pixels(nside, 20000, seed=nside + theta_am)]))
        out = _gpu_convolve(sc, plan, maps)
        assert sc.sc_last_launch_count(plan.handle) == 3
    ref, cnt, _ = O.convolve(nside, T, theta, maps, sel=sel)
    omega64 = 4 * np.pi / npix
    omega = np.float32(omega64)
    for b in range(B):
        s = np.rint(ref[b] / omega64)
        assert np.max(np.abs(ref[b] / omega64 - s)) < 1e-6 and np.max(np.abs(s)) < 2 ** 24
        want = s.astype(np.float32) * omega
        bad = np.nonzero(out[b][sel] != want)[0]
        assert bad.size == 0, (part, sel[bad[:10]], out[b][sel][bad[:10]], want[bad[:10]])


@pytest.mark.parametrize("nside,theta_am,ntab", [(1024, 30, 8192), (1024, 72, 8192), (2048, 20, 16384)])
def test_sym_staging_layouts_agree(sc, nside, theta_am, ntab, monkeypatch):
    """The 16-image sym kernel stages its input runs either as one plane per image by TMA bulk copies (the default,
    sc_sym_pl.cu; lanes skewed so that their 4-byte loads stay 3 positions apart) or as float4-interleaved rotation
    images by 4-byte cp.async (SC_SYM_NOPLANAR).  Same pairs, same weights up to the fp32 rounding of the azimuth (the
    tilings differ, so a pixel's offset is split differently between the integer part and j dphi'): the outputs agree
    to fp32 rounding, and with K == 1 and integer maps bit for bit."""
    theta = theta_am * gen.ARCMIN
    npix = 12 * nside * nside
    rng = np.random.default_rng(nside + theta_am)
    m = rng.standard_normal(npix).astype(np.float32)
    mi = rng.integers(-8, 9, size=npix).astype(np.float32)
    T = np.exp(-np.linspace(4.0, 0.0, ntab))
    res = []
    for noplanar in (False, True):
        if noplanar:
            monkeypatch.setenv("SC_SYM_NOPLANAR", "1")
        with sc.Plan(nside, T, theta, 1) as plan:
            a = _gpu_convolve(sc, plan, [m])[0]
        with sc.Plan(nside, np.ones(ntab), theta, 1) as plan:
            ai = _gpu_convolve(sc, plan, [mi])[0]
        res.append((a, ai))
    np.testing.assert_array_equal(res[0][1], res[1][1])
    assert np.max(np.abs(res[0][0] - res[1][0])) <= 2e-6 * np.max(np.abs(res[0][0]))


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("nside,theta_deg,ntab", [(1, 60.0, 17), (2, 50.0, 2), (3, 89.9, 33), (5, 30.0, 100),
                                                  (8, 75.0, 257), (16, 13.6, 1000), (32, 0.5, 64),
                                                  (11, 7.0, 4096), (64, 90.0, 513)])
def test_edge_geometries_full(sc, path, nside, theta_deg, ntab):
    """Tiny and non-power-of-two Nside, pole-containing discs, whole-ring windows, discs up to a
    hemisphere, 2-node tables, theta_max below the pixel spacing: all pixels, sets and values."""
    npix = 12 * nside * nside
    rng = np.random.default_rng(nside * 1000 + ntab)
    theta = theta_deg * gen.DEG
    # smooth oscillating kernel: fp32 sensitivity |u K'(u)| comparable to the BASELINE configs (a
    # white-noise table would amplify the fp32 rounding of the table coordinate beyond 1e-6)
    _, th = gen.table_nodes(theta, ntab)
    T = np.exp(-3.0 * (th / theta) ** 2) * np.cos(5.0 * th / theta) + 0.1
    maps = [rng.standard_normal(npix).astype(np.float32)]
    ref, cnt, sig = O.convolve(nside, T, theta, maps)
    with sc.Plan(nside, T, theta, 1) as plan:
        _set_path(sc, plan, path)
        assert plan.info()["total_pairs"] == int(cnt.sum())
        _check_counts(sc, plan, cnt, sig)
        out = _gpu_convolve(sc, plan, maps)
    _check_values(out[0], ref[0], f"edge nside {nside} theta {theta_deg}/{path}")


def test_identity_limit(sc):
    """theta_max below the nearest-neighbour distance: count == 1, out = Omega * K(1) * m."""
    nside, theta = 64, 0.2 * gen.DEG
    npix = 12 * nside * nside
    T = np.linspace(0.25, 3.0, 9)
    m = gen.noise_map(npix, 42)
    with sc.Plan(nside, T, theta, 1) as plan:
        cnt, _ = plan.neighbour_counts()
        assert int(cnt.min()) == 1 and int(cnt.max()) == 1
        out = _gpu_convolve(sc, plan, [m])
    want = (4 * np.pi / npix) * 3.0 * m.astype(np.float64)
    np.testing.assert_allclose(out[0], want, rtol=3e-7, atol=0)


def test_batch_chunking_and_host_entry(sc):
    """B = 6 (> maps per launch) through sc_convolve, and the HOST-buffer entry sc_convolve_host,
    give the same numbers as six single-map calls."""
    cfg = gen.config(1)
    T = gen.table_for(cfg)
    maps = [gen.noise_map(cfg.npix, 50 + i) for i in range(6)]
    with sc.Plan(cfg.nside, T, cfg.theta_max, 6) as plan:
        single = [_gpu_convolve(sc, plan, [m])[0] for m in maps]
        batch = _gpu_convolve(sc, plan, maps)
        host = plan.convolve_host(maps)
    ref, _, _ = O.convolve(cfg.nside, T, cfg.theta_max, maps)
    for b in range(6):
        # the host entry runs the same launches as the device entry: bit-identical; a batched launch
        # may use another pixels-per-thread shape than a single-map launch (different fp32 summation
        # order), so batch vs single is held to the oracle bar instead
        np.testing.assert_array_equal(host[b], batch[b])
        _check_values(batch[b], single[b].astype(np.float64), f"batch6 vs single map{b}")
        _check_values(batch[b], ref[b], f"batch6 map{b}")


@pytest.mark.parametrize("nside,theta_deg,ntab,B", [(512, 1.0, 4096, 1),      # belt_kernel<128>, sym 384 variant
                                                   (512, 2.5, 2048, 2),      # belt_kernel<128>, B = 2, two accumulator sets
                                                   (768, 0.8, 4096, 1),      # Nside not a multiple of 512: no belt kernel
                                                   (1024, 1.2, 8192, 1)])    # belt_kernel<256>, discs of ~1500 pixels
def test_other_kernel_variants_sampled(sc, nside, theta_deg, ntab, B):
    """Shapes outside BASELINE.json's five configs that select the other kernel variants: sampled pixels
    (poles, cap/belt boundaries, equator + random) and whole rings around the kernel boundaries."""
    theta = theta_deg * gen.DEG
    npix = 12 * nside * nside
    _, th = gen.table_nodes(theta, ntab)
    T = np.exp(-3.0 * (th / theta) ** 2) * np.cos(4.0 * th / theta) + 0.05
    maps = [gen.noise_map(npix, 300 + nside + b) for b in range(B)]
    tb = O.ring_table(nside)
    with sc.Plan(nside, T, theta, B) as plan:
        part = plan.partition()
        pr, fb = part["polar_rings"], part["first_belt_ring"]
        rings = sorted({1, 2, pr, pr + 1, nside - 1, nside, nside + 1, min(fb, 2 * nside) - 1, min(fb, 2 * nside),
                        2 * nside - 1, 2 * nside, 2 * nside + 1, 4 * nside - min(fb, 2 * nside), 4 * nside - pr,
                        4 * nside - pr - 1, 4 * nside - 1} - {0})
        sel = np.concatenate([np.arange(tb["start"][r - 1], tb["start"][r - 1] + tb["npr"][r - 1]) for r in rings]
                             + [gen.sample_pixels(nside, 3000, seed=nside)])
        sel = np.unique(sel)
        ref, cnt, sig = O.convolve(nside, T, theta, maps, sel=sel)
        c, s = plan.neighbour_counts()
        c, s = c.cpu().numpy(), s.cpu().numpy().view(np.uint64)
        np.testing.assert_array_equal(c[sel], cnt)
        np.testing.assert_array_equal(s[sel], sig)
        out = _gpu_convolve(sc, plan, maps)
        for b in range(B):
            _check_values(out[b][sel], ref[b], f"nside {nside} theta {theta_deg} B {B} map{b} {part}")
            assert np.all(np.isfinite(out[b]))


@pytest.mark.parametrize("ci,world", [(1, 1), (1, 2), (1, 5), (2, 3), (3, 2), (3, 4), (3, 7)])
def test_latitude_bands(sc, ci, world):
    """Latitude bands: the bands' output rows tile the sphere, every band reads only its rows
    + overlap (everything else is poisoned with NaN) and the union of the band results equals sc_convolve
    bit for bit (same per-pixel arithmetic, only the tiling differs)."""
    import torch
    cfg = gen.config(ci)
    T = gen.table_for(cfg)
    m = torch.from_numpy(gen.noise_map(cfg.npix, 500 + ci)).cuda()
    with sc.Plan(cfg.nside, T, cfg.theta_max, 1) as plan:
        full = plan.convolve([m])[0]
        out = torch.full_like(m, float("nan"))
        covered = torch.zeros(cfg.npix, dtype=torch.int32, device="cuda")
        prev_hi = 0
        for rank in range(world):
            bd = plan.band(world, rank)
            assert bd["ring_lo"] == prev_hi + 1 and bd["ring_hi"] >= bd["ring_lo"]
            prev_hi = bd["ring_hi"]
            o, i = bd["out_rows"], bd["in_rows"]
            covered[o[0]:o[1]] += 1
            covered[o[2]:o[3]] += 1
            assert i[0] <= o[0] and i[3] >= o[3]
            poisoned = torch.full_like(m, float("nan"))
            poisoned[i[0]:i[1]] = m[i[0]:i[1]]
            poisoned[i[2]:i[3]] = m[i[2]:i[3]]
            plan.convolve_band(bd["ring_lo"], bd["ring_hi"], [poisoned], [out])
            plan.convolve_band(bd["ring_lo"], bd["ring_hi"], [poisoned], [out])      # cached tile list, same result
        torch.cuda.synchronize()
        assert prev_hi == 2 * cfg.nside
        assert int(covered.min()) == 1 and int(covered.max()) == 1
        assert torch.equal(out, full)
        # the generic path honours bands too
        plan.set_path(sc.SC_PATH_GENERIC)
        out2 = torch.full_like(m, float("nan"))
        for rank in range(world):
            bd = plan.band(world, rank)
            plan.convolve_band(bd["ring_lo"], bd["ring_hi"], [m], [out2])
        torch.cuda.synchronize()
        assert not bool(torch.isnan(out2).any())
        ref = plan.convolve([m])[0]
        assert torch.equal(out2, ref)
        with pytest.raises(sc.ScError):
            plan.band(0, 0)
        with pytest.raises(sc.ScError):
            sc.sc_convolve_band(plan.handle, 5, 4, [m.data_ptr()], [out.data_ptr()])


@pytest.mark.parametrize("ci,world,B", [(1, 2, 1), (2, 3, 2), (3, 4, 1), (3, 8, 1)])
def test_bands_with_simulated_halo_exchange(sc, ci, world, B):
    """The PRODUCT's sc_band_partition output driven through dist.halo_plan with `world` simulated ranks on one GPU:
    every rank has a full-size buffer that is valid in its own rows only (NaN elsewhere), the copies halo_plan prescribes
    are carried out between the buffers, every rank convolves its band, and the union equals sc_convolve bit for bit.
    (The gloo tests exercise the same halo_plan with real point-to-point messages; this one ties it to the kernels.)"""
    import torch
    from paper_1409_4441_b200 import dist as D
    cfg = gen.config(ci)
    T = gen.table_for(cfg)
    maps = [torch.from_numpy(gen.noise_map(cfg.npix, 600 + 7 * ci + b)).cuda() for b in range(B)]
    with sc.Plan(cfg.nside, T, cfg.theta_max, B) as plan:
        full = plan.convolve(maps)
        bands = [plan.band(world, r) for r in range(world)]
        own = [D._ranges(b["out_rows"]) for b in bands]
        bufs = []
        for r in range(world):
            mine = [torch.full_like(m, float("nan")) for m in maps]
            for t, m in zip(mine, maps):
                for lo, hi in own[r]:
                    t[lo:hi] = m[lo:hi]
            bufs.append(mine)
        plans = [D.halo_plan(bands, r) for r in range(world)]
        for r in range(world):
            sends, recvs = plans[r]
            for peer, lo, hi in sends:                          # both sides agree on every message
                assert (r, lo, hi) in plans[peer][1]
            for peer, lo, hi in recvs:
                assert (r, lo, hi) in plans[peer][0]
                assert any(a <= lo and hi <= b for a, b in own[peer])      # the sender owns what it sends
                for t, src in zip(bufs[r], bufs[peer]):
                    t[lo:hi] = src[lo:hi]
        out = [torch.full_like(m, float("nan")) for m in maps]
        for r in range(world):
            for t in bufs[r]:                                   # everything the band reads has arrived
                for lo, hi in D._ranges(bands[r]["in_rows"]):
                    assert not bool(torch.isnan(t[lo:hi]).any())
            plan.convolve_band(bands[r]["ring_lo"], bands[r]["ring_hi"], bufs[r], out)
        torch.cuda.synchronize()
        for o, f in zip(out, full):
            assert torch.equal(o, f)


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("ci,frac,B", [(1, 0.3, 1), (1, 1.0, 2), (2, 0.5, 1), (3, 0.45, 1), (3, 0.97, 2), (4, 0.3, 1)])
def test_north_cap_only(sc, path, ci, frac, B):
    """sc_convolve_cap (the survey area rotated into the polar cap): output rings 1 .. ring_hi only, from
    TRUNCATED buffers that hold just the rows sc_cap_rows names (NaN guard words after the input, a sentinel after the
    output): nothing beyond is read or written, no southern mirror is computed, values and -- with K == 1 and integer
    maps -- the neighbour sets equal the oracle's."""
    import torch
    cfg = gen.config(ci)
    N = cfg.nside
    if path == "generic" and N > 1024:
        pytest.skip("generic path at Nside 2048: minutes")
    ring_hi = max(1, min(2 * N, int(round(frac * 2 * N))))
    T = gen.table_for(cfg)
    maps = [gen.noise_map(cfg.npix, 1200 + 10 * ci + b) for b in range(B)]
    imaps = [np.random.default_rng(77 + b).integers(-8, 9, size=cfg.npix).astype(np.float32) for b in range(B)]
    tb = O.ring_table(N)
    for table, inputs, exact in ((T, maps, False), (np.ones(cfg.n_table), imaps, True)):
        with sc.Plan(N, table, cfg.theta_max, B) as plan:
            _set_path(sc, plan, path)
            rows = plan.cap_rows(ring_hi)
            o1, i1 = rows["out_rows"][1], rows["in_rows"][1]
            assert rows["out_rows"][0] == 0 and rows["in_rows"][0] == 0 and o1 <= i1 <= cfg.npix
            assert o1 == int(tb["start"][ring_hi - 1] + tb["npr"][ring_hi - 1])
            bin_, bout = [], []
            for m in inputs:
                t = torch.full((i1 + 64,), float("nan"), dtype=torch.float32, device="cuda")
                t[:i1] = torch.from_numpy(m[:i1]).cuda()
                bin_.append(t)
                bout.append(torch.full((o1 + 64,), -777.0, dtype=torch.float32, device="cuda"))
            plan.convolve_cap(ring_hi, bin_, bout)
            plan.convolve_cap(ring_hi, bin_, bout)                    # cached tile list, same result
            torch.cuda.synchronize()
            part = plan.partition()
        rings = sorted({1, 2, max(1, min(part["polar_rings"], ring_hi)), min(part["polar_rings"] + 1, ring_hi),
                        min(N, ring_hi), max(1, ring_hi - 1), ring_hi})
        sel = np.unique(np.concatenate([_ring_pixels(tb, rings), np.random.default_rng(ci).integers(0, o1, size=6000)]))
        ref, _, _ = O.convolve(N, table, cfg.theta_max, inputs, sel=sel)
        for b in range(B):
            got = bout[b].cpu().numpy()
            assert np.all(got[o1:] == -777.0)                        # nothing written beyond the cap
            assert np.all(np.isfinite(got[:o1]))                     # nothing read beyond in_rows (NaN guard)
            if exact:
                omega64 = 4 * np.pi / cfg.npix
                want = np.rint(ref[b] / omega64).astype(np.float32) * np.float32(omega64)
                np.testing.assert_array_equal(got[sel], want)
            else:
                _check_values(got[sel], ref[b], f"cap cfg{ci} ring_hi {ring_hi}/{path}/map{b}")
    with sc.Plan(N, T, cfg.theta_max, 1) as plan:
        with pytest.raises(sc.ScError):
            plan.cap_rows(0)
        with pytest.raises(sc.ScError):
            plan.cap_rows(2 * N + 1)


def test_profile_entry_and_partition(sc):
    """sc_convolve_profile runs the same launches as sc_convolve (bit-identical output) and reports a
    positive device time for every kernel the plan uses; sc_plan_partition is consistent with them."""
    import torch
    cfg = gen.config(3)
    T = gen.table_for(cfg)
    m = torch.from_numpy(gen.noise_map(cfg.npix, 77)).cuda()
    with sc.Plan(cfg.nside, T, cfg.theta_max, 1) as plan:
        a = plan.convolve([m])[0]
        b = torch.empty_like(m)
        ms = plan.convolve_profile([m], [b])
        part = plan.partition()
        torch.cuda.synchronize()
        assert torch.equal(a, b)
        N = cfg.nside
        assert 0 < part["polar_rings"] < N and part["polar_rings"] < part["first_belt_ring"] <= 2 * N
        assert set(ms) == set(sc.KERNEL_NAMES)
        assert all(v > 0 for v in ms.values()), ms
        assert sc.sc_last_launch_count(plan.handle) == 3
        plan.set_path(sc.SC_PATH_GENERIC)
        ms = plan.convolve_profile([m], [b])
        assert ms["generic_warp_kernel"] > 0.1 and ms["belt_kernel"] < 0.01 and ms["sym_kernel"] < 0.01


@pytest.mark.parametrize("ci,B", [(3, 1), (3, 5), (2, 2)])
def test_host_entry_pipelined_chunks(sc, ci, B):
    """sc_convolve_host (latitude chunks on three streams, belt + cap kernels launched per chunk) returns
    exactly what sc_convolve computes, also when B exceeds the maps per launch."""
    cfg = gen.config(ci)
    T = gen.table_for(cfg)
    maps = [gen.noise_map(cfg.npix, 700 + 10 * ci + b) for b in range(B)]
    with sc.Plan(cfg.nside, T, cfg.theta_max, B) as plan:
        dev = _gpu_convolve(sc, plan, maps)
        host = plan.convolve_host(maps)
        host2 = plan.convolve_host(maps)                      # event pool reuse
        assert sc.sc_last_launch_count(plan.handle) > 3
    for b in range(B):
        np.testing.assert_array_equal(host[b], dev[b])
        np.testing.assert_array_equal(host2[b], dev[b])


def test_paper_style_split_kernel(sc):
    """A real-space kernel from the paper's least-squares split (PAPER.md:29-58 via workloads/splitfit.py: the
    oscillating, compact part that complements an l-space kernel truncated at l_cut) through the CUDA path:
    sampled pixels against the oracle."""
    from workloads import splitfit
    nside, theta = 256, 4.0 * gen.DEG
    K_ell = splitfit.gaussian_beam_ell(30 * gen.ARCMIN, 3 * nside - 1)
    fit = splitfit.split_fit(K_ell, ell_cut=256, theta_cut=theta, n_nodes=512)
    T = fit["K_hat_theta"]
    assert np.all(np.isfinite(T)) and np.sum(np.diff(np.sign(T)) != 0) >= 3          # it oscillates (Fig. 4)
    maps = [gen.noise_map(12 * nside * nside, 4040)]
    sel = gen.sample_pixels(nside, 8000, seed=41)
    ref, cnt, sig = O.convolve(nside, T, theta, maps, sel=sel)
    with sc.Plan(nside, T, theta, 1) as plan:
        out = _gpu_convolve(sc, plan, maps)
        c, s = plan.neighbour_counts()
    np.testing.assert_array_equal(c.cpu().numpy()[sel], cnt)
    _check_values(out[0][sel], ref[0], "paper-style split kernel")


def _zoned_gauss(theta, n, f, fwhm, ripple):
    x, th = gen.zoned_table_nodes(theta, n, f)
    sigma = fwhm / 2.3548
    return np.exp(-0.5 * (th / sigma) ** 2) * (1.0 + ripple * np.cos(9.0 * th / theta))


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("nside,theta_deg,n,f,B", [(64, 3.4, 4096, 1.0 / 16.0, 1), (128, 2.0, 1024, 0.125, 2),
                                                     (37, 6.0, 64, 0.5, 1), (256, 1.5, 4096, 1.0 / 16.0, 3)])
def test_two_zone_table_full(sc, path, nside, theta_deg, n, f, B):
    """Paper-style two-zone table (reading R11): every pixel against the oracle's
    sco_convolve_zoned, both kernel paths."""
    theta = theta_deg * gen.DEG
    npix = 12 * nside * nside
    T = _zoned_gauss(theta, n, f, 0.6 * theta, 0.3)
    maps = [gen.noise_map(npix, 8100 + nside + b) for b in range(B)]
    ref, cnt, sig = O.convolve(nside, T, theta, maps, zone_frac=f)
    with sc.Plan(nside, T, theta, B, zone_frac=f) as plan:
        _set_path(sc, plan, path)
        _check_counts(sc, plan, cnt, sig)
        out = _gpu_convolve(sc, plan, maps)
    for b in range(B):
        _check_values(out[b], ref[b], f"zoned nside {nside} f {f:.3f} n {n}/{path}/map{b}")


@pytest.mark.parametrize("ci", [3, 4])
def test_two_zone_table_sampled_large(sc, ci):
    """Two-zone table at Nside 1024 / 2048 (sym + belt + polar kernels): sampled pixels; the uniform-table
    result of the same kernel differs by the table's interpolation error only."""
    cfg = gen.config(ci)
    f, n = 1.0 / 16.0, cfg.n_table
    T = _zoned_gauss(cfg.theta_max, n, f, cfg.fwhm, 0.2)
    maps = gen.maps_for(cfg)
    sel = gen.sample_pixels(cfg.nside, 6000, seed=300 + ci)
    ref, cnt, sig = O.convolve(cfg.nside, T, cfg.theta_max, maps, sel=sel, zone_frac=f)
    with sc.Plan(cfg.nside, T, cfg.theta_max, 1, zone_frac=f) as plan:
        c, s = plan.neighbour_counts()
        np.testing.assert_array_equal(c.cpu().numpy()[sel], cnt)
        out = _gpu_convolve(sc, plan, maps)
        host = plan.convolve_host(maps)
    _check_values(out[0][sel], ref[0], f"zoned cfg{ci}")
    np.testing.assert_array_equal(host[0], out[0])


def test_two_zone_arguments(sc):
    T = np.ones(16)
    with pytest.raises(sc.ScError):
        sc.Plan(8, np.ones(15), 0.2, 1, zone_frac=0.1)          # odd n
    with pytest.raises(sc.ScError):
        sc.Plan(8, T, 0.2, 1, zone_frac=1.0)
    with pytest.raises(sc.ScError):
        sc.Plan(8, T, 0.2, 1, zone_frac=0.95)                   # inner zone sparser than the outer one


@pytest.mark.parametrize("nside,theta_deg,B", [(1, 70.0, 1), (4, 30.0, 2), (64, 3.4, 1), (256, 1.5, 5), (1024, 0.5, 1)])
def test_nested_ordering(sc, nside, theta_deg, B):
    """SC_ORDER_NESTED plans: NESTED maps in, NESTED maps out.  The device index map nest -> ring is checked
    against the oracle's independent one (oracle/nested.py) through the results: out_nested[p] must equal the
    oracle's RING result at nest2ring(p), and the neighbour counts follow the same permutation."""
    from oracle import nested
    theta = theta_deg * gen.DEG
    npix = 12 * nside * nside
    n2r = nested.nest2ring(nside)
    _, th = gen.table_nodes(theta, 1024)
    T = np.exp(-3.0 * (th / theta) ** 2) + 0.1
    ring_maps = [gen.noise_map(npix, 8800 + nside + b) for b in range(B)]
    nest_maps = [m[n2r] for m in ring_maps]                    # nest_map[p] = ring_map[nest2ring(p)]
    sel = None if nside <= 256 else gen.sample_pixels(nside, 4000, seed=9)
    ref, cnt, sig = O.convolve(nside, T, theta, ring_maps, sel=sel)
    with sc.Plan(nside, T, theta, B, ordering=sc.SC_ORDER_NESTED) as plan:
        out = _gpu_convolve(sc, plan, nest_maps)
        host = plan.convolve_host(nest_maps)
        c, s = plan.neighbour_counts()
        c = c.cpu().numpy()
    inv = np.empty(npix, np.int64)
    inv[n2r] = np.arange(npix)                                  # ring pixel -> nested pixel
    pix = np.arange(npix) if sel is None else sel
    np.testing.assert_array_equal(c[inv[pix]], cnt)
    for b in range(B):
        _check_values(out[b][inv[pix]], ref[b], f"nested nside {nside} map{b}")
        np.testing.assert_array_equal(host[b], out[b])
    with sc.Plan(nside, T, theta, B) as ring_plan:              # same kernels: bit-identical to the RING plan
        ring_out = _gpu_convolve(sc, ring_plan, ring_maps)
    for b in range(B):
        np.testing.assert_array_equal(out[b], ring_out[b][n2r])


def test_nested_arguments(sc):
    import torch
    T = np.ones(8)
    with pytest.raises(sc.ScError):
        sc.Plan(12, T, 0.2, 1, ordering=sc.SC_ORDER_NESTED)     # not a power of two
    with sc.Plan(8, T, 0.2, 1, ordering=sc.SC_ORDER_NESTED) as plan:
        m = torch.zeros(768, device="cuda")
        with pytest.raises(sc.ScError):
            sc.sc_convolve_band(plan.handle, 1, 4, [m.data_ptr()], [torch.empty_like(m).data_ptr()])


@pytest.mark.parametrize("seed", range(8))
def test_random_shapes_against_oracle(sc, seed):
    """Seeded random (Nside, theta_max, table size, batch): every pixel against the oracle (sets and values),
    and the host entry / latitude bands bit-identical to sc_convolve."""
    import torch
    rng = np.random.default_rng(9000 + seed)
    nside = int(rng.choice([3, 7, 31, 100, 128, 200, 256, 300]))
    npix = 12 * nside * nside
    pix = np.sqrt(4 * np.pi / npix)
    theta = float(min(np.pi / 2, pix * rng.uniform(0.3, 9.0)))
    ntab = int(rng.choice([2, 17, 1000, 4096, 16384]))
    B = int(rng.choice([1, 1, 2, 3, 5]))
    _, th = gen.table_nodes(theta, ntab)
    T = np.exp(-2.5 * (th / theta) ** 2) * np.cos(rng.uniform(0, 6) * th / theta) + 0.02
    maps = [gen.noise_map(npix, 9100 + 10 * seed + b) for b in range(B)]
    ref, cnt, sig = O.convolve(nside, T, theta, maps)
    with sc.Plan(nside, T, theta, B) as plan:
        assert plan.info()["total_pairs"] == int(cnt.sum())
        _check_counts(sc, plan, cnt, sig)
        dm = [torch.from_numpy(m).cuda() for m in maps]
        out = plan.convolve(dm)
        host = plan.convolve_host(maps)
        band_out = [torch.full_like(d, float("nan")) for d in dm]
        world = int(rng.integers(1, 6))
        for rank in range(world):
            bd = plan.band(world, rank)
            plan.convolve_band(bd["ring_lo"], bd["ring_hi"], dm, band_out)
        torch.cuda.synchronize()
    for b in range(B):
        got = out[b].cpu().numpy()
        _check_values(got, ref[b], f"random shape seed {seed}: nside {nside} theta/pix {theta / pix:.2f} ntab {ntab} B {B}")
        np.testing.assert_array_equal(host[b], got)
        np.testing.assert_array_equal(band_out[b].cpu().numpy(), got)


def test_table_too_large_for_shared_memory_falls_back_to_generic(sc):
    """A 40,000-node table (320 KB of cells) does not fit the fast kernels' shared memory: the plan has no
    fast path, every entry point still works (generic kernel) and matches the oracle."""
    nside, theta, ntab = 64, 4.0 * gen.DEG, 40000
    npix = 12 * nside * nside
    _, th = gen.table_nodes(theta, ntab)
    T = np.exp(-2.0 * (th / theta) ** 2) * np.cos(6.0 * th / theta)
    maps = [gen.noise_map(npix, 77), gen.noise_map(npix, 78)]
    ref, cnt, sig = O.convolve(nside, T, theta, maps)
    with sc.Plan(nside, T, theta, 2) as plan:
        part = plan.partition()
        assert part["polar_rings"] == 2 * nside and part["first_belt_ring"] == 2 * nside + 1
        _check_counts(sc, plan, cnt, sig)
        out = _gpu_convolve(sc, plan, maps)
        host = plan.convolve_host(maps)
        import torch
        dm = [torch.from_numpy(m).cuda() for m in maps]
        band_out = [torch.full_like(d, float("nan")) for d in dm]
        for rank in range(3):
            bd = plan.band(3, rank)
            plan.convolve_band(bd["ring_lo"], bd["ring_hi"], dm, band_out)
        torch.cuda.synchronize()
    for b in range(2):
        _check_values(out[b], ref[b], f"large table map{b}")
        np.testing.assert_array_equal(host[b], out[b])
        np.testing.assert_array_equal(band_out[b].cpu().numpy(), out[b])


def test_cuda_graph_capture(sc):
    """sc_convolve only enqueues kernels on the caller's stream (no allocation, no host sync), so it can be
    captured into a CUDA graph and replayed; the replay gives the same bits."""
    import torch
    cfg = gen.config(2)
    T, maps = gen.table_for(cfg), gen.maps_for(cfg)
    with sc.Plan(cfg.nside, T, cfg.theta_max, cfg.batch) as plan:
        dm = [torch.from_numpy(m).cuda() for m in maps]
        ref = plan.convolve(dm)
        out = [torch.empty_like(m) for m in dm]
        g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
        with torch.cuda.stream(s):
            plan.convolve(dm, out)
            s.synchronize()
            with torch.cuda.graph(g, stream=s):
                plan.convolve(dm, out)
        for o in out:
            o.zero_()
        g.replay()
        g.replay()
        torch.cuda.synchronize()
        for a, b in zip(ref, out):
            assert torch.equal(a, b)


def test_knife_edge_host_adjudication(sc, monkeypatch):
    """Widen the knife-edge band so that many pairs are decided on the host with the host libm;
    sets must still equal the oracle's and the override list must be in use."""
    monkeypatch.setenv("SC_KNIFE_EDGE_BAND", "1e-3")
    nside, theta = 32, 6.0 * gen.DEG
    npix = 12 * nside * nside
    T = np.ones(16)
    m = np.random.default_rng(3).integers(-8, 9, size=npix).astype(np.float32)
    ref, cnt, sig = O.convolve(nside, T, theta, [m])
    with sc.Plan(nside, T, theta, 1) as plan:
        info = plan.info()
        assert info["n_knife_edge"] > 0
        assert info["total_pairs"] == int(cnt.sum())
        _check_counts(sc, plan, cnt, sig)
        out = _gpu_convolve(sc, plan, [m])
    omega = np.float32(4 * np.pi / npix)
    want = np.rint(ref[0] / (4 * np.pi / npix)).astype(np.float32) * omega
    np.testing.assert_array_equal(out[0], want)


def test_argument_errors_on_gpu(sc):
    import torch
    cfg = gen.config(1)
    with sc.Plan(cfg.nside, gen.table_for(cfg), cfg.theta_max, 1) as plan:
        a = torch.zeros(cfg.npix, device="cuda")
        with pytest.raises(sc.ScError):            # aliasing
            sc.sc_convolve(plan.handle, [a.data_ptr()], [a.data_ptr()])
        with pytest.raises(sc.ScError):            # misaligned
            sc.sc_convolve(plan.handle, [a.data_ptr() + 4], [torch.empty_like(a).data_ptr()])
        with pytest.raises(sc.ScError):            # empty batch
            sc.sc_convolve(plan.handle, [], [])


@pytest.mark.parametrize("nside,theta_deg,ntab,B,pair", [(64, 3.4, 4096, 1, False), (256, 1.5, 4096, 2, False),
                                                         (512, 1.0, 4096, 1, False), (1024, 0.5, 8192, 1, False),
                                                         (256, 1.5, 4096, 1, True), (1024, 0.5, 8192, 1, True)])
def test_guard_regions_untouched(sc, nside, theta_deg, ntab, B, pair, monkeypatch):
    """Our own bounds check (compute-sanitizer is closed on this GPU pool, profiles/r2_sanitizer.md): every map sits
    inside a larger buffer between guard regions.  Input guards hold NaN -- a read outside the map would poison an
    output --, output guards hold a sentinel that must survive; both the fast kernels and the generic kernel, the
    device and the band entry.  pair: the lane-pair sym instance (SC_SYM_PAIR)."""
    import torch
    if pair:
        monkeypatch.setenv("SC_SYM_PAIR", "1")
    theta = np.deg2rad(theta_deg)
    x, th = gen.table_nodes(theta, ntab)
    T = np.exp(-0.5 * (th / (theta / 3.0)) ** 2)
    npix, G = 12 * nside * nside, 4096                       # guard: 4096 floats on each side (keeps 16-byte alignment)
    SENT = 1234.5
    with sc.Plan(nside, T, theta, B) as plan:
        ins, outs, ibuf, obuf = [], [], [], []
        for b in range(B):
            ib = torch.full((npix + 2 * G,), float("nan"), dtype=torch.float32, device="cuda")
            ib[G:G + npix] = torch.from_numpy(gen.noise_map(npix, 70 + b)).cuda()
            ob = torch.full((npix + 2 * G,), SENT, dtype=torch.float32, device="cuda")
            ibuf.append(ib); obuf.append(ob); ins.append(ib[G:G + npix]); outs.append(ob[G:G + npix])
        for path in PATHS:
            _set_path(sc, plan, path)
            for ob in obuf:
                ob.fill_(SENT)
            plan.convolve(ins, outs)
            torch.cuda.synchronize()
            for ob in obuf:
                assert bool((ob[:G] == SENT).all()) and bool((ob[G + npix:] == SENT).all()), f"{path}: write outside the map"
                assert bool(torch.isfinite(ob[G:G + npix]).all()), f"{path}: read outside the map (NaN guard)"
                assert not bool((ob[G:G + npix] == SENT).any()), f"{path}: pixels left unwritten"
        _set_path(sc, plan, "auto")
        plan.convolve(ins, outs)
        full = [o.clone() for o in outs]
        for rank in range(3):                                     # bands write only their own rows
            band = plan.band(3, rank)
            for ob in obuf:
                ob.fill_(SENT)
            plan.convolve_band(band["ring_lo"], band["ring_hi"], ins, outs)
            torch.cuda.synchronize()
            o0, o1, o2, o3 = band["out_rows"]
            for ob, fo in zip(obuf, full):
                body = ob[G:G + npix]
                assert bool((ob[:G] == SENT).all()) and bool((ob[G + npix:] == SENT).all())
                mask = torch.ones(npix, dtype=torch.bool, device="cuda")
                mask[o0:o1] = False; mask[o2:o3] = False
                assert bool((body[mask] == SENT).all()), "band wrote outside its rows"
                assert bool(torch.equal(body[~mask], fo[~mask])), "band rows differ from the whole-map call"


def test_paper_operating_point_split_kernel(sc):
    """The paper's own operating point (Fig. 3-4: 7' beam, l_max 4096, l_cut 1500, theta_cut 240') with a
    real-space kernel from the least-squares split itself (workloads/splitfit.py, Eq. 1-6) instead of config 6's smooth
    stand-in: an oscillating kernel (33 periods across the disc, sum|K| / |sum K| = 67) over ~61,000 neighbours per pixel
    at Nside 2048.  NOT a BASELINE.json config.  With the fp32 pair geometry this kernel comes out at a relative rms of
    1.8e-6 (K'(theta) theta / K ~ 200 against 6e-8 resolution of 1 - cos theta; the paper reports the same
    single-precision sensitivity as alpha = 5): the plan detects the steep table and forms the table
    coordinate in fp64 (sc_plan_double_coordinate), which brings it under the bars of the BASELINE configs."""
    from workloads import splitfit
    nside, theta = 2048, 240 * gen.ARCMIN
    K_ell = splitfit.gaussian_beam_ell(7 * gen.ARCMIN, 4096)
    fit = splitfit.split_fit(K_ell, ell_cut=1500, theta_cut=theta, n_nodes=512)
    T = fit["K_hat_theta"]
    assert np.all(np.isfinite(T)) and np.sum(np.diff(np.sign(T)) != 0) >= 3          # it oscillates (Fig. 4)
    maps = [gen.noise_map(12 * nside * nside, 4041)]
    sel = gen.sample_pixels(nside, 300, seed=67)
    ref, cnt, sig = O.convolve(nside, T, theta, maps, sel=sel)
    with sc.Plan(nside, T, theta, 1) as plan:
        assert plan.info()["double_coordinate"] == 1
        out = _gpu_convolve(sc, plan, maps)
        assert sc.sc_last_launch_count(plan.handle) == 3          # polar + sym + belt kernels, not the generic fallback
        c, s = plan.neighbour_counts()
    np.testing.assert_array_equal(c.cpu().numpy()[sel], cnt)
    np.testing.assert_array_equal(s.cpu().numpy().view(np.uint64)[sel], sig)
    print("sum|K|/|sum K| =", float(np.sum(np.abs(T)) / abs(np.sum(T))))
    _check_values(out[0][sel], ref[0], "split-fit kernel at the paper's operating point")


@pytest.mark.parametrize("path", PATHS)
@pytest.mark.parametrize("ci,B", [(1, 1), (2, 2), (3, 1)])
def test_double_coordinate_mode_full_maps(sc, path, ci, B, monkeypatch):
    """The fp64 table coordinate forced (SC_HP=1) on BASELINE configs 1-3: every pixel against the oracle through the
    16-image sym instance, the belt stencil (config 3), the warp-per-pixel kernel and the generic kernel; batches run
    one map per launch; counts are untouched by the mode."""
    monkeypatch.setenv("SC_HP", "1")
    cfg = gen.config(ci)
    T = gen.table_for(cfg)
    maps = [gen.noise_map(cfg.npix, 900 + ci + b) for b in range(B)]
    ref, cnt, sig = O.convolve(cfg.nside, T, cfg.theta_max, maps)
    with sc.Plan(cfg.nside, T, cfg.theta_max, B) as plan:
        assert plan.info()["double_coordinate"] == 1
        _set_path(sc, plan, path)
        out = _gpu_convolve(sc, plan, maps)
        if path == "auto":
            _check_counts(sc, plan, cnt, sig)
            host = plan.convolve_host(maps)
            for b in range(B):
                np.testing.assert_array_equal(host[b], out[b])
    for b in range(B):
        _check_values(out[b], ref[b], f"cfg{ci} fp64 coordinate {path} map{b}")


def test_double_coordinate_exact_integer_sums(sc, monkeypatch):
    """Inclusion is untouched by the fp64 coordinate: K == 1, small-integer maps, bit-exact sums (Nside 512: belt taps,
    sym and polar kernels in the mode)."""
    monkeypatch.setenv("SC_HP", "1")
    nside, theta = 512, 1.0 * gen.DEG
    npix = 12 * nside * nside
    rng = np.random.default_rng(5)
    m = rng.integers(-3, 4, npix).astype(np.float32)
    T = np.ones(64)
    sel = gen.sample_pixels(nside, 20000, seed=9)
    ref, cnt, _ = O.convolve(nside, T, theta, [m], sel=sel)
    with sc.Plan(nside, T, theta, 1) as plan:
        assert plan.info()["double_coordinate"] == 1
        out = _gpu_convolve(sc, plan, [m])[0]
    omega = np.float32(4.0 * np.pi / npix)
    want = (np.round(ref[0] / (4.0 * np.pi / npix)).astype(np.float32) * omega).astype(np.float32)
    np.testing.assert_array_equal(out[sel], want)


def test_fma_peak_probe_modes(sc):
    """sc_debug_fma_peak: scalar, packed and the kernels' operand pattern all give a plausible rate (the pattern loop
    cannot beat the constant-operand one), other modes are refused."""
    rates = [sc.sc_debug_fma_peak(packed=m)["fma_per_s"] for m in (0, 1, 2)]
    assert all(1e12 < r < 1e14 for r in rates), rates
    assert rates[2] <= 1.02 * max(rates[:2]), rates
    with pytest.raises(sc.ScError):
        sc.sc_debug_fma_peak(packed=3)
