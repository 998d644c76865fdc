"""sc_neighbour_counts_static (include/sc.h): the neighbour count without any allocation -- its RING-ordered scratch is a
static device array -- against the existing path (sc_debug_neighbour_counts, which takes the scratch from cudaMalloc per
call).  Integer results: bit-exact.  Two calls in a row on different NESTED plans, so that contents left in the shared
array by the first call would show in the second.  Collected last on purpose (the suite runs with pytest -x).
"""
import numpy as np
import pytest

from workloads import gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sc():
    import torch
    assert torch.cuda.is_available()
    import paper_1409_4441_b200 as sc
    return sc


def _plan(sc, nside, theta_deg, ordering, n=256):
    theta = theta_deg * gen.DEG
    x, th = gen.table_nodes(theta, n)
    T = np.exp(-0.5 * (th / (theta / 3.0)) ** 2)
    return sc.Plan(nside, T, theta, 1, ordering=ordering)


def _static_counts(sc, plan):
    import torch
    cnt = torch.full((plan.npix,), -7, dtype=torch.int32, device="cuda")
    sig = torch.full((plan.npix,), -7, dtype=torch.int64, device="cuda")
    sc.sc_neighbour_counts_static(plan.handle, cnt.data_ptr(), sig.data_ptr(), torch.cuda.current_stream().cuda_stream)
    return cnt, sig


def test_static_scratch_counts_two_calls_in_a_row(sc):
    import torch
    cases = [(64, 3.4, sc.SC_ORDER_NESTED), (32, 9.0, sc.SC_ORDER_NESTED), (64, 3.4, sc.SC_ORDER_NESTED),
             (16, 20.0, sc.SC_ORDER_RING)]
    got, want = [], []
    plans = [_plan(sc, *c) for c in cases]
    try:
        for plan in plans:                       # back to back on one stream, nothing in between
            got.append(_static_counts(sc, plan))
        for plan in plans:
            want.append(plan.neighbour_counts())
        torch.cuda.synchronize()
        for (c, s), (cw, sw), case in zip(got, want, cases):
            assert int(cw.min()) >= 1, case
            assert torch.equal(c, cw), case
            assert torch.equal(s, sw), case
        # the count without the signature leaves the signature output alone
        cnt = torch.zeros(plans[0].npix, dtype=torch.int32, device="cuda")
        sc.sc_neighbour_counts_static(plans[0].handle, cnt.data_ptr(), 0, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert torch.equal(cnt, want[0][0])
    finally:
        for plan in plans:
            plan.close()


def test_static_scratch_rejects_maps_beyond_the_array(sc):
    import torch
    assert 12 * 128 * 128 == sc.SC_STATIC_MAX_NPIX
    plan = _plan(sc, 256, 0.8, sc.SC_ORDER_NESTED, n=64)
    try:
        cnt = torch.full((plan.npix,), -7, dtype=torch.int32, device="cuda")
        with pytest.raises(sc.ScError) as ei:
            sc.sc_neighbour_counts_static(plan.handle, cnt.data_ptr(), 0, 0)
        assert ei.value.status == 2 and "static scratch" in str(ei.value)
        torch.cuda.synchronize()
        assert int((cnt != -7).sum()) == 0            # nothing was launched
    finally:
        plan.close()
