"""CPU-only checks of the product library: it builds, loads and exports every symbol that
include/sc.h declares; argument validation that needs no GPU; independence of oracle and product."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "sc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sc_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported():
    import paper_1409_4441_b200 as sc
    l = sc.lib()
    decl = _declared_symbols()
    assert len(decl) >= 10
    for name in decl:
        assert hasattr(l, name), name
    assert sorted(sc.EXPORTS) == decl
    assert "sm_100a" in sc.sc_version()


def test_library_is_built_for_sm_100a():
    import subprocess
    from paper_1409_4441_b200 import build
    out = subprocess.run(["cuobjdump", "-lelf", build.build()], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_invalid_arguments_rejected_without_gpu():
    import paper_1409_4441_b200 as sc
    l = sc.lib()
    kt = np.ones(8)
    h = C.c_void_p(None)
    p = kt.ctypes.data_as(C.c_void_p)
    INVALID, UNSUPPORTED = 1, 2
    assert l.sc_plan_create(C.byref(h), 0, 0, p, 8, 0.1, 1) == INVALID          # nside
    assert l.sc_plan_create(C.byref(h), 8, 0, p, 1, 0.1, 1) == INVALID          # n_table
    assert l.sc_plan_create(C.byref(h), 8, 0, p, 8, 0.0, 1) == INVALID          # theta_max
    assert l.sc_plan_create(C.byref(h), 8, 0, p, 8, 2.0, 1) == INVALID          # theta_max > pi/2
    assert l.sc_plan_create(C.byref(h), 8, 0, None, 8, 0.1, 1) == INVALID       # NULL table
    assert l.sc_plan_create(C.byref(h), 8, 0, p, 8, 0.1, 0) == INVALID          # max_batch
    assert l.sc_plan_create(C.byref(h), 12, 1, p, 8, 0.1, 1) == INVALID         # NESTED needs a power of two
    assert l.sc_plan_create(C.byref(h), 8, 7, p, 8, 0.1, 1) == INVALID          # unknown ordering
    assert l.sc_plan_create(C.byref(h), 20000, 0, p, 8, 0.1, 1) == UNSUPPORTED  # 12 nside^2 >= 2^31
    assert h.value is None
    assert l.sc_plan_destroy(None) == 0
    assert l.sc_convolve(None, None, None, 1, None) == INVALID
    assert l.sc_status_string(4) == b"SC_ERR_CUDA"


def test_no_gpu_means_loud_failure():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_1409_4441_b200 as sc
    with pytest.raises(sc.ScError) as e:
        sc.sc_plan_create(8, sc.SC_ORDER_RING, np.ones(8), 0.1, 1)
    assert e.value.status == 4


def test_product_and_oracle_do_not_touch_each_other():
    """Neither side imports, includes or links the other (prompt rule 3)."""
    pkg = os.path.join(ROOT, "paper_1409_4441_b200")
    for d, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(d, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "sco.h" not in txt and "libsco" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1409_4441_b200 import" not in txt and "import paper_1409_4441_b200" not in txt
            assert "sc.h\"" not in txt.replace("sco.h\"", "") and "libsc.so" not in txt
    gen = open(os.path.join(ROOT, "workloads", "gen.py")).read()
    assert "import oracle" not in gen and "paper_1409_4441_b200" not in gen
