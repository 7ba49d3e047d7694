"""CPU-side checks of the C-ABI library: it builds, loads without a GPU, exports every symbol
include/qsgw.h declares, validates descriptors on the host, and fails loudly (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2506_03477_b200 import build, binding
    build.build()
    return binding.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "qsgw.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(qsgw_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_exported(L):
    names = declared_symbols()
    for must in ("qsgw_zmel_build", "qsgw_chi0_accumulate", "qsgw_chi0_finalize", "qsgw_create",
                 "qsgw_destroy", "qsgw_chi0_run_host"):
        assert must in names
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/qsgw.h but not exported"


def test_version_and_null_handling(L):
    assert b"sm_100a" in L.qsgw_version()
    assert L.qsgw_sync(None) == 1
    assert L.qsgw_reset(None) == 1
    assert L.qsgw_chi0_finalize(None, None) == 1
    L.qsgw_destroy(None)        # no-op
    assert L.qsgw_kernel_launches(None) == 0


def _desc(**kw):
    from paper_2506_03477_b200.binding import _make_desc
    base = dict(orb_per_site=[2, 3], pb_per_site=[3, 2], omega=[0.0, 1.0], n_k=2, max_n_o=2,
                max_n_u=3, precision=0, occ_tol=1e-12, workspace_bytes=0)
    base.update(kw)
    return _make_desc(**base)


@pytest.mark.parametrize("kw,code", [
    (dict(omega=[0.0, 0.0]), 2), (dict(omega=[-1.0, 1.0]), 2), (dict(omega=[1.0, 0.5]), 2),
    (dict(orb_per_site=[2, 0]), 2), (dict(pb_per_site=[0, 2]), 2), (dict(n_k=0), 2),
    (dict(max_n_o=0), 2), (dict(precision=7), 1), (dict(omega=[float("nan")]), 2),
])
def test_create_validates_on_host(L, kw, code):
    d = _desc(**kw)
    h = C.c_void_p()
    rc = L.qsgw_create(C.byref(d), None, C.byref(h))
    assert rc == code and not h.value
    assert len(L.qsgw_last_create_error()) > 0


def test_create_null_args(L):
    h = C.c_void_p()
    assert L.qsgw_create(None, None, C.byref(h)) == 1
    d = _desc()
    assert L.qsgw_create(C.byref(d), None, None) == 1


def test_no_cpu_fallback_without_gpu(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import numpy as np
    import paper_2506_03477_b200 as q
    with pytest.raises(q.QsgwError) as ei:
        q.Chi0Context([2, 3], [3, 2], [0.0, 1.0], 2, 2, 3)
    assert ei.value.code in (5, 6)
    with pytest.raises(q.QsgwError):
        z = np.zeros
        q.chi0_run_host([1], [1], [0.0], z(1, complex), z((1, 1, 1), complex), z((1, 1, 1), complex),
                        z((1, 1)), z((1, 1)), z((1, 1)), z((1, 1)), 1, 1)


def test_product_does_not_import_oracle():
    """The product package must not reference oracle/ (parity would be void)."""
    pkg = os.path.join(ROOT, "paper_2506_03477_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2506_03477_b200" not in txt.replace("(paper_2506_03477_b200)", ""), f
