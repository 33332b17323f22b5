"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol
include/mps_b200.h declares, validates arguments, and fails loudly without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    import __graft_entry__ as ge
    ge.build()
    from paper_2105_01677_b200 import binding
    return binding


def _declared():
    src = open(os.path.join(ROOT, "include", "mps_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(mps_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(B):
    names = _declared()
    assert len(names) >= 25
    for nm in names:
        assert hasattr(B.lib, nm), nm
    assert sorted(B.SYMBOLS) == names
    assert "sm_100a" in B.version()


def test_struct_layout_matches_header(B):
    # 16 int32 then 28 doubles, no padding
    assert C.sizeof(B.MpsParams) == 16 * 4 + 29 * 8
    assert B.MpsParams.l0.offset == 64
    assert C.sizeof(B.MpsStats) == 104
    # field ids in the binding equal the header's enum
    src = open(os.path.join(ROOT, "include", "mps_b200.h")).read()
    for name, fid in B.FIELDS.items():
        tag = ("MPS_F_" if fid < 32 else "MPS_I_") + name.upper()
        m = re.search(tag + r"\s*=\s*(\d+)", src)
        assert m and int(m.group(1)) == fid, tag
    for i, t in enumerate(B.TIMERS):
        m = re.search("MPS_T_" + t.upper() + r"\s*=\s*(\d+)", src)
        assert m and int(m.group(1)) == i, t


def _init_rc(B, **over):
    from paper_2105_01677_b200 import scenes
    p = scenes.default_params(0.01)
    p["domain_max"] = (1.0, 1.0, 1.0)
    p.update(over)
    prm = B.make_params(p)
    h = C.c_void_p()
    buf = np.zeros(8)
    ib = np.zeros(8, np.int32)
    d = buf.ctypes.data_as(C.c_void_p)
    i = ib.ctypes.data_as(C.c_void_p)
    n = over.pop("_n", 8)
    rc = B.lib.mps_init(C.byref(h), C.byref(prm), n, d, d, d, d, d, d, i, i, None)
    return rc, B.lib.mps_last_error(None).decode(), h


@pytest.mark.parametrize("over", [
    dict(dim=4), dict(dim=2, ppe_laplacian=1), dict(ppe_source=3), dict(kernel=2), dict(kernel=1, ppe_source=1), dict(rebin_every=0), dict(_n=0), dict(_n=-5), dict(l0=0.0), dict(dt=-1.0), dict(re_grad=0.5), dict(re_lap=0.001),
    dict(cell_div=0), dict(cell_div=4), dict(key_mode=2), dict(ppe_operator=2), dict(cg_warm_start=-1), dict(n_phases=3), dict(max_neighbours=0),
    dict(grad_variant=4), dict(rho=(0.0, 1.0)), dict(cg_rtol=0.0), dict(domain_max=(0.0, 1.0, 1.0)),
])
def test_bad_parameters_are_rejected(B, over):
    rc, msg, h = _init_rc(B, **over)
    assert rc == B.MPS_ERR_ARG and msg and not h.value


def test_null_pointers_are_rejected(B):
    from paper_2105_01677_b200 import scenes
    p = scenes.default_params(0.01)
    p["domain_max"] = (1.0, 1.0, 1.0)
    prm = B.make_params(p)
    h = C.c_void_p()
    assert B.lib.mps_init(C.byref(h), C.byref(prm), 8, *([None] * 8), None) == B.MPS_ERR_ARG
    assert B.lib.mps_init(None, C.byref(prm), 8, *([None] * 8), None) == B.MPS_ERR_ARG
    for fn in ("mps_bin", "mps_density", "mps_viscosity", "mps_gradient", "mps_sync", "mps_destroy"):
        assert getattr(B.lib, fn)(None) == B.MPS_ERR_ARG
    assert B.lib.mps_step(None, 1, 0) == B.MPS_ERR_ARG


def test_no_gpu_means_loud_failure_not_fallback(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    rc, msg, h = _init_rc(B)
    assert rc == B.MPS_ERR_CUDA and "no CPU fallback" in msg and not h.value
    from paper_2105_01677_b200 import scenes
    with pytest.raises(RuntimeError):
        B.Mps(scenes.small_tank())


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2105_01677_b200")
    banned = ("import oracle", "from oracle", "liborc", "mps_oracle", "orc_")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                for b in banned:
                    assert b not in txt, (f, b)
    txt = open(os.path.join(ROOT, "oracle", "mps_oracle.py")).read() + open(
        os.path.join(ROOT, "oracle", "mps_oracle.cpp")).read()
    for b in ("binding", "libmps_b200", "mps_b200.h", "csrc/"):
        assert b not in txt.replace("paper_2105_01677_b200/csrc", ""), b
