"""No-GPU checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every
symbol include/ds.h declares, and its host-side validation works without a device."""
import ctypes
import os
import re

import pytest

from paper_1004_1932_b200 import ds

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols(header="ds.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ds_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = ds.lib()
    declared = _declared_symbols()
    assert len(declared) >= 12
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/ds.h but not exported by libds.so"
    assert sorted(ds.SYMBOLS) == declared
    # the development hooks live in their own header (include/ds_dev.h), not in the product boundary
    dev = _declared_symbols("ds_dev.h")
    for name in dev:
        assert hasattr(L, name), f"{name} declared in include/ds_dev.h but not exported by libds.so"
    assert sorted(ds.DEV_SYMBOLS) == dev
    assert not set(dev) & set(declared)


def test_version_and_strerror():
    assert "sm_100a" in ds.version()
    L = ds.lib()
    assert L.ds_strerror(0) == b"ok"
    for code in range(-6, 0):
        assert L.ds_strerror(code) not in (b"ok", b"unknown error")
    assert L.ds_strerror(-99) == b"unknown error"


def test_null_and_invalid_arguments_are_rejected_before_any_device_work():
    L = ds.lib()
    h = ctypes.c_void_p()
    assert L.ds_create(None, ctypes.byref(h)) == ds.ERR_NULL
    good = dict(n_dumbbells=4, n_batch=1, precision=ds.F64, tensor=ds.RPY, integrator=ds.HEUN, device=0,
                a=1.0, eta=1.0, ell=10.0, lam=2.0, omega=6.28, k0=1000.0, dt=1e-3, kT=0.0)
    bad = [dict(n_dumbbells=0), dict(n_batch=0), dict(precision=7), dict(tensor=-1), dict(integrator=2),
           dict(a=0.0), dict(eta=-1.0), dict(k0=0.0), dict(dt=float("nan")), dict(ell=4.0),   # ell <= 2a + lam
           dict(lam=8.0), dict(lam=-8.0), dict(omega=-1.0), dict(dt=float("inf")), dict(kT=-1.0), dict(kT=float("nan"))]
    for change in bad:
        kw = dict(good, **change)
        p = ds.Params(kw["n_dumbbells"], kw["n_batch"], kw["precision"], kw["tensor"], kw["integrator"], kw["device"],
                      kw["a"], kw["eta"], kw["ell"], kw["lam"], kw["omega"], kw["k0"], kw["dt"], None, kw["kT"], 0)
        assert L.ds_create(ctypes.byref(p), ctypes.byref(h)) == ds.ERR_INVALID_PARAM, change
        assert not h.value
    for fn, args in [(L.ds_set_state, (None, None, None, 0.0)), (L.ds_get_state, (None, None, None)),
                     (L.ds_forces, (None, None)), (L.ds_mobility_apply, (None, None, None, None, 4)),
                     (L.ds_step, (None, 1)), (L.ds_batch_step, (None, 1)), (L.ds_velocity, (None, None)),
                     (L.ds_set_tuning, (None, 0)), (L.ds_set_stream, (None, None)),
                     (L.ds_dumbbell_coords, (None, None, None)), (L.ds_msd_set_reference, (None,)), (L.ds_msd, (None, None)),
                     (L.ds_avg_rhs, (None, None, None, None, None, None, 4)), (L.ds_avg_step, (None, None, None, None, 4, 0.5, 1))]:
        assert fn(*args) == ds.ERR_NULL
    assert L.ds_destroy(None) == ds.OK
    assert L.ds_launch_count(None) == 0


def test_no_cpu_fallback_without_device():
    """On a box without an sm_100 device the product path fails loudly (no fallback)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("device present")
    with pytest.raises(ds.DsError) as e:
        ds.System(4)
    assert e.value.code == ds.ERR_NO_DEVICE


def test_product_and_oracle_share_no_code():
    """The product package never imports / includes anything under oracle/, and vice versa."""
    imp = re.compile(r"^\s*(from|import)\s+([\w\.]+)", re.M)
    inc = re.compile(r"^\s*#\s*include\s+[\"<]([^\">]+)[\">]", re.M)
    pkg = os.path.join(ROOT, "paper_1004_1932_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            txt = open(os.path.join(dirpath, f), errors="ignore").read() if f.endswith((".py", ".cu", ".cuh", ".h")) else ""
            assert not any(m.group(2).split(".")[0] == "oracle" for m in imp.finditer(txt)), f
            assert not any("oracle" in m.group(1) for m in inc.finditer(txt)), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not any(m.group(2).split(".")[0] == "paper_1004_1932_b200" for m in imp.finditer(txt)), f
            assert not any(("ds.h" in m.group(1)) or ("csrc" in m.group(1)) or ("cuh" in m.group(1)) for m in inc.finditer(txt)), f
