"""CPU-side checks of the C-ABI boundary: the library builds, loads, exports every symbol declared in
include/helios_rt.h, and its host-side validation returns the documented error codes without a GPU
(no compute call is made here)."""
from __future__ import annotations

import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def lib():
    from paper_2203_02293_b200 import build, helios_rt
    build.build()
    return helios_rt.load_library()


def _declared(*headers):
    out = set()
    for h in headers:
        hdr = (ROOT / "include" / h).read_text()
        hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
        out |= set(re.findall(r"\b(helios_rt_[a-zA-Z_0-9]+)\s*\(", hdr))
    return out


def test_exports_every_declared_symbol(lib):
    """libhelios_rt.so exports what helios_rt.h and helios_rt_debug.h declare; libhelios_rt_selftest.so what
    helios_rt_selftest.h declares; and the product library carries none of the test hooks."""
    from paper_2203_02293_b200 import helios_rt
    declared = _declared("helios_rt.h", "helios_rt_debug.h")
    assert declared == set(helios_rt.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    st = helios_rt.load_selftest_library()
    declared_st = _declared("helios_rt_selftest.h")
    assert declared_st == set(helios_rt.SELFTEST_EXPORTS)
    for name in declared_st:
        assert getattr(st, name) is not None
        assert not hasattr(lib, name), f"{name} must not be exported by the product library"


def test_product_library_ignores_the_environment():
    """No getenv in the product sources: a stray variable must not change the kernel that runs."""
    for src in (ROOT / "paper_2203_02293_b200" / "csrc").glob("helios_rt*.cu*"):
        assert "getenv" not in src.read_text(), src
    assert "getenv" not in (ROOT / "paper_2203_02293_b200" / "csrc" / "helios_post.cu").read_text()


def test_strerror(lib):
    assert lib.helios_rt_strerror(0) == b"success"
    assert b"invalid" in lib.helios_rt_strerror(-6)     # HELIOS_RT_ESTUCK
    for code in (-1, -2, -3, -4, -5, -6):
        assert len(lib.helios_rt_strerror(code)) > 5
    assert b"unknown" in lib.helios_rt_strerror(-77)


def test_noalloc_phase_curve_size_limit_is_checked_on_the_host(lib):
    """helios_rt_phase_curve_noalloc refuses a problem whose scratch exceeds the built-in 8 MiB array with ETOOBIG (-5)
    before it touches the device, so the limit can be checked here without a GPU; malformed sizes stay EINVAL."""
    from paper_2203_02293_b200 import helios_rt
    assert helios_rt.PHASE_CURVE_NOALLOC_MAX_BYTES == 8388608
    assert "8388608" in (ROOT / "include" / "helios_rt.h").read_text()
    call = lambda n, nb, na: lib.helios_rt_phase_curve_noalloc(n, nb, na, None, None, None, None, None, None, 0.0, 0.0,
                                                               None, None, None)
    assert call(2562, 781, 64) == -5 and call(10242, 3256, 64) == -5
    assert call(-1, 30, 4) == -1 and call(16, 0, 4) == -1
    assert b"too large" in lib.helios_rt_strerror(-5)


def _cfg():
    from paper_2203_02293_b200 import workloads as W
    cfg, inp, meta = W.make(1)
    return cfg


def _create(cfg, max_columns=8):
    from paper_2203_02293_b200.helios_rt import HeliosRT, HeliosRTError
    try:
        HeliosRT(cfg, max_columns).close()
        return 0
    except HeliosRTError as e:
        return int(re.search(r"error (-?\d+)", str(e)).group(1))


def test_validation_errors_come_before_the_device_check(lib):
    """EINVAL (-1) for malformed configs even on a box without a GPU; a valid config on a GPU-less box
    fails loudly with ENODEV (-4) -- never a silent CPU path."""
    import torch
    good = _cfg()
    rc = _create(good)
    assert rc == (0 if torch.cuda.is_available() else -4)
    bad = dict(good, gauss_w=good["gauss_w"] * 1.01)
    assert _create(bad) == -1
    bad = dict(good, ktab_p=good["ktab_p"][::-1].copy())
    assert _create(bad) == -1
    bad = dict(good, bin_edges=np.concatenate([[0.0], good["bin_edges"][1:]]))
    assert _create(bad) == -1
    bad = dict(good, cloud_w0=np.full_like(good["cloud_w0"], 1.5))
    assert _create(bad) == -1
    bad = dict(good, cloud_g0=np.full_like(good["cloud_g0"], 1.0))
    assert _create(bad) == -1
    k = good["ktab"].copy(); k[0, 0, 0, 0] = 0.0
    assert _create(dict(good, ktab=k)) == -1
    k = good["ktab"].copy(); k[1, 2, 1, 0] = np.nan
    assert _create(dict(good, ktab=k)) == -1
    assert _create(dict(good, n_layers=0)) == -1
    assert _create(dict(good, n_layers=65)) == -1
    assert _create(dict(good, flags=64)) == -1
    assert _create(dict(good, gravity=0.0)) == -1
    assert _create(good, max_columns=0) == -1


def test_null_handles(lib):
    assert lib.helios_rt_destroy(None) == 0
    assert lib.helios_rt_create(None, None) == -1
    h = C.c_void_p()
    assert lib.helios_rt_create(None, C.byref(h)) == -1 and not h
    assert lib.helios_rt_launch_info(None, None) == -1
    assert lib.helios_rt_last_cuda_error(None) == b""


def test_kernel_build_is_reproducible(tmp_path):
    """Two compilations of the headline class with build.py's flags give the same SASS, instruction for instruction
    (with -split-compile other than 1 they do not, and the step time moves by 3 %)."""
    import subprocess
    from paper_2203_02293_b200 import build as B
    src = B.CSRC / "helios_rt_k_iso.cu"
    assert "-split-compile" in B.NVCC_FLAGS and B.NVCC_FLAGS[B.NVCC_FLAGS.index("-split-compile") + 1] == "1"

    def sass(tag):
        obj = tmp_path / f"iso_{tag}.o"
        subprocess.run([B.nvcc(), *B.NVCC_FLAGS, "-c", "-o", str(obj), str(src)], check=True, capture_output=True)
        out = subprocess.run(["cuobjdump", "-sass", str(obj)], check=True, capture_output=True, text=True).stdout
        return [ln.split("*/", 1)[1].split("/*")[0].strip() for ln in out.splitlines() if ln.lstrip().startswith("/*") and "*/" in ln and ";" in ln]

    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=2) as ex:      # side by side, as build.py compiles its translation units
        a, b = ex.map(sass, ("a", "b"))
    assert len(a) > 10000 and a == b
