"""The C-ABI library builds for sm_100a, loads without a GPU, and exports every symbol include/odyssey.h
declares.  No compute calls here (they need a device); argument validation that happens before any
CUDA call is exercised because it is pure host logic."""
import ctypes as C
import os
import re

import pytest

import paper_1601_02063_b200 as ody
from paper_1601_02063_b200 import binding as B
import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "odyssey.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(odyssey_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_all_exported():
    L = ody.load_library()
    declared = _declared_symbols()
    assert len(declared) >= 11
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/odyssey.h but not exported"
    assert set(declared) == set(ody.EXPORTED_SYMBOLS)


def test_struct_layout_matches_header_sizes():
    # 8 doubles + 2 int32 + double + 2 int32 + 3 doubles + 2 int32 = 15*8 = 120 bytes; model: 2 int32 + 16 doubles
    assert C.sizeof(B.Scene) == 120
    assert C.sizeof(B.Model) == 8 + 16 * 8 + 8 + 3 * 8 + 8 + 8


@pytest.mark.parametrize("patch, msg", [
    (dict(a=1.0), "spin"), (dict(nx=0), "nx"), (dict(nx=32769, ny=32768), "2^30"), (dict(rtol=0.0), "rtol"), (dict(tableau=7), "tableau"),
    (dict(x_max=-10.0), "extent"), (dict(max_attempts=0), "max_attempts"),
    (dict(x_min=-2000.0, x_max=2000.0), "r_esc"), (dict(r_obs=50.0, r_esc=55.0, y_min=-300.0, y_max=300.0), "r_esc"),
])
def test_invalid_scene_is_rejected_before_any_cuda_call(patch, msg):
    L = ody.load_library()
    sc = dict(W.C0()["scene"]); sc.update(patch)
    rc = L.odyssey_trace_geodesics(C.byref(B._struct(B.Scene, sc)), None, None, None, None, None, None, None, None)
    assert rc == -1
    assert msg in ody.last_error()


def test_invalid_model_and_frequencies_are_rejected():
    L = ody.load_library()
    w = W.C3(n=8)
    sc, mo = B._struct(B.Scene, w["scene"]), B._struct(B.Model, w["model"])
    nu = (C.c_double * 40)(*([1e9] * 40))
    assert L.odyssey_render_spectrum(C.byref(sc), C.byref(mo), nu, 33, None, None, None, None, None) == -1
    assert L.odyssey_render_spectrum(C.byref(sc), C.byref(mo), nu, 0, None, None, None, None, None) == -1
    nu[3] = -1.0
    assert L.odyssey_render_spectrum(C.byref(sc), C.byref(mo), nu, 8, None, None, None, None, None) == -1
    bad = dict(w["model"]); bad["kind"] = 9
    assert L.odyssey_render_image(C.byref(sc), C.byref(B._struct(B.Model, bad)), C.c_double(1e9),
                                  None, None, None, None, None, None, None, None) == -1
    rk = B._struct(B.Model, dict(w["model"], rt_scheme=W.RT_RK_COMPONENTS))
    assert L.odyssey_render_spectrum(C.byref(sc), C.byref(rk), nu, 4, None, None, None, None, None) == -1
    assert "rt_scheme" in ody.last_error()
    bad_rt = B._struct(B.Model, dict(w["model"], rt_scheme=5))
    assert L.odyssey_render_image(C.byref(sc), C.byref(bad_rt), C.c_double(1e9),
                                  None, None, None, None, None, None, None, None) == -1
    mixed_rk = B._struct(B.Model, dict(w["model"], rt_scheme=W.RT_RK_COMPONENTS)); mixed_rk.precision = 1
    assert L.odyssey_render_image(C.byref(sc), C.byref(mixed_rk), C.c_double(1e9),
                                  None, None, None, None, None, None, None, None) == -1
    mixed = B._struct(B.Model, w["model"]); mixed.precision = 1
    assert L.odyssey_render_spectrum(C.byref(sc), C.byref(mixed), nu, 4, None, None, None, None, None) == -1
    assert "precision" in ody.last_error()
    capped = B._struct(B.Model, W.model_riaf(dtau_max=0.1))
    assert L.odyssey_render_spectrum(C.byref(sc), C.byref(capped), nu, 4, None, None, None, None, None) == -1
    assert "dtau_max" in ody.last_error()
    capped_rk = B._struct(B.Model, W.model_riaf(dtau_max=0.1, rt_scheme=W.RT_RK_COMPONENTS))
    assert L.odyssey_render_image(C.byref(sc), C.byref(capped_rk), C.c_double(1e9),
                                  None, None, None, None, None, None, None, None) == -1
    assert "dtau_max" in ody.last_error()
    spot = B._struct(B.Model, W.model_hot_spot())
    assert L.odyssey_render_image(C.byref(sc), C.byref(spot), C.c_double(1e9),
                                  None, None, None, None, None, None, None, None) == -1
    assert "odyssey_render_hotspot" in ody.last_error()
    tt = (C.c_double * 40)(*([0.0] * 40))
    assert L.odyssey_render_hotspot(C.byref(sc), C.byref(spot), tt, 33, *([None] * 10)) == -1
    assert L.odyssey_render_hotspot(C.byref(sc), C.byref(mo), tt, 4, *([None] * 10)) == -1      # RIAF model in hot-spot mode
    bad_spot = B._struct(B.Model, W.model_hot_spot(r_spot=0.0))
    assert L.odyssey_render_hotspot(C.byref(sc), C.byref(bad_spot), tt, 4, *([None] * 10)) == -1
    nt_bad = B._struct(B.Model, W.model_nt_disk(mbh_msun=0.0))
    assert L.odyssey_render_spectrum(C.byref(sc), C.byref(nt_bad), nu, 4, None, None, None, None, None) == -1
    assert "Novikov-Thorne" in ody.last_error()
    nt = B._struct(B.Model, W.model_nt_disk())
    assert L.odyssey_render_spectrum(C.byref(sc), C.byref(nt), nu, 33, None, None, None, None, None) == -1
    assert L.odyssey_render_image(C.byref(sc), C.byref(nt), C.c_double(0.0), None, None, None, None, None, None, None, None) == -1
    thin = B._struct(B.Model, W.C1()["model"])
    assert L.odyssey_render_spectrum(C.byref(sc), C.byref(thin), nu, 4, None, None, None, None, None) == -1
    assert L.odyssey_render_image(None, None, C.c_double(0.0), None, None, None, None, None, None, None, None) == -1


def test_product_path_fails_loudly_without_a_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(ody.OdysseyError):
        ody.trace_geodesics(W.C0()["scene"])
    # the host-buffer entry point reaches the CUDA runtime and must report an error code, not fall back
    with pytest.raises(ody.OdysseyError):
        ody.trace_geodesics_host(W.C0(n=4)["scene"])


def test_product_sources_do_not_reference_the_oracle():
    pkg = os.path.join(ROOT, "paper_1601_02063_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                for pat in (r"^\s*(from|import)\s+oracle", r"liboracle", r"#include\s+\"[^\"]*oracle", r"oracle[/.]binding"):
                    assert not re.search(pat, text, flags=re.M), f"{f} reaches into oracle/ ({pat})"
