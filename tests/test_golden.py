"""Fixtures under tests/golden/: (1) values PRINTED in the paper, each with its citation, checked against the
oracle; (2) oracle outputs written by tests/golden/make_oracle_golden.py (from oracle/ only), as a
regression guard on the oracle's arithmetic.  The GPU test compares the CUDA path with the same stored
oracle values — the expected values never come from the CUDA path."""
import json
import math
import os

import numpy as np
import pytest

import workloads as W
from oracle import binding as O

HERE = os.path.dirname(os.path.abspath(__file__))
PAPER = json.load(open(os.path.join(HERE, "golden", "paper_values.json")))
ORACLE = json.load(open(os.path.join(HERE, "golden", "oracle_regression.json")))


def _edge(scene, angle, lo=3.0, hi=8.0):
    """Bisect the capture/escape boundary along the image-plane ray at `angle`."""
    cs, sn = math.cos(angle), math.sin(angle)
    for _ in range(46):
        mid = 0.5 * (lo + hi)
        f = O.trace_points(scene, W.model_none(), [], [mid * cs], [mid * sn])["flag"][0]
        lo, hi = (mid, hi) if f == W.FLAG_CAPTURED else (lo, mid)
    return 0.5 * (lo + hi)


def test_paper_shadow_radius_squared_is_27():
    v = PAPER["schwarzschild_shadow_alpha2_plus_beta2"]["value"]
    sc = W.scene(0.0, 90.0, 8, 10.0, r_obs=PAPER["observer_distance"]["r_obs"], rtol=1e-11)
    for ang in (0.0, 1.0, 2.5):
        b = _edge(sc, ang)
        assert b * b == pytest.approx(v, rel=2e-7)          # finite-distance shift at r_obs = 1000 is -5e-8 relative


def test_paper_eq38_as_printed():
    c = PAPER["mahadevan_fit_eq38"]
    for x in (0.05, 1.0, 7.0, 300.0):
        printed = c["prefactor"] / x ** (1 / 6) * (1 + c["c_quarter"] / x ** 0.25 + c["c_half"] / x ** 0.5) \
            * math.exp(-c["exp_coeff"] * x ** (1 / 3))
        assert O.mahadevan_M(x) == pytest.approx(printed, rel=1e-14)


def test_paper_fig5_thin_disk_orientation_and_contour_range():
    f = PAPER["thin_disk_fig5"]
    sc = W.scene(f["spin"], math.degrees(math.acos(f["cos_theta_obs"])), 96, 52.0)
    d = O.render_image(sc, W.model_thin_disk(r_in=0.0, r_out=f["r_out"]))
    g = d["aux0"].reshape(96, 96); r_e = d["aux1"].reshape(96, 96)
    hit = g > 0
    mid = 48
    left, right = g[mid, :48], g[mid, 48:]
    assert left[left > 0].max() > 1.0 > right[right > 0].max()          # approaching (left) side is blue shifted
    # the printed contour levels bracket what the direct image contains
    assert g[hit].min() < f["gamma_contours_min"] + 0.05 and g[hit].max() > f["gamma_contours_max"] - 0.05
    assert f["gamma_contours_min"] - 0.1 < g[hit].min() and g[hit].max() < f["gamma_contours_max"] + 0.1
    assert r_e[hit].min() >= 6.0 - 1e-9 and r_e[hit].max() <= f["r_contours_max"] + 1e-9
    assert r_e[hit].min() < f["r_contours_min"] + 0.5


def test_paper_table1_arithmetic_quoted_in_baseline_md():
    """BASELINE.md's reading of Table 1: the printed last column divides by the photon count twice;
    run time / total steps at 1024^2 is 16.3 ns with ~1505 steps per photon."""
    rows = PAPER["table1"]["rows"]
    for n, ms, steps, printed in rows:
        assert ms * 1e6 / steps / (n * n) == pytest.approx(printed, rel=2e-2, abs=6e-7)
    n, ms, steps, _ = rows[-1]
    assert ms * 1e6 / steps == pytest.approx(16.31, abs=0.01)
    assert steps / (n * n) == pytest.approx(1505, abs=1)


def _cmp(actual, stored, rel):
    a, s = np.asarray(actual, dtype=float).ravel(), np.asarray(stored, dtype=float).ravel()
    assert a.shape == s.shape
    assert np.all(np.abs(a - s) <= rel * np.maximum(np.abs(s), 1e-300))


def test_oracle_regression_values():
    g = O.trace_geodesics(W.C0(n=8)["scene"])
    ref = ORACLE["C0_8x8"]
    assert g["flag"].tolist() == ref["flag"] and g["n_attempt"].tolist() == ref["n_attempt"]
    for k in ("r", "th", "ph"):
        _cmp(g[k], ref[k], 1e-12)
    _cmp(g["t"], ref["t"], 1e-12)
    hs = O.render_hotspot(W.scene(0.5, 60.0, 10, 9.0), W.model_hot_spot(r_spot=1.0, nbins=8), ORACLE["hotspot_10x10"]["t_obs"])
    _cmp(hs["lightcurve"], ORACLE["hotspot_10x10"]["lightcurve"], 1e-10)
    _cmp(hs["t_e"], ORACLE["hotspot_10x10"]["t_e"], 1e-12)
    w = W.C1(n=8)
    d = O.render_image(w["scene"], w["model"])
    assert d["flag"].tolist() == ORACLE["C1_8x8"]["flag"]
    _cmp(d["aux0"], ORACLE["C1_8x8"]["g"], 1e-12)
    w = W.C2(n=8)
    for scheme in (W.RT_PER_STEP, W.RT_RK_COMPONENTS):
        r = O.render_image(w["scene"], dict(w["model"], rt_scheme=scheme), w["nu"][0])
        _cmp(r["image"], ORACLE[f"C2_8x8_rt_scheme{scheme}"]["image"], 1e-10)
    w = W.C3(n=4, nf=4)
    s = O.render_spectrum(w["scene"], w["model"], w["nu"])
    _cmp(s["nuLnu"], ORACLE["C3_4x4_nf4"]["nuLnu"], 1e-10)
    nt = ORACLE["nt_disk"]
    _cmp([O.page_thorne_f(nt["a"], r) for r in nt["r"]], nt["f"], 1e-12)
    _cmp([O.nt_temperature(W.model_nt_disk(), nt["a"], r) for r in nt["r"]], nt["T_eff"], 1e-12)
    sp = O.render_spectrum(W.scene(0.999, 85.0, 9, 25.0), W.model_nt_disk(), nt["nu"])
    assert sp["flag"].tolist() == nt["flag"]
    _cmp(sp["nuLnu"], nt["nuLnu"], 1e-9)
    r = O.render_image(W.C2(n=8)["scene"], W.model_riaf(dtau_max=0.1), 1.0e10)
    assert r["n_attempt"].tolist() == ORACLE["C2_8x8_10GHz_dtau0.1"]["n_attempt"]
    _cmp(r["image"], ORACLE["C2_8x8_10GHz_dtau0.1"]["image"], 1e-10)


@pytest.mark.gpu
def test_cuda_path_against_stored_oracle_values(ody):
    import torch
    out = ody.trace_geodesics(W.C0(n=8)["scene"]); torch.cuda.synchronize()
    ref = ORACLE["C0_8x8"]
    assert out["flag"].cpu().numpy().ravel().tolist() == ref["flag"]
    _cmp(out["theta"].cpu().numpy(), ref["th"], 1e-8)
    _cmp(out["phi"].cpu().numpy(), ref["ph"], 1e-8)
    hs = ody.render_hotspot(W.scene(0.5, 60.0, 10, 9.0), W.model_hot_spot(r_spot=1.0, nbins=8), ORACLE["hotspot_10x10"]["t_obs"])
    torch.cuda.synchronize()
    _cmp(hs["lightcurve"].cpu().numpy(), ORACLE["hotspot_10x10"]["lightcurve"], 1e-6)
    tt = ody.trace_geodesics(W.C0(n=8)["scene"], with_time=True); torch.cuda.synchronize()
    _cmp(tt["t"].cpu().numpy(), ref["t"], 1e-8)
    w = W.C2(n=8)
    for scheme in (W.RT_PER_STEP, W.RT_RK_COMPONENTS):
        r = ody.render_image(w["scene"], dict(w["model"], rt_scheme=scheme), w["nu"][0]); torch.cuda.synchronize()
        img, st = r["image"].cpu().numpy().ravel(), np.asarray(ORACLE[f"C2_8x8_rt_scheme{scheme}"]["image"])
        assert np.abs(img - st).sum() / st.sum() <= 1e-6
    w = W.C3(n=4, nf=4)
    s = ody.render_spectrum(w["scene"], w["model"], w["nu"]); torch.cuda.synchronize()
    _cmp(s["nuLnu"].cpu().numpy(), ORACLE["C3_4x4_nf4"]["nuLnu"], 1e-6)
    nt = ORACLE["nt_disk"]
    sp = ody.render_spectrum(W.scene(0.999, 85.0, 9, 25.0), W.model_nt_disk(), nt["nu"]); torch.cuda.synchronize()
    assert sp["flag"].cpu().numpy().ravel().tolist() == nt["flag"]
    _cmp(sp["nuLnu"].cpu().numpy(), nt["nuLnu"], 1e-6)
    r = ody.render_image(W.C2(n=8)["scene"], W.model_riaf(dtau_max=0.1), 1.0e10); torch.cuda.synchronize()
    img, st = r["image"].cpu().numpy().ravel(), np.asarray(ORACLE["C2_8x8_10GHz_dtau0.1"]["image"])
    assert np.abs(img - st).sum() / st.sum() <= 1e-6
