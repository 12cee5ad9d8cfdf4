"""GPU parity for the emission models: thin-disk line image (C1), RIAF GRRT image (C2), spectrum mode
(C3) and the throughput configuration (C4), against the CPU oracle.  Reduced-size cases compare every
pixel; the BASELINE.json sizes run in the launch configuration bench.py times and are compared on a
strided sub-grid of pixels that the oracle computes one by one."""
import numpy as np
import pytest

import workloads as W
from test_gpu_parity import _np, _sync, _check_image

pytestmark = pytest.mark.gpu


def _sub(a, idx):
    return a[np.asarray(idx[1]), np.asarray(idx[0])]


# ------------------------------------------------------------------------------------------------ C1
def _check_disk(gpu, ref, idx=None, check_hist=True):
    pick = (lambda a: a.ravel()) if idx is None else (lambda a: _sub(a, idx))
    assert np.array_equal(pick(gpu["flag"]), ref["flag"])
    hit = ref["flag"] == W.FLAG_DISK
    assert hit.any()
    g, r_e, img = pick(gpu["aux0"]), pick(gpu["aux1"]), pick(gpu["image"])
    assert np.max(np.abs(g[hit] - ref["aux0"][hit]) / ref["aux0"][hit]) <= 1e-8
    assert np.max(np.abs(r_e[hit] - ref["aux1"][hit]) / ref["aux1"][hit]) <= 1e-8
    assert np.all(g[~hit] == 0.0) and np.all(img[~hit] == 0.0) and np.all(r_e[~hit] == 0.0)
    _check_image(img, ref["image"], "thin-disk image")
    if check_hist and ref.get("hist") is not None:
        h, hr = gpu["hist"], ref["hist"]
        # bin membership can flip only for g within round-off of a bin edge: compare the cumulative profile
        assert abs(h.sum() - hr.sum()) <= 1e-9 * hr.sum()
        assert np.max(np.abs(np.cumsum(h) - np.cumsum(hr))) <= 1e-6 * hr.sum()
        assert np.count_nonzero(np.abs(h - hr) > 1e-9 * hr.max()) <= 2


def test_c1_thin_disk_reduced_every_pixel(ody, orc):
    w = W.C1(n=128)
    out = ody.render_image(w["scene"], w["model"]); _sync()
    gpu = {k: (_np(v) if v is not None else None) for k, v in out.items()}
    ref = orc.render_image(w["scene"], w["model"])
    _check_disk(gpu, ref)


def test_c1_thin_disk_full_size(ody, orc):
    w = W.C1()
    out = ody.render_image(w["scene"], w["model"]); _sync()
    gpu = {k: (_np(v) if v is not None else None) for k, v in out.items()}
    ref = orc.render_image(w["scene"], w["model"])          # 262 144 rays: seconds on the host cores
    _check_disk(gpu, ref)
    # Fig. 5 orientation: the approaching side (left, x < 0) is blue-shifted
    g = gpu["aux0"]
    mid = g.shape[0] // 2
    left, right = g[mid, : g.shape[1] // 2], g[mid, g.shape[1] // 2:]
    assert left[left > 0].max() > 1.0 > right[right > 0].max()


def test_thin_disk_schwarzschild_and_power_options(ody, orc):
    sc = W.scene(0.0, 75.52248781407008, 64, 12.0)          # cos(theta_obs) = 0.25
    mo = W.model_thin_disk(r_in=6.0, r_out=30.0, emis_index=2.0, nbins=50, g_lo=0.3, g_hi=1.5, g_power=4.0)
    out = ody.render_image(sc, mo); _sync()
    gpu = {k: (_np(v) if v is not None else None) for k, v in out.items()}
    ref = orc.render_image(sc, mo)
    _check_disk(gpu, ref)


# ------------------------------------------------------------------------------------------------ C2
def test_c2_riaf_reduced_every_pixel(ody, orc):
    w = W.C2(n=96)
    out = ody.render_image(w["scene"], w["model"], w["nu"][0]); _sync()
    ref = orc.render_image(w["scene"], w["model"], w["nu"][0])
    assert np.array_equal(_np(out["flag"]).ravel(), ref["flag"])
    _check_image(_np(out["image"]).ravel(), ref["image"], "RIAF 230 GHz image")
    tau, tr = _np(out["aux0"]).ravel(), ref["aux0"]
    assert np.max(np.abs(tau - tr) / np.maximum(tr, 1e-6 * tr.max())) <= 1e-4
    assert np.mean(_np(out["n_attempt"]).ravel() == ref["n_attempt"]) >= 0.995


@pytest.mark.parametrize("nu", [1.0e9, 2.0e10, 1.0e12, 1.0e14])
def test_riaf_other_frequencies_including_optically_thick(ody, orc, nu):
    w = W.C2(n=40)
    out = ody.render_image(w["scene"], w["model"], nu); _sync()
    ref = orc.render_image(w["scene"], w["model"], nu)
    assert np.array_equal(_np(out["flag"]).ravel(), ref["flag"])
    _check_image(_np(out["image"]).ravel(), ref["image"], f"RIAF image at {nu:g} Hz")
    if nu <= 2.0e10:
        assert (ref["flag"] == W.FLAG_OPAQUE).any()         # the tau > 30 cutoff is exercised


def test_c2_full_size_sampled(ody, orc):
    w = W.C2()
    out = ody.render_image(w["scene"], w["model"], w["nu"][0]); _sync()
    idx = W.subgrid_indices(w["scene"], 64)
    ref = orc.render_image(w["scene"], w["model"], w["nu"][0], idx=idx)
    assert np.array_equal(_sub(_np(out["flag"]), idx), ref["flag"])
    _check_image(_sub(_np(out["image"]), idx), ref["image"], "C2 sampled")
    img = _np(out["image"])
    assert np.isfinite(img).all() and (img >= 0).all()


# ------------------------------------------------------------------------------------------------ C3
def test_c3_spectrum_reduced_every_pixel(ody, orc):
    w = W.C3(n=48)
    out = ody.render_spectrum(w["scene"], w["model"], w["nu"]); _sync()
    ref = orc.render_spectrum(w["scene"], w["model"], w["nu"])
    imgs = _np(out["images"]).reshape(len(w["nu"]), -1)
    assert np.array_equal(_np(out["flag"]).ravel(), ref["flag"])
    for k, nu in enumerate(w["nu"]):
        if np.abs(ref["images"][k]).max() == 0.0:
            assert np.all(imgs[k] == 0.0)
            continue
        _check_image(imgs[k], ref["images"][k], f"spectrum image k={k} ({nu:.3g} Hz)")
    sed, sr = _np(out["nuLnu"]), ref["nuLnu"]
    assert np.max(np.abs(sed - sr) / np.maximum(sr, 1e-12 * sr.max())) <= 1e-6


def test_spectrum_matches_single_frequency_calls(ody):
    """Frequency k of a spectrum launch = the single-frequency kernel at nu_k, except where another
    frequency kept the ray alive past that kernel's own tau cutoff (frozen: identical) — so identical."""
    w = W.C3(n=32, nf=6)
    spec = ody.render_spectrum(w["scene"], w["model"], w["nu"]); _sync()
    for k, nu in enumerate(w["nu"]):
        one = ody.render_image(w["scene"], w["model"], nu); _sync()
        a, b = _np(spec["images"][k]), _np(one["image"])
        # The two kernels form x_M^(1/12) in a different order (spectrum: (x_M/nu)^(1/12) * nu^(1/12), image: one
        # exponential), and eq. (38)'s exponent -1.8899 x_M^(1/3) reaches -550 at 1e15 Hz (pixel values ~1e-240):
        # a rounding difference of one ulp in x_M^(1/12) is 4 * 550 ulp = 2.4e-13 in such a pixel, per point of
        # the ray.  1e-12 holds wherever the value is above 1e-100; the deep-underflow pixels get 1e-11.
        big = np.abs(b) >= 1e-100
        assert np.allclose(a[big], b[big], rtol=1e-12, atol=0.0)
        assert np.allclose(a[~big], b[~big], rtol=1e-11, atol=0.0)


def test_c3_full_size_sampled(ody, orc):
    w = W.C3()
    out = ody.render_spectrum(w["scene"], w["model"], w["nu"]); _sync()
    idx = W.subgrid_indices(w["scene"], 32)
    ref = orc.render_spectrum(w["scene"], w["model"], w["nu"], idx=idx)
    imgs = _np(out["images"])
    for k in range(len(w["nu"])):
        if np.abs(ref["images"][k]).max() == 0.0:
            continue
        _check_image(_sub(imgs[k], idx), ref["images"][k], f"C3 sampled k={k}")
    # SED = 4 pi nu r_g^2 dx dy sum(I): re-derive from the GPU's own images (property that holds at any size)
    sc = w["scene"]
    area = (sc["x_max"] - sc["x_min"]) / sc["nx"] * (sc["y_max"] - sc["y_min"]) / sc["ny"]
    rg = orc.rg_cm(w["model"]["mbh_msun"])
    sed = 4.0 * np.pi * np.asarray(w["nu"]) * rg * rg * area * imgs.reshape(len(w["nu"]), -1).sum(axis=1)
    assert np.allclose(_np(out["nuLnu"]), sed, rtol=1e-10)


# ------------------------------------------------------------------------------------------------ C4
@pytest.mark.parametrize("a", [0.0, 0.5, 0.9, 0.998])
def test_c4_sweep_spins_sampled_at_1024(ody, orc, a):
    w = W.C4(n=1024, a=a)
    out = ody.render_image(w["scene"], w["model"], w["nu"][0]); _sync()
    idx = W.subgrid_indices(w["scene"], 48)
    ref = orc.render_image(w["scene"], w["model"], w["nu"][0], idx=idx)
    assert np.array_equal(_sub(_np(out["flag"]), idx), ref["flag"])
    _check_image(_sub(_np(out["image"]), idx), ref["image"], f"C4 a={a}")


@pytest.mark.parametrize("a", [0.5, 0.998])
def test_c4_sweep_sampled_at_2048(ody, orc, a):
    w = W.C4(n=2048, a=a)
    out = ody.render_image(w["scene"], w["model"], w["nu"][0]); _sync()
    idx = W.subgrid_indices(w["scene"], 96)
    ref = orc.render_image(w["scene"], w["model"], w["nu"][0], idx=idx)
    assert np.array_equal(_sub(_np(out["flag"]), idx), ref["flag"])
    _check_image(_sub(_np(out["image"]), idx), ref["image"], f"C4 2048^2 a={a}")
    assert np.mean(_sub(_np(out["n_attempt"]), idx) == ref["n_attempt"]) >= 0.995
    img = _np(out["image"])
    assert np.all(np.isfinite(img)) and img.min() >= 0.0


def test_c4_full_size_sampled(ody, orc):
    """4096 x 4096, the exact launch bench.py times: a 128 x 128 grid over the whole frame plus every 8th pixel in both
    directions of the window |x| < 8, |y| < 7 that holds the shadow and the photon ring (81 920 pixels in all,
    each computed by the oracle), and the whole frame finite, non-negative, every pixel written."""
    w = W.C4()
    sc = w["scene"]
    out = ody.render_image(sc, w["model"], w["nu"][0]); _sync()
    ii, jj = W.subgrid_indices(sc, 128)
    n, half = sc["nx"], sc["x_max"]
    lo = lambda v: int((v + half) / (2 * half) * n)
    for j in range(lo(-7.0), lo(7.0), 8):
        for i in range(lo(-8.0), lo(8.0), 8):
            ii.append(i); jj.append(j)
    idx = (ii, jj)
    assert len(ii) >= 256 * 256
    ref = orc.render_image(sc, w["model"], w["nu"][0], idx=idx)
    assert np.array_equal(_sub(_np(out["flag"]), idx), ref["flag"])
    assert {W.FLAG_CAPTURED, W.FLAG_ESCAPED} <= set(np.unique(ref["flag"]))
    _check_image(_sub(_np(out["image"]), idx), ref["image"], "C4 4096^2 sampled")
    assert ref["n_attempt"].max() > 400                                  # the sample reaches the long, winding rays of the ring
    n_att = _np(out["n_attempt"])
    assert n_att.min() > 0 and n_att.max() < sc["max_attempts"]
    assert np.mean(_sub(n_att, idx) == ref["n_attempt"]) >= 0.995
    img = _np(out["image"])
    assert np.all(np.isfinite(img)) and img.min() >= 0.0
    fl = _np(out["flag"])
    assert fl.min() >= 0 and fl.max() <= W.FLAG_MAXSTEP


# ------------------------------------------------------------------------- transfer scheme E' (RK components)
@pytest.mark.parametrize("nu, tableau", [(230.0e9, W.TABLEAU_RKF45), (30.0e9, W.TABLEAU_RKF45), (230.0e9, W.TABLEAU_CASH_KARP)])
def test_rk_component_transfer_scheme_matches_the_oracle(ody, orc, nu, tableau):
    w = W.C2(n=64)
    sc = dict(w["scene"], tableau=tableau)
    mo = dict(w["model"], rt_scheme=W.RT_RK_COMPONENTS)
    out = ody.render_image(sc, mo, nu); _sync()
    ref = orc.render_image(sc, mo, nu)
    assert np.array_equal(_np(out["flag"]).ravel(), ref["flag"])
    _check_image(_np(out["image"]).ravel(), ref["image"], f"RK-component scheme at {nu:g} Hz")
    tau, tr = _np(out["aux0"]).ravel(), ref["aux0"]
    assert np.max(np.abs(tau - tr) / np.maximum(tr, 1e-6 * tr.max())) <= 1e-4
    # same geodesics, same steps as the default scheme
    base = ody.render_image(sc, w["model"], nu); _sync()
    opaque = (ref["flag"] == W.FLAG_OPAQUE) | (_np(base["flag"]).ravel() == W.FLAG_OPAQUE)
    assert np.array_equal(_np(out["n_attempt"]).ravel()[~opaque], _np(base["n_attempt"]).ravel()[~opaque])
    # and the two discretisations agree to their truncation error
    a, b = _np(out["image"]).ravel(), _np(base["image"]).ravel()
    assert np.abs(a - b).sum() / b.sum() < 5e-3


# ------------------------------------------------------- the two spectrum code paths and the overflow fallback
def test_spectrum_two_phase_overflow_fallback_matches_the_oracle(ody, orc):
    """rtol 1e-13: every ray takes > 1023 accepted steps, so the fixed-capacity record pass overflows and the
    library falls back to count + prefix sum + exact-size record."""
    w = W.C3(n=12, nf=5, rtol=1e-13)
    out = ody.render_spectrum(w["scene"], w["model"], w["nu"]); _sync()
    ref = orc.render_spectrum(w["scene"], w["model"], w["nu"])
    assert ref["n_attempt"].min() > 1100
    assert np.array_equal(_np(out["flag"]).ravel(), ref["flag"])
    assert np.mean(_np(out["n_attempt"]).ravel() == ref["n_attempt"]) >= 0.99
    imgs = _np(out["images"]).reshape(len(w["nu"]), -1)
    for k in range(len(w["nu"])):
        _check_image(imgs[k], ref["images"][k], f"overflow fallback k={k}")
    assert np.allclose(_np(out["nuLnu"]), ref["nuLnu"], rtol=1e-6)


def test_fused_spectrum_kernel_on_a_large_image_matches_the_oracle_and_the_two_phase_path(ody, orc):
    """More rays than one band of the two-phase path and fewer than 4 frequencies: the fused multi-frequency
    kernel (accumulators in global scratch) runs.  Checked against the oracle on a strided sub-grid, and against
    the two-phase path on a sub-image rendered separately with the same pixel centres."""
    nx, ny, nf = 640, 480, 3
    sc = W.scene(0.9375, 30.0, nx, 15.0, ny=ny)
    mo, nu = W.model_riaf(), W.log_spaced_frequencies(1e10, 1e12, nf)
    out = ody.render_spectrum(sc, mo, nu); _sync()
    ii = [p * 20 + 10 for q in range(24) for p in range(32)]
    jj = [q * 20 + 10 for q in range(24) for p in range(32)]
    ref = orc.render_spectrum(sc, mo, nu, idx=(ii, jj))
    imgs = _np(out["images"])
    assert np.array_equal(_np(out["flag"])[jj, ii], ref["flag"])
    for k in range(nf):
        _check_image(imgs[k][jj, ii], ref["images"][k], f"fused spectrum k={k}")
    # SED consistency with the kernel's own images
    area = (sc["x_max"] - sc["x_min"]) / nx * (sc["y_max"] - sc["y_min"]) / ny
    rg = orc.rg_cm(mo["mbh_msun"])
    sed = 4.0 * np.pi * np.asarray(nu) * rg * rg * area * imgs.reshape(nf, -1).sum(axis=1)
    assert np.allclose(_np(out["nuLnu"]), sed, rtol=1e-10)
    # the two-phase path on the lower-left 320 x 240 quarter (same pixel centres): identical images
    sub = dict(sc, nx=320, ny=240, x_max=0.0, y_max=0.0)
    small = ody.render_spectrum(sub, mo, nu); _sync()
    a, b = _np(small["images"]), imgs[:, :240, :320]
    assert np.allclose(a, b, rtol=1e-9, atol=1e-300)
    assert np.array_equal(_np(small["flag"]), _np(out["flag"])[:240, :320])


def test_banded_two_phase_spectrum_on_a_large_image_matches_the_oracle_and_the_other_paths(ody, orc):
    """More rays than one band (2 waves of the record kernel's lanes, 151 552 rays) and >= 4 frequencies: the two-phase
    path runs band by band over whole rows — here 236 + 164 rows, the second band ragged.  Checked against the
    oracle on a strided sub-grid that has points in both bands, against the single-band path on a sub-image cut
    across the band boundary, and against the fused kernel frequency by frequency."""
    nx, ny, nf = 640, 400, 16
    sc = W.scene(0.9375, 30.0, nx, 15.0, ny=ny)
    mo, nu = W.model_riaf(), W.log_spaced_frequencies(1e9, 1e14, nf)
    out = ody.render_spectrum(sc, mo, nu); _sync()
    imgs = _np(out["images"])
    ii = [p * 20 + 10 for q in range(20) for p in range(32)]
    jj = [q * 20 + 10 for q in range(20) for p in range(32)]
    ref = orc.render_spectrum(sc, mo, nu, idx=(ii, jj))
    assert np.array_equal(_np(out["flag"])[jj, ii], ref["flag"])
    assert np.mean(_np(out["n_attempt"])[jj, ii] == ref["n_attempt"]) >= 0.995
    for k in range(nf):
        _check_image(imgs[k][jj, ii], ref["images"][k], f"banded spectrum k={k}")
    area = (sc["x_max"] - sc["x_min"]) / nx * (sc["y_max"] - sc["y_min"]) / ny
    rg = orc.rg_cm(mo["mbh_msun"])
    sed = 4.0 * np.pi * np.asarray(nu) * rg * rg * area * imgs.reshape(nf, -1).sum(axis=1)
    assert np.allclose(_np(out["nuLnu"]), sed, rtol=1e-10)
    # rows 200..279 straddle the band boundary (row 236); as an image of their own they fit one band
    dy = (sc["y_max"] - sc["y_min"]) / ny
    sub = dict(sc, ny=80, y_min=sc["y_min"] + 200 * dy, y_max=sc["y_min"] + 280 * dy)
    small = ody.render_spectrum(sub, mo, nu); _sync()
    assert np.allclose(_np(small["images"]), imgs[:, 200:280, :], rtol=1e-9, atol=1e-300)
    assert np.array_equal(_np(small["flag"]), _np(out["flag"])[200:280, :])
    # the fused kernel (fewer than 4 frequencies on the same image) gives the same images
    for lo in (4, 9):
        fused = ody.render_spectrum(sc, mo, nu[lo:lo + 3]); _sync()
        assert np.allclose(_np(fused["images"]), imgs[lo:lo + 3], rtol=1e-9, atol=1e-300)


# ------------------------------------------------------------------------------ parameter and edge-case sweep
@pytest.mark.parametrize("label, scene_kw, model_kw, nu", [
    ("retrograde spin, Cash-Karp", dict(a=-0.8, incl=50.0, tableau=W.TABLEAU_CASH_KARP), dict(), 230e9),
    ("near observer r_obs=200 inside the emitting region", dict(a=0.6, incl=70.0, r_obs=200.0), dict(), 86e9),
    ("j_scale = 4 pi (eq. (37) as printed)", dict(a=0.9375, incl=30.0), dict(j_scale=4.0 * np.pi), 230e9),
    ("thin flow, strong field", dict(a=0.5, incl=80.0), dict(h_over_r=0.1, beta=1.0, n0=3e7), 345e9),
    ("cold flow: K_2 large-argument branch everywhere", dict(a=0.9, incl=45.0), dict(T0=3e9, T_index=-0.5), 22e9),
    ("hot flow: K_2 series everywhere", dict(a=0.9, incl=45.0), dict(T0=3e12, T_index=-0.3, n0=1e5), 230e9),
    ("small tau_max: most rays end OPAQUE", dict(a=0.9375, incl=30.0), dict(tau_max=0.5), 5e9),
    ("no electrons: dark image", dict(a=0.3, incl=20.0), dict(n0=0.0), 230e9),
    ("small emitting region", dict(a=0.998, incl=85.0), dict(r_rt_out=12.0), 230e9),
    ("face-on", dict(a=0.7, incl=0.5), dict(), 230e9),
    ("loose tolerance", dict(a=0.9375, incl=30.0, rtol=1e-5), dict(), 230e9),
    ("tiny tau_max: nearly every ray ends OPAQUE after a few emitting steps (the ring's run-ahead is discarded)", dict(a=0.9375, incl=30.0), dict(tau_max=1e-7), 230e9),
    ("negative tau_max: OPAQUE at the first accepted step", dict(a=0.5, incl=60.0), dict(tau_max=-1.0), 230e9),
    ("few attempts allowed: rays end MAXSTEP with points still in the ring", dict(a=0.9, incl=60.0, max_attempts=120), dict(), 230e9),
    ("observer inside a bright, outward-weighted medium: the start point's coefficients matter", dict(a=0.9375, incl=30.0, r_obs=100.0),
     dict(n0=1e3, n_index=1.0, T0=3e10, T_index=0.0, h_over_r=10.0), 230e9),
])
def test_riaf_parameter_sweep_matches_the_oracle(ody, orc, label, scene_kw, model_kw, nu):
    kw = dict(scene_kw)
    sc = W.scene(kw.pop("a"), kw.pop("incl"), 36, 14.0, **kw)
    mo = W.model_riaf(**model_kw)
    out = ody.render_image(sc, mo, nu); _sync()
    ref = orc.render_image(sc, mo, nu)
    assert np.array_equal(_np(out["flag"]).ravel(), ref["flag"]), label
    assert np.mean(_np(out["n_attempt"]).ravel() == ref["n_attempt"]) >= 0.99, label
    assert np.mean(_np(out["n_accept"]).ravel() == ref["n_accept"]) >= 0.99, label
    tau, tau_ref = _np(out["aux0"]).ravel(), ref["aux0"]
    assert np.allclose(tau, tau_ref, rtol=1e-6, atol=1e-300), label
    img = _np(out["image"]).ravel()
    if ref["image"].max() == 0.0:
        assert np.all(img == 0.0), label
    else:
        _check_image(img, ref["image"], label)
    if "OPAQUE" in label:
        assert np.mean(ref["flag"] == W.FLAG_OPAQUE) > 0.3
    if "MAXSTEP" in label:
        assert np.mean(ref["flag"] == W.FLAG_MAXSTEP) > 0.1


# ------------------------------------------------------------- mixed-precision transfer variant (north_star (c))
@pytest.mark.parametrize("nu", [230.0e9, 30.0e9])
def test_mixed_fp32_transfer_variant_accuracy_against_the_oracle(ody, orc, nu):
    """The variant is 'reported only if it stays inside tolerance' (north_star): this measures it against the
    oracle at the same tolerances as the FP64 path — 1e-6 relative L1, 1e-4 max per-pixel relative."""
    w = W.C2(n=96)
    out = ody.render_image(w["scene"], w["model"], nu, precision=ody.PREC_MIXED_FP32); _sync()
    ref = orc.render_image(w["scene"], w["model"], nu)
    assert np.array_equal(_np(out["flag"]).ravel(), ref["flag"])
    assert np.mean(_np(out["n_attempt"]).ravel() == ref["n_attempt"]) >= 0.995       # the geodesic part is the FP64 one
    _check_image(_np(out["image"]).ravel(), ref["image"], f"mixed FP32 variant at {nu:g} Hz")
    # and it really is a different arithmetic: not bit-identical to the FP64 kernel
    base = ody.render_image(w["scene"], w["model"], nu); _sync()
    a, b = _np(out["image"]).ravel(), _np(base["image"]).ravel()
    l1 = np.abs(a - b).sum() / b.sum()
    assert 1e-10 < l1 < 1e-6


# ----------------------------------------------------------------------------- hot spot (kind 3, reading HS)
@pytest.mark.parametrize("a, incl, n, hw, kw", [
    (0.0, 60.0, 96, 10.0, dict()),                                   # the paper's set-up: Schwarzschild, i = 60 deg, r_spot 0.5 at r_isco
    (0.9, 75.0, 80, 9.0, dict(r_spot=0.4)),
    (0.5, 30.0, 64, 12.0, dict(r_orbit=8.0, r_spot=1.2, phi0=1.0, g_power=3.0, nbins=40)),
])
def test_hot_spot_matches_the_oracle(ody, orc, a, incl, n, hw, kw):
    sc = W.scene(a, incl, n, hw)
    mo = W.model_hot_spot(**kw)
    rs = kw.get("r_orbit", 0.0) or orc.kerr_constants(a)["r_isco"]
    period = 2.0 * np.pi * (rs ** 1.5 + a)
    t_obs = list(np.linspace(0.0, period, 13)[:-1]) + [3.7 * period]
    out = ody.render_hotspot(sc, mo, t_obs); _sync()
    ref = orc.render_hotspot(sc, mo, t_obs)
    gpu = {k: (_np(v) if v is not None else None) for k, v in out.items()}
    assert np.array_equal(gpu["flag"].ravel(), ref["flag"])
    hit = ref["flag"] == W.FLAG_DISK
    for key in ("g", "r_e", "phi_e", "t_e"):
        x, xr = gpu[key].ravel(), ref[key]
        assert np.max(np.abs(x[hit] - xr[hit]) / np.abs(xr[hit])) <= 1e-8, key
        assert np.all(x[~hit] == 0.0), key
    imgs = gpu["images"].reshape(len(t_obs), -1)
    lit = 0
    for k in range(len(t_obs)):
        if ref["images"][k].max() > 0:
            lit += 1
            # the Gaussian turns a 1e-8 relative error of phi_e, t_e into ~1e-7 of the value far out in its wings
            assert np.abs(imgs[k] - ref["images"][k]).sum() / ref["images"][k].sum() <= 1e-6
            on = ref["images"][k] >= 1e-6 * ref["images"][k].max()
            assert np.max(np.abs(imgs[k] - ref["images"][k])[on] / ref["images"][k][on]) <= 1e-4
    assert lit >= 6
    assert np.allclose(gpu["lightcurve"], ref["lightcurve"], rtol=1e-6, atol=1e-12 * ref["lightcurve"].max())
    assert np.allclose(gpu["spectrogram"].sum(axis=1), gpu["lightcurve"], rtol=1e-10, atol=1e-300)
    assert np.max(np.abs(np.cumsum(gpu["spectrogram"], axis=1) - np.cumsum(ref["spectrogram"], axis=1))) <= 1e-6 * ref["lightcurve"].max()
    # host entry point: same numbers
    host = ody.render_hotspot_host(sc, mo, t_obs)
    assert np.array_equal(host["images"], gpu["images"]) and np.array_equal(host["t_e"], gpu["t_e"])
    assert np.allclose(host["lightcurve"], gpu["lightcurve"], rtol=1e-12)


# ------------------------------------------------------- Novikov-Thorne disk (kind 4, eq. (35), reading NT)
KEV_HZ = 2.417989242e17


@pytest.mark.parametrize("a, incl, n, hw, kw", [
    (0.999, 85.0, 128, 25.0, dict()),                                # Fig. 6's set-up: M = 10 M_sun, Mdot = 1e19 g/s, r_out = 50
    (0.0, 45.0, 96, 60.0, dict(r_out=50.0)),
    (0.5, 60.0, 64, 520.0, dict(r_out=500.0, mbh_msun=1.0e7, mdot_gs=1.0e24)),   # a supermassive hole: UV disk
])
def test_nt_disk_spectrum_matches_the_oracle(ody, orc, a, incl, n, hw, kw):
    sc = W.scene(a, incl, n, hw)
    mo = W.model_nt_disk(**kw)
    t_in = orc.nt_temperature(mo, a, 1.5 * orc.kerr_constants(a)["r_isco"])
    kt = 1.380649e-16 * t_in / 6.62607015e-27                        # k T / h of the inner disk, Hz
    nu = list(kt * np.logspace(-3.0, 1.5, 16))
    out = ody.render_spectrum(sc, mo, nu); _sync()
    gpu = {k: _np(v) for k, v in out.items()}
    ref = orc.render_spectrum(sc, mo, nu)
    assert np.array_equal(gpu["flag"].ravel(), ref["flag"])
    assert np.array_equal(gpu["n_attempt"].ravel(), ref["n_attempt"])
    assert (ref["flag"] == W.FLAG_DISK).sum() > 200
    for q in range(len(nu)):
        _check_image(gpu["images"][q].ravel(), ref["images"][q], f"NT disk image at nu[{q}]")
    assert np.max(np.abs(gpu["nuLnu"] - ref["nuLnu"]) / ref["nuLnu"]) <= 1e-6
    # single-frequency image call: same pixels, plus g and r_e of the crossing
    one = ody.render_image(sc, mo, nu[9]); _sync()
    assert np.array_equal(_np(one["image"]), gpu["images"][9])
    thin = orc.render_image(sc, W.model_thin_disk(r_in=mo["r_in"], r_out=mo["r_out"]))
    hit = ref["flag"] == W.FLAG_DISK
    g, r_e = _np(one["aux0"]).ravel(), _np(one["aux1"]).ravel()
    assert np.max(np.abs(g[hit] - thin["aux0"][hit]) / thin["aux0"][hit]) <= 1e-8
    assert np.max(np.abs(r_e[hit] - thin["aux1"][hit]) / thin["aux1"][hit]) <= 1e-8
    # host entry point
    host = ody.render_spectrum_host(sc, mo, nu)
    assert np.array_equal(host["images"], gpu["images"])
    assert np.allclose(host["nuLnu"], gpu["nuLnu"], rtol=1e-12)


def test_nt_disk_degenerate_cases(ody, orc):
    sc = W.scene(0.9, 70.0, 48, 20.0)
    nu = [0.1 * KEV_HZ, 1.0 * KEV_HZ]
    dark = ody.render_spectrum(sc, W.model_nt_disk(mdot_gs=0.0), nu); _sync()      # no accretion: a cold, dark disk
    assert float(dark["images"].abs().max()) == 0.0 and float(dark["nuLnu"].abs().max()) == 0.0
    assert int((dark["flag"] == W.FLAG_DISK).sum()) > 50
    # a disk that reaches inside r_isco: crossings there are flagged DISK but carry no flux (f = 0)
    mo = W.model_nt_disk(r_in=1.6, r_out=30.0)
    out = ody.render_spectrum(sc, mo, nu); _sync()
    ref = orc.render_spectrum(sc, mo, nu)
    assert np.array_equal(_np(out["flag"]).ravel(), ref["flag"])
    for q in range(2):
        _check_image(_np(out["images"])[q].ravel(), ref["images"][q], "NT disk inside r_isco")
    # far Wien tail: expm1 overflows to +inf and the pixel is exactly 0, on both sides
    far = ody.render_spectrum(sc, W.model_nt_disk(), [3.0e4 * KEV_HZ]); _sync()
    assert float(far["images"].max()) == 0.0
    assert orc.render_spectrum(sc, W.model_nt_disk(), [3.0e4 * KEV_HZ])["images"].max() == 0.0


# ------------------------------------------------- optical-depth step cap (reading DT)
@pytest.mark.parametrize("nu, cap, tableau", [(1.0e10, 0.1, W.TABLEAU_RKF45), (1.0e10, 0.5, W.TABLEAU_CASH_KARP),
                                             (5.0e10, 0.02, W.TABLEAU_RKF45), (2.3e11, 0.05, W.TABLEAU_RKF45)])
def test_dtau_step_cap_matches_the_oracle(ody, orc, nu, cap, tableau):
    w = W.C2(n=96)
    sc = dict(w["scene"]); sc["tableau"] = tableau
    mo = W.model_riaf(dtau_max=cap)
    out = ody.render_image(sc, mo, nu); _sync()
    ref = orc.render_image(sc, mo, nu)
    assert np.array_equal(_np(out["flag"]).ravel(), ref["flag"])
    assert np.mean(_np(out["n_attempt"]).ravel() == ref["n_attempt"]) >= 0.995
    _check_image(_np(out["image"]).ravel(), ref["image"], "image with the optical-depth cap")
    tau, tau_ref = _np(out["aux0"]).ravel(), ref["aux0"]
    assert np.max(np.abs(tau - tau_ref) / np.maximum(tau_ref, 1e-30)) <= 1e-6
    # the cap binds in the optically thick cases (many more steps); at 230 GHz (tau <= 0.3 in total) hardly any step
    # is longer than 0.05 optical depths and the step count barely moves
    free = ody.render_image(sc, W.model_riaf(), nu); _sync()
    n_cap, n_free = int(out["n_attempt"].sum()), int(free["n_attempt"].sum())
    if nu <= 5.0e10:
        assert n_cap > 1.05 * n_free
    else:
        assert abs(n_cap - n_free) <= 1e-3 * n_free


# ------------------------------------------------------ rays through the rotation axis (L_z = 0 exactly)
@pytest.mark.parametrize("a, incl", [(0.0, 120.0), (0.9, 100.0), (0.998, 175.0), (0.5, 60.0)])
def test_centre_column_rays_through_the_axis_match_the_oracle(ody, orc, a, incl):
    # an odd number of columns puts x = 0 (L_z = 0) on the centre column: those rays pass through the pole, continue with
    # theta outside [0, pi] and meet the plane at theta = pi/2 + k pi (oracle pin:
    # test_disk_crossing_of_rays_through_the_axis_is_continuous_with_their_neighbours)
    sc = W.scene(a, incl, 41, 18.0, ny=45)
    thin = W.model_thin_disk(r_in=0.0, r_out=60.0)
    out = ody.render_image(sc, thin); _sync()
    gpu = {k: (_np(v) if v is not None else None) for k, v in out.items()}
    ref = orc.render_image(sc, thin)
    _check_disk(gpu, ref, check_hist=False)
    col = ref["flag"].reshape(45, 41)[:, 20]
    assert (col == W.FLAG_DISK).sum() >= 10 and col.max() <= 2
    # hot spot: the azimuth of the crossing carries the k pi
    mo = W.model_hot_spot(r_orbit=8.0, r_spot=2.0)
    mo.update(r_in=0.0, r_out=60.0)
    t_obs = [0.0, 40.0, 90.0]
    hs = ody.render_hotspot(sc, mo, t_obs); _sync()
    hr = orc.render_hotspot(sc, mo, t_obs)
    assert np.array_equal(_np(hs["flag"]).ravel(), hr["flag"])
    hit = hr["flag"] == W.FLAG_DISK
    for key in ("g", "r_e", "phi_e", "t_e"):
        x, xr = _np(hs[key]).ravel(), hr[key]
        assert np.max(np.abs(x[hit] - xr[hit]) / np.maximum(np.abs(xr[hit]), 1.0)) <= 1e-8, key
    for k in range(3):
        if hr["images"][k].max() > 0:
            assert np.abs(_np(hs["images"])[k].ravel() - hr["images"][k]).sum() / hr["images"][k].sum() <= 1e-6
    # Novikov-Thorne disk on the same geometry
    nt = W.model_nt_disk(r_out=60.0)
    nu = [0.3 * KEV_HZ, 2.0 * KEV_HZ]
    sp = ody.render_spectrum(sc, nt, nu); _sync()
    sr = orc.render_spectrum(sc, nt, nu)
    assert np.array_equal(_np(sp["flag"]).ravel(), sr["flag"])
    for q in range(2):
        _check_image(_np(sp["images"])[q].ravel(), sr["images"][q], "NT disk, centre column")
