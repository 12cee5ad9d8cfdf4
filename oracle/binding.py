"""ctypes loader for oracle/liboracle.so — TEST INFRASTRUCTURE (see odyssey_oracle.cpp).

Thin marshalling only: dictionaries from `workloads` -> the oracle's C structs, numpy arrays in and
out.  Never imports the CUDA package.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

c_double_p = C.POINTER(C.c_double)
c_int32_p = C.POINTER(C.c_int32)


class Scene(C.Structure):
    _fields_ = [("a", C.c_double), ("r_obs", C.c_double), ("theta_obs", C.c_double), ("phi_obs", C.c_double),
                ("x_min", C.c_double), ("x_max", C.c_double), ("y_min", C.c_double), ("y_max", C.c_double),
                ("nx", C.c_int32), ("ny", C.c_int32),
                ("rtol", C.c_double),
                ("tableau", C.c_int32), ("pad0", C.c_int32),
                ("h0", C.c_double), ("horizon_eps", C.c_double), ("r_esc", C.c_double),
                ("max_attempts", C.c_int32), ("pad1", C.c_int32)]


class Model(C.Structure):
    _fields_ = [("kind", C.c_int32), ("nbins", C.c_int32),
                ("r_in", C.c_double), ("r_out", C.c_double), ("emis_index", C.c_double),
                ("mbh_msun", C.c_double), ("n0", C.c_double), ("n_index", C.c_double), ("T0", C.c_double),
                ("T_index", C.c_double), ("h_over_r", C.c_double), ("beta", C.c_double),
                ("r_rt_out", C.c_double), ("tau_max", C.c_double), ("j_scale", C.c_double),
                ("g_lo", C.c_double), ("g_hi", C.c_double), ("g_power", C.c_double),
                ("rt_scheme", C.c_int32), ("pad", C.c_int32),
                ("spot_r_orbit", C.c_double), ("spot_size", C.c_double), ("spot_phi0", C.c_double),
                ("mdot_gs", C.c_double), ("dtau_max", C.c_double)]


def _fill(struct, d):
    names = {f[0] for f in struct._fields_}
    for k, v in d.items():
        if k not in names:
            raise KeyError(k)
        setattr(struct, k, v)
    return struct


def make_scene(d):
    return _fill(Scene(), d)


def make_model(d):
    return _fill(Model(), d)


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.oracle_num_threads.restype = C.c_int
        L.oracle_null_ratio.restype = C.c_double
        L.oracle_carter_Q.restype = C.c_double
        L.oracle_error_norm.restype = C.c_double
        L.oracle_bessel_K2.restype = C.c_double
        L.oracle_mahadevan_M.restype = C.c_double
        L.oracle_planck_B.restype = C.c_double
        L.oracle_rg_cm.restype = C.c_double
        L.oracle_flow_gamma.restype = C.c_int
        L.oracle_trace_path.restype = C.c_int
        for name in ("oracle_bessel_K2", "oracle_mahadevan_M", "oracle_rg_cm"):
            getattr(L, name).argtypes = [C.c_double]
        L.oracle_planck_B.argtypes = [C.c_double, C.c_double]
        _lib = L
    return _lib


def _dp(arr):
    return arr.ctypes.data_as(c_double_p) if arr is not None else None


def _ip(arr):
    return arr.ctypes.data_as(c_int32_p) if arr is not None else None


def _vec(v):
    return np.ascontiguousarray(np.asarray(v, dtype=np.float64))


def num_threads():
    return int(lib().oracle_num_threads())


def set_num_threads(n):
    lib().oracle_set_num_threads(C.c_int(int(n)))


def kerr_constants(a):
    out = np.zeros(4)
    lib().oracle_kerr_constants(C.c_double(a), _dp(out))
    return dict(r_h=out[0], r_isco=out[1], E_isco=out[2], L_isco=out[3])


def init_ray(scene, x, y):
    st, cons = np.zeros(5), np.zeros(5)
    lib().oracle_init_ray(C.byref(make_scene(scene)), C.c_double(x), C.c_double(y), _dp(st), _dp(cons))
    return st, dict(E=cons[0], L=cons[1], Q=cons[2], E2_raw=cons[3], L_raw=cons[4])


def rhs(a, E, L, y, with_t=False):
    """Slopes of (r, theta, phi, p_r, p_theta); with_t=True appends dt/dlambda of eq. (9)."""
    y = _vec(y)[:5].copy(); dy = np.zeros(6)
    lib().oracle_rhs(C.c_double(a), C.c_double(E), C.c_double(L), _dp(y), _dp(dy))
    return dy if with_t else dy[:5]


def null_ratio(a, E, L, y):
    y = _vec(y)
    return float(lib().oracle_null_ratio(C.c_double(a), C.c_double(E), C.c_double(L), _dp(y)))


def carter_Q(a, E, L, y):
    y = _vec(y)
    return float(lib().oracle_carter_Q(C.c_double(a), C.c_double(E), C.c_double(L), _dp(y)))


def tableau(which):
    c, A, b5, b4 = np.zeros(6), np.zeros((6, 6)), np.zeros(6), np.zeros(6)
    lib().oracle_tableau(C.c_int(which), _dp(c), _dp(A), _dp(b5), _dp(b4))
    return c, A, b5, b4


def rk_attempt(a, E, L, which, y, h):
    y = _vec(y); ynew, yerr = np.zeros(5), np.zeros(5)
    lib().oracle_rk_attempt(C.c_double(a), C.c_double(E), C.c_double(L), C.c_int(which), _dp(y), C.c_double(h),
                            _dp(ynew), _dp(yerr))
    return ynew, yerr


def error_norm(y, yerr, rtol):
    y, yerr = _vec(y), _vec(yerr)
    return float(lib().oracle_error_norm(_dp(y), _dp(yerr), C.c_double(rtol)))


def flow_gamma(a, r, th, pr, pth, L):
    u = np.zeros(4); g = C.c_double(0.0)
    ok = lib().oracle_flow_gamma(C.c_double(a), C.c_double(r), C.c_double(th), C.c_double(pr), C.c_double(pth),
                                 C.c_double(L), _dp(u), C.byref(g))
    return bool(ok), u, g.value


def bessel_K2(x):
    return float(lib().oracle_bessel_K2(float(x)))


def mahadevan_M(x):
    return float(lib().oracle_mahadevan_M(float(x)))


def planck_B(nu, T):
    return float(lib().oracle_planck_B(float(nu), float(T)))


def rg_cm(mbh_msun):
    return float(lib().oracle_rg_cm(float(mbh_msun)))


def synchrotron(model, a, r, th, nu0):
    out = np.zeros(7)
    lib().oracle_synchrotron(C.byref(make_model(model)), C.c_double(a), C.c_double(r), C.c_double(th),
                             C.c_double(nu0), _dp(out))
    return dict(n_e=out[0], T_e=out[1], B=out[2], Theta_e=out[3], nu_c=out[4], j=out[5], alpha=out[6])


def rt_update(a0, a1, e0, e1, dl, tau_max, tau, T, I):
    st = np.array([tau, T, I], dtype=np.float64)
    lib().oracle_rt_update(C.c_double(a0), C.c_double(a1), C.c_double(e0), C.c_double(e1), C.c_double(dl),
                           C.c_double(tau_max), _dp(st))
    return st[0], st[1], st[2]


def page_thorne_f(a, r):
    L = lib(); L.oracle_page_thorne_f.restype = C.c_double
    return L.oracle_page_thorne_f(C.c_double(a), C.c_double(r))


def nt_temperature(model, a, r):
    L = lib(); L.oracle_nt_temperature.restype = C.c_double
    return L.oracle_nt_temperature(C.byref(make_model(model)), C.c_double(a), C.c_double(r))


def rt_rk_step(which, a, eps, h, tau_max, tau, I):
    st = np.array([tau, I], dtype=np.float64)
    lib().oracle_rt_rk_step(C.c_int(which), _dp(_vec(a)), _dp(_vec(eps)), C.c_double(h), C.c_double(tau_max), _dp(st))
    return float(st[0]), float(st[1])


def trace_points(scene, model, nu, xs, ys):
    xs, ys = _vec(xs), _vec(ys)
    n = xs.size
    nu = _vec(nu); nf = nu.size
    out = dict(flag=np.zeros(n, np.int32), r=np.zeros(n), th=np.zeros(n), ph=np.zeros(n),
               n_attempt=np.zeros(n, np.int32), n_accept=np.zeros(n, np.int32),
               g=np.zeros(n), r_e=np.zeros(n), I=np.zeros((n, nf)), tau=np.zeros((n, nf)), t=np.zeros(n))
    lib().oracle_trace_points(C.byref(make_scene(scene)), C.byref(make_model(model)), C.c_int(nf), _dp(nu), C.c_int(n),
                              _dp(xs), _dp(ys), _ip(out["flag"]), _dp(out["r"]), _dp(out["th"]), _dp(out["ph"]),
                              _ip(out["n_attempt"]), _ip(out["n_accept"]), _dp(out["g"]), _dp(out["r_e"]),
                              _dp(out["I"]), _dp(out["tau"]), _dp(out["t"]))
    return out


def trace_path(scene, model, x, y, max_nodes=20000):
    """Accepted nodes (r, theta, phi, p_r, p_theta, lambda, t) of one ray (geodesic and events only)."""
    nodes = np.zeros((max_nodes, 7)); cons = np.zeros(3); res = np.zeros(3, np.int32)
    n = lib().oracle_trace_path(C.byref(make_scene(scene)), C.byref(make_model(model)), C.c_double(x), C.c_double(y),
                                C.c_int(max_nodes), _dp(nodes), _dp(cons), _ip(res))
    return nodes[:min(n, max_nodes)], dict(E=cons[0], L=cons[1], Q=cons[2]), dict(flag=int(res[0]), n_attempt=int(res[1]),
                                                                                   n_accept=int(res[2]))


def trace_path_rt(scene, model, nu_hz, x, y, max_nodes=20000):
    """trace_path with the transfer at one frequency: also the absorption coefficient at each node."""
    nodes = np.zeros((max_nodes, 7)); absorb = np.zeros(max_nodes); res = np.zeros(3, np.int32)
    n = lib().oracle_trace_path_rt(C.byref(make_scene(scene)), C.byref(make_model(model)), C.c_double(nu_hz),
                                   C.c_double(x), C.c_double(y), C.c_int(max_nodes), _dp(nodes), _dp(absorb), _ip(res))
    n = min(n, max_nodes)
    return nodes[:n], absorb[:n], dict(flag=int(res[0]), n_attempt=int(res[1]), n_accept=int(res[2]))


def _pixels(scene, idx):
    if idx is None:
        return scene["nx"] * scene["ny"], None, None
    ii = np.ascontiguousarray(np.asarray(idx[0], dtype=np.int32))
    jj = np.ascontiguousarray(np.asarray(idx[1], dtype=np.int32))
    return ii.size, ii, jj


def trace_geodesics(scene, idx=None):
    """C0 driver.  idx = (i_list, j_list) restricts to those pixels; default whole grid, row-major [j][i]."""
    n, ii, jj = _pixels(scene, idx)
    out = dict(flag=np.zeros(n, np.int32), r=np.zeros(n), th=np.zeros(n), ph=np.zeros(n),
               n_attempt=np.zeros(n, np.int32), n_accept=np.zeros(n, np.int32), t=np.zeros(n))
    lib().oracle_trace_geodesics(C.byref(make_scene(scene)), C.c_int(n), _ip(ii), _ip(jj),
                                 _ip(out["flag"]), _dp(out["r"]), _dp(out["th"]), _dp(out["ph"]),
                                 _ip(out["n_attempt"]), _ip(out["n_accept"]), _dp(out["t"]))
    return out


def render_image(scene, model, nu_hz=0.0, idx=None):
    n, ii, jj = _pixels(scene, idx)
    nb = int(model.get("nbins", 0))
    out = dict(image=np.zeros(n), aux0=np.zeros(n), aux1=np.zeros(n), flag=np.zeros(n, np.int32),
               n_attempt=np.zeros(n, np.int32), n_accept=np.zeros(n, np.int32),
               hist=np.zeros(nb) if nb > 0 else None)
    lib().oracle_render_image(C.byref(make_scene(scene)), C.byref(make_model(model)), C.c_double(nu_hz), C.c_int(n),
                              _ip(ii), _ip(jj), _dp(out["image"]), _dp(out["aux0"]), _dp(out["aux1"]),
                              _ip(out["flag"]), _ip(out["n_attempt"]), _ip(out["n_accept"]), _dp(out["hist"]))
    return out


def render_hotspot(scene, model, t_obs, idx=None):
    n, ii, jj = _pixels(scene, idx)
    t = _vec(t_obs); nt = t.size
    nb = int(model.get("nbins", 0))
    out = dict(images=np.zeros((nt, n)), lightcurve=np.zeros(nt), spectrogram=np.zeros((nt, nb)) if nb > 0 else None,
               g=np.zeros(n), r_e=np.zeros(n), phi_e=np.zeros(n), t_e=np.zeros(n),
               flag=np.zeros(n, np.int32), n_attempt=np.zeros(n, np.int32))
    lib().oracle_render_hotspot(C.byref(make_scene(scene)), C.byref(make_model(model)), _dp(t), C.c_int(nt), C.c_int(n),
                                _ip(ii), _ip(jj), _dp(out["images"]), _dp(out["lightcurve"]), _dp(out["spectrogram"]),
                                _dp(out["g"]), _dp(out["r_e"]), _dp(out["phi_e"]), _dp(out["t_e"]),
                                _ip(out["flag"]), _ip(out["n_attempt"]))
    return out


def render_spectrum(scene, model, nu_hz, idx=None):
    n, ii, jj = _pixels(scene, idx)
    nu = _vec(nu_hz); nf = nu.size
    out = dict(images=np.zeros((nf, n)), nuLnu=np.zeros(nf), flag=np.zeros(n, np.int32),
               n_attempt=np.zeros(n, np.int32))
    lib().oracle_render_spectrum(C.byref(make_scene(scene)), C.byref(make_model(model)), _dp(nu), C.c_int(nf), C.c_int(n),
                                 _ip(ii), _ip(jj), _dp(out["images"]), _dp(out["nuLnu"]), _ip(out["flag"]),
                                 _ip(out["n_attempt"]))
    return out
