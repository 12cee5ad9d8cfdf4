"""ctypes binding of include/odyssey.h — argument marshalling only.

Every step of the hot path runs inside libodyssey.so's CUDA kernels.  PyTorch is used for device
buffers and the current stream, nothing else.  There is no CPU fallback: if the library cannot be
loaded, or a call returns an error code, OdysseyError is raised.

Scenes and models are the plain dictionaries of `workloads.py` (keys = fields of odyssey_scene /
odyssey_model).  Device calls return dictionaries of torch CUDA tensors shaped [ny, nx]
(or [nf, ny, nx]); host calls return numpy arrays.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

EXPORTED_SYMBOLS = (
    "odyssey_trace_geodesics", "odyssey_render_image", "odyssey_render_spectrum", "odyssey_render_hotspot",
    "odyssey_trace_geodesics_host", "odyssey_render_image_host", "odyssey_render_spectrum_host",
    "odyssey_render_hotspot_host",
    "odyssey_fp64_peak_probe", "odyssey_kernel_info", "odyssey_eval_math", "odyssey_trim_scratch", "odyssey_launch_count",
    "odyssey_last_error", "odyssey_shutdown",
)


class OdysseyError(RuntimeError):
    pass


class Scene(C.Structure):
    _fields_ = [("a", C.c_double), ("r_obs", C.c_double), ("theta_obs", C.c_double), ("phi_obs", C.c_double),
                ("x_min", C.c_double), ("x_max", C.c_double), ("y_min", C.c_double), ("y_max", C.c_double),
                ("nx", C.c_int32), ("ny", C.c_int32), ("rtol", C.c_double),
                ("tableau", C.c_int32), ("pad0", C.c_int32),
                ("h0", C.c_double), ("horizon_eps", C.c_double), ("r_esc", C.c_double),
                ("max_attempts", C.c_int32), ("pad1", C.c_int32)]


class Model(C.Structure):
    _fields_ = [("kind", C.c_int32), ("nbins", C.c_int32),
                ("r_in", C.c_double), ("r_out", C.c_double), ("emis_index", C.c_double),
                ("mbh_msun", C.c_double), ("n0", C.c_double), ("n_index", C.c_double),
                ("T0", C.c_double), ("T_index", C.c_double), ("h_over_r", C.c_double), ("beta", C.c_double),
                ("r_rt_out", C.c_double), ("tau_max", C.c_double), ("j_scale", C.c_double),
                ("g_lo", C.c_double), ("g_hi", C.c_double), ("g_power", C.c_double),
                ("rt_scheme", C.c_int32), ("precision", C.c_int32),
                ("spot_r_orbit", C.c_double), ("spot_size", C.c_double), ("spot_phi0", C.c_double),
                ("mdot_gs", C.c_double), ("dtau_max", C.c_double)]


def _struct(cls, d):
    s = cls()
    names = {f[0] for f in cls._fields_}
    for k, v in d.items():
        if k not in names:
            raise KeyError(f"{cls.__name__} has no field {k!r}")
        setattr(s, k, v)
    return s


_lib = None


def load_library():
    """Load (building first if the sources are newer) libodyssey.so.  Raises OdysseyError if it
    cannot be built or loaded — the product path never falls back to anything else."""
    global _lib
    if _lib is not None:
        return _lib
    try:
        path = _build.build()
    except Exception as e:  # noqa: BLE001
        raise OdysseyError(f"libodyssey.so is missing and could not be built: {e}") from e
    try:
        L = C.CDLL(path)
    except OSError as e:
        raise OdysseyError(f"cannot load {path}: {e}") from e
    vp, dp, ip = C.c_void_p, C.c_void_p, C.c_void_p
    L.odyssey_trace_geodesics.argtypes = [C.POINTER(Scene), ip, dp, dp, dp, dp, ip, ip, vp]
    L.odyssey_render_image.argtypes = [C.POINTER(Scene), C.POINTER(Model), C.c_double, dp, dp, dp, ip, ip, ip, dp, vp]
    L.odyssey_render_spectrum.argtypes = [C.POINTER(Scene), C.POINTER(Model), C.POINTER(C.c_double), C.c_int,
                                          dp, dp, ip, ip, vp]
    L.odyssey_trace_geodesics_host.argtypes = [C.POINTER(Scene), ip, dp, dp, dp, dp, ip, ip]
    L.odyssey_render_image_host.argtypes = [C.POINTER(Scene), C.POINTER(Model), C.c_double, dp, dp, dp, ip, ip, ip, dp]
    L.odyssey_render_spectrum_host.argtypes = [C.POINTER(Scene), C.POINTER(Model), C.POINTER(C.c_double), C.c_int,
                                               dp, dp, ip, ip]
    L.odyssey_fp64_peak_probe.argtypes = [C.c_int, dp, C.POINTER(C.c_double), vp]
    L.odyssey_kernel_info.argtypes = [C.c_int, C.c_int, C.c_int] + [C.POINTER(C.c_int32)] * 5
    L.odyssey_launch_count.restype = C.c_longlong
    L.odyssey_last_error.restype = C.c_char_p
    L.odyssey_shutdown.restype = None
    L.odyssey_eval_math.argtypes = [C.c_int, C.c_int, dp, dp, dp, vp]
    L.odyssey_render_hotspot.argtypes = [C.POINTER(Scene), C.POINTER(Model), C.POINTER(C.c_double), C.c_int,
                                         dp, dp, dp, dp, dp, dp, dp, ip, ip, vp]
    L.odyssey_render_hotspot_host.argtypes = [C.POINTER(Scene), C.POINTER(Model), C.POINTER(C.c_double), C.c_int,
                                              dp, dp, dp, dp, dp, dp, dp, ip, ip]
    L.odyssey_trim_scratch.argtypes = [C.c_ulonglong]
    for name in EXPORTED_SYMBOLS[:12]:
        getattr(L, name).restype = C.c_int
    _lib = L
    return L


def last_error():
    return load_library().odyssey_last_error().decode()


def _check(rc):
    if rc != 0:
        raise OdysseyError(f"odyssey call failed with status {rc}: {last_error()}")


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise OdysseyError("no CUDA device: the Odyssey hot path has no CPU fallback")
    return torch


def _stream(torch):
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def _np_ptr(a):
    return C.c_void_p(a.ctypes.data) if a is not None else None


def trace_geodesics(scene, with_time=False):
    """odyssey_trace_geodesics: flag, r, theta, phi, n_attempt, n_accept (and t with with_time) as [ny, nx] CUDA tensors."""
    torch = _torch()
    L = load_library()
    ny, nx = scene["ny"], scene["nx"]
    f64 = dict(dtype=torch.float64, device="cuda")
    i32 = dict(dtype=torch.int32, device="cuda")
    out = dict(flag=torch.empty((ny, nx), **i32), r=torch.empty((ny, nx), **f64), theta=torch.empty((ny, nx), **f64),
               phi=torch.empty((ny, nx), **f64), n_attempt=torch.empty((ny, nx), **i32),
               n_accept=torch.empty((ny, nx), **i32))
    if with_time:
        out["t"] = torch.empty((ny, nx), **f64)
    _check(L.odyssey_trace_geodesics(C.byref(_struct(Scene, scene)), _ptr(out["flag"]), _ptr(out["r"]),
                                     _ptr(out["theta"]), _ptr(out["phi"]), _ptr(out.get("t")), _ptr(out["n_attempt"]),
                                     _ptr(out["n_accept"]), _stream(torch)))
    return out


PREC_FP64, PREC_MIXED_FP32 = 0, 1


def render_image(scene, model, nu_hz=0.0, out=None, precision=PREC_FP64):
    """odyssey_render_image: image, aux0, aux1, flag, n_attempt, n_accept ([ny, nx]) and hist ([nbins] or None).
    `out` may carry pre-allocated tensors from a previous call (re-used, e.g. by bench.py)."""
    torch = _torch()
    L = load_library()
    ny, nx = scene["ny"], scene["nx"]
    if out is None:
        f64 = dict(dtype=torch.float64, device="cuda")
        nb = int(model.get("nbins", 0)) if model["kind"] == 1 else 0
        out = dict(image=torch.empty((ny, nx), **f64), aux0=torch.empty((ny, nx), **f64),
                   aux1=torch.empty((ny, nx), **f64),
                   flag=torch.empty((ny, nx), dtype=torch.int32, device="cuda"),
                   n_attempt=torch.empty((ny, nx), dtype=torch.int32, device="cuda"),
                   n_accept=torch.empty((ny, nx), dtype=torch.int32, device="cuda"),
                   hist=torch.empty((nb,), **f64) if nb > 0 else None)
    mstruct = _struct(Model, model)
    mstruct.precision = int(precision)
    _check(L.odyssey_render_image(C.byref(_struct(Scene, scene)), C.byref(mstruct), C.c_double(nu_hz),
                                  _ptr(out["image"]), _ptr(out["aux0"]), _ptr(out["aux1"]), _ptr(out["flag"]),
                                  _ptr(out["n_attempt"]), _ptr(out.get("n_accept")), _ptr(out.get("hist")),
                                  _stream(torch)))
    return out


def render_spectrum(scene, model, nu_hz):
    """odyssey_render_spectrum: images [nf, ny, nx], nuLnu [nf], flag, n_attempt."""
    torch = _torch()
    L = load_library()
    ny, nx = scene["ny"], scene["nx"]
    nu = (C.c_double * len(nu_hz))(*[float(v) for v in nu_hz])
    nf = len(nu_hz)
    f64 = dict(dtype=torch.float64, device="cuda")
    out = dict(images=torch.empty((max(nf, 1), ny, nx), **f64), nuLnu=torch.empty((max(nf, 1),), **f64),
               flag=torch.empty((ny, nx), dtype=torch.int32, device="cuda"),
               n_attempt=torch.empty((ny, nx), dtype=torch.int32, device="cuda"))
    _check(L.odyssey_render_spectrum(C.byref(_struct(Scene, scene)), C.byref(_struct(Model, model)), nu, C.c_int(nf),
                                     _ptr(out["images"]), _ptr(out["nuLnu"]), _ptr(out["flag"]),
                                     _ptr(out["n_attempt"]), _stream(torch)))
    return out


def render_hotspot(scene, model, t_obs):
    """odyssey_render_hotspot: images [nt, ny, nx], lightcurve [nt], spectrogram [nt, nbins] or None, and per
    pixel g, r_e, phi_e, t_e, flag, n_attempt."""
    torch = _torch()
    L = load_library()
    ny, nx, nt = scene["ny"], scene["nx"], len(t_obs)
    t = (C.c_double * nt)(*[float(v) for v in t_obs])
    f64 = dict(dtype=torch.float64, device="cuda")
    nb = int(model.get("nbins", 0))
    out = dict(images=torch.empty((max(nt, 1), ny, nx), **f64), lightcurve=torch.empty((max(nt, 1),), **f64),
               spectrogram=torch.empty((max(nt, 1), nb), **f64) if nb > 0 else None,
               g=torch.empty((ny, nx), **f64), r_e=torch.empty((ny, nx), **f64), phi_e=torch.empty((ny, nx), **f64),
               t_e=torch.empty((ny, nx), **f64), flag=torch.empty((ny, nx), dtype=torch.int32, device="cuda"),
               n_attempt=torch.empty((ny, nx), dtype=torch.int32, device="cuda"))
    _check(L.odyssey_render_hotspot(C.byref(_struct(Scene, scene)), C.byref(_struct(Model, model)), t, C.c_int(nt),
                                    _ptr(out["images"]), _ptr(out["lightcurve"]), _ptr(out["spectrogram"]),
                                    _ptr(out["g"]), _ptr(out["r_e"]), _ptr(out["phi_e"]), _ptr(out["t_e"]),
                                    _ptr(out["flag"]), _ptr(out["n_attempt"]), _stream(torch)))
    return out


def render_hotspot_host(scene, model, t_obs):
    L = load_library()
    ny, nx, nt = scene["ny"], scene["nx"], len(t_obs)
    t = (C.c_double * nt)(*[float(v) for v in t_obs])
    nb = int(model.get("nbins", 0))
    out = dict(images=np.empty((max(nt, 1), ny, nx)), lightcurve=np.empty(max(nt, 1)),
               spectrogram=np.empty((max(nt, 1), nb)) if nb > 0 else None,
               g=np.empty((ny, nx)), r_e=np.empty((ny, nx)), phi_e=np.empty((ny, nx)), t_e=np.empty((ny, nx)),
               flag=np.empty((ny, nx), np.int32), n_attempt=np.empty((ny, nx), np.int32))
    _check(L.odyssey_render_hotspot_host(C.byref(_struct(Scene, scene)), C.byref(_struct(Model, model)), t, C.c_int(nt),
                                         _np_ptr(out["images"]), _np_ptr(out["lightcurve"]), _np_ptr(out["spectrogram"]),
                                         _np_ptr(out["g"]), _np_ptr(out["r_e"]), _np_ptr(out["phi_e"]), _np_ptr(out["t_e"]),
                                         _np_ptr(out["flag"]), _np_ptr(out["n_attempt"])))
    return out


def trace_geodesics_host(scene, with_time=False):
    L = load_library()
    ny, nx = scene["ny"], scene["nx"]
    out = dict(flag=np.empty((ny, nx), np.int32), r=np.empty((ny, nx)), theta=np.empty((ny, nx)), phi=np.empty((ny, nx)),
               n_attempt=np.empty((ny, nx), np.int32), n_accept=np.empty((ny, nx), np.int32))
    if with_time:
        out["t"] = np.empty((ny, nx))
    _check(L.odyssey_trace_geodesics_host(C.byref(_struct(Scene, scene)), _np_ptr(out["flag"]), _np_ptr(out["r"]),
                                          _np_ptr(out["theta"]), _np_ptr(out["phi"]), _np_ptr(out.get("t")), _np_ptr(out["n_attempt"]),
                                          _np_ptr(out["n_accept"])))
    return out


def render_image_host(scene, model, nu_hz=0.0, out=None):
    L = load_library()
    ny, nx = scene["ny"], scene["nx"]
    if out is None:
        nb = int(model.get("nbins", 0)) if model["kind"] == 1 else 0
        out = dict(image=np.empty((ny, nx)), aux0=np.empty((ny, nx)), aux1=np.empty((ny, nx)),
                   flag=np.empty((ny, nx), np.int32), n_attempt=np.empty((ny, nx), np.int32),
                   n_accept=np.empty((ny, nx), np.int32), hist=np.empty(nb) if nb > 0 else None)
    _check(L.odyssey_render_image_host(C.byref(_struct(Scene, scene)), C.byref(_struct(Model, model)),
                                       C.c_double(nu_hz), _np_ptr(out["image"]), _np_ptr(out["aux0"]),
                                       _np_ptr(out["aux1"]), _np_ptr(out["flag"]), _np_ptr(out["n_attempt"]),
                                       _np_ptr(out.get("n_accept")), _np_ptr(out.get("hist"))))
    return out


def render_spectrum_host(scene, model, nu_hz):
    L = load_library()
    ny, nx = scene["ny"], scene["nx"]
    nf = len(nu_hz)
    nu = (C.c_double * nf)(*[float(v) for v in nu_hz])
    out = dict(images=np.empty((max(nf, 1), ny, nx)), nuLnu=np.empty(max(nf, 1)),
               flag=np.empty((ny, nx), np.int32), n_attempt=np.empty((ny, nx), np.int32))
    _check(L.odyssey_render_spectrum_host(C.byref(_struct(Scene, scene)), C.byref(_struct(Model, model)), nu,
                                          C.c_int(nf), _np_ptr(out["images"]), _np_ptr(out["nuLnu"]),
                                          _np_ptr(out["flag"]), _np_ptr(out["n_attempt"])))
    return out


def fp64_peak_probe(iters, sink):
    """Enqueue the DFMA microbenchmark on the current stream; returns the flop count of the launch."""
    torch = _torch()
    flop = C.c_double(0.0)
    _check(load_library().odyssey_fp64_peak_probe(C.c_int(int(iters)), _ptr(sink), C.byref(flop), _stream(torch)))
    return flop.value


def eval_math(op, x):
    """odyssey_eval_math on a CUDA float64 tensor; returns (y, y2)."""
    torch = _torch()
    x = x.contiguous()
    y, y2 = torch.empty_like(x), torch.empty_like(x)
    _check(load_library().odyssey_eval_math(C.c_int(int(op)), C.c_int(x.numel()), _ptr(x), _ptr(y), _ptr(y2), _stream(torch)))
    return y, y2


def kernel_info(kind, spectrum=False, tableau=0):
    v = [C.c_int32(0) for _ in range(5)]
    _check(load_library().odyssey_kernel_info(C.c_int(kind), C.c_int(int(spectrum)), C.c_int(tableau),
                                              *[C.byref(x) for x in v]))
    return dict(registers=v[0].value, local_bytes=v[1].value, threads_per_block=v[2].value,
                blocks_per_sm=v[3].value, n_sm=v[4].value)


def trim_scratch(keep_bytes=0):
    """odyssey_trim_scratch: give the library's cached device scratch above keep_bytes back to the driver."""
    _check(load_library().odyssey_trim_scratch(C.c_ulonglong(int(keep_bytes))))


def launch_count():
    return int(load_library().odyssey_launch_count())


def shutdown():
    load_library().odyssey_shutdown()
