"""The kernels' own FP64 elementary functions (paper_1601_02063_b200/csrc/dmath.cuh) against libm /
scipy.  CPU part: the header is compiled for the host (tests/dmath_host.cpp; only the hardware seeds
differ) — this checks the reductions, the polynomial tables and the reconstruction.  GPU part
(-m gpu): the device build through odyssey_eval_math, including the MUFU seeds and K_2."""
import ctypes as C
import os
import subprocess
import tempfile

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
OPS = dict(rcp=0, rsqrt=1, sqrt=2, sincos=3, exp=4, expm1=5, log=6, k2=7)


def _ulps(y, ref):
    return np.max(np.abs(y - ref) / np.spacing(np.abs(ref)))


def _cases():
    rng = np.random.default_rng(7)
    pos = np.exp(rng.uniform(-200, 200, 100000))
    ang = np.concatenate([rng.uniform(-3.3, 3.3, 60000), rng.uniform(-60, 60, 40000), [0.0, np.pi / 2, np.pi, -np.pi / 2]])
    ex = np.concatenate([rng.uniform(-700, 700, 60000), rng.uniform(-1, 1, 40000)])
    em = np.concatenate([rng.uniform(-50, 50, 50000), rng.uniform(-1, 1, 50000),
                         10.0 ** rng.uniform(-18, 0, 2000) * rng.choice([-1, 1], 2000), [0.0]])
    lg = np.concatenate([pos, 1.0 + rng.uniform(-0.3, 0.45, 50000), [1.0, 2.0, 0.5, np.sqrt(2), np.sqrt(0.5)]])
    return pos, ang, ex, em, lg


def _check_all(ev):
    pos, ang, ex, em, lg = _cases()
    assert _ulps(ev("rcp", pos)[0], 1.0 / pos) <= 1.0
    assert _ulps(ev("rsqrt", pos)[0], 1.0 / np.sqrt(pos)) <= 2.0
    assert _ulps(ev("sqrt", pos)[0], np.sqrt(pos)) <= 1.0
    s, c = ev("sincos", ang)
    assert np.max(np.abs(s - np.sin(ang))) <= 2.5e-16 and np.max(np.abs(c - np.cos(ang))) <= 2.5e-16
    small = np.abs(ang) <= 3.3
    assert _ulps(s[small][np.abs(np.sin(ang[small])) > 1e-3], np.sin(ang[small])[np.abs(np.sin(ang[small])) > 1e-3]) <= 4.0
    assert np.all(s * s + c * c - 1.0 < 5e-16)
    assert _ulps(ev("exp", ex)[0], np.exp(ex)) <= 2.0
    assert _ulps(ev("expm1", em)[0][em != 0], np.expm1(em[em != 0])) <= 3.0
    assert ev("expm1", np.array([0.0]))[0][0] == 0.0
    assert _ulps(ev("log", lg)[0][lg != 1.0], np.log(lg[lg != 1.0])) <= 4.0
    assert ev("log", np.array([1.0]))[0][0] == 0.0
    # saturation behaviour the radiative-transfer code relies on
    assert np.all(ev("exp", np.array([-700.5, -1e4, -np.inf]))[0] == 0.0)
    assert np.all(ev("expm1", np.array([-800.0, -1e5]))[0] == -1.0)


@pytest.fixture(scope="module")
def host_lib():
    out = os.path.join(tempfile.mkdtemp(prefix="dmath_"), "dmath_host.so")
    subprocess.run(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-shared", "-fPIC", "-o", out,
                    os.path.join(HERE, "dmath_host.cpp")], check=True)
    return C.CDLL(out)


def test_host_build_of_device_math_matches_libm(host_lib):
    def ev(name, x):
        x = np.ascontiguousarray(x, dtype=np.float64)
        y, y2 = np.zeros_like(x), np.zeros_like(x)
        host_lib.dm_eval(OPS[name], x.size, x.ctypes.data_as(C.c_void_p), y.ctypes.data_as(C.c_void_p),
                         y2.ctypes.data_as(C.c_void_p))
        return y, y2
    _check_all(ev)


@pytest.mark.gpu
def test_device_math_matches_libm(ody):
    import torch

    def ev(name, x):
        t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).cuda()
        y, y2 = ody.eval_math(OPS[name], t)
        torch.cuda.synchronize()
        return y.cpu().numpy(), y2.cpu().numpy()
    _check_all(ev)


@pytest.mark.gpu
def test_device_bessel_k2_matches_scipy(ody):
    import torch
    from scipy import special
    x = np.concatenate([np.exp(np.linspace(np.log(1e-3), np.log(600.0), 20000)), [2.0, 2.0 + 1e-12, 2.0 - 1e-12]])
    y, _ = ody.eval_math(OPS["k2"], torch.from_numpy(x).cuda())
    torch.cuda.synchronize()
    ref = special.kv(2, x)
    rel = np.abs(y.cpu().numpy() - ref) / ref
    assert rel.max() <= 5e-10, rel.max()          # the x > 2 Chebyshev fit is the limit; the series is ~1e-15
    assert rel[x <= 2.0].max() <= 1e-13
