"""The kernels rebuilt with -DODY_DEVICE_CHECKS (device-side assertions on every index into the ray stash, the transfer
ring and the output arrays) run the small configurations of every kernel family; a failed assertion surfaces as a
CUDA error and fails the test.  Also: output buffers carved out of one allocation with sentinel-filled guard bands
between them must come back with the bands untouched (ragged image sizes included).
compute-sanitizer (memcheck / racecheck) is closed on the B200 pool used here: this is the stand-in."""
import os
import subprocess
import sys
import tempfile

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CASES = r'''
import sys
sys.path.insert(0, %r)
import torch, workloads as W
import paper_1601_02063_b200 as ody
ody.load_library()
def done():
    torch.cuda.synchronize()
w = W.C0(n=40); ody.trace_geodesics(w["scene"], with_time=True); done()
w = W.C1(n=56); ody.render_image(w["scene"], w["model"]); done()
for nu in (230e9, 1e10):                                   # thin, and mostly OPAQUE endings through the transfer ring
    w = W.C2(n=72); ody.render_image(dict(w["scene"], ny=50), w["model"], nu); done()
    ody.render_image(w["scene"], w["model"], nu, precision=ody.PREC_MIXED_FP32); done()
w = W.C2(n=33); ody.render_image(w["scene"], dict(w["model"], rt_scheme=W.RT_RK_COMPONENTS), 230e9); done()
ody.render_image(w["scene"], dict(w["model"], dtau_max=0.2), 1e10); done()
w = W.C3(n=40, nf=7); ody.render_spectrum(w["scene"], w["model"], w["nu"]); done()
sc = W.scene(0.5, 60.0, 48, 12.0); ody.render_hotspot(sc, W.model_hot_spot(), [0.0, 30.0, 60.0]); done()
ody.render_spectrum(W.scene(0.9, 70.0, 40, 30.0), W.model_nt_disk(), [1e17, 3e17]); done()
ody.render_image(W.scene(0.9375, 30.0, 1, 15.0), W.model_riaf(), 230e9); done()       # a single pixel
print("CHECKS_OK")
''' % ROOT


def test_small_configurations_under_device_side_index_assertions():
    from paper_1601_02063_b200 import build as B
    lib = os.path.join(tempfile.mkdtemp(prefix="ody_checks_"), "libodyssey_checks.so")
    B.build_variant(lib, ["-DODY_DEVICE_CHECKS"])
    env = dict(os.environ, ODYSSEY_LIB=lib)
    res = subprocess.run([sys.executable, "-c", CASES], capture_output=True, text=True, env=env, timeout=900)
    assert res.returncode == 0 and "CHECKS_OK" in res.stdout, res.stdout[-1500:] + res.stderr[-3000:]


@pytest.mark.parametrize("nx, ny", [(61, 37), (8, 4), (130, 3)])
def test_guard_bands_around_the_output_arrays_stay_untouched(ody, nx, ny):
    import torch
    w = W.C2(n=nx)
    sc = dict(w["scene"], ny=ny)
    n, pad = nx * ny, 512
    buf64 = torch.full((3 * n + 4 * pad,), -777.0, dtype=torch.float64, device="cuda")
    buf32 = torch.full((3 * n + 4 * pad,), -777, dtype=torch.int32, device="cuda")
    cut = lambda b, k: b[pad + k * (n + pad): pad + k * (n + pad) + n].view(ny, nx)
    out = dict(image=cut(buf64, 0), aux0=cut(buf64, 1), aux1=cut(buf64, 2), flag=cut(buf32, 0), n_attempt=cut(buf32, 1),
               n_accept=cut(buf32, 2), hist=None)
    ody.render_image(sc, w["model"], w["nu"][0], out=out)
    torch.cuda.synchronize()
    for b in (buf64, buf32):
        h = b.cpu().numpy()
        inside = np.zeros(h.size, bool)
        for k in range(3):
            inside[pad + k * (n + pad): pad + k * (n + pad) + n] = True
        assert np.all(h[~inside] == -777), "a guard band was written"
        assert not np.any(h[inside] == -777), "an output element was not written"


def test_transfer_ring_does_not_change_a_single_bit(ody):
    """batching the transfer coefficients through the per-warp ring changes which lane evaluates a point and
    when, not the arithmetic or its order per ray.  The library rebuilt without the ring (-DODY_RT_FIFO=0: every lane
    evaluates its own point in the trip that produced it) must give the same image, optical depth, flags and step counts
    bit for bit — thin and optically thick (most rays ending OPAQUE: the ring's run-ahead is discarded)."""
    import torch
    from paper_1601_02063_b200 import build as B
    tmp = tempfile.mkdtemp(prefix="ody_nofifo_")
    lib = os.path.join(tmp, "libodyssey_nofifo.so")
    B.build_variant(lib, ["-DODY_RT_FIFO=0"])
    code = r'''
import sys
sys.path.insert(0, %r)
import numpy as np, torch, workloads as W
import paper_1601_02063_b200 as ody
w = W.C2(n=320)
for tag, nu, kw in (("thin", 230e9, {}), ("thick", 5e9, {"tau_max": 0.5})):
    out = ody.render_image(dict(w["scene"], ny=250), dict(w["model"], **kw), nu); torch.cuda.synchronize()
    np.savez(%r + "/" + tag + ".npz", **{k: v.cpu().numpy() for k, v in out.items() if v is not None})
print("DONE")
''' % (ROOT, tmp)
    res = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, env=dict(os.environ, ODYSSEY_LIB=lib), timeout=900)
    assert res.returncode == 0 and "DONE" in res.stdout, res.stdout[-1000:] + res.stderr[-3000:]
    w = W.C2(n=320)
    for tag, nu, kw in (("thin", 230e9, {}), ("thick", 5e9, {"tau_max": 0.5})):
        out = ody.render_image(dict(w["scene"], ny=250), dict(w["model"], **kw), nu); torch.cuda.synchronize()
        ref = np.load(os.path.join(tmp, tag + ".npz"))
        for k in ("image", "aux0", "flag", "n_attempt", "n_accept"):
            assert np.array_equal(out[k].cpu().numpy(), ref[k]), (tag, k)
        if tag == "thick":
            assert np.mean(ref["flag"] == W.FLAG_OPAQUE) > 0.3
