"""Pins for the optical-depth step cap (reading DT; SURVEY.md §8(f)-2 "a Δτ-limited step cap"): with
model.dtau_max > 0 no step of the per-step transfer scheme is longer than dtau_max optical depths at the absorption
coefficient of its start point; where the medium is thin the cap changes nothing, bit for bit; where it is thick
the image moves TOWARDS the converged one."""
import numpy as np
import pytest

import workloads as W
from oracle import binding as O

SC = W.scene(0.9375, 30.0, 24, 15.0)
THICK, THIN = 1.0e10, 2.3e11


@pytest.mark.parametrize("cap", [0.3, 0.1, 0.02])
def test_no_step_exceeds_the_cap(cap):
    for x, y in ((3.0, 1.0), (-6.5, 0.4), (0.3, -8.0)):
        nodes, absorb, res = O.trace_path_rt(SC, W.model_riaf(dtau_max=cap), THICK, x, y)
        h = np.diff(nodes[:, 5])
        dtau = absorb[:-1] * h                     # the coefficient at the START of each step times its length
        # (lambda is accumulated from ~1e3: its differences carry ~1e-10 relative rounding)
        assert dtau.max() <= cap * (1 + 1e-8)
        assert (dtau > 0.5 * cap).sum() >= 5       # and the cap is what limits the steps in the thick part
        free, _, res0 = O.trace_path_rt(SC, W.model_riaf(), THICK, x, y)
        assert res["n_accept"] > res0["n_accept"]


def test_cap_is_inert_where_the_medium_is_thin():
    a = O.render_image(SC, W.model_riaf(), THIN)
    b = O.render_image(SC, W.model_riaf(dtau_max=0.5), THIN)
    assert a["aux0"].max() < 0.5                   # tau of every ray below the cap: it can never bind
    for k in ("image", "aux0", "flag", "n_attempt", "n_accept"):
        assert np.array_equal(a[k], b[k]), k


def test_cap_moves_the_thick_image_towards_the_converged_one():
    # reference: rtol 1e-11 with a very small cap (two such references, caps 0.01 and 0.003, agree to 5e-6)
    tight = dict(SC); tight["rtol"] = 1e-11
    ref = O.render_image(tight, W.model_riaf(dtau_max=0.01), THICK)["image"]
    errs = []
    for cap in (0.0, 0.3, 0.1):
        img = O.render_image(SC, W.model_riaf(dtau_max=cap), THICK)["image"]
        errs.append(np.abs(img - ref).sum() / ref.sum())
    # measured at rtol 1e-8: 2.2e-3 without the cap, 7.5e-4 at 0.3, 1.4e-4 at 0.1 (below that the geodesic
    # tolerance and the emission region's sharp outer edge set the floor)
    assert errs[0] > 2.0 * errs[1] > 4.0 * errs[2]
    assert errs[0] > 10.0 * errs[2]
    assert errs[2] < 3e-4


def test_cap_is_ignored_by_the_other_models_and_schemes():
    thin = O.render_image(SC, dict(W.model_thin_disk(), dtau_max=0.1))
    thin0 = O.render_image(SC, W.model_thin_disk())
    assert np.array_equal(thin["image"], thin0["image"]) and np.array_equal(thin["n_attempt"], thin0["n_attempt"])
