"""Writes tests/golden/oracle_regression.json from the CPU oracle ALONE (never from the CUDA path): a few
oracle outputs on tiny grids, so that an accidental change to the oracle's arithmetic shows up as a diff.
A deliberate change re-runs this script and names, in its commit message, the PAPER.md passage or
DESIGN.md reading that justifies it.

    python tests/golden/make_oracle_golden.py
"""
import json
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import workloads as W  # noqa: E402
from oracle import binding as O  # noqa: E402


def main():
    out = {"_comment": "written by tests/golden/make_oracle_golden.py from oracle/ only"}
    w = W.C0(n=8)
    g = O.trace_geodesics(w["scene"])
    out["C0_8x8"] = {k: g[k].tolist() for k in ("flag", "r", "th", "ph", "n_attempt", "n_accept")}
    w = W.C1(n=8)
    d = O.render_image(w["scene"], w["model"])
    out["C1_8x8"] = {"flag": d["flag"].tolist(), "g": d["aux0"].tolist(), "r_e": d["aux1"].tolist(),
                     "image": d["image"].tolist()}
    w = W.C2(n=8)
    for scheme in (W.RT_PER_STEP, W.RT_RK_COMPONENTS):
        r = O.render_image(w["scene"], dict(w["model"], rt_scheme=scheme), w["nu"][0])
        out[f"C2_8x8_rt_scheme{scheme}"] = {"flag": r["flag"].tolist(), "image": r["image"].tolist(),
                                            "tau": r["aux0"].tolist(), "n_attempt": r["n_attempt"].tolist()}
    w = W.C3(n=4, nf=4)
    s = O.render_spectrum(w["scene"], w["model"], w["nu"])
    out["C3_4x4_nf4"] = {"nu": list(w["nu"]), "nuLnu": s["nuLnu"].tolist(), "images": s["images"].tolist()}
    sc = W.scene(0.5, 60.0, 10, 9.0)
    hs = O.render_hotspot(sc, W.model_hot_spot(r_spot=1.0, nbins=8), [0.0, 40.0, 80.0])
    out["hotspot_10x10"] = {"t_obs": [0.0, 40.0, 80.0], "lightcurve": hs["lightcurve"].tolist(), "t_e": hs["t_e"].tolist(),
                            "phi_e": hs["phi_e"].tolist(), "images": hs["images"].tolist()}
    g = O.trace_geodesics(W.C0(n=8)["scene"])
    out["C0_8x8"]["t"] = g["t"].tolist()
    # Novikov-Thorne disk (reading NT): f(r), T_eff and a small spectrum of Fig. 6's set-up
    nt = W.model_nt_disk()
    out["nt_disk"] = {"a": 0.999, "r": [1.3, 2.0, 6.0, 30.0],
                      "f": [O.page_thorne_f(0.999, r) for r in (1.3, 2.0, 6.0, 30.0)],
                      "T_eff": [O.nt_temperature(nt, 0.999, r) for r in (1.3, 2.0, 6.0, 30.0)]}
    nu_nt = [2.4e16, 2.4e17, 1.2e18]
    sp = O.render_spectrum(W.scene(0.999, 85.0, 9, 25.0), nt, nu_nt)
    out["nt_disk"].update(nu=nu_nt, nuLnu=sp["nuLnu"].tolist(), images=sp["images"].tolist(), flag=sp["flag"].tolist())
    # optical-depth step cap (reading DT) on the optically thick 10 GHz image
    w = W.C2(n=8)
    r = O.render_image(w["scene"], W.model_riaf(dtau_max=0.1), 1.0e10)
    out["C2_8x8_10GHz_dtau0.1"] = {"image": r["image"].tolist(), "tau": r["aux0"].tolist(), "n_attempt": r["n_attempt"].tolist()}
    with open(os.path.join(HERE, "oracle_regression.json"), "w") as f:
        json.dump(out, f, indent=1)
    print("wrote oracle_regression.json")


if __name__ == "__main__":
    main()
