"""Device-time table for the five BASELINE.json configurations and the C4 sweep.

    python -m paper_1601_02063_b200.timing [--sweep] [--reps 3]

Prints one JSON line per case: milliseconds per call (CUDA events, median of `reps` after one warm-up),
photons, attempted RK steps and ns per photon per attempted step.  The headline number and its roofline
come from bench.py; this is the companion table for the configurations bench.py does not time
(BASELINE.json:configs[0..3] and configs[4]'s sweep over spin and resolution).
"""
import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402


def time_case(ody, torch, name, w, reps):
    sc, mo, nu = w["scene"], w["model"], w["nu"]

    def call():
        if mo["kind"] == W.KIND_HOT_SPOT:
            return ody.render_hotspot(sc, mo, nu)
        if mo["kind"] == W.KIND_NONE:
            return ody.trace_geodesics(sc)
        if len(nu) > 1:
            return ody.render_spectrum(sc, mo, nu)
        return ody.render_image(sc, mo, nu[0] if nu else 0.0)

    out = call()
    torch.cuda.synchronize()
    ms = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        out = call()
        e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    ms.sort()
    t = ms[len(ms) // 2]
    attempts = int(out["n_attempt"].sum(dtype=torch.int64).item())
    rays = sc["nx"] * sc["ny"]
    return {"case": name, "ms": t, "photons": rays, "frequencies": max(len(nu), 1), "attempted_rk_steps": attempts,
            "ns_per_photon_per_step": t * 1e6 / attempts, "images_per_s": 1e3 / t}


def main():
    p = argparse.ArgumentParser()
    p.add_argument("--sweep", action="store_true", help="also the C4 sweep a in {0,0.5,0.9,0.998} x n in {1024,2048,4096}")
    p.add_argument("--reps", type=int, default=3)
    args = p.parse_args()
    import torch
    import paper_1601_02063_b200 as ody
    cases = [("C0", W.C0()), ("C1", W.C1()), ("C2", W.C2()), ("C3", W.C3()), ("C4", W.C4())]
    cases.append(("C2 rt_scheme=RK components", dict(W.C2(), model=W.model_riaf(rt_scheme=W.RT_RK_COMPONENTS))))
    t_obs = [2.0 * 3.141592653589793 * 6.0 ** 1.5 * k / 32 for k in range(32)]
    cases.append(("hot spot a=0 i=60 512^2, 32 phases", dict(scene=W.scene(0.0, 60.0, 512, 10.0), model=W.model_hot_spot(), nu=t_obs)))
    # the set-up of the paper's own timing table (Table 1: geodesics only, a = 0.95, i = 60 deg,
    # 1024^2; the image-plane extent is not stated there: +/-10 M is used)
    cases.append(("paper Table 1 set-up: geodesics only a=0.95 i=60 1024^2", dict(scene=W.scene(0.95, 60.0, 1024, 10.0), model=W.model_none(), nu=[])))
    # Fig. 6's set-up: Novikov-Thorne disk, a = 0.999, i = 85 deg, M = 10 M_sun, Mdot = 1e19 g/s,
    # r_out = 500 r_g; 32 photon energies 0.01-30 keV
    kev = 2.417989242e17
    cases.append(("Fig. 6 set-up: Novikov-Thorne disk a=0.999 i=85 r_out=500, 1024^2 x 32 energies",
                  dict(scene=W.scene(0.999, 85.0, 1024, 520.0), model=W.model_nt_disk(r_out=500.0),
                       nu=W.log_spaced_frequencies(0.01 * kev, 30.0 * kev, 32))))
    if args.sweep:
        for a in (0.0, 0.5, 0.9, 0.998):
            for n in (1024, 2048, 4096):
                cases.append((f"C4 a={a:g} n={n}", W.C4(n=n, a=a)))
    for name, w in cases:
        print(json.dumps(time_case(ody, torch, name, w, args.reps)), flush=True)


if __name__ == "__main__":
    main()
