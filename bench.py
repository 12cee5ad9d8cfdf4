#!/usr/bin/env python
"""bench.py — headline measurement of the Odyssey hot path on B200 (contract: see DESIGN.md §7).

A *step* is one pass of the whole hot path — pixel → initial conditions → adaptive RK geodesic
integration fused with the per-step radiative-transfer update → SoA stores — over one image of the
throughput configuration C4 (BASELINE.json:configs[4]: a = 0.998, i = 85 deg, 4096 x 4096 = 16.8 M
photons, RIAF at 230 GHz, FP64), through the C ABI (odyssey_render_image).

Printed JSON line (rank 0):
  metric/value    ns per photon per RK step = device time / total attempted RK steps (lower is better)
  images_per_s    1 / step time (aggregate over ranks)
  roofline        bound "alu": algorithmic FP64 flop / kernel time vs the DFMA peak
                  measured in this same run by odyssey_fp64_peak_probe
  e2e             the same metric through odyssey_render_image_host (host buffers, copies in the
                  timed region)
  cpu_baseline    the CPU oracle, as it stands, on a bounded strided sample of the same image plane

`--impl reference` times the oracle alone (there is no reference implementation to install: the
reference is a paper).
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as W  # noqa: E402

METRIC = "ns per photon per RK step (FP64)"
UNIT = "ns/photon/step"

# FP64 work per unit: flop per attempted RK step of the geodesic system and per radiative-transfer
# update (one per accepted step, single frequency).  These are flop the kernels EXECUTE (2 x DFMA + DMUL + DADD
# thread instructions, predicated on), counted by ncu on this very workload and kept, with the DRAM traffic, the
# warp execution efficiency and the FP64-pipe utilisation of the same captures, in profiles/r02_flop_counts.json
# (written by bench_counts.py; the file carries a hash of the kernel sources and the line says "stale" when the
# sources have changed since).  SURVEY.md §8(d)'s a-priori hand count (~1500 flop per attempt + ~490 per update)
# is reported beside it as `frac_hand_count`: it is what a straightforward implementation would execute, ~60 %
# more than these kernels do, so it flatters the rate and is NOT the headline fraction.
COUNTS_FILE = os.path.join(ROOT, "profiles", "r02_flop_counts.json")
HAND_FLOP_PER_ATTEMPT, HAND_FLOP_PER_RT_UPDATE = 1500.0, 490.0


def load_counts():
    import bench_counts
    with open(COUNTS_FILE) as f:
        c = json.load(f)
    c["stale"] = c.get("source_hash") != bench_counts.source_hash()
    return c


def parse_args():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=5)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="b200", choices=["b200", "reference"])
    p.add_argument("--n", type=int, default=4096, help="image side (C4 sweep: 1024, 2048, 4096)")
    p.add_argument("--a", type=float, default=0.998, help="spin (C4 sweep: 0, 0.5, 0.9, 0.998)")
    p.add_argument("--model", default="riaf", choices=["riaf", "none"],
                   help="riaf: the fused geodesic + GRRT kernel (the headline); none: geodesics only (the paper's Table 1 workload)")
    p.add_argument("--cpu-sample", type=int, default=448, help="side of the strided sub-grid the oracle is timed on")
    p.add_argument("--no-cpu-baseline", action="store_true")
    p.add_argument("--no-e2e", action="store_true")
    p.add_argument("--no-fp32-variant", action="store_true")
    p.add_argument("--no-extra", action="store_true", help="skip the extra.configs block (C0-C3 and the C4 sweep)")
    p.add_argument("--precision", default="fp64", choices=["fp64", "mixed"],
                   help="mixed: time the mixed-precision transfer variant as the main kernel (for ncu captures)")
    return p.parse_args()


def workload_name(n, a, model="riaf"):
    what = "RIAF 230 GHz" if model == "riaf" else "geodesics only"
    return f"C4: Kerr a={a:g}, i=85deg, {n}x{n} over +/-15M, r_obs=1000M, {what}, RKF45 rtol 1e-8"


def workload(args):
    w = W.C4(n=args.n, a=args.a)
    if args.model == "none":
        w = dict(w, model=W.model_none(), nu=[0.0])
    return w


# ---------------------------------------------------------------------------------------------------
# clocks: sample nvidia-smi DURING the timed region (B200_PROFILING.md recipe)
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for row in self.rows:
            f = [x.strip() for x in row.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline and --impl reference): the only places bench.py executes oracle/
# ---------------------------------------------------------------------------------------------------
def time_oracle_sample(w, n_sub):
    """One pass of the oracle over an n_sub x n_sub grid of pixel centres spanning the same image
    plane as workload w.  Returns (seconds, attempted steps, rays, threads)."""
    from oracle import binding as orc
    sc = W.coarse_scene(w["scene"], n_sub)
    t0 = time.perf_counter()
    out = orc.render_image(sc, w["model"], w["nu"][0])
    dt = time.perf_counter() - t0
    return dt, int(out["n_attempt"].astype("int64").sum()), n_sub * n_sub, orc.num_threads()


def cpu_baseline(w, n_sub):
    dt, attempts, rays, threads = time_oracle_sample(w, n_sub)
    return {"value": dt / attempts * 1e9, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": f"{n_sub}x{n_sub} strided sub-grid of the same image plane, {rays} rays, "
                      f"{attempts} attempted RK steps, {dt:.2f} s wall on {threads} threads",
            "per_core_ns": dt * threads / attempts * 1e9}


def run_reference(args):
    """The reference arm: there is no reference code (the reference is a paper), so the oracle is timed."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import build as oracle_build
    oracle_build.build()
    w = workload(args)
    n_sub = args.cpu_sample
    for _ in range(min(args.warmup, 1)):
        time_oracle_sample(w, 64)
    tot_t, tot_att, threads, rays = 0.0, 0, 1, 0
    for _ in range(args.steps):
        dt, attempts, rays, threads = time_oracle_sample(w, n_sub)
        tot_t += dt; tot_att += attempts
    value = tot_t / tot_att * 1e9
    sample = (f"each step = {n_sub}x{n_sub} strided sub-grid ({rays} rays) of the {args.n}x{args.n} image plane; "
              f"ns/photon/step does not depend on the sampling density")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_t / args.steps * 1e3,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": workload_name(args.n, args.a, args.model), "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------------------------------------------
# rank reduction and headline arithmetic (plain functions: tests/test_bench_multirank.py runs them under
# gloo with world_size 2 on CPU)
# ---------------------------------------------------------------------------------------------------
def reduce_over_ranks(dist, device, times, counts):
    """times: per-rank durations -> MAX over ranks; counts: per-rank work -> SUM over ranks.
    dist is torch.distributed (initialised) or None for a single process."""
    import torch
    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    n = torch.tensor(list(counts), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return t.tolist(), n.tolist()


def headline(total_ms_max, steps, attempts_all, accepts_all, world):
    """Whole-job figures from the max-over-ranks time of `steps` steps and the per-step work summed over
    ranks (every rank renders whole images of its own: weak scaling)."""
    ms_per_step = total_ms_max / steps
    return {"ms_per_step": ms_per_step,
            "value": ms_per_step * 1e6 / attempts_all,                # ns per photon per attempted RK step
            "ns_per_photon_per_accepted_step": ms_per_step * 1e6 / accepts_all,
            "images_per_s": world / (ms_per_step * 1e-3)}


# ---------------------------------------------------------------------------------------------------
# extra.configs: device time of every BASELINE.json configuration and of the C4 sweep (outside the headline's
# timed region; CUDA events on the launching stream, one warm-up, median of 3)
# ---------------------------------------------------------------------------------------------------
def time_extra_configs(ody, torch):
    def timed(call, photons):
        out = call(); torch.cuda.synchronize()
        ms = []
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); out = call(); e1.record(); torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        ms.sort()
        att = int(out["n_attempt"].sum(dtype=torch.int64).item())
        return {"photons": photons, "ms": ms[1], "attempts": att, "ns_per_photon_step": ms[1] * 1e6 / att,
                "images_per_s": 1e3 / ms[1]}

    res = {}
    w = W.C0(); res["C0"] = timed(lambda: ody.trace_geodesics(w["scene"]), w["scene"]["nx"] * w["scene"]["ny"])
    w1 = W.C1(); res["C1"] = timed(lambda: ody.render_image(w1["scene"], w1["model"]), w1["scene"]["nx"] * w1["scene"]["ny"])
    w2 = W.C2(); res["C2"] = timed(lambda: ody.render_image(w2["scene"], w2["model"], w2["nu"][0]), w2["scene"]["nx"] * w2["scene"]["ny"])
    w3 = W.C3(); res["C3"] = dict(timed(lambda: ody.render_spectrum(w3["scene"], w3["model"], w3["nu"]), w3["scene"]["nx"] * w3["scene"]["ny"]),
                                  frequencies=len(w3["nu"]))
    m_rk = dict(w2["model"], rt_scheme=W.RT_RK_COMPONENTS)
    res["C2 rt_scheme=RK components"] = timed(lambda: ody.render_image(w2["scene"], m_rk, w2["nu"][0]), w2["scene"]["nx"] * w2["scene"]["ny"])
    w3f = W.C3(n=1024, nf=3)
    res["C3 flow, 1024^2 x 3 frequencies (fused spectrum kernel)"] = dict(
        timed(lambda: ody.render_spectrum(w3f["scene"], w3f["model"], w3f["nu"]), 1024 * 1024), frequencies=3)
    w8 = W.C3(n=1024, nf=8)
    res["C3 flow, 1024^2 x 8 frequencies (two-phase path in bands)"] = dict(
        timed(lambda: ody.render_spectrum(w8["scene"], w8["model"], w8["nu"]), 1024 * 1024), frequencies=8)
    w32 = W.C3(n=1024)
    res["C3 flow, 1024^2 x 32 frequencies (two-phase path in bands)"] = dict(
        timed(lambda: ody.render_spectrum(w32["scene"], w32["model"], w32["nu"]), 1024 * 1024), frequencies=32)
    ody.trim_scratch(0)
    hs_scene, hs_model = W.scene(0.0, 60.0, 512, 12.0), W.model_hot_spot()
    t_obs = [k * 2.0 * math.pi * (6.0 ** 1.5) / 32 for k in range(32)]
    res["hot spot a=0 i=60 512^2, 32 phases"] = dict(timed(lambda: ody.render_hotspot(hs_scene, hs_model, t_obs), 512 * 512), phases=32)
    tab1 = W.scene(0.95, 60.0, 1024, 10.0)
    res["paper Table 1 set-up: geodesics only a=0.95 i=60 1024^2"] = timed(lambda: ody.trace_geodesics(tab1), 1024 * 1024)
    for a in (0.0, 0.5, 0.9, 0.998):
        for n in (1024, 2048, 4096):
            w4 = W.C4(n=n, a=a)
            res[f"C4 a={a:g} n={n}"] = timed(lambda: ody.render_image(w4["scene"], w4["model"], w4["nu"][0]), n * n)
            torch.cuda.empty_cache()
    return res


# ---------------------------------------------------------------------------------------------------
# the B200 arm
# ---------------------------------------------------------------------------------------------------
def run_b200(args):
    import torch
    import paper_1601_02063_b200 as ody

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the Odyssey hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    ody.load_library()
    # Rays are independent: ranks share nothing; each rank renders one whole image per
    # step (weak scaling, no data-path collective — DESIGN.md §9).
    w = workload(args)
    sc, mo, nu = w["scene"], w["model"], w["nu"][0]
    prec = ody.PREC_MIXED_FP32 if args.precision == "mixed" else ody.PREC_FP64
    out = ody.render_image(sc, mo, nu, precision=prec)
    torch.cuda.synchronize()
    for _ in range(max(args.warmup - 1, 0)):
        ody.render_image(sc, mo, nu, out=out, precision=prec)
    barrier()

    # ---- timed region: exactly K steps, CUDA events on the launching (current) stream
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    launches0 = ody.launch_count()
    barrier()
    ev[0].record()
    for k in range(args.steps):
        ody.render_image(sc, mo, nu, out=out, precision=prec)
        ev[k + 1].record()
    barrier()
    launches = ody.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    step_ms = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    total_ms = ev[0].elapsed_time(ev[args.steps])
    attempts = int(out["n_attempt"].sum(dtype=torch.int64).item())
    accepts = int(out["n_accept"].sum(dtype=torch.int64).item())
    rays = sc["nx"] * sc["ny"]
    out_bytes = sum(v.numel() * v.element_size() for v in out.values() if v is not None)

    # ---- DFMA peak, same run, same clocks regime (burst figure: the probe is timed alone)
    sink = torch.zeros(8, dtype=torch.float64, device="cuda")
    ody.fp64_peak_probe(2000, sink)
    torch.cuda.synchronize()
    best = None
    for _ in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        flop = ody.fp64_peak_probe(20000, sink)
        e1.record()
        torch.cuda.synchronize()
        tf = flop / (e0.elapsed_time(e1) * 1e-3) / 1e12
        best = tf if best is None else max(best, tf)
    peak_tflops = best

    # ---- north_star subsystem (c): the mixed-precision (FP32 polynomial cores) transfer variant, same launch
    # configuration, timed the same way and compared with the FP64 image of the timed steps
    fp32 = None
    if args.model == "riaf" and not args.no_fp32_variant and args.precision == "fp64":
        ref_img = out["image"].clone()
        out32 = ody.render_image(sc, mo, nu, precision=ody.PREC_MIXED_FP32)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            ody.render_image(sc, mo, nu, out=out32, precision=ody.PREC_MIXED_FP32)
        e1.record()
        torch.cuda.synchronize()
        diff = (out32["image"] - ref_img).abs()
        l1 = float(diff.sum() / ref_img.sum())
        mask = ref_img >= 1e-6 * ref_img.max()
        mx = float((diff[mask] / ref_img[mask]).max())
        fp32 = {"ms_per_step": e0.elapsed_time(e1) / args.steps, "rel_l1_vs_fp64": l1, "max_rel_vs_fp64": mx,
                "flags_equal": bool(torch.equal(out32["flag"], out["flag"])),
                "inside_tolerance": bool(l1 <= 1e-6 and mx <= 1e-4),
                "what": "FP32 polynomial cores of exp / expm1 / log / K_2 in the transfer block; geodesic, exponent "
                        "sums and accumulators FP64 (DESIGN.md 8.1)"}

    # ---- end to end through the host-buffer C-ABI call (device alloc + kernel + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        # pinned host buffers for every output of the call (numpy views of page-locked torch tensors)
        ny, nx = sc["ny"], sc["nx"]
        pinned = {k: torch.empty((ny, nx), dtype=dt, pin_memory=True) for k, dt in (
            ("image", torch.float64), ("aux0", torch.float64), ("aux1", torch.float64),
            ("flag", torch.int32), ("n_attempt", torch.int32), ("n_accept", torch.int32))}
        host = {k: v.numpy() for k, v in pinned.items()}
        host["hist"] = None
        ody.render_image_host(sc, mo, nu, out=host)                  # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            ody.render_image_host(sc, mo, nu, out=host)
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        d2h = sum(v.nbytes for v in host.values() if v is not None)
        h2d = 120 + 184 + 8                                           # the two structs and nu_hz (kernel parameters)
        e2e = (e2e_s, d2h, h2d, int(host["n_attempt"].astype("int64").sum()))

    # ---- reduce over ranks: time = max, work = sum
    (total_ms_max, e2e_s_max), (attempts_all, accepts_all, rays_all, launches_all) = reduce_over_ranks(
        dist, "cuda", [total_ms, e2e[0] if e2e else 0.0], [attempts, accepts, rays, launches])
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    head = headline(total_ms_max, args.steps, attempts_all, accepts_all, world)
    ms_per_step, value = head["ms_per_step"], head["value"]
    counts = load_counts()
    flop_geo = counts["flop_per_attempt_geodesic"]
    flop_rt = counts["flop_per_rt_update"] if args.model == "riaf" else 0.0
    flop_step = flop_geo * attempts + flop_rt * accepts                                # per launch (this rank)
    kernel_ms = sum(step_ms) / len(step_ms)
    achieved = flop_step / (kernel_ms * 1e-3) / 1e12
    hand = (HAND_FLOP_PER_ATTEMPT * attempts + (HAND_FLOP_PER_RT_UPDATE if args.model == "riaf" else 0.0) * accepts) / (kernel_ms * 1e-3) / 1e12
    cap = counts["fused_kernel" if args.model == "riaf" else "geodesic_kernel"]
    headline_workload = args.n == 4096 and args.a == 0.998
    info = ody.kernel_info(mo["kind"], False, sc["tableau"])
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": False, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if args.precision == "fp64" else "f64 geodesic + f32 transfer cores", "data": "synthetic",
        "config": {"workload": workload_name(args.n, args.a, args.model), "photons_per_step": int(rays_all),
                   "attempted_rk_steps_per_step": int(attempts_all), "accepted_rk_steps_per_step": int(accepts_all),
                   "attempts_per_photon": attempts_all / rays_all,
                   "l2": "no input arrays (rays are generated from the pixel index); the %d MB of per-step "
                         "outputs exceed the 126 MB L2" % (out_bytes >> 20),
                   "parallelism": "replicas" if world > 1 else "single GPU"},
        "images_per_s": head["images_per_s"],
        "ns_per_photon_per_accepted_step": head["ns_per_photon_per_accepted_step"],
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                     "frac": achieved / peak_tflops,
                     "what": "EXECUTED FP64 flop (2 x DFMA + DMUL + DADD thread instructions, ncu) / CUDA-event kernel time / DFMA peak",
                     "traffic": cap["dram_bytes"] if headline_workload else None,
                     "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
                     "kernel": cap["kernel"], "kernel_ms": kernel_ms,
                     "flop_per_attempt": flop_geo, "flop_per_rt_update": flop_rt,
                     "counts_file": os.path.relpath(COUNTS_FILE, ROOT), "counts_source_hash": counts["source_hash"],
                     "stale": bool(counts["stale"]),
                     "warp_execution_efficiency": cap["warp_execution_efficiency"],
                     "fp64_pipe_utilisation": cap["fp64_pipe_utilisation"],
                     "fp64_share_of_warp_instructions": cap["fp64_share_of_warp_instructions"],
                     "spill_bytes": info["local_bytes"], "local_load_store_instructions_executed": cap["local_load_store_instructions"],
                     "frac_hand_count": hand / peak_tflops,
                     "hand_count": "SURVEY.md 8(d) a-priori count, 1500 flop per attempt + 490 per transfer update: context, not the headline",
                     "peak_source": "odyssey_fp64_peak_probe (DFMA microbenchmark) in this run, best of 5"},
        "kernel_info": info,
        "gpu_launches": int(launches_all),
        "clocks": clocks,
        "paper_context": "~1 ns per photon per RK step claimed on a GTX 780 Ti (FP64, geodesics only); "
                         "its Table 1 gives 25732 ms / 1.578e9 steps = 16.3 ns at 1024^2",
    }
    if fp32:
        fp32["value"] = fp32["ms_per_step"] * 1e6 / attempts
        fp32["unit"] = UNIT
        fp32["speedup_vs_fp64"] = kernel_ms / fp32["ms_per_step"]
        line["fp32_variant"] = fp32
    if e2e:
        _, d2h, h2d, att_host = e2e
        line["e2e"] = {"value": e2e_s_max / args.steps * 1e9 / (att_host * world), "unit": UNIT,
                       "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                       "ms_per_step": e2e_s_max / args.steps * 1e3,
                       "api": "odyssey_render_image_host (pinned host buffers; device scratch, kernel and D2H copies "
                              "of all six output arrays inside the timed region)"}
    if not args.no_extra and world == 1:
        line["extra"] = {"configs": time_extra_configs(ody, torch),
                         "note": "device time per call, CUDA events, median of 3 after one warm-up, outside the headline's timed region; "
                                 "C3 = 32 frequencies per photon-step (two-phase spectrum path); BASELINE.json:configs[0..4]"}
    if not args.no_cpu_baseline and world == 1:                       # the oracle leg runs at N = 1 only
        from oracle import build as oracle_build
        oracle_build.build()
        line["cpu_baseline"] = cpu_baseline(w, args.cpu_sample)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
