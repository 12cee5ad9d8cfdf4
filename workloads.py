"""Deterministic workload definitions C0..C4 (BASELINE.json:configs[0..4]).

This module is the ONLY thing the CPU oracle (`oracle/`) and the CUDA path
(`paper_1601_02063_b200/`) have in common.  It holds plain numbers — scene and model
parameters as dictionaries — and none of the method's arithmetic: no geodesic, no
radiative-transfer, no camera formula lives here.  Every input of the hot path is
generated from (pixel index, these constants); there are no random numbers and no
datasets (rays start on a regular image-plane grid).

Keys mirror the paper's problem statement:
  scene: spin a; observer r_obs, theta_obs, phi_obs; image-plane
         extent and resolution; integrator controls.
  model: emission model parameters (PAPER.md:L223 thin disk; L268-292 synchrotron shell,
         with BASELINE.json:configs[2]'s RIAF profile).
"""
import math

# Flags written per ray (same numbering on both sides; it is part of the output contract).
FLAG_ESCAPED, FLAG_CAPTURED, FLAG_DISK, FLAG_OPAQUE, FLAG_MAXSTEP = 0, 1, 2, 3, 4

KIND_NONE, KIND_THIN_DISK, KIND_RIAF, KIND_HOT_SPOT, KIND_NT_DISK = 0, 1, 2, 3, 4
# How eqs. (30), (31) are advanced (readings E, E'): one exact-attenuation update per accepted
# step (default), or tau and I as two more Runge-Kutta components through the six stages.
RT_PER_STEP, RT_RK_COMPONENTS = 0, 1
TABLEAU_RKF45, TABLEAU_CASH_KARP = 0, 1


def scene(a, incl_deg, n, half_width, *, r_obs=1000.0, rtol=1e-8, tableau=TABLEAU_RKF45,
          ny=None, max_attempts=100000):
    """Scene dictionary.  Pixel centres, x = alpha ascending with i, y = beta ascending with j."""
    return dict(a=float(a), r_obs=float(r_obs), theta_obs=math.radians(incl_deg), phi_obs=0.0,
                x_min=-float(half_width), x_max=float(half_width),
                y_min=-float(half_width), y_max=float(half_width),
                nx=int(n), ny=int(n if ny is None else ny),
                rtol=float(rtol), tableau=int(tableau),
                h0=1.0, horizon_eps=1e-3, r_esc=float(r_obs), max_attempts=int(max_attempts))


def model_none():
    return dict(kind=KIND_NONE, r_in=0.0, r_out=0.0, emis_index=0.0,
                mbh_msun=0.0, n0=0.0, n_index=0.0, T0=0.0, T_index=0.0, h_over_r=1.0, beta=1.0,
                r_rt_out=0.0, tau_max=0.0, j_scale=1.0,
                nbins=0, g_lo=0.0, g_hi=1.0, g_power=0.0, rt_scheme=RT_PER_STEP,
                spot_r_orbit=0.0, spot_size=0.0, spot_phi0=0.0, mdot_gs=0.0, dtau_max=0.0)


def model_thin_disk(r_in=0.0, r_out=50.0, emis_index=3.0, nbins=200, g_lo=0.0, g_hi=2.0, g_power=3.0):
    """Keplerian thin disk r_isco..50 M, emissivity ∝ r^-3 (BASELINE.json:configs[1]).
    r_in <= 0 means r_isco of the scene's spin."""
    m = model_none()
    m.update(kind=KIND_THIN_DISK, r_in=float(r_in), r_out=float(r_out), emis_index=float(emis_index),
             nbins=int(nbins), g_lo=float(g_lo), g_hi=float(g_hi), g_power=float(g_power))
    return m


def model_hot_spot(r_orbit=0.0, r_spot=0.5, phi0=0.0, r_in=0.0, r_out=50.0, g_power=4.0, nbins=100, g_lo=0.0, g_hi=2.0):
    """Keplerian hot spot on the opaque equatorial plane (eq. (36)): Gaussian of width r_spot
    = 0.5 r_g, cut at 4 r_spot, orbiting at r_orbit (<= 0: r_isco of the scene's spin), azimuth phi0 at t = 0."""
    m = model_none()
    m.update(kind=KIND_HOT_SPOT, r_in=float(r_in), r_out=float(r_out), g_power=float(g_power), nbins=int(nbins),
             g_lo=float(g_lo), g_hi=float(g_hi), spot_r_orbit=float(r_orbit), spot_size=float(r_spot), spot_phi0=float(phi0))
    return m


def model_nt_disk(mbh_msun=10.0, mdot_gs=1.0e19, r_in=0.0, r_out=50.0):
    """Novikov-Thorne multi-temperature disk, eq. (35) (Fig. 6 uses M = 10 M_sun,
    Mdot = 1e19 g/s, r_out = 50 or 500 r_g)."""
    m = model_none()
    m.update(kind=KIND_NT_DISK, mbh_msun=float(mbh_msun), mdot_gs=float(mdot_gs), r_in=float(r_in), r_out=float(r_out))
    return m


def model_riaf(mbh_msun=4.0e6, n0=1.0e7, n_index=-1.1, T0=1.0e11, T_index=-0.84, h_over_r=0.3,
               beta=10.0, r_rt_out=500.0, tau_max=30.0, j_scale=1.0, rt_scheme=RT_PER_STEP, dtau_max=0.0):
    """Analytic RIAF-like flow of BASELINE.json:configs[2]; mass and outer radius from PAPER.md:L292."""
    m = model_none()
    m.update(kind=KIND_RIAF, mbh_msun=float(mbh_msun), n0=float(n0), n_index=float(n_index),
             T0=float(T0), T_index=float(T_index), h_over_r=float(h_over_r), beta=float(beta),
             r_rt_out=float(r_rt_out), tau_max=float(tau_max), j_scale=float(j_scale), rt_scheme=int(rt_scheme),
             dtau_max=float(dtau_max))
    return m


def log_spaced_frequencies(nu_lo=1.0e9, nu_hi=1.0e15, nf=32):
    """nf frequencies log-spaced from nu_lo to nu_hi inclusive (BASELINE.json:configs[3])."""
    if nf == 1:
        return [float(nu_lo)]
    return [float(nu_lo) * (float(nu_hi) / float(nu_lo)) ** (k / (nf - 1)) for k in range(nf)]


def C0(n=64, rtol=1e-8):
    """Geodesics only, Schwarzschild, 64x64 over +/-10 M, i = 60 deg (BASELINE.json:configs[0])."""
    return dict(name="C0", scene=scene(0.0, 60.0, n, 10.0, rtol=rtol), model=model_none(), nu=[])


def C1(n=512, rtol=1e-8):
    """Kerr a=0.9, i=60 deg, 512^2 over +/-20 M, thin disk line image (BASELINE.json:configs[1])."""
    return dict(name="C1", scene=scene(0.9, 60.0, n, 20.0, rtol=rtol), model=model_thin_disk(), nu=[])


def C2(n=1024, rtol=1e-8):
    """Kerr a=0.9375, i=30 deg, 1024^2 over +/-15 M, RIAF GRRT at 230 GHz (BASELINE.json:configs[2])."""
    return dict(name="C2", scene=scene(0.9375, 30.0, n, 15.0, rtol=rtol), model=model_riaf(), nu=[230.0e9])


def C3(n=256, rtol=1e-8, nf=32):
    """Spectrum mode: C2's flow and spin, 256^2, 32 frequencies 1e9..1e15 Hz (BASELINE.json:configs[3])."""
    return dict(name="C3", scene=scene(0.9375, 30.0, n, 15.0, rtol=rtol), model=model_riaf(),
                nu=log_spaced_frequencies(nf=nf))


def C4(n=4096, a=0.998, rtol=1e-8):
    """Throughput stress: a=0.998, i=85 deg, 4096^2 over +/-15 M, RIAF at 230 GHz (BASELINE.json:configs[4])."""
    return dict(name="C4", scene=scene(a, 85.0, n, 15.0, rtol=rtol), model=model_riaf(), nu=[230.0e9])


def coarse_scene(sc, n_sub):
    """The same image plane sampled on a coarser n_sub x n_sub grid of pixel centres (used to time
    the oracle on a bounded sample of a large workload; ns per photon per RK step does not depend
    on the sampling density)."""
    out = dict(sc)
    out.update(nx=int(n_sub), ny=int(n_sub))
    return out


def subgrid_indices(sc, n_sub):
    """Pixel indices (i, j) of an n_sub x n_sub strided subset of sc's pixels, row-major.
    Pure indexing: each side turns (i, j) into image-plane coordinates itself."""
    sx, sy = sc["nx"] // n_sub, sc["ny"] // n_sub
    ii, jj = [], []
    for q in range(n_sub):
        for p in range(n_sub):
            ii.append(p * sx + sx // 2)
            jj.append(q * sy + sy // 2)
    return ii, jj
