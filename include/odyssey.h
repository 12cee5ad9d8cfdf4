/* odyssey.h — C ABI of the B200-native Odyssey hot path (arXiv 1601.02063).
 *
 * One image-plane pixel = one photon traced backwards from the observer through Kerr spacetime in
 * Boyer–Lindquist coordinates (§2.1, eqs. (1)-(15)), initial conditions
 * of PAPER.md §2.2 (eqs. (18)-(26)), adaptive embedded 5th-order Runge–Kutta
 * (PAPER.md:L90), with the radiative transfer of PAPER.md §2.3 (eqs. (2), (27)-(31),
 * PAPER.md:L42-46, L149-171) advanced once per accepted step.  Every step of that path runs in the
 * sm_100a kernels of paper_1601_02063_b200/csrc/; there is no CPU fallback.
 *
 * Conventions common to all calls
 *   - Units: G = c = M = 1 for geometry; cgs for radiative quantities.
 *   - Pixel grid: pixel (i, j), 0 <= i < nx, 0 <= j < ny, has image-plane coordinates
 *       x = x_min + (i + 1/2)(x_max - x_min)/nx   (alpha, to the observer's right),
 *       y = y_min + (j + 1/2)(y_max - y_min)/ny   (beta, along the projected spin axis);
 *     per-pixel arrays are row-major [j][i] (index j*nx + i), structure-of-arrays, one array per
 *     quantity.  Per-frequency images are [k][j][i].
 *   - DEVICE entry points (no suffix): every output pointer is a caller-owned DEVICE buffer on the
 *     current CUDA device; a NULL output pointer means "do not write this quantity".  The call
 *     enqueues its work on `cuda_stream` (a cudaStream_t passed as void*, NULL = default stream)
 *     and returns without synchronising; the caller synchronises before reading.
 *   - HOST entry points (suffix _host): same arguments but every output pointer is HOST memory; the
 *     call allocates device scratch, runs the same kernels, copies the results back and returns
 *     after the copies have completed (synchronous).  odyssey_trace_geodesics_host and odyssey_render_image_host
 *     render images of 2^21 pixels and more in up to 16 bands of whole rows that alternate between two streams
 *     of the library's own, so that a band's device->host copies run under the next band's kernel (pinned host
 *     buffers make the copies asynchronous; pageable ones still work); every pixel is bit-identical to the
 *     DEVICE call's.  Concurrent _host calls from several host threads share those two streams.
 *   - The structs and the frequency list are always HOST memory, read during the call only.
 *   - Return value: ODYSSEY_OK (0) or a negative odyssey_status.  After a failure
 *     odyssey_last_error() returns a static, thread-local, NUL-terminated description.
 *     Nothing is printed, nothing throws.
 *   - Scratch: every launch takes what it needs — its work-queue counter, one stash of 32 prepared rays per
 *     warp of the grid (~5 MB in all, whatever the image size), in spectrum mode the per-frequency accumulators
 *     or node lists described there — from a stream-ordered memory pool of the library's own (created lazily per
 *     device, cudaMallocFromPoolAsync / cudaFreeAsync on `cuda_stream`; cached blocks above 12 GiB go back to the
 *     driver at the next synchronisation; odyssey_trim_scratch() returns more, odyssey_shutdown() everything).
 *     Nothing is shared between launches, so any number of calls may be in flight on any number of streams.
 *   - One kernel launch of this library per call (the persistent integrator builds the initial conditions of its
 *     rays itself, a queue tile of 32 pixels at a time); more in spectrum mode.
 *   - All of that is stream-ordered, so a DEVICE call may be captured into a CUDA graph and replayed.  The exception
 *     is the two-phase path of odyssey_render_spectrum, which synchronises the stream inside the call.
 */
#ifndef ODYSSEY_H_
#define ODYSSEY_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum odyssey_status {
    ODYSSEY_OK = 0,
    ODYSSEY_ERR_INVALID_ARGUMENT = -1, /* |a| >= 1, nx/ny <= 0, rtol <= 0, nf outside [1,32], unknown kind/tableau, NULL struct */
    ODYSSEY_ERR_CUDA = -2,             /* a CUDA runtime call or the launch failed; text in odyssey_last_error() */
    ODYSSEY_ERR_UNSUPPORTED_DEVICE = -3 /* current device is not compute capability 10.x */
} odyssey_status;

/* Ray outcome written to `flag` ("captured"; L223 disk; BASELINE.json:configs[2] optical depth). */
enum {
    ODYSSEY_FLAG_ESCAPED = 0,  /* p_r > 0 and r >= r_esc; final state located ON r = r_esc          */
    ODYSSEY_FLAG_CAPTURED = 1, /* r <= r_h + horizon_eps; final state located ON that radius         */
    ODYSSEY_FLAG_DISK = 2,     /* kinds 1, 3: first equatorial crossing with r_in <= r <= r_out       */
    ODYSSEY_FLAG_OPAQUE = 3,   /* kind 2: every frequency has tau > tau_max                           */
    ODYSSEY_FLAG_MAXSTEP = 4   /* max_attempts Runge–Kutta attempts used                              */
};

enum { ODYSSEY_TABLEAU_RKF45 = 0, ODYSSEY_TABLEAU_CASH_KARP = 1 };
enum { ODYSSEY_KIND_NONE = 0, ODYSSEY_KIND_THIN_DISK = 1, ODYSSEY_KIND_RIAF = 2, ODYSSEY_KIND_HOT_SPOT = 3, ODYSSEY_KIND_NT_DISK = 4 };
/* PAPER.md:L171 says the transfer equations are "easily integrated along with the geodesic … piecewise
 * according to these steps".  PER_STEP (default): one update per accepted step, trapezoid in lambda with
 * the exact attenuation across the step.  RK_COMPONENTS: tau and I as two more components of the
 * Runge–Kutta system (coefficients evaluated at all six stages, fifth-order weights, not in the error
 * norm); single-frequency calls only.                                                              */
enum { ODYSSEY_RT_PER_STEP = 0, ODYSSEY_RT_RK_COMPONENTS = 1 };
/* FP64: everything in double precision (default).  MIXED_FP32: the geodesic, every exponent sum, argument
 * reduction and accumulator stay FP64; the polynomial cores of exp / expm1 / log and the K_2 polynomials of the
 * emissivity run in FP32 (relative error ~1e-7 per coefficient).  Inside the image tolerances and a few per cent
 * faster on B200; not the default: the metric is FP64.                                 */
enum { ODYSSEY_PREC_FP64 = 0, ODYSSEY_PREC_MIXED_FP32 = 1 };
#define ODYSSEY_MAX_FREQ 32

/* The observer, the image plane and the integrator controls. */
typedef struct odyssey_scene {
    double a;                  /* spin, |a| < 1                                                  */
    double r_obs;              /* observer distance (PAPER.md:L106 uses 10^3)                    */
    double theta_obs, phi_obs; /* observer inclination and azimuth, radians                      */
    double x_min, x_max, y_min, y_max; /* image-plane extent (edges, not centres)               */
    int32_t nx, ny;            /* resolution                                                     */
    double rtol;               /* per-step tolerance of the scaled max-norm error                */
    int32_t tableau, pad0;     /* ODYSSEY_TABLEAU_*                                              */
    double h0;                 /* first trial step in affine parameter                           */
    double horizon_eps;        /* capture radius = r_h + horizon_eps                             */
    double r_esc;              /* escape radius; the image-plane corners must satisfy sqrt(x^2 + y^2) <= 0.9 r_esc */
    int32_t max_attempts, pad1;
} odyssey_scene;

/* Emission model (PAPER.md:L223 thin disk; L268-292 thermal synchrotron; BASELINE.json:configs[1..2]). */
typedef struct odyssey_model {
    int32_t kind;              /* ODYSSEY_KIND_*                                                 */
    int32_t nbins;             /* kind 1: number of g bins of the line profile (0 = none)        */
    double r_in, r_out;        /* kind 1: disk radii; r_in <= 0 means r_isco(a)                  */
    double emis_index;         /* kind 1: emissivity ∝ r^-emis_index                             */
    double mbh_msun;           /* kind 2: black-hole mass in solar masses (sets r_g in cm)       */
    double n0, n_index;        /* kind 2: n_e = n0 (r/r_h)^n_index exp(-cos^2θ / (2 h_over_r^2)) */
    double T0, T_index;        /* kind 2: T_e = T0 (r/r_h)^T_index                               */
    double h_over_r, beta;     /* kind 2: scale height, magnetisation B^2/8π = n_e m_p c^2/(6 β r) */
    double r_rt_out;           /* kind 2: no emission outside this radius        */
    double tau_max;            /* kind 2: a frequency is frozen once tau > tau_max               */
    double j_scale;            /* kind 2: 1 = per-steradian emissivity; 4π reproduces eq. (37) as printed */
    double g_lo, g_hi;         /* kind 1: histogram range in g                                   */
    double g_power;            /* kind 1: pixel value = g^g_power r_e^-emis_index                */
    int32_t rt_scheme;         /* kind 2: ODYSSEY_RT_* — how eqs. (30), (31) are advanced along the ray */
    int32_t precision;         /* kind 2: ODYSSEY_PREC_* (single-frequency image calls with ODYSSEY_RT_PER_STEP only) */
    double spot_r_orbit;       /* kind 3: radius of the spot's circular equatorial orbit; <= 0 means r_isco(a)  */
    double spot_size;          /* kind 3: r_spot of eq. (36) (the paper uses 0.5 r_g); emission is cut at 4 r_spot */
    double spot_phi0;          /* kind 3: azimuth of the spot centre at coordinate time t = 0                    */
    double mdot_gs;            /* kind 4: accretion rate in g/s (eq. (35)); uses mbh_msun, r_in (<= 0: r_isco), r_out */
    double dtau_max;           /* kind 2, ODYSSEY_RT_PER_STEP, FP64, odyssey_render_image only: > 0 caps the step that follows an
                                  accepted step at dtau_max optical depths, h <= dtau_max / (absorption coefficient at the point
                                  just reached); <= 0: no cap (the default; the step is controlled by the geodesic alone)   */
} odyssey_model;

/* Geodesics only (BASELINE.json:configs[0]; §2.1-2.2).  Per pixel: outcome flag, the
 * final Boyer–Lindquist position (r, theta, phi) — located on the stopping surface — the coordinate
 * time t elapsed along the ray (eq. (9); counted from 0 at the image plane, negative because
 * the ray is traced backwards; integrated only when t is non-NULL, never part of the error norm) and the
 * number of attempted and accepted Runge–Kutta steps ("total number of steps").  */
int odyssey_trace_geodesics(const odyssey_scene* scene,
                            int32_t* flag, double* r, double* theta, double* phi, double* t,
                            int32_t* n_attempt, int32_t* n_accept, void* cuda_stream);

/* One observed frequency nu_hz (ignored by kind 0/1).
 *   kind 1 (eq. (2)): image = g^g_power r_e^-emis_index, aux0 = g, aux1 = r_e of the
 *     first disk crossing (0 where the ray misses); hist[nbins] += image × pixel area in the bin of g
 *     (hist is overwritten, not accumulated across calls).
 *   kind 2 (eqs. (30),(31),(37)-(39)): image = I_nu = nu^3 × invariant intensity (erg s^-1 cm^-2
 *     Hz^-1 sr^-1), aux0 = optical depth tau, aux1 = 0.
 *   kind 4 (eq. (35)): image = I_nu of the Novikov–Thorne disk at nu_hz (see
 *     odyssey_render_spectrum), aux0 = g, aux1 = r_e as for kind 1.
 *   kind 0: image = aux0 = aux1 = 0; flags and step counts as odyssey_trace_geodesics.
 * n_attempt / n_accept: attempted and accepted Runge–Kutta steps per ray (one radiative-transfer
 * update is made per accepted step).                                               */
int odyssey_render_image(const odyssey_scene* scene, const odyssey_model* model, double nu_hz,
                         double* image, double* aux0, double* aux1, int32_t* flag,
                         int32_t* n_attempt, int32_t* n_accept, double* hist, void* cuda_stream);

/* nf <= 32 observed frequencies integrated simultaneously along each geodesic (kind 2 only;
 * BASELINE.json:configs[3]).  images[nf][ny][nx] = I_nu; nuLnu[nf] = 4π nu r_g^2 Δx Δy Σ_pixels I_nu
 * (erg/s; the distance cancels).  nu_hz_host is HOST memory.  rt_scheme must be ODYSSEY_RT_PER_STEP.
 * Two code paths, same results to rounding: images of up to ~1.5e5 rays, and larger images with nf >= 4, take a
 * two-phase path (record the geodesics once, then one lane per (ray, frequency); larger images band by band); it
 * synchronises `cuda_stream` ONCE per band inside the call to read an overflow flag, and uses stream-ordered scratch
 * (64 KB per ray of a band, ~10 GB at most).  Larger images with fewer frequencies take one fused kernel, no
 * synchronisation.
 *
 * kind 4, the relativistic multi-temperature disk of Novikov & Thorne (eq. (35), Fig. 6): an
 * opaque disk on the equatorial plane between r_in (<= 0: r_isco) and r_out whose surface radiates as a blackbody
 * at T_eff(r), sigma T_eff^4 = 3 Mdot M f(r) / (8 pi r^3) in G = c = 1, f = Page & Thorne's zero-torque function
 * (0 at and inside r_isco).  One geodesic pass; at the first crossing, for every frequency,
 * images[k] = I_nu = (2 h nu^3 / c^2) / expm1(h nu / (g k_B T_eff(r_e))) (the invariance of I_nu / nu^3 with the
 * redshift g of eq. (2)), and nuLnu[k] as above.  No stream synchronisation, no scratch beyond the camera pass. */
int odyssey_render_spectrum(const odyssey_scene* scene, const odyssey_model* model,
                            const double* nu_hz_host, int nf,
                            double* images, double* nuLnu, int32_t* flag, int32_t* n_attempt,
                            void* cuda_stream);

/* Orbiting hot spot (§4.4, eq. (36), Figs. 7-8; kind 3, which also uses kind 1's r_in, r_out,
 * g_power, nbins, g_lo, g_hi).  The spot is a Gaussian patch, exp(-d^2 / 2 spot_size^2) for d < 4 spot_size, on the
 * opaque equatorial plane; its centre moves on the prograde circular orbit of radius spot_r_orbit,
 * phi_s(t) = spot_phi0 + t / (r_s^{3/2} + a).  A ray that reaches the plane at (r_e, phi_e) after the coordinate
 * time t_e (eq. (9); negative, the ray is traced backwards from t = 0 at the image plane) shows the spot as it was
 * at t_obs + t_e; d is measured in the pseudo-Cartesian coordinates of eqs. (33), (34).  For each of the nt <= 32
 * observer times t_obs_host[k] (HOST memory): images[k][ny][nx] = g^g_power exp(-d^2/2 spot_size^2),
 * lightcurve[k] = sum(images[k]) x pixel area, spectrogram[k][nbins] = that flux binned over g (NULL or nbins = 0:
 * skipped).  Per pixel: g, r_e, phi_e, t_e of the crossing (0 where the ray misses the plane), flag, n_attempt. */
int odyssey_render_hotspot(const odyssey_scene* scene, const odyssey_model* model, const double* t_obs_host, int nt,
                           double* images, double* lightcurve, double* spectrogram,
                           double* g, double* r_e, double* phi_e, double* t_e, int32_t* flag, int32_t* n_attempt,
                           void* cuda_stream);

/* Host-buffer variants: identical semantics, every output pointer is HOST memory, synchronous. */
int odyssey_trace_geodesics_host(const odyssey_scene* scene,
                                 int32_t* flag, double* r, double* theta, double* phi, double* t,
                                 int32_t* n_attempt, int32_t* n_accept);
int odyssey_render_image_host(const odyssey_scene* scene, const odyssey_model* model, double nu_hz,
                              double* image, double* aux0, double* aux1, int32_t* flag,
                              int32_t* n_attempt, int32_t* n_accept, double* hist);
int odyssey_render_spectrum_host(const odyssey_scene* scene, const odyssey_model* model,
                                 const double* nu_hz_host, int nf,
                                 double* images, double* nuLnu, int32_t* flag, int32_t* n_attempt);
int odyssey_render_hotspot_host(const odyssey_scene* scene, const odyssey_model* model, const double* t_obs_host, int nt,
                                double* images, double* lightcurve, double* spectrogram,
                                double* g, double* r_e, double* phi_e, double* t_e, int32_t* flag, int32_t* n_attempt);

/* FP64 peak probe (BASELINE.json:north_star "measured by a DFMA microbenchmark in the same run"):
 * enqueues a kernel in which every thread runs `iters` rounds of 16 independent DFMA chains
 * on a full-occupancy grid.  *flop_host receives the number of floating-point operations the launch
 * performs (2 per DFMA); sink is a DEVICE buffer of at least 8 bytes.  The caller times it.     */
int odyssey_fp64_peak_probe(int iters, double* sink, double* flop_host, void* cuda_stream);

/* Kernel facts for reports: registers per thread, local (spill) bytes per thread, static shared
 * bytes, threads per block and resident blocks per SM of the kernel that serves (kind, nf > 1).  */
int odyssey_kernel_info(int kind, int spectrum, int tableau, int32_t* regs, int32_t* local_bytes,
                        int32_t* threads_per_block, int32_t* blocks_per_sm, int32_t* n_sm);

/* Diagnostic: evaluate one of the kernels' own FP64 elementary functions (csrc/dmath.cuh) elementwise on
 * n DEVICE doubles: op 0 1/x, 1 x^-1/2, 2 sqrt, 3 sincos (y = sin, y2 = cos), 4 exp, 5 expm1, 6 log,
 * 7 K_2(x) of eq. (37), 8 / 9 the raw hardware seeds of 1/x and x^-1/2.  y2 may be NULL except for op 3.  Used by the tests to check the
 * device arithmetic against libm / scipy on its own, apart from the ray-level parity tests.       */
int odyssey_eval_math(int op, int n, const double* x, double* y, double* y2, void* cuda_stream);

/* Number of kernel launches issued by this library since load (for bench.py's gpu_launches). */
long long odyssey_launch_count(void);

/* Synchronises the current device and returns the library's cached scratch above keep_bytes to the driver
 * (e.g. 0 after a large two-phase spectrum call, before another library needs the memory). */
int odyssey_trim_scratch(unsigned long long keep_bytes);

const char* odyssey_last_error(void);
void odyssey_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* ODYSSEY_H_ */
