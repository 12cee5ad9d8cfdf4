// odyssey_api.cu — the C ABI of include/odyssey.h: argument checks, the constant block, launches.
// No torch types, no CPU fallback: every entry point either enqueues the sm_100a kernels of
// odyssey_kernels.cuh or returns an error code.
#include <cuda_runtime.h>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "../../include/odyssey.h"
#include "odyssey_kernels.cuh"

namespace {

using namespace ody;

// ---- physical constants, cgs (CODATA 2018; IAU nominal GM_sun) ---------------------------------
constexpr double kC = 2.99792458e10, kGMsun = 1.3271244e26, kH = 6.62607015e-27, kKB = 1.380649e-16;
constexpr double kMe = 9.1093837015e-28, kMp = 1.67262192369e-24, kE = 4.80320471257e-10;
constexpr double kPi = 3.14159265358979323846;
constexpr double kG = 6.67430e-8, kSigmaSB = 5.670374419e-5;

thread_local char g_err[512] = "";
std::atomic<long long> g_launches{0};

int fail(int code, const char* fmt, ...) {
    va_list ap; va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define TRY_RC(expr) do { int rc_ = (expr); if (rc_) return rc_; } while (0)
#define CUDA_TRY(expr)                                                                             \
    do { cudaError_t e_ = (expr);                                                                  \
         if (e_ != cudaSuccess) return fail(ODYSSEY_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); } while (0)

// ---- per-device library state: SM count ---------------------------------------------------------
// (Every launch takes its work-queue counter and the warps' ray stashes from stream-ordered scratch of its own, so
// any number of calls may be in flight on any number of streams, and a captured graph owns what it captured.)
constexpr int MAX_DEV = 16;
struct DevState {
    bool ready = false; int n_sm = 0; cudaMemPool_t pool = nullptr;
    cudaStream_t band_stream[2] = {nullptr, nullptr};      // the _host variants' two pipeline streams (created on first use)
    cudaEvent_t band_event[3] = {nullptr, nullptr, nullptr};
};
DevState g_dev[MAX_DEV];
std::mutex g_mu;

int device_state(DevState** out, int* dev_out) {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEV) return fail(ODYSSEY_ERR_CUDA, "device index %d out of range", dev);
    std::lock_guard<std::mutex> lk(g_mu);
    DevState& D = g_dev[dev];
    if (!D.ready) {
        cudaDeviceProp prop;
        CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
        if (prop.major != 10)
            return fail(ODYSSEY_ERR_UNSUPPORTED_DEVICE, "device %d is sm_%d%d; this library is built for sm_100a only", dev, prop.major, prop.minor);
        D.n_sm = prop.multiProcessorCount;
        // Stream-ordered scratch (queue counters, ray stashes, spectrum accumulators and node lists, the _host variants'
        // device buffers) comes from a memory pool of the library's OWN, which keeps freed blocks cached instead of
        // returning them to the driver at every synchronisation; the device's default pool, which belongs to the host
        // application, is not touched.
        cudaMemPoolProps props;
        std::memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        CUDA_TRY(cudaMemPoolCreate(&D.pool, &props));
        // cached scratch above 12 GiB goes back to the driver at the next synchronisation (a band of the two-phase spectrum
        // path holds ~10 GB of node lists and synchronises once per band: a lower threshold would re-allocate them every band)
        unsigned long long keep = 12ull << 30;
        CUDA_TRY(cudaMemPoolSetAttribute(D.pool, cudaMemPoolAttrReleaseThreshold, &keep));
        D.ready = true;
    }
    *out = &D; if (dev_out) *dev_out = dev;
    return ODYSSEY_OK;
}

// stream-ordered allocation from the library's pool on the current device
cudaError_t pool_alloc(void** ptr, size_t bytes, cudaStream_t st) {
    DevState* D = nullptr;
    if (device_state(&D, nullptr) != ODYSSEY_OK) return cudaErrorInitializationError;
    return cudaMallocFromPoolAsync(ptr, bytes, D->pool, st);
}
// give cached blocks above `keep_bytes` back to the driver (after the calls that take gigabytes of scratch)
void pool_trim(size_t keep_bytes) {
    DevState* D = nullptr;
    if (device_state(&D, nullptr) == ODYSSEY_OK && D->pool) cudaMemPoolTrimTo(D->pool, keep_bytes);
}

// ---- Kerr constants (Bardeen, Press & Teukolsky 1972, cited PAPER.md:L223) -----------------------
double isco_radius(double a) {
    const double z1 = 1.0 + std::cbrt(1.0 - a * a) * (std::cbrt(1.0 + a) + std::cbrt(1.0 - a));
    const double z2 = std::sqrt(3.0 * a * a + z1 * z1);
    return 3.0 + z2 - (a >= 0.0 ? 1.0 : -1.0) * std::sqrt((3.0 - z1) * (3.0 + z1 + 2.0 * z2));
}

int check_scene(const odyssey_scene* S) {
    if (!S) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "scene is NULL");
    if (!(std::fabs(S->a) < 1.0)) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "spin |a| = %g must be < 1", S->a);
    if (S->nx <= 0 || S->ny <= 0) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nx = %d, ny = %d must be positive", S->nx, S->ny);
    if ((long long)S->nx * S->ny > (1LL << 30)) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nx*ny exceeds 2^30 pixels");
    if (!(S->rtol > 0.0)) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "rtol = %g must be > 0", S->rtol);
    if (S->tableau != ODYSSEY_TABLEAU_RKF45 && S->tableau != ODYSSEY_TABLEAU_CASH_KARP)
        return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "unknown tableau %d", S->tableau);
    if (!(S->r_obs > 0.0) || !(S->h0 > 0.0) || !(S->r_esc > 0.0) || !(S->horizon_eps >= 0.0) || S->max_attempts <= 0)
        return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "r_obs, h0, r_esc, max_attempts must be positive and horizon_eps >= 0");
    if (S->max_attempts >= (1 << FIFO_ACC_BITS)) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "max_attempts = %d must be below 2^%d", S->max_attempts, FIFO_ACC_BITS);
    if (!(std::fabs(std::sin(S->theta_obs)) > 1e-10))
        return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "observer on the spin axis (theta_obs = %g): the Boyer-Lindquist azimuth of the ray through the image centre is undefined; tilt by >= 1e-9 rad", S->theta_obs);
    if (!(S->x_max > S->x_min) || !(S->y_max > S->y_min))
        return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "image-plane extent is empty");
    {   // every ray must come back out through r = r_esc: a ray whose impact parameter exceeds r_esc turns around
        // outside the escape sphere and its "escape point" (located by Newton iteration on r = r_esc) does not exist
        const double xm = std::fmax(std::fabs(S->x_min), std::fabs(S->x_max)), ym = std::fmax(std::fabs(S->y_min), std::fabs(S->y_max));
        const double b_corner = std::sqrt(xm * xm + ym * ym);
        if (!(b_corner <= 0.9 * S->r_esc))
            return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "image-plane extent: corner impact parameter %g exceeds 0.9 r_esc = %g", b_corner, 0.9 * S->r_esc);
    }
    return ODYSSEY_OK;
}

int check_model(const odyssey_model* M) {
    if (!M) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "model is NULL");
    if (M->kind < ODYSSEY_KIND_NONE || M->kind > ODYSSEY_KIND_NT_DISK) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "unknown model kind %d", M->kind);
    if (M->kind == ODYSSEY_KIND_HOT_SPOT) {
        if (!(M->spot_size > 0.0)) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "spot_size = %g must be > 0", M->spot_size);
        if (M->spot_r_orbit > 0.0 && !(M->spot_r_orbit > 1.0))
            return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "spot_r_orbit = %g must lie outside the horizon (or be <= 0 for r_isco)", M->spot_r_orbit);
    }
    if (M->kind == ODYSSEY_KIND_THIN_DISK || M->kind == ODYSSEY_KIND_HOT_SPOT) {
        if (M->nbins < 0 || M->nbins > 4096) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nbins = %d outside [0, 4096]", M->nbins);
        if (M->nbins > 0 && !(M->g_hi > M->g_lo)) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "g_hi must exceed g_lo");
    }
    if (M->kind == ODYSSEY_KIND_NT_DISK) {
        if (!(M->mbh_msun > 0.0) || !(M->mdot_gs >= 0.0) || !(M->r_out > 0.0))
            return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "Novikov-Thorne disk needs mbh_msun > 0, mdot_gs >= 0, r_out > 0");
    }
    if (M->kind == ODYSSEY_KIND_RIAF) {
        if (M->rt_scheme != ODYSSEY_RT_PER_STEP && M->rt_scheme != ODYSSEY_RT_RK_COMPONENTS)
            return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "unknown rt_scheme %d", M->rt_scheme);
        if (M->precision != ODYSSEY_PREC_FP64 && M->precision != ODYSSEY_PREC_MIXED_FP32)
            return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "unknown precision %d", M->precision);
        if (M->precision == ODYSSEY_PREC_MIXED_FP32 && M->rt_scheme != ODYSSEY_RT_PER_STEP)
            return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "precision MIXED_FP32 needs rt_scheme PER_STEP");
        if (M->dtau_max > 0.0 && (M->rt_scheme != ODYSSEY_RT_PER_STEP || M->precision != ODYSSEY_PREC_FP64))
            return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "dtau_max > 0 needs rt_scheme PER_STEP and precision FP64");
        if (!(M->mbh_msun > 0.0) || !(M->h_over_r > 0.0) || !(M->beta > 0.0) || !(M->T0 > 0.0) || !(M->n0 >= 0.0) ||
            !(M->j_scale >= 0.0))
            return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "RIAF parameters mbh_msun, h_over_r, beta, T0 must be positive, n0 and j_scale non-negative");
    }
    return ODYSSEY_OK;
}

void fill_params(const odyssey_scene& S, const odyssey_model* M, const double* nu, int nf, Params* P) {
    std::memset(P, 0, sizeof(*P));
    P->a = S.a; P->a2 = S.a * S.a;
    P->r_obs = S.r_obs; P->R_obs = std::sqrt(S.r_obs * S.r_obs + S.a * S.a);
    P->sin_obs = std::sin(S.theta_obs); P->cos_obs = std::cos(S.theta_obs);
    P->sin_pobs = std::sin(S.phi_obs); P->cos_pobs = std::cos(S.phi_obs); P->phi_obs = S.phi_obs;
    P->x_min = S.x_min; P->x_span = S.x_max - S.x_min; P->y_min = S.y_min; P->y_span = S.y_max - S.y_min;
    P->pix_area = (P->x_span / S.nx) * (P->y_span / S.ny);
    P->rtol = S.rtol; P->inv_rtol = 1.0 / S.rtol; P->h0 = S.h0;
    P->r_h = 1.0 + std::sqrt(1.0 - S.a * S.a);
    P->r_cap = P->r_h + S.horizon_eps; P->r_esc = S.r_esc;
    P->nx = S.nx; P->ny = S.ny; P->max_attempts = S.max_attempts;
    P->row0 = 0; P->ny_image = S.ny;
    P->tiles_x = (S.nx + TILE_W - 1) / TILE_W;
    const long long tiles_y = (S.ny + TILE_H - 1) / TILE_H;
    P->n_queue = (long long)P->tiles_x * tiles_y * (TILE_W * TILE_H);
    // circular equatorial orbit at the ISCO: specific energy and angular momentum
    P->r_isco = isco_radius(S.a);
    {
        const double r = P->r_isco, sr = std::sqrt(r);
        const double den = std::pow(r, 0.75) * std::sqrt(r * sr - 3.0 * sr + 2.0 * S.a);
        P->E_isco = (r * sr - 2.0 * sr + S.a) / den;
        P->L_isco = (r * r - 2.0 * S.a * sr + S.a * S.a) / den;
    }
    P->kind = M ? M->kind : 0;
    P->nf = nf;
    if (!M) return;
    if (M->kind == ODYSSEY_KIND_HOT_SPOT) {
        const double rs = (M->spot_r_orbit > 0.0) ? M->spot_r_orbit : P->r_isco;
        P->spot_R = std::sqrt(rs * rs + S.a * S.a);
        P->spot_Omega = 1.0 / (rs * std::sqrt(rs) + S.a);
        P->spot_phi0 = M->spot_phi0;
        P->spot_inv2s2 = 1.0 / (2.0 * M->spot_size * M->spot_size);
        P->spot_cut2 = 16.0 * M->spot_size * M->spot_size;
        for (int k = 0; k < nf && k < MAX_FREQ; ++k) P->nu[k] = nu[k];          // the observer times t_obs[k]
    }
    if (M->kind == ODYSSEY_KIND_NT_DISK) {
        // Page & Thorne's f(r) (emission.cuh: nt_temperature): roots of x³ - 3x + 2a and their weights
        const double th = std::acos(S.a) / 3.0;
        const double x[3] = {2.0 * std::cos(th - kPi / 3.0), 2.0 * std::cos(th + kPi / 3.0), -2.0 * std::cos(th)};
        for (int i = 0; i < 3; ++i) {
            const double xi = x[i], xj = x[(i + 1) % 3], xk = x[(i + 2) % 3];
            P->nt_x[i] = xi;
            P->nt_c[i] = 3.0 * (xi - S.a) * (xi - S.a) / (xi * (xi - xj) * (xi - xk));
        }
        P->nt_x0 = std::sqrt(P->r_isco);
        const double Mg = kGMsun * M->mbh_msun / kG;                                   // grams
        P->nt_T4 = 3.0 * M->mdot_gs * std::pow(kC, 6) / (8.0 * kPi * kG * kG * Mg * Mg * kSigmaSB);
        P->h_over_k = kH / kKB;
        P->planck2 = 2.0 * kH / (kC * kC);
        P->r_in = (M->r_in > 0.0) ? M->r_in : P->r_isco;
        P->r_out = M->r_out;
        P->rg_cm = kGMsun * M->mbh_msun / (kC * kC);
        P->sed_coef = 4.0 * kPi * P->rg_cm * P->rg_cm * P->pix_area;
        for (int k = 0; k < nf && k < MAX_FREQ; ++k) { P->nu[k] = nu[k]; P->nu3[k] = nu[k] * nu[k] * nu[k]; }
    }
    if (M->kind == ODYSSEY_KIND_THIN_DISK || M->kind == ODYSSEY_KIND_HOT_SPOT) {
        P->r_in = (M->r_in > 0.0) ? M->r_in : P->r_isco;
        if (M->kind == ODYSSEY_KIND_HOT_SPOT && !(M->r_in > 0.0)) {
            // reading HS: the plane is opaque (and lit) down to the inner edge of the spot, 4 r_spot inside its centre
            // in the pseudo-Cartesian radius of eqs. (33), (34), so that the whole Gaussian of PAPER.md:L259 is seen
            const double R_in = P->spot_R - 4.0 * M->spot_size;
            P->r_in = (R_in > std::fabs(S.a)) ? std::sqrt(R_in * R_in - S.a * S.a) : 0.0;
        }
        P->r_out = M->r_out; P->emis_index = M->emis_index; P->g_power = M->g_power;
        P->g_lo = M->g_lo; P->g_hi = M->g_hi; P->nbins = M->nbins;
    }
    if (M->kind == ODYSSEY_KIND_RIAF) {
        P->n_index = M->n_index; P->T_index = M->T_index;
        P->inv_2h2 = 1.0 / (2.0 * M->h_over_r * M->h_over_r);
        P->ln_rh = std::log(P->r_h);
        P->ln_n0 = std::log(M->n0);                                   // -inf for n0 = 0: no emission
        P->ln_Theta0 = std::log(kKB * M->T0 / (kMe * kC * kC));
        P->ln_nuc0 = std::log(3.0 * kE / (4.0 * kPi * kMe * kC)) + 0.5 * std::log(8.0 * kPi * kMp * kC * kC / (6.0 * M->beta));
        P->ln_j0 = std::log(4.0505 * M->j_scale * kE * kE / (std::sqrt(3.0) * kC));
        P->h_over_mc2 = kH / (kMe * kC * kC);
        P->inv_planck = kC * kC / (2.0 * kH);
        P->r_rt_out = M->r_rt_out; P->tau_max = M->tau_max; P->rt_scheme = M->rt_scheme; P->precision = M->precision;
        if (M->dtau_max > 0.0) { P->rt_scheme = 3; P->dtau_max = M->dtau_max; }
        P->rg_cm = kGMsun * M->mbh_msun / (kC * kC);
        P->sed_coef = 4.0 * kPi * P->rg_cm * P->rg_cm * P->pix_area;
        for (int k = 0; k < nf && k < MAX_FREQ; ++k) { P->nu[k] = nu[k]; P->ln_nu[k] = std::log(nu[k]); P->nu12[k] = std::exp(P->ln_nu[k] / 12.0); P->inu12[k] = 1.0 / P->nu12[k]; P->nu3[k] = nu[k] * nu[k] * nu[k]; }
    }
}

// ---- kernel table ------------------------------------------------------------------------------
#ifndef ODY_MINB_MAIN
#define ODY_MINB_MAIN 5                         // (-DODY_MINB_MAIN=4 builds the 128-register variant of the occupancy comparison in DESIGN.md)
#endif
constexpr int NT_MAIN = 128, MINB_MAIN = ODY_MINB_MAIN;     // 96 registers per thread at most
constexpr int MINB_SPOT = 4;                    // thin disk, hot spot, Novikov-Thorne disk and the coordinate-time variant: 4 blocks per SM keep them free of spills
constexpr int MINB_RK = 4;                      // transfer scheme E' (RK components)
constexpr int NT_SPEC = 128, MINB_SPEC = 4;     // 126 registers, no spills; per-frequency accumulators in a global scratch buffer

typedef void (*KernelFn)(const Params, const Outputs);

KernelFn pick_kernel(int kind, bool spec, int tab, int rts = 0, int prec = 0, bool time = false) {
    if (kind == 3)
        return tab ? odyssey_kernel<3, 1, false, NT_MAIN, MINB_SPOT, 0, 0, 1> : odyssey_kernel<3, 0, false, NT_MAIN, MINB_SPOT, 0, 0, 1>;
    if (kind == 4)
        return tab ? odyssey_kernel<4, 1, false, NT_MAIN, MINB_SPOT> : odyssey_kernel<4, 0, false, NT_MAIN, MINB_SPOT>;
    if (kind == 0 && time)
        return tab ? odyssey_kernel<0, 1, false, NT_MAIN, MINB_SPOT, 0, 0, 1> : odyssey_kernel<0, 0, false, NT_MAIN, MINB_SPOT, 0, 0, 1>;
    if (kind == 2 && !spec && rts == 0 && prec == 1)
        return tab ? odyssey_kernel<2, 1, false, NT_MAIN, MINB_MAIN, 0, 1> : odyssey_kernel<2, 0, false, NT_MAIN, MINB_MAIN, 0, 1>;
    if (kind == 2 && !spec && rts == 1)
        return tab ? odyssey_kernel<2, 1, false, NT_MAIN, MINB_RK, 1> : odyssey_kernel<2, 0, false, NT_MAIN, MINB_RK, 1>;
    if (kind == 2 && !spec && rts == 3)
        return tab ? odyssey_kernel<2, 1, false, NT_MAIN, MINB_MAIN, 3> : odyssey_kernel<2, 0, false, NT_MAIN, MINB_MAIN, 3>;
    if (kind == 2 && !spec && rts == 2)
        return tab ? odyssey_kernel<2, 1, false, NT_MAIN, 4, 2> : odyssey_kernel<2, 0, false, NT_MAIN, 4, 2>;
    if (spec) return tab ? odyssey_kernel<2, 1, true, NT_SPEC, MINB_SPEC> : odyssey_kernel<2, 0, true, NT_SPEC, MINB_SPEC>;
    switch (kind) {
        case 0: return tab ? odyssey_kernel<0, 1, false, NT_MAIN, MINB_MAIN> : odyssey_kernel<0, 0, false, NT_MAIN, MINB_MAIN>;
        case 1: return tab ? odyssey_kernel<1, 1, false, NT_MAIN, MINB_SPOT> : odyssey_kernel<1, 0, false, NT_MAIN, MINB_SPOT>;
        default: return tab ? odyssey_kernel<2, 1, false, NT_MAIN, MINB_MAIN> : odyssey_kernel<2, 0, false, NT_MAIN, MINB_MAIN>;
    }
}

size_t smem_bytes(int kind, bool spec, int nf, int nbins, int rts = 0) {
    if (spec) return (size_t)(smem_per_thread(0) * NT_SPEC + MAX_FREQ) * sizeof(double);
    const size_t stages = (size_t)smem_per_thread(kind == 2 ? rts : 0) * NT_MAIN * sizeof(double);   // stage values + [5][NT] RT state
    if (kind == 1) return stages + (size_t)(nbins > 0 ? nbins : 1) * sizeof(double);
    if (kind == 4) return stages + (size_t)MAX_FREQ * sizeof(double);
    if (uses_fifo(kind, spec, rts)) return stages + (size_t)fifo_doubles_per_block(NT_MAIN) * sizeof(double);
    if (kind == 2 && rts == 1) return stages + (size_t)20 * NT_MAIN * sizeof(double);      // scheme E': the stage states
    return stages;
}

int launch(const Params& P, Outputs O, bool spec, int tab, cudaStream_t st) {
    DevState* D = nullptr;
    int rc = device_state(&D, nullptr);
    if (rc) return rc;
    KernelFn fn = pick_kernel(P.kind, spec, tab, P.rt_scheme, P.precision, O.t != nullptr);
    const int nt = spec ? NT_SPEC : NT_MAIN;
    const size_t sm = smem_bytes(P.kind, spec, P.nf, P.nbins, P.rt_scheme);
    if (sm > 48 * 1024) CUDA_TRY(cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    int per_sm = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, nt, sm));
    if (per_sm < 1) return fail(ODYSSEY_ERR_CUDA, "kernel does not fit on an SM (shared memory %zu B)", sm);
    // persistent grid: every SM full, but no more blocks than there are queue tiles to hand out
    long long blocks = (long long)D->n_sm * per_sm;
    const long long warps_needed = P.n_queue / 32;
    const long long blocks_needed = (warps_needed + nt / 32 - 1) / (nt / 32);
    if (blocks > blocks_needed) blocks = blocks_needed;
    if (blocks < 1) blocks = 1;
    if (O.hist && P.nbins > 0) CUDA_TRY(cudaMemsetAsync(O.hist, 0, sizeof(double) * P.nbins, st));
    if (O.nuLnu) CUDA_TRY(cudaMemsetAsync(O.nuLnu, 0, sizeof(double) * P.nf, st));
    // stream-ordered scratch of this launch: the work-queue counter (its own 256 bytes), one stash of 32 prepared
    // rays per warp of the grid and, in spectrum mode, the per-frequency accumulators [5][nf][blocks * nt]
    const size_t stash_bytes = (size_t)blocks * (nt / 32) * STASH_DOUBLES * sizeof(double);
    const size_t spec_bytes = spec ? sizeof(double) * 5 * (size_t)P.nf * (size_t)blocks * nt : 0;
    char* scratch = nullptr;
    CUDA_TRY(pool_alloc((void**)&scratch, 256 + stash_bytes + spec_bytes, st));
    O.queue = reinterpret_cast<unsigned long long*>(scratch);
    O.stash = reinterpret_cast<double*>(scratch + 256);
    if (spec) O.spec_state = reinterpret_cast<double*>(scratch + 256 + stash_bytes);
    cudaError_t le = cudaMemsetAsync(O.queue, 0, sizeof(unsigned long long), st);
    void* args[] = {(void*)&P, (void*)&O};
    if (le == cudaSuccess) le = cudaLaunchKernel((const void*)fn, dim3((unsigned)blocks), dim3(nt), args, sm, st);
    cudaFreeAsync(scratch, st);
    if (le != cudaSuccess) return fail(ODYSSEY_ERR_CUDA, "cudaLaunchKernel: %s", cudaGetErrorString(le));
    g_launches.fetch_add(1);
    return ODYSSEY_OK;
}

Outputs no_outputs() { Outputs O; std::memset(&O, 0, sizeof(O)); return O; }

// ---- two-phase spectrum path (see spectrum_rt_kernel in odyssey_kernels.cuh) -------------------------------
// Phases: record pass into fixed-capacity node lists, ONE stream synchronisation to read its overflow flag (on
// overflow: count pass, prefix sum, exact-size record pass), then the per-frequency transfer with one lane per
// (ray, frequency).  It wins in two regimes: small images (fewer rays than a few waves of resident lanes, where the
// fused spectrum kernel's run time is the serial time of the longest ray with all frequencies behind each other) and
// many frequencies (the transfer kernel runs every lane on identical work: 1.5 ms per frequency and megaray
// against 3.0 ms fused, for a fixed ~19 ms per megaray of recording).  Images larger than one band are processed
// band by band (whole rows), so the node lists stay at ~10 GB whatever the image size.
constexpr int TWO_PHASE_WAVES = 2;             // rays per band, in waves of the record kernel's resident lanes
#ifndef ODY_TWO_PHASE_MIN_NF
#define ODY_TWO_PHASE_MIN_NF 4
#endif
constexpr int TWO_PHASE_MIN_NF = ODY_TWO_PHASE_MIN_NF;   // larger images with fewer frequencies take the fused kernel (1024^2: 17.5 vs 21.1 ms at 2, 23.8 vs 23.6 at 4, 33.3 vs 29.4 at 8)           // larger images with fewer frequencies take the fused kernel
constexpr long long NODE_CAP = 1024;           // nodes per ray of the first, fixed-capacity attempt (64 KB per ray)

template <int G>
cudaError_t launch_spectrum_rt(const Params& P, const Outputs& O, int blocks, cudaStream_t st) {
    spectrum_rt_kernel<G><<<blocks, 128, 0, st>>>(P, O);
    return cudaGetLastError();
}

int render_spectrum_two_phase(Params P, Outputs user, int tab, cudaStream_t st, bool zero_sed = true) {
    DevState* D = nullptr;
    TRY_RC(device_state(&D, nullptr));
    const size_t n = (size_t)P.nx * P.ny;
    int32_t *iflag = nullptr, *iatt = nullptr, *iacc = nullptr; long long* off = nullptr; double* nodes = nullptr;
    unsigned long long* counter2 = nullptr;                                       // the transfer kernel's own ray counter
    auto release = [&]() {
        if (counter2) cudaFreeAsync(counter2, st);
        if (iflag) cudaFreeAsync(iflag, st); if (iatt) cudaFreeAsync(iatt, st); if (iacc) cudaFreeAsync(iacc, st);
        if (off) cudaFreeAsync(off, st); if (nodes) cudaFreeAsync(nodes, st);
    };
#define TP_TRY(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { release(); return fail(ODYSSEY_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); } } while (0)
    TP_TRY(pool_alloc((void**)&iflag, n * sizeof(int32_t), st));
    TP_TRY(pool_alloc((void**)&iatt, n * sizeof(int32_t), st));
    TP_TRY(pool_alloc((void**)&iacc, n * sizeof(int32_t), st));
    TP_TRY(pool_alloc((void**)&off, (n + 1) * sizeof(long long), st));
    Params Pr = P; Pr.rt_scheme = 2; Pr.nf = 1;
    Outputs O1 = no_outputs();
    O1.flag = iflag; O1.n_attempt = iatt; O1.n_accept = iacc;
    // First try: ONE record pass into fixed-capacity node lists (NODE_CAP nodes per ray) and an overflow flag.
    int32_t* ovf = nullptr;
    TP_TRY(pool_alloc((void**)&ovf, sizeof(int32_t), st));
    TP_TRY(cudaMemsetAsync(ovf, 0, sizeof(int32_t), st));
    int rc = ODYSSEY_OK;
    int32_t overflow = 0;
    if (pool_alloc((void**)&nodes, n * NODE_CAP * NODE_DOUBLES * sizeof(double), st) != cudaSuccess) {
        cudaGetLastError();                                                    // no room for fixed-capacity lists:
        nodes = nullptr; overflow = 1;                                         // size them exactly instead
    } else {
        O1.nodes = nodes; O1.node_cap = NODE_CAP; O1.overflow = ovf;
        rc = launch(Pr, O1, false, tab, st);
    }
    if (rc == ODYSSEY_OK && !overflow) {
        cudaError_t e1 = cudaMemcpyAsync(&overflow, ovf, sizeof(int32_t), cudaMemcpyDeviceToHost, st);
        if (e1 == cudaSuccess) e1 = cudaStreamSynchronize(st);                 // the one synchronisation of this path
        if (e1 != cudaSuccess) rc = fail(ODYSSEY_ERR_CUDA, "two-phase spectrum: %s", cudaGetErrorString(e1));
    }
    cudaFreeAsync(ovf, st);
    if (rc) { release(); return rc; }
    long long node_cap = NODE_CAP;
    if (overflow) {
        // Some ray took more accepted steps than NODE_CAP - 1 (tight tolerances): size the lists exactly —
        // count pass (same kernel, no node buffer), prefix sum, read the total, record again.
        if (nodes) cudaFreeAsync(nodes, st);
        nodes = nullptr;
        O1.nodes = nullptr; O1.node_cap = 0; O1.overflow = nullptr;
        rc = launch(Pr, O1, false, tab, st);
        if (rc) { release(); return rc; }
        node_offsets_kernel<<<1, 1024, 0, st>>>(iacc, (int)n, off);
        TP_TRY(cudaGetLastError());
        g_launches.fetch_add(1);
        long long total = 0;
        TP_TRY(cudaMemcpyAsync(&total, off + n, sizeof(long long), cudaMemcpyDeviceToHost, st));
        TP_TRY(cudaStreamSynchronize(st));
        TP_TRY(pool_alloc((void**)&nodes, (size_t)total * NODE_DOUBLES * sizeof(double), st));
        O1.nodes = nodes; O1.node_offset = off;
        rc = launch(Pr, O1, false, tab, st);
        if (rc) { release(); return rc; }
        node_cap = 0;
    }
    Outputs O2 = no_outputs();
    O2.images = user.images; O2.nuLnu = user.nuLnu; O2.flag = user.flag; O2.n_attempt = user.n_attempt;
    O2.nodes = nodes; O2.node_offset = off; O2.node_cap = node_cap; O2.aux_nacc = iacc; O2.image_stride = user.image_stride;
    TP_TRY(pool_alloc((void**)&counter2, 256, st));
    O2.queue = counter2;
    TP_TRY(cudaMemsetAsync(O2.queue, 0, sizeof(unsigned long long), st));
    if (user.nuLnu && zero_sed) TP_TRY(cudaMemsetAsync(user.nuLnu, 0, sizeof(double) * P.nf, st));
    if (user.flag) TP_TRY(cudaMemcpyAsync(user.flag, iflag, n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    if (user.n_attempt) TP_TRY(cudaMemcpyAsync(user.n_attempt, iatt, n * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    O2.aux_flag = iflag;
    int G = 1; while (G < P.nf) G <<= 1;
    const long long warps = ((long long)n + 32 / G - 1) / (32 / G);
    long long blocks = std::min<long long>((warps + 3) / 4, (long long)D->n_sm * 16);
    if (blocks < 1) blocks = 1;
    cudaError_t le = cudaSuccess;
    switch (G) {
        case 1: le = launch_spectrum_rt<1>(P, O2, (int)blocks, st); break;
        case 2: le = launch_spectrum_rt<2>(P, O2, (int)blocks, st); break;
        case 4: le = launch_spectrum_rt<4>(P, O2, (int)blocks, st); break;
        case 8: le = launch_spectrum_rt<8>(P, O2, (int)blocks, st); break;
        case 16: le = launch_spectrum_rt<16>(P, O2, (int)blocks, st); break;
        default: le = launch_spectrum_rt<32>(P, O2, (int)blocks, st); break;
    }
    TP_TRY(le);
    g_launches.fetch_add(1);
#undef TP_TRY
    release();
    return ODYSSEY_OK;
}

}  // namespace

// ---- host-buffer variants: device scratch, same kernels, copies back, synchronous -------------
namespace {
struct Scratch {
    void* dev[16]; void* host[16]; size_t bytes[16]; int n = 0;
    ~Scratch() { for (int i = 0; i < n; ++i) if (dev[i]) cudaFreeAsync(dev[i], 0); }
    template <class T> int add(T* host_ptr, size_t count, T** out) {
        *out = nullptr;
        if (!host_ptr) return ODYSSEY_OK;
        void* d = nullptr;
        CUDA_TRY(pool_alloc(&d, count * sizeof(T), 0));
        dev[n] = d; host[n] = host_ptr; bytes[n] = count * sizeof(T); ++n;
        *out = (T*)d;
        return ODYSSEY_OK;
    }
    int copy_back() {
        for (int i = 0; i < n; ++i) CUDA_TRY(cudaMemcpyAsync(host[i], dev[i], bytes[i], cudaMemcpyDeviceToHost, 0));
        CUDA_TRY(cudaStreamSynchronize(0));
        return ODYSSEY_OK;
    }
};
#define TRY(expr) do { int rc_ = (expr); if (rc_) return rc_; } while (0)

// The per-pixel work of a _host call, pipelined: the image is cut into bands of whole rows that alternate between two
// streams; a band's device->host copies run while the next band integrates (both kernels are persistent grids, so
// the next band's blocks move in as the previous band's finish: no idle tail between bands).  Same kernels, same
// Params apart from the row window (row0, ny of ny_image), so every pixel is bit-identical to the one-launch result.
// P / O describe the whole image with DEVICE pointers from S; arrays of S with `npix` elements are per-pixel.
constexpr long long BAND_MIN_RAYS = 1 << 20;
constexpr int BAND_MAX = 16;
int run_host_pipelined(const Params& P, const Outputs& O, int tab, Scratch& S, size_t npix) {
    DevState* D = nullptr;
    TRY(device_state(&D, nullptr));
    int nb = (int)std::min<long long>(BAND_MAX, (long long)npix / BAND_MIN_RAYS);
    if (nb > P.ny / (2 * TILE_H)) nb = P.ny / (2 * TILE_H);
    if (nb < 2) {                                                   // small image: one launch, then the copies
        TRY(launch(P, O, false, tab, nullptr));
        return S.copy_back();
    }
    {
        std::lock_guard<std::mutex> lk(g_mu);
        for (int i = 0; i < 2; ++i) if (!D->band_stream[i]) CUDA_TRY(cudaStreamCreateWithFlags(&D->band_stream[i], cudaStreamNonBlocking));
        for (int i = 0; i < 3; ++i) if (!D->band_event[i]) CUDA_TRY(cudaEventCreateWithFlags(&D->band_event[i], cudaEventDisableTiming));
    }
    // the device buffers were allocated in stream 0's order
    CUDA_TRY(cudaEventRecord(D->band_event[2], 0));
    for (int i = 0; i < 2; ++i) CUDA_TRY(cudaStreamWaitEvent(D->band_stream[i], D->band_event[2], 0));
    int rc = ODYSSEY_OK;
    for (int b = 0; b < nb && rc == ODYSSEY_OK; ++b) {
        const int j0 = (int)((long long)P.ny * b / nb) / TILE_H * TILE_H;
        const int j1 = (b + 1 == nb) ? P.ny : (int)((long long)P.ny * (b + 1) / nb) / TILE_H * TILE_H;
        cudaStream_t st = D->band_stream[b & 1];
        Params Pb = P;
        Pb.ny = j1 - j0; Pb.row0 = j0;
        Pb.n_queue = (long long)Pb.tiles_x * ((Pb.ny + TILE_H - 1) / TILE_H) * (TILE_W * TILE_H);
        const size_t shift = (size_t)j0 * P.nx, count = (size_t)(j1 - j0) * P.nx;
        Outputs Ob = O;
        if (O.flag) Ob.flag = O.flag + shift;
        if (O.r) Ob.r = O.r + shift;
        if (O.th) Ob.th = O.th + shift;
        if (O.ph) Ob.ph = O.ph + shift;
        if (O.t) Ob.t = O.t + shift;
        if (O.n_attempt) Ob.n_attempt = O.n_attempt + shift;
        if (O.n_accept) Ob.n_accept = O.n_accept + shift;
        if (O.image) Ob.image = O.image + shift;
        if (O.aux0) Ob.aux0 = O.aux0 + shift;
        if (O.aux1) Ob.aux1 = O.aux1 + shift;
        if (O.images) Ob.images = O.images + shift;
        rc = launch(Pb, Ob, false, tab, st);
        for (int i = 0; i < S.n && rc == ODYSSEY_OK; ++i) {
            if (S.bytes[i] % npix != 0 || S.bytes[i] / npix > 8) continue;          // not a per-pixel array
            const size_t el = S.bytes[i] / npix;
            if (cudaMemcpyAsync((char*)S.host[i] + shift * el, (char*)S.dev[i] + shift * el, count * el, cudaMemcpyDeviceToHost, st) != cudaSuccess)
                rc = fail(ODYSSEY_ERR_CUDA, "device->host copy of band %d failed: %s", b, cudaGetErrorString(cudaGetLastError()));
        }
    }
    // join: the host waits for both streams (also on failure: the buffers are freed in stream 0's order afterwards)
    cudaError_t e0 = cudaStreamSynchronize(D->band_stream[0]), e1 = cudaStreamSynchronize(D->band_stream[1]);
    if (rc == ODYSSEY_OK && (e0 != cudaSuccess || e1 != cudaSuccess))
        rc = fail(ODYSSEY_ERR_CUDA, "pipelined render: %s", cudaGetErrorString(e0 != cudaSuccess ? e0 : e1));
    return rc;
}
}  // namespace

// ================================================================================================
// extern "C" entry points (include/odyssey.h)
// ================================================================================================
extern "C" {

int odyssey_trace_geodesics(const odyssey_scene* scene, int32_t* flag, double* r, double* theta, double* phi, double* t,
                            int32_t* n_attempt, int32_t* n_accept, void* cuda_stream) {
    int rc = check_scene(scene);
    if (rc) return rc;
    Params P; fill_params(*scene, nullptr, nullptr, 0, &P);
    Outputs O = no_outputs();
    O.flag = flag; O.r = r; O.th = theta; O.ph = phi; O.t = t; O.n_attempt = n_attempt; O.n_accept = n_accept;
    return launch(P, O, false, scene->tableau, (cudaStream_t)cuda_stream);
}

int odyssey_render_image(const odyssey_scene* scene, const odyssey_model* model, double nu_hz,
                         double* image, double* aux0, double* aux1, int32_t* flag, int32_t* n_attempt,
                         int32_t* n_accept, double* hist, void* cuda_stream) {
    int rc = check_scene(scene);
    if (rc) return rc;
    rc = check_model(model);
    if (rc) return rc;
    if (model->kind == ODYSSEY_KIND_HOT_SPOT) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "model kind 3 (hot spot) is rendered by odyssey_render_hotspot");
    if ((model->kind == ODYSSEY_KIND_RIAF || model->kind == ODYSSEY_KIND_NT_DISK) && !(nu_hz > 0.0))
        return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nu_hz = %g must be > 0", nu_hz);
    Params P; fill_params(*scene, model, &nu_hz, 1, &P);
    Outputs O = no_outputs();
    if (model->kind == ODYSSEY_KIND_NT_DISK) O.images = image;      // the one-frequency case of the spectrum epilogue
    O.image = image; O.aux0 = aux0; O.aux1 = aux1; O.flag = flag; O.n_attempt = n_attempt; O.n_accept = n_accept;
    O.hist = (model->kind == ODYSSEY_KIND_THIN_DISK && model->nbins > 0) ? hist : nullptr;
    return launch(P, O, false, scene->tableau, (cudaStream_t)cuda_stream);
}

int odyssey_render_spectrum(const odyssey_scene* scene, const odyssey_model* model, const double* nu_hz_host, int nf,
                            double* images, double* nuLnu, int32_t* flag, int32_t* n_attempt, void* cuda_stream) {
    int rc = check_scene(scene);
    if (rc) return rc;
    rc = check_model(model);
    if (rc) return rc;
    if (model->kind != ODYSSEY_KIND_RIAF && model->kind != ODYSSEY_KIND_NT_DISK)
        return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "spectrum mode needs model kind 2 (RIAF) or 4 (Novikov-Thorne disk), got %d", model->kind);
    if (model->kind == ODYSSEY_KIND_NT_DISK) {
        if (nf < 1 || nf > ODYSSEY_MAX_FREQ) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nf = %d outside [1, %d]", nf, ODYSSEY_MAX_FREQ);
        if (!nu_hz_host) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nu_hz_host is NULL");
        for (int k = 0; k < nf; ++k)
            if (!(nu_hz_host[k] > 0.0)) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nu_hz_host[%d] = %g must be > 0", k, nu_hz_host[k]);
        Params P; fill_params(*scene, model, nu_hz_host, nf, &P);
        Outputs O = no_outputs();
        O.images = images; O.nuLnu = nuLnu; O.flag = flag; O.n_attempt = n_attempt;
        return launch(P, O, false, scene->tableau, (cudaStream_t)cuda_stream);      // one geodesic pass, all frequencies at the crossing
    }
    if (model->rt_scheme != ODYSSEY_RT_PER_STEP) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "spectrum mode supports rt_scheme 0 (per-step update) only");
    if (model->dtau_max > 0.0) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "spectrum mode does not support dtau_max (single-frequency image calls only)");
    if (model->precision != ODYSSEY_PREC_FP64) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "spectrum mode supports precision FP64 only");
    if (nf < 1 || nf > ODYSSEY_MAX_FREQ) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nf = %d outside [1, %d]", nf, ODYSSEY_MAX_FREQ);
    if (!nu_hz_host) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nu_hz_host is NULL");
    for (int k = 0; k < nf; ++k)
        if (!(nu_hz_host[k] > 0.0)) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nu_hz_host[%d] = %g must be > 0", k, nu_hz_host[k]);
    Params P; fill_params(*scene, model, nu_hz_host, nf, &P);
    Outputs O = no_outputs();
    O.images = images; O.nuLnu = nuLnu; O.flag = flag; O.n_attempt = n_attempt;
    DevState* D = nullptr;
    rc = device_state(&D, nullptr);
    if (rc) return rc;
    const long long lanes = (long long)D->n_sm * 4 * NT_MAIN;                  // resident lanes of the record kernel
    const long long band_rays = TWO_PHASE_WAVES * lanes;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((long long)scene->nx * scene->ny <= band_rays)
        return render_spectrum_two_phase(P, O, scene->tableau, st);
    if (nf < TWO_PHASE_MIN_NF || scene->nx > band_rays) return launch(P, O, true, scene->tableau, st);   // (bands are whole rows)
    // Larger images, many frequencies: the same two phases band by band (whole rows, about band_rays rays each);
    // one stream synchronisation per band.
    const int rows = (int)std::max<long long>(1, band_rays / scene->nx);
    if (nuLnu) CUDA_TRY(cudaMemsetAsync(nuLnu, 0, sizeof(double) * nf, st));
    for (int j0 = 0; j0 < scene->ny; j0 += rows) {
        Params Pb = P;
        Pb.ny = std::min(rows, scene->ny - j0); Pb.row0 = j0;
        Pb.n_queue = (long long)Pb.tiles_x * ((Pb.ny + TILE_H - 1) / TILE_H) * (TILE_W * TILE_H);
        Outputs Ob = O;
        const size_t shift = (size_t)j0 * scene->nx;
        if (images) Ob.images = images + shift;
        if (flag) Ob.flag = flag + shift;
        if (n_attempt) Ob.n_attempt = n_attempt + shift;
        Ob.image_stride = (long long)scene->nx * scene->ny;
        rc = render_spectrum_two_phase(Pb, Ob, scene->tableau, st, false);
        if (rc) return rc;
    }
    return ODYSSEY_OK;
}

int odyssey_render_hotspot(const odyssey_scene* scene, const odyssey_model* model, const double* t_obs_host, int nt,
                           double* images, double* lightcurve, double* spectrogram,
                           double* g, double* r_e, double* phi_e, double* t_e, int32_t* flag, int32_t* n_attempt,
                           void* cuda_stream) {
    int rc = check_scene(scene);
    if (rc) return rc;
    rc = check_model(model);
    if (rc) return rc;
    if (model->kind != ODYSSEY_KIND_HOT_SPOT) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "hot-spot mode needs model kind 3, got %d", model->kind);
    if (model->spot_r_orbit > 0.0 && !(model->spot_r_orbit > 1.0 + std::sqrt(1.0 - scene->a * scene->a)))
        return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "spot_r_orbit = %g lies inside the horizon of a = %g", model->spot_r_orbit, scene->a);
    if (nt < 1 || nt > ODYSSEY_MAX_FREQ) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nt = %d outside [1, %d]", nt, ODYSSEY_MAX_FREQ);
    if (!t_obs_host) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "t_obs_host is NULL");
    for (int k = 0; k < nt; ++k)
        if (!std::isfinite(t_obs_host[k])) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "t_obs_host[%d] is not finite", k);
    Params P; fill_params(*scene, model, t_obs_host, nt, &P);
    Outputs O = no_outputs();
    O.images = images; O.nuLnu = lightcurve; O.aux0 = g; O.aux1 = r_e; O.ph = phi_e; O.t = t_e;
    O.flag = flag; O.n_attempt = n_attempt;
    const bool spec = spectrogram && model->nbins > 0;
    O.hist = spec ? spectrogram : nullptr;
    if (spec) CUDA_TRY(cudaMemsetAsync(spectrogram, 0, sizeof(double) * (size_t)nt * model->nbins, (cudaStream_t)cuda_stream));
    return launch(P, O, false, scene->tableau, (cudaStream_t)cuda_stream);
}

// ---- host-buffer variants (Scratch defined above) ---------------------------------------------

int odyssey_trace_geodesics_host(const odyssey_scene* scene, int32_t* flag, double* r, double* theta, double* phi, double* t,
                                 int32_t* n_attempt, int32_t* n_accept) {
    TRY(check_scene(scene));
    const size_t n = (size_t)scene->nx * scene->ny;
    Scratch S; int32_t *dflag, *datt, *dacc; double *dr, *dth, *dph, *dt;
    TRY(S.add(flag, n, &dflag)); TRY(S.add(r, n, &dr)); TRY(S.add(theta, n, &dth)); TRY(S.add(phi, n, &dph)); TRY(S.add(t, n, &dt));
    TRY(S.add(n_attempt, n, &datt)); TRY(S.add(n_accept, n, &dacc));
    Params P; fill_params(*scene, nullptr, nullptr, 0, &P);
    Outputs O = no_outputs();
    O.flag = dflag; O.r = dr; O.th = dth; O.ph = dph; O.t = dt; O.n_attempt = datt; O.n_accept = dacc;
    return run_host_pipelined(P, O, scene->tableau, S, n);
}

int odyssey_render_image_host(const odyssey_scene* scene, const odyssey_model* model, double nu_hz,
                              double* image, double* aux0, double* aux1, int32_t* flag, int32_t* n_attempt,
                              int32_t* n_accept, double* hist) {
    TRY(check_scene(scene)); TRY(check_model(model));
    const size_t n = (size_t)scene->nx * scene->ny;
    Scratch S; double *dimg, *da0, *da1, *dhist; int32_t *dflag, *datt, *dacc;
    TRY(S.add(image, n, &dimg)); TRY(S.add(aux0, n, &da0)); TRY(S.add(aux1, n, &da1));
    TRY(S.add(flag, n, &dflag)); TRY(S.add(n_attempt, n, &datt)); TRY(S.add(n_accept, n, &dacc));
    TRY(S.add((model->kind == ODYSSEY_KIND_THIN_DISK && model->nbins > 0) ? hist : nullptr, (size_t)model->nbins, &dhist));
    if (dhist || model->kind == ODYSSEY_KIND_HOT_SPOT || ((model->kind == ODYSSEY_KIND_RIAF || model->kind == ODYSSEY_KIND_NT_DISK) && !(nu_hz > 0.0))) {
        // the line histogram is a sum over the whole image (one launch); invalid arguments are reported by the device call
        TRY(odyssey_render_image(scene, model, nu_hz, dimg, da0, da1, dflag, datt, dacc, dhist, nullptr));
        return S.copy_back();
    }
    Params P; fill_params(*scene, model, &nu_hz, 1, &P);
    Outputs O = no_outputs();
    if (model->kind == ODYSSEY_KIND_NT_DISK) O.images = dimg;
    O.image = dimg; O.aux0 = da0; O.aux1 = da1; O.flag = dflag; O.n_attempt = datt; O.n_accept = dacc;
    return run_host_pipelined(P, O, scene->tableau, S, n);
}

int odyssey_render_spectrum_host(const odyssey_scene* scene, const odyssey_model* model, const double* nu_hz_host, int nf,
                                 double* images, double* nuLnu, int32_t* flag, int32_t* n_attempt) {
    TRY(check_scene(scene)); TRY(check_model(model));
    if (nf < 1 || nf > ODYSSEY_MAX_FREQ) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nf = %d outside [1, %d]", nf, ODYSSEY_MAX_FREQ);
    const size_t n = (size_t)scene->nx * scene->ny;
    Scratch S; double *dimg, *dsed; int32_t *dflag, *datt;
    TRY(S.add(images, n * nf, &dimg)); TRY(S.add(nuLnu, (size_t)nf, &dsed));
    TRY(S.add(flag, n, &dflag)); TRY(S.add(n_attempt, n, &datt));
    TRY(odyssey_render_spectrum(scene, model, nu_hz_host, nf, dimg, dsed, dflag, datt, nullptr));
    return S.copy_back();
}

int odyssey_render_hotspot_host(const odyssey_scene* scene, const odyssey_model* model, const double* t_obs_host, int nt,
                                double* images, double* lightcurve, double* spectrogram,
                                double* g, double* r_e, double* phi_e, double* t_e, int32_t* flag, int32_t* n_attempt) {
    TRY(check_scene(scene)); TRY(check_model(model));
    if (nt < 1 || nt > ODYSSEY_MAX_FREQ) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "nt = %d outside [1, %d]", nt, ODYSSEY_MAX_FREQ);
    const size_t n = (size_t)scene->nx * scene->ny;
    Scratch S; double *dimg, *dlc, *dsp, *dg, *dre, *dph, *dte; int32_t *dflag, *datt;
    TRY(S.add(images, n * nt, &dimg)); TRY(S.add(lightcurve, (size_t)nt, &dlc));
    TRY(S.add(model->nbins > 0 ? spectrogram : nullptr, (size_t)nt * (size_t)(model->nbins > 0 ? model->nbins : 0), &dsp));
    TRY(S.add(g, n, &dg)); TRY(S.add(r_e, n, &dre)); TRY(S.add(phi_e, n, &dph)); TRY(S.add(t_e, n, &dte));
    TRY(S.add(flag, n, &dflag)); TRY(S.add(n_attempt, n, &datt));
    TRY(odyssey_render_hotspot(scene, model, t_obs_host, nt, dimg, dlc, dsp, dg, dre, dph, dte, dflag, datt, nullptr));
    return S.copy_back();
}

// ---- probes and bookkeeping ---------------------------------------------------------------------
int odyssey_fp64_peak_probe(int iters, double* sink, double* flop_host, void* cuda_stream) {
    if (iters <= 0 || !sink) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "iters must be > 0 and sink non-NULL");
    DevState* D = nullptr;
    TRY(device_state(&D, nullptr));
    const int blocks = D->n_sm * 8, threads = 256;                    // 2048 resident threads per SM
    dfma_probe_kernel<<<blocks, threads, 0, (cudaStream_t)cuda_stream>>>(iters, sink);
    CUDA_TRY(cudaGetLastError());
    g_launches.fetch_add(1);
    if (flop_host) *flop_host = 2.0 * PROBE_DFMA_PER_ITER * (double)iters * (double)blocks * threads;
    return ODYSSEY_OK;
}

int odyssey_eval_math(int op, int n, const double* x, double* y, double* y2, void* cuda_stream) {
    if (op < 0 || op > 9 || n < 0 || (n > 0 && (!x || !y)) || (op == 3 && !y2))
        return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "eval_math: op in [0,9], n >= 0, x and y non-NULL (y2 too for op 3)");
    if (n == 0) return ODYSSEY_OK;
    DevState* D = nullptr;
    TRY(device_state(&D, nullptr));
    eval_math_kernel<<<(n + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>(op, n, x, y, y2);
    CUDA_TRY(cudaGetLastError());
    g_launches.fetch_add(1);
    return ODYSSEY_OK;
}

int odyssey_kernel_info(int kind, int spectrum, int tableau, int32_t* regs, int32_t* local_bytes,
                        int32_t* threads_per_block, int32_t* blocks_per_sm, int32_t* n_sm) {
    if (kind < 0 || kind > 4 || (tableau != 0 && tableau != 1)) return fail(ODYSSEY_ERR_INVALID_ARGUMENT, "unknown kind/tableau");
    DevState* D = nullptr;
    TRY(device_state(&D, nullptr));
    const bool spec = spectrum != 0;
    KernelFn fn = pick_kernel(spec ? 2 : kind, spec, tableau);
    cudaFuncAttributes at;
    CUDA_TRY(cudaFuncGetAttributes(&at, (const void*)fn));
    const int nt = spec ? NT_SPEC : NT_MAIN;
    const size_t sm = smem_bytes(spec ? 2 : kind, spec, ODYSSEY_MAX_FREQ, 200);
    if (sm > 48 * 1024) CUDA_TRY(cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    int per_sm = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, nt, sm));
    if (regs) *regs = at.numRegs;
    if (local_bytes) *local_bytes = (int32_t)at.localSizeBytes;
    if (threads_per_block) *threads_per_block = nt;
    if (blocks_per_sm) *blocks_per_sm = per_sm;
    if (n_sm) *n_sm = D->n_sm;
    return ODYSSEY_OK;
}

long long odyssey_launch_count(void) { return g_launches.load(); }

int odyssey_trim_scratch(unsigned long long keep_bytes) {
    DevState* D = nullptr;
    TRY(device_state(&D, nullptr));
    CUDA_TRY(cudaDeviceSynchronize());
    pool_trim((size_t)keep_bytes);
    return ODYSSEY_OK;
}

const char* odyssey_last_error(void) { return g_err; }

void odyssey_shutdown(void) {
    std::lock_guard<std::mutex> lk(g_mu);
    int cur = 0;
    if (cudaGetDevice(&cur) != cudaSuccess) return;
    for (int d = 0; d < MAX_DEV; ++d) {
        if (!g_dev[d].ready) continue;
        cudaSetDevice(d);
        cudaDeviceSynchronize();
        for (int i = 0; i < 2; ++i) if (g_dev[d].band_stream[i]) cudaStreamDestroy(g_dev[d].band_stream[i]);
        for (int i = 0; i < 3; ++i) if (g_dev[d].band_event[i]) cudaEventDestroy(g_dev[d].band_event[i]);
        if (g_dev[d].pool) cudaMemPoolDestroy(g_dev[d].pool);
        g_dev[d] = DevState();
    }
    cudaSetDevice(cur);
}

}  // extern "C"
