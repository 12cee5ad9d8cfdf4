// params.h — the constant block every kernel receives as a __grid_constant__ parameter (constant
// bank; no global __constant__ symbol, so calls on different streams cannot race on it).
// Filled on the host by fill_params() in odyssey_api.cu from the two C-ABI structs.
#pragma once
#include <stdint.h>

namespace ody {

constexpr int MAX_FREQ = 32;
constexpr int TILE_W = 8, TILE_H = 4;          // one queue tile = 8x4 pixels = one warp's first batch
constexpr int STASH_DOUBLES = 7 * 32;          // per warp: the prepared rays of one queue tile (see the refill in odyssey_kernels.cuh)
constexpr int LOCATE_MAX = 8;                  // Newton re-attempts of the event location
constexpr int NODE_DOUBLES = 8;                // two-phase spectrum path: h, fac, E, t0, u0, ycoef, n_attempt (+ 1 pad) per node:
                                               // 64 bytes, written and read as four aligned 16-byte vectors (two whole 32-byte sectors)

struct Params {
    // ---- scene
    double a, a2;
    double r_obs, R_obs;                        // R_obs = sqrt(r_obs^2 + a^2), eq. (19)
    double sin_obs, cos_obs, sin_pobs, cos_pobs, phi_obs;
    double x_min, x_span, y_min, y_span;        // x = x_min + (i + 1/2) x_span / nx
    double pix_area;
    double rtol, inv_rtol, h0, r_h, r_cap, r_esc;
    int32_t nx, ny, tiles_x, max_attempts;
    long long n_queue;                          // tiles_x * tiles_y * 32 queue slots
    // ---- flow (BASELINE.json:configs[2] "plunging inside")
    double r_isco, E_isco, L_isco;
    // ---- thin disk (BASELINE.json:configs[1])
    double r_in, r_out, emis_index, g_power, g_lo, g_hi, bins_per_g;
    int32_t nbins, kind;
    // ---- RIAF thermal synchrotron (eqs. (37)-(39); BASELINE.json:configs[2])
    // (log-space assembly of the emissivity: emission.cuh header)
    double n_index, T_index, inv_2h2;           // n_e ∝ (r/r_h)^n_index exp(-cos²θ inv_2h2), T_e ∝ (r/r_h)^T_index
    double ln_rh;                               // ln r_h
    double ln_n0;                               // ln n0
    double ln_Theta0;                           // ln(k_B T0 / m_e c²)
    double ln_nuc0;                             // ln(3e/(4π m_e c)) + ½ ln(8π m_p c²/(6β)): ν_c = e^ln_nuc0 (n_e/r)^½ Θ_e², eq. (39)
    double ln_j0;                               // ln(4.0505 j_scale e²/(√3 c)): eq. (37) per steradian × the 4.0505 of eq. (38)
    double h_over_mc2;                          // h/(m_e c²): hν0/kT_e = h_over_mc2 ν0 /Θ_e
    double inv_planck;                          // c²/(2h)
    double r_rt_out, tau_max, rg_cm;
    double sed_coef;                            // 4π r_g^2 Δx Δy
    int32_t nf, rt_scheme;                      // rt_scheme: ODYSSEY_RT_* (kind 2); internally 2 = record pass, 3 = per-step with the Δτ cap
    double dtau_max;                            // (rt_scheme 3) cap of the next step's optical depth
    int32_t row0, ny_image;                     // this launch covers image rows [row0, row0 + ny) of ny_image (bands of the two-phase spectrum path)
    int32_t precision, pad3;                    // ODYSSEY_PREC_* (kind 2)
    // ---- hot spot (kind 3; eq. (36)); the observer times t_obs[k] travel in nu[k], nf = their number
    double spot_R, spot_Omega, spot_phi0;       // sqrt(r_s² + a²), 1/(r_s^{3/2} + a), azimuth at t = 0
    double spot_inv2s2, spot_cut2;              // 1/(2 r_spot²), (4 r_spot)²
    // ---- Novikov–Thorne disk (kind 4; eq. (35)): Page & Thorne's f(r) in x = sqrt(r)
    double nt_x0;                               // sqrt(r_isco)
    double nt_x[3], nt_c[3];                    // roots of x³ - 3x + 2a and the weights 3(x_i - a)²/(x_i (x_i - x_j)(x_i - x_k))
    double nt_T4;                               // 3 Mdot c⁶/(8π G² M² σ): T_eff⁴ = nt_T4 f / r³
    double h_over_k;                            // h/k_B
    double planck2;                             // 2h/c²
    double nu[MAX_FREQ];
    double ln_nu[MAX_FREQ];
    double nu12[MAX_FREQ], inu12[MAX_FREQ];     // ν^(1/12) and its reciprocal (eq. (38) in powers of x_M^(1/12))
    double nu3[MAX_FREQ];                       // ν^3 (observed), image = ν^3 × invariant intensity
};

// Output pointers (device memory, any may be null).
struct Outputs {
    int32_t* flag;
    double* r; double* th; double* ph; double* t;
    int32_t* n_attempt; int32_t* n_accept;
    double* image; double* aux0; double* aux1;   // single-frequency image modes
    double* hist;                                // kind 1
    double* images; double* nuLnu;               // spectrum mode
    double* spec_state;                          // spectrum mode: library scratch, [5][nf][grid threads] accumulators
    double* nodes;                               // two-phase spectrum path: library scratch, NODE_DOUBLES per node
    const long long* node_offset;                // two-phase spectrum path: first node of each ray, [npix + 1]
    const int32_t* aux_flag;                     // two-phase spectrum path: the record pass's flags (input of phase 2)
    const int32_t* aux_nacc;                     // two-phase spectrum path: accepted steps per ray (nodes = n_accept + 1)
    long long node_cap;                          // > 0: fixed capacity, ray's nodes start at pix * node_cap (node_offset unused)
    int32_t* overflow;                           // record pass: set to 1 when a ray needs more than node_cap nodes
    unsigned long long* queue;                   // work-queue counter (zeroed before the launch)
    double* stash;                               // library scratch: per warp of the grid, 32 prepared rays x 7 doubles (y, L, pixel index)
    long long image_stride;                      // spectrum_rt_kernel: elements between the images of two frequencies (0: nx * ny)
};

}  // namespace ody
