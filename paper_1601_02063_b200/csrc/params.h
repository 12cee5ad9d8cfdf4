// params.h — the constant block every kernel receives as a __grid_constant__ parameter (constant
// bank; no global __constant__ symbol, so calls on different streams cannot race on it).
// Filled on the host by fill_params() in odyssey_api.cu from the two C-ABI structs.
#pragma once
#include <stdint.h>

namespace ody {

constexpr int MAX_FREQ = 32;
constexpr int TILE_W = 8, TILE_H = 4;          // one queue tile = 8x4 pixels = one warp's first batch
constexpr int LOCATE_MAX = 8;                  // Newton re-attempts of the event location

struct Params {
    // ---- scene
    double a, a2;
    double r_obs, R_obs;                        // R_obs = sqrt(r_obs^2 + a^2), eq. (19)
    double sin_obs, cos_obs, sin_pobs, cos_pobs, phi_obs;
    double x_min, x_span, y_min, y_span;        // x = x_min + (i + 1/2) x_span / nx
    double pix_area;
    double rtol, h0, r_h, r_cap, r_esc;
    int32_t nx, ny, tiles_x, max_attempts;
    long long n_queue;                          // tiles_x * tiles_y * 32 queue slots
    // ---- flow (BASELINE.json:configs[2] "plunging inside")
    double r_isco, E_isco, L_isco;
    // ---- thin disk (BASELINE.json:configs[1])
    double r_in, r_out, emis_index, g_power, g_lo, g_hi, bins_per_g;
    int32_t nbins, kind;
    // ---- RIAF thermal synchrotron (eqs. (37)-(39); BASELINE.json:configs[2])
    double n0, n_index, T0, T_index, inv_2h2;   // exp(-cos^2 θ * inv_2h2)
    double B2_coef;                             // B^2 = B2_coef n_e / r
    double theta_per_K;                         // Θ_e = theta_per_K T_e
    double nuc_coef;                            // ν_c = nuc_coef B Θ_e^2, eq. (39)
    double j_coef;                              // j = j_coef ν0 n_e M(x_M) / K_2(1/Θ_e), eq. (37) per steradian
    double planck_coef;                         // 2h/c^2
    double h_over_k;                            // h/k_B
    double r_rt_out, tau_max, rg_cm;
    double sed_coef;                            // 4π r_g^2 Δx Δy
    int32_t nf, pad;
    double nu[MAX_FREQ];
    double nu3[MAX_FREQ];                       // ν^3 (observed), image = ν^3 × invariant intensity
};

// Output pointers (device memory, any may be null).
struct Outputs {
    int32_t* flag;
    double* r; double* th; double* ph;
    int32_t* n_attempt; int32_t* n_accept;
    double* image; double* aux0; double* aux1;   // single-frequency image modes
    double* hist;                                // kind 1
    double* images; double* nuLnu;               // spectrum mode
    unsigned long long* queue;                   // work-queue counter (zeroed before the launch)
};

}  // namespace ody
