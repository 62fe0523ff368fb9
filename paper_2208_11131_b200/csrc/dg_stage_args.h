// Kernel argument block of the fused stage kernel (filled by dg_api.cu, read by dg_stage.cuh).
#pragma once

struct DgStageArgs {
    const double *w_prev;   // stage input u^(i-1): halo + own reads
    const double *w_n;      // u^n (own cell only)
    double *w_out;          // u^(i) (may alias w_n on the last stage); or dw/dt if rhs_only
    const double *w_aux_in; // SSPRK(5,4) stage 4 only: u^(2); NULL otherwise
    double *w_aux;          // SSPRK(5,4) stage 4 only: aux_a u^(2) + aux_b u^(i-1) + aux_c dt L(u^(i-1)); NULL otherwise
    double *flux;           // projected upper-face fluxes [axis][var][transverse mode][cell] (face kernel -> stage kernel)
    const double *scal;     // device scalars: [0] = dt
    unsigned long long *maxbits;  // [0] = bits of max c_s, [1] = bits of max |v| (non-negative doubles; reset every step),
                                  // [2] = bits of the running max of alpha at the Gauss points (reset by dg_set_state)
    int *flag;              // set to 1 on rho <= 0 or p <= 0
    double *sens_prev;      // [0..N) S^K, [N..2N) G^K of the previous step (AV only)
    double *sens_new;       // same, written on stage 1, committed to sens_prev on the last stage
    int ncells, nx, ny, nz;
    double h, gamma, nu, chi;
    double eta;               // tracer diffusivity (DG_TRACER builds only)
    double f_v, f_tau, f_w, s_onset, alpha_max;
    double rk_a, rk_b, rk_c;  // u^(i) = rk_a u^n + rk_b u^(i-1) + rk_c dt L(u^(i-1))
    double aux_a, aux_b, aux_c;
    int do_sensor, do_wavespeed, commit_sensor, rhs_only;
    int limiter;              // 1: positivity limiter on the stage output inside the stage kernel (dg_stage2_kernel only)
    int total_degree;         // 1: modes with sum_a l_a > n are discarded: their rows stay zero
};
