// Stage kernel, second generation (m x m register tiles, 2 <= m <= 5): the same operator as dg_stage_kernel
// (Eq. 20-21, 200) with
//   * no modal dw/dt accumulator in shared memory: the last projection sweep leaves dw/dt in registers, the lift of
//     the face fluxes (Eq. 20 surface lines) is injected between the projection sweeps -- x faces after P_x (as nodal
//     values in y,z), y faces after P_y (modal in x, nodal in z), z faces after P_z (modal in x,y) -- and the stage
//     combine writes straight to global memory;
//   * the own modes read from global memory directly into the register tiles of the first two expansion sweeps;
//   * six barrier-separated phases in 3D (three in 2D) instead of twelve, ~35 % fewer shared-memory wavefronts, and
//     a per-cell footprint of (V + D*Vc) m^D doubles;
//   * the global inputs of the later phases (face fluxes, u^n, u^(i-1)) are requested before the barrier in front of
//     the phase that needs them, so that one memory round trip covers a thread's items and overlaps the barrier wait;
//   * blocks walk the mesh in (y,z)-blocked order (TilePos / tile_grid in dg_stage.cuh) so that the lower y and z
//     neighbours' face fluxes are still in L2 when they are read.
// The face kernel writes the face fluxes in the matching partially projected form (Cfg::PP in dg_stage.cuh).
// Measured dead ends (profiles/r2b_cfg4.md): persistent blocks with the next tile's modes staged by TMA tensor copies,
// a persistent warp-specialised producer/consumer form (named barriers, second copy of U; bit-identical, 2 % slower per
// step; removed from the source in round 3), L2 prefetch hints, 12 warps per block, two 8-cell
// blocks per SM -- all slower.
#pragma once

#include "dg_stage.cuh"
#include "dg_limiter.cuh"

#ifndef DG_S2_NT3
#define DG_S2_NT3 512
#endif
#ifndef DG_S2_CMAX3
#define DG_S2_CMAX3 16
#endif
#ifndef DG_S2_MINB
#define DG_S2_MINB 1
#endif
#ifndef DG_S2_UNROLL_E
#define DG_S2_UNROLL_E 2
#endif
#ifndef DG_S2_UNROLL_B
#define DG_S2_UNROLL_B 3
#endif

namespace DG_NS {

template <int D, int M, bool VISC, bool AV>
struct Cfg2 {
    using K = Cfg<D, M, VISC, AV>;
    static constexpr int V = K::V, Vc = K::Vc, Np = K::Np, Nf = K::Nf;
    // one block of 16 warps per SM in 3D (measured: 128-byte rows of 16 cells beat two blocks of 8 cells at 128^3);
    // 2D tiles are small, several 8-warp blocks share an SM
    static constexpr int NT = (D == 3) ? DG_S2_NT3 : 256;
    static constexpr int CMAX = (D == 3 && M >= 4) ? DG_S2_CMAX3 : 32;
    // doubles per cell: U (nodal values) + GR (gradients -> fluxes)
    static constexpr int FP = V * Np + D * Vc * Np;
    // Wk[c], wave-speed scratch, sensor partials, S table
    // ... and the positivity limiter's per-cell scratch (fused form, see the kernel's tail)
    static constexpr int lim_doubles(int c) { return (K::Vc + 3) * c + c + (c + 1) / 2 + 2 + K::Vc * c; }
    static constexpr int extra_doubles(int c) {
        return c + 2 * (NT / 32) + (AV ? 4 * (NT / 32) * c : 0) + M * M + 2 + lim_doubles(c);
    }
    static constexpr int pick_c() {
        int c = CMAX;
        while (c > 1 && (c * FP + extra_doubles(c)) * 8 > (227 * 1024) / DG_S2_MINB - 1024) c >>= 1;
        return c;
    }
    static constexpr int C = pick_c();
    static constexpr int kSmemBytes = (C * FP + extra_doubles(C)) * 8;
    static_assert(kSmemBytes <= kSmemMax, "stage kernel 2: per-cell footprint exceeds shared memory");
    static_assert(NT % C == 0, "threads per block must be a multiple of cells per block");
};

// PLAIN: the RK-stage form every time step uses (not rhs_only, full tensor basis, no SSPRK(5,4) auxiliary row): those
// three switches become compile-time constants, which removes their selects from the combine loops.
template <int D, int M, bool VISC, bool AV, bool PLAIN>
__global__ void __launch_bounds__((Cfg2<D, M, VISC, AV>::NT), DG_S2_MINB) dg_stage2_kernel(const DgStageArgs p) {
    using K = Cfg<D, M, VISC, AV>;
    using K2 = Cfg2<D, M, VISC, AV>;
    constexpr int C = K2::C, NT = K2::NT, NTB = NT, V = K::V, Vc = K::Vc, Np = K::Np, Nf = K::Nf;
    constexpr bool GRAD = K::GRAD;
    constexpr int MM = M * M;
    constexpr int kUnrollE = DG_S2_UNROLL_E, kUnrollB = DG_S2_UNROLL_B;
    constexpr int NTILE = Np / MM;               // m x m tiles per slot (m in 3D, 1 in 2D)
    using L = Lay<MM, Np, use_swizzle(M, C), 0>;
    extern __shared__ __align__(128) double smem[];
    double *U = smem;                             // [V][Np][C]   modes -> nodal values -> projected N
    double *GR = U + V * Np * C;                  // [D*Vc][Np][C] gradients -> fluxes (in place)
    double *Wk = GR + D * Vc * Np * C;            // [C]
    double *red = Wk + C;
    double *sens = red + 2 * (NTB / 32);          // [4][NTB/32][C] partial sensor sums (AV only)
    double *sS = sens + (AV ? 4 * (NTB / 32) * C : 0);   // weak-derivative matrix S for run-time row indices
    double *limsc = sS + M * M + 2;                     // limiter scratch (fused form)
    double *ldev = limsc + LimScratch<D, C>::kDoubles;  // [Vc][C] sum_{l>0} |w_l| max|phi_l| of the new state
    const bool lim = (p.limiter != 0);
    const int tid = threadIdx.x;
    if (lim && tid < Vc * C) ldev[tid] = 0.0;
    const int cl = tid % C;
    const double ih = 1.0 / p.h;
    const double pref = (D == 3 ? 0.25 : 0.5) * ih;
    const bool rhs_only = PLAIN ? false : (p.rhs_only != 0);
    const bool total_degree = PLAIN ? false : (p.total_degree != 0);
    const bool has_aux = PLAIN ? false : (p.w_aux != nullptr);
    const double cdt = rhs_only ? 1.0 : p.rk_c * p.scal[0];
    const bool need_n = !rhs_only, need_p = !rhs_only && p.rk_b != 0.0;
    const double cdtp = cdt * pref;
    const bool sens_stage = p.do_sensor != 0;
    if (tid < MM) sS[tid] = c_tab.S[(tid / M) * 8 + tid % M];
    auto cbar = [&]() { __syncthreads(); };       // barrier between the phases
    {   // one tile per block
        const TilePos<D, C> pos(p, cl);
        const int cell0 = pos.cell0;
        const int cg = pos.cg;
        const bool active = pos.active;
        int nbm[D];                               // lower neighbour along each axis (periodic wrap)
#pragma unroll
        for (int a = 0; a < D; ++a) nbm[a] = pos.lower(p, a);
        if (AV && tid < C) {
            // wiggle source of Eq. 45 from the previous step's sensor (readings A14, A15)
            const int c = min(cell0 + tid, p.ncells - 1);
            const double S = p.sens_prev[c];
            const double G = p.sens_prev[p.ncells + c];
            Wk[tid] = (S > p.s_onset) ? p.f_w * fmax(0.0, G) : 0.0;
        }

        // ---- A: own modes, global -> register tile; expansion along x and y (Eq. 21) ----
        for (int it = tid; it < V * NTILE * C; it += NT) {
            const int g = it / C;                 // v*NTILE + lz
            const int v = g / NTILE, lz = g % NTILE;
            double t[MM];
            const double *src = p.w_prev + (size_t)(lz * MM * V + v) * p.ncells + cg;
#pragma unroll
            for (int q = 0; q < MM; ++q) t[q] = __ldg(row_ptr(src, q * V, p.ncells));
            tile_x<DG_SEL_V, M>(t);
            tile_y<DG_SEL_V, M>(t);
            tile_store<M, C, L>(U, g, cl, t);
            if (D == 2 && GRAD && v < Vc) {
                double a[MM];
#pragma unroll
                for (int q = 0; q < MM; ++q) a[q] = t[q];
                tile_x<DG_SEL_DHAT, M>(a);
                tile_store<M, C, L>(GR, g, cl, a);
                tile_y<DG_SEL_DHAT, M>(t);
                tile_store<M, C, L>(GR, Vc * NTILE + g, cl, t);
            }
        }
        cbar();
        if (D == 3) {
            // ---- B: expansion along z, z derivative ----
            constexpr int NKB = (V * MM * C + NT - 1) / NT;
#pragma unroll kUnrollB
            for (int kb = 0; kb < NKB; ++kb) {
                const int it = tid + kb * NT;
                if (it >= V * MM * C) break;
                const int r = it / C;
                const int q = r % MM, v = r / MM;
                double in[M], u[M];
#pragma unroll
                for (int l = 0; l < M; ++l) in[l] = U[L::at2(v, q + l * MM) * C + cl];
                apply1d<DG_SEL_V, M>(in, u);
#pragma unroll
                for (int j = 0; j < M; ++j) U[L::at2(v, q + j * MM) * C + cl] = u[j];
                if (GRAD && v < Vc) {
                    double gz[M];
                    apply1d<DG_SEL_DHAT, M>(u, gz);
#pragma unroll
                    for (int j = 0; j < M; ++j) GR[L::at2(2 * Vc + v, q + j * MM) * C + cl] = gz[j];
                }
            }
            cbar();
            if (GRAD) {
                // ---- D: x and y derivatives of the nodal values, one tile load for both ----
                for (int it = tid; it < Vc * NTILE * C; it += NT) {
                    const int g = it / C;
                    double t[MM], a[MM];
                    tile_load<M, C, L>(U, g, cl, t);
#pragma unroll
                    for (int q = 0; q < MM; ++q) a[q] = t[q];
                    tile_x<DG_SEL_DHAT, M>(a);
                    tile_store<M, C, L>(GR, g, cl, a);
                    tile_y<DG_SEL_DHAT, M>(t);
                    tile_store<M, C, L>(GR, Vc * NTILE + g, cl, t);
                }
                cbar();
            }
        }
        {
            // ---- E: point-wise fluxes G_a = f_a - F_NS,a - eps d_a u (Eq. 24; 315 Eq. 38), alpha source ----
            bool bad = false;
            double amax = 0.0;                                     // max alpha at the Gauss points (diagnostics)
            const double decay = (double)M / (p.f_tau * p.h);      // 1/tau = (n+1) c_s / (f_tau h), Eq. 44
            constexpr int NKE = (Np * C + NT - 1) / NT;
#pragma unroll kUnrollE
            for (int ke = 0; ke < NKE; ++ke) {
                const int it = tid + ke * NT;
                if (it >= Np * C) break;
                const int j = it / C;
                double u[Vc];
#pragma unroll
                for (int v = 0; v < Vc; ++v) u[v] = U[L::at2(v, j) * C + cl];
                const Prim<D> q = primitives<D>(u, p.gamma);
                bad |= !(q.rho > 0.0) || !(q.p > 0.0);
                // the gradient arrays hold d/dxi (reference coordinates): the factor 2/h of the cell map is folded
                // into the two scalars that multiply them, 1/rho (velocity and temperature gradients) and eps
                double g[D][D + 2 + DG_TRACER], dv[D][D];
                double divv = 0.0, epss = 0.0;
                const double gs = 2.0 * ih;
                const double irs = q.ir * gs;
                if (GRAD) {
#pragma unroll
                    for (int b = 0; b < D; ++b)
#pragma unroll
                        for (int v = 0; v < Vc; ++v) g[b][v] = GR[L::at2(b * Vc + v, j) * C + cl];
                    // dv[b][c] = d v_c / d x_b = (d_b(rho v_c) - v_c d_b rho) / rho
#pragma unroll
                    for (int b = 0; b < D; ++b)
#pragma unroll
                        for (int c = 0; c < D; ++c) dv[b][c] = (g[b][1 + c] - q.v[c] * g[b][0]) * irs;
#pragma unroll
                    for (int b = 0; b < D; ++b) divv += dv[b][b];
                }
                if (AV) {
                    const double al = U[L::at2(Vc, j) * C + cl];
                    const double cs = fast_sqrt(p.gamma * q.p * q.ir);
                    if (active) amax = fmax(amax, al);
                    epss = fmin(fmax(al, 0.0), p.alpha_max) * cs * (p.h / (double)M) * gs;        // Eq. 46, A17
                    // Eq. 43-45: shock source + wiggle source - decay; stored pre-scaled by h/2 for the projection
                    const double src = p.f_v * fmax(0.0, -divv) + Wk[cl] - al * (cs * decay);
                    U[L::at2(Vc, j) * C + cl] = 0.5 * p.h * src;
                }
                // Navier-Stokes stress (Eq. 38-39, traceless Pi, reading A7): symmetric, formed once for the D axes
                double Pi[D][D], qh[D];
                if (VISC) {
                    const double mu = p.nu * q.rho, kq = p.chi * (p.gamma - 1.0) * q.rho;
                    const double tt = (2.0 / 3.0) * divv, eir = q.e * q.ir;
#pragma unroll
                    for (int a = 0; a < D; ++a) {
#pragma unroll
                        for (int b = a; b < D; ++b) {
                            Pi[a][b] = mu * (dv[a][b] + dv[b][a] - (a == b ? tt : 0.0));
                            Pi[b][a] = Pi[a][b];
                        }
                    }
#pragma unroll
                    for (int a = 0; a < D; ++a) {
                        // chi (gamma-1) rho d_a u_th,  u_th = e/rho - v^2/2
                        double vdv = 0.0;
#pragma unroll
                        for (int c = 0; c < D; ++c) vdv = fma(q.v[c], dv[a][c], vdv);
                        qh[a] = kq * ((g[a][1 + D] - eir * g[a][0]) * irs - vdv);
                    }
                }
#pragma unroll
                for (int a = 0; a < D; ++a) {
                    double F[Vc];
                    euler_flux<D>(u, q, a, F);
                    if (VISC) {
                        double ev = qh[a];
#pragma unroll
                        for (int b = 0; b < D; ++b) {
                            F[1 + b] -= Pi[a][b];
                            ev = fma(q.v[b], Pi[a][b], ev);
                        }
                        F[1 + D] -= ev;
                        // tracer diffusion eta rho d_a c (Eq. 40); the gradient arrays are in reference coordinates
                        if (DG_TRACER) F[Vc - 1] -= p.eta * gs * (g[a][Vc - 1] - (u[Vc - 1] * q.ir) * g[a][0]);
                    }
                    if (AV) {
#pragma unroll
                        for (int v = 0; v < Vc; ++v) F[v] = fma(-epss, g[a][v], F[v]);
                    }
#pragma unroll
                    for (int v = 0; v < Vc; ++v) GR[L::at2(a * Vc + v, j) * C + cl] = F[v];
                }
            }
            if (bad) atomicOr(p.flag, 1);
            if (AV && p.do_sensor) {
                // running maximum of alpha over the states at the start of every step (dg_get_diagnostics)
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) amax = fmax(amax, __shfl_xor_sync(0xffffffffu, amax, o));
                if ((tid & 31) == 0) red[tid >> 5] = amax;
            }
        }
        // face fluxes of this thread's G items, requested before the barrier: x faces as nodal values (jy, jz), y faces
        // modal in x and nodal in z (Cfg::PP); own cell = upper face, lower neighbour's = lower face
        constexpr int NKG = (V * NTILE * C + NT - 1) / NT;
        double gf[NKG][4][M];
#pragma unroll
        for (int k = 0; k < NKG; ++k) {
            const int g = (tid + k * NT) / C;     // v*NTILE + jz
            const int v = g / NTILE, jz = g % NTILE;
#pragma unroll
            for (int i = 0; i < M; ++i) gf[k][0][i] = gf[k][1][i] = gf[k][2][i] = gf[k][3][i] = 0.0;
            if (g < Vc * NTILE) {
                const double *fx = p.flux + (size_t)((0 * Vc + v) * Nf + jz * M) * p.ncells;
                const double *fy = p.flux + (size_t)((1 * Vc + v) * Nf + jz * M) * p.ncells;
                const double *fx0 = fx + cg, *fx1 = fx + nbm[0], *fy0 = fy + cg, *fy1 = fy + nbm[1];
#pragma unroll
                for (int i = 0; i < M; ++i) {
                    gf[k][0][i] = __ldg(row_ptr(fx0, i, p.ncells));
                    gf[k][1][i] = __ldg(row_ptr(fx1, i, p.ncells));
                    gf[k][2][i] = __ldg(row_ptr(fy0, i, p.ncells));
                    gf[k][3][i] = __ldg(row_ptr(fy1, i, p.ncells));
                }
            }
        }
        cbar();
        if (AV && p.do_sensor && tid == 0) {
            double a = red[0];
            for (int i = 1; i < NT / 32; ++i) a = fmax(a, red[i]);   // NT / 32 = the warps that ran phase E
            atomic_max_nonneg(&p.maxbits[2], a);
        }

        double sA = 0.0, sB = 0.0, dA = 0.0, dB = 0.0;      // shock-sensor sums of Eq. 42 (readings A13/A15)

        // ---- G: weak-form derivative N = sum_a S_a G_a, projection along x and y, lift of the x and y faces ----
#pragma unroll
        for (int k = 0; k < NKG; ++k) {
            const int g = (tid + k * NT) / C;     // v*NTILE + jz
            if (g >= V * NTILE) break;
            const int v = g / NTILE, jz = g % NTILE;
            double n[MM];
            if (v < Vc) {
                double b[MM];
                tile_load<M, C, L>(GR, (0 * Vc + v) * NTILE + jz, cl, n);
                tile_x<DG_SEL_S, M>(n);
                tile_load<M, C, L>(GR, (1 * Vc + v) * NTILE + jz, cl, b);
                tile_y_acc<DG_SEL_S, M>(b, n);
                if (D == 3) {
#pragma unroll
                    for (int kk = 0; kk < NTILE; ++kk) {
                        tile_load<M, C, L>(GR, (2 * Vc + v) * NTILE + kk, cl, b);
                        const double s = sS[jz * M + kk];
#pragma unroll
                        for (int q = 0; q < MM; ++q) n[q] = fma(s, b[q], n[q]);
                    }
                }
                tile_x<DG_SEL_VTG, M>(n);
#pragma unroll
                for (int y = 0; y < M; ++y)
#pragma unroll
                    for (int x = 0; x < M; ++x)
                        n[y * M + x] = fma(-c_tab.Pend[1][x], gf[k][0][y], fma(c_tab.Pend[0][x], gf[k][1][y], n[y * M + x]));
                tile_y<DG_SEL_VTG, M>(n);
#pragma unroll
                for (int y = 0; y < M; ++y)
#pragma unroll
                    for (int x = 0; x < M; ++x)
                        n[y * M + x] = fma(-c_tab.Pend[1][y], gf[k][2][x], fma(c_tab.Pend[0][y], gf[k][3][x], n[y * M + x]));
            } else {
                tile_load<M, C, L>(U, g, cl, n);      // alpha source (slot Vc of U)
                tile_x<DG_SEL_VTG, M>(n);
                tile_y<DG_SEL_VTG, M>(n);
            }
            if (D == 3) {
                tile_store<M, C, L>(U, g, cl, n);
            } else {
                // 2D: dw/dt of this (cell, variable) is complete: stage combine from registers
                const double *bn = p.w_n + (size_t)v * p.ncells + cg;
                const double *bp = p.w_prev + (size_t)v * p.ncells + cg;
                double *bo = p.w_out + (size_t)v * p.ncells + cg;
                double wn[MM], wp[MM];
                double gdev = 0.0;
#pragma unroll
                for (int q = 0; q < MM; ++q) {
                    wn[q] = need_n ? *row_ptr(bn, q * V, p.ncells) : 0.0;
                    wp[q] = need_p ? __ldg(row_ptr(bp, q * V, p.ncells)) : 0.0;
                }
#pragma unroll
                for (int q = 0; q < MM; ++q) {
                    const bool keep = !total_degree || (q % M + q / M <= M - 1);
                    const double Ld = keep ? pref * n[q] : 0.0;
                    double wnew = Ld;
                    if (!rhs_only) wnew = fma(cdt, Ld, fma(p.rk_b, wp[q], p.rk_a * wn[q]));
                    if (active) *row_ptr(bo, q * V, p.ncells) = wnew;
                    if (has_aux && active) {
                        const size_t gi = (size_t)(q * V + v) * p.ncells + cg;
                        p.w_aux[gi] = fma(p.aux_c * p.scal[0], Ld, fma(p.aux_b, wp[q], p.aux_a * p.w_aux_in[gi]));
                    }
                    if (AV && p.do_sensor && v == 0) {
                        const bool top = total_degree ? (q % M + q / M == M - 1) : ((q % M == M - 1) || (q / M == M - 1));
                        sB = fma(wn[q], wn[q], sB);
                        dB = fma(wn[q], Ld, dB);
                        if (top) {
                            sA = fma(wn[q], wn[q], sA);
                            dA = fma(wn[q], Ld, dA);
                        }
                    }
                    n[q] = wnew;
                    if (lim && v < Vc && q != 0) gdev = fma(fabs(wnew), c_tab.Pend[1][q % M] * c_tab.Pend[1][q / M], gdev);
                }
                if (lim && v < Vc) {
                    atomicAdd(&ldev[v * C + cl], gdev);
                    tile_store<M, C, L>(U, g, cl, n);         // new modes: the limiter expands them itself
                } else if (p.do_wavespeed && v < Vc) {
                    tile_x<DG_SEL_V, M>(n);
                    tile_y<DG_SEL_V, M>(n);
                    tile_store<M, C, L>(U, g, cl, n);
                }
            }
        }
        if (D == 3) {
            // ---- H: projection along z, lift of the z faces, stage combine straight to global memory ----
            // every global input of this thread's items (u^n, u^(i-1), the two z-face fluxes) is requested before the
            // barrier, so that one memory round trip covers them all and overlaps the wait for the other warps
            constexpr int NKH = (V * MM * C + NT - 1) / NT;
            constexpr int HP = NKH;              // items per load batch: all of them
#pragma unroll
            for (int k0 = 0; k0 < NKH; k0 += HP) {
            double hwn[HP][M], hwp[HP][M], hfz[HP][2];
#pragma unroll
            for (int k = 0; k < HP; ++k) {
                const int r = (tid + (k0 + k) * NT) / C;
                const int q = r % MM, v = r / MM;     // q = ly*M + lx
                hfz[k][0] = hfz[k][1] = 0.0;
#pragma unroll
                for (int l = 0; l < M; ++l) hwn[k][l] = hwp[k][l] = 0.0;
                if (r < V * MM) {
                    if (v < Vc) {
                        const double *fz = p.flux + (size_t)((2 * Vc + v) * Nf + q) * p.ncells;
                        hfz[k][0] = __ldg(fz + cg);
                        hfz[k][1] = __ldg(fz + nbm[D - 1]);
                    }
                    const double *bn = p.w_n + (size_t)(q * V + v) * p.ncells + cg;
                    const double *bp = p.w_prev + (size_t)(q * V + v) * p.ncells + cg;
#pragma unroll
                    for (int l = 0; l < M; ++l) {
                        if (need_n) hwn[k][l] = *row_ptr(bn, l * MM * V, p.ncells);
                        if (need_p) hwp[k][l] = __ldg(row_ptr(bp, l * MM * V, p.ncells));
                    }
                }
            }
            if (k0 == 0) cbar();
#pragma unroll
            for (int k = 0; k < HP; ++k) {
                const int r = (tid + (k0 + k) * NT) / C;
                if (r >= V * MM) break;
                const int q = r % MM, v = r / MM;
                double *bo = p.w_out + (size_t)(q * V + v) * p.ncells + cg;
                double in[M];
#pragma unroll
                for (int j = 0; j < M; ++j) in[j] = U[L::at2(v, q + j * MM) * C + cl];
                const bool topxy = (q % M == M - 1) || (q / M == M - 1);
                const int lxy = q % M + q / M;
                const double bq = c_tab.Pend[1][q % M] * c_tab.Pend[1][q / M];   // max |P_lx P_ly| on the cell
                double hdev = 0.0;
                double pz[M];
                apply1d<DG_SEL_VTG, M>(in, pz);
#pragma unroll
                for (int l = 0; l < M; ++l) {
                    double acc = pz[l];
                    if (v < Vc) acc = fma(-c_tab.Pend[1][l], hfz[k][0], fma(c_tab.Pend[0][l], hfz[k][1], acc));
                    // total-degree basis: the discarded modes are not test functions of Eq. 20
                    const bool keep = !total_degree || (lxy + l <= M - 1);
                    double Ld, wnew;
                    if (PLAIN) {
                        // prefactor folded into the combine; dw/dt itself is needed by the sensor sums only
                        wnew = fma(cdtp, acc, fma(p.rk_b, hwp[k][l], p.rk_a * hwn[k][l]));
                        Ld = (AV && sens_stage) ? pref * acc : 0.0;
                    } else {
                        Ld = keep ? pref * acc : 0.0;
                        wnew = Ld;
                        if (!rhs_only) wnew = fma(cdt, Ld, fma(p.rk_b, hwp[k][l], p.rk_a * hwn[k][l]));
                    }
                    if (active) *row_ptr(bo, l * MM * V, p.ncells) = wnew;
                    if (has_aux && active) {
                        const size_t gi = (size_t)((l * MM + q) * V + v) * p.ncells + cg;
                        p.w_aux[gi] = fma(p.aux_c * p.scal[0], Ld, fma(p.aux_b, hwp[k][l], p.aux_a * p.w_aux_in[gi]));
                    }
                    if (AV && p.do_sensor && v == 0) {
                        sB = fma(hwn[k][l], hwn[k][l], sB);
                        dB = fma(hwn[k][l], Ld, dB);
                        if (total_degree ? (lxy + l == M - 1) : (topxy || l == M - 1)) {
                            sA = fma(hwn[k][l], hwn[k][l], sA);
                            dA = fma(hwn[k][l], Ld, dA);
                        }
                    }
                    if (p.do_wavespeed || lim) U[L::at2(v, q + l * MM) * C + cl] = wnew;
                    if (lim && v < Vc && (q + l) != 0) hdev = fma(fabs(wnew), bq * c_tab.Pend[1][l], hdev);
                }
                if (lim && v < Vc) atomicAdd(&ldev[v * C + cl], hdev);
            }
            }   // load batches of phase H
        }
        if (AV && p.do_sensor) {
            // lanes of a warp that share a cell (lane = cl + C*j), then one partial per warp and cell in `sens`
            constexpr int NW = NT / 32;
#pragma unroll
            for (int o = C; o < 32; o <<= 1) {
                sA += __shfl_xor_sync(0xffffffffu, sA, o);
                sB += __shfl_xor_sync(0xffffffffu, sB, o);
                dA += __shfl_xor_sync(0xffffffffu, dA, o);
                dB += __shfl_xor_sync(0xffffffffu, dB, o);
            }
            if ((tid & 31) < C) {
                sens[(0 * NW + tid / 32) * C + cl] = sA;
                sens[(1 * NW + tid / 32) * C + cl] = sB;
                sens[(2 * NW + tid / 32) * C + cl] = dA;
                sens[(3 * NW + tid / 32) * C + cl] = dB;
            }
            cbar();
            if (tid < C && cell0 + tid < p.ncells) {
                double s[4] = {0.0, 0.0, 0.0, 0.0};
                for (int k = 0; k < NW; ++k)
#pragma unroll
                    for (int i = 0; i < 4; ++i) s[i] += sens[(i * NW + k) * C + tid];
                const int c = cell0 + tid;
                p.sens_new[c] = s[0] / s[1];
                p.sens_new[p.ncells + c] = (s[0] > 0.0) ? (2.0 * s[2] / s[0] - 2.0 * s[3] / s[1]) : 0.0;
            }
        }
        if (AV && p.commit_sensor && tid < C && cell0 + tid < p.ncells) {
            const int c = cell0 + tid;
            p.sens_prev[c] = p.sens_new[c];
            p.sens_prev[p.ncells + c] = p.sens_new[p.ncells + c];
        }
        if (lim) {
            // ---- positivity limiter on the stage output (Eq. 47; readings L1-L6), fused: the new
            //      modes of the d+2 conserved fields are still in U, the face point values go to the (now free) flux
            //      array; cells with F != 1 re-read their freshly written rows (L2) and scale every mode but the mean ----
            //      Shortcut that cannot change the result: |phi_l| <= prod_a sqrt(2 l_a + 1) on the whole cell, so
            //      rho >= rho_bar - dev_rho, |m_b| <= |m_bar_b| + dev_b, e >= e_bar - dev_e at every evaluation point;
            //      if these bounds already keep rho and p above their floors (with a factor 2 of margin) in all cells
            //      of the block, F = 1 exactly as the full evaluation would find, and the evaluation is skipped.
            __syncthreads();
            int full = 0;
            if (tid < C && cell0 + tid < p.ncells) {
                double mb[Vc], dv_[Vc];
#pragma unroll
                for (int v = 0; v < Vc; ++v) {
                    mb[v] = U[L::at2(v, 0) * C + tid];
                    dv_[v] = ldev[v * C + tid];
                }
                double mm = 0.0, mh = 0.0;
#pragma unroll
                for (int b = 0; b < D; ++b) {
                    mm = fma(mb[1 + b], mb[1 + b], mm);
                    const double hi = fabs(mb[1 + b]) + dv_[1 + b];
                    mh = fma(hi, hi, mh);
                }
                const double pbar = (p.gamma - 1.0) * (mb[1 + D] - 0.5 * mm / mb[0]);
                const double rlo = mb[0] - dv_[0];
                const double plo = (p.gamma - 1.0) * ((mb[1 + D] - dv_[1 + D]) - 0.5 * mh / rlo);
                const bool safe = (mb[0] > 0.0) && (pbar > 0.0) && (rlo > 2.0e-6 * mb[0]) && (plo > 2.0e-6 * pbar);
                full = safe ? 0 : 1;
            }
            full = __syncthreads_or(full);
            const LimScratch<D, C> sc(limsc);
            if (full) limiter_core<D, M, C, NT, true, L>(U, GR, sc, p.gamma, p.flag, cell0, p.ncells, tid);
            const double F = full ? sc.Fc[cl] : 1.0;
            if (F != 1.0 && active) {
                for (int r = tid / C; r < Vc * Np; r += NT / C) {
                    const int v = r % Vc, mode = r / Vc;
                    if (mode == 0) continue;
                    double *q = p.w_out + (size_t)(mode * V + v) * p.ncells + cg;
                    *q = F * __ldcg(q);
                }
            }
            // wave speeds of the limited state (reading L6): u(x) = u_bar + F (u(x) - u_bar) at the volume points
            if (p.do_wavespeed && !full) {
                expand_volume<D, M, C, NT, true, L>(U, Vc, tid);
                wavespeed_points<D, M, C, NT, L>(U, p.gamma, p.flag, red, p.maxbits, tid);
            } else if (p.do_wavespeed) {
                double cmax = 0.0, vmax = 0.0;
                bool bad = false;
                for (int it = tid; it < Np * C; it += NT) {
                    const int j = it / C;
                    double u[Vc];
#pragma unroll
                    for (int v = 0; v < Vc; ++v) {
                        const double x = U[L::at2(v, j) * C + cl], mv = sc.mean[v * C + cl];
                        u[v] = (F == 1.0) ? x : fma(F, x - mv, mv);
                    }
                    const Prim<D> q = primitives<D>(u, p.gamma);
                    bad |= !(q.rho > 0.0) || !(q.p > 0.0);
                    double v2 = 0.0;
#pragma unroll
                    for (int b = 0; b < D; ++b) v2 = fma(q.v[b], q.v[b], v2);
                    const double cs = fast_sqrt(p.gamma * q.p * q.ir);
                    const double vm = fast_sqrt(v2);
                    cmax = (cs > cmax) ? cs : cmax;
                    vmax = (vm > vmax) ? vm : vmax;
                }
                if (bad) atomicOr(p.flag, 4);
                block_max2<NT>(cmax, vmax, red, p.maxbits, tid);
            }
        } else if (p.do_wavespeed) {
            // ---- wave speeds of the new state for the next step's Eq. 23 ----
            __syncthreads();
            if (D == 3) expand_volume<D, M, C, NT, true, L>(U, Vc, tid);
            wavespeed_points<D, M, C, NT, L>(U, p.gamma, p.flag, red, p.maxbits, tid);
        }
    }
}

}  // namespace DG_NS
