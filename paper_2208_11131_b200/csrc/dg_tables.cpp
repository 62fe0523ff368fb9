// Host-side construction of the 1D tables (see dg_tables.h).  long double throughout, rounded once.
#include "dg_tables.h"

#include <cmath>
#include <cstring>

namespace {

typedef long double ld;

// Legendre polynomials Leg_0..Leg_lmax and derivatives at x (Bonnet recurrence).
void legendre(int lmax, ld x, ld *L, ld *dL) {
    L[0] = 1.0L;
    dL[0] = 0.0L;
    if (lmax >= 1) {
        L[1] = x;
        dL[1] = 1.0L;
    }
    for (int l = 1; l < lmax; ++l) {
        L[l + 1] = ((2 * l + 1) * x * L[l] - l * L[l - 1]) / (l + 1);
        dL[l + 1] = dL[l - 1] + (2 * l + 1) * L[l];
    }
}

// Normalised P_l = sqrt(2l+1) Leg_l (Eq. 13) and derivative.
void legendre_norm(int lmax, ld x, ld *P, ld *dP) {
    legendre(lmax, x, P, dP);
    for (int l = 0; l <= lmax; ++l) {
        ld s = sqrtl((ld)(2 * l + 1));
        P[l] *= s;
        dP[l] *= s;
    }
}

// q-point Gauss-Legendre rule on [-1, 1] (ascending nodes), Newton iteration on Leg_q.
void gauss(int q, ld *x, ld *g) {
    const ld pi = acosl(-1.0L);
    ld L[DG_MAXM + 4], dL[DG_MAXM + 4];
    for (int i = 0; i < q; ++i) {
        ld xi = -cosl(pi * (i + 0.75L) / (q + 0.5L));
        for (int it = 0; it < 100; ++it) {
            legendre(q, xi, L, dL);
            ld dx = L[q] / dL[q];
            xi -= dx;
            if (fabsl(dx) < 1e-19L) break;
        }
        legendre(q, xi, L, dL);
        x[i] = xi;
        g[i] = 2.0L / ((1.0L - xi * xi) * dL[q] * dL[q]);
    }
    // exact antisymmetry of the node set
    for (int i = 0; i < q / 2; ++i) {
        ld a = 0.5L * (x[q - 1 - i] - x[i]);
        x[i] = -a;
        x[q - 1 - i] = a;
        ld w = 0.5L * (g[i] + g[q - 1 - i]);
        g[i] = g[q - 1 - i] = w;
    }
    if (q % 2) x[q / 2] = 0.0L;
}

}  // namespace

void dg_build_tables(int m, DgTables *t) {
    std::memset(t, 0, sizeof(*t));
    const int n = m - 1;
    ld x[DG_MAXM], g[DG_MAXM];
    gauss(m, x, g);
    ld V[DG_MAXM][DG_MAXM], D[DG_MAXM][DG_MAXM], Dh[DG_MAXM][DG_MAXM];
    for (int j = 0; j < m; ++j) {
        ld P[DG_MAXM + 2], dP[DG_MAXM + 2];
        legendre_norm(n, x[j], P, dP);
        for (int l = 0; l < m; ++l) {
            V[j][l] = P[l];
            D[j][l] = dP[l];
        }
    }
    // V^T G V = 2 I  =>  V^-1 = 1/2 V^T G;  Dhat = D V^-1
    for (int j = 0; j < m; ++j)
        for (int i = 0; i < m; ++i) {
            ld s = 0.0L;
            for (int l = 0; l < m; ++l) s += D[j][l] * V[i][l];
            Dh[j][i] = 0.5L * s * g[i];
        }
    for (int j = 0; j < m; ++j) {
        t->x[j] = (double)x[j];
        t->g[j] = (double)g[j];
        for (int l = 0; l < m; ++l) {
            t->V[j * 8 + l] = (double)V[j][l];
            t->Dhat[j * 8 + l] = (double)Dh[j][l];
            t->S[j * 8 + l] = (double)(Dh[l][j] * g[l] / g[j]);
            t->VtG[l * 8 + j] = (double)(V[j][l] * g[j]);
        }
    }
    // even-odd forms of the two nodal -> nodal matrices (dg_stage.cuh apply1d): half-sums / half-differences of the
    // mirrored columns, formed in long double
    for (int j = 0; j < m; ++j)
        for (int i = 0; i < m / 2; ++i) {
            const ld sji = Dh[i][j] * g[i] / g[j], sjm = Dh[m - 1 - i][j] * g[m - 1 - i] / g[j];
            t->DhatE[j * 8 + i] = (double)(0.5L * (Dh[j][i] + Dh[j][m - 1 - i]));
            t->DhatO[j * 8 + i] = (double)(0.5L * (Dh[j][i] - Dh[j][m - 1 - i]));
            t->SE[j * 8 + i] = (double)(0.5L * (sji + sjm));
            t->SO[j * 8 + i] = (double)(0.5L * (sji - sjm));
        }
    {
        ld P[DG_MAXM + 2], dP[DG_MAXM + 2];
        legendre_norm(n, -1.0L, P, dP);
        for (int l = 0; l < m; ++l) t->Pend[0][l] = (double)P[l];
        legendre_norm(n, +1.0L, P, dP);
        for (int l = 0; l < m; ++l) t->Pend[1][l] = (double)P[l];
    }
    // Recovery: the two cells' expansions are L2-projected onto one polynomial of degree
    // n+1 over K* (fraction f of each cell).  A^-_{k,l} = int_{-1}^{0} P_k(2 f s + 1) P_l(s) ds and
    // A^+_{k,l} = int_{0}^{1} P_k(2 f s - 1) P_l(s) ds (Eq. 33-34, A9); q_l = 1/2 sum_k [A^- w^- + A^+ w^+]
    // (Eq. 35 with prefactor 1/2 and the full sum, A10); value and normal derivative at s = 0 (Eq. 31).
    const ld f = (n <= 2) ? 0.75L : 1.0L;
    const int q = n + 2;
    ld xq[DG_MAXM + 2], gq[DG_MAXM + 2];
    gauss(q, xq, gq);
    ld P0[DG_MAXM + 2], dP0[DG_MAXM + 2];
    legendre_norm(n + 1, 0.0L, P0, dP0);
    for (int side = 0; side < 2; ++side) {
        for (int k = 0; k < m; ++k) {
            ld R = 0.0L, G = 0.0L;
            for (int l = 0; l <= n + 1; ++l) {
                ld A = 0.0L;
                for (int i = 0; i < q; ++i) {
                    ld s = (side == 0) ? 0.5L * (xq[i] - 1.0L) : 0.5L * (xq[i] + 1.0L);
                    ld xc = (side == 0) ? 2.0L * f * s + 1.0L : 2.0L * f * s - 1.0L;
                    ld Pc[DG_MAXM + 2], dPc[DG_MAXM + 2], Ps[DG_MAXM + 2], dPs[DG_MAXM + 2];
                    legendre_norm(n, xc, Pc, dPc);
                    legendre_norm(n + 1, s, Ps, dPs);
                    A += 0.5L * gq[i] * Pc[k] * Ps[l];
                }
                R += 0.5L * A * P0[l];
                G += 0.5L * A * dP0[l] / f;
            }
            t->Rv[side][k] = (double)R;
            t->Gv[side][k] = (double)G;
        }
    }
}
