// 1D basis / quadrature / recovery tables of the DG operator (S0 of DESIGN.md), built on the host in
// long double and rounded once to fp64.  Every m x m matrix is stored with a fixed row stride of 8 so that
// fully unrolled device loops address it with compile-time offsets (constant-bank operands of DFMA).
//
//   out[r] = sum_c  MAT[r*8 + c] * in[c]       for every matrix below
//
// PAPER.md:125 (Eq. 13) normalised Legendre P_l; 164-171 (Eq. 19) Gauss-Legendre rule with m = n+1 points;
// 287-301 (Eq. 33-35, readings A9/A10) recovery overlap integrals.
#pragma once

#define DG_MAXM 8

struct DgTables {
    double V[DG_MAXM * 8];     // V[j][l]   = P_l(x_j)                     modal -> nodal
    double Dhat[DG_MAXM * 8];  // Dhat[j][i]= (D V^-1)[j][i]               nodal -> d/dxi at the nodes
    double S[DG_MAXM * 8];     // S[j'][j]  = Dhat[j][j'] g_j / g_j'       weak-form derivative, nodal -> nodal
    double VtG[DG_MAXM * 8];   // VtG[l][j] = P_l(x_j) g_j                 weighted nodal -> modal projection
    double DhatE[DG_MAXM * 8]; // (Dhat[j][i] + Dhat[j][m-1-i]) / 2, i < m/2   even-odd form of Dhat (centro-antisymmetric)
    double DhatO[DG_MAXM * 8]; // (Dhat[j][i] - Dhat[j][m-1-i]) / 2
    double SE[DG_MAXM * 8];    // same for S
    double SO[DG_MAXM * 8];
    double Pend[2][8];         // P_l(-1), P_l(+1)                         face traces
    double Rv[2][8];           // R^-_l (left cell), R^+_l (right cell)    recovered interface value
    double Gv[2][8];           // G^-_l, G^+_l                             recovered interface normal derivative * h
    double g[8];               // Gauss weights
    double x[8];               // Gauss nodes
};

// Fill `t` for m = order Gauss points (degree n = m-1).  Recovery fraction f = 3/4 for n <= 2, else 1
// (PAPER.md:301).
void dg_build_tables(int m, DgTables *t);
