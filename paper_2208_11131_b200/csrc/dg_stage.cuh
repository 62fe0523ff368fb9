// Runge-Kutta-stage kernels of the modal DG operator (sm_100a, fp64 CUDA cores).
//
// One SSP-RK stage (Eq. 20-21, 200) = two launches over the whole mesh:
//   dg_face_kernel   every cell owns its D upper faces: one-sided traces and recovery partial sums of both
//                    adjacent cells, HLLC + recovery-based viscous / artificial-viscosity flux
//                     ONCE per face point, projected on the transverse modes -> `flux`
//   dg_stage_kernel  lift of the 2D face fluxes, volume term (Eq. 21 expansion by sum factorisation, Euler /
//                    Navier-Stokes / AV flux, weak-form derivative, projection), shock-sensor bookkeeping, stage
//                    combine and -- on the last stage -- the wave-speed maxima of Eq. 23 for the next step.
// dw/dt never touches HBM; the only intermediate in HBM is the projected face flux (D*Vc*m^(D-1) per cell).
//
// Shared-memory layout per block (doubles):  [slot][point][cell], cell fastest (C cells), so that a warp
// whose lanes are consecutive cells reads/writes conflict-free and global accesses coalesce along `cell`
// (state layout w[(mode*V + var)*Ncells + cell]).
//   stage kernel:  RA  V x Np  own modes -> nodal values (in place);  RX  D*Vc*Np  gradients -> fluxes (in place);
//                  ACC V x Np  dw/dt in modal space
//   face kernel:   RA  V x Np  own modes;  RX  NQ x Nf  traces / recovered state / gradients of one face
// No float atomics in anything that reaches the state, no races: each cell's dw/dt is a fixed-order sum
// (bit-reproducible run to run).  The one exception is harmless by construction: the fused positivity limiter of
// dg_stage2_kernel accumulates the bound sum_{l>0} |w_l| max|phi_l| per cell with a shared-memory atomicAdd(double),
// whose order can change the bound in the last bits -- but the bound only decides whether the full point evaluation
// can be skipped (with a factor 2 of margin), and both branches produce the same F, so no output bit depends on it.
#pragma once

#include <cuda_runtime.h>

#include "dg_tables.h"

#include "dg_stage_args.h"

#define DG_SEL_V 0
#define DG_SEL_DHAT 1
#define DG_SEL_S 2
#define DG_SEL_VTG 3

// passive tracer (Eq. 40): one more conserved row c rho behind the energy.  A compile-time switch of the
// translation unit (dg_stage_inst.cu is built with -DDG_TRACER=0 and =1), so the default kernels are unchanged.
#ifndef DG_TRACER
#define DG_TRACER 0
#endif
// kernels of the two builds live in different namespaces: equal template instantiations from different translation
// units would otherwise be merged by the linker
#if DG_TRACER
#define DG_NS dgkt
#else
#define DG_NS dgk
#endif
#ifndef DG_AOSOA
#define DG_AOSOA 1
#endif
#ifndef DG_EVEN_ODD
#define DG_EVEN_ODD 1
#endif

#ifndef DG_STAGE_NT
#define DG_STAGE_NT 512
#endif
#ifndef DG_STAGE_NT_BIG
#define DG_STAGE_NT_BIG 768
#endif
#ifndef DG_FACE_NT_BIG
#define DG_FACE_NT_BIG 512
#endif
#ifndef DG_STAGE_MINB
#define DG_STAGE_MINB 1
#endif
#ifndef DG_FACE_NT
#define DG_FACE_NT 256
#endif
#ifndef DG_FACE_DIRECT
#define DG_FACE_DIRECT 1
#endif
// row rotation of the pencil-sweep layouts: only where the row index arithmetic is shifts (m = 8); at m = 6 the
// divisions by 6 cost more than the bank conflicts they avoid (stage kernel 2.80 -> 2.50 ms without it)
#ifndef DG_ROT_NONPOW2
#define DG_ROT_NONPOW2 0
#endif
#ifndef DG_ROT_ENABLE
#define DG_ROT_ENABLE 1
#endif
#ifndef DG_FACE_BIG_MINB
#define DG_FACE_BIG_MINB 1
#endif
#ifndef DG_FACE_DIRECT_CMAX
#define DG_FACE_DIRECT_CMAX 16
#endif
#ifndef DG_FACE_DIRECT_MINB
#define DG_FACE_DIRECT_MINB 3
#endif
#ifndef DG_FACE_MINB
#define DG_FACE_MINB 2
#endif

__constant__ DgTables c_tab;

namespace DG_NS {

__host__ __device__ constexpr int ipow(int b, int e) { return e <= 0 ? 1 : b * ipow(b, e - 1); }
__host__ __device__ constexpr int imax(int a, int b) { return a > b ? a : b; }

constexpr int kSmemBudget = (227 * 1024) / DG_STAGE_MINB - 1024;   // DG_STAGE_MINB resident blocks per SM
constexpr int kSmemMax = 227 * 1024;

template <int D, int M, bool VISC, bool AV>
struct Cfg {
    static constexpr bool GRAD = VISC || AV;
    static constexpr int Vc = D + 2 + DG_TRACER;
    static constexpr int V = Vc + (AV ? 1 : 0);
    static constexpr int Np = ipow(M, D);
    static constexpr int Nf = ipow(M, D - 1);
    // face scratch slots: uL(Vc) uR(Vc) [u~(V) gn(Vc) gt((D-1) Vc)]
    static constexpr int NQE = GRAD ? (3 * Vc + V) : 2 * Vc;      // slots expanded modal -> nodal
    static constexpr int NQ = NQE + (GRAD ? (D - 1) * Vc : 0);
    static constexpr int RX = D * Vc * Np;                         // gradients -> fluxes (in place)
    static constexpr int FP = 2 * V * Np + RX;                     // doubles per cell
    // pencil-sweep configurations (3D, m >= 6: 2-4 cells per block): more warps hide the latency of the short row
    // segments (measured at m = 8: 768 threads -13 % against 512)
    static constexpr int NT = (D == 3 && M >= 6) ? DG_STAGE_NT_BIG : DG_STAGE_NT;
    // W^K per cell, wave-speed reduction scratch, partial sensor sums, one mbarrier
    static constexpr int extra_doubles(int c) { return c + 2 * (NT / 32) + (AV ? 4 * (NT / 32) * c : 0) + 2; }
    static constexpr int pick_c() {
        int c = 32;
        while (c > 1 && (c * FP + extra_doubles(c)) * 8 > kSmemBudget) c >>= 1;
        return c;
    }
    static constexpr int C = pick_c();
    static constexpr int kExtraDoubles = extra_doubles(C);
    static constexpr int kSmemBytes = (C * FP + kExtraDoubles) * 8;
    static_assert(kSmemBytes <= kSmemMax, "per-cell footprint exceeds shared memory");
    // A tile of m x m points (the two fastest axes) is swept in registers when it fits (m <= 5).
    static constexpr bool BLK = (M >= 2) && (M * M <= 25);
    // Format of the face-flux buffer.  PP (register-tile configurations, consumed by dg_stage2_kernel): the flux of
    // face axis A is projected on the transverse modes of the axes BELOW A only -- x faces stay nodal, y faces are
    // modal in x (nodal in z), z faces are modal in x and y -- because the stage kernel injects the lift of axis A
    // right after its own projection sweep along A and the remaining sweeps finish the transverse projection.
    // Otherwise (dg_stage_kernel): fully projected on both transverse axes.
    static constexpr bool PP = BLK;
};

// Shared-memory arrays are indexed by a flat point index P = slot*NPTS + p and the cell:  offset = at(P)*C + cell.
// With C = 8 a row of cells is half a 128-byte bank line, and rows whose P differ by a multiple of 2 collide when
// the lanes of a warp walk over planes / slots (strides that are multiples of 16 doubles).  For even m the two rows
// of a pair are exchanged according to the parity of (plane index + slot index), which makes every access pattern
// of the kernels below conflict-free (pencils along any axis, m x m tiles, point-wise, row-wise I/O).
template <int PL, int NPTS, bool SWZ, int ROTM = 0>
struct Lay {
    // ROTM = m (pencil sweeps with few cells per block, m even): the x index of every row of m points is rotated by
    // the row's y index, x' = (x + y) mod m.  Pencils along x of different rows then start in different banks, and
    // every other access pattern still touches the same set of addresses per row.
    static __device__ __forceinline__ int rot(int j) {
        constexpr int R = ROTM > 0 ? ROTM : 1;
        if (ROTM > 0) {
            const int row = j / R;
            int x = j - row * R + row % R;
            if (x >= R) x -= R;
            return row * R + x;
        }
        return j;
    }
    static __device__ __forceinline__ int at(int P) {
        if (SWZ) {
            const int par = P / PL + (NPTS > PL ? P / NPTS : 0);
            return P ^ (par & 1);
        }
        if (ROTM > 0) return (P / NPTS) * NPTS + rot(P % NPTS);
        return P;
    }
    // same as at(slot*NPTS + j); with `slot` a compile-time constant after unrolling this needs one runtime XOR per j
    // (NPTS / PL is even or 1 whenever SWZ is on)
    static __device__ __forceinline__ int at2(int slot, int j) {
        if (SWZ) return slot * NPTS + (j ^ ((j / PL + slot) & 1));
        return slot * NPTS + rot(j);
    }
    // point indices (inside a slot) of the M points of pencil `pen` along an axis of stride STRIDE.  With the row
    // rotation the row index modulo M is known per axis (x sweep: the pencil's row; y sweep: the point's own y = i;
    // z sweep: the pencil's y), so one division per pencil replaces two per point (m = 6: divisions by 6 were 80 %
    // of the stage kernel's instructions).  Not for SWZ layouts (their exchange depends on the slot).
    template <int M, int STRIDE>
    static __device__ __forceinline__ void pencil(int pen, int *idx) {
        if (ROTM > 0 && !SWZ) {
            const int lo = pen % M, hi = pen / M;
            if (STRIDE == 1) {                      // pen = row, lo = row % M
#pragma unroll
                for (int i = 0; i < M; ++i) {
                    int x = i + lo;
                    if (x >= M) x -= M;
                    idx[i] = pen * M + x;
                }
            } else if (STRIDE == M) {               // pen = plane * M + x; point i sits in row plane * M + i
#pragma unroll
                for (int i = 0; i < M; ++i) {
                    int x = lo + i;
                    if (x >= M) x -= M;
                    idx[i] = hi * M * M + i * M + x;
                }
            } else {                                // pen = y * M + x; every point sits in a row with row % M = y
                int x = lo + hi;
                if (x >= M) x -= M;
#pragma unroll
                for (int i = 0; i < M; ++i) idx[i] = i * STRIDE + hi * M + x;
            }
        } else {
            const int pb = (pen / STRIDE) * (STRIDE * M) + (pen % STRIDE);
#pragma unroll
            for (int i = 0; i < M; ++i) idx[i] = rot(pb + i * STRIDE);
        }
    }
    // parity of tile g (PL points per tile): rows q and q^1 of the tile are exchanged when it is 1
    static __device__ __forceinline__ int tile_par(int g) {
        return SWZ ? ((g + (NPTS > PL ? g / (NPTS / PL) : 0)) & 1) : 0;
    }
};
__host__ __device__ constexpr bool use_swizzle(int M, int C) { return (M % 2 == 0) && (C == 8); }
// rotation for the pencil-sweep path (m x m tiles not in registers), few cells per block, even m
__host__ __device__ constexpr int use_rot(int M, int C, bool BLK) {
    return (DG_ROT_ENABLE && !BLK && C < 8 && M % 2 == 0 && M > 1 && (DG_ROT_NONPOW2 || (M & (M - 1)) == 0)) ? M : 0;
}

template <int SEL>
__device__ __forceinline__ double mat(int idx) {
    if (SEL == DG_SEL_V) return c_tab.V[idx];
    if (SEL == DG_SEL_DHAT) return c_tab.Dhat[idx];
    if (SEL == DG_SEL_S) return c_tab.S[idx];
    return c_tab.VtG[idx];
}

// out[r] = sum_c MAT[r][c] in[c] for one pencil of M values in registers (out must not alias in).
// The Legendre basis at the Gauss nodes is parity-symmetric (x_{m-1-j} = -x_j, P_l(-x) = (-1)^l P_l(x)), so
//   V   (modal -> nodal):  out[j], out[m-1-j] = E_j +- O_j,  E_j / O_j = sums over the even / odd modes
//   VtG (nodal -> modal):  even (odd) modes see only in[j] + in[m-1-j]  (in[j] - in[m-1-j])
// which needs m^2/2 + m operations instead of m^2 (m = 4: 12 instead of 16).  Dhat and S map nodal values to nodal
// values and are centro-antisymmetric, MAT[m-1-r][m-1-c] = -MAT[r][c]; their even-odd form (tables DhatE/DhatO, SE/SO:
// half-sums and half-differences of mirrored columns) costs m^2/2 + 2m and is used for m >= 6 only.
template <int SEL, int M>
__device__ __forceinline__ void apply1d(const double *in, double *out) {
    constexpr int H = M / 2;
    if (DG_EVEN_ODD && M >= 2 && SEL == DG_SEL_V) {
#pragma unroll
        for (int j = 0; j < H; ++j) {
            double e = in[0];                       // P_0 = 1 exactly (normalised Legendre): no multiplication
#pragma unroll
            for (int l = 2; l < M; l += 2) e = fma(c_tab.V[j * 8 + l], in[l], e);
            double o = c_tab.V[j * 8 + 1] * in[1];
#pragma unroll
            for (int l = 3; l < M; l += 2) o = fma(c_tab.V[j * 8 + l], in[l], o);
            out[j] = e + o;
            out[M - 1 - j] = e - o;
        }
        if (M % 2) {
            double e = in[0];
#pragma unroll
            for (int l = 2; l < M; l += 2) e = fma(c_tab.V[H * 8 + l], in[l], e);
            out[H] = e;
        }
    } else if (DG_EVEN_ODD && M >= 2 && SEL == DG_SEL_VTG) {
        double sp[H > 0 ? H : 1], sm[H > 0 ? H : 1];
#pragma unroll
        for (int j = 0; j < H; ++j) {
            sp[j] = in[j] + in[M - 1 - j];
            sm[j] = in[j] - in[M - 1 - j];
        }
#pragma unroll
        for (int l = 0; l < M; ++l) {
            const double *s = (l % 2) ? sm : sp;
            double acc = c_tab.VtG[l * 8] * s[0];
#pragma unroll
            for (int j = 1; j < H; ++j) acc = fma(c_tab.VtG[l * 8 + j], s[j], acc);
            if ((M % 2) && (l % 2 == 0)) acc = fma(c_tab.VtG[l * 8 + H], in[H], acc);
            out[l] = acc;
        }
    } else if (DG_EVEN_ODD && M >= 6 && (SEL == DG_SEL_DHAT || SEL == DG_SEL_S)) {
        const double *TE = (SEL == DG_SEL_DHAT) ? c_tab.DhatE : c_tab.SE;
        const double *TO = (SEL == DG_SEL_DHAT) ? c_tab.DhatO : c_tab.SO;
        double sp[H > 0 ? H : 1], sm[H > 0 ? H : 1];
#pragma unroll
        for (int i = 0; i < H; ++i) {
            sp[i] = in[i] + in[M - 1 - i];
            sm[i] = in[i] - in[M - 1 - i];
        }
#pragma unroll
        for (int j = 0; j < H; ++j) {
            double pa = TE[j * 8] * sp[0], qa = TO[j * 8] * sm[0];
#pragma unroll
            for (int i = 1; i < H; ++i) {
                pa = fma(TE[j * 8 + i], sp[i], pa);
                qa = fma(TO[j * 8 + i], sm[i], qa);
            }
            if (M % 2) pa = fma(mat<SEL>(j * 8 + H), in[H], pa);
            out[j] = qa + pa;
            out[M - 1 - j] = qa - pa;
        }
        if (M % 2) {
            double qa = mat<SEL>(H * 8) * sm[0];
#pragma unroll
            for (int i = 1; i < H; ++i) qa = fma(mat<SEL>(H * 8 + i), sm[i], qa);
            out[H] = qa;
        }
    } else {
#pragma unroll
        for (int j = 0; j < M; ++j) {
            double acc = mat<SEL>(j * 8) * in[0];
#pragma unroll
            for (int i = 1; i < M; ++i) acc = fma(mat<SEL>(j * 8 + i), in[i], acc);
            out[j] = acc;
        }
    }
}

// pencil base: index of the first point of pencil `pen` along an axis of stride STRIDE
template <int M, int STRIDE>
__device__ __forceinline__ int pencil_base(int pen) {
    return (pen / STRIDE) * (STRIDE * M) + (pen % STRIDE);
}

// (An fp64 tensor-core form of this sweep for m = 8 -- mma.sync.m8n8k4.f64 over 8 pencils at a time -- was measured
// 14 % slower than the even-odd DFMA sweeps and removed from the source in round 3: profiles/r2_dmma.md.)
// Apply one 1D matrix along one axis to `nslots` arrays of NPTS points (slots s0 .. s0+nslots of src, d0 .. of dst):
//   dst[d0+slot][p] (+)= scale * sum_i MAT[j][i] * (sum_{k<NSUM} src[s0 + k*sum_slots + slot][p_i])
// src == dst (in place) is allowed: a thread owns whole pencils.
template <int SEL, int M, int NPTS, int STRIDE, int C, int NT, int NSUM, bool ADD, bool SCALE, class L>
__device__ __forceinline__ void sweep(const double *src, int s0, int sum_slots, double *dst, int d0, int nslots,
                                      double scale, int tid) {
    constexpr int NPEN = NPTS / M;
    static_assert(NT % C == 0, "threads per block must be a multiple of cells per block");
    const int cell = tid % C;
    const int total = nslots * NPEN;
    constexpr bool FASTIDX = !use_swizzle(M, C);      // SWZ layouts exchange rows depending on the slot: generic path
    for (int r = tid / C; r < total; r += NT / C) {
        const int pen = r % NPEN;
        const int slot = r / NPEN;
        const int pb = pencil_base<M, STRIDE>(pen);
        int idx[M];
        if (FASTIDX) L::template pencil<M, STRIDE>(pen, idx);
        double in[M];
#pragma unroll
        for (int i = 0; i < M; ++i) {
            in[i] = FASTIDX ? src[((s0 + slot) * NPTS + idx[i]) * C + cell] : src[L::at2(s0 + slot, pb + i * STRIDE) * C + cell];
#pragma unroll
            for (int k = 1; k < NSUM; ++k)
                in[i] += FASTIDX ? src[((s0 + k * sum_slots + slot) * NPTS + idx[i]) * C + cell]
                                 : src[L::at2(s0 + k * sum_slots + slot, pb + i * STRIDE) * C + cell];
        }
        double res[M];
        apply1d<SEL, M>(in, res);
#pragma unroll
        for (int j = 0; j < M; ++j) {
            double acc = res[j];
            if (SCALE) acc *= scale;
            double *d = FASTIDX ? dst + ((d0 + slot) * NPTS + idx[j]) * C + cell : dst + L::at2(d0 + slot, pb + j * STRIDE) * C + cell;
            if (ADD)
                *d += acc;
            else
                *d = acc;
        }
    }
}

// ---- m x m register tiles: t[y*M + x] ----
template <int SEL, int M>
__device__ __forceinline__ void tile_x(double *t) {
#pragma unroll
    for (int y = 0; y < M; ++y) {
        double in[M];
#pragma unroll
        for (int i = 0; i < M; ++i) in[i] = t[y * M + i];
        apply1d<SEL, M>(in, t + y * M);
    }
}
template <int SEL, int M>
__device__ __forceinline__ void tile_y(double *t) {
#pragma unroll
    for (int x = 0; x < M; ++x) {
        double in[M];
#pragma unroll
        for (int i = 0; i < M; ++i) in[i] = t[i * M + x];
        double res[M];
        apply1d<SEL, M>(in, res);
#pragma unroll
        for (int j = 0; j < M; ++j) t[j * M + x] = res[j];
    }
}
// acc += (MAT along y) t, plain form (no separate add pass)
template <int SEL, int M>
__device__ __forceinline__ void tile_y_acc(const double *t, double *acc) {
#pragma unroll
    for (int x = 0; x < M; ++x)
#pragma unroll
        for (int j = 0; j < M; ++j)
#pragma unroll
            for (int i = 0; i < M; ++i) acc[j * M + x] = fma(mat<SEL>(j * 8 + i), t[i * M + x], acc[j * M + x]);
}
// tile g (global plane index: P = g*M*M + q) of an array <-> registers; L::PL must be M*M
template <int M, int C, class L>
__device__ __forceinline__ void tile_load(const double *a, int g, int cell, double *t) {
    const int b = L::tile_par(g) * C;
    const double *pe = a + g * (M * M) * C + cell + b;   // even rows: q ^ 1 = q + 1
    const double *po = a + g * (M * M) * C + cell - b;   // odd rows:  q ^ 1 = q - 1
#pragma unroll
    for (int q = 0; q < M * M; ++q) t[q] = ((q & 1) ? po : pe)[q * C];
}
template <int M, int C, class L>
__device__ __forceinline__ void tile_store(double *a, int g, int cell, const double *t) {
    const int b = L::tile_par(g) * C;
    double *pe = a + g * (M * M) * C + cell + b;
    double *po = a + g * (M * M) * C + cell - b;
#pragma unroll
    for (int q = 0; q < M * M; ++q) ((q & 1) ? po : pe)[q * C] = t[q];
}

// ---------------------------------------------------------------------------------------------------
// point-wise physics (Eq. 1-5; 106; 311-323 Eq. 37-39; 375-407 Eq. 43-46)
// ---------------------------------------------------------------------------------------------------
// Reciprocal and square root without the IEEE slow path: hardware seed (>= 20 bits) + Newton steps to ~1 ulp.
// (fp64 division / sqrt compile to ~20-instruction sequences with a branch; these are 6-9 fused operations.)
__device__ __forceinline__ double fast_rcp(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(r, fma(-x, r, 1.0), r);
    r = fma(r, fma(-x, r, 1.0), r);
    return r;
}
__device__ __forceinline__ double fast_sqrt(double x) {
    if (!(x > 1e-280) || !(x < 1e280)) return sqrt(x);   // zero, negative, NaN, extreme magnitudes: library path
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double hx = 0.5 * x;
    y = y * fma(-hx * y, y, 1.5);
    y = y * fma(-hx * y, y, 1.5);
    double s = x * y;
    s = fma(fma(-s, s, x), 0.5 * y, s);
    return s;
}

template <int D>
struct Prim {
    double rho, ir, v[D], p, e;
};

template <int D>
__device__ __forceinline__ Prim<D> primitives(const double *u, double gamma) {
    Prim<D> q;
    q.rho = u[0];
    q.ir = fast_rcp(q.rho);
    double v2 = 0.0;
#pragma unroll
    for (int b = 0; b < D; ++b) {
        q.v[b] = u[1 + b] * q.ir;
        v2 = fma(q.v[b], q.v[b], v2);
    }
    q.e = u[1 + D];
    q.p = (gamma - 1.0) * (q.e - 0.5 * q.rho * v2);
    return q;
}

// Euler flux along axis a (Eq. 4; energy row (e+p) v_a, reading A5)
template <int D>
__device__ __forceinline__ void euler_flux(const double *u, const Prim<D> &q, int a, double *f) {
    const double va = q.v[a];
    f[0] = u[1 + a];
#pragma unroll
    for (int b = 0; b < D; ++b) f[1 + b] = u[1 + a] * q.v[b] + (b == a ? q.p : 0.0);
    f[1 + D] = (q.e + q.p) * va;
    if (DG_TRACER) f[2 + D] = u[2 + D] * va;      // c rho v_a (Eq. 40)
}

// HLLC flux along axis a (Toro's HLLC with Davis wave-speed bounds, reading A6)
template <int D>
__device__ __forceinline__ void hllc_flux(const double *uL, const double *uR, const Prim<D> &L, const Prim<D> &R,
                                          int a, double gamma, double *F) {
    const double cL = fast_sqrt(gamma * L.p * L.ir);
    const double cR = fast_sqrt(gamma * R.p * R.ir);
    const double vnL = L.v[a], vnR = R.v[a];
    const double SL = fmin(vnL - cL, vnR - cR);
    const double SR = fmax(vnL + cL, vnR + cR);
    if (SL >= 0.0) {
        euler_flux<D>(uL, L, a, F);
        return;
    }
    if (SR <= 0.0) {
        euler_flux<D>(uR, R, a, F);
        return;
    }
    const double mL = L.rho * (SL - vnL);
    const double mR = R.rho * (SR - vnR);
    const double Sstar = (R.p - L.p + mL * vnL - mR * vnR) * fast_rcp(mL - mR);
    // F_K + S_K (U*_K - U_K), K = L if S* >= 0 else R
    const bool left = (Sstar >= 0.0);
    const double *u = left ? uL : uR;
    const Prim<D> &K = left ? L : R;
    const double S = left ? SL : SR;
    const double vn = left ? vnL : vnR;
    const double mK = left ? mL : mR;
    double f[D + 2 + DG_TRACER];
    euler_flux<D>(u, K, a, f);
    const double fac = mK * fast_rcp(S - Sstar);
    F[0] = f[0] + S * (fac - u[0]);
#pragma unroll
    for (int b = 0; b < D; ++b) {
        const double us = fac * (b == a ? Sstar : K.v[b]);
        F[1 + b] = f[1 + b] + S * (us - u[1 + b]);
    }
    const double es = fac * (K.e * K.ir + (Sstar - vn) * (Sstar + K.p * fast_rcp(mK)));
    F[1 + D] = f[1 + D] + S * (es - K.e);
    // a passive scalar is carried like a transverse velocity (reading T1): U*_K row = fac c_K
    if (DG_TRACER) F[2 + D] = f[2 + D] + S * (fac * (u[2 + D] * K.ir) - u[2 + D]);
}

// velocity gradient dv[b][c] = d v_c / d x_b = (d_b(rho v_c) - v_c d_b rho) / rho
template <int D>
__device__ __forceinline__ void velocity_gradient(const Prim<D> &q, const double (*g)[D + 2 + DG_TRACER], double (*dv)[D]) {
#pragma unroll
    for (int b = 0; b < D; ++b)
#pragma unroll
        for (int c = 0; c < D; ++c) dv[b][c] = (g[b][1 + c] - q.v[c] * g[b][0]) * q.ir;
}

// Navier-Stokes flux column a (Eq. 38-39, traceless Pi, reading A7), SUBTRACTED from F
template <int D>
__device__ __forceinline__ void ns_flux_sub(const Prim<D> &q, const double (*g)[D + 2 + DG_TRACER], const double (*dv)[D],
                                            double divv, int a, double gamma, double nu, double chi, double *F,
                                            double ctr = 0.0, double eta = 0.0) {
    double evisc = 0.0;
#pragma unroll
    for (int b = 0; b < D; ++b) {
        const double Pi = nu * q.rho * (dv[a][b] + dv[b][a] - (a == b ? (2.0 / 3.0) * divv : 0.0));
        F[1 + b] -= Pi;
        evisc = fma(q.v[b], Pi, evisc);
    }
    double vdv = 0.0;
#pragma unroll
    for (int c = 0; c < D; ++c) vdv = fma(q.v[c], dv[a][c], vdv);
    const double duth = g[a][1 + D] * q.ir - q.e * g[a][0] * (q.ir * q.ir) - vdv;
    F[1 + D] -= evisc + chi * (gamma - 1.0) * q.rho * duth;
    // tracer diffusion eta rho d_a c, grad c = [grad(c rho) - c grad rho] / rho (Eq. 40); ctr = c at this point
    if (DG_TRACER) F[2 + D] -= eta * (g[a][2 + D] - ctr * g[a][0]);
}

__device__ __forceinline__ void atomic_max_nonneg(unsigned long long *addr, double val) {
    atomicMax(addr, (unsigned long long)__double_as_longlong(val));
}

// block-wide max of two non-negative values -> atomicMax on maxbits[0..1]
template <int NT>
__device__ __forceinline__ void block_max2(double a, double b, double *red, unsigned long long *maxbits, int tid) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a = fmax(a, __shfl_xor_sync(0xffffffffu, a, o));
        b = fmax(b, __shfl_xor_sync(0xffffffffu, b, o));
    }
    if ((tid & 31) == 0) {
        red[tid >> 5] = a;
        red[NT / 32 + (tid >> 5)] = b;
    }
    __syncthreads();
    if (tid == 0) {
        for (int i = 1; i < NT / 32; ++i) {
            a = fmax(a, red[i]);
            b = fmax(b, red[NT / 32 + i]);
        }
        atomic_max_nonneg(&maxbits[0], a);
        atomic_max_nonneg(&maxbits[1], b);
    }
}

// expand slots [0, nslots) of `buf` modal -> nodal in place (Eq. 21), all D axes; ends with a barrier
template <int D, int M, int C, int NT, bool BLK, class L>
__device__ __forceinline__ void expand_volume(double *buf, int nslots, int tid) {
    constexpr int Np = ipow(M, D);
    if (BLK) {
        // x and y in registers, one m x m tile per item
        const int ntile = nslots * (Np / (M * M));
        for (int it = tid; it < ntile * C; it += NT) {
            const int cell = it % C, g = it / C;
            double t[M * M];
            tile_load<M, C, L>(buf, g, cell, t);
            tile_x<DG_SEL_V, M>(t);
            tile_y<DG_SEL_V, M>(t);
            tile_store<M, C, L>(buf, g, cell, t);
        }
        __syncthreads();
    } else {
        sweep<DG_SEL_V, M, Np, 1, C, NT, 1, false, false, L>(buf, 0, 0, buf, 0, nslots, 1.0, tid);
        __syncthreads();
        sweep<DG_SEL_V, M, Np, M, C, NT, 1, false, false, L>(buf, 0, 0, buf, 0, nslots, 1.0, tid);
        __syncthreads();
    }
    if (D == 3) {
        sweep<DG_SEL_V, M, Np, M * M, C, NT, 1, false, false, L>(buf, 0, 0, buf, 0, nslots, 1.0, tid);
        __syncthreads();
    }
}

// max c_s and max |v| over the nodal values in RA (Eq. 23 inputs, reading A18)
template <int D, int M, int C, int NT, class L>
__device__ __forceinline__ void wavespeed_points(const double *RA, double gamma, int *flag, double *red,
                                                 unsigned long long *maxbits, int tid) {
    constexpr int Np = ipow(M, D);
    constexpr int Vc = D + 2;
    double cmax = 0.0, vmax = 0.0;
    bool bad = false;
    for (int it = tid; it < Np * C; it += NT) {
        const int cell = it % C;
        const int j = it / C;
        double u[Vc];
#pragma unroll
        for (int v = 0; v < Vc; ++v) u[v] = RA[L::at2(v, j) * C + cell];
        const Prim<D> q = primitives<D>(u, gamma);
        bad |= !(q.rho > 0.0) || !(q.p > 0.0);
        double v2 = 0.0;
#pragma unroll
        for (int b = 0; b < D; ++b) v2 = fma(q.v[b], q.v[b], v2);
        const double cs = fast_sqrt(gamma * q.p * q.ir);
        const double vm = fast_sqrt(v2);
        cmax = (cs > cmax) ? cs : cmax;   // NaN-safe: NaN never becomes the maximum
        vmax = (vm > vmax) ? vm : vmax;
    }
    if (bad) atomicOr(flag, 4);   // flag bits: 1 volume point, 2 face point, 4 wave-speed pass, 8 limiter (cell mean)
    block_max2<NT>(cmax, vmax, red, maxbits, tid);
}

// Block -> tile map.  A tile is C consecutive cells of one x-row.  In 3D, when the mesh divides (nx % C, ny % 8,
// nz % 8), the tiles are visited in groups of 8 y-rows x 8 z-planes (x fastest, then y within the group, then z within
// the group), so that the y and z neighbours of a tile are at most 8 x-rows away in launch order and their rows (state
// for the face kernel, face fluxes for the stage kernel) are still in L2 -- or in flight -- when they are read; 1/8 of
// the tiles per axis reach across a group boundary.  That order is expressed as a 3D grid
//     gridDim = (nx / C, 64 * (ny / 8), nz / 8),   blockIdx.y = 64 * (y group) + 8 * (z in group) + (y in group)
// (blocks are issued x fastest, then y, then z), which gives every thread its (ix, iy, iz) without one integer
// division: the generic 1D map (ragged meshes, tiles that straddle x-rows) costs ~300 instructions per warp.
__host__ __device__ inline bool tile_grid_blocked(int D, int C, int nx, int ny, int nz) {
    return D == 3 && (nx % C) == 0 && (ny % 8) == 0 && (nz % 8) == 0 && (ny / 8) * 64 <= 65535 && (nz / 8) <= 65535;
}
template <int D, int C>
inline dim3 tile_grid(int ncells, int nx, int ny, int nz) {
    if (tile_grid_blocked(D, C, nx, ny, nz)) return dim3(nx / C, 64 * (ny / 8), nz / 8);
    return dim3((ncells + C - 1) / C, 1, 1);
}
// position of lane-cell `cl` of this block: first cell of the tile, clamped global cell index, coordinates
template <int D, int C>
struct TilePos {
    int cell0, cg, ix, iy, iz;
    bool active;
    __device__ __forceinline__ TilePos(const DgStageArgs &p, int cl) {
        if (D == 3 && gridDim.y > 1) {
            const int r = blockIdx.y & 63;
            iy = (blockIdx.y >> 6) * 8 + (r & 7);
            iz = blockIdx.z * 8 + (r >> 3);
            cell0 = (iz * p.ny + iy) * p.nx + blockIdx.x * C;
            ix = blockIdx.x * C + cl;
            cg = cell0 + cl;
            active = true;
        } else {
            cell0 = blockIdx.x * C;
            cg = min(cell0 + cl, p.ncells - 1);
            active = cell0 + cl < p.ncells;
            ix = cg % p.nx;
            iy = (cg / p.nx) % p.ny;
            iz = cg / (p.nx * p.ny);
        }
    }
    // periodic neighbours: lower (-1) / upper (+1) along each axis
    __device__ __forceinline__ int lower(const DgStageArgs &p, int a) const {
        if (a == 0) return cg + ((ix == 0) ? p.nx - 1 : -1);
        if (a == 1) return cg + ((iy == 0) ? (p.ny - 1) * p.nx : -p.nx);
        return cg + ((iz == 0) ? (p.nz - 1) * p.nx * p.ny : -p.nx * p.ny);
    }
    __device__ __forceinline__ int upper(const DgStageArgs &p, int a) const {
        if (a == 0) return cg + ((ix == p.nx - 1) ? 1 - p.nx : 1);
        if (a == 1) return cg + ((iy == p.ny - 1) ? -(p.ny - 1) * p.nx : p.nx);
        return cg + ((iz == p.nz - 1) ? -(p.nz - 1) * p.nx * p.ny : p.nx * p.ny);
    }
};

// address of row `row` (compile-time multiple after unrolling) of a [row][cell] global array: one IMAD.WIDE
__device__ __forceinline__ const double *row_ptr(const double *base, unsigned row, unsigned ncells) {
    return base + (unsigned long long)row * ncells;
}
__device__ __forceinline__ double *row_ptr(double *base, unsigned row, unsigned ncells) {
    return base + (unsigned long long)row * ncells;
}

// Layout of the state and face-flux arrays in global memory.  Default (B = 0): structure of arrays,
// a[row * ncells + cell], the layout of the C-ABI.  Pencil-sweep configurations in 3D (m >= 6) keep only B = 2 or 4
// cells per block in shared memory, and a row segment of B * 8 bytes per request leaves the kernels waiting on
// thousands of 16-byte sectors per tile (measured: 63 % of the m = 8 stage kernel, L2-resident or not).  They use
// an array of B-cell blocks instead, a[((cell / B) * R + row) * B + cell % B] (R rows per array): the rows of a tile are
// adjacent, every request is a full line.  dg_api.cu converts at the boundary (dg_pack_kernel / dg_unpack_kernel).
template <int D, int M>
struct GLay {
    static constexpr int B = (DG_AOSOA && D == 3 && M >= 6) ? Cfg<D, M, true, true>::C : 0;
    // offset of (row 0, cell c) in an array of R rows
    static __host__ __device__ __forceinline__ size_t cell(int c, int R) {
        return B ? ((size_t)(c / (B ? B : 1)) * R * B + c % (B ? B : 1)) : (size_t)c;
    }
    // distance between consecutive rows of one cell
    static __host__ __device__ __forceinline__ unsigned rs(int ncells) { return B ? (unsigned)B : (unsigned)ncells; }
};

// ---- bulk asynchronous copies (TMA engine, 1D): global -> shared, completion on an mbarrier ----
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(void *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, void *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// Own modes of a FULL tile (C cells, 16-byte aligned rows) by bulk copies: one C*8-byte row segment per request,
// global [r = mode*V + v][cell] -> shared [v][mode][cell]; no registers, no LSU queue slots.  Thread 0 must have
// initialised `bar` (count 1) before a __syncthreads(); returns after the data has landed.
template <int V, int Np, int C, int NT, class L>
__device__ __forceinline__ void issue_own_modes_bulk(const double *w, int ncells, int cell0, double *RA, void *bar,
                                                     int tid) {
    if (tid == 0) mbar_expect_tx(bar, (unsigned)(V * Np * C * 8));
    for (int r = tid; r < V * Np; r += NT)
        bulk_g2s(RA + L::at2(r % V, r / V) * C, w + (size_t)r * ncells + cell0, C * 8, bar);
}
// a tile qualifies for bulk copies when it is full and every row segment is 16-byte aligned
template <int C>
__device__ __forceinline__ bool bulk_ok(int cell0, int ncells) {
    return (C % 2 == 0) && (cell0 + C <= ncells) && ((ncells & 1) == 0);
}

// Own modes of the block's cells, global [r = mode*V + v][cell] -> shared [v][mode][cell].  Thread `tid` keeps
// cell tid % C and the modes g, g+G, ... (g = tid / C, G = NT / C) of every variable; its loads are issued in
// batches of up to 12 before the first store (one DRAM round trip per batch).
template <int V, int Np, int C, int NT, class L>
__device__ __forceinline__ void load_own_modes(const double *__restrict__ wcell, unsigned rs, double *RA, int tid) {
    // wcell = address of (row 0, this thread's cell), rs = row stride (GLay)
    constexpr int G = NT / C;
    constexpr int NK = (Np + G - 1) / G;
    constexpr int KB = (12 / V) < 1 ? 1 : (12 / V);          // k-steps per batch
    const unsigned ncells = rs;
    const int cl = tid % C, g = tid / C;
    const double *base = wcell + (size_t)(g * V) * rs;
#pragma unroll
    for (int k0 = 0; k0 < NK; k0 += KB) {
        double t[KB][V];
#pragma unroll
        for (int kk = 0; kk < KB; ++kk)
#pragma unroll
            for (int v = 0; v < V; ++v)
                if (k0 + kk < NK && g + (k0 + kk) * G < Np) t[kk][v] = __ldg(row_ptr(base, (k0 + kk) * G * V + v, ncells));
#pragma unroll
        for (int kk = 0; kk < KB; ++kk)
#pragma unroll
            for (int v = 0; v < V; ++v)
                if (k0 + kk < NK && g + (k0 + kk) * G < Np) RA[L::at2(v, g + (k0 + kk) * G) * C + cl] = t[kk][v];
    }
}

// ---------------------------------------------------------------------------------------------------
// face kernel: the numerical flux of Eq. 20's surface lines, ONCE per face point.
// Cell K owns its D "upper" faces (towards +a): left state = K, right state = K_{a+}.  The result, already
// projected on the transverse modes (sum_k g_k phi_l(xi_k) G^_a), is written to
//     flux[((A*Vc + v)*Nf + lt) * ncells + cell]
// and lifted into both adjacent cells by the stage kernel.
// ---------------------------------------------------------------------------------------------------
template <int D, int M, bool VISC, bool AV>
struct FaceCfg {
    using K = Cfg<D, M, VISC, AV>;
    static constexpr int BIG = (D == 3 && M >= 6);     // one large block per SM (measured at m = 8: -25 %)
    static constexpr int NT = BIG ? DG_FACE_NT_BIG : DG_FACE_NT;
    // DIRECT (3D register-tile configurations): F1 reads the own modes straight from global memory / L1 like the
    // neighbour's (each is used once per axis), so no copy of the tile is staged in shared memory, the block does
    // not wait for it before the first axis, and only the face scratch remains (more cells or blocks per SM)
    static constexpr bool DIRECT = DG_FACE_DIRECT && ((K::BLK && D == 3) || GLay<D, M>::B > 0);
    static constexpr int FP = (DIRECT ? 0 : K::V * K::Np) + K::NQ * K::Nf;   // doubles per cell: [own modes +] one face
    static constexpr int MINB = BIG ? DG_FACE_BIG_MINB : (DIRECT ? DG_FACE_DIRECT_MINB : DG_FACE_MINB);   // resident blocks per SM (register cap)
    static constexpr int CMAX = DIRECT ? DG_FACE_DIRECT_CMAX : 32;
    static constexpr int pick_c() {
        int c = CMAX;
        while (c > 1 && c * FP * 8 > (227 * 1024) / MINB - 2048) c >>= 1;   // MINB resident blocks per SM
        return c;
    }
    static constexpr int C = pick_c();
    static constexpr int kSmemBytes = C * FP * 8 + ((D * C + 1) / 2) * 8 + 16;   // + nbr[D*C] + mbarrier
    static_assert(kSmemBytes <= kSmemMax, "face kernel: per-cell footprint exceeds shared memory");
    static constexpr bool SWZ = use_swizzle(M, C);
    using LV = Lay<M * M, K::Np, SWZ, use_rot(M, C, K::BLK)>;   // own modes (volume array)
    using LF = Lay<K::Nf, K::Nf, SWZ, (D == 3 ? use_rot(M, C, K::BLK) : 0)>;          // face arrays: one tile (3D) / one pencil (2D) per slot
};

template <int D, int M, bool VISC, bool AV, int A>
__device__ __forceinline__ void face_axis(const DgStageArgs &p, const double *RA, double *RX, const int *nbr,
                                          int cell0, int tid) {
    using K = Cfg<D, M, VISC, AV>;
    using FK = FaceCfg<D, M, VISC, AV>;
    using LV = typename FK::LV;
    using LF = typename FK::LF;
    constexpr int C = FK::C, NT = FK::NT, V = K::V, Vc = K::Vc, Nf = K::Nf;
    constexpr bool GRAD = K::GRAD;
    constexpr bool TILE = K::BLK && (D == 3);    // face arrays are m x m tiles
    constexpr int SA = ipow(M, A);               // stride of axis A inside the cell
    constexpr int oUL = 0, oUR = Vc, oUT = 2 * Vc, oGN = 2 * Vc + V, oGT = 3 * Vc + V;
    const double ih = 1.0 / p.h;

    // F1: contract the normal axis (PAPER.md:171 traces; 294-299 recovery partial sums).  A thread keeps one
    // cell (NT % C == 0); all its neighbour loads are issued before the first use.
    {
        static_assert(NT % C == 0, "threads per block must be a multiple of cells per block");
        constexpr int NIT = (V * Nf * C + NT - 1) / NT;
        constexpr int NB = FK::DIRECT ? (NIT % 3 == 0 ? 3 : (NIT % 2 == 0 ? 2 : 1)) : NIT;   // items per load batch
        using GL = GLay<D, M>;
        // Block layout (GL::B > 0): items are numbered in memory order -- cell within its block fastest, then the
        // variable, then the transverse mode -- so that the lanes of a warp read adjacent doubles (row = mode*V + v,
        // address = row*B + cell % B); otherwise lanes = cells and the rows of a thread's items are NT/C apart.
        constexpr bool MO = GL::B > 0;
        constexpr int BB = MO ? GL::B : 1;
        const unsigned grs = GL::rs(p.ncells);
        auto item = [&](int k, int &cell, int &v, int &lt) -> bool {
            if (MO) {
                const int e = tid + k * NT;
                cell = (e / (BB * V * Nf)) * BB + e % BB;
                v = (e / BB) % V;
                lt = (e / (BB * V)) % Nf;
                return e < C * V * Nf;
            }
            const int r = tid / C + k * (NT / C);          // v*Nf + lt
            cell = tid % C;
            v = r / Nf;
            lt = r % Nf;
            return r < V * Nf;
        };
#pragma unroll
        for (int k0 = 0; k0 < NIT; k0 += NB) {
            double nb[NB][M], ow[NB][M];
#pragma unroll
            for (int kk = 0; kk < NB; ++kk) {
                int cell, v, lt;
                if (item(k0 + kk, cell, v, lt)) {
                    const int base = pencil_base<M, SA>(lt);
                    const int nc = nbr[A * C + cell];
                    // the upper x neighbour of every cell but the last one of the tile is the next cell of the tile
                    const bool from_tile = !FK::DIRECT && (A == 0) && (cell < C - 1) && (cell0 + cell + 1 < p.ncells) &&
                                           (nc == cell0 + cell + 1);
                    if (from_tile) {
#pragma unroll
                        for (int l = 0; l < M; ++l) nb[kk][l] = RA[LV::at2(v, base + l * SA) * C + cell + 1];
                    } else {
                        // one IMAD.WIDE per load: base pointer of (first row of the pencil, cell), compile-time row steps
                        const double *wnb = row_ptr(p.w_prev + GL::cell(nc, V * K::Np), base * V + v, grs);
#pragma unroll
                        for (int l = 0; l < M; ++l) nb[kk][l] = __ldg(row_ptr(wnb, l * SA * V, grs));
                    }
                    if (FK::DIRECT) {
                        const double *wow =
                            row_ptr(p.w_prev + GL::cell(min(cell0 + cell, p.ncells - 1), V * K::Np), base * V + v, grs);
#pragma unroll
                        for (int l = 0; l < M; ++l) ow[kk][l] = __ldg(row_ptr(wow, l * SA * V, grs));
                    }
                }
            }
#pragma unroll
            for (int kk = 0; kk < NB; ++kk) {
                int cell, v, lt;
                if (item(k0 + kk, cell, v, lt)) {
                    const int base = pencil_base<M, SA>(lt);
                    double own[M];
#pragma unroll
                    for (int l = 0; l < M; ++l) own[l] = FK::DIRECT ? ow[kk][l] : RA[LV::at2(v, base + l * SA) * C + cell];
                    double uL = 0.0, uR = 0.0, ut = 0.0, gn = 0.0;
#pragma unroll
                    for (int l = 0; l < M; ++l) {
                        uL = fma(c_tab.Pend[1][l], own[l], uL);
                        uR = fma(c_tab.Pend[0][l], nb[kk][l], uR);
                        if (GRAD) {
                            ut = fma(c_tab.Rv[0][l], own[l], ut);
                            ut = fma(c_tab.Rv[1][l], nb[kk][l], ut);
                            gn = fma(c_tab.Gv[0][l], own[l], gn);
                            gn = fma(c_tab.Gv[1][l], nb[kk][l], gn);
                        }
                    }
                    if (v < Vc) {
                        RX[LF::at2(oUL + v, lt) * C + cell] = uL;
                        RX[LF::at2(oUR + v, lt) * C + cell] = uR;
                        if (GRAD) RX[LF::at2(oGN + v, lt) * C + cell] = gn * ih;
                    }
                    if (GRAD) RX[LF::at2(oUT + v, lt) * C + cell] = ut;
                }
            }
        }
    }
    __syncthreads();

    // F2: transverse modal -> nodal on the face (cell basis kept transversally), and the
    // transverse derivatives of the recovered face polynomial
    if (TILE) {
        for (int it = tid; it < K::NQE * C; it += NT) {
            const int cell = it % C, g = it / C;
            double t[M * M];
            tile_load<M, C, LF>(RX, g, cell, t);
            tile_x<DG_SEL_V, M>(t);
            tile_y<DG_SEL_V, M>(t);
            tile_store<M, C, LF>(RX, g, cell, t);
            if (GRAD && g >= oUT && g < oUT + Vc) {
                double a[M * M];
#pragma unroll
                for (int q = 0; q < M * M; ++q) a[q] = t[q];
                tile_x<DG_SEL_DHAT, M>(a);
#pragma unroll
                for (int q = 0; q < M * M; ++q) a[q] *= 2.0 * ih;
                tile_store<M, C, LF>(RX, oGT + (g - oUT), cell, a);
                tile_y<DG_SEL_DHAT, M>(t);
#pragma unroll
                for (int q = 0; q < M * M; ++q) t[q] *= 2.0 * ih;
                tile_store<M, C, LF>(RX, oGT + Vc + (g - oUT), cell, t);
            }
        }
        __syncthreads();
    } else {
        if (M > 1) {
            sweep<DG_SEL_V, M, Nf, 1, C, NT, 1, false, false, LF>(RX, 0, 0, RX, 0, K::NQE, 1.0, tid);
            __syncthreads();
            if (D == 3) {
                sweep<DG_SEL_V, M, Nf, M, C, NT, 1, false, false, LF>(RX, 0, 0, RX, 0, K::NQE, 1.0, tid);
                __syncthreads();
            }
        }
        if (GRAD) {
            sweep<DG_SEL_DHAT, M, Nf, 1, C, NT, 1, false, true, LF>(RX, oUT, 0, RX, oGT, Vc, 2.0 * ih, tid);
            if (D == 3)
                sweep<DG_SEL_DHAT, M, Nf, M, C, NT, 1, false, true, LF>(RX, oUT, 0, RX, oGT + Vc, Vc, 2.0 * ih, tid);
            __syncthreads();
        }
    }

    // F3: numerical flux at every face point; result overwrites the uL slots
    {
        bool bad = false;
        for (int it = tid; it < Nf * C; it += NT) {
            const int cell = it % C;
            const int k = it / C;
            double uL[Vc], uR[Vc], Fh[Vc];
#pragma unroll
            for (int v = 0; v < Vc; ++v) {
                uL[v] = RX[LF::at2(oUL + v, k) * C + cell];
                uR[v] = RX[LF::at2(oUR + v, k) * C + cell];
            }
            const Prim<D> qL = primitives<D>(uL, p.gamma);
            const Prim<D> qR = primitives<D>(uR, p.gamma);
            bad |= !(qL.rho > 0.0) || !(qL.p > 0.0) || !(qR.rho > 0.0) || !(qR.p > 0.0);
            hllc_flux<D>(uL, uR, qL, qR, A, p.gamma, Fh);
            if (GRAD) {
                double ut[Vc], g[D][D + 2 + DG_TRACER];
#pragma unroll
                for (int v = 0; v < Vc; ++v) {
                    ut[v] = RX[LF::at2(oUT + v, k) * C + cell];
#pragma unroll
                    for (int b = 0; b < D; ++b) {
                        const int slot = (b == A) ? (oGN + v) : (oGT + (b < A ? b : b - 1) * Vc + v);
                        g[b][v] = RX[LF::at2(slot, k) * C + cell];
                    }
                }
                const Prim<D> qt = primitives<D>(ut, p.gamma);
                bad |= !(qt.rho > 0.0) || !(qt.p > 0.0);
                if (VISC) {
                    double dv[D][D];
                    velocity_gradient<D>(qt, g, dv);
                    double divv = 0.0;
#pragma unroll
                    for (int b = 0; b < D; ++b) divv += dv[b][b];
                    ns_flux_sub<D>(qt, g, dv, divv, A, p.gamma, p.nu, p.chi, Fh, DG_TRACER ? ut[Vc - 1] * qt.ir : 0.0, p.eta);
                }
                if (AV) {
                    const double al = RX[LF::at2(oUT + Vc, k) * C + cell];
                    const double cst = fast_sqrt(p.gamma * qt.p * qt.ir);
                    const double eps = fmin(fmax(al, 0.0), p.alpha_max) * cst * (p.h / (double)M);   // Eq. 46, A12
#pragma unroll
                    for (int v = 0; v < Vc; ++v) Fh[v] -= eps * g[A][v];
                }
            }
#pragma unroll
            for (int v = 0; v < Vc; ++v) RX[LF::at2(oUL + v, k) * C + cell] = Fh[v];
        }
        if (bad) atomicOr(p.flag, 2);
    }
    __syncthreads();

    // F4: project the face flux on the transverse modes (g_k phi_l(xi_k) of Eq. 20's surface lines) -> global
    // flux array: D * Vc * Nf rows [axis][var][transverse index]
    using GLF = GLay<D, M>;
    const unsigned frs = GLF::rs(p.ncells);
    double *out = p.flux + (size_t)A * Vc * Nf * frs;
    if (TILE) {
        for (int it = tid; it < Vc * C; it += NT) {
            const int cell = it % C, g = it / C;
            double t[M * M];
            tile_load<M, C, LF>(RX, oUL + g, cell, t);
            if (!K::PP || A >= 1) tile_x<DG_SEL_VTG, M>(t);     // tile axes: the two transverse axes in increasing order
            if (!K::PP || A >= 2) tile_y<DG_SEL_VTG, M>(t);
            if (cell0 + cell < p.ncells) {
#pragma unroll
                for (int q = 0; q < M * M; ++q)
                    out[(size_t)(g * Nf + q) * frs + GLF::cell(cell0 + cell, D * Vc * Nf)] = t[q];
            }
        }
    } else {
        if (M > 1 && D == 3) {
            sweep<DG_SEL_VTG, M, Nf, 1, C, NT, 1, false, false, LF>(RX, 0, 0, RX, 0, Vc, 1.0, tid);
            __syncthreads();
        }
        // last projection sweep (or the single-point weight g_0^(D-1) = 2^(D-1)) straight to global memory
        constexpr int STR = (D == 3) ? M : 1;
        constexpr int NPEN = Nf / M;
        for (int it = tid; it < Vc * NPEN * C; it += NT) {
            const int cell = it % C;
            const int r = it / C;
            const int pen = r % NPEN;
            const int v = r / NPEN;
            if (cell0 + cell >= p.ncells) continue;
            const int off = v * Nf + pencil_base<M, STR>(pen);
            double in[M];
#pragma unroll
            for (int i = 0; i < M; ++i) in[i] = RX[LF::at2(v, pencil_base<M, STR>(pen) + i * STR) * C + cell];
            double res[M];
            if (K::PP && D == 2 && A == 0) {
#pragma unroll
                for (int j = 0; j < M; ++j) res[j] = in[j];     // x faces stay nodal in y (see Cfg::PP)
            } else if (M > 1) {
                apply1d<DG_SEL_VTG, M>(in, res);
            } else {
                res[0] = in[0] * (D == 3 ? 4.0 : 2.0);
            }
#pragma unroll
            for (int j = 0; j < M; ++j)
                out[(size_t)(off + j * STR) * frs + GLF::cell(cell0 + cell, D * Vc * Nf)] = res[j];
        }
    }
    __syncthreads();
}

template <int D, int M, bool VISC, bool AV>
__global__ void __launch_bounds__((FaceCfg<D, M, VISC, AV>::NT), (FaceCfg<D, M, VISC, AV>::MINB)) dg_face_kernel(const DgStageArgs p) {
    using K = Cfg<D, M, VISC, AV>;
    using FK = FaceCfg<D, M, VISC, AV>;
    constexpr int C = FK::C, NT = FK::NT, V = K::V, Np = K::Np;
    extern __shared__ __align__(128) double smem[];
    double *RA = smem;
    double *RX = RA + (FK::DIRECT ? 0 : V * Np * C);
    int *nbr = reinterpret_cast<int *>(RX + K::NQ * K::Nf * C);
    double *bar = RX + K::NQ * K::Nf * C + (D * C + 1) / 2;   // mbarrier of the bulk copies, after nbr[D*C]
    const int tid = threadIdx.x;
    const TilePos<D, C> pos(p, tid % C);
    const int cell0 = pos.cell0;
    using GL = GLay<D, M>;
    const bool bulk = !FK::DIRECT && GL::B == 0 && bulk_ok<C>(cell0, p.ncells);
    if (bulk) {
        if (tid == 0) mbar_init(bar, 1);
        __syncthreads();
        issue_own_modes_bulk<V, Np, C, NT, typename FK::LV>(p.w_prev, p.ncells, cell0, RA, bar, tid);
    }
    if (tid < C) {
#pragma unroll
        for (int a = 0; a < D; ++a) nbr[a * C + tid] = pos.upper(p, a);
    }
    if (bulk)
        mbar_wait(bar, 0);
    else if (!FK::DIRECT)
        load_own_modes<V, Np, C, NT, typename FK::LV>(p.w_prev + GL::cell(pos.cg, V * Np), GL::rs(p.ncells), RA, tid);
    __syncthreads();
    face_axis<D, M, VISC, AV, 0>(p, RA, RX, nbr, cell0, tid);
    face_axis<D, M, VISC, AV, 1>(p, RA, RX, nbr, cell0, tid);
    if (D == 3) face_axis<D, M, VISC, AV, (D == 3 ? 2 : 0)>(p, RA, RX, nbr, cell0, tid);
}

// ---------------------------------------------------------------------------------------------------
// the stage kernel
// ---------------------------------------------------------------------------------------------------
template <int D, int M, bool VISC, bool AV>
__global__ void __launch_bounds__((Cfg<D, M, VISC, AV>::NT), DG_STAGE_MINB) dg_stage_kernel(const DgStageArgs p) {
    using K = Cfg<D, M, VISC, AV>;
    constexpr int C = K::C, NT = K::NT, V = K::V, Vc = K::Vc, Np = K::Np;
    constexpr bool GRAD = K::GRAD, BLK = K::BLK;
    using L = Lay<M * M, Np, use_swizzle(M, C), use_rot(M, C, K::BLK)>;
    constexpr int NTILE = Np / (M * M);          // m x m tiles per slot (m in 3D, 1 in 2D)
    extern __shared__ __align__(128) double smem[];
    double *RA = smem;
    double *RX = RA + V * Np * C;
    double *ACC = RX + K::RX * C;
    double *Wk = ACC + V * Np * C;
    double *red = Wk + C;
    double *sens = red + 2 * (NT / 32);           // [4][NT/32][C] partial sensor sums (AV only)
    double *bar = sens + (AV ? 4 * (NT / 32) * C : 0);   // mbarrier of the bulk copies
    const int tid = threadIdx.x;
    const int cell0 = blockIdx.x * C;
    // own modes of a full tile travel global -> RA as bulk asynchronous copies (one request per row segment);
    // with fewer than 8 cells per block (16/32-byte segments, m >= 6) batched plain loads are cheaper here
    using GL = GLay<D, M>;
    constexpr int RW = V * Np, RF = D * Vc * K::Nf;      // rows of a state array / of the flux array
    const unsigned grs = GL::rs(p.ncells);
    const bool bulk = (C >= 8) && GL::B == 0 && bulk_ok<C>(cell0, p.ncells);
    if (bulk) {
        if (tid == 0) mbar_init(bar, 1);
        __syncthreads();
        issue_own_modes_bulk<V, Np, C, NT, L>(p.w_prev, p.ncells, cell0, RA, bar, tid);
    }

    // every thread works on one fixed cell of the block (NT is a multiple of C)
    static_assert(NT % C == 0, "threads per block must be a multiple of cells per block");
    const int cl = tid % C;
    const int cg = min(cell0 + cl, p.ncells - 1);
    int nbm[D];                                  // lower neighbour along each axis (periodic wrap)
    {
        // the integer divisions of cell -> (ix, iy, iz) once per cell of the block, not once per thread
        __shared__ int s_nbm[D][32];
        if (tid < C) {
            const int c = min(cell0 + tid, p.ncells - 1);
            const int ix = c % p.nx;
            const int iy = (c / p.nx) % p.ny;
            const int iz = c / (p.nx * p.ny);
            s_nbm[0][tid] = c + ((ix == 0) ? p.nx - 1 : -1);
            s_nbm[1][tid] = c + ((iy == 0) ? (p.ny - 1) * p.nx : -p.nx);
            if (D == 3) s_nbm[D - 1][tid] = c + ((iz == 0) ? (p.nz - 1) * p.nx * p.ny : -p.nx * p.ny);
        }
        __syncthreads();
#pragma unroll
        for (int a = 0; a < D; ++a) nbm[a] = s_nbm[a][cl];
    }
    // ---- front loads, all in flight before the first barrier: face fluxes of the 2D faces, own modes ----
    constexpr int NFL = Vc * K::Nf;                       // flux values per cell and axis
    constexpr int NLIFT = (NFL * C + NT - 1) / NT;
    double Fp[D][NLIFT], Fm[D][NLIFT];
#pragma unroll
    for (int a = 0; a < D; ++a) {
        const double *fp = p.flux + (size_t)(tid / C) * grs + GL::cell(cg, RF);
        const double *fm = p.flux + (size_t)(tid / C) * grs + GL::cell(nbm[a], RF);
#pragma unroll
        for (int k = 0; k < NLIFT; ++k) {
            if (tid / C + k * (NT / C) < NFL) {
                Fp[a][k] = __ldg(row_ptr(fp, a * NFL + k * (NT / C), grs));
                Fm[a][k] = __ldg(row_ptr(fm, a * NFL + k * (NT / C), grs));
            }
        }
    }
    if (!p.rhs_only && cl % 4 == 0) {
        // u^n is needed only by the stage combine at the very end: start it towards L2 now
        const double *wn = p.w_n + (size_t)(tid / C) * grs + GL::cell(cg, RW);
#pragma unroll 4
        for (int k = 0; tid / C + k * (NT / C) < V * Np; ++k)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(row_ptr(wn, k * (NT / C), grs)));
    }
    if (AV && tid < C) {
        // wiggle source of Eq. 45 from the previous step's sensor (readings A14, A15)
        const double S = p.sens_prev[cg];
        const double G = p.sens_prev[p.ncells + cg];
        Wk[tid] = (S > p.s_onset) ? p.f_w * fmax(0.0, G) : 0.0;
    }
    // own modes -> RA, zero ACC
    for (int r = tid / C; r < V * Np; r += NT / C) ACC[r * C + cl] = 0.0;
    if (bulk)
        mbar_wait(bar, 0);
    else
        load_own_modes<V, Np, C, NT, L>(p.w_prev + GL::cell(cg, RW), grs, RA, tid);   // global slot order: r = mode*V + v
    __syncthreads();

    // ---- surface term: lift the face fluxes of dg_face_kernel along each normal (Eq. 20, readings A3/A4) ----
    //      dw_l -= pref [P_l(+1) F^(a+) - P_l(-1) F^(a-)],  F^(a+) = this cell's upper face, F^(a-) = the lower
    //      neighbour's upper face; every (variable, transverse mode) item owns one modal pencil along the axis
    {
        const double pref = (D == 3 ? 0.25 : 0.5) / p.h;
#pragma unroll
        for (int a = 0; a < D; ++a) {
            const int SA = (a == 0) ? 1 : (a == 1 ? M : M * M);
#pragma unroll
            for (int k = 0; k < NLIFT; ++k) {
                const int r = tid / C + k * (NT / C);     // v*Nf + lt
                if (r < NFL) {
                    const int lt = r % K::Nf;
                    const int v = r / K::Nf;
                    const int base = (lt / SA) * (SA * M) + (lt % SA);
#pragma unroll
                    for (int l = 0; l < M; ++l)
                        ACC[L::at2(v, base + l * SA) * C + cl] +=
                            pref * (c_tab.Pend[0][l] * Fm[a][k] - c_tab.Pend[1][l] * Fp[a][k]);
                }
            }
            __syncthreads();
        }
    }

    // ---- volume term ----
    expand_volume<D, M, C, NT, BLK, L>(RA, V, tid);               // V1: Eq. 21
    const double ih = 1.0 / p.h;
    if (GRAD) {
        // V2: gradients at the Gauss points by analytic differentiation of the basis
        if (BLK) {
            for (int it = tid; it < Vc * NTILE * C; it += NT) {
                const int cell = it % C, g = it / C;
                double t[M * M], a[M * M];
                tile_load<M, C, L>(RA, g, cell, t);
#pragma unroll
                for (int q = 0; q < M * M; ++q) a[q] = t[q];
                tile_x<DG_SEL_DHAT, M>(a);
#pragma unroll
                for (int q = 0; q < M * M; ++q) a[q] *= 2.0 * ih;
                tile_store<M, C, L>(RX, g, cell, a);
                tile_y<DG_SEL_DHAT, M>(t);
#pragma unroll
                for (int q = 0; q < M * M; ++q) t[q] *= 2.0 * ih;
                tile_store<M, C, L>(RX, Vc * NTILE + g, cell, t);
            }
        } else {
            sweep<DG_SEL_DHAT, M, Np, 1, C, NT, 1, false, true, L>(RA, 0, 0, RX, 0, Vc, 2.0 * ih, tid);
            sweep<DG_SEL_DHAT, M, Np, M, C, NT, 1, false, true, L>(RA, 0, 0, RX, Vc, Vc, 2.0 * ih, tid);
        }
        if (D == 3) sweep<DG_SEL_DHAT, M, Np, M * M, C, NT, 1, false, true, L>(RA, 0, 0, RX, 2 * Vc, Vc, 2.0 * ih, tid);
        __syncthreads();
    }
    {
        // V3: point-wise fluxes G_a = f_a - F_NS,a - eps d_a u (Eq. 24; 315 Eq. 38), alpha source
        bool bad = false;
        double amax = 0.0;                                     // max alpha at the Gauss points (diagnostics)
        const double decay = (double)M / (p.f_tau * p.h);      // 1/tau = (n+1) c_s / (f_tau h), Eq. 44
        for (int it = tid; it < Np * C; it += NT) {
            const int cell = it % C;
            const int j = it / C;
            double u[Vc];
#pragma unroll
            for (int v = 0; v < Vc; ++v) u[v] = RA[L::at2(v, j) * C + cell];
            const Prim<D> q = primitives<D>(u, p.gamma);
            bad |= !(q.rho > 0.0) || !(q.p > 0.0);
            double g[D][D + 2 + DG_TRACER], dv[D][D];
            double divv = 0.0, eps = 0.0;
            if (GRAD) {
#pragma unroll
                for (int b = 0; b < D; ++b)
#pragma unroll
                    for (int v = 0; v < Vc; ++v) g[b][v] = RX[L::at2(b * Vc + v, j) * C + cell];
                velocity_gradient<D>(q, g, dv);
#pragma unroll
                for (int b = 0; b < D; ++b) divv += dv[b][b];
            }
            if (AV) {
                const double al = RA[L::at2(Vc, j) * C + cell];
                const double cs = fast_sqrt(p.gamma * q.p * q.ir);
                if (cell0 + cell < p.ncells) amax = fmax(amax, al);
                eps = fmin(fmax(al, 0.0), p.alpha_max) * cs * (p.h / (double)M);        // Eq. 46, A17
                // Eq. 43-45: shock source + wiggle source - decay; stored pre-scaled by h/2 for the projection
                const double src = p.f_v * fmax(0.0, -divv) + Wk[cell] - al * (cs * decay);
                RA[L::at2(Vc, j) * C + cell] = 0.5 * p.h * src;
            }
#pragma unroll
            for (int a = 0; a < D; ++a) {
                double F[Vc];
                euler_flux<D>(u, q, a, F);
                if (VISC) ns_flux_sub<D>(q, g, dv, divv, a, p.gamma, p.nu, p.chi, F, DG_TRACER ? u[Vc - 1] * q.ir : 0.0, p.eta);
                if (AV) {
#pragma unroll
                    for (int v = 0; v < Vc; ++v) F[v] -= eps * g[a][v];
                }
#pragma unroll
                for (int v = 0; v < Vc; ++v) RX[L::at2(a * Vc + v, j) * C + cell] = F[v];
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
    __syncthreads();
    if (AV && p.do_sensor && tid == 0) {
        double a = red[0];
        for (int i = 1; i < NT / 32; ++i) a = fmax(a, red[i]);
        atomic_max_nonneg(&p.maxbits[2], a);
    }
    // Stage-combine inputs u^n and u^(i-1) of this thread's rows: issued before the last projection sweep so that
    // their latency is covered by it (same ownership as load_own_modes: modes g, g+G, ... of every variable).
    constexpr int CG = NT / C;
    constexpr int CNK = (Np + CG - 1) / CG;
    double wn[CNK][V], wp[CNK][V];
#define LOAD_COMBINE_INPUTS()                                                                               \
    do {                                                                                                    \
        const bool need_n = !p.rhs_only, need_p = !p.rhs_only && p.rk_b != 0.0;                             \
        const double *bn = p.w_n + (size_t)((tid / C) * V) * grs + GL::cell(cg, RW);                        \
        const double *bp = p.w_prev + (size_t)((tid / C) * V) * grs + GL::cell(cg, RW);                     \
        _Pragma("unroll") for (int k = 0; k < CNK; ++k) _Pragma("unroll") for (int v = 0; v < V; ++v) {     \
            wn[k][v] = wp[k][v] = 0.0;                                                                      \
            if (tid / C + k * CG < Np) {                                                                    \
                if (need_n) wn[k][v] = *row_ptr(bn, k * CG * V + v, grs);    /* may alias w_out */          \
                if (need_p) wp[k][v] = __ldg(row_ptr(bp, k * CG * V + v, grs));                             \
            }                                                                                               \
        }                                                                                                   \
    } while (0)

    // V4 + V5: weak-form derivative in nodal space, N = sum_a S_a G_a, then projection on the modes,
    //          dw += pref * (x)_a VtG N; alpha row: projection of the source only
    {
        const double pref = (D == 3 ? 0.25 : 0.5) * ih;
        if (BLK) {
            if (D == 3) {
                sweep<DG_SEL_S, M, Np, M * M, C, NT, 1, false, false, L>(RX, 2 * Vc, 0, RX, 2 * Vc, Vc, 1.0, tid);
                __syncthreads();
            }
            // per m x m tile: S_x G_x + S_y G_y (+ S_z G_z), projected along x and y in registers
            for (int it = tid; it < V * NTILE * C; it += NT) {
                const int cell = it % C, g = it / C;
                double n[M * M];
                if (g < Vc * NTILE) {
                    double b[M * M];
                    tile_load<M, C, L>(RX, g, cell, n);
                    tile_x<DG_SEL_S, M>(n);
                    tile_load<M, C, L>(RX, Vc * NTILE + g, cell, b);
                    tile_y<DG_SEL_S, M>(b);
#pragma unroll
                    for (int q = 0; q < M * M; ++q) n[q] += b[q];
                    if (D == 3) {
                        tile_load<M, C, L>(RX, 2 * Vc * NTILE + g, cell, b);
#pragma unroll
                        for (int q = 0; q < M * M; ++q) n[q] += b[q];
                    }
                } else {
                    tile_load<M, C, L>(RA, g, cell, n);      // alpha source (slot Vc of RA)
                }
                tile_x<DG_SEL_VTG, M>(n);
                tile_y<DG_SEL_VTG, M>(n);
                if (D == 3) {
                    if (g < Vc * NTILE)
                        tile_store<M, C, L>(RX, g, cell, n);
                    else
                        tile_store<M, C, L>(RA, g, cell, n);
                } else {
                    double acc[M * M];
                    tile_load<M, C, L>(ACC, g, cell, acc);
#pragma unroll
                    for (int q = 0; q < M * M; ++q) acc[q] = fma(pref, n[q], acc[q]);
                    tile_store<M, C, L>(ACC, g, cell, acc);
                }
            }
            __syncthreads();
            LOAD_COMBINE_INPUTS();
            if (D == 3) {
                sweep<DG_SEL_VTG, M, Np, M * M, C, NT, 1, true, true, L>(RX, 0, 0, ACC, 0, Vc, pref, tid);
                if (AV) sweep<DG_SEL_VTG, M, Np, M * M, C, NT, 1, true, true, L>(RA, Vc, 0, ACC, Vc, 1, pref, tid);
                __syncthreads();
            }
        } else {
            sweep<DG_SEL_S, M, Np, 1, C, NT, 1, false, false, L>(RX, 0, 0, RX, 0, Vc, 1.0, tid);
            sweep<DG_SEL_S, M, Np, M, C, NT, 1, false, false, L>(RX, Vc, 0, RX, Vc, Vc, 1.0, tid);
            if (D == 3) sweep<DG_SEL_S, M, Np, M * M, C, NT, 1, false, false, L>(RX, 2 * Vc, 0, RX, 2 * Vc, Vc, 1.0, tid);
            __syncthreads();
            sweep<DG_SEL_VTG, M, Np, 1, C, NT, D, false, false, L>(RX, 0, Vc, RX, 0, Vc, 1.0, tid);
            if (AV) sweep<DG_SEL_VTG, M, Np, 1, C, NT, 1, false, false, L>(RA, Vc, 0, RA, Vc, 1, 1.0, tid);
            __syncthreads();
            if (D == 3) {
                sweep<DG_SEL_VTG, M, Np, M, C, NT, 1, false, false, L>(RX, 0, 0, RX, 0, Vc, 1.0, tid);
                if (AV) sweep<DG_SEL_VTG, M, Np, M, C, NT, 1, false, false, L>(RA, Vc, 0, RA, Vc, 1, 1.0, tid);
                __syncthreads();
            }
            constexpr int SL = (D == 3) ? M * M : M;
            LOAD_COMBINE_INPUTS();
            sweep<DG_SEL_VTG, M, Np, SL, C, NT, 1, true, true, L>(RX, 0, 0, ACC, 0, Vc, pref, tid);
            if (AV) sweep<DG_SEL_VTG, M, Np, SL, C, NT, 1, true, true, L>(RA, Vc, 0, ACC, Vc, 1, pref, tid);
            __syncthreads();
        }
    }

    // ---- stage combine + shock-sensor sums (Eq. 42, 45; readings A13/A15) ----
    // The sensor is evaluated on stage 1 only, where w_prev == w_n: the density rows of w^n and dw/dt pass through
    // the combine loop; partial sums per thread are reduced per cell in a fixed order.
    const double cdt = p.rhs_only ? 1.0 : p.rk_c * p.scal[0];
    double sA = 0.0, sB = 0.0, dA = 0.0, dB = 0.0;
    {
        constexpr int G = CG;
        constexpr int NK = CNK;
        const int g = tid / C;
        const bool active = cell0 + cl < p.ncells;
        double *bo = p.w_out + (size_t)(g * V) * grs + GL::cell(cg, RW);
#pragma unroll
        for (int k = 0; k < NK; ++k) {
            const int mode = g + k * G;
            int rem = mode, top = 0, lsum = 0;
#pragma unroll
            for (int a = 0; a < D; ++a) {
                top |= (rem % M == M - 1);
                lsum += rem % M;
                rem /= M;
            }
            // total-degree basis: discarded modes are not test functions; the sensor's highest
            // modes are those with sum_a l_a = n
            const bool keep = !p.total_degree || (lsum <= M - 1);
            if (p.total_degree) top = (lsum == M - 1);
#pragma unroll
            for (int v = 0; v < V; ++v) {
                if (mode < Np) {
                    const double Ld = keep ? ACC[L::at2(v, mode) * C + cl] : 0.0;
                    double wnew = Ld;
                    if (!p.rhs_only) wnew = fma(cdt, Ld, fma(p.rk_b, wp[k][v], p.rk_a * wn[k][v]));
                    if (active) *row_ptr(bo, k * G * V + v, grs) = wnew;
                    if (p.w_aux != nullptr && active) {
                        // SSPRK(5,4): the part of the last stage that is known now (u^(2), u^(3), L(u^(3)))
                        const size_t gi = (size_t)((g + k * G) * V + v) * grs + GL::cell(cg, RW);
                        p.w_aux[gi] = fma(p.aux_c * p.scal[0], Ld, fma(p.aux_b, wp[k][v], p.aux_a * p.w_aux_in[gi]));
                    }
                    if (p.do_wavespeed) RA[L::at2(v, mode) * C + cl] = wnew;
                    if (AV && p.do_sensor && v == 0) {
                        const double w = wn[k][v];
                        sB = fma(w, w, sB);
                        dB = fma(w, Ld, dB);
                        if (top && M > 1) {
                            sA = fma(w, w, sA);
                            dA = fma(w, Ld, dA);
                        }
                    }
                }
            }
        }
    }
#undef LOAD_COMBINE_INPUTS
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
        __syncthreads();
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
    // ---- wave speeds of the new state for the next step's Eq. 23 ----
    if (p.do_wavespeed) {
        __syncthreads();
        expand_volume<D, M, C, NT, BLK, L>(RA, Vc, tid);
        wavespeed_points<D, M, C, NT, L>(RA, p.gamma, p.flag, red, p.maxbits, tid);
    }
}

// standalone wave-speed kernel (after dg_set_state): load -> expand -> max
template <int D, int M, bool VISC, bool AV>
__global__ void __launch_bounds__((Cfg<D, M, VISC, AV>::NT), DG_STAGE_MINB) dg_wavespeed_kernel(const DgStageArgs p) {
    using K = Cfg<D, M, VISC, AV>;
    constexpr int C = K::C, NT = K::NT, V = K::V, Vc = K::Vc, Np = K::Np;
    using L = Lay<M * M, Np, use_swizzle(M, C), use_rot(M, C, K::BLK)>;
    extern __shared__ __align__(128) double smem[];
    double *RA = smem;
    double *red = RA + V * Np * C + K::RX * C + V * Np * C + C;
    const int tid = threadIdx.x;
    const int cell0 = blockIdx.x * C;
    load_own_modes<V, Np, C, NT, L>(p.w_prev + GLay<D, M>::cell(min(cell0 + tid % C, p.ncells - 1), V * Np),
                                    GLay<D, M>::rs(p.ncells), RA, tid);
    __syncthreads();
    expand_volume<D, M, C, NT, K::BLK, L>(RA, Vc, tid);
    wavespeed_points<D, M, C, NT, L>(RA, p.gamma, p.flag, red, p.maxbits, tid);
}

}  // namespace DG_NS
