// Positivity limiter (Eq. 47), optional, run on the output of every RK stage.
//
// Per cell: mean density rho_bar = w_0 and mean pressure p_bar (pressure of the cell-mean state); the state is
// evaluated at the union of the m^d volume Gauss points and the m^(d-1) Gauss points of the 2d faces; if
// rho_min < rho_bottom = 1e-6 rho_bar every mode but the mean of every conserved field is multiplied by
// f = (rho_bar - rho_bottom)/(rho_bar - rho_min); then, while p_min < p_bottom = 1e-6 p_bar, the same modes are
// halved.  Scaling the higher modes by F scales the deviation of every point value from the cell mean by F, so the
// point values are expanded once and the pressure loop works on   u(x) = u_bar + F (u_nodal(x) - u_bar).
// The state is rewritten only for cells with F != 1 (smooth flows: the kernel only reads).
//
// Same block structure as the stage kernels: C consecutive cells per block, lanes = cells, [slot][point][cell] shared
// arrays (plain layout: this kernel is not on the default path).
#pragma once

#include "dg_stage.cuh"

namespace DG_NS {

template <int D, int M>
struct LimCfg {
    static constexpr int Vc = D + 2 + DG_TRACER;
    static constexpr int Np = ipow(M, D);
    static constexpr int Nf = ipow(M, D - 1);
    static constexpr int NFS = 2 * D * Vc;                       // face slots: (axis, side, variable)
    static constexpr int NT = 256;
    static constexpr int FP = 2 * Vc * Np + NFS * Nf;            // modal copy + volume point values + face point values
    static constexpr int extra_bytes(int c) { return c * (8 * (Vc + 3) + 8 + 4) + 32; }
    static constexpr int pick_c() {
        int c = 32;
        while (c > 1 && c * FP * 8 + extra_bytes(c) > 110 * 1024) c >>= 1;
        return c;
    }
    static constexpr int C = pick_c();
    static constexpr int kSmemBytes = C * FP * 8 + extra_bytes(C);
    static_assert(kSmemBytes <= kSmemMax, "limiter: per-cell footprint exceeds shared memory");
    static constexpr bool BLK = (M >= 2) && (M * M <= 25);
};

// order-preserving map double -> unsigned 64 bit (for atomicMin on values of either sign)
__device__ __forceinline__ unsigned long long ord_enc(double x) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(x);
    return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double ord_dec(unsigned long long u) {
    const unsigned long long b = (u >> 63) ? (u & 0x7fffffffffffffffull) : ~u;
    return __longlong_as_double((long long)b);
}

// Scratch of the limiter per block of C cells (after the face point values).
template <int D, int C>
struct LimScratch {
    static constexpr int Vc = D + 2 + DG_TRACER;
    double *mean, *Fc, *rbot, *pbot;
    unsigned long long *key;
    int *act;
    __device__ __forceinline__ explicit LimScratch(double *base) {
        mean = base;                                             // [Vc][C]
        Fc = mean + Vc * C;                                      // factor per cell
        rbot = Fc + C;                                           // rho_bottom per cell
        pbot = rbot + C;                                         // p_bottom per cell
        key = reinterpret_cast<unsigned long long *>(pbot + C);
        act = reinterpret_cast<int *>(key + C);                  // 1: cell takes part (inside the mesh, positive means)
    }
    static constexpr int kDoubles = (Vc + 3) * C + C + (C + 1) / 2 + 2;
};

// The limiter proper, shared by dg_limiter_kernel and by the tail of dg_stage2_kernel (fused form).
//   NV  [Vc][Np][C] (layout LV): MODAL coefficients of the block's cells on entry, volume point values on exit
//   NF  [2D*Vc][Nf][C] (plain):  face point values on exit
//   sc.Fc[cell]: the factor F of Eq. 47 (density step, then the halvings of the pressure step) on exit
// `inside(cell)`: the lane-cell lies inside the mesh.  Ends with a barrier; every thread of the block must call it.
template <int D, int M, int C, int NT, bool BLK, class LV>
__device__ __forceinline__ void limiter_core(double *NV, double *NF, const LimScratch<D, C> &sc, double gamma, int *flag,
                                             int cell0, int ncells, int tid) {
    constexpr int Vc = D + 2 + DG_TRACER, Np = ipow(M, D), Nf = ipow(M, D - 1), NFS = 2 * D * Vc;
    constexpr int NPT = Np + 2 * D * Nf;                         // evaluation points per cell
    constexpr int G = NT / C;
    using LF = Lay<Nf, Nf, false, 0>;
    const int cl = tid % C, g = tid / C;
    // face traces: contract the normal axis with P_l(-1) / P_l(+1)
    for (int r = g; r < NFS * Nf; r += G) {
        const int slot = r / Nf, lt = r % Nf;
        const int a = slot / (2 * Vc), s = (slot / Vc) % 2, v = slot % Vc;
        const int SA = (a == 0) ? 1 : (a == 1 ? M : M * M);
        const int base = (lt / SA) * (SA * M) + (lt % SA);
        double t = 0.0;
#pragma unroll
        for (int l = 0; l < M; ++l) t = fma(c_tab.Pend[s][l], NV[LV::at2(v, base + l * SA) * C + cl], t);
        NF[(slot * Nf + lt) * C + cl] = t;
    }
    if (tid < C) {
        double m[Vc];
#pragma unroll
        for (int v = 0; v < Vc; ++v) {
            m[v] = NV[LV::at2(v, 0) * C + tid];                   // mode 0 = cell mean (P_0 = 1)
            sc.mean[v * C + tid] = m[v];
        }
        double mm = 0.0;
#pragma unroll
        for (int b = 0; b < D; ++b) mm = fma(m[1 + b], m[1 + b], mm);
        const double pb = (gamma - 1.0) * (m[1 + D] - 0.5 * mm / m[0]);
        const bool ok = (m[0] > 0.0) && (pb > 0.0);
        if (!ok && cell0 + tid < ncells) atomicOr(flag, 8);       // "a code crash is unavoidable"
        sc.act[tid] = (ok && cell0 + tid < ncells) ? 1 : 0;
        sc.rbot[tid] = 1.0e-6 * m[0];
        sc.pbot[tid] = 1.0e-6 * pb;
        sc.Fc[tid] = 1.0;
        sc.key[tid] = ~0ull;
    }
    __syncthreads();
    // point values: volume (Eq. 21) and the transverse expansion on the faces
    expand_volume<D, M, C, NT, BLK, LV>(NV, Vc, tid);
    if (M > 1) {
        sweep<DG_SEL_V, M, Nf, 1, C, NT, 1, false, false, LF>(NF, 0, 0, NF, 0, NFS, 1.0, tid);
        __syncthreads();
        if (D == 3) {
            sweep<DG_SEL_V, M, Nf, M, C, NT, 1, false, false, LF>(NF, 0, 0, NF, 0, NFS, 1.0, tid);
            __syncthreads();
        }
    }
    // value of variable v at evaluation point q of cell `cell`
    auto at_point = [&](int v, int q, int cell) -> double {
        if (q < Np) return NV[LV::at2(v, q) * C + cell];
        const int qq = q - Np;
        return NF[(((qq / Nf) * Vc + v) * Nf + qq % Nf) * C + cell];
    };

    // ---- density ----
    {
        double lo = 1.0e300;
        for (int q = g; q < NPT; q += G) lo = fmin(lo, at_point(0, q, cl));
        atomicMin(&sc.key[cl], ord_enc(lo));
    }
    __syncthreads();
    if (tid < C) {
        const double rmin = ord_dec(sc.key[tid]);
        const double rb = sc.mean[tid];
        if (sc.act[tid] && rmin < sc.rbot[tid]) sc.Fc[tid] = (rb - sc.rbot[tid]) / (rb - rmin);
    }
    // ---- pressure: halve until p_min >= p_bottom ----
    for (int iter = 0; iter < 64; ++iter) {
        if (tid < C) sc.key[tid] = ~0ull;
        __syncthreads();
        {
            const double F = sc.Fc[cl];
            double m[Vc];
#pragma unroll
            for (int v = 0; v < Vc; ++v) m[v] = sc.mean[v * C + cl];
            double lo = 1.0e300;
            for (int q = g; q < NPT; q += G) {
                double u[Vc];
#pragma unroll
                for (int v = 0; v < Vc; ++v) u[v] = fma(F, at_point(v, q, cl) - m[v], m[v]);
                double mm = 0.0;
#pragma unroll
                for (int b = 0; b < D; ++b) mm = fma(u[1 + b], u[1 + b], mm);
                lo = fmin(lo, (gamma - 1.0) * (u[1 + D] - 0.5 * mm / u[0]));
            }
            atomicMin(&sc.key[cl], ord_enc(lo));
        }
        __syncthreads();
        int again = 0;
        if (tid < C && sc.act[tid] == 1) {
            if (ord_dec(sc.key[tid]) < sc.pbot[tid]) {
                sc.Fc[tid] *= 0.5;
                again = 1;
            } else {
                sc.act[tid] = 2;                                  // settled: never halved again
            }
        }
        if (!__syncthreads_or(again)) break;
    }
}

template <int D, int M>
__global__ void __launch_bounds__(256, 2) dg_limiter_kernel(double *w, int V, int ncells, double gamma, int *flag) {
    using K = LimCfg<D, M>;
    constexpr int C = K::C, NT = K::NT, Vc = K::Vc, Np = K::Np, Nf = K::Nf, NFS = K::NFS;
    using LV = Lay<M * M, Np, false, 0>;
    extern __shared__ __align__(128) double smem[];
    double *RA = smem;                                           // modal copy           [Vc][Np][C]
    double *NV = RA + Vc * Np * C;                               // volume point values  [Vc][Np][C]
    double *NF = NV + Vc * Np * C;                               // face point values    [axis][side][Vc][Nf][C]
    const LimScratch<D, C> sc(NF + NFS * Nf * C);
    static_assert(NT % C == 0, "threads per block must be a multiple of cells per block");
    const int tid = threadIdx.x;
    const int cell0 = blockIdx.x * C;
    const int cl = tid % C, g = tid / C;
    constexpr int G = NT / C;
    const int cg = min(cell0 + cl, ncells - 1);
    const unsigned grs = GLay<D, M>::rs(ncells);
    double *wc = w + GLay<D, M>::cell(cg, V * Np);               // (row 0, this thread's cell), V variables per mode

    for (int mode = g; mode < Np; mode += G) {
#pragma unroll
        for (int v = 0; v < Vc; ++v) {
            const double x = wc[(size_t)(mode * V + v) * grs]   /* rewritten below: no non-coherent load */;
            RA[(v * Np + mode) * C + cl] = x;
            NV[(v * Np + mode) * C + cl] = x;
        }
    }
    __syncthreads();
    limiter_core<D, M, C, NT, K::BLK, LV>(NV, NF, sc, gamma, flag, cell0, ncells, tid);
    // ---- Eq. 47: w_l' = F w_l for every mode but the mean ----
    {
        const double F = sc.Fc[cl];
        if (F != 1.0 && cell0 + cl < ncells) {
            for (int mode = g; mode < Np; mode += G) {
                if (mode == 0) continue;
#pragma unroll
                for (int v = 0; v < Vc; ++v)
                    wc[(size_t)(mode * V + v) * grs] = F * RA[(v * Np + mode) * C + cl];
            }
        }
    }
}

}  // namespace DG_NS
