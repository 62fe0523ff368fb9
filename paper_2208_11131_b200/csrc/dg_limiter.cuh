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

namespace dgk {

template <int D, int M>
struct LimCfg {
    static constexpr int Vc = D + 2;
    static constexpr int Np = ipow(M, D);
    static constexpr int Nf = ipow(M, D - 1);
    static constexpr int NFS = 2 * D * Vc;                       // face slots: (axis, side, variable)
    static constexpr int NT = 256;
    static constexpr int FP = 2 * Vc * Np + NFS * Nf;            // modal copy + volume point values + face point values
    static constexpr int extra_bytes(int c) { return c * (8 * (Vc + 3) + 8 + 4) + 16; }
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

template <int D, int M>
__global__ void __launch_bounds__(256, 2) dg_limiter_kernel(double *w, int V, int ncells, double gamma, int *flag) {
    using K = LimCfg<D, M>;
    constexpr int C = K::C, NT = K::NT, Vc = K::Vc, Np = K::Np, Nf = K::Nf, NFS = K::NFS;
    constexpr int NPT = Np + 2 * D * Nf;                         // evaluation points per cell
    using LV = Lay<M * M, Np, false, 0>;
    using LF = Lay<Nf, Nf, false, 0>;
    extern __shared__ __align__(128) double smem[];
    double *RA = smem;                                           // modal copy           [Vc][Np][C]
    double *NV = RA + Vc * Np * C;                               // volume point values  [Vc][Np][C]
    double *NF = NV + Vc * Np * C;                               // face point values    [axis][side][Vc][Nf][C]
    double *mean = NF + NFS * Nf * C;                            // [Vc][C]
    double *Fc = mean + Vc * C;                                  // factor per cell
    double *rbot = Fc + C;                                       // rho_bottom per cell
    double *pbot = rbot + C;                                     // p_bottom per cell
    unsigned long long *key = reinterpret_cast<unsigned long long *>(pbot + C);
    int *act = reinterpret_cast<int *>(key + C);                 // 1: cell takes part (full tile cell, positive means)
    static_assert(NT % C == 0, "threads per block must be a multiple of cells per block");
    const int tid = threadIdx.x;
    const int cell0 = blockIdx.x * C;
    const int cl = tid % C, g = tid / C;
    constexpr int G = NT / C;
    const int cg = min(cell0 + cl, ncells - 1);

    for (int mode = g; mode < Np; mode += G) {
#pragma unroll
        for (int v = 0; v < Vc; ++v) {
            const double x = w[(size_t)(mode * V + v) * ncells + cg]   /* rewritten below: no non-coherent load */;
            RA[(v * Np + mode) * C + cl] = x;
            NV[(v * Np + mode) * C + cl] = x;
        }
    }
    __syncthreads();
    // face traces: contract the normal axis with P_l(-1) / P_l(+1)
    for (int r = g; r < NFS * Nf; r += G) {
        const int slot = r / Nf, lt = r % Nf;
        const int a = slot / (2 * Vc), s = (slot / Vc) % 2, v = slot % Vc;
        const int SA = (a == 0) ? 1 : (a == 1 ? M : M * M);
        const int base = (lt / SA) * (SA * M) + (lt % SA);
        double t = 0.0;
#pragma unroll
        for (int l = 0; l < M; ++l) t = fma(c_tab.Pend[s][l], RA[(v * Np + base + l * SA) * C + cl], t);
        NF[(slot * Nf + lt) * C + cl] = t;
    }
    if (tid < C) {
        double m[Vc];
#pragma unroll
        for (int v = 0; v < Vc; ++v) {
            m[v] = RA[(v * Np) * C + tid];                        // mode 0 = cell mean (P_0 = 1)
            mean[v * C + tid] = m[v];
        }
        double mm = 0.0;
#pragma unroll
        for (int b = 0; b < D; ++b) mm = fma(m[1 + b], m[1 + b], mm);
        const double pb = (gamma - 1.0) * (m[1 + D] - 0.5 * mm / m[0]);
        const bool ok = (m[0] > 0.0) && (pb > 0.0);
        if (!ok && cell0 + tid < ncells) atomicOr(flag, 8);       // "a code crash is unavoidable"
        act[tid] = (ok && cell0 + tid < ncells) ? 1 : 0;
        rbot[tid] = 1.0e-6 * m[0];
        pbot[tid] = 1.0e-6 * pb;
        Fc[tid] = 1.0;
        key[tid] = ~0ull;
    }
    __syncthreads();
    // point values: volume (Eq. 21) and the transverse expansion on the faces
    expand_volume<D, M, C, NT, K::BLK, LV>(NV, Vc, tid);
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
        if (q < Np) return NV[(v * Np + q) * C + cell];
        const int qq = q - Np;
        return NF[(((qq / Nf) * Vc + v) * Nf + qq % Nf) * C + cell];
    };

    // ---- density ----
    {
        double lo = 1.0e300;
        for (int q = g; q < NPT; q += G) lo = fmin(lo, at_point(0, q, cl));
        atomicMin(&key[cl], ord_enc(lo));
    }
    __syncthreads();
    if (tid < C) {
        const double rmin = ord_dec(key[tid]);
        const double rb = mean[tid];
        if (act[tid] && rmin < rbot[tid]) Fc[tid] = (rb - rbot[tid]) / (rb - rmin);
    }
    // ---- pressure: halve until p_min >= p_bottom ----
    for (int iter = 0; iter < 64; ++iter) {
        if (tid < C) key[tid] = ~0ull;
        __syncthreads();
        {
            const double F = Fc[cl];
            double m[Vc];
#pragma unroll
            for (int v = 0; v < Vc; ++v) m[v] = mean[v * C + cl];
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
            atomicMin(&key[cl], ord_enc(lo));
        }
        __syncthreads();
        int again = 0;
        if (tid < C && act[tid] == 1) {
            if (ord_dec(key[tid]) < pbot[tid]) {
                Fc[tid] *= 0.5;
                again = 1;
            } else {
                act[tid] = 2;                                     // settled: never halved again
            }
        }
        if (!__syncthreads_or(again)) break;
    }
    // ---- Eq. 47: w_l' = F w_l for every mode but the mean ----
    {
        const double F = Fc[cl];
        if (F != 1.0 && cell0 + cl < ncells) {
            for (int mode = g; mode < Np; mode += G) {
                if (mode == 0) continue;
#pragma unroll
                for (int v = 0; v < Vc; ++v)
                    w[(size_t)(mode * V + v) * ncells + cg] = F * RA[(v * Np + mode) * C + cl];
            }
        }
    }
}

}  // namespace dgk
