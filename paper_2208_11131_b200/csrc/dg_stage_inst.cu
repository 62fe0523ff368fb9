// One translation unit per (DG_DIM, DG_M): instantiates the face + stage kernels for the four physics variants
// (Euler, NS, AV, NS+AV) and exports plain launch functions for dg_api.cu.  Compiled 32 times by build.py
// with -DDG_DIM=2|3 -DDG_M=1..8 -DDG_TRACER=0|1 (keeps ptxas work parallel and each image small).
#include "dg_stage.cuh"
#include "dg_stage2.cuh"
#include "dg_dispatch.h"

#ifndef DG_DIM
#error "compile with -DDG_DIM=2|3 -DDG_M=1..8"
#endif

namespace {

// opt in to > 48 KB of dynamic shared memory (once per device context, outside any stream capture)
template <bool VISC, bool AV>
cudaError_t configure() {
    using K = DG_NS::Cfg<DG_DIM, DG_M, VISC, AV>;
    cudaError_t e = cudaFuncSetAttribute(DG_NS::dg_stage_kernel<DG_DIM, DG_M, VISC, AV>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, K::kSmemBytes);
    if (e != cudaSuccess) return e;
    // NB: a kernel template must only ever be instantiated in the translation unit of its own (dim, m): every unit
    // has its own __constant__ tables, and the host stubs of equal instantiations are merged by the linker
    if constexpr (K::PP) {
        e = cudaFuncSetAttribute(DG_NS::dg_stage2_kernel<DG_DIM, DG_M, VISC, AV, false>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 DG_NS::Cfg2<DG_DIM, DG_M, VISC, AV>::kSmemBytes);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(DG_NS::dg_stage2_kernel<DG_DIM, DG_M, VISC, AV, true>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 DG_NS::Cfg2<DG_DIM, DG_M, VISC, AV>::kSmemBytes);
        if (e != cudaSuccess) return e;
    }
    e = cudaFuncSetAttribute(DG_NS::dg_face_kernel<DG_DIM, DG_M, VISC, AV>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             DG_NS::FaceCfg<DG_DIM, DG_M, VISC, AV>::kSmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(DG_NS::dg_limiter_kernel<DG_DIM, DG_M>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             DG_NS::LimCfg<DG_DIM, DG_M>::kSmemBytes);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(DG_NS::dg_wavespeed_kernel<DG_DIM, DG_M, VISC, AV>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, K::kSmemBytes);
}

template <bool VISC, bool AV>
cudaError_t launch(const DgStageArgs &a, cudaStream_t st, int wavespeed_only) {
    using K = DG_NS::Cfg<DG_DIM, DG_M, VISC, AV>;
    const int blocks = (a.ncells + K::C - 1) / K::C;
    // wavespeed_only: 0 = face + stage kernels, 1 = wave-speed kernel, 2 = face kernel only, 3 = stage kernel only
    if (wavespeed_only == 1) {
        DG_NS::dg_wavespeed_kernel<DG_DIM, DG_M, VISC, AV><<<blocks, K::NT, K::kSmemBytes, st>>>(a);
        return cudaGetLastError();
    }
    if (wavespeed_only != 3) {
        using FK = DG_NS::FaceCfg<DG_DIM, DG_M, VISC, AV>;
        const dim3 fgrid = DG_NS::tile_grid<DG_DIM, FK::C>(a.ncells, a.nx, a.ny, a.nz);
        DG_NS::dg_face_kernel<DG_DIM, DG_M, VISC, AV><<<fgrid, FK::NT, FK::kSmemBytes, st>>>(a);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (wavespeed_only != 2) {
        if constexpr (K::PP) {
            // register-tile configurations (2 <= m <= 5): second-generation stage kernel (dg_stage2.cuh)
            using K2 = DG_NS::Cfg2<DG_DIM, DG_M, VISC, AV>;
            const dim3 grid2 = DG_NS::tile_grid<DG_DIM, K2::C>(a.ncells, a.nx, a.ny, a.nz);
            const bool plain = !a.rhs_only && !a.total_degree && a.w_aux == nullptr;
            if (plain)
                DG_NS::dg_stage2_kernel<DG_DIM, DG_M, VISC, AV, true><<<grid2, K2::NT, K2::kSmemBytes, st>>>(a);
            else
                DG_NS::dg_stage2_kernel<DG_DIM, DG_M, VISC, AV, false><<<grid2, K2::NT, K2::kSmemBytes, st>>>(a);
        } else {
            DG_NS::dg_stage_kernel<DG_DIM, DG_M, VISC, AV><<<blocks, K::NT, K::kSmemBytes, st>>>(a);
        }
    }
    return cudaGetLastError();
}

template <bool VISC, bool AV>
void info(int *c, int *nt, int *smem, int *fused_limiter, int *bsz) {
    *fused_limiter = DG_NS::Cfg<DG_DIM, DG_M, VISC, AV>::PP ? 1 : 0;
    *bsz = DG_NS::GLay<DG_DIM, DG_M>::B;
    using K = DG_NS::Cfg<DG_DIM, DG_M, VISC, AV>;
    // block layout: a tile of either kernel must be a whole number of B-cell blocks (the face kernel's memory-order
    // item map and the row addressing of both kernels assume it; a -D override of the tuning macros could break it)
    constexpr int B = DG_NS::GLay<DG_DIM, DG_M>::B;
    static_assert(B == 0 || (K::C % B == 0 && DG_NS::FaceCfg<DG_DIM, DG_M, VISC, AV>::C % B == 0),
                  "cells per block of the stage and face kernels must be multiples of GLay::B");
    if constexpr (K::PP) {
        using K2 = DG_NS::Cfg2<DG_DIM, DG_M, VISC, AV>;
        *c = K2::C;
        *nt = K2::NT;
        *smem = K2::kSmemBytes;
    } else {
        *c = K::C;
        *nt = K::NT;
        *smem = K::kSmemBytes;
    }
}

}  // namespace

cudaError_t DG_FN(dg_launch, DG_DIM, DG_M)(int visc, int av, const DgStageArgs *a, cudaStream_t st,
                                           int wavespeed_only) {
    if (visc && av) return launch<true, true>(*a, st, wavespeed_only);
    if (visc) return launch<true, false>(*a, st, wavespeed_only);
    if (av) return launch<false, true>(*a, st, wavespeed_only);
    return launch<false, false>(*a, st, wavespeed_only);
}

// positivity limiter on a state buffer with V variables per mode (only the d+2 conserved ones are touched)
cudaError_t DG_FN(dg_limit, DG_DIM, DG_M)(double *w, int V, int ncells, double gamma, int *flag, cudaStream_t st) {
    using LK = DG_NS::LimCfg<DG_DIM, DG_M>;
    const int blocks = (ncells + LK::C - 1) / LK::C;
    DG_NS::dg_limiter_kernel<DG_DIM, DG_M><<<blocks, LK::NT, LK::kSmemBytes, st>>>(w, V, ncells, gamma, flag);
    return cudaGetLastError();
}

cudaError_t DG_FN(dg_upload, DG_DIM, DG_M)(const DgTables *t) {
    return cudaMemcpyToSymbol(c_tab, t, sizeof(DgTables));
}

void DG_FN(dg_info, DG_DIM, DG_M)(int visc, int av, int *c, int *nt, int *smem, int *fused_limiter, int *bsz) {
    if (visc && av) return info<true, true>(c, nt, smem, fused_limiter, bsz);
    if (visc) return info<true, false>(c, nt, smem, fused_limiter, bsz);
    if (av) return info<false, true>(c, nt, smem, fused_limiter, bsz);
    return info<false, false>(c, nt, smem, fused_limiter, bsz);
}

cudaError_t DG_FN(dg_config, DG_DIM, DG_M)(int visc, int av) {
    if (visc && av) return configure<true, true>();
    if (visc) return configure<true, false>();
    if (av) return configure<false, true>();
    return configure<false, false>();
}
