// Launch entry points exported by the per-(dim, m) translation units (dg_stage_inst.cu) to dg_api.cu.
#pragma once

#include <cuda_runtime.h>

struct DgStageArgs;
struct DgTables;

// every entry point exists twice: without (t0) and with (t1) the passive-tracer row (-DDG_TRACER=0|1 builds)
#ifndef DG_TRACER
#define DG_TRACER 0
#endif
#define DG_FNT__(name, d, m, t) name##_##d##_##m##_t##t
#define DG_FNT_(name, d, m, t) DG_FNT__(name, d, m, t)
#define DG_FNT(name, d, m, t) DG_FNT_(name, d, m, t)
#define DG_FN(name, d, m) DG_FNT(name, d, m, DG_TRACER)

#define DG_DECLARE_T(d, m, t)                                                                              \
    cudaError_t DG_FNT(dg_launch, d, m, t)(int visc, int av, const DgStageArgs *a, cudaStream_t st,        \
                                           int wavespeed_only);                                             \
    cudaError_t DG_FNT(dg_upload, d, m, t)(const DgTables *tab);                                            \
    void DG_FNT(dg_info, d, m, t)(int visc, int av, int *c, int *nt, int *smem, int *fused_limiter, int *bsz); \
    cudaError_t DG_FNT(dg_config, d, m, t)(int visc, int av);                                               \
    cudaError_t DG_FNT(dg_limit, d, m, t)(double *w, int V, int ncells, double gamma, int *flag, cudaStream_t st);
#define DG_DECLARE(d, m) DG_DECLARE_T(d, m, 0) DG_DECLARE_T(d, m, 1)

#define DG_FOR_ALL_M(X, d) X(d, 1) X(d, 2) X(d, 3) X(d, 4) X(d, 5) X(d, 6) X(d, 7) X(d, 8)

DG_FOR_ALL_M(DG_DECLARE, 2)
DG_FOR_ALL_M(DG_DECLARE, 3)
