// Launch entry points exported by the per-(dim, m) translation units (dg_stage_inst.cu) to dg_api.cu.
#pragma once

#include <cuda_runtime.h>

struct DgStageArgs;
struct DgTables;

#define DG_FN_(name, d, m) name##_##d##_##m
#define DG_FN(name, d, m) DG_FN_(name, d, m)

#define DG_DECLARE(d, m)                                                                               \
    cudaError_t DG_FN(dg_launch, d, m)(int visc, int av, const DgStageArgs *a, cudaStream_t st,       \
                                       int wavespeed_only);                                            \
    cudaError_t DG_FN(dg_upload, d, m)(const DgTables *t);                                             \
    void DG_FN(dg_info, d, m)(int visc, int av, int *c, int *nt, int *smem, int *fused_limiter, int *bsz);                           \
    cudaError_t DG_FN(dg_config, d, m)(int visc, int av);                                              \
    cudaError_t DG_FN(dg_limit, d, m)(double *w, int V, int ncells, double gamma, int *flag, cudaStream_t st);

#define DG_FOR_ALL_M(X, d) X(d, 1) X(d, 2) X(d, 3) X(d, 4) X(d, 5) X(d, 6) X(d, 7) X(d, 8)

DG_FOR_ALL_M(DG_DECLARE, 2)
DG_FOR_ALL_M(DG_DECLARE, 3)
