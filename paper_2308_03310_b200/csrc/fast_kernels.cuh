// fast_kernels.cuh -- register-resident path for M <= 64 (stub: not enabled yet).
#pragma once
#include "common.cuh"
namespace letkf {
static inline bool fast_supported(int) { return false; }
static inline int fast_tridiag_launch(const double*, double*, Workspace, int, int, cudaStream_t) { return -1; }
static inline int fast_apply_launch(double*, Workspace, int, int, cudaStream_t) { return -1; }
static inline int fast_analysis_chunk(const double*, const double*, const double*, const double*, int, int, int,
                                      int, double, double*, double*, double*, int*, Workspace, double*, double*,
                                      double*, cudaStream_t, int*) { return -1; }
}
