// rqr_tall.cuh -- internal interface between the generic tall kernels and the DMMA fast paths.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define RQR_TALL_NOT_HANDLED 12345

// Fast paths: return RQR_TALL_NOT_HANDLED when the shape is not covered, so that the generic
// kernel runs.  *nparts = number of n x n Gram partials written to `part`.
int rqr_trsm_gram_mma(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* V1,
                      int64_t ldq, double* part, int* nparts, cudaStream_t st);
int rqr_apply_mma(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                  double* Q, int64_t ldq, cudaStream_t st);
// 64 < n <= 256 (rqr_tall_panel.cu); `frags` = the workspace's panel fragment region
int rqr_trsm_gram_panel(const double* V, int64_t m, int n, int64_t ldv, const double* R0, double* V1,
                        int64_t ldq, double* part, int* nparts, double* frags, int64_t chunk_rows, cudaStream_t st);
int rqr_apply_panel(const double* V, int64_t m, int n, int64_t ldv, const double* R0, const double* R1,
                    double* Q, int64_t ldq, double* frags, cudaStream_t st);

