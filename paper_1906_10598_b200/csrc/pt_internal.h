// pt_internal.h -- declarations shared by the translation units of libpt.so (not part of the public ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/pt.h"
#include "pt_device.cuh"

namespace pt {

// pt_doppler.cu
int doppler_launch(const double* best, long long B, int D, double T, double los_scale, const int32_t* m, int n_intervals,
                   double* per_block, double* total_phase, double* const* interval_out, cudaStream_t st);

// pt_acquire.cu
int acquire_launch(const float* x, long long B, int N, double fs, int D, const pt_acq_config* a, double* est, double* lo,
                   double* hi, cudaStream_t st);

// pt_retry.cu
int retry_flag_launch(const double* per_block, long long B, double phi_tol, double F_tol_hz, uint32_t* flags, cudaStream_t st);
int retry_box_launch(const uint32_t* flags, const double* best, double* lo, double* hi, long long B, int D, double T, double g,
                     const pt_retry_config* rc, cudaStream_t st);
int retry_compact_launch(const uint32_t* flags, long long B, uint32_t* list, int* count, cudaStream_t st);
int retry_count_launch(const uint32_t* sel, const int* n, long long B, int32_t* attempts, cudaStream_t st);
int retry_abandon_launch(const uint32_t* flags, long long B, uint32_t* status, cudaStream_t st);

// pt_api.cu
void set_error(const char* fmt, ...);
int check_cuda(cudaError_t e, const char* what);

}  // namespace pt
