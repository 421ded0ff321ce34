// ck_internal.h -- host-side handle and the launch interface between ck_api.cu
// (validation, mechanism build, C ABI) and ck_kernels.cu (device code).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "ck_program.h"

struct ck_mech {
  ck::DeviceMech dev{};       // device pointers + sizes, passed to the kernel by value
  int device = 0;
  int blocks_per_sm = 1;
  int num_sms = 1;
  int grid_max = 1;           // persistent grid size = num_sms * blocks_per_sm
  size_t smem_bytes = 0;      // dynamic shared memory per block
  // statistics for ck_mech_info
  int64_t nnz_reac = 0, nnz_prod = 0, nnz_net = 0, nnz_eff = 0;
  int n_three_body = 0, n_lindemann = 0, n_troe = 0;
  // one device allocation holding every table; m_scratch separately
  void *d_tables = nullptr;
  double *d_scratch = nullptr;
  // staging for ck_source_terms_host
  double *d_stage = nullptr;
  int64_t stage_cells = 0;
};

namespace ck {

// Sets the kernel's shared-memory attribute and reports occupancy. Returns cudaError_t.
cudaError_t kernel_configure(int threads, size_t smem_bytes, int *blocks_per_sm);

// Launches the fused source-term kernel on `stream` (asynchronous).
cudaError_t launch_source_terms(const ck_mech *m, const double *T, const double *P,
                                const double *Y, int64_t N, double *wdot, double *dTdt,
                                cudaStream_t stream);

// DFMA throughput microbenchmark (thread-level FMA instructions per second).
cudaError_t measure_fp64_peak(double *fma_per_s, cudaStream_t stream);

}  // namespace ck
