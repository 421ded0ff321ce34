// ck_peaks.cu -- FP64 peak microbenchmarks: the measured rates the
// roofline of this FP64-pipe-bound path is divided by, and the facts the sparse-vs-dense design
// decision rests on:
//   * DFMA issue rate of the whole chip (register-resident chains on every SM);
//   * DMMA.8x8x4 rate (PTX mma.sync.m8n8k4.f64, the only FP64 tensor instruction of sm_100a) --
//     in DFMA equivalents (one DMMA = 256 FMA = 8 warp-wide DFMA);
//   * DMMA and DFMA interleaved in one instruction stream: do they share the pipe?
//   * CUDA libm exp() and log() rates: the 15 / 28 instruction costs of the survey's accounting.
// Each kernel is timed alone with CUDA events on the caller's stream, best of 5 after a warm-up.
#include <cuda_runtime.h>

#include "ck_internal.h"

namespace ck {

namespace {

constexpr int kThreads = 1024, kIters = 4096;

// 8 independent register chains per thread, 64 DFMA per trip
__global__ void __launch_bounds__(kThreads) peak_dfma(double *out, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int u = 0; u < 8; ++u) x[u] = threadIdx.x + u;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int u = 0; u < 8; ++u) x[u] = fma(x[u], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int u = 0; u < 8; ++u) s += x[u];
  if (s == 123.456) out[0] = s;   // never true for the arguments used; keeps the loop alive
}

__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// 8 independent DMMA accumulator pairs per warp; NF independent DFMA per DMMA in the same stream
// (NF = 0: DMMA alone).  8 DMMA (+ 8 NF DFMA) per trip.
template <int NF>
__global__ void __launch_bounds__(kThreads) peak_dmma(double *out, int iters, double a, double b) {
  double c0[8], c1[8], x[NF > 0 ? NF : 1];
#pragma unroll
  for (int u = 0; u < 8; ++u) { c0[u] = threadIdx.x + u; c1[u] = u; }
#pragma unroll
  for (int f = 0; f < (NF > 0 ? NF : 1); ++f) x[f] = threadIdx.x + f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      dmma(c0[u], c1[u], a, b);
#pragma unroll
      for (int f = 0; f < NF; ++f) x[f] = fma(x[f], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int u = 0; u < 8; ++u) s += c0[u] + c1[u];
#pragma unroll
  for (int f = 0; f < NF; ++f) s += x[f];
  if (s == 123.456) out[0] = s;
}

// libm exp / log: 4 independent chains per thread, arguments kept in a fixed range by an fma
template <bool LOG>
__global__ void __launch_bounds__(kThreads) peak_libm(double *out, int iters, double a, double b) {
  double x[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) x[u] = 1.0 + 0.001 * (threadIdx.x + u);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 4; ++u) x[u] = LOG ? fma(log(x[u]), a, b) : fma(exp(x[u]), a, b);
  }
  const double s = (x[0] + x[1]) + (x[2] + x[3]);
  if (s == 123.456) out[0] = s;
}

// legacy tensor-core paths (mma.sync): int8 m16n8k32 and fp16 m16n8k16 with fp32 accumulation, 8
// independent accumulator sets per warp.  What an error-free splitting of M = C E onto the
// low-precision tensor cores would run on (rejected, measured here).
template <bool INT8>
__global__ void __launch_bounds__(kThreads) peak_mma_legacy(double *out, int iters) {
  unsigned a[4] = {threadIdx.x, threadIdx.x * 3u, 7u, 9u}, b[2] = {threadIdx.x * 5u, 11u};
  int ci[8][4];
  float cf[8][4];
#pragma unroll
  for (int u = 0; u < 8; ++u)
#pragma unroll
    for (int v = 0; v < 4; ++v) { ci[u][v] = u + v; cf[u][v] = (float)(u + v); }
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      if (INT8)
        asm volatile("mma.sync.aligned.m16n8k32.row.col.s32.s8.s8.s32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                     : "+r"(ci[u][0]), "+r"(ci[u][1]), "+r"(ci[u][2]), "+r"(ci[u][3])
                     : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
      else
        asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                     : "+f"(cf[u][0]), "+f"(cf[u][1]), "+f"(cf[u][2]), "+f"(cf[u][3])
                     : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
    }
  }
  double s = 0.0;
#pragma unroll
  for (int u = 0; u < 8; ++u)
#pragma unroll
    for (int v = 0; v < 4; ++v) s += INT8 ? (double)ci[u][v] : (double)cf[u][v];
  if (s == 123.456) out[0] = s;
}

template <typename F>
cudaError_t best_ms(F launch, cudaStream_t stream, double *ms_out) {
  cudaEvent_t t0, t1;
  cudaError_t e = cudaEventCreate(&t0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&t1);
  if (e != cudaSuccess) { cudaEventDestroy(t0); return e; }
  launch(64);   // warm-up
  double best = 1e30;
  for (int rep = 0; rep < 5 && e == cudaSuccess; ++rep) {
    cudaEventRecord(t0, stream);
    launch(kIters);
    cudaEventRecord(t1, stream);
    e = cudaEventSynchronize(t1);
    float ms = 0;
    if (e == cudaSuccess) cudaEventElapsedTime(&ms, t0, t1);
    if (e == cudaSuccess && ms < best) best = ms;
  }
  cudaEventDestroy(t0);
  cudaEventDestroy(t1);
  if (e == cudaSuccess) e = cudaGetLastError();
  *ms_out = best;
  return e;
}

}  // namespace

cudaError_t measure_peaks(double out[CK_N_PEAKS], cudaStream_t stream) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  double *d_out = nullptr;
  e = cudaMalloc((void **)&d_out, sizeof(double));
  if (e != cudaSuccess) return e;
  const int blocks = sms * 2;
  const double threads = (double)blocks * kThreads, warps = threads / 32.0;
  double ms = 0;
  for (int i = 0; i < CK_N_PEAKS; ++i) out[i] = 0.0;
  // [0] DFMA, thread-level instructions per second
  e = best_ms([&](int it) { peak_dfma<<<blocks, kThreads, 0, stream>>>(d_out, it, 0.999999, 1e-7); }, stream, &ms);
  if (e == cudaSuccess) out[0] = threads * kIters * 64.0 / (ms * 1e-3);
  // [1] DMMA.8x8x4 alone, warp-level instructions per second
  if (e == cudaSuccess)
    e = best_ms([&](int it) { peak_dmma<0><<<blocks, kThreads, 0, stream>>>(d_out, it, 0.999999, 1e-7); }, stream, &ms);
  if (e == cudaSuccess) out[1] = warps * kIters * 8.0 / (ms * 1e-3);
  // [2], [3] one DMMA + 4 DFMA interleaved: DMMA warp-instructions/s and DFMA thread-instructions/s
  if (e == cudaSuccess)
    e = best_ms([&](int it) { peak_dmma<4><<<blocks, kThreads, 0, stream>>>(d_out, it, 0.999999, 1e-7); }, stream, &ms);
  if (e == cudaSuccess) {
    out[2] = warps * kIters * 8.0 / (ms * 1e-3);
    out[3] = threads * kIters * 32.0 / (ms * 1e-3);
  }
  // [4], [5] CUDA libm exp() and log(), calls per second (thread level)
  if (e == cudaSuccess)
    e = best_ms([&](int it) { peak_libm<false><<<blocks, kThreads, 0, stream>>>(d_out, it, 1e-3, 1.0); }, stream, &ms);
  if (e == cudaSuccess) out[4] = threads * kIters * 4.0 / (ms * 1e-3);
  if (e == cudaSuccess)
    e = best_ms([&](int it) { peak_libm<true><<<blocks, kThreads, 0, stream>>>(d_out, it, 1e-3, 1.5); }, stream, &ms);
  if (e == cudaSuccess) out[5] = threads * kIters * 4.0 / (ms * 1e-3);
  out[6] = (double)sms;
  // [7], [8] legacy mma.sync: int8 m16n8k32 and fp16 m16n8k16, warp-level instructions per second
  if (e == cudaSuccess)
    e = best_ms([&](int it) { peak_mma_legacy<true><<<blocks, kThreads, 0, stream>>>(d_out, it); }, stream, &ms);
  if (e == cudaSuccess) out[7] = warps * kIters * 8.0 / (ms * 1e-3);
  if (e == cudaSuccess)
    e = best_ms([&](int it) { peak_mma_legacy<false><<<blocks, kThreads, 0, stream>>>(d_out, it); }, stream, &ms);
  if (e == cudaSuccess) out[8] = warps * kIters * 8.0 / (ms * 1e-3);
  cudaFree(d_out);
  return e;
}

cudaError_t measure_fp64_peak(double *fma_per_s, cudaStream_t stream) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e != cudaSuccess) return e;
  double *d_out = nullptr;
  e = cudaMalloc((void **)&d_out, sizeof(double));
  if (e != cudaSuccess) return e;
  const int blocks = sms * 2;
  double ms = 0;
  e = best_ms([&](int it) { peak_dfma<<<blocks, kThreads, 0, stream>>>(d_out, it, 0.999999, 1e-7); }, stream, &ms);
  cudaFree(d_out);
  if (e != cudaSuccess) return e;
  *fma_per_s = (double)blocks * kThreads * (double)kIters * 64.0 / (ms * 1e-3);
  return cudaSuccess;
}

}  // namespace ck
