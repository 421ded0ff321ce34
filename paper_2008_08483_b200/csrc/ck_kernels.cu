// ck_kernels.cu -- fused source-term kernel for sm_100a (thread per cell).
//
// One launch evaluates every layer of the paper's ANN form (include/ck.h (1)-(6)) for a
// tile of `threads` cells per block; nothing of size N x R or N x S other than the
// inputs and outputs touches HBM.  Per block, shared memory holds two column arrays
//   col[S][threads]  Y_k/W_k, later ln C_k      (input of the log-rate layers, Eq. 4)
//   wd [S][threads]  accumulators of Eq. 2
// so that thread t only ever touches column t: no bank conflicts (consecutive threads,
// consecutive 8-byte words) and no synchronisation.  Global loads/stores of the SoA
// state are coalesced (thread t <-> cell base + t).  The mechanism is read
// through warp-uniform (broadcast) loads of the reaction program (ck_program.h).
#include <cuda_runtime.h>

#include <cstdint>

#include "ck_internal.h"

namespace ck {

namespace {

__device__ __forceinline__ double ldu(const double *p) { return __ldg(p); }

// Troe / Lindemann factor  Pr/(1+Pr) * F  (textbook form; the paper gives none)
__device__ __noinline__ double falloff_factor(const double *fo, double lnT, double invT, double T,
                                              double ln_kinf, double M) {
  const double ln_k0 = fma(ldu(fo + 1), lnT, fma(ldu(fo + 2), invT, ldu(fo + 0)));
  const double Pr = exp(ln_k0 - ln_kinf) * M;
  double F = 1.0;
  if (ldu(fo + 7) == 3.0) {
    const double alpha = ldu(fo + 3);
    const double Fcent = (1.0 - alpha) * exp(T * ldu(fo + 4)) + alpha * exp(T * ldu(fo + 5)) +
                         exp(ldu(fo + 6) * invT);
    const double lFc = log10(Fcent);
    const double c = -0.4 - 0.67 * lFc;
    const double n = 0.75 - 1.27 * lFc;
    const double lPr = log10(fmax(Pr, 1e-300));
    const double f1 = (lPr + c) / (n - 0.14 * (lPr + c));
    F = exp(2.302585092994045684 * lFc / (1.0 + f1 * f1));
  }
  return Pr / (1.0 + Pr) * F;
}

__global__ void __launch_bounds__(128)
source_terms_kernel(const DeviceMech m, const double *__restrict__ Tg, const double *__restrict__ Pg,
                    const double *__restrict__ Yg, const int64_t N, double *__restrict__ wdot,
                    double *__restrict__ dTdt) {
  extern __shared__ double smem[];
  const int S = m.S;
  const int nt = blockDim.x;
  const int tid = threadIdx.x;
  double *col = smem + tid;              // col[k*nt]
  double *wd = smem + (size_t)S * nt + tid;
  // a free slot of the M scratch for this block's lifetime (ck_program.h)
  __shared__ int s_slot;
  if (tid == 0) {
    int s = blockIdx.x % m.n_slots;
    while (atomicCAS(m.slot_busy + s, 0, 1) != 0) s = (s + 1 == m.n_slots) ? 0 : s + 1;
    __threadfence();   // acquire: the last owner's stores are ordered before this block's
    s_slot = s;
  }
  __syncthreads();
  double *msc = m.m_scratch + (size_t)s_slot * m.n_m_blocks * kMBlock * nt + tid;

  const int64_t n_tiles = (N + nt - 1) / nt;
  for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int64_t i = tile * nt + tid;
    const bool valid = i < N;
    const int64_t ii = valid ? i : N - 1;   // idle lanes recompute the last cell, store nothing

    // ---- (a1-a3) state, temperature features ------------------------------------------
    const double T = Tg[ii], P = Pg[ii];
    const double lnT = log(T), invT = 1.0 / T;
    int range = 0;
    for (int d = 0; d < m.n_ranges - 1; ++d) range += (T > ldu(m.range_T + d)) ? 1 : 0;

    // ---- (a2, a4) Y/W columns, 1/W_mix, cp of the mixture (NASA-7 cp/R) ---
    double inv_Wmix = 0.0, cp_sum = 0.0;
    for (int k = 0; k < S; ++k) {
      // (a mass fraction <= 0 is an absent species: reading Q9)
      const double yw = fmax(Yg[(size_t)k * N + ii], 0.0) * ldu(m.inv_W + k);
      col[(size_t)k * nt] = yw;
      inv_Wmix += yw;
      const double *th = m.thermo + (size_t)k * kThermoStride;
      const double *a = th + ((T <= ldu(th)) ? 1 : 6);
      const double cp_R = fma(fma(fma(fma(ldu(a + 4), T, ldu(a + 3)), T, ldu(a + 2)), T, ldu(a + 1)), T, ldu(a));
      cp_sum = fma(yw, cp_R, cp_sum);
    }
    const double rho = P / (kRu * T * inv_Wmix);

    // ---- (a7) third-body layer M = C E, register tile of kMBlock reactions --------------
    for (int b = 0; b < m.n_m_blocks; ++b) {
      double acc[kMBlock];
#pragma unroll
      for (int q = 0; q < kMBlock; ++q) acc[q] = 0.0;
      const double *e = m.eff + (size_t)b * S * kMBlock;
      for (int k = 0; k < S; ++k) {
        const double c = col[(size_t)k * nt];
#pragma unroll
        for (int q = 0; q < kMBlock; ++q) acc[q] = fma(ldu(e + k * kMBlock + q), c, acc[q]);
      }
#pragma unroll
      for (int q = 0; q < kMBlock; ++q) msc[(size_t)(b * kMBlock + q) * nt] = rho * acc[q];
    }

    // ---- (a2) ln C_k, C floored at 1e-300 (Eq. 4 takes log C) --------------------------
    for (int k = 0; k < S; ++k) {
      const double c = fmax(rho * col[(size_t)k * nt], kCFloor);
      col[(size_t)k * nt] = log(c);
      wd[(size_t)k * nt] = 0.0;
    }

    // ---- (a5, a6, a8-a11) reaction program ------------------------------------------------
    const unsigned char *rec = m.program;
    for (int j = 0; j < m.R; ++j) {
      const int4 h0 = __ldg((const int4 *)rec);        // size, nr, np, nsc
      const int4 h1 = __ldg((const int4 *)rec + 1);    // type, reversible, m_slot, fo_idx
      const double *fwd = (const double *)(rec + sizeof(RecHeader));
      const double *rev = fwd + 4 + 8 * range;
      const double *coef = fwd + 4 + 8 * m.n_ranges;
      const int ncoef = h0.y + h0.z + h0.w;
      const int *offs = (const int *)(coef + ((ncoef + 1) & ~1));

      // Arrhenius layer (Eq. 6) and the folded equilibrium layer (Eq. 7, 10, 11)
      const double ln_kf = fma(ldu(fwd + 1), lnT, fma(ldu(fwd + 2), invT, ldu(fwd)));
      double ln_qf = ln_kf;
      for (int e = 0; e < h0.y; ++e)
        ln_qf = fma(ldu(coef + e), col[(size_t)__ldg(offs + e) * nt], ln_qf);
      double qr = 0.0;
      if (h1.y) {
        const double poly = fma(fma(fma(ldu(rev + 5), T, ldu(rev + 4)), T, ldu(rev + 3)), T, ldu(rev + 2));
        double ln_qr = fma(poly, T, fma(ldu(rev + 1), lnT, fma(ldu(rev + 6), invT, ldu(rev))));
        for (int e = 0; e < h0.z; ++e)
          ln_qr = fma(ldu(coef + h0.y + e), col[(size_t)__ldg(offs + h0.y + e) * nt], ln_qr);
        qr = exp(ln_qr);                               // exp "activation", Eq. 4
      }
      const double qf = exp(ln_qf);
      double phi = 1.0;
      if (h1.x != 0) {
        const double M = msc[(size_t)h1.z * nt];
        phi = (h1.x == 1) ? M
                          : falloff_factor(m.falloff + (size_t)h1.w * kFalloffStride, lnT, invT, T, ln_kf, M);
      }
      const double Q = phi * (qf - qr);
      // net-rate contraction (Eq. 2), scatter form
      const double *cs = coef + h0.y + h0.z;
      const int *os = offs + h0.y + h0.z;
      for (int e = 0; e < h0.w; ++e) {
        double *w = wd + (size_t)__ldg(os + e) * nt;
        *w = fma(ldu(cs + e), Q, *w);
      }
      rec += h0.x;
    }

    // ---- (a12, a13) energy term and stores --------------------------------------------------
    double hw = 0.0;
    for (int k = 0; k < S; ++k) {
      const double w = wd[(size_t)k * nt];
      const double *th = m.thermo + (size_t)k * kThermoStride;
      const double *a = th + ((T <= ldu(th)) ? 11 : 17);
      const double h_RT = fma(ldu(a + 5), invT,
                              fma(fma(fma(fma(ldu(a + 4), T, ldu(a + 3)), T, ldu(a + 2)), T, ldu(a + 1)), T, ldu(a)));
      hw = fma(h_RT, w, hw);
      if (valid) wdot[(size_t)k * N + i] = w;
    }
    // dT/dt = -sum_k h_k wdot_k / (rho cp), h_k = (h/RT) Ru T, cp = Ru sum_k (Y_k/W_k) cp_k/R
    if (valid) dTdt[i] = -(T * hw) / (rho * cp_sum);
  }
  __syncthreads();
  if (tid == 0) {
    __threadfence();   // release: the block's accesses to the slot end before the flag clears
    atomicExch(m.slot_busy + s_slot, 0);
  }
}

}  // namespace

cudaError_t kernel_configure(int threads, size_t smem_bytes, int *blocks_per_sm) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  int optin = 0;
  e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (e != cudaSuccess) return e;
  cudaFuncAttributes attr;
  e = cudaFuncGetAttributes(&attr, source_terms_kernel);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(source_terms_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           optin - (int)attr.sharedSizeBytes);
  if (e != cudaSuccess) return e;
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, source_terms_kernel, threads,
                                                       smem_bytes);
}

cudaError_t launch_source_terms(const ck_mech *m, const double *T, const double *P,
                                const double *Y, int64_t N, double *wdot, double *dTdt,
                                cudaStream_t stream) {
  const int nt = m->dev.threads;
  const int64_t n_tiles = (N + nt - 1) / nt;
  const int grid = (int)(n_tiles < m->grid_max ? n_tiles : m->grid_max);
  source_terms_kernel<<<grid, nt, m->smem_bytes, stream>>>(m->dev, T, P, Y, N, wdot, dTdt);
  return cudaGetLastError();
}

}  // namespace ck
