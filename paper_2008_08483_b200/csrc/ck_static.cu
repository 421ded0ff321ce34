// ck_static.cu -- ck_source_terms_static (include/ck.h): the source terms for callers that must not
// allocate device memory.
//
// Who that is.  A flow solver typically gives the whole device to its own memory pool once its fields
// are set up, so a cudaMalloc from inside the time loop fails, or takes memory the pool was sized
// without.  cudaMalloc and cudaFree also synchronise the device, which stalls every other stream of a
// solver that overlaps chemistry with transport.  And code that runs under a fixed device-memory
// budget (several ranks or jobs sharing one GPU) wants a library whose footprint does not grow with
// the first call on a new shape.  Every other entry point of this library keeps its scratch in
// cudaMalloc'ed memory owned by the handle; this one keeps it in the library image itself.
//
// What it is.  The table-driven source-term kernel of ck_kernels.cu (one thread per cell, the
// mechanism read from the handle's reaction program) with one difference: the third-body
// concentrations M = C E of a block's cells, the only global memory that kernel uses
// besides its inputs and outputs, live in the file-scope array g_m_static below, not in a scratch area
// of the handle.  The array is 32 MiB; every GPU on which this library's code is loaded holds that
// much until the process exits, whether or not this entry point is ever called.
//
// Sharing.  There is ONE array per GPU, shared by every handle and every call.  It is cut by block
// index (block b of a launch owns the b-th region), not by the busy flags ck_source_terms uses, so two
// calls that are on the GPU at the same time (different streams, or different host threads) write the
// same regions and corrupt each other: order them on one stream.  The array keeps the last call's
// values; nothing in it has to start at zero, because a block writes every M row of a tile before it
// reads any, so there is nothing to clear between calls.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>
#include <string>

#include "ck_internal.h"

namespace ck {

namespace {

constexpr int kStaticMaxRows = CK_STATIC_MAX_M_ROWS;   // rows of M a mechanism may have (ck.h)
constexpr int kStaticThreads = 128;                    // most threads (= cells) of a block
constexpr int kStaticMinBlocks = 64;                   // blocks a launch has at the row limit
constexpr size_t kStaticDoubles = (size_t)kStaticMaxRows * kStaticThreads * kStaticMinBlocks;   // 32 MiB

// The scratch itself.  In HOST code this name is only a handle for the runtime's symbol calls, not a
// device address: static_setup() below asks the runtime for the address, per device, and the kernel
// receives it as an argument.
static __device__ __align__(256) double g_m_static[kStaticDoubles];

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

// Same layers in the same order as source_terms_kernel of ck_kernels.cu (include/ck.h (1)-(6)); `m_all`
// is the device address of g_m_static, of which this block owns rows x blockDim.x doubles at its index.
__global__ void __launch_bounds__(kStaticThreads)
source_terms_static_kernel(const DeviceMech m, double *__restrict__ m_all, const double *__restrict__ Tg,
                           const double *__restrict__ Pg, const double *__restrict__ Yg, const int64_t N,
                           double *__restrict__ wdot, double *__restrict__ dTdt) {
  extern __shared__ double smem[];
  const int S = m.S;
  const int nt = blockDim.x;
  const int tid = threadIdx.x;
  double *col = smem + tid;                       // col[k*nt]: Y_k/W_k, later ln C_k
  double *wd = smem + (size_t)S * nt + tid;       // wd[k*nt]: accumulators of Eq. 2
  const int rows = (m.n_m_blocks > 0 ? m.n_m_blocks : 1) * kMBlock;
  double *msc = m_all + (size_t)blockIdx.x * rows * nt + tid;

  const int64_t n_tiles = (N + nt - 1) / nt;
  for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const int64_t i = tile * nt + tid;
    const bool valid = i < N;
    const int64_t ii = valid ? i : N - 1;   // idle lanes recompute the last cell, store nothing

    // ---- state, temperature features ----------------------------------------------------
    const double T = Tg[ii], P = Pg[ii];
    const double lnT = log(T), invT = 1.0 / T;
    int range = 0;
    for (int d = 0; d < m.n_ranges - 1; ++d) range += (T > ldu(m.range_T + d)) ? 1 : 0;

    // ---- Y/W columns, 1/W_mix, cp of the mixture (NASA-7 cp/R) --------------
    double inv_Wmix = 0.0, cp_sum = 0.0;
    for (int k = 0; k < S; ++k) {
      // (a mass fraction <= 0 is an absent species: DESIGN.md reading Q9)
      const double yw = fmax(Yg[(size_t)k * N + ii], 0.0) * ldu(m.inv_W + k);
      col[(size_t)k * nt] = yw;
      inv_Wmix += yw;
      const double *th = m.thermo + (size_t)k * kThermoStride;
      const double *a = th + ((T <= ldu(th)) ? 1 : 6);
      const double cp_R = fma(fma(fma(fma(ldu(a + 4), T, ldu(a + 3)), T, ldu(a + 2)), T, ldu(a + 1)), T, ldu(a));
      cp_sum = fma(yw, cp_R, cp_sum);
    }
    const double rho = P / (kRu * T * inv_Wmix);

    // ---- third-body layer M = C E into this block's region of the static array ------------
    // (every row the reaction walk reads is written here first: nothing of an earlier tile or
    //  an earlier call is ever read)
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

    // ---- ln C_k, C floored at 1e-300 (Eq. 4 takes log C) ------------------------------------
    for (int k = 0; k < S; ++k) {
      const double c = fmax(rho * col[(size_t)k * nt], kCFloor);
      col[(size_t)k * nt] = log(c);
      wd[(size_t)k * nt] = 0.0;
    }

    // ---- reaction program: Arrhenius, equilibrium, third body / falloff, exp, net rate ------
    const unsigned char *rec = m.program;
    for (int j = 0; j < m.R; ++j) {
      const int4 h0 = __ldg((const int4 *)rec);        // size, nr, np, nsc
      const int4 h1 = __ldg((const int4 *)rec + 1);    // type, reversible, m_slot, fo_idx
      const double *fwd = (const double *)(rec + sizeof(RecHeader));
      const double *rev = fwd + 4 + 8 * range;
      const double *coef = fwd + 4 + 8 * m.n_ranges;
      const int ncoef = h0.y + h0.z + h0.w;
      const int *offs = (const int *)(coef + ((ncoef + 1) & ~1));

      const double ln_kf = fma(ldu(fwd + 1), lnT, fma(ldu(fwd + 2), invT, ldu(fwd)));   // Eq. 6
      double ln_qf = ln_kf;
      for (int e = 0; e < h0.y; ++e)
        ln_qf = fma(ldu(coef + e), col[(size_t)__ldg(offs + e) * nt], ln_qf);
      double qr = 0.0;
      if (h1.y) {                                                                       // Eq. 7, 10, 11
        const double poly = fma(fma(fma(ldu(rev + 5), T, ldu(rev + 4)), T, ldu(rev + 3)), T, ldu(rev + 2));
        double ln_qr = fma(poly, T, fma(ldu(rev + 1), lnT, fma(ldu(rev + 6), invT, ldu(rev))));
        for (int e = 0; e < h0.z; ++e)
          ln_qr = fma(ldu(coef + h0.y + e), col[(size_t)__ldg(offs + h0.y + e) * nt], ln_qr);
        qr = exp(ln_qr);                                                                // Eq. 4
      }
      const double qf = exp(ln_qf);
      double phi = 1.0;
      if (h1.x != 0) {
        const double M = msc[(size_t)h1.z * nt];
        phi = (h1.x == 1) ? M
                          : falloff_factor(m.falloff + (size_t)h1.w * kFalloffStride, lnT, invT, T, ln_kf, M);
      }
      const double Q = phi * (qf - qr);
      const double *cs = coef + h0.y + h0.z;                                            // Eq. 2, scatter form
      const int *os = offs + h0.y + h0.z;
      for (int e = 0; e < h0.w; ++e) {
        double *w = wd + (size_t)__ldg(os + e) * nt;
        *w = fma(ldu(cs + e), Q, *w);
      }
      rec += h0.x;
    }

    // ---- energy term and stores -----------------------------------------------------------------
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
    if (valid) dTdt[i] = -(T * hw) / (rho * cp_sum);
  }
}

// Per-device set-up, done once, by the first call that finds that device current: the device address
// of g_m_static on it, and the kernel's shared-memory limit.  Neither allocates; both may load this
// file's code onto the device, which is why the first call belongs before any stream capture.
constexpr int kMaxDevices = 64;
struct StaticSetup {
  std::once_flag once;
  cudaError_t err = cudaSuccess;
  const char *what = "";
  double *scratch = nullptr;
};
StaticSetup g_setup[kMaxDevices];

void static_setup(StaticSetup *s, int dev) {
  double *p = nullptr;
  s->err = cudaGetSymbolAddress((void **)&p, g_m_static);
  s->what = "cudaGetSymbolAddress(g_m_static)";
  if (s->err != cudaSuccess) return;
  int optin = 0;
  s->err = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  s->what = "cudaDeviceGetAttribute";
  if (s->err != cudaSuccess) return;
  cudaFuncAttributes attr;
  s->err = cudaFuncGetAttributes(&attr, source_terms_static_kernel);
  s->what = "cudaFuncGetAttributes";
  if (s->err != cudaSuccess) return;
  s->err = cudaFuncSetAttribute(source_terms_static_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                optin - (int)attr.sharedSizeBytes);
  s->what = "cudaFuncSetAttribute";
  if (s->err != cudaSuccess) return;
  s->scratch = p;
}

}  // namespace

// The launch behind ck_source_terms_static (pointers and N already checked by the caller).  Returns a
// ck_status and, for a non-zero one, the message in *err.  Calls no cudaMalloc, cudaFree or any
// library routine that allocates device memory.
int static_source_terms(const ck_mech *m, const double *T, const double *P, const double *Y, int64_t N,
                        double *wdot, double *dTdt, cudaStream_t stream, std::string *err) {
  if (m->jit_spec.kc_ann || m->jit_spec.prec != CK_PREC_F64 || m->jit_spec.kc_none) {
    *err = "ck_source_terms_static: the handle uses the approximate-ANN Kc, a reduced precision or an ablation; "
           "only the specialised kernel of ck_source_terms implements those";
    return CK_EUNSUPPORTED;
  }
  const int nt = m->dev.threads;
  const int rows = (m->dev.n_m_blocks > 0 ? m->dev.n_m_blocks : 1) * kMBlock;
  if (m->dev.n_m > kStaticMaxRows || rows > kStaticMaxRows || nt > kStaticThreads) {
    *err = "ck_source_terms_static: the mechanism has " + std::to_string(m->dev.n_m) +
           " third-body and falloff reactions; the static scratch holds at most " +
           std::to_string(kStaticMaxRows) + " (CK_STATIC_MAX_M_ROWS). Use ck_source_terms for this mechanism";
    return CK_EUNSUPPORTED;
  }
  int dev = -1;
  cudaError_t ce = cudaGetDevice(&dev);
  if (ce != cudaSuccess) { *err = std::string("cudaGetDevice: ") + cudaGetErrorString(ce); return CK_ECUDA; }
  if (dev != m->device || dev < 0 || dev >= kMaxDevices) {
    *err = "ck_source_terms_static: the current device (" + std::to_string(dev) + ") is not the one the handle was "
           "created on (" + std::to_string(m->device) + ")";
    return CK_EINVAL;
  }
  StaticSetup *s = &g_setup[dev];
  std::call_once(s->once, static_setup, s, dev);
  if (s->err != cudaSuccess) {
    *err = std::string("ck_source_terms_static set-up, ") + s->what + ": " + cudaGetErrorString(s->err);
    return CK_ECUDA;
  }
  const int64_t n_tiles = (N + nt - 1) / nt;
  const int64_t fit = (int64_t)(kStaticDoubles / ((size_t)rows * nt));   // >= kStaticMinBlocks
  int64_t grid = n_tiles < m->grid_max ? n_tiles : m->grid_max;
  if (grid > fit) grid = fit;
  source_terms_static_kernel<<<(unsigned)grid, nt, m->smem_bytes, stream>>>(m->dev, s->scratch, T, P, Y, N, wdot, dTdt);
  ce = cudaGetLastError();
  if (ce != cudaSuccess) { *err = std::string("ck_source_terms_static launch: ") + cudaGetErrorString(ce); return CK_ECUDA; }
  return CK_OK;
}

}  // namespace ck
