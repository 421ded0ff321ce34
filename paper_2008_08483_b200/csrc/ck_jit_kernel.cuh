// ck_jit_kernel.cuh -- mechanism-specialised fused source-term kernel for sm_100a.
//
// This text is compiled at ck_mech_create time by NVRTC.  The mechanism's *structure*
// (which species each reaction reads and writes, small-integer stoichiometric
// coefficients, reaction types) is generated into the function ck_reactions() at the
// marker below, so that
//   * the accumulators of Eq. 2 (wdot_k) live in registers: w[k] with
//     compile-time k, no read-modify-write traffic on shared memory;
//   * the gathers of the log-rate layers (Eq. 4) are shared-memory loads
//     with immediate offsets: ln C_k at col[k*CK_NT + tid];
//   * there is no index decoding, no loop overhead and no branch in the hot path.
// The mechanism's *numbers* (Arrhenius layer of Eq. 6, equilibrium layer of Eq. 11 folded
// onto the Gibbs features per temperature range, thermo tables, efficiencies) stay in
// tables staged in shared memory / L2, read with warp-uniform loads.
//
// Prologue macros defined by the generator (ck_jit.cu):
//   CK_S, CK_R            species, reactions
//   CK_NT                 threads (= cells) per block
//   CK_NRANGES            temperature ranges (distinct T_mid values + 1)
//   CK_NM, CK_NMB         rows of M = C E and their blocks of 8
//   CK_NFO                falloff reactions
//   CK_TAB_SMEM           1: rate tables staged in shared memory, 0: read from global
//   CK_MINB               resident blocks per SM the register budget is sized for
//
// Shared memory:  col[CK_S][CK_NT] | tab[CK_NRANGES][CK_R][10] (if CK_TAB_SMEM) | exp LUT
// Rate table row (per range r, reaction j), 10 doubles:
//   [0] ln A  [1] b  [2] -Ea/R            ln k_f = [0] + [1] ln T + [2]/T        (Eq. 6)
//   [3] r0 [4] r_lnT [5] r_invT [6..9] r_T..r_T4   ln k_r = ln k_f - ln Kc      (Eq. 7, 11)

#define CK_RU 8314.46261815324
#define CK_CFLOOR 1e-300
#define CK_ROW 10

struct CkParams {
  const double *inv_W;     // [S]
  const double *range_T;   // [NRANGES-1]
  const double *thermo;    // [S][24]  (ck_program.h)
  const double *eff;       // [NMB][S][8]
  const double *falloff;   // [NFO][8]
  const double *tab;       // [NRANGES][R][CK_ROW]
  double *m_scratch;       // [grid][NMB*8][NT]
  const double *T, *P, *Y;
  double *wdot, *dTdt;
  long long N;
};

// ---- exp(x): 32-entry table of 2^(j/32) in shared memory + degree-5 polynomial ---------
// x = (32 k + j) ln2/32 + r, |r| <= ln2/64; exp(x) = 2^k 2^(j/32) (1 + r + r^2 p(r)).
// Max relative error 3e-16 + rounding; 10 FP64-pipe instructions.
__device__ __forceinline__ double ck_exp(double x, const double *lut) {
  const double t = fma(x, 46.166241308446828, 6755399441055744.0);
  const int n = __double2loint(t);
  const double nf = t - 6755399441055744.0;
  double r = fma(nf, -0.02166084939249829, x);
  r = fma(nf, -7.2470212932696861e-19, r);
  double p = fma(0.0083333566067988717, r, 0.041666829580991785);
  p = fma(p, r, 0.16666666666632543);
  p = fma(p, r, 0.4999999999976113);
  const double e = fma(p, r * r, r);
  const double tj = lut[n & 31];
  double v = fma(tj, e, tj);
  // scale by 2^k through the exponent field; k clamped so the field stays in [1, 2046]:
  // x <= -708 gives a value <= 9e-308 (true value < 3.4e-308), x >= 709.8 gives ~1.8e308
  const int k = min(max(n >> 5, -1021), 1023);
  v = __hiloint2double(__double2hiint(v) + (k << 20), __double2loint(v));
  return v;
}

// Troe / Lindemann factor Pr/(1+Pr) F (textbook form; PAPER.md:159 gives none)
__device__ __noinline__ double ck_falloff(const double *fo, double lnT, double invT, double T,
                                          double ln_kinf, double M, const double *lut) {
  const double ln_k0 = fma(__ldg(fo + 1), lnT, fma(__ldg(fo + 2), invT, __ldg(fo)));
  const double Pr = ck_exp(ln_k0 - ln_kinf, lut) * M;
  double F = 1.0;
  if (__ldg(fo + 7) == 3.0) {
    const double alpha = __ldg(fo + 3);
    const double Fcent = (1.0 - alpha) * ck_exp(T * __ldg(fo + 4), lut) +
                         alpha * ck_exp(T * __ldg(fo + 5), lut) + ck_exp(__ldg(fo + 6) * invT, lut);
    const double lFc = log10(Fcent);
    const double c = -0.4 - 0.67 * lFc;
    const double n = 0.75 - 1.27 * lFc;
    const double lPr = log10(fmax(Pr, 1e-300));
    const double f1 = (lPr + c) / (n - 0.14 * (lPr + c));
    F = ck_exp(2.302585092994045684 * lFc / (1.0 + f1 * f1), lut);
  }
  return Pr / (1.0 + Pr) * F;
}

struct CkCtx {
  const double *col;    // ln C of this thread's cell: col[k*CK_NT]
  const double *tab;    // rate-table rows of this thread's temperature range
  const double *msc;    // M of this thread's cell: msc[slot*CK_NT]
  const double *fo;     // falloff table
  const double *lut;    // exp table
  double T, lnT, invT;
};

#define CK_LNC(k) (x.col[(k) * CK_NT])
#if CK_TAB_SMEM
#define CK_TAB(j, i) (x.tab[(j) * CK_ROW + (i)])
#else
#define CK_TAB(j, i) (__ldg(x.tab + (j) * CK_ROW + (i)))
#endif
// Arrhenius layer, Eq. 6
#define CK_LNKF(j) fma(CK_TAB(j, 1), x.lnT, fma(CK_TAB(j, 2), x.invT, CK_TAB(j, 0)))
// ln k_r = ln k_f - ln Kc on the Gibbs features, Eq. 7 + Eq. 11 folded at create time
#define CK_LNKR(j)                                                                          \
  fma(fma(fma(fma(CK_TAB(j, 9), x.T, CK_TAB(j, 8)), x.T, CK_TAB(j, 7)), x.T, CK_TAB(j, 6)), \
      x.T, fma(CK_TAB(j, 4), x.lnT, fma(CK_TAB(j, 5), x.invT, CK_TAB(j, 3))))
#define CK_EXP(v) ck_exp((v), x.lut)
#define CK_M(slot) (x.msc[(slot) * CK_NT])
#define CK_FALLOFF(idx, lnkf, M) ck_falloff(x.fo + (idx) * 8, x.lnT, x.invT, x.T, (lnkf), (M), x.lut)

//@@CK_GENERATED_REACTIONS@@
// __device__ __forceinline__ void ck_reactions(const CkCtx &x, double (&w)[CK_S]) { ... }

extern "C" __global__ void __launch_bounds__(CK_NT, CK_MINB) ck_source_terms_jit(const CkParams p) {
  extern __shared__ double smem[];
  const int tid = threadIdx.x;
  double *col = smem + tid;
  double *lut = smem + CK_S * CK_NT;
#if CK_TAB_SMEM
  double *tab = lut + 32;
  for (int i = tid; i < CK_NRANGES * CK_R * CK_ROW; i += CK_NT) tab[i] = p.tab[i];
#else
  const double *tab = p.tab;
#endif
  if (tid < 32) lut[tid] = exp2((double)tid * (1.0 / 32.0));
  __syncthreads();
  double *msc = p.m_scratch + (size_t)blockIdx.x * (CK_NMB * 8) * CK_NT + tid;

  const long long n_tiles = (p.N + CK_NT - 1) / CK_NT;
  for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const long long i = tile * CK_NT + tid;
    const bool valid = i < p.N;
    const long long ii = valid ? i : p.N - 1;

    // (a1-a3) state and temperature features
    const double T = p.T[ii], P = p.P[ii];
    const double lnT = log(T), invT = 1.0 / T;
    int range = 0;
#pragma unroll
    for (int d = 0; d < CK_NRANGES - 1; ++d) range += (T > __ldg(p.range_T + d)) ? 1 : 0;

    // (a2, a4) Y/W columns, 1/W_mix, mixture cp from NASA-7 cp/R
    double inv_Wmix = 0.0, cp_sum = 0.0;
#pragma unroll 4
    for (int k = 0; k < CK_S; ++k) {
      const double yw = p.Y[(size_t)k * p.N + ii] * __ldg(p.inv_W + k);
      col[k * CK_NT] = yw;
      inv_Wmix += yw;
      const double *th = p.thermo + k * 24;
      const double *a = th + ((T <= __ldg(th)) ? 1 : 6);
      const double cp_R = fma(fma(fma(fma(__ldg(a + 4), T, __ldg(a + 3)), T, __ldg(a + 2)), T, __ldg(a + 1)), T, __ldg(a));
      cp_sum = fma(yw, cp_R, cp_sum);
    }
    const double rho = P / (CK_RU * T * inv_Wmix);

    // (a7) third-body layer M = C E: register tile of 8 reactions
#if CK_NM > 0
    for (int b = 0; b < CK_NMB; ++b) {
      double acc[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) acc[q] = 0.0;
      const double2 *e = (const double2 *)(p.eff + (size_t)b * CK_S * 8);
#pragma unroll 2
      for (int k = 0; k < CK_S; ++k) {
        const double c = col[k * CK_NT];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const double2 ev = __ldg(e + k * 4 + q);
          acc[2 * q] = fma(ev.x, c, acc[2 * q]);
          acc[2 * q + 1] = fma(ev.y, c, acc[2 * q + 1]);
        }
      }
#pragma unroll
      for (int q = 0; q < 8; ++q) msc[(b * 8 + q) * CK_NT] = rho * acc[q];
    }
#endif

    // (a2) ln C_k with C floored at 1e-300 (input of Eq. 4)
#pragma unroll 4
    for (int k = 0; k < CK_S; ++k) col[k * CK_NT] = log(fmax(rho * col[k * CK_NT], CK_CFLOOR));

    // (a5, a6, a8-a11) the reaction layers, unrolled for this mechanism
    double w[CK_S];
#pragma unroll
    for (int k = 0; k < CK_S; ++k) w[k] = 0.0;
    CkCtx x;
    x.col = col; x.tab = tab + (size_t)range * (CK_R * CK_ROW); x.msc = msc; x.fo = p.falloff;
    x.lut = lut; x.T = T; x.lnT = lnT; x.invT = invT;
    ck_reactions(x, w);

    // (a12, a13) energy term and coalesced stores
    double hw = 0.0;
#pragma unroll
    for (int k = 0; k < CK_S; ++k) {
      const double *th = p.thermo + k * 24;
      const double *a = th + ((T <= __ldg(th)) ? 11 : 17);
      const double h_RT = fma(__ldg(a + 5), invT,
                              fma(fma(fma(fma(__ldg(a + 4), T, __ldg(a + 3)), T, __ldg(a + 2)), T, __ldg(a + 1)), T, __ldg(a)));
      hw = fma(h_RT, w[k], hw);
      if (valid) p.wdot[(size_t)k * p.N + i] = w[k];
    }
    if (valid) p.dTdt[i] = -(T * hw) / (rho * cp_sum);
  }
}
