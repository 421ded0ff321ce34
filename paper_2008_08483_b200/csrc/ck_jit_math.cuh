// ck_jit_math.cuh -- device math shared by the NVRTC-compiled kernels (pasted into their text at
// build time): exp and ln by table + polynomial, reciprocal by Newton steps, the falloff factor.
// Needs CK_LUT_REP (copies of the exp table), CK_KCONST (coefficients as constant-bank operands or
// literals) and CK_PREC (0 fp64, >= 1 exp mantissa from the fp32 special-function unit).
// falloff table row fo[8]: [0] ln A0 [1] b0 [2] -Ea0/R [3] alpha [4] -1/T*** [5] -1/T* [6] -T**
// [7] kind (2.0 Lindemann, 3.0 Troe)

// Polynomial coefficients live in the constant bank: DFMA reads them as c[bank][imm]
// operands, whereas literals would be rebuilt in (uniform) registers after every branch.
__constant__ double ck_k_exp[8] = {184.6649652337873, 6755399441055744.0, -0.0054152123481245725,
                                   0.0, 0.0, 0.04166668092164609,
                                   0.16666672012284, 0.49999999999996736};
__constant__ double ck_k_fo[12] = {-690.7755278982137, 709.0, -700.0, 1e-300, 0.43429448190325182765, -0.67,
                                   -0.4, -1.27, 0.75, -0.14, 1.0, 0.0};
__constant__ double ck_k_log[8] = {-0.16666666666666666, 0.2, -0.25, 0.33333333333333331, -0.5,
                                   0.693147180369123816490, 1.90821492927058770002e-10, -1.0};

#if CK_KCONST
#define CK_KE(i) ck_k_exp[i]
#define CK_KL(i) ck_k_log[i]
#define CK_KF(i) ck_k_fo[i]
#else
#define CK_KE_0 184.6649652337873
#define CK_KE_1 6755399441055744.0
#define CK_KE_2 -0.0054152123481245725
#define CK_KE_5 0.04166668092164609
#define CK_KE_6 0.16666672012284
#define CK_KE_7 0.49999999999996736
#define CK_KL_0 -0.16666666666666666
#define CK_KL_1 0.2
#define CK_KL_2 -0.25
#define CK_KL_3 0.33333333333333331
#define CK_KL_4 -0.5
#define CK_KL_5 0.693147180369123816490
#define CK_KL_6 1.90821492927058770002e-10
#define CK_KL_7 -1.0
#define CK_KF_0 -690.7755278982137
#define CK_KF_1 709.0
#define CK_KF_2 -700.0
#define CK_KF_3 1e-300
#define CK_KF_4 0.43429448190325182765
#define CK_KF_5 -0.67
#define CK_KF_6 -0.4
#define CK_KF_7 -1.27
#define CK_KF_8 0.75
#define CK_KF_9 -0.14
#define CK_KF_10 1.0
#define CK_KF_11 0.0
#define CK_KE(i) CK_KE_##i
#define CK_KL(i) CK_KL_##i
#define CK_KF(i) CK_KF_##i
#endif

#if CK_PREC >= 1
// ---- exp(x), REDUCED PRECISION (ck_mech_desc.precision = CK_PREC_MIXED; "single or
// half-precision environments"): the exponent is handled in fp64 / integer arithmetic, the mantissa
// 2^f goes through the fp32 special-function unit.
//   tm = x log2(e) + 1.5 2^32 (one fma): the mantissa field of tm then holds round(t 2^20), t = x log2 e;
//   n = floor(t) = that integer >> 20, f = its low 20 bits / 2^20 in [0, 1);
//   2^(1 + f) = MUFU.EX2 of the float 1 + f, whose bits are 0x3f800000 | f << 3 (no conversion);
//   the result 2^(n - 1) 2^(1 + f) is assembled from the float's bits and n (no conversion either).
// ONE FP64-pipe instruction instead of eight.  Relative error <= 2^-21 ln 2 (quantisation of t)
// + 2^-22 (ex2.approx) ~ 6e-7.  Exponent clamped as in the fp64 version.
__device__ __forceinline__ double ck_exp(double x, const double *) {
  const double tm = fma(x, 1.4426950408889634074, 6442450944.0);
  const int lo = __double2loint(tm), hi = __double2hiint(tm) - 0x41f80000;
  const int n = min(max((int)__funnelshift_r((unsigned)lo, (unsigned)hi, 20), -1021), 1022);
  float m;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(m) : "f"(__int_as_float(0x3f800000 | ((lo & 0xfffff) << 3))));
  const unsigned fb = (unsigned)__float_as_int(m);
  return __hiloint2double((int)(fb >> 3) + ((895 + n) << 20), (int)(fb << 29));
}
#else
// ---- exp(x): 128-entry table of 2^(j/128) in shared memory + degree-4 polynomial -------
// x = (128 k + j) ln2/128 + r, |r| <= ln2/256; exp(x) = 2^k 2^(j/128) (1 + r + r^2 p(r)).
// Polynomial error 1.6e-16 relative; the reduction is a single fma with fl(ln2/128), whose
// rounding (6e-19 per step of the table) puts |x| 4e-18 relative error into the result: 4e-16
// at |x| = 100, under the rounding error the argument already carries.
// 8 FP64-pipe instructions.
__device__ __forceinline__ double ck_exp(double x, const double *lut) {
  const double t = fma(x, CK_KE(0), CK_KE(1));
  const int n = __double2loint(t);
  const double nf = t - CK_KE(1);
  const double r = fma(nf, CK_KE(2), x);
  double p = fma(CK_KE(5), r, CK_KE(6));
  p = fma(p, r, CK_KE(7));
  const double e = fma(p, r * r, r);
  // 2^k 2^(j/128): add k to the exponent field of the table entry; k is clamped so the field
  // stays valid: x <= -708 gives a value <= 9e-308 (true value < 3.4e-308), x >= 709.8 ~1.8e308
  const double tj = lut[(n & 127) * CK_LUT_REP];
  const int k = min(max(n >> 7, -1021), 1023);
  const double ts = __hiloint2double(__double2hiint(tj) + (k << 20), __double2loint(tj));
  return fma(ts, e, ts);
}

#endif

#if CK_PREC == 2
// ---- exp(x) of an fp32 argument, returned as fp64 (CK_PREC_F32_RATES): t = x log2 e in fp32,
// n = round(t) by the 1.5 2^23 shifter, 2^(t - n) from MUFU.EX2, the fp64 result assembled from the
// float's bits and n (rates reach e^250: an fp32 result would overflow).  No FP64-pipe instruction.
__device__ __forceinline__ double ck_exp_f32(float x) {
  const float t = x * 1.44269504f;
  const float tm = t + 12582912.0f;
  const int n = min(max(__float_as_int(tm) - 0x4b400000, -1021), 1022);
  float m;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(m) : "f"(t - (tm - 12582912.0f)));
  const unsigned fb = (unsigned)__float_as_int(m);
  return __hiloint2double((int)(fb >> 3) + ((896 + n) << 20), (int)(fb << 29));
}
#endif

// ---- ln(x) for positive normal x: 128-entry table + degree-6 polynomial -----------------
// x = 2^k m, m in [0.70703125, 1.4140625); the top 7 bits of m's position in that range
// pick c_i (no interval straddles 1.0); r = m/c_i - 1 by one fma with the tabulated 1/c_i,
// |r| < 0.0040;  ln x = k ln2 + ln c_i + (r - r^2/2 + ... - r^6/6).
// Absolute error < 3e-16; 11 FP64-pipe instructions and one int->double
// conversion.  x = 0 and denormals give a finite value near -709, never NaN.
__device__ __forceinline__ double ck_log(double x, const double *logtab) {
  const int hi = __double2hiint(x);
  const int t = hi - 0x3fe6a000;
  const double m = __hiloint2double(hi - (t & 0xfff00000), __double2loint(x));
  const double2 c = *(const double2 *)((const char *)logtab + ((t >> 9) & 0x7f0));   // 16 B per entry
  const double r = fma(m, c.x, CK_KL(7));
  double q = fma(CK_KL(0), r, CK_KL(1));
  q = fma(q, r, CK_KL(2));
  q = fma(q, r, CK_KL(3));
  q = fma(q, r, CK_KL(4));
  const double kd = (double)(t >> 20);
  const double p = fma(r * r, q, r);
  return fma(kd, CK_KL(5), c.y) + fma(kd, CK_KL(6), p);
}

// 1/d to about 1 ulp: MUFU.RCP64H seed and two Newton steps (4 FP64-pipe instructions);
// for finite normal d whose reciprocal is normal.
__device__ __forceinline__ double ck_rcp(double d) {
  double x;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
  double e = fma(-d, x, CK_KF(10));
  x = fma(x, e, x);
  e = fma(-d, x, CK_KF(10));
  return fma(x, e, x);
}

// Falloff factor Pr/(1+Pr) F, Lindemann (F = 1) or Troe (textbook form; PAPER.md:159
// gives none), evaluated in logarithms:
//   ln Pr = ln k0 - ln k_inf + ln M, clamped to [ln 1e-300, 709];  Pr/(1+Pr) = 1/(1 + e^(-ln Pr))
//   log10 F = log10 Fcent / (1 + f1^2), f1 = a/b, a = log10 Pr + c, b = n - 0.14 a
//   => F = exp(ln Fcent  b^2 / (a^2 + b^2))
template <bool TROE>
__device__ __forceinline__ double ck_falloff(const double *fo, double lnT, double invT, double T,
                                          double ln_kinf, double M, const double *lut,
                                          const double *logtab) {
  const double ln_k0 = fma(fo[1], lnT, fma(fo[2], invT, fo[0]));
  double lnPr = (ln_k0 - ln_kinf) + ck_log(M, logtab);
  lnPr = fmin(fmax(lnPr, CK_KF(0)), CK_KF(1));
  double phi = ck_rcp(CK_KF(10) + ck_exp(-lnPr, lut));
  if (TROE) {
    // Straight-line code for every reaction of a block (the host puts the Troe reactions of a
    // group first; a Lindemann reaction that shares a block with them takes F = 1 by select),
    // so that the evaluations of a block interleave instead of running one after the other.
    const double alpha = fo[3];
    const double Fcent = (CK_KF(10) - alpha) * ck_exp(fmax(T * fo[4], CK_KF(2)), lut) +
                         alpha * ck_exp(fmax(T * fo[5], CK_KF(2)), lut) +
                         ck_exp(fmax(fo[6] * invT, CK_KF(2)), lut);
    const double L = ck_log(fmax(Fcent, CK_KF(3)), logtab);
    const double lFc = L * CK_KF(4);
    const double c = fma(CK_KF(5), lFc, CK_KF(6));
    const double n = fma(CK_KF(7), lFc, CK_KF(8));
    const double a = fma(lnPr, CK_KF(4), c);
    const double b = fma(CK_KF(9), a, n);
    const double b2 = b * b;
    const double F = ck_exp(L * (b2 * ck_rcp(fma(a, a, b2))), lut);
    phi *= (fo[7] == 3.0) ? F : CK_KF(10);
  }
  return phi;
}

