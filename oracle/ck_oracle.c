/* ck_oracle.c -- plain per-cell, per-reaction CPU oracle.  TEST INFRASTRUCTURE.
 * See ck_oracle.h for scope, citations and pins.  No blocking, no fusion, no log-space
 * tricks: each step below is the definition, in the paper's order and notation.
 * Built by oracle/build.py with: gcc -O2 -fopenmp -shared -fPIC (no -ffast-math).
 */
#include "ck_oracle.h"

#include <math.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* universal gas constant, J/(kmol K): the paper's Omega is in kmol/m^3/s */
#define CK_ORACLE_RU 8314.46261815324
/* DESIGN.md reading Q9: concentrations are floored so that a missing species is a very
 * small positive concentration (the log form needs C > 0) */
#define CK_ORACLE_C_FLOOR 1e-300

/* C^nu: repeated multiplication for small non-negative integer nu, pow otherwise */
static double conc_pow(double c, double nu) {
  if (nu == 0.0) return 1.0;
  if (nu == floor(nu) && nu > 0.0 && nu <= 8.0) {
    double p = c;
    for (int i = 1; i < (int)nu; ++i) p *= c;
    return p;
  }
  return pow(c, nu);
}

/* Arrhenius expression, Eq. 5: k = A T^b exp(-E/(R T)) */
static double arrhenius(double ln_A, double b, double Ea_over_R, double T) {
  return exp(ln_A) * pow(T, b) * exp(-Ea_over_R / T);
}

/* Troe broadening factor F(T, Pr); textbook 4-parameter form (the paper prints none,
 * PAPER.md:159).  T** = +inf gives the 3-parameter form. */
static double troe_F(const double *tp, double T, double Pr) {
  const double alpha = tp[0], T3 = tp[1], T1 = tp[2], T2 = tp[3];
  double Fcent = (1.0 - alpha) * exp(-T / T3) + alpha * exp(-T / T1) + exp(-T2 / T);
  double lFc = log10(Fcent);
  double c = -0.4 - 0.67 * lFc;
  double n = 0.75 - 1.27 * lFc;
  double lPr = log10(Pr > 1e-300 ? Pr : 1e-300);
  double f1 = (lPr + c) / (n - 0.14 * (lPr + c));
  double lF = lFc / (1.0 + f1 * f1);
  return pow(10.0, lF);
}

/* Approximate ANN for log Kc, Eq. 12-14, one cell: lnKc[R] from T.
 * xa, xb: scratch of N_H doubles each. */
static double activation(int kind, double x) {
  if (kind == 0) return x > 0.0 ? x : 0.0;          /* relu, Eq. 13 */
  return x >= 0.0 ? x : exp(x) - 1.0;               /* elu, Eq. 14 */
}

static void ann_log_Kc(const ck_oracle_kc_ann *a, int R, double T, double *xa, double *xb,
                       double *lnKc) {
  const int NH = a->n_hidden;
  const double feat[6] = {log(T), T, T * T, T * T * T, T * T * T * T, 1.0 / T};
  /* X_1 = sigma(X_0 W_0 + B_0), X_0 = standardised features */
  for (int h = 0; h < NH; ++h) {
    double z = a->B[h];
    for (int i = 0; i < a->n_in; ++i)
      z += ((feat[i] - a->in_mean[i]) / a->in_std[i]) * a->W_in[i * NH + h];
    xa[h] = activation(a->activation, z);
  }
  /* X_{l+1} = sigma(X_l W_l + B_l), l = 1 .. N_L - 1 */
  for (int l = 1; l < a->n_layers; ++l) {
    const double *W = a->W_hid + (size_t)(l - 1) * NH * NH;
    for (int h = 0; h < NH; ++h) {
      double z = a->B[l * NH + h];
      for (int g = 0; g < NH; ++g) z += xa[g] * W[g * NH + h];
      xb[h] = activation(a->activation, z);
    }
    for (int h = 0; h < NH; ++h) xa[h] = xb[h];
  }
  /* linear output layer, then de-standardisation */
  for (int j = 0; j < R; ++j) {
    double y = a->B_out[j];
    for (int h = 0; h < NH; ++h) y += xa[h] * a->W_out[h * R + j];
    lnKc[j] = y * a->out_std[j] + a->out_mean[j];
  }
}

/* workspace: per-species and per-reaction scratch for one cell */
typedef struct {
  double *C, *cp_R, *h_RT, *s_R, *g_RT, *Y;      /* [S] */
  double *kf, *Kc, *kr, *M, *qf, *qr, *Q, *wdot; /* [R], wdot [S] */
  double *ann_lnKc, *ann_x;                      /* [R], [2 N_H] (approximate ANN only) */
} cell_ws;

static void one_cell(const ck_oracle_mech *m, double T, double P, const double *Y,
                     int64_t ldY, cell_ws *w, double *rho_out, double *cp_out,
                     double *dTdt_out) {
  const int S = m->S, R = m->R;
  const double Ru = CK_ORACLE_RU;

  /* 1. concentrations: 1/W_mix = sum Y_k/W_k, rho = P W_mix/(Ru T),
   *    C_k = rho Y_k / W_k.  Reading Q9: a mass fraction <= 0 is an absent species (Y_k = 0)
   *    everywhere it enters -- W_mix, C, cp -- and C is then floored for the rate law. */
  double inv_Wmix = 0.0;
  for (int k = 0; k < S; ++k) {
    w->Y[k] = Y[k * ldY] > 0.0 ? Y[k * ldY] : 0.0;
    inv_Wmix += w->Y[k] / m->W[k];
  }
  double rho = P / (Ru * T * inv_Wmix);
  for (int k = 0; k < S; ++k) {
    double c = rho * w->Y[k] / m->W[k];
    w->C[k] = c > CK_ORACLE_C_FLOOR ? c : CK_ORACLE_C_FLOOR;
  }

  /* 2. NASA-7 thermodynamics; low range for T <= T_mid */
  const double T2 = T * T, T3 = T2 * T, T4 = T3 * T, lnT = log(T);
  for (int k = 0; k < S; ++k) {
    const double *a = (T <= m->T_mid[k]) ? m->nasa_lo + 7 * k : m->nasa_hi + 7 * k;
    w->cp_R[k] = a[0] + a[1] * T + a[2] * T2 + a[3] * T3 + a[4] * T4;
    w->h_RT[k] = a[0] + a[1] * T / 2 + a[2] * T2 / 3 + a[3] * T3 / 4 + a[4] * T4 / 5 + a[5] / T;
    w->s_R[k] = a[0] * lnT + a[1] * T + a[2] * T2 / 2 + a[3] * T3 / 3 + a[4] * T4 / 4 + a[6];
    w->g_RT[k] = w->h_RT[k] - w->s_R[k];  /* G = H - S, Eq. 10 */
  }

  for (int k = 0; k < S; ++k) w->wdot[k] = 0.0;

  /* 2b. approximate ANN in place of the exact equilibrium layer */
  if (m->kc_ann)
    ann_log_Kc(m->kc_ann, R, T, w->ann_x, w->ann_x + m->kc_ann->n_hidden, w->ann_lnKc);

  for (int j = 0; j < R; ++j) {
    /* 3. forward constant, Eq. 5; equilibrium constant, Eq. 8:
     *    Kc = (p_ref/(Ru T))^(sum_k nu_kj) exp(-sum_k nu_kj g_k/RT)  */
    double kf = arrhenius(m->ln_A[j], m->b[j], m->Ea_over_R[j], T);
    double dnu_sum = 0.0, dG = 0.0;
    for (int k = 0; k < S; ++k) {
      double nu = m->nu_prod[k * R + j] - m->nu_reac[k * R + j];
      dnu_sum += nu;
      dG += nu * w->g_RT[k];
    }
    double Kc = exp(-dG) * pow(m->p_ref / (Ru * T), dnu_sum);
    if (m->kc_ann) Kc = exp(w->ann_lnKc[j]);

    /* 4. third bodies and falloff */
    const int type = m->rxn_type ? m->rxn_type[j] : 0;
    double phi = 1.0, Mj = 1.0;
    if (type != 0) {
      Mj = 0.0;
      for (int k = 0; k < S; ++k) Mj += (m->eff ? m->eff[k * R + j] : 1.0) * w->C[k];
    }
    if (type == 1) {
      phi = Mj;
    } else if (type == 2 || type == 3) {
      double k_inf = kf;
      double k_0 = arrhenius(m->ln_A0[j], m->b0[j], m->Ea0_over_R[j], T);
      double Pr = k_0 * Mj / k_inf;
      double F = (type == 3) ? troe_F(m->troe + 4 * j, T, Pr) : 1.0;
      kf = k_inf * (Pr / (1.0 + Pr)) * F;
    }

    /* 5. reverse constant, Eq. 7; irreversible -> 0 */
    const int rev = m->reversible ? m->reversible[j] : 1;
    double kr = rev ? kf / Kc : 0.0;

    /* 6. law of mass action, Eq. 3 */
    double qf = kf, qr = kr;
    for (int k = 0; k < S; ++k) {
      if (m->nu_reac[k * R + j] != 0.0) qf *= conc_pow(w->C[k], m->nu_reac[k * R + j]);
      if (m->nu_prod[k * R + j] != 0.0) qr *= conc_pow(w->C[k], m->nu_prod[k * R + j]);
    }
    double Q = phi * (qf - qr);

    /* 7. species production, Eq. 2 */
    for (int k = 0; k < S; ++k)
      w->wdot[k] += (m->nu_prod[k * R + j] - m->nu_reac[k * R + j]) * Q;

    w->kf[j] = kf; w->Kc[j] = Kc; w->kr[j] = kr; w->M[j] = Mj;
    w->qf[j] = qf; w->qr[j] = qr; w->Q[j] = Q;
  }

  /* 8. constant-pressure energy equation: cp = sum Y_k (cp_k/R) Ru/W_k  [J/kg/K],
   *    dT/dt = - sum_k h_k wdot_k / (rho cp),  h_k = (h_k/RT) Ru T  [J/kmol] */
  double cp = 0.0, hw = 0.0;
  for (int k = 0; k < S; ++k) {
    cp += w->Y[k] * w->cp_R[k] * Ru / m->W[k];
    hw += w->h_RT[k] * Ru * T * w->wdot[k];
  }
  *rho_out = rho;
  *cp_out = cp;
  *dTdt_out = -hw / (rho * cp);
}

static int ws_alloc(cell_ws *w, int S, int R, int NH) {
  double *p = (double *)malloc(sizeof(double) * (size_t)(7 * S + 8 * R + 2 * NH));
  if (!p) return -1;
  w->C = p; w->cp_R = p + S; w->h_RT = p + 2 * S; w->s_R = p + 3 * S; w->g_RT = p + 4 * S;
  w->wdot = p + 5 * S; w->Y = p + 6 * S;
  double *q = p + 7 * S;
  w->kf = q; w->Kc = q + R; w->kr = q + 2 * R; w->M = q + 3 * R; w->qf = q + 4 * R;
  w->qr = q + 5 * R; w->Q = q + 6 * R; w->ann_lnKc = q + 7 * R; w->ann_x = q + 8 * R;
  return 0;
}

int ck_oracle_source_terms(const ck_oracle_mech *m, const double *T, const double *P,
                           const double *Y, int64_t N, double *wdot, double *dTdt,
                           int nthreads) {
  const int S = m->S, R = m->R;
  int used = 1;
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
  used = nthreads;
#pragma omp parallel num_threads(nthreads)
#endif
  {
    cell_ws w;
    if (ws_alloc(&w, S, R, m->kc_ann ? m->kc_ann->n_hidden : 0) == 0) {
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
      for (int64_t i = 0; i < N; ++i) {
        double rho, cp, dT;
        one_cell(m, T[i], P[i], Y + i, N, &w, &rho, &cp, &dT);
        for (int k = 0; k < S; ++k) wdot[(int64_t)k * N + i] = w.wdot[k];
        dTdt[i] = dT;
      }
      free(w.C);
    }
  }
  return used;
}

static void copy_out(double *dst, const double *src, int n) {
  if (dst) for (int i = 0; i < n; ++i) dst[i] = src[i];
}

void ck_oracle_cell_detail(const ck_oracle_mech *m, double T, double P, const double *Y,
                           int64_t ldY, double *rho, double *cp_mass,
                           double *C, double *cp_R, double *h_RT, double *s_R, double *g_RT,
                           double *kf, double *Kc, double *kr, double *M, double *qf,
                           double *qr, double *Q, double *wdot, double *dTdt) {
  cell_ws w;
  if (ws_alloc(&w, m->S, m->R, m->kc_ann ? m->kc_ann->n_hidden : 0) != 0) return;
  double r, c, d;
  one_cell(m, T, P, Y, ldY, &w, &r, &c, &d);
  if (rho) *rho = r;
  if (cp_mass) *cp_mass = c;
  if (dTdt) *dTdt = d;
  copy_out(C, w.C, m->S); copy_out(cp_R, w.cp_R, m->S); copy_out(h_RT, w.h_RT, m->S);
  copy_out(s_R, w.s_R, m->S); copy_out(g_RT, w.g_RT, m->S); copy_out(wdot, w.wdot, m->S);
  copy_out(kf, w.kf, m->R); copy_out(Kc, w.Kc, m->R); copy_out(kr, w.kr, m->R);
  copy_out(M, w.M, m->R); copy_out(qf, w.qf, m->R); copy_out(qr, w.qr, m->R);
  copy_out(Q, w.Q, m->R);
  free(w.C);
}
