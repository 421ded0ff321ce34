/* ck_oracle_jac.c -- CPU oracle for the analytic Jacobian of the source term.  TEST
 * INFRASTRUCTURE (see ck_oracle.h for who may use oracle/).
 *
 * What it computes, per cell, in fp64 with plain dense loops (no sparsity, no log-space
 * tricks): the derivative of the function ck_oracle_source_terms evaluates,
 *     f(Y_1..Y_S, T; P) = (wdot_1 .. wdot_S, dT/dt),
 * with respect to (Y_1..Y_S, T) at constant pressure, the Y_l taken as S independent
 * variables (no sum-to-one constraint: the source term is defined for any Y >= 0 and is
 * homogeneous of degree 0 in Y).  This is the "analytic Jacobian" the paper names as the
 * prerequisite of a GPU stiff integrator.
 * The paper prints no Jacobian formulas; every line below is the chain rule applied to the
 * equations the source-term oracle implements, cited where each is differentiated:
 *   Eq. 3  Q_j = phi_j (k_f prod C^nu' - k_r prod C^nu'')
 *       dQ/dC_l |_T = phi (nu'_lj q_f - nu''_lj q_r)/C_l + (dQ/dM) E_lj
 *   Eq. 5  d ln k/dT = (b + (Ea/R)/T)/T
 *   Eq. 8  d ln Kc/dT = sum_k dnu_kj (h_k/RT)/T - (sum_k dnu_kj)/T
 *       (Gibbs-Helmholtz d(g/RT)/dT = -(h/RT)/T for the NASA-7 polynomials)
 *   falloff (textbook Lindemann / Troe, reading Q8):
 *       k = k_inf Gamma(Pr, T), Gamma = Pr/(1+Pr) F, Pr = k_0 M/k_inf
 *       d ln Gamma/d ln Pr = 1/(1+Pr) + d ln F/d ln Pr,   d ln Gamma/dT |_Pr = d ln F/dT |_Pr
 *   Eq. 2  d wdot_k = sum_j dnu_kj dQ_j
 *   PAPER.md:56          C_k = rho Y_k/W_k, rho = P/(Ru T sum_j Y_j/W_j):
 *       dC_k/dY_l = delta_kl rho/W_k - C_k/(W_l sum_j Y_j/W_j),   dC_k/dT = -C_k/T
 *   energy equation (north_star (6)): dT/dt = -sum_k H_k wdot_k / D,
 *       H_k = (h_k/RT) Ru T [J/kmol], dH_k/dT = Cp_k = (cp_k/R) Ru, D = rho cp = sum_k C_k Cp_k.
 * Reading (Q18): the floor on C (Q9), the clamp on Pr (Q8) and the switch of the
 * NASA-7 range at T_mid are not differentiated: the Jacobian is that of the smooth branch
 * the state lies on; states with a floored concentration are outside its contract.
 * The approximate-ANN Kc (kc_ann) is not supported here.
 *
 * Layout: J[N][S+1][S+1], cell-major, row-major per cell; row i < S is wdot_i, row S is
 * dT/dt; column l < S is Y_l, column S is T.
 *
 * Pins (tests/test_oracle_jacobian.py): central finite differences of
 * ck_oracle_source_terms (itself pinned); 50-digit derivatives of the single-reaction closed
 * forms (tests/golden/jacobian_closed_form.json, written by make_jacobian_closed_form.py
 * with mpmath differentiation, elementary / three-body / Lindemann / Troe); Euler's theorem
 * sum_l Y_l J_il = 0; mass and element conservation of every column.
 */
#include <math.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#include "ck_oracle.h"

#define JAC_RU 8314.46261815324
#define JAC_LN10 2.302585092994045684

static double conc_pow_j(double c, double nu) {
  if (nu == 0.0) return 1.0;
  if (nu == floor(nu) && nu > 0.0 && nu <= 8.0) {
    double p = c;
    for (int i = 1; i < (int)nu; ++i) p *= c;
    return p;
  }
  return pow(c, nu);
}

/* One cell.  ws: scratch of 8 S + S S doubles, laid out below. */
static void jac_one_cell(const ck_oracle_mech *m, double T, double P, const double *Y, int64_t ldY,
                         double *ws, double *J) {
  const int S = m->S, R = m->R, n = S + 1;
  const double Ru = JAC_RU;
  double *C = ws, *cpR = C + S, *hRT = cpR + S, *gRT = hRT + S, *dcpR = gRT + S, *wdot = dcpR + S;
  double *JT = wdot + S;          /* [S]   d wdot_i / dT at constant C */
  double *dQdC = JT + S;          /* [S]   dQ_j/dC_l of the reaction in hand */
  double *JC = dQdC + S;          /* [S][S] d wdot_i / dC_l at constant T */

  /* concentrations */
  double s = 0.0;
  for (int k = 0; k < S; ++k) s += Y[k * ldY] / m->W[k];
  const double rho = P / (Ru * T * s);
  for (int k = 0; k < S; ++k) C[k] = rho * Y[k * ldY] / m->W[k];

  /* NASA-7 and the T-derivative of cp/R */
  const double T2 = T * T, T3 = T2 * T, T4 = T3 * T, lnT = log(T);
  for (int k = 0; k < S; ++k) {
    const double *a = (T <= m->T_mid[k]) ? m->nasa_lo + 7 * k : m->nasa_hi + 7 * k;
    cpR[k] = a[0] + a[1] * T + a[2] * T2 + a[3] * T3 + a[4] * T4;
    dcpR[k] = a[1] + 2 * a[2] * T + 3 * a[3] * T2 + 4 * a[4] * T3;
    hRT[k] = a[0] + a[1] * T / 2 + a[2] * T2 / 3 + a[3] * T3 / 4 + a[4] * T4 / 5 + a[5] / T;
    const double sR = a[0] * lnT + a[1] * T + a[2] * T2 / 2 + a[3] * T3 / 3 + a[4] * T4 / 4 + a[6];
    gRT[k] = hRT[k] - sR;
  }

  for (int i = 0; i < S; ++i) { wdot[i] = 0.0; JT[i] = 0.0; }
  for (int i = 0; i < S * S; ++i) JC[i] = 0.0;

  for (int j = 0; j < R; ++j) {
    /* rate constants and their logarithmic T-derivatives (Eq. 5, Eq. 8) */
    double kf = exp(m->ln_A[j]) * pow(T, m->b[j]) * exp(-m->Ea_over_R[j] / T);
    double dlnkf = (m->b[j] + m->Ea_over_R[j] / T) / T;
    double dnu_sum = 0.0, dG = 0.0, dH = 0.0;
    for (int k = 0; k < S; ++k) {
      const double nu = m->nu_prod[k * R + j] - m->nu_reac[k * R + j];
      dnu_sum += nu;
      dG += nu * gRT[k];
      dH += nu * hRT[k];
    }
    const double Kc = exp(-dG) * pow(m->p_ref / (Ru * T), dnu_sum);
    const double dlnKc = dH / T - dnu_sum / T;

    const int type = m->rxn_type ? m->rxn_type[j] : 0;
    double Mj = 1.0;
    if (type != 0) {
      Mj = 0.0;
      for (int k = 0; k < S; ++k) Mj += (m->eff ? m->eff[k * R + j] : 1.0) * C[k];
    }
    double phi = 1.0;          /* multiplies both directions (three-body) */
    double dlnG_dlnPr = 0.0;   /* falloff: d ln Gamma / d ln Pr */
    if (type == 1) phi = Mj;
    if (type == 2 || type == 3) {
      const double k0 = exp(m->ln_A0[j]) * pow(T, m->b0[j]) * exp(-m->Ea0_over_R[j] / T);
      const double dlnk0 = (m->b0[j] + m->Ea0_over_R[j] / T) / T;
      const double Pr = k0 * Mj / kf;
      double F = 1.0, dlnF_dlnPr = 0.0, dlnF_dT = 0.0;
      if (type == 3) {
        const double *tp = m->troe + 4 * j;
        const double alpha = tp[0], T3s = tp[1], T1s = tp[2], T2s = tp[3];
        const double e3 = exp(-T / T3s), e1 = exp(-T / T1s), e2 = exp(-T2s / T);
        const double Fcent = (1.0 - alpha) * e3 + alpha * e1 + e2;
        /* exp(-inf) = 0 and 0 * inf would be NaN: T** = +inf gives the 3-parameter form */
        const double dFcent = -(1.0 - alpha) / T3s * e3 - alpha / T1s * e1 + (isinf(T2s) ? 0.0 : T2s / T2 * e2);
        const double lFc = log10(Fcent), dlFc = dFcent / (Fcent * JAC_LN10);
        const double c = -0.4 - 0.67 * lFc, nn = 0.75 - 1.27 * lFc;
        const double lPr = log10(Pr);
        const double A = lPr + c, B = nn - 0.14 * A;
        const double f1 = A / B, den = 1.0 + f1 * f1;
        F = pow(10.0, lFc / den);
        /* log10 F = lFc / (1 + f1^2) */
        const double df1_dlPr = nn / (B * B);                 /* (B + 0.14 A)/B^2 */
        const double dA_dlFc = -0.67, dB_dlFc = -1.27 - 0.14 * (-0.67);
        const double df1_dlFc = (dA_dlFc * B - A * dB_dlFc) / (B * B);
        const double dlF_df1 = -lFc * 2.0 * f1 / (den * den);
        dlnF_dlnPr = dlF_df1 * df1_dlPr;                      /* d log10 F / d log10 Pr */
        dlnF_dT = JAC_LN10 * dlFc * (1.0 / den + dlF_df1 * df1_dlFc);
      }
      dlnG_dlnPr = 1.0 / (1.0 + Pr) + dlnF_dlnPr;
      /* effective forward constant and its T-derivative at constant C (Pr varies with T) */
      dlnkf = dlnkf + dlnG_dlnPr * (dlnk0 - dlnkf) + dlnF_dT;
      kf = kf * (Pr / (1.0 + Pr)) * F;
    }

    const int rev = m->reversible ? m->reversible[j] : 1;
    double qf = kf, qr = rev ? kf / Kc : 0.0;
    for (int k = 0; k < S; ++k) {
      qf *= conc_pow_j(C[k], m->nu_reac[k * R + j]);
      qr *= conc_pow_j(C[k], m->nu_prod[k * R + j]);
    }
    const double Q = phi * (qf - qr);
    /* dQ/dT at constant C: k_r = k_f/Kc */
    const double dQdT = phi * (qf * dlnkf - qr * (dlnkf - dlnKc));
    /* dQ/dC_l at constant T (Eq. 3 differentiated; third body / falloff through M) */
    for (int l = 0; l < S; ++l) {
      double d = 0.0;
      if (m->nu_reac[l * R + j] != 0.0) d += phi * m->nu_reac[l * R + j] * qf / C[l];
      if (m->nu_prod[l * R + j] != 0.0) d -= phi * m->nu_prod[l * R + j] * qr / C[l];
      const double E = (m->eff ? m->eff[l * R + j] : 1.0);
      if (type == 1) d += E * (qf - qr);
      if (type == 2 || type == 3) d += E * (qf - qr) * dlnG_dlnPr / Mj;
      dQdC[l] = d;
    }
    /* Eq. 2 */
    for (int i = 0; i < S; ++i) {
      const double nu = m->nu_prod[i * R + j] - m->nu_reac[i * R + j];
      if (nu == 0.0) continue;
      wdot[i] += nu * Q;
      JT[i] += nu * dQdT;
      for (int l = 0; l < S; ++l) JC[i * S + l] += nu * dQdC[l];
    }
  }

  /* chain rule to (Y, T) at constant P: dC_k/dY_l = delta_kl rho/W_k - C_k/(s W_l), dC_k/dT = -C_k/T */
  for (int i = 0; i < S; ++i) {
    double g = 0.0;
    for (int k = 0; k < S; ++k) g += JC[i * S + k] * C[k];
    for (int l = 0; l < S; ++l) J[i * n + l] = JC[i * S + l] * rho / m->W[l] - g / (s * m->W[l]);
    J[i * n + S] = JT[i] - g / T;
  }

  /* energy row: dT/dt = -sum_k H_k wdot_k / D */
  double D = 0.0, dD_dT = 0.0, hw = 0.0, cpw = 0.0;
  for (int k = 0; k < S; ++k) {
    D += C[k] * cpR[k] * Ru;
    dD_dT += C[k] * dcpR[k] * Ru;
    hw += hRT[k] * Ru * T * wdot[k];
    cpw += cpR[k] * Ru * wdot[k];
  }
  dD_dT -= D / T;
  const double Tdot = -hw / D;
  for (int l = 0; l < S; ++l) {
    double hj = 0.0;
    for (int k = 0; k < S; ++k) hj += hRT[k] * Ru * T * J[k * n + l];
    const double dD_dYl = rho * cpR[l] * Ru / m->W[l] - D / (s * m->W[l]);
    J[S * n + l] = -hj / D - Tdot * dD_dYl / D;
  }
  {
    double hj = 0.0;
    for (int k = 0; k < S; ++k) hj += hRT[k] * Ru * T * J[k * n + S];
    J[S * n + S] = -(cpw + hj) / D - Tdot * dD_dT / D;
  }
}

int ck_oracle_jacobian(const ck_oracle_mech *m, const double *T, const double *P, const double *Y,
                       int64_t N, double *J, int nthreads) {
  if (m->kc_ann) return -1;
  const int S = m->S;
  const size_t nws = (size_t)8 * S + (size_t)S * S;
  int used = 1;
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
  used = nthreads;
#pragma omp parallel num_threads(nthreads)
#endif
  {
    double *ws = (double *)malloc(sizeof(double) * nws);
    if (ws) {
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
      for (int64_t i = 0; i < N; ++i)
        jac_one_cell(m, T[i], P[i], Y + i, N, ws, J + (size_t)i * (S + 1) * (S + 1));
      free(ws);
    }
  }
  return used;
}
