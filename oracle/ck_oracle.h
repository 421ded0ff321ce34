/* ck_oracle.h -- CPU oracle for the batched chemical source term.  TEST INFRASTRUCTURE.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may use anything under oracle/.  It shares no code, header or table with the CUDA
 * library (paper_2008_08483_b200/, include/ck.h) and neither includes the other.
 *
 * What it computes: the plain definition of the source term in the classic rate-law
 * (product) form, one cell and one reaction at a time, in fp64:
 *   Eq. 1-3   mechanism, species production, law of mass action
 *   Eq. 5   Arrhenius forward rate constant
 *   Eq. 7-8   reverse constant through the equilibrium constant
 *   NASA-7 h, s, cp polynomials with a cutoff temperature
 *   Sec. 2.4 third bodies, falloff, irreversible reactions
 * plus the pieces the paper implies but does not print:
 * concentrations from (T, P, Y), textbook Lindemann / Troe falloff, and the
 * constant-pressure energy equation dT/dt = -sum_k h_k wdot_k / (rho cp).
 *
 * Pins: tests/test_oracle_*.py (closed forms computed at 50 digits, conservation of
 * mass and elements, detailed balance at a constructed equilibrium, thermodynamic
 * identities by finite differences, falloff limits, and a numpy restatement of the
 * paper's matrix equations 2, 4, 6, 10, 11).  Troe's constants and the Troe blending
 * function are pinned only by the 50-digit closed form and its limits -- no external
 * code (Cantera) is available: "parity unpinned" against third-party software.
 */
#ifndef CK_ORACLE_H
#define CK_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Approximate ANN for log Kc (Eq. 12-14, Fig. 2): a drop-in replacement of
 * the exact equilibrium layer.  X_0 = standardised input features of temperature,
 * X_{l+1} = sigma(X_l W_l + B_l) for the N_L hidden layers of N_H neurons (Eq. 12), a linear
 * output layer of width R giving the standardised log Kc~, which is then de-standardised
 * (PAPER.md:141).  n_in = 1: X_0 = [ln T] (Architecture 2); n_in = 6: X_0 = the exact layer's
 * features [ln T, T, T^2, T^3, T^4, 1/T] (Architecture 1).  sigma = relu (Eq. 13) or elu
 * (Eq. 14).  Pins: tests/test_oracle_ann.py (a 50-digit worked example; a network built to
 * reproduce the exact layer; a numpy matrix restatement of Eq. 12). */
typedef struct ck_oracle_kc_ann {
  int32_t n_in, n_layers, n_hidden, activation;  /* activation: 0 relu, 1 elu */
  const double *in_mean, *in_std;  /* [n_in] */
  const double *W_in;              /* [n_in][N_H] */
  const double *B;                 /* [N_L][N_H] */
  const double *W_hid;             /* [N_L-1][N_H (from)][N_H (to)] */
  const double *W_out;             /* [N_H][R] */
  const double *B_out;             /* [R] */
  const double *out_mean, *out_std;/* [R] */
} ck_oracle_kc_ann;

typedef struct ck_oracle_mech {
  int32_t S, R;
  const double *W;          /* [S] kg/kmol */
  const double *nu_reac;    /* [S*R] nu'_kj  at k*R+j */
  const double *nu_prod;    /* [S*R] nu''_kj */
  const double *ln_A;       /* [R] */
  const double *b;          /* [R] */
  const double *Ea_over_R;  /* [R] K */
  const uint8_t *reversible;/* [R] */
  const double *nasa_lo;    /* [S*7] a1..a7, T <= T_mid */
  const double *nasa_hi;    /* [S*7] a1..a7, T >  T_mid */
  const double *T_mid;      /* [S] */
  const uint8_t *rxn_type;  /* [R] 0 elementary, 1 three-body, 2 Lindemann, 3 Troe */
  const double *eff;        /* [S*R] E_kj */
  const double *ln_A0, *b0, *Ea0_over_R; /* [R] low-pressure limit */
  const double *troe;       /* [R*4] alpha, T***, T*, T** */
  double p_ref;             /* Pa */
  const ck_oracle_kc_ann *kc_ann; /* NULL: exact Kc (Eq. 8); else Kc = exp(ANN(T)) */
} ck_oracle_mech;

/* wdot[S][N] (kmol/m^3/s) and dTdt[N] (K/s) from T[N] (K), P[N] (Pa), Y[S][N].
 * nthreads <= 0 -> all OpenMP threads.  Returns the number of threads used. */
int ck_oracle_source_terms(const ck_oracle_mech *m, const double *T, const double *P,
                           const double *Y, int64_t N, double *wdot, double *dTdt,
                           int nthreads);

/* Every intermediate of one cell, for the pins.  Y has stride ldY between species.
 * Any output pointer may be NULL.  Sizes: per-species [S], per-reaction [R]. */
void ck_oracle_cell_detail(const ck_oracle_mech *m, double T, double P, const double *Y,
                           int64_t ldY, double *rho, double *cp_mass,
                           double *C, double *cp_R, double *h_RT, double *s_R, double *g_RT,
                           double *kf, double *Kc, double *kr, double *M, double *qf,
                           double *qr, double *Q, double *wdot, double *dTdt);

/* Analytic Jacobian of (wdot, dT/dt) with respect to (Y, T) at constant P (ck_oracle_jac.c,
 * which states the formulas, the reading and the pins): J[N][S+1][S+1], cell-major; row i < S
 * is wdot_i, row S is dT/dt; column l < S is Y_l, column S is T.  Returns the number of
 * threads used, or -1 if the mechanism carries the approximate-ANN Kc (not supported). */
int ck_oracle_jacobian(const ck_oracle_mech *m, const double *T, const double *P, const double *Y,
                       int64_t N, double *J, int nthreads);

#ifdef __cplusplus
}
#endif
#endif
