// ck_rk4.cu -- the 0-D constant-pressure reactor use of the source term (
// BASELINE.json configs[4]): classic explicit RK4 on y = (T, Y_1..Y_S) of N independent
// cells, ck_source_terms called once per stage.
//
//   dT/dt   = ck_source_terms' energy term,   dY_k/dt = wdot_k W_k / rho,
//   rho     = P / (Ru T sum_k Y_k / W_k),      P constant per cell.
//
// Every state handed to ck_source_terms -- the three intermediate stage states and the
// result of the step -- is first projected onto valid thermochemical states (DESIGN.md
// reading Q14): Y <- max(Y, 0), Y <- Y / sum(Y), T <- min(max(T, 250 K), 5000 K), and the
// slope of a stage is the right-hand side evaluated AT that projected state.
//
// One "stage" kernel per RK stage does everything that is not the source term: the slope
// from (wdot, dT/dt), the running weighted sum of slopes, the next stage state (or the new
// state after stage 4) and its projection.  Thread <-> cell, species rows walked with
// coalesced accesses; a step is 4 x (ck_source_terms + stage kernel), captured once into
// a CUDA graph and replayed n_steps times.
#include <cuda_runtime.h>

#include <cstdint>
#include <string>

#include "../../include/ck.h"
#include "ck_internal.h"

namespace ck {

namespace {

constexpr double kTmin = 250.0, kTmax = 5000.0;

// STAGE 1..4.  a = coefficient of the NEXT stage state (1/2, 1/2, 1; unused for stage 4),
// b = weight of this stage's slope in the step (1/6, 1/3, 1/3, 1/6).
//   in : T0, Y0 (state at the start of the step), Ts, Ys (projected state the slope was
//        evaluated at; for stage 1 these ARE T0, Y0), wdot, dTdt (ck_source_terms there)
//   out: accT, accY += b slope (set at stage 1);
//        stages 1-3: Ts, Ys <- proj(y0 + a dt slope)          (next stage state)
//        stage 4:    T0, Y0 <- proj(y0 + dt acc)              (the step's result)
template <int STAGE>
__global__ void __launch_bounds__(256) rk4_stage_kernel(int S, long long N, const double *__restrict__ inv_W,
                                                        const double *__restrict__ P, double *T0, double *Y0,
                                                        double *Ts, double *Ys, const double *__restrict__ wdot,
                                                        const double *__restrict__ dTdt, double *accT, double *accY,
                                                        double dt) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const double a = (STAGE == 3) ? 1.0 : 0.5;
  const double b = (STAGE == 1 || STAGE == 4) ? (1.0 / 6.0) : (1.0 / 3.0);
  const double *Tin = (STAGE == 1) ? T0 : Ts;
  const double *Yin = (STAGE == 1) ? Y0 : Ys;
  const double Tcur = Tin[i];
  // density of the state the slope belongs to
  double inv_Wmix = 0.0;
  for (int k = 0; k < S; ++k) inv_Wmix = fma(Yin[(size_t)k * N + i], inv_W[k], inv_Wmix);
  const double inv_rho = (kRu * Tcur * inv_Wmix) / P[i];

  const double kT = dTdt[i];
  const double aT = (STAGE == 1) ? b * kT : fma(b, kT, accT[i]);
  double Tn = (STAGE == 4) ? fma(dt, aT, T0[i]) : fma(a * dt, kT, T0[i]);
  Tn = fmin(fmax(Tn, kTmin), kTmax);
  double *Tout = (STAGE == 4) ? T0 : Ts;
  double *Yout = (STAGE == 4) ? Y0 : Ys;
  if (STAGE != 4) accT[i] = aT;
  Tout[i] = Tn;

  double sum = 0.0;
  for (int k = 0; k < S; ++k) {
    const size_t at = (size_t)k * N + i;
    const double kY = wdot[at] * inv_rho / inv_W[k];            // wdot_k W_k / rho
    const double aY = (STAGE == 1) ? b * kY : fma(b, kY, accY[at]);
    if (STAGE != 4) accY[at] = aY;
    double y = (STAGE == 4) ? fma(dt, aY, Y0[at]) : fma(a * dt, kY, Y0[at]);
    y = fmax(y, 0.0);
    sum += y;
    Yout[at] = y;
  }
  const double inv_sum = 1.0 / sum;
  for (int k = 0; k < S; ++k) {
    const size_t at = (size_t)k * N + i;
    Yout[at] *= inv_sum;
  }
}

}  // namespace

cudaError_t launch_rk4_stage(int stage, const ck_mech *m, const double *P, double *T0, double *Y0, double *Ts,
                             double *Ys, const double *wdot, const double *dTdt, double *accT, double *accY,
                             int64_t N, double dt, cudaStream_t stream) {
  const int S = m->dev.S;
  const int threads = 256;
  const unsigned grid = (unsigned)((N + threads - 1) / threads);
  const double *inv_W = m->dev.inv_W;
  switch (stage) {
    case 1: rk4_stage_kernel<1><<<grid, threads, 0, stream>>>(S, N, inv_W, P, T0, Y0, Ts, Ys, wdot, dTdt, accT, accY, dt); break;
    case 2: rk4_stage_kernel<2><<<grid, threads, 0, stream>>>(S, N, inv_W, P, T0, Y0, Ts, Ys, wdot, dTdt, accT, accY, dt); break;
    case 3: rk4_stage_kernel<3><<<grid, threads, 0, stream>>>(S, N, inv_W, P, T0, Y0, Ts, Ys, wdot, dTdt, accT, accY, dt); break;
    default: rk4_stage_kernel<4><<<grid, threads, 0, stream>>>(S, N, inv_W, P, T0, Y0, Ts, Ys, wdot, dTdt, accT, accY, dt); break;
  }
  return cudaGetLastError();
}

}  // namespace ck
