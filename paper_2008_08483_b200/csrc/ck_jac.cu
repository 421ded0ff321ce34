// ck_jac.cu -- analytic Jacobian of the source term, d(wdot, dT/dt)/d(Y, T) at constant P
// (the prerequisite of the GPU stiff integrator the paper
// names as future work).  Host table builder + one fused kernel for sm_100a.
//
// The paper prints no Jacobian; this is the chain rule applied to its layers (DESIGN.md
// section 14 derives every term):
//   Eq. 4  ln q_f = nu'^T ln C + ln k_f, ln q_r = nu''^T ln C + ln k_r
//          =>  dq_f/dC_l = nu'_lj q_f / C_l,  dq_r/dC_l = nu''_lj q_r / C_l
//   Eq. 6  d ln k_f/dT = (b + (Ea/R)/T)/T
//   Eq. 11 d ln Kc/dT = (dnu^T (h/RT) - sum dnu)/T    (Gibbs-Helmholtz on Eq. 10)
//   PAPER.md:157          three-body: dQ/dC_l += E_lj (q_f - q_r); falloff through Pr = k_0 M/k_inf
//   Eq. 2  d wdot_i = sum_j dnu_ij dQ_j
// followed by the change of variables C -> (Y, T) at constant P and the energy row.
//
// Output layout: J[N][S+1][S+1], cell-major and row-major per cell (what a batched linear
// solver takes as a strided batch); row i < S is wdot_i, row S is dT/dt; column l < S is
// Y_l, column S is T.  23 KB per cell at S=53: the kernel is bound by these HBM writes
// (DESIGN.md section 14), so the mapping is chosen for coalesced row stores:
//
//   block = 16 warps, tile of CELLS cells (8, or 4 for big mechanisms), persistent grid.
//   phase A  thread per (species, cell): C, 1/C, ln C, NASA-7 h/RT, cp/R, d(cp/R)/dT, g'.
//   phase M  warp per third-body / falloff reaction: M = sum_k E_kj C_k, lanes over the species
//            (coalesced row of E), the cells' partial sums reduced with a halving butterfly.
//   phase B  thread per (reaction, cell), reactions ordered by type so that warps are
//            homogeneous: the rate layers in log form and the scalars every derivative of Q_j
//            is made of:
//              a = phi q_f, b = phi q_r        dQ/dC_l|sparse = (nu'_lj a - nu''_lj b)/C_l
//              m                               dQ/dC_l|dense  = m E_lj  (stored over M)
//              t = dQ/dT at constant C,        e = sum_l C_l dQ/dC_l = ord' a - ord'' b + m M
//   phase C  warp per row i (species), lanes = columns l, the tile's cells in registers:
//            the row of d wdot_i/dC is gathered (never scattered: no atomics, fixed order)
//            from three host-built lists -- (1) the reactions of row i, staged in shared memory
//            (diagonal, T column, wdot_i and g_i = sum_l C_l dwdot_i/dC_l by Euler's relation,
//            lanes = (cell, part of the list)), (2) the off-diagonal sparse entries grouped by
//            column, (3) the third-body reactions of the row (dense in l: coefficient x row of
//            E) -- then (4) mapped to (Y, T):
//              dwdot_i/dY_l = rho/W_l (dwdot_i/dC_l - g_i/(rho s)),  dwdot_i/dT = t-sum - g_i/T
//            and stored as one coalesced row per cell.
//   phase E  energy row, thread per (cell, column): sum_i H_i x row i read back from L2 in a
//            fixed order, then the quotient rule on dT/dt = -sum_k H_k wdot_k / (rho cp).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "ck_internal.h"

namespace ck {

// Launch shapes: 16 warps per block, one block per SM, tiles of 4 to 32 cells (the most that fit);
// 8 warps and two blocks per SM exist as measured alternatives (CK_JAC_SHAPE; slower).

struct JacRowEnt {   // reaction j of row i: coefficients of a_j, b_j on the diagonal, dnu_ij
  double dnu, cf, cr;   // dnu_ij, dnu_ij nu'_ij, dnu_ij nu''_ij
  int j, tb;            // reaction, its row of E / M (or -1)
};
struct JacOffEnt {   // off-diagonal sparse entry (i, l): coefficients of a_j and b_j
  double cf, cr;        // dnu_ij nu'_lj, dnu_ij nu''_lj
  int j, pad;
};
struct JacRxn {      // per reaction, phase B
  double lnA, b, EaR, lnA0, b0, Ea0R, troe[4];
  double dn, ordf, ordr;   // sum dnu, sum nu', sum nu''
  int type, rev, tb, s0, s1, pad;   // support list [s0, s1) of (species, nu', nu'')
};
struct JacSup { double nuf, nur; int k, pad; };

struct JacTables {
  int S, R, n_tb, SP;          // SP = padded row length of E (multiple of 32)
  const double *invW, *nasa_lo, *nasa_hi, *T_mid;   // [S], [S][7], [S][7], [S]
  const JacRxn *rxn;           // [R]
  const JacSup *sup;           // support lists
  const int *tb_rxn;           // [n_tb] reaction of each row of E
  const double *E;             // [n_tb][SP] efficiencies, zero padded
  const int *row_start;        // [S+1] into row_ent
  const JacRowEnt *row_ent;
  const int *off_start;        // [S][SP+1] into off_ent, segments by column
  const JacOffEnt *off_ent;
  double ln_pref_Ru;           // ln(p_ref / Ru)
};

struct JacMech {
  JacTables t{};
  void *d_blob = nullptr;
  // second kernel (lanes = cells, ck_jac_v2.cuh): tables in the same blob, scratch of its own
  bool v2 = false;
  int v2_mt = 0, v2_nth = 4, v2_nw = 0;
  size_t v2_smem = 0;
  void *v2_tables = nullptr;    // host copy of Jac2Tables (device pointers inside)
  double *d_v2_scratch = nullptr;   // allocated by jac_ensure
  size_t v2_scratch_elems = 0;
  int v2_grid = 1;
  int cells = 8;               // cells per tile
  int warps = 16, minb = 1;    // warps per block, blocks per SM
  size_t smem = 0;
  int grid_max = 1;
};

}  // namespace ck

namespace ck {
namespace {

constexpr double kLn10 = 2.302585092994045684;
constexpr int kJacStage = 64;   // row entries a warp stages in shared memory at a time
enum { SP_C = 0, SP_INVC, SP_LNC, SP_HRT, SP_CPR, SP_DCPR, SP_GP, SP_COUNT };
enum { CS_T = 0, CS_RHO, CS_INVRS, CS_INVT, CS_LNT, CS_D, CS_DDT, CS_INVS, CS_COUNT = 8 };

// doubles of dynamic shared memory
inline size_t jac_smem_doubles(int S, int R, int n_tb, int cells, int kJacWarps) {
  return (size_t)SP_COUNT * S * cells + (size_t)CS_COUNT * cells + (size_t)(n_tb > 0 ? n_tb : 1) * cells +
         (size_t)4 * R * cells + (size_t)S * cells + (size_t)kJacWarps * kJacStage * (sizeof(JacRowEnt) / 8);
}

// Sum over the 32 lanes of v[c], c < CELLS, by a butterfly that halves the number of values a
// lane carries at each step (CELLS - 1 + log2(32 / CELLS) shuffles instead of 5 CELLS).
// Returns the total of cell jac_cell_of_lane<CELLS>(lane), the same on every lane of that cell.
template <int CELLS>
__device__ __forceinline__ int jac_cell_of_lane(int lane) {
  // the butterfly consumes lane bits 4, 3, ... for the cell bits from the top down
  return CELLS == 32 ? lane : CELLS == 16 ? (lane >> 1) & 15 : CELLS == 8 ? (lane >> 2) & 7 : (lane >> 3) & 3;
}
template <int CELLS>
__device__ __forceinline__ double jac_reduce_cells(double (&v)[CELLS], int lane) {
  int o = 16;
#pragma unroll
  for (int w = CELLS; w > 1; w >>= 1, o >>= 1) {
    const bool upper = (lane & o) != 0;
#pragma unroll
    for (int q = 0; q < w / 2; ++q) {
      const double send = upper ? v[q] : v[q + w / 2], keep = upper ? v[q + w / 2] : v[q];
      v[q] = keep + __shfl_xor_sync(0xffffffffu, send, o);
    }
  }
  for (; o > 0; o >>= 1) v[0] += __shfl_xor_sync(0xffffffffu, v[0], o);
  return v[0];
}

template <int CELLS, int CPL, int kJacWarps, int MINB>
__global__ void __launch_bounds__(kJacWarps * 32, MINB)
jacobian_kernel(const JacTables t, const double *__restrict__ Tg, const double *__restrict__ Pg,
                const double *__restrict__ Yg, long long N, double *__restrict__ Jg) {
  extern __shared__ __align__(16) double smem[];
  constexpr int kJacThreads = kJacWarps * 32;
  const int S = t.S, R = t.R, n = S + 1, SP = t.SP;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  double *sp = smem;                                   // [SP_COUNT][S][CELLS]
  double *cs = sp + (size_t)SP_COUNT * S * CELLS;      // [CELLS][CS_COUNT]
  double *Mtb = cs + CS_COUNT * CELLS;                 // [n_tb][CELLS]  M, then m = dQ/dM
  double2 *AB = (double2 *)(Mtb + (size_t)(t.n_tb > 0 ? t.n_tb : 1) * CELLS);   // [R][CELLS] (a, b)
  double *Tt = (double *)AB + (size_t)2 * R * CELLS;   // [R][CELLS]  t = dQ/dT at constant C
  double *Ee = Tt + (size_t)R * CELLS;                 // [R][CELLS]  e = sum_l C_l dQ/dC_l
  double *Wd = Ee + (size_t)R * CELLS;                 // [S][CELLS]  wdot
  JacRowEnt *stg = (JacRowEnt *)(Wd + (size_t)S * CELLS) + warp * kJacStage;   // this warp's staged row entries
#define SPV(a, k, c) sp[((size_t)(a) * S + (k)) * CELLS + (c)]
  // (a, b) of reaction j, cell c lives at AB[j * CELLS + (c ^ (j & (CELLS - 1)))]: lanes that read
  // the same cell of different reactions (phase C (2)) then fall into different banks
#define ABAT(j, c) ((j) * CELLS + ((c) ^ ((j) & (CELLS - 1))))
  constexpr int PARTS = 32 / CELLS;

  const long long n_tiles = (N + CELLS - 1) / CELLS;
  for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const long long cell0 = tile * CELLS;
    // ---- cell scalars: s = sum_k Y_k/W_k, rho; warp c <-> cell c -----------
    for (int c = warp; c < CELLS; c += kJacWarps) {
      const long long cell = cell0 + c < N ? cell0 + c : N - 1;
      double s = 0.0;
      for (int k = lane; k < S; k += 32) s += __ldcs(Yg + (size_t)k * N + cell) * t.invW[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if (lane == 0) {
        const double T = Tg[cell], P = Pg[cell];
        cs[c * CS_COUNT + CS_T] = T;
        cs[c * CS_COUNT + CS_INVRS] = (kRu * T) / P;      // 1 / (rho s)
        cs[c * CS_COUNT + CS_INVS] = 1.0 / s;
        cs[c * CS_COUNT + CS_RHO] = P / (kRu * T * s);
        cs[c * CS_COUNT + CS_INVT] = 1.0 / T;
        cs[c * CS_COUNT + CS_LNT] = log(T);
      }
    }
    __syncthreads();
    // ---- phase A: species layers, thread per (species, cell) -------------------------------
    for (int idx = tid; idx < S * CELLS; idx += kJacThreads) {
      const int k = idx / CELLS, c = idx - k * CELLS;
      const long long cell = cell0 + c < N ? cell0 + c : N - 1;
      const double T = cs[c * CS_COUNT + CS_T], lnT = cs[c * CS_COUNT + CS_LNT], invT = cs[c * CS_COUNT + CS_INVT];
      const double C = fmax(cs[c * CS_COUNT + CS_RHO] * __ldcs(Yg + (size_t)k * N + cell) * t.invW[k], kCFloor);
      SPV(SP_C, k, c) = C;
      SPV(SP_INVC, k, c) = 1.0 / C;
      SPV(SP_LNC, k, c) = log(C);
      const double *a = (T <= t.T_mid[k] ? t.nasa_lo : t.nasa_hi) + 7 * k;
      const double T2 = T * T, T3 = T2 * T, T4 = T3 * T;
      const double cpR = a[0] + a[1] * T + a[2] * T2 + a[3] * T3 + a[4] * T4;
      const double hRT = a[0] + a[1] * T * 0.5 + a[2] * T2 * (1.0 / 3.0) + a[3] * T3 * 0.25 + a[4] * T4 * 0.2 + a[5] * invT;
      const double sR = a[0] * lnT + a[1] * T + a[2] * T2 * 0.5 + a[3] * T3 * (1.0 / 3.0) + a[4] * T4 * 0.25 + a[6];
      SPV(SP_CPR, k, c) = cpR;
      SPV(SP_DCPR, k, c) = a[1] + 2.0 * a[2] * T + 3.0 * a[3] * T2 + 4.0 * a[4] * T3;
      SPV(SP_HRT, k, c) = hRT;
      // g' = g/RT - ln(p_ref/(Ru T)): ln Kc = -dnu^T g' (Eq. 11 with PAPER.md:114's fold)
      SPV(SP_GP, k, c) = hRT - sR - (t.ln_pref_Ru - lnT);
    }
    __syncthreads();
    // D = rho cp = sum_k C_k Cp_k and dD/dT (first at constant C, then the -D/T of dC/dT)
    for (int c = warp; c < CELLS; c += kJacWarps) {
      double D = 0.0, dD = 0.0;
      for (int k = lane; k < S; k += 32) {
        D += SPV(SP_C, k, c) * SPV(SP_CPR, k, c);
        dD += SPV(SP_C, k, c) * SPV(SP_DCPR, k, c);
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        D += __shfl_xor_sync(0xffffffffu, D, o);
        dD += __shfl_xor_sync(0xffffffffu, dD, o);
      }
      if (lane == 0) {
        cs[c * CS_COUNT + CS_D] = D * kRu;
        cs[c * CS_COUNT + CS_DDT] = dD * kRu - D * kRu * cs[c * CS_COUNT + CS_INVT];
      }
    }
    // ---- phase M: third-body layer M = C E: warp per row of E, lanes over the
    //      species (coalesced row of E), the cells' partial sums reduced across the lanes
    for (int r = warp; r < t.n_tb; r += kJacWarps) {
      double v[CELLS];
#pragma unroll
      for (int c = 0; c < CELLS; ++c) v[c] = 0.0;
#pragma unroll
      for (int p = 0; p < CPL; ++p) {
        const int k = lane + 32 * p;
        if (k < S) {
          const double e = __ldg(t.E + (size_t)r * SP + k);
#pragma unroll
          for (int c = 0; c < CELLS; ++c) v[c] = fma(e, SPV(SP_C, k, c), v[c]);
        }
      }
      const double tot = jac_reduce_cells<CELLS>(v, lane);
      if ((lane & (PARTS - 1)) == 0) Mtb[r * CELLS + jac_cell_of_lane<CELLS>(lane)] = tot;
    }
    __syncthreads();
    // ---- phase B: rate layers and the derivative scalars, thread per (reaction, cell) ------
    for (int idx = tid; idx < R * CELLS; idx += kJacThreads) {
      const int j = idx / CELLS, c = idx - j * CELLS;
      const JacRxn &r = t.rxn[j];
      const double lnT = cs[c * CS_COUNT + CS_LNT], invT = cs[c * CS_COUNT + CS_INVT], T = cs[c * CS_COUNT + CS_T];
      const int s0 = r.s0, s1 = r.s1, type = r.type;
      // the first entries of the support list in one batch of independent loads
      JacSup u4[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) u4[q] = t.sup[s0 + q < s1 ? s0 + q : s0];
      // Arrhenius layer (Eq. 6) and its T-derivative
      double lnkf = r.lnA + r.b * lnT - r.EaR * invT;
      double dlnkf = (r.b + r.EaR * invT) * invT;
      // log-rate layers (Eq. 4) and the equilibrium layer (Eq. 11) over the reaction's species
      double sf = 0.0, sr = 0.0, dG = 0.0, dH = 0.0;
      for (int e = s0; e < s1; ++e) {
        JacSup u;
        if (e - s0 < 4) {
          u = u4[0];
#pragma unroll
          for (int q = 1; q < 4; ++q) if (e - s0 == q) u = u4[q];
        } else {
          u = t.sup[e];
        }
        const double lc = SPV(SP_LNC, u.k, c), dnu = u.nur - u.nuf;
        sf = fma(u.nuf, lc, sf);
        sr = fma(u.nur, lc, sr);
        dG = fma(dnu, SPV(SP_GP, u.k, c), dG);
        dH = fma(dnu, SPV(SP_HRT, u.k, c), dH);
      }
      const double dlnKc = (dH - r.dn) * invT;
      double M = 1.0, phi = 1.0, gam = 1.0, dlnG = 0.0;
      if (type != 0) M = Mtb[r.tb * CELLS + c];
      if (type == 1) phi = M;
      if (type >= 2) {
        // falloff (textbook forms): k = k_inf Pr/(1+Pr) F, Pr = k_0 M/k_inf
        const double lnk0 = r.lnA0 + r.b0 * lnT - r.Ea0R * invT;
        const double dlnk0 = (r.b0 + r.Ea0R * invT) * invT;
        const double Pr = exp(lnk0 - lnkf) * M;
        double F = 1.0, dlnF_dlnPr = 0.0, dlnF_dT = 0.0;
        if (type == 3) {
          const double alpha = r.troe[0], T3 = r.troe[1], T1 = r.troe[2], T2 = r.troe[3];
          const double e3 = exp(-T / T3), e1 = exp(-T / T1), e2 = exp(-T2 * invT);
          const double Fc = (1.0 - alpha) * e3 + alpha * e1 + e2;
          const double dFc = -(1.0 - alpha) / T3 * e3 - alpha / T1 * e1 + (isinf(T2) ? 0.0 : T2 * invT * invT * e2);
          const double lFc = log10(Fc), dlFc = dFc / (Fc * kLn10);
          const double cc = -0.4 - 0.67 * lFc, nn = 0.75 - 1.27 * lFc;
          const double A = log10(Pr) + cc, B = nn - 0.14 * A;
          const double f1 = A / B, den = 1.0 + f1 * f1;
          F = exp(kLn10 * lFc / den);
          const double dlF_df1 = -2.0 * lFc * f1 / (den * den);
          dlnF_dlnPr = dlF_df1 * nn / (B * B);
          dlnF_dT = kLn10 * dlFc * (1.0 / den + dlF_df1 * ((-0.67 * B + A * (1.27 - 0.14 * 0.67)) / (B * B)));
        }
        dlnG = 1.0 / (1.0 + Pr) + dlnF_dlnPr;
        dlnkf = dlnkf + dlnG * (dlnk0 - dlnkf) + dlnF_dT;
        gam = Pr / (1.0 + Pr) * F;
      }
      const double qf = exp(lnkf + sf) * gam;
      const double qr = r.rev ? exp(lnkf + dG + sr) * gam : 0.0;   // ln k_r = ln k_f - ln Kc, ln Kc = -dG
      const double a = phi * qf, b = phi * qr;
      double m = 0.0;
      if (type == 1) m = qf - qr;
      if (type >= 2) m = (qf - qr) * dlnG / M;
      AB[ABAT(j, c)] = make_double2(a, b);
      Tt[idx] = a * dlnkf - b * (dlnkf - dlnKc);
      Ee[idx] = r.ordf * a - r.ordr * b + (type != 0 ? m * M : 0.0);
      if (type != 0) Mtb[r.tb * CELLS + c] = m;   // M is dead: its slot carries m = dQ/dM from here on
    }
    __syncthreads();
    // ---- phase C: one warp per row i; lanes = columns, the tile's cells in registers -------
    {
      const int my_c = lane % CELLS, my_part = lane / CELLS;
      double iw[CPL];
#pragma unroll
      for (int p = 0; p < CPL; ++p) iw[p] = (lane + 32 * p < S) ? t.invW[lane + 32 * p] : 0.0;
      for (int i = warp; i < S; i += kJacWarps) {
        const int r0 = t.row_start[i], r1 = t.row_start[i + 1];
        // bounds and first entry of this lane's off-diagonal segments, in flight during (1)
        int e0[CPL], e1[CPL];
        JacOffEnt first[CPL];
#pragma unroll
        for (int p = 0; p < CPL; ++p) {
          const int *seg = t.off_start + (size_t)i * (SP + 1) + lane + 32 * p;
          e0[p] = __ldg(seg);
          e1[p] = __ldg(seg + 1);
        }
#pragma unroll
        for (int p = 0; p < CPL; ++p) first[p] = t.off_ent[e0[p]];   // (the table has a spare entry at its end)
        // (1) the row's reaction list (staged in shared memory, 64 entries at a time), lanes =
        //     (cell, part): diagonal of the sparse part, T column, wdot_i, and
        //     g_i = sum_l C_l dwdot_i/dC_l by Euler's relation reaction by reaction
        double diag = 0.0, tsum = 0.0, wd = 0.0, g = 0.0;
        for (int base = r0; base < r1; base += kJacStage) {
          const int cnt = min(kJacStage, r1 - base);
          __syncwarp();
          for (int q = lane; q < cnt * 4; q += 32) ((double *)stg)[q] = __ldg((const double *)(t.row_ent + base) + q);
          __syncwarp();
          for (int e = my_part; e < cnt; e += PARTS) {
            const JacRowEnt u = stg[e];
            const int at = u.j * CELLS + my_c;
            const double2 ab = AB[ABAT(u.j, my_c)];
            diag = fma(u.cf, ab.x, fma(-u.cr, ab.y, diag));
            tsum = fma(u.dnu, Tt[at], tsum);
            wd = fma(u.dnu, ab.x - ab.y, wd);
            g = fma(u.dnu, Ee[at], g);
          }
        }
#pragma unroll
        for (int o = CELLS; o < 32; o <<= 1) {
          diag += __shfl_xor_sync(0xffffffffu, diag, o);
          tsum += __shfl_xor_sync(0xffffffffu, tsum, o);
          wd += __shfl_xor_sync(0xffffffffu, wd, o);
          g += __shfl_xor_sync(0xffffffffu, g, o);
        }
        if (lane < CELLS) Wd[i * CELLS + lane] = wd;
        // (2) off-diagonal sparse entries of row i, grouped by column (next entry prefetched)
        double acc[CELLS][CPL];
#pragma unroll
        for (int c = 0; c < CELLS; ++c)
#pragma unroll
          for (int p = 0; p < CPL; ++p) acc[c][p] = 0.0;
#pragma unroll
        for (int p = 0; p < CPL; ++p) {
          JacOffEnt u = first[p];
          for (int e = e0[p]; e < e1[p]; ++e) {
            const JacOffEnt un = t.off_ent[e + 1];
            const double2 *ab = AB + (size_t)u.j * CELLS;
            const int sw = u.j & (CELLS - 1);
#pragma unroll
            for (int c = 0; c < CELLS; ++c) {
              const double2 v = ab[c ^ sw];
              acc[c][p] = fma(u.cf, v.x, fma(-u.cr, v.y, acc[c][p]));
            }
            u = un;
          }
        }
        // sparse part / C_l (with the diagonal), then (3) adds the dense part
#pragma unroll
        for (int c = 0; c < CELLS; ++c) {
          const double diag_c = __shfl_sync(0xffffffffu, diag, c);
#pragma unroll
          for (int p = 0; p < CPL; ++p) {
            const int col = lane + 32 * p;
            acc[c][p] = col < S ? (acc[c][p] + (col == i ? diag_c : 0.0)) * SPV(SP_INVC, col, c) : 0.0;
          }
        }
        // (3) third-body / falloff reactions of the row (listed first): coefficient x row of E
        {
          bool done = false;
          for (int base = r0; base < r1 && !done; base += kJacStage) {
            const int cnt = min(kJacStage, r1 - base);
            if (r1 - r0 > kJacStage) {      // a long row: stage this chunk again
              __syncwarp();
              for (int q = lane; q < cnt * 4; q += 32) ((double *)stg)[q] = __ldg((const double *)(t.row_ent + base) + q);
              __syncwarp();
            }
            double evn[CPL];
#pragma unroll
            for (int p = 0; p < CPL; ++p) evn[p] = stg[0].tb >= 0 ? __ldg(t.E + (size_t)stg[0].tb * SP + lane + 32 * p) : 0.0;
            for (int e = 0; e < cnt; ++e) {
              const JacRowEnt u = stg[e];
              if (u.tb < 0) { done = true; break; }
              double ev[CPL];
#pragma unroll
              for (int p = 0; p < CPL; ++p) ev[p] = evn[p];
              const int tbn = e + 1 < cnt ? stg[e + 1].tb : -1;
              if (tbn >= 0) {
#pragma unroll
                for (int p = 0; p < CPL; ++p) evn[p] = __ldg(t.E + (size_t)tbn * SP + lane + 32 * p);
              }
              const double *mm = Mtb + (size_t)u.tb * CELLS;
#pragma unroll
              for (int c = 0; c < CELLS; ++c) {
                const double co = u.dnu * mm[c];
#pragma unroll
                for (int p = 0; p < CPL; ++p) acc[c][p] = fma(co, ev[p], acc[c][p]);
              }
            }
          }
        }
        // (4) C -> (Y, T) at constant P, store the row
#pragma unroll
        for (int c = 0; c < CELLS; ++c) {
          const double tsum_c = __shfl_sync(0xffffffffu, tsum, c);
          const double g_c = __shfl_sync(0xffffffffu, g, c);
          // dwdot_i/dY_l = rho/W_l (dwdot_i/dC_l - g_i/(rho s))
          const double rho = cs[c * CS_COUNT + CS_RHO], gk = g_c * cs[c * CS_COUNT + CS_INVRS];
          const long long cell = cell0 + c;
          if (cell < N) {
            double *row = Jg + ((size_t)cell * n + i) * n;
#pragma unroll
            for (int p = 0; p < CPL; ++p) {
              const int col = lane + 32 * p;
              if (col < S) __stcs(row + col, (acc[c][p] - gk) * (rho * iw[p]));
              else if (col == S) __stcs(row + col, tsum_c - g_c * cs[c * CS_COUNT + CS_INVT]);
            }
          }
        }
      }
    }
    __syncthreads();
    // ---- phase E: energy row, dT/dt = -sum_k H_k wdot_k / D; thread per (cell, column), the
    //      species rows of the tile read back (from L2) in a fixed order
    for (int idx = tid; idx < CELLS * n; idx += kJacThreads) {
      const int c = idx / n, col = idx - c * n;
      const long long cell = cell0 + c;
      if (cell >= N) continue;
      const double RuT = kRu * cs[c * CS_COUNT + CS_T];
      const double *Jc = Jg + (size_t)cell * n * n + col;
      double hj = 0.0, hw = 0.0, cpw = 0.0;
#pragma unroll 8
      for (int i = 0; i < S; ++i) {
        const double H = SPV(SP_HRT, i, c) * RuT, w = Wd[i * CELLS + c];
        hj = fma(H, __ldcg(Jc + (size_t)i * n), hj);
        hw = fma(H, w, hw);
        cpw = fma(SPV(SP_CPR, i, c) * kRu, w, cpw);
      }
      const double D = cs[c * CS_COUNT + CS_D], invD = 1.0 / D, Tdot = -hw * invD;
      double v;
      if (col < S) {
        const double iwc = t.invW[col];
        const double dD = cs[c * CS_COUNT + CS_RHO] * SPV(SP_CPR, col, c) * kRu * iwc - D * iwc * cs[c * CS_COUNT + CS_INVS];
        v = -hj * invD - Tdot * dD * invD;
      } else {
        v = -(cpw + hj) * invD - Tdot * cs[c * CS_COUNT + CS_DDT] * invD;
      }
      __stcs(Jg + ((size_t)cell * n + S) * n + col, v);
    }
    __syncthreads();
  }
#undef SPV
#undef ABAT
}

#include "ck_jac_v2.cuh"

}  // namespace
}  // namespace ck

// ---- host: tables from the mechanism description ---------------------------------------------
namespace ck {

namespace {
template <class T>
size_t blob_add(std::vector<unsigned char> &blob, const std::vector<T> &v) {
  const size_t off = (blob.size() + 255) / 256 * 256;
  blob.resize(off + std::max<size_t>(v.size(), 1) * sizeof(T));
  if (!v.empty()) std::memcpy(blob.data() + off, v.data(), v.size() * sizeof(T));
  return off;
}
}  // namespace

// Builds the device tables of the Jacobian kernel.  Returns "" or an error text; *out stays
// NULL (with "") when the mechanism is not supported (approximate-ANN Kc) or does not fit.
std::string jac_create(const ck_mech_desc *d, int num_sms, size_t smem_block_max, JacMech **out) {
  *out = nullptr;
  if (d->kc_ann) return "";
  const int S = d->n_species, R = d->n_reactions;
  const int cpl = (S + 1 + 31) / 32, SP = 32 * cpl;
  if (cpl > 4) return "";   // S <= 127
  std::vector<double> invW(S), lo(d->nasa_lo, d->nasa_lo + 7 * (size_t)S), hi(d->nasa_hi, d->nasa_hi + 7 * (size_t)S),
      tmid(d->T_mid, d->T_mid + S);
  for (int k = 0; k < S; ++k) invW[k] = 1.0 / d->mol_weight[k];
  // Internal reaction order: by type (elementary, three-body, Lindemann, Troe), so that the warps
  // of phase B (thread per (reaction, cell)) are homogeneous in type; oj = order[j]
  std::vector<int> order;
  for (int ty = 0; ty <= 3; ++ty)
    for (int j = 0; j < R; ++j)
      if ((d->rxn_type ? d->rxn_type[j] : 0) == ty) order.push_back(j);
  std::vector<JacRxn> rxn(R);
  std::vector<JacSup> sup;
  std::vector<int> tb_rxn;
  std::vector<double> E;
  for (int j = 0; j < R; ++j) {
    const int oj = order[j];
    JacRxn &r = rxn[j];
    std::memset(&r, 0, sizeof r);
    r.lnA = d->ln_A[oj]; r.b = d->b[oj]; r.EaR = d->Ea_over_R[oj];
    r.type = d->rxn_type ? d->rxn_type[oj] : 0;
    r.rev = d->reversible ? d->reversible[oj] : 1;
    r.tb = -1;
    r.troe[1] = r.troe[2] = r.troe[3] = 1.0;
    if (r.type >= 2) { r.lnA0 = d->ln_A0[oj]; r.b0 = d->b0[oj]; r.Ea0R = d->Ea0_over_R[oj]; }
    if (r.type == 3) for (int q = 0; q < 4; ++q) r.troe[q] = d->troe[4 * (size_t)oj + q];
    r.s0 = (int)sup.size();
    for (int k = 0; k < S; ++k) {
      const double f = d->nu_reac[(size_t)k * R + oj], p = d->nu_prod[(size_t)k * R + oj];
      if (f == 0.0 && p == 0.0) continue;
      sup.push_back(JacSup{f, p, k, 0});
      r.dn += p - f; r.ordf += f; r.ordr += p;
    }
    r.s1 = (int)sup.size();
    if (r.type != 0) {
      r.tb = (int)tb_rxn.size();
      tb_rxn.push_back(j);
      E.resize(E.size() + SP, 0.0);
      for (int k = 0; k < S; ++k) E[(size_t)r.tb * SP + k] = d->eff ? d->eff[(size_t)k * R + oj] : 1.0;
    }
  }
  // row lists: reactions with dnu_ij != 0, third-body / falloff ones first; off-diagonal
  // entries (i, l != i) grouped by column l, reactions in ascending order (a fixed summation order)
  std::vector<int> row_start(S + 1, 0), off_start((size_t)S * (SP + 1), 0);
  std::vector<JacRowEnt> row_ent;
  std::vector<JacOffEnt> off_ent;
  for (int i = 0; i < S; ++i) {
    row_start[i] = (int)row_ent.size();
    for (int pass = 0; pass < 2; ++pass)
      for (int j = 0; j < R; ++j) {
        const int oj = order[j];
        const double f = d->nu_reac[(size_t)i * R + oj], p = d->nu_prod[(size_t)i * R + oj], dnu = p - f;
        if (dnu == 0.0 || (rxn[j].tb >= 0) != (pass == 0)) continue;
        row_ent.push_back(JacRowEnt{dnu, dnu * f, dnu * p, j, rxn[j].tb});
      }
    for (int l = 0; l < SP; ++l) {
      off_start[(size_t)i * (SP + 1) + l] = (int)off_ent.size();
      if (l >= S || l == i) continue;
      for (int j = 0; j < R; ++j) {
        const int oj = order[j];
        const double dnu = d->nu_prod[(size_t)i * R + oj] - d->nu_reac[(size_t)i * R + oj];
        const double f = d->nu_reac[(size_t)l * R + oj], p = d->nu_prod[(size_t)l * R + oj];
        if (dnu == 0.0 || (f == 0.0 && p == 0.0)) continue;
        off_ent.push_back(JacOffEnt{dnu * f, dnu * p, j, 0});
      }
    }
    off_start[(size_t)i * (SP + 1) + SP] = (int)off_ent.size();
  }
  row_start[S] = (int)row_ent.size();
  off_ent.push_back(JacOffEnt{0.0, 0.0, 0, 0});   // the kernel prefetches one entry past a segment
  off_ent.push_back(JacOffEnt{0.0, 0.0, 0, 0});

  JacMech *jm = new JacMech;
  const int n_tb = (int)tb_rxn.size();
  // launch shape: 8 cells x 16 warps if the tile's shared memory fits, else 4 cells x 16 warps;
  // CK_JAC_SHAPE=cells,warps,blocks_per_sm overrides (measurement knob)
  // the most cells per tile (32, 16, 8, 4) whose tile fits shared memory and whose row
  // accumulators (cells x columns per lane doubles) fit the registers of 512 threads
  jm->cells = 4; jm->warps = 16; jm->minb = 1;
  for (int c : {32, 16, 8})
    if (c * cpl <= 32 && jac_smem_doubles(S, R, n_tb, c, 16) * 8 <= smem_block_max) { jm->cells = c; break; }
  if (const char *e = std::getenv("CK_JAC_SHAPE")) {
    int c = 0, w = 0, b = 0;
    if (std::sscanf(e, "%d,%d,%d", &c, &w, &b) == 3 && (c == 4 || c == 8 || ((c == 16 || c == 32) && c * cpl <= 32)) && (w == 8 || w == 16) && (b == 1 || b == 2) &&
        !(w == 16 && b == 2)) { jm->cells = c; jm->warps = w; jm->minb = b; }
  }
  jm->smem = jac_smem_doubles(S, R, n_tb, jm->cells, jm->warps) * 8;
  if (jm->smem > smem_block_max) { delete jm; return ""; }
  jm->grid_max = num_sms * jm->minb;

  // ---- tables of the second kernel (ck_jac_v2.cuh) -----------------------------------------------
  // rows: reactions of row i with their sparse entries (l, cf, cr) over the reaction's species;
  // dense part: the third-body / falloff reactions of row i in k-steps of 4, E gathered per row as
  // DMMA A fragments
  const int n1 = S + 1;
  const int mt_need = (n1 + 7) / 8;
  int v2_mt = 0, v2_nth = 4, v2_maxt = 512;
  for (int cand : {2, 4, 7, 8, 12, 14, 16})
    if (cand >= mt_need) { v2_mt = cand; break; }
  if (v2_mt > 8) { v2_nth = 2; v2_maxt = 256; } else if (v2_mt > 4) { v2_maxt = 384; }
  std::vector<int> rowj_start(S + 1, 0), ks_start(S + 1, 0);
  std::vector<Jac2RowJ> rowj;
  std::vector<Jac2Ent> ent2;
  std::vector<Jac2Coef> coef2;
  std::vector<double> afrag;
  if (v2_mt) {
    for (int i = 0; i < S; ++i) {
      rowj_start[i] = (int)rowj.size();
      ks_start[i] = (int)coef2.size() / 4;
      std::vector<int> tbs;   // third-body reactions (internal index) of the row
      for (int j = 0; j < R; ++j) {
        const int oj = order[j];
        const double dnu = d->nu_prod[(size_t)i * R + oj] - d->nu_reac[(size_t)i * R + oj];
        if (dnu == 0.0) continue;
        Jac2RowJ rj{dnu, j, (int)ent2.size(), 0, 0};
        for (int l = 0; l < S; ++l) {
          const double f = d->nu_reac[(size_t)l * R + oj], p = d->nu_prod[(size_t)l * R + oj];
          if (f == 0.0 && p == 0.0) continue;
          ent2.push_back(Jac2Ent{dnu * f, dnu * p, l, 0});
        }
        rj.ent1 = (int)ent2.size();
        rowj.push_back(rj);
        if (rxn[j].tb >= 0) tbs.push_back(j);
      }
      const int nks = ((int)tbs.size() + 3) / 4;
      for (int ks = 0; ks < nks; ++ks) {
        const size_t a0 = afrag.size();
        afrag.resize(a0 + (size_t)v2_mt * 32, 0.0);
        for (int qq = 0; qq < 4; ++qq) {
          const int kk = 4 * ks + qq;
          if (kk < (int)tbs.size()) {
            const int j = tbs[kk], oj = order[j];
            coef2.push_back(Jac2Coef{d->nu_prod[(size_t)i * R + oj] - d->nu_reac[(size_t)i * R + oj], rxn[j].tb, 0});
            for (int mt = 0; mt < v2_mt; ++mt)
              for (int gg = 0; gg < 8; ++gg) {
                const int l = 8 * mt + gg;
                if (l < S) afrag[a0 + (size_t)mt * 32 + gg * 4 + qq] = E[(size_t)rxn[j].tb * SP + l];
              }
          } else {
            coef2.push_back(Jac2Coef{0.0, -1, 0});
          }
        }
      }
    }
    rowj_start[S] = (int)rowj.size();
    ks_start[S] = (int)coef2.size() / 4;
  }
  // work of a row (sparse entries, reactions, k-steps of the dense part), for the static balance
  std::vector<int> row_order(S), row_work(S, 0), warp_row_start(17 + 1, 0);
  for (int i = 0; i < S; ++i) row_order[i] = i;
  if (v2_mt)
    for (int i = 0; i < S; ++i) {
      int ents = 0;
      for (int e = rowj_start[i]; e < rowj_start[i + 1]; ++e) ents += rowj[e].ent1 - rowj[e].ent0;
      row_work[i] = ents * 12 + (rowj_start[i + 1] - rowj_start[i]) * 20 + (ks_start[i + 1] - ks_start[i]) * 60 + 400;
    }

  std::vector<unsigned char> blob;
  const size_t o_ro = blob_add(blob, row_order), o_ws = blob_add(blob, warp_row_start);
  const size_t o_rj0 = blob_add(blob, rowj_start), o_rj = blob_add(blob, rowj), o_e2 = blob_add(blob, ent2),
               o_ks = blob_add(blob, ks_start), o_co = blob_add(blob, coef2), o_af = blob_add(blob, afrag);
  const size_t o_invW = blob_add(blob, invW), o_lo = blob_add(blob, lo), o_hi = blob_add(blob, hi),
               o_tmid = blob_add(blob, tmid), o_rxn = blob_add(blob, rxn), o_sup = blob_add(blob, sup),
               o_tbr = blob_add(blob, tb_rxn), o_E = blob_add(blob, E), o_rs = blob_add(blob, row_start),
               o_re = blob_add(blob, row_ent), o_os = blob_add(blob, off_start), o_oe = blob_add(blob, off_ent);
  cudaError_t ce = cudaMalloc(&jm->d_blob, blob.size());
  if (ce == cudaSuccess) ce = cudaMemcpy(jm->d_blob, blob.data(), blob.size(), cudaMemcpyHostToDevice);
  if (ce != cudaSuccess) {
    if (jm->d_blob) cudaFree(jm->d_blob);
    delete jm;
    return std::string("Jacobian tables: ") + cudaGetErrorString(ce);
  }
  const unsigned char *b = (const unsigned char *)jm->d_blob;
  JacTables &t = jm->t;
  t.S = S; t.R = R; t.n_tb = n_tb; t.SP = SP;
  t.invW = (const double *)(b + o_invW); t.nasa_lo = (const double *)(b + o_lo);
  t.nasa_hi = (const double *)(b + o_hi); t.T_mid = (const double *)(b + o_tmid);
  t.rxn = (const JacRxn *)(b + o_rxn); t.sup = (const JacSup *)(b + o_sup);
  t.tb_rxn = (const int *)(b + o_tbr); t.E = (const double *)(b + o_E);
  t.row_start = (const int *)(b + o_rs); t.row_ent = (const JacRowEnt *)(b + o_re);
  t.off_start = (const int *)(b + o_os); t.off_ent = (const JacOffEnt *)(b + o_oe);
  t.ln_pref_Ru = std::log(d->p_ref / kRu);
  // ---- second kernel: warps per block from the shared memory, scratch per block ------------------
  if (v2_mt && !(std::getenv("CK_JAC_KERNEL") && std::string(std::getenv("CK_JAC_KERNEL")) == "v1")) {
    // warps per block: the shape with the most resident warps per SM (shared memory and the
    // kernel's register cap decide); among equals the smaller blocks, whose tiles overlap better
    int nw = 0, v2_bps = 1;
    size_t smem2 = 0;
    const int regs = v2_maxt == 512 ? 128 : (v2_maxt == 384 ? 168 : 255);
    int best_warps = 0;
    for (int cand : {2, 4, 6, 8, 12, 16}) {
      if (cand * 32 > v2_maxt) continue;
      const size_t base = std::max((size_t)cand * n1 * 33, (size_t)6 * S * 32);
      const size_t doubles = base + (size_t)std::max(n_tb, 1) * 32 + (size_t)S * 32 + (size_t)4 * cand * 32;
      if (doubles * 8 > smem_block_max) continue;
      const int bps = (int)std::min<size_t>(std::min<size_t>(16, 233472 / (doubles * 8 + 1024)), 65536 / ((size_t)regs * cand * 32));
      if (bps < 1) continue;
      if (cand * bps > best_warps) { best_warps = cand * bps; nw = cand; v2_bps = bps; smem2 = doubles * 8; }
    }
    if (nw) {
      // rows to warps: longest processing time first (fixed, so results are reproducible)
      std::vector<int> by_work(S);
      for (int i = 0; i < S; ++i) by_work[i] = i;
      std::stable_sort(by_work.begin(), by_work.end(), [&](int x, int y) { return row_work[x] > row_work[y]; });
      std::vector<std::vector<int>> rows_of(nw);
      std::vector<long long> load(nw, 0);
      for (int i : by_work) {
        const int w = (int)(std::min_element(load.begin(), load.end()) - load.begin());
        rows_of[w].push_back(i);
        load[w] += row_work[i];
      }
      std::vector<int> ro, ws(nw + 1, 0);
      for (int w = 0; w < nw; ++w) { ro.insert(ro.end(), rows_of[w].begin(), rows_of[w].end()); ws[w + 1] = (int)ro.size(); }
      ce = cudaMemcpy((void *)(b + o_ro), ro.data(), ro.size() * sizeof(int), cudaMemcpyHostToDevice);
      if (ce == cudaSuccess) ce = cudaMemcpy((void *)(b + o_ws), ws.data(), ws.size() * sizeof(int), cudaMemcpyHostToDevice);
      if (ce != cudaSuccess) { jac_destroy(jm); return std::string("Jacobian tables: ") + cudaGetErrorString(ce); }
      Jac2Tables *u = new Jac2Tables();
      u->warp_row_start = (const int *)(b + o_ws);
      u->rowj_start = (const int *)(b + o_rj0); u->rowj = (const Jac2RowJ *)(b + o_rj); u->ent = (const Jac2Ent *)(b + o_e2);
      u->row_order = (const int *)(b + o_ro);
      u->ks_start = (const int *)(b + o_ks); u->coef = (const Jac2Coef *)(b + o_co); u->afrag = (const double *)(b + o_af);
      u->scratch_per_block = (size_t)4 * R * 32 + (size_t)2 * S * 32 + (size_t)nw * n1 * 32;
      // (the scratch itself, num_sms * v2_bps * scratch_per_block doubles, is allocated by jac_ensure on
      //  the first launch of this kernel: a handle whose calls all go to the specialised kernel, or that
      //  never calls ck_jacobian, does not pay for it)
      u->scratch = nullptr;
      jm->v2_scratch_elems = (size_t)num_sms * v2_bps * u->scratch_per_block;
      jm->v2 = true; jm->v2_mt = v2_mt; jm->v2_nth = v2_nth; jm->v2_nw = nw; jm->v2_smem = smem2;
      jm->v2_tables = u;
      jm->v2_grid = num_sms * v2_bps;
    }
  }
  *out = jm;
  return "";
}

void jac_destroy(JacMech *jm) {
  if (!jm) return;
  if (jm->d_blob) cudaFree(jm->d_blob);
  if (jm->d_v2_scratch) cudaFree(jm->d_v2_scratch);
  delete (Jac2Tables *)jm->v2_tables;
  delete jm;
}

int jac_cells_per_tile(const JacMech *jm) { return jm->v2 ? 32 : jm->cells; }
bool jac_is_v2(const JacMech *jm) { return jm->v2; }

std::string jac_ensure(JacMech *jm) {
  if (!jm->v2 || jm->d_v2_scratch) return "";
  const cudaError_t ce = cudaMalloc((void **)&jm->d_v2_scratch, jm->v2_scratch_elems * sizeof(double));
  if (ce != cudaSuccess) {
    cudaGetLastError();
    return std::string("Jacobian scratch: ") + cudaGetErrorString(ce);
  }
  ((Jac2Tables *)jm->v2_tables)->scratch = jm->d_v2_scratch;
  return "";
}

cudaError_t jac_launch(const JacMech *jm, const double *T, const double *P, const double *Y, int64_t N,
                       double *J, cudaStream_t stream) {
  if (jm->v2) {
    const Jac2Tables &u = *(const Jac2Tables *)jm->v2_tables;
    const int grid = (int)std::min<long long>((N + 31) / 32, jm->v2_grid);
#define CK_JAC2_CASE(MT, NTH, MAXT)                                                                    \
  if (jm->v2_mt == MT) {                                                                               \
    cudaError_t e = cudaFuncSetAttribute(jacobian_kernel_v2<MT, NTH, MAXT>,                            \
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)jm->v2_smem); \
    if (e != cudaSuccess) return e;                                                                    \
    jacobian_kernel_v2<MT, NTH, MAXT><<<grid, jm->v2_nw * 32, jm->v2_smem, stream>>>(jm->t, u, T, P, Y, (long long)N, J); \
    return cudaGetLastError();                                                                         \
  }
    CK_JAC2_CASE(2, 4, 512) CK_JAC2_CASE(4, 4, 512) CK_JAC2_CASE(7, 4, 384) CK_JAC2_CASE(8, 4, 384)
    CK_JAC2_CASE(12, 2, 256) CK_JAC2_CASE(14, 2, 256) CK_JAC2_CASE(16, 2, 256)
#undef CK_JAC2_CASE
    return cudaErrorInvalidConfiguration;
  }
  const int cpl = jm->t.SP / 32;
  const long long tiles = (N + jm->cells - 1) / jm->cells;
  const int grid = (int)std::min<long long>(tiles, jm->grid_max);
#define CK_JAC_CASE(CE, CP, WA, MB)                                                                \
  if (jm->cells == CE && cpl == CP && jm->warps == WA && jm->minb == MB) {                         \
    cudaError_t e = cudaFuncSetAttribute(jacobian_kernel<CE, CP, WA, MB>,                          \
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)jm->smem); \
    if (e != cudaSuccess) return e;                                                                \
    jacobian_kernel<CE, CP, WA, MB><<<grid, WA * 32, jm->smem, stream>>>(jm->t, T, P, Y, (long long)N, J); \
    return cudaGetLastError();                                                                     \
  }
#define CK_JAC_SHAPES(CE, CP) CK_JAC_CASE(CE, CP, 16, 1) CK_JAC_CASE(CE, CP, 8, 1) CK_JAC_CASE(CE, CP, 8, 2)
  CK_JAC_SHAPES(8, 1) CK_JAC_SHAPES(8, 2) CK_JAC_SHAPES(8, 3) CK_JAC_SHAPES(8, 4)
  CK_JAC_SHAPES(4, 1) CK_JAC_SHAPES(4, 2) CK_JAC_SHAPES(4, 3) CK_JAC_SHAPES(4, 4)
  CK_JAC_CASE(32, 1, 16, 1) CK_JAC_CASE(16, 1, 16, 1) CK_JAC_CASE(16, 2, 16, 1)
#undef CK_JAC_SHAPES
#undef CK_JAC_CASE
  return cudaErrorInvalidConfiguration;
}

}  // namespace ck
