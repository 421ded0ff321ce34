// ck_jac_v2.cuh -- second Jacobian kernel (included by ck_jac.cu): lanes = cells.
//
// A block owns a tile of 32 cells; every warp's lane c works on cell c of the tile, and the warps
// split the species (pass 0), the reactions (pass 1) and the rows of J (pass 2) between them.
// Compared with the first kernel (lanes = columns, tiles of 8 cells) no lane idles on a short
// sparse segment, and the dense third-body part of a row,
//     D_il = sum_{j in TB(i)} E_lj (dnu_ij m_j),        m_j = dQ_j/dM_j  per cell,
// is a small GEMM [S x K_i] [K_i x 32 cells] on DMMA.8x8x4 (K_i = third-body / falloff reactions
// of row i, E gathered per row on the host as ready A fragments), which replaces 53 FMAs + 27
// shared-memory loads per (row, reaction) pair by 7 DMMAs per 4 pairs.
//
//   pass 0  species layers: C, 1/C, ln C, NASA-7 h/RT, cp/R, d(cp/R)/dT, g' (warp w: species w,
//           w + NW, ..), cell scalars rho, s, D = rho cp, dD/dT in registers of every warp
//   pass M  M_j = sum_k E_kj C_k, warp per row of E
//   pass 1  rate layers and derivative scalars per reaction (warp w: reactions w, w + NW, ..):
//           a = phi q_f, b = phi q_r, t = dQ/dT|_C, e = sum_l C_l dQ/dC_l to an L2-resident
//           scratch [R][32] (coalesced), m over M in shared memory           (Eq. 4, 6, 11)
//   pass 2  rows (warp w: rows w, w + NW, ..), in the warp's row buffer rb[l][cell]:
//           (1) dense part by DMMA, fragments stored to rb; (2) sparse part, lane = cell: the
//           row's reactions, their (a, b) from the scratch, entries (l, cf, cr) added to rb[l]
//           scaled by 1/C_l, and wdot_i, dwdot_i/dT|_C, g_i by Euler's relation; (3) C -> (Y, T):
//           J_il = rho/W_l (rb[l] - g_i/(rho s)), J_iT = t_i - g_i/T; H_i J_il added to the warp's
//           partial energy-row sums (scratch); (4) rb read transposed: one coalesced row of
//           S + 1 doubles per cell                                             (Eq. 2)
//   pass 3  energy row from the partial sums, quotient rule on dT/dt = -sum H_k wdot_k / D.
// No atomics, fixed summation orders: bitwise reproducible.
#pragma once

struct Jac2RowJ {     // reaction j of row i
  double dnu;
  int j, ent0, ent1, pad;   // entries [ent0, ent1) of Jac2Ent
};
struct Jac2Ent {      // (i, j, l): coefficients of a_j and b_j in the sparse part of J_C[i][l] C_l
  double cf, cr;      // dnu_ij nu'_lj, dnu_ij nu''_lj
  int l, pad;
};
struct Jac2Coef { double dnu; int tb, pad; };   // k-slot of a row's dense part

struct Jac2Tables {
  const int *rowj_start;      // [S + 1]
  const Jac2RowJ *rowj;
  const Jac2Ent *ent;
  const int *row_order;       // [S] rows grouped by the warp that takes them
  const int *warp_row_start;  // [NW + 1] into row_order
  const int *ks_start;        // [S + 1] k-steps (of 4 third-body reactions) of each row
  const Jac2Coef *coef;       // [ks][4]
  const double *afrag;        // [ks][MT][32]: E[l = 8 mt + lane/4][reaction of k-slot 4 ks + lane%4]
  double *scratch;            // per block: a, b, t, e [R][32] | H, Cp [S][32] | esum [NW][S + 1][32]
  size_t scratch_per_block;   // doubles
};

__device__ __forceinline__ void jac2_dmma(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// NTH: cell n-tiles (of 8) per DMMA sweep: 4 (one sweep) while 8 MT fragments fit the registers,
// else 2 (two sweeps over the cells)
template <int MT, int NTH, int MAXT>
__global__ void __launch_bounds__(MAXT, 1)
jacobian_kernel_v2(const JacTables t, const Jac2Tables u, const double *__restrict__ Tg,
                   const double *__restrict__ Pg, const double *__restrict__ Yg, long long N,
                   double *__restrict__ Jg) {
  extern __shared__ __align__(16) double smem[];
  const int S = t.S, R = t.R, n = S + 1, n_tb = t.n_tb;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, NW = blockDim.x >> 5;
  const int g = lane >> 2, q = lane & 3;
  const int RB = n * 33;                                  // doubles of one row buffer
  double *rb = smem + (size_t)warp * RB;                  // this warp's row buffer [n][33]
  // (the pass-0/1 arrays below share the row buffers' space: the larger of the two)
  const size_t base = (size_t)NW * RB > (size_t)6 * S * 32 ? (size_t)NW * RB : (size_t)6 * S * 32;
  double *mtb = smem + base;                              // [n_tb][32]  M, then m
  double *invC = mtb + (size_t)(n_tb > 0 ? n_tb : 1) * 32;   // [S][32]
  double *part = invC + (size_t)S * 32;                   // [4][NW][32] partial sums between warps
  // pass 0 / 1 arrays over the (then unused) row buffers: [S][32] each
  double *aC = smem, *aLNC = aC + (size_t)S * 32, *aHRT = aLNC + (size_t)S * 32, *aGP = aHRT + (size_t)S * 32,
         *aCPR = aGP + (size_t)S * 32, *aDCPR = aCPR + (size_t)S * 32;
  double *scr = u.scratch + (size_t)blockIdx.x * u.scratch_per_block;
  double *sA = scr, *sB = sA + (size_t)R * 32, *sT = sB + (size_t)R * 32, *sE = sT + (size_t)R * 32;
  double *sH = sE + (size_t)R * 32, *sCp = sH + (size_t)S * 32, *sEsum = sCp + (size_t)S * 32 + (size_t)warp * n * 32;

  const long long n_tiles = (N + 31) / 32;
  for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const long long cell0 = tile * 32;
    const long long cell = cell0 + lane < N ? cell0 + lane : N - 1;
    // ---- pass 0: species layers, lane = cell, warp w takes species w, w + NW, ... -----------------
    const double T = __ldg(Tg + cell), P = __ldg(Pg + cell);
    const double lnT = log(T), invT = 1.0 / T;
    const double T2 = T * T, T3 = T2 * T, T4 = T3 * T;
    double s_part = 0.0;
    for (int k = warp; k < S; k += NW) {
      const double yw = __ldcs(Yg + (size_t)k * N + cell) * __ldg(t.invW + k);
      aC[k * 32 + lane] = yw;
      s_part += yw;
      const double *a = (T <= __ldg(t.T_mid + k) ? t.nasa_lo : t.nasa_hi) + 7 * k;
      const double a0 = __ldg(a), a1 = __ldg(a + 1), a2 = __ldg(a + 2), a3 = __ldg(a + 3), a4 = __ldg(a + 4);
      const double cpR = a0 + a1 * T + a2 * T2 + a3 * T3 + a4 * T4;
      const double hRT = a0 + a1 * T * 0.5 + a2 * T2 * (1.0 / 3.0) + a3 * T3 * 0.25 + a4 * T4 * 0.2 + __ldg(a + 5) * invT;
      const double sR = a0 * lnT + a1 * T + a2 * T2 * 0.5 + a3 * T3 * (1.0 / 3.0) + a4 * T4 * 0.25 + __ldg(a + 6);
      aCPR[k * 32 + lane] = cpR;
      aDCPR[k * 32 + lane] = a1 + 2.0 * a2 * T + 3.0 * a3 * T2 + 4.0 * a4 * T3;
      aHRT[k * 32 + lane] = hRT;
      aGP[k * 32 + lane] = hRT - sR - (t.ln_pref_Ru - lnT);   // g' = g/RT - ln(p_ref/(Ru T))
      sH[k * 32 + lane] = hRT * (kRu * T);                     // H_k, J/kmol
      sCp[k * 32 + lane] = cpR * kRu;
    }
    part[warp * 32 + lane] = s_part;
    __syncthreads();
    double s = 0.0;
    for (int w = 0; w < NW; ++w) s += part[w * 32 + lane];
    const double rho = P / (kRu * T * s), invRS = (kRu * T) / P, invS = 1.0 / s;
    double D_part = 0.0, dD_part = 0.0;
    for (int k = warp; k < S; k += NW) {
      const double C = fmax(rho * aC[k * 32 + lane], kCFloor);
      aC[k * 32 + lane] = C;
      invC[k * 32 + lane] = 1.0 / C;
      aLNC[k * 32 + lane] = log(C);
      D_part = fma(C, aCPR[k * 32 + lane], D_part);
      dD_part = fma(C, aDCPR[k * 32 + lane], dD_part);
    }
    part[(NW + warp) * 32 + lane] = D_part;
    part[(2 * NW + warp) * 32 + lane] = dD_part;
    __syncthreads();
    double D = 0.0, dD = 0.0;
    for (int w = 0; w < NW; ++w) { D += part[(NW + w) * 32 + lane]; dD += part[(2 * NW + w) * 32 + lane]; }
    D *= kRu;
    const double dDdT = dD * kRu - D * invT;
    // ---- pass M: M_j = sum_k E_kj C_k, warp per row of E (uniform loads of the row) ----------------
    for (int r = warp; r < n_tb; r += NW) {
      const double2 *e = (const double2 *)(t.E + (size_t)r * t.SP);   // (rows are zero padded to SP)
      double m0 = 0.0, m1 = 0.0, m2 = 0.0, m3 = 0.0;
      int k = 0;
      for (; k + 3 < S; k += 4) {
        const double2 ev = __ldg(e + (k >> 1)), ew = __ldg(e + (k >> 1) + 1);
        m0 = fma(ev.x, aC[k * 32 + lane], m0);
        m1 = fma(ev.y, aC[(k + 1) * 32 + lane], m1);
        m2 = fma(ew.x, aC[(k + 2) * 32 + lane], m2);
        m3 = fma(ew.y, aC[(k + 3) * 32 + lane], m3);
      }
      for (; k < S; ++k) m0 = fma(__ldg(t.E + (size_t)r * t.SP + k), aC[k * 32 + lane], m0);
      mtb[r * 32 + lane] = (m0 + m1) + (m2 + m3);
    }
    __syncthreads();
    // ---- pass 1: rate layers and derivative scalars, warp per reaction, lane = cell ----------------
    for (int j = warp; j < R; j += NW) {
      const JacRxn &r = t.rxn[j];
      const int type = r.type;
      double lnkf = r.lnA + r.b * lnT - r.EaR * invT;               // Eq. 6
      double dlnkf = (r.b + r.EaR * invT) * invT;
      double sf = 0.0, sr = 0.0, dG = 0.0, dH = 0.0;
      {
        // the reaction's species list: lane x loads entry x (one coalesced load), broadcast by shuffles
        const int ns = r.s1 - r.s0;
        for (int e0 = 0; e0 < ns; e0 += 32) {
          const JacSup mine = t.sup[r.s0 + (e0 + lane < ns ? e0 + lane : 0)];
          const int cnt = ns - e0 < 32 ? ns - e0 : 32;
          for (int x = 0; x < cnt; ++x) {
            const int k = __shfl_sync(0xffffffffu, mine.k, x);
            const double nuf = __shfl_sync(0xffffffffu, mine.nuf, x), nur = __shfl_sync(0xffffffffu, mine.nur, x);
            const double lc = aLNC[k * 32 + lane], dnu = nur - nuf;
            sf = fma(nuf, lc, sf);                                    // Eq. 4
            sr = fma(nur, lc, sr);
            dG = fma(dnu, aGP[k * 32 + lane], dG);                    // Eq. 11
            dH = fma(dnu, aHRT[k * 32 + lane], dH);
          }
        }
      }
      const double dlnKc = (dH - r.dn) * invT;
      double M = 1.0, phi = 1.0, gam = 1.0, dlnG = 0.0;
      if (type != 0) M = mtb[r.tb * 32 + lane];
      if (type == 1) phi = M;
      if (type >= 2) {   // falloff (textbook forms): k = k_inf Pr/(1+Pr) F, Pr = k_0 M/k_inf
        const double lnk0 = r.lnA0 + r.b0 * lnT - r.Ea0R * invT;
        const double dlnk0 = (r.b0 + r.Ea0R * invT) * invT;
        const double Pr = exp(lnk0 - lnkf) * M;
        double F = 1.0, dlnF_dlnPr = 0.0, dlnF_dT = 0.0;
        if (type == 3) {
          const double alpha = r.troe[0], T3t = r.troe[1], T1t = r.troe[2], T2t = r.troe[3];
          const double e3 = exp(-T / T3t), e1 = exp(-T / T1t), e2 = exp(-T2t * invT);
          const double Fc = (1.0 - alpha) * e3 + alpha * e1 + e2;
          const double dFc = -(1.0 - alpha) / T3t * e3 - alpha / T1t * e1 + (isinf(T2t) ? 0.0 : T2t * invT * invT * e2);
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
      sA[j * 32 + lane] = a;
      sB[j * 32 + lane] = b;
      sT[j * 32 + lane] = a * dlnkf - b * (dlnkf - dlnKc);
      sE[j * 32 + lane] = r.ordf * a - r.ordr * b + (type != 0 ? m * M : 0.0);
      if (type != 0) mtb[r.tb * 32 + lane] = m;   // M is dead: its slot carries m = dQ/dM from here on
    }
    __syncthreads();   // (also: every warp is done with the pass-0/1 arrays under the row buffers)
    // ---- pass 2: rows, warp w takes rows w, w + NW, ... ---------------------------------------------
    double hw_part = 0.0, cpw_part = 0.0;
    bool first_row = true;
    // the rows of each warp are fixed on the host (longest-processing-time-first over the rows' work):
    // balanced, and the summation order of the energy row does not depend on the run
    const int rw0 = __ldg(u.warp_row_start + warp), rw1 = __ldg(u.warp_row_start + warp + 1);
    for (int slot = rw0; slot < rw1; ++slot) {
      const int i = __ldg(u.row_order + slot);
      // (1) dense part: D[l][cell] = sum_k afrag[l][k] (dnu_k m_k[cell]) on DMMA, into rb
      const int ks0 = __ldg(u.ks_start + i), ks1 = __ldg(u.ks_start + i + 1);
      if (ks1 > ks0) {
#pragma unroll 1
        for (int nh = 0; nh < 4 / NTH; ++nh) {
          double Dc[MT][NTH][2];
#pragma unroll
          for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NTH; ++nt) Dc[mt][nt][0] = Dc[mt][nt][1] = 0.0;
          for (int ks = ks0; ks < ks1; ++ks) {
            const Jac2Coef co = u.coef[ks * 4 + q];
            double bf[NTH];
#pragma unroll
            for (int nt = 0; nt < NTH; ++nt)
              bf[nt] = co.tb >= 0 ? co.dnu * mtb[co.tb * 32 + 8 * (nh * NTH + nt) + g] : 0.0;
            const double *af = u.afrag + ((size_t)ks * MT) * 32 + lane;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
              const double a = __ldg(af + mt * 32);
#pragma unroll
              for (int nt = 0; nt < NTH; ++nt) jac2_dmma(Dc[mt][nt][0], Dc[mt][nt][1], a, bf[nt]);
            }
          }
#pragma unroll
          for (int mt = 0; mt < MT; ++mt)
            if (8 * mt + g < S) {
#pragma unroll
              for (int nt = 0; nt < NTH; ++nt) {
                rb[(8 * mt + g) * 33 + 8 * (nh * NTH + nt) + 2 * q] = Dc[mt][nt][0];
                rb[(8 * mt + g) * 33 + 8 * (nh * NTH + nt) + 2 * q + 1] = Dc[mt][nt][1];
              }
            }
        }
      } else {
        for (int l = 0; l < S; ++l) rb[l * 33 + lane] = 0.0;
      }
      __syncwarp();
      // (2) sparse part and the row's sums, lane = cell
      double wd = 0.0, tsum = 0.0, gsum = 0.0;
      const int j0 = __ldg(u.rowj_start + i), j1 = __ldg(u.rowj_start + i + 1);
      for (int hb = j0; hb < j1; hb += 32) {
        // up to 32 reactions of the row: lane x holds header x.  The scalars (a, b, t, e) and the
        // entries of the NEXT reaction are loaded while this one is worked on (a reaction has at
        // most 32 entries here; longer lists take the tail loop)
        const Jac2RowJ hd = u.rowj[hb + lane < j1 ? hb + lane : j1 - 1];
        const int nh = j1 - hb < 32 ? j1 - hb : 32;
        int jn = __shfl_sync(0xffffffffu, hd.j, 0);
        int x0n = __shfl_sync(0xffffffffu, hd.ent0, 0), x1n = __shfl_sync(0xffffffffu, hd.ent1, 0);
        double a_n = __ldcg(sA + jn * 32 + lane), b_n = __ldcg(sB + jn * 32 + lane);
        double t_n = __ldcg(sT + jn * 32 + lane), e_n = __ldcg(sE + jn * 32 + lane);
        Jac2Ent en_n = u.ent[x0n + lane < x1n ? x0n + lane : x0n];
        for (int h = 0; h < nh; ++h) {
          const double a = a_n, b = b_n, tt = t_n, ee = e_n;
          const Jac2Ent en = en_n;
          const int x0 = x0n, x1 = x1n;
          const double dnu = __shfl_sync(0xffffffffu, hd.dnu, h);
          if (h + 1 < nh) {
            jn = __shfl_sync(0xffffffffu, hd.j, h + 1);
            x0n = __shfl_sync(0xffffffffu, hd.ent0, h + 1); x1n = __shfl_sync(0xffffffffu, hd.ent1, h + 1);
            a_n = __ldcg(sA + jn * 32 + lane); b_n = __ldcg(sB + jn * 32 + lane);
            t_n = __ldcg(sT + jn * 32 + lane); e_n = __ldcg(sE + jn * 32 + lane);
            en_n = u.ent[x0n + lane < x1n ? x0n + lane : x0n];
          }
          wd = fma(dnu, a - b, wd);
          tsum = fma(dnu, tt, tsum);
          gsum = fma(dnu, ee, gsum);
          const int cnt = x1 - x0 < 32 ? x1 - x0 : 32;
          for (int x = 0; x < cnt; ++x) {
            const double cf = __shfl_sync(0xffffffffu, en.cf, x), cr = __shfl_sync(0xffffffffu, en.cr, x);
            const int l = __shfl_sync(0xffffffffu, en.l, x);
            rb[l * 33 + lane] = fma(fma(cf, a, -cr * b), invC[l * 32 + lane], rb[l * 33 + lane]);
          }
          for (int x = x0 + 32; x < x1; ++x) {   // (a reaction of more than 32 species)
            const Jac2Ent e2 = u.ent[x];
            rb[e2.l * 33 + lane] = fma(fma(e2.cf, a, -e2.cr * b), invC[e2.l * 32 + lane], rb[e2.l * 33 + lane]);
          }
        }
      }
      // (3) C -> (Y, T) at constant P:  dwdot_i/dY_l = rho/W_l (dwdot_i/dC_l - g_i/(rho s)),
      //     dwdot_i/dT = dwdot_i/dT|_C - g_i/T;  energy-row partial sums sum_i H_i J_il
      const double H_i = __ldcg(sH + i * 32 + lane), gk = gsum * invRS;
      hw_part = fma(H_i, wd, hw_part);
      cpw_part = fma(__ldcg(sCp + i * 32 + lane), wd, cpw_part);
      for (int l = 0; l < S; ++l) {
        const double v = (rb[l * 33 + lane] - gk) * (rho * __ldg(t.invW + l));
        rb[l * 33 + lane] = v;
        sEsum[l * 32 + lane] = first_row ? H_i * v : fma(H_i, v, sEsum[l * 32 + lane]);
      }
      {
        const double v = tsum - gsum * invT;
        rb[S * 33 + lane] = v;
        sEsum[S * 32 + lane] = first_row ? H_i * v : fma(H_i, v, sEsum[S * 32 + lane]);
      }
      first_row = false;
      __syncwarp();
      // (4) one coalesced row of n doubles per cell
      {
        const int nc = N - cell0 < 32 ? (int)(N - cell0) : 32;
        double *row = Jg + ((size_t)cell0 * n + i) * n + lane;
        const size_t cstride = (size_t)n * n;
        const double *src0 = rb + lane * 33, *src1 = rb + (lane + 32) * 33;
        const bool c0 = lane < n, c1 = lane + 32 < n;
        if (n <= 64) {
#pragma unroll 4
          for (int c = 0; c < nc; ++c, row += cstride) {
            if (c0) __stcs(row, src0[c]);
            if (c1) __stcs(row + 32, src1[c]);
          }
        } else {
          for (int c = 0; c < nc; ++c, row += cstride)
            for (int col = lane; col < n; col += 32) __stcs(row + col - lane, rb[col * 33 + c]);
        }
      }
      __syncwarp();
    }
    if (first_row)   // a warp without rows (more warps than species)
      for (int l = 0; l < n; ++l) sEsum[l * 32 + lane] = 0.0;
    part[warp * 32 + lane] = hw_part;
    part[(NW + warp) * 32 + lane] = cpw_part;
    __syncthreads();
    // ---- pass 3: energy row, dT/dt = -sum_k H_k wdot_k / D (quotient rule) --------------------------
    {
      double hw = 0.0, cpw = 0.0;
      for (int w = 0; w < NW; ++w) { hw += part[w * 32 + lane]; cpw += part[(NW + w) * 32 + lane]; }
      const double invD = 1.0 / D, Tdot = -hw * invD;
      const double *es = scr + (size_t)4 * R * 32 + (size_t)2 * S * 32;
      double *erow = smem;          // row buffer 0 as the energy row [n][33]; its owner is past the barrier
      for (int col = warp; col < n; col += NW) {
        double hj = 0.0;
        for (int w = 0; w < NW; ++w) hj += __ldcg(es + ((size_t)w * n + col) * 32 + lane);
        double v;
        if (col < S) {
          const double iwc = __ldg(t.invW + col);
          const double dDl = rho * __ldcg(sCp + col * 32 + lane) * iwc - D * iwc * invS;
          v = -hj * invD - Tdot * dDl * invD;
        } else {
          v = -(cpw + hj) * invD - Tdot * dDdT * invD;
        }
        erow[col * 33 + lane] = v;
      }
      __syncthreads();
      for (int c = warp; c < 32; c += NW) {
        if (cell0 + c >= N) continue;
        double *row = Jg + ((size_t)(cell0 + c) * n + S) * n;
        for (int col = lane; col < n; col += 32) __stcs(row + col, erow[col * 33 + c]);
      }
    }
    __syncthreads();   // the row buffers and the scratch are rewritten by the next tile
  }
}
