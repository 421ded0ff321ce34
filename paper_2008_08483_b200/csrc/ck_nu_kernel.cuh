// ck_nu_kernel.cuh -- the source term of a SMALL mechanism with every contraction of the paper's
// matrix form on the FP64 tensor-core instruction (DMMA.8x8x4), compiled by NVRTC with the
// sizes as macros.  This is the "tiled contraction path" of the north_star, built where the
// stoichiometric matrices are densest (S=9/R=21: nu'' - nu' is 61 % dense) to be
// measured against the fused sparse kernel of ck_jit_kernel.cuh.
//
//   log Q_f = log C nu' + log K_f,  log Q_r = log C nu'' + log K_r     Eq. 4
//   M = C E                                                             Sec. 2.4
//   Omega = Q_net nu^T                                                  Eq. 2
//
// A warp owns 32 cells.  The three products of a tile of 8 reactions are formed as
// [32 cells x NU_SP4 species] x [NU_SP4 x 8] DMMA sweeps from the cells' ln C and C columns in
// shared memory; the result fragments (lane g*4+q holds cells 8 mt + g, reactions 8 nt + 2 q + e)
// are the layout in which the rate layers then run -- a lane evaluates Eq. 6, 7/11, the
// activations and the third-body / falloff factor for ITS (cell, reaction) pairs -- and the net
// rates, still in that layout, are exactly the A fragments of the Eq. 2 product when its k-slot
// (k-step 2 nt + e, lane q) is made to mean reaction 8 nt + 2 q + e: the host lays the nu^T
// fragments out that way, so no value ever changes lanes.  wdot leaves the tensor layout through
// a shared-memory transpose into the thread <-> cell layout of the prologue and epilogue.
//
// Macros from the host: NU_S, NU_R (reaction slots, a multiple of 8), NU_THREADS, NU_NRANGES,
// CK_LUT_REP = 1, CK_KCONST, CK_PREC = 0.
// Reaction slot s = 8 nt + 2 q + e; tables are indexed by slot (null slots: rate ~ 0).

#define NU_RU 8314.46261815324
#define NU_CFLOOR 1e-300
#define NU_SP4 ((NU_S + 3) / 4 * 4)
#define NU_KS (NU_SP4 / 4)
#define NU_NT (NU_R / 8)
#define NU_NT2 ((NU_S + 7) / 8)
#define NU_LD (NU_THREADS + 8)
#define NU_TROW 12
// shared memory, doubles: lnc[NU_SP4][LD] | cc[NU_SP4][LD] (wdot rows [8 NU_NT2][LD] alias lnc) |
// exp table 128 | log table 256 | thermo[NRANGES][S][12] | tab[NRANGES][R][10] | fo[R][8] |
// b1f, b1r, be [NT][KS][32] each | b2[NT2][2 NT][32] | flags[R] (as doubles: type + 8 * reversible)
#define NU_ROWS (2 * (NU_SP4 > 8 * NU_NT2 ? NU_SP4 : 8 * NU_NT2))
#define NU_FRAG1 (NU_NT * NU_KS * 32)
#define NU_FRAG2 (NU_NT2 * 2 * NU_NT * 32)
#define NU_SMEM_DOUBLES (NU_ROWS * NU_LD + 128 + 256 + NU_NRANGES * NU_S * NU_TROW + NU_NRANGES * NU_R * 10 + NU_R * 8 + 3 * NU_FRAG1 + NU_FRAG2 + NU_R)

struct NuParams {
  const double *thermo;    // [NRANGES][S][12] (as in ck_jit_kernel.cuh)
  const double *logtab;    // [128][2]
  const double *tab;       // [NRANGES][R][10] rate rows by slot
  const double *fo;        // [R][8] falloff rows by slot
  const double *b1f, *b1r, *be;   // nu', nu'', E as B fragments [NT][KS][32]
  const double *b2;        // (nu'' - nu')^T as B fragments [NT2][2 NT][32], k-slot = reaction slot
  const double *flags;     // [R] type + 8 * reversible
  const double *rangeT;    // [NRANGES - 1]
  const double *T, *P, *Y;
  double *wdot, *dTdt;
  long long N;
};

//@@CK_MATH@@

__device__ __forceinline__ void nu_dmma(double &c0, double &c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

extern "C" __global__ void __launch_bounds__(NU_THREADS) ck_source_terms_nu(const NuParams p) {
  extern __shared__ __align__(16) double smem[];
  const int tid = threadIdx.x, lane = tid & 31, g = lane >> 2, q = lane & 3;
  double *lnc = smem, *cc = smem + (NU_ROWS / 2) * NU_LD;
  double *lut = smem + NU_ROWS * NU_LD, *logtab = lut + 128, *thermo = logtab + 256;
  double *tab = thermo + NU_NRANGES * NU_S * NU_TROW, *fo = tab + NU_NRANGES * NU_R * 10;
  double *b1f = fo + NU_R * 8, *b1r = b1f + NU_FRAG1, *be = b1r + NU_FRAG1, *b2 = be + NU_FRAG1;
  double *flags = b2 + NU_FRAG2;
  for (int i = tid; i < 128; i += NU_THREADS) lut[i] = exp2((double)i * (1.0 / 128.0));
  for (int i = tid; i < 256; i += NU_THREADS) logtab[i] = p.logtab[i];
  for (int i = tid; i < NU_NRANGES * NU_S * NU_TROW; i += NU_THREADS) thermo[i] = p.thermo[i];
  for (int i = tid; i < NU_NRANGES * NU_R * 10; i += NU_THREADS) tab[i] = p.tab[i];
  for (int i = tid; i < NU_R * 8; i += NU_THREADS) fo[i] = p.fo[i];
  for (int i = tid; i < NU_FRAG1; i += NU_THREADS) { b1f[i] = p.b1f[i]; b1r[i] = p.b1r[i]; be[i] = p.be[i]; }
  for (int i = tid; i < NU_FRAG2; i += NU_THREADS) b2[i] = p.b2[i];
  for (int i = tid; i < NU_R; i += NU_THREADS) flags[i] = p.flags[i];
  __syncthreads();

  // this warp's columns: cell of this thread at [k * NU_LD + tid], the warp's 32 cells at the
  // warp's base; nothing below crosses warps
  double *mylnc = lnc + tid, *mycc = cc + tid;
  const double *wlnc = lnc + (tid & ~31) + g, *wcc = cc + (tid & ~31) + g;
  const long long n_chunks = (p.N + 31) / 32;
  const long long warp0 = (long long)blockIdx.x * (NU_THREADS / 32) + (tid >> 5);
  const long long warp_stride = (long long)gridDim.x * (NU_THREADS / 32);
  for (long long chunk = warp0; chunk < n_chunks; chunk += warp_stride) {
    const long long i = chunk * 32 + lane;
    const bool valid = i < p.N;
    const long long ii = valid ? i : p.N - 1;
    // ---- thread <-> cell prologue: features, Y/W, cp, rho, C and ln C columns --------------------
    const double T = __ldcs(p.T + ii), P = __ldcs(p.P + ii);
    const double lnT = ck_log(T, logtab), invT = 1.0 / T;
    int range = 0;
#pragma unroll
    for (int d = 0; d < NU_NRANGES - 1; ++d) range += (T > p.rangeT[d]) ? 1 : 0;
    const double *th = thermo + range * (NU_S * NU_TROW);
    double inv_Wmix = 0.0, cp_sum = 0.0;
#pragma unroll
    for (int k = 0; k < NU_S; ++k) {
      const double2 a01 = *(const double2 *)(th + k * NU_TROW), a23 = *(const double2 *)(th + k * NU_TROW + 2);
      const double2 a4w = *(const double2 *)(th + k * NU_TROW + 4);
      const double yw = fmax(__ldcs(p.Y + (size_t)k * p.N + ii), 0.0) * a4w.y;   // Y <= 0: absent (reading Q9)
      mycc[k * NU_LD] = yw;
      inv_Wmix += yw;
      cp_sum = fma(yw, fma(fma(fma(fma(a4w.x, T, a23.y), T, a23.x), T, a01.y), T, a01.x), cp_sum);
    }
    const double rho = P / (NU_RU * T * inv_Wmix);
#pragma unroll
    for (int k = 0; k < NU_S; ++k) {
      const double c = rho * mycc[k * NU_LD];
      mycc[k * NU_LD] = c;                                    // M = C E takes the unfloored C (a zero stays zero)
      mylnc[k * NU_LD] = ck_log(fmax(c, NU_CFLOOR), logtab);   // Eq. 4 takes ln of the floored C
    }
#pragma unroll
    for (int k = NU_S; k < NU_SP4; ++k) { mycc[k * NU_LD] = 0.0; mylnc[k * NU_LD] = 0.0; }
    // features of the four cells whose fragments this lane holds (cells 8 mt + g of the warp)
    double fT[4], flnT[4], finvT[4];
    int frange[4];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt) {
      fT[mt] = __shfl_sync(0xffffffffu, T, 8 * mt + g);
      flnT[mt] = __shfl_sync(0xffffffffu, lnT, 8 * mt + g);
      finvT[mt] = __shfl_sync(0xffffffffu, invT, 8 * mt + g);
      frange[mt] = __shfl_sync(0xffffffffu, range, 8 * mt + g);
    }
    __syncwarp();   // the columns were written by the cells' own threads

    // ---- the contractions and the rate layers, one tile of 8 reactions at a time -----------------
    double w[NU_NT2][4][2];
#pragma unroll
    for (int n2 = 0; n2 < NU_NT2; ++n2)
#pragma unroll
      for (int mt = 0; mt < 4; ++mt) w[n2][mt][0] = w[n2][mt][1] = 0.0;
#pragma unroll 1
    for (int nt = 0; nt < NU_NT; ++nt) {
      double gf[4][2], gr[4][2], mm[4][2];
#pragma unroll
      for (int mt = 0; mt < 4; ++mt) gf[mt][0] = gf[mt][1] = gr[mt][0] = gr[mt][1] = mm[mt][0] = mm[mt][1] = 0.0;
#pragma unroll
      for (int ks = 0; ks < NU_KS; ++ks) {
        const double bf = b1f[(nt * NU_KS + ks) * 32 + lane], br = b1r[(nt * NU_KS + ks) * 32 + lane];
        const double bm = be[(nt * NU_KS + ks) * 32 + lane];
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) {
          const double al = wlnc[(4 * ks + q) * NU_LD + 8 * mt], ac = wcc[(4 * ks + q) * NU_LD + 8 * mt];
          nu_dmma(gf[mt][0], gf[mt][1], al, bf);     // log C nu'
          nu_dmma(gr[mt][0], gr[mt][1], al, br);     // log C nu''
          nu_dmma(mm[mt][0], mm[mt][1], ac, bm);     // C E
        }
      }
      // rate layers of this lane's (cell, reaction) pairs: reactions 8 nt + 2 q + e
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int slot = 8 * nt + 2 * q + e;
        const int flag = (int)flags[slot], type = flag & 7;
        const bool rev = flag >= 8;
        double Q[4];
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) {
          const double *r = tab + ((size_t)frange[mt] * NU_R + slot) * 10;
          const double2 r01 = *(const double2 *)r, r23 = *(const double2 *)(r + 2), r45 = *(const double2 *)(r + 4);
          const double2 r67 = *(const double2 *)(r + 6), r89 = *(const double2 *)(r + 8);
          const double lkf = fma(r01.y, flnT[mt], fma(r23.x, finvT[mt], r01.x));            // Eq. 6
          const double poly = fma(fma(fma(r89.y, fT[mt], r89.x), fT[mt], r67.y), fT[mt], r67.x);
          const double lkr = fma(poly, fT[mt], fma(r45.x, flnT[mt], fma(r45.y, finvT[mt], r23.y)));   // Eq. 7, 11
          double v = ck_exp(lkf + gf[mt][e], lut);                                           // Eq. 4
          const double qr = ck_exp(lkr + gr[mt][e], lut);
          v -= rev ? qr : 0.0;
          Q[mt] = v;
          gf[mt][e] = lkf;   // (kept for the falloff layer)
        }
        if (type == 1) {
#pragma unroll
          for (int mt = 0; mt < 4; ++mt) Q[mt] *= mm[mt][e];
        } else if (type >= 2) {
          const double *f = fo + slot * 8;
#pragma unroll
          for (int mt = 0; mt < 4; ++mt)
            Q[mt] *= ck_falloff<true>(f, flnT[mt], finvT[mt], fT[mt], gf[mt][e], mm[mt][e], lut, logtab);
        }
        // Eq. 2: this lane's Q values are the A fragments of k-step 2 nt + e
#pragma unroll
        for (int n2 = 0; n2 < NU_NT2; ++n2) {
          const double bw = b2[(n2 * 2 * NU_NT + 2 * nt + e) * 32 + lane];
#pragma unroll
          for (int mt = 0; mt < 4; ++mt) nu_dmma(w[n2][mt][0], w[n2][mt][1], Q[mt], bw);
        }
      }
    }
    // ---- wdot out of the tensor layout: rows [species][cell] over the (dead) ln C columns ---------
    __syncwarp();
    double *wrow = lnc + (tid & ~31) + g;
#pragma unroll
    for (int n2 = 0; n2 < NU_NT2; ++n2)
#pragma unroll
      for (int mt = 0; mt < 4; ++mt) {
        wrow[(8 * n2 + 2 * q) * NU_LD + 8 * mt] = w[n2][mt][0];
        wrow[(8 * n2 + 2 * q + 1) * NU_LD + 8 * mt] = w[n2][mt][1];
      }
    __syncwarp();
    // ---- thread <-> cell epilogue: energy term, coalesced stores ---------------------------------
    double hw = 0.0;
#pragma unroll
    for (int k = 0; k < NU_S; ++k) {
      const double2 *a = (const double2 *)(th + k * NU_TROW + 6);
      const double2 a01 = a[0], a23 = a[1], a45 = a[2];
      const double h_RT = fma(a45.y, invT, fma(fma(fma(fma(a45.x, T, a23.y), T, a23.x), T, a01.y), T, a01.x));
      const double wk = mylnc[k * NU_LD];
      hw = fma(h_RT, wk, hw);
      if (valid) __stcs(p.wdot + (size_t)k * p.N + i, wk);
    }
    if (valid) __stcs(p.dTdt + i, -(T * hw) / (rho * cp_sum));
    __syncwarp();   // the columns are rewritten by the next chunk's prologue
  }
}
