// ck_jacj.cu -- host side of the mechanism-specialised Jacobian kernel (ck_jacj_kernel.cuh):
// generates the unique code (reaction walk, column walk, one case per row of J) into the kernel
// text, compiles it with NVRTC (ck_jit.cu), builds the tables of the dense part and launches.
// The reaction order, the folded rate rows and the M = C E fragments are the source-term
// kernel's (ck_api.cu: finalize_jit), so both kernels agree on what "reaction jj" is.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <sstream>
#include <string>
#include <vector>

#include "ck_internal.h"

namespace ck {

namespace {

const char *kJacjText =
#include "ck_jacj_source.inc"
    ;

struct CjCoef { double dnu; int tb, pad; };

// must match CjParams in ck_jacj_kernel.cuh field for field
struct JacjParams {
  const double *eff_frag, *tab, *thermo, *logtab, *bfrag;
  double *scratch;
  const double *T, *P, *Y;
  double *J;
  long long N;
  int tile_cells;
};

std::string lit(double v) {
  char buf[40];
  std::snprintf(buf, sizeof buf, "%.17g", v);
  std::string s(buf);
  if (s.find_first_of(".eEni") == std::string::npos) s += ".0";
  return s;
}

// acc = acc + c * v as source text, c a literal
std::string fma_line(const std::string &acc, double c, const std::string &v) {
  if (c == 1.0) return acc + " += " + v + ";";
  if (c == -1.0) return acc + " -= " + v + ";";
  return acc + " = fma(" + lit(c) + ", " + v + ", " + acc + ");";
}

std::string gather_expr(const std::vector<std::pair<int, double>> &side) {
  if (side.empty()) return "0.0";
  std::string e;
  for (size_t i = 0; i < side.size(); ++i) {
    const std::string c = "CJ_LNC(" + std::to_string(side[i].first) + ")";
    const double nu = side[i].second;
    if (i == 0) e = (nu == 1.0) ? c : (lit(nu) + " * " + c);
    else e = (nu == 1.0) ? (e + " + " + c) : ("fma(" + lit(nu) + ", " + c + ", " + e + ")");
  }
  return e;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (libck.so does not link libcuda)
typedef CUresult (*TmapEncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                 const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                 CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
TmapEncodeFn tmap_encoder() {
  static TmapEncodeFn fn = [] {
    void *f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      f = nullptr;
    cudaGetLastError();
    return (TmapEncodeFn)f;
  }();
  return fn;
}

}  // namespace

struct JacJit {
  cudaLibrary_t lib = nullptr;
  cudaKernel_t kernel = nullptr;
  JacjParams prm{};
  void *d_blob = nullptr;
  double *d_scratch = nullptr;
  int threads = 0, grid_max = 1, n1 = 0, bulk = 0, device = 0;
  size_t smem = 0, scr_rows = 0;
  // until the first ck_jacobian call: the generated text and the host copies of the tables
  std::string src, error;
  std::vector<double> tab16, bfrag;
  bool ready = false;
  int env_tile = 0;            // CK_JACJ_TILE at create time (0 = balanced tiles)
  std::mutex mu;
};

// Returns "" on success (*out set), or the reason the kernel is not available for this mechanism
// (*out NULL; never an error: the table-driven kernels remain).
std::string jacj_create(const ck_mech_desc *d, const JitSpec &spec, const std::vector<double> &tab10,
                        const double *d_thermo, const double *d_logtab, const double *d_eff_frag, int device,
                        int num_sms, size_t smem_blk, JacJit **out) {
  *out = nullptr;
  const int S = spec.S, RP = spec.R, R = d->n_reactions, B = spec.block;
  if (spec.kc_ann || spec.prec != 0) return "approximate-ANN Kc / reduced precision";
  if (!spec.perm.empty() || spec.pair) return "species permuted (accumulators do not fit registers)";
  if (S > 53) return "S > 53: two columns of register accumulators do not fit";
  if (spec.n_m > 640) return "too many third-body reactions for the constant-bank k-slot tables";
  if ((int)spec.rxn.size() != RP || RP % B) return "inconsistent reaction list";
  const int n_ranges = spec.n_ranges, nblk = RP / B, n1 = S + 1;
  if (spec.tab_ranges != n_ranges || spec.row != 10) return "rate table layout";
  const int ntl = (S + 7) / 8;
  int ost = std::max(n1, 8 * ntl);
  while (ost % 4 != 2) ++ost;                      // rows 16-byte aligned, 128-bit row accesses conflict-free
  const int hint = std::getenv("CK_JACJ_HINT") ? std::atoi(std::getenv("CK_JACJ_HINT")) : 1;
  // how rows leave: 2 tensor copies (needs the driver's cuTensorMapEncodeTiled), 1 bulk copies per cell, 0 plain stores
  int bulk = (n1 % 2 == 0) ? 2 : 0;
  if (const char *e = std::getenv("CK_JACJ_BULK")) bulk = std::min(bulk, std::max(0, std::atoi(e)));
  if (bulk == 2 && device >= 0 && !tmap_encoder()) bulk = 1;
  if (bulk == 2) ost = n1;

  // ---- launch shape: the most warps (tile = 32 cells per warp) whose tile fits shared memory ----
  int warps = 0;
  size_t smem = 0;
  // (registers: two columns of accumulators, 4 S, and about 60 beside them at the least; 512 threads x 128
  //  registers when that fits, else 256 x 255)
  int w_max = (4 * S + 60 <= 128) ? 16 : 8;
  if (const char *e = std::getenv("CK_JACJ_WARPS")) w_max = std::min(w_max, std::max(1, std::atoi(e)));
  for (int w = w_max; w >= 1; --w) {
    const size_t ovl = std::max((size_t)n_ranges * RP * 16 + 384, (size_t)w * 32 * ost);
    const size_t doubles = ((size_t)S * (32 * w + 8) + (size_t)n_ranges * S * 12 + 15) / 16 * 16 + ovl;
    if (doubles * 8 + 64 <= smem_blk) { warps = w; smem = doubles * 8; break; }
  }
  if (!warps) return "tile does not fit shared memory";
  const int NT = 32 * warps;
  const int env_chunk = std::getenv("CK_JACJ_CHUNK") ? std::atoi(std::getenv("CK_JACJ_CHUNK")) : 8;
  const int pf_rows = std::getenv("CK_JACJ_PFROWS") ? std::atoi(std::getenv("CK_JACJ_PFROWS")) : 0;
  const int pf_l1 = std::getenv("CK_JACJ_PFL1") ? std::atoi(std::getenv("CK_JACJ_PFL1")) : 8;

  // ---- rate table rows of 16 doubles ----------------------------------------------------------
  std::vector<double> range_T = spec.range_T;
  std::vector<int> rank(S);
  for (int k = 0; k < S; ++k)
    rank[k] = (int)(std::lower_bound(range_T.begin(), range_T.end(), d->T_mid[k]) - range_T.begin());
  std::vector<double> tab16((size_t)n_ranges * RP * 16, 0.0);
  for (int rg = 0; rg < n_ranges; ++rg)
    for (int jj = 0; jj < RP; ++jj) {
      const double *src = &tab10[((size_t)rg * RP + jj) * 10];
      double *row = &tab16[((size_t)rg * RP + jj) * 16];
      for (int i = 0; i < 10; ++i) row[i] = src[i];
      const JitReaction &r = spec.rxn[jj];
      long double ordf = 0, ordr = 0, da1 = 0;
      for (const auto &e : r.reac) ordf += e.second;
      for (const auto &e : r.prod) ordr += e.second;
      for (const auto &e : r.net) {
        const int k = e.first;
        const double *a = (rg > rank[k]) ? d->nasa_hi + 7 * k : d->nasa_lo + 7 * k;
        da1 += (long double)e.second * a[0];
      }
      row[10] = (double)ordf; row[11] = (double)ordr;
      row[12] = 2.0 * row[7]; row[13] = 3.0 * row[8]; row[14] = 4.0 * row[9];
      row[15] = (double)da1;
    }

  // ---- dense part: k-steps of 4 third-body / falloff reactions per row, E gathered as B fragments ----
  std::vector<int> ks_start(S + 2, 0);
  std::vector<CjCoef> coef;
  std::vector<double> bfrag;
  for (int i = 0; i <= S; ++i) {
    ks_start[i] = (int)coef.size() / 4;
    std::vector<std::pair<int, double>> tbs;   // (padded reaction index, coefficient)
    for (int jj = 0; jj < RP; ++jj) {
      const JitReaction &r = spec.rxn[jj];
      if (r.index < 0 || r.m_slot < 0) continue;
      if (i == S) { tbs.emplace_back(jj, 1.0); continue; }
      for (const auto &e : r.net)
        if (e.first == i && e.second != 0.0) tbs.emplace_back(jj, e.second);
    }
    const int nks = ((int)tbs.size() + 3) / 4;
    for (int ks = 0; ks < nks; ++ks) {
      const size_t b0 = bfrag.size();
      bfrag.resize(b0 + (size_t)ntl * 32, 0.0);
      for (int qq = 0; qq < 4; ++qq) {
        const int kk = 4 * ks + qq;
        if (kk >= (int)tbs.size()) { coef.push_back(CjCoef{0.0, -1, 0}); continue; }
        const JitReaction &r = spec.rxn[tbs[kk].first];
        coef.push_back(CjCoef{tbs[kk].second, r.m_slot, 0});
        for (int nt = 0; nt < ntl; ++nt)
          for (int gg = 0; gg < 8; ++gg) {
            const int l = 8 * nt + gg;
            if (l < S)
              bfrag[b0 + (size_t)nt * 32 + gg * 4 + qq] =
                  (d->eff ? d->eff[(size_t)l * R + r.index] : 1.0) / d->mol_weight[l];
          }
      }
    }
  }
  ks_start[S + 1] = (int)coef.size() / 4;
  // k-steps of a species row whose A values are loaded ahead of the sparse part: the longest row's, at most 4
  int kp = 1;
  for (int i = 0; i < S; ++i) kp = std::max(kp, ks_start[i + 1] - ks_start[i]);
  kp = std::min(kp, 4);
  if (const char *e = std::getenv("CK_JACJ_KP")) kp = std::max(1, std::atoi(e));
  if (coef.empty()) coef.push_back(CjCoef{0.0, -1, 0});
  if (bfrag.empty()) bfrag.push_back(0.0);

  // Dead scratch lines are dropped from L2 (discard.global.L2) where the scratch of all blocks fits L2: then
  // they would otherwise be written back behind the output stream (S=9: 2.18 -> 1.23 GB of DRAM traffic per
  // 2^20 cells); where it does not fit (S=53: 457 MB) the lines are gone before they die and the discards only cost time
  int discard = ((size_t)num_sms * ((size_t)4 * RP + (size_t)2 * spec.n_mb * 8 + (size_t)3 * S) * NT * 8 <= ((size_t)100 << 20)) ? 1 : 0;
  if (const char *e = std::getenv("CK_JACJ_DISCARD")) discard = std::atoi(e) != 0;
  // ---- source text -------------------------------------------------------------------------------
  std::ostringstream o;
  o << "#define CJ_S " << S << "\n#define CJ_R " << RP << "\n#define CJ_NT " << NT << "\n#define CJ_NRANGES " << n_ranges
    << "\n#define CJ_B " << B << "\n#define CJ_NBLK " << nblk << "\n#define CJ_G_TB0 " << spec.group_end[1]
    << "\n#define CJ_G_FO0 " << spec.group_end[3] << "\n#define CJ_NM " << spec.n_m << "\n#define CJ_NMB " << spec.n_mb
    << "\n#define CJ_NFO " << spec.n_fo << "\n#define CJ_NTL " << ntl << "\n#define CJ_OST " << ost
    << "\n#define CJ_BULK " << bulk << "\n#define CJ_HINT " << hint << "\n#define CJ_MH " << (std::getenv("CK_JACJ_MH") ? std::atoi(std::getenv("CK_JACJ_MH")) : 4) << "\n#define CJ_KP " << kp << "\n#define CJ_PREF " << (std::getenv("CK_JACJ_PREF") ? std::atoi(std::getenv("CK_JACJ_PREF")) : 6) << "\n#define CJ_DISCARD " << discard << "\n#define CJ_TIMING " << (std::getenv("CK_JACJ_TIMING") ? 1 : 0) << "\n#define CJ_NOALLOC " << (std::getenv("CK_JACJ_NOALLOC") ? std::atoi(std::getenv("CK_JACJ_NOALLOC")) : 0) << "\n#define CJ_STAGGER " << (std::getenv("CK_JACJ_STAGGER") ? std::atoi(std::getenv("CK_JACJ_STAGGER")) : 0) << "\n#define CJ_EXP " << (std::getenv("CK_JACJ_EXP") ? std::atoi(std::getenv("CK_JACJ_EXP")) : 0) << "\n";
  auto emit = [&](const char *name, const std::vector<double> &v) {
    o << "__constant__ double " << name << "[" << (v.empty() ? 1 : v.size()) << "] = {";
    for (size_t i = 0; i < v.size(); ++i) o << (i ? "," : "") << (i % 6 == 0 ? "\n  " : " ") << lit(v[i]);
    if (v.empty()) o << "0.0";
    o << "};\n";
  };
  emit("ck_c_rangeT", spec.range_T);
  emit("ck_c_falloff", spec.falloff);
  {
    std::vector<double> iw(S);
    for (int k = 0; k < S; ++k) iw[k] = 1.0 / d->mol_weight[k];
    emit("cj_c_invW", iw);
  }
  o << "__constant__ int cj_c_ks[" << S + 2 << "] = {";
  for (int i = 0; i < S + 2; ++i) o << (i ? ", " : "") << ks_start[i];
  o << "};\n";
  {
    std::vector<double> dn(coef.size());
    for (size_t i = 0; i < coef.size(); ++i) dn[i] = coef[i].dnu;
    emit("cj_c_dnu", dn);
    o << "__constant__ int cj_c_tb[" << coef.size() << "] = {";
    for (size_t i = 0; i < coef.size(); ++i) o << (i ? "," : "") << (i % 24 == 0 ? "\n  " : " ") << std::max(coef[i].tb, 0);
    o << "};\n";
  }
  const std::string text(kJacjText);
  const std::string marker = "//@@CJ_GENERATED@@";
  const size_t at = text.find(marker);
  o << text.substr(0, at);

  const char *names[6] = {"cj_core<0, 1>", "cj_core<0, 0>", "cj_core<1, 1>", "cj_core<1, 0>", "cj_core<2, 1>", "cj_core<2, 0>"};
  // P1: one switch case per loop trip: energy-row scatters of the previous block, gathers of this one
  o << "__device__ __forceinline__ void cj_reactions(const CjCtx &x, double (&er)[CJ_S], double (&sc)[4]) {\n"
    << "  double gf[CJ_B], gr[CJ_B], ha[CJ_B], hb[CJ_B];\n"
    << "#pragma unroll 1\n  for (int blk = 0; blk <= CJ_NBLK; ++blk) {\n    switch (blk) {\n";
  for (int k = 0; k <= nblk; ++k) {
    o << "      case " << k << ":\n";
    if (k > 0)
      for (int bb = 0; bb < B; ++bb) {
        const JitReaction &r = spec.rxn[(size_t)(k - 1) * B + bb];
        for (const auto &e : r.reac)
          o << "        " << fma_line("er[" + std::to_string(e.first) + "]", e.second, "ha[" + std::to_string(bb) + "]") << "\n";
        if (r.reversible)
          for (const auto &e : r.prod)
            o << "        " << fma_line("er[" + std::to_string(e.first) + "]", -e.second, "hb[" + std::to_string(bb) + "]") << "\n";
      }
    if (k < nblk)
      for (int bb = 0; bb < B; ++bb) {
        const JitReaction &r = spec.rxn[(size_t)k * B + bb];
        o << "        gf[" << bb << "] = " << gather_expr(r.reac) << ";";
        if (r.index >= 0) o << "  // reaction " << r.index;
        o << "\n        gr[" << bb << "] = " << (r.reversible ? gather_expr(r.prod) : std::string("0.0")) << ";\n";
      }
    o << "        break;\n";
  }
  o << "    }\n";
  {
    bool first = true;
    for (int g = 0; g < 6; ++g) {
      const int lo = g ? spec.group_end[g - 1] : 0;
      if (spec.group_end[g] == lo) continue;
      o << "    " << (first ? "if" : "else if") << " (blk < " << spec.group_end[g] << ") " << names[g]
        << "(x, blk, gf, gr, ha, hb, sc);\n";
      first = false;
    }
  }
  o << "  }\n}\n";
  // P1b: tc_i = sum_j dnu_ij t_j, gc_i = sum_j dnu_ij e_j
  o << "__device__ __forceinline__ void cj_columns(const CjCtx &x, double (&tc)[CJ_S], double (&gc)[CJ_S]) {\n"
    << "#pragma unroll 1\n  for (int blk = 0; blk < CJ_NBLK; ++blk) {\n    double t[CJ_B], e[CJ_B];\n"
    << "#if CJ_PREF\n    if (blk + 1 < CJ_NBLK) {\n#pragma unroll\n      for (int b = 0; b < CJ_B; ++b) CJ_PF1(&CJ_SCR2(CJ_R + (blk + 1) * CJ_B + b));\n    }\n#endif\n"
    << "#pragma unroll\n    for (int b = 0; b < CJ_B; ++b) { const double2 te = CJ_TE(blk * CJ_B + b); t[b] = te.x; e[b] = te.y; }\n"
    << "    switch (blk) {\n";
  for (int k = 0; k < nblk; ++k) {
    o << "      case " << k << ":\n";
    for (int bb = 0; bb < B; ++bb) {
      const JitReaction &r = spec.rxn[(size_t)k * B + bb];
      for (const auto &e : r.net) {
        o << "        " << fma_line("tc[" + std::to_string(e.first) + "]", e.second, "t[" + std::to_string(bb) + "]") << " "
          << fma_line("gc[" + std::to_string(e.first) + "]", e.second, "e[" + std::to_string(bb) + "]") << "\n";
      }
    }
    o << "        break;\n";
  }
  o << "    }\n  }\n}\n";
  // P2: sparse part of row i: for every reaction with dnu_ij != 0 the entries dnu_ij nu'_lj a_j - dnu_ij nu''_lj b_j
  o << "__device__ __forceinline__ void cj_row_sparse(const CjCtx &x, const int i, double (&acc)[CJ_S]) {\n  switch (i) {\n";
  const int chunk = std::max(1, env_chunk);
  auto row_list = [&](int i) {
    std::vector<std::pair<int, double>> rows;   // (reaction, dnu) of row i
    for (int jj = 0; jj < RP; ++jj) {
      const JitReaction &r = spec.rxn[jj];
      if (r.index < 0) continue;
      double dnu = 0.0;
      for (const auto &e : r.net) if (e.first == i) dnu = e.second;
      if (dnu != 0.0) rows.emplace_back(jj, dnu);
    }
    return rows;
  };
  for (int i = 0; i < S; ++i) {
    o << "    case " << i << ": {\n";
    const std::vector<std::pair<int, double>> rows = row_list(i);
    // the next row's (a, b) towards L2 (the scratch of the cells in flight does not stay resident)
    if (pf_rows > 0 && i + pf_rows < S) {
      for (const auto &rj : row_list(i + pf_rows)) {
        o << "      CJ_PFAB(" << rj.first << ");\n";
      }
    }
    // the first (a, b) pairs of the next row towards L1: its first loads then do not wait for L2 / DRAM
    if (pf_l1 > 0 && i + 1 < S) {
      const std::vector<std::pair<int, double>> nx = row_list(i + 1);
      for (size_t c = 0; c < nx.size() && (int)c < pf_l1; ++c) o << "      CJ_PF1(&CJ_SCR2(" << nx[c].first << "));\n";
    }
    // the loads of a chunk of reactions first (they keep their order), then the chunk's FMAs
    for (size_t c0 = 0; c0 < rows.size(); c0 += chunk) {
      const size_t c1 = std::min(rows.size(), c0 + chunk);
      o << "      {\n";
      for (size_t c = c0; c < c1; ++c) {
        const int jj = rows[c].first;
        o << "        const double2 ab" << jj << " = CJ_AB(" << jj << ");\n";
      }
      for (size_t c = c0; c < c1; ++c) {
        const int jj = rows[c].first;
        const double dnu = rows[c].second;
        const JitReaction &r = spec.rxn[jj];
        for (const auto &e : r.reac) o << "        " << fma_line("acc[" + std::to_string(e.first) + "]", dnu * e.second, "ab" + std::to_string(jj) + ".x") << "\n";
        if (r.reversible)
          for (const auto &e : r.prod) o << "        " << fma_line("acc[" + std::to_string(e.first) + "]", -dnu * e.second, "ab" + std::to_string(jj) + ".y") << "\n";
      }
      o << "      }\n";
    }
    o << "    } break;\n";
  }
  o << "  }\n}\n";
  o << text.substr(at + marker.size());
  const std::string src = o.str();
  if (const char *e = std::getenv("CK_JACJ_DUMP")) {
    if (FILE *f = std::fopen(e, "w")) {
      std::fwrite(src.data(), 1, src.size(), f);
      std::fclose(f);
    }
  }
  if (device < 0) return "source only";

  // Everything that needs the device -- compiling the text, loading it, the tables and the scratch of
  // the cells in flight (hundreds of MB) -- waits for the first ck_jacobian call (jacj_ensure).
  JacJit *jj = new JacJit;
  jj->src = src;
  jj->tab16.swap(tab16);
  jj->bfrag.swap(bfrag);
  jj->scr_rows = (size_t)4 * RP + (size_t)2 * spec.n_mb * 8 + (size_t)3 * S;
  jj->device = device;
  if (const char *e = std::getenv("CK_JACJ_TILE")) jj->env_tile = std::atoi(e);
  jj->threads = NT; jj->grid_max = num_sms; jj->smem = smem; jj->n1 = n1; jj->bulk = bulk;
  jj->prm.eff_frag = d_eff_frag; jj->prm.thermo = d_thermo; jj->prm.logtab = d_logtab;
  *out = jj;
  return "";
}

// Compiles and loads the kernel, uploads its tables and allocates the scratch, once.  Returns "" or
// the error text (then, and on every later call, the caller falls back to the table-driven kernels).
std::string jacj_ensure(JacJit *jj) {
  std::lock_guard<std::mutex> lock(jj->mu);
  if (jj->ready) return "";
  if (!jj->error.empty()) return jj->error;
  // (tables and scratch belong on the handle's device, whatever device is current in this thread)
  struct DeviceGuard {
    int prev = -1, want;
    explicit DeviceGuard(int w) : want(w) { if (cudaGetDevice(&prev) == cudaSuccess && prev != want) cudaSetDevice(want); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
  } guard(jj->device);
  std::vector<char> cubin;
  cudaError_t ce = cudaSuccess;
  for (int attempt = 0; attempt < 2; ++attempt) {
    const std::string err = jit_compile(jj->src, &cubin, attempt == 0);
    if (!err.empty()) return jj->error = err;
    ce = cudaLibraryLoadData(&jj->lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (ce == cudaSuccess) break;
    cudaGetLastError();
    jj->lib = nullptr;
  }
  if (ce == cudaSuccess) ce = cudaLibraryGetKernel(&jj->kernel, jj->lib, "ck_jacobian_jit");
  if (ce == cudaSuccess)
    ce = cudaKernelSetAttributeForDevice(jj->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)jj->smem, jj->device);
  size_t o_tab = 0, o_bf = 0, bytes = 0;
  auto place = [&](size_t n) { const size_t off = (bytes + 255) / 256 * 256; bytes = off + n; return off; };
  o_tab = place(jj->tab16.size() * 8); o_bf = place(jj->bfrag.size() * 8);
  if (ce == cudaSuccess) ce = cudaMalloc(&jj->d_blob, bytes);
  if (ce == cudaSuccess) ce = cudaMemcpy((char *)jj->d_blob + o_tab, jj->tab16.data(), jj->tab16.size() * 8, cudaMemcpyHostToDevice);
  if (ce == cudaSuccess) ce = cudaMemcpy((char *)jj->d_blob + o_bf, jj->bfrag.data(), jj->bfrag.size() * 8, cudaMemcpyHostToDevice);
  if (ce == cudaSuccess) ce = cudaMalloc((void **)&jj->d_scratch, (size_t)jj->grid_max * jj->scr_rows * jj->threads * sizeof(double));
  if (ce != cudaSuccess) {
    jj->error = std::string("specialised Jacobian kernel: ") + cudaGetErrorString(ce);
    cudaGetLastError();
    if (jj->d_blob) { cudaFree(jj->d_blob); jj->d_blob = nullptr; }
    if (jj->lib) { cudaLibraryUnload(jj->lib); jj->lib = nullptr; }
    return jj->error;
  }
  jj->prm.tab = (const double *)((char *)jj->d_blob + o_tab);
  jj->prm.bfrag = (const double *)((char *)jj->d_blob + o_bf);
  jj->prm.scratch = jj->d_scratch;
  std::string().swap(jj->src);
  std::vector<double>().swap(jj->tab16);
  std::vector<double>().swap(jj->bfrag);
  jj->ready = true;
  return "";
}

void jacj_destroy(JacJit *jj) {
  if (!jj) return;
  if (jj->d_blob) cudaFree(jj->d_blob);
  if (jj->d_scratch) cudaFree(jj->d_scratch);
  if (jj->lib) cudaLibraryUnload(jj->lib);
  delete jj;
}

bool jacj_failed(const JacJit *jj) { return !jj->ready && !jj->error.empty(); }
int jacj_cells(const JacJit *jj) { return jj->threads; }
bool jacj_takes(const JacJit *jj, const double *J) { return jj->bulk == 0 || ((uintptr_t)J & 15u) == 0; }

cudaError_t jacj_launch(const JacJit *jj, const double *T, const double *P, const double *Y, int64_t N, double *J,
                        cudaStream_t stream) {
  JacjParams prm = jj->prm;
  prm.T = T; prm.P = P; prm.Y = Y; prm.J = J; prm.N = N;
  // balanced tiles, as for the source-term kernel: the fewest waves of full tiles, then the tile size
  // (a multiple of 32) that spreads the cells evenly over grid x waves
  const int64_t per_wave = (int64_t)jj->grid_max * jj->threads;
  const int64_t waves = (N + per_wave - 1) / per_wave;
  int64_t tc = (N + waves * jj->grid_max - 1) / (waves * jj->grid_max);
  tc = std::min<int64_t>(jj->threads, (tc + 31) / 32 * 32);
  // (test knob: CK_JACJ_TILE, read at ck_mech_create, forces the tile size; a cell's bits do not depend on it)
  if (jj->env_tile) tc = std::min<int64_t>(jj->threads, std::max(32, jj->env_tile / 32 * 32));
  prm.tile_cells = (int)tc;
  const int64_t tiles = (N + tc - 1) / tc;
  const int grid = (int)std::min<int64_t>(tiles, jj->grid_max);
  // J as a rank-3 tensor (column, row, cell) of doubles; a copy stores one row of 32 cells
  alignas(64) CUtensorMap tmap;
  std::memset(&tmap, 0, sizeof tmap);
  if (jj->bulk == 2) {
    const cuuint64_t n = (cuuint64_t)jj->n1;
    const cuuint64_t dims[3] = {n, n, (cuuint64_t)N}, strides[2] = {n * 8, n * n * 8};
    const cuuint32_t box[3] = {(cuuint32_t)n, 1, 32}, estr[3] = {1, 1, 1};
    const CUresult r = tmap_encoder()(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void *)J, dims, strides, box, estr,
                                      CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                      CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  }
  void *args[] = {&prm, &tmap};
  return cudaLaunchKernel((const void *)jj->kernel, dim3(grid), dim3(jj->threads), args, jj->smem, stream);
}

}  // namespace ck
