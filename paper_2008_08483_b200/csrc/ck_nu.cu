// ck_nu.cu -- host side of the all-DMMA small-mechanism kernel (ck_nu_kernel.cuh): lays nu', nu'',
// E and (nu'' - nu')^T out as DMMA.8x8x4 B fragments, compiles the kernel text for the mechanism's
// sizes with NVRTC and launches it.  Selected by CK_JIT_NU=dmma for mechanisms of at most 16
// species and 64 reactions (the contraction path measured against the sparse one).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <sstream>
#include <string>
#include <vector>

#include "ck_internal.h"

namespace ck {

namespace {
const char *kNuText =
#include "ck_nu_source.inc"
    ;

// must match NuParams in ck_nu_kernel.cuh field for field
struct NuParams {
  const double *thermo, *logtab, *tab, *fo, *b1f, *b1r, *be, *b2, *flags, *rangeT;
  const double *T, *P, *Y;
  double *wdot, *dTdt;
  long long N;
};
}  // namespace

struct NuMech {
  cudaLibrary_t lib = nullptr;
  cudaKernel_t kernel = nullptr;
  void *d_tables = nullptr;
  NuParams prm{};
  int threads = 0, grid_max = 0;
  size_t smem = 0;
};

void nu_destroy(NuMech *nm) {
  if (!nm) return;
  if (nm->lib) cudaLibraryUnload(nm->lib);
  if (nm->d_tables) cudaFree(nm->d_tables);
  delete nm;
}

// tab_orig: [n_ranges][R][10] rate rows in the caller's reaction order; thermo: [n_ranges][S][12];
// falloff: rows of 8 by fo_idx in the caller's order of falloff reactions.  Returns "" or why not.
std::string nu_create(const ck_mech_desc *d, int n_ranges, const std::vector<double> &range_T,
                      const std::vector<double> &tab_orig, const std::vector<double> &thermo,
                      const std::vector<double> &logtab, const std::vector<double> &falloff, int device,
                      int num_sms, size_t smem_block_max, NuMech **out) {
  *out = nullptr;
  const int S = d->n_species, R = d->n_reactions;
  if (S > 16 || R > 64) return "the all-DMMA kernel takes at most 16 species and 64 reactions";
  if (d->kc_ann || d->precision != CK_PREC_F64) return "the all-DMMA kernel has no approximate-ANN or reduced-precision variant";
  const int SP4 = (S + 3) / 4 * 4, KS = SP4 / 4, RP = (R + 7) / 8 * 8, NT = RP / 8, NT2 = (S + 7) / 8;
  // reactions by type (elementary, three-body, falloff), then slot s = 8 nt + 2 q + e with the i-th
  // reaction at nt = i / 8, e = (i % 8) / 4, q = i % 4: consecutive reactions sit on different lanes,
  // so that the few falloff reactions of a tile are evaluated side by side
  std::vector<int> order;
  for (int pass = 0; pass < 3; ++pass)
    for (int j = 0; j < R; ++j) {
      const int t = d->rxn_type ? d->rxn_type[j] : 0;
      if ((pass == 0 && t == 0) || (pass == 1 && t == 1) || (pass == 2 && t >= 2)) order.push_back(j);
    }
  std::vector<int> rxn_of_slot(RP, -1);
  for (int i = 0; i < R; ++i) rxn_of_slot[8 * (i / 8) + 2 * (i % 4) + (i % 8) / 4] = order[i];

  std::vector<double> tab((size_t)n_ranges * RP * 10, 0.0), fo((size_t)RP * 8, 0.0), flags(RP, 8.0);
  std::vector<double> b1f((size_t)NT * KS * 32, 0.0), b1r(b1f.size(), 0.0), be(b1f.size(), 0.0);
  std::vector<double> b2((size_t)NT2 * 2 * NT * 32, 0.0);
  int n_fo = 0;
  std::vector<int> fo_idx(R, -1);
  for (int j = 0; j < R; ++j)
    if (d->rxn_type && d->rxn_type[j] >= 2) fo_idx[j] = n_fo++;
  for (int s = 0; s < RP; ++s) {
    const int j = rxn_of_slot[s];
    for (int r = 0; r < n_ranges; ++r) {
      double *row = &tab[((size_t)r * RP + s) * 10];
      if (j >= 0) std::copy(&tab_orig[((size_t)r * R + j) * 10], &tab_orig[((size_t)r * R + j) * 10] + 10, row);
      else row[0] = row[3] = -5000.0;   // null slot: both rates underflow
    }
    if (j < 0) continue;
    const int type = d->rxn_type ? d->rxn_type[j] : 0;
    flags[s] = type + 8.0 * ((d->reversible ? d->reversible[j] != 0 : true) ? 1 : 0);
    if (type >= 2) std::copy(&falloff[(size_t)fo_idx[j] * 8], &falloff[(size_t)fo_idx[j] * 8] + 8, &fo[(size_t)s * 8]);
  }
  for (int nt = 0; nt < NT; ++nt)
    for (int ks = 0; ks < KS; ++ks)
      for (int lane = 0; lane < 32; ++lane) {
        const int k = 4 * ks + lane % 4, j = rxn_of_slot[8 * nt + lane / 4];
        if (k >= S || j < 0) continue;
        const size_t at = ((size_t)nt * KS + ks) * 32 + lane;
        b1f[at] = d->nu_reac[(size_t)k * R + j];
        b1r[at] = d->nu_prod[(size_t)k * R + j];
        const int type = d->rxn_type ? d->rxn_type[j] : 0;
        if (type != 0) be[at] = d->eff ? d->eff[(size_t)k * R + j] : 1.0;
      }
  for (int n2 = 0; n2 < NT2; ++n2)
    for (int ks2 = 0; ks2 < 2 * NT; ++ks2)
      for (int lane = 0; lane < 32; ++lane) {
        const int k = 8 * n2 + lane / 4, j = rxn_of_slot[8 * (ks2 / 2) + 2 * (lane % 4) + ks2 % 2];
        if (k >= S || j < 0) continue;
        b2[((size_t)n2 * 2 * NT + ks2) * 32 + lane] = d->nu_prod[(size_t)k * R + j] - d->nu_reac[(size_t)k * R + j];
      }
  std::vector<double> rng = range_T;
  if (rng.empty()) rng.push_back(0.0);

  // launch shape: the most threads whose shared memory fits (registers: ~170 per thread)
  int threads = 0;
  size_t smem = 0;
  for (int nt : {384, 256, 128}) {
    const size_t rows = 2 * (size_t)std::max(SP4, 8 * NT2);
    const size_t doubles = rows * (nt + 8) + 128 + 256 + (size_t)n_ranges * S * 12 + (size_t)n_ranges * RP * 10 +
                           (size_t)RP * 8 + 3 * b1f.size() + b2.size() + RP;
    if (doubles * 8 <= smem_block_max) { threads = nt; smem = doubles * 8; break; }
  }
  if (!threads) return "the all-DMMA kernel's tables do not fit shared memory";

  std::ostringstream o;
  o << "#define NU_S " << S << "\n#define NU_R " << RP << "\n#define NU_THREADS " << threads << "\n#define NU_NRANGES "
    << n_ranges << "\n#define CK_LUT_REP 1\n#define CK_KCONST 0\n#define CK_PREC 0\n" << kNuText;
  std::vector<char> cubin;
  NuMech *nm = new NuMech();
  cudaError_t ce = cudaSuccess;
  for (int attempt = 0; attempt < 2; ++attempt) {
    const std::string err = jit_compile(o.str(), &cubin, attempt == 0);
    if (!err.empty()) { nu_destroy(nm); return err; }
    ce = cudaLibraryLoadData(&nm->lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (ce == cudaSuccess) break;
    cudaGetLastError();
    nm->lib = nullptr;
  }
  if (ce == cudaSuccess) ce = cudaLibraryGetKernel(&nm->kernel, nm->lib, "ck_source_terms_nu");
  if (ce == cudaSuccess)
    ce = cudaKernelSetAttributeForDevice(nm->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem, device);
  if (ce != cudaSuccess) { nu_destroy(nm); return std::string("loading the all-DMMA kernel: ") + cudaGetErrorString(ce); }

  // one device allocation for the tables
  std::vector<double> all;
  auto put = [&](const std::vector<double> &v) { const size_t at = all.size(); all.insert(all.end(), v.begin(), v.end()); if (all.size() % 2) all.push_back(0.0); return at; };
  const size_t o_th = put(thermo), o_log = put(logtab), o_tab = put(tab), o_fo = put(fo), o_b1f = put(b1f), o_b1r = put(b1r),
               o_be = put(be), o_b2 = put(b2), o_fl = put(flags), o_rng = put(rng);
  ce = cudaMalloc(&nm->d_tables, all.size() * sizeof(double));
  if (ce == cudaSuccess) ce = cudaMemcpy(nm->d_tables, all.data(), all.size() * sizeof(double), cudaMemcpyHostToDevice);
  if (ce != cudaSuccess) { nu_destroy(nm); return std::string("all-DMMA kernel tables: ") + cudaGetErrorString(ce); }
  const double *base = (const double *)nm->d_tables;
  nm->prm.thermo = base + o_th; nm->prm.logtab = base + o_log; nm->prm.tab = base + o_tab; nm->prm.fo = base + o_fo;
  nm->prm.b1f = base + o_b1f; nm->prm.b1r = base + o_b1r; nm->prm.be = base + o_be; nm->prm.b2 = base + o_b2;
  nm->prm.flags = base + o_fl; nm->prm.rangeT = base + o_rng;
  nm->threads = threads;
  nm->smem = smem;
  nm->grid_max = num_sms * (int)std::max<size_t>(1, std::min<size_t>(65536 / (176 * threads), 233472 / (smem + 1024)));
  *out = nm;
  return "";
}

cudaError_t nu_launch(const NuMech *nm, const double *T, const double *P, const double *Y, int64_t N, double *wdot,
                      double *dTdt, cudaStream_t stream) {
  NuParams prm = nm->prm;
  prm.T = T; prm.P = P; prm.Y = Y; prm.wdot = wdot; prm.dTdt = dTdt; prm.N = N;
  const int64_t warps = (N + 31) / 32, per_block = nm->threads / 32;
  const int grid = (int)std::min<int64_t>((warps + per_block - 1) / per_block, nm->grid_max);
  void *args[] = {&prm};
  return cudaLaunchKernel((const void *)nm->kernel, dim3(grid), dim3(nm->threads), args, nm->smem, stream);
}

int nu_threads(const NuMech *nm) { return nm->threads; }
size_t nu_smem(const NuMech *nm) { return nm->smem; }

}  // namespace ck
