// ck_api.cu -- the C ABI of include/ck.h: validation, mechanism build (host
// preprocessing of the paper's matrices into the device reaction program), launches.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/ck.h"
#include "ck_internal.h"

namespace {

thread_local std::string g_last_error;

int fail(int status, const std::string &msg) {
  g_last_error = msg;
  return status;
}

int fail_cuda(cudaError_t e, const char *what) {
  g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
  return CK_ECUDA;
}

// byte buffer with aligned appends; returns the offset of the appended block
struct Packer {
  std::vector<unsigned char> bytes;
  size_t append(const void *p, size_t n, size_t align = 256) {
    size_t off = (bytes.size() + align - 1) / align * align;
    bytes.resize(off + n);
    if (n) std::memcpy(bytes.data() + off, p, n);
    return off;
  }
};

int validate(const ck_mech_desc *d) {
  if (!d) return fail(CK_EINVAL, "desc is NULL");
  const int S = d->n_species, R = d->n_reactions;
  if (S < 1 || R < 1) return fail(CK_EINVAL, "n_species and n_reactions must be >= 1");
  if (!d->mol_weight || !d->nu_reac || !d->nu_prod || !d->ln_A || !d->b || !d->Ea_over_R ||
      !d->nasa_lo || !d->nasa_hi || !d->T_mid)
    return fail(CK_EINVAL, "a required array pointer is NULL");
  if (!(d->p_ref > 0.0) || !std::isfinite(d->p_ref)) return fail(CK_EINVAL, "p_ref must be > 0");
  for (int k = 0; k < S; ++k) {
    if (!(d->mol_weight[k] > 0.0) || !std::isfinite(d->mol_weight[k]))
      return fail(CK_EINVAL, "mol_weight must be finite and > 0");
    if (!(d->T_mid[k] > 0.0) || !std::isfinite(d->T_mid[k]))
      return fail(CK_EINVAL, "T_mid must be finite and > 0");
    for (int i = 0; i < 7; ++i)
      if (!std::isfinite(d->nasa_lo[k * 7 + i]) || !std::isfinite(d->nasa_hi[k * 7 + i]))
        return fail(CK_EINVAL, "NASA coefficients must be finite");
  }
  for (int j = 0; j < R; ++j) {
    const int type = d->rxn_type ? d->rxn_type[j] : CK_ELEMENTARY;
    if (type < CK_ELEMENTARY || type > CK_TROE)
      return fail(CK_EUNSUPPORTED, "unknown rxn_type code (only 0..3 are supported)");
    if (!std::isfinite(d->ln_A[j]) || !std::isfinite(d->b[j]) || !std::isfinite(d->Ea_over_R[j]))
      return fail(CK_EINVAL, "Arrhenius parameters must be finite");
    double sum_r = 0, sum_p = 0;
    for (int k = 0; k < S; ++k) {
      const double a = d->nu_reac[(size_t)k * R + j], b = d->nu_prod[(size_t)k * R + j];
      if (!(a >= 0.0) || !(b >= 0.0) || !std::isfinite(a) || !std::isfinite(b))
        return fail(CK_EINVAL, "stoichiometric coefficients must be finite and >= 0");
      sum_r += a;
      sum_p += b;
      if (type != CK_ELEMENTARY && d->eff) {
        const double e = d->eff[(size_t)k * R + j];
        if (!(e >= 0.0) || !std::isfinite(e))
          return fail(CK_EINVAL, "third-body efficiencies must be finite and >= 0");
      }
    }
    if (sum_r <= 0.0 || sum_p <= 0.0)
      return fail(CK_EINVAL, "every reaction needs at least one reactant and one product");
    if (type == CK_LINDEMANN || type == CK_TROE) {
      if (!d->ln_A0 || !d->b0 || !d->Ea0_over_R)
        return fail(CK_EINVAL, "falloff reactions need ln_A0, b0 and Ea0_over_R");
      if (!std::isfinite(d->ln_A0[j]) || !std::isfinite(d->b0[j]) || !std::isfinite(d->Ea0_over_R[j]))
        return fail(CK_EINVAL, "low-pressure Arrhenius parameters must be finite");
    }
    if (type == CK_TROE) {
      if (!d->troe) return fail(CK_EINVAL, "Troe reactions need the troe array");
      const double *t = d->troe + 4 * (size_t)j;
      if (!std::isfinite(t[0])) return fail(CK_EINVAL, "Troe alpha must be finite");
      if (!(t[1] > 0.0) || !(t[2] > 0.0) || !(t[3] > 0.0) || std::isnan(t[3]) ||
          !std::isfinite(t[1]) || !std::isfinite(t[2]))
        return fail(CK_EINVAL, "Troe temperatures must be > 0 (T** may be +INF)");
    }
  }
  if (d->precision < CK_PREC_F64 || d->precision > CK_PREC_F32_RATES)
    return fail(CK_EINVAL, "precision must be CK_PREC_F64, CK_PREC_MIXED or CK_PREC_F32_RATES");
  if (const ck_kc_ann *a = d->kc_ann) {
    if ((a->n_in != 1 && a->n_in != 6) || a->n_layers < 1 || a->n_layers > 8 || a->n_hidden < 1 ||
        a->n_hidden > 64 || (a->activation != CK_ANN_RELU && a->activation != CK_ANN_ELU))
      return fail(CK_EINVAL, "kc_ann: n_in must be 1 or 6, 1 <= n_layers <= 8, 1 <= n_hidden <= 64, activation 0 or 1");
    if (!a->in_mean || !a->in_std || !a->W_in || !a->B || !a->W_out || !a->B_out || !a->out_mean ||
        !a->out_std || (a->n_layers > 1 && !a->W_hid))
      return fail(CK_EINVAL, "kc_ann: a weight array pointer is NULL");
    auto finite = [](const double *p, size_t n) {
      for (size_t i = 0; i < n; ++i) if (!std::isfinite(p[i])) return false;
      return true;
    };
    const size_t NI = a->n_in, NH = a->n_hidden, NL = a->n_layers;
    if (!finite(a->in_mean, NI) || !finite(a->in_std, NI) || !finite(a->W_in, NI * NH) || !finite(a->B, NL * NH) ||
        (NL > 1 && !finite(a->W_hid, (NL - 1) * NH * NH)) || !finite(a->W_out, NH * R) || !finite(a->B_out, R) ||
        !finite(a->out_mean, R) || !finite(a->out_std, R))
      return fail(CK_EINVAL, "kc_ann: weights must be finite");
    for (size_t i = 0; i < NI; ++i)
      if (!(a->in_std[i] > 0.0)) return fail(CK_EINVAL, "kc_ann: in_std must be > 0");
    // the hidden layers' weights are constant-bank operands of the kernel (64 KB bank, shared
    // with the falloff table and the compiler's own constants)
    if ((2 * NI + NI * NH + NL * NH + (NL - 1) * NH * NH) * sizeof(double) > 40960)
      return fail(CK_EUNSUPPORTED, "kc_ann: hidden-layer weights exceed 40 KB (e.g. 3 layers of 50 neurons)");
  }
  return CK_OK;
}

// g'_k = g_k/RT - ln(p_ref/(Ru T)) on the features [1, ln T, T, T^2, T^3, T^4, 1/T]
// (Eq. 10 with the standard-concentration term folded into the bias)
void gibbs_feature_row(const double *a, double p_ref, long double out[7]) {
  out[0] = (long double)a[0] - (long double)a[6] - logl((long double)p_ref / (long double)ck::kRu);
  out[1] = 1.0L - (long double)a[0];
  out[2] = -(long double)a[1] / 2.0L;
  out[3] = -(long double)a[2] / 6.0L;
  out[4] = -(long double)a[3] / 12.0L;
  out[5] = -(long double)a[4] / 20.0L;
  out[6] = (long double)a[5];
}

// Everything ck_mech_create derives from the description on the host (no CUDA calls).
struct HostBuild {
  int n_ranges = 1, n_m = 0, n_mb = 0;
  std::vector<double> range_T, inv_W, thermo, eff, eff_frag, falloff, jit_tab;
  int jit_n_m = 0;            // rows of M in the specialised kernel's (padded) order
  int n_ranges_tmp = 1;
  std::vector<double> jit_eff;
  std::vector<double> jit_thermo;   // [n_ranges][S][12], the NASA-7 set holding in each range
  std::vector<double> jit_logtab;   // [128][2]: 1/c_i, ln c_i (ck_log in ck_jit_kernel.cuh)
  std::vector<double> tab_orig, thermo_orig;   // rate rows / thermo rows in the caller's order (ck_nu.cu)
  std::vector<unsigned char> program;
  ck::JitSpec spec;
  std::string jit_why;        // why the mechanism cannot be specialised ("" if it can)
  size_t jit_smem = 0;        // dynamic shared memory of the specialised kernel
  int64_t nnz_reac = 0, nnz_prod = 0, nnz_net = 0, nnz_eff = 0;
  int n_three_body = 0, n_lindemann = 0, n_troe = 0;
};

// B200 (sm_100a) per-SM resources, used when the launch shape has to be chosen without a
// device (ck_mech_jit_source on a build box)
constexpr size_t kSmemPerSm = 233472, kSmemPerBlock = 232448;

int env_int(const char *name, int dflt) {
  const char *e = std::getenv(name);
  return (e && *e) ? std::atoi(e) : dflt;
}

// Launch shape of the specialised kernel.  The kernel wants registers before threads: the
// species accumulators (2 registers per species), the DMMA fragments of M = C E and the
// interleaved exp chains of a reaction block (about 144 registers, "rest"); measured at S=53,
// 256 threads x 255 registers beat 384 x 168 by 14 %.
//  * All accumulators in registers (S <= 103): the most resident threads whose register cap
//    reaches 2 S + rest (or 255), else the largest cap.
//  * Otherwise hot/cold: the s_reg most scattered-to species accumulate in registers, the
//    rest in per-thread columns of shared memory (read-modify-write, no FP64-pipe cost);
//    the most resident threads, then the most register accumulators.
// Shared memory (ln C columns + cold accumulators + tables) must fit.  Fills spec.threads /
// min_blocks / tab_in_smem / s_reg and returns "", or returns the reason it cannot.
std::string choose_jit_shape(ck::JitSpec &spec, size_t smem_sm, size_t smem_blk, size_t *smem_out) {
  const int S = spec.S, R = spec.R;
  const bool fits = 2 * S + 48 <= 255;
  // registers beside the accumulators: the interleaved exp chains of a block (two per reaction)
  // dominate, so smaller blocks need fewer (measured at S=9 with blocks of 2: 512 threads x 128
  // registers 0.183 ms, 384 x 168 0.196 ms)
  const int rest_dflt = !fits ? 166 : (spec.block <= 2 ? 100 : (spec.block == 3 ? 124 : 144));
  const int rest = std::max(48, env_int("CK_JIT_REST", rest_dflt));
  const int sreg_forced = std::min(S, env_int("CK_JIT_SREG", -1));   // tuning / test knob
  const size_t tab_elem = spec.prec == CK_PREC_F32_RATES ? sizeof(float) : sizeof(double);
  const size_t tab_bytes = (size_t)spec.tab_ranges * R * spec.row * tab_elem;   // R includes padding
  const int nt_forced = env_int("CK_JIT_NT", 0), b_forced = env_int("CK_JIT_MINB", 0);
  {
    // copies of the exp table: a power of two in 1..16 (lane l reads copy l & (rep - 1))
    const int rep = env_int("CK_JIT_LUTREP", 1);
    spec.lut_rep = 1;
    while (spec.lut_rep * 2 <= std::min(rep, 16)) spec.lut_rep *= 2;
  }
  int best_nt = 0, best_b = 0, best_cap = 0, best_sreg = 0;
  bool best_tab = false;
  size_t best_smem = 0;
  auto smem_of = [&](int nt, int s_reg, bool tab_smem) {
    return (size_t)(S + (S - s_reg) + spec.ann_nhp) * (nt + 8) * 8 + (128 * spec.lut_rep + 256) * 8 + (size_t)spec.n_ranges * S * 12 * 8 +
           (tab_smem ? tab_bytes : (size_t)(nt / 32) * 2 * spec.tab_ranges * spec.block * spec.row * tab_elem) + 16;
  };
  const bool all_regs = sreg_forced < 0 ? fits : (sreg_forced == S);
  if (all_regs) {
    const int regs_wanted = std::min(255, 2 * S + rest);
    for (int nt : {512, 448, 384, 320, 256, 192, 128, 64}) {
      if (nt_forced && nt != nt_forced) continue;
      for (int b = 1; b <= 4; ++b)
        for (int tab_smem = 1; tab_smem >= 0; --tab_smem) {
          if (b_forced && b != b_forced) continue;
          const int regcap = std::min(255, (65536 / (nt * b)) / 8 * 8);
          if (regcap < 2 * S + 48) continue;
          const size_t smem = smem_of(nt, S, tab_smem != 0);
          if (smem > smem_blk || b * (smem + 1024) > smem_sm) continue;
          const int cap = std::min(regcap, regs_wanted);
          // registers, then resident threads, then larger blocks, then the table resident in smem
          const bool better = cap > best_cap || (cap == best_cap && nt * b > best_nt * best_b) ||
                              (cap == best_cap && nt * b == best_nt * best_b && nt > best_nt) ||
                              (cap == best_cap && nt == best_nt && b == best_b && (tab_smem != 0) > best_tab);
          if (better) { best_nt = nt; best_b = b; best_cap = cap; best_tab = tab_smem != 0; best_smem = smem; best_sreg = S; }
        }
    }
  } else {
    for (int nt : {512, 448, 384, 320, 256, 192, 128, 64})
      for (int b = 1; b <= 2; ++b)
        for (int tab_smem = 1; tab_smem >= 0; --tab_smem) {
          if ((nt_forced && nt != nt_forced) || (b_forced && b != b_forced)) continue;
          const int regcap = std::min(255, (65536 / (nt * b)) / 8 * 8);
          const int s_reg = sreg_forced >= 0 ? sreg_forced : std::min(S, (regcap - rest) / 2);
          if (s_reg < 0 || 2 * s_reg + 48 > regcap) continue;
          if (sreg_forced < 0 && s_reg < S / 4) continue;
          const size_t smem = smem_of(nt, s_reg, tab_smem != 0);
          if (smem > smem_blk || b * (smem + 1024) > smem_sm) continue;
          const bool better = nt * b > best_nt * best_b ||
                              (nt * b == best_nt * best_b && (tab_smem != 0) > best_tab) ||
                              (nt * b == best_nt * best_b && (tab_smem != 0) == best_tab && s_reg > best_sreg);
          if (better) { best_nt = nt; best_b = b; best_tab = tab_smem != 0; best_smem = smem; best_sreg = s_reg; }
        }
  }
  // Two threads per cell (CK_PAIR): for mechanisms whose accumulators do not fit one thread's
  // registers, 2 x cells threads share the cells' columns and split the accumulators, which puts
  // twice the warps on a scheduler for the same shared memory.  CK_JIT_PAIR=1 forces it on any
  // mechanism (tests), =0 disables it.  Not combined with the approximate ANN.
  const int pair_env = env_int("CK_JIT_PAIR", -1);
  bool pair = false;
  if (!spec.kc_ann && pair_env != 0 && (pair_env == 1 || !all_regs)) {
    int p_nt = 0, p_sreg = 0;
    bool p_tab = false;
    size_t p_smem = 0;
    for (int nt : {512, 384, 256, 128})
      for (int tab_smem = 1; tab_smem >= 0; --tab_smem) {
        if (nt_forced && nt != nt_forced) continue;
        const int cells = nt / 2;
        const int regcap = std::min(255, (65536 / nt) / 8 * 8);
        int s_reg = std::min((S + 1) / 2, (regcap - rest) / 2);
        if (sreg_forced >= 0) s_reg = std::min((S + 1) / 2, sreg_forced);
        if (s_reg < 0 || 2 * s_reg + 48 > regcap) continue;
        if (sreg_forced < 0 && 2 * s_reg < S / 4) continue;
        const int n_cold = std::max(0, S - 2 * s_reg);
        const size_t smem = (size_t)(S + n_cold) * (cells + 8) * 8 + (128 * spec.lut_rep + 256) * 8 +
                            (size_t)spec.n_ranges * S * 12 * 8 +
                            (tab_smem ? tab_bytes : (size_t)(nt / 32) * 2 * spec.tab_ranges * spec.block * spec.row * tab_elem) +
                            (size_t)(4 * spec.block + 8) * cells * 8 + 16;
        if (smem > smem_blk || smem + 1024 > smem_sm) continue;
        const bool better = nt > p_nt || (nt == p_nt && (tab_smem != 0) > p_tab);
        if (better) { p_nt = nt; p_sreg = s_reg; p_tab = tab_smem != 0; p_smem = smem; }
      }
    // worth it only if it puts more threads on the SM than the one-thread-per-cell shape
    if (p_nt > 0 && (pair_env == 1 || p_nt > best_nt * best_b)) {
      pair = true;
      best_nt = p_nt; best_b = 1; best_tab = p_tab; best_sreg = p_sreg; best_smem = p_smem;
    }
  }
  if (best_nt == 0) return "no launch shape fits registers and shared memory";
  spec.pair = pair;
  spec.threads = best_nt; spec.min_blocks = best_b; spec.tab_in_smem = best_tab; spec.s_reg = best_sreg;
  // tuning knobs for A/B runs under ncu (defaults are the measured best)
  if (const char *e = std::getenv("CK_JIT_M")) spec.m_dmma = std::string(e) != "dfma";
  if (const char *e = std::getenv("CK_JIT_MHINT")) spec.m_hint = std::atoi(e) != 0;
  if (const char *e = std::getenv("CK_JIT_SYNC")) spec.sync_every = std::atoi(e);
  if (const char *e = std::getenv("CK_JIT_KCONST")) spec.kconst = std::atoi(e) != 0;
  spec.straight = env_int("CK_JIT_STRAIGHT", 0);
  spec.pin = env_int("CK_JIT_PIN", 0);
  // (CK_JIT_KC=none, the ablation that removes the equilibrium layer, changes the RESULT: it is
  //  honoured only together with CK_ALLOW_ABLATION=1, see setup_jit, and shows in ck_mech_info 18)
  if (const char *e = std::getenv("CK_JIT_KC")) spec.kc_none = std::string(e) == "none";
  *smem_out = best_smem;
  return "";
}

// The specialised kernel walks the reactions in blocks of kJitBlock that are homogeneous
// in (type, reversible): a compact, instruction-cache resident "core" evaluates the rate
// layers of a whole block (Eq. 4, 6, 7, 11 and Sec. 2.4), and only the gathers / scatters
// of each block are unique generated code.  Here the reactions are sorted into those
// (blocks of 4 reactions by default)
// groups, every group is padded to whole blocks with null reactions (rate ~ 0, no species),
// and the rate table, falloff table and efficiency fragments are laid out in that order.

void finalize_jit(const ck_mech_desc *d, HostBuild *hb, const std::vector<double> &falloff_orig,
                  size_t smem_sm, size_t smem_blk) {
  const int S = d->n_species, R = d->n_reactions;
  ck::JitSpec &spec = hb->spec;
  const int n_ranges = hb->n_ranges_tmp;
  const int tab_ranges = spec.tab_ranges, ROW = spec.row;
  std::vector<ck::JitReaction> orig;
  orig.swap(spec.rxn);
  const std::vector<double> tab_orig = hb->jit_tab;

  // blocks of 4 reactions; 6 when the accumulators do not all fit in registers: that shape has
  // one warp per scheduler and needs the longer independent chains (measured)
  int kJitBlock = (2 * S + 48 > 255) ? 6 : 4;   // tuning knob CK_JIT_B (1..8)
  if (R <= 64 && kJitBlock == 4) {
    // Small mechanisms: every group is padded to whole blocks with null reactions that cost as
    // much as real ones (at S=9/R=21 blocks of 4 evaluate 24 slots, two of them Troe, for 21
    // reactions): take the block size in 2..4 with the least padded work (three-body 1.2, falloff 4
    // elementary reactions' worth).  Measured at S=9/R=21: 0.195 ms with blocks of 2, 0.224 with 4.
    double best = 0.0;
    for (int b = 2; b <= 4; ++b) {
      int n[3] = {0, 0, 0}, nr[3] = {0, 0, 0};
      for (int j = 0; j < R; ++j) {
        const int t = orig[j].type == 0 ? 0 : (orig[j].type == 1 ? 1 : 2);
        (orig[j].reversible ? n[t] : nr[t])++;
      }
      const double wgt[3] = {1.0, 1.2, 4.0};
      double cost = 0.0;
      for (int t = 0; t < 3; ++t) cost += wgt[t] * b * ((n[t] + b - 1) / b + (nr[t] + b - 1) / b);
      if (b == 2 || cost < best) { best = cost; kJitBlock = b; }
    }
  }
  if (const char *e = std::getenv("CK_JIT_B")) kJitBlock = std::min(8, std::max(1, std::atoi(e)));
  auto group_of = [](const ck::JitReaction &r) {
    const int t = r.type == 0 ? 0 : (r.type == 1 ? 1 : 2);
    return 2 * t + (r.reversible ? 0 : 1);
  };
  std::vector<int> order;                 // original reaction index, or -1 for a null reaction
  spec.block = kJitBlock;
  for (int g = 0; g < 6; ++g) {
    // within a falloff group the Troe reactions first: the kernel decides Troe / Lindemann per
    // block from its first reaction
    const size_t g0 = order.size();
    for (int pass = 0; pass < 2; ++pass) {
      const size_t p0 = order.size();
      for (int j = 0; j < R; ++j)
        if (group_of(orig[j]) == g && (orig[j].type == 3) == (pass == 0)) order.push_back(j);
      // Within the pass, reactions that gather the same species are put into the same block: their
      // ln C loads are then shared (one LDS instead of two: less unique code, less load latency).
      // Greedy: a block takes, one after the other, the remaining reaction that shares the most
      // species with what the block already reads (ties: input order).  CK_JIT_CLUSTER=0 turns it off.
      if (env_int("CK_JIT_CLUSTER", 1) != 0 && order.size() - p0 > (size_t)kJitBlock) {
        std::vector<int> rest(order.begin() + p0, order.end()), out;
        std::vector<char> in_blk(S, 0);
        while (!rest.empty()) {
          const size_t pos_in_blk = (g0 + (order.size() - rest.size() - g0)) % kJitBlock;   // position within the group's blocks
          (void)pos_in_blk;
          if ((out.size() + (p0 - g0)) % kJitBlock == 0) std::fill(in_blk.begin(), in_blk.end(), 0);
          size_t best = 0;
          int best_share = -1;
          for (size_t c = 0; c < rest.size(); ++c) {
            int share = 0;
            for (const auto &e : orig[rest[c]].reac) share += in_blk[e.first];
            for (const auto &e : orig[rest[c]].prod) share += in_blk[e.first];
            if (share > best_share) { best_share = share; best = c; }
          }
          const int j = rest[best];
          rest.erase(rest.begin() + best);
          out.push_back(j);
          for (const auto &e : orig[j].reac) in_blk[e.first] = 1;
          for (const auto &e : orig[j].prod) in_blk[e.first] = 1;
        }
        std::copy(out.begin(), out.end(), order.begin() + p0);
        // then pairwise swaps between blocks while the number of distinct species read per block,
        // summed over the blocks, goes down (a fixed, deterministic sweep order)
        auto blk_cost = [&](size_t blk_first) {   // distinct species gathered by the block starting at this position
          std::fill(in_blk.begin(), in_blk.end(), 0);
          int n = 0;
          for (size_t q = blk_first; q < blk_first + (size_t)kJitBlock && q < order.size(); ++q) {
            if (q < g0) continue;
            const ck::JitReaction &r = orig[order[q]];
            for (const auto &e : r.reac) if (!in_blk[e.first]) { in_blk[e.first] = 1; ++n; }
            if (r.reversible) for (const auto &e : r.prod) if (!in_blk[e.first]) { in_blk[e.first] = 1; ++n; }
          }
          return n;
        };
        auto first_of = [&](size_t pos) { return g0 + (pos - g0) / kJitBlock * kJitBlock; };
        for (int sweep = 0; sweep < 8; ++sweep) {
          bool improved = false;
          for (size_t a = p0; a < order.size(); ++a)
            for (size_t b = a + 1; b < order.size(); ++b) {
              const size_t fa = first_of(a), fb = first_of(b);
              if (fa == fb) continue;
              const int before = blk_cost(fa) + blk_cost(fb);
              std::swap(order[a], order[b]);
              if (blk_cost(fa) + blk_cost(fb) < before) improved = true;
              else std::swap(order[a], order[b]);
            }
          if (!improved) break;
        }
      }
    }
    while (order.size() % kJitBlock) order.push_back(-1);
    spec.group_end[g] = (int)order.size() / kJitBlock;
  }
  const int RP = (int)order.size();
  spec.R = RP;
  hb->jit_tab.assign((size_t)tab_ranges * RP * ROW, 0.0);
  spec.falloff.clear();
  std::vector<int> m_rows;                // original reaction of each M row (-1: null)
  for (int jj = 0; jj < RP; ++jj) {
    const int j = order[jj];
    const int g = [&] { int gg = 0; while (jj / kJitBlock >= spec.group_end[gg]) ++gg; return gg; }();
    ck::JitReaction r;
    if (j >= 0) r = orig[j];
    r.index = j;
    r.type = g / 2 == 0 ? 0 : (g / 2 == 1 ? 1 : (j >= 0 ? orig[j].type : 2));
    r.reversible = (g % 2 == 0);
    for (int rg = 0; rg < tab_ranges; ++rg) {
      double *row = &hb->jit_tab[((size_t)rg * RP + jj) * ROW];
      if (j >= 0) {
        const double *src = &tab_orig[((size_t)rg * R + j) * ROW];
        for (int i = 0; i < ROW; ++i) row[i] = src[i];
      } else {
        row[0] = -5000.0;   // null reaction: ln q = -5000, the rate underflows to ~1e-307
        if (!spec.kc_ann) row[3] = -5000.0;   // (with the ANN, ln k_r = ln k_f + row[3] + ...)
      }
    }
    if (g >= 2) {           // third-body and falloff reactions: a row of M each, in this order
      r.m_slot = (int)m_rows.size();
      m_rows.push_back(j);
    }
    if (g >= 4) {           // falloff rows in this order (null: Lindemann with k0 tiny)
      r.fo_idx = (int)(spec.falloff.size() / ck::kFalloffStride);
      if (j >= 0) {
        const double *src = &falloff_orig[(size_t)orig[j].fo_idx * ck::kFalloffStride];
        spec.falloff.insert(spec.falloff.end(), src, src + ck::kFalloffStride);
      } else {
        const double row[ck::kFalloffStride] = {-100.0, 0, 0, 0, 0, 0, 0, 2.0};
        spec.falloff.insert(spec.falloff.end(), row, row + ck::kFalloffStride);
      }
    }
    spec.rxn.push_back(std::move(r));
  }
  // ---- launch shape, and which accumulators live in registers --------------------------
  hb->jit_why = choose_jit_shape(spec, smem_sm, smem_blk, &hb->jit_smem);
  if (!hb->jit_why.empty()) spec.s_reg = S;
  // Internal species order: by the number of scatters into the species (Eq. 2), descending,
  // so that the register accumulators serve the most updates; identity if all are in registers.
  std::vector<int> perm(S), inv(S);
  for (int k = 0; k < S; ++k) perm[k] = k;
  if (spec.pair || spec.s_reg < S) {
    std::vector<int> hits(S, 0);
    for (const ck::JitReaction &r : spec.rxn)
      for (const auto &e : r.net) hits[e.first]++;
    std::stable_sort(perm.begin(), perm.end(), [&](int a, int b) { return hits[a] > hits[b]; });
    spec.perm = perm;
  }
  for (int k = 0; k < S; ++k) inv[perm[k]] = k;
  spec.mol_weight.resize(S);
  for (int k = 0; k < S; ++k) spec.mol_weight[k] = d->mol_weight[perm[k]];
  for (ck::JitReaction &r : spec.rxn) {
    for (auto &e : r.reac) e.first = inv[e.first];
    for (auto &e : r.prod) e.first = inv[e.first];
    for (auto &e : r.net) e.first = inv[e.first];
  }
  {
    const std::vector<double> th = hb->jit_thermo;
    for (int r = 0; r < n_ranges; ++r)
      for (int k = 0; k < S; ++k)
        std::copy(&th[((size_t)r * S + perm[k]) * 12], &th[((size_t)r * S + perm[k]) * 12] + 12,
                  &hb->jit_thermo[((size_t)r * S + k) * 12]);
  }
  // E as DMMA.8x8x4 B fragments: [n-tile][k-step][lane], lane holds
  // E[4 ks + lane%4][8 nt + lane/4] (species in internal order), zero padded in both directions
  const int n_m = (int)m_rows.size();
  const int n_mb = ((n_m + 7) / 8 + 1) & ~1, k_steps = (S + 3) / 4;   // pairs of n-tiles
  hb->jit_n_m = n_m;
  spec.n_m = n_m;
  spec.n_mb = n_mb;
  spec.n_fo = (int)(spec.falloff.size() / ck::kFalloffStride);
  hb->eff_frag.assign((size_t)std::max(n_mb, 1) * k_steps * 32, 0.0);
  for (int nt = 0; nt < n_mb; ++nt)
    for (int ks = 0; ks < k_steps; ++ks)
      for (int lane = 0; lane < 32; ++lane) {
        const int k = 4 * ks + lane % 4, row = 8 * nt + lane / 4;
        if (k < S && row < n_m && m_rows[row] >= 0)
          hb->eff_frag[((size_t)nt * k_steps + ks) * 32 + lane] =
              d->eff ? d->eff[(size_t)perm[k] * R + m_rows[row]] : 1.0;
      }
  // the DFMA variant's layout [block of 8 rows][species][8]
  hb->jit_eff.assign((size_t)std::max(n_mb, 1) * S * 8, 0.0);
  for (int row = 0; row < n_m; ++row)
    if (m_rows[row] >= 0)
      for (int k = 0; k < S; ++k)
        hb->jit_eff[((size_t)(row / 8) * S + k) * 8 + row % 8] =
            d->eff ? d->eff[(size_t)perm[k] * R + m_rows[row]] : 1.0;
}

void build_host(const ck_mech_desc *d, HostBuild *hb, size_t smem_sm = kSmemPerSm, size_t smem_blk = kSmemPerBlock) {
  const int S = d->n_species, R = d->n_reactions;
  HostBuild *m = hb;   // statistics are accumulated on the same names as in ck_mech
  // ---- temperature ranges from the distinct T_mid values --------------
  std::vector<double> &range_T = hb->range_T;
  range_T.assign(d->T_mid, d->T_mid + S);
  std::sort(range_T.begin(), range_T.end());
  range_T.erase(std::unique(range_T.begin(), range_T.end()), range_T.end());
  const int n_ranges = (int)range_T.size() + 1;
  std::vector<int> rank(S);
  for (int k = 0; k < S; ++k)
    rank[k] = (int)(std::lower_bound(range_T.begin(), range_T.end(), d->T_mid[k]) - range_T.begin());

  // ---- per-species tables -------------------------------------------------------------
  std::vector<double> &inv_W = hb->inv_W, &thermo = hb->thermo;
  inv_W.assign(S, 0.0);
  thermo.assign((size_t)S * ck::kThermoStride, 0.0);
  std::vector<long double> gfeat((size_t)S * 2 * 7);
  for (int k = 0; k < S; ++k) {
    inv_W[k] = 1.0 / d->mol_weight[k];
    double *t = &thermo[(size_t)k * ck::kThermoStride];
    const double *lo = d->nasa_lo + 7 * k, *hi = d->nasa_hi + 7 * k;
    t[0] = d->T_mid[k];
    for (int i = 0; i < 5; ++i) { t[1 + i] = lo[i]; t[6 + i] = hi[i]; }
    for (int i = 0; i < 5; ++i) { t[11 + i] = lo[i] / (i + 1); t[17 + i] = hi[i] / (i + 1); }
    t[16] = lo[5];
    t[22] = hi[5];
    gibbs_feature_row(lo, d->p_ref, &gfeat[((size_t)k * 2 + 0) * 7]);
    gibbs_feature_row(hi, d->p_ref, &gfeat[((size_t)k * 2 + 1) * 7]);
  }

  // ---- reaction program ------------------------------------------------------------------
  std::vector<unsigned char> &program = hb->program;
  std::vector<double> &falloff = hb->falloff;
  std::vector<int> m_rows;       // reaction index of each row of M
  ck::JitSpec &spec = hb->spec;
  spec.S = S; spec.R = R; spec.n_ranges = n_ranges;
  spec.prec = d->precision;
  const ck_kc_ann *ann = d->kc_ann;
  spec.kc_ann = ann != nullptr;
  if (ann) {
    spec.ann_nin = ann->n_in; spec.ann_nl = ann->n_layers; spec.ann_nh = ann->n_hidden;
    spec.ann_act = ann->activation; spec.ann_nhp = (ann->n_hidden + 1) & ~1;
    spec.tab_ranges = 1; spec.row = 4 + spec.ann_nhp;
    // constant-bank block of the hidden layers: mean | 1/std | W_in | B | W_hid
    const int NI = ann->n_in, NH = ann->n_hidden, NL = ann->n_layers;
    spec.ann_const.assign(ann->in_mean, ann->in_mean + NI);
    for (int i = 0; i < NI; ++i) spec.ann_const.push_back(1.0 / ann->in_std[i]);
    spec.ann_const.insert(spec.ann_const.end(), ann->W_in, ann->W_in + (size_t)NI * NH);
    spec.ann_const.insert(spec.ann_const.end(), ann->B, ann->B + (size_t)NL * NH);
    spec.ann_const.insert(spec.ann_const.end(), ann->W_hid, ann->W_hid + (size_t)(NL - 1) * NH * NH);
  } else {
    // (fp32 rate layers: rows of 12 floats, three 16-byte loads)
    spec.tab_ranges = n_ranges; spec.row = spec.prec == CK_PREC_F32_RATES ? 12 : 10;
  }
  const int ROW = spec.row;
  std::vector<double> &jit_tab = hb->jit_tab;
  jit_tab.assign((size_t)spec.tab_ranges * R * ROW, 0.0);
  for (int j = 0; j < R; ++j) {
    const int type = d->rxn_type ? d->rxn_type[j] : CK_ELEMENTARY;
    const int rev = d->reversible ? (d->reversible[j] != 0) : 1;
    std::vector<int> off_r, off_p, off_s;
    std::vector<double> c_r, c_p, c_s;
    for (int k = 0; k < S; ++k) {
      const double a = d->nu_reac[(size_t)k * R + j], b = d->nu_prod[(size_t)k * R + j];
      if (a != 0.0) { off_r.push_back(k); c_r.push_back(a); }
      if (b != 0.0) { off_p.push_back(k); c_p.push_back(b); }
      if (b - a != 0.0) { off_s.push_back(k); c_s.push_back(b - a); }
    }
    m->nnz_reac += (int64_t)off_r.size();
    m->nnz_prod += (int64_t)off_p.size();
    m->nnz_net += (int64_t)off_s.size();

    ck::RecHeader h{};
    h.nr = (int)off_r.size(); h.np = (int)off_p.size(); h.nsc = (int)off_s.size();
    h.type = type; h.reversible = rev; h.m_slot = -1; h.fo_idx = -1;
    if (type != CK_ELEMENTARY) {
      h.m_slot = (int)m_rows.size();
      m_rows.push_back(j);
      for (int k = 0; k < S; ++k)
        if (!d->eff || d->eff[(size_t)k * R + j] != 0.0) m->nnz_eff++;
    }
    if (type == CK_THREE_BODY) m->n_three_body++;
    if (type == CK_LINDEMANN || type == CK_TROE) {
      h.fo_idx = (int)(falloff.size() / ck::kFalloffStride);
      double row[ck::kFalloffStride] = {d->ln_A0[j], d->b0[j], -d->Ea0_over_R[j], 0, 0, 0, 0,
                                        (double)type};
      if (type == CK_TROE) {
        const double *t = d->troe + 4 * (size_t)j;
        row[3] = t[0]; row[4] = -1.0 / t[1]; row[5] = -1.0 / t[2];
        row[6] = std::isinf(t[3]) ? -1e300 : -t[3];   // exp(-T**/T) -> 0 for T** = +INF
        m->n_troe++;
      } else {
        m->n_lindemann++;
      }
      falloff.insert(falloff.end(), row, row + ck::kFalloffStride);
    }

    std::vector<double> dbl;
    dbl.push_back(d->ln_A[j]); dbl.push_back(d->b[j]); dbl.push_back(-d->Ea_over_R[j]);
    dbl.push_back(0.0);
    for (int r = 0; r < n_ranges; ++r) {
      long double f[7] = {(long double)d->ln_A[j], (long double)d->b[j], 0, 0, 0, 0,
                          -(long double)d->Ea_over_R[j]};
      for (size_t e = 0; e < off_s.size(); ++e) {
        const int k = off_s[e];
        const int variant = (r > rank[k]) ? 1 : 0;   // T > T_mid[k] throughout range r
        const long double *g = &gfeat[((size_t)k * 2 + variant) * 7];
        for (int i = 0; i < 7; ++i) f[i] += (long double)c_s[e] * g[i];
      }
      for (int i = 0; i < 7; ++i) dbl.push_back((double)f[i]);
      dbl.push_back(0.0);
      // row of the specialised kernel's rate table (ck_jit_kernel.cuh)
      if (ann) continue;
      double *row = &jit_tab[((size_t)r * R + j) * ROW];
      row[0] = d->ln_A[j]; row[1] = d->b[j]; row[2] = -d->Ea_over_R[j];
      row[3] = (double)f[0]; row[4] = (double)f[1]; row[5] = (double)f[6];
      row[6] = (double)f[2]; row[7] = (double)f[3]; row[8] = (double)f[4]; row[9] = (double)f[5];
    }
    if (ann) {
      // approximate ANN (Eq. 12): ln Kc~_j = mu_j + sigma_j (B_out,j + sum_h x_h W_out[h][j]);
      // ln k_r = ln k_f - ln Kc~ (Eq. 7): output layer and de-standardisation folded into the row
      double *row = &jit_tab[(size_t)j * ROW];
      row[0] = d->ln_A[j]; row[1] = d->b[j]; row[2] = -d->Ea_over_R[j];
      row[3] = -(ann->out_mean[j] + ann->out_std[j] * ann->B_out[j]);
      for (int h = 0; h < ann->n_hidden; ++h) row[4 + h] = -ann->out_std[j] * ann->W_out[(size_t)h * R + j];
    }
    {
      ck::JitReaction jr;
      jr.index = j; jr.type = type; jr.reversible = rev; jr.m_slot = h.m_slot; jr.fo_idx = h.fo_idx;
      for (size_t e = 0; e < off_r.size(); ++e) jr.reac.emplace_back(off_r[e], c_r[e]);
      for (size_t e = 0; e < off_p.size(); ++e) jr.prod.emplace_back(off_p[e], c_p[e]);
      for (size_t e = 0; e < off_s.size(); ++e) jr.net.emplace_back(off_s[e], c_s[e]);
      spec.rxn.push_back(std::move(jr));
    }
    dbl.insert(dbl.end(), c_r.begin(), c_r.end());
    dbl.insert(dbl.end(), c_p.begin(), c_p.end());
    dbl.insert(dbl.end(), c_s.begin(), c_s.end());
    if (dbl.size() % 2) dbl.push_back(0.0);
    std::vector<int32_t> ints;
    ints.insert(ints.end(), off_r.begin(), off_r.end());
    ints.insert(ints.end(), off_p.begin(), off_p.end());
    ints.insert(ints.end(), off_s.begin(), off_s.end());
    while (ints.size() % 4) ints.push_back(0);

    h.size_bytes = (int32_t)(sizeof(h) + dbl.size() * sizeof(double) + ints.size() * sizeof(int32_t));
    const size_t at = program.size();
    program.resize(at + h.size_bytes);
    std::memcpy(&program[at], &h, sizeof(h));
    std::memcpy(&program[at + sizeof(h)], dbl.data(), dbl.size() * sizeof(double));
    std::memcpy(&program[at + sizeof(h) + dbl.size() * sizeof(double)], ints.data(),
                ints.size() * sizeof(int32_t));
  }

  // ---- third-body efficiency matrix, blocked for the register-tiled M = C E -----------
  const int n_m = (int)m_rows.size();
  const int n_mb = (n_m + ck::kMBlock - 1) / ck::kMBlock;
  std::vector<double> &eff = hb->eff;
  eff.assign((size_t)std::max(n_mb, 1) * S * ck::kMBlock, 0.0);
  for (int s = 0; s < n_m; ++s) {
    const int j = m_rows[s];
    for (int k = 0; k < S; ++k)
      eff[((size_t)(s / ck::kMBlock) * S + k) * ck::kMBlock + (s % ck::kMBlock)] =
          d->eff ? d->eff[(size_t)k * R + j] : 1.0;
  }
  spec.inv_W = inv_W; spec.range_T = range_T;
  // NASA-7 rows per temperature range: species k is on its high set in range r iff r > rank[k]
  hb->jit_thermo.assign((size_t)n_ranges * S * 12, 0.0);
  for (int r = 0; r < n_ranges; ++r)
    for (int k = 0; k < S; ++k) {
      const double *a = (r > rank[k]) ? d->nasa_hi + 7 * k : d->nasa_lo + 7 * k;
      double *row = &hb->jit_thermo[((size_t)r * S + k) * 12];
      for (int i = 0; i < 5; ++i) { row[i] = a[i]; row[6 + i] = a[i] / (i + 1); }
      row[5] = inv_W[k];
      row[11] = a[5];
    }
  // ln table: interval i covers m in [lo_i, lo_i + width) on the hi-word grid from 0x3fe6a000
  hb->jit_logtab.assign(256, 0.0);
  for (int i = 0; i < 128; ++i) {
    auto from_hi = [](uint32_t hi) {
      const uint64_t bits = (uint64_t)hi << 32;
      double v;
      std::memcpy(&v, &bits, sizeof v);
      return v;
    };
    const double lo = from_hi(0x3fe6a000u + (uint32_t)i * 8192u), hi = from_hi(0x3fe6a000u + (uint32_t)(i + 1) * 8192u);
    const double inv_c = 1.0 / (0.5 * (lo + hi));
    hb->jit_logtab[2 * i] = inv_c;
    hb->jit_logtab[2 * i + 1] = (double)(-logl((long double)inv_c));
  }
  hb->n_ranges_tmp = n_ranges;
  hb->tab_orig = jit_tab;
  hb->thermo_orig = hb->jit_thermo;
  finalize_jit(d, hb, falloff, smem_sm, smem_blk);
  if (falloff.empty()) falloff.resize(ck::kFalloffStride, 0.0);
  if (range_T.empty()) range_T.push_back(0.0);

  hb->n_ranges = n_ranges; hb->n_m = n_m; hb->n_mb = n_mb;
}

// Decides whether to use the specialised kernel (env CK_KERNEL = auto | generic | jit),
// compiles and loads it.  Returns CK_OK also when it falls back to the generic kernel in
// auto mode (m->jit_note says why).
// M scratch of the kernel in use: n_slots slots of slot_elems doubles + the slot flags (zeroed)
int alloc_scratch(ck_mech *m, int n_slots, size_t slot_elems) {
  cudaError_t ce = cudaMalloc((void **)&m->d_scratch, (size_t)n_slots * slot_elems * sizeof(double));
  if (ce == cudaSuccess) ce = cudaMalloc((void **)&m->d_slot_busy, (size_t)n_slots * sizeof(int));
  if (ce != cudaSuccess) return fail(CK_ENOMEM, std::string("cudaMalloc M scratch: ") + cudaGetErrorString(ce));
  ce = cudaMemset(m->d_slot_busy, 0, (size_t)n_slots * sizeof(int));
  if (ce != cudaSuccess) return fail_cuda(ce, "cudaMemset slot flags");
  return CK_OK;
}

int setup_jit(ck_mech *m, ck::JitSpec &spec, const std::string &why, size_t smem, size_t smem_sm, size_t smem_blk) {
  const char *mode_env = std::getenv("CK_KERNEL");
  std::string mode = mode_env ? mode_env : "auto";
  if (spec.kc_ann) {
    // the approximate-ANN layer exists only in the specialised kernel
    if (mode == "generic") return fail(CK_EUNSUPPORTED, "kc_ann needs the specialised kernel (CK_KERNEL=generic)");
    mode = "jit";
  }
  if (spec.prec == CK_PREC_F32_RATES && spec.kc_ann)
    return fail(CK_EUNSUPPORTED, "CK_PREC_F32_RATES is not combined with the approximate-ANN Kc");
  if (spec.prec != CK_PREC_F64) {
    // so do the reduced-precision variants
    if (mode == "generic") return fail(CK_EUNSUPPORTED, "reduced precision needs the specialised kernel (CK_KERNEL=generic)");
    mode = "jit";
  }
  if (spec.kc_none && env_int("CK_ALLOW_ABLATION", 0) != 1)
    return fail(CK_EINVAL, "CK_JIT_KC=none removes the equilibrium layer (a measurement-only ablation whose "
                           "results are not the source term); set CK_ALLOW_ABLATION=1 to build it");
  if (mode == "generic") {
    if (spec.kc_none) return fail(CK_EINVAL, "CK_JIT_KC=none exists only in the specialised kernel");
    m->jit_note = "CK_KERNEL=generic";
    return CK_OK;
  }
  if (mode != "auto" && mode != "jit") return fail(CK_EINVAL, "CK_KERNEL must be auto, generic or jit");
  const bool required = (mode == "jit");
  auto give_up = [&](const std::string &why) {
    m->jit_note = why;
    return required ? fail(CK_EUNSUPPORTED, "CK_KERNEL=jit but " + why) : (int)CK_OK;
  };
  if (!why.empty()) return give_up(why);

  const std::string src = ck::jit_generate_source(spec);
  if (const char *e = std::getenv("CK_JIT_DUMP")) {
    if (FILE *f = std::fopen(e, "w")) {
      std::fwrite(src.data(), 1, src.size(), f);
      std::fclose(f);
    }
  }
  std::vector<char> cubin;
  cudaError_t ce = cudaSuccess;
  for (int attempt = 0; attempt < 2; ++attempt) {
    // second attempt: the cubin came from the on-disk cache and would not load -- compile afresh
    const std::string err = ck::jit_compile(src, &cubin, /*use_cache=*/attempt == 0);
    if (!err.empty()) return give_up(err);
    ce = cudaLibraryLoadData(&m->jit_lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (ce == cudaSuccess) break;
    cudaGetLastError();
    m->jit_lib = nullptr;
  }
  if (ce != cudaSuccess) return give_up(std::string("cudaLibraryLoadData: ") + cudaGetErrorString(ce));
  ce = cudaLibraryGetKernel(&m->jit_kernel, m->jit_lib, "ck_source_terms_jit");
  if (ce == cudaSuccess)
    ce = cudaKernelSetAttributeForDevice(m->jit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem, m->device);
  if (ce != cudaSuccess) {
    cudaLibraryUnload(m->jit_lib);
    m->jit_lib = nullptr; m->jit_kernel = nullptr;
    return give_up(std::string("loading the specialised kernel: ") + cudaGetErrorString(ce));
  }
  m->jit_threads = spec.threads; m->jit_blocks_per_sm = spec.min_blocks; m->jit_smem = smem;
  m->jit_cells = spec.pair ? spec.threads / 2 : spec.threads;
  m->jit_spec = spec;
  m->jit_grid_max = m->num_sms * spec.min_blocks;
  // M = C E scratch in slots (ck_jit_kernel.cuh): one per block that can be resident on the device.
  // Shared memory bounds the resident blocks per SM from above (registers can only lower it).
  const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(std::min<size_t>(32, 2048 / spec.threads), smem_sm / (smem + 1024)));
  // A slot is sized for this (the main) shape; the small-batch shapes below and the RK4 stage variant
  // work on tiles of at most as many cells and index the slots with the same stride, so slot s is the
  // same bytes in every kernel of the handle and one set of busy flags guards it.
  const size_t slot_elems = (size_t)std::max(spec.n_mb, 1) * ck::kMBlock * m->jit_cells;
  if (int st = alloc_scratch(m, m->num_sms * per_sm, slot_elems)) return st;
  m->jit_params.m_scratch = m->d_scratch;
  m->jit_params.slot_busy = m->d_slot_busy;
  m->jit_params.n_slots = m->num_sms * per_sm;
  m->jit_params.slot_elems = (int)slot_elems;

  // ---- the small-batch shape (CK_SPLIT = 8 threads per cell, tiles of 32 cells): one warp no longer
  //      walks the whole mechanism alone when the batch is a few thousand cells.  Same tables, same
  //      scratch slots.  For mechanisms whose accumulators all sit in registers, of 32 reactions or
  //      more; CK_JIT_SPLIT=0 turns it off, a failure to build it is not an error.
  //      CK_JIT_SPLIT=k builds only the shape with k threads per cell (0: none); default 8, 4 and 2.
  const int only = env_int("CK_JIT_SPLIT", -1);
  if (only != 0 && !spec.pair && spec.s_reg == spec.S && !spec.kc_ann && spec.tab_in_smem && spec.R >= 32 && per_sm == 1)
    for (int split : {8, 4, 2}) {
      if (only > 0 && split != only) continue;
      ck::JitSpec s2 = spec;
      s2.split = split; s2.threads = 256; s2.min_blocks = 1;
      const size_t tab_elem = spec.prec == CK_PREC_F32_RATES ? sizeof(float) : sizeof(double);
      const size_t smem2 = (size_t)spec.S * (256 / split + 8) * 8 + (128 * spec.lut_rep + 256) * 8 + (size_t)spec.n_ranges * spec.S * 12 * 8 +
                           (size_t)spec.tab_ranges * spec.R * spec.row * tab_elem + (size_t)(spec.S + 4) * 256 * 8 + 16;
      std::vector<char> cubin2;
      const int at = m->n_split;
      if (smem2 + 64 <= smem_blk && ck::jit_compile(ck::jit_generate_source(s2), &cubin2).empty() &&
          cudaLibraryLoadData(&m->split_lib[at], cubin2.data(), nullptr, nullptr, 0, nullptr, nullptr, 0) == cudaSuccess) {
        if (cudaLibraryGetKernel(&m->split_kernel[at], m->split_lib[at], "ck_source_terms_jit") == cudaSuccess &&
            cudaKernelSetAttributeForDevice(m->split_kernel[at], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2, m->device) == cudaSuccess) {
          m->split_smem[at] = smem2; m->split_cells[at] = 256 / split;
          m->n_split++;
        } else {
          cudaLibraryUnload(m->split_lib[at]);
          m->split_lib[at] = nullptr; m->split_kernel[at] = nullptr;
        }
      }
      cudaGetLastError();
    }
  return CK_OK;
}

}  // namespace

extern "C" const char *ck_last_error(void) { return g_last_error.c_str(); }

extern "C" int ck_mech_create(const ck_mech_desc *d, ck_mech **out) {
  if (!out) return fail(CK_EINVAL, "out is NULL");
  *out = nullptr;
  if (int st = validate(d)) return st;
  const int S = d->n_species, R = d->n_reactions;

  ck_mech *m = new (std::nothrow) ck_mech();
  if (!m) return fail(CK_ENOMEM, "host allocation failed");
  cudaError_t ce = cudaGetDevice(&m->device);
  if (ce != cudaSuccess) { delete m; return fail_cuda(ce, "cudaGetDevice"); }
  cudaDeviceProp prop;
  ce = cudaGetDeviceProperties(&prop, m->device);
  if (ce != cudaSuccess) { delete m; return fail_cuda(ce, "cudaGetDeviceProperties"); }
  m->num_sms = prop.multiProcessorCount;
  // environment knobs of the per-call paths, read here once (see ck_mech in ck_internal.h)
  m->env_tile = env_int("CK_JIT_TILE", 0);
  m->env_host_chunks = env_int("CK_HOST_CHUNKS", 0);
  m->env_rk4_fused = env_int("CK_RK4_FUSED", 1) != 0;
  { const char *e = std::getenv("CK_JAC_KERNEL"); m->env_jac_v3_required = e && std::string(e) == "v3"; }

  // ---- launch shape: as many resident cells per SM as shared memory allows ----------
  int best_threads = 0, best_bps = 0;
  size_t best_smem = 0;
  for (int threads : {128, 64, 32}) {
    size_t smem = (size_t)2 * S * threads * sizeof(double);
    if (smem + 64 > (size_t)prop.sharedMemPerBlockOptin) continue;   // (+ the kernel's static shared memory)
    int bps = 0;
    ce = ck::kernel_configure(threads, smem, &bps);
    if (ce != cudaSuccess) { delete m; return fail_cuda(ce, "kernel_configure"); }
    if (bps * threads > best_bps * best_threads) {
      best_threads = threads; best_bps = bps; best_smem = smem;
    }
  }
  if (best_threads == 0) {
    delete m;
    return fail(CK_EUNSUPPORTED, "n_species too large for the shared-memory resident kernel");
  }
  ce = ck::kernel_configure(best_threads, best_smem, &best_bps);   // leave the attribute set
  if (ce != cudaSuccess) { delete m; return fail_cuda(ce, "kernel_configure"); }
  m->blocks_per_sm = best_bps;
  m->smem_bytes = best_smem;
  m->grid_max = m->num_sms * best_bps;

  HostBuild hb;
  build_host(d, &hb, (size_t)prop.sharedMemPerMultiprocessor, (size_t)prop.sharedMemPerBlockOptin);
  const int n_ranges = hb.n_ranges, n_m = hb.n_m, n_mb = hb.n_mb;
  m->nnz_reac = hb.nnz_reac; m->nnz_prod = hb.nnz_prod; m->nnz_net = hb.nnz_net; m->nnz_eff = hb.nnz_eff;
  m->n_three_body = hb.n_three_body; m->n_lindemann = hb.n_lindemann; m->n_troe = hb.n_troe;
  std::vector<double> &inv_W = hb.inv_W, &range_T = hb.range_T, &thermo = hb.thermo, &eff = hb.eff,
                      &eff_frag = hb.eff_frag, &falloff = hb.falloff, &jit_tab = hb.jit_tab;
  std::vector<unsigned char> &program = hb.program;
  ck::JitSpec &spec = hb.spec;

  // ---- one device allocation for all tables -------------------------------------------
  Packer pk;
  const size_t o_invW = pk.append(inv_W.data(), inv_W.size() * sizeof(double));
  const size_t o_rng = pk.append(range_T.data(), range_T.size() * sizeof(double));
  const size_t o_thermo = pk.append(thermo.data(), thermo.size() * sizeof(double));
  const size_t o_eff = pk.append(eff.data(), eff.size() * sizeof(double));
  const size_t o_fo = pk.append(falloff.data(), falloff.size() * sizeof(double));
  const size_t o_prog = pk.append(program.data(), program.size());
  std::vector<float> jit_tab32;
  if (spec.prec == CK_PREC_F32_RATES) jit_tab32.assign(jit_tab.begin(), jit_tab.end());
  const size_t o_jtab = jit_tab32.empty() ? pk.append(jit_tab.data(), jit_tab.size() * sizeof(double))
                                          : pk.append(jit_tab32.data(), jit_tab32.size() * sizeof(float));
  const size_t o_efrag = pk.append(eff_frag.data(), eff_frag.size() * sizeof(double));
  const size_t o_jeff = pk.append(hb.jit_eff.data(), hb.jit_eff.size() * sizeof(double));
  const size_t o_jthermo = pk.append(hb.jit_thermo.data(), hb.jit_thermo.size() * sizeof(double));
  const size_t o_jlog = pk.append(hb.jit_logtab.data(), hb.jit_logtab.size() * sizeof(double));
  ce = cudaMalloc(&m->d_tables, pk.bytes.size());
  if (ce != cudaSuccess) { delete m; return fail(CK_ENOMEM, std::string("cudaMalloc tables: ") + cudaGetErrorString(ce)); }
  ce = cudaMemcpy(m->d_tables, pk.bytes.data(), pk.bytes.size(), cudaMemcpyHostToDevice);
  if (ce != cudaSuccess) { ck_mech_destroy(m); return fail_cuda(ce, "cudaMemcpy tables"); }
  unsigned char *base = (unsigned char *)m->d_tables;
  ck::DeviceMech &dm = m->dev;
  dm.S = S; dm.R = R; dm.n_ranges = n_ranges; dm.n_m = n_m; dm.n_m_blocks = n_mb;
  dm.threads = best_threads;
  dm.inv_W = (const double *)(base + o_invW);
  dm.range_T = (const double *)(base + o_rng);
  dm.thermo = (const double *)(base + o_thermo);
  dm.eff = (const double *)(base + o_eff);
  dm.falloff = (const double *)(base + o_fo);
  dm.program = base + o_prog;

  // ---- mechanism-specialised kernel (ck_jit.cu); the generic kernel stays as fallback ---
  m->jit_params.eff = (const double *)(base + o_jeff);
  m->jit_params.eff_frag = (const double *)(base + o_efrag);
  m->jit_params.tab = (const double *)(base + o_jtab);
  m->jit_params.thermo = (const double *)(base + o_jthermo);
  m->jit_params.logtab = (const double *)(base + o_jlog);
  if (int st = setup_jit(m, spec, hb.jit_why, hb.jit_smem, (size_t)prop.sharedMemPerMultiprocessor,
                         (size_t)prop.sharedMemPerBlockOptin)) { ck_mech_destroy(m); return st; }
  if (!m->jit_kernel) {
    // generic kernel in use: its own M scratch, one slot per resident block
    if (int st = alloc_scratch(m, m->grid_max, (size_t)std::max(n_mb, 1) * ck::kMBlock * best_threads)) { ck_mech_destroy(m); return st; }
    dm.m_scratch = m->d_scratch;
    dm.slot_busy = m->d_slot_busy;
    dm.n_slots = m->grid_max;
  }
  m->jit_s_reg = spec.pair ? std::min(2 * spec.s_reg, S) : spec.s_reg;
  // ---- the all-DMMA small-mechanism kernel (ck_nu.cu), on request ---------------------------
  if (const char *e = std::getenv("CK_JIT_NU")) {
    if (std::string(e) == "dmma") {
      const std::string err = ck::nu_create(d, n_ranges, hb.range_T, hb.tab_orig, hb.thermo_orig, hb.jit_logtab, hb.falloff,
                                            m->device, m->num_sms, (size_t)prop.sharedMemPerBlockOptin, &m->nu);
      if (!err.empty()) { ck_mech_destroy(m); return fail(CK_EUNSUPPORTED, "CK_JIT_NU=dmma: " + err); }
    }
  }
  // ---- tables of the Jacobian kernel (ck_jac.cu) ------------------------------------------
  {
    const std::string err = ck::jac_create(d, m->num_sms, (size_t)prop.sharedMemPerBlockOptin, &m->jac);
    if (!err.empty()) { ck_mech_destroy(m); return fail(CK_ECUDA, err); }
  }
  // ---- the mechanism-specialised Jacobian kernel (ck_jacj.cu); CK_JAC_KERNEL=v1|v2 keeps the
  //      table-driven ones, =v3 requires this one --------------------------------------------
  {
    const char *e = std::getenv("CK_JAC_KERNEL");
    const std::string which = e ? e : "";
    // CK_JACJ_EXP skips passes of the kernel or feeds it constants, CK_JACJ_TIMING makes it print cycle
    // counters: measurement-only builds whose J is not the Jacobian, behind the same guard as CK_JIT_KC=none
    const bool jac_ablation = env_int("CK_JACJ_EXP", 0) != 0 || std::getenv("CK_JACJ_TIMING") != nullptr;
    if (jac_ablation && env_int("CK_ALLOW_ABLATION", 0) != 1) {
      ck_mech_destroy(m);
      return fail(CK_EINVAL, "CK_JACJ_EXP / CK_JACJ_TIMING build a measurement-only Jacobian kernel whose results "
                             "are not the Jacobian; set CK_ALLOW_ABLATION=1 to build it");
    }
    if (which != "v1" && which != "v2" && m->jac) {
      m->jacj_note = ck::jacj_create(d, spec, hb.jit_tab, m->jit_params.thermo, m->jit_params.logtab,
                                     m->jit_params.eff_frag, m->device, m->num_sms,
                                     (size_t)prop.sharedMemPerBlockOptin, &m->jacj);
      m->jac_ablation = jac_ablation && m->jacj;
      if (!m->jacj && which == "v3") {
        const std::string why = m->jacj_note;
        ck_mech_destroy(m);
        return fail(CK_EUNSUPPORTED, "CK_JAC_KERNEL=v3 but " + why);
      }
    }
  }
  *out = m;
  return CK_OK;
}

extern "C" void ck_mech_destroy(ck_mech *m) {
  if (!m) return;
  if (m->d_tables) cudaFree(m->d_tables);
  if (m->d_scratch) cudaFree(m->d_scratch);
  if (m->d_slot_busy) cudaFree(m->d_slot_busy);
  ck::jac_destroy(m->jac);
  ck::jacj_destroy(m->jacj);
  ck::nu_destroy(m->nu);
  if (m->d_stage) cudaFree(m->d_stage);
  if (m->host_in) cudaStreamDestroy(m->host_in);
  if (m->host_out) cudaStreamDestroy(m->host_out);
  for (cudaEvent_t e : m->host_ev) if (e) cudaEventDestroy(e);
  if (m->rk4_graph) cudaGraphExecDestroy(m->rk4_graph);
  if (m->rk4_lib) cudaLibraryUnload(m->rk4_lib);
  for (cudaLibrary_t l : m->split_lib) if (l) cudaLibraryUnload(l);
  if (m->d_rk4) cudaFree(m->d_rk4);
  if (m->jit_lib) cudaLibraryUnload(m->jit_lib);
  delete m;
}

namespace {
int jit_tiling(const ck_mech *m, int64_t N, int *tile_cells);
}

extern "C" int ck_source_terms(const ck_mech *m, const double *T, const double *P,
                               const double *Y, int64_t N, double *wdot, double *dTdt,
                               void *stream) {
  if (!m) return fail(CK_EINVAL, "mechanism handle is NULL");
  if (N < 0) return fail(CK_EINVAL, "N must be >= 0");
  if (N == 0) return CK_OK;
  if (!T || !P || !Y || !wdot || !dTdt) return fail(CK_EINVAL, "a state or result pointer is NULL");
  if (((uintptr_t)T | (uintptr_t)P | (uintptr_t)Y | (uintptr_t)wdot | (uintptr_t)dTdt) & 7u)
    return fail(CK_EINVAL, "pointers must be 8-byte aligned");
  cudaError_t ce;
  if (m->nu) {
    ce = ck::nu_launch(m->nu, T, P, Y, N, wdot, dTdt, (cudaStream_t)stream);
  } else if (m->n_split > 0 && N <= (int64_t)m->split_cells[m->n_split - 1] * m->num_sms) {
    // small batch: one wave of tiles, the most threads per cell whose tiles hold the batch
    int v = 0;
    while (N > (int64_t)m->split_cells[v] * m->num_sms) ++v;
    ck::JitParams prm = m->jit_params;
    prm.T = T; prm.P = P; prm.Y = Y; prm.wdot = wdot; prm.dTdt = dTdt; prm.N = N;
    int64_t tc = (N + m->num_sms - 1) / m->num_sms;
    tc = std::min<int64_t>(m->split_cells[v], (tc + 31) / 32 * 32);
    prm.tile_cells = (int)tc;
    void *args[] = {&prm};
    ce = cudaLaunchKernel((const void *)m->split_kernel[v], dim3((unsigned)((N + tc - 1) / tc)), dim3(256), args,
                          m->split_smem[v], (cudaStream_t)stream);
  } else if (m->jit_kernel) {
    ck::JitParams prm = m->jit_params;
    prm.T = T; prm.P = P; prm.Y = Y; prm.wdot = wdot; prm.dTdt = dTdt; prm.N = N;
    // Balanced tiles: the fewest waves of full tiles the grid needs, then the tile size that
    // spreads the cells evenly over grid x waves (a multiple of the warp size), so that a batch
    // just past a multiple of the grid does not pay for a nearly empty last wave and a small
    // batch uses every SM.
    const int grid = jit_tiling(m, N, &prm.tile_cells);
    void *args[] = {&prm};
    ce = cudaLaunchKernel((const void *)m->jit_kernel, dim3(grid), dim3(m->jit_threads), args,
                          m->jit_smem, (cudaStream_t)stream);
  } else {
    ce = ck::launch_source_terms(m, T, P, Y, N, wdot, dTdt, (cudaStream_t)stream);
  }
  if (ce != cudaSuccess) return fail_cuda(ce, "ck_source_terms launch");
  return CK_OK;
}

// The no-allocation variant (ck_static.cu): argument checks here as for ck_source_terms, the kernel,
// its static scratch and the per-device set-up there.
extern "C" int ck_source_terms_static(const ck_mech *m, const double *T, const double *P, const double *Y,
                                      int64_t N, double *wdot, double *dTdt, void *stream) {
  if (!m) return fail(CK_EINVAL, "mechanism handle is NULL");
  if (N < 0) return fail(CK_EINVAL, "N must be >= 0");
  if (N == 0) return CK_OK;
  if (!T || !P || !Y || !wdot || !dTdt) return fail(CK_EINVAL, "a state or result pointer is NULL");
  if (((uintptr_t)T | (uintptr_t)P | (uintptr_t)Y | (uintptr_t)wdot | (uintptr_t)dTdt) & 7u)
    return fail(CK_EINVAL, "pointers must be 8-byte aligned");
  std::string err;
  const int st = ck::static_source_terms(m, T, P, Y, N, wdot, dTdt, (cudaStream_t)stream, &err);
  return st == CK_OK ? CK_OK : fail(st, err);
}

extern "C" int ck_jacobian(const ck_mech *m, const double *T, const double *P, const double *Y,
                           int64_t N, double *J, void *stream) {
  if (!m) return fail(CK_EINVAL, "mechanism handle is NULL");
  if (N < 0) return fail(CK_EINVAL, "N must be >= 0");
  if (N == 0) return CK_OK;
  if (!T || !P || !Y || !J) return fail(CK_EINVAL, "a state or result pointer is NULL");
  if (((uintptr_t)T | (uintptr_t)P | (uintptr_t)Y | (uintptr_t)J) & 7u)
    return fail(CK_EINVAL, "pointers must be 8-byte aligned");
  if (!m->jac)
    return fail(CK_EUNSUPPORTED, "ck_jacobian: not available for this mechanism (approximate-ANN Kc, S > 127, "
                                 "or the tile does not fit shared memory)");
  // the specialised kernel is compiled, and its scratch allocated, on the first call; if that fails
  // the table-driven kernels take this and every later call (ck_mech_note-style: jacj_note says why)
  bool jit = m->jacj && ck::jacj_takes(m->jacj, J);
  if (jit) {
    const std::string err = ck::jacj_ensure(m->jacj);
    if (!err.empty()) {
      if (m->env_jac_v3_required) return fail(CK_EUNSUPPORTED, "CK_JAC_KERNEL=v3 but " + err);
      jit = false;
    }
  }
  if (!jit) {
    const std::string err = ck::jac_ensure(m->jac);
    if (!err.empty()) return fail(CK_ENOMEM, err);
  }
  const cudaError_t ce = jit ? ck::jacj_launch(m->jacj, T, P, Y, N, J, (cudaStream_t)stream)
                             : ck::jac_launch(m->jac, T, P, Y, N, J, (cudaStream_t)stream);
  if (ce != cudaSuccess) return fail_cuda(ce, "ck_jacobian launch");
  return CK_OK;
}

extern "C" int ck_source_terms_host(ck_mech *m, const double *T, const double *P,
                                    const double *Y, int64_t N, double *wdot, double *dTdt,
                                    void *stream) {
  if (!m) return fail(CK_EINVAL, "mechanism handle is NULL");
  if (N < 0) return fail(CK_EINVAL, "N must be >= 0");
  if (N == 0) return CK_OK;
  if (!T || !P || !Y || !wdot || !dTdt) return fail(CK_EINVAL, "a state or result pointer is NULL");
  const int64_t S = m->dev.S;
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t ce;
  if (m->stage_cells < N) {
    if (m->d_stage) { cudaFree(m->d_stage); m->d_stage = nullptr; m->stage_cells = 0; }
    ce = cudaMalloc((void **)&m->d_stage, (size_t)(2 * S + 3) * N * sizeof(double));
    if (ce != cudaSuccess) return fail(CK_ENOMEM, std::string("cudaMalloc staging: ") + cudaGetErrorString(ce));
    m->stage_cells = N;
  }
  // Chunks of cells pipelined over three streams: chunk c's rows go up on the handle's
  // copy-in stream while chunk c-1 computes on `stream` and chunk c-2's results come down on
  // the copy-out stream (PCIe is full duplex, so the two copy directions overlap as well).
  // Each chunk has its own compact SoA region of the staging buffer: T | P | Y[S] | wdot[S] | dTdt.
  int64_t n_chunks = N / 65536;
  if (n_chunks > CK_HOST_CHUNKS) n_chunks = CK_HOST_CHUNKS;
  if (m->env_host_chunks) n_chunks = m->env_host_chunks;
  if (n_chunks < 1) n_chunks = 1;
  if (n_chunks > CK_HOST_CHUNKS) n_chunks = CK_HOST_CHUNKS;
  if (n_chunks > 1 && !m->host_in) {
    if ((ce = cudaStreamCreateWithFlags(&m->host_in, cudaStreamNonBlocking)) != cudaSuccess ||
        (ce = cudaStreamCreateWithFlags(&m->host_out, cudaStreamNonBlocking)) != cudaSuccess)
      return fail_cuda(ce, "cudaStreamCreate (host pipeline)");
    for (int i = 0; i < 2 * CK_HOST_CHUNKS + 2; ++i)
      if ((ce = cudaEventCreateWithFlags(&m->host_ev[i], cudaEventDisableTiming)) != cudaSuccess)
        return fail_cuda(ce, "cudaEventCreate (host pipeline)");
  }
  const int64_t per = ((N + n_chunks - 1) / n_chunks + 255) & ~(int64_t)255;   // keeps rows 16-byte aligned
  const size_t pitch = (size_t)N * sizeof(double);
  cudaStream_t s_in = n_chunks > 1 ? m->host_in : st, s_out = n_chunks > 1 ? m->host_out : st;
  if (n_chunks > 1) {
    // the copies start after whatever the caller has queued on `stream`
    cudaEvent_t e0 = m->host_ev[2 * CK_HOST_CHUNKS];
    if ((ce = cudaEventRecord(e0, st)) != cudaSuccess || (ce = cudaStreamWaitEvent(s_in, e0, 0)) != cudaSuccess ||
        (ce = cudaStreamWaitEvent(s_out, e0, 0)) != cudaSuccess)
      return fail_cuda(ce, "host pipeline start");
  }
  int c = 0;
  for (int64_t c0 = 0; c0 < N; c0 += per, ++c) {
    const int64_t n = (N - c0 < per) ? (N - c0) : per;
    double *dT = m->d_stage + (size_t)(2 * S + 3) * c0, *dP = dT + n, *dY = dP + n, *dW = dY + S * n, *dD = dW + S * n;
    const size_t w = (size_t)n * sizeof(double);
    if ((ce = cudaMemcpyAsync(dT, T + c0, w, cudaMemcpyHostToDevice, s_in)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(dP, P + c0, w, cudaMemcpyHostToDevice, s_in)) != cudaSuccess ||
        (ce = cudaMemcpy2DAsync(dY, w, Y + c0, pitch, w, (size_t)S, cudaMemcpyHostToDevice, s_in)) != cudaSuccess)
      return fail_cuda(ce, "host to device copy");
    if (n_chunks > 1 && ((ce = cudaEventRecord(m->host_ev[2 * c], s_in)) != cudaSuccess ||
                         (ce = cudaStreamWaitEvent(st, m->host_ev[2 * c], 0)) != cudaSuccess))
      return fail_cuda(ce, "host pipeline (copy-in event)");
    if (int rc = ck_source_terms(m, dT, dP, dY, n, dW, dD, stream)) return rc;
    if (n_chunks > 1 && ((ce = cudaEventRecord(m->host_ev[2 * c + 1], st)) != cudaSuccess ||
                         (ce = cudaStreamWaitEvent(s_out, m->host_ev[2 * c + 1], 0)) != cudaSuccess))
      return fail_cuda(ce, "host pipeline (kernel event)");
    if ((ce = cudaMemcpy2DAsync(wdot + c0, pitch, dW, w, w, (size_t)S, cudaMemcpyDeviceToHost, s_out)) != cudaSuccess ||
        (ce = cudaMemcpyAsync(dTdt + c0, dD, w, cudaMemcpyDeviceToHost, s_out)) != cudaSuccess)
      return fail_cuda(ce, "device to host copy");
  }
  if (n_chunks > 1) {
    // `stream` ends after the last copy-out, so that the caller's later work is ordered behind it
    cudaEvent_t e1 = m->host_ev[2 * CK_HOST_CHUNKS + 1];
    if ((ce = cudaEventRecord(e1, s_out)) != cudaSuccess || (ce = cudaStreamWaitEvent(st, e1, 0)) != cudaSuccess)
      return fail_cuda(ce, "host pipeline end");
  }
  if ((ce = cudaStreamSynchronize(st)) != cudaSuccess) return fail_cuda(ce, "cudaStreamSynchronize");
  return CK_OK;
}

namespace {

// The explicit-RK4 stage variant of the specialised kernel (CK_RK4 in ck_jit_kernel.cuh),
// compiled on first use.  Leaves m->rk4_kernel NULL if there is no specialised kernel, if
// CK_RK4_FUSED=0, or if the compilation fails (the separate stage kernels are used then).
void ensure_rk4_kernel(ck_mech *m) {
  if (m->rk4_tried) return;
  m->rk4_tried = true;
  if (!m->jit_kernel || m->jit_spec.pair) return;   // (the two-threads-per-cell kernel has no stage variant)
  if (!m->env_rk4_fused) return;
  ck::JitSpec spec = m->jit_spec;
  spec.rk4 = true;
  std::vector<char> cubin;
  if (!ck::jit_compile(ck::jit_generate_source(spec), &cubin).empty()) return;
  if (cudaLibraryLoadData(&m->rk4_lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0) != cudaSuccess) {
    m->rk4_lib = nullptr;
    return;
  }
  if (cudaLibraryGetKernel(&m->rk4_kernel, m->rk4_lib, "ck_source_terms_jit") != cudaSuccess ||
      cudaKernelSetAttributeForDevice(m->rk4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)m->jit_smem,
                                      m->device) != cudaSuccess) {
    cudaLibraryUnload(m->rk4_lib);
    m->rk4_lib = nullptr; m->rk4_kernel = nullptr;
  }
  cudaGetLastError();
}

// tile size and grid of a launch of the specialised kernel (balanced tiles, see ck_source_terms)
int jit_tiling(const ck_mech *m, int64_t N, int *tile_cells) {
  const int64_t nt = m->jit_cells;
  const int64_t waves = ((N + nt - 1) / nt + m->jit_grid_max - 1) / m->jit_grid_max;
  int64_t tc = (N + m->jit_grid_max * waves - 1) / (m->jit_grid_max * waves);
  tc = std::min<int64_t>(nt, (tc + 31) / 32 * 32);
  if (m->env_tile) tc = std::min<int64_t>(nt, std::max(32, m->env_tile / 32 * 32));   // (test knob, read at create)
  *tile_cells = (int)tc;
  return (int)std::min<int64_t>((N + tc - 1) / tc, m->jit_grid_max);
}

// one RK4 step on `st`: 4 fused stage launches, or 4 x (source terms + stage kernel)
int rk4_enqueue_step(ck_mech *m, double *T, const double *P, double *Y, int64_t N, double dt, cudaStream_t st) {
  const int64_t S = m->dev.S;
  double *Ts = m->d_rk4, *Ys = Ts + N, *wd = Ys + S * N, *dT = wd + S * N, *aT = dT + N, *aY = aT + N;
  if (m->rk4_kernel) {
    for (int stage = 1; stage <= 4; ++stage) {
      ck::JitParams prm = m->jit_params;
      prm.T = stage == 1 ? T : Ts; prm.P = P; prm.Y = stage == 1 ? Y : Ys; prm.N = N;
      prm.wdot = nullptr; prm.dTdt = nullptr;
      prm.rk_stage = stage; prm.rk_dt = dt; prm.rk_T0 = T; prm.rk_Y0 = Y; prm.rk_accT = aT; prm.rk_accY = aY;
      prm.rk_Tout = stage == 4 ? T : Ts; prm.rk_Yout = stage == 4 ? Y : Ys;
      const int grid = jit_tiling(m, N, &prm.tile_cells);
      void *args[] = {&prm};
      cudaError_t ce = cudaLaunchKernel((const void *)m->rk4_kernel, dim3(grid), dim3(m->jit_threads), args,
                                        m->jit_smem, st);
      if (ce != cudaSuccess) return fail_cuda(ce, "rk4 fused stage launch");
    }
    return CK_OK;
  }
  for (int stage = 1; stage <= 4; ++stage) {
    const double *Tin = stage == 1 ? T : Ts, *Yin = stage == 1 ? Y : Ys;
    if (int rc = ck_source_terms(m, Tin, P, Yin, N, wd, dT, (void *)st)) return rc;
    cudaError_t ce = ck::launch_rk4_stage(stage, m, P, T, Y, Ts, Ys, wd, dT, aT, aY, N, dt, st);
    if (ce != cudaSuccess) return fail_cuda(ce, "rk4 stage kernel launch");
  }
  return CK_OK;
}

}  // namespace

extern "C" int ck_rk4_integrate(ck_mech *m, double *T, const double *P, double *Y, int64_t N, double dt,
                                int64_t n_steps, int use_graph, void *stream) {
  if (!m) return fail(CK_EINVAL, "mechanism handle is NULL");
  if (N < 0 || n_steps < 0) return fail(CK_EINVAL, "N and n_steps must be >= 0");
  if (!(dt > 0.0) || !std::isfinite(dt)) return fail(CK_EINVAL, "dt must be finite and > 0");
  if (N == 0 || n_steps == 0) return CK_OK;
  if (!T || !P || !Y) return fail(CK_EINVAL, "a state pointer is NULL");
  if (((uintptr_t)T | (uintptr_t)P | (uintptr_t)Y) & 7u) return fail(CK_EINVAL, "pointers must be 8-byte aligned");
  const int64_t S = m->dev.S;
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t ce;
  if (m->rk4_cells < N) {
    if (m->rk4_graph) { cudaGraphExecDestroy(m->rk4_graph); m->rk4_graph = nullptr; }
    if (m->d_rk4) { cudaFree(m->d_rk4); m->d_rk4 = nullptr; m->rk4_cells = 0; }
    // N even keeps every row 16-byte aligned for the bulk loads of the source-term kernel
    ce = cudaMalloc((void **)&m->d_rk4, (size_t)(3 * S + 3) * N * sizeof(double));
    if (ce != cudaSuccess) return fail(CK_ENOMEM, std::string("cudaMalloc rk4 workspace: ") + cudaGetErrorString(ce));
    m->rk4_cells = N;
  }
  ensure_rk4_kernel(m);
  if (!use_graph) {
    for (int64_t s = 0; s < n_steps; ++s)
      if (int rc = rk4_enqueue_step(m, T, P, Y, N, dt, st)) return rc;
    return CK_OK;
  }
  const bool same = m->rk4_graph && m->rk4_key[0] == T && m->rk4_key[1] == P && m->rk4_key[2] == Y &&
                    m->rk4_key_N == N && m->rk4_key_dt == dt;
  if (!same) {
    if (m->rk4_graph) { cudaGraphExecDestroy(m->rk4_graph); m->rk4_graph = nullptr; }
    // capture on a private stream so that a legacy/default `stream` argument also works
    cudaStream_t cap = nullptr;
    if ((ce = cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking)) != cudaSuccess) return fail_cuda(ce, "cudaStreamCreate");
    cudaGraph_t graph = nullptr;
    ce = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    int rc = CK_OK;
    if (ce == cudaSuccess) {
      rc = rk4_enqueue_step(m, T, P, Y, N, dt, cap);
      ce = cudaStreamEndCapture(cap, &graph);
    }
    if (ce == cudaSuccess && rc == CK_OK) ce = cudaGraphInstantiate(&m->rk4_graph, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    cudaStreamDestroy(cap);
    if (rc != CK_OK) return rc;
    if (ce != cudaSuccess) { m->rk4_graph = nullptr; return fail_cuda(ce, "capturing the RK4 step"); }
    m->rk4_key[0] = T; m->rk4_key[1] = P; m->rk4_key[2] = Y; m->rk4_key_N = N; m->rk4_key_dt = dt;
  }
  for (int64_t s = 0; s < n_steps; ++s)
    if ((ce = cudaGraphLaunch(m->rk4_graph, st)) != cudaSuccess) return fail_cuda(ce, "cudaGraphLaunch");
  return CK_OK;
}

extern "C" int64_t ck_mech_info(const ck_mech *m, int what) {
  if (!m) return -1;
  switch (what) {
    case 0: return m->dev.S;
    case 1: return m->dev.R;
    case 2: return m->nnz_reac;
    case 3: return m->nnz_prod;
    case 4: return m->nnz_net;
    case 5: return m->n_three_body;
    case 6: return m->n_lindemann;
    case 7: return m->n_troe;
    case 8: return m->dev.n_ranges;
    case 9: return m->nu ? ck::nu_threads(m->nu) : (m->jit_kernel ? m->jit_threads : m->dev.threads);
    case 10: return m->jit_kernel ? m->jit_blocks_per_sm : m->blocks_per_sm;
    case 11: return (int64_t)(m->nu ? ck::nu_smem(m->nu) : (m->jit_kernel ? m->jit_smem : m->smem_bytes));
    case 12: return 1;
    case 13: return m->nnz_eff;
    case 14: return m->jit_kernel ? 1 : 0;
    case 15: return m->jit_kernel ? m->jit_s_reg : 0;
    case 16: return (m->jacj && !ck::jacj_failed(m->jacj)) ? ck::jacj_cells(m->jacj) : (m->jac ? ck::jac_cells_per_tile(m->jac) : 0);
    case 17: return (m->jit_kernel && m->jit_spec.pair) ? 1 : 0;
    case 18: return ((m->jit_kernel && m->jit_spec.kc_none) || m->jac_ablation) ? 1 : 0;
    case 19: return m->jit_kernel ? m->jit_spec.prec : 0;
    case 20: return m->nu ? 1 : 0;
    case 21: return m->n_split ? (int64_t)m->split_cells[m->n_split - 1] * m->num_sms : 0;
    case 22: return (m->jacj && !ck::jacj_failed(m->jacj)) ? 3 : (m->jac ? (ck::jac_cells_per_tile(m->jac) == 32 && ck::jac_is_v2(m->jac) ? 2 : 1) : 0);
    default: return -1;
  }
}

extern "C" const char *ck_mech_note(const ck_mech *m) { return m ? m->jit_note.c_str() : ""; }

extern "C" int64_t ck_mech_jit_source(const ck_mech_desc *d, char *buf, int64_t cap) {
  if (validate(d)) return -1;
  HostBuild hb;
  build_host(d, &hb);
  if (!hb.jit_why.empty()) { fail(CK_EUNSUPPORTED, hb.jit_why); return -1; }
  // (CK_JIT_SOURCE_SPLIT=K: the text of the small-batch shape instead, for offline inspection)
  if (const int k = env_int("CK_JIT_SOURCE_SPLIT", 0)) { hb.spec.split = k; hb.spec.threads = 256; hb.spec.min_blocks = 1; }
  // (CK_JACJ_DUMP=path: also write the text of the specialised Jacobian kernel there)
  if (std::getenv("CK_JACJ_DUMP")) {
    ck::JacJit *jj = nullptr;
    ck::jacj_create(d, hb.spec, hb.jit_tab, nullptr, nullptr, nullptr, -1, 148, kSmemPerBlock, &jj);
  }
  const std::string src = ck::jit_generate_source(hb.spec);
  if (buf && cap > 0) {
    const size_t n = std::min((size_t)cap - 1, src.size());
    std::memcpy(buf, src.data(), n);
    buf[n] = '\0';
  }
  return (int64_t)src.size() + 1;
}

extern "C" int ck_measure_fp64_peak(double *fma_per_s, void *stream) {
  if (!fma_per_s) return fail(CK_EINVAL, "fma_per_s is NULL");
  cudaError_t ce = ck::measure_fp64_peak(fma_per_s, (cudaStream_t)stream);
  if (ce != cudaSuccess) return fail_cuda(ce, "ck_measure_fp64_peak");
  return CK_OK;
}

extern "C" int ck_measure_peaks(double *out, void *stream) {
  if (!out) return fail(CK_EINVAL, "out is NULL");
  cudaError_t ce = ck::measure_peaks(out, (cudaStream_t)stream);
  if (ce != cudaSuccess) return fail_cuda(ce, "ck_measure_peaks");
  return CK_OK;
}
