// ck_jit.cu -- run-time specialisation of the fused kernel to one mechanism.
//
// generate_source() writes the unrolled reaction list (ck_reactions) for the mechanism
// into the hand-written kernel text of ck_jit_kernel.cuh; NVRTC compiles it for sm_100a;
// the CUDA runtime's library API loads the cubin.  NVRTC is opened with dlopen so that
// libck.so itself has no link-time dependency on it (the library must load, and report
// errors through the ABI, on machines without NVRTC or without a GPU).
#include <cuda_runtime.h>
#include <dlfcn.h>
#include <nvrtc.h>
#include <sys/stat.h>
#include <unistd.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <fstream>
#include <sstream>
#include <string>
#include <vector>

#include "ck_internal.h"

namespace ck {

namespace {

const char *kKernelText =
#include "ck_jit_source.inc"
    ;

struct Nvrtc {
  void *handle = nullptr;
  decltype(&nvrtcCreateProgram) CreateProgram = nullptr;
  decltype(&nvrtcCompileProgram) CompileProgram = nullptr;
  decltype(&nvrtcDestroyProgram) DestroyProgram = nullptr;
  decltype(&nvrtcGetCUBINSize) GetCUBINSize = nullptr;
  decltype(&nvrtcGetCUBIN) GetCUBIN = nullptr;
  decltype(&nvrtcGetProgramLogSize) GetProgramLogSize = nullptr;
  decltype(&nvrtcGetProgramLog) GetProgramLog = nullptr;
  decltype(&nvrtcGetErrorString) GetErrorString = nullptr;
  decltype(&nvrtcVersion) Version = nullptr;
  bool ok = false;
};

Nvrtc &nvrtc() {
  static Nvrtc n = [] {
    Nvrtc r;
    const char *names[] = {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12",
                           "/usr/local/cuda/lib64/libnvrtc.so"};
    for (const char *nm : names) {
      r.handle = dlopen(nm, RTLD_NOW | RTLD_LOCAL);
      if (r.handle) break;
    }
    if (!r.handle) return r;
#define CK_SYM(f) r.f = (decltype(r.f))dlsym(r.handle, "nvrtc" #f)
    CK_SYM(CreateProgram); CK_SYM(CompileProgram); CK_SYM(DestroyProgram); CK_SYM(GetCUBINSize);
    CK_SYM(GetCUBIN); CK_SYM(GetProgramLogSize); CK_SYM(GetProgramLog); CK_SYM(GetErrorString);
    CK_SYM(Version);
#undef CK_SYM
    r.ok = r.CreateProgram && r.CompileProgram && r.DestroyProgram && r.GetCUBINSize && r.GetCUBIN &&
           r.GetProgramLogSize && r.GetProgramLog && r.GetErrorString && r.Version;
    return r;
  }();
  return n;
}

std::string lit(double v) {
  char buf[40];
  std::snprintf(buf, sizeof buf, "%.17g", v);
  std::string s(buf);
  if (s.find_first_of(".eEni") == std::string::npos) s += ".0";
  return s;
}

// nu^T ln C of one side of a reaction as an expression: sums and fmas of CK_LNC(k) (or, for the
// species in `pinned`, of the register copy lcp<k> made at the top of ck_reactions)
std::string gather_expr(const std::vector<std::pair<int, double>> &side, const std::vector<char> &pinned) {
  if (side.empty()) return "CK_LIT(0.0)";
  std::string e;
  for (size_t i = 0; i < side.size(); ++i) {
    const std::string c = pinned[side[i].first] ? "lcp" + std::to_string(side[i].first)
                                                 : "CK_LNC(" + std::to_string(side[i].first) + ")";
    const double nu = side[i].second;
    const std::string l = "CK_LIT(" + lit(nu) + ")";
    if (i == 0) e = (nu == 1.0) ? c : (l + " * " + c);
    else e = (nu == 1.0) ? (e + " + " + c) : ("fma(" + l + ", " + c + ", " + e + ")");
  }
  return e;
}

uint64_t fnv1a(const std::string &s, uint64_t h) {
  for (unsigned char c : s) { h ^= c; h *= 1099511628211ull; }
  return h;
}

// Directory of the cubin cache, or "" for no cache: $CK_JIT_CACHE if set ("" disables), else
// $HOME/.cache/ck_jit; without HOME there is no cache (a predictable path under /tmp could be
// planted by another user).  Created 0700.
std::string cache_dir() {
  const char *e = std::getenv("CK_JIT_CACHE");
  if (e && !*e) return "";
  std::string d = e ? e : "";
  if (d.empty()) {
    const char *home = std::getenv("HOME");
    if (!home || !*home) return "";
    d = std::string(home) + "/.cache/ck_jit";
    ::mkdir((d.substr(0, d.find_last_of('/'))).c_str(), 0700);
  }
  ::mkdir(d.c_str(), 0700);
  return d;
}

// Cache file = header {magic, payload bytes, FNV-1a of the payload} + cubin.  A file that does
// not verify (truncated, corrupt, foreign) is removed and the kernel is compiled again.
struct CacheHeader {
  char magic[8];
  uint64_t size, hash;
};
const char kCacheMagic[8] = {'C', 'K', 'J', 'I', 'T', '0', '0', '2'};

uint64_t fnv1a_bytes(const char *p, size_t n) {
  uint64_t h = 1469598103934665603ull;
  for (size_t i = 0; i < n; ++i) { h ^= (unsigned char)p[i]; h *= 1099511628211ull; }
  return h;
}

bool cache_read(const std::string &path, std::vector<char> *cubin) {
  std::ifstream in(path, std::ios::binary);
  if (!in) return false;
  CacheHeader h;
  in.read((char *)&h, sizeof h);
  bool ok = in.gcount() == (std::streamsize)sizeof h && std::memcmp(h.magic, kCacheMagic, 8) == 0 &&
            h.size > 0 && h.size < (1ull << 30);
  if (ok) {
    cubin->resize((size_t)h.size);
    in.read(cubin->data(), (std::streamsize)h.size);
    ok = in.gcount() == (std::streamsize)h.size && in.peek() == std::ifstream::traits_type::eof() &&
         fnv1a_bytes(cubin->data(), cubin->size()) == h.hash;
  }
  in.close();
  if (!ok) {
    cubin->clear();
    ::unlink(path.c_str());
  }
  return ok;
}

void cache_write(const std::string &path, const std::vector<char> &cubin) {
  const std::string tmp = path + ".tmp" + std::to_string((long)getpid());
  std::ofstream out(tmp, std::ios::binary);
  CacheHeader h;
  std::memcpy(h.magic, kCacheMagic, 8);
  h.size = cubin.size();
  h.hash = fnv1a_bytes(cubin.data(), cubin.size());
  out.write((const char *)&h, sizeof h);
  out.write(cubin.data(), (std::streamsize)cubin.size());
  out.close();
  if (out) std::rename(tmp.c_str(), path.c_str());
  else ::unlink(tmp.c_str());
}

}  // namespace

std::string jit_generate_source(const JitSpec &s) {
  std::ostringstream o;
  o << "#define CK_S " << s.S << "\n#define CK_R " << s.R << "\n#define CK_NT " << s.threads
    << "\n#define CK_MINB " << s.min_blocks << "\n#define CK_NRANGES " << s.n_ranges
    << "\n#define CK_NM " << s.n_m << "\n#define CK_NMB " << s.n_mb
    << "\n#define CK_NFO " << s.n_fo << "\n#define CK_TAB_SMEM " << (s.tab_in_smem ? 1 : 0)
    << "\n#define CK_M_DMMA " << (s.m_dmma ? 1 : 0) << "\n#define CK_M_HINT " << (s.m_hint ? 1 : 0) << "\n#define CK_PREC " << s.prec << "\n#define CK_SPLIT " << s.split << "\n#define CK_KCONST " << (s.kconst ? 1 : 0) << "\n#define CK_SYNC_EVERY " << s.sync_every
    << "\n#define CK_B " << s.block << "\n#define CK_NBLK " << (int)s.rxn.size() / s.block
    << "\n#define CK_G_TB0 " << s.group_end[1] << "\n#define CK_G_FO0 " << s.group_end[3]
    << "\n#define CK_TAB_NRANGES " << s.tab_ranges << "\n#define CK_ROW " << s.row
    << "\n#define CK_RK4 " << (s.rk4 ? 1 : 0) << "\n#define CK_KC_ANN " << (s.kc_ann ? 1 : 0) << "\n#define CK_KC_NONE " << (s.kc_none ? 1 : 0)
    << "\n#define CK_PAIR " << (s.pair ? 1 : 0) << "\n#define CK_LUT_REP " << s.lut_rep << "\n#define CK_SREG " << s.s_reg << "\n#define CK_PERM " << (s.perm.empty() ? 0 : 1) << "\n";
  if (!s.perm.empty()) {
    o << "__constant__ int ck_c_perm[" << s.perm.size() << "] = {";
    for (size_t i = 0; i < s.perm.size(); ++i) o << (i ? "," : "") << (i % 16 == 0 ? "\n  " : " ") << s.perm[i];
    o << "};\n";
  }
  auto emit = [&](const char *name, const std::vector<double> &v) {
    o << "__constant__ double " << name << "[" << (v.empty() ? 1 : v.size()) << "] = {";
    for (size_t i = 0; i < v.size(); ++i) o << (i ? "," : "") << (i % 6 == 0 ? "\n  " : " ") << lit(v[i]);
    if (v.empty()) o << "0.0";
    o << "};\n";
  };
  if (s.kc_ann) {
    o << "#define CK_ANN_NIN " << s.ann_nin << "\n#define CK_ANN_NL " << s.ann_nl << "\n#define CK_ANN_NH "
      << s.ann_nh << "\n#define CK_ANN_NHP " << s.ann_nhp << "\n#define CK_ANN_ACT " << s.ann_act << "\n";
    emit("ck_c_ann", s.ann_const);
  }
  if (s.rk4) emit("ck_c_W", s.mol_weight);
  emit("ck_c_rangeT", s.range_T);
  emit("ck_c_falloff", s.falloff);
  const std::string text(kKernelText);
  const std::string marker = "//@@CK_GENERATED_REACTIONS@@";
  const size_t at = text.find(marker);
  o << text.substr(0, at);
  const int B = s.block, nblk = (int)s.rxn.size() / B;
  const int nhot = s.pair ? std::min(2 * s.s_reg, s.S) : s.s_reg;
  // the s.pin species that the gathers read most often keep their ln C in a register for the whole walk
  std::vector<char> pinned(s.S, 0);
  if (s.pin > 0 && !s.pair && s.split <= 1) {
    std::vector<int> cnt(s.S, 0), idx(s.S);
    for (const JitReaction &r : s.rxn) {
      for (const auto &e : r.reac) cnt[e.first]++;
      if (r.reversible) for (const auto &e : r.prod) cnt[e.first]++;
    }
    for (int k = 0; k < s.S; ++k) idx[k] = k;
    std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return cnt[a] > cnt[b]; });
    for (int i = 0; i < std::min(s.pin, s.S); ++i) pinned[idx[i]] = 1;
  }
  // accumulator of internal species sp, and (pair mode) the half of the cell's thread pair that owns it
  auto acc_of = [&](int sp, int *owner) {
    if (sp < nhot) {
      *owner = s.pair ? (sp & 1) : 0;
      return "w[" + std::to_string(s.pair ? sp >> 1 : sp) + "]";
    }
    const int c = sp - nhot;
    *owner = s.pair ? (c & 1) : 0;
    return "CK_WC(" + std::to_string(c) + ")";
  };
  // scatters of block k (Eq. 2) restricted to the species owned by `half` (-1: all), q from `qsrc`
  auto scatters = [&](int k, int half, const std::string &qsrc) {
    for (int bb = 0; bb < B; ++bb) {
      const JitReaction &r = s.rxn[(size_t)k * B + bb];
      const std::string q = qsrc + std::to_string(bb) + (qsrc == "q[" ? "]" : "");
      for (size_t e = 0; e < r.net.size(); ++e) {
        int owner = 0;
        const std::string acc = acc_of(r.net[e].first, &owner);
        if (half >= 0 && owner != half) continue;
        const double c = r.net[e].second;
        if (c == 1.0) o << "        " << acc << " += " << q << ";\n";
        else if (c == -1.0) o << "        " << acc << " -= " << q << ";\n";
        else o << "        " << acc << " = fma(" << lit(c) << ", " << q << ", " << acc << ");\n";
      }
    }
  };
  auto gathers = [&](int k) {
    for (int bb = 0; bb < B; ++bb) {
      const JitReaction &r = s.rxn[(size_t)k * B + bb];
      o << "        gf[" << bb << "] = " << gather_expr(r.reac, pinned) << ";";
      if (r.index >= 0) o << "  // reaction " << r.index;
      o << "\n        gr[" << bb << "] = " << (r.reversible ? gather_expr(r.prod, pinned) : std::string("CK_LIT(0.0)")) << ";\n";
    }
  };
  const char *names[6] = {"ck_core<0, 1>", "ck_core<0, 0>", "ck_core<1, 1>", "ck_core<1, 0>",
                          "ck_core<2, 1>", "ck_core<2, 0>"};
  auto dispatch = [&](const char *indent, const char *slot) {
    bool first = true;
    for (int g = 0; g < 6; ++g) {
      const int lo = g ? s.group_end[g - 1] : 0;
      if (s.group_end[g] == lo) continue;
      o << indent << (first ? "if" : "else if") << " (blk < " << s.group_end[g] << ") " << names[g]
        << "(x, blk, " << slot << ", gf, gr, q);\n";
      first = false;
    }
  };
  o << "__device__ __forceinline__ void ck_reactions(const CkCtx &x, double (&w)[CK_SREG > 0 ? CK_SREG : 1]) {\n"
    << "  ck_real gf[CK_B], gr[CK_B];\n  double q[CK_B];\n";
  for (int k = 0; k < s.S; ++k)
    if (pinned[k]) o << "  const ck_real lcp" << k << " = CK_LNC(" << k << ");\n";
  if (s.split > 1) {
    // Small-batch shape: part x.half of a cell's CK_SPLIT threads walks blocks x.half, x.half + K, ..;
    // a block's gathers, its rate core and its scatters (into this thread's own accumulators of
    // every species) follow each other, two switches per block.
    o << "#pragma unroll 1\n  for (int blk = x.half; blk < CK_NBLK; blk += CK_SPLIT) {\n    switch (blk) {\n";
    for (int k = 0; k < nblk; ++k) {
      o << "      case " << k << ":\n";
      gathers(k);
      o << "        break;\n";
    }
    o << "    }\n";
    dispatch("    ", "0");
    o << "    switch (blk) {\n";
    for (int k = 0; k < nblk; ++k) {
      o << "      case " << k << ":\n";
      scatters(k, -1, "q[");
      o << "        break;\n";
    }
    o << "    }\n  }\n}\n";
  } else if (!s.pair && s.straight > 0 && s.tab_in_smem) {
    // Straight-line walk: gathers, the rate core (inlined with the block number as a literal)
    // and scatters of every block one after the other, no loop, no switch: the instruction
    // stream is sequential, so the fetch unit's prefetcher can run ahead of it.
    for (int k = 0; k < nblk; ++k) {
      int g = 0;
      while (k >= s.group_end[g]) ++g;
      o << "  {\n";
      gathers(k);
      o << "    " << names[g] << "(x, " << k << ", 0, gf, gr, q);\n";
      scatters(k, -1, "q[");
      o << "  }\n";
    }
    o << "}\n";
  } else if (!s.pair) {
    // One switch case per loop trip: the scatters of the previous block (Eq. 2) and the
    // gathers of this one (Eq. 4), so that the unique code is walked in address order with one
    // indirect branch per block; trip CK_NBLK only scatters the last block.
    o << "#if !CK_TAB_SMEM\n  ck_ring_issue(x, 0, 0);\n#endif\n"
      << "#pragma unroll 1\n  for (int blk = 0; blk <= CK_NBLK; ++blk) {\n"
      << "#if !CK_TAB_SMEM\n    ck_ring_issue(x, blk + 1, (blk + 1) & 1);\n#endif\n"
      << "    switch (blk) {\n";
    for (int k = 0; k <= nblk; ++k) {
      o << "      case " << k << ":\n";
      if (k > 0) scatters(k - 1, -1, "q[");
      if (k < nblk) gathers(k);
      o << "        break;\n";
    }
    o << "    }\n#if !CK_TAB_SMEM\n    ck_ring_wait();\n#endif\n";
    dispatch("    ", "blk & 1");
    if (s.sync_every > 0)
      o << "    if (blk % " << s.sync_every << " == " << s.sync_every - 1 << ") __syncthreads();\n";
    o << "  }\n}\n";
  } else {
    // Two threads per cell: trip pr handles the pair of blocks (2 pr, 2 pr + 1).  Half h gathers and
    // evaluates block 2 pr + h and publishes its q in the exchange buffer; after the pair's barrier
    // (next trip) each half scatters BOTH blocks into the species it owns: its own q from
    // registers, the other half's from shared memory.  One switch per half.
    o << "#if !CK_TAB_SMEM\n  ck_ring_issue(x, x.half, 0);\n#endif\n"
      << "#pragma unroll 1\n  for (int pr = 0; pr <= (CK_NBLK + 1) / 2; ++pr) {\n"
      << "    const int blk = 2 * pr + x.half;\n"
      << "#if !CK_TAB_SMEM\n    ck_ring_issue(x, blk + 2, (pr + 1) & 1);\n#endif\n";
    for (int h = 0; h < 2; ++h) {
      o << (h == 0 ? "    if (x.half == 0) {\n" : "    } else {\n") << "    switch (pr) {\n";
      for (int k = 0; k <= (nblk + 1) / 2; ++k) {
        o << "      case " << k << ": {\n";
        if (k > 0) {
          for (int bb = 0; bb < B; ++bb)
            o << "        const double o" << bb << " = CK_XQ(" << ((k - 1) & 1) << ", " << (1 - h) << ", " << bb << ");\n";
          if (2 * (k - 1) + h < nblk) scatters(2 * (k - 1) + h, h, "q[");
          if (2 * (k - 1) + (1 - h) < nblk) scatters(2 * (k - 1) + (1 - h), h, "o");
        }
        if (2 * k + h < nblk) gathers(2 * k + h);
        o << "      } break;\n";
      }
      o << "    }\n";
    }
    o << "    }\n#if !CK_TAB_SMEM\n    ck_ring_wait();\n#endif\n"
      << "    if (blk < CK_NBLK) {\n";
    dispatch("      ", "pr & 1");
    o << "#pragma unroll\n      for (int b = 0; b < CK_B; ++b) CK_XQ(pr & 1, x.half, b) = q[b];\n"
      << "    }\n    ck_pair_sync(x.bar);\n  }\n}\n";
  }
  o << text.substr(at + marker.size());
  return o.str();
}

// Compiles `src` to a cubin for sm_100a.  Returns "" on success, else an error message.
// use_cache = false skips the lookup (the caller's retry after a cached cubin failed to load);
// the freshly compiled cubin still replaces the cache entry.
std::string jit_compile(const std::string &src, std::vector<char> *cubin, bool use_cache) {
  Nvrtc &n = nvrtc();
  if (!n.ok) return "NVRTC (libnvrtc.so.12) could not be loaded";
  int major = 0, minor = 0;
  n.Version(&major, &minor);

  // cubin cache keyed by the source text and the NVRTC version
  std::string path;
  const std::string dir = cache_dir();
  if (!dir.empty()) {
    char name[96];
    const uint64_t h1 = fnv1a(src, 1469598103934665603ull), h2 = fnv1a(src, 0x9E3779B97F4A7C15ull);
    std::snprintf(name, sizeof name, "/ck_%016llx%016llx_nvrtc%d_%d.ckbin", (unsigned long long)h1,
                  (unsigned long long)h2, major, minor);
    path = dir + name;
    if (use_cache && cache_read(path, cubin)) return "";
  }

  nvrtcProgram prog;
  nvrtcResult rc = n.CreateProgram(&prog, src.c_str(), "ck_source_terms_jit.cu", 0, nullptr, nullptr);
  if (rc != NVRTC_SUCCESS) return std::string("nvrtcCreateProgram: ") + n.GetErrorString(rc);
  const char *opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo", "--fmad=true"};
  rc = n.CompileProgram(prog, (int)(sizeof opts / sizeof opts[0]), opts);
  if (rc != NVRTC_SUCCESS) {
    size_t ls = 0;
    n.GetProgramLogSize(prog, &ls);
    std::string log(ls, '\0');
    if (ls) n.GetProgramLog(prog, &log[0]);
    n.DestroyProgram(&prog);
    return std::string("nvrtcCompileProgram: ") + n.GetErrorString(rc) + "\n" + log;
  }
  size_t sz = 0;
  rc = n.GetCUBINSize(prog, &sz);
  if (rc == NVRTC_SUCCESS) {
    cubin->resize(sz);
    rc = n.GetCUBIN(prog, cubin->data());
  }
  n.DestroyProgram(&prog);
  if (rc != NVRTC_SUCCESS) return std::string("nvrtcGetCUBIN: ") + n.GetErrorString(rc);
  if (!path.empty()) cache_write(path, *cubin);
  return "";
}

}  // namespace ck
