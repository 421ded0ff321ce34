// ck_internal.h -- host-side handle and the launch interface between ck_api.cu
// (validation, mechanism build, C ABI) and ck_kernels.cu (device code).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <utility>
#include <vector>

#include "../../include/ck.h"
#include "ck_program.h"

#define CK_HOST_CHUNKS 16   // most chunks ck_source_terms_host splits a batch into

namespace ck {

// Kernel argument of the mechanism-specialised kernel; must match CkParams in
// ck_jit_kernel.cuh field for field.
struct JitParams {
  const double *eff, *eff_frag, *tab, *thermo, *logtab;
  double *m_scratch;
  int *slot_busy;
  int n_slots;
  int slot_elems;              // doubles per slot, one value for every shape built on the handle
  const double *T, *P, *Y;
  double *wdot, *dTdt;
  long long N;
  int tile_cells;
  int rk_stage;
  double rk_dt;
  const double *rk_T0, *rk_Y0;
  double *rk_accT, *rk_accY;
  double *rk_Tout, *rk_Yout;
};

struct JitReaction {
  int index = 0, type = 0, reversible = 1, m_slot = -1, fo_idx = -1;
  std::vector<std::pair<int, double>> reac, prod, net;   // (species, coefficient)
};

struct JitSpec {
  int S = 0, R = 0, threads = 0, min_blocks = 1, n_ranges = 1, n_m = 0, n_fo = 0;
  int n_mb = 0;                // blocks of 8 rows of M, padded to an even count
  bool tab_in_smem = true;
  bool m_dmma = true;          // M = C E on DMMA.8x8x4 (else register-tiled DFMA)
  bool m_hint = true;          // M scratch accesses carry an L2 evict_last policy
  int split = 1;               // small-batch shape: threads per cell (CK_SPLIT in ck_jit_kernel.cuh)
  int prec = 0;                // ck_mech_desc.precision: 0 fp64, 1 mixed (CK_PREC in ck_jit_kernel.cuh)
  int sync_every = 0;          // block barrier every n reaction blocks (0 = never)
  int block = 4;               // reactions per block of the core
  int s_reg = 0;               // register accumulators per thread (internal species order); rest in smem
  bool pair = false;           // two threads per cell (CK_PAIR in ck_jit_kernel.cuh): threads = 2 x cells
  std::vector<int> perm;       // internal species -> row of Y / wdot; empty = identity
  int tab_ranges = 1, row = 10;  // rate table: ranges and doubles per row
  bool rk4 = false;            // the explicit-RK4 stage variant of the kernel (ck_rk4_integrate)
  std::vector<double> mol_weight;  // [S], internal order (RK4 variant)
  bool kc_none = false;        // measurement-only ablation: no equilibrium layer (CK_JIT_KC=none)
  bool kc_ann = false;         // approximate ANN for ln Kc in place of the exact layer
  int ann_nin = 0, ann_nl = 0, ann_nh = 0, ann_nhp = 0, ann_act = 0;
  std::vector<double> ann_const;   // mean | 1/std | W_in | B | W_hid
  int lut_rep = 1;             // interleaved copies of the exp table (16: conflict-free lookups)
  bool kconst = false;         // polynomial coefficients as constant-bank operands (else literals)
  int pin = 0;                 // species whose ln C the reaction walk keeps in registers (the most gathered ones)
  int straight = 0;            // n > 0: the reaction walk in straight-line code, rate core inlined per block (measurement knob CK_JIT_STRAIGHT)
  int group_end[6] = {0, 0, 0, 0, 0, 0};   // end block of (elementary, three-body, falloff) x (rev, irrev)
  std::vector<JitReaction> rxn;
  std::vector<double> inv_W, range_T, falloff;   // constant-bank tables
};

struct JacMech;   // device tables of the Jacobian kernel (ck_jac.cu)
// Builds them; returns "" (with *out NULL if the mechanism is unsupported there) or an error text.
std::string jac_create(const ck_mech_desc *d, int num_sms, size_t smem_block_max, JacMech **out);
void jac_destroy(JacMech *jm);
int jac_cells_per_tile(const JacMech *jm);
bool jac_is_v2(const JacMech *jm);
// First launch of the second table-driven kernel: allocates its scratch ("" or the error text); a no-op later
// and for the first kernel.
std::string jac_ensure(JacMech *jm);
cudaError_t jac_launch(const JacMech *jm, const double *T, const double *P, const double *Y, int64_t N,
                       double *J, cudaStream_t stream);

// The mechanism-specialised Jacobian kernel (ck_jacj.cu / ck_jacj_kernel.cuh), NVRTC-compiled.
// jacj_create generates the kernel text and its tables (no device work) and returns "" with *out set, or
// returns why the kernel is not available (*out NULL; the table-driven kernels of ck_jac.cu remain).
// device < 0: only generate the source (CK_JACJ_DUMP).
struct JacJit;
std::string jacj_create(const ck_mech_desc *d, const JitSpec &spec, const std::vector<double> &tab10,
                        const double *d_thermo, const double *d_logtab, const double *d_eff_frag, int device,
                        int num_sms, size_t smem_blk, JacJit **out);
// First use: compiles and loads the kernel, uploads its tables, allocates its scratch ("" or the error text).
std::string jacj_ensure(JacJit *jj);
void jacj_destroy(JacJit *jj);
int jacj_cells(const JacJit *jj);
// true once jacj_ensure has failed: the table-driven kernels serve the handle from then on
bool jacj_failed(const JacJit *jj);
// false if J is not aligned for the kernel's bulk row stores (16 bytes): the table-driven kernels take the call
bool jacj_takes(const JacJit *jj, const double *J);
cudaError_t jacj_launch(const JacJit *jj, const double *T, const double *P, const double *Y, int64_t N, double *J,
                        cudaStream_t stream);

// The all-DMMA small-mechanism kernel (ck_nu.cu / ck_nu_kernel.cuh).
struct NuMech;
std::string nu_create(const ck_mech_desc *d, int n_ranges, const std::vector<double> &range_T,
                      const std::vector<double> &tab_orig, const std::vector<double> &thermo,
                      const std::vector<double> &logtab, const std::vector<double> &falloff, int device,
                      int num_sms, size_t smem_block_max, NuMech **out);
void nu_destroy(NuMech *nm);
cudaError_t nu_launch(const NuMech *nm, const double *T, const double *P, const double *Y, int64_t N, double *wdot,
                      double *dTdt, cudaStream_t stream);
int nu_threads(const NuMech *nm);
size_t nu_smem(const NuMech *nm);

std::string jit_generate_source(const JitSpec &spec);
// Compiles to a cubin for sm_100a with NVRTC; returns "" on success, else the error text.
// use_cache = false: do not read the on-disk cubin cache (it is still refreshed).
std::string jit_compile(const std::string &src, std::vector<char> *cubin, bool use_cache = true);

}  // namespace ck

struct ck_mech {
  ck::DeviceMech dev{};       // device pointers + sizes, passed to the kernel by value
  int device = 0;
  int blocks_per_sm = 1;
  int num_sms = 1;
  int grid_max = 1;           // persistent grid size = num_sms * blocks_per_sm
  size_t smem_bytes = 0;      // dynamic shared memory per block
  // statistics for ck_mech_info
  int64_t nnz_reac = 0, nnz_prod = 0, nnz_net = 0, nnz_eff = 0;
  int n_three_body = 0, n_lindemann = 0, n_troe = 0;
  // one device allocation holding every table; m_scratch separately
  void *d_tables = nullptr;
  double *d_scratch = nullptr;    // M = C E scratch of the kernel in use (slots, ck_program.h)
  int *d_slot_busy = nullptr;
  // mechanism-specialised kernel (NULL kernel => the generic kernel is used)
  cudaLibrary_t jit_lib = nullptr;
  cudaKernel_t jit_kernel = nullptr;
  ck::JitParams jit_params{};
  int jit_threads = 0, jit_blocks_per_sm = 0, jit_grid_max = 0, jit_s_reg = 0;
  int jit_cells = 0;          // cells per block of the specialised kernel (= threads, or half with pair)
  size_t jit_smem = 0;
  ck::JitSpec jit_spec;       // kept to compile the RK4 stage variant on first use
  // the small-batch shape of the specialised kernel (CK_SPLIT threads per cell, tiles of 32 cells),
  // used by ck_source_terms when the batch fits one wave of such tiles
  // (up to three of them: 8, 4 and 2 threads per cell, tiles of 32, 64 and 128 cells)
  cudaLibrary_t split_lib[3] = {nullptr, nullptr, nullptr};
  cudaKernel_t split_kernel[3] = {nullptr, nullptr, nullptr};
  size_t split_smem[3] = {0, 0, 0};
  int split_cells[3] = {0, 0, 0};
  int n_split = 0;
  cudaLibrary_t rk4_lib = nullptr;
  cudaKernel_t rk4_kernel = nullptr;
  bool rk4_tried = false;
  std::string jit_note;       // why the specialised kernel is not in use, if so
  // analytic Jacobian (ck_jacobian): NULL if unsupported for this mechanism
  ck::JacMech *jac = nullptr;
  ck::JacJit *jacj = nullptr;   // the mechanism-specialised Jacobian kernel, used when present
  std::string jacj_note;        // why it is not, if so
  bool jac_ablation = false;    // it was built with CK_JACJ_EXP / CK_JACJ_TIMING (CK_ALLOW_ABLATION=1): J is not the Jacobian
  // all-DMMA small-mechanism kernel (CK_JIT_NU=dmma), used by ck_source_terms when present
  ck::NuMech *nu = nullptr;
  // staging for ck_source_terms_host
  double *d_stage = nullptr;
  int64_t stage_cells = 0;
  // ... and its copy/compute pipeline: copy-in and copy-out streams, per chunk one event after
  // the copy-in and one after the kernel, plus a start and an end event
  cudaStream_t host_in = nullptr, host_out = nullptr;
  cudaEvent_t host_ev[2 * CK_HOST_CHUNKS + 2] = {};
  // ck_rk4_integrate: workspace (stage state, slopes, weighted slope sums) and the captured step
  double *d_rk4 = nullptr;
  int64_t rk4_cells = 0;
  cudaGraphExec_t rk4_graph = nullptr;
  // Environment knobs of the calls below, read ONCE by ck_mech_create: the asynchronous entry points
  // (ck_source_terms, ck_jacobian, ck_rk4_integrate, ck_source_terms_host) never call getenv.
  int env_tile = 0;               // CK_JIT_TILE: forced tile size of the specialised kernel (test knob; 0 = balanced)
  int env_host_chunks = 0;        // CK_HOST_CHUNKS (0 = unset: by batch size)
  bool env_rk4_fused = true;      // CK_RK4_FUSED=0: unfused RK4 stages
  bool env_jac_v3_required = false;   // CK_JAC_KERNEL=v3: a failed specialisation is an error
  const void *rk4_key[3] = {nullptr, nullptr, nullptr};   // T, P, Y the graph was captured for
  int64_t rk4_key_N = 0;
  double rk4_key_dt = 0.0;
};

namespace ck {

// Sets the kernel's shared-memory attribute and reports occupancy. Returns cudaError_t.
cudaError_t kernel_configure(int threads, size_t smem_bytes, int *blocks_per_sm);

// Launches the fused source-term kernel on `stream` (asynchronous).
cudaError_t launch_source_terms(const ck_mech *m, const double *T, const double *P,
                                const double *Y, int64_t N, double *wdot, double *dTdt,
                                cudaStream_t stream);

// ck_source_terms_static's launch (ck_static.cu): the table-driven kernel with its M scratch in a
// file-scope device array.  Returns a ck_status; *err carries the message of a non-zero one.
int static_source_terms(const ck_mech *m, const double *T, const double *P, const double *Y, int64_t N,
                        double *wdot, double *dTdt, cudaStream_t stream, std::string *err);

// One RK4 stage's update kernel (ck_rk4.cu); stage = 1..4.
cudaError_t launch_rk4_stage(int stage, const ck_mech *m, const double *P, double *T0, double *Y0, double *Ts,
                             double *Ys, const double *wdot, const double *dTdt, double *accT, double *accY,
                             int64_t N, double dt, cudaStream_t stream);

// DFMA throughput microbenchmark (thread-level FMA instructions per second), ck_peaks.cu.
cudaError_t measure_fp64_peak(double *fma_per_s, cudaStream_t stream);
// All FP64 microbenchmarks of ck_peaks.cu; out as documented at ck_measure_peaks in ck.h.
#define CK_N_PEAKS 10
cudaError_t measure_peaks(double out[CK_N_PEAKS], cudaStream_t stream);

}  // namespace ck
