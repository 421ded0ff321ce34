/* ck.h -- C ABI of the B200-native batched chemical source-term library.
 *
 * The library evaluates, for N independent reacting cells, the paper's ANN-form source
 * term (Barwey & Raman, arXiv 2008.08483; line numbers are /root/reference/PAPER.md):
 *
 *   (1) Arrhenius layer      ln k_f = [ln A, b, -Ea/R] . [1, ln T, 1/T]        Eq. 5-6, l.72-83
 *   (2) NASA-7 thermo layer  g/RT, h/RT, cp/R from X_G = [ln T, T..T^4, 1/T]   Eq. 10,  l.101-108
 *   (3) equilibrium layer    ln Kc = -nu^T (g/RT - ln(p_ref/(Ru T)))           Eq. 8-11, l.93-114
 *                            ln k_r = ln k_f - ln Kc                           Eq. 7,   l.87-91
 *   (4) third bodies M = C E, Lindemann / Troe falloff                         Sec. 2.4, l.157-159
 *   (5) log-rate layers      q_f = exp(nu'^T ln C + ln k_f),
 *                            q_r = exp(nu''^T ln C + ln k_r)                   Eq. 4,   l.58
 *   (6) net-rate contraction wdot = (nu'' - nu') (q_f - q_r)                   Eq. 2,   l.49-51
 *       energy term          dT/dt = -sum_k h_k wdot_k / (rho cp)              l.185 (const.-P reactor)
 *
 * Every step runs in hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 * Units are SI-kmol: T [K], P [Pa], W [kg/kmol], C [kmol/m^3], wdot [kmol/m^3/s],
 * Ru = 8314.46261815324 J/(kmol K).  All floating point is IEEE fp64.
 *
 * Error behaviour: every function returns CK_OK (0) or a positive ck_status; nothing
 * throws or aborts across this boundary.  ck_last_error() returns a thread-local,
 * human-readable message for the last non-zero status on the calling thread.
 */
#ifndef CK_H
#define CK_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum ck_status {
  CK_OK = 0,
  CK_EINVAL = 1,       /* bad argument (NULL, negative size, invalid mechanism data) */
  CK_ENOMEM = 2,       /* host or device allocation failed */
  CK_ECUDA = 3,        /* a CUDA runtime call failed; see ck_last_error() */
  CK_EUNSUPPORTED = 4  /* unknown reaction type, or a mechanism too large for the kernels */
} ck_status;

/* reaction types (Sec. 2.4) */
enum { CK_ELEMENTARY = 0, CK_THREE_BODY = 1, CK_LINDEMANN = 2, CK_TROE = 3 };

typedef struct ck_mech ck_mech; /* opaque; owns device memory on the device current at create */

/* Approximate ANN for log Kc (Sec. 2.3, Eq. 12-14, Fig. 2): a drop-in
 * replacement of the exact equilibrium layer (3).  X_0 = standardised input features of
 * temperature, X_{l+1} = sigma(X_l W_l + B_l) for l = 0 .. N_L-1 (N_L hidden layers of N_H
 * neurons), a linear output layer of width R giving the standardised log Kc~, then
 * log Kc~_j = out_mean[j] + out_std[j] * y_j (standardisation: PAPER.md:141).
 *   n_in = 1: X_0 = [ln T]                              (Architecture 2, the one the paper runs)
 *   n_in = 6: X_0 = [ln T, T, T^2, T^3, T^4, 1/T]       (Architecture 1, the exact layer's features)
 * standardised as (x - in_mean) / in_std.  All arrays are HOST pointers, row-major, copied.
 * The hidden layers' weights (everything but W_out, B_out, out_*) must fit 40 KB (they are
 * constant-bank operands of the kernel): e.g. 3 layers of 50 neurons; else CK_EUNSUPPORTED.
 * The weights come from the caller (the paper trains them; training is not part
 * of this library).  Everything else of the path is unchanged: k_r = k_f / Kc~ (Eq. 7). */
enum { CK_ANN_RELU = 0 /* Eq. 13 */, CK_ANN_ELU = 1 /* Eq. 14 */ };
typedef struct ck_kc_ann {
  int32_t n_in;           /* 1 or 6 */
  int32_t n_layers;       /* N_L hidden layers, 1..8 */
  int32_t n_hidden;       /* N_H neurons per hidden layer, 1..64 */
  int32_t activation;     /* CK_ANN_RELU or CK_ANN_ELU */
  const double *in_mean;  /* [n_in] */
  const double *in_std;   /* [n_in] > 0 */
  const double *W_in;     /* [n_in][N_H]         input i -> neuron h at i*N_H + h */
  const double *B;        /* [N_L][N_H]          bias of hidden layer l */
  const double *W_hid;    /* [N_L-1][N_H][N_H]   layer l: neuron g -> neuron h at (l*N_H + g)*N_H + h;
                                                  may be NULL if N_L == 1 */
  const double *W_out;    /* [N_H][R]            neuron h -> reaction j at h*R + j */
  const double *B_out;    /* [R] */
  const double *out_mean; /* [R] */
  const double *out_std;  /* [R] */
} ck_kc_ann;

/* Arithmetic of the rate layers (ck_mech_desc.precision).  CK_PREC_F64 is the product: IEEE fp64
 * throughout, the north_star tolerance holds.  The others are the reduced-precision variants the
 * paper names as future work ("single or half-precision environments"; SURVEY.md
 * section 8(f) item 4); state, results, M = C E and the accumulation of Eq. 2 stay fp64 in all of them:
 *   CK_PREC_MIXED      the exp activations of Eq. 4 (and of the falloff layer) take their mantissa
 *                      2^f from the fp32 special-function unit, the exponent is handled in fp64 /
 *                      integer arithmetic; every rate carries a relative error <= ~6e-7, whatever its
 *                      magnitude (no overflow: the synthetic configs' rates reach e^250);
 *   CK_PREC_F32_RATES  additionally ln C, the gathers of Eq. 4 and the Arrhenius / equilibrium
 *                      layers (Eq. 6, 11) run in fp32: a rate carries an ABSOLUTE error of about
 *                      1e-7 |ln q| x (terms) in its logarithm, i.e. 1e-5 .. 1e-4 relative.
 * Both need the mechanism-specialised kernel (CK_EUNSUPPORTED otherwise); measured errors and
 * times: DESIGN.md section 15, bench.py --precision. */
enum { CK_PREC_F64 = 0, CK_PREC_MIXED = 1, CK_PREC_F32_RATES = 2 };

/* Mechanism description.  All pointers are HOST pointers; the arrays are copied by
 * ck_mech_create and stay owned by the caller.  S = n_species, R = n_reactions.
 * Matrices are row-major with the species index first: element (k, j) at k*R + j. */
typedef struct ck_mech_desc {
  int32_t n_species;         /* S >= 1 */
  int32_t n_reactions;       /* R >= 1 */
  const double *mol_weight;  /* [S]   W_k > 0, kg/kmol */
  const double *nu_reac;     /* [S*R] nu'_kj  >= 0; real values allowed */
  const double *nu_prod;     /* [S*R] nu''_kj >= 0 */
  const double *ln_A;        /* [R]   ln of the pre-exponential factor (Eq. 5-6), SI-kmol units */
  const double *b;           /* [R]   temperature exponent */
  const double *Ea_over_R;   /* [R]   activation temperature Ea/R, K */
  const uint8_t *reversible; /* [R]   1/0; NULL => all reversible */
  const double *nasa_lo;     /* [S*7] a1..a7 of species k at k*7, used for T <= T_mid[k] */
  const double *nasa_hi;     /* [S*7] a1..a7, used for T > T_mid[k] */
  const double *T_mid;       /* [S]   cutoff temperature, K */
  const uint8_t *rxn_type;   /* [R]   CK_ELEMENTARY..CK_TROE; NULL => all elementary */
  const double *eff;         /* [S*R] third-body efficiencies E_kj; read only in
                                      columns with rxn_type != 0; NULL => all 1 */
  const double *ln_A0;       /* [R]   low-pressure-limit Arrhenius set; read where rxn_type is */
  const double *b0;          /* [R]   CK_LINDEMANN or CK_TROE (the main set is then k_inf);   */
  const double *Ea0_over_R;  /* [R]   may be NULL if there is no falloff reaction             */
  const double *troe;        /* [R*4] alpha, T***, T*, T** at j*4; T** = +INF gives the
                                      3-parameter form; read where rxn_type == CK_TROE */
  double p_ref;              /* Pa, standard-state pressure of the NASA data (Eq. 8) */
  const ck_kc_ann *kc_ann;   /* NULL: exact equilibrium layer; else log Kc from this network.
                                Needs the mechanism-specialised kernel (CK_EUNSUPPORTED if it
                                cannot be built) */
  int32_t precision;         /* CK_PREC_F64 (0, the default of a zeroed struct), CK_PREC_MIXED or
                                CK_PREC_F32_RATES */
} ck_mech_desc;

/* Validate `desc`, build the device-resident mechanism (sorted reaction program, folded
 * equilibrium-layer coefficients, thermo tables, efficiency matrix) on the current CUDA
 * device and return an opaque handle in *out.  Synchronous.
 * Kernel variant: by default (environment CK_KERNEL unset or "auto") a kernel specialised
 * to the mechanism's structure is compiled with NVRTC for sm_100a (species accumulators in
 * registers for S <= 103, the most updated ones in registers and the rest in shared memory
 * beyond that), falling back to the generic table-driven kernel if no launch shape fits or
 * NVRTC is unavailable; CK_KERNEL=generic forces the generic kernel,
 * CK_KERNEL=jit makes a failed specialisation an error (in auto mode ck_mech_note() says why
 * the generic kernel is in use).  Compiled cubins are cached under $CK_JIT_CACHE (default
 * $HOME/.cache/ck_jit, created 0700; empty string, or no HOME, disables the cache); a cache
 * file carries its size and hash, and one that does not verify or load is removed and rebuilt.
 * Errors: CK_EINVAL (NULL pointers, S/R < 1, W <= 0, negative or non-finite nu, a reaction
 * without reactants or without products, T_mid <= 0, non-positive Troe temperatures,
 * p_ref <= 0), CK_EUNSUPPORTED (unknown rxn_type; S or R beyond the kernels' limits),
 * CK_ENOMEM, CK_ECUDA.  On error *out is set to NULL. */
int ck_mech_create(const ck_mech_desc *desc, ck_mech **out);

/* Source terms of N cells.  T, P, Y, wdot, dTdt are DEVICE pointers, fp64, 8-byte aligned:
 *   T[N] K, P[N] Pa, Y[S][N] mass fractions with species k at Y + k*N (SoA);
 *   wdot[S][N] kmol/m^3/s (Eq. 2), dTdt[N] K/s.
 * `stream` is a cudaStream_t (NULL = default stream).  The call is asynchronous on
 * `stream`, allocates nothing, synchronises nothing and is deterministic run to run.
 * Inputs are not modified; outputs must not alias inputs.  Re-entrant: calls that share one
 * handle may run at the same time on different streams (and from different host threads) as
 * long as their output buffers are distinct.  N == 0 is a
 * successful no-op.  A mass fraction Y_k <= 0 is an absent species: it enters W_mix, cp, M and
 * C as 0, and concentrations are then floored at 1e-300 kmol/m^3 for the log form (DESIGN.md
 * reading Q9); T must be finite and > 0, P > 0; inputs are not screened for NaN.
 * Errors: CK_EINVAL (NULL handle or pointer with N > 0, N < 0), CK_ECUDA. */
int ck_source_terms(const ck_mech *m, const double *T, const double *P, const double *Y,
                    int64_t N, double *wdot, double *dTdt, void *stream);

/* ck_source_terms for callers that cannot allocate device memory: same arguments, same layout,
 * same results to rounding (Eq. 2-11 as listed at the top of this file), but no byte of global
 * memory beyond the handle's tables, the inputs and the outputs comes from an allocator.
 *
 * Who needs it: a solver that hands the whole device to its own memory pool after set-up, so that
 * a later cudaMalloc fails or eats into memory the pool was sized without; a solver that overlaps
 * chemistry with other work on other streams, which cudaMalloc / cudaFree would stall because they
 * synchronise the device; a process that shares a GPU under a fixed memory budget and needs the
 * library's footprint known up front.  Create the handle (ck_mech_create does allocate its tables)
 * during set-up; call this from the time loop.
 *
 * How: it runs the table-driven kernel, one thread per cell (about 6-10 x slower than the
 * specialised kernel of ck_source_terms; this entry point is about where the memory lives, not
 * about speed).  That kernel's only scratch, the third-body concentrations M = C E of the cells a
 * block works on, sits in a fixed array of 32 MiB inside the library image.  Every
 * GPU this library's code is loaded on holds those 32 MiB until the process exits, used or not.
 * Limit: a mechanism may have at most CK_STATIC_MAX_M_ROWS third-body + falloff reactions (rows
 * of M); beyond that the call returns CK_EUNSUPPORTED and says so in ck_last_error(), as it does
 * for handles with the approximate-ANN Kc or a reduced precision (those exist only in the
 * specialised kernel).  N is not limited.
 *
 * First call on a device: it looks up the array's device address and sets the kernel's
 * shared-memory limit (once per device, no allocation, but the CUDA runtime may load the
 * library's code onto the device at that moment).  Make that first call during set-up, before any
 * stream capture; the handle's device must be the current one (CK_EINVAL otherwise).
 *
 * The array is shared by all handles and all calls on a device and is divided by block index, so
 * NOT re-entrant: two calls that can be on the GPU at the same time (different streams or host
 * threads) overwrite each other's M values and return wrong rates without any error.  Order all
 * calls of this function on a device on one stream (or with events).  The array keeps whatever the
 * last call left; nothing in it needs clearing, because a block writes every M row of a tile
 * before it reads one.  It does not interfere with ck_source_terms, ck_jacobian or
 * ck_rk4_integrate, which keep using the handle's own scratch.
 * Asynchronous on `stream`, deterministic run to run.  Calls no cudaMalloc, cudaFree or other
 * allocating routine, on the first call or later.
 * Errors: CK_EINVAL (as ck_source_terms; wrong current device), CK_EUNSUPPORTED (above), CK_ECUDA. */
#define CK_STATIC_MAX_M_ROWS 512
int ck_source_terms_static(const ck_mech *m, const double *T, const double *P, const double *Y,
                           int64_t N, double *wdot, double *dTdt, void *stream);

/* Same computation with HOST buffers: copies T, P, Y to the device, runs
 * ck_source_terms and copies wdot, dTdt back, then synchronises `stream`.  Batches of
 * 2^17 cells or more are split into up to 16 chunks of cells that are pipelined: a chunk's
 * rows are copied up on a stream owned by the handle while the previous chunk computes on
 * `stream` and the one before is copied back on a second owned stream; the work starts
 * after everything queued on `stream` at the call and `stream` ends after the last copy
 * (environment CK_HOST_CHUNKS=n, read by ck_mech_create, overrides the chunk count, 1 = everything on `stream`).
 * Pinned host memory makes the copies asynchronous; pageable memory also works.
 * Device staging buffers, the two copy streams and their events are owned by the handle and grow
 * on demand: unlike ck_source_terms, calls of this function on ONE handle must not overlap. */
int ck_source_terms_host(ck_mech *m, const double *T, const double *P, const double *Y,
                         int64_t N, double *wdot, double *dTdt, void *stream);

/* The 0-D constant-pressure reactor use of the source term (BASELINE.json
 * configs[4]): n_steps steps of the classic explicit 4-stage Runge-Kutta scheme with step dt
 * [s] on y = (T, Y_1..Y_S) of N independent cells, in place, P[N] constant:
 *   dT/dt = ck_source_terms' energy term,  dY_k/dt = wdot_k W_k / rho,
 *   rho = P / (Ru T sum_k Y_k / W_k);
 *   k1 = f(y), k2 = f(p(y + dt/2 k1)), k3 = f(p(y + dt/2 k2)), k4 = f(p(y + dt k3)),
 *   y <- p(y + dt/6 (k1 + 2 k2 + 2 k3 + k4)),
 * where p projects onto valid thermochemical states: Y <- max(Y, 0), Y <- Y / sum(Y),
 * T <- min(max(T, 250 K), 5000 K) (reading Q14: BASELINE's dt = 1e-9 s is far
 * outside explicit stability for its rate constants, so every state handed to the source
 * term is projected).  ck_source_terms runs once per stage (4 per step); one more kernel per
 * stage forms slopes, weighted sums, the next stage state and its projection.
 * T, P, Y are DEVICE pointers laid out as for ck_source_terms; T and Y are updated in place.
 * use_graph != 0: the step is captured once into a CUDA graph (re-captured when T, P, Y, N or
 * dt change) and replayed n_steps times; use_graph == 0: plain launches.  Asynchronous on
 * `stream`; the workspace ((3S+3) N doubles) is owned by the handle and grows on demand
 * (that allocation synchronises), so calls on ONE handle must not overlap.  N == 0 or
 * n_steps == 0 is a successful no-op.
 * Errors: CK_EINVAL (NULL handle/pointer, negative sizes, dt <= 0), CK_ENOMEM, CK_ECUDA. */
int ck_rk4_integrate(ck_mech *m, double *T, const double *P, double *Y, int64_t N, double dt,
                     int64_t n_steps, int use_graph, void *stream);

/* Analytic Jacobian of the source term (the prerequisite of
 * the GPU stiff integrator PAPER.md:277 names): for each of N cells the (S+1) x (S+1) matrix
 *   J = d(wdot_0 .. wdot_{S-1}, dT/dt) / d(Y_0 .. Y_{S-1}, T)      at constant P,
 * the Y_l taken as S independent variables (the source term is defined for any Y > 0 and is
 * homogeneous of degree 0 in Y, so sum_l Y_l J_il = 0).  It is the chain rule applied to the
 * paper's layers: Eq. 4 dq/dC_l = nu_lj q/C_l; Eq. 6
 * d ln k_f/dT = (b + (Ea/R)/T)/T; Eq. 11 d ln Kc/dT = (dnu^T h/RT - sum dnu)/T;
 * third bodies and falloff through M and Pr; Eq. 2; then
 * C_k = rho Y_k / W_k with rho = P/(Ru T sum_j Y_j/W_j) and the quotient rule on
 * dT/dt = -sum_k h_k wdot_k/(rho cp).  The floor on C, the clamp on Pr and the NASA-7 range
 * switch are not differentiated (reading Q18): T, P and every Y_k must be > 0.
 * T, P, Y: DEVICE pointers laid out as for ck_source_terms.  J: DEVICE, [N][S+1][S+1]
 * doubles, cell-major and row-major per cell (a strided batch of matrices, lda = S+1); row
 * i < S is wdot_i, row S is dT/dt; column l < S is Y_l, column S is T; every entry is written.
 * Asynchronous on `stream`, deterministic run to run (no atomics).  The FIRST call on a handle compiles
 * the mechanism-specialised kernel (NVRTC; cached on disk like the source-term kernel) and allocates its
 * scratch (that synchronises); later calls allocate nothing.  Calls on ONE
 * handle must be ordered on one stream: the per-(reaction, cell) scalars of the cells in flight
 * live in a scratch area the handle owns (ck_source_terms has no such restriction).
 * N == 0 is a successful no-op.  Errors: CK_EINVAL (NULL handle or pointer with N > 0, N < 0,
 * misaligned pointer), CK_EUNSUPPORTED (mechanism with the approximate-ANN Kc, S > 127, or
 * a tile that does not fit shared memory), CK_ECUDA. */
int ck_jacobian(const ck_mech *m, const double *T, const double *P, const double *Y, int64_t N,
                double *J, void *stream);

/* Free the handle and its device memory.  NULL is a no-op. */
void ck_mech_destroy(ck_mech *m);

/* Message for the last non-zero status returned on this thread ("" if none). */
const char *ck_last_error(void);

/* Introspection (for the harness: roofline accounting and launch reporting).
 * what: 0 S, 1 R, 2 nnz(nu'), 3 nnz(nu''), 4 nnz(nu''-nu'), 5 #three-body, 6 #Lindemann,
 *       7 #Troe, 8 #temperature ranges, 9 threads per block, 10 blocks per SM,
 *       11 dynamic shared memory per block (bytes), 12 kernels launched per
 *       ck_source_terms call, 13 nnz(E) counted over third-body and falloff columns,
 *       14 kernel variant in use (0 generic table-driven kernel, 1 mechanism-specialised),
 *       15 species whose accumulators the specialised kernel keeps in registers (the other
 *       S - that many accumulate in shared memory; 0 for the generic kernel),
 *       16 cells per tile of the Jacobian kernel in use (0 if ck_jacobian is unsupported here),
 *       17 1 if the specialised kernel runs two threads per cell (then 9 counts both, and a
 *       block works on half that many cells),
 *       18 1 if the handle was built as a measurement-only ABLATION whose results are not the
 *       source term (environment CK_JIT_KC=none together with CK_ALLOW_ABLATION=1: the
 *       equilibrium layer removed, used by bench.py --ann to cost that layer; or CK_JACJ_EXP /
 *       CK_JACJ_TIMING with CK_ALLOW_ABLATION=1: the specialised Jacobian kernel with passes skipped or
 *       printing cycle counters, J is then not the Jacobian; without CK_ALLOW_ABLATION=1 ck_mech_create
 *       refuses all of these with CK_EINVAL); 0 otherwise,
 *       19 the handle's precision (CK_PREC_*),
 *       20 1 if ck_source_terms runs the all-DMMA small-mechanism kernel (environment
 *       CK_JIT_NU=dmma, at most 16 species and 64 reactions: every contraction of Eq. 2 and 4
 *       and M = C E as dense DMMA.8x8x4 products; same results to rounding),
 *       21 the largest N for which ck_source_terms uses a small-batch shape of the specialised
 *       kernel (8, 4 or 2 threads per cell in tiles of 32, 64 or 128 cells, whichever holds the
 *       batch in one wave; 0 if no such shape was built),
 *       22 the kernel ck_jacobian runs: 0 none (unsupported here), 1 the first table-driven kernel
 *       (lanes = columns), 2 the second (lanes = cells), 3 the mechanism-specialised kernel
 *       (NVRTC-compiled at create time; mechanisms of at most 53 species at fp64 without the
 *       approximate-ANN Kc; environment CK_JAC_KERNEL=v1|v2 keeps the table-driven ones).
 * Returns -1 for a NULL handle or unknown `what`. */
int64_t ck_mech_info(const ck_mech *m, int what);

/* Why the mechanism-specialised kernel is NOT in use on this handle ("" if it is): the NVRTC or
 * load error, "no launch shape fits ...", or "CK_KERNEL=generic".  The string lives as long as
 * the handle.  NULL handle: "". */
const char *ck_mech_note(const ck_mech *m);

/* The CUDA source of the mechanism-specialised kernel ck_mech_create would compile for
 * `desc` on a B200 (generated reaction list inside the hand-written kernel text of
 * csrc/ck_jit_kernel.cuh).  Needs no GPU.  Writes at most cap bytes (NUL terminated) to
 * buf (may be NULL) and returns the size needed including the NUL, or -1 if the
 * description is invalid or the mechanism cannot be specialised (see ck_last_error()). */
int64_t ck_mech_jit_source(const ck_mech_desc *desc, char *buf, int64_t cap);

/* Measured FP64 FMA throughput of the current device, in FMA instructions (thread level)
 * per second: a register-resident DFMA loop on every SM, timed with CUDA events on
 * `stream`.  Used as the roofline denominator for this FP64-pipe-bound path.
 * Returns CK_OK and writes *fma_per_s, or CK_ECUDA. */
int ck_measure_fp64_peak(double *fma_per_s, void *stream);

/* The FP64 microbenchmarks behind the roofline and the sparse-vs-dense design decision
 * (DESIGN.md section 6), each kernel timed alone with CUDA events on
 * `stream` (best of 5).  Writes 10 doubles to the HOST array `out`:
 *   [0] DFMA           thread-level instructions / s (= ck_measure_fp64_peak)
 *   [1] DMMA.8x8x4     warp-level instructions / s, alone (one = 256 FMA = 8 warp-wide DFMA)
 *   [2] DMMA.8x8x4     warp-level instructions / s when 4 independent DFMA follow each DMMA
 *   [3] DFMA           thread-level instructions / s in that same interleaved stream
 *   [4] exp()  [5] log()   CUDA libm calls / s (thread level): the costs the survey's roofline
 *                          accounting charges for an exponential / a logarithm
 *   [6] number of SMs
 *   [7] legacy mma.sync int8 m16n8k32, [8] legacy mma.sync fp16 m16n8k16 (fp32 accumulate): warp-level
 *       instructions / s -- the paths an error-free splitting of M = C E onto low-precision tensor
 *       cores would run on (measured to decide against it)   [9] 0 (reserved)
 * Returns CK_OK, CK_EINVAL (NULL out) or CK_ECUDA. */
int ck_measure_peaks(double *out, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* CK_H */
