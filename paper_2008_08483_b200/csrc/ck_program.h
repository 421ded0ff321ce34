// ck_program.h -- internal layout of the device-resident mechanism ("reaction program").
// Shared by the host builder (ck_build.cu) and the kernels (ck_kernels.cu); not part of
// the public ABI (include/ck.h) and not shared with oracle/.
//
// ck_mech_create turns the dense matrices of the paper (nu', nu'', E)
// into a compact stream of per-reaction records that a thread-per-cell kernel walks with
// warp-uniform (broadcast) reads:
//
//   record := RecHeader | fwd[4] | rev[n_ranges][8] | coef[nr+np+nsc] (even count)
//             | offs[nr+np+nsc] (int32, count padded to a multiple of 4)
//
//   fwd   = { ln A, b, -Ea/R, 0 }                       Arrhenius layer, Eq. 6
//   rev   = ln k_r = fwd - ln Kc folded onto the Gibbs features of Eq. 10:
//           r0 + r1 ln T + r2 T + r3 T^2 + r4 T^3 + r5 T^4 + r6 / T, one row per
//           temperature range (ranges are delimited by the distinct T_mid values).
//           This is Eq. 11's two-layer linear net -(X_G W_G + B_G) nu collapsed into one
//           layer X_G (-W_G nu) - B_G nu at create time, with the standard-concentration
//           term in the bias as PAPER.md:114 does.
//   coef  = nu'_k (reactants), nu''_k (products), nu''_k - nu'_k (scatter list)
//   offs  = species indices of the three lists
#pragma once
#include <cstdint>

namespace ck {

constexpr double kRu = 8314.46261815324;   // J/(kmol K)
constexpr double kCFloor = 1e-300;         // kmol/m^3 (reading Q9)
constexpr int kMBlock = 8;                 // reactions per register block of M = C E
constexpr int kThermoStride = 24;          // doubles per species in the thermo table
constexpr int kFalloffStride = 8;          // doubles per falloff reaction

struct RecHeader {        // 32 bytes
  int32_t size_bytes;     // whole record, multiple of 16
  int32_t nr, np, nsc;    // list lengths
  int32_t type;           // CK_ELEMENTARY .. CK_TROE
  int32_t reversible;
  int32_t m_slot;         // row of the M scratch (type != 0), else -1
  int32_t fo_idx;         // row of the falloff table (type >= 2), else -1
};

// thermo table row (per species), doubles:
//  [0] T_mid  [1..5] cp/R lo a1..a5  [6..10] cp/R hi  [11..16] h/RT lo: a1, a2/2, a3/3,
//  a4/4, a5/5, a6  [17..22] h/RT hi  [23] pad
// falloff table row: [0] ln A0 [1] b0 [2] -Ea0/R [3] alpha [4] -1/T*** [5] -1/T* [6] -T**
//  [7] kind (2.0 Lindemann, 3.0 Troe)

struct DeviceMech {
  int32_t S, R;
  int32_t n_ranges;           // number of temperature ranges (distinct T_mid values + 1)
  int32_t n_m;                // third-body + falloff reactions (rows of M)
  int32_t n_m_blocks;         // ceil(n_m / kMBlock)
  int32_t threads;            // threads (= cells) per block
  const double *inv_W;        // [S]
  const double *range_T;      // [n_ranges - 1] ascending
  const double *thermo;       // [S][kThermoStride]
  const double *eff;          // [n_m_blocks][S][kMBlock], zero padded
  const double *falloff;      // [n_fo][kFalloffStride]
  const unsigned char *program;  // R records back to back
  // M = C E scratch (L2 resident): n_slots slots of [n_m_blocks * kMBlock][threads] doubles.  A block
  // takes a free slot for its lifetime (slot_busy[s]: 0 free, 1 taken), so launches that overlap on
  // different streams never share one; n_slots >= the blocks that can be resident on the device.
  double *m_scratch;
  int *slot_busy;
  int32_t n_slots;
};

}  // namespace ck
