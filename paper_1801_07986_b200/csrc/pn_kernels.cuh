// pn_kernels.cuh -- sm_100a kernels of the limited-1PN hot path (arXiv:1801.07986).
// Product code: shares nothing with oracle/.  Citations: /root/reference/PAPER.md:<line>.
//
// Kernels (DESIGN.md section 6 has the roofline of each); the parts are included at the end of this file, in this order:
//   pn_common.cuh, pn_pair_fp64.cuh, pn_pair_cross.cuh, pn_pair_fp32.cuh, pn_epilogue.cuh, pn_small.cuh, pn_energy.cuh
//   S1  pair_fp64_kernel          star-star Newtonian, every ordered pair, tiled (PN_PAIR_TILED)
//       pair_sym_fp64_kernel      the same, every unordered pair once (Newton's third law), general / equal-mass form; the
//                                 j-side sums travel through the lanes of a warp in Gray-code order (N_s >= 3072)
//       pair_cross_fp64_kernel, pair_cross_sym_kernel   NEXT-1/2: S1 + the O(N^2) sums of the Cross terms, Eqs. 2.6 and 2.3, on
//                                 ordered / unordered pairs (cross_prep/sum: O(N))
//       pair_fp32_kernel, pair_sym_fp32_kernel   fp32-pair / fp64-accumulate variant (packed f32x2 arithmetic; split kernels:
//                                 two-float records)
//   S2-S4  epilogue_kernel        partial-sum reduction, BH <-> star Newtonian + 1PN, a_1 reduction, fused RK4 stage update
//   S1-S4  small_path_kernel      N_s < 3072: a whole pn_step call (or one pn_accel) in ONE cooperative launch
//   S5  energy_prep / energy_pair / energy_final   Eq. 2.7, compensated
//   NEXT-3  momentum_prep / momentum_pair / momentum_final   Eq. 2.8, compensated
//   pack / unpack (AoS <-> internal layout)
//
// Internal data layout (all fp64, star index s = body index - 1, padded to NP):
//   JRec  jrec[NP]      : stage position + mass constants of star s, 48 B, 16 B aligned.  This is the record the
//                         O(N^2) pair kernels read; pad records have gm = 0, x = 1e100.
//   double v[3][NP]     : stage velocity, SoA
//   double x0/v0[3][NP] : state at the beginning of the RK4 step;  double sx/sv[3][NP] : weighted sum of k's
//   double part[S][3][NP]: partial star-star accelerations, one slot per j-chunk (tiled) or j-group (symmetric), each entry
//                         written by exactly one block; summed in fixed order by the epilogue (7 or 8 components per slot
//                         in Cross mode)
//   BhState             : the massive object's stage state, step state, k-sums (a handful of doubles)
#pragma once
#include "pn_common.cuh"
#include "pn_pair_fp64.cuh"
#include "pn_pair_cross.cuh"
#include "pn_pair_fp32.cuh"
#include "pn_epilogue.cuh"
#include "pn_small.cuh"
#include "pn_energy.cuh"
