// fused.h -- the fused Chebyshev step of Algorithm 2 for FP32-storage blocks (real or complex).
//
// One step  R_X <- a H S^-1approx R_Y - a c R_Y - zeta zeta1 R_X + a Y Lambda_Y  is computed without ever
// writing T = S^-1approx R_Y or H T to memory:
//   * the recurrence state is kept as  Rt = M_D^-1 R  (and Yt = M_D^-1 Y), so that T = Rt - M_D^-1 C W with
//     W^a = Delta^a_Sinv C^a^dagger Rt  (Eq. 28) needs no diagonal scaling at gather time;
//   * the low-rank terms are folded into the cell contraction as extra K rows ("K-extension"): for every
//     (cell e, atom b) whose assembled projector support touches e,
//         Y_e += [ -H^e (M_D^-1 C^b)|_e ,  C^{e,b} ] [ W^b ; D^b P2^b ],
//     with P2^b = C^b^dagger T = P1^b - sum_a G^{ba} W^a,  G^{ba} = C^b^dagger M_D^-1 C^a  (exact algebra);
//   * the bracket  -a c Rt_Y - zeta zeta1 Rt_X + a Yt Lambda_Y (FP64 add, L374)  is written by the cell kernel itself: the
//     first writer of every node (cell_tcgen05.cu, ordered assembly) stores bracket + its share of  a M_D^-1 H T,  the
//     other cells sharing the node add theirs afterwards, in cell order.
#pragma once
#include "common.h"

struct FusedPlan;

// Build (on first use) the K-extension blocks, the neighbour couplings G^{ab} Delta^b_Sinv and scratch for block
// width B.  Needs mesh, FP64 cell matrices and atoms.  Synchronises the stream the first time and when B grows.
pawfe_status fused_prepare(pawfe_ctx* c, int B);
// The same plus everything else the fused path would allocate on first use for precision mode prec (pawfe_prepare).
pawfe_status fused_prepare_all(pawfe_ctx* c, pawfe_prec prec, int B, bool with_block);
// Drop the plan (cell matrices or atoms changed).
void fused_invalidate(pawfe_ctx* c);
bool fused_supported(pawfe_ctx* c, pawfe_prec prec, int B);

// Algorithm 2 in FP32 storage with the tcgen05 contraction: PAWFE_TF32 (one TF32 pass; real and complex contexts) or
// PAWFE_FP32 (real contexts: three passes on hi/lo operand splits, FP32-accurate).  Coefficients come from
// filter_scalars (api_filter.cu).  X: [dof][vec] float (real) or float2 (complex), ld >= B in those scalars; complex
// blocks need B and ld even and a 16-byte aligned X.  workspace as pawfe_filter_workspace.  HX, SX: null, or the
// caller's FP64 products H X and S X (layout of X, FP64 scalars): step 2 then applies no operator.
pawfe_status fused_filter(pawfe_ctx* c, pawfe_prec prec, int m, const double* ds /*device scalars*/, const double* as,
                          const double* acs, const double* zzs, double z_over_e, void* X, long ld, int B,
                          void* workspace, const void* HX = nullptr, const void* SX = nullptr);

// Y = H X (tcgen05 contraction, non-local term through the K-extension).  X, Y as float blocks (complex: interleaved,
// ldx / ldy in floats), 16-byte aligned, ldx % 4 == ldy % 4 == 0; B vectors.
pawfe_status fused_apply_H(pawfe_ctx* c, pawfe_prec prec, const float* X, long ldx, float* Y, long ldy, int B);
// Y = H S^-1approx X in the kernel configuration of the filter's step (same argument rules).
pawfe_status fused_apply_HSinv(pawfe_ctx* c, pawfe_prec prec, const float* X, long ldx, float* Y, long ldy, int B);
