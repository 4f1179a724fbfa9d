// apply_impl.h -- templated operator applications defined (and explicitly instantiated) in api_apply.cu.
//   TX: storage scalar of the input block, TY: of the output block, TC: compute / operator scalar.
#pragma once
#include "common.h"

template <typename TX, typename TY, typename TC>
pawfe_status pawfe_apply_HS(pawfe_ctx* c, int op /*0 = H, 1 = S*/, bool tf32, const TX* X, long ldx, TY* Y,
                            long ldy, int B);
// Y -= (S X) Lambda in FP64 without storing S X (api_apply.cu).
template <typename TX, typename TD>
pawfe_status pawfe_sub_SX_lambda(pawfe_ctx* c, const TX* X, long ldx, TD* Y, long ldy, int B, const double* lam,
                                 const double* neg_lam);
template <typename TX, typename TY, typename TC>
pawfe_status pawfe_apply_Sinv_impl(pawfe_ctx* c, const TX* X, long ldx, TY* Y, long ldy, int B);

// H apply in the storage type selected by prec (float / double, complex if the context is); picks the
// tcgen05 kernel for the TF32 mode when it supports the shape.
pawfe_status pawfe_apply_H_any(pawfe_ctx* c, pawfe_prec prec, const void* X, long ldx, void* Y, long ldy, int B);

// Y += sum_e P_e^T H^e (P_e X) in FP64 on the DMMA pipe, real contexts (no zeroing of Y, no non-local term).
template <typename RX>
pawfe_status pawfe_cell_product_fp64(pawfe_ctx* c, const RX* X, long ldx, double* Y, long ldy, int B);
