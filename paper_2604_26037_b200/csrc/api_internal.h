// api_internal.h -- functions shared between the API translation units (not exported).
#pragma once
#include "common.h"

// Make sure the projection scratch (2 x [natoms][npj][B] scalars of the widest type) exists.
pawfe_status pawfe_ensure_P(pawfe_ctx* ctx, int B);

// Recompute FP32 copies / Delta_Sinv after the couplings changed (host h_dS, device G needed).
pawfe_status pawfe_upload_couplings(pawfe_ctx* ctx, const double* D, const double* dS,
                                    const std::vector<double>& G /* natoms*npj*npj*cw */);
