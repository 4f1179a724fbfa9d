// cell_tcgen05.h -- TF32 cell contraction Y_e = H^e T_e on tcgen05 tensor cores (PAPER.md:L347 step iii;
// TF32: L11, L27).  Host-side entry points used by the API translation units.
#pragma once
#include "common.h"

// Split of the n output nodes of a cell into NH halves of NT columns (NT a multiple of 16) used by the kernel.
void tc_shape(const pawfe_ctx* ctx, int* NH, int* NT);

// Drop any cached tensor maps / plans (called when the cell matrices are rebuilt or freed).
void tc_invalidate(pawfe_ctx* ctx);

// True if the tensor-core kernel handles this context's (p, scalar type) and block width B.
bool tc_supported(const pawfe_ctx* ctx, int B);

// True if, in addition, these blocks meet the kernel's alignment rules (16-byte aligned pointers, leading
// dimensions and B multiples of 4) and the tensor map could be built.
bool tc_usable(pawfe_ctx* ctx, const void* X, long ldx, const void* Y, long ldy, int B);

// Optional K-extension of the contraction (fused.h): cell e gets, after its own n input rows, one 32-row chunk
// per listed (cell, atom) entry x in [ext_start[e], ext_start[e+1]): input rows Wcat[ext_atom[x]][0..32)[vec],
// matrix block Bext[x][I][0..32) (I = output node).  This adds the low-rank projector terms to the product
// inside the same MMA accumulation.  ksteps = ceil(used rows / 8).
struct TcExt {
  int scale_mode;              // 0: Y += alpha * acc;  1: Y += alpha * M_D^-1[J] * acc
  long nchunks;
  const int* ext_start; const int* ext_atom;
  const float* Bext;           // [chunk][half][NT][32] floats, rows 128-byte swizzled (api_fused.cu k_build_ext)
  const float* Wcat; long ldw;
  int ksteps;
  const float* Hstream;        // null: the context's re-tiled cell matrices; else an array of the same layout (tc_hstream_lo)
};

// dst[i] = src[i] - trunc_tf32(src[i]): the part of an FP32 value the tensor core drops (3xTF32 split, FP32 mode).
pawfe_status tc_lo_part(pawfe_ctx* ctx, const float* src, float* dst, long count);
// The low parts of the re-tiled cell-matrix stream (built on first use; same layout as the stream itself).
pawfe_status tc_hstream_lo(pawfe_ctx* ctx, const float** out);

// Y += alpha * [M_D^-1] sum_e P_e^T (H^e (P_e X) + extension terms) for a real FP32 block, TF32 multiply, FP32
// accumulate.  X, Y: device [dof][vec] float, leading dimensions ldx, ldy.  Y must already hold the values to
// add to (assembly is by atomic adds).  ext may be null.
pawfe_status tc_cell_apply(pawfe_ctx* ctx, const float* X, long ldx, float* Y, long ldy, int B, float alpha,
                           const TcExt* ext = nullptr);
