// cell_tcgen05.h -- TF32 cell contraction Y_e = H^e T_e on tcgen05 tensor cores (PAPER.md:L347 step iii;
// TF32: L11, L27) with extraction (step i) in front and an ORDERED, conflict-free assembly (step iv) behind.
// Host-side entry points used by the API translation units.
#pragma once
#include "common.h"

// Split of the n output nodes of a cell into NH halves of NT columns (NT a multiple of 16) used by the kernel.
void tc_shape(const pawfe_ctx* ctx, int* NH, int* NT);

// Drop any cached plans (called when the cell matrices are rebuilt or freed).
void tc_invalidate(pawfe_ctx* ctx);

// True if the tensor-core kernel handles this context's (p, scalar type) and block width B.
bool tc_supported(const pawfe_ctx* ctx, int B);

// True if, in addition, these blocks meet the kernel's alignment rules (16-byte aligned pointers, leading
// dimensions and B multiples of 4) and the plan could be built.
bool tc_usable(pawfe_ctx* ctx, const void* X, long ldx, const void* Y, long ldy, int B);

// Build the plan now (re-tiled cell-matrix stream, cell order, dependency lists, completion flags) instead of on the
// first apply: pawfe_prepare.
pawfe_status tc_prepare(pawfe_ctx* ctx);

// Optional K-extension of the contraction (fused.h): cell e gets, after its own n input rows, one 32-row chunk
// per listed (cell, atom) entry x in [ext_start[e], ext_start[e+1]): input rows Wcat[ext_atom[x]][0..32)[vec],
// matrix block Bext[x][I][0..32) (I = output node).  This adds the low-rank projector terms to the product
// inside the same MMA accumulation.  ksteps = ceil(used rows / 8).
struct TcExt {
  int scale_mode;              // 0: acc scaled by alpha;  1: by alpha * M_D^-1[J]
  long nchunks;
  const int* ext_start; const int* ext_atom;
  const float* Bext;           // [chunk][half][NT][32] floats, rows 128-byte swizzled (api_fused.cu k_build_ext)
  const float* Wcat; long ldw;
  int ksteps;
  const float* Hstream;        // null: the context's re-tiled cell matrices; else an array of the same layout (tc_hstream_lo)
};

// What the assembly does with the scaled accumulator s = alpha [M_D^-1] acc of output node J (Fig. 2 step iv, L347).
// Every node has exactly ONE first writer per launch (the cell that comes first in the plan's cell order among the
// <= 8 cells sharing it); the other cells add their contribution after it, in cell order (see cell_tcgen05.cu).
enum TcEpiMode {
  TC_EPI_STORE = 0,     // Y[J] = sum of s                 first writer stores (0 on Dirichlet rows), the others add
  TC_EPI_ADD = 1,       // Y[J] += sum of s                everybody adds (Y holds the values to add to)
  TC_EPI_BRACKET = 2    // Alg. 2 step 4 (L272, L374):     first writer stores
                        //   Y[J] = fp32(-ac X[J] - zz1 Y[J]) + Yt[J] aLam[v] (FP64 add) + s,   the others add s
                        // (X = R_Y, Y = R_X in the scaled variables; X, Y, Yt share one leading dimension)
};
struct TcEpi {
  int mode;
  const double* Yt;      // [dof][ld] FP64 residual source (scaled), TC_EPI_BRACKET only
  const double* aLam;    // device, per vector: a * Lambda_Y
  float ac, zz1;
  int cw;                // real columns per vector (2 for complex contexts): aLam index = column / cw
};

// dst[i] = src[i] - trunc_tf32(src[i]): the part of an FP32 value the tensor core drops (3xTF32 split, FP32 mode).
pawfe_status tc_lo_part(pawfe_ctx* ctx, const float* src, float* dst, long count);
// The low parts of the re-tiled cell-matrix stream (built by tc_prepare_lo; same layout as the stream itself).
pawfe_status tc_hstream_lo(pawfe_ctx* ctx, const float** out);

// [M_D^-1-scaled] sum_e P_e^T (H^e (P_e X) + extension terms) for a real FP32 block, TF32 multiply, FP32 accumulate,
// assembled into Y as `epi` says (null: TC_EPI_ADD).  X, Y: device [dof][vec] float, leading dimensions ldx, ldy;
// complex contexts: the interleaved (re, im) block seen as a real block of 2B columns.  ext may be null.
pawfe_status tc_cell_apply(pawfe_ctx* ctx, const float* X, long ldx, float* Y, long ldy, int B, float alpha,
                           const TcExt* ext = nullptr, const TcEpi* epi = nullptr);
