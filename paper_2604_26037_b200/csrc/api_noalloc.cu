// api_noalloc.cu -- pawfe_apply_Sinv_noalloc: Y = S^-1approx X (Eq. 28) for callers that cannot allocate
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// The ordinary pawfe_apply_Sinv keeps its projections P^a = C^a^dagger M_D^-1 X and couplings W^a = -Delta^a_Sinv P^a in a
// scratch block that pawfe_ensure_P grows with cudaMalloc.  This variant runs the same four steps (diagonal scaling,
// atom-local projection, coupling, low-rank scatter: kernels_simt.cuh / kernels_stream.cuh) with P and W in a FILE-SCOPE
// static device array of PAWFE_NOALLOC_SCRATCH_BYTES, which every GPU that loads libpawfe.so holds until the process exits.
// It calls no cudaMalloc / cudaFree and no allocating library routine; blocks that need more scratch are rejected.
//
// In host code the array's name is only a host-side stand-in for the symbol: its DEVICE address is looked up once per
// device with cudaGetSymbolAddress (that device current) and cached; kernels are given that pointer.
// Every call shares the array and it keeps the last call's contents: the part a call uses is cleared first, and calls
// that overlap on the GPU (two streams, two contexts on one device) race on it.
#include "common.h"
#include "host_util.h"
#include "kernels_simt.cuh"
#include "kernels_stream.cuh"
#include <map>
#include <mutex>

#define PAWFE_NOALLOC_SCRATCH_BYTES (1u << 20)   // 1 MiB: e.g. 64 atoms x 9 projectors x 200 vectors in FP32 (0.92 MB)

static __device__ __align__(256) unsigned char g_noalloc_scratch[PAWFE_NOALLOC_SCRATCH_BYTES];

namespace {

// device address of g_noalloc_scratch on the context's device (looked up on the first call per device; no allocation)
pawfe_status scratch_address(pawfe_ctx* c, unsigned char** out) {
  static std::mutex mu;
  static std::map<int, unsigned char*> addr;
  std::lock_guard<std::mutex> lock(mu);
  auto it = addr.find(c->device);
  if (it == addr.end()) {
    unsigned char* p = nullptr;
    CUDA_TRY(c, cudaSetDevice(c->device));
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) {
      c->err = std::string("pawfe_apply_Sinv_noalloc: cudaGetSymbolAddress failed: ") + cudaGetErrorString(e);
      return PAWFE_ECUDA;
    }
    it = addr.emplace(c->device, p).first;
  }
  *out = it->second;
  return PAWFE_OK;
}

// TS: storage scalar of X and Y; TC: scalar of the operator data and of P, W
template <typename TS, typename TC>
pawfe_status sinv_noalloc(pawfe_ctx* c, const TS* X, TS* Y, long ld, int B, const TC* Cd, const TC* dSinv) {
  typedef typename ScalarTraits<TS>::real RS;
  const int cw = ScalarTraits<TS>::cplx ? 2 : 1;
  const size_t half = (size_t)c->natoms * c->npj * B * sizeof(TC);   // P, then W
  if (2 * half > PAWFE_NOALLOC_SCRATCH_BYTES) {
    c->err = "pawfe_apply_Sinv_noalloc: this block needs " + std::to_string(2 * half) + " bytes of projection scratch, the static "
             "array holds " + std::to_string((size_t)PAWFE_NOALLOC_SCRATCH_BYTES) + ": narrow the block or use pawfe_apply_Sinv";
    return PAWFE_EINVAL;
  }
  unsigned char* scratch = nullptr;
  TRY(scratch_address(c, &scratch));
  // Y = M_D^-1 X (Dirichlet wall rows become 0)
  k_scale_mdinv<RS, RS><<<4 * c->sm_count, 256, 0, c->stream>>>(c->md, (const RS*)X, ld * cw, (RS*)Y, ld * cw, B * cw);
  KERNEL_CHECK(c, "k_scale_mdinv");
  if (c->npairs == 0) return PAWFE_OK;
  // the array keeps what the previous call left: clear the part this call uses
  CUDA_TRY(c, cudaMemsetAsync(scratch, 0, 2 * half, c->stream));
  TC* P = reinterpret_cast<TC*>(scratch);
  TC* W = reinterpret_cast<TC*>(scratch + half);
  const size_t smem = (size_t)c->n * 16 + 4 * PAWFE_MAX_NPJ * 32 * sizeof(TC);   // <= 40 KB: no attribute call needed
  k_proj<TS, TC><<<dim3(c->natoms, ceil_div(B, 32)), 128, smem, c->stream>>>(
      c->md, 0, c->d_atom_pair_start, c->d_pair_cell, Cd, c->npj, X, ld, B, 1, P, B);
  KERNEL_CHECK(c, "k_proj");
  k_coupling<TC><<<dim3(c->natoms, ceil_div(B, 128)), 128, 0, c->stream>>>(dSinv, c->npj, P, B, B, -1.0, W);
  KERNEL_CHECK(c, "k_coupling");
  k_nl_scatter<TS, TC><<<dim3((unsigned)c->npairs, ceil_div(B, 32)), 128, 0, c->stream>>>(
      c->md, 0, c->d_pair_cell, c->d_pair_atom, Cd, c->npj, W, B, B, 1, Y, ld);
  KERNEL_CHECK(c, "k_nl_scatter");
  return PAWFE_OK;
}

}  // namespace

extern "C" pawfe_status pawfe_apply_Sinv_noalloc(pawfe_ctx* c, pawfe_prec prec, const void* X, void* Y, long ld, int B) {
  if (!c) return PAWFE_EINVAL;
  if (!X || !Y || B < 1 || B > 512 || ld < B) { c->err = "bad block arguments"; return PAWFE_EINVAL; }
  if (prec != PAWFE_FP64 && prec != PAWFE_FP32 && prec != PAWFE_TF32) { c->err = "bad precision mode"; return PAWFE_EINVAL; }
  if (!c->have_mesh || !c->have_atoms) { c->err = "operators not set up"; return PAWFE_ESTATE; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  const bool f64 = prec == PAWFE_FP64;
  if (c->cplx)
    return f64 ? sinv_noalloc<double2, double2>(c, (const double2*)X, (double2*)Y, ld, B, (const double2*)c->d_Cd64, (const double2*)c->d_dSinv64)
               : sinv_noalloc<float2, float2>(c, (const float2*)X, (float2*)Y, ld, B, (const float2*)c->d_Cd32, (const float2*)c->d_dSinv32);
  return f64 ? sinv_noalloc<double, double>(c, (const double*)X, (double*)Y, ld, B, (const double*)c->d_Cd64, (const double*)c->d_dSinv64)
             : sinv_noalloc<float, float>(c, (const float*)X, (float*)Y, ld, B, (const float*)c->d_Cd32, (const float*)c->d_dSinv32);
}
