// api_apply.cu -- operator applications A X, A in {H, S, S^-1approx} (section 4.3; Eq. 28)
// as sequences of kernel launches on the context's stream.  No allocation, no host synchronisation
// (except growing the projection scratch the first time a wider block is seen).
#include "common.h"
#include "host_util.h"
#include "kernels_simt.cuh"
#include "kernels_stream.cuh"
#include "cell_dmma.cuh"
#include "nonlocal_f32.cuh"
#include "setup_fp64.cuh"
#include "api_internal.h"
#include "apply_impl.h"
#include "fused.h"
#include <algorithm>
#include <type_traits>

namespace {

template <typename TC> struct OpData;
template <> struct OpData<double> {
  static const double* H(const pawfe_ctx* c) { return (const double*)c->d_H64; }
  static const double* Mref(const pawfe_ctx* c) { return c->d_Mref64; }
  static int lda(const pawfe_ctx* c) { return c->n; }
  static const double* Cd(const pawfe_ctx* c) { return (const double*)c->d_Cd64; }
  static const double* D(const pawfe_ctx* c) { return (const double*)c->d_D64; }
  static const double* dS(const pawfe_ctx* c) { return (const double*)c->d_dS64; }
  static const double* dSinv(const pawfe_ctx* c) { return (const double*)c->d_dSinv64; }
};
template <> struct OpData<double2> {
  static const double2* H(const pawfe_ctx* c) { return (const double2*)c->d_H64; }
  static const double2* Mref(const pawfe_ctx* c) { return (const double2*)c->d_Mref64; }
  static int lda(const pawfe_ctx* c) { return c->n; }
  static const double2* Cd(const pawfe_ctx* c) { return (const double2*)c->d_Cd64; }
  static const double2* D(const pawfe_ctx* c) { return (const double2*)c->d_D64; }
  static const double2* dS(const pawfe_ctx* c) { return (const double2*)c->d_dS64; }
  static const double2* dSinv(const pawfe_ctx* c) { return (const double2*)c->d_dSinv64; }
};
template <> struct OpData<float> {
  static const float* H(const pawfe_ctx* c) { return (const float*)c->d_H32; }
  static const float* Mref(const pawfe_ctx* c) { return c->d_Mref32; }
  static int lda(const pawfe_ctx* c) { return c->ldk; }
  static const float* Cd(const pawfe_ctx* c) { return (const float*)c->d_Cd32; }
  static const float* D(const pawfe_ctx* c) { return (const float*)c->d_D32; }
  static const float* dS(const pawfe_ctx* c) { return (const float*)c->d_dS32; }
  static const float* dSinv(const pawfe_ctx* c) { return (const float*)c->d_dSinv32; }
};
template <> struct OpData<float2> {
  static const float2* H(const pawfe_ctx* c) { return (const float2*)c->d_H32; }
  static const float2* Mref(const pawfe_ctx* c) { return (const float2*)c->d_Mref32; }
  static int lda(const pawfe_ctx* c) { return c->ldk; }
  static const float2* Cd(const pawfe_ctx* c) { return (const float2*)c->d_Cd32; }
  static const float2* D(const pawfe_ctx* c) { return (const float2*)c->d_D32; }
  static const float2* dS(const pawfe_ctx* c) { return (const float2*)c->d_dS32; }
  static const float2* dSinv(const pawfe_ctx* c) { return (const float2*)c->d_dSinv32; }
};

template <typename TY>
pawfe_status zero_block(pawfe_ctx* c, TY* Y, long ldy, int B) {
  if (ldy == B) CUDA_TRY(c, cudaMemsetAsync(Y, 0, (size_t)c->M * B * sizeof(TY), c->stream));
  else CUDA_TRY(c, cudaMemset2DAsync(Y, ldy * sizeof(TY), 0, (size_t)B * sizeof(TY), c->M, c->stream));
  return PAWFE_OK;
}

// FP64 cell product on the DMMA pipe (cell_dmma.cuh).  RX: real type of the input block.
template <typename RX, bool CPLX, int MT>
pawfe_status launch_dmma_mt(pawfe_ctx* c, const double* A, long cell_stride, const RX* X, long ldx, double* Y, long ldy,
                            int Wr, double alpha) {
  auto kern = dmma::k_cell_dmma<RX, CPLX, MT>;
  const size_t smem = dmma::smem_bytes<RX, CPLX, MT>(c->n);
  TRY(pawfe_ensure_smem(c, (const void*)kern, smem));
  kern<<<(unsigned)ceil_div(Wr, dmma::kTN) * (unsigned)c->ncell, dmma::kThreads, smem, c->stream>>>(c->md, A, cell_stride, X, ldx, Y, ldy, Wr, alpha);
  KERNEL_CHECK(c, "k_cell_dmma");
  return PAWFE_OK;
}
template <typename RX, bool CPLX>
pawfe_status launch_dmma(pawfe_ctx* c, const double* A, long cell_stride, const RX* X, long ldx, double* Y, long ldy,
                         int Wr, double alpha) {
  const int n = c->n;
  if (n <= 32) return launch_dmma_mt<RX, CPLX, 1>(c, A, cell_stride, X, ldx, Y, ldy, Wr, alpha);
  if (n <= 64) return launch_dmma_mt<RX, CPLX, 2>(c, A, cell_stride, X, ldx, Y, ldy, Wr, alpha);
  if (n <= 128) return launch_dmma_mt<RX, CPLX, 4>(c, A, cell_stride, X, ldx, Y, ldy, Wr, alpha);
  if (n <= 224) return launch_dmma_mt<RX, CPLX, 7>(c, A, cell_stride, X, ldx, Y, ldy, Wr, alpha);
  if (n <= 352) {
    // n = 343 (p = 6): MT = 11 is one row block at one CTA per SM (two row blocks at two CTAs per SM, MT = 5 / 6, were not
    // faster: DESIGN.md section 7)
    return launch_dmma_mt<RX, CPLX, 11>(c, A, cell_stride, X, ldx, Y, ldy, Wr, alpha);
  }
  return launch_dmma_mt<RX, CPLX, 8>(c, A, cell_stride, X, ldx, Y, ldy, Wr, alpha);
}

template <typename TX, typename TY, typename TC, bool TF32>
pawfe_status launch_cell(pawfe_ctx* c, const TC* A, long cell_stride, int lda, const TX* X, long ldx, TY* Y,
                         long ldy, int B, int in_scale, double alpha) {
  if constexpr (sizeof(typename ScalarTraits<TC>::real) == 8) {
    // FP64 compute: DMMA kernel (lda == n, no input scaling on this path)
    constexpr bool CP = ScalarTraits<TC>::cplx;
    constexpr int cw = CP ? 2 : 1;
    typedef typename ScalarTraits<TX>::real RX;
    return launch_dmma<RX, CP>(c, (const double*)A, cell_stride, (const RX*)X, ldx * cw, (double*)Y, ldy * cw, B * cw, alpha);
  } else {
  constexpr int BV = (sizeof(TC) == 16) ? 16 : 32;
  size_t smem = (size_t)c->n * 16 + (size_t)c->n * BV * sizeof(TC);
  auto kern = k_cell_simt<TX, TY, TC, BV, TF32>;
  TRY(pawfe_ensure_smem(c, (const void*)kern, smem));
  kern<<<dim3(c->ncell, ceil_div(B, BV)), 256, smem, c->stream>>>(c->md, A, cell_stride, lda, X, ldx, Y, ldy, B,
                                                                  in_scale, alpha);
  KERNEL_CHECK(c, "k_cell_simt");
  return PAWFE_OK;
  }
}

// Fast FP32-storage non-local path (nonlocal_f32.cuh): real or complex interleaved blocks as Wr = B * cw real columns.
template <int NPJ, bool CPLX>
pawfe_status nonlocal_f32_t(pawfe_ctx* c, const float* Delta, double scale, const float* X, long ldx, int in_scale,
                            float* Y, long ldy, int out_scale, int B) {
  constexpr int cw = CPLX ? 2 : 1;
  typedef typename std::conditional<CPLX, float2, float>::type TC;
  const int n = c->n, Wr = B * cw;
  float* P = (float*)c->d_P;
  float* W = P + (size_t)c->natoms * NPJ * Wr;
  CUDA_TRY(c, cudaMemsetAsync(P, 0, (size_t)c->natoms * NPJ * Wr * sizeof(float), c->stream));
  dim3 grid((unsigned)c->npairs, ceil_div(Wr, 128));
  const size_t head = (size_t)(n + 1) / 2 * 16 + (size_t)(n + 3) / 4 * 16;
  {
    const size_t smem = head + ((size_t)NPJ * n * cw + 3) / 4 * 16 + (size_t)NPJ * 128 * 4;
    TRY(pawfe_ensure_smem(c, (const void*)k_projF<NPJ, CPLX>, smem));
    k_projF<NPJ, CPLX><<<grid, 256, smem, c->stream>>>(c->md, c->d_pair_cell, c->d_pair_atom, (const float*)c->d_Cd32, X, ldx * cw, Wr,
                                                      in_scale, P, (long)Wr);
    KERNEL_CHECK(c, "k_projF");
  }
  k_coupling<TC><<<dim3(c->natoms, ceil_div(B, 128)), 128, 0, c->stream>>>((const TC*)Delta, NPJ, (const TC*)P, B, B, scale, (TC*)W);
  KERNEL_CHECK(c, "k_coupling");
  {
    const size_t smem = head + ((size_t)NPJ * n * cw + 3) / 4 * 16;
    TRY(pawfe_ensure_smem(c, (const void*)k_scatterF<NPJ, CPLX>, smem));
    k_scatterF<NPJ, CPLX><<<grid, 256, smem, c->stream>>>(c->md, c->d_pair_cell, c->d_pair_atom, (const float*)c->d_Cd32, W, (long)Wr, NPJ, Wr,
                                                         out_scale, 1.0f, Y, ldy * cw);
    KERNEL_CHECK(c, "k_scatterF");
  }
  return PAWFE_OK;
}
template <bool CPLX>
pawfe_status nonlocal_f32(pawfe_ctx* c, const float* Delta, double scale, const float* X, long ldx, int in_scale, float* Y,
                          long ldy, int out_scale, int B) {
  switch (c->npj) {
#define CASE_NL(N) case N: return nonlocal_f32_t<N, CPLX>(c, Delta, scale, X, ldx, in_scale, Y, ldy, out_scale, B);
    CASE_NL(1) CASE_NL(2) CASE_NL(3) CASE_NL(4) CASE_NL(5) CASE_NL(6) CASE_NL(7) CASE_NL(8)
    CASE_NL(9) CASE_NL(10) CASE_NL(11) CASE_NL(12) CASE_NL(13) CASE_NL(14) CASE_NL(15) CASE_NL(16)
#undef CASE_NL
  }
  return PAWFE_EINVAL;
}

}  // namespace

// Y (+)= nonlocal part:  Y += out_scale o C (scale * Delta (C^dagger (in_scale o X)))
template <typename TX, typename TY, typename TC>
pawfe_status pawfe_apply_nonlocal(pawfe_ctx* c, const TC* Delta, double scale, const TX* X, long ldx, int in_scale,
                                  TY* Y, long ldy, int out_scale, int B, const double* colscale) {
  if (c->npairs == 0) return PAWFE_OK;
  TRY(pawfe_ensure_P(c, B));
  if constexpr (std::is_same<TX, TC>::value && std::is_same<TY, TC>::value &&
                (std::is_same<TC, float>::value || std::is_same<TC, float2>::value)) {
    constexpr int cw = ScalarTraits<TC>::cplx ? 2 : 1;
    // 16-byte pieces: rows and the block width must be multiples of 4 floats
    if (!colscale && ((ldx * cw) & 3) == 0 && ((ldy * cw) & 3) == 0 && ((B * cw) & 3) == 0 && ((uintptr_t)X & 15) == 0 && ((uintptr_t)Y & 15) == 0)
      return nonlocal_f32<ScalarTraits<TC>::cplx>(c, (const float*)Delta, scale, (const float*)X, ldx, in_scale, (float*)Y, ldy, out_scale, B);
  }
  TC* P = (TC*)c->d_P;
  TC* W = P + (size_t)c->natoms * c->npj * B;
  size_t smem = (size_t)c->n * 16 + 4 * PAWFE_MAX_NPJ * 32 * sizeof(TC);
  k_proj<TX, TC><<<dim3(c->natoms, ceil_div(B, 32)), 128, smem, c->stream>>>(
      c->md, 0, c->d_atom_pair_start, c->d_pair_cell, OpData<TC>::Cd(c), c->npj, X, ldx, B, in_scale, P, B);
  KERNEL_CHECK(c, "k_proj");
  k_coupling<TC><<<dim3(c->natoms, ceil_div(B, 128)), 128, 0, c->stream>>>(Delta, c->npj, P, B, B, scale, W, colscale);
  KERNEL_CHECK(c, "k_coupling");
  k_nl_scatter<TY, TC><<<dim3((unsigned)c->npairs, ceil_div(B, 32)), 128, 0, c->stream>>>(
      c->md, 0, c->d_pair_cell, c->d_pair_atom, OpData<TC>::Cd(c), c->npj, W, B, B, out_scale, Y, ldy);
  KERNEL_CHECK(c, "k_nl_scatter");
  return PAWFE_OK;
}

// Y = H X (op 0) or S X (op 1)
template <typename TX, typename TY, typename TC>
pawfe_status pawfe_apply_HS(pawfe_ctx* c, int op, bool tf32, const TX* X, long ldx, TY* Y, long ldy, int B) {
  TRY(zero_block(c, Y, ldy, B));
  const TC* A = op == 0 ? OpData<TC>::H(c) : OpData<TC>::Mref(c);
  long stride = op == 0 ? (long)c->n * OpData<TC>::lda(c) : 0;
  const bool timed = (op == 0) && sizeof(typename ScalarTraits<TC>::real) == sizeof(typename ScalarTraits<TX>::real);  // the loop's contraction
  if (timed) prof_begin(c);
  pawfe_status st;
  if (tf32 && op == 0) st = launch_cell<TX, TY, TC, true>(c, A, stride, OpData<TC>::lda(c), X, ldx, Y, ldy, B, 0, 1.0);
  else st = launch_cell<TX, TY, TC, false>(c, A, stride, OpData<TC>::lda(c), X, ldx, Y, ldy, B, 0, 1.0);
  if (timed) prof_end(c);
  TRY(st);
  const TC* Delta = op == 0 ? OpData<TC>::D(c) : OpData<TC>::dS(c);
  return pawfe_apply_nonlocal<TX, TY, TC>(c, Delta, 1.0, X, ldx, 0, Y, ldy, 0, B, nullptr);
}

// Y = S^-1approx X = M_D^-1 X - M_D^-1 C Delta_Sinv C^dagger M_D^-1 X   (Eq. 28)
template <typename TX, typename TY, typename TC>
pawfe_status pawfe_apply_Sinv_impl(pawfe_ctx* c, const TX* X, long ldx, TY* Y, long ldy, int B) {
  typedef typename ScalarTraits<TX>::real RX;
  typedef typename ScalarTraits<TY>::real RY;
  const int cw = ScalarTraits<TX>::cplx ? 2 : 1;
  if constexpr (std::is_same<RX, float>::value && std::is_same<RY, float>::value) {
    if (((ldx * cw) & 3) == 0 && ((ldy * cw) & 3) == 0 && ((B * cw) & 3) == 0 && ((uintptr_t)X & 15) == 0 && ((uintptr_t)Y & 15) == 0) {
      k_scale_mdinv_f4<<<8 * c->sm_count, 256, 0, c->stream>>>(c->md, (const float4*)X, ldx * cw / 4, (float4*)Y, ldy * cw / 4, B * cw / 4);
      KERNEL_CHECK(c, "k_scale_mdinv_f4");
      return pawfe_apply_nonlocal<TX, TY, TC>(c, OpData<TC>::dSinv(c), -1.0, X, ldx, 1, Y, ldy, 1, B, nullptr);
    }
  }
  k_scale_mdinv<RX, RY><<<4 * c->sm_count, 256, 0, c->stream>>>(c->md, (const RX*)X, ldx * cw, (RY*)Y, ldy * cw, B * cw);
  KERNEL_CHECK(c, "k_scale_mdinv");
  return pawfe_apply_nonlocal<TX, TY, TC>(c, OpData<TC>::dSinv(c), -1.0, X, ldx, 1, Y, ldy, 1, B, nullptr);
}

template <typename RX>
pawfe_status pawfe_cell_product_fp64(pawfe_ctx* c, const RX* X, long ldx, double* Y, long ldy, int B) {
  return launch_dmma<RX, false>(c, (const double*)c->d_H64, (long)c->n * c->n, X, ldx, Y, ldy, B, 1.0);
}
template pawfe_status pawfe_cell_product_fp64<float>(pawfe_ctx*, const float*, long, double*, long, int);
template pawfe_status pawfe_cell_product_fp64<double>(pawfe_ctx*, const double*, long, double*, long, int);

// Y -= (S X) Lambda, S = M + C dS C^dagger (Eq. 16), FP64, without storing S X: the mass part by three 1-D sweeps of
// M^e = (hx hy hz / 8) M1 (x) M1 (x) M1 (setup_fp64.cuh: k_mass_sf), the non-local part with the Ritz value folded into
// the coupling.  neg_lam / lam: device, [B] doubles (-Lambda and Lambda).  Y: FP64 block with leading dimension ldy.
template <typename TX, typename TD>
pawfe_status pawfe_sub_SX_lambda(pawfe_ctx* c, const TX* X, long ldx, TD* Y, long ldy, int B, const double* lam,
                                 const double* neg_lam) {
  typedef typename ScalarTraits<TX>::real RX;
  constexpr int cw = ScalarTraits<TX>::cplx ? 2 : 1;
  const size_t smem = (size_t)c->n * kMassCT * 8 + (size_t)c->n * 8;
  TRY(pawfe_ensure_smem(c, (const void*)k_mass_sf<RX, kMassCT>, smem));
  k_mass_sf<RX, kMassCT><<<dim3(c->ncell, ceil_div(B * cw, kMassCT)), 256, smem, c->stream>>>(
      c->md, c->d_M1, c->h[0] * c->h[1] * c->h[2] / 8.0, (const RX*)X, ldx * cw, (double*)Y, ldy * cw, B * cw, neg_lam, cw);
  KERNEL_CHECK(c, "k_mass_sf");
  return pawfe_apply_nonlocal<TX, TD, TD>(c, OpData<TD>::dS(c), -1.0, X, ldx, 0, Y, ldy, 0, B, lam);
}
template pawfe_status pawfe_sub_SX_lambda<float, double>(pawfe_ctx*, const float*, long, double*, long, int, const double*, const double*);
template pawfe_status pawfe_sub_SX_lambda<double, double>(pawfe_ctx*, const double*, long, double*, long, int, const double*, const double*);
template pawfe_status pawfe_sub_SX_lambda<float2, double2>(pawfe_ctx*, const float2*, long, double2*, long, int, const double*, const double*);
template pawfe_status pawfe_sub_SX_lambda<double2, double2>(pawfe_ctx*, const double2*, long, double2*, long, int, const double*, const double*);

// explicit instantiations used by the other translation units
#define INST(TX, TY, TC)                                                                                          \
  template pawfe_status pawfe_apply_HS<TX, TY, TC>(pawfe_ctx*, int, bool, const TX*, long, TY*, long, int);       \
  template pawfe_status pawfe_apply_Sinv_impl<TX, TY, TC>(pawfe_ctx*, const TX*, long, TY*, long, int);
INST(double, double, double)
INST(float, double, double)
INST(float, float, float)
INST(double2, double2, double2)
INST(float2, double2, double2)
INST(float2, float2, float2)
#undef INST

// ================================================================================================
// C ABI
// ================================================================================================
static pawfe_status check_apply(pawfe_ctx* c, pawfe_prec prec, const void* X, void* Y, long ld, int B, bool need_pot) {
  if (!c || !X || !Y || B < 1 || B > 512 || ld < B) { if (c) c->err = "bad block arguments"; return PAWFE_EINVAL; }
  if (prec != PAWFE_FP64 && prec != PAWFE_FP32 && prec != PAWFE_TF32) return PAWFE_EINVAL;
  if (!c->have_mesh || !c->have_atoms || (need_pot && !c->have_pot)) { c->err = "operators not set up"; return PAWFE_ESTATE; }
  if (need_pot && prec == PAWFE_FP64 && !c->have_h64) { c->err = "FP64 cell matrices were not kept (keep_fp64 = 0)"; return PAWFE_ESTATE; }
  cudaError_t e = cudaSetDevice(c->device);
  if (e != cudaSuccess) { c->err = cudaGetErrorString(e); return PAWFE_ECUDA; }
  return PAWFE_OK;
}

extern "C" pawfe_status pawfe_apply_H(pawfe_ctx* c, pawfe_prec prec, const void* X, void* Y, long ld, int B) {
  TRY(check_apply(c, prec, X, Y, ld, B, true));
  return pawfe_apply_H_any(c, prec, X, ld, Y, ld, B);
}
extern "C" pawfe_status pawfe_apply_S(pawfe_ctx* c, pawfe_prec prec, const void* X, void* Y, long ld, int B) {
  TRY(check_apply(c, prec, X, Y, ld, B, false));
  bool f64 = prec == PAWFE_FP64;
  if (c->cplx) return f64 ? pawfe_apply_HS<double2, double2, double2>(c, 1, false, (const double2*)X, ld, (double2*)Y, ld, B)
                          : pawfe_apply_HS<float2, float2, float2>(c, 1, false, (const float2*)X, ld, (float2*)Y, ld, B);
  return f64 ? pawfe_apply_HS<double, double, double>(c, 1, false, (const double*)X, ld, (double*)Y, ld, B)
             : pawfe_apply_HS<float, float, float>(c, 1, false, (const float*)X, ld, (float*)Y, ld, B);
}
extern "C" pawfe_status pawfe_apply_Sinv(pawfe_ctx* c, pawfe_prec prec, const void* X, void* Y, long ld, int B) {
  TRY(check_apply(c, prec, X, Y, ld, B, false));
  bool f64 = prec == PAWFE_FP64;
  if (c->cplx) return f64 ? pawfe_apply_Sinv_impl<double2, double2, double2>(c, (const double2*)X, ld, (double2*)Y, ld, B)
                          : pawfe_apply_Sinv_impl<float2, float2, float2>(c, (const float2*)X, ld, (float2*)Y, ld, B);
  return f64 ? pawfe_apply_Sinv_impl<double, double, double>(c, (const double*)X, ld, (double*)Y, ld, B)
             : pawfe_apply_Sinv_impl<float, float, float>(c, (const float*)X, ld, (float*)Y, ld, B);
}

// H apply in the storage type of `prec`; the TF32 mode of a real context runs the tcgen05 kernel when it
// supports the shape, otherwise the SIMT kernel with TF32-rounded operands.
pawfe_status pawfe_apply_H_any(pawfe_ctx* c, pawfe_prec prec, const void* X, long ldx, void* Y, long ldy, int B) {
  if (prec == PAWFE_FP64) {
    if (c->cplx) return pawfe_apply_HS<double2, double2, double2>(c, 0, false, (const double2*)X, ldx, (double2*)Y, ldy, B);
    return pawfe_apply_HS<double, double, double>(c, 0, false, (const double*)X, ldx, (double*)Y, ldy, B);
  }
  bool tf32 = prec == PAWFE_TF32;
  if (c->cplx) {
    if (tc_usable(c, X, 2 * ldx, Y, 2 * ldy, 2 * B) && fused_supported(c, prec, B))
      return fused_apply_H(c, prec, (const float*)X, 2 * ldx, (float*)Y, 2 * ldy, B);
    if (tf32 && tc_usable(c, X, 2 * ldx, Y, 2 * ldy, 2 * B)) {
      // complex TF32: interleaved (re, im) columns as a real block of 2B columns; P / Q accumulators in the kernel;
      // every row is stored by its first writer (no zero fill)
      TcEpi st_epi; st_epi.mode = TC_EPI_STORE; st_epi.Yt = nullptr; st_epi.aLam = nullptr; st_epi.ac = st_epi.zz1 = 0.f; st_epi.cw = 2;
      prof_begin(c);
      pawfe_status st = tc_cell_apply(c, (const float*)X, 2 * ldx, (float*)Y, 2 * ldy, 2 * B, 1.0f, nullptr, &st_epi);
      prof_end(c);
      TRY(st);
      return pawfe_apply_nonlocal<float2, float2, float2>(c, OpData<float2>::D(c), 1.0, (const float2*)X, ldx, 0, (float2*)Y, ldy, 0, B, nullptr);
    }
    return pawfe_apply_HS<float2, float2, float2>(c, 0, tf32, (const float2*)X, ldx, (float2*)Y, ldy, B);
  }
  if (tc_usable(c, X, ldx, Y, ldy, B) && fused_supported(c, prec, B))
    return fused_apply_H(c, prec, (const float*)X, ldx, (float*)Y, ldy, B);
  if (tf32 && tc_usable(c, X, ldx, Y, ldy, B)) {
    TcEpi st_epi; st_epi.mode = TC_EPI_STORE; st_epi.Yt = nullptr; st_epi.aLam = nullptr; st_epi.ac = st_epi.zz1 = 0.f; st_epi.cw = 1;
    prof_begin(c);
    pawfe_status st = tc_cell_apply(c, (const float*)X, ldx, (float*)Y, ldy, B, 1.0f, nullptr, &st_epi);
    prof_end(c);
    TRY(st);
    return pawfe_apply_nonlocal<float, float, float>(c, OpData<float>::D(c), 1.0, (const float*)X, ldx, 0, (float*)Y, ldy, 0, B, nullptr);
  }
  return pawfe_apply_HS<float, float, float>(c, 0, tf32, (const float*)X, ldx, (float*)Y, ldy, B);
}

// Y = H S^-1approx X.  FP32 / TF32 blocks that meet the tensor-core kernel's alignment rules run the fused step's kernel
// configuration (fused_apply_HSinv); everything else S^-1approx then H through a context-owned block T.
extern "C" pawfe_status pawfe_apply_HSinv(pawfe_ctx* c, pawfe_prec prec, const void* X, void* Y, long ld, int B) {
  TRY(check_apply(c, prec, X, Y, ld, B, true));
  const int cw = c->cplx ? 2 : 1;
  if (prec != PAWFE_FP64 && tc_usable(c, X, cw * ld, Y, cw * ld, cw * B) && fused_supported(c, prec, B))
    return fused_apply_HSinv(c, prec, (const float*)X, cw * ld, (float*)Y, cw * ld, B);
  const size_t es = (prec == PAWFE_FP64 ? 8 : 4) * (size_t)cw;
  const size_t need = (size_t)c->M * B * es;
  if (need > c->tmpblk_bytes) {   // first use / wider block (pawfe_prepare sizes it ahead)
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    cudaFree(c->d_tmpblk); c->d_tmpblk = nullptr; c->tmpblk_bytes = 0;
    char* q = nullptr; TRY(dev_alloc(c, &q, need)); c->d_tmpblk = q; c->tmpblk_bytes = need;
  }
  void* T = c->d_tmpblk;
  if (c->cplx) {
    if (prec == PAWFE_FP64) TRY((pawfe_apply_Sinv_impl<double2, double2, double2>(c, (const double2*)X, ld, (double2*)T, B, B)));
    else TRY((pawfe_apply_Sinv_impl<float2, float2, float2>(c, (const float2*)X, ld, (float2*)T, B, B)));
  } else {
    if (prec == PAWFE_FP64) TRY((pawfe_apply_Sinv_impl<double, double, double>(c, (const double*)X, ld, (double*)T, B, B)));
    else TRY((pawfe_apply_Sinv_impl<float, float, float>(c, (const float*)X, ld, (float*)T, B, B)));
  }
  return pawfe_apply_H_any(c, prec, T, B, Y, ld, B);
}

extern "C" const char* pawfe_cell_kernel_name(const pawfe_ctx* c, pawfe_prec prec, int B) {
  if (!c) return "none";
  if (prec == PAWFE_FP64) return "dmma_fp64";
  if (prec == PAWFE_FP32) return tc_supported(c, B) ? "tcgen05_3xtf32" : "simt_fp32";
  if (tc_supported(c, B)) return "tcgen05_tf32";
  return "simt_tf32_emulated";
}

extern "C" pawfe_status pawfe_col_norms(pawfe_ctx* c, pawfe_prec prec, const void* X, long ld, int B, double* out) {
  if (!c || !X || !out || B < 1 || ld < B) return PAWFE_EINVAL;
  if (!c->have_mesh) return PAWFE_ESTATE;
  CUDA_TRY(c, cudaSetDevice(c->device));
  CUDA_TRY(c, cudaMemsetAsync(out, 0, B * sizeof(double), c->stream));
  const int cw = c->cplx ? 2 : 1;
  dim3 grid(ceil_div(B, 32), std::min<long>(4 * c->sm_count, (c->M + 7) / 8)), block(32, 8);
  if (prec == PAWFE_FP64) k_col_sumsq<double><<<grid, block, 0, c->stream>>>(c->M, B, cw, (const double*)X, ld, out);
  else k_col_sumsq<float><<<grid, block, 0, c->stream>>>(c->M, B, cw, (const float*)X, ld, out);
  KERNEL_CHECK(c, "k_col_sumsq");
  k_sqrt_inplace<<<ceil_div(B, 128), 128, 0, c->stream>>>(out, B);
  KERNEL_CHECK(c, "k_sqrt_inplace");
  return PAWFE_OK;
}

extern "C" pawfe_status pawfe_cell_timing(pawfe_ctx* c, int enable) {
  if (!c) return PAWFE_EINVAL;
  c->prof_on = enable != 0;
  c->prof_used = 0;
  c->prof_setup_used = 0;
  return PAWFE_OK;
}

extern "C" pawfe_status pawfe_cell_timing_read(pawfe_ctx* c, long* launches, double* ms) {
  if (!c || !launches || !ms) return PAWFE_EINVAL;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  double tot = 0.0;
  for (size_t i = 0; i + 1 < c->prof_used; i += 2) {
    float t = 0.f;
    CUDA_TRY(c, cudaEventElapsedTime(&t, c->prof_ev[i], c->prof_ev[i + 1]));
    tot += t;
  }
  *launches = (long)(c->prof_used / 2);
  *ms = tot;
  return PAWFE_OK;
}

extern "C" pawfe_status pawfe_setup_timing_read(pawfe_ctx* c, long* calls, double* ms) {
  if (!c || !calls || !ms) return PAWFE_EINVAL;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  double tot = 0.0;
  for (size_t i = 0; i + 1 < c->prof_setup_used; i += 2) {
    float t = 0.f;
    CUDA_TRY(c, cudaEventElapsedTime(&t, c->prof_setup_ev[i], c->prof_setup_ev[i + 1]));
    tot += t;
  }
  *calls = (long)(c->prof_setup_used / 2);
  *ms = tot;
  return PAWFE_OK;
}
