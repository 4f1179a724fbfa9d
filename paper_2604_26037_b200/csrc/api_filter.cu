// api_filter.cu -- Algorithm 2 of the paper: the residual-based Chebyshev filter,
// orchestrated on the host as a stream of kernel launches.  Mixed precision as in section 4.4 (L374):
// residual set-up and the residual-source term in FP64, the bracket and H S^-1approx in the mode's precision.
#include "common.h"
#include "host_util.h"
#include "kernels_stream.cuh"
#include "api_internal.h"
#include "apply_impl.h"
#include "fused.h"
#include "setup_fp64.cuh"
#include <algorithm>
#include <cstring>
#include <type_traits>

namespace {

inline size_t align256(size_t x) { return (x + 255) / 256 * 256; }

struct WsLayout {
  size_t y64, sx_t, ht, rx, ry, total;
};

// storage bytes per scalar: ss (4/8 real, 8/16 complex); FP64 scalar bytes: sd
WsLayout ws_layout(long M, int B, size_t ss, size_t sd) {
  WsLayout w;
  const size_t ldw = ((size_t)B + 3) / 4 * 4;  // the fused path pads rows to a multiple of 4 elements
  size_t blk_s = align256((size_t)M * ldw * ss), blk_d = align256((size_t)M * ldw * sd);
  if (2 * ss <= sd) blk_d = std::max(blk_d, 2 * blk_s);
  w.y64 = 0;
  w.sx_t = blk_d;                       // S X (FP64) during set-up, then T (and H T when 2 ss <= sd)
  size_t off = 2 * blk_d;
  if (2 * ss <= sd) w.ht = w.sx_t + blk_s; else { w.ht = off; off += blk_s; }
  w.rx = off; off += blk_s;
  w.ry = off; off += blk_s;
  w.total = off;
  return w;
}

pawfe_status ensure_scalars(pawfe_ctx* c, size_t doubles) {
  if (doubles <= c->scal_doubles) return PAWFE_OK;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (c->h_pinned) cudaFreeHost(c->h_pinned);
  cudaFree(c->d_scal);
  c->h_pinned = nullptr; c->d_scal = nullptr; c->scal_doubles = 0;
  size_t cap = std::max<size_t>(doubles, 64 * 512);
  CUDA_TRY(c, cudaMallocHost((void**)&c->h_pinned, cap * pawfe_ctx::kScalSlots * sizeof(double)));
  CUDA_TRY(c, cudaMalloc((void**)&c->d_scal, cap * pawfe_ctx::kScalSlots * sizeof(double)));
  for (int i = 0; i < pawfe_ctx::kScalSlots; ++i)
    if (!c->scal_ev[i]) CUDA_TRY(c, cudaEventCreateWithFlags(&c->scal_ev[i], cudaEventDisableTiming));
  c->scal_doubles = cap;
  return PAWFE_OK;
}

// Step 1 and the Lambda recurrences of Alg. 2 on the host in FP64 (L257, L264, L275).  Fills a pinned staging slot,
// starts its copy to the device and returns the per-step coefficients:
//   device scalars ds: [0, B) Lambda;  [(th-1) B, th B) a_th Lambda_Y (th = 2..m);  [m B, (m+1) B) final Lambda_Y;
//   [(m+1) B, (m+2) B) -Lambda
struct FilterScalars {
  const double* ds = nullptr;
  std::vector<double> as, acs, zzs;
  double z_over_e = 0.0;
};

pawfe_status filter_scalars(pawfe_ctx* c, int m, double b0, double bW, double bU, const double* lambda, int B,
                            FilterScalars* out) {
  const double e = 0.5 * (bU - bW), cc = 0.5 * (bU + bW);
  double zeta = e / (b0 - cc);
  const double gamma = 2.0 / zeta;
  TRY(ensure_scalars(c, (size_t)(m + 2) * B));
  const int slot = c->scal_next;
  c->scal_next = (slot + 1) % pawfe_ctx::kScalSlots;
  CUDA_TRY(c, cudaEventSynchronize(c->scal_ev[slot]));  // the slot's previous copy has been consumed
  double* hs = c->h_pinned + (size_t)slot * c->scal_doubles;
  double* ds = c->d_scal + (size_t)slot * c->scal_doubles;
  std::vector<double> LX(B, 1.0), LY(B);
  out->as.assign(m + 1, 0.0); out->acs.assign(m + 1, 0.0); out->zzs.assign(m + 1, 0.0);
  const double z_over_e = zeta / e;
  for (int v = 0; v < B; ++v) { hs[v] = lambda[v]; LY[v] = z_over_e * (lambda[v] - cc); }
  for (int th = 2; th <= m; ++th) {
    double zeta1 = 1.0 / (gamma - zeta);
    double a = 2.0 * zeta1 / e;
    out->as[th] = a; out->acs[th] = a * cc; out->zzs[th] = zeta * zeta1;
    double* aL = hs + (size_t)(th - 1) * B;
    for (int v = 0; v < B; ++v) {
      aL[v] = a * LY[v];
      double lx = a * LY[v] * lambda[v] - a * cc * LY[v] - zeta * zeta1 * LX[v];
      LX[v] = LY[v]; LY[v] = lx;  // swap
    }
    zeta = zeta1;
  }
  for (int v = 0; v < B; ++v) { hs[(size_t)m * B + v] = LY[v]; hs[(size_t)(m + 1) * B + v] = -lambda[v]; }
  CUDA_TRY(c, cudaMemcpyAsync(ds, hs, (size_t)(m + 2) * B * sizeof(double), cudaMemcpyHostToDevice, c->stream));
  CUDA_TRY(c, cudaEventRecord(c->scal_ev[slot], c->stream));
  out->ds = ds; out->z_over_e = z_over_e;
  return PAWFE_OK;
}

// TS: storage scalar (float / double / float2 / double2), TD: FP64 scalar of the same kind
template <typename TS, typename TD>
pawfe_status filter_impl(pawfe_ctx* c, pawfe_prec prec, int m, double b0, double bW, double bU, TS* X,
                         const double* lambda, long ld, int B, void* workspace, const void* HXin = nullptr,
                         const void* SXin = nullptr) {
  typedef typename ScalarTraits<TS>::real RS;
  const int cw = ScalarTraits<TS>::cplx ? 2 : 1;
  const int W = B * cw;
  const long total = c->M * (long)W;
  WsLayout wl = ws_layout(c->M, B, sizeof(TS), sizeof(TD));
  char* ws = (char*)workspace;
  TD* Y64 = (TD*)(ws + wl.y64);
  TD* SX64 = (TD*)(ws + wl.sx_t);
  TS* T = (TS*)(ws + wl.sx_t);
  TS* HT = (TS*)(ws + wl.ht);
  TS* RX = (TS*)(ws + wl.rx);
  TS* RY = (TS*)(ws + wl.ry);

  FilterScalars fs;
  TRY(filter_scalars(c, m, b0, bW, bU, lambda, B, &fs));
  const double* ds = fs.ds;
  const std::vector<double>&as = fs.as, &acs = fs.acs, &zzs = fs.zzs;
  const double z_over_e = fs.z_over_e;

  const int gs = 8 * c->sm_count;
  // ---- step 2: Y = H X - S X Lambda in FP64 (L260, L374) ----
  prof_setup_mark(c, true);
  if (HXin && SXin) {   // the caller's products (pawfe_cheb_filter_hs): no operator application
    k_residual_from_products<<<gs, 256, 0, c->stream>>>(c->M, (long)W, W, cw, (const double*)HXin, (const double*)SXin, ld * cw, ds, (double*)Y64);
    KERNEL_CHECK(c, "k_residual_from_products");
  } else {
    TRY((pawfe_apply_HS<TS, TD, TD>(c, 0, false, X, ld, Y64, B, B)));
    (void)SX64;   // S X is not stored: Y -= (S X) Lambda directly (mass part by 1-D sweeps, Lambda folded into the coupling)
    TRY((pawfe_sub_SX_lambda<TS, TD>(c, X, ld, Y64, B, B, ds, ds + (size_t)(m + 1) * B)));
  }
  // ---- step 3 ----
  k_residual_init<RS><<<gs, 256, 0, c->stream>>>(c->M, W, cw, (double*)Y64, (const double*)nullptr, ds, z_over_e,
                                                 (RS*)RX, (RS*)RY);
  KERNEL_CHECK(c, "k_residual_init");
  prof_setup_mark(c, false);
  // ---- step 4 ----
  for (int th = 2; th <= m; ++th) {
    TRY((pawfe_apply_Sinv_impl<TS, TS, TS>(c, RY, B, T, B, B)));
    TRY(pawfe_apply_H_any(c, prec, T, B, HT, B, B));
    if constexpr (std::is_same<RS, float>::value) {
      if ((W & 3) == 0) {
        k_recurrence_f4<<<gs, 256, 0, c->stream>>>(total / 4, W / 4, cw, (const float4*)HT, (const float4*)RY, (float4*)RX,
                                                   (const double2*)Y64, ds + (size_t)(th - 1) * B, (float)as[th], (float)acs[th], (float)zzs[th]);
        KERNEL_CHECK(c, "k_recurrence_f4");
        std::swap(RX, RY);
        continue;
      }
    }
    k_recurrence<RS><<<gs, 256, 0, c->stream>>>(total, W, cw, (const RS*)HT, (const RS*)RY, (RS*)RX,
                                                (const double*)Y64, ds + (size_t)(th - 1) * B, as[th], acs[th], zzs[th]);
    KERNEL_CHECK(c, "k_recurrence");
    std::swap(RX, RY);
  }
  // ---- step 5: Psi_f = S^-1approx R_Y + X Lambda_Y (L282) ----
  TRY((pawfe_apply_Sinv_impl<TS, TS, TS>(c, RY, B, T, B, B)));
  k_recover<RS><<<gs, 256, 0, c->stream>>>(c->md, W, cw, (const RS*)T, (RS*)X, ld * cw, ds + (size_t)m * B);
  KERNEL_CHECK(c, "k_recover");
  return PAWFE_OK;
}

pawfe_status check_filter(pawfe_ctx* c, pawfe_prec prec, int m, double b0, double bW, double bU, const void* X,
                          const double* lambda, long ld, int B) {
  if (!c) return PAWFE_EINVAL;
  if (!X || !lambda || B < 1 || B > 512 || ld < B || m < 1 || m > 512) { c->err = "bad filter arguments"; return PAWFE_EINVAL; }
  if (!(bU > bW) || !(b0 < bW)) { c->err = "need b0 < bW < bU"; return PAWFE_EINVAL; }
  if (prec != PAWFE_FP64 && prec != PAWFE_FP32 && prec != PAWFE_TF32) return PAWFE_EINVAL;
  if (!c->have_mesh || !c->have_atoms || !c->have_pot) { c->err = "operators not set up"; return PAWFE_ESTATE; }
  if (!c->have_h64) { c->err = "the filter's residual set-up needs the FP64 cell matrices (keep_fp64 = 1)"; return PAWFE_ESTATE; }
  return PAWFE_OK;
}

// bytes of workspace of the generic sequence (fused = false) or of the fused step
size_t filter_ws_bytes(pawfe_ctx* c, pawfe_prec prec, int B, bool fused) {
  size_t cw = c->cplx ? 2 : 1;
  size_t ss = (prec == PAWFE_FP64 ? 8 : 4) * cw, sd = 8 * cw;
  size_t bytes = ws_layout(c->M, B, ss, sd).total;
  if (fused) {
    // fused step (fused.h): Yt (FP64) + Rt_X + Rt_Y (FP32) as real blocks of B * cw columns; S X, T and H T are never
    // stored.  Never more than the generic layout, so a block the fused path turns down (alignment) still fits.
    const size_t ldw = ((size_t)B * cw + 3) / 4 * 4;
    bytes = align256((size_t)c->M * ldw * 8) + (prec == PAWFE_FP32 ? 3 : 2) * align256((size_t)c->M * ldw * 4);
  }
  return bytes;
}

// complex blocks take the fused step only with an even width (16-byte pieces of interleaved columns)
bool fused_width_ok(pawfe_ctx* c, pawfe_prec prec, int B) { return fused_supported(c, prec, B) && (!c->cplx || !(B & 1)); }

}  // namespace

extern "C" pawfe_status pawfe_filter_workspace(pawfe_ctx* c, pawfe_prec prec, int B, size_t* bytes) {
  if (!c || !bytes || B < 1 || B > 512) return PAWFE_EINVAL;
  if (!c->have_mesh) return PAWFE_ESTATE;
  // complex blocks with an odd leading dimension or a misaligned pointer fall back to the unfused sequence, which needs
  // more: complex contexts are always told the larger figure, so a workspace of this size fits every (ld, X)
  const size_t fused = filter_ws_bytes(c, prec, B, fused_width_ok(c, prec, B));
  *bytes = c->cplx ? std::max(fused, filter_ws_bytes(c, prec, B, false)) : fused;
  return PAWFE_OK;
}

// Allocate now what the hot calls would otherwise allocate on first use (include/pawfe.h).
extern "C" pawfe_status pawfe_prepare(pawfe_ctx* c, pawfe_prec prec, int Bmax, int mmax) {
  if (!c || Bmax < 1 || Bmax > 512 || mmax < 1 || mmax > 512) return PAWFE_EINVAL;
  if (prec != PAWFE_FP64 && prec != PAWFE_FP32 && prec != PAWFE_TF32) return PAWFE_EINVAL;
  if (!c->have_mesh || !c->have_atoms || !c->have_pot) { c->err = "operators not set up"; return PAWFE_ESTATE; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  TRY(ensure_scalars(c, (size_t)(mmax + 2) * Bmax));
  TRY(pawfe_ensure_P(c, Bmax));
  if (prec != PAWFE_FP64 && tc_supported(c, Bmax)) TRY(tc_prepare(c));
  if (fused_supported(c, prec, Bmax)) TRY(fused_prepare_all(c, prec, Bmax, true));
  const size_t need = (size_t)c->M * Bmax * (prec == PAWFE_FP64 ? 8 : 4) * (c->cplx ? 2 : 1);
  if (need > c->tmpblk_bytes) {
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    cudaFree(c->d_tmpblk); c->d_tmpblk = nullptr; c->tmpblk_bytes = 0;
    char* q = nullptr; TRY(dev_alloc(c, &q, need)); c->d_tmpblk = q; c->tmpblk_bytes = need;
  }
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return PAWFE_OK;
}

static pawfe_status cheb_filter_impl(pawfe_ctx* c, pawfe_prec prec, int m, double b0, double bW, double bU,
                                     void* X, const double* lambda, long ld, int B, void* workspace,
                                     size_t workspace_bytes, const void* HX, const void* SX) {
  TRY(check_filter(c, prec, m, b0, bW, bU, X, lambda, ld, B));
  if ((HX != nullptr) != (SX != nullptr)) { c->err = "give both H X and S X, or neither"; return PAWFE_EINVAL; }
  // complex blocks with an odd leading dimension or a misaligned pointer run the generic sequence (larger workspace)
  const bool fused = fused_width_ok(c, prec, B) && (!c->cplx || (!(ld & 1) && !((uintptr_t)X & 15)));
  const size_t need = filter_ws_bytes(c, prec, B, fused);
  if (!workspace || workspace_bytes < need || ((uintptr_t)workspace & 255)) {
    c->err = fused ? "workspace too small or misaligned"
                   : "workspace too small or misaligned (blocks the fused step cannot take need the generic sequence's workspace)";
    return PAWFE_EINVAL;
  }
  CUDA_TRY(c, cudaSetDevice(c->device));
  if (c->cplx) {
    if (prec == PAWFE_FP64) return filter_impl<double2, double2>(c, prec, m, b0, bW, bU, (double2*)X, lambda, ld, B, workspace, HX, SX);
    if (fused) {
      FilterScalars fs;
      TRY(filter_scalars(c, m, b0, bW, bU, lambda, B, &fs));
      return fused_filter(c, prec, m, fs.ds, fs.as.data(), fs.acs.data(), fs.zzs.data(), fs.z_over_e, X, ld, B, workspace, HX, SX);
    }
    return filter_impl<float2, double2>(c, prec, m, b0, bW, bU, (float2*)X, lambda, ld, B, workspace, HX, SX);
  }
  if (prec == PAWFE_FP64) return filter_impl<double, double>(c, prec, m, b0, bW, bU, (double*)X, lambda, ld, B, workspace, HX, SX);
  if (fused) {
    FilterScalars fs;
    TRY(filter_scalars(c, m, b0, bW, bU, lambda, B, &fs));
    return fused_filter(c, prec, m, fs.ds, fs.as.data(), fs.acs.data(), fs.zzs.data(), fs.z_over_e, X, ld, B, workspace, HX, SX);
  }
  return filter_impl<float, double>(c, prec, m, b0, bW, bU, (float*)X, lambda, ld, B, workspace, HX, SX);
}

extern "C" pawfe_status pawfe_cheb_filter(pawfe_ctx* c, pawfe_prec prec, int m, double b0, double bW, double bU,
                                          void* X, const double* lambda, long ld, int B, void* workspace,
                                          size_t workspace_bytes) {
  return cheb_filter_impl(c, prec, m, b0, bW, bU, X, lambda, ld, B, workspace, workspace_bytes, nullptr, nullptr);
}

// Algorithm 2 with step 2 taken from products the caller already holds
extern "C" pawfe_status pawfe_cheb_filter_hs(pawfe_ctx* c, pawfe_prec prec, int m, double b0, double bW, double bU,
                                             void* X, const double* HX, const double* SX, const double* lambda, long ld,
                                             int B, void* workspace, size_t workspace_bytes) {
  if (!c) return PAWFE_EINVAL;
  if (!HX || !SX) { c->err = "pawfe_cheb_filter_hs needs H X and S X"; return PAWFE_EINVAL; }
  return cheb_filter_impl(c, prec, m, b0, bW, bU, X, lambda, ld, B, workspace, workspace_bytes, HX, SX);
}

extern "C" pawfe_status pawfe_cheb_filter_host(pawfe_ctx* c, pawfe_prec prec, int m, double b0, double bW,
                                               double bU, void* X_host, const double* lambda, long ld, int B) {
  TRY(check_filter(c, prec, m, b0, bW, bU, X_host, lambda, ld, B));
  CUDA_TRY(c, cudaSetDevice(c->device));
  size_t es = (prec == PAWFE_FP64 ? 8 : 4) * (c->cplx ? 2 : 1);
  const size_t blk = (size_t)c->M * ld * es;
  const size_t need = filter_ws_bytes(c, prec, B, fused_width_ok(c, prec, B) && (!c->cplx || !(ld & 1)));
  if (blk > c->hostblk_bytes) {
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    cudaFree(c->d_hostblk); c->d_hostblk = nullptr; c->hostblk_bytes = 0;
    char* p = nullptr; TRY(dev_alloc(c, &p, blk)); c->d_hostblk = p; c->hostblk_bytes = blk;
  }
  if (need > c->hostws_bytes) {
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    cudaFree(c->d_hostws); c->d_hostws = nullptr; c->hostws_bytes = 0;
    char* p = nullptr; TRY(dev_alloc(c, &p, need)); c->d_hostws = p; c->hostws_bytes = need;
  }
  CUDA_TRY(c, cudaMemcpyAsync(c->d_hostblk, X_host, blk, cudaMemcpyHostToDevice, c->stream));
  TRY(pawfe_cheb_filter(c, prec, m, b0, bW, bU, c->d_hostblk, lambda, ld, B, c->d_hostws, c->hostws_bytes));
  CUDA_TRY(c, cudaMemcpyAsync(X_host, c->d_hostblk, blk, cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return PAWFE_OK;
}

// Pipelined over two device blocks: H2D of block k+1 and D2H of block k-1 on the copy streams under block k's filter.
extern "C" pawfe_status pawfe_cheb_filter_host_set(pawfe_ctx* c, pawfe_prec prec, int m, double b0, double bW, double bU,
                                                   void* const* X_host, const double* const* lambda, const long* ld,
                                                   const int* B, int nblk) {
  if (!c) return PAWFE_EINVAL;
  if (nblk < 1 || !X_host || !lambda || !ld || !B) { c->err = "bad block-set arguments"; return PAWFE_EINVAL; }
  const size_t es = (prec == PAWFE_FP64 ? 8 : 4) * (c->cplx ? 2 : 1);
  size_t blk_max = 0, need_max = 0;
  for (int k = 0; k < nblk; ++k) {
    TRY(check_filter(c, prec, m, b0, bW, bU, X_host[k], lambda[k], ld[k], B[k]));
    blk_max = std::max(blk_max, (size_t)c->M * ld[k] * es);
    need_max = std::max(need_max, filter_ws_bytes(c, prec, B[k], fused_width_ok(c, prec, B[k]) && (!c->cplx || !(ld[k] & 1))));
  }
  CUDA_TRY(c, cudaSetDevice(c->device));
  auto grow = [&](void** p, size_t* have, size_t want) -> pawfe_status {
    if (want <= *have) return PAWFE_OK;
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    cudaFree(*p); *p = nullptr; *have = 0;
    char* q = nullptr; TRY(dev_alloc(c, &q, want)); *p = q; *have = want;
    return PAWFE_OK;
  };
  TRY(grow(&c->d_hostblk, &c->hostblk_bytes, blk_max));
  if (nblk > 1) TRY(grow(&c->d_hostblk2, &c->hostblk2_bytes, blk_max));
  TRY(grow(&c->d_hostws, &c->hostws_bytes, need_max));
  if (!c->s_h2d) {
    CUDA_TRY(c, cudaStreamCreateWithFlags(&c->s_h2d, cudaStreamNonBlocking));
    CUDA_TRY(c, cudaStreamCreateWithFlags(&c->s_d2h, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_h2d[i], cudaEventDisableTiming));
      CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_filt[i], cudaEventDisableTiming));
      CUDA_TRY(c, cudaEventCreateWithFlags(&c->ev_d2h[i], cudaEventDisableTiming));
    }
  }
  void* dblk[2] = {c->d_hostblk, c->d_hostblk2};
  // the copy streams start after whatever the caller has queued on the context's stream
  CUDA_TRY(c, cudaEventRecord(c->ev_filt[0], c->stream));
  CUDA_TRY(c, cudaStreamWaitEvent(c->s_h2d, c->ev_filt[0], 0));
  auto h2d = [&](int k) -> pawfe_status {
    const int b = k & 1;
    if (k >= 2) CUDA_TRY(c, cudaStreamWaitEvent(c->s_h2d, c->ev_d2h[b], 0));   // block k-2 has left this device block
    CUDA_TRY(c, cudaMemcpyAsync(dblk[b], X_host[k], (size_t)c->M * ld[k] * es, cudaMemcpyHostToDevice, c->s_h2d));
    CUDA_TRY(c, cudaEventRecord(c->ev_h2d[b], c->s_h2d));
    return PAWFE_OK;
  };
  TRY(h2d(0));
  for (int k = 0; k < nblk; ++k) {
    const int b = k & 1;
    if (k + 1 < nblk) TRY(h2d(k + 1));     // queued before block k's filter: runs under it
    CUDA_TRY(c, cudaStreamWaitEvent(c->stream, c->ev_h2d[b], 0));
    TRY(pawfe_cheb_filter(c, prec, m, b0, bW, bU, dblk[b], lambda[k], ld[k], B[k], c->d_hostws, c->hostws_bytes));
    CUDA_TRY(c, cudaEventRecord(c->ev_filt[b], c->stream));
    CUDA_TRY(c, cudaStreamWaitEvent(c->s_d2h, c->ev_filt[b], 0));
    CUDA_TRY(c, cudaMemcpyAsync(X_host[k], dblk[b], (size_t)c->M * ld[k] * es, cudaMemcpyDeviceToHost, c->s_d2h));
    CUDA_TRY(c, cudaEventRecord(c->ev_d2h[b], c->s_d2h));
  }
  CUDA_TRY(c, cudaStreamSynchronize(c->s_d2h));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return PAWFE_OK;
}
