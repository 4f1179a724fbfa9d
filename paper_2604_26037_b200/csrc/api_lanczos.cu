// api_lanczos.cu -- pawfe_lanczos_bound: upper bound b_U of the spectrum of the operator Algorithm 2 iterates, H S^-1approx
// (Alg. 1 steps 1-2; L179; reading R17).  The paper's "k-step generalised
// Lanczos" (its ref. 25) is not available; this is a k-step Lanczos on H S^-1approx in the S^-1approx inner product
// <x, y> = Re x^dagger S^-1approx y, in which H S^-1approx is self-adjoint:
//     v_1 = keep o v0 / ||.||;   w = H S^-1approx v_j - beta_{j-1} v_{j-1};   alpha_j = <v_j, w>;   w -= alpha_j v_j;
//     beta_j = sqrt(<w, w>);   v_{j+1} = w / beta_j;          b_U = 1.02 (theta_max(T_k) + beta_k)
// in FP64 with the library's own applies (one-column blocks).  Not a hot call: allocates five vectors, synchronises per step.
#include "common.h"
#include "host_util.h"
#include "kernels_stream.cuh"
#include "apply_impl.h"
#include <algorithm>
#include <cmath>
#include <vector>

namespace {

// out[0] += Re sum_i conj(x_i) y_i over W reals per row (complex: interleaved, so this is the plain real dot product)
__global__ void __launch_bounds__(256)
k_dot_real(long total, const double* __restrict__ x, const double* __restrict__ y, double* __restrict__ out) {
  __shared__ double red[8];
  double s = 0.0;
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) s = fma(x[i], y[i], s);
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += red[w];
    atomicAdd(out, t);
  }
}
// y = a x + b y
__global__ void k_axpby(long total, double a, const double* x, double b, double* y) {   // (x may be y)
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) y[i] = a * x[i] + b * y[i];
}
// y = keep o x (rows where M_D^-1 is stored as 0, the Dirichlet walls, become 0)
__global__ void k_keep_rows(MeshDev md, int W, const double* __restrict__ x, double* __restrict__ y) {
  const long total = md.M * (long)W;
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x)
    y[i] = mdinv_of_row(md, i / W) != 0.0 ? x[i] : 0.0;
}

// largest eigenvalue of the symmetric tridiagonal (alpha, beta) by bisection on the Sturm count
double tridiag_max_eig(const std::vector<double>& a, const std::vector<double>& b) {
  const int k = (int)a.size();
  double lo = a[0], hi = a[0];
  for (int i = 0; i < k; ++i) {
    const double r = (i > 0 ? std::fabs(b[i - 1]) : 0.0) + (i + 1 < k ? std::fabs(b[i]) : 0.0);
    lo = std::min(lo, a[i] - r); hi = std::max(hi, a[i] + r);
  }
  auto count_below = [&](double x) {   // eigenvalues < x
    int cnt = 0;
    double d = 1.0;
    for (int i = 0; i < k; ++i) {
      const double off = i > 0 ? b[i - 1] * b[i - 1] : 0.0;
      d = a[i] - x - (i > 0 ? off / d : 0.0);
      if (d == 0.0) d = 1e-300;
      if (d < 0.0) ++cnt;
    }
    return cnt;
  };
  for (int it = 0; it < 200 && hi - lo > 1e-15 * std::max(1.0, std::fabs(hi)); ++it) {
    const double mid = 0.5 * (lo + hi);
    if (count_below(mid) >= k) hi = mid; else lo = mid;   // all k eigenvalues below mid: the largest is below mid
  }
  return 0.5 * (lo + hi);
}

template <typename TD>
pawfe_status lanczos_impl(pawfe_ctx* c, int k, const TD* v0, double* bU, double* theta_max, double* beta_last, int* steps) {
  const int cw = ScalarTraits<TD>::cplx ? 2 : 1;
  const long total = c->M * (long)cw;
  TD *v = nullptr, *vp = nullptr, *w = nullptr, *t = nullptr;
  double* d_s = nullptr;
  pawfe_status st = PAWFE_OK;
  auto cleanup = [&]() { cudaFree(v); cudaFree(vp); cudaFree(w); cudaFree(t); cudaFree(d_s); };
#define TRYL(x) do { st = (x); if (st != PAWFE_OK) { cleanup(); return st; } } while (0)
#define CUDAL(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { c->err = std::string(#x) + ": " + cudaGetErrorString(e_); cleanup(); return PAWFE_ECUDA; } } while (0)
  TRYL(dev_alloc(c, &v, (size_t)c->M)); TRYL(dev_alloc(c, &vp, (size_t)c->M)); TRYL(dev_alloc(c, &w, (size_t)c->M));
  TRYL(dev_alloc(c, &t, (size_t)c->M)); TRYL(dev_alloc(c, &d_s, 1));
  const int gs = 4 * c->sm_count;
  auto ip = [&](const TD* x, const TD* y, double* out) -> pawfe_status {   // <x, y> = Re x^dagger S^-1approx y
    TRY((pawfe_apply_Sinv_impl<TD, TD, TD>(c, y, 1, t, 1, 1)));
    CUDA_TRY(c, cudaMemsetAsync(d_s, 0, sizeof(double), c->stream));
    k_dot_real<<<gs, 256, 0, c->stream>>>(total, (const double*)x, (const double*)t, d_s);
    KERNEL_CHECK(c, "k_dot_real");
    CUDA_TRY(c, cudaMemcpyAsync(out, d_s, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return PAWFE_OK;
  };
  k_keep_rows<<<gs, 256, 0, c->stream>>>(c->md, cw, (const double*)v0, (double*)v);
  c->launches++;
  CUDAL(cudaGetLastError());
  double nrm2 = 0.0;
  TRYL(ip(v, v, &nrm2));
  if (!(nrm2 > 0.0)) { c->err = "pawfe_lanczos_bound: the start vector vanishes on the free dofs"; cleanup(); return PAWFE_EINVAL; }
  k_axpby<<<gs, 256, 0, c->stream>>>(total, 0.0, (const double*)v, 1.0 / std::sqrt(nrm2), (double*)v);
  CUDAL(cudaMemsetAsync(vp, 0, (size_t)c->M * sizeof(TD), c->stream));
  c->launches++;
  std::vector<double> alphas, betas;
  double beta = 0.0;
  for (int j = 0; j < k; ++j) {
    TRYL((pawfe_apply_Sinv_impl<TD, TD, TD>(c, v, 1, t, 1, 1)));            // t = S^-1approx v
    TRYL((pawfe_apply_HS<TD, TD, TD>(c, 0, false, t, 1, w, 1, 1)));         // w = H t
    k_axpby<<<gs, 256, 0, c->stream>>>(total, -beta, (const double*)vp, 1.0, (double*)w);
    c->launches++;
    double alpha = 0.0, b2 = 0.0;
    TRYL(ip(v, w, &alpha));
    k_axpby<<<gs, 256, 0, c->stream>>>(total, -alpha, (const double*)v, 1.0, (double*)w);
    c->launches++;
    TRYL(ip(w, w, &b2));
    beta = std::sqrt(std::max(b2, 0.0));
    alphas.push_back(alpha); betas.push_back(beta);
    if (beta < 1e-14) break;
    std::swap(vp, v);                                                          // vprev = v
    k_axpby<<<gs, 256, 0, c->stream>>>(total, 1.0 / beta, (const double*)w, 0.0, (double*)v);   // v = w / beta
    c->launches++;
  }
  CUDAL(cudaStreamSynchronize(c->stream));
  cleanup();
#undef TRYL
#undef CUDAL
  std::vector<double> off(betas.begin(), betas.end() - 1);
  const double th = tridiag_max_eig(alphas, off);
  *theta_max = th; *beta_last = betas.back(); *steps = (int)alphas.size();
  *bU = 1.02 * (th + betas.back());
  return PAWFE_OK;
}

}  // namespace

extern "C" pawfe_status pawfe_lanczos_bound(pawfe_ctx* c, int k, const void* v0, double* bU, double* theta_max, double* beta_k,
                                            int* steps_done) {
  if (!c) return PAWFE_EINVAL;
  if (!v0 || !bU || k < 1 || k > 256) { c->err = "bad Lanczos arguments"; return PAWFE_EINVAL; }
  if (!c->have_mesh || !c->have_atoms || !c->have_pot) { c->err = "operators not set up"; return PAWFE_ESTATE; }
  if (!c->have_h64) { c->err = "pawfe_lanczos_bound works in FP64: keep_fp64 = 1 needed"; return PAWFE_ESTATE; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  double th = 0.0, bl = 0.0;
  int steps = 0;
  pawfe_status st = c->cplx ? lanczos_impl<double2>(c, k, (const double2*)v0, bU, &th, &bl, &steps)
                            : lanczos_impl<double>(c, k, (const double*)v0, bU, &th, &bl, &steps);
  if (st != PAWFE_OK) return st;
  if (theta_max) *theta_max = th;
  if (beta_k) *beta_k = bl;
  if (steps_done) *steps_done = steps;
  return PAWFE_OK;
}
