// api_setup.cu -- operator set-up calls of the C ABI: cell matrices from the Gaussian local potential
// (Eq. 13 / Eq. 32) and the atom / projector data (Eq. 16-17, 34; Eq. 28-29).
#include "common.h"
#include "fe_tables.h"
#include "host_util.h"
#include "fe_setup.cuh"
#include "api_internal.h"
#include <algorithm>
#include <cmath>

using namespace pawfe;

// ================================================================================================
// local potential -> cell matrices
// ================================================================================================
extern "C" pawfe_status pawfe_local_potential_gaussians(pawfe_ctx* c, int natoms, const double* pos,
                                                        const double* Z, const double* sigma, int keep_fp64) {
  if (!c || natoms < 0 || (natoms > 0 && (!pos || !Z || !sigma))) return PAWFE_EINVAL;
  if (!c->have_mesh) { c->err = "mesh not created"; return PAWFE_ESTATE; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  pawfe_free_pot(c);
  const int n = c->n, n1 = c->n1, p = c->p, nq = p + 2, cw = c->cplx ? 2 : 1;
  const long nq3 = (long)nq * nq * nq;

  // 1-D tables
  std::vector<double> xq, wq, Lq, dLq;
  gauss_legendre_rule(nq, xq, wq);
  lagrange_basis(c->xi, xq, Lq, dLq);  // [n1][nq]

  // reference matrices: Kre = 1/2 K^e + 1/2 |k|^2 M^e,  Kim = - sum_d k_d G_d^e   (Eq. 13; reading R6 of DESIGN.md)
  const double hx = 0.5 * c->h[0], hy = 0.5 * c->h[1], hz = 0.5 * c->h[2];
  std::vector<double> Kre((size_t)n * n, 0.0), Kim((size_t)n * n, 0.0);
  kron3(n1, c->K1, c->M1, c->M1, 0.5 * hy * hz / hx, Kre);
  kron3(n1, c->M1, c->K1, c->M1, 0.5 * hx * hz / hy, Kre);
  kron3(n1, c->M1, c->M1, c->K1, 0.5 * hx * hy / hz, Kre);
  if (c->cplx) {
    double k2 = c->kpt[0] * c->kpt[0] + c->kpt[1] * c->kpt[1] + c->kpt[2] * c->kpt[2];
    kron3(n1, c->M1, c->M1, c->M1, 0.5 * k2 * hx * hy * hz, Kre);
    kron3(n1, c->G1, c->M1, c->M1, -c->kpt[0] * hy * hz, Kim);
    kron3(n1, c->M1, c->G1, c->M1, -c->kpt[1] * hx * hz, Kim);
    kron3(n1, c->M1, c->M1, c->G1, -c->kpt[2] * hx * hy, Kim);
  }

  double *d_xq = nullptr, *d_wq = nullptr, *d_Lq = nullptr, *d_Kre = nullptr, *d_Kim = nullptr;
  double *d_pos = nullptr, *d_Z = nullptr, *d_sig = nullptr, *d_WV = nullptr, *d_scratch = nullptr;
  pawfe_status st = PAWFE_OK;
  auto cleanup = [&]() {
    cudaFree(d_xq); cudaFree(d_wq); cudaFree(d_Lq); cudaFree(d_Kre); cudaFree(d_Kim);
    cudaFree(d_pos); cudaFree(d_Z); cudaFree(d_sig); cudaFree(d_WV); cudaFree(d_scratch);
  };
#define TRYC(x) do { st = (x); if (st != PAWFE_OK) { cleanup(); pawfe_free_pot(c); return st; } } while (0)
#define CUDAC(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { c->err = std::string(#call) + ": " + cudaGetErrorString(e_); cleanup(); pawfe_free_pot(c); return PAWFE_ECUDA; } } while (0)
  TRYC(upload(c, &d_xq, xq)); TRYC(upload(c, &d_wq, wq)); TRYC(upload(c, &d_Lq, Lq));
  TRYC(upload(c, &d_Kre, Kre)); TRYC(upload(c, &d_Kim, Kim));
  std::vector<double> vpos(pos, pos + 3 * (size_t)natoms), vZ(Z, Z + natoms), vs(sigma, sigma + natoms);
  if (natoms > 0) { TRYC(upload(c, &d_pos, vpos)); TRYC(upload(c, &d_Z, vZ)); TRYC(upload(c, &d_sig, vs)); }
  TRYC(dev_alloc(c, &d_WV, (size_t)c->ncell * nq3));

  SetupGeom g;
  for (int d = 0; d < 3; ++d) { g.h[d] = c->h[d]; g.box[d] = c->box[d]; }
  g.periodic = (c->bc == PAWFE_PERIODIC);
  k_potential_wv<<<c->ncell, 256, 0, c->stream>>>(c->md, g, nq, d_xq, d_wq, natoms, d_pos, d_Z, d_sig, d_WV);
  c->launches++;
  CUDAC(cudaGetLastError());

  size_t h32_elems = (size_t)c->ncell * n * c->ldk * cw;
  float* H32 = nullptr; double* H64 = nullptr;
  TRYC(dev_alloc(c, &H32, h32_elems));
  c->d_H32 = H32;
  CUDAC(cudaMemsetAsync(H32, 0, h32_elems * sizeof(float), c->stream));
  if (keep_fp64) {
    TRYC(dev_alloc(c, &H64, (size_t)c->ncell * n * n * cw));
    c->d_H64 = H64;
  }
  int grid = std::min(c->ncell, 2 * c->sm_count);
  TRYC(dev_alloc(c, &d_scratch, (size_t)grid * nq * n1 * n1 * n1 * n1));
  size_t smem = ((size_t)n1 * n1 * nq + nq3 + (size_t)nq * nq * n1 * n1) * sizeof(double);
  if (c->cplx) {
    CUDAC(cudaFuncSetAttribute(k_build_hcell<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_build_hcell<true><<<grid, 256, smem, c->stream>>>(c->md, nq, d_Lq, d_WV, d_Kre, d_Kim, d_scratch, H64, H32, c->ldk);
  } else {
    CUDAC(cudaFuncSetAttribute(k_build_hcell<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_build_hcell<false><<<grid, 256, smem, c->stream>>>(c->md, nq, d_Lq, d_WV, d_Kre, d_Kim, d_scratch, H64, H32, c->ldk);
  }
  c->launches++;
  CUDAC(cudaGetLastError());
  CUDAC(cudaStreamSynchronize(c->stream));
  cleanup();
#undef TRYC
#undef CUDAC
  c->have_pot = true;
  c->have_h64 = keep_fp64 != 0;
  return PAWFE_OK;
}

namespace {
// FP32 copy of the FP64 cell matrices with the padded row stride ldk (columns >= n are zero): [cell][n][ldk] scalars
__global__ void k_h64_to_h32(const double* __restrict__ H64, int n, int ldk, int cw, long rows, float* __restrict__ H32) {
  const long total = rows * ldk * cw;
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    const int q = (int)(i % cw);
    const long t = i / cw;
    const int k = (int)(t % ldk);
    const long row = t / ldk;                      // cell * n + I
    H32[i] = k < n ? (float)H64[(row * n + k) * cw + q] : 0.f;
  }
}
}  // namespace

// User- (or oracle-) built cell matrices instead of pawfe_local_potential_gaussians.
extern "C" pawfe_status pawfe_set_cell_matrices(pawfe_ctx* c, const double* Hcell, int is_device, int keep_fp64) {
  if (!c || !Hcell) return PAWFE_EINVAL;
  if (!c->have_mesh) { c->err = "mesh not created"; return PAWFE_ESTATE; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  pawfe_free_pot(c);
  const int n = c->n, cw = c->cplx ? 2 : 1;
  const size_t e64 = (size_t)c->ncell * n * n * cw, e32 = (size_t)c->ncell * n * c->ldk * cw;
  double* H64 = nullptr; float* H32 = nullptr;
  TRY(dev_alloc(c, &H64, e64));
  c->d_H64 = H64;
  cudaError_t e = cudaMemcpyAsync(H64, Hcell, e64 * sizeof(double), is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream);
  if (e != cudaSuccess) { c->err = std::string("pawfe_set_cell_matrices copy: ") + cudaGetErrorString(e); pawfe_free_pot(c); return PAWFE_ECUDA; }
  pawfe_status st = dev_alloc(c, &H32, e32);
  if (st != PAWFE_OK) { pawfe_free_pot(c); return st; }
  c->d_H32 = H32;
  k_h64_to_h32<<<8 * c->sm_count, 256, 0, c->stream>>>(H64, n, c->ldk, cw, (long)c->ncell * n, H32);
  c->launches++;
  e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) { c->err = std::string("pawfe_set_cell_matrices: ") + cudaGetErrorString(e); pawfe_free_pot(c); return PAWFE_ECUDA; }
  if (!keep_fp64) { cudaFree(c->d_H64); c->d_H64 = nullptr; }
  c->have_pot = true;
  c->have_h64 = keep_fp64 != 0;
  return PAWFE_OK;
}

extern "C" pawfe_status pawfe_get_cell_matrix(pawfe_ctx* c, long cell, double* out) {
  if (!c || !out) return PAWFE_EINVAL;
  if (!c->have_pot || !c->have_h64) { c->err = "FP64 cell matrices not kept"; return PAWFE_ESTATE; }
  if (cell < 0 || cell >= c->ncell) return PAWFE_EINVAL;
  size_t sz = (size_t)c->n * c->n * (c->cplx ? 2 : 1);
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  CUDA_TRY(c, cudaMemcpy(out, (double*)c->d_H64 + cell * sz, sz * sizeof(double), cudaMemcpyDeviceToHost));
  return PAWFE_OK;
}
