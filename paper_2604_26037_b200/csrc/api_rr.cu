// api_rr.cu -- the two Rayleigh-Ritz kernels of Algorithm 1 that are the method's own:
//   RR-Projection (Alg. 1 step 4):  G = X^dagger Y  (B x B; Y = H X or S X), only the blocks of the LOWER
//     triangle are computed ("exploits the Hermiticity of the projected matrices"), the upper ones are mirrored;
//   RR-SR (Alg. 1 step 6, L248, L406-L408):  X_out = X Q  with the DIAGONAL blocks of Q applied in FP64 and the OFF-DIAGONAL
//     blocks in FP32 ("mixed precision subspace rotation": the rotation is close to the identity near convergence).
// The dense B x B generalised eigenproblem in between (RR-GHEP, L404: ELPA in the paper) is a library call in harness.py.
// FP64 blocks [dof][vec], real or complex (interleaved).  Plain register-tiled FMA kernels (there is no FP64 kind of tcgen05);
// every sum is taken in a fixed order (row slabs are reduced slab by slab), so the results are bit-reproducible.
// Not hot calls of the filter: pawfe_rr_project allocates its slab partials per call.
#include "common.h"
#include "host_util.h"
#include <algorithm>

namespace {

constexpr int kT = 64;      // tile edge (vectors) of G and Q blocks: the "block" of the mixed-precision rotation
constexpr int kRC = 16;     // rows (projection) / inner vectors (rotation) per shared-memory chunk

template <bool CPLX> struct Acc;
template <> struct Acc<false> {
  typedef double T;
  static __device__ __forceinline__ void fma_conj(double& c, double a, double b) { c = fma(a, b, c); }      // c += conj(a) b
  static __device__ __forceinline__ void fma_(double& c, double a, double b) { c = fma(a, b, c); }          // c += a b
  static __device__ __forceinline__ double zero() { return 0.0; }
  static __device__ __forceinline__ double conj(double a) { return a; }
  static __device__ __forceinline__ double add(double a, double b) { return a + b; }
  static __device__ __forceinline__ double real_part(double a) { return a; }
};
template <> struct Acc<true> {
  typedef double2 T;
  static __device__ __forceinline__ void fma_conj(double2& c, double2 a, double2 b) {
    c.x = fma(a.x, b.x, c.x); c.x = fma(a.y, b.y, c.x); c.y = fma(a.x, b.y, c.y); c.y = fma(-a.y, b.x, c.y);
  }
  static __device__ __forceinline__ void fma_(double2& c, double2 a, double2 b) {
    c.x = fma(a.x, b.x, c.x); c.x = fma(-a.y, b.y, c.x); c.y = fma(a.x, b.y, c.y); c.y = fma(a.y, b.x, c.y);
  }
  static __device__ __forceinline__ double2 zero() { return make_double2(0.0, 0.0); }
  static __device__ __forceinline__ double2 conj(double2 a) { return make_double2(a.x, -a.y); }
  static __device__ __forceinline__ double2 add(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
  static __device__ __forceinline__ double2 real_part(double2 a) { return make_double2(a.x, 0.0); }
};

// partial[slab][tile][i][j] = sum over the slab's rows J of conj(X[J][ib kT + i]) Y[J][jb kT + j], lower tiles (ib >= jb) only.
//   grid = (ntiles, nslab), block = 256 = 16 x 16 threads, each a 4 x 4 sub-tile.
template <bool CPLX>
__global__ void __launch_bounds__(256)
k_rr_project(long M, long rows_per_slab, int B, const typename Acc<CPLX>::T* __restrict__ X, const typename Acc<CPLX>::T* __restrict__ Y,
             long ld, typename Acc<CPLX>::T* __restrict__ partial) {
  typedef typename Acc<CPLX>::T T;
  __shared__ T Xs[kRC][kT], Ys[kRC][kT];
  int ib = 0, t = blockIdx.x;                       // tile index -> (ib, jb) of the lower triangle, row by row
  while (t > ib) { t -= ib + 1; ++ib; }
  const int jb = t;
  const int ti = threadIdx.x >> 4, tj = threadIdx.x & 15;
  const long J0 = blockIdx.y * rows_per_slab, J1 = min(M, J0 + rows_per_slab);
  T acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = Acc<CPLX>::zero();
  for (long J = J0; J < J1; J += kRC) {
    __syncthreads();
    for (int i = threadIdx.x; i < kRC * kT; i += 256) {
      const int r = i / kT, v = i % kT;
      const bool row = J + r < J1;
      Xs[r][v] = (row && ib * kT + v < B) ? X[(J + r) * ld + ib * kT + v] : Acc<CPLX>::zero();
      Ys[r][v] = (row && jb * kT + v < B) ? Y[(J + r) * ld + jb * kT + v] : Acc<CPLX>::zero();
    }
    __syncthreads();
#pragma unroll 4
    for (int r = 0; r < kRC; ++r) {
      T xa[4], yb[4];
#pragma unroll
      for (int a = 0; a < 4; ++a) { xa[a] = Xs[r][ti * 4 + a]; yb[a] = Ys[r][tj * 4 + a]; }
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) Acc<CPLX>::fma_conj(acc[a][b], xa[a], yb[b]);
    }
  }
  T* out = partial + ((long)blockIdx.y * gridDim.x + blockIdx.x) * kT * kT;
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) out[(ti * 4 + a) * kT + tj * 4 + b] = acc[a][b];
}

// G = sum of the slab partials, slab by slab (fixed order); the upper triangle is the conjugate transpose of the lower one
template <bool CPLX>
__global__ void k_rr_reduce(int ntiles, int nslab, int B, const typename Acc<CPLX>::T* __restrict__ partial,
                            typename Acc<CPLX>::T* __restrict__ G) {
  typedef typename Acc<CPLX>::T T;
  int ib = 0, t = blockIdx.x;
  while (t > ib) { t -= ib + 1; ++ib; }
  const int jb = t;
  for (int e = threadIdx.x; e < kT * kT; e += blockDim.x) {
    const int i = ib * kT + e / kT, j = jb * kT + e % kT;
    if (i >= B || j >= B) continue;
    T s = Acc<CPLX>::zero();
    for (int sl = 0; sl < nslab; ++sl) s = Acc<CPLX>::add(s, partial[((long)sl * ntiles + blockIdx.x) * kT * kT + e]);
    if (ib == jb && j > i) continue;               // diagonal tile: keep its lower part, mirrored below
    if (i == j) s = Acc<CPLX>::real_part(s);         // a Hermitian matrix has a real diagonal (the sum is real only to rounding)
    G[(long)i * B + j] = s;
    if (i != j) G[(long)j * B + i] = Acc<CPLX>::conj(s);
  }
}

// Xout[J][jb kT + j] = sum_i X[J][i] Q[i][jb kT + j]; i-blocks other than jb in FP32 when mixed (products and the sum inside a
// block in FP32, blocks added in FP64).  grid = (ceil(M / 64), ceil(B / kT)), block = 256 = 16 x 16 threads, 4 x 4 each.
template <bool CPLX>
__global__ void __launch_bounds__(256)
k_rr_rotate(long M, int B, int mixed, const typename Acc<CPLX>::T* __restrict__ X, long ldx, const typename Acc<CPLX>::T* __restrict__ Q,
            typename Acc<CPLX>::T* __restrict__ Xout, long ldo) {
  typedef typename Acc<CPLX>::T T;
  constexpr int cw = CPLX ? 2 : 1;
  __shared__ T Xs[64][kRC + 1], Qs[kRC][kT];
  const long J0 = blockIdx.x * 64L;
  const int jb = blockIdx.y;
  const int ti = threadIdx.x >> 4, tj = threadIdx.x & 15;
  T acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = Acc<CPLX>::zero();
  const int nib = (B + kT - 1) / kT;
  for (int ib = 0; ib < nib; ++ib) {
    const bool lowp = mixed && ib != jb;
    float facc[4][4][cw];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = 0; b < 4; ++b)
#pragma unroll
        for (int q = 0; q < cw; ++q) facc[a][b][q] = 0.f;
    for (int i0 = ib * kT; i0 < min(B, (ib + 1) * kT); i0 += kRC) {
      __syncthreads();
      for (int e = threadIdx.x; e < 64 * kRC; e += 256) {
        const int r = e / kRC, k = e % kRC;
        Xs[r][k] = (J0 + r < M && i0 + k < B) ? X[(J0 + r) * ldx + i0 + k] : Acc<CPLX>::zero();
      }
      for (int e = threadIdx.x; e < kRC * kT; e += 256) {
        const int k = e / kT, v = e % kT;
        Qs[k][v] = (i0 + k < B && jb * kT + v < B) ? Q[(long)(i0 + k) * B + jb * kT + v] : Acc<CPLX>::zero();
      }
      __syncthreads();
#pragma unroll 4
      for (int k = 0; k < kRC; ++k) {
        T xa[4], qb[4];
#pragma unroll
        for (int a = 0; a < 4; ++a) { xa[a] = Xs[ti * 4 + a][k]; qb[a] = Qs[k][tj * 4 + a]; }
        if (!lowp) {
#pragma unroll
          for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) Acc<CPLX>::fma_(acc[a][b], xa[a], qb[b]);
        } else {
          const double* xd = reinterpret_cast<const double*>(xa);
          const double* qd = reinterpret_cast<const double*>(qb);
#pragma unroll
          for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
              if constexpr (CPLX) {
                const float xr = (float)xd[2 * a], xi = (float)xd[2 * a + 1], qr = (float)qd[2 * b], qi = (float)qd[2 * b + 1];
                facc[a][b][0] = fmaf(xr, qr, facc[a][b][0]); facc[a][b][0] = fmaf(-xi, qi, facc[a][b][0]);
                facc[a][b][cw - 1] = fmaf(xr, qi, facc[a][b][cw - 1]); facc[a][b][cw - 1] = fmaf(xi, qr, facc[a][b][cw - 1]);
              } else {
                facc[a][b][0] = fmaf((float)xd[a], (float)qd[b], facc[a][b][0]);
              }
            }
        }
      }
    }
    if (lowp) {
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          double* d = reinterpret_cast<double*>(&acc[a][b]);
#pragma unroll
          for (int q = 0; q < cw; ++q) d[q] += (double)facc[a][b][q];
        }
    }
  }
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    const long J = J0 + ti * 4 + a;
    if (J >= M) continue;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int j = jb * kT + tj * 4 + b;
      if (j < B) Xout[J * ldo + j] = acc[a][b];
    }
  }
}

template <bool CPLX>
pawfe_status project_impl(pawfe_ctx* c, const void* X, const void* Y, long ld, int B, void* G) {
  typedef typename Acc<CPLX>::T T;
  const int nb = (B + kT - 1) / kT, ntiles = nb * (nb + 1) / 2;
  const int nslab = (int)std::max<long>(1, std::min<long>((4L * c->sm_count + ntiles - 1) / ntiles, (c->M + 1023) / 1024));
  const long rps = ((c->M + nslab - 1) / nslab + kRC - 1) / kRC * kRC;
  T* partial = nullptr;
  TRY(dev_alloc(c, &partial, (size_t)nslab * ntiles * kT * kT));
  k_rr_project<CPLX><<<dim3(ntiles, nslab), 256, 0, c->stream>>>(c->M, rps, B, (const T*)X, (const T*)Y, ld, partial);
  c->launches++;
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) {
    k_rr_reduce<CPLX><<<ntiles, 256, 0, c->stream>>>(ntiles, nslab, B, partial, (T*)G);
    c->launches++;
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);   // the partials are freed below
  cudaFree(partial);
  if (e != cudaSuccess) { c->err = std::string("pawfe_rr_project: ") + cudaGetErrorString(e); return PAWFE_ECUDA; }
  return PAWFE_OK;
}

}  // namespace

extern "C" pawfe_status pawfe_rr_project(pawfe_ctx* c, const void* X, const void* Y, long ld, int B, void* G) {
  if (!c) return PAWFE_EINVAL;
  if (!X || !Y || !G || B < 1 || B > 8192 || ld < B) { c->err = "bad Rayleigh-Ritz projection arguments"; return PAWFE_EINVAL; }
  if (!c->have_mesh) { c->err = "mesh not created"; return PAWFE_ESTATE; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  return c->cplx ? project_impl<true>(c, X, Y, ld, B, G) : project_impl<false>(c, X, Y, ld, B, G);
}

extern "C" pawfe_status pawfe_rr_rotate(pawfe_ctx* c, int mixed, const void* X, long ldx, const void* Q, void* Xout, long ldo, int B) {
  if (!c) return PAWFE_EINVAL;
  if (!X || !Q || !Xout || X == Xout || B < 1 || B > 8192 || ldx < B || ldo < B) { c->err = "bad subspace rotation arguments"; return PAWFE_EINVAL; }
  if (!c->have_mesh) { c->err = "mesh not created"; return PAWFE_ESTATE; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  const dim3 grid((unsigned)((c->M + 63) / 64), (unsigned)((B + kT - 1) / kT));
  if (c->cplx) k_rr_rotate<true><<<grid, 256, 0, c->stream>>>(c->M, B, mixed, (const double2*)X, ldx, (const double2*)Q, (double2*)Xout, ldo);
  else k_rr_rotate<false><<<grid, 256, 0, c->stream>>>(c->M, B, mixed, (const double*)X, ldx, (const double*)Q, (double*)Xout, ldo);
  KERNEL_CHECK(c, "k_rr_rotate");
  return PAWFE_OK;
}
