// kernels_stream.cuh -- bandwidth-bound kernels of Algorithm 2: residual set-up,
// the three-term recurrence with the FP64 residual-source add (L374), recovery, column norms, and the
// diagonal part of S^-1approx (M_D^-1, L228).  A complex block is treated as a real block with
// cw = 2 reals per element; all coefficients are real.
#pragma once
#include "common.h"

__device__ inline double mdinv_of_row(const MeshDev& md, long J) {
  int iz = (int)(J % md.N[2]);
  long t = J / md.N[2];
  int iy = (int)(t % md.N[1]);
  int ix = (int)(t / md.N[1]);
  return md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz];
}

// Y = M_D^-1 X  (rows), W = B*cw reals per row
template <typename TX, typename TY>
__global__ void k_scale_mdinv(MeshDev md, const TX* __restrict__ X, long ldx, TY* __restrict__ Y,
                              long ldy, int W) {
  long total = md.M * (long)W;
  for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total;
       idx += (long)gridDim.x * blockDim.x) {
    long J = idx / W; int c = (int)(idx % W);
    double s = mdinv_of_row(md, J);
    Y[J * ldy + c] = (TY)((double)X[J * ldx + c] * s);
  }
}

// Y *= M_D^-1 in place
template <typename TY>
__global__ void k_scale_mdinv_inplace(MeshDev md, TY* __restrict__ Y, long ldy, int W) {
  long total = md.M * (long)W;
  for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total;
       idx += (long)gridDim.x * blockDim.x) {
    long J = idx / W; int c = (int)(idx % W);
    double s = mdinv_of_row(md, J);
    Y[J * ldy + c] = (TY)((double)Y[J * ldy + c] * s);
  }
}

// Alg. 2 steps 2-3 (L260-L264):  Y <- HX - SX Lambda (in place in HX, FP64);  R_Y = (zeta/e) Y;  R_X = 0.
//   lam: [B] doubles (device).  HX, SX: FP64 blocks with leading dimension W.  RX, RY storage TS.
template <typename TS>
__global__ void k_residual_init(long M, int W, int cw, double* __restrict__ HX,
                                const double* __restrict__ SX, const double* __restrict__ lam,
                                double z_over_e, TS* __restrict__ RX, TS* __restrict__ RY) {
  long total = M * (long)W;
  for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total;
       idx += (long)gridDim.x * blockDim.x) {
    int c = (int)(idx % W);
    double y = SX ? HX[idx] - SX[idx] * lam[c / cw] : HX[idx];
    HX[idx] = y;
    RY[idx] = (TS)(z_over_e * y);
    RX[idx] = (TS)0;
  }
}

// Alg. 2 step 4 (L272):  R_X <- a HT - a c R_Y - zeta zeta1 R_X  [TS arithmetic]  + a Y LamY [FP64 add]
//   aLamY: [B] doubles = a * Lambda_Y (device).
template <typename TS>
__global__ void k_recurrence(long total, int W, int cw, const TS* __restrict__ HT,
                             const TS* __restrict__ RY, TS* __restrict__ RX,
                             const double* __restrict__ Y, const double* __restrict__ aLamY,
                             double a, double ac, double zz1) {
  for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total;
       idx += (long)gridDim.x * blockDim.x) {
    int c = (int)(idx % W);
    TS br = (TS)a * HT[idx] - (TS)ac * RY[idx] - (TS)zz1 * RX[idx];
    RX[idx] = (TS)((double)br + Y[idx] * aLamY[c / cw]);
  }
}

// Alg. 2 step 5 (L282):  X <- T + X LamY  with T = S^-1approx R_Y (leading dimension W), X leading dim ldx
template <typename TS>
__global__ void k_recover(MeshDev md, int W, int cw, const TS* __restrict__ T, TS* __restrict__ X, long ldx,
                          const double* __restrict__ lamY) {
  long total = md.M * (long)W;
  for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total;
       idx += (long)gridDim.x * blockDim.x) {
    long J = idx / W; int c = (int)(idx % W);
    double x = (double)X[J * ldx + c];
    double keep = mdinv_of_row(md, J) != 0.0 ? 1.0 : 0.0;  // Dirichlet boundary rows are written as 0
    X[J * ldx + c] = (TS)(keep * ((double)T[idx] + x * lamY[c / cw]));
  }
}

// out[v] += sum_J |X[J][v]|^2 over a slab of rows; host takes the square root afterwards.
//   grid = (ceil(B/32), nslabs), block = (32, 8).  FP64 accumulation (L290).
template <typename TS>
__global__ void k_col_sumsq(long M, int B, int cw, const TS* __restrict__ X, long ldx,
                            double* __restrict__ out) {
  __shared__ double red[8][33];
  int v = blockIdx.x * 32 + threadIdx.x;
  double acc = 0.0;
  if (v < B) {
    for (long J = blockIdx.y * (long)blockDim.y + threadIdx.y; J < M; J += (long)gridDim.y * blockDim.y) {
      for (int q = 0; q < cw; ++q) {
        double x = (double)X[(J * ldx + v) * cw + q];
        acc += x * x;
      }
    }
  }
  red[threadIdx.y][threadIdx.x] = acc;
  __syncthreads();
  if (threadIdx.y == 0 && v < B) {
    double s = 0.0;
    for (int i = 0; i < 8; ++i) s += red[i][threadIdx.x];
    atomicAdd(&out[v], s);
  }
}

static __global__ void k_sqrt_inplace(double* x, int n) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) x[i] = sqrt(x[i]);
}

// ---- float4-vectorised variants for FP32 storage (W % 4 == 0, 16-byte aligned rows); one row factor per thread row ----
// Y = M_D^-1 X, 4 consecutive columns per thread.  Wq = W / 4; ldxq, ldyq = leading dimensions / 4.
static __global__ void __launch_bounds__(256)
k_scale_mdinv_f4(MeshDev md, const float4* __restrict__ X, long ldxq, float4* __restrict__ Y, long ldyq, int Wq) {
  const long total = md.M * (long)Wq;
  for (long q = blockIdx.x * (long)blockDim.x + threadIdx.x; q < total; q += (long)gridDim.x * blockDim.x) {
    const long J = q / Wq;
    const int c = (int)(q - J * Wq);
    const float s = (float)mdinv_of_row(md, J);
    const float4 x = X[J * ldxq + c];
    Y[J * ldyq + c] = make_float4(x.x * s, x.y * s, x.z * s, x.w * s);
  }
}

// Alg. 2 step 4 (L272) for FP32 storage, 4 consecutive real columns per thread (all blocks have leading dimension W):
//   R_X <- a HT - a c R_Y - zeta zeta1 R_X  [FP32]  + a Y LamY [FP64 add]
static __global__ void __launch_bounds__(256)
k_recurrence_f4(long nquads, int Wq, int cw, const float4* __restrict__ HT, const float4* __restrict__ RY,
                float4* __restrict__ RX, const double2* __restrict__ Y, const double* __restrict__ aLamY, float a,
                float ac, float zz1) {
  for (long q = blockIdx.x * (long)blockDim.x + threadIdx.x; q < nquads; q += (long)gridDim.x * blockDim.x) {
    const int c0 = (int)(q % Wq) * 4;
    const float4 h = HT[q], ry = RY[q], rx = RX[q];
    const double2 y0 = Y[2 * q], y1 = Y[2 * q + 1];
    const double l0 = aLamY[c0 / cw], l1 = aLamY[(c0 + 1) / cw], l2 = aLamY[(c0 + 2) / cw], l3 = aLamY[(c0 + 3) / cw];
    float4 o;
    o.x = (float)((double)(a * h.x - ac * ry.x - zz1 * rx.x) + y0.x * l0);
    o.y = (float)((double)(a * h.y - ac * ry.y - zz1 * rx.y) + y0.y * l1);
    o.z = (float)((double)(a * h.z - ac * ry.z - zz1 * rx.z) + y1.x * l2);
    o.w = (float)((double)(a * h.w - ac * ry.w - zz1 * rx.w) + y1.y * l3);
    RX[q] = o;
  }
}
