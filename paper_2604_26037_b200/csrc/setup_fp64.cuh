// setup_fp64.cuh -- FP64 kernels of the residual set-up of Algorithm 2 ("full precision"):
//     Y = H X - S X Lambda,   S = M + sum_a C^a dS^a C^a^T                     (Eq. 16)
// for real contexts, fused so that S X is never stored:
//   * the H^e X_e part is the DMMA cell product (cell_dmma.cuh);
//   * the mass part  -(M^e X_e) Lambda  uses M^e = (hx hy hz / 8) M1 (x) M1 (x) M1 (Eq. 33) applied as
//     three 1-D sweeps (same matrix, same result up to rounding; 16x fewer flops than the dense n x n product);
//   * the two non-local parts share ONE projection P = C^T X:  Y += C (D P - dS P Lambda).
#pragma once
#include "common.h"

// Y[J][v] += coef[v / cw] * (M^e X_e)[I][v] over all cells (coef = null: +1; cw = 2: interleaved complex columns).
//   grid = (ncell, ceil(W/CT)), block = 256.  dynamic smem: n * CT doubles + n longs.  M1: [n1][n1] doubles (device).
//   CT = 16 columns per CTA: 47 KB of shared memory, so four CTAs per SM overlap their gather / sweep / reduction phases
//   (the kernel is latency-bound: ncu, profiles/r01_ncu_small_kernels.md).
constexpr int kMassCT = 16;
template <typename RX, int CT>
__global__ void __launch_bounds__(256, 4)
k_mass_sf(MeshDev md, const double* __restrict__ M1, double scale, const RX* __restrict__ X, long ldx,
          double* __restrict__ Y, long ldy, int W, const double* __restrict__ coef, int cw = 1) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = md.n, n1 = md.n1, n2 = n1 * n1;
  double* U = reinterpret_cast<double*>(smem_raw);    // [n][CT]
  long* nodeJ = reinterpret_cast<long*>(U + (size_t)n * CT);
  __shared__ double m1s[PAWFE_MAX_N1 * PAWFE_MAX_N1];
  const int v0 = blockIdx.y * CT;
  int cx, cy, cz;
  mesh_cell_coords(md, blockIdx.x, &cx, &cy, &cz);
  for (int I = threadIdx.x; I < n; I += blockDim.x) {
    int c = I % n1, b = (I / n1) % n1, a = I / n2, ix, iy, iz;
    long J = mesh_node(md, cx, cy, cz, a, b, c, &ix, &iy, &iz);
    if (md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz] == 0.0) J = -1;
    nodeJ[I] = J;
  }
  for (int i = threadIdx.x; i < n2; i += blockDim.x) m1s[i] = M1[i];
  __syncthreads();
#pragma unroll 4
  for (int i = threadIdx.x; i < n * CT; i += blockDim.x) {
    const int I = i / CT, col = i % CT;
    const long J = nodeJ[I];
    U[i] = (J >= 0 && v0 + col < W) ? (double)X[J * ldx + v0 + col] : 0.0;
  }
  __syncthreads();
  // three sweeps: direction d has stride n1^(2-d); a work item is one line (n1 values) of one column
  for (int d = 2; d >= 0; --d) {
    const int stride = d == 2 ? 1 : (d == 1 ? n1 : n2);
    for (int i = threadIdx.x; i < n2 * CT; i += blockDim.x) {
      const int col = i % CT, line = i / CT;
      const int q0 = line / n1, q1 = line % n1;   // the two fixed indices
      int base;
      if (d == 2) base = (q0 * n1 + q1) * n1;          // (a, b, .)
      else if (d == 1) base = q0 * n2 + q1;            // (a, ., c)
      else base = q0 * n1 + q1;                        // (., b, c)
      double t[PAWFE_MAX_N1];
#pragma unroll
      for (int k = 0; k < PAWFE_MAX_N1; ++k) t[k] = k < n1 ? U[(base + k * stride) * CT + col] : 0.0;
#pragma unroll
      for (int r = 0; r < PAWFE_MAX_N1; ++r)
        if (r < n1) {
          double s = 0.0;
#pragma unroll
          for (int k = 0; k < PAWFE_MAX_N1; ++k) if (k < n1) s = fma(m1s[r * n1 + k], t[k], s);
          U[(base + r * stride) * CT + col] = s;
        }
    }
    __syncthreads();
  }
  for (int i = threadIdx.x; i < n * CT; i += blockDim.x) {
    const int I = i / CT, col = i % CT;
    const long J = nodeJ[I];
    if (J >= 0 && v0 + col < W) atomicAdd(Y + J * ldy + v0 + col, (coef ? coef[(v0 + col) / cw] : 1.0) * scale * U[i]);
  }
}

// P[a][al][v] += sum_I C^{e,a}[I][al] X[J(e,I)][v] in FP64.  grid = (npairs, ceil(B/64)), block = 256 (8 warps over
// rows, lane = 2 consecutive vectors).  dynamic smem: n longs + NPJ*n doubles + 8 bytes + NPJ*64 doubles.  P zero on entry.
template <int NPJ, typename RX>
__global__ void __launch_bounds__(256)
k_proj64(MeshDev md, const int* __restrict__ pair_cell, const int* __restrict__ pair_atom,
         const double* __restrict__ Cd, const RX* __restrict__ X, long ldx, int B, double* __restrict__ P, long ldp) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = md.n, n1 = md.n1;
  long* nodeJ = reinterpret_cast<long*>(smem_raw);
  double* Cs = reinterpret_cast<double*>(nodeJ + n);   // [NPJ][n]
  double* red = Cs + ((size_t)NPJ * n + ((n + (size_t)NPJ * n) & 1));   // [NPJ][64], 16-byte aligned
  const int pr = blockIdx.x, a = pair_atom[pr];
  int cx, cy, cz;
  mesh_cell_coords(md, pair_cell[pr], &cx, &cy, &cz);
  for (int I = threadIdx.x; I < n; I += blockDim.x) {
    int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1), ix, iy, iz;
    long J = mesh_node(md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
    if (md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz] == 0.0) J = -1;
    nodeJ[I] = J;
  }
  for (int i = threadIdx.x; i < NPJ * n; i += blockDim.x) Cs[i] = Cd[(long)pr * NPJ * n + i];
  for (int i = threadIdx.x; i < NPJ * 64; i += blockDim.x) red[i] = 0.0;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int v = blockIdx.y * 64 + lane * 2;
  double a0[NPJ], a1[NPJ];
#pragma unroll
  for (int al = 0; al < NPJ; ++al) a0[al] = a1[al] = 0.0;
  if (v < B) {
    const bool two = v + 1 < B;
    for (int I0 = w; I0 < n; I0 += 32) {
      double x0[4], x1[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int I = I0 + 8 * u;
        const long J = I < n ? nodeJ[I] : -1;
        x0[u] = J >= 0 ? (double)X[J * ldx + v] : 0.0;
        x1[u] = (J >= 0 && two) ? (double)X[J * ldx + v + 1] : 0.0;
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int I = min(I0 + 8 * u, n - 1);
#pragma unroll
        for (int al = 0; al < NPJ; ++al) {
          const double cv = Cs[al * n + I];
          a0[al] = fma(cv, x0[u], a0[al]); a1[al] = fma(cv, x1[u], a1[al]);
        }
      }
    }
  }
  // cross-warp sum in shared memory, one warp per round (fixed order; shared-memory FP64 atomics are CAS loops)
  for (int r = 0; r < 8; ++r) {
    if (w == r && v < B) {
#pragma unroll
      for (int al = 0; al < NPJ; ++al) {
        double2* q = reinterpret_cast<double2*>(red + al * 64 + lane * 2);
        double2 t = *q;
        t.x += a0[al]; t.y += a1[al];
        *q = t;
      }
    }
    __syncthreads();
  }
  for (int i = threadIdx.x; i < NPJ * 64; i += blockDim.x) {
    const int al = i >> 6, vv = blockIdx.y * 64 + (i & 63);
    if (vv < B) atomicAdd(P + ((long)a * NPJ + al) * ldp + vv, red[i]);
  }
}

// W[a][al][v] = sum_be (D^a[al][be] - lam[v] dS^a[al][be]) P[a][be][v].  grid = (natoms, ceil(B/128)), block = 128.
static __global__ void k_couple64(int npj, const double* __restrict__ P, long ldp, int B, const double* __restrict__ D,
                                  const double* __restrict__ dS, const double* __restrict__ lam, double* __restrict__ Wd) {
  const int a = blockIdx.x, v = blockIdx.y * blockDim.x + threadIdx.x;
  if (v >= B) return;
  double p[PAWFE_MAX_NPJ];
#pragma unroll
  for (int be = 0; be < PAWFE_MAX_NPJ; ++be) p[be] = be < npj ? P[((long)a * npj + be) * ldp + v] : 0.0;
  const double l = lam[v];
  for (int al = 0; al < npj; ++al) {
    double s = 0.0;
#pragma unroll
    for (int be = 0; be < PAWFE_MAX_NPJ; ++be)
      if (be < npj) s = fma(D[((long)a * npj + al) * npj + be] - l * dS[((long)a * npj + al) * npj + be], p[be], s);
    Wd[((long)a * npj + al) * ldp + v] = s;
  }
}

// Y[J][v] += sum_al C^{e,a}[I][al] W[a][al][v] in FP64.  grid = (npairs, ceil(B/64)), block = 256.
//   dynamic smem: n longs + NPJ*n doubles.
template <int NPJ>
__global__ void __launch_bounds__(256)
k_scatter64(MeshDev md, const int* __restrict__ pair_cell, const int* __restrict__ pair_atom,
            const double* __restrict__ Cd, const double* __restrict__ Wd, long ldp, int B, double* __restrict__ Y, long ldy) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = md.n, n1 = md.n1;
  long* nodeJ = reinterpret_cast<long*>(smem_raw);
  double* Cs = reinterpret_cast<double*>(nodeJ + n);
  const int pr = blockIdx.x, a = pair_atom[pr];
  int cx, cy, cz;
  mesh_cell_coords(md, pair_cell[pr], &cx, &cy, &cz);
  for (int I = threadIdx.x; I < n; I += blockDim.x) {
    int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1), ix, iy, iz;
    long J = mesh_node(md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
    if (md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz] == 0.0) J = -1;
    nodeJ[I] = J;
  }
  for (int i = threadIdx.x; i < NPJ * n; i += blockDim.x) Cs[i] = Cd[(long)pr * NPJ * n + i];
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int v = blockIdx.y * 64 + lane * 2;
  if (v >= B) return;
  const bool two = v + 1 < B;
  double w0[NPJ], w1[NPJ];
#pragma unroll
  for (int al = 0; al < NPJ; ++al) {
    w0[al] = Wd[((long)a * NPJ + al) * ldp + v];
    w1[al] = two ? Wd[((long)a * NPJ + al) * ldp + v + 1] : 0.0;
  }
  for (int I = w; I < n; I += 8) {
    const long J = nodeJ[I];
    if (J < 0) continue;
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int al = 0; al < NPJ; ++al) { const double cv = Cs[al * n + I]; s0 = fma(cv, w0[al], s0); s1 = fma(cv, w1[al], s1); }
    atomicAdd(Y + J * ldy + v, s0);
    if (two) atomicAdd(Y + J * ldy + v + 1, s1);
  }
}

// Alg. 2 steps 2-3 (L260-L264) in the scaled variables:  Yt = M_D^-1 Y (FP64, in place);  Rt_Y = (zeta/e) Yt;  Rt_X = 0.
// 4 consecutive columns per thread (ldw % 4 == 0, arrays 16-byte aligned); pad columns are written as 0.
static __global__ void __launch_bounds__(256)
k_residual_init3(MeshDev md, long ldw, int B, double* __restrict__ Y, double z_over_e,
                 float* __restrict__ RX, float* __restrict__ RY) {
  const int ldq = (int)(ldw / 4);
  const long nquads = md.M * ldq;
  const int N1 = md.N[1], N2 = md.N[2];
  double2* Y2 = reinterpret_cast<double2*>(Y);
  for (long q = blockIdx.x * (long)blockDim.x + threadIdx.x; q < nquads; q += (long)gridDim.x * blockDim.x) {
    const int J = (int)(q / ldq);
    const int v = (int)(q - (long)J * ldq) * 4;
    const int iz = J % N2, t = J / N2;
    const double s = md.mdinv1[0][t / N1] * md.mdinv1[1][t % N1] * md.mdinv1[2][iz];
    double2 y0 = Y2[2 * q], y1 = Y2[2 * q + 1];
    y0.x = v < B ? s * y0.x : 0.0;
    y0.y = v + 1 < B ? s * y0.y : 0.0;
    y1.x = v + 2 < B ? s * y1.x : 0.0;
    y1.y = v + 3 < B ? s * y1.y : 0.0;
    Y2[2 * q] = y0;
    Y2[2 * q + 1] = y1;
    reinterpret_cast<float4*>(RY)[q] = make_float4((float)(z_over_e * y0.x), (float)(z_over_e * y0.y),
                                                   (float)(z_over_e * y1.x), (float)(z_over_e * y1.y));
    reinterpret_cast<float4*>(RX)[q] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
}

// Alg. 2 step 2 (L260) from products the caller already holds (pawfe_cheb_filter_hs: H Psi and S Psi of the last
// Rayleigh-Ritz, rotated with the Ritz vectors, L402-L408):  Y = HX - SX Lambda, FP64.  HX, SX: [dof][ldx] doubles (complex:
// interleaved, cw = 2 reals per vector); Y: [dof][ldw]; columns >= W of Y are left to k_residual_init3 (written as 0 there).
static __global__ void __launch_bounds__(256)
k_residual_from_products(long M, long ldw, int W, int cw, const double* __restrict__ HX, const double* __restrict__ SX,
                         long ldx, const double* __restrict__ lam, double* __restrict__ Y) {
  const long total = M * (long)W;
  for (long idx = blockIdx.x * (long)blockDim.x + threadIdx.x; idx < total; idx += (long)gridDim.x * blockDim.x) {
    const long J = idx / W;
    const int v = (int)(idx - J * W);
    Y[J * ldw + v] = HX[J * ldx + v] - SX[J * ldx + v] * lam[v / cw];
  }
}
