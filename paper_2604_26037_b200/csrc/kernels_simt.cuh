// kernels_simt.cuh -- generic (any scalar type) kernels of the operator action A X of PAPER.md section 4.3
// (L337-L347, Fig. 2): (i) extraction, (ii) partial non-local projection, (iii) cell-level product,
// (iv) assembly.  These are the FP64 reference-mode and FP32 kernels; the TF32 cell contraction on
// tcgen05 tensor cores lives in cell_tcgen05.cu.
#pragma once
#include "common.h"

// ------------------------------------------------------------------------------------------------
// cell-level product: Y += alpha * sum_e P_e^T A^e (s o P_e X)   (steps i, iii, iv)
//   Amat: [cell][n][lda] (cell_stride = n*lda) or one shared reference matrix (cell_stride = 0)
//   in_scale: 0 = none, 1 = M_D^-1 on the gathered rows.  Dirichlet boundary rows are gathered as 0
//   and never written.  Y must have been initialised by the caller (assembly is by atomic adds).
//   grid = (ncell, ceil(B / BV)), block = 256.
// ------------------------------------------------------------------------------------------------
template <typename TX, typename TY, typename TC, int BV, bool TF32>
__global__ void __launch_bounds__(256)
k_cell_simt(MeshDev md, const TC* __restrict__ Amat, long cell_stride, int lda,
            const TX* __restrict__ X, long ldx, TY* __restrict__ Y, long ldy, int B,
            int in_scale, double alpha) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = md.n, n1 = md.n1;
  long* nodeJ = reinterpret_cast<long*>(smem_raw);                   // [n]
  double* nodeS = reinterpret_cast<double*>(nodeJ + n);              // [n]  M_D^-1 (0 = masked)
  TC* Xs = reinterpret_cast<TC*>(nodeS + n);                         // [n][BV]
  const int e = blockIdx.x;
  const int v0 = blockIdx.y * BV;
  int cx, cy, cz;
  mesh_cell_coords(md, e, &cx, &cy, &cz);
  for (int I = threadIdx.x; I < n; I += blockDim.x) {
    int c = I % n1, b = (I / n1) % n1, a = I / (n1 * n1);
    int ix, iy, iz;
    nodeJ[I] = mesh_node(md, cx, cy, cz, a, b, c, &ix, &iy, &iz);
    nodeS[I] = md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz];
  }
  __syncthreads();
  const int tx = threadIdx.x % BV, ty = threadIdx.x / BV;
  constexpr int ROWG = 256 / BV;
  const int v = v0 + tx;
  for (int I = ty; I < n; I += ROWG) {
    TC x = s_zero(TC());
    double s = nodeS[I];
    if (v < B && s != 0.0) {
      s_cvt(x, X[nodeJ[I] * ldx + v]);
      if (in_scale) x = s_scale(x, s);
    }
    if (TF32) {
      float* xf = reinterpret_cast<float*>(&x);
      for (int q = 0; q < (int)(sizeof(TC) / sizeof(float)); ++q) xf[q] = tf32_round(xf[q]);
    }
    Xs[I * BV + tx] = x;
  }
  __syncthreads();
  const TC* A = Amat + (long)e * cell_stride;
  constexpr int RT = 4;
  for (int i0 = 0; i0 < n; i0 += ROWG * RT) {
    TC acc[RT];
    const TC* Ar[RT];
#pragma unroll
    for (int r = 0; r < RT; ++r) {
      acc[r] = s_zero(TC());
      int i = i0 + ty + ROWG * r;
      Ar[r] = A + (long)(i < n ? i : 0) * lda;
    }
    for (int k = 0; k < n; ++k) {
      TC x = Xs[k * BV + tx];
#pragma unroll
      for (int r = 0; r < RT; ++r) {
        TC hv = Ar[r][k];
        if (TF32) {
          float* hf = reinterpret_cast<float*>(&hv);
          for (int q = 0; q < (int)(sizeof(TC) / sizeof(float)); ++q) hf[q] = tf32_round(hf[q]);
        }
        s_fma(acc[r], hv, x);
      }
    }
#pragma unroll
    for (int r = 0; r < RT; ++r) {
      int i = i0 + ty + ROWG * r;
      if (i < n && v < B && nodeS[i] != 0.0) {
        TY out;
        s_cvt(out, s_scale(acc[r], alpha));
        s_atomic_add(&Y[nodeJ[i] * ldy + v], out);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// (ii) partial non-local projection  P^a = sum_e C^{e,a dagger} (s o X_e)   (L345; Eq. 34)
//   Cd: [pair][npj][n] rows of C^{e,a dagger}; pairs of atom a are [aps[a], aps[a+1]).
//   P: [atom][npj][ldp].  in_scale: 0 none, 1 M_D^-1.  grid = (natoms_in_range, ceil(B/32)), block 128.
// ------------------------------------------------------------------------------------------------
template <typename TX, typename TC>
__global__ void __launch_bounds__(128)
k_proj(MeshDev md, int atom0, const int* __restrict__ aps, const int* __restrict__ pair_cell,
       const TC* __restrict__ Cd, int npj, const TX* __restrict__ X, long ldx, int B, int in_scale,
       TC* __restrict__ P, int ldp) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n = md.n, n1 = md.n1;
  long* nodeJ = reinterpret_cast<long*>(smem_raw);
  double* nodeS = reinterpret_cast<double*>(nodeJ + n);
  TC* red = reinterpret_cast<TC*>(nodeS + n);  // [4][PAWFE_MAX_NPJ][32]
  const int a = atom0 + blockIdx.x;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int v = blockIdx.y * 32 + lane;
  TC acc[PAWFE_MAX_NPJ];
#pragma unroll
  for (int al = 0; al < PAWFE_MAX_NPJ; ++al) acc[al] = s_zero(TC());
  for (int pr = aps[a]; pr < aps[a + 1]; ++pr) {
    int cx, cy, cz;
    mesh_cell_coords(md, pair_cell[pr], &cx, &cy, &cz);
    __syncthreads();
    for (int I = threadIdx.x; I < n; I += blockDim.x) {
      int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1);
      int ix, iy, iz;
      nodeJ[I] = mesh_node(md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
      nodeS[I] = md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz];
    }
    __syncthreads();
    const TC* Cp = Cd + (long)pr * npj * n;
    for (int I = w; I < n; I += 4) {
      double s = nodeS[I];
      if (s == 0.0 || v >= B) continue;
      TC x;
      s_cvt(x, X[nodeJ[I] * ldx + v]);
      if (in_scale) x = s_scale(x, s);
#pragma unroll
      for (int al = 0; al < PAWFE_MAX_NPJ; ++al)
        if (al < npj) s_fma(acc[al], Cp[(long)al * n + I], x);
    }
  }
  __syncthreads();
#pragma unroll
  for (int al = 0; al < PAWFE_MAX_NPJ; ++al)
    if (al < npj) red[(w * PAWFE_MAX_NPJ + al) * 32 + lane] = acc[al];
  __syncthreads();
  for (int al = w; al < npj; al += 4) {
    TC s = red[(0 * PAWFE_MAX_NPJ + al) * 32 + lane];
    for (int ww = 1; ww < 4; ++ww) s = s_add(s, red[(ww * PAWFE_MAX_NPJ + al) * 32 + lane]);
    if (v < B) P[((long)a * npj + al) * ldp + v] = s;
  }
}

// W^a = scale * Delta^a P^a  (npj x npj times npj x B).  grid = (natoms, ceil(B/128)), block 128.
// colscale (optional, device, [B] doubles): extra real factor per vector, e.g. the Ritz values Lambda.
template <typename TC>
__global__ void k_coupling(const TC* __restrict__ Delta, int npj, const TC* __restrict__ P, int ldp,
                           int B, double scale, TC* __restrict__ W, const double* __restrict__ colscale = nullptr) {
  const int a = blockIdx.x;
  const int v = blockIdx.y * blockDim.x + threadIdx.x;
  if (v >= B) return;
  TC p[PAWFE_MAX_NPJ];
#pragma unroll
  for (int be = 0; be < PAWFE_MAX_NPJ; ++be)
    if (be < npj) p[be] = P[((long)a * npj + be) * ldp + v];
  for (int al = 0; al < npj; ++al) {
    TC s = s_zero(TC());
#pragma unroll
    for (int be = 0; be < PAWFE_MAX_NPJ; ++be)
      if (be < npj) s_fma(s, Delta[((long)a * npj + al) * npj + be], p[be]);
    W[((long)a * npj + al) * ldp + v] = s_scale(s, colscale ? scale * colscale[v] : scale);
  }
}

// Y += out_scale_J * sum_alpha conj(Cd[pair][alpha][I]) W^a[alpha]   (remaining non-local part, L347)
//   out_scale: 0 none, 1 M_D^-1.  grid = (npairs_in_range, ceil(B/32)), block 128.
template <typename TY, typename TC>
__global__ void __launch_bounds__(128)
k_nl_scatter(MeshDev md, int pair0, const int* __restrict__ pair_cell, const int* __restrict__ pair_atom,
             const TC* __restrict__ Cd, int npj, const TC* __restrict__ W, int ldp, int B,
             int out_scale, TY* __restrict__ Y, long ldy) {
  const int n = md.n, n1 = md.n1;
  const int pr = pair0 + blockIdx.x;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int v = blockIdx.y * 32 + lane;
  if (v >= B) return;
  const int a = pair_atom[pr];
  int cx, cy, cz;
  mesh_cell_coords(md, pair_cell[pr], &cx, &cy, &cz);
  TC wv[PAWFE_MAX_NPJ];
#pragma unroll
  for (int al = 0; al < PAWFE_MAX_NPJ; ++al)
    if (al < npj) wv[al] = W[((long)a * npj + al) * ldp + v];
  const TC* Cp = Cd + (long)pr * npj * n;
  for (int I = w; I < n; I += 4) {
    int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1);
    int ix, iy, iz;
    long J = mesh_node(md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
    double s = md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz];
    if (s == 0.0) continue;
    TC acc = s_zero(TC());
#pragma unroll
    for (int al = 0; al < PAWFE_MAX_NPJ; ++al)
      if (al < npj) s_fma_conj(acc, Cp[(long)al * n + I], wv[al]);
    if (out_scale) acc = s_scale(acc, s);
    TY out;
    s_cvt(out, acc);
    s_atomic_add(&Y[J * ldy + v], out);
  }
}
