// fe_setup.cuh -- device kernels that BUILD the operators (not on the hot path; "<1% of SCF time",
// PAPER.md:L321): local potential at quadrature points, cell matrices H^e (Eq. 13 / Eq. 32,
// L311), and cell-level projector blocks C^{e,a dagger} (Eq. 34).  All FP64, sum-factorised over
// the tensor-product basis so that the cost per cell is O(n^2 n_q) instead of O(n^2 n_q^3).
#pragma once
#include "common.h"

struct SetupGeom {
  double h[3], box[3];
  int periodic;
};

// WV[cell][q] = w_qx w_qy w_qz detJ V(x_q),  V(x) = - sum_a sum_images Z_a exp(-|x-R_a-L|^2 / 2 sigma_a^2)
//   xq, wq: [nq] Gauss-Legendre rule on [-1,1].  grid = ncell, block = 256.
static __global__ void k_potential_wv(MeshDev md, SetupGeom g, int nq, const double* __restrict__ xq,
                               const double* __restrict__ wq, int natoms, const double* __restrict__ pos,
                               const double* __restrict__ Z, const double* __restrict__ sig,
                               double* __restrict__ WV) {
  const int e = blockIdx.x;
  int cx, cy, cz;
  mesh_cell_coords(md, e, &cx, &cy, &cz);
  const double detJ = g.h[0] * g.h[1] * g.h[2] / 8.0;
  const int nq3 = nq * nq * nq;
  const int nimg = g.periodic ? 1 : 0;
  for (int q = threadIdx.x; q < nq3; q += blockDim.x) {
    int qz = q % nq, qy = (q / nq) % nq, qx = q / (nq * nq);
    double x = g.h[0] * (cx + 0.5 * (xq[qx] + 1.0));
    double y = g.h[1] * (cy + 0.5 * (xq[qy] + 1.0));
    double z = g.h[2] * (cz + 0.5 * (xq[qz] + 1.0));
    double V = 0.0;
    for (int a = 0; a < natoms; ++a) {
      double inv2s2 = 1.0 / (2.0 * sig[a] * sig[a]);
      for (int sx = -nimg; sx <= nimg; ++sx)
        for (int sy = -nimg; sy <= nimg; ++sy)
          for (int sz = -nimg; sz <= nimg; ++sz) {
            double dx = x - (pos[3 * a + 0] + sx * g.box[0]);
            double dy = y - (pos[3 * a + 1] + sy * g.box[1]);
            double dz = z - (pos[3 * a + 2] + sz * g.box[2]);
            V -= Z[a] * exp(-(dx * dx + dy * dy + dz * dz) * inv2s2);
          }
    }
    WV[(long)e * nq3 + q] = wq[qx] * wq[qy] * wq[qz] * detJ * V;
  }
}

// H^e_IJ = Kre_IJ + i Kim_IJ + sum_q N_I(x_q) N_J(x_q) WV_q,   N_I = l_a(qx) l_b(qy) l_c(qz).
//   Lq: [n1][nq] basis values at the 1-D quadrature points.  Kre = 1/2 K^e + 1/2|k|^2 M^e, Kim = -sum k_d G_d^e.
//   scratch: [gridDim.x][nq * n1^4] doubles.  Outputs: H64 [cell][n][n] (may be null), H32 [cell][n][ldk].
//   dynamic smem: (n1*n1*nq + nq^3 + nq*nq*n1*n1) doubles.  grid-stride over cells, block = 256.
template <bool CPLX>
__global__ void __launch_bounds__(256)
k_build_hcell(MeshDev md, int nq, const double* __restrict__ Lq, const double* __restrict__ WV,
              const double* __restrict__ Kre, const double* __restrict__ Kim,
              double* __restrict__ scratch, double* __restrict__ H64, float* __restrict__ H32, int ldk) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n1 = md.n1, n = md.n;
  const int n2 = n1 * n1;
  double* LL = reinterpret_cast<double*>(smem_raw);  // [n1][n1][nq]
  double* WVs = LL + n2 * nq;                        // [nq^3]
  double* T1 = WVs + nq * nq * nq;                   // [nq][nq][n1][n1]
  double* T2 = scratch + (long)blockIdx.x * nq * n2 * n2;  // [nq][b][b'][c][c']
  for (int i = threadIdx.x; i < n2 * nq; i += blockDim.x) {
    int q = i % nq, c2 = (i / nq) % n1, c = i / (nq * n1);
    LL[i] = Lq[c * nq + q] * Lq[c2 * nq + q];
  }
  const int cw = CPLX ? 2 : 1;
  for (int e = blockIdx.x; e < md.ncell; e += gridDim.x) {
    __syncthreads();
    for (int q = threadIdx.x; q < nq * nq * nq; q += blockDim.x) WVs[q] = WV[(long)e * nq * nq * nq + q];
    __syncthreads();
    // stage 1: contract qz
    for (int i = threadIdx.x; i < nq * nq * n2; i += blockDim.x) {
      int cc = i % n2, qxy = i / n2;
      double s = 0.0;
      for (int qz = 0; qz < nq; ++qz) s += LL[cc * nq + qz] * WVs[qxy * nq + qz];
      T1[i] = s;
    }
    __syncthreads();
    // stage 2: contract qy -> T2[qx][bb'][cc']
    for (int i = threadIdx.x; i < nq * n2 * n2; i += blockDim.x) {
      int cc = i % n2, bb = (i / n2) % n2, qx = i / (n2 * n2);
      double s = 0.0;
      for (int qy = 0; qy < nq; ++qy) s += LL[bb * nq + qy] * T1[(qx * nq + qy) * n2 + cc];
      T2[i] = s;
    }
    __syncthreads();
    // stage 3: contract qx, add the kinetic / k-dependent reference matrices, store
    for (long idx = threadIdx.x; idx < (long)n * n; idx += blockDim.x) {
      int J = (int)(idx % n), I = (int)(idx / n);
      int c = I % n1, b = (I / n1) % n1, a = I / n2;
      int c2 = J % n1, b2 = (J / n1) % n1, a2 = J / n2;
      double s = 0.0;
      const double* t2 = T2 + ((long)(b * n1 + b2)) * n2 + (c * n1 + c2);
      const double* ll = LL + (a * n1 + a2) * nq;
      for (int qx = 0; qx < nq; ++qx) s += ll[qx] * t2[(long)qx * n2 * n2];
      double re = s + Kre[idx];
      double im = CPLX ? Kim[idx] : 0.0;
      if (H64) {
        H64[((long)e * n * n + idx) * cw] = re;
        if (CPLX) H64[((long)e * n * n + idx) * cw + 1] = im;
      }
      long o = ((long)e * n + I) * ldk + J;
      H32[o * cw] = (float)re;
      if (CPLX) H32[o * cw + 1] = (float)im;
    }
  }
}

// real orthonormal solid harmonics r^l Y_lm(d), l <= 2 (the textbook real Y_lm; m = -l..l)
__device__ inline double solid_harmonic_dev(int l, int m, double x, double y, double z) {
  const double pi = 3.14159265358979323846;
  if (l == 0) return 0.5 / sqrt(pi);
  if (l == 1) {
    double c = sqrt(3.0 / (4.0 * pi));
    return c * (m == -1 ? y : (m == 0 ? z : x));
  }
  double c = sqrt(15.0 / (4.0 * pi));
  switch (m) {
    case -2: return c * x * y;
    case -1: return c * y * z;
    case 0:  return sqrt(5.0 / (16.0 * pi)) * (3.0 * z * z - (x * x + y * y + z * z));
    case 1:  return c * x * z;
    default: return 0.5 * c * (x * x - y * y);
  }
}

struct ProjTable {
  int npj;
  int l[PAWFE_MAX_NPJ], m[PAWFE_MAX_NPJ];
  double sigma[PAWFE_MAX_NPJ], amp[PAWFE_MAX_NPJ];
  double rc;
  double kpt[3];
};

// (C^{e,a dagger})_{alpha I} = sum_q w_q detJ e^{i k.(R_a + d_q)} N_I(x_q) p_alpha(d_q),  d_q = minimum image of
// x_q - R_a (periodic) -- Eq. 34 (L318) on an nq^3 Gauss-Legendre grid.  One CTA per (cell, atom) pair.
//   Lq: [n1][nq].  Output Cd64 [pair][npj][n] (complex interleaved if CPLX).
//   dynamic smem: cw * (nq^3 + nq*nq*n1 + nq*n1*n1) doubles.
template <bool CPLX>
__global__ void __launch_bounds__(256)
k_build_proj(MeshDev md, SetupGeom g, int nq, const double* __restrict__ xq, const double* __restrict__ wq,
             const double* __restrict__ Lq, ProjTable pt, const double* __restrict__ pos,
             const int* __restrict__ pair_cell, const int* __restrict__ pair_atom,
             double* __restrict__ Cd64) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int cw = CPLX ? 2 : 1;
  const int n1 = md.n1, n = md.n;
  double* F = reinterpret_cast<double*>(smem_raw);   // [nq^3][cw]
  double* A1 = F + (long)nq * nq * nq * cw;           // [qx][qy][c][cw]
  double* A2 = A1 + (long)nq * nq * n1 * cw;          // [qx][b][c][cw]
  const int pr = blockIdx.x;
  const int e = pair_cell[pr], at = pair_atom[pr];
  int cx, cy, cz;
  mesh_cell_coords(md, e, &cx, &cy, &cz);
  const double detJ = g.h[0] * g.h[1] * g.h[2] / 8.0;
  const double R[3] = {pos[3 * at], pos[3 * at + 1], pos[3 * at + 2]};
  const int nq3 = nq * nq * nq;
  for (int al = 0; al < pt.npj; ++al) {
    __syncthreads();
    const double inv2s2 = 1.0 / (2.0 * pt.sigma[al] * pt.sigma[al]);
    for (int q = threadIdx.x; q < nq3; q += blockDim.x) {
      int qz = q % nq, qy = (q / nq) % nq, qx = q / (nq * nq);
      double d[3];
      d[0] = g.h[0] * (cx + 0.5 * (xq[qx] + 1.0)) - R[0];
      d[1] = g.h[1] * (cy + 0.5 * (xq[qy] + 1.0)) - R[1];
      d[2] = g.h[2] * (cz + 0.5 * (xq[qz] + 1.0)) - R[2];
      if (g.periodic)
        for (int k = 0; k < 3; ++k) d[k] -= g.box[k] * rint(d[k] / g.box[k]);
      double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
      double val = 0.0;
      if (r2 < pt.rc * pt.rc) {
        double cut = 1.0 - r2 / (pt.rc * pt.rc);
        val = pt.amp[al] * exp(-r2 * inv2s2) * cut * cut *
              solid_harmonic_dev(pt.l[al], pt.m[al], d[0], d[1], d[2]) * wq[qx] * wq[qy] * wq[qz] * detJ;
      }
      if (CPLX) {
        double ph = (R[0] + d[0]) * pt.kpt[0] + (R[1] + d[1]) * pt.kpt[1] + (R[2] + d[2]) * pt.kpt[2];
        double sn, cs;
        sincos(ph, &sn, &cs);
        F[2 * q] = val * cs; F[2 * q + 1] = val * sn;
      } else {
        F[q] = val;
      }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nq * nq * n1; i += blockDim.x) {   // contract qz
      int c = i % n1, qxy = i / n1;
      for (int w = 0; w < cw; ++w) {
        double s = 0.0;
        for (int qz = 0; qz < nq; ++qz) s += Lq[c * nq + qz] * F[(qxy * nq + qz) * cw + w];
        A1[i * cw + w] = s;
      }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nq * n1 * n1; i += blockDim.x) {   // contract qy
      int c = i % n1, b = (i / n1) % n1, qx = i / (n1 * n1);
      for (int w = 0; w < cw; ++w) {
        double s = 0.0;
        for (int qy = 0; qy < nq; ++qy) s += Lq[b * nq + qy] * A1[((qx * nq + qy) * n1 + c) * cw + w];
        A2[i * cw + w] = s;
      }
    }
    __syncthreads();
    for (int I = threadIdx.x; I < n; I += blockDim.x) {              // contract qx
      int bc = I % (n1 * n1), a = I / (n1 * n1);
      for (int w = 0; w < cw; ++w) {
        double s = 0.0;
        for (int qx = 0; qx < nq; ++qx) s += Lq[a * nq + qx] * A2[(qx * n1 * n1 + bc) * cw + w];
        Cd64[(((long)pr * pt.npj + al) * n + I) * cw + w] = s;
      }
    }
  }
}

// generic FP64 -> FP32 copy
static __global__ void k_f64_to_f32(const double* __restrict__ s, float* __restrict__ d, long nelem) {
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < nelem; i += (long)gridDim.x * blockDim.x)
    d[i] = (float)s[i];
}
