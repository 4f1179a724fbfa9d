// nonlocal_f32.cuh -- pair-parallel kernels of the non-local PAW terms (Fig. 2 steps ii-iii; Eq. 16,
// Eq. 28) for FP32 storage, real or complex (interleaved) blocks seen as Wr = B * cw real columns:
//   k_projF   :  P[a][al][.] += sum_I Cd[pair][al][I] * (s_I X[J(e,I)][.])        Cd = rows of C^{e,a dagger} (Eq. 34)
//   k_scatterF:  Y[J(e,I)][.] += scale * s_I * sum_al conj(Cd[pair][al][I]) * W[a][al][.]     (W rows: [a][wrows][ldp])
// with s_I = M_D^-1 at the node when the scale flag is set (S^-1approx, Eq. 28), else 1.  One CTA per (cell, atom)
// pair and 128 real columns; 8 warps over the cell's rows, one 16-byte piece per lane; four loads in flight per thread.
#pragma once
#include "common.h"

template <int NPJ, bool CPLX>
__global__ void __launch_bounds__(256, (NPJ <= 9 ? 3 : 2))
k_projF(MeshDev md, const int* __restrict__ pair_cell, const int* __restrict__ pair_atom, const float* __restrict__ Cd,
        const float* __restrict__ X, long ldx /*floats*/, int Wr, int in_scale, float* __restrict__ P, long ldp /*floats*/) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int cw = CPLX ? 2 : 1;
  const int n = md.n, n1 = md.n1;
  long* nodeO = reinterpret_cast<long*>(smem_raw);                      // byte offset of the node's row, -1: masked
  float* nodeS = reinterpret_cast<float*>(nodeO + (n + 1) / 2 * 2);     // input scale
  float* Cs = nodeS + (n + 3) / 4 * 4;                                  // [NPJ][n][cw]
  float* red = Cs + ((size_t)NPJ * n * cw + 3) / 4 * 4;                 // [NPJ][128]
  const int pr = blockIdx.x, a = pair_atom[pr];
  int cx, cy, cz;
  mesh_cell_coords(md, pair_cell[pr], &cx, &cy, &cz);
  for (int I = threadIdx.x; I < n; I += blockDim.x) {
    int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1), ix, iy, iz;
    long J = mesh_node(md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
    const double mi = md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz];
    nodeO[I] = (mi == 0.0) ? -1 : J * ldx * 4;
    nodeS[I] = in_scale ? (float)mi : 1.f;
  }
  for (int i = threadIdx.x; i < NPJ * n * cw; i += blockDim.x) Cs[i] = Cd[(long)pr * NPJ * n * cw + i];
  for (int i = threadIdx.x; i < NPJ * 128; i += blockDim.x) red[i] = 0.f;
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int v = blockIdx.y * 128 + lane * 4;
  float4 acc[NPJ];
#pragma unroll
  for (int al = 0; al < NPJ; ++al) acc[al] = make_float4(0.f, 0.f, 0.f, 0.f);
  if (v < Wr) {
    const char* xv = reinterpret_cast<const char*>(X + v);
    for (int I0 = w; I0 < n; I0 += 32) {
      float4 x[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int I = I0 + 8 * u;
        const long off = I < n ? nodeO[I] : -1;
        x[u] = off >= 0 ? __ldg(reinterpret_cast<const float4*>(xv + off)) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int I = min(I0 + 8 * u, n - 1);   // x[u] is zero beyond n
        const float s = nodeS[I];
        const float4 xs = make_float4(s * x[u].x, s * x[u].y, s * x[u].z, s * x[u].w);
#pragma unroll
        for (int al = 0; al < NPJ; ++al) {
          if (CPLX) {
            const float2 cv = *reinterpret_cast<const float2*>(&Cs[(al * n + I) * 2]);
            acc[al].x = fmaf(cv.x, xs.x, acc[al].x); acc[al].x = fmaf(-cv.y, xs.y, acc[al].x);
            acc[al].y = fmaf(cv.x, xs.y, acc[al].y); acc[al].y = fmaf(cv.y, xs.x, acc[al].y);
            acc[al].z = fmaf(cv.x, xs.z, acc[al].z); acc[al].z = fmaf(-cv.y, xs.w, acc[al].z);
            acc[al].w = fmaf(cv.x, xs.w, acc[al].w); acc[al].w = fmaf(cv.y, xs.z, acc[al].w);
          } else {
            const float cv = Cs[al * n + I];
            acc[al].x = fmaf(cv, xs.x, acc[al].x); acc[al].y = fmaf(cv, xs.y, acc[al].y);
            acc[al].z = fmaf(cv, xs.z, acc[al].z); acc[al].w = fmaf(cv, xs.w, acc[al].w);
          }
        }
      }
    }
  }
  // cross-warp sum in shared memory, one warp per round (fixed order; shared-memory float atomics are CAS loops)
  for (int r = 0; r < 8; ++r) {
    if (w == r && v < Wr) {
#pragma unroll
      for (int al = 0; al < NPJ; ++al) {
        float4* q = reinterpret_cast<float4*>(red + al * 128 + lane * 4);
        float4 t = *q;
        t.x += acc[al].x; t.y += acc[al].y; t.z += acc[al].z; t.w += acc[al].w;
        *q = t;
      }
    }
    __syncthreads();
  }
  for (int i = threadIdx.x; i < NPJ * 32; i += blockDim.x) {
    const int al = i >> 5, vv = blockIdx.y * 128 + (i & 31) * 4;
    if (vv < Wr) {
      const float4 val = *reinterpret_cast<const float4*>(&red[al * 128 + (i & 31) * 4]);
      float* dst = P + ((long)a * NPJ + al) * ldp + vv;
      asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(val.x), "f"(val.y), "f"(val.z), "f"(val.w) : "memory");
    }
  }
}

template <int NPJ, bool CPLX>
__global__ void __launch_bounds__(256, (NPJ <= 9 ? 3 : 2))
k_scatterF(MeshDev md, const int* __restrict__ pair_cell, const int* __restrict__ pair_atom, const float* __restrict__ Cd,
           const float* __restrict__ W, long ldp /*floats*/, int wrows /*rows of W per atom*/, int Wr, int out_scale, float scale,
           float* __restrict__ Y, long ldy /*floats*/) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int cw = CPLX ? 2 : 1;
  const int n = md.n, n1 = md.n1;
  long* nodeO = reinterpret_cast<long*>(smem_raw);
  float* nodeS = reinterpret_cast<float*>(nodeO + (n + 1) / 2 * 2);
  float* Cs = nodeS + (n + 3) / 4 * 4;
  const int pr = blockIdx.x, a = pair_atom[pr];
  int cx, cy, cz;
  mesh_cell_coords(md, pair_cell[pr], &cx, &cy, &cz);
  for (int I = threadIdx.x; I < n; I += blockDim.x) {
    int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1), ix, iy, iz;
    long J = mesh_node(md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
    const double mi = md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz];
    nodeO[I] = (mi == 0.0) ? -1 : J * ldy * 4;
    nodeS[I] = scale * (out_scale ? (float)mi : 1.f);
  }
  for (int i = threadIdx.x; i < NPJ * n * cw; i += blockDim.x) Cs[i] = Cd[(long)pr * NPJ * n * cw + i];
  __syncthreads();
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int v = blockIdx.y * 128 + lane * 4;
  if (v >= Wr) return;
  float4 wv[NPJ];
#pragma unroll
  for (int al = 0; al < NPJ; ++al) wv[al] = *reinterpret_cast<const float4*>(W + ((long)a * wrows + al) * ldp + v);
  char* yv = reinterpret_cast<char*>(Y + v);
  for (int I = w; I < n; I += 8) {
    const long off = nodeO[I];
    if (off < 0) continue;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int al = 0; al < NPJ; ++al) {
      if (CPLX) {   // conj(Cd) * W
        const float2 cv = *reinterpret_cast<const float2*>(&Cs[(al * n + I) * 2]);
        acc.x = fmaf(cv.x, wv[al].x, acc.x); acc.x = fmaf(cv.y, wv[al].y, acc.x);
        acc.y = fmaf(cv.x, wv[al].y, acc.y); acc.y = fmaf(-cv.y, wv[al].x, acc.y);
        acc.z = fmaf(cv.x, wv[al].z, acc.z); acc.z = fmaf(cv.y, wv[al].w, acc.z);
        acc.w = fmaf(cv.x, wv[al].w, acc.w); acc.w = fmaf(-cv.y, wv[al].z, acc.w);
      } else {
        const float cv = Cs[al * n + I];
        acc.x = fmaf(cv, wv[al].x, acc.x); acc.y = fmaf(cv, wv[al].y, acc.y);
        acc.z = fmaf(cv, wv[al].z, acc.z); acc.w = fmaf(cv, wv[al].w, acc.w);
      }
    }
    const float s = nodeS[I];
    float* dst = reinterpret_cast<float*>(yv + off);
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(dst), "f"(s * acc.x), "f"(s * acc.y), "f"(s * acc.z), "f"(s * acc.w) : "memory");
  }
}
