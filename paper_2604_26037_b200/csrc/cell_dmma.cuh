// cell_dmma.cuh -- FP64 cell-level product on the double-precision tensor pipe (DMMA.8x8x4):
//     Y += alpha * sum_e P_e^T A^e (P_e X)          (Fig. 2 steps i, iii, iv)
// used by the FP64 reference mode and by the full-precision residual set-up of Algorithm 2 (L260, L374).
//
// One CTA = one cell x one tile of 64 real columns (64 real vectors or 32 complex ones).  The cell matrix is
// streamed in K chunks through a 3-stage cp.async ring together with the gathered rows of X; 8 warps = 4 row
// groups x 2 column halves, each warp owns MT x 4 DMMA tiles (8 rows x 8 columns) in registers, row tile mt*4 + rg of
// the row block (interleaved, so the tiles of a ragged last row block spread evenly over the row groups).  Row blocks
// of 32 MT rows are processed one after the other when n > 32 MT.  MT <= 6: two CTAs per SM (16 warps feed the DMMA pipe).
//   complex:  Y = Hr X + Hi (iX); with interleaved (re, im) columns, iX is the pair (-im, re), so one
//   accumulator set and two DMMAs per tile and k step do the complex product.
#pragma once
#include "common.h"
#include "ptx_sm100.cuh"
#include <type_traits>

namespace dmma {

constexpr int kTN = 64;       // real columns per CTA
constexpr int kStages = 3;
constexpr int kThreads = 256;
constexpr int kStrideB32 = 72;  // floats per staged X row (conflict-free fragment loads)
constexpr int kStrideB64 = 68;  // doubles per staged X row

template <bool CPLX> struct Cfg {
  static constexpr int KC = CPLX ? 8 : 16;            // k rows per stage
  static constexpr int strideA = (KC + 4) * (CPLX ? 2 : 1);  // doubles per staged matrix row
};

template <typename RX, bool CPLX, int MT>
size_t smem_bytes(int n) {
  const size_t a = (size_t)32 * MT * Cfg<CPLX>::strideA * 8;
  const size_t b = (size_t)Cfg<CPLX>::KC * (sizeof(RX) == 4 ? kStrideB32 * 4 : kStrideB64 * 8);
  return kStages * (a + b) + (size_t)n * 8 + 16;
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src, uint32_t src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async4(uint32_t dst, const void* src, uint32_t src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}

// Amat: [cell][n][n] doubles (complex: interleaved), cell_stride in scalars (0 = one shared matrix).
// X: RX reals, ldx in reals; Y: doubles, ldy in reals; Wr = real columns (B or 2B).
template <typename RX, bool CPLX, int MT>
__global__ void __launch_bounds__(kThreads, (MT <= 6 ? 2 : 1))
k_cell_dmma(MeshDev md, const double* __restrict__ Amat, long cell_stride, const RX* __restrict__ X, long ldx,
            double* __restrict__ Y, long ldy, int Wr, double alpha) {
  constexpr int KC = Cfg<CPLX>::KC, strideA = Cfg<CPLX>::strideA, cw = CPLX ? 2 : 1;
  constexpr int RB = 32 * MT;                       // rows per row block
  constexpr int strideB = sizeof(RX) == 4 ? kStrideB32 : kStrideB64;
  constexpr size_t aBytes = (size_t)RB * strideA * 8, bBytes = (size_t)KC * strideB * sizeof(RX);
  extern __shared__ __align__(16) unsigned char smem_raw[];
  unsigned char* stage0 = smem_raw;
  long* nodeJ = reinterpret_cast<long*>(smem_raw + kStages * (aBytes + bBytes));
  const int n = md.n, n1 = md.n1;
  // column tile fastest: the CTAs that share a cell matrix are scheduled together and the re-reads hit L2
  const int ntile = (Wr + kTN - 1) / kTN;
  const int e = blockIdx.x / ntile, v0 = (blockIdx.x % ntile) * kTN;
  {
    int cx, cy, cz;
    mesh_cell_coords(md, e, &cx, &cy, &cz);
    for (int I = threadIdx.x; I < n; I += kThreads) {
      int c = I % n1, b = (I / n1) % n1, a = I / (n1 * n1), ix, iy, iz;
      long J = mesh_node(md, cx, cy, cz, a, b, c, &ix, &iy, &iz);
      if (md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz] == 0.0) J = -1;  // Dirichlet boundary
      nodeJ[I] = J;
    }
  }
  __syncthreads();
  const double* A = Amat + (long)e * cell_stride * cw;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int rg = warp & 3, vh = warp >> 2;
  const int nchunks = (n + KC - 1) / KC;
  // n-tiles (8 real columns) of this warp that hold any column of the block: the others are skipped (ragged last tile)
  int ntv = 0;
  for (int nt = 0; nt < 4; ++nt) if (v0 + vh * 32 + nt * 8 < Wr) ntv = nt + 1;

  for (int r0 = 0; r0 < n; r0 += RB) {
    double acc[MT][4][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    constexpr int RPP = kThreads / KC, NJ = RB / RPP;   // rows per sweep of the CTA, sweeps per chunk
    static_assert(RB % RPP == 0, "row block must be a multiple of the rows per sweep");
    const int ak = threadIdx.x % KC, arow0 = threadIdx.x / KC;
    const double* srcA = A + ((long)(r0 + arow0) * n + ak) * cw;
    const uint32_t dstA = (uint32_t)(arow0 * strideA + ak * cw) * 8;
    const int nrow_valid = n - r0 - arow0;              // row arow0 + RPP j of the block exists iff RPP j < nrow_valid
    const long rstep = (long)RPP * n * cw;

    auto issue = [&](int ch) {
      unsigned char* st = stage0 + (size_t)(ch % kStages) * (aBytes + bBytes);
      const uint32_t abase = ptx::smem_u32(st), bbase = abase + (uint32_t)aBytes;
      const int k0 = ch * KC;
      // matrix rows: thread t copies element ak = t % KC of the rows arow0 + RPP j (RPP = kThreads / KC rows per sweep);
      // source and destination advance by constants, so a copy costs a pointer add and a select (the index arithmetic of
      // the generic loop took ~45% of the warps' time: profiles/r01_ncu_small_kernels.md)
      {
        const bool kok = k0 + ak < n;
        const double* sj = srcA + (long)k0 * cw;
#pragma unroll
        for (int j = 0; j < NJ; ++j) {
          const bool ok = kok && (RPP * j < nrow_valid);
          const uint32_t dst = abase + dstA + (uint32_t)(j * RPP * strideA * 8);
          if (CPLX) ptx::cp_async16(dst, ok ? sj : A, ok ? 16u : 0u);
          else cp_async8(dst, ok ? sj : A, ok ? 8u : 0u);
          sj += rstep;
        }
      }
      // gathered X rows: KC rows x 64 reals
      if (sizeof(RX) == 4) {
        for (int i = threadIdx.x; i < KC * (kTN / 2); i += kThreads) {
          const int k = i / (kTN / 2), c2 = (i % (kTN / 2)) * 2;
          const long J = (k0 + k < n) ? nodeJ[k0 + k] : -1;
          const int v = v0 + c2;
          // pairs of floats: 8-byte copies need even ldx and an 8-byte aligned base; fall back to 4-byte copies
          const bool ok = J >= 0 && v < Wr;
          const RX* src = ok ? X + J * ldx + v : X;
          const uint32_t dst = bbase + (uint32_t)(k * strideB + c2) * 4;
          if (((ldx & 1) == 0) && ((reinterpret_cast<uintptr_t>(X) & 7) == 0)) {
            cp_async8(dst, src, ok ? (v + 1 < Wr ? 8u : 4u) : 0u);
          } else {
            cp_async4(dst, src, ok ? 4u : 0u);
            const bool ok1 = ok && v + 1 < Wr;
            cp_async4(dst + 4, ok1 ? src + 1 : X, ok1 ? 4u : 0u);
          }
        }
      } else {
        for (int i = threadIdx.x; i < KC * kTN; i += kThreads) {
          const int k = i / kTN, c1 = i % kTN;
          const long J = (k0 + k < n) ? nodeJ[k0 + k] : -1;
          const int v = v0 + c1;
          const bool ok = J >= 0 && v < Wr;
          cp_async8(bbase + (uint32_t)(k * strideB + c1) * 8, ok ? X + J * ldx + v : X, ok ? 8u : 0u);
        }
      }
      ptx::cp_async_commit();
    };

    // row tiles of this warp inside the cell's rows (warp-uniform; fewer than MT only in a ragged last row block)
    int mtv = 0;
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) if (r0 + (mt * 4 + rg) * 8 < n) mtv = mt + 1;

    // the DMMAs of one staged chunk.  FULLN: all four n-tiles of the warp hold columns; MTVC >= 0: the number of valid row
    // tiles is the compile-time value (straight-line DMMAs: predicated mma.sync costs a WARPSYNC and a reload bubble per
    // group of four, profiles/r01_ncu_small_kernels.md), -1: run-time value mtv.
    auto mma_chunk = [&](auto fulln, auto mtvc, const double* As, const RX* Bs) {
      constexpr bool FULLN = decltype(fulln)::value;
      constexpr int MTVC = decltype(mtvc)::value;
#pragma unroll
      for (int ks = 0; ks < KC / 4; ++ks) {
        const int kk = ks * 4 + (lane & 3);
        double b[4], bi[4];
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) {
          const int col = vh * 32 + nt * 8 + (lane >> 2);
          if (CPLX) {
            const RX re = Bs[kk * strideB + (col & ~1)], im = Bs[kk * strideB + (col | 1)];
            b[nt] = (col & 1) ? (double)im : (double)re;
            bi[nt] = (col & 1) ? (double)re : -(double)im;
          } else {
            b[nt] = (double)Bs[kk * strideB + col];
          }
        }
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
          if (MTVC >= 0 ? mt < MTVC : mt < mtv) {             // warp-uniform
            const int row = (mt * 4 + rg) * 8 + (lane >> 2);   // row tiles interleaved over the 4 row groups
            if (CPLX) {
              const double2 a2 = *reinterpret_cast<const double2*>(As + row * strideA + kk * 2);
#pragma unroll
              for (int nt = 0; nt < 4; ++nt)
                if (FULLN || nt < ntv) {
                  dmma884(acc[mt][nt][0], acc[mt][nt][1], a2.x, b[nt]);
                  dmma884(acc[mt][nt][0], acc[mt][nt][1], a2.y, bi[nt]);
                }
            } else {
              const double a1 = As[row * strideA + kk];
#pragma unroll
              for (int nt = 0; nt < 4; ++nt)
                if (FULLN || nt < ntv) dmma884(acc[mt][nt][0], acc[mt][nt][1], a1, b[nt]);
            }
          }
        }
      }
    };

    issue(0);
    if (nchunks > 1) issue(1); else ptx::cp_async_commit();
    for (int ch = 0; ch < nchunks; ++ch) {
      ptx::cp_async_wait<1>();
      __syncthreads();  // chunk ch has landed for everyone; everyone is done with chunk ch - 1
      if (ch + 2 < nchunks) issue(ch + 2); else ptx::cp_async_commit();
      const unsigned char* st = stage0 + (size_t)(ch % kStages) * (aBytes + bBytes);
      const double* As = reinterpret_cast<const double*>(st);
      const RX* Bs = reinterpret_cast<const RX*>(st + aBytes);
      if (ntv == 4 && mtv == MT) mma_chunk(std::true_type(), std::integral_constant<int, MT>(), As, Bs);
      else if (ntv == 4 && mtv == MT - 1) mma_chunk(std::true_type(), std::integral_constant<int, MT - 1>(), As, Bs);
      else if (ntv == 4) mma_chunk(std::true_type(), std::integral_constant<int, -1>(), As, Bs);
      else if (ntv > 0) mma_chunk(std::false_type(), std::integral_constant<int, -1>(), As, Bs);
    }
    ptx::cp_async_wait<0>();
    __syncthreads();  // ring free for the next row block
    // assembly (step iv): atomic adds of the 8 x 8 tiles
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
      const int I = r0 + (mt * 4 + rg) * 8 + (lane >> 2);
      const long J = I < n ? nodeJ[I] : -1;
      if (J < 0) continue;
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) {
        const int v = v0 + vh * 32 + nt * 8 + 2 * (lane & 3);
        if (v < Wr) atomicAdd(Y + J * ldy + v, alpha * acc[mt][nt][0]);
        if (v + 1 < Wr) atomicAdd(Y + J * ldy + v + 1, alpha * acc[mt][nt][1]);
      }
    }
  }
}

}  // namespace dmma
