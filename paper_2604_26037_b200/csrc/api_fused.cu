// api_fused.cu -- fused Chebyshev step of Algorithm 2 for FP32-storage blocks (see fused.h):
// plan construction (K-extension blocks, neighbour couplings), the atom-local projection and coupling kernels
// (Fig. 2 step ii; Eq. 28-29), the step loop (the bracket of L272 / L374 is written by the cell kernel's
// first writers, cell_tcgen05.cu), recovery (L282).
#include "fused.h"
#include "cell_tcgen05.h"
#include "host_util.h"
#include "api_internal.h"
#include "apply_impl.h"
#include "setup_fp64.cuh"
#include "nonlocal_f32.cuh"
#include "ptx_sm100.cuh"
#include "kernels_stream.cuh"
#include <algorithm>
#include <cmath>
#include <set>

struct FusedPlan {
  bool ok = false;
  long nchunks = 0;
  int* d_ext_start = nullptr;   // [ncell + 1]
  int* d_ext_atom = nullptr;    // [nchunks]
  float* d_Bext = nullptr;      // [nchunks][n][32]
  int* d_nb_start = nullptr;    // [natoms + 1]
  int* d_nb_atom = nullptr;     // [nnb]
  float* d_GD = nullptr;        // [nnb][npj][npj]:  G^{ab} Delta^b_Sinv
  int* d_cps = nullptr;         // [ncell + 1] cell -> its (cell, atom) pairs
  int* d_cpi = nullptr;         // [npairs] pair indices by cell
  int* d_pcells = nullptr; int npcells = 0;   // cells that have at least one pair (grid of k_proj_cell)
  int ext_ksteps = 4;
  // scratch for block width <= Bcap
  int Bcap = 0; long ldw = 0;
  float* d_P1 = nullptr;        // [natoms][npj][ldw]
  float* d_Ppart = nullptr;     // [npairs][npj][ldw] per-pair partial projections (summed in pair order by k_psum)
  uint4* d_CdF = nullptr;       // [npairs][ceil(n/8)][32]: the pairs' blocks as mma.sync A fragments, rounded to TF32 (k_build_cdf)
  float* d_Wcat = nullptr;      // [natoms][32][ldw]: rows [0,npj) W, [npj,2npj) D P2, rest 0
  float* d_Wcat_lo = nullptr;   // low parts of Wcat (FP32 mode, 3xTF32 split)
  float* d_Bext_lo = nullptr;   // low parts of d_Bext (built on first FP32-mode use)
  float* d_xlo = nullptr; size_t xlo_elems = 0;   // low parts of the input block of fused_apply_H / _HSinv in FP32 mode
  float* d_xs = nullptr; size_t xs_elems = 0;     // M_D^-1 X of fused_apply_HSinv
  // second stream for work that is independent inside a step (projection || bracket prepass; mass / non-local || DMMA)
  cudaStream_t aux = nullptr; cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  bool no_aux = false;          // PAWFE_NO_AUX=1: everything on the context's stream (timing experiments)
  double* d_P64 = nullptr;      // [natoms][npj][ldw] FP64 projections of the residual set-up
  double* d_W64 = nullptr;      // [natoms][npj][ldw] (D - Lambda dS) P
};

namespace {

inline long roundup4(long x) { return (x + 3) / 4 * 4; }

// ---- pair lookup: index of (atom, cell) in the pair list (pairs sorted by atom, then cell), or -1 ----
__device__ inline int find_pair(const int* __restrict__ aps, const int* __restrict__ pair_cell, int atom, int cell) {
  int lo = aps[atom], hi = aps[atom + 1] - 1;
  while (lo <= hi) {
    int mid = (lo + hi) >> 1, pc = pair_cell[mid];
    if (pc == cell) return mid;
    if (pc < cell) lo = mid + 1; else hi = mid - 1;
  }
  return -1;
}

// ------------------------------------------------------------------------------------------------
// Set-up: one CTA per K-extension chunk x = (cell e, atom b).  TD = double (real) or double2 (complex context).
//   Zs[I][be] = M_D^-1[J] * (assembled C^b)[J][be] at the nodes J of cell e  (sum over the <= 8 cells sharing J);
//               C^b = (C^b dagger)^dagger, i.e. conj of the stored rows Cd = C^{e,b dagger} (Eq. 34)
//   block[I][be]       = - sum_J H^e[I][J] Zs[J][be]                         (be < npj)
//   block[I][npj + be] = C^{e,b}[I][be] = conj(Cd[pair][be][I]) if (e, b) is a pair, else 0
//   G[slot(a, b)][al][be] += sum_I Cd^{e,a}[al][I] Zs[I][be]   for every pair (e, a)   (G^{ab} = C^a^dagger M_D^-1 C^b)
// Output layout [x][half][comp][NT rows][32] floats (comp: Re, Im), rows 128-byte swizzled (16-byte piece j of row r at
// j ^ (r % 8)), the block format of the cell kernel; rows I >= n stay zero.  block = 256; smem: n * npj TD.
// ------------------------------------------------------------------------------------------------
__device__ inline double  t_conj(double a)  { return a; }
__device__ inline double2 t_conj(double2 a) { return make_double2(a.x, -a.y); }
__device__ inline double  t_re(double a)  { return a; }
__device__ inline double  t_re(double2 a) { return a.x; }
__device__ inline double  t_im(double)    { return 0.0; }
__device__ inline double  t_im(double2 a) { return a.y; }
__device__ inline void t_atomic_add(double* p, double v) { atomicAdd(p, v); }
__device__ inline void t_atomic_add(double2* p, double2 v) { atomicAdd(&p->x, v.x); atomicAdd(&p->y, v.y); }
__device__ inline double  t_warp_sum(double s)  { for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o); return s; }
__device__ inline double2 t_warp_sum(double2 s) { return make_double2(t_warp_sum(s.x), t_warp_sum(s.y)); }

template <typename TD>
__global__ void __launch_bounds__(256)
k_build_ext(MeshDev md, const int* __restrict__ ext_cell, const int* __restrict__ ext_atom,
            const int* __restrict__ aps, const int* __restrict__ pair_cell, const TD* __restrict__ Cd64,
            int npj, const TD* __restrict__ H64, const int* __restrict__ cell_pair_start,
            const int* __restrict__ cell_pair_idx, const int* __restrict__ pair_atom,
            const int* __restrict__ nb_start, const int* __restrict__ nb_atom, int NH, int NT,
            float* __restrict__ Bext, TD* __restrict__ G) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int ncomp = ScalarTraits<TD>::cplx ? 2 : 1;
  TD* Zs = reinterpret_cast<TD*>(smem_raw);  // [n][npj]
  const int n = md.n, n1 = md.n1, p = md.p;
  const int x = blockIdx.x;
  const int e = ext_cell[x], b = ext_atom[x];
  int cx, cy, cz;
  mesh_cell_coords(md, e, &cx, &cy, &cz);
  const int cc[3] = {cx, cy, cz};
  // ---- phase 1: assembled, M_D^-1-scaled projector values of atom b at this cell's nodes ----
  for (int I = threadIdx.x; I < n; I += blockDim.x) {
    const int loc[3] = {I / (n1 * n1), (I / n1) % n1, I % n1};
    int ix, iy, iz;
    mesh_node(md, cx, cy, cz, loc[0], loc[1], loc[2], &ix, &iy, &iz);
    const double mi = md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz];
    // incidences of this node: per direction the own cell, plus the neighbour across a face the node lies on
    int ncand[3], ccell[3][2], cloc[3][2];
    for (int d = 0; d < 3; ++d) {
      ncand[d] = 1; ccell[d][0] = cc[d]; cloc[d][0] = loc[d];
      if (loc[d] == 0 || loc[d] == p) {
        int nbc = loc[d] == 0 ? cc[d] - 1 : cc[d] + 1;
        const int nbl = loc[d] == 0 ? p : 0;
        if (md.periodic) nbc = (nbc + md.nc[d]) % md.nc[d];
        if (nbc >= 0 && nbc < md.nc[d]) { ccell[d][1] = nbc; cloc[d][1] = nbl; ncand[d] = 2; }
      }
    }
    for (int be = 0; be < npj; ++be) Zs[I * npj + be] = s_zero(TD());
    if (mi != 0.0) {
      for (int qx = 0; qx < ncand[0]; ++qx)
        for (int qy = 0; qy < ncand[1]; ++qy)
          for (int qz = 0; qz < ncand[2]; ++qz) {
            const int e2 = (ccell[0][qx] * md.nc[1] + ccell[1][qy]) * md.nc[2] + ccell[2][qz];
            const int pr = find_pair(aps, pair_cell, b, e2);
            if (pr < 0) continue;
            const int I2 = (cloc[0][qx] * n1 + cloc[1][qy]) * n1 + cloc[2][qz];
            for (int be = 0; be < npj; ++be)
              Zs[I * npj + be] = s_add(Zs[I * npj + be], t_conj(Cd64[((long)pr * npj + be) * n + I2]));
          }
      for (int be = 0; be < npj; ++be) Zs[I * npj + be] = s_scale(Zs[I * npj + be], mi);
    }
  }
  __syncthreads();
  // ---- phase 2: K-extension block ----
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int prb = find_pair(aps, pair_cell, b, e);
  const TD* He = H64 + (long)e * n * n;
  auto bidx = [&](int I, int k, int comp) -> long {
    const int half = I / NT, r = I - half * NT;
    return ((((long)x * NH + half) * ncomp + comp) * NT + r) * 32 + ((((k >> 2) ^ (r & 7)) << 2) | (k & 3));
  };
  for (int I = w; I < n; I += nw) {
    TD acc[PAWFE_MAX_NPJ];
#pragma unroll
    for (int be = 0; be < PAWFE_MAX_NPJ; ++be) acc[be] = s_zero(TD());
    for (int J = lane; J < n; J += 32) {
      const TD h = He[(long)I * n + J];
#pragma unroll
      for (int be = 0; be < PAWFE_MAX_NPJ; ++be)
        if (be < npj) s_fma(acc[be], h, Zs[J * npj + be]);
    }
#pragma unroll
    for (int be = 0; be < PAWFE_MAX_NPJ; ++be)
      if (be < npj) {
        const TD s = t_warp_sum(acc[be]);
        if (lane == 0) {
          Bext[bidx(I, be, 0)] = (float)(-t_re(s));
          if (ncomp == 2) Bext[bidx(I, be, 1)] = (float)(-t_im(s));
        }
      }
    for (int k = npj + lane; k < 32; k += 32) {
      float vr = 0.f, vi = 0.f;
      if (k < 2 * npj && prb >= 0) {
        const TD cv = t_conj(Cd64[((long)prb * npj + (k - npj)) * n + I]);
        vr = (float)t_re(cv); vi = (float)t_im(cv);
      }
      Bext[bidx(I, k, 0)] = vr;
      if (ncomp == 2) Bext[bidx(I, k, 1)] = vi;
    }
  }
  // ---- phase 3: G^{ab} contributions of this cell ----
  for (int q = cell_pair_start[e]; q < cell_pair_start[e + 1]; ++q) {
    const int pr = cell_pair_idx[q], a = pair_atom[pr];
    int slot = -1;
    for (int s = nb_start[a]; s < nb_start[a + 1]; ++s) if (nb_atom[s] == b) { slot = s; break; }
    if (slot < 0) continue;
    for (int ab = w; ab < npj * npj; ab += nw) {
      const int al = ab / npj, be = ab % npj;
      TD s = s_zero(TD());
      for (int I = lane; I < n; I += 32) s_fma(s, Cd64[((long)pr * npj + al) * n + I], Zs[I * npj + be]);
      s = t_warp_sum(s);
      if (lane == 0) t_atomic_add(&G[((long)slot * npj + al) * npj + be], s);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// (ii) partial non-local projection, CELL-parallel:  Ppart[pair][al][v] = sum_I C^{e,a}[I][al] X[J(e,I)][v]  for every pair of
//   the cell.  One CTA per (cell that has pairs, tile of 64 real columns): the cell's rows are brought to shared memory ONCE
//   (cp.async, 16 bytes per thread and row piece) and every pair of the cell is projected from there (a pair-parallel
//   kernel reads the rows once per pair: config 4 has 45k pairs on 22k such cells, 16 GB per step instead of 8 GB).
//   256 threads = 16 row groups x 16 column quads; the row groups are summed in a fixed order (shuffle, then warp by warp in
//   shared memory), so the per-pair partials are bit-reproducible; k_psum adds them pair by pair.
//   CPLX: interleaved (re, im) columns, Cd complex [pair][NPJ][n][2].  dynamic smem: see proj_cell_smem().
// ------------------------------------------------------------------------------------------------
constexpr int kPcVT = 64;   // real columns per CTA
// floats reserved for a pair's block (plus the alignment shift, whole 16-byte pieces) or the reduction scratch, whichever is larger
template <int NPJ, bool CPLX>
__host__ __device__ constexpr size_t proj_cell_cs_floats(int n) {
  return ((size_t)NPJ * (CPLX ? 2 : 1) * n + 3 + 3) / 4 * 4 > (size_t)4 * NPJ * kPcVT ? ((size_t)NPJ * (CPLX ? 2 : 1) * n + 3 + 3) / 4 * 4 : (size_t)4 * NPJ * kPcVT;
}
template <int NPJ, bool CPLX>
__global__ void __launch_bounds__(256, 2)
k_proj_cell(MeshDev md, const int* __restrict__ pcells, const int* __restrict__ cps, const int* __restrict__ cpi,
            const float* __restrict__ Cd, long cd_total, const float* __restrict__ X, long ldx, int Wr, float* __restrict__ Ppart,
            long ldp) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int cw = CPLX ? 2 : 1;
  constexpr int kCnt = NPJ * cw;                                            // floats of a pair's block per node
  const int n = md.n, n1 = md.n1;
  float* tile = reinterpret_cast<float*>(smem_raw);                         // [n][64]
  float* Csraw = tile + (size_t)n * kPcVT;                                  // the pair's block [NPJ][n][cw], shifted by <= 3 floats (see below)
  float* red = Csraw;                                                       // [4][NPJ][64], reuses the block's space once a pair's FMAs are done
  long* nodeO = reinterpret_cast<long*>(Csraw + proj_cell_cs_floats<NPJ, CPLX>(n));   // [n] element offset of the node's row, -1: masked
  const int e = pcells[blockIdx.x];
  const int v0 = blockIdx.y * kPcVT;
  {
    int cx, cy, cz;
    mesh_cell_coords(md, e, &cx, &cy, &cz);
    for (int I = threadIdx.x; I < n; I += 256) {
      int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1), ix, iy, iz;
      const long J = mesh_node(md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
      nodeO[I] = md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz] != 0.0 ? J * ldx : -1;
    }
  }
  __syncthreads();
  // rows -> shared memory (Dirichlet wall rows and columns beyond the block: zero fill)
  const uint32_t tile_a = ptx::smem_u32(tile), cs_a = ptx::smem_u32(Csraw);
  for (int i = threadIdx.x; i < n * (kPcVT / 4); i += 256) {
    const int I = i >> 4, q = i & 15;
    const long off = nodeO[I];
    const bool ok = off >= 0 && v0 + 4 * q < Wr;
    ptx::cp_async16(tile_a + (uint32_t)(I * kPcVT + 4 * q) * 4, ok ? X + off + v0 + 4 * q : X, ok ? 16u : 0u);
  }
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int vq = threadIdx.x & 15, rg = threadIdx.x >> 4;   // column quad, row group (rows rg, rg + 16, ...)
  for (int q = cps[e]; q < cps[e + 1]; ++q) {
    const int pr = cpi[q];
    __syncthreads();   // everyone is done with the block / red of the previous pair
    // the pair's block by 16-byte copies: a block starts at a multiple of 4 bytes only (n is odd), so the copy starts at the
    // 16-byte boundary below it and the block is read from Csraw + sh; nothing is read beyond the end of the array
    const long start = (long)pr * kCnt * n;
    const int sh = (int)(start & 3);
    const float* src = Cd + (start - sh);
    const int cnt4 = (kCnt * n + sh + 3) / 4;
    for (int i = threadIdx.x; i < cnt4; i += 256) {
      const long left = cd_total - (start - sh) - 4L * i;                   // floats of the array from this piece on
      ptx::cp_async16(cs_a + 16u * i, src + 4 * i, left >= 4 ? 16u : (uint32_t)(4 * left));
    }
    ptx::cp_async_commit();
    const float* Cs = Csraw + sh;
    ptx::cp_async_wait<0>();
    __syncthreads();
    float4 acc[NPJ];
#pragma unroll
    for (int al = 0; al < NPJ; ++al) acc[al] = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int I = rg; I < n; I += 16) {
      const float4 x = *reinterpret_cast<const float4*>(&tile[I * kPcVT + 4 * vq]);
#pragma unroll
      for (int al = 0; al < NPJ; ++al) {
        if (CPLX) {
          const float2 cv = *reinterpret_cast<const float2*>(&Cs[(al * n + I) * 2]);
          acc[al].x = fmaf(cv.x, x.x, acc[al].x); acc[al].x = fmaf(-cv.y, x.y, acc[al].x);
          acc[al].y = fmaf(cv.x, x.y, acc[al].y); acc[al].y = fmaf(cv.y, x.x, acc[al].y);
          acc[al].z = fmaf(cv.x, x.z, acc[al].z); acc[al].z = fmaf(-cv.y, x.w, acc[al].z);
          acc[al].w = fmaf(cv.x, x.w, acc[al].w); acc[al].w = fmaf(cv.y, x.z, acc[al].w);
        } else {
          const float cv = Cs[al * n + I];
          acc[al].x = fmaf(cv, x.x, acc[al].x); acc[al].y = fmaf(cv, x.y, acc[al].y);
          acc[al].z = fmaf(cv, x.z, acc[al].z); acc[al].w = fmaf(cv, x.w, acc[al].w);
        }
      }
    }
    // the warp's two row groups (lanes l and l ^ 16), then warp w + 4 onto warp w, then the four sums in order
#pragma unroll
    for (int al = 0; al < NPJ; ++al) {
      acc[al].x += __shfl_xor_sync(0xffffffffu, acc[al].x, 16); acc[al].y += __shfl_xor_sync(0xffffffffu, acc[al].y, 16);
      acc[al].z += __shfl_xor_sync(0xffffffffu, acc[al].z, 16); acc[al].w += __shfl_xor_sync(0xffffffffu, acc[al].w, 16);
    }
    __syncthreads();   // all reads of Cs are done: red may overwrite it
    if (w >= 4 && lane < 16) {
#pragma unroll
      for (int al = 0; al < NPJ; ++al) *reinterpret_cast<float4*>(&red[((w - 4) * NPJ + al) * kPcVT + 4 * vq]) = acc[al];
    }
    __syncthreads();
    if (w < 4 && lane < 16) {
#pragma unroll
      for (int al = 0; al < NPJ; ++al) {
        float4* r4 = reinterpret_cast<float4*>(&red[(w * NPJ + al) * kPcVT + 4 * vq]);
        const float4 u = *r4;
        *r4 = make_float4(acc[al].x + u.x, acc[al].y + u.y, acc[al].z + u.z, acc[al].w + u.w);
      }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NPJ * 16; i += 256) {
      const int al = i >> 4, qq = i & 15;
      if (v0 + 4 * qq < Wr) {
        float4 t = *reinterpret_cast<const float4*>(&red[al * kPcVT + 4 * qq]);
#pragma unroll
        for (int ww = 1; ww < 4; ++ww) {
          const float4 u = *reinterpret_cast<const float4*>(&red[(ww * NPJ + al) * kPcVT + 4 * qq]);
          t.x += u.x; t.y += u.y; t.z += u.z; t.w += u.w;
        }
        *reinterpret_cast<float4*>(Ppart + ((long)pr * NPJ + al) * ldp + v0 + 4 * qq) = t;
      }
    }
  }
  ptx::cp_async_wait<0>();
}
template <int NPJ, bool CPLX>
size_t proj_cell_smem(int n) {
  return ((size_t)n * kPcVT + proj_cell_cs_floats<NPJ, CPLX>(n)) * sizeof(float) + (size_t)n * sizeof(long);
}

// The pairs' blocks in the order mma.sync m16n8k8 wants its A fragments, rounded to TF32 (round to nearest), zero beyond the
// npj projectors and the n nodes:  CdF[pair][ks][part][lane] = { C[g][8ks+t], C[g+8][8ks+t], C[g][8ks+t+4], C[g+8][8ks+t+4] },
// g = lane >> 2, t = lane & 3, C[al][I] = Cd[pair][al][I]; complex contexts (cw = 2): part 0 = Re C, part 1 = Im C.
// Built once per plan.
__global__ void __launch_bounds__(256)
k_build_cdf(long total, int npj, int n, int nks, int cw, const float* __restrict__ Cd, uint4* __restrict__ CdF) {
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    const int lane = (int)(i & 31), g = lane >> 2, t = lane & 3;
    long sl = i >> 5;
    const int part = (int)(sl % cw);
    sl /= cw;
    const int ks = (int)(sl % nks);
    const long pr = sl / nks;
    auto val = [&](int row, int col) -> uint32_t {
      return row < npj && col < n ? ptx::cvt_rna_tf32(Cd[((pr * npj + row) * n + col) * cw + part]) : 0u;
    };
    const int c0 = ks * 8 + t;
    CdF[i] = make_uint4(val(g, c0), val(g + 8, c0), val(g, c0 + 4), val(g + 8, c0 + 4));
  }
}

// The same projection on the tensor cores, for the TF32 mode: per pair P(16 x 64) += A(16 x 8) B(8 x 64) over
// the 43 (p = 6) row slices of 8 nodes, warp w taking slices w, w + 8, ... (mma.sync m16n8k8, TF32 operands, FP32 accumulate:
// the precision the cell kernel next to it multiplies in).  A = the pair's block, read straight from global memory one pair
// ahead, as ready-made fragments (k_build_cdf: one coalesced 16-byte load per lane and slice, each used by one warp only); B = the cell's rows in shared
// memory, 16-byte pieces XOR-swizzled by (row & 3) so that the four k rows of a fragment load fall on different banks.
// The eight warps' partial tiles are summed in the fixed order of k_proj_cell (w + 4 onto w, then 0..3): bit-reproducible.
constexpr int kPmRedLd = 72;   // floats per row of the reduction scratch (72 mod 32 = 8: the float2 stores of a tile do not collide)
// CPLX (interleaved (re, im) columns): P = Cr X + Ci X' with X'[2v] = -X[2v+1], X'[2v+1] = X[2v], i.e. a second MMA per tile whose
// B fragment is read from the neighbouring column (g ^ 1) with the sign of the even columns flipped.
template <int NPJ, int MAXJ, bool CPLX>   // MAXJ: row slices per warp, ceil(ceil(n / 8) / 8)
__global__ void __launch_bounds__(256, 2)
k_proj_cell_mma(MeshDev md, const int* __restrict__ pcells, const int* __restrict__ cps, const int* __restrict__ cpi,
                const uint4* __restrict__ CdF, const float* __restrict__ X, long ldx, int Wr, float* __restrict__ Ppart, long ldp) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  static_assert(NPJ <= 16, "one m16 tile");
  const int n = md.n, n1 = md.n1;
  const int nks = (n + 7) / 8;
  float* tile = reinterpret_cast<float*>(smem_raw);                         // [8 nks][64], swizzled; rows >= n are zero
  float* red = tile + (size_t)nks * 8 * kPcVT;                              // [4][NPJ][72]
  long* nodeO = reinterpret_cast<long*>(red + 4 * NPJ * kPmRedLd);          // [n]
  const int e = pcells[blockIdx.x];
  const int v0 = blockIdx.y * kPcVT;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, g = lane >> 2, t = lane & 3;
  constexpr int cw = CPLX ? 2 : 1;
  uint32_t a[MAXJ][4], ai[CPLX ? MAXJ : 1][4];
  // slice j of a pair's block: rows g, g + 8 (projector), columns 8 ks + t, + 4 (node); complex: Re then Im
  auto load_a = [&](const uint4* Cp, int j) {                               // Cp: the pair's fragments + lane
    const int ks = w + 8 * j;
    const uint4 v = ks < nks ? __ldg(Cp + 32 * cw * ks) : make_uint4(0u, 0u, 0u, 0u);
    a[j][0] = v.x; a[j][1] = v.y; a[j][2] = v.z; a[j][3] = v.w;
    if (CPLX) {
      const uint4 u = ks < nks ? __ldg(Cp + 32 * (cw * ks + 1)) : make_uint4(0u, 0u, 0u, 0u);
      ai[j][0] = u.x; ai[j][1] = u.y; ai[j][2] = u.z; ai[j][3] = u.w;
    }
  };
  const int q0 = cps[e], q1 = cps[e + 1];
  {
    const uint4* Cp = CdF + (long)cpi[q0] * nks * (32 * cw) + lane;
#pragma unroll
    for (int j = 0; j < MAXJ; ++j) load_a(Cp, j);
  }
  {
    int cx, cy, cz;
    mesh_cell_coords(md, e, &cx, &cy, &cz);
    for (int I = threadIdx.x; I < n; I += 256) {
      int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1), ix, iy, iz;
      const long J = mesh_node(md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
      nodeO[I] = md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz] != 0.0 ? J * ldx : -1;
    }
  }
  __syncthreads();
  const uint32_t tile_a = ptx::smem_u32(tile);
  for (int i = threadIdx.x; i < nks * 8 * (kPcVT / 4); i += 256) {
    const int I = i >> 4, q = i & 15;
    const long off = I < n ? nodeO[I] : -1;
    const bool ok = off >= 0 && v0 + 4 * q < Wr;
    ptx::cp_async16(tile_a + (uint32_t)(I * kPcVT + 4 * (q ^ ((I & 3) << 1))) * 4, ok ? X + off + v0 + 4 * q : X, ok ? 16u : 0u);
  }
  ptx::cp_async_commit();
  ptx::cp_async_wait<0>();
  __syncthreads();
  // byte address of (row 8 ks + t, logical column 8 nt + g) = rowb + o[nt & 3] + 128 (nt >> 2); row + 4: + 1024
  const uint32_t o0 = (uint32_t)((((0 ^ t) << 3) + g) * 4), o1 = (uint32_t)((((1 ^ t) << 3) + g) * 4),
                 o2 = (uint32_t)((((2 ^ t) << 3) + g) * 4), o3 = (uint32_t)((((3 ^ t) << 3) + g) * 4);
  const uint32_t sgn = (g & 1) ? 0u : 0x80000000u;                         // complex: column g ^ 1 (offset ^ 4), even columns negated
  for (int q = q0; q < q1; ++q) {
    const int pr = cpi[q];
    const uint4* Cnext = q + 1 < q1 ? CdF + (long)cpi[q + 1] * nks * (32 * cw) + lane : nullptr;
    float acc[8][4];
#pragma unroll
    for (int nt = 0; nt < 8; ++nt) acc[nt][0] = acc[nt][1] = acc[nt][2] = acc[nt][3] = 0.f;
#pragma unroll
    for (int j = 0; j < MAXJ; ++j) {
      const int ks = w + 8 * j;
      if (ks < nks) {                                                        // (warp-uniform)
        const uint32_t rowb = tile_a + (uint32_t)((ks * 8 + t) * kPcVT) * 4;
#define PM_MMA(NT, O)                                                                                             \
        ptx::mma_m16n8k8_tf32(acc[NT], a[j], ptx::lds_u32_off<128 * ((NT) >> 2)>(rowb + (O)),                     \
                              ptx::lds_u32_off<1024 + 128 * ((NT) >> 2)>(rowb + (O)));                            \
        if (CPLX)                                                                                                 \
          ptx::mma_m16n8k8_tf32(acc[NT], ai[j], ptx::lds_u32_off<128 * ((NT) >> 2)>(rowb + ((O) ^ 4u)) ^ sgn,     \
                                ptx::lds_u32_off<1024 + 128 * ((NT) >> 2)>(rowb + ((O) ^ 4u)) ^ sgn);
        PM_MMA(0, o0) PM_MMA(1, o1) PM_MMA(2, o2) PM_MMA(3, o3) PM_MMA(4, o0) PM_MMA(5, o1) PM_MMA(6, o2) PM_MMA(7, o3)
#undef PM_MMA
      }
      if (Cnext) load_a(Cnext, j);                                           // the next pair's slice, in flight behind this pair's work
    }
    if (w >= 4) {
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        float* r0 = red + ((size_t)(w - 4) * NPJ + g) * kPmRedLd + nt * 8 + 2 * t;
        if (g < NPJ) *reinterpret_cast<float2*>(r0) = make_float2(acc[nt][0], acc[nt][1]);
        if (g + 8 < NPJ) *reinterpret_cast<float2*>(r0 + 8 * kPmRedLd) = make_float2(acc[nt][2], acc[nt][3]);
      }
    }
    __syncthreads();
    if (w < 4) {
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        float* r0 = red + ((size_t)w * NPJ + g) * kPmRedLd + nt * 8 + 2 * t;
        float2 u;
        if (g < NPJ) {
          u = *reinterpret_cast<float2*>(r0);
          *reinterpret_cast<float2*>(r0) = make_float2(acc[nt][0] + u.x, acc[nt][1] + u.y);
        }
        if (g + 8 < NPJ) {
          u = *reinterpret_cast<float2*>(r0 + 8 * kPmRedLd);
          *reinterpret_cast<float2*>(r0 + 8 * kPmRedLd) = make_float2(acc[nt][2] + u.x, acc[nt][3] + u.y);
        }
      }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < NPJ * 16; i += 256) {
      const int al = i >> 4, qq = i & 15;
      if (v0 + 4 * qq < Wr) {
        float4 s = *reinterpret_cast<const float4*>(&red[(size_t)al * kPmRedLd + 4 * qq]);
#pragma unroll
        for (int ww = 1; ww < 4; ++ww) {
          const float4 u = *reinterpret_cast<const float4*>(&red[((size_t)ww * NPJ + al) * kPmRedLd + 4 * qq]);
          s.x += u.x; s.y += u.y; s.z += u.z; s.w += u.w;
        }
        *reinterpret_cast<float4*>(Ppart + ((long)pr * NPJ + al) * ldp + v0 + 4 * qq) = s;
      }
    }
    __syncthreads();   // red is free for the next pair
  }
}
template <int NPJ>
size_t proj_cell_mma_smem(int n) {
  return ((size_t)((n + 7) / 8) * 8 * kPcVT + 4 * NPJ * kPmRedLd) * sizeof(float) + (size_t)n * sizeof(long);
}

// P[a][al][.] = sum over the atom's pairs, in pair order, of the per-pair partial projections (k_proj_cell):
// the ordered replacement of their cross-CTA reductions.  grid = (natoms * npj, ceil(Wq / 128)), block = 128; Wq = quads
// of 4 real columns that hold data; ldq = leading dimension / 4.
__global__ void __launch_bounds__(128)
k_psum(int npj, const int* __restrict__ aps, const float4* __restrict__ Ppart, long ldq, int Wq, float4* __restrict__ P) {
  const int a = blockIdx.x / npj, al = blockIdx.x - a * npj;
  const int q = blockIdx.y * 128 + threadIdx.x;
  if (q >= Wq) return;
  float4 s = make_float4(0.f, 0.f, 0.f, 0.f);
  const int p0 = aps[a], p1 = aps[a + 1];
  int pr = p0;
  for (; pr + 4 <= p1; pr += 4) {   // four loads in flight, added in pair order
    float4 t[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) t[u] = Ppart[((long)(pr + u) * npj + al) * ldq + q];
#pragma unroll
    for (int u = 0; u < 4; ++u) { s.x += t[u].x; s.y += t[u].y; s.z += t[u].z; s.w += t[u].w; }
  }
  for (; pr < p1; ++pr) {
    const float4 t = Ppart[((long)pr * npj + al) * ldq + q];
    s.x += t.x; s.y += t.y; s.z += t.z; s.w += t.w;
  }
  P[((long)a * npj + al) * ldq + q] = s;
}

// ------------------------------------------------------------------------------------------------
// Couplings per atom and vector (Eq. 28-29, Eq. 16):
//   W^a = Delta^a_Sinv P1^a;  P2^a = P1^a - sum_{b in nb(a)} (G^{ab} Delta^b_Sinv) P1^b;  W2^a = D^a P2^a.
//   mode 0: both (filter step);  mode 1: W only (recovery, S^-1approx alone);  mode 2: plain H (W = 0, W2 = D P1).
//   Wcat[a][k][v]: k < npj -> W, npj <= k < 2 npj -> W2; columns B <= v < Bpad (the pad columns of a ragged block the cell
//   kernel's 16-byte gathers touch) are written as 0.  grid = (natoms, ceil(Bpad/32)), block = 32 * npj: one thread per
//   (output row al, vector), so the dependent chain per thread is one dot product per neighbour instead of npj of them;
//   P1 slices, G^{ab} Delta^b_Sinv and P2 go through shared memory.
// ------------------------------------------------------------------------------------------------
constexpr int kCoupleLanes = 32;
template <typename T>   // float (real context) or float2 (complex context); ldp, ldw in units of T
__global__ void __launch_bounds__(kCoupleLanes * PAWFE_MAX_NPJ)
k_couple(int npj, int mode, const T* __restrict__ P1, long ldp, int B, int Bpad, const T* __restrict__ dSinv,
         const T* __restrict__ D, const int* __restrict__ nb_start, const int* __restrict__ nb_atom,
         const T* __restrict__ GD, T* __restrict__ Wcat, long ldw) {
  // every operand is staged once per CTA: thread (al, lane) fetches ONE element of an atom's npj x 32 slice of P1 and
  // (tid < npj^2) one element of the neighbour's G^{ab} Delta^b_Sinv, one neighbour ahead of the products that read them
  // from shared memory.  The order of the additions is the one of the definition above (be = 0 .. npj-1, neighbours in list order).
  __shared__ T own[PAWFE_MAX_NPJ][kCoupleLanes];
  __shared__ T p2s[PAWFE_MAX_NPJ][kCoupleLanes];
  __shared__ T pbs[2][PAWFE_MAX_NPJ][kCoupleLanes];
  __shared__ T gs[2][PAWFE_MAX_NPJ * PAWFE_MAX_NPJ];
  const int a = blockIdx.x;
  const int tid = threadIdx.x, lane = tid % kCoupleLanes, al = tid / kCoupleLanes;   // al < npj
  const int v = blockIdx.y * kCoupleLanes + lane, nn = npj * npj;
  const bool ok = v < B, wr = v < Bpad;   // wr && !ok: pad column, every product below is zero
  const int s0 = mode == 0 ? nb_start[a] : 0, s1 = mode == 0 ? nb_start[a + 1] : 0;
  T pre = s_zero(T()), gpre = s_zero(T());
  auto fetch = [&](int s) {
    const int b = nb_atom[s];
    pre = ok ? P1[((long)b * npj + al) * ldp + v] : s_zero(T());
    if (tid < nn) gpre = GD[(long)s * nn + tid];
  };
  if (s0 < s1) fetch(s0);
  T p2 = ok ? P1[((long)a * npj + al) * ldp + v] : s_zero(T());
  own[al][lane] = p2;
  __syncthreads();
  T* Wa = Wcat + (long)a * 32 * ldw;
  if (mode != 2) {
    const T* S = dSinv + ((long)a * npj + al) * npj;
    T s = s_zero(T());
#pragma unroll
    for (int be = 0; be < PAWFE_MAX_NPJ; ++be) if (be < npj) s_fma(s, S[be], own[be][lane]);
    if (wr) Wa[(long)al * ldw + v] = s;
  } else if (wr) {
    Wa[(long)al * ldw + v] = s_zero(T());
  }
  if (mode == 1) return;
  for (int s = s0; s < s1; ++s) {
    const int buf = (s - s0) & 1;
    pbs[buf][al][lane] = pre;
    if (tid < nn) gs[buf][tid] = gpre;
    __syncthreads();   // (two buffers: the writes of neighbour s + 2 come after the barrier of s + 1, past every read of s)
    if (s + 1 < s1) fetch(s + 1);
    const T* g = &gs[buf][al * npj];
    T t = s_zero(T());
#pragma unroll
    for (int be = 0; be < PAWFE_MAX_NPJ; ++be) if (be < npj) s_fma(t, g[be], pbs[buf][be][lane]);
    p2 = s_add(p2, s_scale(t, -1.0));
  }
  p2s[al][lane] = p2;
  __syncthreads();
  const T* Da = D + ((long)a * npj + al) * npj;
  T w2 = s_zero(T());
#pragma unroll
  for (int be = 0; be < PAWFE_MAX_NPJ; ++be) if (be < npj) s_fma(w2, Da[be], p2s[be][lane]);
  if (wr) Wa[(long)(npj + al) * ldw + v] = w2;
}


// Alg. 2 step 5 (L282) in one ORDERED pass:  X <- keep * (Rt_Y + X Lambda_Y) - M_D^-1 C W   (W = rows [0, npj) of Wcat).
// Every node has one owner cell (local index < p in each direction; the upper wall planes of a Dirichlet mesh go to the last
// cells); the owner's CTA sums, for each of its nodes, the low-rank contributions of ALL (cell, atom) pairs whose cell
// contains the node -- the owner cell and the up to 7 cells below it -- in a fixed order (octant, then pair), and stores
// the row once.  No atomics: the result is bit-reproducible, and the diagonal part needs no kernel of its own.
//   grid = (ncell, ceil(Wr / 128)), block = 256: warp = node, lane = 4 consecutive real columns.  VEC: 16-byte accesses
//   (ldx % 4 == 0, X 16-byte aligned); otherwise scalar accesses with a guard on the block's last quad.
template <bool CPLX, bool VEC>
__global__ void __launch_bounds__(256)
k_recover_ordered(MeshDev md, const int* __restrict__ cps, const int* __restrict__ cpi, const int* __restrict__ pair_atom,
                  const float* __restrict__ Cd, int npj, const float* __restrict__ Wcat, long ldwc, const float* __restrict__ RY,
                  long ldw, float* __restrict__ X, long ldx, int Wr, const double* __restrict__ lamY) {
  constexpr int cw = CPLX ? 2 : 1;
  const int n = md.n, n1 = md.n1, p = md.p;
  const int e = blockIdx.x;
  int cc[3];
  mesh_cell_coords(md, e, &cc[0], &cc[1], &cc[2]);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int v = blockIdx.y * 128 + lane * 4;
  if (v >= Wr) return;
  double lam[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) lam[u] = v + u < Wr ? lamY[(v + u) / cw] : 0.0;
  const bool last[3] = {!md.periodic && cc[0] == md.nc[0] - 1, !md.periodic && cc[1] == md.nc[1] - 1, !md.periodic && cc[2] == md.nc[2] - 1};
  for (int I = w; I < n; I += 8) {
    const int loc[3] = {I / (n1 * n1), (I / n1) % n1, I % n1};
    if ((loc[0] == p && !last[0]) || (loc[1] == p && !last[1]) || (loc[2] == p && !last[2])) continue;   // another cell owns it
    int ix, iy, iz;
    const long J = mesh_node(md, cc[0], cc[1], cc[2], loc[0], loc[1], loc[2], &ix, &iy, &iz);
    const double mi = md.mdinv1[0][ix] * md.mdinv1[1][iy] * md.mdinv1[2][iz];
    float* xp = X + J * ldx + v;
    float xo[4] = {0.f, 0.f, 0.f, 0.f};
    if (mi != 0.0) {   // (Dirichlet wall rows are written as 0)
      const float4 ry = *reinterpret_cast<const float4*>(RY + J * ldw + v);   // ldw % 4 == 0, pad columns readable
      float xi[4];
      if (VEC) { const float4 t = *reinterpret_cast<const float4*>(xp); xi[0] = t.x; xi[1] = t.y; xi[2] = t.z; xi[3] = t.w; }
      else {
#pragma unroll
        for (int u = 0; u < 4; ++u) xi[u] = v + u < Wr ? xp[u] : 0.f;
      }
      xo[0] = (float)((double)ry.x + (double)xi[0] * lam[0]); xo[1] = (float)((double)ry.y + (double)xi[1] * lam[1]);
      xo[2] = (float)((double)ry.z + (double)xi[2] * lam[2]); xo[3] = (float)((double)ry.w + (double)xi[3] * lam[3]);
      const float s = -(float)mi;
      for (int oct = 0; oct < 8; ++oct) {
        const int d[3] = {oct & 1, (oct >> 1) & 1, (oct >> 2) & 1};
        if ((d[0] && loc[0] != 0) || (d[1] && loc[1] != 0) || (d[2] && loc[2] != 0)) continue;   // the node is not on that face
        int c2[3], l2[3];
        bool ok = true;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          c2[k] = cc[k] - d[k];
          l2[k] = d[k] ? p : loc[k];
          if (c2[k] < 0) { if (md.periodic) c2[k] += md.nc[k]; else ok = false; }
        }
        if (!ok) continue;
        const int e2 = (c2[0] * md.nc[1] + c2[1]) * md.nc[2] + c2[2];
        const int I2 = (l2[0] * n1 + l2[1]) * n1 + l2[2];
        for (int q = cps[e2]; q < cps[e2 + 1]; ++q) {
          const int pr = cpi[q], at = pair_atom[pr];
          float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
          for (int al = 0; al < npj; ++al) {
            const float4 wv = *reinterpret_cast<const float4*>(Wcat + ((long)at * 32 + al) * ldwc + v);
            if (CPLX) {   // conj(Cd) * W on interleaved (re, im) columns
              const float2 cv = *reinterpret_cast<const float2*>(Cd + (((long)pr * npj + al) * n + I2) * 2);
              acc.x = fmaf(cv.x, wv.x, acc.x); acc.x = fmaf(cv.y, wv.y, acc.x);
              acc.y = fmaf(cv.x, wv.y, acc.y); acc.y = fmaf(-cv.y, wv.x, acc.y);
              acc.z = fmaf(cv.x, wv.z, acc.z); acc.z = fmaf(cv.y, wv.w, acc.z);
              acc.w = fmaf(cv.x, wv.w, acc.w); acc.w = fmaf(-cv.y, wv.z, acc.w);
            } else {
              const float cv = Cd[((long)pr * npj + al) * n + I2];
              acc.x = fmaf(cv, wv.x, acc.x); acc.y = fmaf(cv, wv.y, acc.y);
              acc.z = fmaf(cv, wv.z, acc.z); acc.w = fmaf(cv, wv.w, acc.w);
            }
          }
          xo[0] += s * acc.x; xo[1] += s * acc.y; xo[2] += s * acc.z; xo[3] += s * acc.w;
        }
      }
    }
    if (VEC) *reinterpret_cast<float4*>(xp) = make_float4(xo[0], xo[1], xo[2], xo[3]);
    else {
#pragma unroll
      for (int u = 0; u < 4; ++u) if (v + u < Wr) xp[u] = xo[u];
    }
  }
}

void free_plan(FusedPlan* p) {
  if (!p) return;
  cudaFree(p->d_ext_start); cudaFree(p->d_ext_atom); cudaFree(p->d_Bext);
  cudaFree(p->d_nb_start); cudaFree(p->d_nb_atom); cudaFree(p->d_GD); cudaFree(p->d_cps); cudaFree(p->d_cpi); cudaFree(p->d_pcells);
  cudaFree(p->d_P1); cudaFree(p->d_Ppart); cudaFree(p->d_Wcat); cudaFree(p->d_P64); cudaFree(p->d_W64);
  cudaFree(p->d_Wcat_lo); cudaFree(p->d_Bext_lo); cudaFree(p->d_xlo); cudaFree(p->d_CdF);
  if (p->aux) cudaStreamDestroy(p->aux);
  if (p->ev_fork) cudaEventDestroy(p->ev_fork);
  if (p->ev_join) cudaEventDestroy(p->ev_join);
  delete p;
}

pawfe_status build_plan(pawfe_ctx* c, FusedPlan* p) {
  const int ncell = c->ncell, natoms = c->natoms, npj = c->npj, n = c->n;
  const bool per = c->bc == PAWFE_PERIODIC;
  // host copies of the pair list
  std::vector<int> pc(c->npairs), pa(c->npairs);
  if (c->npairs) {
    CUDA_TRY(c, cudaMemcpy(pc.data(), c->d_pair_cell, c->npairs * sizeof(int), cudaMemcpyDeviceToHost));
    CUDA_TRY(c, cudaMemcpy(pa.data(), c->d_pair_atom, c->npairs * sizeof(int), cudaMemcpyDeviceToHost));
  }
  // cell -> pairs
  std::vector<int> cps(ncell + 1, 0), cpi(c->npairs);
  for (long q = 0; q < c->npairs; ++q) cps[pc[q] + 1]++;
  for (int e = 0; e < ncell; ++e) cps[e + 1] += cps[e];
  {
    std::vector<int> fill(cps.begin(), cps.end() - 1);
    for (long q = 0; q < c->npairs; ++q) cpi[fill[pc[q]]++] = (int)q;
  }
  {
    std::vector<int> pcs;
    for (int e = 0; e < ncell; ++e) if (cps[e + 1] > cps[e]) pcs.push_back(e);
    p->npcells = (int)pcs.size();
    if (!pcs.empty()) TRY(upload(c, &p->d_pcells, pcs));
  }
  // K-extension entries: every cell sharing a node with a pair cell of the atom (the pair cells and their 26 neighbours)
  std::vector<std::vector<int>> cell_atoms(ncell);
  for (int a = 0; a < natoms; ++a) {
    std::set<int> cells;
    for (int q = c->h_atom_pair_start[a]; q < c->h_atom_pair_start[a + 1]; ++q) {
      int cx, cy, cz;
      mesh_cell_coords(c->md, pc[q], &cx, &cy, &cz);
      for (int dx = -1; dx <= 1; ++dx)
        for (int dy = -1; dy <= 1; ++dy)
          for (int dz = -1; dz <= 1; ++dz) {
            int x = cx + dx, y = cy + dy, z = cz + dz;
            if (per) { x = (x + c->nc[0]) % c->nc[0]; y = (y + c->nc[1]) % c->nc[1]; z = (z + c->nc[2]) % c->nc[2]; }
            else if (x < 0 || y < 0 || z < 0 || x >= c->nc[0] || y >= c->nc[1] || z >= c->nc[2]) continue;
            cells.insert((x * c->nc[1] + y) * c->nc[2] + z);
          }
    }
    for (int e : cells) cell_atoms[e].push_back(a);
  }
  std::vector<int> es(ncell + 1, 0), ea, ec;
  for (int e = 0; e < ncell; ++e) {
    for (int a : cell_atoms[e]) { ea.push_back(a); ec.push_back(e); }
    es[e + 1] = (int)ea.size();
  }
  p->nchunks = (long)ea.size();
  // neighbour atoms: b in nb(a) iff some pair cell of a is an extension cell of b
  std::vector<std::set<int>> nbs(natoms);
  for (int e = 0; e < ncell; ++e)
    for (int q = cps[e]; q < cps[e + 1]; ++q)
      for (int b : cell_atoms[e]) nbs[pa[cpi[q]]].insert(b);
  std::vector<int> ns(natoms + 1, 0), na;
  for (int a = 0; a < natoms; ++a) { for (int b : nbs[a]) na.push_back(b); ns[a + 1] = (int)na.size(); }
  const long nnb = (long)na.size();
  p->ext_ksteps = (2 * npj + 7) / 8;
  if (p->nchunks == 0) {   // no atoms near any cell: only the cell -> pairs lists (all empty) are needed, by the recovery kernel
    TRY(upload(c, &p->d_cps, cps)); TRY(upload(c, &p->d_cpi, cpi));
    p->ok = true; return PAWFE_OK;
  }

  int* d_ec = nullptr;
  int *&d_cps = p->d_cps, *&d_cpi = p->d_cpi;   // kept: the ordered recovery kernel walks the cells' pairs
  double* d_G = nullptr;
  pawfe_status st = PAWFE_OK;
  auto cleanup = [&]() { cudaFree(d_ec); cudaFree(d_G); };
#define TRYP(xx) do { st = (xx); if (st != PAWFE_OK) { cleanup(); return st; } } while (0)
  TRYP(upload(c, &p->d_ext_start, es)); TRYP(upload(c, &p->d_ext_atom, ea)); TRYP(upload(c, &d_ec, ec));
  TRYP(upload(c, &d_cps, cps)); TRYP(upload(c, &d_cpi, cpi));
  TRYP(upload(c, &p->d_nb_start, ns)); TRYP(upload(c, &p->d_nb_atom, na));
  int NH = 1, NT = n;
  tc_shape(c, &NH, &NT);
  const int cw = c->cplx ? 2 : 1;
  const size_t per2 = (size_t)npj * npj;
  const size_t bext_elems = (size_t)p->nchunks * NH * NT * 32 * cw;
  TRYP(dev_alloc(c, &p->d_Bext, bext_elems));
  cudaMemsetAsync(p->d_Bext, 0, bext_elems * sizeof(float), c->stream);
  TRYP(dev_alloc(c, &d_G, (size_t)nnb * per2 * cw));
  cudaMemsetAsync(d_G, 0, (size_t)nnb * per2 * cw * sizeof(double), c->stream);
  size_t smem = (size_t)n * npj * sizeof(double) * cw;
  cudaError_t e;
  if (c->cplx) {
    e = cudaFuncSetAttribute(k_build_ext<double2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess)
      k_build_ext<double2><<<(unsigned)p->nchunks, 256, smem, c->stream>>>(
          c->md, d_ec, p->d_ext_atom, c->d_atom_pair_start, c->d_pair_cell, (const double2*)c->d_Cd64, npj,
          (const double2*)c->d_H64, d_cps, d_cpi, c->d_pair_atom, p->d_nb_start, p->d_nb_atom, NH, NT, p->d_Bext, (double2*)d_G);
  } else {
    e = cudaFuncSetAttribute(k_build_ext<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess)
      k_build_ext<double><<<(unsigned)p->nchunks, 256, smem, c->stream>>>(
          c->md, d_ec, p->d_ext_atom, c->d_atom_pair_start, c->d_pair_cell, (const double*)c->d_Cd64, npj,
          (const double*)c->d_H64, d_cps, d_cpi, c->d_pair_atom, p->d_nb_start, p->d_nb_atom, NH, NT, p->d_Bext, d_G);
  }
  if (e == cudaSuccess) { c->launches++; e = cudaGetLastError(); }
  std::vector<double> G((size_t)nnb * per2 * cw);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e == cudaSuccess) e = cudaMemcpy(G.data(), d_G, G.size() * sizeof(double), cudaMemcpyDeviceToHost);
  cleanup();
  if (e != cudaSuccess) { c->err = std::string("fused plan build: ") + cudaGetErrorString(e); return PAWFE_ECUDA; }
#undef TRYP
  // GD^{ab} = G^{ab} Delta^b_Sinv (complex arithmetic when cw = 2); cross-check the diagonal blocks against G^a of atoms_create
  std::vector<float> GD((size_t)nnb * per2 * cw);
  for (int a = 0; a < natoms; ++a)
    for (int s = ns[a]; s < ns[a + 1]; ++s) {
      const int b = na[s];
      const double* g = &G[(size_t)s * per2 * cw];
      if (b == a) {
        double dmax = 0, gmax = 0;
        for (size_t i = 0; i < per2 * cw; ++i) { dmax = std::max(dmax, std::fabs(g[i] - c->h_G[a * per2 * cw + i])); gmax = std::max(gmax, std::fabs(g[i])); }
        if (dmax > 1e-9 * std::max(gmax, 1e-300)) { c->err = "fused plan: G^{aa} from the extension blocks disagrees with atoms_create"; return PAWFE_ECUDA; }
      }
      const double* si = &c->h_dSinv[(size_t)b * per2 * cw];
      for (int i = 0; i < npj; ++i)
        for (int j = 0; j < npj; ++j) {
          double tr = 0, ti = 0;
          for (int k = 0; k < npj; ++k) {
            const double gr = g[(i * npj + k) * cw], gi = cw == 2 ? g[(i * npj + k) * cw + 1] : 0.0;
            const double sr = si[(k * npj + j) * cw], sim = cw == 2 ? si[(k * npj + j) * cw + 1] : 0.0;
            tr += gr * sr - gi * sim; ti += gr * sim + gi * sr;
          }
          GD[((size_t)s * per2 + i * npj + j) * cw] = (float)tr;
          if (cw == 2) GD[((size_t)s * per2 + i * npj + j) * cw + 1] = (float)ti;
        }
    }
  TRY(upload(c, &p->d_GD, GD));
  p->ok = true;
  return PAWFE_OK;
}

// Scratch of the fused path for blocks of up to Bvec vectors: projections, couplings (and their low parts for the FP32
// mode), FP64 projections of the residual set-up.  Grows on the first call and when a wider block arrives (stream
// synchronisation + allocation: pawfe_prepare does this ahead of the hot calls).
pawfe_status ensure_scratch(pawfe_ctx* c, FusedPlan* p, int Bvec) {
  const int B = Bvec * (c->cplx ? 2 : 1);   // real columns
  if (B <= p->Bcap) return PAWFE_OK;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  if (p->aux) CUDA_TRY(c, cudaStreamSynchronize(p->aux));
  cudaFree(p->d_P1); cudaFree(p->d_Ppart); cudaFree(p->d_Wcat); cudaFree(p->d_P64); cudaFree(p->d_W64); cudaFree(p->d_Wcat_lo);
  p->d_Wcat_lo = nullptr; p->d_Ppart = nullptr;
  p->d_P1 = p->d_Wcat = nullptr; p->d_P64 = p->d_W64 = nullptr; p->Bcap = 0;
  const long ldw = roundup4(B);
  const size_t na = (size_t)std::max(1, c->natoms);
  TRY(dev_alloc(c, &p->d_P1, na * c->npj * ldw));
  TRY(dev_alloc(c, &p->d_Ppart, (size_t)std::max<long>(1, c->npairs) * c->npj * ldw));
  TRY(dev_alloc(c, &p->d_Wcat, na * 32 * ldw));
  TRY(dev_alloc(c, &p->d_Wcat_lo, na * 32 * ldw));
  TRY(dev_alloc(c, &p->d_P64, na * c->npj * ldw));
  TRY(dev_alloc(c, &p->d_W64, na * c->npj * ldw));
  CUDA_TRY(c, cudaMemsetAsync(p->d_Wcat, 0, na * 32 * ldw * sizeof(float), c->stream));
  p->Bcap = B; p->ldw = ldw;
  return PAWFE_OK;
}

// a block-sized scratch array of the plan (low parts / scaled copy of an apply's input block)
pawfe_status ensure_block(pawfe_ctx* c, FusedPlan* p, float** buf, size_t* have, size_t want) {
  if (*have >= want) return PAWFE_OK;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  cudaFree(*buf); *buf = nullptr; *have = 0;
  TRY(dev_alloc(c, buf, want));
  *have = want;
  return PAWFE_OK;
}

// P1 = C^T X (X already in the scaled variables), then the couplings in `mode` (see k_couple).
// X: the block as floats (complex: interleaved), ldx in floats; B vectors.
// the fragment-ordered TF32 copy of the projector blocks (n <= 512): built on the first TF32 projection of a
// plan, or ahead of the hot calls by pawfe_prepare(PAWFE_TF32, ..)
bool proj_mma_usable(const pawfe_ctx* c, const FusedPlan* p) { return c->n <= 512 && p->npcells > 0; }
pawfe_status ensure_cdf(pawfe_ctx* c, FusedPlan* p) {
  if (p->d_CdF || !proj_mma_usable(c, p)) return PAWFE_OK;
  const int nks = (c->n + 7) / 8;
  const int cw = c->cplx ? 2 : 1;
  const long total = (long)c->npairs * nks * cw * 32;
  TRY(dev_alloc(c, &p->d_CdF, (size_t)total));
  k_build_cdf<<<8 * c->sm_count, 256, 0, c->stream>>>(total, c->npj, c->n, nks, cw, (const float*)c->d_Cd32, p->d_CdF);
  KERNEL_CHECK(c, "k_build_cdf");
  return PAWFE_OK;
}

// tf32: the caller multiplies in TF32 (PAWFE_TF32 mode): a real context then projects on the tensor cores (k_proj_cell_mma).
pawfe_status project_and_couple(pawfe_ctx* c, FusedPlan* p, bool tf32, const float* X, long ldx, int B, int mode) {
  if (c->npairs == 0) return PAWFE_OK;
  const int n = c->n, npj = c->npj;
  // per-pair partial projections, then their sum in pair order (no cross-CTA reductions: bit-reproducible)
  auto psum = [&](int Wr) -> pawfe_status {
    const int Wq = (Wr + 3) / 4;
    k_psum<<<dim3((unsigned)(c->natoms * npj), ceil_div(Wq, 128)), 128, 0, c->stream>>>(
        npj, c->d_atom_pair_start, (const float4*)p->d_Ppart, p->ldw / 4, Wq, (float4*)p->d_P1);
    KERNEL_CHECK(c, "k_psum");
    return PAWFE_OK;
  };
  // Cell-parallel projection into per-pair partials (every pair belongs to exactly one cell of the list).  It replaced round
  // 1's pair-parallel kernels, which read a cell's rows once per pair (profiles/r02_projection_kernels.md, configs 1 / 2 / 3 / 4:
  // 0.29 / 3.15 / 1.76 / 7.65 ms per step -> FP32 FMA 0.27 / 2.59 / 1.24 / 4.45 -> tensor cores 0.20 / 1.59 / 0.93 / 2.33).
  const int Wr = B * (c->cplx ? 2 : 1);
  if (tf32 && proj_mma_usable(c, p)) {
    TRY(ensure_cdf(c, p));
    const dim3 grid((unsigned)p->npcells, ceil_div(Wr, kPcVT));
#define LAUNCH_PM(N, J)                                                                                                     \
    do {                                                                                                                    \
      if (c->cplx) {                                                                                                        \
        TRY(pawfe_ensure_smem(c, (const void*)k_proj_cell_mma<N, J, true>, smem));                                          \
        k_proj_cell_mma<N, J, true><<<grid, 256, smem, c->stream>>>(c->md, p->d_pcells, p->d_cps, p->d_cpi, p->d_CdF, X, ldx,    \
                                                                    Wr, p->d_Ppart, p->ldw);                                \
      } else {                                                                                                              \
        TRY(pawfe_ensure_smem(c, (const void*)k_proj_cell_mma<N, J, false>, smem));                                         \
        k_proj_cell_mma<N, J, false><<<grid, 256, smem, c->stream>>>(c->md, p->d_pcells, p->d_cps, p->d_cpi, p->d_CdF, X, ldx,   \
                                                                     Wr, p->d_Ppart, p->ldw);                               \
      }                                                                                                                     \
    } while (0)
#define CASE_PM(N)                                                                                                          \
    case N: {                                                                                                               \
      const size_t smem = proj_cell_mma_smem<N>(n);                                                                         \
      if (n <= 384) LAUNCH_PM(N, 6); else LAUNCH_PM(N, 8);                                                                  \
    } break;
    switch (npj) {
      CASE_PM(1) CASE_PM(2) CASE_PM(3) CASE_PM(4) CASE_PM(5) CASE_PM(6) CASE_PM(7) CASE_PM(8)
      CASE_PM(9) CASE_PM(10) CASE_PM(11) CASE_PM(12) CASE_PM(13) CASE_PM(14) CASE_PM(15) CASE_PM(16)
    }
#undef LAUNCH_PM
#undef CASE_PM
    KERNEL_CHECK(c, "k_proj_cell_mma");
  } else if (p->npcells > 0) {
    const dim3 grid((unsigned)p->npcells, ceil_div(Wr, kPcVT));
#define LAUNCH_PC(N, CP)                                                                                                   \
    do {                                                                                                                    \
      const size_t smem = proj_cell_smem<N, CP>(n);                                                                         \
      TRY(pawfe_ensure_smem(c, (const void*)k_proj_cell<N, CP>, smem));                                                     \
      k_proj_cell<N, CP><<<grid, 256, smem, c->stream>>>(c->md, p->d_pcells, p->d_cps, p->d_cpi, (const float*)c->d_Cd32,        \
                                                          (long)c->npairs * N * n * (CP ? 2 : 1), X, ldx, Wr, p->d_Ppart, p->ldw); \
    } while (0)
#define CASE_PC(N) case N: if (c->cplx) LAUNCH_PC(N, true); else LAUNCH_PC(N, false); break;
    switch (npj) {
      CASE_PC(1) CASE_PC(2) CASE_PC(3) CASE_PC(4) CASE_PC(5) CASE_PC(6) CASE_PC(7) CASE_PC(8)
      CASE_PC(9) CASE_PC(10) CASE_PC(11) CASE_PC(12) CASE_PC(13) CASE_PC(14) CASE_PC(15) CASE_PC(16)
    }
#undef CASE_PC
#undef LAUNCH_PC
    KERNEL_CHECK(c, "k_proj_cell");
  }
  if (c->cplx) {
    TRY(psum(2 * B));
    const int Bpad = (int)(roundup4(2 * B) / 2);
    k_couple<float2><<<dim3(c->natoms, ceil_div(Bpad, kCoupleLanes)), kCoupleLanes * npj, 0, c->stream>>>(
        npj, mode, (const float2*)p->d_P1, p->ldw / 2, B, Bpad, (const float2*)c->d_dSinv32, (const float2*)c->d_D32, p->d_nb_start,
        p->d_nb_atom, (const float2*)p->d_GD, (float2*)p->d_Wcat, p->ldw / 2);
    KERNEL_CHECK(c, "k_couple");
    return PAWFE_OK;
  }
  TRY(psum(B));
  const int Bpad = (int)roundup4(B);
  k_couple<float><<<dim3(c->natoms, ceil_div(Bpad, kCoupleLanes)), kCoupleLanes * npj, 0, c->stream>>>(
      npj, mode, p->d_P1, p->ldw, B, Bpad, (const float*)c->d_dSinv32, (const float*)c->d_D32, p->d_nb_start, p->d_nb_atom,
      p->d_GD, p->d_Wcat, p->ldw);
  KERNEL_CHECK(c, "k_couple");
  return PAWFE_OK;
}

// Y += C (D P - dS P Lambda), P = C^T X, all FP64 (non-local parts of H X - S X Lambda with one projection)
template <int NPJ>
pawfe_status setup_nonlocal64_t(pawfe_ctx* c, FusedPlan* p, const float* X, long ldx, int B, const double* lam,
                                double* Y, long ldy) {
  const int n = c->n;
  CUDA_TRY(c, cudaMemsetAsync(p->d_P64, 0, (size_t)c->natoms * NPJ * p->ldw * sizeof(double), c->stream));
  dim3 grid((unsigned)c->npairs, ceil_div(B, 64));
  {
    const size_t smem = (size_t)n * 8 + (size_t)NPJ * n * 8 + 8 + (size_t)NPJ * 64 * 8;
    TRY(pawfe_ensure_smem(c, (const void*)k_proj64<NPJ, float>, smem));
    k_proj64<NPJ, float><<<grid, 256, smem, c->stream>>>(c->md, c->d_pair_cell, c->d_pair_atom, (const double*)c->d_Cd64, X, ldx, B, p->d_P64, p->ldw);
    KERNEL_CHECK(c, "k_proj64");
  }
  k_couple64<<<dim3(c->natoms, ceil_div(B, 128)), 128, 0, c->stream>>>(NPJ, p->d_P64, p->ldw, B, (const double*)c->d_D64,
                                                                       (const double*)c->d_dS64, lam, p->d_W64);
  KERNEL_CHECK(c, "k_couple64");
  {
    const size_t smem = (size_t)n * 8 + (size_t)NPJ * n * 8;
    TRY(pawfe_ensure_smem(c, (const void*)k_scatter64<NPJ>, smem));
    k_scatter64<NPJ><<<grid, 256, smem, c->stream>>>(c->md, c->d_pair_cell, c->d_pair_atom, (const double*)c->d_Cd64, p->d_W64, p->ldw, B, Y, ldy);
    KERNEL_CHECK(c, "k_scatter64");
  }
  return PAWFE_OK;
}
pawfe_status setup_nonlocal64(pawfe_ctx* c, FusedPlan* p, const float* X, long ldx, int B, const double* lam, double* Y, long ldy) {
  switch (c->npj) {
#define CASE_NL(N) case N: return setup_nonlocal64_t<N>(c, p, X, ldx, B, lam, Y, ldy);
    CASE_NL(1) CASE_NL(2) CASE_NL(3) CASE_NL(4) CASE_NL(5) CASE_NL(6) CASE_NL(7) CASE_NL(8)
    CASE_NL(9) CASE_NL(10) CASE_NL(11) CASE_NL(12) CASE_NL(13) CASE_NL(14) CASE_NL(15) CASE_NL(16)
#undef CASE_NL
  }
  return PAWFE_EINVAL;
}

TcExt make_ext(const FusedPlan* p, int scale_mode) {
  TcExt x;
  x.scale_mode = scale_mode; x.nchunks = p->nchunks; x.ext_start = p->d_ext_start; x.ext_atom = p->d_ext_atom;
  x.Bext = p->d_Bext; x.Wcat = p->d_Wcat; x.ldw = p->ldw; x.ksteps = p->ext_ksteps;
  x.Hstream = nullptr;
  return x;
}

}  // namespace

void fused_invalidate(pawfe_ctx* c) {
  if (c->fused) { free_plan((FusedPlan*)c->fused); c->fused = nullptr; }
}

bool fused_supported(pawfe_ctx* c, pawfe_prec prec, int B) {
  return (prec == PAWFE_TF32 || prec == PAWFE_FP32) && c->have_h64 && c->have_atoms && tc_supported(c, B) && 2 * c->npj <= 32;
}

// run work on the plan's auxiliary stream, ordered after everything enqueued so far on the context's stream
#define FORK_AUX(c, p) do { if ((p)->no_aux) break; CUDA_TRY(c, cudaEventRecord((p)->ev_fork, (c)->stream)); CUDA_TRY(c, cudaStreamWaitEvent((p)->aux, (p)->ev_fork, 0)); } while (0)
#define JOIN_AUX(c, p) do { if ((p)->no_aux) break; CUDA_TRY(c, cudaEventRecord((p)->ev_join, (p)->aux)); CUDA_TRY(c, cudaStreamWaitEvent((c)->stream, (p)->ev_join, 0)); } while (0)
struct StreamSwap {   // kernels launched while this lives go to `s`
  pawfe_ctx* c; cudaStream_t keep;
  StreamSwap(pawfe_ctx* c_, cudaStream_t s) : c(c_), keep(c_->stream) { c->stream = s; }
  ~StreamSwap() { c->stream = keep; }
};

pawfe_status fused_prepare(pawfe_ctx* c, int B) {
  FusedPlan* p = (FusedPlan*)c->fused;
  if (!p) {
    TRY(tc_prepare(c));
    p = new FusedPlan();
    c->fused = p;
    // highest priority: the auxiliary kernels are short and latency-bound; their CTAs should take every slot that frees up
    // next to the long kernel of the main stream instead of queueing behind its whole grid
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    if (cudaStreamCreateWithPriority(&p->aux, cudaStreamNonBlocking, prio_hi) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming) != cudaSuccess) {
      cudaGetLastError(); fused_invalidate(c); c->err = "fused plan: stream / event creation failed"; return PAWFE_ECUDA;
    }
    p->no_aux = getenv("PAWFE_NO_AUX") != nullptr;   // read once, here: everything on the context's stream (timing experiments)
    pawfe_status st = build_plan(c, p);
    if (st != PAWFE_OK) { fused_invalidate(c); return st; }
  }
  return ensure_scratch(c, p, B);
}

// Everything the fused path allocates lazily, now: plan, scratch for blocks of up to B vectors, and for PAWFE_FP32 the low
// parts of the operand streams and a block-sized scratch; with_block: the block-sized scratch of pawfe_apply_HSinv too.
pawfe_status fused_prepare_all(pawfe_ctx* c, pawfe_prec prec, int B, bool with_block) {
  TRY(fused_prepare(c, B));
  FusedPlan* p = (FusedPlan*)c->fused;
  const size_t blk = (size_t)c->M * roundup4((long)B * (c->cplx ? 2 : 1));
  if (prec == PAWFE_FP32) {
    const float* hlo = nullptr;
    TRY(tc_hstream_lo(c, &hlo));
    if (p->nchunks > 0 && !p->d_Bext_lo) {
      int NH = 1, NT = c->n;
      tc_shape(c, &NH, &NT);
      const size_t cnt = (size_t)p->nchunks * NH * NT * 32 * (c->cplx ? 2 : 1);
      TRY(dev_alloc(c, &p->d_Bext_lo, cnt));
      TRY(tc_lo_part(c, p->d_Bext, p->d_Bext_lo, (long)cnt));
    }
    if (with_block) TRY(ensure_block(c, p, &p->d_xlo, &p->xlo_elems, blk));
  }
  if (prec == PAWFE_TF32) TRY(ensure_cdf(c, p));
  if (with_block) TRY(ensure_block(c, p, &p->d_xs, &p->xs_elems, blk));
  return PAWFE_OK;
}

// One cell-level pass: Y <- epi(alpha [M_D^-1] (H_loc X + K-extension terms)).  TF32: one launch.  FP32 (PAPER.md:L374
// "FP32"): three launches with the operands split into the part the tensor core keeps (hi = trunc_tf32) and the rest (lo):
//   hi x hi + lo x hi + hi x lo   (the dropped lo x lo term is ~2^-22 relative), FP32 accumulation throughout;
// the first launch runs the caller's epilogue, the other two add to its result.
// xlo: scratch for the low parts of X (same shape).  Wcat holds the couplings of this step.
pawfe_status cell_pass(pawfe_ctx* c, FusedPlan* p, pawfe_prec prec, const float* X, long ldx, float* Y, long ldy, int B,
                       float alpha, int scale_mode, const TcEpi& epi, float* xlo) {
  TcExt x = make_ext(p, scale_mode);
  prof_begin(c);
  pawfe_status st = tc_cell_apply(c, X, ldx, Y, ldy, B, alpha, &x, &epi);
  if (st == PAWFE_OK && prec == PAWFE_FP32) {
    const float* hlo = nullptr;
    st = tc_hstream_lo(c, &hlo);
    if (st == PAWFE_OK && p->nchunks > 0 && !p->d_Bext_lo) {   // first FP32-mode use without pawfe_prepare
      int NH = 1, NT = c->n;
      tc_shape(c, &NH, &NT);
      const size_t cnt = (size_t)p->nchunks * NH * NT * 32 * (c->cplx ? 2 : 1);
      st = dev_alloc(c, &p->d_Bext_lo, cnt);
      if (st == PAWFE_OK) st = tc_lo_part(c, p->d_Bext, p->d_Bext_lo, (long)cnt);
    }
    if (st == PAWFE_OK) st = tc_lo_part(c, X, xlo, c->M * ldx);
    if (st == PAWFE_OK && c->natoms > 0) st = tc_lo_part(c, p->d_Wcat, p->d_Wcat_lo, (long)c->natoms * 32 * p->ldw);
    TcEpi add; add.mode = TC_EPI_ADD; add.Yt = nullptr; add.aLam = nullptr; add.ac = add.zz1 = 0.f; add.cw = 1;
    if (st == PAWFE_OK) {           // lo(X) x hi(H)
      TcExt x2 = x; x2.Wcat = p->d_Wcat_lo;
      st = tc_cell_apply(c, xlo, ldx, Y, ldy, B, alpha, &x2, &add);
    }
    if (st == PAWFE_OK) {           // hi(X) x lo(H)
      TcExt x3 = x; x3.Bext = p->d_Bext_lo; x3.Hstream = hlo;
      st = tc_cell_apply(c, X, ldx, Y, ldy, B, alpha, &x3, &add);
    }
  }
  prof_end(c);
  return st;
}

static TcEpi epi_plain(int mode) {
  TcEpi e; e.mode = mode; e.Yt = nullptr; e.aLam = nullptr; e.ac = e.zz1 = 0.f; e.cw = 1;
  return e;
}

// Y = H X: every row of Y is stored by its first writer (no zero-fill), the non-local term rides in the K-extension
pawfe_status fused_apply_H(pawfe_ctx* c, pawfe_prec prec, const float* X, long ldx, float* Y, long ldy, int B) {
  TRY(fused_prepare(c, B));
  FusedPlan* p = (FusedPlan*)c->fused;
  if (prec == PAWFE_FP32) TRY(ensure_block(c, p, &p->d_xlo, &p->xlo_elems, (size_t)c->M * ldx));
  const int Wr = B * (c->cplx ? 2 : 1);   // X, Y as float blocks: ldx, ldy in floats, Wr real columns
  TRY(project_and_couple(c, p, prec == PAWFE_TF32, X, ldx, B, 2));
  return cell_pass(c, p, prec, X, ldx, Y, ldy, Wr, 1.0f, 0, epi_plain(TC_EPI_STORE), p->d_xlo);
}

// Y = H S^-1approx X (the operator the filter iterates, Alg. 1 step 2 L244 / Eq. 30) in exactly the kernel
// configuration of the filter's step: Xs = M_D^-1 X, P1 = C^T Xs, couplings W / W2, one cell pass with both halves of
// the K-extension.  X, Y as float blocks (complex: interleaved; ldx, ldy in floats).
pawfe_status fused_apply_HSinv(pawfe_ctx* c, pawfe_prec prec, const float* X, long ldx, float* Y, long ldy, int B) {
  TRY(fused_prepare(c, B));
  FusedPlan* p = (FusedPlan*)c->fused;
  const int Wr = B * (c->cplx ? 2 : 1);
  const long lds = roundup4(Wr);
  TRY(ensure_block(c, p, &p->d_xs, &p->xs_elems, (size_t)c->M * lds));
  if (prec == PAWFE_FP32) TRY(ensure_block(c, p, &p->d_xlo, &p->xlo_elems, (size_t)c->M * lds));
  if (lds != Wr) CUDA_TRY(c, cudaMemsetAsync(p->d_xs, 0, (size_t)c->M * lds * sizeof(float), c->stream));   // pad columns
  k_scale_mdinv_f4<<<8 * c->sm_count, 256, 0, c->stream>>>(c->md, (const float4*)X, ldx / 4, (float4*)p->d_xs, lds / 4, Wr / 4);
  KERNEL_CHECK(c, "k_scale_mdinv_f4");
  TRY(project_and_couple(c, p, prec == PAWFE_TF32, p->d_xs, lds, B, 0));
  return cell_pass(c, p, prec, p->d_xs, lds, Y, ldy, Wr, 1.0f, 0, epi_plain(TC_EPI_STORE), p->d_xlo);
}

// Step 2 of Alg. 2 for real contexts (L260, L374), FP64, S X never stored:  Yt <- H X - S X Lambda  (unscaled; the caller
// scales).  The DMMA product runs on the context's stream, the mass sweeps and the FP64 non-local part (both add into Yt
// with FP64 atomics) on the auxiliary stream; on any failure the auxiliary stream is joined before returning.
static pawfe_status residual_setup_real(pawfe_ctx* c, FusedPlan* p, const float* X, long ld, int B, double* Yt, long ldw,
                                        const double* lam, const double* neg_lam) {
  CUDA_TRY(c, cudaMemsetAsync(Yt, 0, (size_t)c->M * ldw * sizeof(double), c->stream));
  FORK_AUX(c, p);                                                 // Yt is zero from here on for both streams
  pawfe_status st = pawfe_cell_product_fp64<float>(c, X, ld, Yt, ldw, B);
  {
    StreamSwap sw(c, p->no_aux ? c->stream : p->aux);
    if (st == PAWFE_OK) {
      const size_t smem = (size_t)c->n * kMassCT * 8 + (size_t)c->n * 8;
      st = pawfe_ensure_smem(c, (const void*)k_mass_sf<float, kMassCT>, smem);
      if (st == PAWFE_OK) {
        k_mass_sf<float, kMassCT><<<dim3(c->ncell, ceil_div(B, kMassCT)), 256, smem, c->stream>>>(
            c->md, c->d_M1, c->h[0] * c->h[1] * c->h[2] / 8.0, X, ld, Yt, ldw, B, neg_lam);
        c->launches++;
        if (cudaGetLastError() != cudaSuccess) { c->err = "k_mass_sf launch failed"; st = PAWFE_ECUDA; }
      }
    }
    if (st == PAWFE_OK && c->npairs > 0) st = setup_nonlocal64(c, p, X, ld, B, lam, Yt, ldw);
  }
  if (st != PAWFE_OK) { if (!p->no_aux) cudaStreamSynchronize(p->aux); return st; }
  JOIN_AUX(c, p);
  return PAWFE_OK;
}

// X: the block in the context's FP32 storage scalar (float, or float2 interleaved), ld and B in those scalars.  Inside, every
// array is a real block of Wr = B * cw columns (cw = 2 for complex contexts) with leading dimension ldw = roundup4(Wr).
// HX, SX: null (step 2 computed here, L260) or the caller's FP64 blocks H X and S X in X's layout (leading dimension ld,
// FP64 scalars): step 2 is then Y = HX - SX Lambda without any operator application (pawfe_cheb_filter_hs).
pawfe_status fused_filter(pawfe_ctx* c, pawfe_prec prec, int m, const double* ds, const double* as, const double* acs,
                          const double* zzs, double z_over_e, void* Xv, long ld, int B, void* workspace,
                          const void* HX, const void* SX) {
  TRY(fused_prepare(c, B));
  FusedPlan* p = (FusedPlan*)c->fused;
  const int cw = c->cplx ? 2 : 1;
  const int Wr = B * cw;
  float* X = (float*)Xv;
  const long ldx = ld * cw;
  // workspace arrays use this block's own padded leading dimension; P1 / Wcat use the plan's (widest block seen)
  const long ldw = roundup4(Wr);
  const size_t blk_s = ((size_t)c->M * ldw * 4 + 255) / 256 * 256, blk_d = ((size_t)c->M * ldw * 8 + 255) / 256 * 256;
  char* ws = (char*)workspace;
  double* Yt = (double*)ws;
  float* RX = (float*)(ws + blk_d);
  float* RY = (float*)(ws + blk_d + blk_s);
  float* XLO = (float*)(ws + blk_d + 2 * blk_s);   // FP32 mode only (pawfe_filter_workspace adds the block)
  const int gs = 8 * c->sm_count;
  const double* lam = ds;
  const double* neg_lam = ds + (size_t)(m + 1) * B;
  // ---- step 2 (FP64, L260, L374): Y = H X - S X Lambda ----
  prof_setup_mark(c, true);
  if (HX && SX) {
    k_residual_from_products<<<gs, 256, 0, c->stream>>>(c->M, ldw, Wr, cw, (const double*)HX, (const double*)SX, ldx, lam, Yt);
    KERNEL_CHECK(c, "k_residual_from_products");
  } else if (c->cplx) {
    // complex: the generic FP64 applies (DMMA cell product, mass sweeps, Ritz values folded into the coupling)
    TRY((pawfe_apply_HS<float2, double2, double2>(c, 0, false, (const float2*)X, ld, (double2*)Yt, ldw / 2, B)));
    TRY((pawfe_sub_SX_lambda<float2, double2>(c, (const float2*)X, ld, (double2*)Yt, ldw / 2, B, lam, neg_lam)));
  } else {
    TRY(residual_setup_real(c, p, X, ld, B, Yt, ldw, lam, neg_lam));
  }
  // ---- step 3 in the scaled variables: Yt = M_D^-1 Y, Rt_Y = (zeta/e) Yt, Rt_X = 0 (pad columns 0) ----
  k_residual_init3<<<gs, 256, 0, c->stream>>>(c->md, ldw, Wr, Yt, z_over_e, RX, RY);
  KERNEL_CHECK(c, "k_residual_init3");
  prof_setup_mark(c, false);
  // ---- step 4: one projection + coupling pass and ONE cell kernel per step; the cell kernel's first writers store the
  //      bracket  -a c Rt_Y - zeta zeta1 Rt_X [FP32] + Yt (a Lambda_Y) [FP64 add, L374]  plus their own share of
  //      a M_D^-1 H T, the other cells add theirs in cell order ----
  for (int th = 2; th <= m; ++th) {
    TRY(project_and_couple(c, p, prec == PAWFE_TF32, RY, ldw, B, 0));
    TcEpi epi;
    epi.mode = TC_EPI_BRACKET; epi.Yt = Yt; epi.aLam = ds + (size_t)(th - 1) * B; epi.ac = (float)acs[th]; epi.zz1 = (float)zzs[th]; epi.cw = cw;
    TRY(cell_pass(c, p, prec, RY, ldw, RX, ldw, Wr, (float)as[th], 1, epi, XLO));
    std::swap(RX, RY);
  }
  // ---- step 5: Psi_f = S^-1approx R_Y + X Lambda_Y = Rt_Y - M_D^-1 C W + X Lambda_Y ----
  TRY(project_and_couple(c, p, prec == PAWFE_TF32, RY, ldw, B, 1));
  {
    const bool vec = (ldx & 3) == 0 && (reinterpret_cast<uintptr_t>(X) & 15) == 0;
    const dim3 grid((unsigned)c->ncell, ceil_div(Wr, 128));
    const double* lamY = ds + (size_t)m * B;
#define LAUNCH_REC(CP, VE) k_recover_ordered<CP, VE><<<grid, 256, 0, c->stream>>>(c->md, p->d_cps, p->d_cpi, c->d_pair_atom, \
        (const float*)c->d_Cd32, c->npj, p->d_Wcat, p->ldw, RY, ldw, X, ldx, Wr, lamY)
    if (c->cplx) { if (vec) LAUNCH_REC(true, true); else LAUNCH_REC(true, false); }
    else { if (vec) LAUNCH_REC(false, true); else LAUNCH_REC(false, false); }
#undef LAUNCH_REC
    KERNEL_CHECK(c, "k_recover_ordered");
  }
  return PAWFE_OK;
}
