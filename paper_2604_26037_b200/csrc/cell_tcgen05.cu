// cell_tcgen05.cu -- the cell-level contraction of the operator action (Fig. 2 step iii) fused
// with extraction (step i, L343) and assembly (step iv, L347), on tcgen05 tensor cores in TF32 with FP32
// accumulation in tensor memory (TF32: L11, L27; FP32 storage: L374).
//
// Formulation.  Per cell e and per tile of 128 vectors the kernel computes the TRANSPOSED product
//     Y_e^T (128 vec x n) = X_e^T (128 vec x n) * H^e^T (n x n)
// so that the MMA M dimension (128 TMEM lanes) is the vector index and the N dimension the output node:
//   * operand A = X_e^T is "MN-major": a K-chunk is 32 gathered node rows of 128 contiguous vectors, exactly the
//     shape of the global [dof][vec] block, copied by cp.async into the canonical 128-byte-swizzled layout;
//   * operand B = H^e is "K-major": rows of the row-major cell matrix, streamed by TMA (2-D tiled map, 128-byte
//     swizzle) -- each cell matrix is read once per (vector tile, node half);
//   * the accumulator (128 lanes x NT columns) is read back lane = vector, so one warp-wide reduction per node
//     writes 32 consecutive vectors = one coalesced 128-byte segment of the global row.
// n = (p+1)^3 output nodes are split into NH = 1 or 2 halves of NT <= 256 columns (NT a multiple of 16) so that
// two CTAs fit one SM (2 x 256 TMEM columns, 2 x <= 110 KB shared memory): while one CTA drains its accumulator
// the other one runs its MMAs.  Persistent CTAs loop over (cell, vector tile, node half) tiles.
//
// Warp roles (192 threads): warps 0-3 gather producers, then epilogue; warp 4 TMA producer; warp 5 TMEM owner and
// MMA issuer.  Pipelines: full[s] / empty[s] per shared-memory stage, accum for the accumulator.
#include "cell_tcgen05.h"
#include "ptx_sm100.cuh"
#include <cstdio>
#include <cstdlib>
#include <algorithm>

namespace {

constexpr int kStages = 2;
constexpr int kChunkK = 32;             // K rows per pipeline stage (= 128 bytes of a K-major tf32 row)
constexpr int kTileV = 128;             // vectors per tile (MMA M)
constexpr int kABytes = kChunkK * kTileV * 4;  // 16 KB
constexpr int kThreads = 192;

struct TcArgs {
  MeshDev md;
  const float* X; long ldx;
  float* Y; long ldy;
  int B; float alpha;
  int n, NH, NT, kchunks, ksteps_last, nvt, ntiles;
  uint32_t tmem_cols, idesc;
  int scale_mode;            // 0: Y += alpha * acc;  1: Y += alpha * M_D^-1[J] * acc
  // K-extension chunks (fused.h): per cell a CSR list of 32-row chunks whose A rows come from Wcat[atom]
  const int* ext_start; const int* ext_atom; const float* Wcat; long ldw; int ext_ksteps;
  int dbg;
};

struct TcPlan {
  CUtensorMap tmapH;
  CUtensorMap tmapE;             // K-extension blocks [chunk * n + I][32], built on first use for ext_ptr
  const void* ext_ptr = nullptr;
  int NT = 0, NH = 0;
  bool ok = false;
};

__global__ void __launch_bounds__(kThreads, 2)
k_cell_tcgen05(const __grid_constant__ CUtensorMap tmapH, const __grid_constant__ CUtensorMap tmapE, const TcArgs a) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const int bbytes = a.NT * 128;
  uint8_t* sA = smem;                                  // [kStages][16 KB]
  uint8_t* sB = smem + kStages * kABytes;              // [kStages][NT * 128 B]
  long* nodeJ = reinterpret_cast<long*>(sB + kStages * bbytes);          // [NH * NT] global row or -1
  float* nodeS = reinterpret_cast<float*>(nodeJ + a.NH * a.NT);          // [NH * NT] output scale per node
  uint64_t* full = reinterpret_cast<uint64_t*>(nodeS + a.NH * a.NT);      // [kStages]
  uint64_t* empty = full + kStages;                                       // [kStages]
  uint64_t* accum = empty + kStages;                                      // [1]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(accum + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) { ptx::mbar_init(&full[s], 128 + 1); ptx::mbar_init(&empty[s], 1); }
    ptx::mbar_init(accum, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 4 && lane == 0) { ptx::prefetch_tmap(&tmapH); if (a.ext_start) ptx::prefetch_tmap(&tmapE); }
  if (warp == 5) ptx::tmem_alloc(tmem_slot, a.tmem_cols);
  ptx::tc_fence_before_sync();
  __syncthreads();
  ptx::tc_fence_after_sync();
  const uint32_t tmem_base = *tmem_slot;

  uint32_t it = 0;        // running chunk counter (same sequence in every role)
  uint32_t tile_iter = 0;
  const int n1 = a.md.n1;
  for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x, ++tile_iter) {
    const int per_cell = a.nvt * a.NH;
    const int cell = tile / per_cell;
    const int rem = tile - cell * per_cell;
    const int vt = rem / a.NH, half = rem - vt * a.NH;
    const int v0 = vt * kTileV;
    const int ext0 = a.ext_start ? a.ext_start[cell] : 0;
    const int nchunks = a.kchunks + (a.ext_start ? a.ext_start[cell + 1] - ext0 : 0);

    __syncthreads();  // previous tile's readers of nodeJ are done
    {
      int cx, cy, cz;
      mesh_cell_coords(a.md, cell, &cx, &cy, &cz);
      for (int I = threadIdx.x; I < a.NH * a.NT; I += kThreads) {
        long J = -1;
        float sc = 0.f;
        if (I < a.n) {
          int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1);
          int ix, iy, iz;
          J = mesh_node(a.md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
          const double mi = a.md.mdinv1[0][ix] * a.md.mdinv1[1][iy] * a.md.mdinv1[2][iz];
          if (mi == 0.0) J = -1;  // Dirichlet boundary
          sc = a.scale_mode ? (float)((double)a.alpha * mi) : a.alpha;
        }
        nodeJ[I] = J;
        nodeS[I] = sc;
      }
    }
    __syncthreads();

    if (warp < 4) {
      // ================= gather producers: X rows -> swizzled MN-major A tiles =================
      const int t = threadIdx.x;  // 0..127
      for (int c = 0; c < nchunks; ++c) {
        const uint32_t s = (it + c) % kStages, ph = ((it + c) / kStages) & 1;
        ptx::mbar_wait(&empty[s], ph ^ 1);
        const uint32_t abase = ptx::smem_u32(sA + s * kABytes);
        const bool isext = c >= a.kchunks;
        const float* wrows = isext ? a.Wcat + (long)a.ext_atom[ext0 + c - a.kchunks] * 32 * a.ldw : nullptr;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const int op = i * 128 + t;
          const int row = op >> 5, c16all = op & 31;   // one warp covers one 512-byte row
          const int k = c * kChunkK + row;
          const int v = v0 + c16all * 4;
          const float* src;
          bool ok;
          if (!isext) {
            long J = (k < a.n) ? nodeJ[k] : -1;
            ok = (J >= 0) && (v < a.B);
            src = ok ? (a.X + J * a.ldx + v) : a.X;
          } else {
            ok = v < a.B;
            src = ok ? (wrows + (long)row * a.ldw + v) : a.X;
          }
          // MN-major tf32 layout (128-byte swizzle, 32-byte atoms): 32-vector column block cb at cb * 4096;
          // row r at r * 128; its four 32-byte chunks q stored at q ^ (r % 4)
          const uint32_t dst = abase + (c16all >> 3) * 4096 + row * 128 +
                               (((((c16all & 7) >> 1) ^ (row & 3)) << 5) | ((c16all & 1) << 4));
          ptx::cp_async16(dst, src, ok ? 16u : 0u);
        }
        ptx::cp_async_commit();
        if (c >= 1) {
          ptx::cp_async_wait<1>();
          ptx::fence_proxy_async_smem();
          ptx::mbar_arrive(&full[(it + c - 1) % kStages]);
        }
      }
      ptx::cp_async_wait<0>();
      ptx::fence_proxy_async_smem();
      ptx::mbar_arrive(&full[(it + nchunks - 1) % kStages]);

      // ================= epilogue: TMEM -> scaled atomic adds into Y (assembly) =================
      ptx::mbar_wait(accum, tile_iter & 1);
      ptx::tc_fence_after_sync();
      const int v = v0 + warp * 32 + lane;
      const bool vok = v < a.B;
      for (int col0 = 0; col0 < a.NT; col0 += 16) {
        if (half * a.NT + col0 >= a.n) break;
        uint32_t r[16];
        ptx::tmem_ld16(tmem_base + ((uint32_t)(warp * 32) << 16) + (uint32_t)col0, r);
        ptx::tmem_ld_wait();
#ifdef PAWFE_TC_DEBUG
        if (blockIdx.x == 0 && threadIdx.x == 0 && col0 == 0)
          printf("epi: tmem_base=%x r0=%g r1=%g r2=%g r15=%g J0=%ld v=%d vok=%d alpha=%g NT=%d n=%d\n", tmem_base, __uint_as_float(r[0]),
                 __uint_as_float(r[1]), __uint_as_float(r[2]), __uint_as_float(r[15]), nodeJ[0], v, (int)vok, a.alpha, a.NT, a.n);
#endif
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const long J = nodeJ[half * a.NT + col0 + j];
          if (J >= 0 && vok) atomicAdd(a.Y + J * a.ldy + v, nodeS[half * a.NT + col0 + j] * __uint_as_float(r[j]));
        }
      }
      ptx::tc_fence_before_sync();
    } else if (warp == 4) {
      // ================= TMA producer: H^e row block, one K chunk per stage =================
      if (lane == 0) {
        for (int c = 0; c < nchunks; ++c) {
          const uint32_t s = (it + c) % kStages, ph = ((it + c) / kStages) & 1;
          ptx::mbar_wait(&empty[s], ph ^ 1);
          ptx::mbar_arrive_expect_tx(&full[s], (uint32_t)bbytes);
          if (c < a.kchunks)
            ptx::tma_load_2d(ptx::smem_u32(sB + s * bbytes), &tmapH, c * kChunkK, cell * a.n + half * a.NT, &full[s]);
          else
            ptx::tma_load_2d(ptx::smem_u32(sB + s * bbytes), &tmapE, 0, (ext0 + c - a.kchunks) * a.n + half * a.NT, &full[s]);
        }
      }
    } else {
      // ================= MMA issuer =================
      if (lane == 0) {
        for (int c = 0; c < nchunks; ++c) {
          const uint32_t s = (it + c) % kStages, ph = ((it + c) / kStages) & 1;
          ptx::mbar_wait(&full[s], ph);
          ptx::tc_fence_after_sync();
          const uint32_t abase = ptx::smem_u32(sA + s * kABytes), bbase = ptx::smem_u32(sB + s * bbytes);
          const int ksteps = (c == a.kchunks - 1) ? a.ksteps_last : (c >= a.kchunks ? a.ext_ksteps : kChunkK / 8);
#ifdef PAWFE_TC_DEBUG
          if (blockIdx.x == 0 && c == 0) {
            const float* Af = reinterpret_cast<const float*>(sA + s * kABytes);
            const float* Bf = reinterpret_cast<const float*>(sB + s * bbytes);
            printf("mma: idesc=%x ksteps=%d kchunks=%d A[0]=%g A[1]=%g B[0]=%g B[1]=%g abase=%x bbase=%x\n", a.idesc, ksteps,
                   a.kchunks, Af[0], Af[1], Bf[0], Bf[1], abase, bbase);
          }
#endif
          for (int ks = 0; ks < ksteps; ++ks) {
            // A (MN-major, 128B swizzle / 32B atoms): 4 blocks of 32 vectors 4096 B apart (LBO); K atoms of 4 rows
            // 512 B apart (SBO); one K step = 8 rows = 1024 B
            uint64_t adesc = ptx::smem_desc(abase + ks * 1024, 4096, 512, 1);
#ifdef PAWFE_TC_DEBUG
            if (a.dbg & 1) adesc = ptx::smem_desc_sw128(bbase + ks * 32, 16, 1024);  // A := B tile, K-major
            if (a.dbg & 2) adesc = ptx::smem_desc(abase + ks * 1024, 512, 4096, 1);  // swapped LBO/SBO
#endif
            // B (K-major, SW128): 8-row groups 1024 B apart (SBO); 8 tf32 = 32 B per K step inside the 128-B row
            const uint64_t bdesc = ptx::smem_desc_sw128(bbase + ks * 32, 16, 1024);
            ptx::mma_tf32_ss(tmem_base, adesc, bdesc, a.idesc, (c > 0 || ks > 0) ? 1u : 0u);
          }
          ptx::mma_commit(&empty[s]);
        }
        ptx::mma_commit(accum);
      }
      __syncwarp();
    }
    it += nchunks;
  }
  __syncthreads();
  if (warp == 5) ptx::tmem_dealloc(tmem_base, a.tmem_cols);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

void shape_for(const pawfe_ctx* c, int* NH, int* NT) {
  *NH = c->n > 256 ? 2 : 1;
  int per = (c->n + *NH - 1) / *NH;
  *NT = (per + 15) / 16 * 16;
}

size_t smem_bytes(int NH, int NT) {
  return (size_t)kStages * (kABytes + NT * 128) + (size_t)NH * NT * 12 + (2 * kStages + 1) * 8 + 16;
}

TcPlan* get_plan(pawfe_ctx* c) {
  if (c->tc_plan) return (TcPlan*)c->tc_plan;
  TcPlan* p = new TcPlan();
  c->tc_plan = p;
  shape_for(c, &p->NH, &p->NT);
  EncodeTiledFn enc = get_encode();
  if (!enc || !c->d_H32) return p;
  cuuint64_t dims[2] = {(cuuint64_t)c->ldk, (cuuint64_t)c->ncell * c->n};
  cuuint64_t strides[1] = {(cuuint64_t)c->ldk * sizeof(float)};
  cuuint32_t box[2] = {(cuuint32_t)kChunkK, (cuuint32_t)p->NT};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = enc(&p->tmapH, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, c->d_H32, dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return p;
  // the attribute is per function, not per context: only ever raise it
  static size_t smem_attr = 0;
  size_t smem = smem_bytes(p->NH, p->NT);
  if (smem > smem_attr) {
    if (cudaFuncSetAttribute(k_cell_tcgen05, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
      cudaGetLastError();
      return p;
    }
    smem_attr = smem;
  }
  p->ok = true;
  return p;
}

}  // namespace

void tc_invalidate(pawfe_ctx* c) {
  if (c->tc_plan) { delete (TcPlan*)c->tc_plan; c->tc_plan = nullptr; }
}

bool tc_supported(const pawfe_ctx* c, int B) {
  if (c->cplx || !c->have_pot || B < 1) return false;
  if (c->n < 16) return false;
  return true;
}

bool tc_usable(pawfe_ctx* c, const void* X, long ldx, const void* Y, long ldy, int B) {
  if (!tc_supported(c, B)) return false;
  if ((ldx & 3) || (ldy & 3) || (B & 3) || ((uintptr_t)X & 15) || ((uintptr_t)Y & 15)) return false;
  return get_plan(c)->ok;
}

pawfe_status tc_cell_apply(pawfe_ctx* c, const float* X, long ldx, float* Y, long ldy, int B, float alpha,
                           const TcExt* ext) {
  TcPlan* p = get_plan(c);
  if (!p->ok) { c->err = "tcgen05 cell kernel: tensor map / attribute set-up failed"; return PAWFE_EUNSUPPORTED; }
  TcArgs a;
  a.md = c->md; a.X = X; a.ldx = ldx; a.Y = Y; a.ldy = ldy; a.B = B; a.alpha = alpha;
  a.n = c->n; a.NH = p->NH; a.NT = p->NT;
  a.kchunks = (c->ldk + kChunkK - 1) / kChunkK;
  a.ksteps_last = (c->ldk - (a.kchunks - 1) * kChunkK) / 8;
  a.nvt = (B + kTileV - 1) / kTileV;
  a.ntiles = c->ncell * a.nvt * a.NH;
  uint32_t cols = 32;
  while ((int)cols < a.NT) cols <<= 1;
  a.tmem_cols = cols;
  a.idesc = ptx::idesc_tf32(kTileV, a.NT, /*A MN-major*/ 1, /*B K-major*/ 0);
  a.scale_mode = 0;
  a.ext_start = nullptr; a.ext_atom = nullptr; a.Wcat = nullptr; a.ldw = 0; a.ext_ksteps = 0;
  if (ext) {
    a.scale_mode = ext->scale_mode;
    if (ext->nchunks > 0) {
      if (p->ext_ptr != ext->Bext) {
        EncodeTiledFn enc = get_encode();
        cuuint64_t dims[2] = {32, (cuuint64_t)ext->nchunks * c->n};
        cuuint64_t strides[1] = {32 * sizeof(float)};
        cuuint32_t box[2] = {(cuuint32_t)kChunkK, (cuuint32_t)p->NT};
        cuuint32_t estr[2] = {1, 1};
        CUresult r = enc(&p->tmapE, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, (void*)ext->Bext, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { c->err = "tcgen05 cell kernel: K-extension tensor map failed"; return PAWFE_ECUDA; }
        p->ext_ptr = ext->Bext;
      }
      a.ext_start = ext->ext_start; a.ext_atom = ext->ext_atom; a.Wcat = ext->Wcat; a.ldw = ext->ldw;
      a.ext_ksteps = ext->ksteps;
    }
  }
  a.dbg = 0;
#ifdef PAWFE_TC_DEBUG
  a.dbg = getenv("PAWFE_TC_DBG") ? atoi(getenv("PAWFE_TC_DBG")) : 0;
  if (a.dbg & 1) a.idesc = ptx::idesc_tf32(kTileV, a.NT, 0, 0);
#endif
  int grid = std::min(a.ntiles, 2 * c->sm_count);
  k_cell_tcgen05<<<grid, kThreads, smem_bytes(p->NH, p->NT), c->stream>>>(p->tmapH, a.ext_start ? p->tmapE : p->tmapH, a);
  KERNEL_CHECK(c, "k_cell_tcgen05");
  return PAWFE_OK;
}
