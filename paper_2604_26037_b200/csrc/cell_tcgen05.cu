// cell_tcgen05.cu -- the cell-level contraction of the operator action (Fig. 2 step iii) fused
// with extraction (step i, L343) and assembly (step iv, L347), on tcgen05 tensor cores in TF32 with FP32
// accumulation in tensor memory (TF32: L11, L27; FP32 storage: L374).
//
// Formulation.  Per cell e, node half and tile of 128 vectors the kernel computes the TRANSPOSED product
//     Y_e^T (128 vec x NT) = X_e^T (128 vec x n) * H^e^T (n x NT)
// so that the MMA M dimension (128 TMEM lanes) is the vector index and the N dimension the output node:
//   * operand A = X_e^T is "MN-major": a K chunk is 32 gathered node rows of 128 contiguous vectors, exactly the
//     shape of the global [dof][vec] block, copied by cp.async into the 128-byte-swizzle / 32-byte-atom layout;
//   * operand B = H^e is "K-major": stored re-tiled and pre-swizzled ([cell][half][K chunk][NT][32 floats]) so that
//     each chunk is ONE contiguous cp.async.bulk copy that lands in the SW128 K-major layout;
//   * the accumulator (128 lanes x NT columns) is read back lane = vector, transposed through shared memory and
//     added to the global rows with 16-byte vector reductions (4 vectors of one node per thread).
// n = (p+1)^3 output nodes are split into NH = 1 or 2 halves of NT <= 256 columns (NT a multiple of 16).  Optional
// K-extension chunks (fused.h) append low-rank projector terms to the same accumulation.
//
// One persistent CTA per SM, 10 warps: 0-3 epilogue, 4-7 gather producers, 8 bulk-copy producer, 9 MMA issuer and
// TMEM owner.  Pipelines: full[s] / empty[s] per shared-memory stage, accum_full[b] / accum_empty[b] per
// accumulator buffer (two buffers: the epilogue of one vector tile runs under the MMAs of the next).
#include "cell_tcgen05.h"
#include "ptx_sm100.cuh"
#include <cstdio>
#include <cstdlib>
#include <algorithm>

namespace {

constexpr int kChunkK = 32;             // K rows per pipeline stage (= 128 bytes of a K-major tf32 row)
constexpr int kTileV = 128;             // vectors per MMA (M)
constexpr int kABytes = kChunkK * kTileV * 4;  // 16 KB per vector tile and stage
constexpr int kThreads = 320;           // warps 0-3 epilogue, 4-7 gather, 8 TMA, 9 MMA / TMEM owner
constexpr int kMaxStages = 6;

struct TcArgs {
  MeshDev md;
  const float* X; long ldx;
  float* Y; long ldy;
  int B; float alpha;
  int n, NH, NT, kchunks, ksteps_last;
  int nvt;       // vector tiles of 128 in the block (processed one after the other inside a tile)
  int ntiles;    // ncell * NH
  int stages;
  int ncomp;     // 1: real cell matrices; 2: complex (two B blocks Re, Im and two accumulators P, Q per buffer)
  uint32_t tmem_cols, acc_stride, idesc;   // two accumulators of NT columns, acc_stride apart
  int scale_mode;            // 0: Y += alpha * acc;  1: Y += alpha * M_D^-1[J] * acc
  // K-extension chunks (fused.h): per cell a CSR list of 32-row chunks whose A rows come from Wcat[atom]
  const int* ext_start; const int* ext_atom; const float* Wcat; long ldw; int ext_ksteps;
  const float* H32t; const float* Bext;   // pre-swizzled, block-contiguous operand streams
  int dbg;  // timing experiments only (PAWFE_TC_DBG): 1 plain stores, 2 no output, 4 no gather loads
};

struct TcPlan {
  float* d_H32t_lo = nullptr;    // low parts (value - trunc_tf32(value)) of d_H32t, FP32 mode only
  long h32t_elems = 0;
  float* d_H32t = nullptr;       // cell matrices re-tiled for streaming: [cell][half][K chunk][NT rows][32] floats
  int NT = 0, NH = 0;
  bool ok = false;
};

// Re-tile the row-major FP32 cell matrices so that every (cell, half, K chunk) block the kernel loads is one
// contiguous NT x 128-byte region of HBM (row-major [cell][n][ldk] gives NT scattered 128-byte pieces per load,
// which costs DRAM page locality).  Rows >= n and columns >= n are zero.
__global__ void k_retile_h32(const float* __restrict__ H, int n, int ldk, int NH, int NT, int kchunks, int ncomp,
                             long total, float* __restrict__ out) {
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
    const int kk = (int)(i & 31);
    long t = i >> 5;
    const int r = (int)(t % NT); t /= NT;
    const int comp = (int)(t % ncomp); t /= ncomp;   // complex: [chunk][Re block][Im block]
    const int ch = (int)(t % kchunks); t /= kchunks;
    const int half = (int)(t % NH);
    const long cell = t / NH;
    const int I = half * NT + r, k = ch * 32 + kk;
    // 128-byte-swizzled image: 16-byte piece j of row r is stored at piece j ^ (r % 8), so that a plain contiguous
    // bulk copy of the block lands in shared memory in the layout the K-major SW128 matrix descriptor expects
    const long o = (i & ~31L) + ((((kk >> 2) ^ (r & 7)) << 2) | (kk & 3));
    out[o] = (I < n && k < n) ? H[((cell * n + I) * ldk + k) * ncomp + comp] : 0.f;
  }
}

__device__ __forceinline__ void bar_sync_128(int id) { asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory"); }

// Persistent CTAs (one per SM) loop over tiles (cell, node half); inside a tile over the vector tiles of 128
// ("subtiles").  The first vector tile of a tile streams its H^e half from HBM, the following ones re-read it
// from L2.  Accumulators are double-buffered in tensor memory (subtile parity), so the assembly epilogue of one
// subtile runs under the loads and MMAs of the next.  Roles are decoupled through mbarriers only.
__global__ void __launch_bounds__(kThreads, 1)
k_cell_tcgen05(const TcArgs a) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const int bbytes1 = a.NT * 128;                       // one matrix block (Re or Im)
  const int bbytes = a.ncomp * bbytes1;
  const int sbytes = kABytes + bbytes;                  // one stage: [A][B (Re)][B (Im)]
  long* gJ = reinterpret_cast<long*>(smem + a.stages * sbytes);           // [NH * NT] gather rows: byte offset or -1
  long* eJ = gJ + a.NH * a.NT;                                            // [NT] output rows of this half
  float* eS = reinterpret_cast<float*>(eJ + a.NT);                        // [NT] output scale
  float* stage_epi = eS + a.NT;                                           // [4 warps][32 nodes][32 vectors]
  uint64_t* full = reinterpret_cast<uint64_t*>(stage_epi + 4 * 32 * 32);  // [stages]
  uint64_t* empty = full + kMaxStages;                                    // [stages]
  uint64_t* accum_full = empty + kMaxStages;                              // [2]
  uint64_t* accum_empty = accum_full + 2;                                 // [2]
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(accum_empty + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < a.stages; ++s) { ptx::mbar_init(&full[s], 128 + 1); ptx::mbar_init(&empty[s], 1); }
    for (int b = 0; b < 2; ++b) { ptx::mbar_init(&accum_full[b], 1); ptx::mbar_init(&accum_empty[b], 128); }
    ptx::fence_barrier_init();
  }
  if (warp == 9) ptx::tmem_alloc(tmem_slot, a.tmem_cols);
  ptx::tc_fence_before_sync();
  __syncthreads();
  ptx::tc_fence_after_sync();
  const uint32_t tmem_base = *tmem_slot;
  const int n1 = a.md.n1;

  uint32_t it = 0;        // running chunk counter (same sequence in every role)
  uint32_t sub_iter = 0;  // running subtile counter: accumulator buffer = sub_iter & 1
  for (int tile = blockIdx.x; tile < a.ntiles; tile += gridDim.x) {
    const int cell = tile / a.NH;
    const int half = tile - cell * a.NH;
    const int ext0 = a.ext_start ? a.ext_start[cell] : 0;
    const int nchunks = a.kchunks + (a.ext_start ? a.ext_start[cell + 1] - ext0 : 0);
    int cx, cy, cz;
    mesh_cell_coords(a.md, cell, &cx, &cy, &cz);

    if (warp < 4) {
      // ================= epilogue: TMEM -> scaled vector reductions into Y (assembly, Fig. 2 step iv) =================
      bar_sync_128(2);   // previous tile's readers of eJ / eS are done
      for (int I = threadIdx.x; I < a.NT; I += 128) {
        const int Ig = half * a.NT + I;
        long J = -1;
        float sc = 0.f;
        if (Ig < a.n) {
          int c = Ig % n1, b = (Ig / n1) % n1, aa = Ig / (n1 * n1), ix, iy, iz;
          J = mesh_node(a.md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
          const double mi = a.md.mdinv1[0][ix] * a.md.mdinv1[1][iy] * a.md.mdinv1[2][iz];
          J = (mi == 0.0) ? -1 : J * a.ldy * 4;  // byte offset of the output row; -1: Dirichlet boundary
          sc = a.scale_mode ? (float)((double)a.alpha * mi) : a.alpha;
        }
        eJ[I] = J; eS[I] = sc;
      }
      bar_sync_128(2);
      const int ncols = min(a.NT, a.n - half * a.NT);
      // Each warp owns 32 vectors (TMEM lanes).  32 output nodes at a time: TMEM -> registers (lane = vector) ->
      // scaled -> staging tile [node][vector] in shared memory -> each thread takes 4 consecutive vectors of one
      // node and issues ONE 16-byte vector reduction (REDG.128): 4x fewer atomic lane-operations than scalar adds.
      float* stg = stage_epi + warp * (32 * 32);
      const int sub = lane >> 3, v4 = (lane & 7) * 4;
      for (int vt = 0; vt < a.nvt; ++vt) {
        const uint32_t buf = (sub_iter + vt) & 1, use = (sub_iter + vt) >> 1;
        ptx::mbar_wait(&accum_full[buf], use & 1);
        ptx::tc_fence_after_sync();
        const int vb = vt * kTileV + warp * 32;
        const bool vok = vb + v4 < a.B;             // B % 4 == 0: a float4 is all in or all out
        char* yv = reinterpret_cast<char*>(a.Y + vb + v4);
        if (vb < a.B && !(a.dbg & 16) && a.ncomp == 2) {
          // complex: columns are interleaved (re, im); with P = X^T Hr^T and Q = X^T Hi^T,
          //   Y_re = P_re - Q_im,  Y_im = P_im + Q_re  ->  y = P + (lane odd ? +1 : -1) * Q of the partner lane
          const float sg = (lane & 1) ? 1.f : -1.f;
          for (int col0 = 0; col0 < ncols; col0 += 16) {
            uint32_t r[16], q[16];
            const uint32_t taddr = tmem_base + ((uint32_t)(warp * 32) << 16) + buf * a.acc_stride + (uint32_t)col0;
            ptx::tmem_ld16(taddr, r);
            ptx::tmem_ld16(taddr + a.NT, q);
            ptx::tmem_ld_wait();
            const int nq = min(16, ncols - col0);
#pragma unroll
            for (int k = 0; k < 16; k += 4) {
              const float4 sc = *reinterpret_cast<const float4*>(&eS[col0 + k]);
              const float scs[4] = {sc.x, sc.y, sc.z, sc.w};
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                const float qp = __shfl_xor_sync(0xffffffffu, __uint_as_float(q[k + u]), 1);
                stg[(k + u) * 32 + lane] = scs[u] * fmaf(sg, qp, __uint_as_float(r[k + u]));
              }
            }
            __syncwarp();
            if (vok) {
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                const int k = sub + 4 * i;
                if (k < nq) {
                  const long off = eJ[col0 + k];
                  if (off >= 0) ptx::red_add_v4(reinterpret_cast<float*>(yv + off), *reinterpret_cast<const float4*>(&stg[k * 32 + v4]));
                }
              }
            }
            __syncwarp();
          }
        } else if (vb < a.B && !(a.dbg & 16)) {
          for (int col0 = 0; col0 < ncols; col0 += 32) {
            uint32_t r[32];
            const uint32_t taddr = tmem_base + ((uint32_t)(warp * 32) << 16) + buf * a.acc_stride + (uint32_t)col0;
            ptx::tmem_ld16(taddr, *reinterpret_cast<uint32_t(*)[16]>(&r[0]));
            if (col0 + 16 < ncols) ptx::tmem_ld16(taddr + 16, *reinterpret_cast<uint32_t(*)[16]>(&r[16]));
            ptx::tmem_ld_wait();
            const int nq = min(32, ncols - col0);
#pragma unroll
            for (int q = 0; q < 32; q += 4) {
              if (q < nq) {
                const float4 sc = *reinterpret_cast<const float4*>(&eS[col0 + q]);
                stg[(q + 0) * 32 + lane] = sc.x * __uint_as_float(r[q + 0]);
                stg[(q + 1) * 32 + lane] = sc.y * __uint_as_float(r[q + 1]);
                stg[(q + 2) * 32 + lane] = sc.z * __uint_as_float(r[q + 2]);
                stg[(q + 3) * 32 + lane] = sc.w * __uint_as_float(r[q + 3]);
              }
            }
            __syncwarp();
            if (vok) {
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                const int q = sub + 4 * i;
                if (q < nq) {
                  const long off = eJ[col0 + q];
                  if (off >= 0) {
                    const float4 val = *reinterpret_cast<const float4*>(&stg[q * 32 + v4]);
                    if (a.dbg & 1) *reinterpret_cast<float4*>(yv + off) = val;
                    else if (!(a.dbg & 2)) ptx::red_add_v4(reinterpret_cast<float*>(yv + off), val);
                  }
                }
              }
            }
            __syncwarp();
          }
        }
        ptx::tc_fence_before_sync();
        ptx::mbar_arrive(&accum_empty[buf]);
      }
    } else if (warp < 8) {
      // ================= gather producers: X rows -> swizzled MN-major A tiles (Fig. 2 step i) =================
      const int t = threadIdx.x - 128;  // 0..127
      bar_sync_128(1);   // previous tile's readers of gJ are done
      for (int I = t; I < a.NH * a.NT; I += 128) {
        long J = -1;
        if (I < a.n) {
          int c = I % n1, b = (I / n1) % n1, aa = I / (n1 * n1), ix, iy, iz;
          J = mesh_node(a.md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
          J = (a.md.mdinv1[0][ix] * a.md.mdinv1[1][iy] * a.md.mdinv1[2][iz] == 0.0) ? -1 : J * a.ldx * 4;  // byte offset
        }
        gJ[I] = J;
      }
      bar_sync_128(1);
      // per-thread constants: this thread always copies 16-byte column `lane` of rows wg, wg + 4, ... of a chunk
      const int wg = t >> 5;                               // row within each group of 4
      const int vl = lane * 4;                             // first vector of the 16-byte piece inside the tile
      // MN-major tf32 layout (128-byte swizzle, 32-byte atoms): 32-vector column block cb at cb * 4096; row r at
      // r * 128; its four 32-byte chunks q stored at q ^ (r % 4); r % 4 == wg for every row this thread copies
      const uint32_t dst_thread = (lane >> 3) * 4096 + wg * 128 + (((((lane & 7) >> 1) ^ wg) << 5) | ((lane & 1) << 4));
      uint32_t itc = it;
      for (int vt = 0; vt < a.nvt; ++vt) {
        const int v = vt * kTileV + vl;
        const bool vok = v < a.B;
        const char* xv = reinterpret_cast<const char*>(a.X + v);
        for (int c = 0; c < nchunks; ++c, ++itc) {
          const uint32_t s = itc % a.stages, ph = (itc / a.stages) & 1;
          ptx::mbar_wait(&empty[s], ph ^ 1);
          const uint32_t abase = ptx::smem_u32(smem + s * sbytes) + dst_thread;
          if (c < a.kchunks) {
            const long* offs = gJ + c * kChunkK + wg;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const long off = (c * kChunkK + wg + 4 * i < a.NH * a.NT) ? offs[4 * i] : -1;
              const bool ok = vok && off >= 0;
              if (!(a.dbg & 4)) ptx::cp_async16(abase + i * 512, ok ? xv + off : reinterpret_cast<const char*>(a.X), ok ? 16u : 0u);
            }
          } else {
            const float* wrows = a.Wcat + ((long)a.ext_atom[ext0 + c - a.kchunks] * 32 + wg) * a.ldw + v;
#pragma unroll
            for (int i = 0; i < 8; ++i)
              ptx::cp_async16(abase + i * 512, vok ? wrows + (long)(4 * i) * a.ldw : a.X, vok ? 16u : 0u);
          }
          // arrival on full[s] fires when all of this thread's copies above have landed: no wait here, the thread
          // goes straight on to the next chunk (gated only by that stage being free)
          ptx::cp_async_mbar_arrive_noinc(&full[s]);
        }
      }
    } else if (warp == 8) {
      // ================= TMA producer: H^e row block (or K-extension block), one K chunk per stage =================
      if (lane == 0) {
        uint32_t itc = it;
        for (int vt = 0; vt < a.nvt; ++vt)
          for (int c = 0; c < nchunks; ++c, ++itc) {
            const uint32_t s = itc % a.stages, ph = (itc / a.stages) & 1;
            ptx::mbar_wait(&empty[s], ph ^ 1);
            ptx::mbar_arrive_expect_tx(&full[s], (uint32_t)bbytes);
            const uint32_t dst = ptx::smem_u32(smem + s * sbytes + kABytes);
            // both operand streams are stored pre-swizzled and block-contiguous: one linear bulk copy per chunk
            const float* src = (c < a.kchunks)
                ? a.H32t + ((long)((cell * a.NH + half) * a.kchunks + c) * a.NT) * 32 * a.ncomp
                : a.Bext + ((long)(ext0 + c - a.kchunks) * a.NH + half) * a.NT * 32 * a.ncomp;
            if (a.dbg & 64) { ptx::bulk_load(dst, src, (uint32_t)bbytes / 2, &full[s]); ptx::bulk_load(dst + bbytes / 2, src, (uint32_t)bbytes / 2, &full[s]); }
            else ptx::bulk_load(dst, src, (uint32_t)bbytes, &full[s]);
          }
      }
      __syncwarp();
    } else {
      // ================= MMA issuer =================
      if (lane == 0) {
        uint32_t itc = it;
        for (int vt = 0; vt < a.nvt; ++vt) {
          const uint32_t buf = (sub_iter + vt) & 1, use = (sub_iter + vt) >> 1;
          ptx::mbar_wait(&accum_empty[buf], (use & 1) ^ 1);   // buffer drained by the epilogue of two subtiles ago
          ptx::tc_fence_after_sync();
          const uint32_t dtm = tmem_base + buf * a.acc_stride;
          for (int c = 0; c < nchunks; ++c, ++itc) {
            const uint32_t s = itc % a.stages, ph = (itc / a.stages) & 1;
            ptx::mbar_wait(&full[s], ph);
            if (!(a.dbg & 32)) ptx::fence_proxy_async_smem();   // cp.async (generic proxy) writes of the A tile -> tensor-core (async proxy) reads
            ptx::tc_fence_after_sync();
            const uint32_t abase = ptx::smem_u32(smem + s * sbytes), bbase = abase + kABytes;
            const int ksteps = (c == a.kchunks - 1) ? a.ksteps_last : (c >= a.kchunks ? a.ext_ksteps : kChunkK / 8);
            for (int ks = 0; ks < ksteps; ++ks) {
              // A (MN-major, 128B swizzle / 32B atoms): 4 blocks of 32 vectors 4096 B apart (LBO); K atoms of 4 rows
              // 512 B apart (SBO); one K step = 8 rows = 1024 B
              const uint64_t adesc = ptx::smem_desc(abase + ks * 1024, 4096, 512, 1);
              // B (K-major, SW128): 8-row groups 1024 B apart (SBO); 8 tf32 = 32 B per K step inside the 128-B row
              const uint64_t bdesc = ptx::smem_desc_sw128(bbase + ks * 32, 16, 1024);
              if (!(a.dbg & 8)) ptx::mma_tf32_ss(dtm, adesc, bdesc, a.idesc, (c > 0 || ks > 0) ? 1u : 0u);
              if (a.ncomp == 2) {
                const uint64_t bdesc2 = ptx::smem_desc_sw128(bbase + bbytes1 + ks * 32, 16, 1024);
                ptx::mma_tf32_ss(dtm + (uint32_t)a.NT, adesc, bdesc2, a.idesc, (c > 0 || ks > 0) ? 1u : 0u);
              }
            }
            ptx::mma_commit(&empty[s]);
          }
          ptx::mma_commit(&accum_full[buf]);
        }
      }
      __syncwarp();
    }
    it += (uint32_t)(nchunks * a.nvt);
    sub_iter += (uint32_t)a.nvt;
  }
  __syncthreads();
  if (warp == 9) ptx::tmem_dealloc(tmem_base, a.tmem_cols);
}

void shape_for(const pawfe_ctx* c, int* NH, int* NT) {
  // two accumulator buffers of ncomp * NT columns must fit the 512 TMEM columns
  const int maxnt = c->cplx ? 128 : 256;
  *NH = (c->n + maxnt - 1) / maxnt;
  int per = (c->n + *NH - 1) / *NH;
  *NT = (per + 15) / 16 * 16;
}

size_t smem_fixed_(int NH, int NT) { return (size_t)NH * NT * 8 + (size_t)NT * 12 + 4 * 32 * 32 * 4 + (2 * kMaxStages + 4) * 8 + 16; }
size_t smem_fixed(int NH, int NT) { return smem_fixed_(NH, NT); }
int stages_for(int NH, int NT, int ncomp) {
  const size_t budget = 227 * 1024 - 1024;  // dynamic shared memory per CTA, less the alignment slack
  int st = (int)((budget - smem_fixed(NH, NT)) / (size_t)(kABytes + ncomp * NT * 128));
  return std::min(st, kMaxStages);
}
size_t smem_bytes(int NH, int NT, int ncomp) {
  return (size_t)stages_for(NH, NT, ncomp) * (kABytes + ncomp * NT * 128) + smem_fixed(NH, NT);
}

TcPlan* get_plan(pawfe_ctx* c) {
  if (c->tc_plan) return (TcPlan*)c->tc_plan;
  TcPlan* p = new TcPlan();
  c->tc_plan = p;
  shape_for(c, &p->NH, &p->NT);
  if (!c->d_H32) return p;
  const int ncomp = c->cplx ? 2 : 1;
  const int kchunks = (c->ldk + kChunkK - 1) / kChunkK;
  const long elems = (long)c->ncell * p->NH * kchunks * ncomp * p->NT * 32;
  if (cudaMalloc((void**)&p->d_H32t, (size_t)elems * sizeof(float)) != cudaSuccess) { cudaGetLastError(); p->d_H32t = nullptr; return p; }
  p->h32t_elems = elems;
  k_retile_h32<<<8 * c->sm_count, 256, 0, c->stream>>>((const float*)c->d_H32, c->n, c->ldk, p->NH, p->NT, kchunks, ncomp, elems, p->d_H32t);
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) return p;
  // the attribute is per function, not per context: only ever raise it
  static size_t smem_attr = 0;
  size_t smem = smem_bytes(p->NH, p->NT, ncomp);
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

void tc_shape(const pawfe_ctx* c, int* NH, int* NT) { shape_for(c, NH, NT); }

namespace {
__global__ void k_lo_part(const float* __restrict__ src, float* __restrict__ dst, long count) {
  for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < count; i += (long)gridDim.x * blockDim.x) {
    const float v = src[i];
    dst[i] = v - __uint_as_float(__float_as_uint(v) & 0xffffe000u);   // kind::tf32 keeps sign, exponent, 10 mantissa bits
  }
}
}  // namespace

pawfe_status tc_lo_part(pawfe_ctx* c, const float* src, float* dst, long count) {
  k_lo_part<<<8 * c->sm_count, 256, 0, c->stream>>>(src, dst, count);
  KERNEL_CHECK(c, "k_lo_part");
  return PAWFE_OK;
}

pawfe_status tc_hstream_lo(pawfe_ctx* c, const float** out) {
  TcPlan* p = get_plan(c);
  if (!p->ok) { c->err = "tcgen05 cell kernel: plan set-up failed"; return PAWFE_EUNSUPPORTED; }
  if (!p->d_H32t_lo) {
    if (cudaMalloc((void**)&p->d_H32t_lo, (size_t)p->h32t_elems * sizeof(float)) != cudaSuccess) {
      cudaGetLastError(); p->d_H32t_lo = nullptr; c->err = "out of memory for the low parts of the cell matrices"; return PAWFE_ENOMEM;
    }
    pawfe_status st = tc_lo_part(c, p->d_H32t, p->d_H32t_lo, p->h32t_elems);
    if (st != PAWFE_OK) return st;
  }
  *out = p->d_H32t_lo;
  return PAWFE_OK;
}

void tc_invalidate(pawfe_ctx* c) {
  if (c->tc_plan) { cudaFree(((TcPlan*)c->tc_plan)->d_H32t_lo); cudaFree(((TcPlan*)c->tc_plan)->d_H32t); delete (TcPlan*)c->tc_plan; c->tc_plan = nullptr; }
}

bool tc_supported(const pawfe_ctx* c, int B) {
  if (!c->have_pot || B < 1) return false;
  if (c->n < 16) return false;
  return true;
}

bool tc_usable(pawfe_ctx* c, const void* X, long ldx, const void* Y, long ldy, int B) {
  if (!tc_supported(c, B)) return false;
  if ((ldx & 3) || (ldy & 3) || (B & 3) || ((uintptr_t)X & 15) || ((uintptr_t)Y & 15)) return false;
  return get_plan(c)->ok;
}

// Complex contexts: X, Y are the interleaved (re, im) blocks seen as real blocks, B = 2 x vectors, ldx / ldy in floats.
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
  a.ntiles = c->ncell * a.NH;
  a.ncomp = c->cplx ? 2 : 1;
  a.stages = stages_for(p->NH, p->NT, a.ncomp);
  uint32_t cols = 32;
  while ((int)cols < a.ncomp * a.NT) cols <<= 1;
  a.acc_stride = cols;
  a.tmem_cols = 2 * cols;
  a.idesc = ptx::idesc_tf32(kTileV, a.NT, /*A MN-major*/ 1, /*B K-major*/ 0);
  a.scale_mode = 0;
  a.H32t = (ext && ext->Hstream) ? ext->Hstream : p->d_H32t; a.Bext = nullptr;
  a.ext_start = nullptr; a.ext_atom = nullptr; a.Wcat = nullptr; a.ldw = 0; a.ext_ksteps = 0;
  if (ext) {
    a.scale_mode = ext->scale_mode;
    if (ext->nchunks > 0) {
      a.ext_start = ext->ext_start; a.ext_atom = ext->ext_atom; a.Wcat = ext->Wcat; a.ldw = ext->ldw; a.Bext = ext->Bext;
      a.ext_ksteps = ext->ksteps;
    }
  }
  { const char* d = getenv("PAWFE_TC_DBG"); a.dbg = d ? atoi(d) : 0; }
  int grid = std::min(a.ntiles, c->sm_count);
  k_cell_tcgen05<<<grid, kThreads, smem_bytes(p->NH, p->NT, a.ncomp), c->stream>>>(a);
  KERNEL_CHECK(c, "k_cell_tcgen05");
  return PAWFE_OK;
}
