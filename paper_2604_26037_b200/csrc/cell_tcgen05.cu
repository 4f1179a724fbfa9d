// cell_tcgen05.cu -- the cell-level contraction of the operator action (Fig. 2 step iii) fused
// with extraction (step i, L343), assembly (step iv, L347) and -- inside the filter -- the bracket of Algorithm 2
// step 4 (L272, L374), on tcgen05 tensor cores in TF32 with FP32 accumulation in tensor memory (TF32: L11, L27; FP32
// storage: L374).
//
// Formulation.  Per cell e, node half and tile of 128 vectors the kernel computes the TRANSPOSED product
//     Y_e^T (128 vec x NT) = X_e^T (128 vec x n) * H^e^T (n x NT)
// so that the MMA M dimension (128 TMEM lanes) is the vector index and the N dimension the output node:
//   * operand A = X_e^T is "MN-major": a K chunk is 32 gathered node rows of 128 contiguous vectors, exactly the
//     shape of the global [dof][vec] block, copied by cp.async into the 128-byte-swizzle / 32-byte-atom layout;
//   * operand B = H^e is "K-major": stored re-tiled and pre-swizzled ([cell][half][K chunk][NT][32 floats]) so that
//     each chunk is ONE contiguous cp.async.bulk copy that lands in the SW128 K-major layout;
//   * the accumulator (128 lanes x NT columns) is read back lane = vector and transposed through shared memory; each
//     thread then owns 4 consecutive vectors of one output node (16 bytes of its global row).
// n = (p+1)^3 output nodes are split into NH = 1 or 2 halves of NT <= 256 columns (NT a multiple of 16).  Optional
// K-extension chunks (fused.h) append low-rank projector terms to the same accumulation.
//
// Ordered assembly ("conflict-free scatter-add").  The plan fixes a cell ORDER (blocks of cells, inside a block the 8
// parity colours one after the other: same-colour cells share no node).  Of the <= 8 cells that share a node the one
// that comes first in the order is the node's FIRST WRITER: its first-writer warps store the row's initial value with
// plain 16-byte stores (inside the filter they stream R_Y, R_X, Y of the row through the bulk-copy engine and store the
// whole bracket of Alg. 2 step 4, so no separate bracket pass and no zero-fill exist) while the tile's MMAs run.  Every
// cell then adds its contribution with 16-byte vector reductions, the first writer after its own initial value, the
// others only when every neighbour that precedes them in the order has finished (one completion
// counter per cell, release / acquire at gpu scope).  Tiles are handed to the persistent CTAs in that same order, so
// the wait graph is acyclic and the lowest unfinished tile never waits; contributions reach every node in cell order,
// which makes the FP32 sums bit-reproducible from launch to launch.
//
// One persistent CTA per SM, 22 warps: 0-7 assembly (two per TMEM lane quadrant), 8-11 gather producers, 12 bulk-copy
// producer, 13 MMA issuer and TMEM owner, 14-21 first writers.  Pipelines: full[s] / empty[s] per shared-memory stage,
// accum_full[b] / accum_empty[b] per accumulator buffer (two buffers: the assembly of one vector tile runs under the MMAs
// of the next), br_done[t] / epi_free[t] between first writers and assembly (the first writers run up to 4 tiles ahead).
#include "cell_tcgen05.h"
#include "host_util.h"
#include "ptx_sm100.cuh"
#include <cstdio>
#include <cstdlib>
#include <algorithm>
#include <vector>

namespace {

constexpr int kChunkK = 32;             // K rows per pipeline stage (= 128 bytes of a K-major tf32 row)
constexpr int kTileV = 128;             // vectors per MMA (M)
constexpr int kABytes = kChunkK * kTileV * 4;  // 16 KB per vector tile and stage
constexpr int kEpiWarps = 8;            // two per TMEM lane quadrant (warp % 4), alternating column groups: the assembly is a
                                        // chain of dependent TMEM / shared / global operations, two warps per scheduler overlap it
constexpr int kEpiThreads = 32 * kEpiWarps;
constexpr int kGatherWarps = 4;
constexpr int kGatherThreads = 32 * kGatherWarps;
constexpr int kWarpTma = kEpiWarps + kGatherWarps, kWarpMma = kWarpTma + 1;
constexpr int kBrWarps = 8;              // first-writer warps: stream the initial value (bracket of Alg. 2 step 4, or 0) of the rows this tile writes first
constexpr int kBrThreads = 32 * kBrWarps;
constexpr int kBrSlots = 4;              // rows in flight per first-writer warp (ring of row slots in shared memory, filled by bulk copies)
constexpr int kBrRowBytes = 2048;        // one row slot: R_Y 512 B | R_X 512 B | Y 1024 B for 128 vectors
constexpr int kBrRingBytes = kBrWarps * kBrSlots * kBrRowBytes;
constexpr int kBrAhead = 4;              // tiles the first-writer warps may run ahead of the assembly (ring of br_done / epi_free barriers)
constexpr int kWarpBr = kWarpMma + 1;
constexpr int kThreads = 32 * (kWarpBr + kBrWarps);   // warps 0-7 assembly, 8-11 gather, 12 TMA, 13 MMA / TMEM owner, 14-21 first writers
constexpr int kMaxStages = 8;
// default block of the cell order (cells per direction; see cell_order): PAWFE_TC_ORDER_BLOCK=bx,by,bz overrides it at plan creation
constexpr int kOrderBlock[3] = {8, 8, 8};   // 64 cells per colour: enough independent tiles between a cell and the neighbours it waits for (profiles/r02_cell_kernel_ordered.md)

// Timing experiments (switching parts of the kernel OFF gives WRONG results) exist only in builds with -DPAWFE_TC_DEBUG
// (PAWFE_TC_DEBUG=1 python -m paper_2604_26037_b200.build); the shipped kernel has none of these branches.
#ifdef PAWFE_TC_DEBUG
#define TC_DBG(a, bit) (((a).dbg & (bit)) != 0)
#else
#define TC_DBG(a, bit) false
#endif

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
  int scale_mode;            // 0: s = alpha * acc;  1: s = alpha * M_D^-1[J] * acc
  // K-extension chunks (fused.h): per cell a CSR list of 32-row chunks whose A rows come from Wcat[atom]
  const int* ext_start; const int* ext_atom; const float* Wcat; long ldw; int ext_ksteps;
  const float* H32t; const float* Bext;   // pre-swizzled, block-contiguous operand streams
  // ordered assembly (see the header of this file)
  const int* order;        // tile sequence -> cell
  const int* dep_start;    // [ncell + 1]: cell -> its neighbours that precede it in the order
  const int* dep;
  const uint32_t* early;   // [ncell]: bit ((dx+1)*3 + (dy+1))*3 + (dz+1) set if that neighbour cell exists and precedes the cell
  int* flag;               // [ncell] completion counters; a cell is finished in this launch when its counter reaches flag_target
  int flag_target;
  // epilogue
  int epi_mode;            // TcEpiMode
  const double* Yt; const double* aLam; float ac, zz1; int cw;
  int dbg;                 // PAWFE_TC_DEBUG builds only: 2 no output, 4 no gather loads, 8 no MMAs, 16 no epilogue, 32 no first-writer
                           // stream, 64 no waiting for neighbours, 512 no L2 hint on the bulk copies, 4096 no bulk copies
};

struct TcPlan {
  float* d_H32t_lo = nullptr;    // low parts (value - trunc_tf32(value)) of d_H32t, FP32 mode only
  long h32t_elems = 0;
  float* d_H32t = nullptr;       // cell matrices re-tiled for streaming: [cell][half][K chunk][NT rows][32] floats
  int* d_order = nullptr;        // cell visiting order
  int* d_dep_start = nullptr; int* d_dep = nullptr;
  uint32_t* d_early = nullptr;
  int* d_flag = nullptr;
  int flag_base = 0;             // value every completion counter holds between launches
  int NT = 0, NH = 0;
  bool nopair = false;           // PAWFE_TC_NOPAIR (read once, at plan creation)
  int stage_cap = kMaxStages;    // PAWFE_TC_STAGES
  int dbg = 0;                   // PAWFE_TC_DBG (PAWFE_TC_DEBUG builds only)
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

__device__ __forceinline__ void bar_sync_epi(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(kEpiThreads) : "memory"); }
__device__ __forceinline__ void bar_sync_gather(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(kGatherThreads) : "memory"); }

__device__ __forceinline__ void bar_sync_br(int id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(kBrThreads) : "memory"); }

// Output node I of (cell, half): byte offset of its row in Y (a multiple of 16) | bit 0: this cell is the node's FIRST
// WRITER (no cell sharing the node precedes it in the order) | bit 1: masked (Dirichlet wall row, or I beyond n); *sc: scale.
__device__ __forceinline__ long node_entry(const TcArgs& a, int cx, int cy, int cz, int half, int I, uint32_t early, float* sc) {
  const int n1 = a.md.n1;
  const int Ig = half * a.NT + I;
  *sc = 0.f;
  if (Ig >= a.n) return 2;          // no node: masked, never written
  int c = Ig % n1, b = (Ig / n1) % n1, aa = Ig / (n1 * n1), ix, iy, iz;
  const long J = mesh_node(a.md, cx, cy, cz, aa, b, c, &ix, &iy, &iz);
  const double mi = a.md.mdinv1[0][ix] * a.md.mdinv1[1][iy] * a.md.mdinv1[2][iz];
  // cells sharing this node: offsets (0 | sx, 0 | sy, 0 | sz) with s = -1 / +1 on the low / high face of the cell
  const int sx = aa == 0 ? -1 : (aa == a.md.p ? 1 : 0), sy = b == 0 ? -1 : (b == a.md.p ? 1 : 0), sz = c == 0 ? -1 : (c == a.md.p ? 1 : 0);
  uint32_t share = 0;
#pragma unroll
  for (int u = 1; u < 8; ++u) {
    if (((u & 1) && !sx) || ((u & 2) && !sy) || ((u & 4) && !sz)) continue;
    const int dx = (u & 1) ? sx : 0, dy = (u & 2) ? sy : 0, dz = (u & 4) ? sz : 0;
    share |= 1u << (((dx + 1) * 3 + (dy + 1)) * 3 + (dz + 1));
  }
  *sc = a.scale_mode ? (float)((double)a.alpha * mi) : a.alpha;
  return (J * a.ldy * 4) | ((early & share) == 0 ? 1 : 0) | (mi == 0.0 ? 2 : 0);
}

// Persistent CTAs (one per SM) loop over tiles (cell, node half); inside a tile over the vector tiles of 128
// ("subtiles").  Accumulators are double-buffered in tensor memory (subtile parity), so the assembly epilogue of one
// subtile runs under the loads and MMAs of the next.  Roles are decoupled through mbarriers only.
//   PAIR = false: one CTA per tile; the first vector tile streams its H^e half from HBM, the following ones re-read it
//     from L2.
//   PAIR = true (blocks wider than 128 columns): the two CTAs of a cluster (one TPC) work on the same tile with
//     tcgen05.mma.cta_group::2, M = 256: CTA r gathers and assembles vector tile 2j + r and loads only rows
//     [r NT/2, (r+1) NT/2) of every matrix block, so each H^e block crosses L2 -> SM once per pair instead of once per
//     vector tile.  The leader (rank 0) issues the MMAs for both; rank 1's owner warp forwards "stage full" to it.
template <bool PAIR, bool CPLX>
__global__ void __launch_bounds__(kThreads, 1)
k_cell_tcgen05(const TcArgs a) {
  constexpr int ncomp = CPLX ? 2 : 1;   // complex: two matrix blocks (Re, Im) per stage and two accumulators per buffer
  extern __shared__ __align__(1024) uint8_t smem[];
  const int bbytes1 = (PAIR ? a.NT / 2 : a.NT) * 128;   // this CTA's rows of one matrix block (Re or Im)
  const int bbytes = ncomp * bbytes1;
  const int sbytes = kABytes + bbytes;                  // one stage: [A][B (Re)][B (Im)]
  int* gR = reinterpret_cast<int*>(smem + a.stages * sbytes);             // [kchunks * 32] gather rows: node index or -1
  long* eJ = reinterpret_cast<long*>(gR) + a.NH * a.NT;                   // [NT] output rows of this half: byte offset | flags
  float* eS = reinterpret_cast<float*>(eJ + a.NT);                        // [NT] output scale
  float* stage_epi = eS + a.NT;                                           // [epilogue warps][32 nodes][32 vectors]
  uint64_t* full = reinterpret_cast<uint64_t*>(stage_epi + kEpiWarps * 32 * 32);  // [stages]
  uint64_t* empty = full + kMaxStages;                                    // [stages]
  uint64_t* full_peer = empty + kMaxStages;                               // [stages] leader: rank 1's stage is full
  uint64_t* accum_full = full_peer + kMaxStages;                          // [2]
  uint64_t* accum_empty = accum_full + 2;                                 // [2]
  uint64_t* br_done = accum_empty + 2;                                    // [kBrAhead] first-writer rows of a tile are initialised (tile_iter % kBrAhead)
  uint64_t* epi_free = br_done + kBrAhead;                                // [kBrAhead] the assembly of that tile is done
  uint32_t* bL = reinterpret_cast<uint32_t*>(epi_free + kBrAhead);               // [NT] rows the first-writer warps' tile writes first (byte offset / 16)
  int* bN = reinterpret_cast<int*>(bL + a.NT);                            // their number
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bN + 4);
  uint64_t* br_bar = reinterpret_cast<uint64_t*>(tmem_slot + 4);          // [first-writer warps][slots] a row's operands have landed
  uint8_t* br_ring = reinterpret_cast<uint8_t*>(br_bar + kBrWarps * kBrSlots);   // [first-writer warps][slots][2048] (16-byte aligned)

  // the shuffle tells the compiler that the warp index is warp-uniform: role branches become uniform branches and the
  // operands computed inside them can live in uniform registers
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  const uint32_t rank = PAIR ? ptx::cluster_ctarank() : 0u;
  if (threadIdx.x == 0) {
    for (int s = 0; s < a.stages; ++s) { ptx::mbar_init(&full[s], kGatherThreads + 1); ptx::mbar_init(&empty[s], 1); ptx::mbar_init(&full_peer[s], 1); }
    // accum_empty: PAIR: one arrival per epilogue warp of both CTAs, on the leader's barrier
    for (int b = 0; b < 2; ++b) { ptx::mbar_init(&accum_full[b], 1); ptx::mbar_init(&accum_empty[b], PAIR ? 2 * kEpiWarps : kEpiThreads); }
    for (int b = 0; b < kBrAhead; ++b) { ptx::mbar_init(&br_done[b], kBrWarps); ptx::mbar_init(&epi_free[b], kEpiWarps); }
    for (int b = 0; b < kBrWarps * kBrSlots; ++b) ptx::mbar_init(&br_bar[b], 1);
    ptx::fence_barrier_init();
  }
  if (PAIR) ptx::cluster_sync();   // both CTAs' barriers exist before any remote arrival or multicast commit
  if (warp == kWarpMma) { if (PAIR) ptx::tmem_alloc_pair(tmem_slot, a.tmem_cols); else ptx::tmem_alloc(tmem_slot, a.tmem_cols); }
  ptx::tc_fence_before_sync();
  __syncthreads();
  ptx::tc_fence_after_sync();
  const uint32_t tmem_base = __shfl_sync(0xffffffffu, *tmem_slot, 0);
  const int n1 = a.md.n1;
  const int nsub = PAIR ? (a.nvt + 1) / 2 : a.nvt;   // subtiles per tile; subtile j of CTA r is vector tile 2j + r (PAIR) or j
  // 32-bit shared-memory addresses of the stage ring and the barriers (8 bytes per barrier)
  const uint32_t sm0 = ptx::smem_u32(smem);
  const uint32_t full_a = ptx::smem_u32(full), empty_a = ptx::smem_u32(empty), fpeer_a = ptx::smem_u32(full_peer);
  const uint32_t accf_a = ptx::smem_u32(accum_full), acce_a = ptx::smem_u32(accum_empty);
  // gather threads: local (a, b, c) of the up to four cell nodes whose row index this thread computes per tile
  constexpr int kDec = 512 / kGatherThreads;   // n <= 512
  int gdec[kDec];
  for (int k = 0; k < kDec; ++k) gdec[k] = -1;
  if (warp >= kEpiWarps && warp < kWarpTma) {
    for (int k = 0; k < kDec; ++k) {
      const int I = (int)threadIdx.x - kEpiThreads + kGatherThreads * k;
      if (I < a.n) gdec[k] = (I / (n1 * n1)) | (((I / n1) % n1) << 8) | ((I % n1) << 16);
    }
  }
  const uint64_t pol_stream = ptx::policy_evict_first();   // data read once per launch: cell-matrix blocks, residual source
  const uint64_t pol_keep = ptx::policy_evict_last();      // the rows of Y: written first, then added to by up to 7 later cells

  uint32_t st_s = 0, st_ph = 0;   // running stage index and phase of this role's walk over the ring (same sequence in every role)
  uint32_t sub_iter = 0;          // running subtile counter: accumulator buffer = sub_iter & 1
  uint32_t brc = 0;               // first-writer warps: running count of rows issued (slot = brc % kBrSlots, phase from brc / kBrSlots)
  uint32_t tile_iter = 0;         // running tile counter of this CTA: br_done / epi_free barrier = tile_iter % kBrAhead
  const bool init_rows = a.epi_mode != TC_EPI_ADD;   // the first-writer warps have work
  for (int tile = PAIR ? blockIdx.x >> 1 : blockIdx.x; tile < a.ntiles; tile += PAIR ? gridDim.x >> 1 : gridDim.x) {
    const int cseq = tile / a.NH;
    const int half = tile - cseq * a.NH;
    const int cell = __shfl_sync(0xffffffffu, a.order[cseq], 0);
    // (values read from memory are made warp-uniform explicitly, see the note on `warp`)
    const int ext0 = __shfl_sync(0xffffffffu, a.ext_start ? a.ext_start[cell] : 0, 0);
    const int nchunks = a.kchunks + __shfl_sync(0xffffffffu, a.ext_start ? a.ext_start[cell + 1] - ext0 : 0, 0);
    int cx, cy, cz;
    mesh_cell_coords(a.md, cell, &cx, &cy, &cz);

    if (warp < kEpiWarps) {
      // ================= epilogue: TMEM -> ordered assembly into Y (Fig. 2 step iv) =================
      // (the previous tile ended with a barrier of the epilogue warps: eJ / eS are free)
      const uint32_t early = a.early[cell];
      for (int I = threadIdx.x; I < a.NT; I += kEpiThreads) {
        float sc;
        eJ[I] = node_entry(a, cx, cy, cz, half, I, early, &sc);
        eS[I] = sc;
      }
      // ordered assembly: every neighbour that precedes this cell in the order has finished writing
      if (warp == 0) {
        const int d0 = a.dep_start[cell], nd = a.dep_start[cell + 1] - d0;   // at most 26
        if (lane < nd && !TC_DBG(a, 64)) {
          const int* f = a.flag + a.dep[d0 + lane];
          while (ptx::ld_acquire_gpu(f) < a.flag_target) __nanosleep(64);
        }
        __syncwarp();
      }
      bar_sync_epi(2);
      const int ncols = min(a.NT, a.n - half * a.NT);
      // Each warp owns 32 vectors (TMEM lanes).  32 output nodes at a time: TMEM -> registers (lane = vector) ->
      // scaled -> staging tile [node][vector] in shared memory -> each thread takes 4 consecutive vectors of one
      // node: ONE 16-byte store (first writer) or vector reduction (REDG.128) per node and thread.
      float* stg = stage_epi + warp * (32 * 32);
      const int quad = warp & 3, grp = warp >> 2;   // TMEM lanes [32 quad, 32 quad + 32); column groups grp, grp + 2, ...
      const int sub = lane >> 3, v4 = (lane & 7) * 4;
      // the rows this tile writes first hold their initial value (bracket of Alg. 2 step 4, or 0): first-writer warps
      if (init_rows) ptx::mbar_wait_relaxed(&br_done[tile_iter % kBrAhead], (tile_iter / kBrAhead) & 1, 2000);
      for (int j = 0; j < nsub; ++j) {
        const uint32_t buf = (sub_iter + j) & 1, use = (sub_iter + j) >> 1;
        ptx::mbar_wait_relaxed(&accum_full[buf], use & 1, 2000);
        ptx::tc_fence_after_sync();
        const int vt = PAIR ? 2 * j + (int)rank : j;
        const int vb = vt * kTileV + quad * 32;
        const bool vok = vb + v4 < a.B;             // B % 4 == 0: a float4 is all in or all out
        char* yv = reinterpret_cast<char*>(a.Y + vb + v4);
        if (vb < a.B && !TC_DBG(a, 16) && CPLX) {
          // complex: columns are interleaved (re, im); with P = X^T Hr^T and Q = X^T Hi^T,
          //   Y_re = P_re - Q_im,  Y_im = P_im + Q_re  ->  y = P + (lane odd ? +1 : -1) * Q of the partner lane
          const float sg = (lane & 1) ? 1.f : -1.f;
          for (int col0 = 16 * grp; col0 < ncols; col0 += 16 * (kEpiWarps / 4)) {
            uint32_t r[16], q[16];
            const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + buf * a.acc_stride + (uint32_t)col0;
            ptx::tmem_ld16(taddr, r);
            ptx::tmem_ld16(taddr + a.NT, q);
            ptx::tmem_ld_wait();
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
            if (vok && !TC_DBG(a, 2)) {
              const int nq = min(16, ncols - col0);
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                const int k = sub + 4 * i;
                const long e = k < nq ? eJ[col0 + k] : 2;
                if (!(e & 2)) { if (TC_DBG(a, 2048)) ptx::red_add_v4(reinterpret_cast<float*>(yv + (e & ~15L)), *reinterpret_cast<const float4*>(&stg[k * 32 + v4])); else ptx::red_add_v4_hint(reinterpret_cast<float*>(yv + (e & ~15L)), *reinterpret_cast<const float4*>(&stg[k * 32 + v4]), pol_keep); }
              }
            }
            __syncwarp();
          }
        } else if (vb < a.B && !TC_DBG(a, 16)) {
          for (int col0 = 32 * grp; col0 < ncols; col0 += 32 * (kEpiWarps / 4)) {
            uint32_t r[32];
            const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + buf * a.acc_stride + (uint32_t)col0;
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
            if (vok && !TC_DBG(a, 2)) {
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                const int q = sub + 4 * i;
                const long e = q < nq ? eJ[col0 + q] : 2;
                if (!(e & 2)) { if (TC_DBG(a, 2048)) ptx::red_add_v4(reinterpret_cast<float*>(yv + (e & ~15L)), *reinterpret_cast<const float4*>(&stg[q * 32 + v4])); else ptx::red_add_v4_hint(reinterpret_cast<float*>(yv + (e & ~15L)), *reinterpret_cast<const float4*>(&stg[q * 32 + v4]), pol_keep); }
              }
            }
            __syncwarp();
          }
        }
        ptx::tc_fence_before_sync();
        if (PAIR) {
          __syncwarp();
          if (lane == 0) { if (rank == 0) ptx::mbar_arrive(&accum_empty[buf]); else ptx::mbar_arrive_remote(&accum_empty[buf], 0); }
        } else {
          ptx::mbar_arrive(&accum_empty[buf]);
        }
      }
      // this CTA's share of the tile is written: count it on the cell.  The barrier orders every assembly thread's writes
      // (and, through br_done, the first-writer warps' stores) before thread 0's release at gpu scope, which is cumulative
      // (the grid-synchronisation pattern: barrier, then ONE thread fences and signals); the other warps go on to the next
      // tile instead of each draining its own reductions with a fence.
      if (init_rows) { __syncwarp(); if (lane == 0) ptx::mbar_arrive(&epi_free[tile_iter % kBrAhead]); }
      bar_sync_epi(2);
      if (threadIdx.x == 0) { __threadfence(); ptx::red_release_gpu_add(a.flag + cell, 1); }
    } else if (warp < kWarpTma) {
      // ================= gather producers: X rows -> swizzled MN-major A tiles (Fig. 2 step i) =================
      // (the loops of the three producer / issuer roles are kept lean: one warp per scheduler runs them, so every
      //  dependent instruction costs its full latency; stage index and phase are running counters, shared-memory
      //  addresses are 32-bit values computed once, and the row indices of a chunk are read before the wait)
      const int t = threadIdx.x - kEpiThreads;  // 0 .. kGatherThreads - 1
      bar_sync_gather(1);   // previous tile's readers of gR are done
      for (int k = 0; k < kDec; ++k) {
        const int I = t + kGatherThreads * k;
        if (I >= a.kchunks * kChunkK) break;
        int J = -1;
        if (gdec[k] >= 0) {
          int ix = cx * a.md.p + (gdec[k] & 0xff), iy = cy * a.md.p + ((gdec[k] >> 8) & 0xff), iz = cz * a.md.p + (gdec[k] >> 16);
          bool masked = false;
          if (a.md.periodic) {
            if (ix >= a.md.N[0]) ix -= a.md.N[0];
            if (iy >= a.md.N[1]) iy -= a.md.N[1];
            if (iz >= a.md.N[2]) iz -= a.md.N[2];
          } else {   // Dirichlet walls: the rows where M_D^-1 is stored as 0
            masked = ix == 0 || iy == 0 || iz == 0 || ix == a.md.N[0] - 1 || iy == a.md.N[1] - 1 || iz == a.md.N[2] - 1;
          }
          if (!masked) J = (ix * a.md.N[1] + iy) * a.md.N[2] + iz;
        }
        gR[I] = J;
      }
      bar_sync_gather(1);
      // per-thread constants: this thread always copies 16-byte column `lane` of rows wg, wg + 8, ... of a chunk
      constexpr int kRows = kChunkK / kGatherWarps;        // rows of a chunk per thread
      const int wg = t >> 5;                               // first row; wg % 4 is the row's place in its group of 4
      const int vl = lane * 4;                             // first vector of the 16-byte piece inside the tile
      // MN-major tf32 layout (128-byte swizzle, 32-byte atoms): 32-vector column block cb at cb * 4096; row r at
      // r * 128; its four 32-byte chunks q stored at q ^ (r % 4); r % 4 == wg for every row this thread copies
      const uint32_t dst_thread = sm0 + (lane >> 3) * 4096 + wg * 128 + (((((lane & 7) >> 1) ^ (wg & 3)) << 5) | ((lane & 1) << 4));
      const long ldx4 = a.ldx * 4;
      for (int j = 0; j < nsub; ++j) {
        const int vt = PAIR ? 2 * j + (int)rank : j;
        const int v = vt * kTileV + vl;
        const bool vok = v < a.B;
        const char* xv = reinterpret_cast<const char*>(a.X + v);
        const int* rows_t = gR + wg;
        for (int c = 0; c < a.kchunks; ++c, rows_t += kChunkK) {
          int rows[kRows];
#pragma unroll
          for (int i = 0; i < kRows; ++i) rows[i] = rows_t[kGatherWarps * i];
          ptx::mbar_wait(empty_a + 8 * st_s, st_ph ^ 1);
          const uint32_t abase = dst_thread + st_s * sbytes;
#pragma unroll
          for (int i = 0; i < kRows; ++i) {
            const bool ok = vok && rows[i] >= 0;
            if (!TC_DBG(a, 4)) ptx::cp_async16(abase + i * (128 * kGatherWarps), ok ? xv + rows[i] * ldx4 : reinterpret_cast<const char*>(a.X), ok ? 16u : 0u);
          }
          // arrival on full[s] fires when all of this thread's copies above have landed: no wait here, the thread
          // goes straight on to the next chunk (gated only by that stage being free)
          ptx::cp_async_mbar_arrive_noinc(full_a + 8 * st_s);
          if (++st_s == (uint32_t)a.stages) { st_s = 0; st_ph ^= 1; }
        }
        for (int c = a.kchunks; c < nchunks; ++c) {
          const float* wrows = a.Wcat + ((long)a.ext_atom[ext0 + c - a.kchunks] * 32 + wg) * a.ldw + v;
          ptx::mbar_wait(empty_a + 8 * st_s, st_ph ^ 1);
          const uint32_t abase = dst_thread + st_s * sbytes;
#pragma unroll
          for (int i = 0; i < kRows; ++i)
            ptx::cp_async16(abase + i * (128 * kGatherWarps), vok ? wrows + (long)(kGatherWarps * i) * a.ldw : a.X, vok ? 16u : 0u);
          ptx::cp_async_mbar_arrive_noinc(full_a + 8 * st_s);
          if (++st_s == (uint32_t)a.stages) { st_s = 0; st_ph ^= 1; }
        }
      }
    } else if (warp == kWarpTma) {
      // ================= TMA producer: H^e row block (or K-extension block), one K chunk per stage =================
      // (the whole warp runs the loop so that every operand stays warp-uniform -- the bulk-copy and MMA instructions take
      //  their operands from uniform registers, and per-thread values would each cost an election + broadcast sequence;
      //  only the instructions with side effects are issued by one lane)
      {
        // both operand streams are stored pre-swizzled and block-contiguous: one linear bulk copy per chunk and component;
        // PAIR: this CTA's half of the rows of every component block (NT / 2 is a multiple of 8: the swizzle phase is kept)
        const long comp_stride = (long)a.NT * 32, chunk_stride = comp_stride * ncomp;
        const long my_rows = PAIR ? (long)rank * (a.NT / 2) * 32 : 0;
        const float* hsrc0 = a.H32t + (long)(cell * a.NH + half) * a.kchunks * chunk_stride + my_rows;
        for (int j = 0; j < nsub; ++j) {
          const float* src = hsrc0;
          for (int c = 0; c < nchunks; ++c, src += chunk_stride) {
            if (c == a.kchunks) src = a.Bext + ((long)ext0 * a.NH + half) * chunk_stride + my_rows;
            const long step = c >= a.kchunks ? (long)(a.NH - 1) * chunk_stride : 0;   // extension blocks: [entry][half]
            ptx::mbar_wait(empty_a + 8 * st_s, st_ph ^ 1);
            const uint32_t dst = sm0 + st_s * sbytes + kABytes;
            if (ptx::elect_one()) {
              ptx::mbar_arrive_expect_tx(full_a + 8 * st_s, TC_DBG(a, 4096) ? 0u : (uint32_t)bbytes);
              if (TC_DBG(a, 4096)) {
              } else if (TC_DBG(a, 512)) {
#pragma unroll
                for (int comp = 0; comp < ncomp; ++comp)
                  ptx::bulk_load(dst + comp * bbytes1, src + comp * comp_stride, (uint32_t)bbytes1, full_a + 8 * st_s);
              } else if (PAIR || !CPLX) {
#pragma unroll
                for (int comp = 0; comp < ncomp; ++comp)
                  ptx::bulk_load_hint(dst + comp * bbytes1, src + comp * comp_stride, (uint32_t)bbytes1, full_a + 8 * st_s, pol_stream);
              } else {
                ptx::bulk_load_hint(dst, src, (uint32_t)bbytes, full_a + 8 * st_s, pol_stream);
              }
            }
            src += step;
            if (++st_s == (uint32_t)a.stages) { st_s = 0; st_ph ^= 1; }
          }
        }
      }
      __syncwarp();
    } else if (warp == kWarpMma) {
      // ================= MMA issuer =================
      if (PAIR && rank == 1) {
        // rank 1 issues no MMAs: tell the leader when a stage of THIS CTA holds its operands
        {
          const uint32_t peer_a = ptx::map_to_rank(fpeer_a, 0);
          for (int cnt = nchunks * nsub; cnt > 0; --cnt) {
            ptx::mbar_wait(full_a + 8 * st_s, st_ph);
            if (ptx::elect_one()) {
              ptx::fence_proxy_async_smem();   // cp.async (generic proxy) writes -> tensor-core (async proxy) reads
              // relaxed: the operands were complete in THIS CTA's shared memory when full[s] flipped (observed above), the
              // arrival is issued after that wait, and the leader's MMA is issued after it has seen the arrival; a
              // release at cluster scope costs a full memory barrier per chunk (measured: +0.2 ms per launch)
              ptx::mbar_arrive_cluster_relaxed(peer_a + 8 * st_s);
            }
            if (++st_s == (uint32_t)a.stages) { st_s = 0; st_ph ^= 1; }
          }
        }
      } else {
        const uint64_t adesc_c = ptx::smem_desc(0, 4096, 512, 1);
        const uint64_t bdesc_c = ptx::smem_desc_sw128(0, 16, 1024);
        for (int j = 0; j < nsub; ++j) {
          const uint32_t buf = (sub_iter + j) & 1, use = (sub_iter + j) >> 1;
          if (PAIR) ptx::mbar_wait_cluster(acce_a + 8 * buf, (use & 1) ^ 1);
          else ptx::mbar_wait(acce_a + 8 * buf, (use & 1) ^ 1);   // buffer drained by the epilogue of two subtiles ago
          ptx::tc_fence_after_sync();
          const uint32_t dtm = tmem_base + buf * a.acc_stride;
          for (int c = 0; c < nchunks; ++c) {
            ptx::mbar_wait(full_a + 8 * st_s, st_ph);
            if (PAIR) ptx::mbar_wait_cluster(fpeer_a + 8 * st_s, st_ph);
            ptx::fence_proxy_async_smem();   // cp.async (generic proxy) writes of the A tile -> tensor-core (async proxy) reads
            ptx::tc_fence_after_sync();
            // descriptors: constant fields | stage address in 16-byte units (stage bases are 1024-byte aligned)
            //   A (MN-major, 128B swizzle / 32B atoms): 4 blocks of 32 vectors 4096 B apart (LBO); K atoms of 4 rows
            //     512 B apart (SBO); one K step = 8 rows = 1024 B = 64 units
            //   B (K-major, SW128): 8-row groups 1024 B apart (SBO); 8 tf32 = 32 B = 2 units per K step
            const uint32_t a16 = (sm0 + st_s * sbytes) >> 4;
            const uint64_t ad = adesc_c | (uint64_t)(a16 & 0x3FFF);
            const uint64_t bd = bdesc_c | (uint64_t)((a16 + (kABytes >> 4)) & 0x3FFF);
            const int ksteps = (c == a.kchunks - 1) ? a.ksteps_last : (c >= a.kchunks ? a.ext_ksteps : kChunkK / 8);
            if (ptx::elect_one()) {
#pragma unroll
              for (int ks = 0; ks < kChunkK / 8; ++ks) {
                if (ks < ksteps && !TC_DBG(a, 8)) {
                  const uint32_t acc = (c | ks) != 0 ? 1u : 0u;
                  if (PAIR) ptx::mma_tf32_ss_pair(dtm, ad + ks * 64, bd + ks * 2, a.idesc, acc);
                  else ptx::mma_tf32_ss(dtm, ad + ks * 64, bd + ks * 2, a.idesc, acc);
                  if (CPLX) {
                    if (PAIR) ptx::mma_tf32_ss_pair(dtm + (uint32_t)a.NT, ad + ks * 64, bd + (bbytes1 >> 4) + ks * 2, a.idesc, acc);
                    else ptx::mma_tf32_ss(dtm + (uint32_t)a.NT, ad + ks * 64, bd + (bbytes1 >> 4) + ks * 2, a.idesc, acc);
                  }
                }
              }
              if (PAIR) ptx::mma_commit_pair(empty_a + 8 * st_s); else ptx::mma_commit(empty_a + 8 * st_s);
            }
            __syncwarp();
            if (++st_s == (uint32_t)a.stages) { st_s = 0; st_ph ^= 1; }
          }
          if (ptx::elect_one()) { if (PAIR) ptx::mma_commit_pair(accf_a + 8 * buf); else ptx::mma_commit(accf_a + 8 * buf); }
          __syncwarp();
        }
      }
      __syncwarp();
    } else if (init_rows) {
      // ================= first-writer warps: initial value of the rows this tile writes first =================
      // Streams  Y[J] = fp32(-ac X[J] - zz1 Y[J]) + Yt[J] aLam (FP64 add)  (bracket of Alg. 2 step 4, L272 / L374) or 0
      // (TC_EPI_STORE) into the rows whose first writer is this cell, under the MMAs of the tile; the assembly warps then
      // ADD the tile's contributions to every row.  A warp takes one node row at a time (32 lanes x 16 bytes = 128 vectors),
      // kBrSlots rows in flight.  No waiting for other cells: nobody else touches these rows before this cell is finished.
      const int t = threadIdx.x - 32 * kWarpBr, bw = t >> 5;
      if (tile_iter >= kBrAhead)   // the assembly of kBrAhead tiles ago has seen its br_done phase (no data dependence: these rows are this cell's alone)
        ptx::mbar_wait_relaxed(&epi_free[tile_iter % kBrAhead], ((tile_iter / kBrAhead) & 1) ^ 1, 2000);
      bar_sync_br(3);   // previous tile's readers of the row list are done
      if (t == 0) *bN = 0;
      bar_sync_br(3);
      const bool bracket = a.epi_mode == TC_EPI_BRACKET;
      {
        // compact list of the rows this tile writes first (bracket mode: without the Dirichlet wall rows, which stay 0 in
        // both recurrence states); order within the list does not matter.  Entry = byte offset of the row / 16.
        const uint32_t early = a.early[cell];
        for (int I = t; I < a.NT; I += kBrThreads) {
          float sc;
          const long e = node_entry(a, cx, cy, cz, half, I, early, &sc);
          if ((e & 1) && !(bracket && (e & 2))) bL[atomicAdd(bN, 1)] = (uint32_t)(e >> 4);
        }
      }
      bar_sync_br(3);
      const int nr = TC_DBG(a, 32) ? 0 : ((int)*bN - bw + kBrWarps - 1) / kBrWarps;   // rows of this warp: bw, bw + kBrWarps, ...
      const uint32_t* rows = bL + bw;
      const uint32_t ring = ptx::smem_u32(br_ring) + (uint32_t)(bw * kBrSlots * kBrRowBytes);
      const uint32_t rbar = ptx::smem_u32(br_bar) + (uint32_t)(bw * kBrSlots * 8);
      for (int j = 0; j < nsub; ++j) {
        const int v0 = (PAIR ? 2 * j + (int)rank : j) * kTileV;
        if (v0 >= a.B) continue;                       // (warp-uniform)
        const int v = v0 + lane * 4;
        const bool lane_ok = v < a.B;                  // B % 4 == 0: a float4 is all in or all out
        char* yg = reinterpret_cast<char*>(a.Y + v);
        if (!bracket) {                                // TC_EPI_STORE: zero (incl. Dirichlet wall rows)
          if (lane_ok)
            for (int i = 0; i < nr; ++i) ptx::stg_f4(yg + ((long)rows[kBrWarps * i] << 4), make_float4(0.f, 0.f, 0.f, 0.f));
          continue;
        }
        const char* xg0 = reinterpret_cast<const char*>(a.X + v0);
        const char* yg0 = reinterpret_cast<const char*>(a.Y + v0);
        const char* tg0 = reinterpret_cast<const char*>(a.Yt + v0);
        // bytes of a R_Y / R_X row piece of this vector tile; a ragged width is rounded up to whole 16-byte pieces (the pad
        // columns exist: leading dimensions are multiples of 4)
        const uint32_t rowb = (uint32_t)(min(kTileV, ((a.B + 3) & ~3) - v0) * 4);
        double l[4] = {0.0, 0.0, 0.0, 0.0};
        if (lane_ok) {
#pragma unroll
          for (int u = 0; u < 4; ++u) l[u] = a.aLam[(v + u) / a.cw];
        }
        // Operands of kBrSlots rows in flight, brought by the bulk-copy engine (three linear copies per row, issued by one
        // lane, completion on the slot's mbarrier): they occupy neither registers nor the load / store unit's miss tracking,
        // which the gather producers of the A tiles need.
        auto issue = [&](int i) {                      // row i of this warp into slot (brc + i) % kBrSlots
          if (i < nr && !TC_DBG(a, 256)) {
            const uint32_t s2 = (brc + (uint32_t)i) % kBrSlots;
            if (ptx::elect_one()) {
              const long off = (long)rows[kBrWarps * i] << 4;
              const uint32_t dst = ring + s2 * kBrRowBytes, bar = rbar + s2 * 8;
              ptx::mbar_arrive_expect_tx(bar, 4u * rowb);
              ptx::bulk_load(dst, xg0 + off, rowb, bar);
              ptx::bulk_load(dst + 512, yg0 + off, rowb, bar);
              ptx::bulk_load_hint(dst + 1024, tg0 + 2 * off, 2u * rowb, bar, pol_stream);
            }
          }
        };
#pragma unroll 1
        for (int i = 0; i < kBrSlots; ++i) issue(i);
#pragma unroll 2
        for (int i = 0; i < nr; ++i) {
          const uint32_t s2 = (brc + (uint32_t)i) % kBrSlots, ph = ((brc + (uint32_t)i) / kBrSlots) & 1;
          if (!TC_DBG(a, 256)) ptx::mbar_wait(rbar + s2 * 8, ph);     // row i has landed
          if (lane_ok) {
            const uint32_t src = ring + s2 * kBrRowBytes;
            const float4 ry = ptx::lds_f4(src + lane * 16), rx = ptx::lds_f4(src + 512 + lane * 16);
            const double2 ya = ptx::lds_d2(src + 1024 + lane * 32), yb = ptx::lds_d2(src + 1040 + lane * 32);
            float4 o;
            // bracket in FP32, residual-source term added in FP64, stored FP32 (L374)
            o.x = (float)((double)(-a.ac * ry.x - a.zz1 * rx.x) + ya.x * l[0]);
            o.y = (float)((double)(-a.ac * ry.y - a.zz1 * rx.y) + ya.y * l[1]);
            o.z = (float)((double)(-a.ac * ry.z - a.zz1 * rx.z) + yb.x * l[2]);
            o.w = (float)((double)(-a.ac * ry.w - a.zz1 * rx.w) + yb.y * l[3]);
            if (!TC_DBG(a, 128)) { if (TC_DBG(a, 2048)) ptx::stg_f4(yg + ((long)rows[kBrWarps * i] << 4), o); else ptx::stg_f4_hint(yg + ((long)rows[kBrWarps * i] << 4), o, pol_keep); }
          }
          __syncwarp();                                // every lane has read the slot before it is refilled
          issue(i + kBrSlots);
        }
        brc += (uint32_t)nr;                           // (rows beyond nr were never issued: the slot sequence continues at nr)
      }
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(&br_done[tile_iter % kBrAhead]);   // release: the stores above precede the assembly's reductions
    }
    sub_iter += (uint32_t)nsub;
    ++tile_iter;
  }
  ptx::tc_fence_before_sync();
  if (PAIR) ptx::cluster_sync(); else __syncthreads();   // PAIR: the peer's MMAs, commits and remote arrivals are done too
  ptx::tc_fence_after_sync();
  if (warp == kWarpMma) { if (PAIR) ptx::tmem_dealloc_pair(tmem_base, a.tmem_cols); else ptx::tmem_dealloc(tmem_base, a.tmem_cols); }
}

void shape_for(const pawfe_ctx* c, int* NH, int* NT) {
  // two accumulator buffers of ncomp * NT columns must fit the 512 TMEM columns
  const int maxnt = c->cplx ? 128 : 256;
  *NH = (c->n + maxnt - 1) / maxnt;
  int per = (c->n + *NH - 1) / *NH;
  *NT = (per + 15) / 16 * 16;
}

size_t smem_fixed(int NH, int NT) { return (size_t)NH * NT * 8 + (size_t)NT * 16 + kEpiWarps * 32 * 32 * 4 + (3 * kMaxStages + 4 + 2 * kBrAhead + kBrWarps * kBrSlots) * 8 + 32 + kBrRingBytes; }
// brows: rows of a matrix block one CTA holds per stage (NT, or NT / 2 for CTA pairs)
int stages_for(int NH, int NT, int ncomp, int brows) {
  const size_t budget = 227 * 1024 - 1024;  // dynamic shared memory per CTA, less the alignment slack
  int st = (int)((budget - smem_fixed(NH, NT)) / (size_t)(kABytes + ncomp * brows * 128));
  return std::min(st, kMaxStages);
}
size_t smem_bytes(int NH, int NT, int ncomp, int brows) {
  return (size_t)stages_for(NH, NT, ncomp, brows) * (kABytes + ncomp * brows * 128) + smem_fixed(NH, NT);
}

// Cell order of the ordered assembly: blocks of bs[0] x bs[1] x bs[2] cells (even sizes) one after the other; inside a
// block the 8 parity colours (cx % 2, cy % 2, cz % 2) one after the other.  Cells of one colour share no node, so the
// cells a cell has to wait for (its neighbours earlier in the order) were handed out well before it.  Smaller blocks
// keep the rows neighbouring cells share in L2 between their first and their last contribution; larger ones leave more
// independent tiles between a cell and the neighbours it waits for.
void cell_order(const pawfe_ctx* c, const int bs[3], std::vector<int>* order) {
  order->clear();
  order->reserve(c->ncell);
  for (int bx = 0; bx < c->nc[0]; bx += bs[0])
    for (int by = 0; by < c->nc[1]; by += bs[1])
      for (int bz = 0; bz < c->nc[2]; bz += bs[2])
        for (int col = 0; col < 8; ++col)
          for (int x = bx + (col & 1); x < std::min(bx + bs[0], c->nc[0]); x += 2)
            for (int y = by + ((col >> 1) & 1); y < std::min(by + bs[1], c->nc[1]); y += 2)
              for (int z = bz + ((col >> 2) & 1); z < std::min(bz + bs[2], c->nc[2]); z += 2)
                order->push_back((x * c->nc[1] + y) * c->nc[2] + z);
}

// For every cell: the neighbours (cells sharing a node) that precede it in the order, as a list and as a 27-bit mask
void order_dependencies(const pawfe_ctx* c, const std::vector<int>& order, std::vector<int>* dep_start, std::vector<int>* dep,
                        std::vector<uint32_t>* early) {
  const int ncell = c->ncell;
  const bool per = c->bc == PAWFE_PERIODIC;
  std::vector<int> pos(ncell);
  for (int s = 0; s < ncell; ++s) pos[order[s]] = s;
  dep_start->assign(ncell + 1, 0); dep->clear(); early->assign(ncell, 0u);
  for (int e = 0; e < ncell; ++e) {
    const int cz = e % c->nc[2], cy = (e / c->nc[2]) % c->nc[1], cx = e / (c->nc[1] * c->nc[2]);
    const size_t first = dep->size();
    for (int dx = -1; dx <= 1; ++dx)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dz = -1; dz <= 1; ++dz) {
          if (!dx && !dy && !dz) continue;
          int x = cx + dx, y = cy + dy, z = cz + dz;
          if (per) { x = (x + c->nc[0]) % c->nc[0]; y = (y + c->nc[1]) % c->nc[1]; z = (z + c->nc[2]) % c->nc[2]; }
          else if (x < 0 || y < 0 || z < 0 || x >= c->nc[0] || y >= c->nc[1] || z >= c->nc[2]) continue;
          const int e2 = (x * c->nc[1] + y) * c->nc[2] + z;
          if (e2 == e || pos[e2] > pos[e]) continue;
          (*early)[e] |= 1u << (((dx + 1) * 3 + (dy + 1)) * 3 + (dz + 1));
          if (std::find(dep->begin() + first, dep->end(), e2) == dep->end()) dep->push_back(e2);   // (two cells per direction: one cell, two offsets)
        }
    (*dep_start)[e + 1] = (int)dep->size();
  }
}

void free_plan(TcPlan* p) {
  if (!p) return;
  cudaFree(p->d_H32t_lo); cudaFree(p->d_H32t); cudaFree(p->d_order); cudaFree(p->d_dep_start); cudaFree(p->d_dep);
  cudaFree(p->d_early); cudaFree(p->d_flag);
  delete p;
}

// A plan that could not be completed is dropped again (the next call retries) and the cause is returned.
pawfe_status build_plan(pawfe_ctx* c, TcPlan** out) {
  *out = nullptr;
  if (!c->d_H32) { c->err = "tcgen05 cell kernel: no FP32 cell matrices"; return PAWFE_ESTATE; }
  TcPlan* p = new TcPlan();
  shape_for(c, &p->NH, &p->NT);
  // tuning switches are read once, here (never on the hot path)
  p->nopair = getenv("PAWFE_TC_NOPAIR") != nullptr;
  { const char* d = getenv("PAWFE_TC_STAGES"); if (d && atoi(d) >= 2) p->stage_cap = std::min(kMaxStages, atoi(d)); }
  { const char* d = getenv("PAWFE_TC_NT"); const int maxnt = c->cplx ? 128 : 256; if (d && atoi(d) >= p->NT && atoi(d) <= maxnt && atoi(d) % 16 == 0) p->NT = atoi(d); }
#ifdef PAWFE_TC_DEBUG
  { const char* d = getenv("PAWFE_TC_DBG"); p->dbg = d ? atoi(d) : 0; }
#endif
  pawfe_status st = PAWFE_OK;
  auto fail = [&](pawfe_status s) { free_plan(p); return s; };
  {
    int bs[3] = {c->nc[0], c->nc[1], c->nc[2]};   // default: the whole mesh is one block (colour after colour)
    if (const char* d = getenv("PAWFE_TC_ORDER_BLOCK")) {
      int b0 = 0, b1 = 0, b2 = 0;
      const int k = sscanf(d, "%d,%d,%d", &b0, &b1, &b2);
      if (k == 1) b1 = b2 = b0;
      if (k >= 1 && b0 >= 2 && b1 >= 2 && b2 >= 2 && !(b0 & 1) && !(b1 & 1) && !(b2 & 1)) { bs[0] = b0; bs[1] = b1; bs[2] = b2; }
    } else {
      for (int d = 0; d < 3; ++d) bs[d] = std::min(c->nc[d] + (c->nc[d] & 1), kOrderBlock[d]);
    }
    std::vector<int> order, dep_start, dep;
    std::vector<uint32_t> early;
    cell_order(c, bs, &order);
    order_dependencies(c, order, &dep_start, &dep, &early);
    if (dep.empty()) dep.push_back(0);
    if ((st = upload(c, &p->d_order, order)) != PAWFE_OK) return fail(st);
    if ((st = upload(c, &p->d_dep_start, dep_start)) != PAWFE_OK) return fail(st);
    if ((st = upload(c, &p->d_dep, dep)) != PAWFE_OK) return fail(st);
    if ((st = upload(c, &p->d_early, early)) != PAWFE_OK) return fail(st);
    if ((st = dev_alloc(c, &p->d_flag, (size_t)c->ncell)) != PAWFE_OK) return fail(st);
    if (cudaMemsetAsync(p->d_flag, 0, (size_t)c->ncell * sizeof(int), c->stream) != cudaSuccess) { cudaGetLastError(); return fail(PAWFE_ECUDA); }
  }
  const int ncomp = c->cplx ? 2 : 1;
  const int kchunks = (c->ldk + kChunkK - 1) / kChunkK;
  const long elems = (long)c->ncell * p->NH * kchunks * ncomp * p->NT * 32;
  if ((st = dev_alloc(c, &p->d_H32t, (size_t)elems)) != PAWFE_OK) return fail(st);
  p->h32t_elems = elems;
  k_retile_h32<<<8 * c->sm_count, 256, 0, c->stream>>>((const float*)c->d_H32, c->n, c->ldk, p->NH, p->NT, kchunks, ncomp, elems, p->d_H32t);
  c->launches++;
  if (cudaGetLastError() != cudaSuccess) { c->err = "k_retile_h32 launch failed"; return fail(PAWFE_ECUDA); }
  const void* k1 = c->cplx ? (const void*)k_cell_tcgen05<false, true> : (const void*)k_cell_tcgen05<false, false>;
  const void* k2 = c->cplx ? (const void*)k_cell_tcgen05<true, true> : (const void*)k_cell_tcgen05<true, false>;
  if ((st = pawfe_ensure_smem(c, k1, smem_bytes(p->NH, p->NT, ncomp, p->NT))) != PAWFE_OK) return fail(st);
  if ((st = pawfe_ensure_smem(c, k2, smem_bytes(p->NH, p->NT, ncomp, p->NT / 2))) != PAWFE_OK) return fail(st);
  p->ok = true;
  *out = p;
  return PAWFE_OK;
}

pawfe_status get_plan(pawfe_ctx* c, TcPlan** out) {
  if (!c->tc_plan) {
    TcPlan* p = nullptr;
    TRY(build_plan(c, &p));
    c->tc_plan = p;
  }
  *out = (TcPlan*)c->tc_plan;
  return PAWFE_OK;
}

}  // namespace

void tc_shape(const pawfe_ctx* c, int* NH, int* NT) {
  if (c->tc_plan) { *NH = ((TcPlan*)c->tc_plan)->NH; *NT = ((TcPlan*)c->tc_plan)->NT; return; }
  shape_for(c, NH, NT);
}

pawfe_status tc_prepare(pawfe_ctx* c) {
  TcPlan* p = nullptr;
  return get_plan(c, &p);
}

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
  TcPlan* p = nullptr;
  TRY(get_plan(c, &p));
  if (!p->d_H32t_lo) {   // first FP32-mode use (pawfe_prepare does this ahead of the hot calls)
    TRY(dev_alloc(c, &p->d_H32t_lo, (size_t)p->h32t_elems));
    pawfe_status st = tc_lo_part(c, p->d_H32t, p->d_H32t_lo, p->h32t_elems);
    if (st != PAWFE_OK) { cudaFree(p->d_H32t_lo); p->d_H32t_lo = nullptr; return st; }
  }
  *out = p->d_H32t_lo;
  return PAWFE_OK;
}

void tc_invalidate(pawfe_ctx* c) {
  if (c->tc_plan) { free_plan((TcPlan*)c->tc_plan); c->tc_plan = nullptr; }
}

bool tc_supported(const pawfe_ctx* c, int B) {
  if (!c->have_pot || B < 1) return false;
  if (c->n < 16) return false;
  return true;
}

bool tc_usable(pawfe_ctx* c, const void* X, long ldx, const void* Y, long ldy, int B) {
  if (!tc_supported(c, B)) return false;
  if ((ldx & 3) || (ldy & 3) || (B & 3) || ((uintptr_t)X & 15) || ((uintptr_t)Y & 15)) return false;
  TcPlan* p = nullptr;
  return get_plan(c, &p) == PAWFE_OK;
}

// Complex contexts: X, Y are the interleaved (re, im) blocks seen as real blocks, B = 2 x vectors, ldx / ldy in floats.
pawfe_status tc_cell_apply(pawfe_ctx* c, const float* X, long ldx, float* Y, long ldy, int B, float alpha,
                           const TcExt* ext, const TcEpi* epi) {
  TcPlan* p = nullptr;
  TRY(get_plan(c, &p));
  TcArgs a;
  a.md = c->md; a.X = X; a.ldx = ldx; a.Y = Y; a.ldy = ldy; a.B = B; a.alpha = alpha;
  a.n = c->n; a.NH = p->NH; a.NT = p->NT;
  a.kchunks = (c->ldk + kChunkK - 1) / kChunkK;
  a.ksteps_last = (c->ldk - (a.kchunks - 1) * kChunkK) / 8;
  a.nvt = (B + kTileV - 1) / kTileV;
  a.ntiles = c->ncell * a.NH;
  a.ncomp = c->cplx ? 2 : 1;
  // blocks wider than one vector tile: CTA pairs (cta_group::2), both vector tiles of a pair against one load of H^e
  const bool pair = a.nvt > 1 && c->sm_count >= 2 && !p->nopair;
  const int brows = pair ? p->NT / 2 : p->NT;
  a.stages = std::min(stages_for(p->NH, p->NT, a.ncomp, brows), p->stage_cap);
  uint32_t cols = 32;
  while ((int)cols < a.ncomp * a.NT) cols <<= 1;
  a.acc_stride = cols;
  a.tmem_cols = 2 * cols;
  a.idesc = ptx::idesc_tf32(pair ? 2 * kTileV : kTileV, a.NT, /*A MN-major*/ 1, /*B K-major*/ 0);
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
  a.epi_mode = epi ? epi->mode : TC_EPI_ADD;
  a.Yt = nullptr; a.aLam = nullptr; a.ac = 0.f; a.zz1 = 0.f; a.cw = 1;
  if (a.epi_mode == TC_EPI_BRACKET) {
    if (ldx != ldy || !epi->Yt || !epi->aLam || epi->cw < 1) { c->err = "tcgen05 cell kernel: the bracket epilogue needs X, Y, Yt with one leading dimension"; return PAWFE_EINVAL; }
    a.Yt = epi->Yt; a.aLam = epi->aLam; a.ac = epi->ac; a.zz1 = epi->zz1; a.cw = epi->cw;
  }
  // ordered assembly: one counter per cell; every CTA working on a (cell, half) tile counts once
  a.order = p->d_order; a.dep_start = p->d_dep_start; a.dep = p->d_dep; a.early = p->d_early; a.flag = p->d_flag;
  p->flag_base += a.NH * (pair ? 2 : 1);
  a.flag_target = p->flag_base;
  a.dbg = p->dbg;
  const size_t smem = smem_bytes(p->NH, p->NT, a.ncomp, brows);
  if (pair) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * (unsigned)std::min(a.ntiles, c->sm_count / 2));
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (c->cplx) CUDA_TRY(c, cudaLaunchKernelEx(&cfg, k_cell_tcgen05<true, true>, a));
    else CUDA_TRY(c, cudaLaunchKernelEx(&cfg, k_cell_tcgen05<true, false>, a));
    c->launches++;
    return PAWFE_OK;
  }
  int grid = std::min(a.ntiles, c->sm_count);
  if (c->cplx) k_cell_tcgen05<false, true><<<grid, kThreads, smem, c->stream>>>(a);
  else k_cell_tcgen05<false, false><<<grid, kThreads, smem, c->stream>>>(a);
  KERNEL_CHECK(c, "k_cell_tcgen05");
  return PAWFE_OK;
}
