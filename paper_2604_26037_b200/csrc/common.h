// common.h -- context, scalar helpers and kernel-launch declarations shared by the libpawfe.so sources.
// Product code: never includes or links anything under oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>
#include "../../include/pawfe.h"

#define PAWFE_MAX_NPJ 16
#define PAWFE_MAX_N1 8      // p <= 7
#define PAWFE_MAX_NQ3 18    // 2 (p + 2)

// ------------------------------------------------------------------------------------------------
// scalar helpers: real (float/double) and complex (float2/double2, interleaved re, im)
// ------------------------------------------------------------------------------------------------
template <typename T> struct ScalarTraits;
template <> struct ScalarTraits<float>   { typedef float real;  static const bool cplx = false; };
template <> struct ScalarTraits<double>  { typedef double real; static const bool cplx = false; };
template <> struct ScalarTraits<float2>  { typedef float real;  static const bool cplx = true; };
template <> struct ScalarTraits<double2> { typedef double real; static const bool cplx = true; };

__host__ __device__ inline float  s_zero(float)   { return 0.f; }
__host__ __device__ inline double s_zero(double)  { return 0.0; }
__host__ __device__ inline float2 s_zero(float2)  { return make_float2(0.f, 0.f); }
__host__ __device__ inline double2 s_zero(double2){ return make_double2(0.0, 0.0); }

// acc += a * b
__device__ inline void s_fma(float& acc, float a, float b)    { acc = fmaf(a, b, acc); }
__device__ inline void s_fma(double& acc, double a, double b) { acc = fma(a, b, acc); }
__device__ inline void s_fma(float2& acc, float2 a, float2 b) {
  acc.x = fmaf(a.x, b.x, acc.x); acc.x = fmaf(-a.y, b.y, acc.x);
  acc.y = fmaf(a.x, b.y, acc.y); acc.y = fmaf(a.y, b.x, acc.y);
}
__device__ inline void s_fma(double2& acc, double2 a, double2 b) {
  acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a) * b
__device__ inline void s_fma_conj(float& acc, float a, float b)    { acc = fmaf(a, b, acc); }
__device__ inline void s_fma_conj(double& acc, double a, double b) { acc = fma(a, b, acc); }
__device__ inline void s_fma_conj(float2& acc, float2 a, float2 b) {
  acc.x = fmaf(a.x, b.x, acc.x); acc.x = fmaf(a.y, b.y, acc.x);
  acc.y = fmaf(a.x, b.y, acc.y); acc.y = fmaf(-a.y, b.x, acc.y);
}
__device__ inline void s_fma_conj(double2& acc, double2 a, double2 b) {
  acc.x = fma(a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y); acc.y = fma(-a.y, b.x, acc.y);
}
// real scale
__device__ inline float   s_scale(float a, double r)   { return a * (float)r; }
__device__ inline double  s_scale(double a, double r)  { return a * r; }
__device__ inline float2  s_scale(float2 a, double r)  { float f = (float)r; return make_float2(a.x * f, a.y * f); }
__device__ inline double2 s_scale(double2 a, double r) { return make_double2(a.x * r, a.y * r); }
__device__ inline float   s_add(float a, float b)     { return a + b; }
__device__ inline double  s_add(double a, double b)   { return a + b; }
__device__ inline float2  s_add(float2 a, float2 b)   { return make_float2(a.x + b.x, a.y + b.y); }
__device__ inline double2 s_add(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }

// conversions between storage and compute scalars
__device__ inline void s_cvt(float& d, float s)     { d = s; }
__device__ inline void s_cvt(float& d, double s)    { d = (float)s; }
__device__ inline void s_cvt(double& d, float s)    { d = (double)s; }
__device__ inline void s_cvt(double& d, double s)   { d = s; }
__device__ inline void s_cvt(float2& d, float2 s)   { d = s; }
__device__ inline void s_cvt(float2& d, double2 s)  { d = make_float2((float)s.x, (float)s.y); }
__device__ inline void s_cvt(double2& d, float2 s)  { d = make_double2((double)s.x, (double)s.y); }
__device__ inline void s_cvt(double2& d, double2 s) { d = s; }

__device__ inline void s_atomic_add(float* p, float v)   { atomicAdd(p, v); }
__device__ inline void s_atomic_add(double* p, double v) { atomicAdd(p, v); }
__device__ inline void s_atomic_add(float2* p, float2 v) {
  atomicAdd(&p->x, v.x); atomicAdd(&p->y, v.y);
}
__device__ inline void s_atomic_add(double2* p, double2 v) {
  atomicAdd(&p->x, v.x); atomicAdd(&p->y, v.y);
}

// round an FP32 value to TF32 (10-bit mantissa, round to nearest, ties away) -- what the tensor core
// multiplier sees in kind::tf32; used by the SIMT emulation of the TF32 mode.
__device__ inline float tf32_round(float x) {
  uint32_t u;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"(x));
  return __uint_as_float(u);
}

// ------------------------------------------------------------------------------------------------
// mesh description passed by value to kernels
// ------------------------------------------------------------------------------------------------
struct MeshDev {
  int nc[3];       // cells per direction
  int N[3];        // stored nodes per direction
  int p, n1, n;    // order, p+1, (p+1)^3
  int periodic;    // 1 periodic, 0 Dirichlet
  long M;          // stored nodes
  int ncell;
  const double* mdinv1[3];  // device: per-direction factor of M_D^-1 (0 at Dirichlet boundary nodes)
  const double* md1[3];     // device: per-direction factor of M_D
};

// global node of cell (cx,cy,cz), local (a,b,c)
__host__ __device__ inline long mesh_node(const MeshDev& m, int cx, int cy, int cz, int a, int b, int c,
                                          int* ix_, int* iy_, int* iz_) {
  int ix = cx * m.p + a, iy = cy * m.p + b, iz = cz * m.p + c;
  if (m.periodic) {
    if (ix >= m.N[0]) ix -= m.N[0];
    if (iy >= m.N[1]) iy -= m.N[1];
    if (iz >= m.N[2]) iz -= m.N[2];
  }
  *ix_ = ix; *iy_ = iy; *iz_ = iz;
  return ((long)ix * m.N[1] + iy) * m.N[2] + iz;
}
__host__ __device__ inline void mesh_cell_coords(const MeshDev& m, int e, int* cx, int* cy, int* cz) {
  *cz = e % m.nc[2];
  *cy = (e / m.nc[2]) % m.nc[1];
  *cx = e / (m.nc[1] * m.nc[2]);
}

// ------------------------------------------------------------------------------------------------
// context
// ------------------------------------------------------------------------------------------------
struct pawfe_ctx {
  int device = 0;
  cudaStream_t stream = 0;
  std::string err;
  long launches = 0;
  int sm_count = 148;

  // mesh
  bool have_mesh = false;
  int nc[3] = {0, 0, 0};
  double box[3] = {0, 0, 0}, h[3] = {0, 0, 0};
  int p = 0, n1 = 0, n = 0, bc = 0;
  bool cplx = false;
  double kpt[3] = {0, 0, 0};
  int N[3] = {0, 0, 0};
  long M = 0;
  int ncell = 0;
  int ldk = 0;  // row stride (elements) of the FP32 cell matrices: n rounded up to a multiple of 8
  std::vector<double> xi, wgll, K1, M1, G1;  // host 1-D tables
  double* d_md1 = nullptr;     // device: [N0+N1+N2] M_D factors, then [N0+N1+N2] M_D^-1 factors
  MeshDev md{};
  double* d_M1 = nullptr;      // device: 1-D consistent mass matrix M1 [n1][n1] on the reference interval
  double* d_Mref64 = nullptr;  // reference mass cell matrix M^e (n x n), real
  float* d_Mref32 = nullptr;   // same in FP32 with row stride ldk

  // local operator
  bool have_pot = false;
  bool have_h64 = false;
  void* d_H64 = nullptr;  // [cell][n][n] double (complex: double2)
  void* d_H32 = nullptr;  // [cell][n][ldk] float (complex: float2)

  // atoms
  bool have_atoms = false;
  int natoms = 0, npj = 0;
  double rc = 0;
  std::vector<double> pos;
  std::vector<int> proj_l, proj_m;
  std::vector<double> proj_sigma, proj_amp;
  long npairs = 0;
  int* d_pair_cell = nullptr;        // [npairs]
  int* d_pair_atom = nullptr;        // [npairs]
  int* d_atom_pair_start = nullptr;  // [natoms+1], pairs sorted by atom
  std::vector<int> h_atom_pair_start;
  void* d_Cd64 = nullptr;  // [pair][npj][n]: rows of C^{e,a dagger} (Eq. 34), double / double2
  void* d_Cd32 = nullptr;  // same, float / float2
  std::vector<double> h_dS;          // natoms*npj*npj real
  std::vector<double> h_G;           // natoms*npj*npj scalars: G^a = C^a^dagger M_D^-1 C^a
  int sinv_variant = 0;              // which G^a enters Delta_Sinv (Eq. 29): 0 = C^a^dagger M_D^-1 C^a, 1 = <p_alpha|p_beta> (L228)
  std::vector<double> h_dSinv;       // natoms*npj*npj scalars: Delta^a_Sinv (Eq. 29)
  void* d_D64 = nullptr; void* d_dS64 = nullptr; void* d_dSinv64 = nullptr;  // [atom][npj][npj] scalar
  void* d_D32 = nullptr; void* d_dS32 = nullptr; void* d_dSinv32 = nullptr;
  void* d_P = nullptr;   // projection scratch: 2 x [natoms][npj][512] scalar (FP64-complex sized)
  size_t P_bytes = 0;

  // filter scalars
  static const int kScalSlots = 4;   // ring of pinned staging slots, each guarded by an event
  double* h_pinned = nullptr;  // pinned staging for lambda / coefficient tables [kScalSlots][scal_doubles]
  double* d_scal = nullptr;    // device copies [kScalSlots][scal_doubles]
  size_t scal_doubles = 0;
  cudaEvent_t scal_ev[4] = {nullptr, nullptr, nullptr, nullptr};
  int scal_next = 0;

  void* tc_plan = nullptr;  // cell_tcgen05.cu: cached tensor map and tile shape
  void* fused = nullptr;    // api_fused.cu: FusedPlan (K-extension blocks, neighbour couplings, scratch)

  // optional CUDA-event timing of the cell-contraction launches of the filter loop (pawfe_cell_timing)
  bool prof_on = false;
  std::vector<cudaEvent_t> prof_ev;  // pairs (start, stop)
  size_t prof_used = 0;
  std::vector<cudaEvent_t> prof_setup_ev;  // pairs around the residual set-up (Alg. 2 steps 2-3) of every filter call
  size_t prof_setup_used = 0;

  void* d_tmpblk = nullptr; size_t tmpblk_bytes = 0;   // block T of the unfused pawfe_apply_HSinv

  // host-buffer filter (pawfe_cheb_filter_host)
  void* d_hostblk = nullptr; size_t hostblk_bytes = 0;
  void* d_hostws = nullptr;  size_t hostws_bytes = 0;
  void* h_stage = nullptr;   size_t stage_bytes = 0;
  // pipelined host-buffer filter over a block set (pawfe_cheb_filter_host_set): second device block, copy streams, events
  void* d_hostblk2 = nullptr; size_t hostblk2_bytes = 0;
  cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
  cudaEvent_t ev_h2d[2] = {nullptr, nullptr}, ev_filt[2] = {nullptr, nullptr}, ev_d2h[2] = {nullptr, nullptr};
};

#define CUDA_TRY(ctx, call)                                                                   \
  do {                                                                                        \
    cudaError_t e_ = (call);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                        \
      return (e_ == cudaErrorMemoryAllocation) ? PAWFE_ENOMEM : PAWFE_ECUDA;                  \
    }                                                                                         \
  } while (0)

#define KERNEL_CHECK(ctx, name)                                                               \
  do {                                                                                        \
    (ctx)->launches++;                                                                        \
    cudaError_t e_ = cudaGetLastError();                                                      \
    if (e_ != cudaSuccess) {                                                                  \
      (ctx)->err = std::string(name) + " launch: " + cudaGetErrorString(e_);                  \
      return PAWFE_ECUDA;                                                                     \
    }                                                                                         \
  } while (0)

static inline int ceil_div(long a, long b) { return (int)((a + b - 1) / b); }
