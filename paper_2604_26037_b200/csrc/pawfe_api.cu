// pawfe_api.cu -- C ABI of libpawfe.so (include/pawfe.h): context, operator set-up, host orchestration of
// the operator applications (section 4.3) and of Algorithm 2 (L250-L282).
// Product code: there is no CPU fallback; every arithmetic step of the path runs in the kernels of
// kernels_simt.cuh / kernels_stream.cuh / cell_tcgen05.cu.
#include "common.h"
#include "fe_tables.h"
#include "host_util.h"
#include "fused.h"
#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <mutex>

using namespace pawfe;

pawfe_status pawfe_ensure_smem(pawfe_ctx* c, const void* func, size_t bytes) {
  static std::mutex mu;
  // per (device, kernel): the limit set so far (default 48 KB needs no call); cudaFuncSetAttribute acts on the current device
  static std::map<std::pair<int, const void*>, size_t> limit;
  std::lock_guard<std::mutex> lock(mu);
  size_t& cur = limit[std::make_pair(c->device, func)];
  if (bytes <= cur || bytes <= 48 * 1024) return PAWFE_OK;
  CUDA_TRY(c, cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  cur = bytes;
  return PAWFE_OK;
}

void pawfe_free_mesh(pawfe_ctx* c) {
  cudaFree(c->d_md1); c->d_md1 = nullptr;
  cudaFree(c->d_M1); c->d_M1 = nullptr;
  cudaFree(c->d_Mref64); c->d_Mref64 = nullptr;
  cudaFree(c->d_Mref32); c->d_Mref32 = nullptr;
  c->have_mesh = false;
}
void pawfe_free_pot(pawfe_ctx* c) {
  cudaFree(c->d_H64); c->d_H64 = nullptr;
  cudaFree(c->d_H32); c->d_H32 = nullptr;
  c->have_pot = false; c->have_h64 = false;
  tc_invalidate(c);
  fused_invalidate(c);
}
void pawfe_free_atoms(pawfe_ctx* c) {
  fused_invalidate(c);
  cudaFree(c->d_pair_cell); cudaFree(c->d_pair_atom); cudaFree(c->d_atom_pair_start);
  cudaFree(c->d_Cd64); cudaFree(c->d_Cd32);
  cudaFree(c->d_D64); cudaFree(c->d_dS64); cudaFree(c->d_dSinv64);
  cudaFree(c->d_D32); cudaFree(c->d_dS32); cudaFree(c->d_dSinv32);
  cudaFree(c->d_P);
  c->d_pair_cell = c->d_pair_atom = c->d_atom_pair_start = nullptr;
  c->d_Cd64 = c->d_Cd32 = nullptr;
  c->d_D64 = c->d_dS64 = c->d_dSinv64 = c->d_D32 = c->d_dS32 = c->d_dSinv32 = nullptr;
  c->d_P = nullptr; c->P_bytes = 0;
  c->have_atoms = false; c->npairs = 0; c->natoms = 0;
}

// ================================================================================================
// lifetime
// ================================================================================================
extern "C" pawfe_status pawfe_create(pawfe_ctx** out, int device, void* cuda_stream) {
  if (!out) return PAWFE_EINVAL;
  *out = nullptr;
  pawfe_ctx* c = new (std::nothrow) pawfe_ctx();
  if (!c) return PAWFE_ENOMEM;
  *out = c;  // returned even on failure so that pawfe_last_error can be read; caller destroys it
  c->device = device;
  c->stream = (cudaStream_t)cuda_stream;
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    c->err = "no CUDA device: libpawfe has no CPU fallback";
    return PAWFE_EUNSUPPORTED;
  }
  if (device < 0 || device >= ndev) { c->err = "bad device index"; return PAWFE_EINVAL; }
  CUDA_TRY(c, cudaSetDevice(device));
  cudaDeviceProp prop;
  CUDA_TRY(c, cudaGetDeviceProperties(&prop, device));
  if (prop.major != 10) {
    c->err = std::string("device is sm_") + std::to_string(prop.major * 10 + prop.minor) +
             "; libpawfe is built for sm_100a (B200) only";
    return PAWFE_EUNSUPPORTED;
  }
  c->sm_count = prop.multiProcessorCount;
  return PAWFE_OK;
}

extern "C" pawfe_status pawfe_destroy(pawfe_ctx* c) {
  if (!c) return PAWFE_EINVAL;
  if (c->have_mesh || c->d_md1) cudaSetDevice(c->device);
  pawfe_free_atoms(c); pawfe_free_pot(c); pawfe_free_mesh(c);
  if (c->h_pinned) cudaFreeHost(c->h_pinned);
  cudaFree(c->d_scal);
  for (int i = 0; i < pawfe_ctx::kScalSlots; ++i) if (c->scal_ev[i]) cudaEventDestroy(c->scal_ev[i]);
  cudaFree(c->d_hostblk); cudaFree(c->d_hostws); cudaFree(c->d_hostblk2); cudaFree(c->d_tmpblk);
  if (c->s_h2d) cudaStreamDestroy(c->s_h2d);
  if (c->s_d2h) cudaStreamDestroy(c->s_d2h);
  for (int i = 0; i < 2; ++i) {
    if (c->ev_h2d[i]) cudaEventDestroy(c->ev_h2d[i]);
    if (c->ev_filt[i]) cudaEventDestroy(c->ev_filt[i]);
    if (c->ev_d2h[i]) cudaEventDestroy(c->ev_d2h[i]);
  }
  if (c->h_stage) cudaFreeHost(c->h_stage);
  for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
  for (cudaEvent_t e : c->prof_setup_ev) cudaEventDestroy(e);
  delete c;
  return PAWFE_OK;
}

extern "C" const char* pawfe_last_error(const pawfe_ctx* c) { return c ? c->err.c_str() : "null context"; }

extern "C" pawfe_status pawfe_set_stream(pawfe_ctx* c, void* s) {
  if (!c) return PAWFE_EINVAL;
  c->stream = (cudaStream_t)s;
  return PAWFE_OK;
}

extern "C" pawfe_status pawfe_num_dofs(const pawfe_ctx* c, long* M) {
  if (!c || !M) return PAWFE_EINVAL;
  if (!c->have_mesh) return PAWFE_ESTATE;
  *M = c->M;
  return PAWFE_OK;
}
extern "C" pawfe_status pawfe_num_pairs(const pawfe_ctx* c, long* np) {
  if (!c || !np) return PAWFE_EINVAL;
  if (!c->have_atoms) return PAWFE_ESTATE;
  *np = c->npairs;
  return PAWFE_OK;
}
extern "C" pawfe_status pawfe_launch_count(const pawfe_ctx* c, long* n) {
  if (!c || !n) return PAWFE_EINVAL;
  *n = c->launches;
  return PAWFE_OK;
}

// ================================================================================================
// mesh
// ================================================================================================
extern "C" pawfe_status pawfe_mesh_create(pawfe_ctx* c, const int ncells[3], const double box[3], int p,
                                          pawfe_bc bc, const double* kpt) {
  if (!c || !ncells || !box) return PAWFE_EINVAL;
  if (p < 2 || p > 7) { c->err = "FE order p must be in [2, 7]"; return PAWFE_EUNSUPPORTED; }
  for (int d = 0; d < 3; ++d) {
    if (ncells[d] < 1 || !(box[d] > 0)) { c->err = "bad mesh size"; return PAWFE_EINVAL; }
    if (bc == PAWFE_PERIODIC && (ncells[d] % 2)) { c->err = "periodic meshes need an even cell count"; return PAWFE_EINVAL; }
  }
  CUDA_TRY(c, cudaSetDevice(c->device));
  pawfe_free_atoms(c); pawfe_free_pot(c); pawfe_free_mesh(c);
  c->p = p; c->n1 = p + 1; c->n = c->n1 * c->n1 * c->n1; c->bc = (int)bc;
  c->cplx = (kpt != nullptr);
  c->ldk = (c->n + 31) / 32 * 32;  // 128-byte rows: every TMA box row of the FP32 cell matrices is one aligned line
  long M = 1; int ncell = 1;
  for (int d = 0; d < 3; ++d) {
    c->nc[d] = ncells[d]; c->box[d] = box[d]; c->h[d] = box[d] / ncells[d];
    c->N[d] = ncells[d] * p + (bc == PAWFE_DIRICHLET ? 1 : 0);
    c->kpt[d] = kpt ? kpt[d] : 0.0;
    M *= c->N[d]; ncell *= ncells[d];
  }
  c->M = M; c->ncell = ncell;
  gll_rule(p, c->xi, c->wgll);
  matrices_1d(p, c->K1, c->M1, c->G1);

  // lumped mass M_D (L228): per-direction factors  md1_d[i] = (h_d / 2) * sum of GLL weights meeting at node i
  long Ntot = c->N[0] + c->N[1] + c->N[2];
  std::vector<double> md(2 * Ntot, 0.0);
  long off = 0;
  for (int d = 0; d < 3; ++d) {
    for (int cc = 0; cc < c->nc[d]; ++cc)
      for (int a = 0; a <= p; ++a) {
        int i = cc * p + a;
        if (bc == PAWFE_PERIODIC) i %= c->N[d];
        md[off + i] += 0.5 * c->h[d] * c->wgll[a];
      }
    for (int i = 0; i < c->N[d]; ++i) {
      bool boundary = (bc == PAWFE_DIRICHLET) && (i == 0 || i == c->N[d] - 1);
      md[Ntot + off + i] = boundary ? 0.0 : 1.0 / md[off + i];
    }
    off += c->N[d];
  }
  TRY(upload(c, &c->d_md1, md));
  TRY(upload(c, &c->d_M1, c->M1));
  MeshDev& m = c->md;
  off = 0;
  for (int d = 0; d < 3; ++d) {
    m.nc[d] = c->nc[d]; m.N[d] = c->N[d];
    m.md1[d] = c->d_md1 + off; m.mdinv1[d] = c->d_md1 + Ntot + off;
    off += c->N[d];
  }
  m.p = p; m.n1 = c->n1; m.n = c->n; m.periodic = (bc == PAWFE_PERIODIC); m.M = M; m.ncell = ncell;

  // reference mass cell matrix M^e = (hx hy hz / 8) M1 x M1 x M1 (Eq. 33), in the context's scalar type
  const int n = c->n, cw = c->cplx ? 2 : 1;
  std::vector<double> Me((size_t)n * n, 0.0);
  kron3(c->n1, c->M1, c->M1, c->M1, c->h[0] * c->h[1] * c->h[2] / 8.0, Me);
  std::vector<double> Me64((size_t)n * n * cw, 0.0);
  std::vector<float> Me32((size_t)n * c->ldk * cw, 0.f);
  for (int I = 0; I < n; ++I)
    for (int J = 0; J < n; ++J) {
      Me64[((size_t)I * n + J) * cw] = Me[(size_t)I * n + J];
      Me32[((size_t)I * c->ldk + J) * cw] = (float)Me[(size_t)I * n + J];
    }
  TRY(upload(c, &c->d_Mref64, Me64));
  TRY(upload(c, &c->d_Mref32, Me32));
  c->have_mesh = true;
  return PAWFE_OK;
}
