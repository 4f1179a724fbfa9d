// api_atoms.cu -- atoms and projectors: (cell, atom) pair list, projector blocks C^{e,a dagger} (Eq. 34),
// G^a = C^a^dagger M_D^-1 C^a and Delta^a_Sinv = (I + dS^a G^a)^-1 dS^a (Eq. 29; reading R10).
#include "common.h"
#include "fe_tables.h"
#include "host_util.h"
#include "fe_setup.cuh"
#include "kernels_simt.cuh"
#include "api_internal.h"
#include "fused.h"
#include <algorithm>
#include <cmath>

using namespace pawfe;

namespace {

// zero the rows of Z touched by the pairs [pair0, pair0 + gridDim.x): Z[J][0..W)
__global__ void k_zero_pair_rows(MeshDev md, int pair0, const int* __restrict__ pair_cell,
                                 double* __restrict__ Z, int W) {
  int cx, cy, cz;
  mesh_cell_coords(md, pair_cell[pair0 + blockIdx.x], &cx, &cy, &cz);
  const int n1 = md.n1;
  for (int i = threadIdx.x; i < md.n * W; i += blockDim.x) {
    int I = i / W, w = i % W;
    int c = I % n1, b = (I / n1) % n1, a = I / (n1 * n1);
    int ix, iy, iz;
    long J = mesh_node(md, cx, cy, cz, a, b, c, &ix, &iy, &iz);
    Z[J * W + w] = 0.0;
  }
}

template <typename T64, typename T32>
pawfe_status upload_coupling_arrays(pawfe_ctx* c, const std::vector<double>& v, void** d64, void** d32) {
  // v: natoms*npj*npj*cw doubles in the context's scalar layout
  cudaFree(*d64); cudaFree(*d32); *d64 = *d32 = nullptr;
  double* a64 = nullptr; float* a32 = nullptr;
  TRY(upload(c, &a64, v));
  std::vector<float> vf(v.begin(), v.end());
  TRY(upload(c, &a32, vf));
  *d64 = a64; *d32 = a32;
  return PAWFE_OK;
}

}  // namespace

pawfe_status pawfe_ensure_P(pawfe_ctx* c, int B) {
  size_t need = (size_t)2 * c->natoms * c->npj * B * sizeof(double2);
  if (need <= c->P_bytes) return PAWFE_OK;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  cudaFree(c->d_P); c->d_P = nullptr; c->P_bytes = 0;
  char* p = nullptr;
  TRY(dev_alloc(c, &p, need));
  c->d_P = p; c->P_bytes = need;
  return PAWFE_OK;
}

pawfe_status pawfe_upload_couplings(pawfe_ctx* c, const double* D, const double* dS,
                                    const std::vector<double>& G) {
  const int npj = c->npj, cw = c->cplx ? 2 : 1;
  const size_t per = (size_t)npj * npj;
  std::vector<double> vD(c->natoms * per * cw, 0.0), vS(c->natoms * per * cw, 0.0), vI(c->natoms * per * cw, 0.0);
  for (size_t i = 0; i < c->natoms * per; ++i) {
    if (D) vD[i * cw] = D[i];
    vS[i * cw] = dS[i];
  }
  // Delta_Sinv = (I + dS G)^-1 dS per atom, complex arithmetic (imaginary parts vanish for a real context)
  for (int a = 0; a < c->natoms; ++a) {
    std::vector<double> A(2 * per, 0.0), Bm(2 * per, 0.0), X;
    for (int i = 0; i < npj; ++i)
      for (int j = 0; j < npj; ++j) {
        double sr = 0, si = 0;
        for (int k = 0; k < npj; ++k) {
          double d = dS[a * per + i * npj + k];
          sr += d * G[(a * per + k * npj + j) * cw];
          if (cw == 2) si += d * G[(a * per + k * npj + j) * cw + 1];
        }
        A[2 * (i * npj + j)] = sr + (i == j ? 1.0 : 0.0);
        A[2 * (i * npj + j) + 1] = si;
        Bm[2 * (i * npj + j)] = dS[a * per + i * npj + j];
      }
    if (!solve_complex(npj, A, Bm, X)) { c->err = "I + dS G is singular"; return PAWFE_EINVAL; }
    for (size_t i = 0; i < per; ++i) {
      vI[(a * per + i) * cw] = X[2 * i];
      if (cw == 2) vI[(a * per + i) * cw + 1] = X[2 * i + 1];
    }
  }
  c->h_dSinv = vI;
  if (D) TRY((upload_coupling_arrays<double, float>(c, vD, &c->d_D64, &c->d_D32)));
  TRY((upload_coupling_arrays<double, float>(c, vS, &c->d_dS64, &c->d_dS32)));
  TRY((upload_coupling_arrays<double, float>(c, vI, &c->d_dSinv64, &c->d_dSinv32)));
  return PAWFE_OK;
}

template <typename TC>
static pawfe_status compute_G(pawfe_ctx* c, std::vector<double>& G) {
  // G^a = C^a^dagger M_D^-1 C^a by scattering the atom's projector columns into a zeroed global block Z
  // (width npj), projecting M_D^-1 Z back onto the same atom, and zeroing the touched rows again.
  const int npj = c->npj, n = c->n, cw = c->cplx ? 2 : 1;
  const size_t per = (size_t)npj * npj;
  double *Z = nullptr, *Id = nullptr, *Gd = nullptr;
  pawfe_status st;
  if ((st = dev_alloc(c, &Z, (size_t)c->M * npj * cw)) != PAWFE_OK) return st;
  std::vector<double> hid(c->natoms * per * cw, 0.0);
  for (int a = 0; a < c->natoms; ++a)
    for (int i = 0; i < npj; ++i) hid[(a * per + i * npj + i) * cw] = 1.0;
  if ((st = upload(c, &Id, hid)) != PAWFE_OK) { cudaFree(Z); return st; }
  if ((st = dev_alloc(c, &Gd, c->natoms * per * cw)) != PAWFE_OK) { cudaFree(Z); cudaFree(Id); return st; }
  cudaMemsetAsync(Z, 0, (size_t)c->M * npj * cw * sizeof(double), c->stream);
  size_t smem = (size_t)n * 16 + 4 * PAWFE_MAX_NPJ * 32 * sizeof(TC);
  for (int a = 0; a < c->natoms; ++a) {
    int p0 = c->h_atom_pair_start[a], np = c->h_atom_pair_start[a + 1] - p0;
    if (np == 0) { cudaMemsetAsync(Gd + a * per * cw, 0, per * cw * sizeof(double), c->stream); continue; }
    k_nl_scatter<TC, TC><<<dim3(np, 1), 128, 0, c->stream>>>(
        c->md, p0, c->d_pair_cell, c->d_pair_atom, (const TC*)c->d_Cd64, npj, (const TC*)Id, npj, npj, 0,
        (TC*)Z, (long)npj);
    k_proj<TC, TC><<<dim3(1, 1), 128, smem, c->stream>>>(
        c->md, a, c->d_atom_pair_start, c->d_pair_cell, (const TC*)c->d_Cd64, npj, (const TC*)Z, (long)npj,
        npj, 1, (TC*)Gd, npj);
    k_zero_pair_rows<<<np, 128, 0, c->stream>>>(c->md, p0, c->d_pair_cell, Z, npj * cw);
    c->launches += 3;
  }
  G.assign(c->natoms * per * cw, 0.0);
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e == cudaSuccess) e = cudaMemcpy(G.data(), Gd, G.size() * sizeof(double), cudaMemcpyDeviceToHost);
  cudaFree(Z); cudaFree(Id); cudaFree(Gd);
  if (e != cudaSuccess) { c->err = std::string("compute_G: ") + cudaGetErrorString(e); return PAWFE_ECUDA; }
  return PAWFE_OK;
}

extern "C" pawfe_status pawfe_atoms_create(pawfe_ctx* c, int natoms, const double* pos, int nproj,
                                           const int* proj_l, const int* proj_m, const double* proj_sigma,
                                           const double* proj_amp, double rc, const double* D, const double* dS) {
  if (!c || natoms < 0 || nproj < 1 || nproj > PAWFE_MAX_NPJ) return PAWFE_EINVAL;
  if (natoms > 0 && (!pos || !D || !dS)) return PAWFE_EINVAL;
  if (!proj_l || !proj_m || !proj_sigma || !proj_amp || !(rc > 0)) return PAWFE_EINVAL;
  if (!c->have_mesh) { c->err = "mesh not created"; return PAWFE_ESTATE; }
  for (int al = 0; al < nproj; ++al)
    if (proj_l[al] < 0 || proj_l[al] > 2 || std::abs(proj_m[al]) > proj_l[al]) { c->err = "projector (l, m) out of range (l <= 2)"; return PAWFE_EUNSUPPORTED; }
  if (c->bc == PAWFE_PERIODIC)
    for (int d = 0; d < 3; ++d)
      if (!(rc < 0.5 * c->box[d])) { c->err = "rc must be < box/2 for periodic meshes"; return PAWFE_EINVAL; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  pawfe_free_atoms(c);
  c->natoms = natoms; c->npj = nproj; c->rc = rc; c->sinv_variant = 0;
  c->pos.assign(pos, pos + 3 * (size_t)natoms);
  c->proj_l.assign(proj_l, proj_l + nproj); c->proj_m.assign(proj_m, proj_m + nproj);
  c->proj_sigma.assign(proj_sigma, proj_sigma + nproj); c->proj_amp.assign(proj_amp, proj_amp + nproj);
  c->h_dS.assign(dS, dS + (size_t)natoms * nproj * nproj);

  // ---- (cell, atom) pairs: cells whose box comes within rc of the atom (minimum image when periodic) ----
  std::vector<int> pc, pa, aps(natoms + 1, 0);
  const bool per = (c->bc == PAWFE_PERIODIC);
  for (int a = 0; a < natoms; ++a) {
    std::vector<std::pair<int, double>> cand[3];  // per direction: (cell index, squared 1-D distance)
    for (int d = 0; d < 3; ++d) {
      double x = pos[3 * a + d];
      for (int cc = 0; cc < c->nc[d]; ++cc) {
        double lo = cc * c->h[d], hi = (cc + 1) * c->h[d], best = 1e300;
        for (int s = (per ? -1 : 0); s <= (per ? 1 : 0); ++s) {
          double xs = x + s * c->box[d];
          double dd = xs < lo ? lo - xs : (xs > hi ? xs - hi : 0.0);
          best = std::min(best, dd);
        }
        if (best < rc) cand[d].push_back({cc, best * best});
      }
    }
    std::vector<int> cells;
    for (auto& ex : cand[0]) for (auto& ey : cand[1]) for (auto& ez : cand[2])
      if (ex.second + ey.second + ez.second < rc * rc)
        cells.push_back((ex.first * c->nc[1] + ey.first) * c->nc[2] + ez.first);
    std::sort(cells.begin(), cells.end());
    for (int e : cells) { pc.push_back(e); pa.push_back(a); }
    aps[a + 1] = (int)pc.size();
  }
  c->npairs = (long)pc.size();
  c->h_atom_pair_start = aps;
  TRY(upload(c, &c->d_atom_pair_start, aps));
  const int n = c->n, cw = c->cplx ? 2 : 1;
  if (c->npairs > 0) {
    TRY(upload(c, &c->d_pair_cell, pc));
    TRY(upload(c, &c->d_pair_atom, pa));
    size_t celems = (size_t)c->npairs * nproj * n * cw;
    double* Cd64 = nullptr; float* Cd32 = nullptr;
    TRY(dev_alloc(c, &Cd64, celems)); c->d_Cd64 = Cd64;
    TRY(dev_alloc(c, &Cd32, celems)); c->d_Cd32 = Cd32;

    const int nq = 2 * (c->p + 2);
    std::vector<double> xq, wq, Lq, dLq;
    gauss_legendre_rule(nq, xq, wq);
    lagrange_basis(c->xi, xq, Lq, dLq);
    double *d_xq = nullptr, *d_wq = nullptr, *d_Lq = nullptr, *d_pos = nullptr;
    TRY(upload(c, &d_xq, xq)); TRY(upload(c, &d_wq, wq)); TRY(upload(c, &d_Lq, Lq)); TRY(upload(c, &d_pos, c->pos));
    ProjTable pt;
    pt.npj = nproj; pt.rc = rc;
    for (int al = 0; al < nproj; ++al) { pt.l[al] = proj_l[al]; pt.m[al] = proj_m[al]; pt.sigma[al] = proj_sigma[al]; pt.amp[al] = proj_amp[al]; }
    for (int d = 0; d < 3; ++d) pt.kpt[d] = c->kpt[d];
    SetupGeom g;
    for (int d = 0; d < 3; ++d) { g.h[d] = c->h[d]; g.box[d] = c->box[d]; }
    g.periodic = per;
    size_t smem = (size_t)cw * ((size_t)nq * nq * nq + (size_t)nq * nq * c->n1 + (size_t)nq * c->n1 * c->n1) * sizeof(double);
    cudaError_t e;
    if (c->cplx) {
      e = cudaFuncSetAttribute(k_build_proj<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e == cudaSuccess)
        k_build_proj<true><<<(int)c->npairs, 256, smem, c->stream>>>(c->md, g, nq, d_xq, d_wq, d_Lq, pt, d_pos, c->d_pair_cell, c->d_pair_atom, Cd64);
    } else {
      e = cudaFuncSetAttribute(k_build_proj<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e == cudaSuccess)
        k_build_proj<false><<<(int)c->npairs, 256, smem, c->stream>>>(c->md, g, nq, d_xq, d_wq, d_Lq, pt, d_pos, c->d_pair_cell, c->d_pair_atom, Cd64);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) {
      k_f64_to_f32<<<4 * c->sm_count, 256, 0, c->stream>>>(Cd64, Cd32, (long)celems);
      e = cudaGetLastError();
    }
    c->launches += 2;
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(d_xq); cudaFree(d_wq); cudaFree(d_Lq); cudaFree(d_pos);
    if (e != cudaSuccess) { c->err = std::string("projector build: ") + cudaGetErrorString(e); return PAWFE_ECUDA; }
  }
  std::vector<double> G((size_t)natoms * nproj * nproj * cw, 0.0);
  if (c->npairs > 0) {
    if (c->cplx) TRY(compute_G<double2>(c, G)); else TRY(compute_G<double>(c, G));
  }
  c->h_G = G;
  TRY(pawfe_upload_couplings(c, D, dS, G));
  c->have_atoms = true;
  return PAWFE_OK;
}

namespace {
// G^a of the variant in force (same for every atom in variant 1): natoms*npj*npj*cw doubles
//   variant 1 (text after Eq. 29): C^a^dagger M^-1 C^a ~ <p_alpha|p_beta> = int p_alpha p_beta d^3x
//     = delta_ll' delta_mm' amp amp' int_0^rc r^(2l) exp(-r^2/2s^2) exp(-r^2/2s'^2) (1-(r/rc)^2)^4 r^2 dr   (orthonormal Y_lm),
//     by a 96-point Gauss-Legendre rule on [0, rc].
std::vector<double> sinv_G(const pawfe_ctx* c) {
  if (c->sinv_variant == 0) return c->h_G;
  const int npj = c->npj, cw = c->cplx ? 2 : 1;
  std::vector<double> x, w, O((size_t)npj * npj, 0.0);
  gauss_legendre_rule(96, x, w);
  for (int a = 0; a < npj; ++a)
    for (int b = 0; b < npj; ++b) {
      if (c->proj_l[a] != c->proj_l[b] || c->proj_m[a] != c->proj_m[b]) continue;
      double s = 0.0;
      for (size_t q = 0; q < x.size(); ++q) {
        const double r = 0.5 * c->rc * (x[q] + 1.0), cut = 1.0 - (r / c->rc) * (r / c->rc);
        const double f = std::pow(r, 2 * c->proj_l[a]) * std::exp(-r * r / (2 * c->proj_sigma[a] * c->proj_sigma[a])) *
                         std::exp(-r * r / (2 * c->proj_sigma[b] * c->proj_sigma[b])) * cut * cut * cut * cut * r * r;
        s += 0.5 * c->rc * w[q] * f;
      }
      O[(size_t)a * npj + b] = c->proj_amp[a] * c->proj_amp[b] * s;
    }
  std::vector<double> G((size_t)c->natoms * npj * npj * cw, 0.0);
  for (int at = 0; at < c->natoms; ++at)
    for (size_t i = 0; i < (size_t)npj * npj; ++i) G[((size_t)at * npj * npj + i) * cw] = O[i];
  return G;
}
}  // namespace

extern "C" pawfe_status pawfe_get_pairs(pawfe_ctx* c, int* pair_cell, int* pair_atom) {
  if (!c || !pair_cell || !pair_atom) return PAWFE_EINVAL;
  if (!c->have_atoms) return PAWFE_ESTATE;
  if (c->npairs == 0) return PAWFE_OK;
  CUDA_TRY(c, cudaSetDevice(c->device));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  CUDA_TRY(c, cudaMemcpy(pair_cell, c->d_pair_cell, c->npairs * sizeof(int), cudaMemcpyDeviceToHost));
  CUDA_TRY(c, cudaMemcpy(pair_atom, c->d_pair_atom, c->npairs * sizeof(int), cudaMemcpyDeviceToHost));
  return PAWFE_OK;
}

// User- (or oracle-) built projector blocks for the library's pair list: replaces C^{e,a dagger}, then G^a, Delta_Sinv
// and the FP32 copies are rebuilt from them exactly as pawfe_atoms_create does.
extern "C" pawfe_status pawfe_set_projector_blocks(pawfe_ctx* c, const double* Cd, int is_device) {
  if (!c || !Cd) return PAWFE_EINVAL;
  if (!c->have_atoms) return PAWFE_ESTATE;
  CUDA_TRY(c, cudaSetDevice(c->device));
  fused_invalidate(c);
  const int cw = c->cplx ? 2 : 1;
  const size_t celems = (size_t)c->npairs * c->npj * c->n * cw;
  if (celems > 0) {
    CUDA_TRY(c, cudaMemcpyAsync(c->d_Cd64, Cd, celems * sizeof(double), is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    k_f64_to_f32<<<4 * c->sm_count, 256, 0, c->stream>>>((const double*)c->d_Cd64, (float*)c->d_Cd32, (long)celems);
    KERNEL_CHECK(c, "k_f64_to_f32");
  }
  std::vector<double> G((size_t)c->natoms * c->npj * c->npj * cw, 0.0);
  if (c->npairs > 0) {
    if (c->cplx) TRY(compute_G<double2>(c, G)); else TRY(compute_G<double>(c, G));
  }
  c->h_G = G;
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return pawfe_upload_couplings(c, nullptr, c->h_dS.data(), sinv_G(c));
}

// Which G^a enters Delta^a_Sinv = (dS^a^-1 + G^a)^-1 (Eq. 29): recomputes Delta_Sinv and drops the fused plan.
extern "C" pawfe_status pawfe_set_sinv_variant(pawfe_ctx* c, int variant) {
  if (!c) return PAWFE_EINVAL;
  if (variant != 0 && variant != 1) { c->err = "S^-1approx variant must be 0 or 1"; return PAWFE_EINVAL; }
  if (!c->have_atoms) { c->err = "atoms not created"; return PAWFE_ESTATE; }
  CUDA_TRY(c, cudaSetDevice(c->device));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  fused_invalidate(c);
  c->sinv_variant = variant;
  return pawfe_upload_couplings(c, nullptr, c->h_dS.data(), sinv_G(c));
}

extern "C" pawfe_status pawfe_update_coupling(pawfe_ctx* c, const double* D) {
  if (!c || !D) return PAWFE_EINVAL;
  if (!c->have_atoms) return PAWFE_ESTATE;
  CUDA_TRY(c, cudaSetDevice(c->device));
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return pawfe_upload_couplings(c, D, c->h_dS.data(), sinv_G(c));
}

extern "C" pawfe_status pawfe_get_sinv_coupling(pawfe_ctx* c, double* out) {
  if (!c || !out) return PAWFE_EINVAL;
  if (!c->have_atoms) return PAWFE_ESTATE;
  size_t sz = (size_t)c->natoms * c->npj * c->npj * (c->cplx ? 2 : 1);
  CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  CUDA_TRY(c, cudaMemcpy(out, c->d_dSinv64, sz * sizeof(double), cudaMemcpyDeviceToHost));
  return PAWFE_OK;
}
