/*
 * pawfe.h -- C ABI of libpawfe.so: the R-ChFSI filter hot path of PAW-FE (arxiv/paper_2604_26037)
 * on one NVIDIA B200 (sm_100a).
 *
 * Citations are lines of the paper text with the section / equation / algorithm they
 * fall in.  The library computes, with its own CUDA kernels only (there is no CPU fallback):
 *
 *   H = H_loc + sum_a C^a D^a C^a^dagger,   S = M + sum_a C^a dS^a C^a^dagger      (Eq. 13, 16; L125-L138)
 *   S^-1approx = M_D^-1 - sum_a M_D^-1 C^a Delta^a_Sinv C^a^dagger M_D^-1           (Eq. 28-29; L219-L228)
 *   Algorithm 2: residual-based Chebyshev filter of degree m on [bW, bU]          (L250-L282)
 *
 * on a uniform hexahedral spectral-element mesh (tensor-product GLL Lagrange basis of order p,
 * L116, L307) through the cell-matrix strategy of section 4.3 (L337-L347): gather to cells, dense
 * cell-matrix x cell-vector-block contraction, scatter-add assembly, plus atom-local projector
 * contractions for the non-local PAW terms.
 *
 * Conventions
 *  - Every function returns a pawfe_status and never throws across the ABI; pawfe_last_error()
 *    gives the text of the last failure on that context.
 *  - "host" / "device" is stated for every pointer.  Device pointers must belong to the context's
 *    device.  All work is enqueued on the context's CUDA stream.  Hot calls (apply_*, cheb_filter*, col_norms) do not
 *    synchronise the host and allocate nothing ONCE pawfe_prepare has been called for their (prec, B, m); without it
 *    the library's internal plans and scratch (re-tiled operand streams, projection scratch, coefficient staging) are
 *    built on the first call that needs them and re-grown when a wider block arrives, which synchronises the stream.
 *  - The library OWNS the operators (cell matrices, projector blocks, couplings, lumped mass) and
 *    frees them in pawfe_destroy.  The CALLER owns all vector blocks and the filter workspace.
 *  - Vector blocks are row-major [dof][vec] ("vec" contiguous), leading dimension ld in ELEMENTS.
 *    Real contexts: element = double (PAWFE_FP64) or float (PAWFE_FP32 / PAWFE_TF32).
 *    Complex contexts (k-point given): element = interleaved (re, im) pair of that type.
 *  - Node numbering is lexicographic over the stored node grid: J = (ix*Ny + iy)*Nz + iz, with
 *    i = c*p + a for cell c and local GLL index a.  Periodic: N_d = ncells_d*p.  Dirichlet:
 *    N_d = ncells_d*p + 1 nodes are STORED, boundary rows are ignored on input and written as 0.
 *  - A device that is not compute capability 10.x gives PAWFE_EUNSUPPORTED.
 */
#ifndef PAWFE_H
#define PAWFE_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default) /* the library is built with -fvisibility=hidden */
#endif

typedef struct pawfe_ctx pawfe_ctx; /* opaque, owned by the library */

typedef enum {
  PAWFE_OK = 0,
  PAWFE_EINVAL = 1,       /* bad argument */
  PAWFE_ENOMEM = 2,       /* device or host allocation failed */
  PAWFE_ECUDA = 3,        /* a CUDA call or kernel failed; see pawfe_last_error */
  PAWFE_ESTATE = 4,       /* call made before the data it needs exists */
  PAWFE_EUNSUPPORTED = 5  /* not an sm_100 device, or an unsupported (p, B, precision) */
} pawfe_status;

/* Arithmetic of the cell contraction (section 4.4; L11, L27 for TF32):
 *   FP64: every step in double (reference mode).
 *   FP32: FP32 storage, FP32-accurate arithmetic inside H S^-1approx.  The cell contraction runs on tcgen05 tensor cores
 *         as three TF32 passes on operands split into the part kind::tf32 keeps and the rest (hi*hi + lo*hi + hi*lo,
 *         FP32 accumulation; ~1e-6 relative per product), real and complex contexts alike; blocks that do not meet the
 *         tensor-core path's alignment rules use FP32 FMAs.
 *   TF32: FP32 storage; operands of the cell contraction truncated to TF32 inside tcgen05 tensor
 *         cores, FP32 accumulation (~7e-4 relative per product).  In the fused filter step and pawfe_apply_HSinv the
 *         projection C^dagger X is a TF32 tensor-core product too (projector blocks rounded to nearest, FP32
 *         accumulation).  Nothing else is TF32. */
typedef enum { PAWFE_FP64 = 0, PAWFE_FP32 = 1, PAWFE_TF32 = 2 } pawfe_prec;
typedef enum { PAWFE_PERIODIC = 0, PAWFE_DIRICHLET = 1 } pawfe_bc;

/* ---- lifetime ------------------------------------------------------------------------------ */

/* Create a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t (NULL = the legacy
 * default stream); the caller keeps ownership of the stream. */
pawfe_status pawfe_create(pawfe_ctx** out, int device, void* cuda_stream);
pawfe_status pawfe_destroy(pawfe_ctx* ctx);
/* Text of the last error on this context ("" if none).  Valid until the next call on ctx. */
const char* pawfe_last_error(const pawfe_ctx* ctx);
/* Change the stream later calls are enqueued on. */
pawfe_status pawfe_set_stream(pawfe_ctx* ctx, void* cuda_stream);

/* ---- mesh and cell operators (Eq. 12-13; Eq. 31-33; M_D of L228) -------- */

/* Uniform mesh of box[0] x box[1] x box[2] bohr with ncells[d] cells per direction, FE order p
 * (2 <= p <= 7; p+1 GLL nodes per direction per cell).  kpt: host, 3 doubles (Bloch vector in
 * 1/bohr) or NULL for a real (Gamma, no phase) context.  Periodic meshes need an even ncells[d].
 * Builds the 1-D GLL / Gauss-Legendre tables, the reference cell matrices and the lumped mass. */
pawfe_status pawfe_mesh_create(pawfe_ctx* ctx, const int ncells[3], const double box[3], int p,
                               pawfe_bc bc, const double* kpt);

/* Local potential V(x) = - sum_a sum_images Z_a exp(-|x - R_a - L|^2 / (2 sigma_a^2)); periodic:
 * the 27 nearest images; Dirichlet: none (stands in for V_eff + V_z of Eq. 2).
 * pos: host, 3*natoms doubles; Z, sigma: host, natoms doubles.
 * Builds on the device, in FP64 arithmetic, every cell matrix
 *   H^e = 1/2 K^e + V^e + 1/2 |k|^2 M^e - i sum_d k_d G_d^e                (Eq. 13 / Eq. 32)
 * with V^e on a (p+2)^3 Gauss-Legendre grid, and stores it as FP32 (always) and FP64 (if
 * keep_fp64 != 0; needed by PAWFE_FP64 applies and by the residual set-up of the filter).
 * Synchronises the host. */
pawfe_status pawfe_local_potential_gaussians(pawfe_ctx* ctx, int natoms, const double* pos,
                                             const double* Z, const double* sigma, int keep_fp64);

/* Cell matrices supplied by the caller instead (e.g. built by an independent implementation, to run the library's
 * kernels on them): Hcell = [cell][I][J] doubles, cell = (cx*ncy + cy)*ncz + cz, I = (a*(p+1) + b)*(p+1) + c, complex
 * contexts interleaved (re, im); host (is_device = 0) or device memory.  Replaces H^e of every cell; the mass cell
 * matrix stays the mesh's M^e = (hx hy hz / 8) M1 x M1 x M1.  FP32 copies are derived; keep_fp64 as above.
 * Synchronises the host. */
pawfe_status pawfe_set_cell_matrices(pawfe_ctx* ctx, const double* Hcell, int is_device, int keep_fp64);

/* ---- atoms and projectors (Eq. 16-17; Eq. 34; Eq. 28-29) ----------- */

/* One species: nproj projectors p_alpha(d) = amp * r^l exp(-r^2 / 2 sigma^2) (1-(r/rc)^2)^2 Y_lm(d/r)
 * for r < rc (real orthonormal Y_lm, l <= 2), 0 otherwise.  proj_l, proj_m: host, nproj ints;
 * proj_sigma, proj_amp: host, nproj doubles.  pos: host, 3*natoms doubles.
 * D (= Delta_H) and dS (= Delta_S): host, natoms*nproj*nproj doubles, real symmetric per atom.
 * Builds the cell-level projector blocks C^{e,a} (Eq. 34) on a (2(p+2))^3 Gauss-Legendre grid for
 * every (cell, atom) pair whose cell meets the atom's sphere (minimum image when periodic; phase
 * e^{ik.(R_a + d)} when complex), G^a = C^a^dagger M_D^-1 C^a and
 * Delta^a_Sinv = (I + dS^a G^a)^-1 dS^a (Eq. 29).  Needs rc < min(box)/2 when periodic.
 * Synchronises the host. */
pawfe_status pawfe_atoms_create(pawfe_ctx* ctx, int natoms, const double* pos, int nproj,
                                const int* proj_l, const int* proj_m, const double* proj_sigma,
                                const double* proj_amp, double rc, const double* D, const double* dS);

/* The (cell, atom) pairs the library holds projector blocks for, in its own order (pairs sorted by atom, then cell):
 * pair_cell, pair_atom: host, pawfe_num_pairs ints each. */
pawfe_status pawfe_get_pairs(pawfe_ctx* ctx, int* pair_cell, int* pair_atom);
/* Projector blocks supplied by the caller for exactly those pairs: Cd = [pair][alpha][I] doubles = (C^{e,a dagger})_{alpha I}
 * (Eq. 34; complex interleaved), host or device.  G^a, Delta^a_Sinv and the FP32 copies are rebuilt from them.
 * Synchronises the host. */
pawfe_status pawfe_set_projector_blocks(pawfe_ctx* ctx, const double* Cd, int is_device);

/* Which G^a enters Delta^a_Sinv = (dS^a^-1 + G^a)^-1 of Eq. 29 (L225-L228): variant 0 (default) G^a = C^a^dagger M_D^-1 C^a
 * (exact Woodbury inverse of M_D + C dS C^dagger for one atom); variant 1 the paper's cheaper alternative (text after Eq. 29,
 * L228) G^a ~ <p_alpha|p_beta>, the overlap matrix of the projector functions (mesh-independent; radial quadrature on the
 * host).  Recomputes Delta_Sinv; pawfe_atoms_create resets the variant to 0.  Synchronises the host. */
pawfe_status pawfe_set_sinv_variant(pawfe_ctx* ctx, int variant);

/* Replace D (Delta_H changes every SCF step, Eq. 18).  host, natoms*nproj*nproj. */
pawfe_status pawfe_update_coupling(pawfe_ctx* ctx, const double* D);

/* ---- queries ------------------------------------------------------------------------------- */

pawfe_status pawfe_num_dofs(const pawfe_ctx* ctx, long* M);          /* stored nodes */
pawfe_status pawfe_num_pairs(const pawfe_ctx* ctx, long* npairs);    /* (cell, atom) pairs */
/* Copy one FP64 cell matrix H^e (n x n, row-major, complex interleaved if k-point) to host memory.
 * Needs keep_fp64.  For tests; synchronises. */
pawfe_status pawfe_get_cell_matrix(pawfe_ctx* ctx, long cell, double* out_host);
/* Copy Delta_Sinv (natoms*nproj*nproj, complex interleaved if k-point) to host.  For tests. */
pawfe_status pawfe_get_sinv_coupling(pawfe_ctx* ctx, double* out_host);

/* ---- operator applications on a block (section 4.3) ------------------------------ */

/* Y = A X for A in {H, S, S^-1approx}.  X, Y: device, [dof][vec] with leading dimension ld >= B,
 * element type given by prec (see Conventions); X and Y must not overlap.  1 <= B <= 512.
 * Boundary (Dirichlet) rows of X are ignored, those of Y are written as 0. */
pawfe_status pawfe_apply_H(pawfe_ctx* ctx, pawfe_prec prec, const void* X, void* Y, long ld, int B);
pawfe_status pawfe_apply_S(pawfe_ctx* ctx, pawfe_prec prec, const void* X, void* Y, long ld, int B);
pawfe_status pawfe_apply_Sinv(pawfe_ctx* ctx, pawfe_prec prec, const void* X, void* Y, long ld, int B);
/* Y = H S^-1approx X, the operator Algorithm 2 iterates (Alg. 1 step 2 L244; Eq. 30; T of Eq. 39 L367 is never
 * stored).  FP32 / TF32 blocks with 16-byte aligned X, Y and ld, B multiples of 4 (complex: of 2) run exactly the kernel
 * sequence of one filter step (projection, couplings, one cell contraction with the low-rank terms inside). */
pawfe_status pawfe_apply_HSinv(pawfe_ctx* ctx, pawfe_prec prec, const void* X, void* Y, long ld, int B);

/* Y = S^-1approx X without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, serving
 * loops, harnesses that forbid it).  Same result as pawfe_apply_Sinv up to the order of floating-point sums; same arguments.
 * The projections and couplings (2 * natoms * nproj * B scalars of the precision mode's type; complex contexts: pairs)
 * live in a static device array of 1 MiB (1,048,576 bytes) that every GPU that loads the library holds until the process
 * exits; a block that needs more gives PAWFE_EINVAL with the sizes in pawfe_last_error (narrow B, or use pawfe_apply_Sinv).
 * The call does no cudaMalloc / cudaFree and calls no allocating library routine; its FIRST call on a device looks the
 * array's address up (cudaGetSymbolAddress, no allocation): make that call once outside graph capture.
 * All calls on a device share the array and it keeps the last call's contents (the part in use is cleared first):
 * calls that overlap on the GPU (other streams, other contexts on the same device) race on it. */
pawfe_status pawfe_apply_Sinv_noalloc(pawfe_ctx* ctx, pawfe_prec prec, const void* X, void* Y, long ld, int B);

/* Build every internal plan and scratch array the hot calls need for blocks of up to Bmax vectors, Chebyshev degree up to
 * mmax, in precision mode prec (see Conventions).  Optional; synchronises the host.  Call again after the operators
 * change or for a wider block. */
pawfe_status pawfe_prepare(pawfe_ctx* ctx, pawfe_prec prec, int Bmax, int mmax);

/* ---- Algorithm 2 (L250-L282) --------------------------------------------------------------- */

/* Bytes of device workspace pawfe_cheb_filter needs for block width B (any leading dimension, any alignment of X). */
pawfe_status pawfe_filter_workspace(pawfe_ctx* ctx, pawfe_prec prec, int B, size_t* bytes);

/* Residual-based Chebyshev filter of degree m >= 1:
 *   step 1  e = (bU-bW)/2, c = (bU+bW)/2, zeta = e/(b0-c), gamma = 2/zeta                    (L257)
 *   step 2  Y = H X - S X Lambda                      always FP64 arithmetic                  (L260, L374)
 *   step 3  R_X = 0, R_Y = (zeta/e) Y, Lambda_X = 1, Lambda_Y = (zeta/e)(Lambda - c)           (L262-L264)
 *   step 4  for theta = 2..m: zeta1 = 1/(gamma - zeta);
 *             R_X <- (2 zeta1/e) H S^-1approx R_Y - (2 zeta1 c/e) R_Y - zeta zeta1 R_X  [prec]
 *                    + (2 zeta1/e) Y Lambda_Y                                        [FP64 add, L374]
 *             Lambda_X likewise; swap; zeta <- zeta1                                          (L269-L279)
 *   step 5  X <- S^-1approx R_Y + X Lambda_Y                                                    (L282)
 * X: device, in Psi_in / out Psi_f, [dof][vec], leading dimension ld, element type by prec.
 * lambda: HOST, B doubles.  workspace: device, >= pawfe_filter_workspace bytes, 256-byte aligned.
 * Needs b0 < bW < bU (strictly: a one-vector block needs bW above its Ritz value) and 1 <= m <= 512; PAWFE_EINVAL otherwise.
 * The B scalars are copied to the device asynchronously from an internal pinned buffer (the call waits on the host only
 * for the staging slot used four calls earlier). */
pawfe_status pawfe_cheb_filter(pawfe_ctx* ctx, pawfe_prec prec, int m, double b0, double bW, double bU,
                               void* X, const double* lambda, long ld, int B,
                               void* workspace, size_t workspace_bytes);

/* Algorithm 2 with step 2 taken from products the caller already holds: HX = H Psi_in and SX = S Psi_in (device, FP64
 * scalars, layout and leading dimension of X; complex interleaved), e.g. the H Psi_f Q, S Psi_f Q of the last Rayleigh-Ritz
 * step (L402-L408): Y = HX - SX Lambda costs no operator application (L260, L290).  Everything else as pawfe_cheb_filter. */
pawfe_status pawfe_cheb_filter_hs(pawfe_ctx* ctx, pawfe_prec prec, int m, double b0, double bW, double bU,
                                  void* X, const double* HX, const double* SX, const double* lambda, long ld, int B,
                                  void* workspace, size_t workspace_bytes);

/* Same call with HOST vector block X_host (B columns, leading dimension ld): copies it to an
 * internal device block, filters, copies Psi_f back, and synchronises.  The internal block and
 * workspace are allocated on first use for the largest B seen. */
pawfe_status pawfe_cheb_filter_host(pawfe_ctx* ctx, pawfe_prec prec, int m, double b0, double bW,
                                    double bU, void* X_host, const double* lambda, long ld, int B);

/* Algorithm 2 over nblk HOST vector blocks, one after the other (the blocks of one pass over the vector set, L378:
 * "blocks of wavefunctions" are filtered independently).  Block k: X_host[k] (B[k] columns, leading dimension ld[k],
 * element type by prec), Ritz values lambda[k] (HOST, B[k] doubles); the bounds are shared.  Same results as nblk calls
 * of pawfe_cheb_filter_host, but pipelined over two internal device blocks: block k+1's host-to-device copy and block
 * k-1's device-to-host copy run on the library's copy streams under block k's filter.  The host blocks should be
 * pinned (pageable memory works but serialises the copies).  Synchronises before returning.
 * PAWFE_EINVAL: nblk < 1, a null pointer, or arguments pawfe_cheb_filter rejects. */
pawfe_status pawfe_cheb_filter_host_set(pawfe_ctx* ctx, pawfe_prec prec, int m, double b0, double bW, double bU,
                                        void* const* X_host, const double* const* lambda, const long* ld,
                                        const int* B, int nblk);

/* Upper bound b_U of the spectrum of H S^-1approx, the operator the filter iterates (Alg. 1 steps 1-2, L243-L244; L179): k-step
 * Lanczos on H S^-1approx in the inner product <x, y> = Re x^dagger S^-1approx y (in which it is self-adjoint), FP64, with the
 * library's own applies; b_U = 1.02 (theta_max(T_k) + beta_k).  v0: DEVICE, start vector, M FP64 scalars of the context's kind
 * (complex interleaved); Dirichlet wall rows are ignored.  bU: HOST out.  theta_max, beta_k, steps_done: HOST out, optional
 * (largest Ritz value of the tridiagonal matrix, last off-diagonal, Lanczos steps taken: fewer than k on breakdown).
 * 1 <= k <= 256.  Not a hot call: allocates five work vectors and synchronises once per step.  Needs keep_fp64. */
pawfe_status pawfe_lanczos_bound(pawfe_ctx* ctx, int k, const void* v0, double* bU, double* theta_max, double* beta_k,
                                 int* steps_done);

/* ---- Rayleigh-Ritz kernels of Algorithm 1 (L246-L248; section 4.5) ----------------------- */

/* RR-Projection: G = X^dagger Y (B x B), FP64.  X, Y: device, FP64 blocks [dof][vec] with leading dimension ld (complex:
 * interleaved).  Only the 64 x 64 blocks of the LOWER triangle are computed (L402); the upper triangle is written as the
 * conjugate transpose, so G is exactly Hermitian: meant for Y = H X or Y = S X.  G: device, B * B FP64 scalars, row-major.
 * Sums are taken in a fixed order (bit-reproducible).  1 <= B <= 8192.  Allocates its partial sums per call and
 * synchronises the stream before returning. */
pawfe_status pawfe_rr_project(pawfe_ctx* ctx, const void* X, const void* Y, long ld, int B, void* G);

/* RR-SR, subspace rotation: Xout = X Q.  X, Xout: device FP64 blocks (leading dimensions ldx, ldo), must not overlap;
 * Q: device, B * B FP64 scalars, row-major.  mixed = 0: all products in FP64.  mixed != 0: the paper's mixed-precision
 * rotation (L406-L408): the 64 x 64 DIAGONAL blocks of Q in FP64, the OFF-DIAGONAL blocks in FP32 (operands rounded to
 * FP32, FP32 sums inside a block, blocks added in FP64): exact to FP64 level when Q is close to block-diagonal, i.e.
 * near convergence; ~1e-7 relative in general. */
pawfe_status pawfe_rr_rotate(pawfe_ctx* ctx, int mixed, const void* X, long ldx, const void* Q, void* Xout, long ldo, int B);

/* Column 2-norms ||x_i||_2, i < B, accumulated in FP64 (L290).  X: device, element type by prec;
 * out: DEVICE, B doubles. */
pawfe_status pawfe_col_norms(pawfe_ctx* ctx, pawfe_prec prec, const void* X, long ld, int B, double* out);

/* Count of kernels this context has launched so far (bench.py's gpu_launches). */
pawfe_status pawfe_launch_count(const pawfe_ctx* ctx, long* n);

/* CUDA-event timing of the cell-contraction launches inside H S^-1approx (the FP32 / TF32 cell kernel of
 * pawfe_apply_H and of step 4 of the filter): enable != 0 starts recording one event pair per launch on
 * the context's stream and resets the counters; 0 stops.  pawfe_cell_timing_read synchronises the stream
 * and returns the number of launches recorded and the sum of their durations in milliseconds. */
pawfe_status pawfe_cell_timing(pawfe_ctx* ctx, int enable);
pawfe_status pawfe_cell_timing_read(pawfe_ctx* ctx, long* launches, double* ms);
/* While pawfe_cell_timing is enabled every filter call also brackets its residual set-up (Alg. 2 steps 2-3, L260-L264: the
 * FP64 products and the scaling into R_Y) with an event pair: number of filter calls recorded and the sum of their set-up
 * times in milliseconds (bench.py's recurrence-only throughput = total minus this).  Synchronises the stream. */
pawfe_status pawfe_setup_timing_read(pawfe_ctx* ctx, long* calls, double* ms);

/* Name of the cell-contraction kernel variant a given (prec, B) runs ("tcgen05_tf32", "simt_fp32",
 * "dmma_fp64", ...).  Static string. */
const char* pawfe_cell_kernel_name(const pawfe_ctx* ctx, pawfe_prec prec, int B);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif /* PAWFE_H */
