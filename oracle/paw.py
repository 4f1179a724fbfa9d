"""PAW non-local pieces of the oracle (TEST INFRASTRUCTURE; see oracle/__init__.py).

Projector functions, projector-basis integrals C^a (Eq. 17 / Eq. 34),
and the approximate inverse overlap couplings (Eq. 28-29).
"""
from __future__ import annotations

import math

import numpy as np
import scipy.sparse as sp

from .fe import Mesh, cell_quadrature, lumped_mass


def solid_harmonic(l: int, m: int, d: np.ndarray) -> np.ndarray:
    """r^l Y_lm(d/|d|): real orthonormal spherical harmonics times r^l, l <= 2 (C1.5)."""
    x, y, z = d[:, 0], d[:, 1], d[:, 2]
    if l == 0:
        return np.full(len(d), 0.5 / math.sqrt(math.pi))
    if l == 1:
        c = math.sqrt(3.0 / (4.0 * math.pi))
        return c * {-1: y, 0: z, 1: x}[m]
    if l == 2:
        c = math.sqrt(15.0 / (4.0 * math.pi))
        if m == -2:
            return c * x * y
        if m == -1:
            return c * y * z
        if m == 0:
            return math.sqrt(5.0 / (16.0 * math.pi)) * (3.0 * z * z - (x * x + y * y + z * z))
        if m == 1:
            return c * x * z
        if m == 2:
            return 0.5 * c * (x * x - y * y)
    raise ValueError("l <= 2 only")


def projector_values(sysd, d: np.ndarray) -> np.ndarray:
    """p_alpha(d) = amp_alpha exp(-r^2 / 2 sigma_alpha^2) (1 - (r/rc)^2)^2 r^l Y_lm(dhat), r < rc, else 0.
    d: (nq, 3) -> (nproj, nq)."""
    r2 = np.sum(d * d, axis=1)
    inside = r2 < sysd.rc ** 2
    cut = np.where(inside, (1.0 - r2 / sysd.rc ** 2) ** 2, 0.0)
    out = np.zeros((len(sysd.proj_l), len(d)))
    for al in range(len(sysd.proj_l)):
        l, m = int(sysd.proj_l[al]), int(sysd.proj_m[al])
        out[al] = sysd.proj_amp[al] * np.exp(-r2 / (2.0 * sysd.proj_sigma[al] ** 2)) * cut * solid_harmonic(l, m, d)
    return out


def atom_cell_block(mesh: Mesh, sysd, a: int, cx, cy, cz, kpt=None, nq3=None):
    """Cell contribution to C^{a dagger}: (C^{e,a dagger})_{alpha I} =
        sum_r sum_q w_q e^{i k.(x_q - L_r)} N_I(x_q) p_alpha(x_q - R_a - L_r) detJ      (Eq. 34)
    on an n_q3 = 2(p+2) per-direction Gauss-Legendre grid (reading R8).  Since rc < L/2 at most one image
    is non-zero at a point: d = minimum-image (x_q - R_a); the phase is evaluated at the unwrapped point
    x_q - L_r = R_a + d (reading R7).  Returns None if the cell does not meet the sphere, else
    an (nproj, n) array (complex if kpt is given)."""
    nq3 = nq3 or 2 * (mesh.p + 2)
    pts, W, L1, _ = cell_quadrature(mesh, nq3, cx, cy, cz)
    d = pts - sysd.pos[a]
    if mesh.bc == "periodic":
        d -= mesh.box * np.round(d / mesh.box)
    if not np.any(np.sum(d * d, axis=1) < sysd.rc ** 2):
        return None
    P = projector_values(sysd, d) * W                       # (nproj, nq^3)
    if kpt is not None:
        P = P * np.exp(1j * ((sysd.pos[a] + d) @ kpt))
    n1 = mesh.n1
    F = P.reshape(len(sysd.proj_l), nq3, nq3, nq3)
    # sum_q N_I(x_q) F_q with N_I = l_a(qx) l_b(qy) l_c(qz)
    Cd = np.einsum("pxyz,ax,by,cz->pabc", F, L1, L1, L1)
    return Cd.reshape(len(sysd.proj_l), n1 ** 3)


def build_C(mesh: Mesh, sysd, kpt=None, atoms=None):
    """Explicit sparse C (M x natoms*nproj): column block a holds C^a = (C^{a dagger})^dagger (Eq. 16-17).
    Dirichlet boundary rows are zeroed.  Also returns the (cell, atom) pair list."""
    npj = len(sysd.proj_l)
    natoms = len(sysd.pos)
    atoms = range(natoms) if atoms is None else atoms
    rows, cols, vals, pairs = [], [], [], []
    hmax = float(np.max(mesh.h))
    for a in atoms:
        for cx in range(mesh.ncells[0]):
            for cy in range(mesh.ncells[1]):
                for cz in range(mesh.ncells[2]):
                    # cheap reject: cell centre farther than rc + half diagonal
                    cen = mesh.cell_origin(cx, cy, cz) + 0.5 * mesh.h
                    dc = cen - sysd.pos[a]
                    if mesh.bc == "periodic":
                        dc -= mesh.box * np.round(dc / mesh.box)
                    if np.linalg.norm(dc) > sysd.rc + 0.5 * math.sqrt(3.0) * hmax:
                        continue
                    Cd = atom_cell_block(mesh, sysd, a, cx, cy, cz, kpt)
                    if Cd is None:
                        continue
                    pairs.append((mesh.cell_index(cx, cy, cz), a))
                    J = mesh.cell_nodes(cx, cy, cz)
                    rows.append(np.tile(J, npj))
                    cols.append(np.repeat(a * npj + np.arange(npj), mesh.n))
                    vals.append(np.conj(Cd).reshape(-1))
    dtype = complex if kpt is not None else float
    if rows:
        C = sp.coo_matrix((np.concatenate(vals).astype(dtype),
                           (np.concatenate(rows), np.concatenate(cols))),
                          shape=(mesh.M, natoms * npj)).tocsr()
    else:
        C = sp.csr_matrix((mesh.M, natoms * npj), dtype=dtype)
    if mesh.bc == "dirichlet":
        C = (sp.diags(mesh.interior_mask().astype(float)) @ C).tocsr()
    return C, pairs


def block_diag_coupling(blocks: np.ndarray):
    """sparse block-diagonal matrix of per-atom n_pj x n_pj couplings."""
    return sp.block_diag([sp.csr_matrix(b) for b in blocks], format="csr")


def projector_overlap_matrix(sysd) -> np.ndarray:
    """<p_alpha|p_beta> = int p_alpha(d) p_beta(d) d^3d over the cutoff sphere: the matrix the paper says C^a^dagger M^-1 C^a
    "can be approximated by" (text after Eq. 29).  Real orthonormal Y_lm make it block diagonal in (l, m);
    the radial integral is taken by adaptive quadrature."""
    import scipy.integrate as si
    npj = len(sysd.proj_l)
    O = np.zeros((npj, npj))
    for a in range(npj):
        for b in range(npj):
            if sysd.proj_l[a] != sysd.proj_l[b] or sysd.proj_m[a] != sysd.proj_m[b]:
                continue
            l, sa, sb, rc = int(sysd.proj_l[a]), sysd.proj_sigma[a], sysd.proj_sigma[b], sysd.rc
            f = lambda r: (r ** l * math.exp(-r * r / (2 * sa * sa)) * (1 - (r / rc) ** 2) ** 2) * \
                          (r ** l * math.exp(-r * r / (2 * sb * sb)) * (1 - (r / rc) ** 2) ** 2) * r * r
            O[a, b] = sysd.proj_amp[a] * sysd.proj_amp[b] * si.quad(f, 0.0, rc, epsabs=1e-14, epsrel=1e-13)[0]
    return O


def sinv_couplings(C, md_inv: np.ndarray, dS: np.ndarray, G_override=None):
    """Delta^a_Sinv = (dS^a^-1 + C^a^dagger M_D^-1 C^a)^-1   (Eq. 29), evaluated as
    (I + dS^a G^a)^-1 dS^a (reading R10: same matrix, no inverse of dS^a).  Cross-atom blocks of
    C^dagger M_D^-1 C are dropped (approximation (ii)).  G_override: use this n_pj x n_pj matrix as G^a of every atom
    instead (the <p_alpha|p_beta> variant of L228: projector_overlap_matrix)."""
    natoms, npj, _ = dS.shape
    out = np.zeros((natoms, npj, npj), dtype=C.dtype)
    G = []
    for a in range(natoms):
        Ca = C[:, a * npj:(a + 1) * npj]
        Ga = (Ca.conj().T @ sp.diags(md_inv) @ Ca).toarray() if G_override is None else np.asarray(G_override, dtype=C.dtype)
        G.append(Ga)
        out[a] = np.linalg.solve(np.eye(npj) + dS[a] @ Ga, dS[a].astype(C.dtype))
    return out, np.array(G)
