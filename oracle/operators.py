"""Assembled PAW-FE operators H, S and the approximate inverse overlap (TEST INFRASTRUCTURE).

H = H_loc + sum_a C^a D^a C^a^dagger,  S = M + sum_a C^a dS^a C^a^dagger           (Eq. 16, PAPER.md:L137;
                                                                       reading R1 for the lost Eq. 14)
S^-1 approx = M_D^-1 - sum_a M_D^-1 C^a Delta^a_Sinv C^a^dagger M_D^-1               (Eq. 28)
All explicit sparse matrices in FP64; applications are products of the explicit factors.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp

from . import fe, paw


class PawOperators:
    def __init__(self, sysd, with_potential: bool = True, with_nonlocal: bool = True):
        cfg = sysd.cfg
        self.sysd = sysd
        self.cfg = cfg
        self.mesh = fe.Mesh(cfg.ncells, cfg.box, cfg.p, cfg.bc)
        mesh = self.mesh
        self.kpt = cfg.kpoint
        self.dtype = complex if self.kpt is not None else float
        self.mask = mesh.interior_mask()
        self.ref = fe.reference_cell_matrices(mesh)
        self.with_potential = with_potential

        self.Hloc = fe.assemble(mesh, self.H_cell, dtype=self.dtype)
        self.M = fe.assemble(mesh, lambda cx, cy, cz: self.ref[1])
        self.md = fe.lumped_mass(mesh)
        self.md_inv = np.where(self.mask, 1.0 / self.md, 0.0)

        npj = len(sysd.proj_l)
        if with_nonlocal:
            self.C, self.pairs = paw.build_C(mesh, sysd, self.kpt)
            self.D = sysd.D
            self.dS = sysd.dS
        else:
            self.C = sp.csr_matrix((mesh.M, len(sysd.pos) * npj), dtype=self.dtype)
            self.pairs = []
            self.D = np.zeros_like(sysd.D)
            self.dS = np.zeros_like(sysd.dS)
        self.Ch = self.C.conj().T.tocsr()
        self.Dbig = paw.block_diag_coupling(self.D)
        self.dSbig = paw.block_diag_coupling(self.dS)
        self.dSinv, self.G = paw.sinv_couplings(self.C, self.md_inv, self.dS)
        self.dSinvbig = paw.block_diag_coupling(self.dSinv)

    # -- cell matrices ---------------------------------------------------------------------
    def H_cell(self, cx, cy, cz):
        return fe.hamiltonian_cell_matrix(self.mesh, self.sysd, cx, cy, cz, self.kpt, self.ref,
                                          self.with_potential)

    def M_cell(self, cx, cy, cz):
        return self.ref[1]

    # -- operator applications ---------------------------------------------------------------
    def apply_H(self, X):
        """Y = H X = H_loc X + C (D (C^dagger X))   (Eq. 13, 16)."""
        return self.Hloc @ X + self.C @ (self.Dbig @ (self.Ch @ X))

    def apply_S(self, X):
        """Y = S X = M X + C (dS (C^dagger X))   (Eq. 13, 16)."""
        return self.M @ X + self.C @ (self.dSbig @ (self.Ch @ X))

    def apply_Sinv(self, X):
        """Y = M_D^-1 X - M_D^-1 C (Delta_Sinv (C^dagger (M_D^-1 X)))   (Eq. 28; T of Eq. 39)."""
        T = self.md_inv[:, None] * X
        return T - self.md_inv[:, None] * (self.C @ (self.dSinvbig @ (self.Ch @ T)))

    # -- dense forms for tiny meshes ---------------------------------------------------------
    def dense_H(self):
        return (self.Hloc + self.C @ self.Dbig @ self.Ch).toarray()

    def dense_S(self):
        return (self.M + self.C @ self.dSbig @ self.Ch).toarray()

    def free(self):
        """indices of free (non-Dirichlet) dofs"""
        return np.nonzero(self.mask)[0]


def apply_H_rows(sysd, X, cells):
    """Sampled rows of H X at full size: for each listed cell (cx,cy,cz) return the global node ids of
    the cell and (H X) at those nodes, computed one by one from the definitions without forming H:

      (H X)_J = sum_{e contains J} (H^e X_e)_{I(J)}  +  sum_a C^a_J (D^a (C^a^dagger X)).

    Only the 27 cells around each sampled cell and the atoms whose sphere meets them are evaluated.
    """
    cfg = sysd.cfg
    mesh = fe.Mesh(cfg.ncells, cfg.box, cfg.p, cfg.bc)
    kpt = cfg.kpoint
    ref = fe.reference_cell_matrices(mesh)
    mask = mesh.interior_mask()
    Xm = X * mask[:, None]
    npj = len(sysd.proj_l)
    out = []
    for (cx, cy, cz) in cells:
        J0 = mesh.cell_nodes(cx, cy, cz)
        pos_in = {int(j): i for i, j in enumerate(J0)}
        acc = np.zeros((mesh.n, X.shape[1]), dtype=np.result_type(X.dtype, complex if kpt is not None else float))
        seen = set()
        for dx in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for dz in (-1, 0, 1):
                    c = [cx + dx, cy + dy, cz + dz]
                    if cfg.bc == "periodic":
                        c = [c[i] % mesh.ncells[i] for i in range(3)]
                    elif any(c[i] < 0 or c[i] >= mesh.ncells[i] for i in range(3)):
                        continue
                    if tuple(c) in seen:
                        continue
                    seen.add(tuple(c))
                    J = mesh.cell_nodes(*c)
                    hit = [(pos_in[int(j)], i) for i, j in enumerate(J) if int(j) in pos_in]
                    if not hit:
                        continue
                    He = fe.hamiltonian_cell_matrix(mesh, sysd, c[0], c[1], c[2], kpt, ref)
                    Ye = He @ Xm[J]
                    for (i0, i) in hit:
                        acc[i0] += Ye[i]
        # non-local part: atoms whose sphere can reach the sampled cell
        cen = mesh.cell_origin(cx, cy, cz) + 0.5 * mesh.h
        for a in range(len(sysd.pos)):
            dc = cen - sysd.pos[a]
            if cfg.bc == "periodic":
                dc -= mesh.box * np.round(dc / mesh.box)
            if np.linalg.norm(dc) > sysd.rc + np.sqrt(3.0) * float(np.max(mesh.h)):
                continue
            Ca, _ = paw.build_C(mesh, sysd, kpt, atoms=[a])
            Ca = Ca[:, a * npj:(a + 1) * npj]
            P = Ca.conj().T @ X
            acc += Ca[J0] @ (sysd.D[a] @ P)
        out.append((J0, acc * mask[J0][:, None]))
    return out
