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
    def __init__(self, sysd, with_potential: bool = True, with_nonlocal: bool = True, sinv_variant: int = 0):
        """sinv_variant: 0 = G^a = C^a^dagger M_D^-1 C^a in Eq. 29 (default); 1 = G^a = <p_alpha|p_beta>"""
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
        self.dSinv, self.G = paw.sinv_couplings(self.C, self.md_inv, self.dS,
                                                paw.projector_overlap_matrix(sysd) if sinv_variant == 1 else None)
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
            # cheap reject, rigorous: a node of the sampled cell gets weight from any of the 27 cells around it, whose farthest
            # point is 1.5 sqrt(3) h from the sampled cell's centre
            if np.linalg.norm(dc) > sysd.rc + 1.5 * np.sqrt(3.0) * float(np.max(mesh.h)):
                continue
            Ca, _ = paw.build_C(mesh, sysd, kpt, atoms=[a])
            Ca = Ca[:, a * npj:(a + 1) * npj]
            P = Ca.conj().T @ X
            acc += Ca[J0] @ (sysd.D[a] @ P)
        out.append((J0, acc * mask[J0][:, None]))
    return out


def _box_cells_near_atom(mesh, cfg, pos_a, rc):
    """Cells whose box comes within rc of the atom (minimum image when periodic): a cheap geometric SUPERSET of the cells
    that hold projector weight; the exact set is decided by paw.atom_cell_block (None = no quadrature point inside rc)."""
    per = cfg.bc == "periodic"
    cand = []
    for d in range(3):
        lo = np.arange(mesh.ncells[d]) * mesh.h[d]
        hi = lo + mesh.h[d]
        best = np.full(mesh.ncells[d], np.inf)
        for s in ((-1, 0, 1) if per else (0,)):
            xs = pos_a[d] + s * mesh.box[d]
            best = np.minimum(best, np.where(xs < lo, lo - xs, np.where(xs > hi, xs - hi, 0.0)))
        cand.append([(c, best[c] ** 2) for c in range(mesh.ncells[d]) if best[c] < rc])
    return [(cx, cy, cz) for cx, dx in cand[0] for cy, dy in cand[1] for cz, dz in cand[2] if dx + dy + dz < rc * rc]


def _cell_neighbourhood(mesh, cfg, c):
    out = set()
    for dx in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dz in (-1, 0, 1):
                q = [c[0] + dx, c[1] + dy, c[2] + dz]
                if cfg.bc == "periodic":
                    q = [q[i] % mesh.ncells[i] for i in range(3)]
                elif any(q[i] < 0 or q[i] >= mesh.ncells[i] for i in range(3)):
                    continue
                out.add(tuple(q))
    return out


def atom_pair_blocks(sysd, a):
    """[(cell (cx, cy, cz), C^{e,a dagger} block)] over the cells that hold weight of atom a (paw.atom_cell_block, Eq. 34).
    Module-level and free of shared state so that a test can evaluate many atoms in parallel worker processes."""
    cfg = sysd.cfg
    mesh = fe.Mesh(cfg.ncells, cfg.box, cfg.p, cfg.bc)
    out = []
    for c in sorted(_box_cells_near_atom(mesh, cfg, sysd.pos[a], sysd.rc)):
        Cd = paw.atom_cell_block(mesh, sysd, a, c[0], c[1], c[2], cfg.kpoint)
        if Cd is not None:
            out.append((c, Cd))
    return out


def atoms_near_cells(sysd, cells, radius):
    """atoms whose (minimum-image) distance to the centre of one of the cells is below radius"""
    cfg = sysd.cfg
    mesh = fe.Mesh(cfg.ncells, cfg.box, cfg.p, cfg.bc)
    out = []
    for a in range(len(sysd.pos)):
        for c in cells:
            d = mesh.cell_origin(*c) + 0.5 * mesh.h - sysd.pos[a]
            if cfg.bc == "periodic":
                d -= mesh.box * np.round(d / mesh.box)
            if np.linalg.norm(d) < radius:
                out.append(a)
                break
    return out


def apply_HSinv_rows(sysd, X, cells, op="HSinv", cache=None):
    """Sampled rows of  H S^-1approx X  (the operator Algorithm 2 iterates: Alg. 1 step 2; Eq. 28; Eq. 30,
    L230) at full size, from the definitions, without forming any global matrix:

        T      = M_D^-1 X - M_D^-1 sum_b C^b Delta^b_Sinv (C^b^dagger M_D^-1 X)                       (Eq. 28)
        (H T)_J = sum_{e contains J} (H^e T_e)_{I(J)} + sum_a C^a_J (D^a (C^a^dagger T))              (Eq. 13, 16)

    for the nodes J of each listed cell (cx, cy, cz).  T is evaluated only where it is needed: on the nodes of the 27 cells
    around the sampled cell and on the supports of the atoms a that reach the sampled cell; the atoms b that enter T there are
    all atoms whose projector cells touch (share a node with) those regions.  X needs only row indexing: X[J] for an integer
    index array J must return the (len(J), B) rows as a NumPy array (a NumPy array does; tests pass a device-tensor wrapper).
    op="H" returns the rows of H X instead (T = X on the free dofs): the same evaluation as apply_H_rows, for an X that can
    only be indexed by rows.  cache: an optional dict that keeps the projector blocks and cell matrices between calls on the
    same system (they do not depend on X or op); cache["blocks"][a] may be pre-filled with atom_pair_blocks(sysd, a).
    Returns [(J0, rows)] like apply_H_rows."""
    if op not in ("HSinv", "H"):
        raise ValueError(op)
    cfg = sysd.cfg
    mesh = fe.Mesh(cfg.ncells, cfg.box, cfg.p, cfg.bc)
    kpt = cfg.kpoint
    ref = fe.reference_cell_matrices(mesh)
    mask = mesh.interior_mask()
    md_inv = np.where(mask, 1.0 / fe.lumped_mass(mesh), 0.0)
    npj = len(sysd.proj_l)
    natoms = len(sysd.pos)
    dtype = complex if kpt is not None else float
    box_cells = [set(_box_cells_near_atom(mesh, cfg, sysd.pos[a], sysd.rc)) for a in range(natoms)]
    cache = {} if cache is None else cache
    pairs_of = cache.setdefault("atom_pairs", {})      # atom -> [(J, C^{e,a})], evaluated on demand
    He_of = cache.setdefault("He", {})                 # cell -> H^e

    def atom_pairs(a):
        """[(cell nodes J, C^{e,a} = conj(block)^T with Dirichlet rows zeroed)] over the cells that hold weight of atom a"""
        if a not in pairs_of:
            raw = cache.get("blocks", {}).get(a)
            if raw is None:
                raw = atom_pair_blocks(sysd, a)
            out = []
            for c, Cd in raw:
                J = mesh.cell_nodes(*c)
                out.append((J, np.conj(Cd).T * mask[J][:, None]))
            pairs_of[a] = out
        return pairs_of[a]

    def rows_in(J, nodes):
        """positions (in J, in the sorted array nodes) of the entries of J that occur in nodes"""
        k = np.searchsorted(nodes, J)
        k[k == len(nodes)] = 0
        ii = np.nonzero(nodes[k] == J)[0]
        return ii, k[ii]

    def project(a, rows_of):
        """C^a^dagger V for a vector field given by rows_of(J) -> V[J]"""
        P = np.zeros((npj, ncol), dtype=dtype)
        for J, Ce in atom_pairs(a):
            P += Ce.conj().T @ rows_of(J)
        return P

    out = []
    for c0 in cells:
        c0 = tuple(int(v) for v in c0)
        J0 = mesh.cell_nodes(*c0)
        ncol = np.asarray(X[J0[:1]]).shape[1]
        near = _cell_neighbourhood(mesh, cfg, c0)
        # atoms with weight on a node of the sampled cell: the assembled C^a_J sums over EVERY cell that contains J (Eq. 16-17),
        # so an atom that only reaches a neighbour cell still contributes at the shared face / edge / corner nodes
        A0 = [a for a in range(natoms) if box_cells[a] & near]
        region = set(near)                                                     # cells on whose nodes T is needed
        for a in A0:
            region |= box_cells[a]
        touch = set()
        for c in region:
            touch |= _cell_neighbourhood(mesh, cfg, c)                         # cells sharing a node with the region
        Bset = [b for b in range(natoms) if box_cells[b] & touch] if op == "HSinv" else []
        # W^b = Delta^b_Sinv C^b^dagger M_D^-1 X, with Delta^b_Sinv = (I + dS^b G^b)^-1 dS^b, G^b = C^b^dagger M_D^-1 C^b (Eq. 29, R10)
        W = {}
        for b in Bset:
            prs = atom_pairs(b)
            if not prs:
                continue
            # assemble the atom's sparse column block on its own nodes (a node shared by two of its cells gets both parts)
            nodes = np.unique(np.concatenate([J for J, _ in prs]))          # sorted
            Cb = np.zeros((len(nodes), npj), dtype=dtype)
            for J, Ce in prs:
                np.add.at(Cb, np.searchsorted(nodes, J), Ce)
            G = Cb.conj().T @ (md_inv[nodes][:, None] * Cb)
            dSinv = np.linalg.solve(np.eye(npj) + sysd.dS[b] @ G, sysd.dS[b].astype(dtype))
            P1 = Cb.conj().T @ (md_inv[nodes][:, None] * np.asarray(X[nodes]))
            W[b] = (nodes, Cb, dSinv @ P1)

        def T_rows(J):
            J = np.asarray(J)
            if op == "H":
                return mask[J][:, None] * np.asarray(X[J]).astype(dtype)
            t = md_inv[J][:, None] * np.asarray(X[J]).astype(dtype)
            for b, (nodes, Cb, Wb) in W.items():
                ii, kk = rows_in(J, nodes)
                if len(ii):
                    t[ii] -= md_inv[J[ii]][:, None] * (Cb[kk] @ Wb)
            return t

        pos_in = {int(j): i for i, j in enumerate(J0)}
        acc = np.zeros((mesh.n, ncol), dtype=dtype)
        for c in sorted(near):
            J = mesh.cell_nodes(*c)
            hit = [(pos_in[int(j)], i) for i, j in enumerate(J) if int(j) in pos_in]
            if not hit:
                continue
            if c not in He_of:
                He_of[c] = fe.hamiltonian_cell_matrix(mesh, sysd, c[0], c[1], c[2], kpt, ref)
            Ye = He_of[c] @ (T_rows(J) * mask[J][:, None])
            for (i0, i) in hit:
                acc[i0] += Ye[i]
        for a in A0:
            prs = atom_pairs(a)
            if not prs:
                continue
            P2 = project(a, T_rows)
            for J, Ce in prs:
                hit = [(pos_in[int(j)], i) for i, j in enumerate(J) if int(j) in pos_in]
                for (i0, i) in hit:
                    acc[i0] += Ce[i] @ (sysd.D[a] @ P2)
        out.append((J0, acc * mask[J0][:, None]))
    return out
