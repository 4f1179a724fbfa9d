"""Spectral finite-element pieces of the oracle (TEST INFRASTRUCTURE; see oracle/__init__.py).

Follows PAPER.md section 2.2 (L116-L128, Eq. 12-13) and section 4.1 (L296-L321, Eq. 31-33):
C0 Lagrange basis on Gauss-Lobatto-Legendre nodes, tensor-product hexahedral cells, Gauss-Legendre
quadrature, cell matrices H^e, M^e, and their assembly into explicit sparse matrices.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp
from numpy.polynomial import legendre as npleg


# ----------------------------------------------------------------------------------------------
# 1-D rules and basis
# ----------------------------------------------------------------------------------------------

def gll(p: int):
    """p+1 Gauss-Lobatto-Legendre nodes on [-1,1] and weights.

    Nodes: roots of (1 - x^2) P_p'(x); weights w_a = 2 / (p (p+1) P_p(x_a)^2)  (
    DESIGN.md C1.1).  Interior roots from the companion matrix of P_p', polished by Newton.
    """
    Pp = npleg.Legendre.basis(p)
    dP = Pp.deriv()
    d2P = dP.deriv()
    xi = np.sort(np.real(dP.roots()))
    for _ in range(3):
        xi = xi - dP(xi) / d2P(xi)
    x = np.concatenate(([-1.0], xi, [1.0]))
    w = 2.0 / (p * (p + 1) * Pp(x) ** 2)
    return x, w


def gauss_legendre(n: int):
    """n-point Gauss-Legendre rule on [-1,1] (library primitive; exact to degree 2n-1)."""
    return npleg.leggauss(n)


def lagrange(nodes: np.ndarray, x: np.ndarray):
    """Values L[a, i] = l_a(x_i) and derivatives dL[a, i] = l_a'(x_i) of the Lagrange basis on `nodes`.

    l_a(x) = prod_{b != a} (x - xi_b) / (xi_a - xi_b)                      (Eq. 12 basis)
    l_a'(x) = sum_{c != a} 1/(xi_a - xi_c) prod_{b != a, c} (x - xi_b)/(xi_a - xi_b)
    """
    n = len(nodes)
    x = np.atleast_1d(np.asarray(x, dtype=float))
    L = np.ones((n, len(x)))
    dL = np.zeros((n, len(x)))
    for a in range(n):
        for b in range(n):
            if b != a:
                L[a] *= (x - nodes[b]) / (nodes[a] - nodes[b])
        for c in range(n):
            if c == a:
                continue
            term = np.full(len(x), 1.0 / (nodes[a] - nodes[c]))
            for b in range(n):
                if b != a and b != c:
                    term *= (x - nodes[b]) / (nodes[a] - nodes[b])
            dL[a] += term
    return L, dL


def matrices_1d(p: int):
    """Reference-interval matrices K1 = int l_a' l_b', M1 = int l_a l_b, G1 = int l_a l_b'.

    Integrated exactly by Gauss-Legendre with p+2 points (degree 2p needs >= p+1).
    """
    xi, _ = gll(p)
    xq, wq = gauss_legendre(p + 2)
    L, dL = lagrange(xi, xq)
    K1 = (dL * wq) @ dL.T
    M1 = (L * wq) @ L.T
    G1 = (L * wq) @ dL.T
    return K1, M1, G1


# ----------------------------------------------------------------------------------------------
# mesh
# ----------------------------------------------------------------------------------------------

class Mesh:
    """Uniform hexahedral mesh of a box [0,Lx]x[0,Ly]x[0,Lz]; lexicographic nodes (C1.1).

    Global node (ix,iy,iz), i = c*p + a; J = (ix*Ny + iy)*Nz + iz.  Periodic: i mod (nc*p).
    Dirichlet: nc*p+1 nodes per direction are STORED; boundary nodes are masked (reading R19/R-BC).
    """

    def __init__(self, ncells, box, p, bc="periodic"):
        self.ncells = tuple(int(n) for n in ncells)
        self.box = np.array(box, dtype=float)
        self.p = int(p)
        self.bc = bc
        self.n1 = p + 1
        self.n = self.n1 ** 3
        self.h = self.box / np.array(self.ncells)
        extra = 1 if bc == "dirichlet" else 0
        self.N = tuple(nc * p + extra for nc in self.ncells)
        self.M = self.N[0] * self.N[1] * self.N[2]
        self.ncell_total = self.ncells[0] * self.ncells[1] * self.ncells[2]
        self.xi, self.wgll = gll(p)

    def cell_index(self, cx, cy, cz):
        return (cx * self.ncells[1] + cy) * self.ncells[2] + cz

    def cell_coords(self, e):
        cz = e % self.ncells[2]
        cy = (e // self.ncells[2]) % self.ncells[1]
        cx = e // (self.ncells[1] * self.ncells[2])
        return cx, cy, cz

    def cell_nodes(self, cx, cy, cz):
        """Global node ids of cell (cx,cy,cz), cell-local order I = (a*n1 + b)*n1 + c."""
        p, n1 = self.p, self.n1
        a = np.arange(n1)
        ix = cx * p + a
        iy = cy * p + a
        iz = cz * p + a
        if self.bc == "periodic":
            ix, iy, iz = ix % self.N[0], iy % self.N[1], iz % self.N[2]
        J = (ix[:, None, None] * self.N[1] + iy[None, :, None]) * self.N[2] + iz[None, None, :]
        return J.reshape(-1)

    def cell_origin(self, cx, cy, cz):
        return np.array([cx, cy, cz]) * self.h

    def interior_mask(self):
        """1 for free dofs, 0 for Dirichlet boundary nodes (all ones when periodic)."""
        if self.bc != "dirichlet":
            return np.ones(self.M, dtype=bool)
        m = []
        for N in self.N:
            v = np.ones(N, dtype=bool)
            v[0] = v[-1] = False
            m.append(v)
        return (m[0][:, None, None] & m[1][None, :, None] & m[2][None, None, :]).reshape(-1)

    def node_coords(self):
        """Coordinates of all stored nodes, shape (M, 3)."""
        c1 = []
        for d in range(3):
            x = np.zeros(self.N[d])
            for c in range(self.ncells[d]):
                for a in range(self.n1):
                    i = c * self.p + a
                    if self.bc == "periodic":
                        i %= self.N[d]
                    x[i] = self.h[d] * (c + 0.5 * (self.xi[a] + 1.0))
            if self.bc == "periodic":
                x[0] = 0.0
            c1.append(x)
        X, Y, Z = np.meshgrid(c1[0], c1[1], c1[2], indexing="ij")
        return np.stack([X.reshape(-1), Y.reshape(-1), Z.reshape(-1)], axis=1)


# ----------------------------------------------------------------------------------------------
# potential and cell matrices
# ----------------------------------------------------------------------------------------------

def gaussian_potential(x, pos, Z, sigma, box, periodic: bool):
    """V(x) = - sum_a sum_images Z_a exp(-|x - R_a - L_r|^2 / (2 sigma_a^2))  (C1.4).

    Stands in for V_eff + V_z of Eq. 2.  Periodic: the 27 nearest images.
    x: (nq, 3).  Returns (nq,).
    """
    V = np.zeros(len(x))
    shifts = [-1, 0, 1] if periodic else [0]
    for a in range(len(pos)):
        for sx in shifts:
            for sy in shifts:
                for sz in shifts:
                    R = pos[a] + np.array([sx, sy, sz]) * box
                    d2 = np.sum((x - R) ** 2, axis=1)
                    V -= Z[a] * np.exp(-d2 / (2.0 * sigma[a] ** 2))
    return V


def cell_quadrature(mesh: Mesh, nq: int, cx, cy, cz):
    """Gauss-Legendre tensor grid in cell (cx,cy,cz): points (nq^3,3), weights*detJ (nq^3,), 1-D basis."""
    xq, wq = gauss_legendre(nq)
    L1, dL1 = lagrange(mesh.xi, xq)
    o = mesh.cell_origin(cx, cy, cz)
    px = o[0] + 0.5 * mesh.h[0] * (xq + 1.0)
    py = o[1] + 0.5 * mesh.h[1] * (xq + 1.0)
    pz = o[2] + 0.5 * mesh.h[2] * (xq + 1.0)
    X, Y, Z = np.meshgrid(px, py, pz, indexing="ij")
    pts = np.stack([X.reshape(-1), Y.reshape(-1), Z.reshape(-1)], axis=1)
    detJ = mesh.h[0] * mesh.h[1] * mesh.h[2] / 8.0
    W = (wq[:, None, None] * wq[None, :, None] * wq[None, None, :]).reshape(-1) * detJ
    return pts, W, L1, dL1


def shape_at_quadrature(L1):
    """N[I, q] = l_a(q_x) l_b(q_y) l_c(q_z), I = (a*n1+b)*n1+c, q = (qx*nq+qy)*nq+qz."""
    return np.kron(np.kron(L1, L1), L1)


def reference_cell_matrices(mesh: Mesh):
    """Kinetic, mass and gradient cell matrices of the (uniform) cell (Eq. 32-33).

    Jacobian diag(h/2).  K^e = sum_d (2/h_d) prod_{d' != d}(h_d'/2) [K1 in slot d, M1 elsewhere];
    M^e = (hx hy hz / 8) M1 x M1 x M1;  G_d^e = prod_{d' != d}(h_d'/2) [G1 in slot d, M1 elsewhere].
    """
    K1, M1, G1 = matrices_1d(mesh.p)
    hx, hy, hz = 0.5 * mesh.h
    k3 = lambda A, B, C: np.kron(np.kron(A, B), C)
    Ke = (hy * hz / hx) * k3(K1, M1, M1) + (hx * hz / hy) * k3(M1, K1, M1) + (hx * hy / hz) * k3(M1, M1, K1)
    Me = hx * hy * hz * k3(M1, M1, M1)
    Gx = hy * hz * k3(G1, M1, M1)
    Gy = hx * hz * k3(M1, G1, M1)
    Gz = hx * hy * k3(M1, M1, G1)
    return Ke, Me, (Gx, Gy, Gz)


def potential_cell_matrix(mesh: Mesh, sysd, cx, cy, cz, nq2=None):
    """V^e_IJ = sum_q w_q N_I(x_q) N_J(x_q) V(x_q) detJ on an n_q2 = p+2 per-direction grid
    (Eq. 32 third line; reading R8)."""
    nq2 = nq2 or (mesh.p + 2)
    pts, W, L1, _ = cell_quadrature(mesh, nq2, cx, cy, cz)
    V = gaussian_potential(pts, sysd.pos, sysd.Z, sysd.sigmaV, mesh.box, mesh.bc == "periodic")
    Nq = shape_at_quadrature(L1)
    return (Nq * (W * V)) @ Nq.T


def hamiltonian_cell_matrix(mesh: Mesh, sysd, cx, cy, cz, kpt=None, ref=None, with_potential=True):
    """H^e = 1/2 K^e + V^e + 1/2 |k|^2 M^e - i sum_d k_d G_d^e   (Eq. 13; reading R6:
    the k-term is  -i k . N_I grad N_J  as in Eq. 13, not Eq. 32's extraction)."""
    Ke, Me, G = ref if ref is not None else reference_cell_matrices(mesh)
    He = 0.5 * Ke
    if with_potential:
        He = He + potential_cell_matrix(mesh, sysd, cx, cy, cz)
    if kpt is not None:
        He = He + 0.5 * float(np.dot(kpt, kpt)) * Me - 1j * (kpt[0] * G[0] + kpt[1] * G[1] + kpt[2] * G[2])
    return He


def assemble(mesh: Mesh, cell_matrix_fn, dtype=float):
    """Assemble cell matrices into an explicit CSR matrix over the STORED node grid:
    A = sum_e P_e^T A^e P_e with P_e the cell->node gather.
    Dirichlet: boundary rows and columns are zeroed afterwards."""
    rows, cols, vals = [], [], []
    for cx in range(mesh.ncells[0]):
        for cy in range(mesh.ncells[1]):
            for cz in range(mesh.ncells[2]):
                J = mesh.cell_nodes(cx, cy, cz)
                Ae = cell_matrix_fn(cx, cy, cz)
                rows.append(np.repeat(J, mesh.n))
                cols.append(np.tile(J, mesh.n))
                vals.append(np.asarray(Ae, dtype=dtype).reshape(-1))
    A = sp.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))),
                      shape=(mesh.M, mesh.M)).tocsr()
    if mesh.bc == "dirichlet":
        m = sp.diags(mesh.interior_mask().astype(float))
        A = (m @ A @ m).tocsr()
    return A


def lumped_mass(mesh: Mesh):
    """M_D: diagonal mass from GLL quadrature, (M_D)_JJ = sum_{e contains J} detJ w_a w_b w_c
    (PAPER.md:L228 approximation (i))."""
    md = np.zeros(mesh.M)
    detJ = mesh.h[0] * mesh.h[1] * mesh.h[2] / 8.0
    w3 = (mesh.wgll[:, None, None] * mesh.wgll[None, :, None] * mesh.wgll[None, None, :]).reshape(-1) * detJ
    for cx in range(mesh.ncells[0]):
        for cy in range(mesh.ncells[1]):
            for cz in range(mesh.ncells[2]):
                np.add.at(md, mesh.cell_nodes(cx, cy, cz), w3)
    return md


def apply_cellwise(mesh: Mesh, cell_matrix_fn, X):
    """sum_e scatter(A^e gather(X)): the paper's 4-step AX without the non-local part
    (Fig. 2 steps i, iii, iv).  Used to pin cell-wise == assembled."""
    Y = np.zeros((mesh.M, X.shape[1]), dtype=np.result_type(X.dtype, float))
    mask = mesh.interior_mask()
    Xm = X * mask[:, None]
    first = True
    for cx in range(mesh.ncells[0]):
        for cy in range(mesh.ncells[1]):
            for cz in range(mesh.ncells[2]):
                J = mesh.cell_nodes(cx, cy, cz)
                Ae = cell_matrix_fn(cx, cy, cz)
                if first and np.iscomplexobj(Ae):
                    Y = Y.astype(complex)
                first = False
                np.add.at(Y, J, Ae @ Xm[J])
    return Y * mask[:, None]
