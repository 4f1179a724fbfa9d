"""Pins of the oracle's PAW pieces: projector integrals, Woodbury inverse."""
import dataclasses
import math

import numpy as np
import scipy.integrate as si
import scipy.sparse as sp

from oracle import fe, paw
from oracle.operators import PawOperators
from pawfe_inputs import get_config, make_system, projector_table


def _radial(sysd, al, power):
    """int_0^rc amp f(r) r^power dr with f the radial part WITHOUT r^l (independent adaptive quadrature)."""
    s, amp, rc = sysd.proj_sigma[al], sysd.proj_amp[al], sysd.rc
    f = lambda r: amp * math.exp(-r * r / (2 * s * s)) * (1 - (r / rc) ** 2) ** 2 * r ** power
    return si.quad(f, 0.0, rc, epsabs=1e-14, epsrel=1e-13)[0]


def test_solid_harmonics_orthonormal_on_sphere():
    # Gauss-Legendre in cos(theta) x uniform in phi: exact for these low-degree polynomials
    ct, wt = np.polynomial.legendre.leggauss(8)
    ph = np.arange(16) * 2 * np.pi / 16
    st = np.sqrt(1 - ct ** 2)
    d = np.stack([np.outer(st, np.cos(ph)).ravel(), np.outer(st, np.sin(ph)).ravel(),
                  np.outer(ct, np.ones(16)).ravel()], axis=1)
    w = np.outer(wt, np.full(16, 2 * np.pi / 16)).ravel()
    lm = [(0, 0)] + [(1, m) for m in (-1, 0, 1)] + [(2, m) for m in range(-2, 3)]
    Y = np.array([paw.solid_harmonic(l, m, d) for l, m in lm])     # r = 1
    G = (Y * w) @ Y.T
    assert np.allclose(G, np.eye(9), atol=1e-13)


def test_projector_amplitudes_unit_norm():
    l, m, sg, amp = projector_table(13, 3.0)
    assert list(l) == [0, 0, 1, 1, 1, 1, 1, 1, 2, 2, 2, 2, 2]
    for al in range(13):
        f = lambda r: (amp[al] * r ** l[al] * math.exp(-r * r / (2 * sg[al] ** 2)) * (1 - (r / 3.0) ** 2) ** 2) ** 2 * r * r
        assert abs(si.quad(f, 0, 3.0, epsabs=1e-14)[0] - 1.0) < 1e-10


def _centered_system():
    """config-0 mesh, Dirichlet storage (no wrap), one atom well inside the box -> moments are unambiguous."""
    cfg = dataclasses.replace(get_config(0), bc="dirichlet", natoms=1, nproj=9, wall_margin=6.0,
                              ncells=(5, 5, 5), box=(15.0, 15.0, 15.0))
    sysd = make_system(cfg)
    return cfg, sysd


def test_projector_integrals_partition_of_unity_and_moments():
    """sum_J C_J,alpha = int p_alpha (closed radial form for s, 0 for l>0), and first/second moments
    sum_J C_J,alpha x_J = int p_alpha x  pin the (l, m) -> axis mapping and the node ordering."""
    cfg, sysd = _centered_system()
    mesh = fe.Mesh(cfg.ncells, cfg.box, cfg.p, "periodic")   # periodic storage: no rows masked
    # the sphere stays inside cells 1..3 per direction, so no basis function that sees it wraps
    assert np.all(sysd.pos[0] - sysd.rc >= 3.0) and np.all(sysd.pos[0] + sysd.rc <= 12.0)
    C, pairs = paw.build_C(mesh, sysd)
    C = C.toarray()
    X = mesh.node_coords() - sysd.pos[0]
    # fix the wrapped plane: periodic storage puts node 0 at x=0, fine since atom is interior
    s0 = C.sum(axis=0)
    exact_s = (0.5 / math.sqrt(math.pi)) * 4 * math.pi * _radial(sysd, 0, 2)
    assert abs(s0[0] - exact_s) < 1e-6 * abs(exact_s)      # quadrature error of the C^1 cutoff
    assert np.all(np.abs(s0[1:]) < 1e-5)      # exact 0; what is left is quadrature error
    # p-type: alpha = 1,2,3 <-> m = -1,0,1 <-> y, z, x
    c1 = math.sqrt(3 / (4 * math.pi)) * (4 * math.pi / 3)
    mom = X.T @ C                                            # (3, nproj)
    for al, axis in ((1, 1), (2, 2), (3, 0)):
        exact = c1 * _radial(sysd, al, 4)
        assert abs(mom[axis, al] - exact) < 1e-5 * abs(exact)
        for other in range(3):
            if other != axis:
                assert abs(mom[other, al]) < 1e-5
    # d-type second moments: m=-2 <-> xy, m=-1 <-> yz, m=1 <-> xz
    c2 = math.sqrt(15 / (4 * math.pi)) * (4 * math.pi / 15)
    for al, (i, j) in ((4, (0, 1)), (5, (1, 2)), (7, (0, 2))):
        got = (X[:, i] * X[:, j]) @ C[:, al]
        exact = c2 * _radial(sysd, al, 6)
        assert abs(got - exact) < 1e-5 * abs(exact)
    # m=0: int p (3z^2 - r^2), m=2: int p (x^2 - y^2)
    got = (3 * X[:, 2] ** 2 - np.sum(X * X, axis=1)) @ C[:, 6]
    exact = math.sqrt(5 / (16 * math.pi)) * (16 * math.pi / 5) * _radial(sysd, 6, 6)
    assert abs(got - exact) < 1e-5 * abs(exact)
    got = (X[:, 0] ** 2 - X[:, 1] ** 2) @ C[:, 8]
    exact = 0.5 * math.sqrt(15 / (4 * math.pi)) * (16 * math.pi / 15) * _radial(sysd, 8, 6)
    assert abs(got - exact) < 1e-5 * abs(exact)


def test_projector_periodic_wrap_matches_unwrapped():
    """Translating the atom across the periodic boundary only permutes rows of C (translation by whole
    cells is a symmetry of the uniform periodic mesh)."""
    cfg = dataclasses.replace(get_config(0), natoms=1)
    sysd = make_system(cfg)
    mesh = fe.Mesh(cfg.ncells, cfg.box, cfg.p, cfg.bc)
    sysd.pos[0] = np.array([3.9, 1.0, 6.5])
    C1, _ = paw.build_C(mesh, sysd)
    sysd2 = dataclasses.replace(sysd, pos=sysd.pos + np.array([4.0, 0.0, 4.0]))   # one cell in x and z
    sysd2.pos[0] %= np.array(cfg.box)
    C2, _ = paw.build_C(mesh, sysd2)
    N = mesh.N
    idx = np.arange(mesh.M).reshape(N)
    perm = np.roll(np.roll(idx, -cfg.p, axis=0), -cfg.p, axis=2).reshape(-1)   # row J of C2 = row perm of C1
    A1 = C1.toarray()
    A2 = C2.toarray()
    assert np.abs(A2[idx.reshape(-1)] - A1[perm]).max() < 1e-13
    assert np.abs(A1).max() > 1e-3


def test_complex_projector_phase():
    """C(k) entries carry e^{-ik.x}: for a smooth plane wave u = e^{iGx}, C^dagger u ~ int p e^{i(k+G).x}
    whose s-channel value is the radial Fourier (sinc) transform -- pins the sign and origin of the phase."""
    cfg = dataclasses.replace(get_config(0), natoms=1, kfrac=(0.25, 0.0, 0.0), p=6)
    sysd = make_system(cfg)
    sysd.pos[0] = np.array([7.5, 4.0, 4.0])        # sphere wraps across x = L
    mesh = fe.Mesh(cfg.ncells, cfg.box, cfg.p, cfg.bc)
    kpt = cfg.kpoint
    C, _ = paw.build_C(mesh, sysd, kpt)
    X = mesh.node_coords()
    G = 2 * np.pi / cfg.box[0] * np.array([1.0, 0, 0])
    u = np.exp(1j * X @ G)                          # periodic part
    got = (C.conj().T @ u)[0]
    q = np.linalg.norm(kpt + G)
    s, amp, rc = sysd.proj_sigma[0], sysd.proj_amp[0], sysd.rc
    f = lambda r: amp * math.exp(-r * r / (2 * s * s)) * (1 - (r / rc) ** 2) ** 2 * r * r * (math.sin(q * r) / (q * r))
    radial = si.quad(f, 0, rc, epsabs=1e-14)[0]
    exact = (0.5 / math.sqrt(math.pi)) * 4 * math.pi * radial * np.exp(1j * (kpt + G) @ sysd.pos[0])
    assert abs(got - exact) < 2e-5 * abs(exact)     # FE interpolation error of the plane wave (p=6, h=4)


def test_sinv_is_exact_woodbury_inverse_single_atom():
    """For one atom, Eq. 28-29 is exactly (M_D + C dS C^T)^-1 (pin C3.7)."""
    cfg = dataclasses.replace(get_config(0), natoms=1)
    sysd = make_system(cfg)
    ops = PawOperators(sysd)
    rng = np.random.default_rng(3)
    X = rng.standard_normal((ops.mesh.M, 4))
    Shat = sp.diags(ops.md) + ops.C @ ops.dSbig @ ops.Ch
    err = np.linalg.norm(ops.apply_Sinv(Shat @ X) - X) / np.linalg.norm(X)
    assert err < 1e-13
    err = np.linalg.norm(Shat @ ops.apply_Sinv(X) - X) / np.linalg.norm(X)
    assert err < 1e-13


def test_sinv_two_atoms_drops_cross_blocks(cfg0_ops):
    """With two atoms the inverse is exact only up to the dropped cross blocks (approximation (ii))."""
    ops = cfg0_ops
    rng = np.random.default_rng(4)
    X = rng.standard_normal((ops.mesh.M, 4))
    Shat = sp.diags(ops.md) + ops.C @ ops.dSbig @ ops.Ch
    err = np.linalg.norm(ops.apply_Sinv(Shat @ X) - X) / np.linalg.norm(X)
    npj = ops.dS.shape[1]
    cross = (ops.Ch[:npj] @ sp.diags(ops.md_inv) @ ops.C[:, npj:]).toarray()
    assert err < 10 * np.abs(cross).max() + 1e-13
    # symmetric operator
    A = ops.apply_Sinv(np.eye(ops.mesh.M))
    assert np.abs(A - A.T).max() < 1e-13
    assert np.linalg.eigvalsh(0.5 * (A + A.T))[0] > 0
