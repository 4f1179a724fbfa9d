"""Pins of Alg. 2 / Alg. 1 in the oracle."""
import numpy as np
import scipy.linalg as sla
import scipy.sparse as sp
import scipy.sparse.linalg as spla

from oracle import chfsi
from pawfe_inputs import random_block


def _bounds(ops):
    H, S = ops.dense_H(), ops.dense_S()
    lam = sla.eigh(H, S, eigvals_only=True)
    return H, S, lam


def test_residual_filter_equals_plain_filter_with_exact_inverse(cfg0_ops):
    """Alg. 2 with the EXACT S^-1 is "mathematically equivalent" to Eq. 19-20."""
    ops = cfg0_ops
    H, S, lam = _bounds(ops)
    Sinv = np.linalg.inv(S)
    X = chfsi.s_orthonormalise(ops.apply_S, random_block(ops.cfg, 6))
    X, rv = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, X)
    m, b0, bW, bU = 10, lam[0] - 0.1, lam[40], lam[-1] * 1.01
    Y1 = chfsi.filter_residual(ops.apply_H, ops.apply_S, lambda R: Sinv @ R, X, rv, m, b0, bW, bU)
    Y2 = chfsi.filter_plain(lambda V: Sinv @ (H @ V), X, m, b0, bW, bU)
    assert np.linalg.norm(Y1 - Y2) < 1e-11 * np.linalg.norm(Y2)
    # and the result does not depend on the Lambda_in estimates (they cancel exactly)
    Y3 = chfsi.filter_residual(ops.apply_H, ops.apply_S, lambda R: Sinv @ R, X, rv + 0.3, m, b0, bW, bU)
    assert np.linalg.norm(Y3 - Y2) < 1e-10 * np.linalg.norm(Y2)


def test_eigenpair_is_fixed_point_with_chebyshev_gain(cfg0_ops):
    """Exact eigenpair in => Y = 0 => output psi * T_m((lam-c)/e) / T_m((b0-c)/e), with
    T_m(x) = cosh(m acosh|x|) sign(x)^m outside [-1,1]; holds for the APPROXIMATE inverse too (C3.10)."""
    ops = cfg0_ops
    H, S, lam = _bounds(ops)
    w, V = sla.eigh(H, S)
    m, b0, bW, bU = 9, w[0] - 0.05, w[30], w[-1] * 1.01
    X = V[:, :5]
    out = chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, X, w[:5], m, b0, bW, bU)
    e, c = 0.5 * (bU - bW), 0.5 * (bU + bW)

    def T(x):
        return np.cosh(m * np.arccosh(abs(x))) * np.sign(x) ** m
    gain = np.array([T((w[i] - c) / e) / T((b0 - c) / e) for i in range(5)])
    assert np.linalg.norm(out - X * gain[None, :]) < 1e-9 * np.linalg.norm(X)
    assert np.allclose(chfsi.scaled_chebyshev(w[:5], m, b0, bW, bU), gain, rtol=1e-11)


def test_filter_degree_one(cfg0_ops):
    """m = 1: loop empty, returns Sinv R_1 + X Lambda_1 (reading R22)."""
    ops = cfg0_ops
    X = random_block(ops.cfg, 3)
    lam = np.array([0.1, 0.2, 0.3])
    b0, bW, bU = -1.0, 1.0, 20.0
    out = chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, X, lam, 1, b0, bW, bU)
    e, c = 0.5 * (bU - bW), 0.5 * (bU + bW)
    z = e / (b0 - c)
    ref = ops.apply_Sinv((z / e) * (ops.apply_H(X) - ops.apply_S(X) * lam)) + X * ((z / e) * (lam - c))
    assert np.linalg.norm(out - ref) < 1e-13 * np.linalg.norm(ref)


def test_lanczos_bound_is_an_upper_bound(cfg0_ops):
    ops = cfg0_ops
    A = ops.apply_Sinv(ops.dense_H())               # S^-1approx H
    true_max = np.max(np.real(np.linalg.eigvals(A)))
    bU = chfsi.lanczos_upper_bound(ops.apply_H, ops.apply_Sinv, ops.mesh.M, k=10, seed=1)
    assert bU >= true_max
    assert bU < 3.0 * true_max
    # the approximate inverse has a smaller top eigenvalue than the exact one (reading R17)
    exact_max = sla.eigh(ops.dense_H(), ops.dense_S(), eigvals_only=True)[-1]
    assert true_max < exact_max


def test_full_loop_matches_dense_eigensolve(cfg0_ops):
    """Alg. 1 on config 0 (degree 10, 30 outer iterations, 16 vectors): lowest 12 Ritz values equal
    the dense generalised eigenvalues (north_star pin; C3.11, reading R18)."""
    ops = cfg0_ops
    cfg = ops.cfg
    H, S, lam = _bounds(ops)
    bU = chfsi.lanczos_upper_bound(ops.apply_H, ops.apply_Sinv, ops.mesh.M, k=10, seed=1)
    X0 = random_block(cfg, cfg.nvec)
    hist = []
    X, rv = chfsi.chfsi_loop(ops.apply_H, ops.apply_S, ops.apply_Sinv, X0, cfg.degree, bU, cfg.outer,
                             history=hist)
    ncheck = (3 * cfg.nvec) // 4
    assert np.max(np.abs(rv[:ncheck] - lam[:ncheck])) < 1e-10
    assert np.max(np.abs(hist[9][:ncheck] - lam[:ncheck])) < 1e-5     # already close after 10
    rn = chfsi.residual_norms(ops.apply_H, ops.apply_S, X, rv)
    assert np.max(rn[:ncheck]) < 1e-7                                  # 1e-7..1e-9
    # S-orthonormal output
    G = X.T @ ops.apply_S(X)
    assert np.abs(G - np.eye(cfg.nvec)).max() < 1e-10
