"""R-ChFSI: Algorithm 2 (the filter), Algorithm 1 (outer loop), bounds, brute force (TEST INFRASTRUCTURE).

Everything in FP64, written line by line in the paper's order and notation.
"""
from __future__ import annotations

import numpy as np
import scipy.linalg as sla


def cheb_coefficients(b0, bW, bU):
    """Alg. 2 step 1: e, c, zeta = e/(b0 - c), gamma = 2/zeta  (readings R2, R4)."""
    e = 0.5 * (bU - bW)
    c = 0.5 * (bU + bW)
    zeta = e / (b0 - c)
    gamma = 2.0 / zeta
    return e, c, zeta, gamma


def filter_residual(apply_H, apply_S, apply_Sinv, X, lam, m, b0, bW, bU):
    """Algorithm 2: residual-based Chebyshev filtered block.

    X: (M, B) block Psi_in, lam: (B,) estimates Lambda_in.  Returns Psi_f (M, B).
    """
    lam = np.asarray(lam, dtype=float)
    e, c, zeta, gamma = cheb_coefficients(b0, bW, bU)                 # step 1
    zeta1 = zeta
    Y = apply_H(X) - apply_S(X) * lam[None, :]                        # step 2
    RX = np.zeros_like(Y)                                             # step 3
    RY = (zeta1 / e) * Y
    LX = np.ones_like(lam)
    LY = (zeta1 / e) * (lam - c)
    for _theta in range(2, m + 1):                                    # step 4
        zeta1 = 1.0 / (gamma - zeta)
        a = 2.0 * zeta1 / e
        RX = a * apply_H(apply_Sinv(RY)) - a * c * RY - zeta * zeta1 * RX + a * Y * LY[None, :]
        LX = a * LY * lam - a * c * LY - zeta * zeta1 * LX
        RX, RY = RY, RX
        LX, LY = LY, LX
        zeta = zeta1
    return apply_Sinv(RY) + X * LY[None, :]                           # step 5


def filter_plain(apply_SinvH, X, m, b0, bW, bU):
    """Plain scaled Chebyshev filter on S^-1 H, Eq. 19-20:
    X_0 = Psi, X_1 = (zeta_1/e)(S^-1 H - c I) Psi,
    X_{t+1} = (2 zeta_{t+1}/e) S^-1 H X_t - (2 zeta_{t+1} c/e) X_t - zeta_t zeta_{t+1} X_{t-1},
    zeta_{t+1} = 1/(2/zeta_1 - zeta_t).  Used only to pin Alg. 2 ("mathematically equivalent", L217)."""
    e, c, zeta1, gamma = cheb_coefficients(b0, bW, bU)
    Xp = X
    Xc = (zeta1 / e) * (apply_SinvH(X) - c * X)
    zeta = zeta1
    for _t in range(2, m + 1):
        zn = 1.0 / (gamma - zeta)
        Xn = (2.0 * zn / e) * apply_SinvH(Xc) - (2.0 * zn * c / e) * Xc - zeta * zn * Xp
        Xp, Xc = Xc, Xn
        zeta = zn
    return Xc


def scaled_chebyshev(x, m, b0, bW, bU):
    """C_m(x~, b0~) = T_m((x-c)/e) / T_m((b0-c)/e) for scalars (Eq. 19), by the scalar recurrence."""
    e, c, _, _ = cheb_coefficients(b0, bW, bU)

    def T(t):
        t = np.asarray(t, dtype=float)
        tp, tc = np.ones_like(t), t.copy()
        if m == 0:
            return tp
        for _ in range(2, m + 1):
            tp, tc = tc, 2.0 * t * tc - tp
        return tc
    return T((np.asarray(x) - c) / e) / T((b0 - c) / e)


def lanczos_upper_bound(apply_H, apply_Sinv, M, k=10, seed=0, dtype=float, mask=None, v0=None):
    """Upper bound b_U of the spectrum of the iterated operator H S^-1approx (same spectrum as
    S^-1approx H; Alg. 1 steps 1-2; reading R17).  k-step Lanczos in the
    S^-1approx inner product <x,y> = x^dagger S^-1approx y, in which H S^-1approx is self-adjoint;
    b_U = 1.02 * (theta_max + beta_k).  v0: optional start vector (default: seeded standard normal)."""
    if v0 is None:
        rng = np.random.default_rng(seed)
        v = rng.standard_normal((M, 1)).astype(dtype)
    else:                                   # start vector given (the random numbers the method draws are passed in)
        v = np.array(v0, dtype=dtype).reshape(M, 1)
    if mask is not None:
        v = v * mask[:, None]
    ip = lambda x, y: np.real(np.vdot(x, apply_Sinv(y)))
    v = v / np.sqrt(ip(v, v))
    vprev = np.zeros_like(v)
    beta = 0.0
    alphas, betas = [], []
    for _ in range(k):
        w = apply_H(apply_Sinv(v)) - beta * vprev
        alpha = ip(v, w)
        w = w - alpha * v
        beta = np.sqrt(max(ip(w, w), 0.0))
        alphas.append(alpha)
        betas.append(beta)
        if beta < 1e-14:
            break
        vprev, v = v, w / beta
    T = np.diag(alphas) + np.diag(betas[:-1], 1) + np.diag(betas[:-1], -1)
    theta = np.linalg.eigvalsh(T)
    return 1.02 * (theta[-1] + betas[-1])


def s_orthonormalise(apply_S, X):
    """X <- X L^-dagger with L L^dagger = X^dagger S X."""
    G = X.conj().T @ apply_S(X)
    L = np.linalg.cholesky(0.5 * (G + G.conj().T))
    return np.linalg.solve(L, X.conj().T).conj().T


def rayleigh_ritz(apply_H, apply_S, X):
    """Alg. 1 steps 4-6: H^p = X^dagger H X, S^p = X^dagger S X,
    H^p Q = S^p Q Lambda, X <- X Q."""
    HX = apply_H(X)
    SX = apply_S(X)
    Hp = X.conj().T @ HX
    Sp = X.conj().T @ SX
    Hp = 0.5 * (Hp + Hp.conj().T)
    Sp = 0.5 * (Sp + Sp.conj().T)
    lam, Q = sla.eigh(Hp, Sp)
    return X @ Q, lam


def residual_norms(apply_H, apply_S, X, lam):
    """|| H x_i - lambda_i S x_i ||_2 per column."""
    R = apply_H(X) - apply_S(X) * lam[None, :]
    return np.sqrt(np.sum(np.abs(R) ** 2, axis=0))


def chfsi_loop(apply_H, apply_S, apply_Sinv, X0, m, bU, outer, block=None, history=None):
    """Algorithm 1 repeated `outer` times (reading R16: b0 = lowest, bW = highest Ritz value of the
    previous Rayleigh-Ritz; initial (Psi, Lambda) from a Rayleigh-Ritz on the S-orthonormalised block)."""
    X = s_orthonormalise(apply_S, X0)
    X, lam = rayleigh_ritz(apply_H, apply_S, X)
    B = block or X.shape[1]
    for _it in range(outer):
        b0, bW = lam[0], lam[-1]
        Xf = np.empty_like(X)
        for s in range(0, X.shape[1], B):
            Xf[:, s:s + B] = filter_residual(apply_H, apply_S, apply_Sinv, X[:, s:s + B], lam[s:s + B],
                                             m, b0, bW, bU)
        X, lam = rayleigh_ritz(apply_H, apply_S, Xf)
        if history is not None:
            history.append(lam.copy())
    return X, lam


def dense_eigh(H, S, free=None):
    """Brute force: lowest eigenvalues of the dense pencil (H, S) on the free dofs."""
    if free is not None:
        H = H[np.ix_(free, free)]
        S = S[np.ix_(free, free)]
    return sla.eigh(0.5 * (H + H.conj().T), 0.5 * (S + S.conj().T), eigvals_only=True)
