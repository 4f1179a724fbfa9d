"""Harness around the filter: the steps of Algorithm 1 that are NOT on the hot path
this library builds -- S-orthonormalisation, Rayleigh-Ritz (steps 4-6), residual norms (L290).  The tall products run in
the library (RR-Projection pawfe_rr_project, subspace rotation pawfe_rr_rotate, the H / S / S^-1approx applications, the
Lanczos bound); only the small dense B x B algebra (Cholesky, eigh: RR-GHEP, a library call in the paper too) is torch.  They exist so that tests and bench.py can drive the filter with the
inputs Algorithm 2 expects (an S-orthonormal Ritz block, its Ritz values, [b0, bW, bU]).
section 8(f) lists moving them into the library as NEXT-1 / NEXT-2.
"""
from __future__ import annotations

import numpy as np
import torch

from .binding import Context, FP64


def _as_complex(t: torch.Tensor, cplx: bool) -> torch.Tensor:
    return torch.view_as_complex(t) if cplx else t


class Harness:
    """FP64 helper operations on blocks stored in the library's layout ([M, B] or [M, B, 2])."""

    def __init__(self, ctx: Context, M: int, cplx: bool, mixed_rotation: bool = False):
        """mixed_rotation: the paper's mixed-precision subspace rotation (FP64 diagonal / FP32 off-diagonal blocks, L406-L408)"""
        self.ctx, self.M, self.cplx, self.mixed = ctx, M, cplx, mixed_rotation

    def _empty_like(self, X):
        return torch.empty_like(X)

    def apply(self, which: str, X: torch.Tensor) -> torch.Tensor:
        B = X.shape[1]
        Y = torch.empty_like(X)
        getattr(self.ctx, "apply_" + which)(FP64, X, Y, B, B)
        return Y

    def gram(self, X: torch.Tensor, Y: torch.Tensor) -> torch.Tensor:
        """X^dagger Y (B x B), FP64, for Y = H X or S X (Hermitian result): pawfe_rr_project."""
        B = X.shape[1]
        X, Y = X.contiguous(), Y.contiguous()
        G = torch.empty((B, B, 2) if self.cplx else (B, B), dtype=torch.float64, device=X.device)
        self.ctx.rr_project(X, Y, B, B, G)
        return _as_complex(G, self.cplx)

    def rotate(self, X: torch.Tensor, Q: torch.Tensor) -> torch.Tensor:
        """X Q: pawfe_rr_rotate (mixed precision if the harness was created with mixed_rotation)."""
        B = X.shape[1]
        X = X.contiguous()
        Qd = (torch.view_as_real(Q.to(torch.complex128).resolve_conj().contiguous()) if self.cplx else Q.to(torch.float64)).contiguous()
        out = torch.empty_like(X)
        self.ctx.rr_rotate(self.mixed, X, B, Qd, out, B, B)
        return out

    def s_orthonormalise(self, X: torch.Tensor) -> torch.Tensor:
        G = self.gram(X, self.apply("S", X))
        G = 0.5 * (G + G.conj().T)
        L = torch.linalg.cholesky(G)
        Linv_h = torch.linalg.inv(L).conj().T
        return self.rotate(X, Linv_h)

    def rayleigh_ritz(self, X: torch.Tensor):
        """H^p Q = S^p Q Lambda with H^p = X^dagger H X, S^p = X^dagger S X; X <- X Q (Alg. 1 steps 4-6)."""
        Hp = self.gram(X, self.apply("H", X))
        Sp = self.gram(X, self.apply("S", X))
        Hp = 0.5 * (Hp + Hp.conj().T)
        Sp = 0.5 * (Sp + Sp.conj().T)
        L = torch.linalg.cholesky(Sp)
        Li = torch.linalg.inv(L)
        A = Li @ Hp @ Li.conj().T
        lam, U = torch.linalg.eigh(0.5 * (A + A.conj().T))
        Q = Li.conj().T @ U
        return self.rotate(X, Q), lam.cpu().numpy()

    def residual_norms(self, X: torch.Tensor, lam: np.ndarray) -> np.ndarray:
        B = X.shape[1]
        HX, SX = self.apply("H", X), self.apply("S", X)
        l = torch.from_numpy(np.asarray(lam, dtype=np.float64)).to(X.device)
        R = HX - SX * (l[None, :, None] if self.cplx else l[None, :])
        out = torch.zeros(B, dtype=torch.float64, device=X.device)
        self.ctx.col_norms(FP64, R.contiguous(), B, B, out)
        return out.cpu().numpy()

    def upper_bound(self, k: int = 10, seed: int = 0) -> float:
        """b_U for the iterated operator H S^-1approx: k-step Lanczos in the S^-1approx inner product,
        b_U = 1.02 (theta_max + beta_k) (reading R17), inside the library (pawfe_lanczos_bound); only the
        seeded start vector is drawn here."""
        g = torch.Generator(device="cpu").manual_seed(seed)
        shape = (self.M, 1, 2) if self.cplx else (self.M, 1)
        v = torch.randn(shape, dtype=torch.float64, generator=g).cuda()
        return self.ctx.lanczos_bound(k, v)[0]


def cast_block(X64: torch.Tensor, prec: int) -> torch.Tensor:
    return X64 if prec == FP64 else X64.to(torch.float32)


def chfsi_loop(ctx: Context, hz: Harness, X0: torch.Tensor, prec: int, m: int, bU: float, outer: int,
               block: int | None = None, history=None):
    """Algorithm 1 repeated `outer` times with the library's filter (reading R16: b0 = lowest, bW = highest
    Ritz value of the previous Rayleigh-Ritz).  X0: FP64 block in library layout.  Returns (X, lam)."""
    X = hz.s_orthonormalise(X0)
    X, lam = hz.rayleigh_ritz(X)
    N = X.shape[1]
    B = block or N
    nbytes = ctx.filter_workspace(prec, B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device=X.device)
    for _ in range(outer):
        b0, bW = float(lam[0]), float(lam[-1])
        Xf = torch.empty_like(X)
        for s in range(0, N, B):
            w = min(B, N - s)
            blk = cast_block(X[:, s:s + w].contiguous(), prec)
            ctx.cheb_filter(prec, m, b0, bW, bU, blk, lam[s:s + w], w, w, ws, nbytes)
            Xf[:, s:s + w] = blk.to(torch.float64)
        X, lam = hz.rayleigh_ritz(Xf)
        if history is not None:
            history.append(lam.copy())
    return X, lam
