"""Helpers shared by the round-2 GPU parity tests (tests/test_gpu_parity_r2.py, tests/test_gpu_fullsize_r2.py).

Error measures (a relative Frobenius norm alone cannot see one wrong row in 10^5):
  relerr(a, b)      ||a - b||_F / ||b||_F                                  the north_star's per-product measure
  rowerr(a, b)      max_J ||a_J - b_J||_2 / (||b||_F / sqrt(rows))          a single bad row of RMS size gives O(1)
"""
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from pawfe_inputs import get_config, make_system, random_block, twin  # noqa: E402,F401

TOL = {"fp64": 1e-12, "fp32": 1e-5, "tf32": 5e-3}
# per-row bound: a row's error may exceed the block's RMS error by the tail of its distribution over ~1e5 rows
ROW_FACTOR = 6.0


def need_gpu():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")


def to_dev(x, prec, cplx):
    """numpy (M, B) real/complex -> torch CUDA tensor in the library's element layout."""
    real = np.float64 if prec == "fp64" else np.float32
    a = np.stack([x.real, x.imag], axis=-1).astype(real) if cplx else x.astype(real)
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def to_host(t, cplx):
    a = t.cpu().numpy().astype(np.float64)
    return a[..., 0] + 1j * a[..., 1] if cplx else a


def relerr(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def rowerr(a, b):
    rms = np.linalg.norm(b) / np.sqrt(b.shape[0])
    return float(np.max(np.linalg.norm(a - b, axis=1)) / rms)


def check(got, want, tol, what):
    e, r = relerr(got, want), rowerr(got, want)
    rep = os.environ.get("PAWFE_TEST_REPORT")          # optional log of the measured errors (profiles/r02_parity_margins.md)
    if rep:
        with open(rep, "a") as f:
            f.write(f"{what}\trelerr={e:.3e}\trowerr={r:.3e}\ttol={tol:.1e}\n")
    assert e < tol, (what, "relerr", e)
    assert r < ROW_FACTOR * tol, (what, "rowerr", r)
    return e


def bounds(ops, lam):
    from oracle.chfsi import lanczos_upper_bound
    bU = lanczos_upper_bound(ops.apply_H, ops.apply_Sinv, ops.mesh.M, k=10, seed=1, dtype=ops.dtype, mask=ops.mask)
    return lam[0] - 0.1, lam[-1] + 0.05, bU


def ritz_block(ops, cfg, B, stream):
    """S-orthonormal Ritz block and Ritz values of a seeded random block (what Algorithm 2 expects as input)."""
    from oracle import chfsi
    X0 = random_block(cfg, B, stream=stream) * ops.mask[:, None]
    X = chfsi.s_orthonormalise(ops.apply_S, X0)
    return chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, X)


def run_filter(ctx, prec, m, b0, bW, bU, Xd, lam, B, ld=None):
    from paper_2604_26037_b200 import PREC
    ld = ld or B
    nbytes = ctx.filter_workspace(PREC[prec], B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.cheb_filter(PREC[prec], m, b0, bW, bU, Xd, lam, ld, B, ws, nbytes)
    torch.cuda.synchronize()
    return Xd


def run_filter_hs(ctx, prec, m, b0, bW, bU, Xd, HX, SX, lam, B, ld=None):
    """pawfe_cheb_filter_hs: step 2 from the given FP64 products (no operator application, no FP64 atomics)"""
    from paper_2604_26037_b200 import PREC
    ld = ld or B
    nbytes = ctx.filter_workspace(PREC[prec], B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.cheb_filter_hs(PREC[prec], m, b0, bW, bU, Xd, HX, SX, lam, ld, B, ws, nbytes)
    torch.cuda.synchronize()
    return Xd


def fp64_products(ctx, Xd, ld, B):
    """H X and S X of an FP32-stored device block in FP64 with the library's own applies (what a Rayleigh-Ritz step holds)"""
    from paper_2604_26037_b200 import FP64
    X64 = Xd.double().contiguous()
    HX, SX = torch.zeros_like(X64), torch.zeros_like(X64)
    ctx.apply_H(FP64, X64, HX, ld, B)
    ctx.apply_S(FP64, X64, SX, ld, B)
    torch.cuda.synchronize()
    return HX, SX


class DeviceRows:
    """Row source for oracle.operators.apply_*_rows: X[J] fetches the rows J of a device block as float64 / complex128."""

    def __init__(self, t, cplx):
        self.t, self.cplx = t, cplx
        self.shape = (t.shape[0], t.shape[1])

    def __getitem__(self, J):
        idx = torch.from_numpy(np.ascontiguousarray(np.asarray(J, dtype=np.int64))).cuda()
        return to_host(self.t[idx], self.cplx)
