"""BASELINE.json configs 2, 3 and 4 at FULL size (4.74M / 1.73M / 7.19M dofs), in the launch configuration bench.py times
(TF32, the config's block width, CTA-pair kernel, 27+ tiles per persistent CTA), against the oracle on sampled rows:

  * H X and H S^-1approx X on all nodes of sampled cells -- the first and the last cell of the launch order, a wall cell
    (config 4), cells that hold atoms -- by oracle.operators.apply_HSinv_rows (Eq. 13, 16, 28-29 evaluated row by row).
    H S^-1approx X runs exactly the kernel sequence of one Chebyshev step (projection, couplings, fused cell kernel with both
    halves of the K-extension), so the low-rank correction inside the fused step is checked at scale.
  * a property of the whole filter call that holds at any size: with H Psi = S Psi Lambda handed in (pawfe_cheb_filter_hs)
    the residual vanishes and Algorithm 2 returns Psi C_m(Lambda) exactly (fixed point), where
    C_m is the scaled Chebyshev polynomial of Eq. 19 -- a closed form for every one of the 10^9 output elements.

Inputs are generated on the device (seeded torch.Generator, U[-0.5, 0.5]); only the sampled rows travel to the host.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from gpu_helpers import TOL, DeviceRows, need_gpu, relerr, rowerr, to_host  # noqa: E402
from pawfe_inputs import get_config, make_system  # noqa: E402


def _prefill_blocks(sysd, cells):
    """the oracle's projector blocks (paw.atom_cell_block via operators.atom_pair_blocks) of every atom that can matter for
    the sampled cells, evaluated by worker processes on the host cores: the same oracle code, only run in parallel"""
    import multiprocessing as mp
    import os
    from oracle.operators import atom_pair_blocks, atoms_near_cells
    h = sysd.cfg.box[0] / sysd.cfg.ncells[0]
    atoms = atoms_near_cells(sysd, cells, 3.0 * sysd.rc + 5.0 * h)        # superset of what apply_HSinv_rows asks for
    nproc = max(1, min(12, len(os.sched_getaffinity(0)) - 1, len(atoms)))
    with mp.get_context("spawn").Pool(nproc) as pool:
        blocks = pool.starmap(atom_pair_blocks, [(sysd, a) for a in atoms])
    return {"blocks": dict(zip(atoms, blocks))}


def _sample_cells(cfg, sysd, k_atoms):
    nc = cfg.ncells[0]
    h = cfg.box[0] / nc
    cells = [(0, 0, 0), (nc - 1, nc - 1, nc - 1)]       # first and last cell of the launch order (periodic: both wrap)
    if cfg.bc == "dirichlet":
        cells.append((nc // 2, 0, nc - 1))              # a wall cell away from the corners
    for a in range(k_atoms):                            # cells that contain an atom: strongest non-local weight
        cells.append(tuple(int(min(nc - 1, max(0, np.floor(sysd.pos[a][d] / h)))) for d in range(3)))
    out = []
    for c in cells:
        if c not in out:
            out.append(c)
    return out


@pytest.mark.parametrize("cid,k_atoms", [(3, 1), (2, 1), (4, 1)])
def test_full_size_sampled_rows_H_and_HSinv(cid, k_atoms):
    need_gpu()
    from oracle.operators import apply_HSinv_rows
    from paper_2604_26037_b200 import TF32, context_from_system
    cfg = get_config(cid)
    sysd = make_system(cfg)
    ctx = context_from_system(sysd, device=0, stream=torch.cuda.current_stream().cuda_stream)
    try:
        M, B = ctx.num_dofs(), cfg.block - cfg.block % 4        # 248 of config 2's 250 columns: the tensor-core applies take multiples of 4
        cplx = cfg.complex
        gen = torch.Generator(device="cuda").manual_seed(cfg.seed + 7)
        shape = (M, B, 2) if cplx else (M, B)
        X = torch.rand(shape, dtype=torch.float32, device="cuda", generator=gen) - 0.5
        Y = torch.empty_like(X)
        src = DeviceRows(X, cplx)
        cells = _sample_cells(cfg, sysd, k_atoms)
        cache = _prefill_blocks(sysd, cells)             # projector blocks and cell matrices are shared by the two operators
        assert ctx.cell_kernel_name(TF32, B) == "tcgen05_tf32"
        for op, fn in (("H", ctx.apply_H), ("HSinv", ctx.apply_HSinv)):
            Y.fill_(float("nan"))
            fn(TF32, X, Y, B, B)
            torch.cuda.synchronize()
            want = apply_HSinv_rows(sysd, src, cells, op=op, cache=cache)
            for (J, ref), c in zip(want, cells):
                got = DeviceRows(Y, cplx)[J]
                assert np.all(np.isfinite(got)), (cid, op, c)
                if np.linalg.norm(ref) == 0.0:           # (cannot happen for interior cells; wall rows are zero inside ref)
                    assert np.linalg.norm(got) == 0.0
                    continue
                e, r = relerr(got, ref), rowerr(got, ref)
                assert e < TOL["tf32"], (cid, op, c, e)
                live = np.linalg.norm(ref, axis=1) > 0    # Dirichlet wall rows: written as exact zeros
                assert np.all(got[~live] == 0.0), (cid, op, c)
                assert r < 6 * TOL["tf32"], (cid, op, c, r)
    finally:
        ctx.destroy()


def _scaled_chebyshev(x, m, b0, bW, bU):
    """C_m(x) = T_m((x - c)/e) / T_m((b0 - c)/e), closed form (|t| >= 1: cosh, else cos); Eq. 19, PAPER.md:L164-L172"""
    e, c = 0.5 * (bU - bW), 0.5 * (bU + bW)

    def T(t):
        t = np.asarray(t, dtype=float)
        out = np.empty_like(t)
        big = np.abs(t) >= 1.0
        out[big] = np.sign(t[big]) ** m * np.cosh(m * np.arccosh(np.abs(t[big])))
        out[~big] = np.cos(m * np.arccos(t[~big]))
        return out
    return T((np.asarray(x) - c) / e) / T(np.array([(b0 - c) / e]))[0]


@pytest.mark.parametrize("cid", [4, 3])
def test_full_size_filter_fixed_point(cid):
    """H Psi = S Psi Lambda given => Y = 0 => Psi_f = Psi C_m(Lambda) (Lambda recurrence of Alg. 2 steps 3-4 + recovery, in the
    bench's launch configuration; the cell kernel runs on an all-zero residual and must leave it zero)."""
    need_gpu()
    from paper_2604_26037_b200 import TF32, context_from_system
    cfg = get_config(cid)
    sysd = make_system(cfg)
    ctx = context_from_system(sysd, device=0, stream=torch.cuda.current_stream().cuda_stream)
    try:
        M, B, m = ctx.num_dofs(), cfg.block, 8
        cplx = cfg.complex
        gen = torch.Generator(device="cuda").manual_seed(cfg.seed + 8)
        shape = (M, B, 2) if cplx else (M, B)
        X = torch.rand(shape, dtype=torch.float32, device="cuda", generator=gen) - 0.5
        lam = np.linspace(-0.4, 2.5, B)
        b0, bW, bU = -0.5, 2.6, 340.0
        lam_t = torch.from_numpy(lam).cuda()
        SX = torch.rand(shape, dtype=torch.float64, device="cuda", generator=gen) - 0.5        # any block: only HX - SX Lambda matters
        HX = SX * (lam_t[None, :, None] if cplx else lam_t[None, :])
        nbytes = ctx.filter_workspace(TF32, B)
        ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        X0 = X.clone()
        ctx.cheb_filter_hs(TF32, m, b0, bW, bU, X, HX, SX, lam, B, B, ws, nbytes)
        torch.cuda.synchronize()
        del HX, SX, ws
        gain = torch.from_numpy(_scaled_chebyshev(lam, m, b0, bW, bU)).cuda()
        # free dofs: rows where S^-1approx does not vanish; Dirichlet wall rows are written as 0
        one = torch.ones((M, 4, 2) if cplx else (M, 4), dtype=torch.float32, device="cuda")
        msk = torch.empty_like(one)
        ctx.apply_Sinv(TF32, one, msk, 4, 4)
        torch.cuda.synchronize()
        free = (msk.reshape(M, -1).abs().sum(dim=1) > 0)
        want = X0.double() * (gain[None, :, None] if cplx else gain[None, :]) * (free[:, None, None] if cplx else free[:, None])
        err = float((X.double() - want).norm() / want.norm())
        worst = float((X.double() - want).abs().max() / want.abs().max())
        assert err < 2e-7 and worst < 1e-6, (cid, err, worst)                                  # one FP32 rounding of the product
        if cfg.bc == "dirichlet":
            assert int((~free).sum()) == M - 191 ** 3
            assert float(X[~free].abs().max()) == 0.0
    finally:
        ctx.destroy()
