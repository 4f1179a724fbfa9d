"""GPU parity: libpawfe.so (through the C ABI) against the FP64 CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json's north_star: per product FP64 <= 1e-12, FP32 <= 1e-5,
TF32 <= 5e-3 (relative Frobenius error on the seeded random block); FP64 filter call <= 1e-10.

Cases: BASELINE.json configs[0] (full) and reduced-cell twins of configs 1-4 (same p, h, potential,
projector set, boundary condition and k-point), sized so the oracle finishes in seconds while every
kernel still sees several cells, vector tiles and a ragged tail.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from pawfe_inputs import get_config, make_system, random_block, twin  # noqa: E402

TOL = {"fp64": 1e-12, "fp32": 1e-5, "tf32": 5e-3}


def _cases():
    return {
        "cfg0": get_config(0),
        "cfg1_twin": twin(get_config(1), nc=4, natoms=3, nvec=40, block=40, degree=6),
        "cfg2_twin": twin(get_config(2), nc=4, natoms=3, nvec=24, block=24, degree=5),
        "cfg3_twin": twin(get_config(3), nc=4, natoms=3, nvec=20, block=20, degree=5),
        "cfg4_twin": twin(get_config(4), nc=4, natoms=3, nvec=24, block=24, degree=5),
    }


_CACHE = {}


def _setup(name):
    if name in _CACHE:
        return _CACHE[name]
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from oracle.operators import PawOperators
    from paper_2604_26037_b200 import context_from_system
    cfg = _cases()[name]
    sysd = make_system(cfg)
    ops = PawOperators(sysd)
    ctx = context_from_system(sysd, device=0, stream=torch.cuda.current_stream().cuda_stream)
    _CACHE[name] = (cfg, sysd, ops, ctx)
    return _CACHE[name]


def _to_dev(x, prec, cplx):
    """numpy (M, B) real/complex -> torch CUDA tensor in the library's element layout."""
    real = np.float64 if prec == "fp64" else np.float32
    if cplx:
        a = np.stack([x.real, x.imag], axis=-1).astype(real)
    else:
        a = x.astype(real)
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _to_host(t, cplx):
    a = t.cpu().numpy().astype(np.float64)
    return a[..., 0] + 1j * a[..., 1] if cplx else a


def _relerr(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


CASES = ["cfg0", "cfg1_twin", "cfg2_twin", "cfg3_twin", "cfg4_twin"]


@pytest.mark.parametrize("name", CASES)
def test_cell_matrices_and_couplings(name):
    cfg, sysd, ops, ctx = _setup(name)
    n = ops.mesh.n
    for e in sorted({0, ops.mesh.ncell_total // 2, ops.mesh.ncell_total - 1}):
        He = ops.H_cell(*ops.mesh.cell_coords(e))
        got = ctx.get_cell_matrix(e, n)
        assert _relerr(got, He) < 1e-13, (name, e)
    got = ctx.get_sinv_coupling(cfg.natoms, cfg.nproj)
    assert _relerr(got, ops.dSinv) < 1e-11
    assert ctx.num_pairs() >= len(ops.pairs)


@pytest.mark.parametrize("prec", ["fp64", "fp32", "tf32"])
@pytest.mark.parametrize("name", CASES)
def test_apply_H_S_Sinv(name, prec):
    from paper_2604_26037_b200 import PREC
    cfg, sysd, ops, ctx = _setup(name)
    B = cfg.block
    X = random_block(cfg, B) * ops.mask[:, None]
    Xd = _to_dev(X, prec, cfg.complex)
    Yd = torch.empty_like(Xd)
    for opname, fn, ref in (("H", ctx.apply_H, ops.apply_H), ("S", ctx.apply_S, ops.apply_S),
                            ("Sinv", ctx.apply_Sinv, ops.apply_Sinv)):
        Yd.fill_(float("nan"))
        fn(PREC[prec], Xd, Yd, B, B)
        torch.cuda.synchronize()
        got = _to_host(Yd, cfg.complex)
        want = ref(X) * ops.mask[:, None]
        err = _relerr(got, want)
        tol = TOL[prec] if not (opname != "H" and prec == "tf32") else TOL["fp32"]  # only the H contraction is TF32
        assert err < tol, (name, prec, opname, err)


@pytest.mark.parametrize("name", CASES)
def test_apply_with_padded_ld_and_ignored_boundary(name):
    """ld > B, and garbage in Dirichlet boundary rows of X must not change the result."""
    from paper_2604_26037_b200 import FP64
    cfg, sysd, ops, ctx = _setup(name)
    B, ld = 5, 8
    X = random_block(cfg, B, stream=3)
    want = ops.apply_H(X * ops.mask[:, None]) * ops.mask[:, None]
    Xp = np.zeros((X.shape[0], ld), dtype=X.dtype)
    Xp[:, :B] = X  # boundary rows keep their random values
    Xd = _to_dev(Xp, "fp64", cfg.complex)
    Yd = torch.full_like(Xd, 7.0)
    ctx.apply_H(FP64, Xd, Yd, ld, B)
    torch.cuda.synchronize()
    got = _to_host(Yd, cfg.complex)
    assert _relerr(got[:, :B], want) < 1e-12
    assert np.all(got[:, B:] == 7.0 * (1 + 1j if cfg.complex else 1))


def _bounds(ops, lam):
    from oracle.chfsi import lanczos_upper_bound
    bU = lanczos_upper_bound(ops.apply_H, ops.apply_Sinv, ops.mesh.M, k=10, seed=1, dtype=ops.dtype, mask=ops.mask)
    return lam[0] - 0.1, lam[-1] + 0.05, bU


@pytest.mark.parametrize("prec", ["fp64", "fp32", "tf32"])
@pytest.mark.parametrize("name", CASES)
def test_filter_call(name, prec):
    """One Algorithm-2 call against the oracle's filter_residual on an S-orthonormal Ritz block."""
    from oracle import chfsi
    from paper_2604_26037_b200 import PREC
    cfg, sysd, ops, ctx = _setup(name)
    B, m = cfg.block, cfg.degree
    X0 = random_block(cfg, B, stream=1) * ops.mask[:, None]
    X = chfsi.s_orthonormalise(ops.apply_S, X0)
    X, lam = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, X)
    b0, bW, bU = _bounds(ops, lam)
    want = chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, X, lam, m, b0, bW, bU)
    Xd = _to_dev(X, prec, cfg.complex)
    nbytes = ctx.filter_workspace(PREC[prec], B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.cheb_filter(PREC[prec], m, b0, bW, bU, Xd, lam, B, B, ws, nbytes)
    torch.cuda.synchronize()
    got = _to_host(Xd, cfg.complex)
    err = _relerr(got, want)
    tol = {"fp64": 1e-10, "fp32": 5e-5, "tf32": 1e-2}[prec]
    assert err < tol, (name, prec, err)


def test_col_norms():
    from paper_2604_26037_b200 import FP32, FP64
    cfg, sysd, ops, ctx = _setup("cfg3_twin")
    B = 7
    X = random_block(cfg, B, stream=5)
    want = np.sqrt(np.sum(np.abs(X) ** 2, axis=0))
    for prec, name in ((FP64, "fp64"), (FP32, "fp32")):
        Xd = _to_dev(X, name, cfg.complex)
        out = torch.zeros(B, dtype=torch.float64, device="cuda")
        ctx.col_norms(prec, Xd, B, B, out)
        torch.cuda.synchronize()
        assert np.allclose(out.cpu().numpy(), want, rtol=1e-6 if name == "fp32" else 1e-13)


# ------------------------------------------------------------------------------------------------
# BASELINE.json configs[1] at FULL size, in the launch configuration bench.py times (B = 200, TF32 mode)
# ------------------------------------------------------------------------------------------------
_FULL = {}


def _full_cfg1():
    if "ctx" not in _FULL:
        if not torch.cuda.is_available():
            pytest.skip("no CUDA device")
        from paper_2604_26037_b200 import context_from_system
        cfg = get_config(1)
        sysd = make_system(cfg)
        _FULL["cfg"], _FULL["sys"] = cfg, sysd
        _FULL["ctx"] = context_from_system(sysd, device=0, stream=torch.cuda.current_stream().cuda_stream)
    return _FULL["cfg"], _FULL["sys"], _FULL["ctx"]


def test_full_size_cfg1_H_sampled_rows():
    """H X at 884,736 dofs x 200 vectors (tcgen05 kernel, two vector tiles, K-extension) against the oracle's
    row-by-row evaluation (oracle.operators.apply_H_rows) on the nodes of two sampled cells."""
    from oracle.operators import apply_H_rows
    from paper_2604_26037_b200 import TF32, FP32, FP64
    cfg, sysd, ctx = _full_cfg1()
    B = cfg.block
    X = random_block(cfg, B, stream=11)
    cells = [(0, 0, 0), (7, 15, 3)]          # a corner cell (periodic wrap) and an interior one
    want = apply_H_rows(sysd, X, cells)
    for prec, name, tol in ((TF32, "tf32", TOL["tf32"]), (FP32, "fp32", TOL["fp32"]), (FP64, "fp64", TOL["fp64"])):
        Xd = _to_dev(X, name, False)
        Yd = torch.empty_like(Xd)
        ctx.apply_H(prec, Xd, Yd, B, B)
        torch.cuda.synchronize()
        for J, ref in want:
            got = Yd[torch.from_numpy(np.asarray(J)).cuda()].cpu().numpy().astype(np.float64)
            assert _relerr(got, ref) < tol, (name, _relerr(got, ref))


def test_full_size_cfg1_filter_properties():
    """Properties of one full-size TF32 filter call that hold at any size: (i) columns are filtered independently, so
    a 64-column call reproduces the first 64 columns of the 200-column call (different tile shapes, ragged tail);
    (ii) the output is finite and (iii) scaling the input block scales the output (linearity in X for fixed Lambda)."""
    from paper_2604_26037_b200 import TF32
    from paper_2604_26037_b200.harness import Harness
    cfg, sysd, ctx = _full_cfg1()
    B, m = cfg.block, 6
    M = ctx.num_dofs()
    hz = Harness(ctx, M, False)
    gen = torch.Generator(device="cuda").manual_seed(cfg.seed)
    X0 = torch.rand((M, B), dtype=torch.float64, device="cuda", generator=gen) - 0.5
    X, lam = hz.rayleigh_ritz(hz.s_orthonormalise(X0))
    bU = hz.upper_bound(k=10, seed=1)
    b0, bW = float(lam[0]) - 0.1, 0.5 * (float(lam[0]) - 0.1 + bU)
    nbytes = ctx.filter_workspace(TF32, B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    A = X.to(torch.float32).contiguous()
    ctx.cheb_filter(TF32, m, b0, bW, bU, A, lam, B, B, ws, nbytes)
    Bsub = X[:, :64].to(torch.float32).contiguous()
    ctx.cheb_filter(TF32, m, b0, bW, bU, Bsub, lam[:64], 64, 64, ws, nbytes)
    C2 = (2.0 * X).to(torch.float32).contiguous()
    ctx.cheb_filter(TF32, m, b0, bW, bU, C2, lam, B, B, ws, nbytes)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(A).all())
    nrm = A[:, :64].double().norm()
    assert float((A[:, :64].double() - Bsub.double()).norm() / nrm) < 1e-4
    assert float((C2.double() - 2.0 * A.double()).norm() / (2.0 * A.double().norm())) < 1e-4


@pytest.mark.parametrize("B", [10, 130])
def test_filter_ragged_block_width(B):
    """Block widths that are not a multiple of 4 (config 2 has B = 250) or just over one vector tile: the workspace
    rows are padded to a multiple of 4 and the pad columns must stay inert."""
    from oracle import chfsi
    from paper_2604_26037_b200 import TF32
    cfg, sysd, ops, ctx = _setup("cfg1_twin")
    m = 5
    X0 = random_block(cfg, B, stream=21) * ops.mask[:, None]
    X = chfsi.s_orthonormalise(ops.apply_S, X0)
    X, lam = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, X)
    b0, bW, bU = _bounds(ops, lam)
    want = chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, X, lam, m, b0, bW, bU)
    Xd = _to_dev(X, "tf32", False)
    nbytes = ctx.filter_workspace(TF32, B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.cheb_filter(TF32, m, b0, bW, bU, Xd, lam, B, B, ws, nbytes)
    torch.cuda.synchronize()
    assert _relerr(_to_host(Xd, False), want) < 1e-2


@pytest.mark.parametrize("name,B", [("cfg2_twin", 136), ("cfg3_twin", 80), ("cfg4_twin", 256)])
@pytest.mark.parametrize("prec", ["tf32", "fp32"])
def test_apply_H_wide_blocks(name, B, prec):
    """Block widths that need two or more 128-column tiles on the twins: p = 7 (two node halves of 256 columns, both
    TMEM buffers full), complex (P / Q accumulators, 160 real columns), Dirichlet with the full config-4 width."""
    from paper_2604_26037_b200 import PREC
    cfg, sysd, ops, ctx = _setup(name)
    X = random_block(cfg, B, stream=31) * ops.mask[:, None]
    Xd = _to_dev(X, prec, cfg.complex)
    Yd = torch.full_like(Xd, float("nan"))
    ctx.apply_H(PREC[prec], Xd, Yd, B, B)
    torch.cuda.synchronize()
    want = ops.apply_H(X) * ops.mask[:, None]
    assert _relerr(_to_host(Yd, cfg.complex), want) < TOL[prec], (name, prec)


@pytest.mark.parametrize("name,B", [("cfg2_twin", 136), ("cfg3_twin", 80)])
def test_filter_wide_blocks(name, B):
    from oracle import chfsi
    from paper_2604_26037_b200 import TF32
    cfg, sysd, ops, ctx = _setup(name)
    m = 4
    X0 = random_block(cfg, B, stream=33) * ops.mask[:, None]
    X = chfsi.s_orthonormalise(ops.apply_S, X0)
    X, lam = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, X)
    b0, bW, bU = _bounds(ops, lam)
    want = chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, X, lam, m, b0, bW, bU)
    Xd = _to_dev(X, "tf32", cfg.complex)
    nbytes = ctx.filter_workspace(TF32, B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.cheb_filter(TF32, m, b0, bW, bU, Xd, lam, B, B, ws, nbytes)
    torch.cuda.synchronize()
    assert _relerr(_to_host(Xd, cfg.complex), want) < 1e-2


def test_filter_complex_odd_width_generic_sequence():
    """A complex block of odd width cannot be cut into 16-byte pieces of interleaved columns: the library runs the
    unfused sequence (and asks for its larger workspace); the result is the same filter."""
    from oracle import chfsi
    from paper_2604_26037_b200 import TF32
    cfg, sysd, ops, ctx = _setup("cfg3_twin")
    B, m = 7, 4
    X0 = random_block(cfg, B, stream=35) * ops.mask[:, None]
    X = chfsi.s_orthonormalise(ops.apply_S, X0)
    X, lam = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, X)
    b0, bW, bU = _bounds(ops, lam)
    want = chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, X, lam, m, b0, bW, bU)
    Xd = _to_dev(X, "tf32", True)
    nbytes = ctx.filter_workspace(TF32, B)
    assert nbytes >= ctx.filter_workspace(TF32, B + 1)      # complex contexts are always told the unfused sequence's size
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.cheb_filter(TF32, m, b0, bW, bU, Xd, lam, B, B, ws, nbytes)
    torch.cuda.synchronize()
    assert _relerr(_to_host(Xd, True), want) < 1e-2


@pytest.mark.parametrize("name,prec", [("cfg1_twin", "fp32"), ("cfg3_twin", "tf32"), ("cfg0", "fp64")])
def test_filter_host_block_set(name, prec):
    """pawfe_cheb_filter_host_set: three pinned HOST blocks of different widths (the third reuses the first device
    block of the two-block pipeline) against the oracle's filter of each block; also equal to the device-block call."""
    from oracle import chfsi
    from paper_2604_26037_b200 import PREC
    cfg, sysd, ops, ctx = _setup(name)
    m = 4
    widths = [cfg.block, max(2, cfg.block // 2), cfg.block - 2]
    Xs, lams, wants = [], [], []
    for k, B in enumerate(widths):
        X0 = random_block(cfg, B, stream=40 + k) * ops.mask[:, None]
        X = chfsi.s_orthonormalise(ops.apply_S, X0)
        X, lam = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, X)
        Xs.append(X); lams.append(lam)
    b0 = min(l[0] for l in lams) - 0.1
    bW = max(l[-1] for l in lams) + 0.05
    bU = _bounds(ops, lams[0])[2]
    for X, lam in zip(Xs, lams):
        wants.append(chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, X, lam, m, b0, bW, bU))
    host = [_to_dev(X, prec, cfg.complex).cpu().pin_memory() for X in Xs]
    dev = [h.cuda() for h in host]
    ctx.cheb_filter_host_set(PREC[prec], m, b0, bW, bU, [h.data_ptr() for h in host], lams, widths, widths)
    tol = {"fp64": 1e-10, "fp32": 5e-5, "tf32": 1e-2}[prec]
    for k, B in enumerate(widths):
        got = _to_host(host[k], cfg.complex)
        assert _relerr(got, wants[k]) < tol, (name, prec, k, _relerr(got, wants[k]))
        nbytes = ctx.filter_workspace(PREC[prec], B)
        ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        ctx.cheb_filter(PREC[prec], m, b0, bW, bU, dev[k], lams[k], B, B, ws, nbytes)
        torch.cuda.synchronize()
        # same kernels on the same data.  FP32 storage: the ordered path is bit-reproducible except for the FP64 residual set-up,
        # whose FP64 atomics can move the last bit of the FP32 R_Y (1e-7 level after m steps).  FP64 mode: the FP64 assembly is
        # by atomics whose order differs from run to run: ~1e-15 per product, amplified by the degree-4 recurrence (the gate
        # was 1e-13 before commit 61383d5, which a run with an unlucky atomic order exceeded; 1e-12 = the per-product bar)
        assert _relerr(_to_host(dev[k], cfg.complex), got) < (1e-12 if prec == "fp64" else 1e-5)


# ---- degenerate and extreme cases --------------------------------------------------------------------------------

@pytest.mark.parametrize("name,prec", [("cfg1_twin", "tf32"), ("cfg1_twin", "fp64"), ("cfg3_twin", "tf32"), ("cfg4_twin", "fp32")])
def test_filter_degree_one(name, prec):
    """m = 1 (reading R22): the step loop is empty, Psi_f = S^-1approx R_1 + X Lambda_1 from the FP64 residual alone."""
    from oracle import chfsi
    from paper_2604_26037_b200 import PREC
    cfg, sysd, ops, ctx = _setup(name)
    B = cfg.block
    X0 = random_block(cfg, B, stream=51) * ops.mask[:, None]
    X = chfsi.s_orthonormalise(ops.apply_S, X0)
    X, lam = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, X)
    b0, bW, bU = _bounds(ops, lam)
    want = chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, X, lam, 1, b0, bW, bU)
    Xd = _to_dev(X, prec, cfg.complex)
    nbytes = ctx.filter_workspace(PREC[prec], B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.cheb_filter(PREC[prec], 1, b0, bW, bU, Xd, lam, B, B, ws, nbytes)
    torch.cuda.synchronize()
    assert _relerr(_to_host(Xd, cfg.complex), want) < {"fp64": 1e-10, "fp32": 5e-5, "tf32": 5e-5}[prec]


@pytest.mark.parametrize("name", ["cfg1_twin", "cfg4_twin"])
def test_single_vector_block(name):
    """B = 1: one column (workspace rows padded to 4, one partially filled vector tile)."""
    from oracle import chfsi
    from paper_2604_26037_b200 import FP32, TF32
    cfg, sysd, ops, ctx = _setup(name)
    X = random_block(cfg, 1, stream=52) * ops.mask[:, None]
    Xd = _to_dev(X, "fp32", False)
    Yd = torch.empty_like(Xd)
    ctx.apply_H(FP32, Xd, Yd, 1, 1)
    torch.cuda.synchronize()
    assert _relerr(_to_host(Yd, False), ops.apply_H(X) * ops.mask[:, None]) < TOL["fp32"]
    Xs = chfsi.s_orthonormalise(ops.apply_S, X)
    Xs, lam = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, Xs)
    b0, bW, bU = _bounds(ops, lam)
    m = 4
    want = chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, Xs, lam, m, b0, bW, bU)
    Xd = _to_dev(Xs, "tf32", False)
    nbytes = ctx.filter_workspace(TF32, 1)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.cheb_filter(TF32, m, b0, bW, bU, Xd, lam, 1, 1, ws, nbytes)
    torch.cuda.synchronize()
    assert _relerr(_to_host(Xd, False), want) < 1e-2


def test_maximum_block_width():
    """B = 512, the widest block the library accepts (four vector tiles per cell): H X in every mode, one filter call."""
    from oracle import chfsi
    from paper_2604_26037_b200 import PREC, TF32
    cfg, sysd, ops, ctx = _setup("cfg1_twin")
    B = 512
    X = random_block(cfg, B, stream=53) * ops.mask[:, None]
    want = ops.apply_H(X) * ops.mask[:, None]
    for prec in ("fp64", "fp32", "tf32"):
        Xd = _to_dev(X, prec, False)
        Yd = torch.full_like(Xd, float("nan"))
        ctx.apply_H(PREC[prec], Xd, Yd, B, B)
        torch.cuda.synchronize()
        assert _relerr(_to_host(Yd, False), want) < TOL[prec], prec
    Xs = chfsi.s_orthonormalise(ops.apply_S, X)
    Xs, lam = chfsi.rayleigh_ritz(ops.apply_H, ops.apply_S, Xs)
    b0, bW, bU = _bounds(ops, lam)
    m = 3
    wantf = chfsi.filter_residual(ops.apply_H, ops.apply_S, ops.apply_Sinv, Xs, lam, m, b0, bW, bU)
    Xd = _to_dev(Xs, "tf32", False)
    nbytes = ctx.filter_workspace(TF32, B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    ctx.cheb_filter(TF32, m, b0, bW, bU, Xd, lam, B, B, ws, nbytes)
    torch.cuda.synchronize()
    assert _relerr(_to_host(Xd, False), wantf) < 1e-2


def test_error_behaviour():
    """Every call returns a status (include/pawfe.h): bad arguments are PAWFE_EINVAL, calls before set-up PAWFE_ESTATE; the
    block is left untouched."""
    from paper_2604_26037_b200 import Context, PawfeError, PERIODIC, TF32
    cfg, sysd, ops, ctx = _setup("cfg1_twin")
    B = 8
    X = _to_dev(random_block(cfg, B, stream=54), "tf32", False)
    X0 = X.clone()
    lam = np.linspace(-1.0, 0.0, B)
    nbytes = ctx.filter_workspace(TF32, B)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    with pytest.raises(PawfeError, match="EINVAL"):
        ctx.cheb_filter(TF32, 4, -2.0, 1.0, 0.5, X, lam, B, B, ws, nbytes)          # bW >= bU
    with pytest.raises(PawfeError, match="EINVAL"):
        ctx.cheb_filter(TF32, 4, 0.5, 0.0, 10.0, X, lam, B, B, ws, nbytes)          # b0 >= bW
    with pytest.raises(PawfeError, match="EINVAL"):
        ctx.cheb_filter(TF32, 0, -2.0, 0.5, 10.0, X, lam, B, B, ws, nbytes)         # m < 1
    with pytest.raises(PawfeError, match="EINVAL"):
        ctx.cheb_filter(TF32, 4, -2.0, 0.5, 10.0, X, lam, B - 1, B, ws, nbytes)     # ld < B
    with pytest.raises(PawfeError, match="EINVAL"):
        ctx.cheb_filter(TF32, 4, -2.0, 0.5, 10.0, X, lam, B, B, ws, nbytes // 2)    # workspace too small
    with pytest.raises(PawfeError, match="EINVAL"):
        ctx.filter_workspace(TF32, 513)                                             # B beyond the maximum
    torch.cuda.synchronize()
    assert torch.equal(X, X0)
    bare = Context(0, torch.cuda.current_stream().cuda_stream)
    bare.mesh_create(cfg.ncells, cfg.box, cfg.p, PERIODIC, None)
    Y = torch.empty_like(X)
    with pytest.raises(PawfeError, match="ESTATE"):
        bare.apply_H(TF32, X, Y, B, B)                                              # no potential, no atoms yet
    bare.destroy()


@pytest.mark.parametrize("prec", ["fp64", "fp32", "tf32"])
def test_full_loop_eigenvalues_cfg0(prec):
    """north_star: converged lowest eigenvalues of the full R-ChFSI loop (Algorithm 1 around the library's filter: config 0,
    degree 10, 30 outer iterations, 16 vectors) within 1e-6 Ha of the oracle's dense FP64 solve eigh(H, S), in every
    precision mode; Rayleigh-Ritz in FP64 with the library's own applies (paper_2604_26037_b200/harness.py)."""
    from oracle import chfsi
    from paper_2604_26037_b200 import PREC
    from paper_2604_26037_b200.harness import Harness, chfsi_loop
    cfg, sysd, ops, ctx = _setup("cfg0")
    want = chfsi.dense_eigh(ops.dense_H(), ops.dense_S())
    hz = Harness(ctx, ops.mesh.M, cfg.complex)
    bU = hz.upper_bound(k=10, seed=1)
    assert bU >= np.max(np.real(np.linalg.eigvals(ops.apply_Sinv(ops.dense_H()))))   # an upper bound of the filtered operator
    X0 = torch.from_numpy(random_block(cfg, cfg.nvec)).cuda()
    X, lam = chfsi_loop(ctx, hz, X0, PREC[prec], cfg.degree, bU, cfg.outer)
    ncheck = (3 * cfg.nvec) // 4     # reading R18
    err = np.max(np.abs(np.asarray(lam)[:ncheck] - want[:ncheck]))
    # north_star's bar is 1e-6 Ha; measured 2.5e-14 in all three modes (Rayleigh-Ritz is FP64, the filter only has to span
    # the subspace), so the gate is held far tighter than the bar
    assert err < 1e-10, (prec, err)
