"""pawfe_apply_Sinv_noalloc (include/pawfe.h): S^-1approx X with its projection scratch in the library's static 1 MiB device
array, against the existing pawfe_apply_Sinv on the same inputs, on two calls in a row (the second narrower than the first,
so the array still holds the first call's values where the second does not write).

Collected last on purpose (file name): the suite runs with `pytest -x`, and a failure here must not hide other tests.
Needs nothing from the other test files: builds its own contexts, uses no oracle (the reference is the existing path, which
tests/test_gpu_parity.py::test_apply_H_S_Sinv compares with the oracle).
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from pawfe_inputs import get_config, make_system, random_block, twin  # noqa: E402

# tolerances of tests/test_gpu_parity.py (north_star: per product FP64 <= 1e-12, FP32 <= 1e-5); both paths compute the same
# sums in different orders
TOL = {"fp64": 1e-12, "fp32": 1e-5}
SCRATCH_BYTES = 1 << 20


def _ctx(which):
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2604_26037_b200 import context_from_system
    base = get_config(1 if which == "real" else 3)
    cfg = twin(base, nc=4, natoms=8, nvec=24, block=24)
    sysd = make_system(cfg)
    return cfg, context_from_system(sysd, device=0, stream=torch.cuda.current_stream().cuda_stream)


def _to_dev(x, prec, cplx):
    real = np.float64 if prec == "fp64" else np.float32
    a = np.stack([x.real, x.imag], axis=-1).astype(real) if cplx else x.astype(real)
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _relerr(a, b):
    a, b = a.double(), b.double()
    return float((a - b).norm() / b.norm())


@pytest.mark.parametrize("which", ["real", "complex"])
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_apply_Sinv_noalloc_matches_apply_Sinv_twice(which, prec):
    from paper_2604_26037_b200 import PREC
    cfg, ctx = _ctx(which)
    try:
        free_after_first = None
        for call, (B, ld, stream) in enumerate([(24, 24, 71), (10, 12, 72)]):   # second call: narrower, padded ld
            X = random_block(cfg, ld, stream=stream)
            Xd = _to_dev(X, prec, cfg.complex)
            want = torch.full_like(Xd, 3.0)
            got = torch.full_like(Xd, 3.0)
            ctx.apply_Sinv(PREC[prec], Xd, want, ld, B)
            ctx.apply_Sinv_noalloc(PREC[prec], Xd, got, ld, B)
            torch.cuda.synchronize()
            err = _relerr(got[:, :B], want[:, :B])
            assert err < TOL[prec], (which, prec, call, err)
            assert float(want[:, :B].double().norm()) > 0
            assert torch.equal(got[:, B:], torch.full_like(got[:, B:], 3.0))          # pad columns untouched
            free_now, _ = torch.cuda.mem_get_info()
            if free_after_first is None:
                free_after_first = free_now
            else:   # nothing was allocated between the first and the second call (torch's own blocks are cached)
                assert free_now >= free_after_first - (2 << 20), (free_after_first, free_now)
    finally:
        ctx.destroy()


def test_apply_Sinv_noalloc_rejects_blocks_beyond_the_static_array():
    """8 atoms x 9 projectors, complex FP64: 2 * 8 * 9 * B * 16 bytes > 1 MiB for B = 512; B = 400 (921,600 bytes) still fits."""
    from paper_2604_26037_b200 import FP64, PawfeError
    cfg, ctx = _ctx("complex")
    try:
        assert 2 * cfg.natoms * cfg.nproj * 512 * 16 > SCRATCH_BYTES >= 2 * cfg.natoms * cfg.nproj * 400 * 16
        X = _to_dev(random_block(cfg, 512, stream=73), "fp64", True)
        Y = torch.full_like(X, 5.0)
        with pytest.raises(PawfeError, match=r"EINVAL.*1048576"):
            ctx.apply_Sinv_noalloc(FP64, X, Y, 512, 512)
        torch.cuda.synchronize()
        assert torch.equal(Y, torch.full_like(Y, 5.0))                               # a rejected call writes nothing
        want = torch.empty_like(X)
        ctx.apply_Sinv(FP64, X, want, 512, 400)
        ctx.apply_Sinv_noalloc(FP64, X, Y, 512, 400)
        torch.cuda.synchronize()
        assert _relerr(Y[:, :400], want[:, :400]) < TOL["fp64"]
    finally:
        ctx.destroy()
