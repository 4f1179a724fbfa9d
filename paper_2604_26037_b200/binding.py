"""Thin ctypes binding of libpawfe.so (include/pawfe.h).  Argument marshalling only: every step of the
path runs in the library's CUDA kernels.  PyTorch is used by callers for device memory and streams.

The binding fails loudly if the library is missing or no sm_100 device is present: there is no CPU
fallback, and nothing here imports the test oracle.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpawfe.so")

FP64, FP32, TF32 = 0, 1, 2
PERIODIC, DIRICHLET = 0, 1
PREC = {"fp64": FP64, "fp32": FP32, "tf32": TF32}
_STATUS = {0: "OK", 1: "EINVAL", 2: "ENOMEM", 3: "ECUDA", 4: "ESTATE", 5: "EUNSUPPORTED"}

# every symbol include/pawfe.h declares
SYMBOLS = [
    "pawfe_create", "pawfe_destroy", "pawfe_last_error", "pawfe_set_stream", "pawfe_mesh_create",
    "pawfe_local_potential_gaussians", "pawfe_atoms_create", "pawfe_update_coupling", "pawfe_num_dofs",
    "pawfe_num_pairs", "pawfe_get_cell_matrix", "pawfe_get_sinv_coupling", "pawfe_apply_H", "pawfe_apply_S",
    "pawfe_apply_Sinv", "pawfe_filter_workspace", "pawfe_cheb_filter", "pawfe_cheb_filter_host", "pawfe_cheb_filter_host_set",
    "pawfe_col_norms", "pawfe_launch_count", "pawfe_cell_kernel_name", "pawfe_cell_timing",
    "pawfe_cell_timing_read", "pawfe_set_cell_matrices", "pawfe_get_pairs", "pawfe_set_projector_blocks",
    "pawfe_apply_HSinv", "pawfe_prepare", "pawfe_cheb_filter_hs", "pawfe_apply_Sinv_noalloc", "pawfe_setup_timing_read", "pawfe_lanczos_bound", "pawfe_rr_project",
    "pawfe_rr_rotate", "pawfe_set_sinv_variant",
]


class PawfeError(RuntimeError):
    pass


_lib = None


def load_library(path: Optional[str] = None) -> C.CDLL:
    """dlopen libpawfe.so (built in-tree by paper_2604_26037_b200/build.py) and set the prototypes."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise PawfeError(f"{p} not found: build it with `python -m paper_2604_26037_b200.build` "
                         "(there is no CPU fallback)")
    lib = C.CDLL(p)
    vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    lib.pawfe_create.argtypes = [C.POINTER(vp), C.c_int, vp]
    lib.pawfe_destroy.argtypes = [vp]
    lib.pawfe_last_error.argtypes = [vp]
    lib.pawfe_last_error.restype = C.c_char_p
    lib.pawfe_set_stream.argtypes = [vp, vp]
    lib.pawfe_mesh_create.argtypes = [vp, ip, dp, C.c_int, C.c_int, dp]
    lib.pawfe_local_potential_gaussians.argtypes = [vp, C.c_int, dp, dp, dp, C.c_int]
    lib.pawfe_atoms_create.argtypes = [vp, C.c_int, dp, C.c_int, ip, ip, dp, dp, C.c_double, dp, dp]
    lib.pawfe_update_coupling.argtypes = [vp, dp]
    lib.pawfe_num_dofs.argtypes = [vp, C.POINTER(C.c_long)]
    lib.pawfe_num_pairs.argtypes = [vp, C.POINTER(C.c_long)]
    lib.pawfe_get_cell_matrix.argtypes = [vp, C.c_long, dp]
    lib.pawfe_get_sinv_coupling.argtypes = [vp, dp]
    lib.pawfe_set_cell_matrices.argtypes = [vp, vp, C.c_int, C.c_int]
    lib.pawfe_get_pairs.argtypes = [vp, ip, ip]
    lib.pawfe_set_projector_blocks.argtypes = [vp, vp, C.c_int]
    lib.pawfe_prepare.argtypes = [vp, C.c_int, C.c_int, C.c_int]
    lib.pawfe_set_sinv_variant.argtypes = [vp, C.c_int]
    lib.pawfe_cheb_filter_hs.argtypes = [vp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, vp, vp, vp, dp,
                                         C.c_long, C.c_int, vp, C.c_size_t]
    for f in (lib.pawfe_apply_H, lib.pawfe_apply_S, lib.pawfe_apply_Sinv, lib.pawfe_apply_HSinv, lib.pawfe_apply_Sinv_noalloc):
        f.argtypes = [vp, C.c_int, vp, vp, C.c_long, C.c_int]
    lib.pawfe_filter_workspace.argtypes = [vp, C.c_int, C.c_int, C.POINTER(C.c_size_t)]
    lib.pawfe_cheb_filter.argtypes = [vp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, vp, dp,
                                      C.c_long, C.c_int, vp, C.c_size_t]
    lib.pawfe_cheb_filter_host.argtypes = [vp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, vp, dp,
                                           C.c_long, C.c_int]
    lib.pawfe_cheb_filter_host_set.argtypes = [vp, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                               C.POINTER(C.c_void_p), C.POINTER(dp), C.POINTER(C.c_long),
                                               C.POINTER(C.c_int), C.c_int]
    lib.pawfe_col_norms.argtypes = [vp, C.c_int, vp, C.c_long, C.c_int, vp]
    lib.pawfe_launch_count.argtypes = [vp, C.POINTER(C.c_long)]
    lib.pawfe_cell_timing.argtypes = [vp, C.c_int]
    lib.pawfe_cell_timing_read.argtypes = [vp, C.POINTER(C.c_long), C.POINTER(C.c_double)]
    lib.pawfe_setup_timing_read.argtypes = [vp, C.POINTER(C.c_long), C.POINTER(C.c_double)]
    lib.pawfe_lanczos_bound.argtypes = [vp, C.c_int, vp, dp, dp, dp, ip]
    lib.pawfe_rr_project.argtypes = [vp, vp, vp, C.c_long, C.c_int, vp]
    lib.pawfe_rr_rotate.argtypes = [vp, C.c_int, vp, C.c_long, vp, vp, C.c_long, C.c_int]
    lib.pawfe_cell_kernel_name.argtypes = [vp, C.c_int, C.c_int]
    lib.pawfe_cell_kernel_name.restype = C.c_char_p
    for s in SYMBOLS:
        if s not in ("pawfe_last_error", "pawfe_cell_kernel_name"):
            getattr(lib, s).restype = C.c_int
    if path is None:
        _lib = lib
    return lib


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _iptr(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_int))


def _f64(x) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


def _i32(x) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(x, dtype=np.int32))


class Context:
    """One pawfe_ctx.  Method names follow include/pawfe.h without the prefix.  Block arguments are
    torch CUDA tensors (or raw device pointers as ints); the binding only passes their data_ptr()."""

    def __init__(self, device: int = 0, stream: int = 0):
        self.lib = load_library()
        self._h = C.c_void_p()
        st = self.lib.pawfe_create(C.byref(self._h), int(device), C.c_void_p(int(stream) or None))
        if st != 0:
            msg = self.lib.pawfe_last_error(self._h).decode() if self._h else ""
            if self._h:
                self.lib.pawfe_destroy(self._h)
                self._h = C.c_void_p()
            raise PawfeError(f"pawfe_create: {_STATUS.get(st, st)}: {msg}")
        self.complex = False

    def _check(self, st: int, what: str):
        if st != 0:
            raise PawfeError(f"{what}: {_STATUS.get(st, st)}: {self.lib.pawfe_last_error(self._h).decode()}")

    def destroy(self):
        if self._h:
            self.lib.pawfe_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # ---- set-up ----
    def set_stream(self, stream: int):
        self._check(self.lib.pawfe_set_stream(self._h, C.c_void_p(int(stream) or None)), "pawfe_set_stream")

    def mesh_create(self, ncells: Sequence[int], box: Sequence[float], p: int, bc: int, kpt=None):
        nc, bx = _i32(ncells), _f64(box)
        k = _f64(kpt) if kpt is not None else None
        self._check(self.lib.pawfe_mesh_create(self._h, _iptr(nc), _dptr(bx), int(p), int(bc),
                                               _dptr(k) if k is not None else None), "pawfe_mesh_create")
        self.complex = kpt is not None

    def local_potential_gaussians(self, pos, Z, sigma, keep_fp64: bool = True):
        pos, Z, sigma = _f64(pos), _f64(Z), _f64(sigma)
        self._check(self.lib.pawfe_local_potential_gaussians(self._h, len(Z), _dptr(pos), _dptr(Z), _dptr(sigma),
                                                             int(keep_fp64)), "pawfe_local_potential_gaussians")

    def atoms_create(self, pos, proj_l, proj_m, proj_sigma, proj_amp, rc: float, D, dS):
        pos, D, dS = _f64(pos), _f64(D), _f64(dS)
        l, m, sg, am = _i32(proj_l), _i32(proj_m), _f64(proj_sigma), _f64(proj_amp)
        self._check(self.lib.pawfe_atoms_create(self._h, len(pos.reshape(-1, 3)), _dptr(pos), len(l), _iptr(l),
                                                _iptr(m), _dptr(sg), _dptr(am), float(rc), _dptr(D), _dptr(dS)),
                    "pawfe_atoms_create")

    def set_cell_matrices(self, Hcell: np.ndarray, keep_fp64: bool = True):
        """Hcell: host array [cell][n][n], float64 or complex128 (pawfe_set_cell_matrices)."""
        H = np.ascontiguousarray(Hcell, dtype=np.complex128 if self.complex else np.float64)
        self._check(self.lib.pawfe_set_cell_matrices(self._h, C.c_void_p(H.ctypes.data), 0, int(keep_fp64)),
                    "pawfe_set_cell_matrices")

    def get_pairs(self):
        n = self.num_pairs()
        pc, pa = np.zeros(max(n, 1), dtype=np.int32), np.zeros(max(n, 1), dtype=np.int32)
        self._check(self.lib.pawfe_get_pairs(self._h, _iptr(pc), _iptr(pa)), "pawfe_get_pairs")
        return pc[:n], pa[:n]

    def set_projector_blocks(self, Cd: np.ndarray):
        """Cd: host array [pair][nproj][n], float64 or complex128 (pawfe_set_projector_blocks)."""
        A = np.ascontiguousarray(Cd, dtype=np.complex128 if self.complex else np.float64)
        self._check(self.lib.pawfe_set_projector_blocks(self._h, C.c_void_p(A.ctypes.data), 0),
                    "pawfe_set_projector_blocks")

    def prepare(self, prec: int, Bmax: int, mmax: int):
        self._check(self.lib.pawfe_prepare(self._h, int(prec), int(Bmax), int(mmax)), "pawfe_prepare")

    def set_sinv_variant(self, variant: int):
        """0: G^a = C^dagger M_D^-1 C (Eq. 29); 1: G^a = <p_alpha|p_beta> (L228)."""
        self._check(self.lib.pawfe_set_sinv_variant(self._h, int(variant)), "pawfe_set_sinv_variant")

    def update_coupling(self, D):
        D = _f64(D)
        self._check(self.lib.pawfe_update_coupling(self._h, _dptr(D)), "pawfe_update_coupling")

    # ---- queries ----
    def num_dofs(self) -> int:
        v = C.c_long()
        self._check(self.lib.pawfe_num_dofs(self._h, C.byref(v)), "pawfe_num_dofs")
        return v.value

    def num_pairs(self) -> int:
        v = C.c_long()
        self._check(self.lib.pawfe_num_pairs(self._h, C.byref(v)), "pawfe_num_pairs")
        return v.value

    def launch_count(self) -> int:
        v = C.c_long()
        self._check(self.lib.pawfe_launch_count(self._h, C.byref(v)), "pawfe_launch_count")
        return v.value

    def cell_timing(self, enable: bool):
        self._check(self.lib.pawfe_cell_timing(self._h, int(enable)), "pawfe_cell_timing")

    def cell_timing_read(self):
        n, ms = C.c_long(), C.c_double()
        self._check(self.lib.pawfe_cell_timing_read(self._h, C.byref(n), C.byref(ms)), "pawfe_cell_timing_read")
        return n.value, ms.value

    def setup_timing_read(self):
        n, ms = C.c_long(), C.c_double()
        self._check(self.lib.pawfe_setup_timing_read(self._h, C.byref(n), C.byref(ms)), "pawfe_setup_timing_read")
        return n.value, ms.value

    def cell_kernel_name(self, prec: int, B: int) -> str:
        return self.lib.pawfe_cell_kernel_name(self._h, int(prec), int(B)).decode()

    def get_cell_matrix(self, cell: int, n: int) -> np.ndarray:
        out = np.empty((n, n, 2) if self.complex else (n, n), dtype=np.float64)
        self._check(self.lib.pawfe_get_cell_matrix(self._h, int(cell), _dptr(out)), "pawfe_get_cell_matrix")
        return out[..., 0] + 1j * out[..., 1] if self.complex else out

    def get_sinv_coupling(self, natoms: int, npj: int) -> np.ndarray:
        out = np.empty((natoms, npj, npj, 2) if self.complex else (natoms, npj, npj), dtype=np.float64)
        self._check(self.lib.pawfe_get_sinv_coupling(self._h, _dptr(out)), "pawfe_get_sinv_coupling")
        return out[..., 0] + 1j * out[..., 1] if self.complex else out

    # ---- hot calls ----
    @staticmethod
    def _ptr(t) -> C.c_void_p:
        return C.c_void_p(t if isinstance(t, int) else t.data_ptr())

    def apply_H(self, prec: int, X, Y, ld: int, B: int):
        self._check(self.lib.pawfe_apply_H(self._h, int(prec), self._ptr(X), self._ptr(Y), int(ld), int(B)), "pawfe_apply_H")

    def apply_S(self, prec: int, X, Y, ld: int, B: int):
        self._check(self.lib.pawfe_apply_S(self._h, int(prec), self._ptr(X), self._ptr(Y), int(ld), int(B)), "pawfe_apply_S")

    def apply_Sinv(self, prec: int, X, Y, ld: int, B: int):
        self._check(self.lib.pawfe_apply_Sinv(self._h, int(prec), self._ptr(X), self._ptr(Y), int(ld), int(B)), "pawfe_apply_Sinv")

    def apply_Sinv_noalloc(self, prec: int, X, Y, ld: int, B: int):
        """S^-1approx X with its scratch in the library's static 1 MiB device array (no allocation; include/pawfe.h)."""
        self._check(self.lib.pawfe_apply_Sinv_noalloc(self._h, int(prec), self._ptr(X), self._ptr(Y), int(ld), int(B)),
                    "pawfe_apply_Sinv_noalloc")

    def apply_HSinv(self, prec: int, X, Y, ld: int, B: int):
        self._check(self.lib.pawfe_apply_HSinv(self._h, int(prec), self._ptr(X), self._ptr(Y), int(ld), int(B)), "pawfe_apply_HSinv")

    def cheb_filter_hs(self, prec: int, m: int, b0: float, bW: float, bU: float, X, HX, SX, lam, ld: int, B: int,
                       workspace, workspace_bytes: int):
        lam = _f64(lam)
        self._check(self.lib.pawfe_cheb_filter_hs(self._h, int(prec), int(m), float(b0), float(bW), float(bU),
                                                  self._ptr(X), self._ptr(HX), self._ptr(SX), _dptr(lam), int(ld), int(B),
                                                  self._ptr(workspace), int(workspace_bytes)), "pawfe_cheb_filter_hs")

    def filter_workspace(self, prec: int, B: int) -> int:
        v = C.c_size_t()
        self._check(self.lib.pawfe_filter_workspace(self._h, int(prec), int(B), C.byref(v)), "pawfe_filter_workspace")
        return v.value

    def cheb_filter(self, prec: int, m: int, b0: float, bW: float, bU: float, X, lam, ld: int, B: int,
                    workspace, workspace_bytes: int):
        lam = _f64(lam)
        self._check(self.lib.pawfe_cheb_filter(self._h, int(prec), int(m), float(b0), float(bW), float(bU),
                                               self._ptr(X), _dptr(lam), int(ld), int(B), self._ptr(workspace),
                                               int(workspace_bytes)), "pawfe_cheb_filter")

    def cheb_filter_host(self, prec: int, m: int, b0: float, bW: float, bU: float, X_host_ptr: int, lam,
                         ld: int, B: int):
        lam = _f64(lam)
        self._check(self.lib.pawfe_cheb_filter_host(self._h, int(prec), int(m), float(b0), float(bW), float(bU),
                                                    C.c_void_p(int(X_host_ptr)), _dptr(lam), int(ld), int(B)),
                    "pawfe_cheb_filter_host")

    def cheb_filter_host_set(self, prec: int, m: int, b0: float, bW: float, bU: float, X_host_ptrs, lams, lds, Bs):
        """Algorithm 2 over a set of HOST blocks, copies pipelined under the filters (pawfe_cheb_filter_host_set)."""
        n = len(X_host_ptrs)
        lams = [_f64(x) for x in lams]
        xs = (C.c_void_p * n)(*[int(p) for p in X_host_ptrs])
        ls = (C.POINTER(C.c_double) * n)(*[_dptr(x) for x in lams])
        ldv = (C.c_long * n)(*[int(x) for x in lds])
        bv = (C.c_int * n)(*[int(x) for x in Bs])
        self._check(self.lib.pawfe_cheb_filter_host_set(self._h, int(prec), int(m), float(b0), float(bW), float(bU),
                                                        xs, ls, ldv, bv, n), "pawfe_cheb_filter_host_set")

    def lanczos_bound(self, k: int, v0):
        """b_U of H S^-1approx from a k-step Lanczos started at the FP64 device vector v0 (pawfe_lanczos_bound).
        Returns (bU, theta_max, beta_k, steps)."""
        bU, th, bk, st = C.c_double(), C.c_double(), C.c_double(), C.c_int()
        self._check(self.lib.pawfe_lanczos_bound(self._h, int(k), self._ptr(v0), C.byref(bU), C.byref(th), C.byref(bk), C.byref(st)),
                    "pawfe_lanczos_bound")
        return bU.value, th.value, bk.value, st.value

    def rr_project(self, X, Y, ld: int, B: int, G):
        """G = X^dagger Y (FP64, lower-triangle blocks computed, mirrored; pawfe_rr_project)"""
        self._check(self.lib.pawfe_rr_project(self._h, self._ptr(X), self._ptr(Y), int(ld), int(B), self._ptr(G)), "pawfe_rr_project")

    def rr_rotate(self, mixed: bool, X, ldx: int, Q, Xout, ldo: int, B: int):
        """Xout = X Q (FP64; mixed: FP32 off-diagonal blocks; pawfe_rr_rotate)"""
        self._check(self.lib.pawfe_rr_rotate(self._h, int(bool(mixed)), self._ptr(X), int(ldx), self._ptr(Q), self._ptr(Xout),
                                             int(ldo), int(B)), "pawfe_rr_rotate")

    def col_norms(self, prec: int, X, ld: int, B: int, out):
        self._check(self.lib.pawfe_col_norms(self._h, int(prec), self._ptr(X), int(ld), int(B), self._ptr(out)),
                    "pawfe_col_norms")


def context_from_system(sysd, device: int = 0, stream: int = 0, keep_fp64: bool = True) -> Context:
    """Create a context and set up mesh, potential and atoms from a pawfe_inputs.System (data only)."""
    cfg = sysd.cfg
    ctx = Context(device, stream)
    ctx.mesh_create(cfg.ncells, cfg.box, cfg.p, PERIODIC if cfg.bc == "periodic" else DIRICHLET, cfg.kpoint)
    ctx.local_potential_gaussians(sysd.pos, sysd.Z, sysd.sigmaV, keep_fp64)
    ctx.atoms_create(sysd.pos, sysd.proj_l, sysd.proj_m, sysd.proj_sigma, sysd.proj_amp, sysd.rc, sysd.D, sysd.dS)
    return ctx
