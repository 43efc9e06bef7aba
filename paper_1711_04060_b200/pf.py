"""Thin ctypes binding of libpf_b200.so (include/pf.h).  Argument marshalling only: every step of
the hot path runs in the CUDA kernels behind the C ABI.  torch is used for device memory and streams.

The module-level functions carry the names of the C entry points; `Grid` is a convenience owner of
the handle and its workspace tensor.  There is no CPU fallback: if the library is missing or no CUDA
device is present, calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# PF_B200_LIB: another build of the same sources (e.g. the -DPF_EXPERIMENT_PLAIN_DOT measurement of profiles/r2_plain_dot.md)
LIB_PATH = os.environ.get("PF_B200_LIB") or os.path.join(_HERE, "libpf_b200.so")

PF_OK, PF_NOT_CONVERGED, PF_INNER_NOT_CONVERGED = 0, 1, 2
PF_ERR_ARG, PF_ERR_CUDA, PF_ERR_BREAKDOWN, PF_ERR_NONPHYSICAL, PF_ERR_WORKSPACE = -1, -2, -3, -4, -5
PF_BC_DIRICHLET, PF_BC_NEUMANN = 0, 1
(PF_OPT_STENCIL, PF_OPT_OMEGA_PF, PF_OPT_LINEAR_TOL, PF_OPT_LINEAR_MAXIT, PF_OPT_CHECK_INTERVAL,
 PF_OPT_WATER_MOLAR, PF_OPT_MAX_OUTER, PF_OPT_PRECOND, PF_OPT_HISTORY, PF_OPT_KERNELS, PF_OPT_PROFILE,
 PF_OPT_GRAPH, PF_OPT_NORM, PF_OPT_CHARGE_MODEL, PF_OPT_DIAG_FROM_CODE, PF_OPT_SOLVER, PF_OPT_STERIC_MODE,
 PF_OPT_TILE_ROWS, PF_OPT_SEGMENTS) = range(1, 20)
STERIC_SIMULTANEOUS, STERIC_LAGGED = 0, 1
SOLVER_TABLE3, SOLVER_MERGED = 0, 1
CHARGES_DEPOSITED, CHARGES_SINGULAR = 0, 1
NORM_REL_L2, NORM_ABS_INF = 0, 1
STENCIL_AUTO, STENCIL_STORED, STENCIL_ONTHEFLY = 0, 1, 2
KERNELS_AUTO, KERNELS_DIRECT, KERNELS_TILED, KERNELS_COOP = 0, 1, 2, 3

EXPORTS = [
    "pf_grid_create", "pf_grid_set_fixed_nodes", "pf_grid_workspace_bytes", "pf_grid_set_workspace", "pf_grid_set_option",
    "pf_solve_linear", "pf_solve_linear_host", "pf_grid_stage_host", "pf_solve_pf", "pf_fermi_pointwise", "pf_grid_history",
    "pf_grid_linear_iters", "pf_grid_increments", "pf_grid_fault_repeats", "pf_grid_laplace_iters", "pf_grid_stencil", "pf_grid_palette_size", "pf_grid_code_layout", "pf_grid_copy_array",
    "pf_grid_profile", "pf_launch_count", "pf_coop_plan", "pf_tile_plan", "pf_grid_relax", "pf_relax_noalloc", "pf_grid_destroy", "pf_last_error", "pf_version",
]


class pf_bc(ctypes.Structure):
    _fields_ = [("type", ctypes.c_int * 6), ("value", ctypes.c_double * 6)]


class pf_charge(ctypes.Structure):
    _fields_ = [("x", ctypes.c_double), ("y", ctypes.c_double), ("z", ctypes.c_double), ("q", ctypes.c_double)]


class PFError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"pf error {code}: {msg}")
        self.code = code


_lib = None
_vp, _dp, _ip = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)


def load():
    """dlopen the in-tree library; raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1711_04060_b200.build` "
                           "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    L.pf_grid_create.argtypes = [ctypes.POINTER(_vp), ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                 _vp, ctypes.POINTER(pf_charge), ctypes.c_int, ctypes.POINTER(pf_bc), _vp]
    L.pf_grid_create.restype = ctypes.c_int
    L.pf_grid_set_fixed_nodes.argtypes = [_vp, ctypes.POINTER(ctypes.c_longlong), _dp, ctypes.c_int]
    L.pf_grid_workspace_bytes.argtypes = [_vp]
    L.pf_grid_workspace_bytes.restype = ctypes.c_size_t
    L.pf_grid_set_workspace.argtypes = [_vp, _vp, ctypes.c_size_t]
    L.pf_grid_set_option.argtypes = [_vp, ctypes.c_int, ctypes.c_double]
    L.pf_solve_linear.argtypes = [_vp, _vp, _vp, _vp, ctypes.c_double, ctypes.c_int, _ip, _dp, _dp]
    L.pf_solve_linear_host.argtypes = [_vp, _vp, _vp, _vp, ctypes.c_double, ctypes.c_int, _ip, _dp, _dp]
    L.pf_grid_stage_host.argtypes = [_vp, _vp, _vp]
    L.pf_solve_pf.argtypes = [_vp, ctypes.c_int, _dp, _dp, _dp, ctypes.c_double, ctypes.c_double, _vp, _vp, _vp,
                              _ip, _ip]
    L.pf_fermi_pointwise.argtypes = [_vp, ctypes.c_int, _dp, _dp, _dp, _vp, _vp, _vp, _vp, _vp]
    L.pf_grid_history.argtypes = [_vp, _dp, ctypes.c_int]
    L.pf_grid_linear_iters.argtypes = [_vp, _ip, ctypes.c_int]
    L.pf_grid_increments.argtypes = [_vp, _dp, ctypes.c_int]
    L.pf_grid_fault_repeats.argtypes = [_vp]
    L.pf_grid_relax.argtypes = [_vp, ctypes.c_double, _vp, _vp, _dp]
    L.pf_relax_noalloc.argtypes = [ctypes.c_longlong, ctypes.c_double, _vp, _vp, _vp, _vp]
    L.pf_grid_laplace_iters.argtypes = [_vp]
    L.pf_grid_stencil.argtypes = [_vp]
    L.pf_grid_palette_size.argtypes = [_vp]
    L.pf_grid_copy_array.argtypes = [_vp, ctypes.c_int, _vp]
    L.pf_grid_code_layout.argtypes = [_vp, _ip, _ip, ctypes.POINTER(ctypes.c_size_t)]
    L.pf_grid_profile.argtypes = [_vp, _dp, ctypes.POINTER(ctypes.c_longlong)]
    L.pf_launch_count.restype = ctypes.c_longlong
    L.pf_coop_plan.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_size_t, _ip]
    L.pf_tile_plan.argtypes = [ctypes.c_int] * 6 + [_ip]
    L.pf_grid_destroy.argtypes = [_vp]
    L.pf_grid_destroy.restype = None
    L.pf_last_error.argtypes = [_vp]
    L.pf_last_error.restype = ctypes.c_char_p
    L.pf_version.restype = ctypes.c_char_p
    _lib = L
    return L


def _check(handle, rc: int) -> int:
    if rc < 0:
        raise PFError(rc, load().pf_last_error(handle).decode())
    return rc


def _dev_ptr(t: Optional[torch.Tensor], n: Optional[int] = None, dtype=torch.float64) -> Optional[int]:
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise ValueError("expected a contiguous CUDA tensor of dtype %s" % dtype)
    if n is not None and t.numel() != n:
        raise ValueError(f"expected {n} elements, got {t.numel()}")
    return t.data_ptr()


def _host_doubles(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(-1))


# ---- functions named after the C entry points ---------------------------------------------------

def pf_version() -> str:
    return load().pf_version().decode()


def pf_grid_create(nx: int, ny: int, nz: int, h: float, eps_map: torch.Tensor, charges, bc_type, bc_value,
                   stream: Optional[torch.cuda.Stream] = None):
    """eps_map: CUDA float64 tensor of nx*ny*nz (borrowed); charges: (M,4) host array x,y,z,q."""
    L = load()
    ch = np.ascontiguousarray(np.asarray(charges, dtype=np.float64).reshape(-1, 4))
    bc = pf_bc()
    for f in range(6):
        bc.type[f] = int(bc_type[f])
        bc.value[f] = float(bc_value[f])
    handle = _vp()
    s = (stream or torch.cuda.current_stream()).cuda_stream
    rc = L.pf_grid_create(ctypes.byref(handle), nx, ny, nz, float(h), _dev_ptr(eps_map, nx * ny * nz),
                          ch.ctypes.data_as(ctypes.POINTER(pf_charge)) if ch.shape[0] else None, int(ch.shape[0]),
                          ctypes.byref(bc), _vp(s))
    _check(None, rc)
    return handle


def pf_grid_set_fixed_nodes(handle, idx, val) -> None:
    """Omega_f: nodes (linear indices) whose potential is prescribed; call before pf_grid_set_workspace."""
    idx = np.ascontiguousarray(np.asarray(idx, dtype=np.int64).reshape(-1))
    val = _host_doubles(val)
    if idx.size != val.size:
        raise ValueError("idx and val need the same length")
    _check(handle, load().pf_grid_set_fixed_nodes(handle, idx.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)),
                                                  val.ctypes.data_as(_dp), int(idx.size)))


def pf_grid_workspace_bytes(handle) -> int:
    return int(load().pf_grid_workspace_bytes(handle))


def pf_grid_set_workspace(handle, workspace: torch.Tensor) -> None:
    _check(handle, load().pf_grid_set_workspace(handle, _dev_ptr(workspace, dtype=torch.uint8), workspace.numel()))


def pf_grid_set_option(handle, key: int, value: float) -> None:
    _check(handle, load().pf_grid_set_option(handle, int(key), float(value)))


def pf_solve_linear(handle, n: int, rhs: torch.Tensor, x: torch.Tensor, tol: float, maxit: int,
                    sigma: Optional[torch.Tensor] = None, true_residual: bool = True) -> dict:
    it, rr, tr = ctypes.c_int(0), ctypes.c_double(0), ctypes.c_double(0)
    rc = load().pf_solve_linear(handle, _dev_ptr(rhs, n), _dev_ptr(x, n), _dev_ptr(sigma, n), float(tol), int(maxit),
                                ctypes.byref(it), ctypes.byref(rr), ctypes.byref(tr) if true_residual else None)
    _check(handle, rc)
    return dict(status=rc, iters=it.value, relres=rr.value, true_relres=tr.value if true_residual else None)


def pf_solve_linear_host(handle, n: int, rhs_host: torch.Tensor, x_host: torch.Tensor, tol: float, maxit: int,
                         sigma: Optional[torch.Tensor] = None, true_residual: bool = True) -> dict:
    """rhs_host, x_host: CPU float64 tensors (pinned for speed); copies run inside the call."""
    for t in (rhs_host, x_host):
        if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != n:
            raise ValueError("expected contiguous CPU float64 tensors of n elements")
    it, rr, tr = ctypes.c_int(0), ctypes.c_double(0), ctypes.c_double(0)
    rc = load().pf_solve_linear_host(handle, rhs_host.data_ptr(), x_host.data_ptr(), _dev_ptr(sigma, n), float(tol),
                                     int(maxit), ctypes.byref(it), ctypes.byref(rr),
                                     ctypes.byref(tr) if true_residual else None)
    _check(handle, rc)
    return dict(status=rc, iters=it.value, relres=rr.value, true_relres=tr.value if true_residual else None)


def pf_grid_stage_host(handle, n: int, rhs_host: torch.Tensor, x_host: torch.Tensor) -> None:
    """Start the upload of the (pinned) host buffers of the next pf_solve_linear_host on the grid's copy stream."""
    for t in (rhs_host, x_host):
        if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != n:
            raise ValueError("expected contiguous CPU float64 tensors of n elements")
    _check(handle, load().pf_grid_stage_host(handle, rhs_host.data_ptr(), x_host.data_ptr()))


def pf_solve_pf(handle, n: int, valence, bath_conc, radii, l_c: float, tol: float, phi: torch.Tensor,
                conc: Optional[torch.Tensor] = None, steric: Optional[torch.Tensor] = None) -> dict:
    z, cb, a = _host_doubles(valence), _host_doubles(bath_conc), _host_doubles(radii)
    K = z.size
    if cb.size != K or a.size != K + 1:
        raise ValueError("valence/bath_conc need K entries, radii K+1 (water last)")
    outer, lin = ctypes.c_int(0), ctypes.c_int(0)
    rc = load().pf_solve_pf(handle, K, z.ctypes.data_as(_dp), cb.ctypes.data_as(_dp), a.ctypes.data_as(_dp),
                            float(l_c), float(tol), _dev_ptr(phi, n), _dev_ptr(conc, (K + 1) * n),
                            _dev_ptr(steric, n), ctypes.byref(outer), ctypes.byref(lin))
    _check(handle, rc)
    its = (ctypes.c_int * (2 * outer.value + 1))()
    m = load().pf_grid_linear_iters(handle, its, len(its))
    return dict(status=rc, outer_iters=outer.value, linear_iters=lin.value, lin_iters_hist=list(its[:m]),
                incr_hist=pf_grid_increments(handle, outer.value))


def pf_fermi_pointwise(handle, n: int, valence, bath_conc, radii, phi: torch.Tensor,
                       rho=None, sigma=None, steric=None, conc=None) -> None:
    z, cb, a = _host_doubles(valence), _host_doubles(bath_conc), _host_doubles(radii)
    K = z.size
    rc = load().pf_fermi_pointwise(handle, K, z.ctypes.data_as(_dp), cb.ctypes.data_as(_dp), a.ctypes.data_as(_dp),
                                   _dev_ptr(phi, n), _dev_ptr(rho, n), _dev_ptr(sigma, n), _dev_ptr(steric, n),
                                   _dev_ptr(conc, (K + 1) * n))
    _check(handle, rc)


def pf_grid_history(handle, cap: int) -> np.ndarray:
    buf = np.empty(cap, dtype=np.float64)
    m = _check(handle, load().pf_grid_history(handle, buf.ctypes.data_as(_dp), cap))
    return buf[:m]


def pf_grid_increments(handle, cap: int) -> np.ndarray:
    """||Phi - Phi0||_inf of every outer iteration of the last pf_solve_pf."""
    buf = np.empty(max(cap, 1), dtype=np.float64)
    k = _check(handle, load().pf_grid_increments(handle, buf.ctypes.data_as(_dp), int(buf.size)))
    return buf[:k].copy()


def pf_grid_profile(handle) -> dict:
    ms = (ctypes.c_double * 3)()
    cnt = (ctypes.c_longlong * 3)()
    _check(handle, load().pf_grid_profile(handle, ms, cnt))
    return {name: dict(ms=ms[j], launches=cnt[j]) for j, name in enumerate(("k1", "k2", "k3"))}


def pf_launch_count() -> int:
    return int(load().pf_launch_count())


def pf_coop_plan(nx: int, ny: int, nz: int, max_blocks: int = 148, smem_cap: int = 228352) -> Optional[dict]:
    """Brick decomposition of the cooperative kernel (host arithmetic only); None when none fits."""
    out = (ctypes.c_int * 8)()
    if load().pf_coop_plan(nx, ny, nz, max_blocks, smem_cap, out) != PF_OK:
        return None
    keys = ("nbx", "nby", "nbz", "vmax", "hmax", "nhmax", "threads", "smem")
    return dict(zip(keys, list(out)))


def pf_tile_plan(nx: int, ny: int, nz: int, tile_rows: int, sm_count: int = 148, mode: int = -1) -> dict:
    """Decomposition of the persistent tiled kernels (host arithmetic only; include/pf_debug.h)."""
    out = (ctypes.c_int * 9)()
    rc = load().pf_tile_plan(nx, ny, nz, tile_rows, sm_count, mode, out)
    if rc != PF_OK:
        raise PFError(rc, "pf_tile_plan: invalid argument")
    keys = ("mode", "ntx", "ntiles", "depth", "nitems", "zrest", "erest", "q", "blocks")
    return dict(zip(keys, list(out)))


def pf_grid_laplace_iters(handle) -> int:
    return load().pf_grid_laplace_iters(handle)


def pf_grid_relax(handle, n: int, omega_pf: float, phi0: torch.Tensor, phi: torch.Tensor) -> float:
    """Row N5 through pf_solve_pf's own kernel and scratch; phi is relaxed in place, the increment is returned."""
    d = ctypes.c_double(0)
    _check(handle, load().pf_grid_relax(handle, float(omega_pf), _dev_ptr(phi0, n), _dev_ptr(phi, n), ctypes.byref(d)))
    return d.value


def pf_relax_noalloc(n: int, omega_pf: float, phi0: Optional[torch.Tensor], phi: Optional[torch.Tensor],
                     incr_out: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> None:
    """The no-allocation entry point (include/pf_noalloc.h): needs no grid; phi is relaxed in place and the increment
    written to the 1-element CUDA tensor incr_out; only enqueues work on the stream."""
    s = (stream or torch.cuda.current_stream()).cuda_stream
    rc = load().pf_relax_noalloc(int(n), float(omega_pf), None if phi0 is None else phi0.data_ptr(),
                                 None if phi is None else phi.data_ptr(), _dev_ptr(incr_out, 1), _vp(s))
    _check(None, rc)


def pf_grid_fault_repeats(handle) -> int:
    return load().pf_grid_fault_repeats(handle)


def pf_grid_stencil(handle) -> int:
    return load().pf_grid_stencil(handle)


def pf_grid_palette_size(handle) -> int:
    return load().pf_grid_palette_size(handle)


def pf_grid_code_layout(handle) -> dict:
    bits, pitch, nbytes = ctypes.c_int(0), ctypes.c_int(0), ctypes.c_size_t(0)
    _check(handle, load().pf_grid_code_layout(handle, ctypes.byref(bits), ctypes.byref(pitch), ctypes.byref(nbytes)))
    return dict(bits=bits.value, pitch=pitch.value, bytes=nbytes.value)


def pf_grid_copy_array(handle, which: int, n: int) -> torch.Tensor:
    """Copy of an assembled device array (tests): 0 diag, 1..6 off-diagonals, 7 fixed charges, 8 / 11 stencil
    codes (raw bytes), 9 PF1 diag, 10 / 12 coefficient tables (16 doubles)."""
    if which in (8, 11):
        out = torch.empty(pf_grid_code_layout(handle)["bytes"], dtype=torch.uint8, device="cuda")
    elif which in (10, 12):
        out = torch.empty(16, dtype=torch.float64, device="cuda")
    else:
        out = torch.empty(n, dtype=torch.float64, device="cuda")
    _check(handle, load().pf_grid_copy_array(handle, which, out.data_ptr()))
    return out


def decode_offdiagonals(handle, nx: int, ny: int, nz: int, pf1: bool = False):
    """Off-diagonals A1..A6 (numpy, 6 x N) that the on-the-fly stencil codes and table stand for."""
    lay = pf_grid_code_layout(handle)
    raw = pf_grid_copy_array(handle, 11 if pf1 else 8, 0).cpu().numpy()
    tab = pf_grid_copy_array(handle, 12 if pf1 else 10, 0).cpu().numpy()
    dt = np.uint16 if lay["bits"] == 16 else np.uint32
    fb = 2 if lay["bits"] == 16 else 4
    codes = raw[: lay["pitch"] * ny * nz * (lay["bits"] // 8)].view(dt).reshape(nz, ny, lay["pitch"])[:, :, :nx]
    codes = codes.reshape(-1).astype(np.uint32)
    return np.stack([tab[(codes >> (fb * d)) & ((1 << fb) - 1)] for d in range(6)])


def pf_grid_destroy(handle) -> None:
    load().pf_grid_destroy(handle)


# ---- convenience owner ------------------------------------------------------------------------

class Grid:
    """Owns a pf_grid handle, the borrowed eps tensor and the torch-allocated workspace."""

    def __init__(self, nx, ny, nz, h, eps, charges, bc_type, bc_value, stencil=STENCIL_AUTO, kernels=KERNELS_AUTO,
                 options: Optional[dict] = None, stream: Optional[torch.cuda.Stream] = None, fixed_nodes=None):
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: paper_1711_04060_b200 has no CPU fallback")
        self.nx, self.ny, self.nz, self.h = nx, ny, nz, h
        self.n = nx * ny * nz
        self.eps = torch.as_tensor(eps, dtype=torch.float64).reshape(-1).cuda().contiguous()
        self.handle = pf_grid_create(nx, ny, nz, h, self.eps, charges, bc_type, bc_value, stream)
        pf_grid_set_option(self.handle, PF_OPT_STENCIL, stencil)
        if kernels != KERNELS_AUTO:
            pf_grid_set_option(self.handle, PF_OPT_KERNELS, kernels)
        for k, v in (options or {}).items():
            pf_grid_set_option(self.handle, k, v)
        if fixed_nodes is not None:
            pf_grid_set_fixed_nodes(self.handle, fixed_nodes[0], fixed_nodes[1])
        self.workspace = torch.empty(pf_grid_workspace_bytes(self.handle), dtype=torch.uint8, device="cuda")
        pf_grid_set_workspace(self.handle, self.workspace)

    @classmethod
    def from_workload(cls, w, **kw):
        return cls(w.nx, w.ny, w.nz, w.h, w.eps, w.charges, w.bc_type, w.bc_value, **kw)

    def set_option(self, key, value):
        pf_grid_set_option(self.handle, key, value)

    def solve_linear(self, rhs, x=None, tol=1e-10, maxit=10000, sigma=None, true_residual=True):
        rhs = torch.as_tensor(rhs, dtype=torch.float64).reshape(-1).cuda().contiguous()
        x = torch.zeros(self.n, dtype=torch.float64, device="cuda") if x is None else x
        out = pf_solve_linear(self.handle, self.n, rhs, x, tol, maxit, sigma, true_residual)
        out["x"] = x
        return out

    def solve_pf(self, valence, bath_conc, radii, l_c, tol, want_conc=True):
        K = len(valence)
        phi = torch.empty(self.n, dtype=torch.float64, device="cuda")
        conc = torch.empty((K + 1) * self.n, dtype=torch.float64, device="cuda") if want_conc else None
        steric = torch.empty(self.n, dtype=torch.float64, device="cuda") if want_conc else None
        out = pf_solve_pf(self.handle, self.n, valence, bath_conc, radii, l_c, tol, phi, conc, steric)
        out.update(phi=phi, conc=None if conc is None else conc.view(K + 1, self.n), steric=steric)
        return out

    def history(self, cap):
        return pf_grid_history(self.handle, cap)

    def close(self):
        if self.handle is not None:
            pf_grid_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
