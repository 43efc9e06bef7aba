"""ctypes wrapper of the CPU oracle (oracle/pf_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It never imports the CUDA
package and the CUDA package never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pf_oracle.cpp")
_LIB = os.path.join(_HERE, "libpf_oracle.so")
_lib = None

c_dp = ctypes.POINTER(ctypes.c_double)
c_ip = ctypes.POINTER(ctypes.c_int)
c_u8p = ctypes.POINTER(ctypes.c_uint8)


def _sanitized() -> bool:
    return os.environ.get("PF_ORACLE_SANITIZE", "") not in ("", "0")


def build(force: bool = False) -> str:
    """Compile the oracle: g++ -O2 -ffp-contract=off (every operation rounded as written).

    PF_ORACLE_SANITIZE=1 builds (and lib() then loads) a second library with -fsanitize=address,undefined; the
    interpreter then needs the sanitizer runtime preloaded, see profiles/r2_sanitizer.md for the command."""
    if _sanitized():
        out = os.path.join(_HERE, "libpf_oracle_san.so")
        if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
            cmd = ["g++", "-std=c++17", "-O1", "-g", "-fno-omit-frame-pointer", "-ffp-contract=off",
                   "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fPIC", "-shared", _SRC, "-o", out]
            subprocess.run(cmd, check=True)
        return out
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.pfo_kappa.restype = ctypes.c_double
        _lib.pfo_kT_over_e_volt.restype = ctypes.c_double
        _lib.pfo_molar_to_per_A3.restype = ctypes.c_double
        _lib.pfo_dot.restype = ctypes.c_double
        _lib.pfo_coulomb_potential.restype = ctypes.c_double
        _lib.pfo_coulomb_gradient.restype = ctypes.c_double
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(c_dp)


def _i(a):
    return None if a is None else a.ctypes.data_as(c_ip)


def _u8(a):
    return None if a is None else a.ctypes.data_as(c_u8p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _bc(bc_type, bc_value):
    return np.ascontiguousarray(bc_type, dtype=np.int32), np.ascontiguousarray(bc_value, dtype=np.float64)


def kappa() -> float:
    return lib().pfo_kappa()


def kT_over_e_volt() -> float:
    return lib().pfo_kT_over_e_volt()


def molar_to_per_A3() -> float:
    return lib().pfo_molar_to_per_A3()


def dot(a, b) -> float:
    a = _f64(a)
    b = _f64(b)
    return lib().pfo_dot(ctypes.c_int64(a.size), _d(a), _d(b))


def _fix(fixed_nodes, n):
    """(mask uint8[n], values float64[n]) of Omega_f from (indices, values), or (None, None)."""
    if fixed_nodes is None:
        return None, None
    idx, val = fixed_nodes
    mask = np.zeros(n, dtype=np.uint8)
    vals = np.zeros(n)
    mask[np.asarray(idx, dtype=np.int64)] = 1
    vals[np.asarray(idx, dtype=np.int64)] = np.asarray(val, dtype=np.float64)
    return mask, vals


def assemble_poisson(nx, ny, nz, h, bc_type, bc_value, eps, sigma=None, fixed_nodes=None) -> np.ndarray:
    """Rows of -div(eps grad u) + sigma u in the paper's A0..A6 format; returns (7, N)."""
    n = nx * ny * nz
    t, v = _bc(bc_type, bc_value)
    eps = _f64(eps)
    sigma = None if sigma is None else _f64(sigma)
    A = np.empty((7, n), dtype=np.float64)
    fm, fv = _fix(fixed_nodes, n)
    lib().pfo_assemble_poisson(nx, ny, nz, ctypes.c_double(h), _i(t), _d(v), _d(eps), _d(sigma), _d(A), _u8(fm), _d(fv))
    return A


def solvent_mask(eps) -> np.ndarray:
    eps = _f64(eps)
    m = np.empty(eps.size, dtype=np.uint8)
    lib().pfo_solvent_mask(ctypes.c_int64(eps.size), _d(eps), _u8(m))
    return m


def assemble_pf1(nx, ny, nz, h, bc_type, bc_value, eps, solvent, lc) -> np.ndarray:
    n = nx * ny * nz
    t, v = _bc(bc_type, bc_value)
    eps = _f64(eps)
    solvent = np.ascontiguousarray(solvent, dtype=np.uint8)
    A = np.empty((7, n), dtype=np.float64)
    lib().pfo_assemble_pf1(nx, ny, nz, ctypes.c_double(h), _i(t), _d(v), _d(eps), _u8(solvent),
                           ctypes.c_double(lc), _d(A))
    return A


def dia_spmv(nx, ny, nz, A, x) -> np.ndarray:
    A = _f64(A)
    x = _f64(x)
    y = np.empty(nx * ny * nz, dtype=np.float64)
    lib().pfo_dia_spmv(nx, ny, nz, _d(A), _d(x), _d(y))
    return y


def set_dirichlet(nx, ny, nz, bc_type, bc_value, x, fixed_nodes=None) -> np.ndarray:
    t, v = _bc(bc_type, bc_value)
    x = _f64(x).copy()
    fm, fv = _fix(fixed_nodes, nx * ny * nz)
    lib().pfo_set_dirichlet(nx, ny, nz, _i(t), _d(v), _d(x), _u8(fm), _d(fv))
    return x


def deposit_charges(nx, ny, nz, h, charges) -> np.ndarray:
    ch = _f64(charges).reshape(-1, 4)
    b = np.zeros(nx * ny * nz, dtype=np.float64)
    lib().pfo_deposit_charges(nx, ny, nz, ctypes.c_double(h), _d(ch), int(ch.shape[0]), _d(b))
    return b


NORM_REL_L2, NORM_ABS_INF = 0, 1     # stopping test: BASELINE's relative 2-norm / the paper's absolute maximum norm
SOLVER_TABLE3, SOLVER_MERGED = 0, 1  # Table 3 as written / the merged two-reduction rearrangement (reading M1)
STERIC_SIMULTANEOUS, STERIC_LAGGED = 0, 1   # Eq (1) solved per node (Q11) / S^trc from the previous outer iteration (G1)


def bicgstab(nx, ny, nz, A, b, x0=None, tol=1e-10, maxit=10000, precond=True, history=False, norm=NORM_REL_L2):
    """Table 3 (+Jacobi).  Returns dict(x, status, iters, relres, true_relres[, hist])."""
    A = _f64(A)
    b = _f64(b)
    n = nx * ny * nz
    x = np.zeros(n) if x0 is None else _f64(x0).copy()
    it = ctypes.c_int(0)
    rr = ctypes.c_double(0)
    tr = ctypes.c_double(0)
    hist = np.full(maxit + 1, np.nan) if history else None
    st = lib().pfo_bicgstab(nx, ny, nz, _d(A), _d(b), _d(x), ctypes.c_double(tol), int(maxit),
                            int(bool(precond)), ctypes.byref(it), ctypes.byref(rr), ctypes.byref(tr), _d(hist),
                            int(norm))
    out = dict(x=x, status=st, iters=it.value, relres=rr.value, true_relres=tr.value)
    if history:
        out["hist"] = hist[: it.value + 1]
    return out


def bicgstab_merged(nx, ny, nz, A, b, x0=None, tol=1e-10, maxit=10000, precond=True, history=False, norm=NORM_REL_L2,
                    rho_direct=False):
    """The merged two-reduction BiCGSTAB (reading M1; SURVEY 8(d) "fully merged").  Same outputs as bicgstab();
    with rho_direct=True also out["rho_rec"][i] = the rho_i the recurrence used, (rhat_{i-1} - alpha r~.v) - omega r~.t,
    and out["rho_direct"][i] = the directly reduced r~.r_i of every iterate."""
    A = _f64(A)
    b = _f64(b)
    n = nx * ny * nz
    x = np.zeros(n) if x0 is None else _f64(x0).copy()
    it = ctypes.c_int(0)
    rr = ctypes.c_double(0)
    tr = ctypes.c_double(0)
    hist = np.full(maxit + 1, np.nan) if history else None
    rd = np.full(maxit + 1, np.nan) if rho_direct else None
    rc = np.full(maxit + 1, np.nan) if rho_direct else None
    st = lib().pfo_bicgstab_merged(nx, ny, nz, _d(A), _d(b), _d(x), ctypes.c_double(tol), int(maxit),
                                   int(bool(precond)), ctypes.byref(it), ctypes.byref(rr), ctypes.byref(tr), _d(hist),
                                   int(norm), _d(rc), _d(rd))
    out = dict(x=x, status=st, iters=it.value, relres=rr.value, true_relres=tr.value)
    if history:
        out["hist"] = hist[: it.value + 1]
    if rho_direct:
        out["rho_direct"] = rd[: it.value + 1]
        out["rho_rec"] = rc[: it.value + 1]
    return out


def solve_linear(nx, ny, nz, h, bc_type, bc_value, eps, rhs, x0=None, sigma=None, tol=1e-10,
                 maxit=10000, precond=True, history=False, norm=NORM_REL_L2, fixed_nodes=None, solver=SOLVER_TABLE3):
    """What pf_solve_linear computes: the grid's Poisson operator, Dirichlet data forced.
    solver: SOLVER_TABLE3 (Table 3 of the paper) or SOLVER_MERGED (the two-reduction rearrangement, reading M1)."""
    n = nx * ny * nz
    t, v = _bc(bc_type, bc_value)
    eps = _f64(eps)
    rhs = _f64(rhs)
    sigma = None if sigma is None else _f64(sigma)
    x = np.zeros(n) if x0 is None else _f64(x0).copy()
    it = ctypes.c_int(0)
    rr = ctypes.c_double(0)
    tr = ctypes.c_double(0)
    hist = np.full(maxit + 1, np.nan) if history else None
    fm, fv = _fix(fixed_nodes, n)
    st = lib().pfo_solve_linear(nx, ny, nz, ctypes.c_double(h), _i(t), _d(v), _d(eps), _d(sigma), _d(rhs),
                                _d(x), ctypes.c_double(tol), int(maxit), int(bool(precond)),
                                ctypes.byref(it), ctypes.byref(rr), ctypes.byref(tr), _d(hist), int(norm),
                                _u8(fm), _d(fv), int(solver))
    out = dict(x=x, status=st, iters=it.value, relres=rr.value, true_relres=tr.value)
    if history:
        out["hist"] = hist[: it.value + 1]
    return out


def fermi_pointwise(valence, bath_molar, radii, phi, solvent=None, water_molar=55.5):
    """Eq (1) solved per node.  Returns dict(rho, sigma, S, conc[(K+1),N], gammaB, status)."""
    valence = _f64(valence)
    bath = _f64(bath_molar)
    radii = _f64(radii)
    K = valence.size
    phi = _f64(phi).reshape(-1)
    n = phi.size
    solvent = np.ones(n, dtype=np.uint8) if solvent is None else np.ascontiguousarray(solvent, dtype=np.uint8)
    rho = np.empty(n)
    sigma = np.empty(n)
    S = np.empty(n)
    conc = np.empty((K + 1, n))
    gB = ctypes.c_double(0)
    st = lib().pfo_fermi_pointwise(int(K), _d(valence), _d(bath), _d(radii), ctypes.c_double(water_molar),
                                   ctypes.c_int64(n), _d(phi), _u8(solvent), _d(rho), _d(sigma), _d(S),
                                   _d(conc), ctypes.byref(gB))
    return dict(rho=rho, sigma=sigma, S=S, conc=conc, gammaB=gB.value, status=st)


def solve_pf(nx, ny, nz, h, bc_type, bc_value, eps, charges, valence, bath_molar, radii, l_c, tol,
             omega_pf=0.3, lin_tol=1e-10, lin_maxit=10000, max_outer=200, water_molar=55.5, norm=NORM_REL_L2,
             fixed_override=None, fixed_nodes=None, solver=SOLVER_TABLE3, want_fields=True, steric_mode=STERIC_SIMULTANEOUS):
    """The outer loop of Table 2 / Table 4 (R5).  want_fields=False skips the final evaluation of C_k and S^trc
    (out["conc"], out["steric"] are then None): at 512^3 it costs a minute and 4 GB that a truncated run does not need."""
    n = nx * ny * nz
    t, v = _bc(bc_type, bc_value)
    eps = _f64(eps)
    ch = _f64(charges).reshape(-1, 4)
    valence = _f64(valence)
    bath = _f64(bath_molar)
    radii = _f64(radii)
    K = valence.size
    phi = np.zeros(n)
    psi = np.zeros(n)
    conc = np.zeros((K + 1, n)) if want_fields else None
    steric = np.zeros(n) if want_fields else None
    outer = ctypes.c_int(0)
    lin = ctypes.c_int(0)
    cap = 2 * max_outer + 1
    lhist = np.zeros(cap, dtype=np.int32)
    ihist = np.zeros(max_outer, dtype=np.float64)
    fm, fv = _fix(fixed_nodes, n)
    st = lib().pfo_solve_pf(nx, ny, nz, ctypes.c_double(h), _i(t), _d(v), _d(eps), _d(ch), int(ch.shape[0]),
                            int(K), _d(valence), _d(bath), _d(radii), ctypes.c_double(water_molar),
                            ctypes.c_double(l_c), ctypes.c_double(tol), ctypes.c_double(omega_pf),
                            ctypes.c_double(lin_tol), int(lin_maxit), int(max_outer), int(norm),
                            _d(phi), _d(psi), _d(conc), _d(steric), ctypes.byref(outer), ctypes.byref(lin),
                            _i(lhist), int(cap), _d(ihist), _d(None if fixed_override is None else _f64(fixed_override)),
                            _u8(fm), _d(fv), int(solver), int(steric_mode))
    return dict(phi=phi, psi=psi, conc=conc, steric=steric, status=st, outer_iters=outer.value,
                linear_iters=lin.value, lin_iters_hist=lhist[: 2 * outer.value + 1].copy(),
                incr_hist=ihist[: outer.value].copy())


def pf_residuals(nx, ny, nz, h, bc_type, bc_value, eps, charges, valence, bath_molar, radii, l_c,
                 phi, psi, water_molar=55.5):
    t, v = _bc(bc_type, bc_value)
    eps = _f64(eps)
    ch = _f64(charges).reshape(-1, 4)
    valence = _f64(valence)
    bath = _f64(bath_molar)
    radii = _f64(radii)
    phi = _f64(phi)
    psi = _f64(psi)
    r1 = ctypes.c_double(0)
    r2 = ctypes.c_double(0)
    st = lib().pfo_pf_residuals(nx, ny, nz, ctypes.c_double(h), _i(t), _d(v), _d(eps), _d(ch), int(ch.shape[0]),
                                int(valence.size), _d(valence), _d(bath), _d(radii), ctypes.c_double(water_molar),
                                ctypes.c_double(l_c), _d(phi), _d(psi), ctypes.byref(r1), ctypes.byref(r2))
    return dict(status=st, res_pf1=r1.value, res_pf2=r2.value)


def coulomb_potential(charges, eps_m, x, y, z) -> float:
    ch = _f64(charges).reshape(-1, 4)
    return lib().pfo_coulomb_potential(_d(ch), int(ch.shape[0]), ctypes.c_double(eps_m), ctypes.c_double(x),
                                       ctypes.c_double(y), ctypes.c_double(z))


def coulomb_gradient(charges, eps_m, x, y, z, axis) -> float:
    ch = _f64(charges).reshape(-1, 4)
    return lib().pfo_coulomb_gradient(_d(ch), int(ch.shape[0]), ctypes.c_double(eps_m), ctypes.c_double(x),
                                      ctypes.c_double(y), ctypes.c_double(z), int(axis))


def interface_rhs(nx, ny, nz, h, eps, solvent, J) -> np.ndarray:
    """b^IF from the flux jumps J (6 x N, stored at the Omega_m node of each interface face)."""
    b = np.zeros(nx * ny * nz)
    lib().pfo_interface_rhs(nx, ny, nz, ctypes.c_double(h), _d(_f64(eps)),
                            _u8(np.ascontiguousarray(solvent, dtype=np.uint8)), _d(_f64(J).reshape(-1)), _d(b))
    return b


def singular_setup(nx, ny, nz, h, eps, charges, lin_tol=1e-10, lin_maxit=10000, want_jumps=False):
    """phi^L, phi* (on Omega_m), b^IF of the singular-charge decomposition (Eqs 5-10)."""
    n = nx * ny * nz
    ch = _f64(charges).reshape(-1, 4)
    phiL, phistar, bIF = np.zeros(n), np.zeros(n), np.zeros(n)
    J = np.zeros(6 * n) if want_jumps else None
    it = ctypes.c_int(0)
    st = lib().pfo_singular_setup(nx, ny, nz, ctypes.c_double(h), _d(_f64(eps)), _d(ch), int(ch.shape[0]),
                                  ctypes.c_double(lin_tol), int(lin_maxit), _d(phiL), _d(phistar), _d(bIF), _d(J),
                                  ctypes.byref(it))
    out = dict(status=st, phiL=phiL, phistar=phistar, bIF=bIF, laplace_iters=it.value)
    if want_jumps:
        out["J"] = J.reshape(6, n)
    return out


def dia_to_dense(nx, ny, nz, A) -> np.ndarray:
    A = _f64(A)
    n = nx * ny * nz
    D = np.empty((n, n))
    lib().pfo_dia_to_dense(nx, ny, nz, _d(A), _d(D))
    return D


def dense_lu_solve(dense, b) -> np.ndarray:
    a = _f64(dense).copy()
    b = _f64(b)
    n = b.size
    x = np.empty(n)
    rc = lib().pfo_dense_lu_solve(ctypes.c_int64(n), _d(a), _d(b), _d(x))
    if rc:
        raise RuntimeError("singular matrix in oracle dense LU")
    return x
