"""Pins of the oracle's merged two-reduction BiCGSTAB (oracle/pf_oracle.cpp bicgstab_merged; SURVEY.md 8(d) "fully
merged", 8(f) #3; reading M1 of DESIGN.md).  No paper prints this recurrence, so it is pinned by what the
mathematics fixes: the solution of A x = b (dense LU), the identity it rests on (rho_i = r~.r_i), equivalence
with Table 3 in exact arithmetic (same early history, same solution), and an independent numpy transcription."""
import numpy as np
import pytest

from paper_1711_04060_b200 import workloads as W

D, NEU = W.DIRICHLET, W.NEUMANN


def _random_problem(n, seed):
    rng = np.random.default_rng(seed)
    N = n ** 3
    return rng.choice([2.0, 80.0], size=N), rng.uniform(0.0, 5.0, size=N), rng.standard_normal(N)


@pytest.mark.parametrize("bt,bv", [([D] * 6, [0.3, -0.2, 0.0, 1.0, 0.5, -1.0]),
                                   ([NEU, NEU, NEU, NEU, D, D], [0, 0, 0, 0, 0.0, 2.0])])
@pytest.mark.parametrize("precond", [True, False])
def test_merged_dense_lu_8cubed(oracle, bt, bv, precond):
    """The merged recurrence converges to the solution of A x = b: dense LU with partial pivoting on 8^3."""
    n, h = 8, 0.5
    eps, sigma, rhs = _random_problem(n, 11)
    A = oracle.assemble_poisson(n, n, n, h, bt, bv, eps, sigma)
    b = oracle.set_dirichlet(n, n, n, bt, bv, rhs)
    x_lu = np.linalg.solve(oracle.dia_to_dense(n, n, n, A), b)
    x0 = oracle.set_dirichlet(n, n, n, bt, bv, np.zeros(n ** 3))
    r = oracle.bicgstab_merged(n, n, n, A, b, x0=x0, tol=1e-13, precond=precond)
    assert r["status"] == 0
    assert np.linalg.norm(r["x"] - x_lu) <= 1e-10 * np.linalg.norm(x_lu)
    # r stays the true residual of A x = b while well above the rounding floor (right preconditioning)
    r9 = oracle.bicgstab_merged(n, n, n, A, b, x0=x0, tol=1e-9, precond=precond)
    assert r9["status"] == 0 and r9["relres"] <= 1e-9
    assert abs(r9["relres"] - r9["true_relres"]) <= 1e-3 * r9["relres"]


def _merged_numpy(matvec, b, x0, tol, maxit, keep_bracket=True, record=None):
    """Independent transcription of the merged recurrence (M = I) in numpy, plain dot products.
    keep_bracket=False is SURVEY 8(d)'s rho_i = -omega r~.t (the bracket dropped)."""
    x = x0.copy()
    r = b - matvec(x)
    rt = r.copy()
    bn = np.linalg.norm(b)
    hist = [np.linalg.norm(r) / bn]
    rho = rhat = rt @ r
    p = r.copy()
    v = matvec(p)
    rtv = rt @ v
    for _ in range(maxit):
        alpha = rho / rtv
        s = r - alpha * v
        t = matvec(s)
        omega = (t @ s) / (t @ t)
        rtt = rt @ t
        x = x + alpha * p + omega * s
        r = s - omega * t
        hist.append(np.linalg.norm(r) / bn)
        rho_new = ((rhat - alpha * rtv) if keep_bracket else 0.0) - omega * rtt
        rhat = rt @ r
        if record is not None:
            record.append(abs(rho_new - rhat) / (np.linalg.norm(rt) * np.linalg.norm(r)))
        if hist[-1] <= tol:
            break
        beta = (rho_new / rho) * (alpha / omega)
        rho = rho_new
        p = r + beta * (p - omega * v)
        v = matvec(p)
        rtv = rt @ v
    return x, np.array(hist)


def test_merged_equals_numpy_transcription(oracle):
    n, h = 10, 0.5
    bt, bv = [D] * 6, [0.0] * 6
    eps, sigma, rhs = _random_problem(n, 3)
    A = oracle.assemble_poisson(n, n, n, h, bt, bv, eps, sigma)
    b = oracle.set_dirichlet(n, n, n, bt, bv, rhs)
    mv = lambda u: oracle.dia_spmv(n, n, n, A, u)
    x_np, hist_np = _merged_numpy(mv, b, np.zeros(n ** 3), 1e-10, 500)
    r = oracle.bicgstab_merged(n, n, n, A, b, tol=1e-10, maxit=500, precond=False, history=True)
    assert r["status"] == 0
    m = min(25, len(hist_np), len(r["hist"]))
    assert np.allclose(r["hist"][:m], hist_np[:m], rtol=1e-6)
    assert abs(r["iters"] - (len(hist_np) - 1)) <= max(3, 0.1 * r["iters"])
    assert np.linalg.norm(r["x"] - x_np) <= 1e-8 * np.linalg.norm(x_np)
    # Jacobi = the same recurrence on A D^-1 in y = D x
    rj = oracle.bicgstab_merged(n, n, n, A, b, tol=1e-11, precond=True, history=True)
    mvj = lambda y: oracle.dia_spmv(n, n, n, A, y / A[0])
    y_np, hist_j = _merged_numpy(mvj, b, np.zeros(n ** 3), 1e-11, 500)
    m = min(20, len(hist_j), len(rj["hist"]))
    assert rj["status"] == 0 and np.allclose(rj["hist"][:m], hist_j[:m], rtol=1e-6)
    assert np.linalg.norm(y_np / A[0] - rj["x"]) <= 1e-8 * np.linalg.norm(rj["x"])


@pytest.mark.parametrize("cfg", ["config0_24", "config1_32"])
def test_merged_identity_and_agreement_with_table3(oracle, cfg):
    """(a) The identity the merged form rests on: rho_i = -omega r~.t equals the directly reduced r~.r_i up to the
    rounding of s and r.  (b) Table 3 and the merged form are the same method: same residual history while rounding
    has not separated them, same solution to solver tolerance, iteration counts close."""
    if cfg == "config0_24":
        w = W.config0(n=24)
        rhs = oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges)
    else:
        w = W.config1(n=32, ncharges=60)
        rhs = w.rhs
    A = oracle.assemble_poisson(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps)
    b = oracle.set_dirichlet(w.nx, w.ny, w.nz, w.bc_type, w.bc_value, rhs)
    x0 = oracle.set_dirichlet(w.nx, w.ny, w.nz, w.bc_type, w.bc_value, np.zeros(w.n))
    ref = oracle.bicgstab(w.nx, w.ny, w.nz, A, b, x0=x0, tol=1e-10, history=True)
    mer = oracle.bicgstab_merged(w.nx, w.ny, w.nz, A, b, x0=x0, tol=1e-10, history=True, rho_direct=True)
    assert ref["status"] == 0 and mer["status"] == 0
    assert mer["true_relres"] <= 1.05e-10
    # (b)
    m = 12
    assert np.allclose(mer["hist"][:m], ref["hist"][:m], rtol=1e-8)
    assert np.linalg.norm(mer["x"] - ref["x"]) <= 1e-8 * np.linalg.norm(ref["x"])
    assert abs(mer["iters"] - ref["iters"]) <= max(3, 0.15 * ref["iters"])
    # (a) re-run the recurrence's own rho from the library-level pieces: r~.r_i of the iterates vs the history
    rd = mer["rho_direct"]
    assert np.all(np.isfinite(rd)) and rd[0] == oracle.dot(b - oracle.dia_spmv(w.nx, w.ny, w.nz, A, x0),
                                                          b - oracle.dia_spmv(w.nx, w.ny, w.nz, A, x0))
    # one more solve capped one iteration earlier gives r_i, hence rho_i, of iterate k from outside the solver
    k = 7
    xk = oracle.bicgstab_merged(w.nx, w.ny, w.nz, A, b, x0=x0, tol=0.0, maxit=k)["x"]
    r0 = b - oracle.dia_spmv(w.nx, w.ny, w.nz, A, x0)
    rk = b - oracle.dia_spmv(w.nx, w.ny, w.nz, A, xk)
    scale = np.linalg.norm(r0) * np.linalg.norm(rk)
    assert abs(oracle.dot(r0, rk) - rd[k]) <= 1e-9 * scale       # true residual of x_k vs recurrence residual


def test_merged_rho_identity_in_the_recurrence(oracle):
    """Reading M1: rho_i = (rhat_{i-1} - alpha r~.v) - omega r~.t tracks the directly reduced r~.r_i to rounding
    for the whole solve, in the oracle and in an independent numpy transcription; with the bracket dropped (exact
    arithmetic says it is 0) the error of rho is never corrected, grows relative to |r~||r_i| as the residual
    shrinks, and the solve stalls -- which is why the oracle keeps the bracket."""
    n, h = 12, 0.5
    bt, bv = [D] * 6, [0.0] * 6
    eps, sigma, rhs = _random_problem(n, 5)
    A = oracle.assemble_poisson(n, n, n, h, bt, bv, eps, sigma)
    b = oracle.set_dirichlet(n, n, n, bt, bv, rhs)
    mv = lambda y: oracle.dia_spmv(n, n, n, A, y / A[0])
    with_b, without_b = [], []
    _, hist_with = _merged_numpy(mv, b, np.zeros(n ** 3), 1e-12, 300, True, with_b)
    _, hist_without = _merged_numpy(mv, b, np.zeros(n ** 3), 1e-12, 300, False, without_b)
    assert hist_with[-1] <= 1e-12 and max(with_b) <= 1e-12           # tracks r~.r_i down to convergence
    assert max(without_b) >= 1e3 * max(with_b)                       # the dropped bracket is what corrects rho
    out = oracle.bicgstab_merged(n, n, n, A, b, tol=1e-12, rho_direct=True, history=True)
    assert out["status"] == 0
    # the oracle's own rho against r~.r_i, both relative to |r~| |r_i| (|r~| = |r_0| = hist[0] |b|, |r_i| = hist[i] |b|)
    bn2 = oracle.dot(b, b)
    scale = out["hist"][0] * out["hist"][1:] * bn2
    err = np.abs(out["rho_rec"][1:] - out["rho_direct"][1:]) / scale
    assert err.max() <= 1e-12
    assert abs(out["iters"] - (len(hist_with) - 1)) <= max(3, 0.15 * out["iters"])


def test_merged_degenerate_cases(oracle):
    n, h = 8, 0.5
    bt, bv = [D] * 6, [0.0] * 6
    eps, sigma, rhs = _random_problem(n, 2)
    A = oracle.assemble_poisson(n, n, n, h, bt, bv, eps, sigma)
    b = oracle.set_dirichlet(n, n, n, bt, bv, rhs)
    z = oracle.bicgstab_merged(n, n, n, A, np.zeros(n ** 3))
    assert z["status"] == 0 and z["iters"] == 0 and np.all(z["x"] == 0)
    m0 = oracle.bicgstab_merged(n, n, n, A, b, maxit=0)
    assert m0["status"] == 1 and m0["iters"] == 0
    sol = oracle.bicgstab_merged(n, n, n, A, b, tol=1e-13)["x"]
    w = oracle.bicgstab_merged(n, n, n, A, b, x0=sol, tol=1e-8)
    assert w["status"] == 0 and w["iters"] == 0
    fixed = oracle.bicgstab_merged(n, n, n, A, b, tol=0.0, maxit=7)
    assert fixed["status"] == 1 and fixed["iters"] == 7
    bad = b.copy(); bad[3 + n * (3 + n * 3)] = np.nan
    assert oracle.bicgstab_merged(n, n, n, A, bad, tol=1e-6, maxit=10)["status"] == -3


def test_merged_through_solve_linear_and_pf(oracle):
    """The library-level calls route to the merged solver: same solution as Table 3 to solver tolerance; the PF
    loop converges to the same fields (1e-7) with it."""
    w = W.config1(n=24, ncharges=40)
    a = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=1e-11)
    m = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=1e-11, solver=oracle.SOLVER_MERGED)
    assert a["status"] == 0 and m["status"] == 0
    assert np.linalg.norm(a["x"] - m["x"]) <= 1e-8 * np.linalg.norm(a["x"])
    w = W.config0(n=16)
    sp = w.species
    pa = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                         sp.radii, w.l_c, 1e-8)
    pm = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                         sp.radii, w.l_c, 1e-8, solver=oracle.SOLVER_MERGED)
    assert pa["status"] == 0 and pm["status"] == 0 and pa["outer_iters"] == pm["outer_iters"]
    assert np.linalg.norm(pa["phi"] - pm["phi"]) <= 1e-7 * np.linalg.norm(pa["phi"])
