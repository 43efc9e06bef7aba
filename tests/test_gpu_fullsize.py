"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (on-the-fly
stencil, tiled TMA kernels chosen by `auto`).  The oracle cannot run these solves to the end in test
time, so the checks are: the first iterations element by element against the oracle (same iterate, same
residual history), and properties that hold at any size evaluated with the ORACLE's operator on the
GPU's result (true residual, fixed-point residuals of the split PF system, physical invariants).
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1711_04060_b200 import workloads as wl  # noqa: E402


@pytest.fixture(scope="module")
def pf():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1711_04060_b200 import build as _build, pf as _pf
    _build.build()      # no-op when libpf_b200.so is newer than its sources; needs nvcc otherwise
    _pf.load()
    return _pf


def rel_l2(a, b):
    d = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (d if d > 0 else 1.0)


def oracle_true_relres(oracle, w, A, b, x):
    r = b - oracle.dia_spmv(w.nx, w.ny, w.nz, A, x)
    return np.sqrt(oracle.dot(r, r)) / np.sqrt(oracle.dot(b, b))


def test_config3_256_bench_configuration(pf, oracle):
    """configs[3] (256^3, 16.8 M unknowns), the bench's dense random right-hand side."""
    w = wl.config3()
    assert w.n == 256 ** 3
    rhs = np.random.default_rng(3).standard_normal(w.n)
    A = oracle.assemble_poisson(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps)
    b = oracle.set_dirichlet(w.nx, w.ny, w.nz, w.bc_type, w.bc_value, rhs.copy())
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY, options={pf.PF_OPT_HISTORY: 256})
    # (1) six iterations element by element
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, rhs, tol=0.0, maxit=6, history=True)
    out = g.solve_linear(rhs, tol=0.0, maxit=6)
    assert out["iters"] == 6 == ref["iters"]
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-12
    assert np.allclose(g.history(7), ref["hist"], rtol=1e-10)
    # sampled entries, one by one
    idx = np.random.default_rng(0).integers(0, w.n, 4096)
    xs = out["x"][torch.as_tensor(idx, device="cuda")].cpu().numpy()
    assert np.allclose(xs, ref["x"][idx], rtol=1e-11, atol=1e-13 * np.abs(ref["x"]).max())
    # (2) the 200 fixed iterations the bench times: the reported residuals are those of the oracle's operator
    out = g.solve_linear(rhs, tol=0.0, maxit=200)
    assert out["status"] == 1 and out["iters"] == 200
    tr = oracle_true_relres(oracle, w, A, b, out["x"].cpu().numpy())
    assert abs(out["true_relres"] - tr) <= 1e-6 * tr
    assert abs(out["relres"] - tr) <= 1e-3 * tr          # recurrence residual tracks the true one
    hist = g.history(201)
    assert hist[200] < 1e-3 * hist[0]                     # it converges
    g.close()


def test_config3_256_solve_to_tolerance(pf, oracle):
    """configs[3] (i): one Jacobi-BiCGSTAB solve to 1e-10, the deposited charges as right-hand side."""
    w = wl.config3()
    rhs = oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges)
    A = oracle.assemble_poisson(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps)
    b = oracle.set_dirichlet(w.nx, w.ny, w.nz, w.bc_type, w.bc_value, rhs.copy())
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY)
    assert np.array_equal(pf.pf_grid_copy_array(g.handle, 0, w.n).cpu().numpy(), A[0])
    assert np.array_equal(pf.pf_grid_copy_array(g.handle, 7, w.n).cpu().numpy(), rhs)
    out = g.solve_linear(rhs, tol=1e-10)
    g.close()
    assert out["status"] == 0, out
    x = out["x"].cpu().numpy()
    tr = oracle_true_relres(oracle, w, A, b, x)
    print(f"256^3 solve: {out['iters']} iterations, true relres gpu {out['true_relres']:.3e} oracle operator {tr:.3e}")
    assert tr <= 1.05e-10 and abs(out["true_relres"] - tr) <= 1e-4 * tr
    assert np.all(x.reshape(w.nz, w.ny, w.nx)[0] == 0.0) and np.all(x.reshape(w.nz, w.ny, w.nx)[-1] == 0.0)


def test_config2_128_pf_properties(pf, oracle):
    """configs[2] (128^3, Na+/Ca2+/Cl-/water, +50 mV): the converged GPU fields satisfy the oracle's
    discrete split system and the physical invariants of Eq (1)."""
    w = wl.config2(volt_mv=50.0)
    sp = w.species
    g = pf.Grid.from_workload(w)
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol)
    psi = pf.pf_grid_copy_array(g.handle, 13, w.n).cpu().numpy()
    g.close()
    assert out["status"] == 0, out
    phi = out["phi"].cpu().numpy()
    res = oracle.pf_residuals(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence,
                              sp.bath_molar, sp.radii, w.l_c, phi, psi)
    print(f"128^3 PF: {out['outer_iters']} outer, {out['linear_iters']} linear iterations, "
          f"fixed-point residuals PF1 {res['res_pf1']:.2e} PF2 {res['res_pf2']:.2e}")
    # the outer loop stops on an increment of 1e-8 with contraction ~0.3: residuals of the order of the tolerance
    assert res["res_pf1"] < 1e-7 and res["res_pf2"] < 1e-7
    conc = out["conc"].cpu().numpy()
    solvent = oracle.solvent_mask(w.eps).astype(bool)
    vol = 4.0 * np.pi * np.asarray(sp.radii) ** 3 / 3.0
    occ = (vol[:, None] * conc).sum(0)
    assert np.all(conc >= 0.0) and np.all(conc[:, ~solvent] == 0.0)
    assert occ.max() < 1.0                                   # excluded volume fraction stays below 1
    assert np.all(conc < 1.0 / vol[:, None])                 # saturation
    # pointwise kernel at the converged potential against the oracle, element by element
    ref = oracle.fermi_pointwise(sp.valence, sp.bath_molar, sp.radii, phi, solvent.astype(np.uint8))
    assert np.allclose(conc, ref["conc"], rtol=1e-10, atol=0)
    assert np.allclose(out["steric"].cpu().numpy(), ref["S"], rtol=1e-10, atol=1e-13)
    z3 = phi.reshape(w.nz, w.ny, w.nx)
    # Dirichlet data (the relaxation w V + (1-w) V of Table 2 step 5 may move V by one rounding)
    assert np.all(z3[0] == 0.0) and np.allclose(z3[-1], w.bc_value[5], rtol=1e-14, atol=0)


# ---- configs[4]: 512^3, 134 M unknowns, one vector = 1.07 GB, workspace 22 GB --------------------------------------
# The oracle needs 3-4 s per iteration here and 7.5 GB per matrix, so both sides run the same small fixed numbers of
# iterations and are compared element by element; the 100 iterations the bench times are
# checked through the oracle's operator.

def test_config4_512_linear(pf, oracle):
    w = wl.config4()
    assert w.n == 512 ** 3
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY, options={pf.PF_OPT_HISTORY: 128})
    # (1) five iterations element by element, residual history, sampled entries one by one
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=0.0, maxit=5, history=True)
    out = g.solve_linear(w.rhs, tol=0.0, maxit=5)
    assert out["iters"] == 5 == ref["iters"]
    x = out["x"].cpu().numpy()
    assert rel_l2(x, ref["x"]) <= 1e-12
    assert np.allclose(g.history(6), ref["hist"], rtol=1e-10)
    idx = np.random.default_rng(0).integers(0, w.n, 4096)
    assert np.allclose(x[idx], ref["x"][idx], rtol=1e-11, atol=1e-13 * np.abs(ref["x"]).max())
    del ref, x
    # (2) assembly: the diagonal bit for bit
    A = oracle.assemble_poisson(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps)
    assert np.array_equal(pf.pf_grid_copy_array(g.handle, 0, w.n).cpu().numpy(), A[0])
    # (3) the 100 fixed iterations of the bench: reported residuals are those of the oracle's operator on the result
    b = oracle.set_dirichlet(w.nx, w.ny, w.nz, w.bc_type, w.bc_value, w.rhs.copy())
    out = g.solve_linear(w.rhs, tol=0.0, maxit=100)
    assert out["status"] == 1 and out["iters"] == 100
    tr = oracle_true_relres(oracle, w, A, b, out["x"].cpu().numpy())
    print(f"512^3: 100 iterations, true relres gpu {out['true_relres']:.6e}, oracle operator {tr:.6e}")
    assert abs(out["true_relres"] - tr) <= 1e-6 * tr
    assert abs(out["relres"] - tr) <= 1e-3 * tr
    hist = g.history(101)
    assert hist[100] < 1e-2 * hist[0]
    g.close()


def test_config4_512_pf_step(pf, oracle):
    """One outer PF step (Na+/Cl-/water, 100 mM) with the same fixed number of iterations per linear solve on both
    sides: phi within 1e-7 (element-wise agreement is far better: the iterates match to rounding), the pointwise
    fields against the oracle on a sample of nodes."""
    w = wl.config4()
    sp = w.species
    lin_it = 4
    ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                          sp.radii, w.l_c, w.nonlinear_tol, lin_tol=0.0, lin_maxit=lin_it, max_outer=1, want_fields=False)
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY,
                              options={pf.PF_OPT_LINEAR_TOL: 0.0, pf.PF_OPT_LINEAR_MAXIT: lin_it, pf.PF_OPT_MAX_OUTER: 1})
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol)
    psi = pf.pf_grid_copy_array(g.handle, 13, w.n).cpu().numpy()
    g.close()
    assert out["status"] == 1 == ref["status"] and out["outer_iters"] == 1 == ref["outer_iters"]
    assert out["linear_iters"] == 3 * lin_it == ref["linear_iters"]
    phi = out["phi"].cpu().numpy()
    d_phi, d_psi = rel_l2(phi, ref["phi"]), rel_l2(psi, ref["psi"])
    print(f"512^3 PF step: rel L2 diff phi {d_phi:.2e}, Psi {d_psi:.2e}, increment gpu {out['incr_hist'][0]:.6e} "
          f"oracle {ref['incr_hist'][0]:.6e}")
    assert d_phi <= 1e-7 and d_psi <= 1e-7
    assert np.isclose(out["incr_hist"][0], ref["incr_hist"][0], rtol=1e-9)
    # pointwise fields at the returned potential: a sample of 2 M nodes through the oracle's Eq (1)
    idx = np.sort(np.random.default_rng(1).choice(w.n, 2_000_000, replace=False))
    solvent = oracle.solvent_mask(w.eps)[idx]
    fr = oracle.fermi_pointwise(sp.valence, sp.bath_molar, sp.radii, phi[idx], solvent)
    conc = out["conc"].cpu().numpy()
    assert np.allclose(conc[:, idx], fr["conc"], rtol=1e-10, atol=0)
    assert np.allclose(out["steric"].cpu().numpy()[idx], fr["S"], rtol=1e-10, atol=1e-13)
    vol = 4.0 * np.pi * np.asarray(sp.radii) ** 3 / 3.0
    assert (vol[:, None] * conc[:, idx]).sum(0).max() < 1.0


# ---- the PF loop through the TILED kernels (the family the bench times) against the oracle, element by element -------

def _pf_tiled_vs_oracle(pf, oracle, w, max_outer, lin_maxit, solver=0):
    sp = w.species
    ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                          sp.radii, w.l_c, w.nonlinear_tol, lin_tol=w.linear_tol, lin_maxit=lin_maxit, max_outer=max_outer,
                          solver=solver)
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY, kernels=pf.KERNELS_TILED,
                              options={pf.PF_OPT_LINEAR_MAXIT: lin_maxit, pf.PF_OPT_MAX_OUTER: max_outer,
                                       pf.PF_OPT_SOLVER: solver})
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol)
    psi = pf.pf_grid_copy_array(g.handle, 13, w.n).cpu().numpy()
    assert pf.pf_grid_fault_repeats(g.handle) == 0         # every solve stayed on the tiled kernels
    g.close()
    assert out["status"] == ref["status"] and out["outer_iters"] == ref["outer_iters"]
    assert abs(out["linear_iters"] - ref["linear_iters"]) <= 0.02 * ref["linear_iters"]
    d = rel_l2(out["phi"].cpu().numpy(), ref["phi"])
    dc = [rel_l2(out["conc"][k].cpu().numpy(), ref["conc"][k]) for k in range(len(sp.valence) + 1)]
    print(f"{w.name}: outer {out['outer_iters']}, linear iterations gpu/oracle {out['linear_iters']}/{ref['linear_iters']}, "
          f"rel L2 diff phi {d:.2e}, Psi {rel_l2(psi, ref['psi']):.2e}, C_k {max(dc):.2e}")
    assert d <= 1e-7 and max(dc) <= 1e-7 and rel_l2(psi, ref["psi"]) <= 1e-7
    assert rel_l2(out["steric"].cpu().numpy(), ref["steric"]) <= 1e-7
    assert np.allclose(out["incr_hist"], ref["incr_hist"], rtol=1e-3)
    return out, ref


def test_pf_tiled_config2_64_against_oracle(pf, oracle):
    """configs[2] geometry at 64^3 (Na+/Ca2+/Cl-/water, +50 mV, lateral Neumann), linear solves to 1e-10, thirty outer
    iterations on both sides (the increment contracts by ~0.95 per iteration: convergence to 1e-8 takes hundreds)."""
    _pf_tiled_vs_oracle(pf, oracle, wl.config2(n=64, volt_mv=50.0), max_outer=30, lin_maxit=10000)


@pytest.mark.parametrize("solver", [0, 1])
def test_pf_tiled_config2_128_truncated_against_oracle(pf, oracle, solver):
    """configs[2] at its own size (128^3), two outer iterations with ten iterations per linear solve on both sides;
    Table 3 and the merged recurrence, each against its oracle counterpart.  (Ten, not more: an unconverged BiCGSTAB
    iterate is an ill-conditioned function of its input -- with 50 iterations per solve the last-bit differences between
    libm's and CUDA's exp in the right-hand sides grow to 1e-7 after one outer iteration and 7e-4 after two, identically
    in the direct and the tiled kernels, while with 10 the fields agree to 3e-12.  Converged solves are compared at
    64^3 above and, through the fixed-point residuals of the oracle's operators, at 128^3 in
    test_config2_128_pf_properties.)"""
    _pf_tiled_vs_oracle(pf, oracle, wl.config2(volt_mv=50.0), max_outer=2, lin_maxit=10, solver=solver)


def test_config3_256_decompositions_and_geometries_same_bits(pf):
    """At the bench's size the persistent kernels get their work from the plans of tests/test_tile_plan.py: 13-row tiles
    -> 80 tiles, mode 2 (a deep lower layer, a shallower upper one, the rest in pieces); 16-row tiles -> 64 tiles, mode 1
    (two layers in step + a rest group).  Whatever the plan and the tile height, the iterates have the same bits as with
    equal chunks (the default is also compared with the oracle above), for both solvers."""
    w = wl.config3()
    rng = np.random.default_rng(31)
    rhs = torch.from_numpy(rng.standard_normal(w.n)).cuda()
    assert pf.pf_tile_plan(256, 256, 256, 13, 148, -1)["mode"] == 2 and pf.pf_tile_plan(256, 256, 256, 16, 148, -1)["mode"] == 1
    for solver in (0, 1):
        ref = None
        for rows, seg, diag in ((0, 0, 1), (0, -1, 1), (16, -1, 1), (16, 0, 2), (13, 2, 2)):
            g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY, kernels=pf.KERNELS_TILED,
                                      options={pf.PF_OPT_SOLVER: solver, pf.PF_OPT_TILE_ROWS: rows, pf.PF_OPT_SEGMENTS: seg,
                                               pf.PF_OPT_DIAG_FROM_CODE: diag, pf.PF_OPT_HISTORY: 64})
            o = g.solve_linear(rhs, tol=0.0, maxit=12, true_residual=False)
            h = g.history(64)
            assert pf.pf_grid_fault_repeats(g.handle) == 0
            g.close()
            if ref is None:
                ref = (o["x"].clone(), h)
                continue
            assert o["iters"] == 12 and torch.equal(o["x"], ref[0]) and np.array_equal(h, ref[1]), (solver, rows, seg, diag)
