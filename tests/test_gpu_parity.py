"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are BASELINE.json's: linear solves -- relative L2 difference
of the potential <= 1e-9, true relative residual <= 1e-10, iteration counts within +-2 %; assembly
and index work bit-exact; full PF -- relative L2 difference of phi and of each C_k <= 1e-7.
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
    _pf.load()          # fails loudly if the library has not been built
    return _pf


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64).reshape(-1)
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    d = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (d if d > 0 else 1.0)


def ragged_workload(nx=37, ny=20, nz=11, seed=7, mixed_bc=True):
    """Small box whose sizes are multiples of nothing, two-valued eps, Neumann + Dirichlet faces."""
    rng = wl.SplitMix64(seed)
    eps = wl.sphere_eps(rng, nx, ny, nz, 0.5, fill=0.3, r_lo=1.0, r_hi=2.5)
    n = nx * ny * nz
    rhs = np.array([rng.uniform_range(-1.0, 1.0) for _ in range(n)])
    if mixed_bc:
        t = np.array([wl.NEUMANN, wl.DIRICHLET, wl.NEUMANN, wl.NEUMANN, wl.DIRICHLET, wl.DIRICHLET], dtype=np.int32)
        v = np.array([0.0, 0.7, 0.0, 0.0, -0.3, 1.9])
    else:
        t = np.zeros(6, dtype=np.int32)
        v = np.zeros(6)
    return wl.Workload("ragged", nx, ny, nz, 0.5, eps, np.zeros((0, 4)), t, v, rhs=rhs)


# ---- rows L1, L2: assembly, bit-exact -------------------------------------------------------------

@pytest.mark.parametrize("which", ["cfg0", "cfg2_small", "cfg3_64", "ragged"])
def test_assembly_bit_exact(pf, oracle, which):
    # cfg3_64: 1536 charges, chunks with and without node conflicts in the parallel in-order deposition
    w = {"cfg0": lambda: wl.config0(), "cfg2_small": lambda: wl.config2(n=32, volt_mv=50.0),
         "cfg3_64": lambda: wl.config3(n=64), "ragged": lambda: ragged_workload()}[which]()
    A = oracle.assemble_poisson(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps)
    fixed = oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges)
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_STORED)
    assert np.array_equal(pf.pf_grid_copy_array(g.handle, 0, w.n).cpu().numpy(), A[0])
    for d in range(1, 7):
        assert np.array_equal(pf.pf_grid_copy_array(g.handle, d, w.n).cpu().numpy(), A[d]), f"A{d}"
    assert np.array_equal(pf.pf_grid_copy_array(g.handle, 7, w.n).cpu().numpy(), fixed)
    g.close()
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY)
    assert pf.pf_grid_stencil(g.handle) == 2 and pf.pf_grid_palette_size(g.handle) == 2
    assert pf.pf_grid_code_layout(g.handle)["bits"] == 16
    assert np.array_equal(pf.pf_grid_copy_array(g.handle, 0, w.n).cpu().numpy(), A[0])
    # the packed stencil codes + coefficient table stand for exactly the oracle's A1..A6
    offd = pf.decode_offdiagonals(g.handle, w.nx, w.ny, w.nz)
    for d in range(1, 7):
        assert np.array_equal(offd[d - 1], A[d]), f"decoded A{d}"
    g.close()


@pytest.mark.parametrize("levels", [3, 4])
def test_assembly_codes_four_level_map(pf, oracle, levels):
    """Maps with 3 or 4 distinct eps values use 32-bit codes (4-bit fields); decoded rows and the PF1
    operator are bit-exact, and a solve through the tiled kernels matches the oracle."""
    w = ragged_workload(nx=40, ny=18, nz=12, seed=21)
    rng = wl.SplitMix64(22)
    vals = [2.0, 4.0, 20.0, 78.5][:levels]
    w.eps = np.array([vals[int(rng.uniform() * levels) % levels] for _ in range(w.n)])
    A = oracle.assemble_poisson(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps)
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY, kernels=2)
    assert pf.pf_grid_code_layout(g.handle)["bits"] == 32 and pf.pf_grid_palette_size(g.handle) == levels
    offd = pf.decode_offdiagonals(g.handle, w.nx, w.ny, w.nz)
    for d in range(1, 7):
        assert np.array_equal(offd[d - 1], A[d]), f"decoded A{d}"
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=1e-10)
    out = g.solve_linear(w.rhs, tol=1e-10)
    assert out["status"] == 0 and abs(out["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9
    g.close()


def test_assembly_pf1_codes(pf, oracle):
    """PF1 operator (row N2): diagonal and decoded off-diagonals bit-exact after a (capped) PF solve."""
    w = wl.config0()
    sp = w.species
    solvent = oracle.solvent_mask(w.eps)
    A1 = oracle.assemble_pf1(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, solvent, w.l_c)
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_ONTHEFLY,
                              options={pf.PF_OPT_MAX_OUTER: 1, pf.PF_OPT_LINEAR_MAXIT: 2})
    g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, want_conc=False)
    assert np.array_equal(pf.pf_grid_copy_array(g.handle, 9, w.n).cpu().numpy(), A1[0])
    offd = pf.decode_offdiagonals(g.handle, w.nx, w.ny, w.nz, pf1=True)
    for d in range(1, 7):
        assert np.array_equal(offd[d - 1], A1[d]), f"decoded PF1 A{d}"
    g.close()


def test_palette_overflow_falls_back_to_stored(pf, oracle):
    w = ragged_workload(mixed_bc=False)
    rng = wl.SplitMix64(11)
    w.eps = np.array([rng.uniform_range(2.0, 80.0) for _ in range(w.n)])   # every node its own eps
    g = pf.Grid.from_workload(w)
    assert pf.pf_grid_stencil(g.handle) == 1 and pf.pf_grid_palette_size(g.handle) > 4
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=1e-10)
    out = g.solve_linear(w.rhs, tol=1e-10)
    assert out["status"] == 0 and abs(out["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9
    g.close()


# ---- rows L3-L8: linear solves ------------------------------------------------------------------------

def _linear_case(pf, oracle, w, stencil, kernels=0, precond=True, sigma=None, tol=1e-10, x0=None, maxit=10000):
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, x0=x0, sigma=sigma, tol=tol,
                              maxit=maxit, precond=precond, history=True)
    g = pf.Grid.from_workload(w, stencil=stencil, kernels=kernels,
                              options={pf.PF_OPT_PRECOND: 1 if precond else 0, pf.PF_OPT_HISTORY: maxit + 1})
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda") if x0 is None else torch.tensor(x0, device="cuda")
    sg = None if sigma is None else torch.tensor(sigma, device="cuda")
    out = g.solve_linear(w.rhs, x=x, tol=tol, maxit=maxit, sigma=sg)
    hist = g.history(maxit + 1)
    out["fault_repeats"] = pf.pf_grid_fault_repeats(g.handle)
    g.close()
    return ref, out, hist


@pytest.mark.parametrize("stencil", [1, 2])
def test_linear_config1_64(pf, oracle, stencil):
    """BASELINE configs[1]: 64^3, random-sphere eps 2/80, 500 Gaussian charges, tol 1e-10."""
    w = wl.config1()
    ref, out, hist = _linear_case(pf, oracle, w, stencil)
    assert ref["status"] == 0 and out["status"] == 0
    assert abs(out["iters"] - ref["iters"]) <= 0.02 * ref["iters"], (out["iters"], ref["iters"])
    assert out["true_relres"] <= 1e-10 * 1.0000001 or out["true_relres"] <= 1.05e-10
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9
    # the residual histories track each other while both run
    m = min(len(hist), len(ref["hist"]))
    assert m > 10 and np.allclose(hist[: m // 2], ref["hist"][: m // 2], rtol=1e-6)


@pytest.mark.parametrize("stencil", [1, 2])
@pytest.mark.parametrize("precond", [True, False])
def test_linear_ragged_mixed_bc(pf, oracle, stencil, precond):
    w = ragged_workload()
    ref, out, _ = _linear_case(pf, oracle, w, stencil, precond=precond)
    assert ref["status"] == 0 and out["status"] == 0
    assert abs(out["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    assert out["true_relres"] <= 1.05e-10
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9


@pytest.mark.parametrize("stencil", [1, 2])
@pytest.mark.parametrize("precond", [True, False])
def test_tiled_kernels_ragged_even(pf, oracle, stencil, precond):
    """Partial tiles in x and y, several z chunks, mixed bc: tiled == direct bit for bit, both == oracle."""
    w = ragged_workload(nx=70, ny=37, nz=19, seed=9)
    ref, out_t, hist_t = _linear_case(pf, oracle, w, stencil, kernels=2, precond=precond)
    _, out_d, hist_d = _linear_case(pf, oracle, w, stencil, kernels=1, precond=precond)
    assert out_t["status"] == 0 and out_t["iters"] == out_d["iters"] and out_t["fault_repeats"] == 0
    assert torch.equal(out_t["x"], out_d["x"])
    assert np.array_equal(hist_t, hist_d)
    assert abs(out_t["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    assert out_t["true_relres"] <= 1.05e-10
    assert rel_l2(out_t["x"].cpu().numpy(), ref["x"]) <= 1e-9


def test_tiled_kernels_neumann_channel(pf, oracle):
    """configs[3] geometry at 64^3 (lateral Neumann, Dirichlet 0/V in z, charges as RHS), tiled kernels."""
    w = wl.config3(n=64)
    w.rhs = oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges)
    w.bc_value = w.bc_value.copy(); w.bc_value[5] = 1.9
    ref, out, _ = _linear_case(pf, oracle, w, 2, kernels=2)
    assert ref["status"] == 0 and out["status"] == 0
    assert abs(out["iters"] - ref["iters"]) <= 0.02 * ref["iters"], (out["iters"], ref["iters"])
    assert out["true_relres"] <= 1.05e-10
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9


def test_linear_with_sigma_and_warm_start(pf, oracle):
    w = ragged_workload()
    rng = wl.SplitMix64(3)
    sigma = np.array([rng.uniform_range(0.0, 5.0) for _ in range(w.n)])
    x0 = np.array([rng.uniform_range(-1.0, 1.0) for _ in range(w.n)])
    ref, out, _ = _linear_case(pf, oracle, w, 2, sigma=sigma, x0=x0)
    assert ref["status"] == 0 and out["status"] == 0
    assert abs(out["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9


def test_linear_fixed_iterations_match_iterate(pf, oracle):
    """tol = 0: exactly maxit iterations on both sides; the iterates themselves agree."""
    w = wl.config1(n=32, ncharges=50)
    ref, out, hist = _linear_case(pf, oracle, w, 2, tol=0.0, maxit=20)
    assert ref["status"] == 1 and out["status"] == 1 and out["iters"] == 20 == ref["iters"]
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-12
    assert np.allclose(hist, ref["hist"], rtol=1e-10)


def test_linear_degenerate_cases(pf, oracle):
    w = ragged_workload(mixed_bc=False)
    g = pf.Grid.from_workload(w)
    # b = 0 with zero Dirichlet data: x = 0 after 0 iterations (Q3)
    x = torch.ones(w.n, dtype=torch.float64, device="cuda")
    out = g.solve_linear(np.zeros(w.n), x=x)
    assert out["status"] == 0 and out["iters"] == 0 and float(x.abs().max()) == 0.0
    # maxit = 0: not converged, x = x0 with Dirichlet values forced
    x = torch.full((w.n,), 0.5, dtype=torch.float64, device="cuda")
    out = g.solve_linear(w.rhs, x=x, maxit=0)
    assert out["status"] == 1 and out["iters"] == 0
    ref = oracle.set_dirichlet(w.nx, w.ny, w.nz, w.bc_type, w.bc_value, np.full(w.n, 0.5))
    assert np.array_equal(x.cpu().numpy(), ref)
    # warm start at the solution: converged before the first iteration
    sol = g.solve_linear(w.rhs, tol=1e-12)["x"]
    out = g.solve_linear(w.rhs, x=sol.clone(), tol=1e-8)
    assert out["status"] == 0 and out["iters"] == 0
    g.close()


@pytest.mark.parametrize("kernels", [1, 2, 3])
@pytest.mark.parametrize("norm", [0, 1])
@pytest.mark.parametrize("bad", ["nan", "overflow"])
def test_non_finite_input_is_a_breakdown_not_a_success(pf, oracle, kernels, norm, bad):
    """Reading D7: a NaN (or a sum of squares that overflows) fails every comparison, so it must not pass the
    maximum-norm stopping test as 'converged' nor run silently to maxit: all three kernel families and the oracle
    report a breakdown after zero iterations."""
    w = ragged_workload(nx=64, ny=32, nz=16, seed=4, mixed_bc=False)      # fits tiled and cooperative kernels
    rhs = w.rhs.copy()
    rhs[5 + w.nx * (7 + w.ny * 8)] = np.nan if bad == "nan" else 1e200     # interior node; 1e200^2 overflows: ||b|| = inf
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, rhs, tol=1e-6, maxit=50, norm=norm)
    assert ref["status"] == -3 and ref["iters"] == 0
    g = pf.Grid.from_workload(w, kernels=kernels, options={pf.PF_OPT_NORM: norm})
    with pytest.raises(pf.PFError) as e:
        g.solve_linear(rhs, tol=1e-6, maxit=50)
    assert e.value.code == pf.PF_ERR_BREAKDOWN
    # the grid stays usable
    out = g.solve_linear(w.rhs, tol=1e-8 if norm == 0 else 1e-6)
    assert out["status"] == 0
    g.close()


def test_pf_reports_cut_off_inner_solves(pf, oracle):
    """pf_solve_pf whose increment meets a loose tolerance while every linear solve stopped at its cap returns
    PF_INNER_NOT_CONVERGED (2), like the oracle, not PF_OK."""
    w = wl.config0(n=24)
    sp = w.species
    ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                          sp.radii, w.l_c, 1e3, lin_maxit=3, max_outer=5)
    g = pf.Grid.from_workload(w, options={pf.PF_OPT_LINEAR_MAXIT: 3, pf.PF_OPT_MAX_OUTER: 5})
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, 1e3)
    g.close()
    assert ref["status"] == 2 and out["status"] == pf.PF_INNER_NOT_CONVERGED
    assert out["outer_iters"] == ref["outer_iters"] == 1 and out["linear_iters"] == ref["linear_iters"] == 9
    assert rel_l2(out["phi"].cpu().numpy(), ref["phi"]) <= 1e-12


def test_linear_host_buffers(pf, oracle):
    w = ragged_workload()
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=1e-10)
    g = pf.Grid.from_workload(w)
    rhs_h = torch.tensor(w.rhs).pin_memory()
    x_h = torch.zeros(w.n, dtype=torch.float64).pin_memory()
    out = pf.pf_solve_linear_host(g.handle, w.n, rhs_h, x_h, 1e-10, 10000)
    g.close()
    assert out["status"] == 0 and rel_l2(x_h.numpy(), ref["x"]) <= 1e-9


def test_linear_host_buffers_staged_upload(pf, oracle):
    """pf_grid_stage_host: the upload runs on the grid's copy stream while a PF solve uses the grid; the host solve that
    follows recognises the staged pair and gives the bits of the plain host solve.  Another pair is uploaded as usual."""
    w = wl.config0(n=32)
    sp = w.species
    rhs = np.random.default_rng(2).standard_normal(w.n)
    g = pf.Grid.from_workload(w, kernels=pf.KERNELS_TILED)
    rhs_h = torch.tensor(rhs).pin_memory()
    x_plain = torch.zeros(w.n, dtype=torch.float64).pin_memory()
    a = pf.pf_solve_linear_host(g.handle, w.n, rhs_h, x_plain, 1e-10, 10000)
    x_staged = torch.zeros(w.n, dtype=torch.float64).pin_memory()
    pf.pf_grid_stage_host(g.handle, w.n, rhs_h, x_staged)
    g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, 1e-3, want_conc=False)      # uses the PF scratch meanwhile
    b = pf.pf_solve_linear_host(g.handle, w.n, rhs_h, x_staged, 1e-10, 10000)
    assert a["status"] == 0 == b["status"] and a["iters"] == b["iters"]
    assert torch.equal(x_plain, x_staged)
    # staged for one pair, solved with another: the other pair is uploaded, the result is that pair's
    x_other = torch.zeros(w.n, dtype=torch.float64).pin_memory()
    pf.pf_grid_stage_host(g.handle, w.n, rhs_h, x_staged)
    c = pf.pf_solve_linear_host(g.handle, w.n, (2.0 * rhs_h).pin_memory(), x_other, 1e-10, 10000)
    assert c["status"] == 0 and rel_l2(x_other.numpy(), 2.0 * x_plain.numpy()) <= 1e-9
    g.close()


# ---- row N1: pointwise Fermi kernel --------------------------------------------------------------

@pytest.mark.parametrize("species", ["nacl", "nacacl", "nosteric"])
def test_fermi_pointwise(pf, oracle, species):
    w = wl.config0()
    sp = {"nacl": wl.NACL, "nacacl": wl.NACACL, "nosteric": wl.NACL}[species]
    radii = np.zeros_like(sp.radii) if species == "nosteric" else sp.radii
    rng = wl.SplitMix64(5)
    phi = np.array([rng.uniform_range(-12.0, 12.0) for _ in range(w.n)])
    phi[:8] = [0.0, 50.0, -50.0, 500.0, -500.0, 1e-9, 20.0, -20.0]
    solvent = oracle.solvent_mask(w.eps)
    ref = oracle.fermi_pointwise(sp.valence, sp.bath_molar, radii, phi, solvent)
    g = pf.Grid.from_workload(w)
    K = len(sp.valence)
    dev = lambda m: torch.empty(m, dtype=torch.float64, device="cuda")
    rho, sigma, S, conc = dev(w.n), dev(w.n), dev(w.n), dev((K + 1) * w.n)
    pf.pf_fermi_pointwise(g.handle, w.n, sp.valence, sp.bath_molar, radii, torch.tensor(phi, device="cuda"),
                          rho, sigma, S, conc)
    g.close()
    assert np.allclose(S.cpu().numpy(), ref["S"], rtol=1e-11, atol=1e-13)
    assert np.allclose(conc.cpu().numpy().reshape(K + 1, -1), ref["conc"], rtol=1e-10, atol=0)
    assert np.allclose(rho.cpu().numpy(), ref["rho"], rtol=1e-9, atol=1e-18)
    assert np.allclose(sigma.cpu().numpy(), ref["sigma"], rtol=1e-10, atol=0)
    assert np.all(conc.cpu().numpy().reshape(K + 1, -1)[:, solvent == 0] == 0.0)


# ---- rows N1-N5: the full nonlinear solve ----------------------------------------------------------

def _pf_case(pf, oracle, w, stencil=0):
    sp = w.species
    ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence,
                          sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, lin_tol=w.linear_tol)
    g = pf.Grid.from_workload(w, stencil=stencil)
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol)
    g.close()
    return ref, out


@pytest.mark.parametrize("stencil", [1, 2])
def test_pf_config0_32(pf, oracle, stencil):
    """BASELINE configs[0]: 32^3 PF with Na+/Cl-/water, l_c = 1.2, linear 1e-10, nonlinear 1e-8."""
    w = wl.config0()
    ref, out = _pf_case(pf, oracle, w, stencil)
    assert ref["status"] == 0 and out["status"] == 0
    assert out["outer_iters"] == ref["outer_iters"]
    assert abs(out["linear_iters"] - ref["linear_iters"]) <= 0.02 * ref["linear_iters"], \
        (out["linear_iters"], ref["linear_iters"])
    assert rel_l2(out["phi"].cpu().numpy(), ref["phi"]) <= 1e-7
    conc = out["conc"].cpu().numpy()
    for k in range(conc.shape[0]):
        assert rel_l2(conc[k], ref["conc"][k]) <= 1e-7, k
    assert np.allclose(out["steric"].cpu().numpy(), ref["steric"], rtol=1e-6, atol=1e-9)
    # the increments ||Phi - Phi0||_inf of the outer loop follow the oracle's
    assert np.allclose(out["incr_hist"], ref["incr_hist"], rtol=1e-3, atol=0)   # linear solves stop at 1e-10


def test_pf_channel_neumann_small(pf, oracle):
    """configs[2]'s geometry and species (Na+, Ca2+, Cl-, +50 mV, lateral Neumann) at 32^3."""
    w = wl.config2(n=32, volt_mv=50.0)
    ref, out = _pf_case(pf, oracle, w)
    assert ref["status"] == 0 and out["status"] == 0
    assert out["outer_iters"] == ref["outer_iters"]
    assert abs(out["linear_iters"] - ref["linear_iters"]) <= 0.02 * ref["linear_iters"]
    assert rel_l2(out["phi"].cpu().numpy(), ref["phi"]) <= 1e-7
    conc = out["conc"].cpu().numpy()
    for k in range(conc.shape[0]):
        assert rel_l2(conc[k], ref["conc"][k]) <= 1e-7, k


@pytest.mark.parametrize("kernels", [0, 2])
def test_pf_lagged_steric_mode(pf, oracle, kernels):
    """PF_OPT_STERIC_MODE = 1 (readings G1, G2): S^trc of the previous outer iteration.  (a) configs[0]'s
    geometry at 32^3 with the charges scaled to 0.1 e, where the lagged loop converges: phi, C_k, S^trc against the
    oracle's lagged loop; (b) three outer iterations at full strength, where Gamma_0 meets its floor next to the charges."""
    sp = wl.NACL
    for scale, max_outer, tol in ((0.2, 400, 1e-8), (1.0, 3, 1e-8)):
        w = wl.config0()
        w.charges = w.charges.copy()
        w.charges[:, 3] *= scale
        ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                              sp.radii, w.l_c, tol, max_outer=max_outer, steric_mode=oracle.STERIC_LAGGED)
        g = pf.Grid.from_workload(w, kernels=kernels, options={pf.PF_OPT_STERIC_MODE: 1, pf.PF_OPT_MAX_OUTER: max_outer})
        out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, tol)
        g.close()
        assert out["status"] == ref["status"] == (0 if scale < 1 else 1) and out["outer_iters"] == ref["outer_iters"]
        assert abs(out["linear_iters"] - ref["linear_iters"]) <= 0.02 * ref["linear_iters"]
        assert rel_l2(out["phi"].cpu().numpy(), ref["phi"]) <= 1e-7
        for k in range(3):
            assert rel_l2(out["conc"][k].cpu().numpy(), ref["conc"][k]) <= 1e-7
        assert rel_l2(out["steric"].cpu().numpy(), ref["steric"]) <= 1e-7
        if scale == 1.0:
            assert ref["steric"].min() < -20.0               # ln(1e-12 / Gamma^B): the floor


def test_pf_errors(pf):
    w = wl.config0(n=16)
    g = pf.Grid.from_workload(w)
    with pytest.raises(pf.PFError) as e:
        g.solve_pf([1.0, -1.0], [0.1, 0.2], [0.95, 1.81, 1.4], 1.2, 1e-8)     # not neutral
    assert e.value.code == pf.PF_ERR_NONPHYSICAL
    with pytest.raises(pf.PFError) as e:
        g.solve_pf([1.0, -1.0], [0.1, 0.1], [9.0, 9.0, 9.0], 1.2, 1e-8)       # Gamma^B <= 0
    assert e.value.code == pf.PF_ERR_NONPHYSICAL
    g.close()


@pytest.mark.parametrize("shape", [(32, 16, 8), (34, 17, 9), (64, 16, 40), (130, 33, 21), (96, 48, 64), (256, 20, 12)])
def test_tiled_equals_direct_on_many_shapes(pf, shape):
    """Smallest supported grid, partial tiles in x and/or y, one plane per block up to several chunks:
    the TMA-tiled kernels (mbarrier ring, halo warps, zero-filled out-of-grid nodes) give the same bits as
    the one-thread-per-node kernels, iterate and residual history, for both stencil variants."""
    nx, ny, nz = shape
    w = ragged_workload(nx=nx, ny=ny, nz=nz, seed=31 + nx)
    for stencil in (1, 2):
        res = []
        for kernels in (1, 2):
            g = pf.Grid.from_workload(w, stencil=stencil, kernels=kernels, options={pf.PF_OPT_HISTORY: 32})
            out = g.solve_linear(w.rhs, tol=0.0, maxit=25)
            res.append((out["x"].clone(), g.history(26), out["true_relres"]))
            g.close()
        assert torch.equal(res[0][0], res[1][0]), (shape, stencil)
        assert np.array_equal(res[0][1], res[1][1]) and res[0][2] == res[1][2]


@pytest.mark.parametrize("case", ["tiny_rhs_entries", "huge_diagonal"])
def test_division_range_fault_falls_back(pf, oracle, case):
    """Operands outside the range of the tiled kernels' branch-free division (DESIGN D4) raise the fault flag;
    the solve is repeated by the kernels that divide with __ddiv_rn and still matches the oracle."""
    w = ragged_workload(nx=70, ny=37, nz=19, seed=9)
    sigma = None
    if case == "tiny_rhs_entries":
        w.rhs = w.rhs.copy()
        w.rhs[24390:24400] = 1e-300                   # interior nodes: quotients below 2^-900 in the first iteration
    else:
        sigma = np.zeros(w.n)
        sigma[7000:7004] = 1e20                       # diagonal above 2^60
    ref, out_t, _ = _linear_case(pf, oracle, w, 2, kernels=2, sigma=sigma)
    _, out_d, _ = _linear_case(pf, oracle, w, 2, kernels=1, sigma=sigma)
    assert ref["status"] == 0 and out_t["status"] == 0
    assert torch.equal(out_t["x"], out_d["x"]) and out_t["iters"] == out_d["iters"]
    assert out_t["fault_repeats"] == 1 and out_d["fault_repeats"] == 0
    if case == "tiny_rhs_entries":
        assert abs(out_t["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    # huge_diagonal: products in the inner products span 1e40, beyond what twice the working precision
    # resolves, so the reduced scalars depend on the summation order and the iteration paths separate
    # (DESIGN section 4); the converged solutions still agree
    assert out_t["true_relres"] <= 1.05e-10
    assert rel_l2(out_t["x"].cpu().numpy(), ref["x"]) <= 1e-9


# ---- the paper's own parameter set ----------------------------------------------

@pytest.mark.parametrize("kernels", [1, 2])
def test_linear_paper_stopping_test(pf, oracle, kernels):
    """Table 3 steps 18-19 as written: stop when ||r||_inf < 1e-6, absolute."""
    w = ragged_workload(nx=70, ny=37, nz=19, seed=9)
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=1e-6, history=True,
                              norm=oracle.NORM_ABS_INF)
    g = pf.Grid.from_workload(w, stencil=2, kernels=kernels, options={pf.PF_OPT_NORM: pf.NORM_ABS_INF,
                                                                       pf.PF_OPT_HISTORY: 4096})
    out = g.solve_linear(w.rhs, tol=1e-6)
    hist = g.history(4096)
    g.close()
    assert ref["status"] == 0 and out["status"] == 0 and out["iters"] == ref["iters"]
    assert out["relres"] < 1e-6 and np.all(hist[:-1] >= 1e-6)
    assert np.allclose(hist, ref["hist"], rtol=1e-8)               # absolute maximum norms, iteration by iteration
    assert abs(out["true_relres"] - ref["true_relres"]) <= 1e-6 * ref["true_relres"]
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9


def test_pf_paper_parameters(pf, oracle):
    """Linear tolerance 1e-6 in the maximum norm for every system, Newton ErrTol 1e-3, omega_PF 0.3."""
    w = wl.config0()
    sp = w.species
    ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                          sp.radii, w.l_c, 1e-3, omega_pf=0.3, lin_tol=1e-6, norm=oracle.NORM_ABS_INF)
    g = pf.Grid.from_workload(w, options={pf.PF_OPT_NORM: pf.NORM_ABS_INF, pf.PF_OPT_LINEAR_TOL: 1e-6,
                                          pf.PF_OPT_OMEGA_PF: 0.3})
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, 1e-3)
    g.close()
    assert ref["status"] == 0 and out["status"] == 0 and out["outer_iters"] == ref["outer_iters"]
    # the right-hand sides come from exp/log of two different math libraries: a solve whose residual hovers at
    # the threshold may stop an iteration or two apart; totals agree within BASELINE's 2 %
    assert abs(out["linear_iters"] - ref["linear_iters"]) <= 0.02 * ref["linear_iters"]
    assert np.max(np.abs(np.array(out["lin_iters_hist"]) - ref["lin_iters_hist"])) <= 10
    assert rel_l2(out["phi"].cpu().numpy(), ref["phi"]) <= 1e-7
    assert np.allclose(out["incr_hist"], ref["incr_hist"], rtol=1e-4, atol=0)


# ---- odd nx: the tiled kernels on the box widened by one column of identity rows ---------------------------

@pytest.mark.parametrize("shape", [(33, 16, 8), (65, 17, 9), (131, 33, 21), (97, 48, 64)])
def test_tiled_kernels_odd_nx(pf, oracle, shape):
    """An odd nx cannot be described to the TMA unit; the solve is embedded in the box with one more column of
    decoupled identity rows.  Same bits as the one-thread-per-node kernels on the original box:
    iterate, residual history, true residual; with a warm start and a sigma shift as well."""
    nx, ny, nz = shape
    w = ragged_workload(nx=nx, ny=ny, nz=nz, seed=77 + nx)
    rng = wl.SplitMix64(5)
    sigma = np.array([rng.uniform_range(0.0, 3.0) for _ in range(w.n)])
    x0 = np.array([rng.uniform_range(-1.0, 1.0) for _ in range(w.n)])
    for sg, start, stencil in ((None, None, 2), (sigma, x0, 2), (sigma, None, 1)):     # 1: stored coefficients
        res = []
        for kernels in (1, 2):
            g = pf.Grid.from_workload(w, stencil=stencil, kernels=kernels, options={pf.PF_OPT_HISTORY: 64})
            x = torch.zeros(w.n, dtype=torch.float64, device="cuda") if start is None else torch.tensor(start, device="cuda")
            out = g.solve_linear(w.rhs, x=x, tol=0.0, maxit=30, sigma=None if sg is None else torch.tensor(sg, device="cuda"))
            res.append((out["x"].clone(), g.history(64), out["true_relres"], out["iters"]))
            g.close()
        assert torch.equal(res[0][0], res[1][0]), shape
        assert np.array_equal(res[0][1], res[1][1]) and res[0][2] == res[1][2] and res[0][3] == res[1][3] == 30
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=1e-10)
    g = pf.Grid.from_workload(w, stencil=2, kernels=2)
    out = g.solve_linear(w.rhs, tol=1e-10)
    g.close()
    assert out["status"] == 0 and abs(out["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    assert out["true_relres"] <= 1.05e-10 and rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9


def test_odd_nx_auto_and_pf(pf):
    """Auto mode on a large odd-nx box takes the widened tiled path (same bits as the direct kernels); b = 0 gives
    x = 0; a PF solve on an odd-nx box is the same with both families."""
    w = ragged_workload(nx=129, ny=96, nz=80, seed=3)
    res = []
    for kernels in (1, 0):
        g = pf.Grid.from_workload(w, stencil=2, kernels=kernels)
        out = g.solve_linear(w.rhs, tol=0.0, maxit=12)
        res.append(out["x"].clone())
        g.close()
    assert torch.equal(res[0], res[1])
    w0 = ragged_workload(nx=65, ny=40, nz=37, seed=4, mixed_bc=False)
    g = pf.Grid.from_workload(w0, stencil=2, kernels=2)
    x = torch.ones(w0.n, dtype=torch.float64, device="cuda")
    z = g.solve_linear(np.zeros(w0.n), x=x)                       # Q3 through the widened path
    assert z["status"] == 0 and z["iters"] == 0 and float(x.abs().max()) == 0.0
    g.close()
    w = wl.config0(n=33)
    sp = w.species
    out = []
    for kernels in (1, 2):
        g = pf.Grid.from_workload(w, stencil=2, kernels=kernels)
        out.append(g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, 1e-6))
        g.close()
    assert out[0]["outer_iters"] == out[1]["outer_iters"] and out[0]["lin_iters_hist"] == out[1]["lin_iters_hist"]
    assert torch.equal(out[0]["phi"], out[1]["phi"])


def test_eps_scan(pf):
    """The scan of the permittivity map: palette sizes 1..5+ with the values scattered so that every thread meets
    them in a different order; maps with a negative, zero, NaN or infinite entry are rejected at grid creation."""
    w = ragged_workload(nx=40, ny=33, nz=21, seed=13)
    rng = np.random.default_rng(5)
    vals = [2.0, 4.5, 20.0, 78.5, 80.0, 33.0]
    for count in range(1, 7):
        w.eps = rng.choice(vals[:count], size=w.n)
        w.eps[: count] = vals[:count]                       # every value present
        g = pf.Grid.from_workload(w)
        assert pf.pf_grid_palette_size(g.handle) == min(count, 5), count      # 5 = "more than four"
        assert pf.pf_grid_stencil(g.handle) == (2 if count <= 4 else 1)
        g.close()
    for bad in (-2.0, 0.0, float("nan"), float("inf")):
        w.eps = np.full(w.n, 2.0)
        w.eps[w.n // 3] = bad
        with pytest.raises(pf.PFError) as e:
            pf.Grid.from_workload(w)
        assert e.value.code == pf.PF_ERR_ARG, bad


def test_linear_unaligned_views(pf):
    """rhs, x and sigma given as views that start 8 bytes into a larger allocation: same bits as with aligned
    tensors (the iterate is solved in the workspace copy so that the tiled kernels still apply)."""
    w = ragged_workload(nx=70, ny=37, nz=19, seed=9)
    rng = wl.SplitMix64(8)
    sigma = np.array([rng.uniform_range(0.0, 2.0) for _ in range(w.n)])
    g = pf.Grid.from_workload(w, stencil=2, kernels=2)
    ref = g.solve_linear(w.rhs, tol=0.0, maxit=20, sigma=torch.tensor(sigma, device="cuda"))
    big = [torch.zeros(w.n + 1, dtype=torch.float64, device="cuda") for _ in range(3)]
    rhs_v, x_v, sg_v = (b[1:] for b in big)
    assert rhs_v.data_ptr() % 16 == 8
    rhs_v.copy_(torch.tensor(w.rhs)); sg_v.copy_(torch.tensor(sigma))
    out = pf.pf_solve_linear(g.handle, w.n, rhs_v, x_v, 0.0, 20, sigma=sg_v)
    assert out["iters"] == 20 and out["true_relres"] == ref["true_relres"]
    assert torch.equal(x_v, ref["x"])
    assert pf.pf_grid_fault_repeats(g.handle) == 0
    g.close()


@pytest.mark.parametrize("kernels", [1, 2])
def test_device_loop_equals_polled_launches(pf, kernels):
    """PF_OPT_GRAPH 0 (stream launches, host polls), 1 (graph replays of polling chunks), 2 (one graph whose WHILE
    node repeats the iterations on the device until the solve is over) and 3 (2 or 1 by the expected length of the
    solve) run the same kernels on the same state: same
    iterate, residual history, iteration count and status -- for solves that end inside a loop body, at its last
    iteration, at maxit (odd and even, below and above one body), before the first iteration, and with the first
    iterations bracketed by profiling events."""
    w = ragged_workload(nx=66, ny=35, nz=23, seed=77)
    cases = [dict(tol=1e-10, maxit=10000), dict(tol=0.0, maxit=1), dict(tol=0.0, maxit=7), dict(tol=0.0, maxit=8),
             dict(tol=0.0, maxit=16), dict(tol=0.0, maxit=21), dict(tol=1e-3, maxit=10000), dict(tol=1e30, maxit=10)]
    res = {}
    for mode in (0, 1, 2, 3):
        g = pf.Grid.from_workload(w, kernels=kernels, options={pf.PF_OPT_GRAPH: mode, pf.PF_OPT_HISTORY: 512})
        res[mode] = []
        for c in cases:
            out = g.solve_linear(w.rhs, **c)
            res[mode].append((out["x"].clone(), g.history(512), out["iters"], out["status"], out["true_relres"]))
        g.set_option(pf.PF_OPT_PROFILE, 3)           # four iterations launched one by one, the rest in the loop
        out = g.solve_linear(w.rhs, tol=1e-10)
        res[mode].append((out["x"].clone(), g.history(512), out["iters"], out["status"], out["true_relres"]))
        g.close()
    assert res[0][0][3] == 0 and res[0][0][2] > 16       # the converged case runs over several bodies
    # every iteration count 9..24 ends somewhere else in a body of 8 and in a polling chunk of 16
    for k, ref in enumerate(res[0]):
        for mode in (1, 2, 3):
            got = res[mode][k]
            assert torch.equal(got[0], ref[0]), (mode, k)
            assert np.array_equal(got[1], ref[1]) and got[2:] == ref[2:], (mode, k)


def test_device_loop_every_exit_position(pf):
    """The solve ends at every position of a loop body: maxit = 9..25 with tol = 0, and tolerances that stop the
    solve at consecutive iteration counts; the launch counter follows the bodies that ran."""
    w = ragged_workload(nx=40, ny=24, nz=16, seed=78)
    g1 = pf.Grid.from_workload(w, kernels=2, options={pf.PF_OPT_GRAPH: 1, pf.PF_OPT_HISTORY: 64})
    g2 = pf.Grid.from_workload(w, kernels=2, options={pf.PF_OPT_GRAPH: 2, pf.PF_OPT_HISTORY: 64})
    fixed = set()
    for maxit in range(9, 26):
        a = g1.solve_linear(w.rhs, tol=0.0, maxit=maxit)
        n0 = pf.pf_launch_count()
        b = g2.solve_linear(w.rhs, tol=0.0, maxit=maxit, true_residual=False)
        launched = pf.pf_launch_count() - n0
        assert a["iters"] == b["iters"] == maxit and torch.equal(a["x"], b["x"]), maxit
        # the whole bodies of 8 iterations below maxit in the loop, the rest as stream launches: nothing runs
        # beyond iteration maxit; + the solve's fixed launches (Dirichlet values into b and x, residual kernel,
        # finalize, x = x0 + M^-1 y)
        fixed.add(launched - 3 * maxit)
    assert len(fixed) == 1 and 3 <= fixed.pop() <= 8
    hist = g1.history(64)
    hist = hist[np.isfinite(hist)]
    for it in range(10, 19):                       # stop right after iteration `it`
        tol = float(np.sqrt(hist[it] * hist[it - 1])) if hist[it] < hist[it - 1] else None
        if tol is None:
            continue
        a = g1.solve_linear(w.rhs, tol=tol)
        b = g2.solve_linear(w.rhs, tol=tol)
        assert a["iters"] == b["iters"] and a["status"] == b["status"] == 0 and torch.equal(a["x"], b["x"]), it
    g1.close(); g2.close()


def test_device_loop_pf_and_odd_nx(pf):
    """A whole PF solve (three operators, warm starts, sigma diagonal; tiled kernels, and the widened box of an odd
    nx) gives the same bits, outer and linear iteration counts whether its inner solves run as polled launches,
    in the device-side loop or in the mode the library picks by itself; stored coefficients included."""
    for w, stencil in ((wl.config2(n=40, volt_mv=50.0), 2), (wl.config0(n=33), 2), (wl.config0(n=34), 1)):
        sp = w.species
        out = {}
        for mode in (0, 2, 3):
            g = pf.Grid.from_workload(w, stencil=stencil, kernels=2, options={pf.PF_OPT_GRAPH: mode})
            out[mode] = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, 1e-6)
            g.close()
        for mode in (2, 3):
            assert out[mode]["status"] == out[0]["status"] == 0
            assert out[mode]["outer_iters"] == out[0]["outer_iters"]
            assert out[mode]["lin_iters_hist"] == out[0]["lin_iters_hist"], (w.name, mode)
            assert torch.equal(out[mode]["phi"], out[0]["phi"]) and torch.equal(out[mode]["conc"], out[0]["conc"])


@pytest.mark.parametrize("shape", [(32, 16, 8), (34, 17, 9), (130, 33, 21), (96, 48, 64), (65, 17, 9)])
def test_diagonal_from_codes(pf, shape):
    """PF_OPT_DIAG_FROM_CODE: the tiled k1 that takes the Poisson diagonal from the table indexed by the node's
    stencil code (identity rows, Neumann and Dirichlet faces, partial tiles, the widened box of an odd nx) gives the
    bits of the k1 that reads A0, with and without the Jacobi preconditioner; a solve with a sigma diagonal and the
    PF operators keep reading A0 and are unchanged."""
    nx, ny, nz = shape
    w = ragged_workload(nx=nx, ny=ny, nz=nz, seed=11 + nx, mixed_bc=(nx % 3 != 0))
    sigma = torch.rand(w.n, dtype=torch.float64, device="cuda")
    for precond in (1, 0):
        res = []
        for diag in (0, 1):
            g = pf.Grid.from_workload(w, stencil=2, kernels=2, options={pf.PF_OPT_DIAG_FROM_CODE: diag,
                                                                       pf.PF_OPT_PRECOND: precond, pf.PF_OPT_HISTORY: 64})
            out = g.solve_linear(w.rhs, tol=0.0, maxit=25)
            h = g.history(26)
            outs = g.solve_linear(w.rhs, tol=0.0, maxit=9, sigma=sigma)
            res.append((out["x"].clone(), h, out["true_relres"], outs["x"].clone()))
            g.close()
        assert torch.equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1]), (shape, precond)
        assert res[0][2] == res[1][2] and torch.equal(res[0][3], res[1][3]), (shape, precond)
