"""GPU tests of the merged two-reduction BiCGSTAB (PF_OPT_SOLVER = 1; SURVEY.md 8(d) "fully merged", 8(f) #3; reading M1):
two kernels per iteration (K2M: s, t = A M^-1 s | K31: r, y, p, v = A M^-1 p fused).  Its parity reference is the
oracle's bicgstab_merged() -- the same recurrence, statement for statement -- at BASELINE.json's tolerances: relative
L2 difference of the potential <= 1e-9, true relative residual <= 1e-10, iteration counts within +-2 %; PF <= 1e-7.
The tiled TMA kernels must give the same bits as the one-thread-per-node kernels."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1711_04060_b200 import workloads as wl  # noqa: E402
from test_gpu_parity import ragged_workload, rel_l2  # noqa: E402


@pytest.fixture(scope="module")
def pf():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_1711_04060_b200 import build as _build, pf as _pf
    _build.build()
    _pf.load()
    return _pf


def _solve(pf, w, kernels, stencil=2, precond=1, tol=1e-10, maxit=10000, norm=0, x0=None, sigma=None, solver=1, graph=None,
           diag_code=None):
    opts = {pf.PF_OPT_PRECOND: precond, pf.PF_OPT_HISTORY: 4096, pf.PF_OPT_NORM: norm, pf.PF_OPT_SOLVER: solver}
    if graph is not None:
        opts[pf.PF_OPT_GRAPH] = graph
    if diag_code is not None:
        opts[pf.PF_OPT_DIAG_FROM_CODE] = diag_code
    g = pf.Grid.from_workload(w, stencil=stencil, kernels=kernels, options=opts)
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda") if x0 is None else torch.tensor(x0, device="cuda")
    sg = None if sigma is None else torch.tensor(sigma, device="cuda")
    out = g.solve_linear(w.rhs, x=x, tol=tol, maxit=maxit, sigma=sg)
    out["hist"] = g.history(4096)
    out["fault_repeats"] = pf.pf_grid_fault_repeats(g.handle)
    g.close()
    return out


def _oracle(oracle, w, precond=True, tol=1e-10, maxit=10000, norm=0, x0=None, sigma=None):
    return oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, x0=x0, sigma=sigma, tol=tol,
                               maxit=maxit, precond=precond, history=True, norm=norm, solver=oracle.SOLVER_MERGED)


@pytest.mark.parametrize("stencil", [1, 2])
@pytest.mark.parametrize("precond", [1, 0])
def test_merged_direct_kernels_against_oracle(pf, oracle, stencil, precond):
    w = ragged_workload()                                 # 37 x 20 x 11, Neumann + Dirichlet faces
    ref = _oracle(oracle, w, precond=bool(precond))
    out = _solve(pf, w, pf.KERNELS_DIRECT, stencil=stencil, precond=precond)
    assert ref["status"] == 0 and out["status"] == 0
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9
    assert out["true_relres"] <= 1.05e-10
    assert abs(out["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    m = min(len(out["hist"]), len(ref["hist"]), 30)
    assert np.allclose(out["hist"][:m], ref["hist"][:m], rtol=1e-9)


@pytest.mark.parametrize("shape", [(32, 16, 8), (34, 17, 9), (64, 16, 40), (130, 33, 21), (96, 48, 64), (65, 17, 9)])
@pytest.mark.parametrize("precond", [1, 0])
def test_merged_tiled_equals_direct(pf, shape, precond):
    """Tiled K2M / K31 (diagonal from the codes, K31D, and read from memory, K31) give the bits of the direct kernels."""
    nx, ny, nz = shape
    w = ragged_workload(nx=nx, ny=ny, nz=nz, seed=31 + nx)
    a = _solve(pf, w, pf.KERNELS_DIRECT, precond=precond, maxit=120)
    for diag_code in (1, 0):
        b = _solve(pf, w, pf.KERNELS_TILED, precond=precond, maxit=120, diag_code=diag_code)
        assert a["status"] == b["status"] and a["iters"] == b["iters"] and b["fault_repeats"] == 0
        assert torch.equal(a["x"], b["x"])
        assert np.array_equal(a["hist"], b["hist"])
        assert a["relres"] == b["relres"] and a["true_relres"] == b["true_relres"]


def test_merged_tiled_four_level_map_and_sigma(pf, oracle):
    """4-bit stencil codes (uint32), a sigma diagonal (so the diagonal is read, K31), a warm start."""
    w = ragged_workload(nx=66, ny=34, nz=18, seed=12)
    rng = np.random.default_rng(5)
    w.eps = np.where(w.eps > 10, rng.choice([80.0, 40.0], size=w.n), rng.choice([2.0, 4.0], size=w.n))
    sigma = rng.uniform(0.0, 3.0, size=w.n)
    x0 = rng.standard_normal(w.n)
    ref = _oracle(oracle, w, sigma=sigma, x0=x0)
    a = _solve(pf, w, pf.KERNELS_DIRECT, sigma=sigma, x0=x0)
    b = _solve(pf, w, pf.KERNELS_TILED, sigma=sigma, x0=x0)
    assert ref["status"] == 0 and a["status"] == 0 and b["status"] == 0
    assert torch.equal(a["x"], b["x"]) and a["iters"] == b["iters"] and np.array_equal(a["hist"], b["hist"])
    assert rel_l2(b["x"].cpu().numpy(), ref["x"]) <= 1e-9 and b["true_relres"] <= 1.05e-10
    assert abs(b["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])


@pytest.mark.parametrize("stencil", [1, 2])
def test_merged_config1_64(pf, oracle, stencil):
    """configs[1] (64^3, spheres eps 2/80, 500 Gaussian charges) with kernels = auto (tiled for the on-the-fly stencil,
    direct for stored coefficients)."""
    w = wl.config1()
    ref = _oracle(oracle, w)
    out = _solve(pf, w, pf.KERNELS_AUTO, stencil=stencil)
    assert ref["status"] == 0 and out["status"] == 0
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9
    assert out["true_relres"] <= 1.05e-10
    assert abs(out["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    m = min(len(out["hist"]), len(ref["hist"]))
    assert np.allclose(out["hist"][:40], ref["hist"][:40], rtol=1e-9)
    print(f"merged 64^3 stencil {stencil}: iterations gpu/oracle {out['iters']}/{ref['iters']}, hist compared {m}")


def test_merged_fixed_iterations_match_iterate(pf, oracle):
    w = wl.config1()
    for k in (1, 2, 7):
        ref = _oracle(oracle, w, tol=0.0, maxit=k)
        out = _solve(pf, w, pf.KERNELS_TILED, tol=0.0, maxit=k)
        assert out["iters"] == k == ref["iters"] and out["status"] == 1
        assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-12
        assert np.allclose(out["hist"], ref["hist"], rtol=1e-10)


@pytest.mark.parametrize("kernels", [1, 2])
def test_merged_launch_modes_give_the_same_bits(pf, kernels):
    """Stream launches, polled graph chunks, the device-side loop (whose bodies end with the finalize that sets the
    condition) and auto: same iterates, at exit positions that fall on every place of a body."""
    w = ragged_workload(nx=64, ny=32, nz=16, seed=4, mixed_bc=False)
    for tol, maxit in ((1e-10, 10000), (0.0, 1), (0.0, 8), (0.0, 9), (0.0, 16), (0.0, 17), (0.0, 31), (1e-3, 10000)):
        base = _solve(pf, w, kernels, tol=tol, maxit=maxit, graph=0)
        for graph in (1, 2, 3):
            o = _solve(pf, w, kernels, tol=tol, maxit=maxit, graph=graph)
            assert o["status"] == base["status"] and o["iters"] == base["iters"], (tol, maxit, graph)
            assert torch.equal(o["x"], base["x"]) and np.array_equal(o["hist"], base["hist"]), (tol, maxit, graph)


def test_merged_degenerate_cases(pf, oracle):
    w = ragged_workload(nx=64, ny=32, nz=16, seed=4, mixed_bc=False)
    for kernels in (1, 2):
        g = pf.Grid.from_workload(w, kernels=kernels, options={pf.PF_OPT_SOLVER: 1})
        x = torch.ones(w.n, dtype=torch.float64, device="cuda")
        out = g.solve_linear(np.zeros(w.n), x=x)
        assert out["status"] == 0 and out["iters"] == 0 and float(x.abs().max()) == 0.0
        x = torch.full((w.n,), 0.5, dtype=torch.float64, device="cuda")
        out = g.solve_linear(w.rhs, x=x, maxit=0)
        assert out["status"] == 1 and out["iters"] == 0
        assert np.array_equal(x.cpu().numpy(), oracle.set_dirichlet(w.nx, w.ny, w.nz, w.bc_type, w.bc_value, np.full(w.n, 0.5)))
        sol = g.solve_linear(w.rhs, tol=1e-12)["x"]
        out = g.solve_linear(w.rhs, x=sol.clone(), tol=1e-8)
        assert out["status"] == 0 and out["iters"] == 0
        bad = w.rhs.copy()
        bad[5 + w.nx * (7 + w.ny * 8)] = np.nan
        with pytest.raises(pf.PFError) as e:
            g.solve_linear(bad, tol=1e-6, maxit=50)
        assert e.value.code == pf.PF_ERR_BREAKDOWN
        g.close()
    g = pf.Grid.from_workload(w, options={pf.PF_OPT_SOLVER: 1})
    with pytest.raises(pf.PFError):
        pf.pf_grid_set_option(g.handle, pf.PF_OPT_KERNELS, pf.KERNELS_COOP)
        g.solve_linear(w.rhs)
    g.close()


def test_merged_paper_stopping_test(pf, oracle):
    """Norm mode 1 (Table 3 steps 18-19: ||r||_inf < tol, absolute) with the merged recurrence."""
    w = ragged_workload(nx=64, ny=32, nz=16, seed=4)
    ref = _oracle(oracle, w, tol=1e-6, norm=1)
    for kernels in (1, 2):
        out = _solve(pf, w, kernels, tol=1e-6, norm=1)
        assert out["status"] == 0 == ref["status"] and out["iters"] == ref["iters"]
        assert np.allclose(out["hist"], ref["hist"], rtol=1e-8)
        assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9


@pytest.mark.parametrize("kernels", [0, 2])
def test_merged_pf_config0_32(pf, oracle, kernels):
    """Full nonlinear PF solve of configs[0] (32^3) with every linear solve through the merged recurrence:
    phi and each C_k within 1e-7 of the oracle's PF loop run with its merged solver."""
    w = wl.config0()
    sp = w.species
    ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                          sp.radii, w.l_c, w.nonlinear_tol, max_outer=1000, solver=oracle.SOLVER_MERGED)
    g = pf.Grid.from_workload(w, kernels=kernels, options={pf.PF_OPT_SOLVER: 1})
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol)
    g.close()
    assert ref["status"] == 0 and out["status"] == 0
    assert out["outer_iters"] == ref["outer_iters"]
    assert abs(out["linear_iters"] - ref["linear_iters"]) <= 0.02 * ref["linear_iters"]
    assert rel_l2(out["phi"].cpu().numpy(), ref["phi"]) <= 1e-7
    for k in range(len(sp.valence) + 1):
        assert rel_l2(out["conc"][k].cpu().numpy(), ref["conc"][k]) <= 1e-7
    print(f"merged PF 32^3 kernels {kernels}: outer {out['outer_iters']}, linear gpu/oracle {out['linear_iters']}/{ref['linear_iters']}")


@pytest.mark.parametrize("rows", [13, 16])
@pytest.mark.parametrize("solver", [0, 1])
def test_both_tile_geometries_equal_direct(pf, rows, solver):
    """PF_OPT_TILE_ROWS: the tiled kernels are compiled for tiles of 16 rows (19 warps) and of 13 rows (16 warps, 128
    registers); the default picks per kernel and grid size.  Forced either way they give the bits of the direct kernels,
    on shapes with partial tiles in x and y for both heights, Poisson (diagonal from the codes) and with a sigma."""
    for shape in ((64, 29, 12), (130, 33, 21), (66, 53, 40)):
        nx, ny, nz = shape
        w = ragged_workload(nx=nx, ny=ny, nz=nz, seed=77 + ny)
        sigma = np.random.default_rng(ny).uniform(0.0, 2.0, size=w.n)
        for sg in (None, sigma):
            outs = []
            for kernels, r in ((pf.KERNELS_DIRECT, 0), (pf.KERNELS_TILED, rows)):
                g = pf.Grid.from_workload(w, stencil=2, kernels=kernels,
                                          options={pf.PF_OPT_SOLVER: solver, pf.PF_OPT_TILE_ROWS: r, pf.PF_OPT_HISTORY: 256})
                o = g.solve_linear(w.rhs, tol=1e-10, maxit=150, sigma=None if sg is None else torch.tensor(sg, device="cuda"))
                o["hist"] = g.history(256)
                assert pf.pf_grid_fault_repeats(g.handle) == 0
                g.close()
                outs.append(o)
            a, b = outs
            assert a["status"] == b["status"] and a["iters"] == b["iters"]
            assert torch.equal(a["x"], b["x"]) and np.array_equal(a["hist"], b["hist"])
            assert a["true_relres"] == b["true_relres"]


@pytest.mark.parametrize("solver", [0, 1])
def test_segment_plans_and_k2_diagonal_table_equal_direct(pf, solver):
    """PF_OPT_SEGMENTS (how tiles x z ranges are handed to the persistent blocks) and PF_OPT_DIAG_FROM_CODE = 2 (k2 / K2M
    take the diagonal and the divisor's half of the Jacobi division from the code table as k1 / K31 do) change no bit:
    forced either way the tiled kernels give the iterates of the direct kernels, on shapes where the two-group plan
    exists (several layers, a rest group of one to a few blocks with segments that cross tiles) and where it does not."""
    for shape in ((64, 29, 200), (130, 33, 96), (66, 53, 40), (128, 64, 61), (320, 208, 40)):
        nx, ny, nz = shape
        w = ragged_workload(nx=nx, ny=ny, nz=nz, seed=5 + nz)
        ref = None
        # (320 x 208 x 40 on 148 SMs: 80 tiles of 13 rows -- the plan of mode 2; 65 tiles of 16 rows -- mode 1)
        for kernels, seg, diag, rows in ((pf.KERNELS_DIRECT, -1, 1, 0), (pf.KERNELS_TILED, 0, 1, 0), (pf.KERNELS_TILED, 1, 1, 0),
                                         (pf.KERNELS_TILED, 1, 2, 16), (pf.KERNELS_TILED, 0, 2, 13), (pf.KERNELS_TILED, -1, 2, 0),
                                         (pf.KERNELS_TILED, 1, 0, 13), (pf.KERNELS_TILED, 2, 1, 13), (pf.KERNELS_TILED, 2, 2, 0)):
            g = pf.Grid.from_workload(w, stencil=2, kernels=kernels,
                                      options={pf.PF_OPT_SOLVER: solver, pf.PF_OPT_SEGMENTS: seg, pf.PF_OPT_TILE_ROWS: rows,
                                               pf.PF_OPT_DIAG_FROM_CODE: diag, pf.PF_OPT_HISTORY: 256})
            o = g.solve_linear(w.rhs, tol=1e-10, maxit=120)
            o["hist"] = g.history(256)
            assert pf.pf_grid_fault_repeats(g.handle) == 0
            g.close()
            if ref is None:
                ref = o
                continue
            assert o["status"] == ref["status"] and o["iters"] == ref["iters"], (shape, seg, diag, rows)
            assert torch.equal(o["x"], ref["x"]) and np.array_equal(o["hist"], ref["hist"]), (shape, seg, diag, rows)
