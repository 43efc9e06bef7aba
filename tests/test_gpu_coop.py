"""GPU tests of the cooperative single-kernel solver (PF_OPT_KERNELS = 3):
one persistent kernel per solve, one brick of the box per SM, the vectors in shared memory, three grid-wide
barriers per iteration.  Its arithmetic is Table 3 statement for statement, so it must give the same bits as the
one-thread-per-node kernels and meet the same tolerances against the CPU oracle (BASELINE.json: relative L2
difference <= 1e-9, true relative residual <= 1e-10, iteration counts within 2 %; PF <= 1e-7).
"""
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


def _solve(pf, w, kernels, stencil=2, precond=1, tol=1e-10, maxit=10000, norm=0, x0=None, sigma=None):
    g = pf.Grid.from_workload(w, stencil=stencil, kernels=kernels,
                              options={pf.PF_OPT_PRECOND: precond, pf.PF_OPT_HISTORY: 4096, pf.PF_OPT_NORM: norm})
    x = torch.zeros(w.n, dtype=torch.float64, device="cuda") if x0 is None else torch.tensor(x0, device="cuda")
    sg = None if sigma is None else torch.tensor(sigma, device="cuda")
    out = g.solve_linear(w.rhs, x=x, tol=tol, maxit=maxit, sigma=sg)
    out["hist"] = g.history(4096)
    g.close()
    return out


# one brick per block with ragged splits in every direction, a single plane of bricks, the smallest box, boxes
# whose bricks have one node along an axis, 148 blocks and fewer
SHAPES = [(3, 3, 3), (5, 4, 3), (37, 20, 11), (33, 35, 31), (64, 16, 40), (40, 40, 40), (7, 150, 9), (64, 64, 64)]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("precond", [1, 0])
def test_coop_equals_direct(pf, shape, precond):
    nx, ny, nz = shape
    w = ragged_workload(nx=nx, ny=ny, nz=nz, seed=51 + nx)
    a = _solve(pf, w, pf.KERNELS_DIRECT, precond=precond, tol=1e-10, maxit=300)
    b = _solve(pf, w, pf.KERNELS_COOP, precond=precond, tol=1e-10, maxit=300)
    assert a["status"] == b["status"] and a["iters"] == b["iters"]
    assert torch.equal(a["x"], b["x"])
    assert np.array_equal(a["hist"], b["hist"])
    assert a["relres"] == b["relres"] and a["true_relres"] == b["true_relres"]


@pytest.mark.parametrize("which", ["cfg0", "cfg1", "ragged_sigma_warm"])
def test_coop_against_oracle(pf, oracle, which):
    sigma = x0 = None
    if which == "cfg0":
        w = wl.config0()
        w.rhs = oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges)
    elif which == "cfg1":
        w = wl.config1()
    else:
        w = ragged_workload()
        rng = wl.SplitMix64(3)
        sigma = np.array([rng.uniform_range(0.0, 5.0) for _ in range(w.n)])
        x0 = np.array([rng.uniform_range(-1.0, 1.0) for _ in range(w.n)])
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, x0=x0, sigma=sigma, tol=1e-10,
                              history=True)
    out = _solve(pf, w, pf.KERNELS_COOP, x0=x0, sigma=sigma)
    assert ref["status"] == 0 and out["status"] == 0
    assert abs(out["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"]), (out["iters"], ref["iters"])
    assert out["true_relres"] <= 1.05e-10
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9
    m = min(len(out["hist"]), len(ref["hist"]))
    assert np.allclose(out["hist"][: m // 2], ref["hist"][: m // 2], rtol=1e-6)


def test_coop_paper_stopping_test(pf, oracle):
    """Table 3 steps 18-19 as written (absolute maximum norm < 1e-6): the maximum is reduced with the sums."""
    w = ragged_workload(nx=70, ny=37, nz=19, seed=9)
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=1e-6, history=True,
                              norm=oracle.NORM_ABS_INF)
    out = _solve(pf, w, pf.KERNELS_COOP, tol=1e-6, norm=pf.NORM_ABS_INF)
    assert ref["status"] == 0 and out["status"] == 0 and out["iters"] == ref["iters"]
    assert np.allclose(out["hist"], ref["hist"], rtol=1e-8)
    assert rel_l2(out["x"].cpu().numpy(), ref["x"]) <= 1e-9


def test_coop_degenerate_cases(pf, oracle):
    w = ragged_workload(mixed_bc=False)
    g = pf.Grid.from_workload(w, stencil=2, kernels=pf.KERNELS_COOP)
    x = torch.ones(w.n, dtype=torch.float64, device="cuda")
    out = g.solve_linear(np.zeros(w.n), x=x)                        # b = 0: x = 0, no iterations (Q3)
    assert out["status"] == 0 and out["iters"] == 0 and float(x.abs().max()) == 0.0
    x = torch.full((w.n,), 0.5, dtype=torch.float64, device="cuda")
    out = g.solve_linear(w.rhs, x=x, maxit=0)                       # maxit = 0: x = x0 with Dirichlet values forced
    assert out["status"] == 1 and out["iters"] == 0
    ref = oracle.set_dirichlet(w.nx, w.ny, w.nz, w.bc_type, w.bc_value, np.full(w.n, 0.5))
    assert np.array_equal(x.cpu().numpy(), ref)
    sol = g.solve_linear(w.rhs, tol=1e-12)["x"]
    out = g.solve_linear(w.rhs, x=sol.clone(), tol=1e-8)            # warm start at the solution
    assert out["status"] == 0 and out["iters"] == 0
    out = g.solve_linear(w.rhs, tol=0.0, maxit=7)                   # exactly maxit iterations
    assert out["status"] == 1 and out["iters"] == 7
    g.close()


def test_coop_pf_solve(pf, oracle):
    """configs[0]: the nonlinear PF loop with every linear solve in the cooperative kernel: same bits as with the
    one-thread-per-node kernels, and the oracle's potential and concentrations within 1e-7."""
    w = wl.config0()
    sp = w.species
    res = []
    for kernels in (pf.KERNELS_DIRECT, pf.KERNELS_COOP):
        g = pf.Grid.from_workload(w, stencil=2, kernels=kernels)
        res.append(g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol))
        g.close()
    a, b = res
    assert a["status"] == 0 and b["status"] == 0
    assert a["outer_iters"] == b["outer_iters"] and a["lin_iters_hist"] == b["lin_iters_hist"]
    assert torch.equal(a["phi"], b["phi"]) and torch.equal(a["conc"], b["conc"])
    ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                          sp.radii, w.l_c, w.nonlinear_tol)
    assert ref["status"] == 0 and b["outer_iters"] == ref["outer_iters"]
    assert rel_l2(b["phi"].cpu().numpy(), ref["phi"]) <= 1e-7
    K = len(sp.valence)
    conc = b["conc"].cpu().numpy()
    for k in range(K + 1):
        assert rel_l2(conc[k], ref["conc"][k]) <= 1e-7, k


def test_coop_not_applicable(pf):
    w = ragged_workload(nx=128, ny=96, nz=80, seed=5)               # bricks would not fit an SM's shared memory
    g = pf.Grid.from_workload(w, stencil=2, kernels=pf.KERNELS_COOP)
    with pytest.raises(pf.PFError) as e:
        g.solve_linear(w.rhs, maxit=5)
    assert e.value.code == pf.PF_ERR_ARG
    g.close()
    w = ragged_workload()
    g = pf.Grid.from_workload(w, stencil=pf.STENCIL_STORED, kernels=pf.KERNELS_COOP)      # needs the code form
    with pytest.raises(pf.PFError):
        g.solve_linear(w.rhs, maxit=5)
    g.close()


def test_coop_random_shapes_repeatable(pf):
    """Twelve seeded random box shapes, each solved three times by the cooperative kernel: every run gives the bits
    of the one-thread-per-node kernels (a race in the barrier or in the halo reads would show up as a run-to-run
    difference)."""
    rng = np.random.default_rng(123)
    for trial in range(12):
        nx, ny, nz = (int(v) for v in rng.integers(3, 64, size=3))
        w = ragged_workload(nx=nx, ny=ny, nz=nz, seed=1000 + trial)
        ref = _solve(pf, w, pf.KERNELS_DIRECT, maxit=300)
        g = pf.Grid.from_workload(w, stencil=2, kernels=pf.KERNELS_COOP, options={pf.PF_OPT_HISTORY: 4096})
        for _ in range(3):
            x = torch.zeros(w.n, dtype=torch.float64, device="cuda")
            out = g.solve_linear(w.rhs, x=x, tol=1e-10, maxit=300)
            assert out["iters"] == ref["iters"] and torch.equal(out["x"], ref["x"]), (nx, ny, nz)
            assert np.array_equal(g.history(4096), ref["hist"])
        g.close()
