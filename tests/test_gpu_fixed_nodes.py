"""GPU parity for Omega_f (nodes with prescribed potential; readings F1-F3) against the oracle."""
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
    _build.build()
    _pf.load()
    return _pf


def rel_l2(a, b):
    d = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (d if d > 0 else 1.0)


def _sites(w, count, seed):
    """`count` distinct solvent nodes strictly inside the box, with potentials in [-3, 1]."""
    rng = wl.SplitMix64(seed)
    eps3 = w.eps.reshape(w.nz, w.ny, w.nx)
    idx, vals = [], []
    while len(idx) < count:
        x = 1 + int(rng.uniform() * (w.nx - 2)); y = 1 + int(rng.uniform() * (w.ny - 2)); z = 1 + int(rng.uniform() * (w.nz - 2))
        i = x + w.nx * (y + w.ny * z)
        if eps3[z, y, x] > 40.0 and i not in idx:
            idx.append(i); vals.append(rng.uniform_range(-3.0, 1.0))
    return np.array(idx), np.array(vals)


@pytest.mark.parametrize("stencil,kernels", [(1, 1), (2, 1), (2, 2)])
def test_linear_solve_with_fixed_nodes(pf, oracle, stencil, kernels):
    w = wl.config2(n=48, volt_mv=50.0)
    w.rhs = oracle.deposit_charges(w.nx, w.ny, w.nz, w.h, w.charges)
    fixed = _sites(w, 40, 5)
    A = oracle.assemble_poisson(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, fixed_nodes=fixed)
    ref = oracle.solve_linear(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.rhs, tol=1e-10, fixed_nodes=fixed)
    g = pf.Grid.from_workload(w, stencil=stencil, kernels=kernels, fixed_nodes=fixed)
    assert np.array_equal(pf.pf_grid_copy_array(g.handle, 0, w.n).cpu().numpy(), A[0])
    offd = (np.stack([pf.pf_grid_copy_array(g.handle, d, w.n).cpu().numpy() for d in range(1, 7)]) if stencil == 1
            else pf.decode_offdiagonals(g.handle, w.nx, w.ny, w.nz))
    assert np.array_equal(offd, A[1:])
    out = g.solve_linear(w.rhs, tol=1e-10)
    g.close()
    assert ref["status"] == 0 and out["status"] == 0
    assert abs(out["iters"] - ref["iters"]) <= max(1, 0.02 * ref["iters"])
    x = out["x"].cpu().numpy()
    assert np.array_equal(x[fixed[0]], fixed[1]) and rel_l2(x, ref["x"]) <= 1e-9 and out["true_relres"] <= 1.05e-10


def test_pf_solve_with_fixed_nodes(pf, oracle):
    w = wl.config0()
    sp = w.species
    fixed = _sites(w, 12, 9)
    ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                          sp.radii, w.l_c, w.nonlinear_tol, lin_tol=w.linear_tol, max_outer=1000, fixed_nodes=fixed)
    g = pf.Grid.from_workload(w, fixed_nodes=fixed)
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol)
    psi = pf.pf_grid_copy_array(g.handle, 13, w.n).cpu().numpy()
    g.close()
    assert ref["status"] == 0 and out["status"] == 0 and out["outer_iters"] == ref["outer_iters"]
    assert abs(out["linear_iters"] - ref["linear_iters"]) <= 0.02 * ref["linear_iters"]
    phi = out["phi"].cpu().numpy()
    conc = out["conc"].cpu().numpy()
    assert rel_l2(phi, ref["phi"]) <= 1e-7 and rel_l2(psi, ref["psi"]) <= 1e-7
    for k in range(conc.shape[0]):
        assert rel_l2(conc[k], ref["conc"][k]) <= 1e-7, k
    assert np.allclose(phi[fixed[0]], fixed[1], rtol=1e-14) and np.all(psi[fixed[0]] == 0.0)
    assert np.all(conc[:, fixed[0]] == 0.0)


def test_fixed_node_errors(pf):
    w = wl.config0(n=16)
    eps = torch.as_tensor(w.eps).cuda()
    h = pf.pf_grid_create(w.nx, w.ny, w.nz, w.h, eps, w.charges, w.bc_type, w.bc_value)
    with pytest.raises(pf.PFError):
        pf.pf_grid_set_fixed_nodes(h, [w.n], [0.0])
    with pytest.raises(pf.PFError):
        pf.pf_grid_set_fixed_nodes(h, [5], [float("nan")])
    pf.pf_grid_destroy(h)
