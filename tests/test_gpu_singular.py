"""GPU parity of the singular-charge decomposition (charge model 1; Eqs (5)-(10)) against the
oracle: phi^L, phi*, b^IF element by element, then the nonlinear PF solve on top of b^IF."""
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


@pytest.mark.parametrize("which,kernels", [("cfg0", 2), ("cfg0", 1), ("cfg2_48", 2)])
def test_setup_matches_oracle(pf, oracle, which, kernels):
    """Coulomb sums, Laplace solve and interface vector: the same operations in the same order on both sides."""
    w = wl.config0() if which == "cfg0" else wl.config2(n=48, volt_mv=50.0)
    ref = oracle.singular_setup(w.nx, w.ny, w.nz, w.h, w.eps, w.charges, lin_tol=1e-10)
    g = pf.Grid.from_workload(w, kernels=kernels, options={pf.PF_OPT_CHARGE_MODEL: pf.CHARGES_SINGULAR})
    phiL = pf.pf_grid_copy_array(g.handle, 14, w.n).cpu().numpy()
    phistar = pf.pf_grid_copy_array(g.handle, 15, w.n).cpu().numpy()
    bIF = pf.pf_grid_copy_array(g.handle, 7, w.n).cpu().numpy()
    its = pf.pf_grid_laplace_iters(g.handle)
    g.close()
    assert ref["status"] == 0 and abs(its - ref["laplace_iters"]) <= max(1, 0.02 * ref["laplace_iters"])
    assert np.array_equal(phistar, ref["phistar"])                     # bit-exact: same sums in the same order
    assert rel_l2(phiL, ref["phiL"]) <= 1e-9                           # a linear solve: BASELINE's gate
    solvent = oracle.solvent_mask(w.eps).astype(bool)
    assert np.all(phiL[solvent] == 0.0)
    # b^IF amplifies differences of phi^L by eps/h^2: compare relative to its own scale
    assert np.abs(bIF - ref["bIF"]).max() <= 1e-8 * np.abs(ref["bIF"]).max()
    assert np.array_equal(bIF == 0.0, ref["bIF"] == 0.0)


def test_pf_solve_with_singular_charges(pf, oracle):
    """configs[0] with the charges entering through b^IF; the result is the TOTAL potential of Eq (5)."""
    w = wl.config0()
    sp = w.species
    s = oracle.singular_setup(w.nx, w.ny, w.nz, w.h, w.eps, w.charges, lin_tol=1e-10)
    ref = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                          sp.radii, w.l_c, w.nonlinear_tol, lin_tol=w.linear_tol, max_outer=1000, fixed_override=s["bIF"])
    total = ref["phi"] + s["phistar"] + s["phiL"]
    g = pf.Grid.from_workload(w, options={pf.PF_OPT_CHARGE_MODEL: pf.CHARGES_SINGULAR})
    out = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol)
    g.close()
    assert ref["status"] == 0 and out["status"] == 0 and out["outer_iters"] == ref["outer_iters"]
    assert abs(out["linear_iters"] - ref["linear_iters"]) <= 0.02 * ref["linear_iters"]
    assert rel_l2(out["phi"].cpu().numpy(), total) <= 1e-7
    conc = out["conc"].cpu().numpy()
    for k in range(conc.shape[0]):
        assert rel_l2(conc[k], ref["conc"][k]) <= 1e-7, k
    # the decomposition and the deposition model describe the same physics: in the solvent, away from the
    # membrane, the two potentials agree to discretisation error
    g = pf.Grid.from_workload(w)
    dep = g.solve_pf(sp.valence, sp.bath_molar, sp.radii, w.l_c, w.nonlinear_tol, want_conc=False)["phi"].cpu().numpy()
    g.close()
    solvent = oracle.solvent_mask(w.eps).astype(bool)
    scale = np.abs(dep[solvent]).max()
    assert np.abs(out["phi"].cpu().numpy() - dep)[solvent].max() <= 0.15 * scale


def test_uniform_map_is_rejected(pf):
    w = wl.config0(n=16)
    w.eps = np.full(w.n, 78.5)
    with pytest.raises(pf.PFError) as e:
        pf.Grid.from_workload(w, options={pf.PF_OPT_CHARGE_MODEL: pf.CHARGES_SINGULAR})
    assert e.value.code == pf.PF_ERR_ARG
