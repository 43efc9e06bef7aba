"""Pins for the oracle's operator assembly (rows L1, L2 of 8(a)).

None of these re-types the oracle's own formula: they check it against the paper's SMIB
coefficients (Eqs 17-18), against algebraic invariants, and against the closed-form solution
of a two-dielectric slab.
"""
import numpy as np
import pytest

D, NEU = 0, 1


def _idx(nx, ny, ix, iy, iz):
    return ix + nx * (iy + ny * iz)


def _golden_table1():
    import os
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "table1_constants.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) >= 2:
                out[line[0]] = float(line[1])
    return out


def test_constants_match_table1(oracle):
    """kappa = e^2/(eps_0 k_B T) and k_B T/e recomputed here from the paper's printed Table 1 values
    (tests/golden/table1_constants.txt); reading R0."""
    g = _golden_table1()
    kappa = g["e"] ** 2 / (g["eps_0"] * 100.0 * g["k_B"] * g["T"]) * 1e10      # F/cm -> F/m, m -> A
    assert abs(oracle.kappa() - kappa) <= 1e-12 * kappa
    assert abs(oracle.kappa() - 7048.03) < 0.01
    assert abs(oracle.kT_over_e_volt() - g["k_B"] * g["T"] / g["e"]) < 1e-18
    assert abs(oracle.kT_over_e_volt() * 1e3 - 25.683) < 1e-3
    assert abs(oracle.molar_to_per_A3() - 6.02214076e-4) < 1e-18
    # the species tables of the workloads use the paper's radii
    from paper_1711_04060_b200 import workloads as W
    assert W.NACACL.radii.tolist() == [g["a_Na"], g["a_Ca"], g["a_Cl"], g["a_H2O"]]
    assert W.NACL.radii.tolist() == [g["a_Na"], g["a_Cl"], g["a_H2O"]]


def test_smib_rows_equal_paper_eqs_17_18(oracle):
    """Rows at the two nodes straddling the interface equal Eqs (17)-(18)."""
    nx, ny, nz, h = 10, 3, 3, 0.5
    em, es = 2.0, 78.45                      # Table 1's eps_m, eps_s
    l = 4                                    # x_l in Omega_m, x_{l+1} in Omega_s
    eps = np.empty((nz, ny, nx))
    eps[:, :, : l + 1] = em
    eps[:, :, l + 1:] = es
    bt, bv = [D, D, NEU, NEU, NEU, NEU], [0.0] * 6
    A = oracle.assemble_poisson(nx, ny, nz, h, bt, bv, eps.ravel())
    # paper's coefficients, typed from the paper
    c1 = (em - es) / (em + es)
    c2 = 2 * es / (em + es)
    d1 = 2 * em / (em + es)
    d2 = (es - em) / (em + es)
    i = _idx(nx, ny, l, 1, 1)
    j = _idx(nx, ny, l + 1, 1, 1)
    lateral_m = 4 * em / h ** 2              # the y and z parts of the 7-point row (same medium)
    lateral_s = 4 * es / h ** 2
    # Eq (17): eps_m [ -phi_{l-1} + (2-c1) phi_l - c2 phi_{l+1} ] / dx^2
    assert np.isclose(A[2, i], -em / h ** 2, rtol=1e-14)
    assert np.isclose(A[1, i], -em * c2 / h ** 2, rtol=1e-14)
    assert np.isclose(A[0, i] - lateral_m, em * (2 - c1) / h ** 2, rtol=1e-13)
    # Eq (18): eps_s [ -d1 phi_l + (2-d2) phi_{l+1} - phi_{l+2} ] / dx^2
    assert np.isclose(A[2, j], -es * d1 / h ** 2, rtol=1e-14)
    assert np.isclose(A[1, j], -es / h ** 2, rtol=1e-14)
    assert np.isclose(A[0, j] - lateral_s, es * (2 - d2) / h ** 2, rtol=1e-13)
    # the two interface couplings are the same number (flux form, symmetric)
    assert A[1, i] == A[2, j]


def test_row_sums_and_boundary_rows(oracle):
    rng = np.random.default_rng(5)
    nx, ny, nz, h = 7, 6, 5, 0.5
    eps = rng.choice([2.0, 80.0], size=nx * ny * nz)
    sigma = rng.uniform(0, 3, size=nx * ny * nz)
    bt, bv = [NEU, NEU, D, NEU, D, D], [0, 0, 1.5, 0, -2.0, 0.25]
    A = oracle.assemble_poisson(nx, ny, nz, h, bt, bv, eps, sigma)
    for iz in range(nz):
        for iy in range(ny):
            for ix in range(nx):
                i = _idx(nx, ny, ix, iy, iz)
                dirichlet = iy == 0 or iz == 0 or iz == nz - 1
                if dirichlet:
                    assert A[0, i] == 1.0 and np.all(A[1:, i] == 0.0)
                    continue
                # row sum = sigma_i (flux form, zero-Neumann faces simply dropped)
                assert np.isclose(A[:, i].sum(), sigma[i], rtol=0, atol=1e-10 * abs(A[0, i]))
                assert np.all(A[1:, i] <= 0.0) and A[0, i] > 0
                # omitted outward faces on Neumann sides
                if ix == 0:
                    assert A[2, i] == 0.0
                if ix == nx - 1:
                    assert A[1, i] == 0.0
                if iy == ny - 1:
                    assert A[4, i] == 0.0
    # set_dirichlet: first Dirichlet face in the order -x,+x,-y,+y,-z,+z wins
    x = oracle.set_dirichlet(nx, ny, nz, bt, bv, np.full(nx * ny * nz, 9.0))
    x3 = x.reshape(nz, ny, nx)
    assert np.all(x3[:, 0, :] == 1.5)
    assert np.all(x3[0, 1:, :] == -2.0) and np.all(x3[-1, 1:, :] == 0.25)
    assert np.all(x3[1:-1, 1:, :] == 9.0)


def test_symmetry_on_unknowns(oracle):
    """x^T A y = y^T A x for vectors vanishing on Dirichlet nodes (symmetric)."""
    rng = np.random.default_rng(6)
    nx, ny, nz, h = 9, 8, 7, 0.5
    n = nx * ny * nz
    eps = rng.choice([4.0, 78.5], size=n)
    sigma = rng.uniform(0, 1, size=n)
    bt, bv = [NEU, NEU, NEU, NEU, D, D], [0.0] * 6
    A = oracle.assemble_poisson(nx, ny, nz, h, bt, bv, eps, sigma)
    x = oracle.set_dirichlet(nx, ny, nz, bt, bv, rng.standard_normal(n))
    y = oracle.set_dirichlet(nx, ny, nz, bt, bv, rng.standard_normal(n))
    xAy = x @ oracle.dia_spmv(nx, ny, nz, A, y)
    yAx = y @ oracle.dia_spmv(nx, ny, nz, A, x)
    assert abs(xAy - yAx) <= 1e-12 * abs(xAy)
    # PF1 operator with a single-valued solvent eps is symmetric too
    solv = (eps > 40).astype(np.uint8)
    A1 = oracle.assemble_pf1(nx, ny, nz, h, bt, bv, eps, solv, 1.2)
    m = solv.reshape(nz, ny, nx).copy()
    m[0], m[-1], m[:, 0], m[:, -1], m[:, :, 0], m[:, :, -1] = 0, 0, 0, 0, 0, 0
    x = rng.standard_normal(n) * m.ravel()
    y = rng.standard_normal(n) * m.ravel()
    xAy = x @ oracle.dia_spmv(nx, ny, nz, A1, y)
    yAx = y @ oracle.dia_spmv(nx, ny, nz, A1, x)
    assert abs(xAy - yAx) <= 1e-12 * abs(xAy)


def test_pf1_rows(oracle):
    """PF1 rows: (eps lc^2/h^2)(6 u_i - sum u_nb) + eps u_i on interior solvent nodes (Eq 12)."""
    nx = ny = nz = 6
    h, lc = 0.5, 1.2
    n = nx * ny * nz
    eps = np.full(n, 78.5)
    eps3 = eps.reshape(nz, ny, nx)
    eps3[2, 2, 2] = 4.0
    solv = oracle.solvent_mask(eps)
    assert solv.sum() == n - 1
    bt, bv = [NEU, NEU, NEU, NEU, D, D], [0.0] * 6
    A = oracle.assemble_pf1(nx, ny, nz, h, bt, bv, eps, solv, lc)
    i = _idx(nx, ny, 3, 3, 3)
    c = 78.5 * lc ** 2 / h ** 2
    assert np.allclose(A[1:, i], -c, rtol=1e-15)
    assert np.isclose(A[0, i], 6 * c + 78.5, rtol=1e-15)
    # the PF1 symbol: applied to a constant field on the unknowns it returns eps*const
    # identity rows: the membrane node and every box-boundary node, Neumann faces included (Q15)
    for i in (_idx(nx, ny, 2, 2, 2), _idx(nx, ny, 0, 3, 3), _idx(nx, ny, 3, 5, 2), _idx(nx, ny, 3, 3, 0)):
        assert A[0, i] == 1.0 and np.all(A[1:, i] == 0.0)


def test_solvent_mask_reading_q17(oracle):
    assert np.all(oracle.solvent_mask(np.full(10, 3.0)) == 1)           # uniform => all solvent
    m = oracle.solvent_mask(np.array([2.0, 80.0, 41.0, 40.9, 80.0]))
    assert m.tolist() == [0, 1, 0, 0, 1]                                # eps > midpoint (41) only


@pytest.mark.parametrize("l", [3, 10])
def test_two_dielectric_slab_closed_form(oracle, l):
    """1-D slab: piecewise-linear phi with eps1 phi1' = eps2 phi2', interface at a face midpoint.

    Series-resistance closed form: the drop across each grid interval is J/eps_interval with
    1/eps of the interface interval = (1/eps1 + 1/eps2)/2; this is the continuum solution with
    the interface at z = (l + 1/2) h, sampled at the nodes.
    """
    nx = ny = 3
    nz, h, V = 21, 0.5, 1.7
    e1, e2 = 2.0, 80.0
    eps = np.empty((nz, ny, nx))
    eps[: l + 1] = e1
    eps[l + 1:] = e2
    bt, bv = [NEU, NEU, NEU, NEU, D, D], [0, 0, 0, 0, 0.0, V]
    n = nx * ny * nz
    r = oracle.solve_linear(nx, ny, nz, h, bt, bv, eps.ravel(), np.zeros(n), tol=1e-14, maxit=2000)
    assert r["status"] == 0
    # continuum solution with the interface at zi
    zi = (l + 0.5) * h
    L = (nz - 1) * h
    J = V / (zi / e1 + (L - zi) / e2)
    z = np.arange(nz) * h
    exact = np.where(z <= zi, J * z / e1, J * zi / e1 + J * (z - zi) / e2)
    phi = r["x"].reshape(nz, ny, nx)
    assert np.abs(phi - exact[:, None, None]).max() < 1e-11 * V
    # flux continuity across the interface, eps1 phi1' = eps2 phi2'
    f1 = e1 * (phi[l, 1, 1] - phi[l - 1, 1, 1])
    f2 = e2 * (phi[l + 3, 1, 1] - phi[l + 2, 1, 1])
    assert np.isclose(f1, f2, rtol=1e-9)


def test_charge_deposition(oracle):
    """Trilinear deposition conserves total charge and its first moment (Eq 3 discretised)."""
    nx = ny = nz = 8
    h = 0.5
    ch = np.array([[1.3, 2.05, 0.77, 0.5], [2.9, 1.0, 3.2, -0.5], [1.3, 2.05, 0.77, 0.25]])
    b = oracle.deposit_charges(nx, ny, nz, h, ch).reshape(nz, ny, nx)
    kap = oracle.kappa()
    # sum_i b_i h^3 / kappa = total charge
    assert np.isclose(b.sum() * h ** 3 / kap, ch[:, 3].sum(), rtol=1e-13)
    z, y, x = np.meshgrid(np.arange(nz) * h, np.arange(ny) * h, np.arange(nx) * h, indexing="ij")
    for ax, col in ((x, 0), (y, 1), (z, 2)):
        assert np.isclose((b * ax).sum() * h ** 3 / kap, (ch[:, 3] * ch[:, col]).sum(), rtol=1e-12)
    # a charge sitting exactly on a node goes to that node only
    b1 = oracle.deposit_charges(nx, ny, nz, h, np.array([[1.0, 1.5, 2.0, 1.0]])).reshape(nz, ny, nx)
    assert np.isclose(b1[4, 3, 2], kap / h ** 3, rtol=1e-15) and np.count_nonzero(b1) == 1
