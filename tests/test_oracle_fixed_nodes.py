"""Pins of the oracle's Omega_f support (interior nodes whose potential an atomic model prescribes;
PAPER.md:213, 224-226; readings F1-F3 of DESIGN.md).  All -m "not gpu"."""
import numpy as np

from paper_1711_04060_b200 import workloads as W

D, NEU = 0, 1


def test_shell_of_fixed_nodes_equals_a_smaller_dirichlet_box(oracle):
    """Prescribing g on the node layer next to the box boundary is the same problem as a box two nodes smaller
    with Dirichlet g on its faces: the two solutions agree on the inner box to solver tolerance."""
    n, h, g = 13, 0.5, 0.8
    rng = W.SplitMix64(3)
    eps3 = np.array([2.0 if rng.uniform() < 0.3 else 80.0 for _ in range(n ** 3)]).reshape(n, n, n)
    rhs3 = np.array([rng.uniform_range(-1, 1) for _ in range(n ** 3)]).reshape(n, n, n)
    shell = np.zeros((n, n, n), dtype=bool)
    shell[1:-1, 1:-1, 1:-1] = True
    shell[2:-2, 2:-2, 2:-2] = False
    idx = np.flatnonzero(shell.reshape(-1))
    big = oracle.solve_linear(n, n, n, h, [D] * 6, [0.0] * 6, eps3.reshape(-1), rhs3.reshape(-1), tol=1e-13,
                              fixed_nodes=(idx, np.full(idx.size, g)))
    m = n - 2
    small = oracle.solve_linear(m, m, m, h, [D] * 6, [g] * 6, eps3[1:-1, 1:-1, 1:-1].reshape(-1),
                                rhs3[1:-1, 1:-1, 1:-1].reshape(-1), tol=1e-13)
    assert big["status"] == 0 and small["status"] == 0
    inner = big["x"].reshape(n, n, n)[1:-1, 1:-1, 1:-1]
    assert np.abs(inner - small["x"].reshape(m, m, m)).max() < 1e-10
    assert np.all(big["x"].reshape(n, n, n)[shell] == g)
    # rows: identity at the fixed nodes, neighbours keep their coupling (Q20)
    A = oracle.assemble_poisson(n, n, n, h, [D] * 6, [0.0] * 6, eps3.reshape(-1), fixed_nodes=(idx, np.full(idx.size, g)))
    assert np.all(A[0, idx] == 1.0) and np.all(A[1:, idx] == 0.0)
    A0 = oracle.assemble_poisson(n, n, n, h, [D] * 6, [0.0] * 6, eps3.reshape(-1))
    free = np.ones(n ** 3, dtype=bool); free[idx] = False
    assert np.array_equal(A[:, free], A0[:, free])


def test_fixed_plane_1d_closed_form(oracle):
    """A plane of prescribed potential V between two grounded ends, no charge, uniform eps: piecewise linear."""
    nx = ny = 4; nz = 25; h = 0.5; k = 9; V = 1.7
    eps = np.full(nx * ny * nz, 78.5)
    plane = np.zeros((nz, ny, nx), dtype=bool); plane[k] = True
    idx = np.flatnonzero(plane.reshape(-1))
    bt, bv = [NEU, NEU, NEU, NEU, D, D], [0.0] * 6
    r = oracle.solve_linear(nx, ny, nz, h, bt, bv, eps, np.zeros_like(eps), tol=1e-14, fixed_nodes=(idx, np.full(idx.size, V)))
    z = np.arange(nz)
    exact = np.where(z <= k, V * z / k, V * (nz - 1 - z) / (nz - 1 - k))
    assert np.abs(r["x"].reshape(nz, ny, nx) - exact[:, None, None]).max() < 1e-12


def test_pf_excludes_fixed_nodes_from_the_continuum_model(oracle):
    """Table 2 solves PF1 and PF2 outside Omega_f: there Psi = 0, no Fermi distribution (C = 0), phi = phi_b; the
    rest of the field feels the prescribed values."""
    w = W.config0(n=16)
    sp = w.species
    c = w.nx // 2
    sites = [(c, c, c - 1), (c, c, c), (c, c, c + 1)]                       # three nodes inside the pore
    idx = np.array([x + w.nx * (y + w.ny * z) for x, y, z in sites])
    vals = np.array([-2.0, -3.0, -2.5])
    solvent = oracle.solvent_mask(w.eps).astype(bool)
    assert np.all(solvent[idx])
    r = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                        sp.radii, w.l_c, 1e-8, max_outer=600, fixed_nodes=(idx, vals))
    r0 = oracle.solve_pf(w.nx, w.ny, w.nz, w.h, w.bc_type, w.bc_value, w.eps, w.charges, sp.valence, sp.bath_molar,
                         sp.radii, w.l_c, 1e-8, max_outer=600)
    assert r["status"] == 0 and r0["status"] == 0
    assert np.allclose(r["phi"][idx], vals, rtol=1e-14) and np.all(r["psi"][idx] == 0.0)
    assert np.all(r["conc"][:, idx] == 0.0) and np.all(r["steric"][idx] == 0.0)
    assert np.abs(r["phi"] - r0["phi"]).max() > 0.5                          # the sites matter
    # a neighbour of a site is an ordinary solvent node: Eq (1) holds there
    nb = idx[0] - 1
    ref = oracle.fermi_pointwise(sp.valence, sp.bath_molar, sp.radii, r["phi"][nb:nb + 1])
    assert np.allclose(r["conc"][:, nb], ref["conc"][:, 0], rtol=1e-12)
