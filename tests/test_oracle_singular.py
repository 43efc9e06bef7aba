"""Pins of the oracle's singular-charge decomposition (Eqs (5)-(10), flux-jump terms c0, d0 of Eqs (17)-(18);
PAPER.md:85-111, 148-156): closed forms, Gauss's law, the Born ion, and agreement with the independent
charge-deposition model away from the charges.  All -m "not gpu"."""
import numpy as np
import pytest

D, NEU = 0, 1


def _sphere_eps(n, h, R, eps_m=2.0, eps_s=80.0):
    c = (n - 1) * h / 2.0
    ax = np.arange(n) * h - c
    r2 = ax[:, None, None] ** 2 + ax[None, :, None] ** 2 + ax[None, None, :] ** 2
    return np.where(r2 <= R * R, eps_m, eps_s).reshape(-1), c


def test_coulomb_sum_against_numpy(oracle):
    """Eq (5) in the units of R0: phi* = kappa/(4 pi eps_m) sum q_j/|r - r_j|; gradient by central differences."""
    rng = np.random.default_rng(0)
    ch = np.column_stack([rng.uniform(0, 10, (7, 3)), rng.uniform(-1, 1, 7)])
    for p in rng.uniform(-3, 13, (5, 3)):
        ref = oracle.kappa() / (4 * np.pi * 3.5) * np.sum(ch[:, 3] / np.linalg.norm(p - ch[:, :3], axis=1))
        assert np.isclose(oracle.coulomb_potential(ch, 3.5, *p), ref, rtol=1e-13)
        for ax in range(3):
            e = np.zeros(3); e[ax] = 1e-5
            fd = (oracle.coulomb_potential(ch, 3.5, *(p + e)) - oracle.coulomb_potential(ch, 3.5, *(p - e))) / 2e-5
            assert np.isclose(oracle.coulomb_gradient(ch, 3.5, *p, ax), fd, rtol=1e-6)
    assert np.isclose(oracle.kappa() / (4 * np.pi), 560.9, rtol=1e-3)     # e^2/(4 pi eps0 kT) = 560.9 A at 298.15 K


@pytest.mark.parametrize("e1,e2", [(2.0, 80.0), (4.0, 78.5)])
def test_flux_jump_rows_1d_closed_form(oracle, e1, e2):
    """c0, d0 of Eqs (17)-(18): two dielectrics, interface at a face midpoint, prescribed jump
    [eps phi'] = eps2 phi2' - eps1 phi1' = J, Dirichlet 0 / V.  The exact solution is piecewise linear and the
    scheme reproduces it to rounding: pins the sign and the eps-weighted split of the jump between the two rows."""
    nx = ny = 4; nz = 21; h = 0.5; k = 8; V = 1.3; J = 0.7
    eps = np.empty((nz, ny, nx)); eps[:k] = e1; eps[k:] = e2
    eps = eps.reshape(-1)
    bt, bv = [NEU, NEU, NEU, NEU, D, D], [0, 0, 0, 0, 0.0, V]
    solvent = oracle.solvent_mask(eps)
    Jf = np.zeros((6, nx * ny * nz))
    plane = np.zeros((nz, ny, nx), dtype=bool); plane[k - 1] = True
    Jf[5, plane.reshape(-1)] = J                                   # face "up" (d = 6) of the last Omega_m plane
    b = oracle.interface_rhs(nx, ny, nz, h, eps, solvent, Jf)
    A = oracle.assemble_poisson(nx, ny, nz, h, bt, bv, eps)
    b = oracle.set_dirichlet(nx, ny, nz, bt, bv, b)
    x0 = oracle.set_dirichlet(nx, ny, nz, bt, bv, np.zeros_like(b))
    sol = oracle.bicgstab(nx, ny, nz, A, b, x0=x0, tol=1e-14)["x"].reshape(nz, ny, nx)
    zf, L = (k - 0.5) * h, (nz - 1) * h
    # a1 zf + a2 (L - zf) = V,  e2 a2 - e1 a1 = J
    a1 = (e2 * V - J * (L - zf)) / (e2 * zf + e1 * (L - zf))
    a2 = (J + e1 * a1) / e2
    z = np.arange(nz) * h
    exact = np.where(z < zf, a1 * z, a1 * zf + a2 * (z - zf))
    assert np.abs(sol - exact[:, None, None]).max() < 1e-10 * max(1.0, np.abs(exact).max())


def test_gauss_law_and_harmonic_phiL(oracle):
    """A closed molecule (sphere) with three charges inside: phi^L is discretely harmonic, the jumps of its
    normal derivative sum to zero exactly, the Coulomb flux through the staircase surface gives the enclosed
    charge, and b^IF carries the same total source as the deposited point charges: sum b^IF h^3 = kappa sum q."""
    n, h, R = 33, 0.5, 5.0
    eps, c = _sphere_eps(n, h, R)
    ch = np.array([[c + 0.7, c - 0.4, c + 0.2, 0.8], [c - 1.1, c + 0.6, c - 0.9, -0.5], [c + 0.1, c + 1.3, c + 0.8, 0.4]])
    s = oracle.singular_setup(n, n, n, h, eps, ch, lin_tol=1e-13, want_jumps=True)
    assert s["status"] == 0
    solvent = oracle.solvent_mask(eps).reshape(n, n, n).astype(bool)
    u = s["phiL"].reshape(n, n, n)
    m = ~solvent
    core = m[1:-1, 1:-1, 1:-1].copy()
    for sl in ((slice(2, None), slice(1, -1), slice(1, -1)), (slice(None, -2), slice(1, -1), slice(1, -1)),
               (slice(1, -1), slice(2, None), slice(1, -1)), (slice(1, -1), slice(None, -2), slice(1, -1)),
               (slice(1, -1), slice(1, -1), slice(2, None)), (slice(1, -1), slice(1, -1), slice(None, -2))):
        core &= m[sl]
    lap = (u[2:, 1:-1, 1:-1] + u[:-2, 1:-1, 1:-1] + u[1:-1, 2:, 1:-1] + u[1:-1, :-2, 1:-1] + u[1:-1, 1:-1, 2:]
           + u[1:-1, 1:-1, :-2] - 6 * u[1:-1, 1:-1, 1:-1]) / h ** 2
    assert core.sum() > 1000 and np.abs(lap[core]).max() < 1e-8 * np.abs(u).max() / h ** 2
    assert np.all(u[solvent] == 0.0) and np.all(s["phistar"].reshape(n, n, n)[solvent] == 0.0)
    total = s["bIF"].sum() * h ** 3
    assert np.isclose(total, oracle.kappa() * ch[:, 3].sum(), rtol=2e-3)
    fixed = oracle.deposit_charges(n, n, n, h, ch)
    assert np.isclose(fixed.sum() * h ** 3, oracle.kappa() * ch[:, 3].sum(), rtol=1e-12)
    # b^IF lives on the two node layers next to the interface only
    assert np.count_nonzero(s["bIF"]) < 0.2 * n ** 3 and np.count_nonzero(s["bIF"]) > 100


def test_born_ion_and_agreement_with_deposition(oracle):
    """One charge at the centre of a sphere (eps 2 inside, 80 outside), no mobile ions.  (a) Born: the reaction
    potential phi~ + phi^L at the ion equals kappa q/(4 pi R)(1/eps_s - 1/eps_m) up to the staircase surface and
    the finite box; (b) outside the sphere the total potential kappa q/(4 pi eps_s r); (c) the deposition model
    of reading Q22, an independent discretisation of the same problem, agrees with the decomposition in the solvent."""
    n, h, R, q = 49, 0.5, 4.0, 1.0
    eps, c = _sphere_eps(n, h, R)
    ch = np.array([[c, c, c, q]])
    bt, bv = [D] * 6, [0.0] * 6
    s = oracle.singular_setup(n, n, n, h, eps, ch, lin_tol=1e-12)
    tilde = oracle.solve_linear(n, n, n, h, bt, bv, eps, s["bIF"], tol=1e-12)["x"].reshape(n, n, n)
    ic = (n - 1) // 2
    born = oracle.kappa() * q / (4 * np.pi * R) * (1 / 80.0 - 1 / 2.0)
    box = oracle.kappa() * q / (4 * np.pi * 80.0 * c)                # what the grounded box removes, roughly
    rf = tilde[ic, ic, ic] + s["phiL"].reshape(n, n, n)[ic, ic, ic]
    assert abs(rf - born) < 0.03 * abs(born) + box            # measured: 2.2 % at h = 0.5, 1.7 % at h = 0.375
    # (b) along the x axis outside the sphere
    for i in (ic + 12, ic + 16):
        r = (i - ic) * h
        exact = oracle.kappa() * q / (4 * np.pi * 80.0) * (1 / r - 1 / c)    # grounded at distance ~c
        assert abs(tilde[ic, ic, i] - exact) < 0.15 * abs(exact) + 0.02
    # (c) deposition model on the same grid
    dep = oracle.solve_linear(n, n, n, h, bt, bv, eps, oracle.deposit_charges(n, n, n, h, ch), tol=1e-12)["x"].reshape(n, n, n)
    solvent = oracle.solvent_mask(eps).reshape(n, n, n).astype(bool)
    far = solvent.copy(); far[:2] = far[-2:] = False; far[:, :2] = far[:, -2:] = False; far[:, :, :2] = far[:, :, -2:] = False
    rel = np.abs(tilde - dep)[far].max() / np.abs(dep[far]).max()
    assert rel < 0.03                                        # measured 1.3 %
