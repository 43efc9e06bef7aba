"""Pins for the oracle's pointwise Fermi update (row N1 of 8(a)).

Eq (1):  C_k = C_k^B exp(-z_k phi + (v_k/v_0) S),  S = ln(Gamma/Gamma^B),
Gamma = 1 - sum_k v_k C_k.  The pins: the paper's own statements (phi = 0 gives the bath,
PAPER.md:47; saturation C_k < 1/v_k), a closed form for equal radii, the
Boltzmann limit, the three definitions holding simultaneously on the outputs, and an independent
bracketing root-finder (scipy brentq) on the scalar equation for Gamma.
"""
import numpy as np
import pytest

from paper_1711_04060_b200 import workloads as W

MOLAR = 6.02214076e-4          # 1 mol/L in 1/A^3 (typed here, not read from the oracle)
WATER = 55.5


def _vol(radii):
    return 4.0 * np.pi * np.asarray(radii) ** 3 / 3.0


def _bath(species, water=WATER):
    cb = np.append(species.bath_molar, water) * MOLAR
    v = _vol(species.radii)
    return cb, v, 1.0 - (v * cb).sum()


@pytest.mark.parametrize("species", [W.NACL, W.NACACL])
def test_phi_zero_gives_bath(oracle, species):
    """phi = 0 yields Gamma = Gamma^B, hence S = 0 and C = C^B."""
    cb, v, gB = _bath(species)
    r = oracle.fermi_pointwise(species.valence, species.bath_molar, species.radii, np.zeros(5))
    assert r["status"] == 0
    assert abs(r["gammaB"] - gB) < 1e-15
    assert np.abs(r["S"]).max() < 5e-15
    assert np.allclose(r["conc"], cb[:, None], rtol=1e-14, atol=0)
    assert np.abs(r["rho"]).max() < 1e-17                     # neutral bath
    # survey Q12: Gamma^B = 0.61412 (config 0), 0.61409 (config 2) with 55.5 mol/L water
    assert abs(gB - (0.61412 if species is W.NACL else 0.61409)) < 1e-5


def test_equal_radii_closed_form(oracle):
    """All radii equal => v_k/v_0 = 1 and Eq (1) solves in closed form (Bikerman-type):
    Gamma/Gamma^B = 1/(Gamma^B + sum_j v C_j^B e^{-z_j phi})."""
    val, bath, a = np.array([1.0, 2.0, -1.0]), np.array([0.1, 0.05, 0.2]), 1.3
    radii = np.full(4, a)
    cb = np.append(bath, WATER) * MOLAR
    z = np.append(val, 0.0)
    v = _vol(a)
    gB = 1.0 - v * cb.sum()
    phi = np.array([-7.0, -1.0, 0.0, 0.3, 2.5, 11.0])
    r = oracle.fermi_pointwise(val, bath, radii, phi)
    denom = gB + (v * cb[:, None] * np.exp(-z[:, None] * phi[None, :])).sum(0)
    assert np.allclose(r["S"], -np.log(denom), rtol=1e-12, atol=1e-14)
    assert np.allclose(r["conc"], cb[:, None] * np.exp(-z[:, None] * phi[None, :]) / denom, rtol=1e-12)


@pytest.mark.parametrize("species", [W.NACL, W.NACACL])
def test_three_definitions_hold_simultaneously(oracle, species):
    """On the outputs: Gamma := 1 - sum v_k C_k > 0, S = ln(Gamma/Gamma^B), and each C_k obeys Eq (1).
    (The 'total excluded volume fraction stays below 1' invariant of the north star.)"""
    cb, v, gB = _bath(species)
    z = np.append(species.valence, 0.0)
    v0 = v.mean()
    phi = np.array([-500.0, -50.0, -12.0, -3.0, -0.5, 0.0, 0.7, 4.0, 20.0, 50.0, 500.0])
    r = oracle.fermi_pointwise(species.valence, species.bath_molar, species.radii, phi)
    occ = (v[:, None] * r["conc"]).sum(0)
    gam_from_S = gB * np.exp(r["S"])
    assert np.all(np.isfinite(r["S"])) and np.all(occ > 0.0)   # Gamma = Gamma^B e^S > 0 ...
    # ... occ may ROUND to 1 when Gamma < 1e-16; exp() of an argument ~1e3 carries ~1e-13 relative error
    assert np.all(occ <= 1.0 + 1e-12)
    assert np.all(occ[np.abs(phi) <= 12.0] < 1.0)
    assert np.abs(occ + gam_from_S - 1.0).max() < 1e-12
    # Eq (1) itself, evaluated here in log form to survive phi = +-500
    logc = np.log(cb)[:, None] - z[:, None] * phi[None, :] + (v / v0)[:, None] * r["S"][None, :]
    ok = logc > -700.0                                     # below that exp() underflows to 0
    assert np.all(r["conc"][~ok] < 1e-300)
    assert np.allclose(np.log(r["conc"][ok]), logc[ok], rtol=1e-13, atol=1e-11)
    # C_k < 1/v_k for arbitrary phi
    assert np.all(r["conc"] <= (1.0 / v)[:, None] * (1 + 1e-12))
    assert np.all(r["conc"][:, np.abs(phi) <= 12.0] < (1.0 / v)[:, None])
    # charge density and the inexact-Newton derivative: rho = sum z C,
    # rho' = -sum z^2 C with S held fixed; sigma = -kappa rho'
    K = len(species.valence)
    assert np.allclose(r["rho"], (species.valence[:, None] * r["conc"][:K]).sum(0), rtol=1e-13)
    assert np.allclose(r["sigma"], oracle.kappa() * (species.valence[:, None] ** 2 * r["conc"][:K]).sum(0), rtol=1e-13)


@pytest.mark.parametrize("species", [W.NACL, W.NACACL])
def test_against_bracketing_root_finder(oracle, species):
    """Independent solve: eliminate C_k and find Gamma in (0,1) with brentq on
    F(G) = 1 - G - sum_k v_k C_k^B e^{-z_k phi} (G/Gamma^B)^{v_k/v_0}   (monotone decreasing)."""
    from scipy.optimize import brentq
    cb, v, gB = _bath(species)
    z = np.append(species.valence, 0.0)
    lam = v / v.mean()
    phis = np.array([-30.0, -8.0, -2.0, -0.1, 0.4, 3.0, 9.0, 25.0])
    r = oracle.fermi_pointwise(species.valence, species.bath_molar, species.radii, phis)
    for j, phi in enumerate(phis):
        F = lambda G: 1.0 - G - float(np.sum(v * cb * np.exp(-z * phi + lam * np.log(G / gB))))
        G = brentq(F, 1e-300, 1.0, xtol=1e-300, rtol=4 * np.finfo(float).eps, maxiter=500)
        assert abs(r["S"][j] - np.log(G / gB)) < 1e-10 * max(1.0, abs(r["S"][j]))


def test_boltzmann_limit(oracle):
    """Steric switched off (all radii 0, Q25): S = 0 and C_k = C_k^B e^{-z_k phi} exactly;
    tiny radii approach it.  Also pins rho' by a finite difference (sign and z^2)."""
    val, bath = np.array([1.0, -1.0]), np.array([0.1, 0.1])
    phi = np.array([-3.0, -0.2, 0.0, 1.1, 4.0])
    r = oracle.fermi_pointwise(val, bath, np.zeros(3), phi)
    assert r["status"] == 0 and np.all(r["S"] == 0.0) and r["gammaB"] == 1.0
    assert np.allclose(r["conc"][:2], (bath * MOLAR)[:, None] * np.exp(-val[:, None] * phi[None, :]), rtol=1e-15)
    assert np.allclose(r["rho"], -2 * 0.1 * MOLAR * np.sinh(phi), rtol=1e-13, atol=1e-20)
    d = 1e-6
    rp = oracle.fermi_pointwise(val, bath, np.zeros(3), phi + d)["rho"]
    rm = oracle.fermi_pointwise(val, bath, np.zeros(3), phi - d)["rho"]
    assert np.allclose(-(rp - rm) / (2 * d) * oracle.kappa(), r["sigma"], rtol=1e-8)
    small = oracle.fermi_pointwise(val, bath, np.array([1e-3, 1e-3, 1e-3]), phi)
    assert np.allclose(small["conc"][:2], r["conc"][:2], rtol=1e-6)
    assert np.abs(small["S"]).max() < 1e-6


def test_outside_solvent_and_nonphysical(oracle):
    """Distribution defined only in Omega_s; Q26 neutrality; Gamma^B > 0."""
    sp = W.NACL
    phi = np.array([1.0, 1.0, -2.0])
    r = oracle.fermi_pointwise(sp.valence, sp.bath_molar, sp.radii, phi, solvent=np.array([1, 0, 1], np.uint8))
    assert np.all(r["conc"][:, 1] == 0) and r["sigma"][1] == 0 and r["rho"][1] == 0 and r["S"][1] == 0
    assert r["conc"][0, 0] > 0 and r["sigma"][0] > 0
    bad = oracle.fermi_pointwise(np.array([1.0, -1.0]), np.array([0.1, 0.2]), sp.radii, phi)
    assert bad["status"] == -4                                   # non-neutral bath
    bad = oracle.fermi_pointwise(sp.valence, sp.bath_molar, np.array([0.95, 1.81, 2.5]), phi)
    assert bad["status"] == -4                                   # water alone overfills: Gamma^B <= 0
