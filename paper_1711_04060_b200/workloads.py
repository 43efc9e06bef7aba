"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests, cpu_baseline) and the CUDA path
(tests, bench.py).  It holds none of the method's arithmetic: it only produces
the *inputs* of the method -- a relative-permittivity map eps[N], a list of
point charges, boundary-condition descriptors, species tables and (for the
linear-solve configs) a right-hand side.  Assembly, charge deposition, the
Krylov solver and the Fermi update live in `oracle/` and in `csrc/` separately.

The paper's own workload (NCX_Mj, PDB 3v5u) is not available;
these channel-like grids stand in for it (same scale and structure: a low-eps
slab with an aqueous pore, partial charges in the low-eps region, two baths).

Layout: linear index i = ix + nx*(iy + ny*iz), x fastest.
Node (ix,iy,iz) sits at (ix*h, iy*h, iz*h) Angstrom.

Random numbers: a self-contained splitmix64 counter generator so that every
input is reproducible bit for bit from the seed on any machine.
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Tuple

import numpy as np

_MASK = (1 << 64) - 1

# Nominal scale applied to the smeared charge density of the linear-solve
# configs so the potentials come out in k_BT/e-like magnitudes.  It is an input
# scale only (the solve is linear in it); it is NOT read by oracle or kernels.
RHS_SCALE = 7048.0

DIRICHLET = 0
NEUMANN = 1


class SplitMix64:
    """splitmix64: state += golden; z = mix(state).  Public-domain algorithm."""

    def __init__(self, seed: int):
        self.state = seed & _MASK

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & _MASK
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        return z ^ (z >> 31)

    def uniform(self) -> float:
        """Uniform in [0,1) with 53 random bits."""
        return (self.next_u64() >> 11) * (1.0 / 9007199254740992.0)

    def uniform_range(self, a: float, b: float) -> float:
        return a + (b - a) * self.uniform()


@dataclasses.dataclass
class Species:
    """Ion table for pf_solve_pf: K ions then water (radius only)."""
    names: List[str]
    valence: np.ndarray      # K
    bath_molar: np.ndarray   # K, mol/L
    radii: np.ndarray        # K+1, Angstrom, water last


@dataclasses.dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    h: float
    eps: np.ndarray                   # N float64, relative permittivity per node
    charges: np.ndarray               # (M,4) float64: x,y,z [A], q [e]
    bc_type: np.ndarray               # 6 int32: faces -x,+x,-y,+y,-z,+z
    bc_value: np.ndarray              # 6 float64 (k_BT/e)
    rhs: Optional[np.ndarray] = None  # N float64 (linear-solve configs)
    species: Optional[Species] = None
    l_c: float = 0.0
    linear_tol: float = 1e-10
    nonlinear_tol: float = 1e-8
    seed: int = 0

    @property
    def n(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def shape(self) -> Tuple[int, int, int]:
        return (self.nz, self.ny, self.nx)


# --------------------------------------------------------------------------
# geometry helpers (pure input construction)
# --------------------------------------------------------------------------

def _axes(nx, ny, nz, h):
    x = np.arange(nx, dtype=np.float64) * h
    y = np.arange(ny, dtype=np.float64) * h
    z = np.arange(nz, dtype=np.float64) * h
    return x, y, z


def channel_eps(nx, ny, nz, h, slab_thick, pore_radius, eps_membrane=4.0,
                eps_water=78.5) -> np.ndarray:
    """Slab of eps_membrane centred in z, pierced by a cylinder of water along z."""
    x, y, z = _axes(nx, ny, nz, h)
    xc, yc, zc = 0.5 * (nx - 1) * h, 0.5 * (ny - 1) * h, 0.5 * (nz - 1) * h
    in_slab = np.abs(z - zc) <= 0.5 * slab_thick                      # nz
    r2 = (x[None, :] - xc) ** 2 + (y[:, None] - yc) ** 2              # ny,nx
    in_pore = r2 < pore_radius ** 2
    eps = np.full((nz, ny, nx), eps_water, dtype=np.float64)
    memb = in_slab[:, None, None] & (~in_pore)[None, :, :]
    eps[memb] = eps_membrane
    return eps.reshape(-1)


def channel_charges(rng: SplitMix64, count, nx, ny, nz, h, slab_thick, r_in,
                    r_out=None, q_abs=0.5) -> np.ndarray:
    """+-q_abs charges at uniform positions inside the slab, outside the pore.

    r_out=None: anywhere in the slab outside r_in (config 0) but at least two
    cells away from the lateral box faces; otherwise inside the annulus
    r_in <= r <= r_out (configs 2, 3).  Rejection sampling; the slab is shrunk
    by one cell in z so that all 8 deposit corners are membrane nodes.
    """
    xc, yc, zc = 0.5 * (nx - 1) * h, 0.5 * (ny - 1) * h, 0.5 * (nz - 1) * h
    lo_x, hi_x = 2 * h, (nx - 3) * h
    lo_y, hi_y = 2 * h, (ny - 3) * h
    half = 0.5 * slab_thick - h
    out = np.zeros((count, 4), dtype=np.float64)
    k = 0
    while k < count:
        px = rng.uniform_range(lo_x, hi_x)
        py = rng.uniform_range(lo_y, hi_y)
        pz = rng.uniform_range(zc - half, zc + half)
        sign = 1.0 if rng.uniform() < 0.5 else -1.0
        r = np.hypot(px - xc, py - yc)
        if r < r_in + h:
            continue
        if r_out is not None and r > r_out:
            continue
        out[k] = (px, py, pz, sign * q_abs)
        k += 1
    return out


def sphere_eps(rng: SplitMix64, nx, ny, nz, h, fill=0.30, r_lo=2.0, r_hi=6.0,
               eps_in=2.0, eps_out=80.0) -> np.ndarray:
    """Random overlapping spheres of eps_in until >= `fill` of the nodes are inside."""
    inside = np.zeros((nz, ny, nx), dtype=bool)
    n = nx * ny * nz
    count = 0
    Lx, Ly, Lz = (nx - 1) * h, (ny - 1) * h, (nz - 1) * h
    while count < fill * n:
        cx = rng.uniform_range(0.0, Lx)
        cy = rng.uniform_range(0.0, Ly)
        cz = rng.uniform_range(0.0, Lz)
        r = rng.uniform_range(r_lo, r_hi)
        i0, i1 = max(0, int(np.floor((cx - r) / h))), min(nx - 1, int(np.ceil((cx + r) / h)))
        j0, j1 = max(0, int(np.floor((cy - r) / h))), min(ny - 1, int(np.ceil((cy + r) / h)))
        k0, k1 = max(0, int(np.floor((cz - r) / h))), min(nz - 1, int(np.ceil((cz + r) / h)))
        xs = np.arange(i0, i1 + 1) * h - cx
        ys = np.arange(j0, j1 + 1) * h - cy
        zs = np.arange(k0, k1 + 1) * h - cz
        ball = (zs[:, None, None] ** 2 + ys[None, :, None] ** 2 + xs[None, None, :] ** 2) <= r * r
        sub = inside[k0:k1 + 1, j0:j1 + 1, i0:i1 + 1]
        count += int(np.count_nonzero(ball & ~sub))
        sub |= ball
    eps = np.where(inside, eps_in, eps_out).astype(np.float64)
    return eps.reshape(-1)


def gaussian_rhs(rng: SplitMix64, count, nx, ny, nz, h, sigma_cells=1.0,
                 support=4, scale=RHS_SCALE) -> np.ndarray:
    """Sum of `count` Gaussian-smeared charges, q ~ U[-1,1] e.

    Each Gaussian is truncated at +-support cells around its nearest node and
    renormalised so that its discrete weights sum to exactly q;
    the field is the charge density q*w/h^3 times `scale`.  Centres stay
    support+1 cells away from the box faces.  Boundary nodes are left at 0
    (they carry the Dirichlet value g = 0).
    """
    rho = np.zeros((nz, ny, nx), dtype=np.float64)
    m = support + 1
    for _ in range(count):
        cx = rng.uniform_range(m, nx - 1 - m)      # in cell units
        cy = rng.uniform_range(m, ny - 1 - m)
        cz = rng.uniform_range(m, nz - 1 - m)
        q = rng.uniform_range(-1.0, 1.0)
        ix, iy, iz = int(round(cx)), int(round(cy)), int(round(cz))
        ax = np.arange(ix - support, ix + support + 1)
        ay = np.arange(iy - support, iy + support + 1)
        az = np.arange(iz - support, iz + support + 1)
        wx = np.exp(-0.5 * ((ax - cx) / sigma_cells) ** 2)
        wy = np.exp(-0.5 * ((ay - cy) / sigma_cells) ** 2)
        wz = np.exp(-0.5 * ((az - cz) / sigma_cells) ** 2)
        w = wz[:, None, None] * wy[None, :, None] * wx[None, None, :]
        w *= q / w.sum()
        rho[az[0]:az[-1] + 1, ay[0]:ay[-1] + 1, ax[0]:ax[-1] + 1] += w
    rho *= scale / h ** 3
    return rho.reshape(-1)


def _bc(types, values):
    return np.asarray(types, dtype=np.int32), np.asarray(values, dtype=np.float64)


# --------------------------------------------------------------------------
# the five configs
# --------------------------------------------------------------------------

NACL = Species(["Na+", "Cl-"], np.array([1.0, -1.0]), np.array([0.1, 0.1]),
               np.array([0.95, 1.81, 1.4]))
NACACL = Species(["Na+", "Ca2+", "Cl-"], np.array([1.0, 2.0, -1.0]),
                 np.array([0.1, 0.001, 0.102]), np.array([0.95, 0.99, 1.81, 1.4]))

# +50 mV in k_BT/e with Table 1's constants: the oracle and
# the library compute k_BT/e themselves; tests pass volts through this input.
def millivolt_to_kT(mv: float) -> float:
    kB, T, e = 1.38e-23, 298.15, 1.602e-19
    return mv * 1e-3 * e / (kB * T)


def config0(n: int = 32) -> Workload:
    """32^3 PF smallest instance (BASELINE.json configs[0])."""
    h = 0.5
    rng = SplitMix64(0)
    eps = channel_eps(n, n, n, h, slab_thick=8.0, pore_radius=3.0)
    ch = channel_charges(rng, 20, n, n, n, h, slab_thick=8.0, r_in=3.0)
    t, v = _bc([DIRICHLET] * 6, [0.0] * 6)
    return Workload("cfg0_pf_32", n, n, n, h, eps, ch, t, v, species=NACL, l_c=1.2,
                    linear_tol=1e-10, nonlinear_tol=1e-8, seed=0)


def config1(n: int = 64, seed: int = 1, ncharges: int = 500) -> Workload:
    """64^3 single linear solve on a two-region random-sphere eps field."""
    h = 0.5
    rng = SplitMix64(seed)
    eps = sphere_eps(rng, n, n, n, h)
    rhs = gaussian_rhs(rng, ncharges, n, n, n, h)
    t, v = _bc([DIRICHLET] * 6, [0.0] * 6)
    return Workload(f"cfg1_linear_{n}", n, n, n, h, eps, np.zeros((0, 4)), t, v, rhs=rhs,
                    linear_tol=1e-10, seed=seed)


def _channel(name, n, slab, pore, ncharges, seed, volt_mv, species) -> Workload:
    h = 0.5
    rng = SplitMix64(seed)
    eps = channel_eps(n, n, n, h, slab_thick=slab, pore_radius=pore)
    ch = channel_charges(rng, ncharges, n, n, n, h, slab_thick=slab, r_in=pore, r_out=4.0 * pore)
    t, v = _bc([NEUMANN, NEUMANN, NEUMANN, NEUMANN, DIRICHLET, DIRICHLET],
               [0.0, 0.0, 0.0, 0.0, 0.0, millivolt_to_kT(volt_mv)])
    return Workload(name, n, n, n, h, eps, ch, t, v, species=species, l_c=1.2,
                    linear_tol=1e-10, nonlinear_tol=1e-8, seed=seed)


def config2(n: int = 128, volt_mv: float = 0.0) -> Workload:
    """128^3 full nonlinear PF on the channel geometry, 0 / +50 mV."""
    scale = n / 128.0
    return _channel(f"cfg2_pf_{n}_{int(volt_mv)}mV", n, 30.0 * scale, 5.0 * scale,
                    max(8, int(round(300 * scale ** 3))) if n != 128 else 300, 2, volt_mv, NACACL)


def config3(n: int = 256) -> Workload:
    """256^3 throughput linear solve on the scaled channel geometry."""
    scale = n / 256.0
    nch = 1536 if n == 256 else max(8, int(round(1536 * scale ** 3)))
    return _channel(f"cfg3_linear_{n}", n, 60.0 * scale, 8.0 * scale, nch, 3, 0.0, NACACL)


def config4(n: int = 512) -> Workload:
    """512^3 bandwidth stress: cfg-1 generator, seed 4, plus NaCl species for one PF step.

    The linear solve uses the Gaussian-smeared right-hand side; the PF step needs fixed charges in the
    library's own form (point charges, deposited by the method), so the workload also carries the same number
    of point charges q ~ U[-1,1] e at uniform positions at least five cells inside the box (own seed)."""
    ncharges = 500 if n >= 256 else 100
    w = config1(n=n, seed=4, ncharges=ncharges)
    w.name = f"cfg4_stress_{n}"
    w.species = NACL
    w.l_c = 1.2
    rng = SplitMix64(1004)
    L = (n - 1) * w.h
    ch = np.zeros((ncharges, 4))
    for k in range(ncharges):
        ch[k, 0] = rng.uniform_range(5 * w.h, L - 5 * w.h)
        ch[k, 1] = rng.uniform_range(5 * w.h, L - 5 * w.h)
        ch[k, 2] = rng.uniform_range(5 * w.h, L - 5 * w.h)
        ch[k, 3] = rng.uniform_range(-1.0, 1.0)
    w.charges = ch
    return w
