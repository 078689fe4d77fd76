"""Seeded synthetic inputs for BASELINE.json's five configurations.

This module holds NONE of the method's arithmetic: it only draws geometry,
charges and QEq parameters.  Both the CUDA path (tests, bench.py) and the
oracle's tests consume the fp32 arrays it returns; neither side's code lives
here.  The inputs stand in for the paper's "randomly generated water-like
systems" and water clusters, which
are not available; the recipe is DESIGN.md section 4.

Seeds: 20250321 + cfg (positions), +100 (chi, J), +200 (velocities),
+300+k (k-th perturbation).
"""
from dataclasses import dataclass, field

import numpy as np

SEED0 = 20250321
KE_EV_A = 14.3996454784255          # eV*Angstrom/e^2
D_OH = 0.9572                       # Angstrom
THETA_HOH = 104.52                  # degrees
Q_O, Q_H = -0.834, 0.417            # e
MASS_O, MASS_H = 15.999, 1.008      # amu
K_REP, R_REP = 10.0, 2.9            # eV/A^2, A: O-O soft-sphere repulsion of the MD stand-in


@dataclass
class Config:
    index: int
    name: str
    kind: str            # "water" | "nacl"
    n_lattice: int       # molecules (water) or ion sites (nacl) per axis
    L: float             # cubic box edge, Angstrom
    rc: float            # real-space cutoff
    alpha: float         # Ewald splitting parameter, 1/Angstrom
    grid: int            # PME grid points per axis
    order: int = 6
    skin: float = 0.0    # list cutoff = rc + skin
    workload: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def n_atoms(self) -> int:
        return 3 * self.n_lattice ** 3 if self.kind == "water" else self.n_lattice ** 3

    @property
    def box(self):
        return np.array([self.L, self.L, self.L], dtype=np.float64)

    @property
    def r_list(self) -> float:
        return self.rc + self.skin


CONFIGS = [
    Config(0, "water216", "water", 6, 18.62, 9.0, 0.35, 24, 6, 0.0,
           "1 nl_build + 1 coulomb + 1 qeq_solve"),
    Config(1, "nacl8000", "nacl", 20, 56.4, 10.0, 0.32, 64, 6, 0.0,
           "1 nl_build + 1 coulomb (jittered) + Madelung check (sigma 0)",
           extra=dict(a=5.64, sigma=0.1)),
    Config(2, "water8000", "water", 20, 62.1, 9.0, 0.35, 72, 6, 0.0,
           "50 QEq Krylov iterations, each one PME Coulomb evaluation"),
    Config(3, "water32768", "water", 32, 99.4, 9.0, 0.35, 108, 6, 1.0,
           "evaluations with a rebuild every 10, sigma 0.02 A perturbations"),
    Config(4, "water110592", "water", 48, 149.0, 9.0, 0.35, 160, 6, 1.0,
           "100 shadow-QEq XL-BOMD steps, 0.5 fs, 4 Krylov updates, rebuild every 10"),
]


def _water_frame():
    h = np.deg2rad(THETA_HOH) / 2.0
    return np.array([[0.0, 0.0, 0.0],
                     [D_OH * np.sin(h), D_OH * np.cos(h), 0.0],
                     [-D_OH * np.sin(h), D_OH * np.cos(h), 0.0]])


def water_box(n: int, L: float, seed: int):
    """n^3 rigid 3-site waters, O on an n^3 lattice with +-0.3 A jitter, random orientation.

    Draw order per molecule: rng.uniform(-0.3, 0.3, 3) then rng.normal(size=4)
    (unit quaternion), molecules in m = (ix*n+iy)*n+iz order, atom order O,H,H.
    Positions are left unwrapped.  Returns fp64 positions [3 n^3, 3], charges.
    """
    rng = np.random.default_rng(seed)
    a = L / n
    frame = _water_frame()
    nm = n ** 3
    pos = np.empty((nm, 3, 3))
    m = 0
    for ix in range(n):
        for iy in range(n):
            for iz in range(n):
                o = (np.array([ix, iy, iz]) + 0.5) * a + rng.uniform(-0.3, 0.3, 3)
                w, x, y, z = (lambda v: v / np.linalg.norm(v))(rng.normal(size=4))
                R = np.array([
                    [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                    [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                    [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])
                pos[m] = o + frame @ R.T
                m += 1
    q = np.tile(np.array([Q_O, Q_H, Q_H]), nm)
    return pos.reshape(-1, 3), q


def nacl_box(n_sites: int, a: float, sigma: float, seed: int):
    """Rock salt: simple-cubic sites (i,j,k)*a/2, q = (-1)^(i+j+k), Gaussian jitter sigma."""
    rng = np.random.default_rng(seed)
    r0 = a / 2.0
    idx = np.stack(np.meshgrid(np.arange(n_sites), np.arange(n_sites), np.arange(n_sites),
                               indexing="ij"), axis=-1).reshape(-1, 3)
    pos = idx.astype(np.float64) * r0
    if sigma > 0:
        pos = pos + rng.normal(0.0, sigma, pos.shape)
    q = np.where(idx.sum(axis=1) % 2 == 0, 1.0, -1.0)
    return pos, q


def make(cfg_index: int, sigma=None):
    """fp32 positions [N,3] and charges [N] of configuration cfg_index (see CONFIGS)."""
    c = CONFIGS[cfg_index]
    seed = SEED0 + c.index
    if c.kind == "water":
        pos, q = water_box(c.n_lattice, c.L, seed)
    else:
        s = c.extra["sigma"] if sigma is None else sigma
        pos, q = nacl_box(c.n_lattice, c.extra["a"], s, seed)
    return np.ascontiguousarray(pos, dtype=np.float32), np.ascontiguousarray(q, dtype=np.float32)


def qeq_params(n_atoms: int, seed: int = SEED0 + 100):
    """cfg 0/2 QEq parameters: J ~ U(5,10) eV/e^2 then chi ~ U(-1,1) eV/e (that draw order)."""
    rng = np.random.default_rng(seed)
    J = rng.uniform(5.0, 10.0, n_atoms)
    chi = rng.uniform(-1.0, 1.0, n_atoms)
    return chi.astype(np.float32), J.astype(np.float32)


def qeq_params_water_pd(n_atoms: int):
    """cfg 4 per-element parameters: chi_O = +16.4, chi_H = -16.4 eV/e,
    u = 60 eV/e^2.  C is positive definite (k_e*A has eigenvalues down to about -20 eV/e^2) and the
    unshielded point-charge model stays bound with the harmonic stand-in (q_O ~ -0.51 e); with
    u = 30 (q_O ~ -0.84 e) the intramolecular O-H Coulomb attraction wins within ~10 steps."""
    chi = np.tile(np.array([16.4, -16.4, -16.4], dtype=np.float32), n_atoms // 3)
    u = np.full(n_atoms, 60.0, dtype=np.float32)
    return chi, u


def masses_water(n_atoms: int):
    return np.tile(np.array([MASS_O, MASS_H, MASS_H], dtype=np.float32), n_atoms // 3)


def velocities(masses, T=300.0, seed: int = SEED0 + 200):
    """Maxwell-Boltzmann velocities in Angstrom/fs, centre-of-mass motion removed."""
    kB = 8.617333e-5           # eV/K
    conv = 0.00964853          # (eV/amu) -> (A/fs)^2
    rng = np.random.default_rng(seed)
    m = np.asarray(masses, dtype=np.float64)
    v = rng.normal(size=(m.size, 3)) * np.sqrt(kB * T / m * conv)[:, None]
    v -= (m[:, None] * v).sum(axis=0) / m.sum()
    return v.astype(np.float32)


def perturb(pos, k: int, sigma: float = 0.02, cfg_index: int = 3):
    """cfg 3: add N(0, sigma^2) to every coordinate (k-th perturbation)."""
    rng = np.random.default_rng(SEED0 + cfg_index + 300 + k)
    return (np.asarray(pos, dtype=np.float64) + rng.normal(0.0, sigma, np.shape(pos))).astype(np.float32)
