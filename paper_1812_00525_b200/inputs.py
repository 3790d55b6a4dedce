"""Seeded synthetic inputs for the CLTx hot path -- the ONLY module shared by the CUDA path's
tests/bench and the CPU oracle's tests.  It holds the workload recipe (grids, analytic reference
states, seeded perturbations, physics constants) and none of the method's arithmetic: no stencil,
no RHS, no time stepping.  numpy only; imports neither the CUDA binding nor ``oracle``.

The five configurations are BASELINE.json's ``configs`` (stand-ins for the paper's NOVA/EFIT
equilibrium + m/n = 2/1 tearing-mode case, which is not available):

* box R in [2, 4], Z in [-1, 1], full torus, node counts include the two frozen layers per R/Z side
  and the box edge is a node (reading R1);
* reference state ("equilibrium" of eqs (11)-(14), L105-117): rho0 = 1, p0 = 0.01 (1 - r^2/2),
  r^2 = (R-3)^2 + Z^2, v0 = 0, B_phi0 = 3/R, B_R0 = -(1/R) dpsi/dZ, B_Z0 = (1/R) dpsi/dR with
  psi = 0.1 (1 - r^2)  (configs 1-4)  or  psi = -(1/3) ln(1 + r^2), i.e. q(r) = 1.5 + 1.5 r^2
  (config 5, reading G14);
* state = reference + env(R,Z) * sum_{m=1..3} sum_{n=0..2} a cos(m theta - n phi + chi) per field,
  a ~ U(-1e-4, 1e-4), chi ~ U(0, 2 pi), theta = atan2(Z, R-3),
  env = sin^2(pi (R-Rmin)/(Rmax-Rmin)) sin^2(pi (Z-Zmin)/(Zmax-Zmin))  (readings G11, G12);
  config 5 instead adds 1e-5 env cos(2 theta - phi + chi) to B_R and B_Z only;
* the 72 (a, chi) pairs are drawn in the order field -> m -> n -> (a, chi) from SplitMix64
  (double = (x >> 11) * 2^-53), seed = 181200525 + config index (1-based);
* Gamma = 5/3, eta = nu = D = kappa = 1e-5, CFL = 0.5; the fixed time step handed to both sides is
  the CFL number times the smallest cell-crossing time of the initial state (formula of PAPER.md
  Fig. 4; reading R8) -- a run parameter, computed here once.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 181200525
_MASK = (1 << 64) - 1


class SplitMix64:
    """Counter-based generator (Steele/Lea/Flood 2014); doubles are (x >> 11) * 2**-53."""

    def __init__(self, seed: int):
        self.s = seed & _MASK

    def next_u64(self) -> int:
        self.s = (self.s + 0x9E3779B97F4A7C15) & _MASK
        z = self.s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        return z ^ (z >> 31)

    def next_double(self) -> float:
        return (self.next_u64() >> 11) * (2.0 ** -53)

    def uniform(self, lo: float, hi: float) -> float:
        return lo + (hi - lo) * self.next_double()


@dataclass(frozen=True)
class Config:
    index: int
    name: str
    nR: int
    nphi: int
    nZ: int
    steps: int
    Rmin: float = 2.0
    Rmax: float = 4.0
    Zmin: float = -1.0
    Zmax: float = 1.0
    phi_extent: float = 0.0          # 0 = full torus (2 pi)
    gamma: float = 5.0 / 3.0
    eta: float = 1e-5
    nu: float = 1e-5
    D: float = 1e-5
    kappa: float = 1e-5
    cfl: float = 0.5
    kind: str = "multimode"          # or "tearing" (config 5)

    @property
    def nodes(self) -> int:
        return self.nR * self.nphi * self.nZ

    @property
    def interior(self) -> int:
        return (self.nR - 4) * self.nphi * (self.nZ - 4)

    @property
    def shape(self):
        return (8, self.nphi, self.nZ, self.nR)


CONFIGS = {
    1: Config(1, "tiny-32x16x32", 32, 16, 32, 10),
    2: Config(2, "128x16x128", 128, 16, 128, 100),
    3: Config(3, "256x32x256", 256, 32, 256, 100),
    4: Config(4, "512x64x512", 512, 64, 512, 50),
    5: Config(5, "tearing-256x32x256", 256, 32, 256, 2000, kind="tearing"),
}


def grid_axes(cfg: Config):
    """R_i = Rmin + i*dR, Z_k = Zmin + k*dZ, phi_j = j*dphi (plain double arithmetic)."""
    dR = (cfg.Rmax - cfg.Rmin) / (cfg.nR - 1)
    dZ = (cfg.Zmax - cfg.Zmin) / (cfg.nZ - 1)
    Lphi = cfg.phi_extent if cfg.phi_extent != 0.0 else 2.0 * np.pi
    dphi = Lphi / cfg.nphi
    R = cfg.Rmin + np.arange(cfg.nR, dtype=np.float64) * dR
    Z = cfg.Zmin + np.arange(cfg.nZ, dtype=np.float64) * dZ
    phi = np.arange(cfg.nphi, dtype=np.float64) * dphi
    return R, Z, phi


def reference_state(cfg: Config) -> np.ndarray:
    """U0[8][nZ][nR]: the axisymmetric reference state of the config (see module docstring).

    Not a Grad-Shafranov solution (reading G13): eqs (11)-(14) drop its force residual by construction.
    """
    R, Z, _ = grid_axes(cfg)
    RR, ZZ = np.meshgrid(R, Z, indexing="xy")          # [nZ][nR]
    x = RR - 3.0
    r2 = x * x + ZZ * ZZ
    U0 = np.zeros((8, cfg.nZ, cfg.nR))
    U0[0] = 1.0
    U0[1] = 0.01 * (1.0 - 0.5 * r2)
    if cfg.kind == "tearing":
        dpsi_dR = -(2.0 / 3.0) * x / (1.0 + r2)
        dpsi_dZ = -(2.0 / 3.0) * ZZ / (1.0 + r2)
    else:
        dpsi_dR = -0.2 * x
        dpsi_dZ = -0.2 * ZZ
    U0[5] = -dpsi_dZ / RR
    U0[6] = 3.0 / RR
    U0[7] = dpsi_dR / RR
    return U0


def envelope(cfg: Config) -> np.ndarray:
    R, Z, _ = grid_axes(cfg)
    eR = np.sin(np.pi * (R - cfg.Rmin) / (cfg.Rmax - cfg.Rmin)) ** 2
    eZ = np.sin(np.pi * (Z - cfg.Zmin) / (cfg.Zmax - cfg.Zmin)) ** 2
    return eZ[:, None] * eR[None, :]                   # [nZ][nR]


def initial_state(cfg: Config, U0: np.ndarray | None = None) -> np.ndarray:
    """U[8][nphi][nZ][nR] = reference state + seeded perturbation (module docstring)."""
    if U0 is None:
        U0 = reference_state(cfg)
    R, Z, phi = grid_axes(cfg)
    RR, ZZ = np.meshgrid(R, Z, indexing="xy")
    theta = np.arctan2(ZZ, RR - 3.0)                   # [nZ][nR]
    env = envelope(cfg)
    rng = SplitMix64(SEED_BASE + cfg.index)
    U = np.repeat(U0[:, None, :, :], cfg.nphi, axis=1).copy()
    ph = phi[:, None, None]
    if cfg.kind == "tearing":
        for m in (5, 7):                               # B_R, B_Z
            chi = rng.uniform(0.0, 2.0 * np.pi)
            U[m] += 1e-5 * env[None] * np.cos(2.0 * theta[None] - ph + chi)
        return U
    for f in range(8):
        pert = np.zeros((cfg.nphi, cfg.nZ, cfg.nR))
        for m in (1, 2, 3):
            for n in (0, 1, 2):
                a = rng.uniform(-1e-4, 1e-4)
                chi = rng.uniform(0.0, 2.0 * np.pi)
                pert += a * np.cos(m * theta[None] - n * ph + chi)
        U[f] += env[None] * pert
    return U


def cfl_time_step(cfg: Config, U: np.ndarray) -> float:
    """Run parameter dt = CFL * min over interior nodes of the cell-crossing times (Fig. 4)."""
    R, _, _ = grid_axes(cfg)
    dR = (cfg.Rmax - cfg.Rmin) / (cfg.nR - 1)
    dZ = (cfg.Zmax - cfg.Zmin) / (cfg.nZ - 1)
    Lphi = cfg.phi_extent if cfg.phi_extent != 0.0 else 2.0 * np.pi
    dphi = Lphi / cfg.nphi
    s = (slice(None), slice(None), slice(2, cfg.nZ - 2), slice(2, cfg.nR - 2))
    Ui = U[s]
    c = np.sqrt(np.abs(cfg.gamma * Ui[1] / Ui[0] + (Ui[5] ** 2 + Ui[6] ** 2 + Ui[7] ** 2) / Ui[0]))
    Ri = R[2:cfg.nR - 2][None, None, :]
    t = np.minimum(np.minimum(dR / (np.abs(Ui[2]) + c), dZ / (np.abs(Ui[4]) + c)), Ri * dphi / (np.abs(Ui[3]) + c))
    return float(cfg.cfl * t.min())


@dataclass
class Problem:
    cfg: Config
    U0: np.ndarray
    U: np.ndarray
    dt: float
    extra: dict = field(default_factory=dict)


def make_problem(index: int) -> Problem:
    cfg = CONFIGS[index]
    U0 = reference_state(cfg)
    U = initial_state(cfg, U0)
    return Problem(cfg, U0, U, cfl_time_step(cfg, U))


def custom_config(nR, nphi, nZ, index=99, steps=1, **kw) -> Config:
    """A config with the same recipe at another grid size (parity cases with ragged tiles)."""
    return Config(index, f"custom-{nR}x{nphi}x{nZ}", nR, nphi, nZ, steps, **kw)


def make_custom_problem(nR, nphi, nZ, index=99, rotation=0.0, amplitude_scale=1.0, poloidal=None, **kw) -> Problem:
    """Same recipe on an arbitrary grid.  ``rotation`` = Omega adds a rigid toroidal rotation
    v0 = Omega R phi^ to the reference state (exercises the toroidal v0 terms of eqs (11)-(13)).
    ``poloidal`` = (a, b) adds a compressible poloidal flow  v0_R = a sin(pi x) cos(pi z),
    v0_Z = b cos(2 pi x) sin(pi z) + b/2  (x, z = box coordinates in [0, 1]): div v0, grad v0_R, grad v0_Z,
    (v0.grad)v0 and the R/Z parts of v0 x B0 are all non-zero, on the frozen layers too."""
    cfg = custom_config(nR, nphi, nZ, index=index, **kw)
    U0 = reference_state(cfg)
    if rotation != 0.0:
        R, _, _ = grid_axes(cfg)
        U0[3] = rotation * R[None, :]
    if poloidal is not None:
        a, b = poloidal
        R, Z, _ = grid_axes(cfg)
        x = ((R - cfg.Rmin) / (cfg.Rmax - cfg.Rmin))[None, :]
        z = ((Z - cfg.Zmin) / (cfg.Zmax - cfg.Zmin))[:, None]
        U0[2] = a * np.sin(np.pi * x) * np.cos(np.pi * z)
        U0[4] = b * np.cos(2.0 * np.pi * x) * np.sin(np.pi * z) + 0.5 * b
    U = initial_state(cfg, U0)
    if amplitude_scale != 1.0:
        U = U0[:, None] + amplitude_scale * (U - U0[:, None])
    return Problem(cfg, U0, U, cfl_time_step(cfg, U))
