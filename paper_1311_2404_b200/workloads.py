"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle with the *same* arrays.  It holds
none of the method's arithmetic (no equilibrium, no collision, no streaming): it only draws
fields with numpy.random.Generator(PCG64(seed)) in fp64 and builds node masks.  It imports
neither the oracle nor the CUDA binding.

Every workload stands in for a workload of the paper (which uses no public dataset):
  c1  Taylor-Green vortex, D2Q9            <- PAPER.md section 3.7, 256^2 there
  c2  force-driven channel, D3Q19 LBGK     <- duct flow of section 4.2
  c3  MRT with 5 % random solid obstacles  <- MRT bar of Fig. 7 with complex geometry
  c4  duct with four side walls, fp64      <- duct flow, DP case
  c5  Shan-Chen spinodal decomposition     <- 254x100x100 periodic binary box

Arrays are C-order [z][y][x] (x fastest); u is [D][z][y][x].
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

D2Q9, D3Q19 = 0, 1
BGK, MRT, SC2, REG, LES = 0, 1, 2, 3, 4   # LBGK | MRT | Shan-Chen 2 x LBGK | regularized LBGK | LBGK + Smagorinsky
F32, F64 = 0, 1
FLUID, SOLID, WALL_FULLWAY, VELOCITY = 0, 1, 2, 3   # node types of the geometry mask
FORCE_GUO, FORCE_EDM = 0, 1


def mrt_rates_d3q19(tau: float) -> list:
    """c3 rate vector, reading A7 (moment order of reading A5)."""
    s = 1.0 / tau
    return [0.0, 1.19, 1.4, 0.0, 1.2, 0.0, 1.2, 0.0, 1.2, s, 1.4, s, 1.4, s, s, s, 1.98, 1.98, 1.98]


def mrt_rates_d2q9(tau: float) -> list:
    s = 1.0 / tau
    return [0.0, 1.63, 1.14, 0.0, 1.92, 0.0, 1.92, s, s]


@dataclass
class Workload:
    name: str
    lattice: int
    model: int
    precision: int
    nx: int
    ny: int
    nz: int
    tau: tuple
    steps: int
    force: tuple = (0.0, 0.0, 0.0)
    rates: list | None = None
    sc_G: float = 0.0
    sc_psi: int = 0
    bc_velocity: tuple = (0.0, 0.0, 0.0)
    force_scheme: int = 0                          # 0 Guo (eq. 17), 1 Exact Difference Method (eq. 18)
    smagorinsky_cs: float = 0.0                    # C_S of eq. (9), model LES only
    seed: int | None = None
    mask: np.ndarray | None = None                 # uint8 [nz][ny][nx], 0 FLUID 1 SOLID
    rho: list = field(default_factory=list)        # per component, fp64 [nz][ny][nx]
    u: list = field(default_factory=list)          # per component, fp64 [D][nz][ny][nx]

    @property
    def D(self):
        return 2 if self.lattice == D2Q9 else 3

    @property
    def Q(self):
        return 9 if self.lattice == D2Q9 else 19

    @property
    def sites(self):
        return self.nx * self.ny * self.nz

    @property
    def ncomp(self):
        return 2 if self.model == SC2 else 1

    def params(self) -> dict:
        return dict(lattice=self.lattice, model=self.model, nx=self.nx, ny=self.ny, nz=self.nz,
                    tau=self.tau, rates=self.rates, force=self.force, sc_G=self.sc_G, sc_psi=self.sc_psi,
                    bc_velocity=self.bc_velocity, force_scheme=self.force_scheme,
                    smagorinsky_cs=self.smagorinsky_cs)


def c1_taylor_green(n: int = 128, steps: int = 1000, u0: float = 0.01, tau: float = 0.8,
                    precision: int = F32) -> Workload:
    k = 2.0 * np.pi / n
    y, x = np.meshgrid(np.arange(n, dtype=np.float64), np.arange(n, dtype=np.float64), indexing="ij")
    ux = -u0 * np.cos(k * x) * np.sin(k * y)
    uy = u0 * np.sin(k * x) * np.cos(k * y)
    w = Workload("c1_taylor_green_d2q9_bgk", D2Q9, BGK, precision, n, n, 1, (tau, tau), steps)
    w.mask = np.zeros((1, n, n), np.uint8)
    w.rho = [np.ones((1, n, n))]
    w.u = [np.stack([ux, uy])[:, None, :, :].copy()]
    return w


def c2_channel(nx: int = 256, ny: int = 256, nz: int = 256, steps: int = 2000, tau: float = 0.6,
               g: float = 1e-6, seed: int = 20131102, precision: int = F32) -> Workload:
    rng = np.random.Generator(np.random.PCG64(seed))
    w = Workload("c2_channel_d3q19_bgk", D3Q19, BGK, precision, nx, ny, nz, (tau, tau), steps,
                 force=(g, 0.0, 0.0), seed=seed)
    mask = np.zeros((nz, ny, nx), np.uint8)
    mask[:, 0, :] = 1
    mask[:, ny - 1, :] = 1
    u = rng.uniform(-1e-3, 1e-3, (3, nz, ny, nx))
    u[:, mask == 1] = 0.0
    w.mask, w.rho, w.u = mask, [np.ones((nz, ny, nx))], [u]
    return w


def c3_mrt_obstacles(nx: int = 384, ny: int = 384, nz: int = 384, steps: int = 500, tau: float = 0.55,
                     solid_fraction: float = 0.05, seed: int = 20131103, precision: int = F32) -> Workload:
    rng = np.random.Generator(np.random.PCG64(seed))
    w = Workload("c3_obstacles_d3q19_mrt", D3Q19, MRT, precision, nx, ny, nz, (tau, tau), steps,
                 rates=mrt_rates_d3q19(tau), seed=seed)
    mask = (rng.random((nz, ny, nx)) < solid_fraction).astype(np.uint8)
    u = np.zeros((3, nz, ny, nx))
    u[0] = 0.05
    u[:, mask == 1] = 0.0
    w.mask, w.rho, w.u = mask, [np.ones((nz, ny, nx))], [u]
    return w


def c4_duct(nx: int = 512, ny: int = 256, nz: int = 256, steps: int = 500, tau: float = 0.52,
            g: float = 1e-7, precision: int = F64) -> Workload:
    w = Workload("c4_duct_d3q19_bgk", D3Q19, BGK, precision, nx, ny, nz, (tau, tau), steps,
                 force=(g, 0.0, 0.0))
    mask = np.zeros((nz, ny, nx), np.uint8)
    mask[:, 0, :] = 1
    mask[:, ny - 1, :] = 1
    mask[0, :, :] = 1
    mask[nz - 1, :, :] = 1
    w.mask, w.rho, w.u = mask, [np.ones((nz, ny, nx))], [np.zeros((3, nz, ny, nx))]
    return w


def c5_shan_chen(nx: int = 256, ny: int = 256, nz: int = 256, steps: int = 1000, G: float = 0.9,
                 seed: int = 20131105, precision: int = F32) -> Workload:
    rng = np.random.Generator(np.random.PCG64(seed))
    w = Workload("c5_spinodal_d3q19_sc2", D3Q19, SC2, precision, nx, ny, nz, (1.0, 1.0), steps,
                 sc_G=G, sc_psi=0, seed=seed)
    n = rng.uniform(-0.01, 0.01, (nz, ny, nx))
    w.mask = np.zeros((nz, ny, nx), np.uint8)
    w.rho = [1.0 + n, 1.0 - n]
    w.u = [np.zeros((3, nz, ny, nx)), np.zeros((3, nz, ny, nx))]
    return w


def ldc_cavity(nx: int = 256, ny: int = 256, nz: int = 256, steps: int = 1000, Re: float = 1000.0,
               U: float = 0.05, precision: int = F32, model: int = BGK) -> Workload:
    """Lid-driven cavity, the paper's single-fluid benchmark case (254^3 interior, Re = 1000,
    full bounce-back walls, equilibrium-velocity lid).  Box = interior + one node of wall all round:
    x, z faces and the floor y = 0 are full-way walls, the lid row y = ny-2 moves at (U, 0, 0) and is
    backed by a SOLID row y = ny-1 (which also separates it from the floor on the torus)."""
    nu = U * (nx - 2) / Re
    tau = 3.0 * nu + 0.5
    w = Workload("ldc_cavity_d3q19", D3Q19, model, precision, nx, ny, nz, (tau, tau), steps,
                 rates=mrt_rates_d3q19(tau) if model == MRT else None, bc_velocity=(U, 0.0, 0.0))
    mask = np.zeros((nz, ny, nx), np.uint8)
    mask[:, ny - 2, :] = VELOCITY
    mask[:, 0, :] = WALL_FULLWAY
    mask[:, :, 0] = WALL_FULLWAY
    mask[:, :, nx - 1] = WALL_FULLWAY
    mask[0, :, :] = WALL_FULLWAY
    mask[nz - 1, :, :] = WALL_FULLWAY
    mask[:, ny - 1, :] = SOLID
    w.mask, w.rho, w.u = mask, [np.ones((nz, ny, nx))], [np.zeros((3, nz, ny, nx))]
    return w


def binary_poiseuille(nx: int = 64, ny: int = 256, steps: int = 400000, g: float = 1e-7, G: float = 1.5,
                      density: float = 0.8, minority: float = 0.06, precision: int = F64) -> Workload:
    """Shan-Chen binary Poiseuille flow of the paper's section 5.3: 64 x 256 D2Q9, half-way
    bounce-back walls at y = +-L, fluid of viscosity nu_1 = 1/24 in the core |y| <= L/2 and nu_0 = 1/6
    outside, G = 1.5, body force through the Exact Difference Method, starting from rest.
    Component 0 is the outer fluid, component 1 the core fluid; each phase carries a small amount of
    the other component (`minority`, as a fraction of `density`), since the Shan-Chen model permits
    residual mixing.
    The paper gives G = 1.5 but not the densities.  With psi = rho only the product G * density enters the
    dynamics: at density 1 (G rho = 1.5) the minority density goes negative at the interface and an
    asymmetric mode grows after ~2e5 steps; G rho <= 1.2 stays symmetric to round-off and positive.  So the
    paper's G is kept and the phases are initialised at density 0.8 (reading A22; measured scan in
    section 7).  psi = 1 - exp(-rho) at G = 1.5 does not keep the two fluids apart at all."""
    nu0, nu1 = 1.0 / 6.0, 1.0 / 24.0
    w = Workload("binary_poiseuille_d2q9_sc2", D2Q9, SC2, precision, nx, ny, 1, (3 * nu0 + 0.5, 3 * nu1 + 0.5), steps,
                 force=(g, 0.0, 0.0), sc_G=G, sc_psi=0, force_scheme=FORCE_EDM)
    mask = np.zeros((1, ny, nx), np.uint8)
    mask[:, 0, :] = SOLID
    mask[:, ny - 1, :] = SOLID
    y = np.arange(ny) - (ny - 1) / 2.0
    L = (ny - 2) / 2.0
    core = (np.abs(y) <= L / 2)[None, :, None] * np.ones((1, ny, nx), bool)
    w.mask = mask
    w.rho = [np.where(core, minority * density, density), np.where(core, density, minority * density)]
    w.u = [np.zeros((2, 1, ny, nx)), np.zeros((2, 1, ny, nx))]
    return w


def random_types(lattice: int, nx: int, ny: int, nz: int, seed: int, ncomp: int = 1):
    """Seeded state with all four node types mixed at random (parity tests of the boundary nodes)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    _, rho, u = random_state(lattice, nx, ny, nz, seed + 1, ncomp=ncomp)
    mask = rng.choice(np.array([FLUID] * 7 + [SOLID, WALL_FULLWAY, VELOCITY], np.uint8), size=(nz, ny, nx))
    return mask, rho, u


def random_state(lattice: int, nx: int, ny: int, nz: int, seed: int, solid_fraction: float = 0.0,
                 du: float = 0.02, drho: float = 0.02, ncomp: int = 1):
    """Generic seeded (mask, rho[], u[]) for parity tests at arbitrary (ragged) sizes."""
    rng = np.random.Generator(np.random.PCG64(seed))
    D = 2 if lattice == D2Q9 else 3
    mask = (rng.random((nz, ny, nx)) < solid_fraction).astype(np.uint8)
    rho, u = [], []
    for _ in range(ncomp):
        rho.append(1.0 + rng.uniform(-drho, drho, (nz, ny, nx)))
        uu = rng.uniform(-du, du, (D, nz, ny, nx))
        uu[:, mask == 1] = 0.0
        u.append(uu)
    return mask, rho, u


CONFIGS = {
    "c1": c1_taylor_green,
    "c2": c2_channel,
    "c3": c3_mrt_obstacles,
    "c4": c4_duct,
    "c5": c5_shan_chen,
    "ldc": ldc_cavity,
}
