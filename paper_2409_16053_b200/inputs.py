"""Seeded synthetic inputs: mesh descriptions and initial states for the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic (no c2p, reconstruction, Riemann solver, update, ghost fill, dt): it only lays out a
MeshBlock list (paper §2, "MeshBlockPack", "[m][n][k][j][i]") and
evaluates analytic initial conditions at cell centres (uniform Cartesian mesh), converting
(rho, v, P) to the conserved vector of Eq.(4) once.  The recipe for every config is
restated in DESIGN.md ("Input recipe").  Everything is float64; torch is used only as an array
library so that the 512^3 config can be generated directly in device memory.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Callable, List, Sequence, Tuple

import numpy as np
import torch

GAMMA = 5.0 / 3.0          # BASELINE.json: all configs
CFL = 0.3                  # BASELINE.json: all configs
RECON_PLM, RECON_PPM4, RECON_PPMX, RECON_WENOZ = 0, 1, 2, 3
RSOLVER_HLLC = 0


# --------------------------------------------------------------------------------------------
# Mesh: a static list of MeshBlocks (level, lx1, lx2, lx3) on a periodic box
# --------------------------------------------------------------------------------------------
def _morton(l1: int, l2: int, l3: int) -> int:
    key = 0
    for b in range(21):
        key |= ((l1 >> b) & 1) << (3 * b) | ((l2 >> b) & 1) << (3 * b + 1) | ((l3 >> b) & 1) << (3 * b + 2)
    return key


@dataclass
class Mesh:
    """Root grid of nrb[d] blocks of nx[d] cells; blocks = leaves (level, lx1, lx2, lx3)."""
    nrb: Tuple[int, int, int]
    nx: Tuple[int, int, int]
    ng: int
    blocks: List[Tuple[int, int, int, int]]
    xmin: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    xmax: Tuple[float, float, float] = (1.0, 1.0, 1.0)
    # boundary condition per face (x1min, x1max, x2min, x2max, x3min, x3max): 0 periodic, 1 outflow, 2 reflect
    bc: Tuple[int, int, int, int, int, int] = (0, 0, 0, 0, 0, 0)

    @property
    def nmb(self) -> int:
        return len(self.blocks)

    @property
    def nt(self) -> Tuple[int, int, int]:
        return tuple(n + 2 * self.ng for n in self.nx)

    @property
    def ncells_active(self) -> int:
        return self.nmb * self.nx[0] * self.nx[1] * self.nx[2]

    def state_shape(self) -> Tuple[int, int, int, int, int]:
        n1, n2, n3 = self.nt
        return (self.nmb, 5, n3, n2, n1)

    def dx(self, level: int) -> Tuple[float, float, float]:
        return tuple((self.xmax[d] - self.xmin[d]) / (self.nrb[d] * self.nx[d] * (1 << level)) for d in range(3))

    def centres(self, m: int, device="cpu"):
        """Active-cell centre coordinates (x1[nx1], x2[nx2], x3[nx3]) of block m."""
        level, *lx = self.blocks[m]
        dx = self.dx(level)
        out = []
        for d in range(3):
            g = torch.arange(self.nx[d], dtype=torch.float64, device=device) + float(lx[d] * self.nx[d])
            out.append(self.xmin[d] + (g + 0.5) * dx[d])
        return tuple(out)

    def cell_volume(self, m: int) -> float:
        d = self.dx(self.blocks[m][0])
        return d[0] * d[1] * d[2]


def uniform_mesh(nrb: Sequence[int], nx: Sequence[int], ng: int) -> Mesh:
    """Single-level mesh, blocks in Morton (Z) order of their logical location."""
    locs = [(l1, l2, l3) for l3 in range(nrb[2]) for l2 in range(nrb[1]) for l1 in range(nrb[0])]
    locs.sort(key=lambda l: _morton(*l))
    return Mesh(tuple(nrb), tuple(nx), ng, [(0, *l) for l in locs])


def smr_mesh(nrb: Sequence[int], nx: Sequence[int], ng: int, lo: Sequence[int], hi: Sequence[int]) -> Mesh:
    """Two-level static refinement: root blocks with lo[d] <= l_d < hi[d] are replaced by their 8 children."""
    blocks = []
    for l3 in range(nrb[2]):
        for l2 in range(nrb[1]):
            for l1 in range(nrb[0]):
                l = (l1, l2, l3)
                if all(lo[d] <= l[d] < hi[d] for d in range(3)):
                    for c in range(8):
                        blocks.append((1, 2 * l1 + (c & 1), 2 * l2 + ((c >> 1) & 1), 2 * l3 + ((c >> 2) & 1)))
                else:
                    blocks.append((0, l1, l2, l3))
    # Z-order across levels: sort by the Morton key of the location expressed at the finest level
    blocks.sort(key=lambda b: (_morton(*(x << (1 - b[0]) for x in b[1:])), b[0]))
    return Mesh(tuple(nrb), tuple(nx), ng, blocks)


# --------------------------------------------------------------------------------------------
# State assembly
# --------------------------------------------------------------------------------------------
PrimFn = Callable[[torch.Tensor, torch.Tensor, torch.Tensor], Tuple[torch.Tensor, ...]]


def make_state(mesh: Mesh, prim_fn: PrimFn, gamma: float = GAMMA, device="cpu") -> torch.Tensor:
    """U[m][n][k][j][i] (ghosts included, zero) from prim_fn(x1,x2,x3)->(rho,v1,v2,v3,P) at cell centres.

    Conserved vector of Eq.(4): (rho, rho v, E) with E = P/(gamma-1) + rho v^2/2.
    """
    U = torch.zeros(mesh.state_shape(), dtype=torch.float64, device=device)
    ng = mesh.ng
    n1, n2, n3 = mesh.nx
    for m in range(mesh.nmb):
        x1, x2, x3 = mesh.centres(m, device)
        X3, X2, X1 = x3[:, None, None], x2[None, :, None], x1[None, None, :]
        rho, v1, v2, v3, P = (torch.broadcast_to(torch.as_tensor(q, dtype=torch.float64, device=device), (n3, n2, n1))
                              for q in prim_fn(X1, X2, X3))
        act = U[m, :, ng:ng + n3, ng:ng + n2, ng:ng + n1]
        act[0] = rho
        act[1] = rho * v1
        act[2] = rho * v2
        act[3] = rho * v3
        act[4] = P / (gamma - 1.0) + 0.5 * rho * (v1 * v1 + v2 * v2 + v3 * v3)
    return U


# --------------------------------------------------------------------------------------------
# Random Fourier-mode fields (configs 1, 3 and the SMR parity input)
# --------------------------------------------------------------------------------------------
@dataclass
class ModeField:
    """sum_m a * sin(2 pi k_m . x + phi_m): 16 integer wave-vectors with 0 < |k|_2 <= 4, no replacement."""
    k: np.ndarray        # (nmode, 3) int
    phi: np.ndarray      # (nmode,)
    scale: float = 1.0

    def __call__(self, X1, X2, X3):
        out = None
        for (k1, k2, k3), ph in zip(self.k.tolist(), self.phi.tolist()):
            term = torch.sin(2.0 * math.pi * (k1 * X1 + k2 * X2 + k3 * X3) + ph)
            out = term if out is None else out + term
        return self.scale * out


def _draw_modes(rng: np.random.Generator, nmode: int = 16, kmax: int = 4) -> ModeField:
    cand = [(a, b, c) for a in range(-kmax, kmax + 1) for b in range(-kmax, kmax + 1) for c in range(-kmax, kmax + 1)
            if 0 < a * a + b * b + c * c <= kmax * kmax]
    idx = rng.choice(len(cand), size=nmode, replace=False)
    k = np.array([cand[i] for i in idx], dtype=np.int64)
    phi = rng.uniform(0.0, 2.0 * math.pi, size=nmode)
    return ModeField(k, phi)


@dataclass
class RandomModes:
    """Three velocity-component fields (rng 16053) and one density field (rng 16054), SURVEY Q19."""
    v: List[ModeField]
    g: ModeField

    @staticmethod
    def draw(mach: float, gamma: float = GAMMA, ncal: int = 64, rho_amp: float = 0.05) -> "RandomModes":
        rv = np.random.default_rng(16053)
        v = [_draw_modes(rv) for _ in range(3)]
        g = _draw_modes(np.random.default_rng(16054))
        # calibration on a fixed ncal^3 cell-centred lattice of the unit box (all |k| <= 4 are resolved)
        x = (torch.arange(ncal, dtype=torch.float64) + 0.5) / ncal
        X3, X2, X1 = x[:, None, None], x[None, :, None], x[None, None, :]
        v2 = sum((f(X1, X2, X3) ** 2).mean().item() for f in v)
        cs0 = math.sqrt(gamma * 1.0 / 1.0)
        for f in v:
            f.scale = mach * cs0 / math.sqrt(v2)
        g.scale = rho_amp / g(X1, X2, X3).abs().max().item()
        return RandomModes(v, g)


# --------------------------------------------------------------------------------------------
# Workloads
# --------------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    mesh: Mesh
    recon: int
    nsteps: int
    prim_fn: PrimFn
    gamma: float = GAMMA
    cfl: float = CFL
    rsolver: int = RSOLVER_HLLC
    note: str = ""

    def state(self, device="cpu") -> torch.Tensor:
        return make_state(self.mesh, self.prim_fn, self.gamma, device)


def sound_wave_prim(amp: float = 1e-6, direction: int = 0, gamma: float = GAMMA, literal: bool = False) -> PrimFn:
    """Right-going sound-wave eigenmode: rho0=1, P0=1/gamma, c_s=1."""
    def fn(X1, X2, X3):
        x = (X1, X2, X3)[direction]
        s = torch.sin(2.0 * math.pi * x)
        rho = 1.0 + amp * s
        vel = [torch.zeros_like(s)] * 3
        vel[direction] = amp * s
        P = 1.0 / gamma + (0.0 if literal else amp) * s
        return (rho, vel[0], vel[1], vel[2], P)
    return fn


def sedov_prim(centre=(0.5, 0.5, 0.5), r0=0.05, p_in=100.0, p_out=1e-2) -> PrimFn:
    def fn(X1, X2, X3):
        r2 = (X1 - centre[0]) ** 2 + (X2 - centre[1]) ** 2 + (X3 - centre[2]) ** 2
        P = torch.where(r2 < r0 * r0, torch.full_like(r2, p_in), torch.full_like(r2, p_out))
        z = torch.zeros_like(r2)
        return (torch.ones_like(r2), z, z, z, P)
    return fn


SHU_OSHER_GAMMA = 1.4


def shu_osher_prim(direction: int = 0, mach: float = 3.0, gamma: float = SHU_OSHER_GAMMA) -> PrimFn:
    """Shock - entropy-wave interaction tube of the paper's Fig. 1 right (200 cells, density at t = 0.047).
    A Mach-3 shock at x = -0.08 on [-0.1, 0.1] runs into gas at rest with density 1 + 0.2 sin(50 pi x), P = 1
    (Q32: the classic tube on [-1, 1] to t = 0.47 scaled by 1/10, which is what t = 0.047 implies; the
    Euler equations are invariant under that scaling).  The post-shock state is evaluated from the Rankine-Hugoniot
    relations for `mach` here, not typed in."""
    c1 = math.sqrt(gamma * 1.0 / 1.0)
    r2 = (gamma + 1.0) * mach * mach / ((gamma - 1.0) * mach * mach + 2.0)
    p2 = 1.0 + 2.0 * gamma / (gamma + 1.0) * (mach * mach - 1.0)
    u2 = mach * c1 * (1.0 - 1.0 / r2)

    def fn(X1, X2, X3):
        x = (X1, X2, X3)[direction]
        left = x < -0.08
        rho = torch.where(left, torch.full_like(x, r2), 1.0 + 0.2 * torch.sin(50.0 * math.pi * x))
        vel = [torch.zeros_like(x)] * 3
        vel[direction] = torch.where(left, torch.full_like(x, u2), torch.zeros_like(x))
        P = torch.where(left, torch.full_like(x, p2), torch.ones_like(x))
        return (rho, vel[0], vel[1], vel[2], P)
    return fn


def shu_osher_mesh(N: int, ng: int, nblocks: int = 1) -> Mesh:
    """N x 4 x 4 cells on [-0.1, 0.1] x [0, 1]^2 in `nblocks` blocks along x1, outflow ends."""
    m = uniform_mesh((nblocks, 1, 1), (N // nblocks, 4, 4), ng)
    m.xmin, m.xmax, m.bc = (-0.1, 0.0, 0.0), (0.1, 1.0, 1.0), (1, 1, 0, 0, 0, 0)
    return m


def modes_prim(mach: float, shear: bool, rho_pert: bool) -> PrimFn:
    rm = RandomModes.draw(mach)

    def fn(X1, X2, X3):
        v1, v2, v3 = (f(X1, X2, X3) for f in rm.v)
        if shear:  # double shear layer in x2 (BASELINE.json config 3): +-0.5 across |y|<0.25, tanh width 0.01
            y = X2 - 0.5
            v1 = v1 + 0.5 * (torch.tanh((y + 0.25) / 0.01) - torch.tanh((y - 0.25) / 0.01) - 1.0)
        rho = 1.0 + rm.g(X1, X2, X3) if rho_pert else torch.ones_like(v1)
        return (rho, v1, v2, v3, torch.ones_like(v1))
    return fn


def config0(literal: bool = False) -> Workload:
    return Workload("cfg0_soundwave_1x32", uniform_mesh((1, 1, 1), (32, 32, 32), 2), RECON_PLM, 10,
                    sound_wave_prim(literal=literal))


def config1(nrb: int = 4, nx: int = 32) -> Workload:
    return Workload(f"cfg1_modes_{nrb**3}x{nx}", uniform_mesh((nrb,) * 3, (nx,) * 3, 2), RECON_PLM, 20,
                    modes_prim(0.3, shear=False, rho_pert=True))


def config2(nx: int = 32, n: int = 256) -> Workload:
    nrb = n // nx
    return Workload(f"cfg2_sedov_{nrb**3}x{nx}", uniform_mesh((nrb,) * 3, (nx,) * 3, 2), RECON_PLM, 20, sedov_prim())


def config3(nrb: int = 4, nx: int = 128) -> Workload:
    return Workload(f"cfg3_shear_modes_{nrb**3}x{nx}_ppm", uniform_mesh((nrb,) * 3, (nx,) * 3, 3), RECON_PPM4, 10,
                    modes_prim(1.0, shear=True, rho_pert=False))


def _smr(nx: int = 32) -> Mesh:
    return smr_mesh((4, 4, 4), (nx,) * 3, 2, (1, 1, 1), (3, 3, 3))


def config4(nx: int = 32) -> Workload:
    return Workload(f"cfg4_smr_sedov_120x{nx}", _smr(nx), RECON_PLM, 20,
                    sedov_prim(centre=(0.55, 0.5, 0.5), r0=0.03))


def smr_parity(nx: int = 32) -> Workload:
    """SURVEY finding 3: config-1 field on the config-4 mesh so that level boundaries carry structure."""
    return Workload(f"smr_modes_120x{nx}", _smr(nx), RECON_PLM, 4, modes_prim(0.3, shear=False, rho_pert=True))


def table1() -> Workload:
    """Shape of the paper's Table 1 GPU workload: 512x256x256 in 128^3 blocks, linear wave."""
    return Workload("table1_soundwave_16x128", uniform_mesh((4, 2, 2), (128, 128, 128), 2), RECON_PLM, 10,
                    sound_wave_prim())


# --------------------------------------------------------------------------------------------
# MHD states: 8 variables per cell, the last three the face-centred field
# --------------------------------------------------------------------------------------------
def make_state_mhd(mesh: Mesh, prim_fn: PrimFn, A_fn, B0=(0.0, 0.0, 0.0), gamma: float = GAMMA, device="cpu") -> torch.Tensor:
    """U[m][8][k][j][i] = (rho, rho v, E, b1, b2, b3) with b_d the area-averaged field on the LOWER d-face of each cell
    ("area-averages on cell-faces").  The faces come from a vector potential evaluated on the cell EDGES,
    b = curl A by Stokes' theorem, plus a uniform field B0, so that the discrete divergence vanishes to round-off;
    A_fn(x1, x2, x3) -> (A1, A2, A3) at arbitrary points.  E = P/(gamma-1) + rho v^2/2 + B^2/2 with the
    cell-centred B the mean of the two faces.  Faces are set on the active cells and on the first ghost layer above them
    (the upper face of the last active cell); ghost cells otherwise stay zero (the ghost fill writes them)."""
    n1, n2, n3 = mesh.nx
    ng = mesh.ng
    U = torch.zeros((mesh.nmb, 8) + tuple(mesh.state_shape()[2:]), dtype=torch.float64, device=device)
    for m in range(mesh.nmb):
        level, *lx = mesh.blocks[m]
        dx = mesh.dx(level)
        xc = mesh.centres(m, device)                                   # cell centres of the active cells
        # face / edge coordinates: nx+1 lower-face positions per direction
        xf = [mesh.xmin[d] + (torch.arange(mesh.nx[d] + 1, dtype=torch.float64, device=device) + float(lx[d] * mesh.nx[d])) * dx[d]
              for d in range(3)]

        def grid(a1, a2, a3):
            return a1[None, None, :], a2[None, :, None], a3[:, None, None]

        def A(comp, a1, a2, a3):
            X1, X2, X3 = grid(a1, a2, a3)
            return torch.broadcast_to(torch.as_tensor(A_fn(X1, X2, X3)[comp], dtype=torch.float64, device=device),
                                      (a3.numel(), a2.numel(), a1.numel()))
        # b1 on x1-faces (x1f, x2c, x3c): dA3/dx2 - dA2/dx3, differences of edge values over the face
        A3 = A(2, xf[0], xf[1], xc[2]); A2 = A(1, xf[0], xc[1], xf[2])
        b1 = (A3[:, 1:, :] - A3[:, :-1, :]) / dx[1] - (A2[1:, :, :] - A2[:-1, :, :]) / dx[2] + B0[0]
        # b2 on x2-faces (x1c, x2f, x3c): dA1/dx3 - dA3/dx1
        A1 = A(0, xc[0], xf[1], xf[2]); A3 = A(2, xf[0], xf[1], xc[2])
        b2 = (A1[1:, :, :] - A1[:-1, :, :]) / dx[2] - (A3[:, :, 1:] - A3[:, :, :-1]) / dx[0] + B0[1]
        # b3 on x3-faces (x1c, x2c, x3f): dA2/dx1 - dA1/dx2
        A2 = A(1, xf[0], xc[1], xf[2]); A1 = A(0, xc[0], xf[1], xf[2])
        b3 = (A2[:, :, 1:] - A2[:, :, :-1]) / dx[0] - (A1[:, 1:, :] - A1[:, :-1, :]) / dx[1] + B0[2]
        U[m, 5, ng:ng + n3, ng:ng + n2, ng:ng + n1 + 1] = b1
        U[m, 6, ng:ng + n3, ng:ng + n2 + 1, ng:ng + n1] = b2
        U[m, 7, ng:ng + n3 + 1, ng:ng + n2, ng:ng + n1] = b3
        X1, X2, X3 = grid(*xc)
        rho, v1, v2, v3, P = (torch.broadcast_to(torch.as_tensor(q, dtype=torch.float64, device=device), (n3, n2, n1))
                              for q in prim_fn(X1, X2, X3))
        bc1 = 0.5 * (b1[:, :, 1:] + b1[:, :, :-1]); bc2 = 0.5 * (b2[:, 1:, :] + b2[:, :-1, :]); bc3 = 0.5 * (b3[1:, :, :] + b3[:-1, :, :])
        act = U[m, :, ng:ng + n3, ng:ng + n2, ng:ng + n1]
        act[0] = rho; act[1] = rho * v1; act[2] = rho * v2; act[3] = rho * v3
        act[4] = P / (gamma - 1.0) + 0.5 * rho * (v1 * v1 + v2 * v2 + v3 * v3) + 0.5 * (bc1 * bc1 + bc2 * bc2 + bc3 * bc3)
    return U


def mhd_workload(name: str, ng: int = 3):
    """MHD workloads of bench.py and the full-size GPU test: the seeded Mach-0.5 random-mode velocity field and
    5 % density modes of the hydro configs, P = 1, a tangled field from a vector potential plus a mean field, on a uniform periodic
    pack of 8 MeshBlocks, ng = 3 (4 for PPM4 / PPMX / WENOZ).  -> (mesh, prim_fn, A_fn, B0) for make_state_mhd."""
    nrb, nx = {"mhd_256": (2, 128), "mhd_128": (2, 64), "mhd_64": (2, 32)}[name]
    mesh = uniform_mesh((nrb,) * 3, (nx,) * 3, ng)
    rm = RandomModes.draw(0.5)
    k = 2 * math.pi

    def prim(X1, X2, X3):
        v1, v2, v3 = (f(X1, X2, X3) for f in rm.v)
        return (1.0 + rm.g(X1, X2, X3), v1, v2, v3, torch.ones_like(v1))

    def A(X1, X2, X3):
        return (0.05 * torch.sin(k * X2) * torch.cos(2 * k * X3) + 0 * X1, 0.05 * torch.sin(k * X3 + 0.3) * torch.cos(k * X1) + 0 * X2,
                0.05 * torch.cos(2 * k * X1 + 0.7) * torch.sin(k * X2) + 0 * X3)
    return mesh, prim, A, (0.4, 0.3, 0.2)
