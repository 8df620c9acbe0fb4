"""Pins for the MHD + constrained-transport oracle (oracle/orc_mhd.cpp; paper P:116).

Nothing here compares the oracle with itself:
  * HLLD: consistency with the physical flux of Eq.(5), mirror symmetry, a stationary contact across which the density jumps
    while the field threads it, supersonic upwinding;
  * the hydrodynamic limit: with B = 0 the Sod tube converges to the exact Riemann solution (solver in test_oracle_scheme);
  * div B = 0 to round-off, conservation of mass, momentum, energy and of the mean field, on a 3-D multi-block periodic mesh
    with a field from a vector potential;
  * a uniform magnetised state in motion is preserved bit for bit;
  * a plane-parallel problem (Brio-Wu states) stays plane-parallel bit for bit, and run along x2 or x3 it matches x1;
  * "For PPM4 and PLM reconstruction, all waves converge at second-order" -- fast, Alfven and slow waves whose
    eigenvectors are computed here numerically from the primitive-variable Jacobian of Eq.(5).
"""
import math

import numpy as np
import pytest
import torch

from paper_2409_16053_b200 import inputs as I

G53 = 5.0 / 3.0


@pytest.fixture(scope="module")
def om():
    from oracle import orc_mhd
    orc_mhd.build()
    return orc_mhd


def phys_flux(g, bx, W):
    r, u, v, w, e, by, bz = W
    p = (g - 1) * e
    b2 = bx * bx + by * by + bz * bz
    pt = p + 0.5 * b2
    E = e + 0.5 * r * (u * u + v * v + w * w) + 0.5 * b2
    vb = u * bx + v * by + w * bz
    return np.array([r * u, r * u * u + pt - bx * bx, r * u * v - bx * by, r * u * w - bx * bz, (E + pt) * u - bx * vb,
                     by * u - bx * v, bz * u - bx * w])


def rand_state(rng):
    return [10 ** rng.uniform(-1, 1), *rng.normal(size=3), 10 ** rng.uniform(-1, 1), *rng.normal(size=2)]


# ---------------------------------------------------------------- HLLD -----------------------------
def test_hlld_consistency(om):
    rng = np.random.default_rng(1)
    for _ in range(300):
        W, bx = rand_state(rng), rng.normal() * rng.integers(0, 2)        # (half of the cases with Bx = 0)
        F, Fx = om.hlld(G53, bx, W, W), phys_flux(G53, bx, W)
        assert np.abs(F - Fx).max() <= 1e-13 * (np.abs(Fx).max() + 1.0)


def test_hlld_mirror_symmetry(om):
    # x -> -x together with B -> -B (an invariance of Eq.(5)): L <-> R, u -> -u, Bx -> -Bx, transverse components unchanged;
    # then every flux component but the normal momentum changes sign
    rng = np.random.default_rng(2)
    sign = np.array([-1.0, 1.0, -1.0, -1.0, -1.0, -1.0, -1.0])
    for _ in range(300):
        WL, WR, bx = rand_state(rng), rand_state(rng), rng.normal()
        F = om.hlld(G53, bx, WL, WR)
        ML, MR = list(WR), list(WL)
        ML[1], MR[1] = -ML[1], -MR[1]
        Fm = om.hlld(G53, -bx, ML, MR)
        assert np.abs(Fm - sign * F).max() <= 1e-12 * (np.abs(F).max() + 1.0)


def test_hlld_keeps_a_stationary_contact_and_upwinds_supersonic_flow(om):
    # density jumps, everything else continuous, gas at rest, field threading the contact: only the stresses remain
    bx, by, bz, ug = 0.8, -0.6, 0.3, 1.5
    WL, WR = [1.0, 0, 0, 0, ug, by, bz], [0.1, 0, 0, 0, ug, by, bz]
    F = om.hlld(G53, bx, WL, WR)
    pt = (G53 - 1) * ug + 0.5 * (bx * bx + by * by + bz * bz)
    np.testing.assert_allclose(F, [0.0, pt - bx * bx, -bx * by, -bx * bz, 0.0, 0.0, 0.0], atol=1e-15)
    assert F[0] == 0.0
    # faster than the fast speed to the right / left: the upwind physical flux
    rng = np.random.default_rng(3)
    WL, WR = rand_state(rng), rand_state(rng)
    WL[1], WR[1] = 30.0, 31.0
    np.testing.assert_allclose(om.hlld(G53, 0.7, WL, WR), phys_flux(G53, 0.7, WL), rtol=1e-14)
    WL[1], WR[1] = -31.0, -30.0
    np.testing.assert_allclose(om.hlld(G53, 0.7, WL, WR), phys_flux(G53, 0.7, WR), rtol=1e-14)


def fast_speed(g, bx, W):
    r, u, v, w, e, by, bz = W
    gp, b2 = g * (g - 1) * e, bx * bx + by * by + bz * bz
    return math.sqrt(0.5 * ((gp + b2) + math.sqrt((gp + b2) ** 2 - 4 * gp * bx * bx)) / r)


@pytest.mark.parametrize("solver", ["llf", "hlle"])
def test_llf_and_hlle_for_mhd(om, solver):
    """P:103 names LLF and the HLL family; in MHD variables: consistency with Eq.(5), the mirror symmetry of Eq.(5), closed forms
    of the dissipation on a stationary contact (LLF: -(lambda/2) dU with lambda = max(|u| + cf); HLLE between +-max cf: the same
    value), HLLE upwinds supersonic flow exactly; in the scheme both carry linear waves at second order with more dissipation than
    HLLD (error at N = 32 between 1 and 3 times HLLD's)."""
    rng = np.random.default_rng(11)
    sign = np.array([-1.0, 1.0, -1.0, -1.0, -1.0, -1.0, -1.0])
    for _ in range(200):
        W, bx = rand_state(rng), rng.normal() * rng.integers(0, 2)
        F, Fx = om.hlld(G53, bx, W, W, solver), phys_flux(G53, bx, W)
        assert np.abs(F - Fx).max() <= 1e-13 * (np.abs(Fx).max() + 1.0)
        WL, WR = rand_state(rng), rand_state(rng)
        F = om.hlld(G53, bx, WL, WR, solver)
        ML, MR = list(WR), list(WL)
        ML[1], MR[1] = -ML[1], -MR[1]
        assert np.abs(om.hlld(G53, -bx, ML, MR, solver) - sign * F).max() <= 1e-12 * (np.abs(F).max() + 1.0)
    bx, by, bz, ug = 0.8, -0.6, 0.3, 1.5
    WL, WR = [1.0, 0, 0, 0, ug, by, bz], [0.1, 0, 0, 0, ug, by, bz]
    lam = max(fast_speed(G53, bx, WL), fast_speed(G53, bx, WR))
    pt = (G53 - 1) * ug + 0.5 * (bx * bx + by * by + bz * bz)
    F = om.hlld(G53, bx, WL, WR, solver)                     # U_R - U_L = (-0.9, 0, 0, 0, 0, 0, 0): only the mass flux is smeared
    np.testing.assert_allclose(F, [0.5 * lam * 0.9, pt - bx * bx, -bx * by, -bx * bz, 0.0, 0.0, 0.0], rtol=1e-14, atol=1e-15)
    if solver == "hlle":
        WL, WR = rand_state(rng), rand_state(rng)
        WL[1], WR[1] = 30.0, 31.0
        np.testing.assert_allclose(om.hlld(G53, 0.7, WL, WR, solver), phys_flux(G53, 0.7, WL), rtol=1e-14)
        WL[1], WR[1] = -31.0, -30.0
        np.testing.assert_allclose(om.hlld(G53, 0.7, WL, WR, solver), phys_flux(G53, 0.7, WR), rtol=1e-14)
    # in the scheme: second-order convergence of a fast and a slow linear wave, with more dissipation than HLLD
    rs = {"llf": 1, "hlle": 2}[solver]
    for family in ("fast", "slow"):
        e16, e32 = (wave_error(om, family, N, rsolver=rs) for N in (16, 32))
        d32 = wave_error(om, family, 32)
        assert 1.2 <= math.log2(e16 / e32) <= 2.4 and d32 <= e32 * (1 + 1e-9) and e32 < 3.0 * d32, (family, e16, e32, d32)


# ---------------------------------------------------------------- helpers --------------------------
ZERO_A = lambda X1, X2, X3: (0 * X1 + 0 * X2 + 0 * X3,) * 3


def act(mesh):
    g = mesh.ng
    return (slice(None), slice(None), slice(g, -g), slice(g, -g), slice(g, -g))


def divb(mesh, U):
    g, (n1, n2, n3) = mesh.ng, mesh.nx
    dx = mesh.dx(0)
    b1, b2, b3 = U[:, 5], U[:, 6], U[:, 7]
    s = (slice(None), slice(g, g + n3), slice(g, g + n2), slice(g, g + n1))
    up1 = (slice(None), slice(g, g + n3), slice(g, g + n2), slice(g + 1, g + n1 + 1))
    up2 = (slice(None), slice(g, g + n3), slice(g + 1, g + n2 + 1), slice(g, g + n1))
    up3 = (slice(None), slice(g + 1, g + n3 + 1), slice(g, g + n2), slice(g, g + n1))
    return (b1[up1] - b1[s]) / dx[0] + (b2[up2] - b2[s]) / dx[1] + (b3[up3] - b3[s]) / dx[2]


def run(om, mesh, U0, gamma=G53, cfl=0.3, nsteps=None, tend=None, threads=4, recon=0, nstages=2, rsolver=0):
    p = om.OrcMhdPack(mesh, gamma, threads=threads, recon=recon, nstages=nstages, rsolver=rsolver)
    p.load(U0)
    t, n = 0.0, 0
    while (nsteps is None or n < nsteps) and (tend is None or t < tend):
        dt = p.new_dt(cfl)
        if tend is not None and t + dt > tend:
            dt = tend - t
        p.step(cfl, dt)
        t += dt
        n += 1
    assert p.floor_count() == 0
    p.fill_ghosts()
    out = p.current().copy()
    p.close()
    return out


def tri(x):
    """Periodic triangle wave with slope +1 on [0.25, 0.75) and -1 elsewhere: the integral of the double Brio-Wu field."""
    x = x - torch.floor(x)
    return torch.where((x >= 0.25) & (x < 0.75), x - 0.5, torch.where(x < 0.25, -x, 1.0 - x))


def brio_wu(N, d, ng=3):
    """Two mirrored Brio-Wu problems on a periodic line along direction d (left state on [0.25, 0.75)), gamma = 2."""
    nx = [4, 4, 4]
    nx[d] = N
    mesh = I.uniform_mesh((1, 1, 1), tuple(nx), ng)
    d2 = (d + 2) % 3

    def prim(X1, X2, X3):
        x = (X1, X2, X3)[d] + 0 * X1 + 0 * X2 + 0 * X3
        inside = (x >= 0.25) & (x < 0.75)
        z = torch.zeros_like(x)
        return (torch.where(inside, 1.0, 0.125).to(torch.float64), z, z, z, torch.where(inside, 1.0, 0.1).to(torch.float64))

    def A(X1, X2, X3):
        x = (X1, X2, X3)[d] + 0 * X1 + 0 * X2 + 0 * X3
        out = [torch.zeros_like(x)] * 3
        out[d2] = -tri(x)                                   # B_{d+1} = -dA_{d+2}/dx_d = +1 inside, -1 outside
        return tuple(out)

    B0 = [0.0, 0.0, 0.0]
    B0[d] = 0.75
    return mesh, I.make_state_mhd(mesh, prim, A, tuple(B0), gamma=2.0).numpy()


# ---------------------------------------------------------------- scheme ---------------------------
def test_hydrodynamic_limit_sod_against_the_exact_solution(om):
    from tests.test_oracle_scheme import exact_riemann, sod_sample
    g = 1.4
    ps, us = exact_riemann(g, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    errs = {}
    for N in (128, 256):
        mesh = I.uniform_mesh((1, 1, 1), (N, 4, 4), 3)

        def prim(X1, X2, X3):
            x = X1 + 0 * X2 + 0 * X3
            inside = (x >= 0.25) & (x < 0.75)
            z = torch.zeros_like(x)
            return (torch.where(inside, 1.0, 0.125).to(torch.float64), z, z, z, torch.where(inside, 1.0, 0.1).to(torch.float64))

        U0 = I.make_state_mhd(mesh, prim, ZERO_A, gamma=g).numpy()
        U = run(om, mesh, U0, gamma=g, tend=0.1)
        prof = U[0, :, 3, 3, 3:-3]
        x = (np.arange(N) + 0.5) / N
        right = x >= 0.5
        rho_ex, _ = sod_sample(g, (x[right] - 0.75) / 0.1, ps, us)
        errs[N] = np.abs(prof[0, right] - rho_ex).mean()
        assert np.all(U[:, 5:] == 0.0)                                     # no field is generated
        assert np.abs(prof[0] - prof[0, ::-1]).max() <= 1e-13              # the two halves mirror each other
    assert errs[256] < 5e-3 and 0.7 <= math.log2(errs[128] / errs[256]) <= 1.15, errs


def test_divb_conservation_and_mean_field_on_a_multiblock_mesh(om):
    mesh = I.uniform_mesh((2, 2, 1), (8, 6, 10), 3)
    k = 2 * math.pi

    def A(X1, X2, X3):
        return (0.1 * torch.sin(k * X2) * torch.cos(k * X3) + 0 * X1, 0.1 * torch.sin(k * X3 + 0.3) * torch.cos(k * X1) + 0 * X2,
                0.1 * torch.cos(k * X1 + 0.7) * torch.sin(k * X2) + 0 * X3)

    prim = lambda X1, X2, X3: (1.0 + 0.2 * torch.sin(k * X1) * torch.cos(k * X2) + 0 * X3, 0.3 * torch.sin(k * X2) + 0 * X1 + 0 * X3,
                               -0.2 * torch.cos(k * X3) + 0 * X1 + 0 * X2, 0.1 * torch.sin(k * X1 + 1.0) + 0 * X2 + 0 * X3,
                               0.6 + 0 * X1 + 0 * X2 + 0 * X3)
    U0 = I.make_state_mhd(mesh, prim, A, (0.3, -0.2, 0.1)).numpy()
    assert np.abs(divb(mesh, U0)).max() <= 1e-13
    U = run(om, mesh, U0, nsteps=6)
    assert np.abs(divb(mesh, U)).max() <= 2e-13                            # (|B|/dx ~ 10: a few ulp of that)
    a = act(mesh)
    for n in range(8):                                                    # mass, momentum, energy and the mean field
        t0, t1 = U0[a][:, n].sum(), U[a][:, n].sum()
        scale = np.abs(U0[a][:, n]).sum() + 1.0
        assert abs(t1 - t0) <= 1e-13 * scale, (n, t0, t1)
    assert np.abs(U[a] - U0[a]).max() > 1e-3                               # (something happened)


def test_corner_emfs_are_continuous_where_a_mass_flux_changes_sign(om):
    """Q36 (ramped upwind switch): a 3-D field whose x1 velocity vanishes on a plane.  Shifting that velocity by +-1e-14 -- the
    size of a rounding difference between two arithmetics -- must move the result of a step by a comparable amount; with a
    sharp switch on the sign of the mass flux the two runs pick opposite sides there and differ by ~1e-4."""
    mesh = I.uniform_mesh((1, 1, 1), (8, 6, 12), 3)
    k = 2 * math.pi

    def A(X1, X2, X3):
        return (0.1 * torch.sin(k * X2) * torch.cos(2 * k * X3) + 0 * X1, 0.1 * torch.sin(k * X3 + 0.3) * torch.cos(k * X1) + 0 * X2,
                0.1 * torch.cos(2 * k * X1 + 0.7) * torch.sin(k * X2) + 0 * X3)

    outs = []
    for eps in (1e-14, -1e-14, 1e-3):
        prim = lambda X1, X2, X3: (1.0 + 0.3 * torch.sin(k * X1) * torch.cos(k * X2) + 0 * X3,
                                   eps + 0 * X1 + 0 * X2 + 0 * X3,              # x1 mass fluxes at round-off level everywhere
                                   -0.5 * torch.cos(k * X3) * torch.sin(2 * k * X1) + 0 * X2,
                                   0.5 * torch.sin(k * X1 + 1.0) * torch.sin(k * X2) + 0 * X3, 0.6 + 0 * X1 + 0 * X2 + 0 * X3)
        U0 = I.make_state_mhd(mesh, prim, A, (0.4, -0.3, 0.2)).numpy()
        p = om.OrcMhdPack(mesh, G53)
        p.load(U0)
        p.step(0.3, 2e-3)
        outs.append(p.current()[act(mesh)].copy())
        p.close()
    assert np.abs(outs[0] - outs[1]).max() <= 1e-12                         # (measured 2.5e-14; a sharp switch gives ~1e-4)
    assert np.abs(outs[0] - outs[2]).max() > 1e-6                           # (the velocity does matter once it is not round-off)


def assemble(mesh, U):
    """Active cells of every block -> one global (8, N3, N2, N1) array (a face field sits on the lower face of its cell)."""
    g, nx = mesh.ng, mesh.nx
    G = np.empty((8, mesh.nrb[2] * nx[2], mesh.nrb[1] * nx[1], mesh.nrb[0] * nx[0]))
    for m, (_, l1, l2, l3) in enumerate(mesh.blocks):
        G[:, l3 * nx[2]:(l3 + 1) * nx[2], l2 * nx[1]:(l2 + 1) * nx[1], l1 * nx[0]:(l1 + 1) * nx[0]] = U[m][:, g:-g, g:-g, g:-g]
    return G


@pytest.mark.parametrize("recon,ng", [(0, 3), (3, 4)])
def test_block_decomposition_does_not_change_the_result(om, recon, ng):
    """The same periodic problem cut into 1, 4 and 12 MeshBlocks (the pack is an implementation device, not part of the
    scheme): bit-identical global states after three steps -- ghost fill, face ownership at block boundaries and the corner EMFs
    computed independently by neighbouring blocks all have to agree for that."""
    k = 2 * math.pi

    def A(X1, X2, X3):
        return (0.1 * torch.sin(k * X2) * torch.cos(k * X3) + 0 * X1, 0.1 * torch.sin(k * X3 + 0.3) * torch.cos(k * X1) + 0 * X2,
                0.1 * torch.cos(k * X1 + 0.7) * torch.sin(k * X2) + 0 * X3)

    prim = lambda X1, X2, X3: (1.0 + 0.2 * torch.sin(k * X1) * torch.cos(k * X2) + 0 * X3, 0.3 * torch.sin(k * X2 + 0.1) + 0 * X1 + 0 * X3,
                               -0.2 * torch.cos(k * X3) + 0 * X1 + 0 * X2, 0.1 * torch.sin(k * X1 + 1.0) + 0 * X2 + 0 * X3,
                               0.6 + 0 * X1 + 0 * X2 + 0 * X3)
    outs = []
    for nrb, nx in (((1, 1, 1), (16, 12, 8)), ((2, 2, 1), (8, 6, 8)), ((2, 3, 2), (8, 4, 4))):
        mesh = I.uniform_mesh(nrb, nx, ng)
        U0 = I.make_state_mhd(mesh, prim, A, (0.3, -0.2, 0.1)).numpy()
        p = om.OrcMhdPack(mesh, G53, recon=recon)
        p.load(U0)
        for _ in range(3):
            p.step(0.3, 2e-3)
        outs.append(assemble(mesh, p.current()))
        p.close()
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
    assert np.abs(outs[0][0] - 1.0).max() > 0.1                             # (a non-trivial state)


def test_uniform_magnetised_state_is_preserved_bit_exactly(om):
    mesh = I.uniform_mesh((2, 1, 2), (6, 8, 4), 3)
    prim = lambda X1, X2, X3: (1.3 + 0 * X1 + 0 * X2 + 0 * X3, 0.4 + 0 * X1 + 0 * X2 + 0 * X3, -0.7 + 0 * X1 + 0 * X2 + 0 * X3,
                               0.2 + 0 * X1 + 0 * X2 + 0 * X3, 0.9 + 0 * X1 + 0 * X2 + 0 * X3)
    U0 = I.make_state_mhd(mesh, prim, ZERO_A, (0.5, -0.3, 0.8)).numpy()
    U = run(om, mesh, U0, nsteps=2)
    a = act(mesh)
    assert np.array_equal(U[a], U0[a])


def test_plane_parallel_brio_wu_stays_plane_parallel_and_is_direction_independent(om):
    profs = []
    for d in range(3):
        mesh, U0 = brio_wu(64, d)
        U = run(om, mesh, U0, gamma=2.0, tend=0.05)
        A = U[0][:, 3:-3, 3:-3, 3:-3]                                       # (n, k, j, i)
        line = np.moveaxis(A, 3 - d, 1)                                     # (n, along, t, t)
        assert np.array_equal(line, np.broadcast_to(line[:, :, :1, :1], line.shape))       # transverse planes identical
        prof = line[:, :, 0, 0]
        d1, d2 = (d + 1) % 3, (d + 2) % 3
        profs.append(prof[[0, 1 + d, 1 + d1, 1 + d2, 4, 5 + d, 5 + d1, 5 + d2]])            # rotated into the x1 frame
        assert np.all(prof[5 + d] == 0.75)                                  # the normal field of a 1-D problem never changes
        assert np.abs(prof[0] - prof[0, ::-1]).max() <= 1e-13 and prof[0].min() > 0.1 and prof[0].max() <= 1.0 + 1e-12
    for p in profs[1:]:
        assert np.abs(p - profs[0]).max() <= 1e-13
    # the compound structure has formed: the tangential field has changed sign across the fan and v_x > 0.3 somewhere
    assert (profs[0][1] / profs[0][0]).max() > 0.3 and profs[0][6].min() < -0.9 and profs[0][6].max() > 0.9


# ---------------------------------------------------------------- linear waves -------------
def mhd_eigenmode(family):
    """Right-going eigenvector of the primitive Jacobian d(rho, u, v, w, p, By, Bz)/dt + A d/dx = 0 of Eq.(5) about the
    Gardiner-Stone background (rho = 1, p = 1/gamma, B = (1, sqrt 2, 1/2), at rest): speeds 2, 1, 1/2."""
    g, r, p, bx, by, bz = G53, 1.0, 1.0 / G53, 1.0, math.sqrt(2.0), 0.5
    A = np.zeros((7, 7))
    A[0, 1] = r
    A[1, 4], A[1, 5], A[1, 6] = 1 / r, by / r, bz / r
    A[2, 5] = -bx / r
    A[3, 6] = -bx / r
    A[4, 1] = g * p
    A[5, 1], A[5, 2] = by, -bx
    A[6, 1], A[6, 3] = bz, -bx
    lam, R = np.linalg.eig(A)
    speed = {"fast": 2.0, "alfven": 1.0, "slow": 0.5}[family]
    k = int(np.argmin(np.abs(lam - speed)))
    assert abs(lam[k].real - speed) < 1e-12 and abs(lam[k].imag) < 1e-12
    v = R[:, k].real
    return speed, v / np.abs(v).max(), (r, p, bx, by, bz)


def wave_error(om, family, N, amp=1e-6, recon=0, nstages=2, rsolver=0):
    speed, R, (r0, p0, bx, by0, bz0) = mhd_eigenmode(family)
    mesh = I.uniform_mesh((1, 1, 1), (N, 4, 4), 3 if recon == 0 else 4)
    k = 2 * math.pi

    def prim(X1, X2, X3):
        s = torch.sin(k * X1) + 0 * X2 + 0 * X3
        return (r0 + amp * R[0] * s, amp * R[1] * s, amp * R[2] * s, amp * R[3] * s, p0 + amp * R[4] * s)

    def A(X1, X2, X3):                                   # dBy = -dA3/dx1, dBz = +dA2/dx1
        c = torch.cos(k * X1) / k + 0 * X2 + 0 * X3
        return (0 * c, -amp * R[6] * c, amp * R[5] * c)

    U0 = I.make_state_mhd(mesh, prim, A, (bx, by0, bz0)).numpy()
    U = run(om, mesh, U0, tend=1.0 / speed, recon=recon, nstages=nstages, rsolver=rsolver)
    a = act(mesh)
    return math.sqrt(sum(np.abs(U[a][0, n] - U0[a][0, n]).mean() ** 2 for n in range(8)))


def test_higher_order_options_reproduce_the_papers_convergence_orders(om):
    """"While fourth-order convergence is observed for RK3+PPMX and RK3+WENOZ for slow and Alfven waves, the fast wave only
    converges at second-order even in one-dimension.  For PPM4 and PLM reconstruction, all waves converge at second-order".
    WENOZ / PPMX + SSPRK(3,3): Alfven and slow errors fall by >= 2^3.5 per doubling, the fast wave's by 2^1.7 .. 2^3; PPM4 + RK2:
    second order, below PLM's error at the same resolution.  (Measured rates at N = 16 -> 32 -> 64: WENOZ Alfven 4.8 / 4.4, slow 5.0,
    fast 2.5; PPMX Alfven 3.96 / 3.99, slow 3.96, fast 3.3 then 2.3; PPM4 1.6-2.2.  The test runs the cheapest pairs of these.)"""
    W = lambda family, N: wave_error(om, family, N, recon=3, nstages=3)
    X = lambda family, N: wave_error(om, family, N, recon=2, nstages=3)
    a16, a32 = W("alfven", 16), W("alfven", 32)
    assert math.log2(a16 / a32) >= 3.5, (a16, a32)
    x16, x32 = X("alfven", 16), X("alfven", 32)
    assert math.log2(x16 / x32) >= 3.5, (x16, x32)
    s16, s32, y16, y32 = W("slow", 12), W("slow", 24), X("slow", 12), X("slow", 24)
    assert math.log2(s16 / s32) >= 3.5 and math.log2(y16 / y32) >= 3.5, (s16, s32, y16, y32)
    f16, f32, g32, g64 = W("fast", 16), W("fast", 32), X("fast", 32), X("fast", 64)
    assert 1.7 <= math.log2(f16 / f32) <= 3.0 and 1.7 <= math.log2(g32 / g64) <= 3.0, (f16, f32, g32, g64)
    p16, p32 = (wave_error(om, "alfven", N, recon=1) for N in (16, 32))
    l32 = wave_error(om, "alfven", 32)
    assert 1.4 <= math.log2(p16 / p32) <= 2.6 and p32 < l32 and a32 < 0.1 * p32 and x32 < 0.1 * p32, (p16, p32, l32, a32, x32)


@pytest.mark.parametrize("family", ["fast", "alfven", "slow"])
def test_linear_mhd_waves_converge_at_second_order(om, family):
    e = {N: wave_error(om, family, N) for N in (16, 32, 64)}
    assert e[64] < e[32] < e[16] < 1e-6
    assert 3.0 <= e[32] / e[64] <= 5.0, (family, e)


def oblique_wave_error(om, family, N, amp=1e-6):
    """The same eigenmodes propagating at tan(theta) = 2 to the x1 axis on a 2N x N (x 4) grid of square cells
    (the setup of Gardiner & Stone 2005, restated): wavelength 1/sqrt 5 fits the 1 x 1/2 periodic box once in each direction."""
    speed, R, (r0, p0, bpar, bp10, bp20) = mhd_eigenmode(family)
    ct, st = 1.0 / math.sqrt(5.0), 2.0 / math.sqrt(5.0)
    lam = ct
    mesh = I.uniform_mesh((4, 2, 1), (N // 2, N // 2, 4), 3)       # (8 blocks only spread the oracle over threads)
    mesh.xmax = (1.0, 0.5, 4.0 / (2 * N))                 # cubic cells
    k = 2 * math.pi / lam

    def rot(par, perp1, perp2):                            # (k-hat, e-perp, z) components -> (x1, x2, x3)
        return (par * ct - perp1 * st, par * st + perp1 * ct, perp2)

    def prim(X1, X2, X3):
        s = torch.sin(k * (X1 * ct + X2 * st)) + 0 * X3
        v = rot(amp * R[1] * s, amp * R[2] * s, amp * R[3] * s)
        return (r0 + amp * R[0] * s, v[0], v[1], v[2], p0 + amp * R[4] * s)

    def A(X1, X2, X3):
        c = torch.cos(k * (X1 * ct + X2 * st)) / k + 0 * X3
        # in-plane perturbation dB_perp1 e_perp = curl(A3 z) with A3' = -dB_perp1; dB3 = d(A2)/dx1
        return (0 * c, -amp * R[6] * c / ct, amp * R[5] * c)

    U0 = I.make_state_mhd(mesh, prim, A, rot(bpar, bp10, bp20)).numpy()
    assert np.abs(divb(mesh, U0)).max() <= 1e-12
    U = run(om, mesh, U0, tend=lam / speed, threads=8)
    a = act(mesh)
    return math.sqrt(sum(np.abs(U[a][:, n] - U0[a][:, n]).mean() ** 2 for n in range(8)))


@pytest.mark.parametrize("family", ["fast", "alfven", "slow"])
def test_oblique_linear_waves_converge_at_second_order(om, family):
    """Multi-dimensional CT (Q35, Q36): with the corner EMFs wrong (a dropped or mis-signed upwind term, a wrong face) the wave
    is damped or distorted at first order or grows; with them right the unsplit scheme keeps its second order obliquely."""
    e = {N: oblique_wave_error(om, family, N) for N in (32, 64)}              # 29, 57 cells per wavelength
    assert e[64] < e[32] < 1e-6
    assert 3.0 <= e[32] / e[64] <= 5.0, (family, e)        # (14 -> 29 cells per wavelength is pre-asymptotic, as in 1-D: 2.6)
