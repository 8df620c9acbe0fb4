"""Pins for the oracle's LLF, HLLE and Roe fluxes (paper P:103 lists "LLF ... HLLE, HLLC ...").
Each is checked against what mathematics fixes for ANY consistent two-state solver of its kind, not against a
retyped formula: consistency with the physical flux, exact upwinding where it must upwind, exact resolution of an
isolated shock (HLLE: Roe's property U makes u~ + c~ the exact shock speed), closed forms on a stationary contact,
mirror symmetry bit for bit, direction permutation, and at scheme level convergence of Sod's problem to the exact
Riemann solution, conservation and the bit-exact mirror image of the two half problems."""
import math

import numpy as np
import pytest

from paper_2409_16053_b200 import inputs as I
from tests.test_oracle_units import G53, phys_flux, ulp_diff
from tests.test_oracle_scheme import exact_riemann, sod_run, sod_sample

SOLVERS = ["llf", "hlle", "roe"]


def flux(orc, name, g, d, WL, WR):
    return getattr(orc, name)(g, d, WL, WR)


def rand_state(rng):
    return [10 ** rng.uniform(-1, 1), *rng.normal(size=3), 10 ** rng.uniform(-1, 1)]


@pytest.mark.parametrize("name", SOLVERS)
@pytest.mark.parametrize("d", [0, 1, 2])
def test_consistency(orc, name, d):
    rng = np.random.default_rng(40 + d)
    for _ in range(200):
        W = rand_state(rng)
        F, Fx = flux(orc, name, G53, d, W, W), phys_flux(G53, d, W)
        assert np.abs(F - Fx).max() <= 8 * np.spacing(np.abs(Fx).max())


@pytest.mark.parametrize("name", SOLVERS)
@pytest.mark.parametrize("d", [0, 1, 2])
def test_mirror_symmetry(orc, name, d):
    rng = np.random.default_rng(50 + d)
    for _ in range(300):
        WL, WR = rand_state(rng), rand_state(rng)
        F = flux(orc, name, G53, d, WL, WR)
        ML, MR = list(WR), list(WL)
        ML[1 + d], MR[1 + d] = -ML[1 + d], -MR[1 + d]
        sign = -np.ones(5)
        sign[1 + d] = 1.0
        Fm = flux(orc, name, G53, d, ML, MR)
        if name == "roe":       # a1 and a5 are not evaluated by mirror-image expressions: symmetric to rounding only
            assert np.abs(Fm - sign * F).max() <= 1e-13 * max(1.0, np.abs(F).max())
        else:
            assert np.array_equal(Fm, sign * F)


@pytest.mark.parametrize("name", SOLVERS)
def test_direction_permutation(orc, name):
    WL, WR = [1.0, 0.3, -0.2, 0.1, 1.5], [0.8, -0.1, 0.4, 0.25, 0.9]
    F0 = flux(orc, name, G53, 0, WL, WR)
    for d in (1, 2):
        perm = lambda W: [W[0]] + [W[1 + (c - d) % 3] for c in range(3)] + [W[4]]
        Fd = flux(orc, name, G53, d, perm(WL), perm(WR))
        back = [Fd[0]] + [Fd[1 + (c + d) % 3] for c in range(3)] + [Fd[4]]
        assert np.array_equal(np.array(back), F0)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hlle_supersonic_upwinds_exactly(orc, d):
    WL, WR = [1.0, 0.1, -0.2, 0.3, 0.9], [1.2, 0.2, 0.1, -0.1, 0.8]
    WL[1 + d], WR[1 + d] = 5.0, 5.5
    F, Fx = orc.hlle(G53, d, WL, WR), phys_flux(G53, d, WL)
    assert np.abs(F - Fx).max() <= 2 * np.spacing(np.abs(Fx).max())
    WL[1 + d], WR[1 + d] = -5.5, -5.0
    F, Fx = orc.hlle(G53, d, WL, WR), phys_flux(G53, d, WR)
    assert np.abs(F - Fx).max() <= 2 * np.spacing(np.abs(Fx).max())


@pytest.mark.parametrize("name", ["hlle", "roe"])
def test_isolated_shock_is_resolved_exactly(orc, name):
    """Right-moving shock obeying Rankine-Hugoniot: F_R - F_L = S (U_R - U_L) and the Roe averages give
    u~ + c~ = S exactly (Roe's property U), so the HLLE flux collapses to F(W_L) whatever the left speed estimate
    is, and Roe's flux does because dU is parallel to K5 alone."""
    g = 1.4
    rR, pR, uR, ps = 1.0, 1.0, 0.0, 4.0
    cR = math.sqrt(g * pR / rR)
    S = uR + cR * math.sqrt((g + 1) / (2 * g) * ps / pR + (g - 1) / (2 * g))
    rL = rR * ((ps / pR + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pR + 1))
    uL = S * (1 - rR / rL)
    WL, WR = [rL, uL, 0, 0, ps / (g - 1)], [rR, uR, 0, 0, pR / (g - 1)]
    np.testing.assert_allclose(flux(orc, name, g, 0, WL, WR), phys_flux(g, 0, WL), rtol=1e-12, atol=1e-13)


def test_stationary_contact_closed_forms(orc):
    """u = 0, equal pressure, rho_L != rho_R.  LLF: mass flux -a/2 (rho_R - rho_L) with a = max(c_L, c_R), momentum
    flux p, energy flux 0 (equal E).  HLLE: Roe u~ = 0, c~^2 = (gamma-1) H~ with H~ the sqrt(rho)-weighted mean of
    gamma u_g / rho; b-+ = -+max(c_K, c~); mass flux b+ b- (rho_R - rho_L) / (b+ - b-)."""
    g, ug, rL, rR = 1.4, 2.5, 1.0, 0.25
    p = (g - 1) * ug
    cL, cR = math.sqrt(g * p / rL), math.sqrt(g * p / rR)
    F = orc.llf(g, 0, [rL, 0, 0, 0, ug], [rR, 0, 0, 0, ug])
    assert F[0] == pytest.approx(-0.5 * max(cL, cR) * (rR - rL), rel=1e-15)
    assert ulp_diff(F[1], p) <= 1 and F[2] == 0.0 and F[3] == 0.0 and F[4] == 0.0
    sL, sR = math.sqrt(rL), math.sqrt(rR)
    Ht = (sL * g * ug / rL + sR * g * ug / rR) / (sL + sR)
    ct = math.sqrt((g - 1) * Ht)
    bm, bp = -max(cL, ct), max(cR, ct)
    F = orc.hlle(g, 0, [rL, 0, 0, 0, ug], [rR, 0, 0, 0, ug])
    assert F[0] == pytest.approx(bp * bm * (rR - rL) / (bp - bm), rel=1e-14)
    assert F[1] == pytest.approx(p, rel=1e-15) and F[2] == 0.0 and F[3] == 0.0 and abs(F[4]) <= 1e-15


def test_roe_keeps_a_contact_with_shear_exactly(orc):
    """u = 0, equal pressure, jumps in density AND transverse velocity: only the l2 = u~ = 0 waves carry the jump, so
    Roe's flux is (0, p, 0, 0, 0) -- nothing is smeared (HLLE and LLF diffuse this contact, HLLC keeps the density)."""
    g, ug = 1.4, 2.5
    for d in range(3):
        WL, WR = [1.0, 0, 0, 0, ug], [0.25, 0, 0, 0, ug]
        WL[1 + (d + 1) % 3], WR[1 + (d + 1) % 3] = 0.3, -0.2
        F = orc.roe(g, d, WL, WR)
        expect = np.zeros(5); expect[1 + d] = (g - 1) * ug
        assert np.abs(F - expect).max() <= 4e-16


@pytest.mark.parametrize("rsolver,name", [(1, "llf"), (2, "hlle"), (3, "roe")])
def test_sod_converges_to_the_exact_solution(orc, rsolver, name):
    g = 1.4
    ps, us = exact_riemann(g, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    errs = {}
    for N in (128, 256, 512):
        U0, U = sod_run(orc, N, I.RECON_PLM, 2, rsolver=rsolver)
        x = (np.arange(N) + 0.5) / N
        right = x >= 0.5
        rho_ex, d = sod_sample(g, (x[right] - 0.75) / 0.1, ps, us)
        errs[N] = np.abs(U[0, right] - rho_ex).mean()
        if name == "roe":
            assert np.abs(U[0] - U[0, ::-1]).max() <= 1e-12 and np.abs(U[1] + U[1, ::-1]).max() <= 1e-12
        else:
            assert np.array_equal(U[0], U[0, ::-1]) and np.array_equal(U[4], U[4, ::-1]) and np.array_equal(U[1], -U[1, ::-1])
        assert abs(U[0].sum() - U0[0].sum()) <= 1e-13 * U0[0].sum()
    r1, r2 = math.log2(errs[128] / errs[256]), math.log2(errs[256] / errs[512])
    assert 0.6 <= r1 <= 1.15 and 0.6 <= r2 <= 1.15, (errs, r1, r2)
    # the same solution as HLLC: errors within a factor 2.5 of each other.  LLF / HLLE smear the contact more than HLLC
    # (error above it); Roe, which resolves the contact exactly and carries less numerical viscosity at the shock than
    # HLLC's bounding wave speeds, ends slightly BELOW it -- hence the lower bound 0.9 (widened from 1.0 when Roe was added)
    _, Uc = sod_run(orc, 256, I.RECON_PLM, 2, rsolver=0)
    x = (np.arange(256) + 0.5) / 256
    rho_ex, _ = sod_sample(g, (x[x >= 0.5] - 0.75) / 0.1, ps, us)
    e_hllc = np.abs(Uc[0, x >= 0.5] - rho_ex).mean()
    assert 0.9 * e_hllc <= errs[256] <= 2.5 * e_hllc, (e_hllc, errs[256])


@pytest.mark.parametrize("rsolver", [1, 2, 3])
def test_uniform_state_and_conservation(orc, rsolver):
    w = I.config1(nrb=2, nx=8)
    p = orc.OrcPack(w.mesh, w.gamma, w.recon, rsolver=rsolver)
    U0 = w.state().numpy()
    p.load(U0)
    for _ in range(10):
        p.step(w.cfl)
    from tests import parity as P
    t0, t1 = P.totals(w.mesh, U0), P.totals(w.mesh, p.current())
    norm = P.momentum_norm(w.mesh, U0, w.gamma)
    assert (np.abs(t1 - t0) / np.array([t0[0], norm, norm, norm, t0[4]])).max() <= 1e-13
    mesh = I.uniform_mesh((2, 1, 1), (8, 8, 8), 2)
    prim = lambda X1, X2, X3: (1.3 + 0 * X1, 0.4 + 0 * X1, -0.7 + 0 * X1, 0.2 + 0 * X1, 0.9 + 0 * X1)
    Uu = I.make_state(mesh, prim).numpy()
    q = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM, rsolver=rsolver)
    q.load(Uu)
    q.step(0.3)
    a = P.active(mesh)
    # LLF / HLLE fluxes of identical states are the physical flux, identical on both faces: nothing changes
    assert np.array_equal(q.current()[a], Uu[a])
