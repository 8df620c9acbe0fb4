"""Scheme-level pins of the oracle (SURVEY 8(c) "Pins"): what the paper and the mathematics fix.

* exact Riemann solution of Sod's problem (solver written here, Newton on the pressure function)
* second-order convergence of a sound-wave eigenmode after one period (Fig.1 left)
* conservation on periodic domains, preservation of uniform states
* mirror / axis-permutation symmetry, decomposition invariance
* closed-form CFL time step (Eq.(3))
"""
import json
import math
import os

import numpy as np
import pytest
import torch

from paper_2409_16053_b200 import inputs as I

GOLD_A = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "appendix_a.json")))
GOLD_C = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "appendix_c.json")))


def act(mesh):
    g = mesh.ng
    return (slice(None), slice(None), slice(g, -g), slice(g, -g), slice(g, -g))


def run(orc, mesh, U0, recon, gamma=I.GAMMA, cfl=0.3, nsteps=None, tend=None, rsolver=0):
    p = orc.OrcPack(mesh, gamma, recon, rsolver=rsolver)
    p.load(U0)
    t, n = 0.0, 0
    while True:
        if nsteps is not None and n >= nsteps:
            break
        if tend is not None and t >= tend:
            break
        dt = p.new_dt(cfl)
        if tend is not None and t + dt > tend:
            dt = tend - t
        p.step(cfl, dt)
        t += dt
        n += 1
    assert p.floor_count() == 0
    out = p.current().copy()
    p.close()
    return out


# ------------------------------------------------------------------ exact Riemann solver ----------
def exact_riemann(g, rL, uL, pL, rR, uR, pR):
    """Textbook exact solution (two-shock / two-rarefaction pressure functions, Newton iteration)."""
    cL, cR = math.sqrt(g * pL / rL), math.sqrt(g * pR / rR)

    def f(p, rK, pK, cK):
        if p > pK:
            A, B = 2.0 / ((g + 1) * rK), (g - 1) / (g + 1) * pK
            return (p - pK) * math.sqrt(A / (p + B)), math.sqrt(A / (p + B)) * (1 - 0.5 * (p - pK) / (p + B))
        return (2 * cK / (g - 1)) * ((p / pK) ** ((g - 1) / (2 * g)) - 1), (1 / (rK * cK)) * (p / pK) ** (-(g + 1) / (2 * g))

    p = 0.5 * (pL + pR)
    for _ in range(100):
        fl, dfl = f(p, rL, pL, cL)
        fr, dfr = f(p, rR, pR, cR)
        pn = p - (fl + fr + (uR - uL)) / (dfl + dfr)
        pn = max(pn, 1e-12)
        if abs(pn - p) < 1e-15 * p:
            p = pn
            break
        p = pn
    u = 0.5 * (uL + uR) + 0.5 * (f(p, rR, pR, cR)[0] - f(p, rL, pL, cL)[0])
    return p, u


def sod_sample(g, xi, ps, us):
    """Density of the Sod solution (left rarefaction, right shock) at similarity coordinate xi = x/t."""
    rL, pL, rR, pR = 1.0, 1.0, 0.125, 0.1
    cL = math.sqrt(g * pL / rL)
    rsL = rL * (ps / pL) ** (1 / g)
    csL = cL * (ps / pL) ** ((g - 1) / (2 * g))
    rsR = rR * ((ps / pR + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * ps / pR + 1))
    S = math.sqrt(g * pR / rR) * math.sqrt((g + 1) / (2 * g) * ps / pR + (g - 1) / (2 * g))
    head, tail = -cL, us - csL
    rho = np.where(xi < head, rL,
          np.where(xi < tail, rL * (2 / (g + 1) + (g - 1) / ((g + 1) * cL) * (0.0 - xi)) ** (2 / (g - 1)),
          np.where(xi < us, rsL, np.where(xi < S, rsR, rR))))
    return rho, dict(rhostar_L=rsL, rhostar_R=rsR, shock=S, head=head, tail=tail)


@pytest.mark.parametrize("key,g", [("gamma_1.4", 1.4), ("gamma_5/3", 5.0 / 3.0)])
def test_exact_riemann_fixture_is_reproduced_by_independent_solver(key, g):
    ps, us = exact_riemann(g, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    _, d = sod_sample(g, np.array([0.0]), ps, us)
    ref = GOLD_A["exact_riemann"][key]
    assert ps == pytest.approx(ref["pstar"], rel=1e-11)
    assert us == pytest.approx(ref["ustar"], rel=1e-11)
    for k in ("rhostar_L", "rhostar_R", "shock", "head", "tail"):
        assert d[k] == pytest.approx(ref[k], rel=1e-11)


def sod_run(orc, N, recon, ng, direction=0, rsolver=0):
    """Periodic line with two mirrored Sod problems: left state on [0.25,0.75)."""
    g = 1.4
    nx = [4, 4, 4]
    nx[direction] = N
    mesh = I.uniform_mesh((1, 1, 1), tuple(nx), ng)

    def prim(X1, X2, X3):
        x = (X1, X2, X3)[direction]
        inside = (x >= 0.25) & (x < 0.75)
        rho = torch.where(inside, 1.0, 0.125).to(torch.float64)
        P = torch.where(inside, 1.0, 0.1).to(torch.float64)
        z = torch.zeros_like(rho)
        return (rho, z, z, z, P)

    U0 = I.make_state(mesh, prim, gamma=g).numpy()
    U = run(orc, mesh, U0, recon, gamma=g, cfl=0.3, tend=0.1, rsolver=rsolver)
    a = [ng, ng, ng]
    sl = [0, slice(None), ng, ng, ng]
    sl[4 - direction] = slice(ng, -ng)
    return U0[tuple(sl)], U[tuple(sl)]          # (5, N) profiles along the sweep direction


@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3)])
def test_sod_against_exact_solution(orc, recon, ng):
    g = 1.4
    ps, us = exact_riemann(g, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    errs = {}
    for N in (128, 256, 512):
        U0, U = sod_run(orc, N, recon, ng)
        x = (np.arange(N) + 0.5) / N
        right = x >= 0.5                                   # Riemann problem centred on 0.75
        rho_ex, d = sod_sample(g, (x[right] - 0.75) / 0.1, ps, us)
        errs[N] = np.abs(U[0, right] - rho_ex).mean()
        # the two halves mirror each other bit-exactly: rho, E even; momentum odd
        assert np.array_equal(U[0], U[0, ::-1]) and np.array_equal(U[4], U[4, ::-1])
        assert np.array_equal(U[1], -U[1, ::-1])
        # mass conserved to round-off
        assert abs(U[0].sum() - U0[0].sum()) <= 1e-13 * U0[0].sum()
        if N == 512:
            xi = (x - 0.75) / 0.1
            plateau_R = (xi > us + 0.25) & (xi < d["shock"] - 0.25)
            plateau_L = (xi > d["tail"] + 0.25) & (xi < us - 0.25)
            assert plateau_R.sum() >= 5 and plateau_L.sum() >= 5
            assert np.abs(U[0, plateau_R] / d["rhostar_R"] - 1).max() < 1e-3
            assert np.abs(U[0, plateau_L] / d["rhostar_L"] - 1).max() < 1e-3
            assert np.abs(U[1, plateau_R] / U[0, plateau_R] / us - 1).max() < 1e-3
    r1 = math.log2(errs[128] / errs[256])
    r2 = math.log2(errs[256] / errs[512])
    assert 0.7 <= r1 <= 1.15 and 0.7 <= r2 <= 1.15, (errs, r1, r2)


def test_sod_is_direction_independent_bit_exact(orc):
    base = sod_run(orc, 64, I.RECON_PLM, 2, 0)[1]
    for d in (1, 2):
        prof = sod_run(orc, 64, I.RECON_PLM, 2, d)[1]
        assert np.array_equal(prof[0], base[0]) and np.array_equal(prof[4], base[4])
        assert np.array_equal(prof[1 + d], base[1])        # normal momentum


# ------------------------------------------------------------------ sound wave convergence --------
def wave_error(orc, N, recon, ng, cfl, direction=0):
    nx = [4, 4, 4]
    nx[direction] = N
    mesh = I.uniform_mesh((1, 1, 1), tuple(nx), ng)
    U0 = I.make_state(mesh, I.sound_wave_prim(direction=direction)).numpy()
    U = run(orc, mesh, U0, recon, cfl=cfl, tend=1.0)
    a = act(mesh)
    return math.sqrt(sum(np.abs(U[a][0, n] - U0[a][0, n]).mean() ** 2 for n in range(5)))


def test_sound_wave_second_order_plm(orc):
    e = {N: wave_error(orc, N, I.RECON_PLM, 2, 0.3) for N in (32, 64, 128, 256)}
    for N, ref in GOLD_C["plm_cfl0.3"].items():              # written by tests/golden/make_appendix_c.py (stand-alone 1-D numpy)
        if int(N) in e:
            assert e[int(N)] == pytest.approx(ref, rel=1e-6)
    for N in (64, 128):
        assert 3.5 <= e[N] / e[2 * N] <= 4.2, e


def test_sound_wave_second_order_ppm4(orc):
    e = {N: wave_error(orc, N, I.RECON_PPM4, 3, 0.1) for N in (32, 64, 128)}
    # PPM4 + SSPRK(2,2) amplifies round-off differences on this 1e-6-amplitude wave (limiter decisions flip at the
    # grid scale: two implementations that agree to 1e-16 after one step differ by 3e-10 after the 320 steps of a
    # period, measured), so the stand-alone script's errors are reproduced to a fraction of a per cent only
    for N, ref in GOLD_C["ppm4_cfl0.1"].items():
        assert e[int(N)] == pytest.approx(ref, rel=1e-2)
    for N in (32, 64):
        assert 3.6 <= e[N] / e[2 * N] <= 4.3, e


@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3), (I.RECON_PPMX, 3), (I.RECON_WENOZ, 3)])
def test_sound_wave_along_x2_x3_matches_x1(orc, recon, ng):
    e1 = wave_error(orc, 32, recon, ng, 0.3, 0)
    assert wave_error(orc, 32, recon, ng, 0.3, 1) == e1
    assert wave_error(orc, 32, recon, ng, 0.3, 2) == e1


# ------------------------------------------------------------------ invariants --------------------
def totals(mesh, U):
    a = act(mesh)
    return np.array([math.fsum(U[a][:, n].ravel()) for n in range(5)])


@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3), (I.RECON_PPMX, 3), (I.RECON_WENOZ, 3)])
def test_conservation_on_periodic_multiblock_mesh(orc, recon, ng):
    mesh = I.uniform_mesh((2, 2, 2), (16, 16, 16), ng)
    U0 = I.make_state(mesh, I.modes_prim(0.5, shear=False, rho_pert=True)).numpy()
    U = run(orc, mesh, U0, recon, nsteps=20)
    t0, t1 = totals(mesh, U0), totals(mesh, U)
    a = act(mesh)
    rho, mom = U0[a][:, 0], U0[a][:, 1:4]
    norm_m = math.fsum((np.sqrt((mom ** 2).sum(1)) + rho * math.sqrt(I.GAMMA)).ravel())   # ~ sum rho(|v|+c_s)
    assert abs(t1[0] - t0[0]) <= 1e-13 * t0[0]
    assert abs(t1[4] - t0[4]) <= 1e-13 * t0[4]
    assert np.abs(t1[1:4] - t0[1:4]).max() <= 1e-13 * norm_m
    assert np.abs(U[a] - U0[a]).max() > 1e-3               # the state did evolve


@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3), (I.RECON_PPMX, 3), (I.RECON_WENOZ, 3)])
def test_uniform_state_is_preserved_bit_exactly(orc, recon, ng):
    mesh = I.uniform_mesh((2, 1, 1), (8, 8, 8), ng)
    prim = lambda X1, X2, X3: (1.3 + 0 * X1, 0.4 + 0 * X1, -0.7 + 0 * X1, 0.2 + 0 * X1, 0.9 + 0 * X1)
    U0 = I.make_state(mesh, prim).numpy()
    p = orc.OrcPack(mesh, I.GAMMA, recon)
    p.load(U0)
    dt = p.new_dt(0.3)
    a = act(mesh)
    for stage in (1, 2):
        p.fill_ghosts()
        p.hydro_stage(stage, dt)
        assert np.array_equal(p.current()[a], U0[a])
    # closed-form dt: CFL * min_d dx_d / (|v_d| + c_s) with dx = (1/16, 1/8, 1/8)
    cs = math.sqrt(I.GAMMA * 0.9 / 1.3)
    expect = 0.3 * min((1 / 16) / (0.4 + cs), (1 / 8) / (0.7 + cs), (1 / 8) / (0.2 + cs))
    assert dt == pytest.approx(expect, rel=1e-14)


def test_dt_uses_each_directions_own_dx_and_is_a_min(orc):
    mesh = I.uniform_mesh((1, 1, 1), (8, 16, 4), 2)            # dx = 1/8, 1/16, 1/4
    prim = lambda X1, X2, X3: (1.0 + 0 * X1, 0.1 + 0 * X1, 0.0 * X1, 3.0 + 0 * X1, 0.6 + 0 * X1)
    U0 = I.make_state(mesh, prim).numpy()
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    p.load(U0)
    cs = 1.0
    expect = 0.3 * min((1 / 8) / (0.1 + cs), (1 / 16) / (0.0 + cs), (1 / 4) / (3.0 + cs))
    assert p.new_dt(0.3) == pytest.approx(expect, rel=1e-14)
    # one hot, fast cell controls the minimum
    U0[0, 4, 5, 7, 3] *= 50.0
    p.load(U0)
    assert p.new_dt(0.3) < expect


def test_dt_on_a_two_level_mesh_uses_each_levels_own_dx(orc):
    """Eq.(3), P:107-110 with 'uniform time stepping' over all levels; reading Q9: every leaf block enters with
    its OWN level's dx.  (the level-dependent dx of orc_new_dt had no CPU pin.)
    A 'level-0 dx everywhere' oracle fails case 1 (dt twice too large), a 'finest dx everywhere' oracle fails case 2."""
    nx, ng = 8, 2
    mesh = I.smr_mesh((2, 2, 2), (nx, nx, nx), ng, (0, 0, 0), (1, 1, 1))     # one root block refined: 7 + 8 blocks
    assert sorted(set(b[0] for b in mesh.blocks)) == [0, 1]
    rho, v, P = 1.3, (0.4, -0.7, 0.2), 0.9
    prim = lambda X1, X2, X3: (rho + 0 * X1, v[0] + 0 * X1, v[1] + 0 * X1, v[2] + 0 * X1, P + 0 * X1)
    U0 = I.make_state(mesh, prim).numpy()
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    p.load(U0)
    cs = math.sqrt(I.GAMMA * P / rho)
    dx0 = 1.0 / (2 * nx)
    # case 1: uniform state -> the fine level decides: CFL (dx0/2) / (max_d |v_d| + c_s)
    assert p.new_dt(0.3) == pytest.approx(0.3 * (dx0 / 2) / (0.7 + cs), rel=1e-14)
    # case 2: one fast cell that sits in a level-0 block only: the answer is the COARSE candidate dx0/(|v1| + c_s)
    m0 = [m for m, b in enumerate(mesh.blocks) if b[0] == 0][3]
    vfast = 40.0
    U1 = U0.copy()
    k, j, i = ng + 3, ng + 1, ng + 5
    U1[m0, 1, k, j, i] = rho * vfast
    U1[m0, 4, k, j, i] = P / (I.GAMMA - 1) + 0.5 * rho * (vfast ** 2 + v[1] ** 2 + v[2] ** 2)
    p.load(U1)
    assert p.new_dt(0.3) == pytest.approx(0.3 * dx0 / (vfast + cs), rel=1e-13)
    # case 3: the same fast cell in a level-1 block: the fine candidate, half of case 2
    m1 = [m for m, b in enumerate(mesh.blocks) if b[0] == 1][5]
    U2 = U0.copy()
    U2[m1, 1, k, j, i] = rho * vfast
    U2[m1, 4, k, j, i] = P / (I.GAMMA - 1) + 0.5 * rho * (vfast ** 2 + v[1] ** 2 + v[2] ** 2)
    p.load(U2)
    assert p.new_dt(0.3) == pytest.approx(0.3 * (dx0 / 2) / (vfast + cs), rel=1e-13)
    # a NaN momentum anywhere in the active cells is reported, not skipped (a NaN density or energy is
    # caught by the floors of reading Q7, which are written as !(x >= floor))
    U3 = U0.copy()
    U3[m0, 2, k, j, i] = float("nan")
    p.load(U3)
    with pytest.raises(orc.OrcError):
        p.new_dt(0.3)
    p.close()


# ------------------------------------------------------------------ strong shocks -------------
def two_shock_sample(g, L, R, ps, us, xi):
    """rho, u, p of a two-shock Riemann solution at xi = x/t (both outer waves shocks: ps > pL, pR)."""
    (rL, uL, pL), (rR, uR, pR) = L, R
    cL, cR = math.sqrt(g * pL / rL), math.sqrt(g * pR / rR)
    mu = (g - 1) / (g + 1)
    rsL = rL * (ps / pL + mu) / (mu * ps / pL + 1)
    rsR = rR * (ps / pR + mu) / (mu * ps / pR + 1)
    SL = uL - cL * math.sqrt((g + 1) / (2 * g) * ps / pL + (g - 1) / (2 * g))
    SR = uR + cR * math.sqrt((g + 1) / (2 * g) * ps / pR + (g - 1) / (2 * g))
    rho = np.where(xi < SL, rL, np.where(xi < us, rsL, np.where(xi < SR, rsR, rR)))
    u = np.where(xi < SL, uL, np.where(xi < SR, us, uR))
    pr = np.where(xi < SL, pL, np.where(xi < SR, ps, pR))
    return rho, u, pr, dict(SL=SL, SR=SR, rsL=rsL, rsR=rsR)


@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3)])
def test_colliding_supersonic_streams_converge_to_the_exact_two_shock_solution(orc, recon, ng):
    """Two Mach-3 / Mach-2.5 streams colliding head-on (the regime of the paper's supersonic-turbulence and blast runs,
    P:142): with the round-1 pressure-based HLLC speeds the first face flux was 0/0.  The run must stay finite,
    floor-free, and converge in L1 to the exact solution (two shocks, a contact), with the star pressure and
    velocity on the plateaus between the shocks within 3 % (post-shock oscillations behind slowly moving strong shocks are a known feature of Godunov-type schemes)."""
    g = 1.4
    L = (1.0, 3.0 * math.sqrt(g * 1.0 / 1.0), 1.0)
    R = (2.0, -2.5 * math.sqrt(g * 0.5 / 2.0), 0.5)
    ps, us = exact_riemann(g, L[0], L[1], L[2], R[0], R[1], R[2])
    assert ps > 10 * L[2]                                  # strong shocks on both sides
    tend = 0.05
    errs = {}
    for N in (128, 256, 512):
        mesh = I.uniform_mesh((1, 1, 1), (N, 4, 4), ng)
        mesh = __import__("dataclasses").replace(mesh, bc=(1, 1, 0, 0, 0, 0))       # outflow ends along x1

        def prim(X1, X2, X3):
            left = X1 < 0.5
            f = lambda a, b: torch.where(left, a, b).to(torch.float64)
            z = torch.zeros_like(X1)
            return (f(L[0], R[0]), f(L[1], R[1]), z, z, f(L[2], R[2]))

        U0 = I.make_state(mesh, prim, gamma=g).numpy()
        U = run(orc, mesh, U0, recon, gamma=g, cfl=0.3, tend=tend)     # asserts floor_count == 0
        prof = U[0, :, ng, ng, ng:-ng]
        assert np.all(np.isfinite(prof))
        x = (np.arange(N) + 0.5) / N
        xi = (x - 0.5) / tend
        rho_ex, u_ex, p_ex, d = two_shock_sample(g, L, R, ps, us, xi)
        assert -0.5 / tend < d["SL"] and d["SR"] < 0.5 / tend          # both shocks still inside the tube
        errs[N] = np.abs(prof[0] - rho_ex).mean()
        if N == 512:
            rho, u = prof[0], prof[1] / prof[0]
            pr = (g - 1) * (prof[4] - 0.5 * rho * u * u)
            width = d["SR"] - d["SL"]
            plateau = (xi > d["SL"] + 0.15 * width) & (xi < d["SR"] - 0.15 * width)
            assert plateau.sum() >= 20
            assert np.abs(pr[plateau] / ps - 1).max() < 3e-2
            assert np.abs(u[plateau] - us).max() < 3e-2 * abs(L[1])
            # densities away from the contact (start-up 'wall heating' leaves a dip AT the contact in every
            # shock-capturing scheme): the outer third of each post-shock region
            left_third = (xi > d["SL"] + 0.1 * width) & (xi < d["SL"] + 0.3 * width) & (xi < us - 0.1 * width)
            right_third = (xi < d["SR"] - 0.1 * width) & (xi > d["SR"] - 0.3 * width) & (xi > us + 0.1 * width)
            assert left_third.sum() >= 5 and right_third.sum() >= 5
            assert np.abs(rho[left_third] / d["rsL"] - 1).max() < 3e-2
            assert np.abs(rho[right_third] / d["rsR"] - 1).max() < 3e-2
    assert errs[256] < 0.75 * errs[128] and errs[512] < 0.75 * errs[256], errs


@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3), (I.RECON_PPMX, 3), (I.RECON_WENOZ, 3)])
def test_decomposition_invariance_bit_exact(orc, recon, ng):
    """Same global field cut into 1x32^3, 8x16^3 and 64x8^3 blocks gives identical active cells."""
    results = []
    for nrb, nx in ((1, 32), (2, 16), (4, 8)):
        mesh = I.uniform_mesh((nrb,) * 3, (nx,) * 3, ng)
        U0 = I.make_state(mesh, I.modes_prim(0.8, shear=False, rho_pert=True)).numpy()
        U = run(orc, mesh, U0, recon, nsteps=3)
        glob = np.zeros((5, 32, 32, 32))
        for m, (_, l1, l2, l3) in enumerate(mesh.blocks):
            glob[:, l3 * nx:(l3 + 1) * nx, l2 * nx:(l2 + 1) * nx, l1 * nx:(l1 + 1) * nx] = U[m][:, ng:-ng, ng:-ng, ng:-ng]
        results.append(glob)
    assert np.array_equal(results[0], results[1])
    assert np.array_equal(results[0], results[2])


@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3), (I.RECON_PPMX, 3), (I.RECON_WENOZ, 3)])
def test_mirror_symmetry_bit_exact_and_axis_permutation(orc, recon, ng):
    mesh = I.uniform_mesh((1, 1, 1), (16, 16, 16), ng)
    U0 = I.make_state(mesh, I.modes_prim(0.8, shear=False, rho_pert=True)).numpy()
    U = run(orc, mesh, U0, recon, nsteps=3)
    # mirror along x1: reverse i, negate rho*v1
    M0 = U0[..., ::-1].copy()
    M0[:, 1] *= -1
    M = run(orc, mesh, M0, recon, nsteps=3)
    back = M[..., ::-1].copy()
    back[:, 1] *= -1
    a = act(mesh)
    assert np.array_equal(back[a], U[a])
    # cyclic axis permutation x1->x2->x3->x1: equal up to summation order (<= 1e-14)
    P0 = np.ascontiguousarray(np.transpose(U0, (0, 1, 3, 4, 2)))[:, [0, 3, 1, 2, 4]]
    P = run(orc, mesh, np.ascontiguousarray(P0), recon, nsteps=3)
    backp = np.transpose(P[:, [0, 2, 3, 1, 4]], (0, 1, 4, 2, 3))
    assert np.abs(backp[a] - U[a]).max() <= 1e-13
