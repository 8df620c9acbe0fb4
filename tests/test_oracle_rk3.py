"""Pins for the oracle's SSPRK(3,3) option (paper P:105: "SSP Runge-Kutta ... RK1 through RK4"; SURVEY 8(f) f2;
coefficients: DESIGN.md Q27).  The coefficients are pinned by the temporal order they must produce: on a FIXED grid
the spatial discretisation is the same for every dt, so the difference to a tiny-dt reference on that grid is purely
the time integrator's error -- it must fall 8x per halving of dt for three stages (4x for the default two), to the
extent the van Leer limiter's kinks at extrema allow (measured 7.5 and 6.5; a wrong weight gives 2x).  Plus
conservation to round-off and the uniform state to round-off (3/4 u + 1/4 u is not exactly u in floating point)."""
import math

import numpy as np
import torch

from paper_2409_16053_b200 import inputs as I
from tests import parity as P


def _setup():
    mesh = I.uniform_mesh((1, 1, 1), (32, 4, 4), 2)

    def prim(X1, X2, X3):
        s = torch.sin(2 * math.pi * X1)
        return (1.0 + 0.2 * s, 0.3 + 0.1 * s, 0 * X1, 0 * X1, 1.0 + 0.1 * s)

    return mesh, I.make_state(mesh, prim).numpy()


def _run(orc, mesh, U0, nstages, nsteps, T=0.05):
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    p.load(U0)
    if nstages != 2:
        p.set_integrator(nstages)
    for _ in range(nsteps):
        p.step(0.3, T / nsteps)
    return p.current()[P.active(mesh)].copy()


def test_temporal_order_on_a_fixed_grid(orc):
    mesh, U0 = _setup()
    ref = _run(orc, mesh, U0, 3, 1024)
    err = {n: {k: np.abs(_run(orc, mesh, U0, n, k) - ref).max() for k in (8, 16, 32)} for n in (2, 3)}
    assert 3.7 <= err[2][8] / err[2][16] <= 4.3 and 3.7 <= err[2][16] / err[2][32] <= 4.3, err
    assert 6.5 <= err[3][8] / err[3][16] <= 8.5 and 5.5 <= err[3][16] / err[3][32] <= 8.5, err
    assert err[3][8] < err[2][8] / 5 and err[3][32] < err[2][32] / 15, err


def test_forward_euler_is_first_order_and_alternates_the_registers(orc):
    """RK1 of the paper's list: error to the tiny-dt reference halves with dt; A and B alternate."""
    mesh, U0 = _setup()
    ref = _run(orc, mesh, U0, 3, 1024)
    e = {k: np.abs(_run(orc, mesh, U0, 1, k) - ref).max() for k in (16, 32, 64)}
    assert 1.9 <= e[16] / e[32] <= 2.2 and 1.9 <= e[32] / e[64] <= 2.2, e
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    p.load(U0)
    p.set_integrator(1)
    p.step(0.3, 1e-3)
    assert p.current() is p.ub
    t0, t1 = P.totals(mesh, U0), P.totals(mesh, p.current())
    assert abs(t1[0] - t0[0]) <= 1e-14 * t0[0] and abs(t1[4] - t0[4]) <= 1e-14 * t0[4]
    import pytest
    with pytest.raises(orc.OrcError):
        p.set_integrator(2)                 # U^n sits in B after an odd number of Euler steps
    p.step(0.3, 1e-3)
    assert p.current() is p.ua
    p.set_integrator(2)


def test_rk3_conserves_and_keeps_a_uniform_state_to_round_off(orc):
    w = I.config1(nrb=2, nx=8)
    p = orc.OrcPack(w.mesh, w.gamma, w.recon)
    U0 = w.state().numpy()
    p.load(U0)
    p.set_integrator(3)
    for _ in range(8):
        p.step(w.cfl)
    t0, t1 = P.totals(w.mesh, U0), P.totals(w.mesh, p.current())
    norm = P.momentum_norm(w.mesh, U0, w.gamma)
    assert (np.abs(t1 - t0) / np.array([t0[0], norm, norm, norm, t0[4]])).max() <= 1e-13
    assert p.floor_count() == 0
    mesh = I.uniform_mesh((2, 1, 1), (8, 8, 8), 2)
    prim = lambda X1, X2, X3: (1.3 + 0 * X1, 0.4 + 0 * X1, -0.7 + 0 * X1, 0.2 + 0 * X1, 0.9 + 0 * X1)
    Uu = I.make_state(mesh, prim).numpy()
    q = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    q.load(Uu)
    q.set_integrator(3)
    for _ in range(3):
        q.step(0.3)
    a = P.active(mesh)
    assert np.abs(q.current()[a] / Uu[a] - 1).max() <= 4e-16


def test_stage_order_is_enforced(orc):
    import pytest
    mesh, U0 = _setup()
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    p.load(U0)
    p.fill_ghosts()
    with pytest.raises(orc.OrcError):
        p.hydro_stage(3, 1e-3)              # two-stage integrator
    p.set_integrator(3)
    with pytest.raises(orc.OrcError):
        p.hydro_stage(2, 1e-3)              # stage 1 first
    for s in (1, 2, 3):
        p.fill_ghosts()
        p.hydro_stage(s, 1e-3)
    assert p.current() is p.ua
