"""Pins for the oracle's first-order flux correction (paper P:118; reading DESIGN.md Q31).

  * positivity: two streams receding at Mach 10 (and colliding across the periodic boundary) drive the internal energy --
    with WENOZ also the density -- negative with every reconstruction (the floors fire thousands of times); with FOFC the
    floors never fire, density and internal energy stay positive, and the totals are conserved to round-off (the replaced
    fluxes are single-valued);
  * inertness: on a smooth input no cell is flagged and the results are bit-identical with the switch on or off;
  * what is replaced: after one stage only flagged cells and their face neighbours differ from the uncorrected run, and a flagged cell's new value is U_in - dt/dx [F_LLF(i+1/2) - F_LLF(i-1/2)] with the Rusanov flux of
    the CELL-CENTRED states, evaluated here in numpy.
"""
import math

import numpy as np
import pytest
import torch

from paper_2409_16053_b200 import inputs as I
from tests import parity as P

G = I.GAMMA


def receding(mach):
    c = math.sqrt(G)
    return lambda X1, X2, X3: (torch.ones_like(X1), torch.where(X1 < 0.5, -mach * c, mach * c) * torch.ones_like(X1),
                               0 * X1, 0 * X1, torch.ones_like(X1))


def eint(U):
    return U[:, 4] - 0.5 * (U[:, 1:4] ** 2).sum(1) / U[:, 0]


@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3), (I.RECON_WENOZ, 3)])
def test_positivity_where_the_floors_fire_without_it(orc, recon, ng):
    mesh = I.uniform_mesh((2, 1, 1), (32, 4, 4), ng)
    U0 = I.make_state(mesh, receding(10.0)).numpy()
    a = P.active(mesh)
    res = {}
    for on in (False, True):
        p = orc.OrcPack(mesh, G, recon, threads=2)
        p.set_fofc(on)
        p.load(U0)
        for _ in range(30):
            p.step(0.3)
        res[on] = (p.floor_count(), p.fofc_count(), p.current()[a].copy())
        p.close()
    assert res[False][0] > 1000 and res[False][1] == 0          # the uncorrected scheme lives on its floors here
    floors, nflag, U = res[True]
    assert floors == 0 and nflag > 0
    assert U[:, 0].min() > 0.0 and eint(U).min() > 0.0 and np.all(np.isfinite(U))
    t0, t1 = P.totals(mesh, U0), P.totals(mesh, res[True][2] if False else np.pad(U, ((0, 0), (0, 0), (ng, ng), (ng, ng), (ng, ng))))
    assert abs(t1[0] - t0[0]) <= 1e-13 * t0[0] and abs(t1[4] - t0[4]) <= 1e-13 * t0[4]


@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3)])
def test_inert_on_smooth_input(orc, recon, ng):
    w = I.config1(nrb=2, nx=8)
    w.mesh = I.uniform_mesh((2, 2, 2), (8, 8, 8), ng)
    U0 = w.state().numpy()
    out = []
    for on in (False, True):
        p = orc.OrcPack(w.mesh, w.gamma, recon, threads=P.NTHREADS)
        p.set_fofc(on)
        p.load(U0)
        for _ in range(3):
            p.step(w.cfl)
        assert p.fofc_count() == 0
        out.append(p.current().copy())
        p.close()
    assert np.array_equal(out[0], out[1])


def llf_numpy(WL, WR):
    """Rusanov flux along x1 of primitive states (rho, u, v, w, u_g), restated from the textbook form."""
    def cons_flux(W):
        r, u, v, w, e = W
        p = (G - 1) * e
        E = e + 0.5 * r * (u * u + v * v + w * w)
        return np.array([r, r * u, r * v, r * w, E]), np.array([r * u, r * u * u + p, r * u * v, r * u * w, (E + p) * u]), np.sqrt(G * p / r)
    UL, FL, cL = cons_flux(WL)
    UR, FR, cR = cons_flux(WR)
    a = np.maximum(np.abs(WL[1]) + cL, np.abs(WR[1]) + cR)
    return 0.5 * ((FL + FR) - a * (UR - UL))


def test_flagged_cells_take_the_first_order_llf_update(orc):
    ng, N = 3, 32
    mesh = I.uniform_mesh((1, 1, 1), (N, 4, 4), ng)
    U0 = I.make_state(mesh, receding(10.0)).numpy()
    dt = None
    res = {}
    for on in (False, True):
        p = orc.OrcPack(mesh, G, I.RECON_PPM4)
        p.set_fofc(on)
        p.load(U0)
        dt = 4.0 * p.new_dt(0.3)      # (beyond the CFL limit on purpose: the first stage then already drives cells negative)
        p.fill_ghosts()
        p.hydro_stage(1, dt)
        res[on] = (p.current()[0][:, ng, ng, ng:-ng].copy(), p.fofc_count())
        p.close()
    tent, fixed = res[False][0], res[True][0]
    flagged = ~(tent[0] > 0) | ~((tent[4] - 0.5 * (tent[1:4] ** 2).sum(0) / tent[0]) > 0)
    assert flagged.sum() >= 2 and res[True][1] == flagged.sum() * 16      # (4 x 4 identical columns)
    changed = np.abs(fixed - tent).max(0) > 0
    near = flagged | np.roll(flagged, 1) | np.roll(flagged, -1)
    # only flagged cells and their face neighbours may differ (a neighbour whose shared face separates two equal states
    # keeps its value: there LLF and the high-order flux are both the physical flux), and every flagged cell does
    assert np.all(near[changed]) and np.all(changed[flagged])
    # the flagged cells' new values, from the cell-centred states of U_in
    u = U0[0][:, ng, ng, ng:-ng]
    W = np.array([u[0], u[1] / u[0], u[2] / u[0], u[3] / u[0], u[4] - 0.5 * (u[1:4] ** 2).sum(0) / u[0]])
    Flo = llf_numpy(np.roll(W, 1, axis=1), W)                # flux at the lower face of every cell
    expect = u - dt * N * (np.roll(Flo, -1, axis=1) - Flo)
    assert np.abs(fixed[:, flagged] - expect[:, flagged]).max() <= 1e-13 * np.abs(expect).max()
