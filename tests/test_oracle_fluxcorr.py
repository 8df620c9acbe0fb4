"""Pins for the oracle's flux correction at coarse-fine faces (paper P:57: the AMR framework
"includes ... flux correction"; north_star's stage list omits it, so it is an option that is off by default).

What fixes it without an implementation to compare against:
  * conservation: on a periodic two-level mesh whose level boundaries carry structure, the totals of all five
    conserved variables stay constant to round-off with the correction and drift at the 1e-6 level without it
    (a wrong face, sign, fine-flux choice or a missing face breaks the telescoping);
  * the corrected coarse flux is a MEAN of fine fluxes: a uniform state (v != 0) stays bit-identical;
  * it touches level boundaries only: on a single-level mesh the switch changes nothing, bit for bit, and on the
    two-level mesh only the coarse cells that touch a fine block differ from the uncorrected result after one stage;
  * 1-D data along x1 stay 1-D: the four fine fluxes through a coarse x1-face are identical there, so the transverse
    profiles remain bit-identical.
"""
import numpy as np
import pytest

from paper_2409_16053_b200 import inputs as I
from tests import parity as P


def act(mesh):
    return P.active(mesh)


def drift(w, orc, on, nsteps):
    po = orc.OrcPack(w.mesh, w.gamma, w.recon, threads=P.NTHREADS)
    U0 = w.state().numpy()
    po.load(U0)
    po.set_flux_correction(on)
    for _ in range(nsteps):
        po.step(w.cfl)
    assert po.floor_count() == 0
    t0, t1 = P.totals(w.mesh, U0), P.totals(w.mesh, po.current())
    norm = P.momentum_norm(w.mesh, U0, w.gamma)
    return np.abs(t1 - t0) / np.array([t0[0], norm, norm, norm, t0[4]])


def test_smr_conserves_to_round_off_only_with_flux_correction(orc):
    w = I.smr_parity(nx=8)                    # config-4 mesh (120 blocks), random-mode field on the level boundaries
    with_fc, without = drift(w, orc, True, 6), drift(w, orc, False, 6)
    assert with_fc.max() <= 1e-14, with_fc
    assert without.min() >= 1e-9, without     # the uncorrected scheme is visibly non-conservative here


def test_uniform_state_with_velocity_is_preserved_bit_exactly(orc):
    mesh = I.smr_mesh((2, 2, 2), (8, 8, 8), 2, (0, 0, 0), (1, 1, 1))
    prim = lambda X1, X2, X3: (1.3 + 0 * X1, 0.4 + 0 * X1, -0.7 + 0 * X1, 0.2 + 0 * X1, 0.9 + 0 * X1)
    U0 = I.make_state(mesh, prim).numpy()
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    p.load(U0)
    p.set_flux_correction(True)
    dt = p.new_dt(0.3)
    for stage in (1, 2):
        p.fill_ghosts()
        p.hydro_stage(stage, dt)
        assert np.array_equal(p.current()[act(mesh)], U0[act(mesh)])


def test_switch_is_inert_on_a_single_level_mesh(orc):
    w = I.config1(nrb=2, nx=8)
    res = []
    for on in (False, True):
        p = orc.OrcPack(w.mesh, w.gamma, w.recon)
        p.load(w.state().numpy())
        p.set_flux_correction(on)
        for _ in range(2):
            p.step(w.cfl)
        res.append(p.current().copy())
    assert np.array_equal(res[0], res[1])


def test_only_coarse_cells_next_to_fine_blocks_change(orc):
    w = I.smr_parity(nx=8)
    mesh, g, nx = w.mesh, w.mesh.ng, 8
    res = []
    for on in (False, True):
        p = orc.OrcPack(mesh, w.gamma, w.recon, threads=P.NTHREADS)
        p.load(w.state().numpy())
        p.set_flux_correction(on)
        dt = p.new_dt(w.cfl)
        p.fill_ghosts()
        p.hydro_stage(1, dt)
        res.append(p.current().copy())
    diff = np.any(res[0] != res[1], axis=1)                      # (nmb, k, j, i)
    nchanged = 0
    for m, (lev, l1, l2, l3) in enumerate(mesh.blocks):
        d = diff[m][g:-g, g:-g, g:-g]
        if lev == 1:
            assert not d.any()                                   # fine blocks keep their own fluxes
            continue
        allowed = np.zeros_like(d)
        # refined region = root blocks 1..2 in every direction; a coarse block touches it across a face iff it
        # is one block away in exactly one direction and inside [1, 2] in the other two
        l = (l1, l2, l3)
        for dirn in range(3):
            others = [l[e] for e in range(3) if e != dirn]
            if all(1 <= o <= 2 for o in others):
                sl = [slice(None)] * 3
                if l[dirn] == 0:
                    sl[2 - dirn] = slice(nx - 1, nx); allowed[tuple(sl)] = True
                if l[dirn] == 3:
                    sl[2 - dirn] = slice(0, 1); allowed[tuple(sl)] = True
        assert not (d & ~allowed).any(), (m, l)
        nchanged += int(d.sum())
    assert nchanged == 6 * 16 * 16            # every coarse cell on the surface of the 16^3-coarse-cell refined cube


def test_one_dimensional_data_stay_one_dimensional(orc):
    mesh = I.smr_mesh((4, 2, 2), (8, 8, 8), 2, (1, 0, 0), (3, 2, 2))      # refined slab in x1, full extent in x2, x3
    import torch
    tprim = lambda X1, X2, X3: (1.0 + 0.3 * torch.sin(2 * torch.pi * X1), 0.5 + 0 * X1, 0 * X1, 0 * X1,
                                1.0 + 0.2 * torch.cos(2 * torch.pi * X1))
    U0 = I.make_state(mesh, tprim).numpy()
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    p.load(U0)
    p.set_flux_correction(True)
    for _ in range(3):
        p.step(0.3)
    U = p.current()
    g = mesh.ng
    for m in range(mesh.nmb):
        a = U[m][:, g:-g, g:-g, g:-g]
        assert np.array_equal(a, np.broadcast_to(a[:, :1, :1, :], a.shape)), m
        assert np.all(a[2] == 0.0) and np.all(a[3] == 0.0)
