"""GPU parity of the MHD + constrained-transport path (include/ak_mhd.h, csrc/mhd/ak_mhd.cu) against the
oracle (oracle/orc_mhd.cpp) through the C-ABI binding: ghost cells bit-exact, states within the tolerances of the hydro path
(Q14-style metric <= 1e-12 per stage, <= 1e-9 over the run), div B to round-off on the GPU, conserved totals, dt.
"""
import math

import numpy as np
import pytest
import torch

from paper_2409_16053_b200 import inputs as I
from tests import parity as P
from tests.test_oracle_mhd import G53, ZERO_A, act, brio_wu, divb

pytestmark = pytest.mark.gpu
TOL_STAGE, TOL_RUN = 1e-12, 1e-9


@pytest.fixture(scope="module")
def om():
    from oracle import orc_mhd
    orc_mhd.build()
    return orc_mhd


@pytest.fixture(scope="module")
def akm():
    from paper_2409_16053_b200 import ak_mhd
    ak_mhd.lib()
    assert torch.cuda.is_available()
    return ak_mhd


def q_mhd(Ug, Uo, gamma):
    """Per cell max of |d rho|/rho, |d m|/(rho (|v| + c_f)), |dE|/E, |d b|/(|B| + sqrt(rho) c_f-scale); denominators from the oracle."""
    rho, m, E, b = Uo[:, 0], Uo[:, 1:4], Uo[:, 4], Uo[:, 5:8]
    b2 = (b ** 2).sum(1)
    p = np.maximum((gamma - 1.0) * (E - 0.5 * (m ** 2).sum(1) / rho - 0.5 * b2), 0.0)
    cf = np.sqrt((gamma * p + b2) / rho)
    vmag = np.sqrt((m ** 2).sum(1)) / rho
    d = np.abs(Ug - Uo)
    e = np.maximum(d[:, 0] / rho, d[:, 4] / E)
    e = np.maximum(e, d[:, 1:4].max(1) / (rho * (vmag + cf)))
    e = np.maximum(e, d[:, 5:8].max(1) / (np.sqrt(rho) * (vmag + cf)))
    return float(e.max())


def turbulent_state(mesh, mach=0.5, shift=(0.0, 0.0, 0.0)):
    """Smooth 3-D field with a tangled magnetic field.  Unshifted it has planes of exact symmetry on the grid (a velocity that vanishes
    on a plane of cell centres: the case the ramped upwind switch of Q36 exists for); `shift` moves the pattern off the grid."""
    k = 2 * math.pi

    def A(X1, X2, X3):
        X1, X2, X3 = X1 + shift[0], X2 + shift[1], X3 + shift[2]
        return (0.1 * torch.sin(k * X2) * torch.cos(2 * k * X3) + 0 * X1, 0.1 * torch.sin(k * X3 + 0.3) * torch.cos(k * X1) + 0 * X2,
                0.1 * torch.cos(2 * k * X1 + 0.7) * torch.sin(k * X2) + 0 * X3)

    def prim(X1, X2, X3):
        X1, X2, X3 = X1 + shift[0], X2 + shift[1], X3 + shift[2]
        return (1.0 + 0.3 * torch.sin(k * X1) * torch.cos(k * X2) + 0 * X3,
                mach * torch.sin(k * X2 + 0.2) * torch.cos(k * X3) + 0 * X1,
                -mach * torch.cos(k * X3) * torch.sin(2 * k * X1) + 0 * X2,
                mach * torch.sin(k * X1 + 1.0) * torch.sin(k * X2) + 0 * X3, 0.6 + 0 * X1 + 0 * X2 + 0 * X3)
    return I.make_state_mhd(mesh, prim, A, (0.4, -0.3, 0.2))


def lockstep(om, akm, mesh, U0, gamma, nsteps, cfl=0.3, exact=False, recon=0, nstages=2, rsolver=0):
    po = om.OrcMhdPack(mesh, gamma, threads=P.NTHREADS, recon=recon, nstages=nstages, rsolver=rsolver)
    pg = akm.MhdPack(mesh, gamma, exact=exact, recon=recon, nstages=nstages, rsolver=rsolver)
    po.load(U0.numpy())
    pg.load(U0)
    a = act(mesh)
    errs = []
    for step in range(nsteps):
        dt = po.new_dt(cfl)
        dtg = pg.new_dt(cfl)
        assert abs(dtg - dt) <= 1e-13 * dt, (step, dt, dtg)
        for stage in range(1, nstages + 1):
            po.fill_ghosts(); pg.fill_ghosts()
            if step == 0:
                ug = pg.current().cpu().numpy()
                chk = om.OrcMhdPack(mesh, gamma)
                chk.load(ug); chk.fill_ghosts()
                assert np.array_equal(chk.current(), ug), f"ghost fill differs at stage {stage}"
                chk.close()
            po.stage(stage, dt); pg.stage(stage, dt)
            if step == 0:
                e = q_mhd(pg.current().cpu().numpy()[a], po.current()[a], gamma)
                assert e <= TOL_STAGE * stage, f"stage {stage}: {e:.3e}"
        errs.append(q_mhd(pg.current().cpu().numpy()[a], po.current()[a], gamma))
    assert po.floor_count() == 0 and pg.floor_count() == 0
    return errs, po, pg


@pytest.mark.parametrize("exact", [False, True])
@pytest.mark.parametrize("nrb,nx", [((2, 2, 2), (16, 16, 16)), ((2, 1, 3), (24, 10, 6)), ((1, 1, 1), (4, 6, 8)), ((2, 2, 2), (32, 32, 32))])
def test_turbulent_field_matches_the_oracle(om, akm, nrb, nx, exact):
    """Default arithmetic (MUFU-seeded reciprocals / square roots): within the hydro path's tolerances; verification mode
    (akm_pack_set_exact: IEEE division / sqrt in the definition's order): bit-identical to the oracle."""
    mesh = I.uniform_mesh(nrb, nx, 3)
    U0 = turbulent_state(mesh)
    errs, po, pg = lockstep(om, akm, mesh, U0, G53, 6 if nx[0] < 32 else 3, exact=exact)
    P.report(f"[parity] MHD turbulent field nmb={mesh.nmb} nx={nx} exact={exact}: worst per step {max(errs):.3e} (bar {TOL_RUN:.0e}), first step {errs[0]:.3e}")
    assert max(errs) <= TOL_RUN
    if exact:
        assert max(errs) == 0.0
    pg.fill_ghosts()
    ug = pg.current().cpu().numpy()
    assert np.abs(divb(mesh, ug)).max() <= 2e-13                          # div B on the GPU state
    a = act(mesh)
    for n in range(8):                                                   # totals incl. the mean field, GPU vs initial
        scale = np.abs(U0.numpy()[a][:, n]).sum() + 1.0
        assert abs(ug[a][:, n].sum() - U0.numpy()[a][:, n].sum()) <= 1e-12 * scale, n
    # free-running: each side computes its own dt
    p2 = akm.MhdPack(mesh, G53, exact=exact)
    p2.load(U0)
    nst = 6 if nx[0] < 32 else 3
    for _ in range(nst):
        p2.step(0.3)
    assert q_mhd(p2.current().cpu().numpy()[a], po.current()[a], G53) <= TOL_RUN
    assert p2.launch_count() == nst * (2 + 2 * 7)                          # dt_init + dt + 2 x (fill + 6 stage kernels) per step


@pytest.mark.parametrize("exact", [False, True])
@pytest.mark.parametrize("recon,nstages", [(1, 2), (2, 3), (3, 2), (3, 3), (0, 3)])
@pytest.mark.parametrize("nrb,nx", [((2, 2, 2), (16, 16, 16)), ((2, 1, 3), (24, 10, 6))])
def test_higher_order_options_match_the_oracle(om, akm, nrb, nx, recon, nstages, exact):
    """PPM4 / PPMX / WENOZ reconstruction and SSPRK(3,3) (the options of the paper's MHD tests and runs; ng = 4): same bars as
    the PLM + RK2 path, bit-identical in the verification flavour."""
    mesh = I.uniform_mesh(nrb, nx, 4)
    # PPMX switches between its extremum and its monotone limiter where two neighbouring cells are equal: a discontinuous function of
    # the data there (Q30), so a field with exact mirror symmetries on the grid lets 1 ulp decide O(1e-7) -- in the default flavour
    # the pattern is moved off the grid for it; the verification flavour takes the symmetric field (bit-identical either way)
    shift = (0.0137, 0.0291, 0.0173) if (recon == 2 and not exact) else (0.0, 0.0, 0.0)
    U0 = turbulent_state(mesh, shift=shift)
    errs, po, pg = lockstep(om, akm, mesh, U0, G53, 4, exact=exact, recon=recon, nstages=nstages)
    name = f"{['PLM', 'PPM4', 'PPMX', 'WENOZ'][recon]} + SSPRK{nstages}"
    P.report(f"[parity] MHD {name} nmb={mesh.nmb} nx={nx} exact={exact}: worst per step {max(errs):.3e} (bar {TOL_RUN:.0e}), first step {errs[0]:.3e}")
    assert max(errs) <= TOL_RUN and (max(errs) == 0.0 or not exact)
    pg.fill_ghosts()
    ug = pg.current().cpu().numpy()
    assert np.abs(divb(mesh, ug)).max() <= 2e-13
    a = act(mesh)
    for n in range(8):
        scale = np.abs(U0.numpy()[a][:, n]).sum() + 1.0
        assert abs(ug[a][:, n].sum() - U0.numpy()[a][:, n].sum()) <= 1e-12 * scale, n
    assert pg.launch_count() == 4 * (2 + nstages * 7) + 1                  # (+ the fill above)
    with pytest.raises(akm.AkmError):
        akm.MhdPack(I.uniform_mesh((1, 1, 1), (8, 8, 8), 3), G53, recon=recon or 1)   # ng < 4


@pytest.mark.parametrize("exact", [False, True])
@pytest.mark.parametrize("rsolver", [1, 2])
def test_llf_and_hlle_match_the_oracle(om, akm, rsolver, exact):
    """LLF and HLLE for MHD (PLM, RK2) on the ragged 6-block pack and along a Brio-Wu tube: same bars as HLLD."""
    mesh = I.uniform_mesh((2, 1, 3), (24, 10, 6), 3)
    U0 = turbulent_state(mesh)
    errs, po, pg = lockstep(om, akm, mesh, U0, G53, 5, exact=exact, rsolver=rsolver)
    mesh1, B0 = brio_wu(64, 1)
    p1 = om.OrcMhdPack(mesh1, 2.0, threads=P.NTHREADS, rsolver=rsolver)
    g1 = akm.MhdPack(mesh1, 2.0, exact=exact, rsolver=rsolver)
    p1.load(B0); g1.load(torch.from_numpy(B0))
    t = 0.0
    while t < 0.05:
        dt = min(p1.new_dt(0.3), 0.05 - t)
        p1.step(0.3, dt); g1.step(0.3, dt)
        t += dt
    a = act(mesh1)
    e = q_mhd(g1.current().cpu().numpy()[a], p1.current()[a], 2.0)
    P.report(f"[parity] MHD {['', 'LLF', 'HLLE'][rsolver]} exact={exact}: turbulent field worst per step {max(errs):.3e}, Brio-Wu {e:.3e} (bar {TOL_RUN:.0e})")
    assert max(errs) <= TOL_RUN and e <= TOL_RUN and (not exact or (max(errs) == 0.0 and e == 0.0))
    assert g1.floor_count() == 0 and pg.floor_count() == 0
    with pytest.raises(akm.AkmError) as ei:                                # LLF / HLLE are built with PLM only
        akm.MhdPack(I.uniform_mesh((1, 1, 1), (8, 8, 8), 4), G53, recon=1, rsolver=rsolver)
    assert "PLM only" in str(ei.value)


@pytest.mark.parametrize("exact", [False, True])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_brio_wu_on_the_gpu(om, akm, d, exact):
    mesh, U0 = brio_wu(64, d)
    U0 = torch.from_numpy(U0)
    po = om.OrcMhdPack(mesh, 2.0, threads=P.NTHREADS)
    pg = akm.MhdPack(mesh, 2.0, exact=exact)
    po.load(U0.numpy()); pg.load(U0)
    t = 0.0
    while t < 0.05:
        dt = min(po.new_dt(0.3), 0.05 - t)
        po.step(0.3, dt); pg.step(0.3, dt)
        t += dt
    a = act(mesh)
    e = q_mhd(pg.current().cpu().numpy()[a], po.current()[a], 2.0)
    P.report(f"[parity] MHD Brio-Wu along x{d + 1}, 64 cells, exact={exact}: {e:.3e}")
    assert e <= TOL_RUN and pg.floor_count() == 0 and (e == 0.0 or not exact)


@pytest.mark.parametrize("recon,nstages,exact", [(1, 2, False), (3, 3, False), (3, 3, True)])
def test_brio_wu_with_the_higher_order_options_on_the_gpu(om, akm, recon, nstages, exact):
    """P:156 (Fig. 3 right: the Brio-Wu tube with different methods): two mirrored tubes of 200 cells each, PPM4 + RK2 and WENOZ + RK3,
    to t = 0.05 (~170 steps): finite, floor-free, density within its initial bounds.  Verification flavour: bit-identical to the
    oracle at the end.  Default flavour: within the run tolerance after 40 steps (twice the length of the configs' runs); over the
    whole run WENOZ's nonlinear weights amplify the 1-ulp differences at the discontinuities (measured 9e-9 at the end against
    6e-14 for PPM4), so the end state is held to 1e-6 and reported."""
    mesh, U0 = brio_wu(400, 0, ng=4)
    U0 = torch.from_numpy(U0)
    po = om.OrcMhdPack(mesh, 2.0, threads=P.NTHREADS, recon=recon, nstages=nstages)
    pg = akm.MhdPack(mesh, 2.0, recon=recon, nstages=nstages, exact=exact)
    po.load(U0.numpy()); pg.load(U0)
    a = act(mesh)
    t, n, e40 = 0.0, 0, None
    while t < 0.05:
        dt = min(po.new_dt(0.3), 0.05 - t)
        po.step(0.3, dt); pg.step(0.3, dt)
        t += dt
        n += 1
        if n == 40:
            e40 = q_mhd(pg.current().cpu().numpy()[a], po.current()[a], 2.0)
    ug = pg.current().cpu().numpy()[a]
    e = q_mhd(ug, po.current()[a], 2.0)
    P.report(f"[parity] MHD Brio-Wu 2 x 200 cells, {['PLM', 'PPM4', 'PPMX', 'WENOZ'][recon]} + SSPRK{nstages}, exact={exact}: after 40 steps {e40:.3e} (bar {TOL_RUN:.0e}), after {n} steps {e:.3e}")
    assert n > 40 and e40 <= TOL_RUN and e <= 1e-6 and (e == 0.0 or not exact)
    assert pg.floor_count() == 0 and po.floor_count() == 0 and np.isfinite(ug).all()
    assert ug[0, 0].min() > 0.1 and ug[0, 0].max() <= 1.0 + 1e-12            # density stays within the initial bounds


def test_uniform_state_dt_and_errors_on_the_gpu(om, akm):
    mesh = I.uniform_mesh((2, 1, 2), (6, 8, 4), 3)
    prim = lambda X1, X2, X3: (1.3 + 0 * X1 + 0 * X2 + 0 * X3, 0.4 + 0 * X1 + 0 * X2 + 0 * X3, -0.7 + 0 * X1 + 0 * X2 + 0 * X3,
                               0.2 + 0 * X1 + 0 * X2 + 0 * X3, 0.9 + 0 * X1 + 0 * X2 + 0 * X3)
    U0 = I.make_state_mhd(mesh, prim, ZERO_A, (0.5, -0.3, 0.8))
    pg = akm.MhdPack(mesh, G53)
    pg.load(U0)
    po = om.OrcMhdPack(mesh, G53)
    po.load(U0.numpy())
    assert pg.new_dt(0.3) == po.new_dt(0.3)                              # same state, same bits
    pg.step(0.3); pg.step(0.3)
    a = act(mesh)
    assert np.array_equal(pg.current().cpu().numpy()[a], U0.numpy()[a])  # preserved bit for bit
    with pytest.raises(akm.AkmError):
        pg.stage(1, 1e-3)                                                # ghosts not filled
    pg.fill_ghosts()
    with pytest.raises(akm.AkmError):
        pg.stage(2, 1e-3)                                                # stage 2 before stage 1
    pg.stage(1, 1e-3)
    assert akm.lib().akm_pack_set_integrator(pg._h, 3) == -2             # the integrator cannot change inside a step
    assert akm.lib().akm_pack_set_recon(pg._h, 7) == -3 and akm.lib().akm_pack_set_recon(pg._h, 3) == -1   # unknown code; ng = 3
    pg.fill_ghosts(); pg.stage(2, 1e-3)
    assert akm.lib().akm_pack_set_integrator(pg._h, 3) == 0
    with pytest.raises(akm.AkmError):
        pg.fill_ghosts(); pg.stage(1, 1e-3); pg.fill_ghosts(); pg.stage(2, 1e-3); pg.fill_ghosts(); pg.stage(3, 1e-3); pg.stage(1, 1e-3)   # ghosts not refilled
    bad = U0.clone()
    bad[0, 2, 4, 5, 6] = float("nan")
    pg.load(bad)
    with pytest.raises(akm.AkmError) as ei:
        pg.new_dt(0.3)
    assert "non-finite" in str(ei.value)
    with pytest.raises(akm.AkmError):
        akm.MhdPack(I.uniform_mesh((1, 1, 1), (8, 8, 8), 2), G53)        # ng < 3


def _assemble8(mesh, U):
    """Active cells of every block -> global (8, N3, N2, N1) on the device; a face field sits on the lower face of its cell, so the
    periodic global array holds every face exactly once."""
    g, nx = mesh.ng, mesh.nx
    G = torch.empty((8, mesh.nrb[2] * nx[2], mesh.nrb[1] * nx[1], mesh.nrb[0] * nx[0]), dtype=U.dtype, device=U.device)
    for m, (_, l1, l2, l3) in enumerate(mesh.blocks):
        G[:, l3 * nx[2]:(l3 + 1) * nx[2], l2 * nx[1]:(l2 + 1) * nx[1], l1 * nx[0]:(l1 + 1) * nx[0]] = U[m][:, g:-g, g:-g, g:-g]
    return G


def _dt_reference_mhd(G, gamma, dx, cfl):
    """cfl * min dx_d / (|v_d| + c_f,d) with torch ops on the assembled global state (not the library's kernels)."""
    rho, mom, E = G[0], G[1:4], G[4]
    B = torch.stack([0.5 * (G[5 + d] + torch.roll(G[5 + d], -1, dims=2 - d)) for d in range(3)])
    b2 = (B ** 2).sum(0)
    p = (gamma - 1.0) * (E - 0.5 * (mom ** 2).sum(0) / rho - 0.5 * b2)
    gp = gamma * p
    best = math.inf
    for d in range(3):
        disc = torch.clamp((gp + b2) ** 2 - 4.0 * gp * B[d] ** 2, min=0.0)
        cf = torch.sqrt((gp + b2 + torch.sqrt(disc)) / (2.0 * rho))
        best = min(best, float((dx[d] / (mom[d].abs() / rho + cf)).min()))
    return cfl * best


def test_mhd_256_full_size_sampled(om, akm):
    """The workload bench.py times (`--workload mhd_256`: 8 MeshBlocks of 128^3, default arithmetic, the same launches): TWO steps on
    the GPU, checked on sampled 64^3 sub-boxes that the oracle advances one by one as small periodic blocks with the same dx and dt
    sequence.  One stage reaches at most 4 cells (PLM 2, cell-centred field 1, corner EMFs 1), two steps 16: the sub-box interior
    >= 20 cells from its faces is exact (24^3 cells and faces compared per box; boxes on the corner where the 8 blocks meet, on the
    periodic wrap, inside a block).  Plus what holds at any size: div B, totals, no floors, each dt against torch on the global state."""
    mesh, prim, A, B0 = I.mhd_workload("mhd_256")
    dev = torch.device("cuda", 0)
    U0 = I.make_state_mhd(mesh, prim, A, B0, device=dev)
    pg = akm.MhdPack(mesh, I.GAMMA, device=dev)
    pg.load(U0)
    G0 = _assemble8(mesh, U0)
    del U0
    nsteps, n, pad = 2, 64, 20
    origins = [(96, 96, 96), (224, 224, 224), (30, 140, 200), (150, 10, 70)]
    idx = lambda G, o: [(torch.arange(n, device=G.device) + o[d]) % G.shape[3 - d] for d in range(3)]
    sub = lambda G, o: G.index_select(1, idx(G, o)[2]).index_select(2, idx(G, o)[1]).index_select(3, idx(G, o)[0]).cpu().numpy()
    subs0 = [sub(G0, o) for o in origins]
    tot0 = G0.sum(dim=(1, 2, 3)).cpu().numpy()
    abs0 = G0.abs().sum(dim=(1, 2, 3)).cpu().numpy()
    dx = mesh.dx(0)
    dt_ref = _dt_reference_mhd(G0, I.GAMMA, dx, I.CFL)
    del G0
    dts = []
    for step in range(nsteps):
        dt = pg.new_dt(I.CFL)
        assert abs(dt - dt_ref) <= 1e-13 * dt_ref, (step, dt, dt_ref)
        pg.step(I.CFL, dt)
        dts.append(dt)
        G1 = _assemble8(mesh, pg.current())
        dt_ref = _dt_reference_mhd(G1, I.GAMMA, dx, I.CFL)
    assert pg.floor_count() == 0
    tot1 = G1.sum(dim=(1, 2, 3)).cpu().numpy()
    assert (np.abs(tot1 - tot0) / (abs0 + 1.0)).max() <= 1e-12                # mass, momentum, energy, mean field
    div = sum((torch.roll(G1[5 + d], -1, dims=2 - d) - G1[5 + d]) / dx[d] for d in range(3))
    assert float(div.abs().max()) <= 1e-11                                   # (|B| / dx ~ 250: a few ulp of that)
    sub_mesh = I.Mesh((1, 1, 1), (n, n, n), 3, [(0, 0, 0, 0)], xmax=(n * dx[0], n * dx[1], n * dx[2]))
    assert sub_mesh.dx(0) == dx
    worst = 0.0
    for o, s0 in zip(origins, subs0):
        po = om.OrcMhdPack(sub_mesh, I.GAMMA, threads=P.NTHREADS)
        u = np.zeros(sub_mesh.state_shape()[:1] + (8,) + sub_mesh.state_shape()[2:])
        u[0][:, 3:-3, 3:-3, 3:-3] = s0
        po.load(u)
        for dt in dts:
            po.step(I.CFL, dt)
        ref = po.current()[0][:, 3 + pad:-3 - pad, 3 + pad:-3 - pad, 3 + pad:-3 - pad]
        got = sub(G1, o)[:, pad:-pad, pad:-pad, pad:-pad]
        e = q_mhd(got[None], ref[None], I.GAMMA)
        worst = max(worst, e)
        assert e <= 2 * nsteps * TOL_STAGE, (o, e)
        po.close()
    P.report(f"[parity] MHD mhd_256 full size (8 x 128^3, bench launch configuration): worst sampled difference after {nsteps} steps = {worst:.2e}")


def _gpu_wave_error(akm, family, N, recon, nstages, amp=1e-6):
    """L1 error of a 1-D linear MHD wave after one period on the CUDA path alone (the eigenvector comes from numpy, the reference is
    the initial state): a property of the scheme that needs no oracle."""
    from tests.test_oracle_mhd import mhd_eigenmode
    speed, R, (r0, p0, bx, by0, bz0) = mhd_eigenmode(family)
    mesh = I.uniform_mesh((1, 1, 1), (N, 4, 4), 4)
    k = 2 * math.pi

    def prim(X1, X2, X3):
        s = torch.sin(k * X1) + 0 * X2 + 0 * X3
        return (r0 + amp * R[0] * s, amp * R[1] * s, amp * R[2] * s, amp * R[3] * s, p0 + amp * R[4] * s)

    def A(X1, X2, X3):
        c = torch.cos(k * X1) / k + 0 * X2 + 0 * X3
        return (0 * c, -amp * R[6] * c, amp * R[5] * c)

    U0 = I.make_state_mhd(mesh, prim, A, (bx, by0, bz0))
    pg = akm.MhdPack(mesh, G53, recon=recon, nstages=nstages)
    pg.load(U0)
    t, tend = 0.0, 1.0 / speed
    while t < tend:
        dt = min(pg.new_dt(0.3), tend - t)
        pg.step(0.3, dt)
        t += dt
    a = act(mesh)
    U = pg.current().cpu().numpy()
    assert pg.floor_count() == 0
    return math.sqrt(sum(np.abs(U[a][0, n] - U0.numpy()[a][0, n]).mean() ** 2 for n in range(8)))


def test_the_papers_mhd_convergence_orders_on_the_gpu(akm):
    """P:152 on the CUDA path itself (default arithmetic): RK3 + WENOZ and RK3 + PPMX converge at fourth order on the Alfven and slow
    waves, the fast wave at second order; PLM + RK2 at second order."""
    for family in ("alfven", "slow"):
        for recon in (3, 2):
            e16, e32 = (_gpu_wave_error(akm, family, N, recon, 3) for N in (16, 32))
            assert math.log2(e16 / e32) >= 3.5, (family, recon, e16, e32)
    f16, f32 = (_gpu_wave_error(akm, "fast", N, 3, 3) for N in (16, 32))
    assert 1.7 <= math.log2(f16 / f32) <= 3.0, (f16, f32)
    p32, p64 = (_gpu_wave_error(akm, "alfven", N, 0, 2) for N in (32, 64))
    assert 1.6 <= math.log2(p32 / p64) <= 2.4, (p32, p64)
    P.report(f"[property] MHD linear waves on the GPU: WENOZ + RK3 fast-wave rate {math.log2(f16 / f32):.2f}, PLM + RK2 Alfven rate {math.log2(p32 / p64):.2f}; "
             f"Alfven / slow with WENOZ / PPMX + RK3 >= 3.5")


@pytest.mark.parametrize("recon,ng", [(0, 3), (3, 4)])
def test_block_decomposition_does_not_change_the_result_on_the_gpu(akm, recon, ng):
    """The same periodic problem cut into 1, 4 and 12 MeshBlocks gives bit-identical global states on the CUDA path (default
    arithmetic): every face and corner is computed from the same numbers in the same order whichever block owns it."""
    from tests.test_oracle_mhd import assemble
    outs = []
    for nrb, nx in (((1, 1, 1), (16, 12, 8)), ((2, 2, 1), (8, 6, 8)), ((2, 3, 2), (8, 4, 4))):
        mesh = I.uniform_mesh(nrb, nx, ng)
        U0 = turbulent_state(mesh, shift=(0.0137, 0.0291, 0.0173))
        pg = akm.MhdPack(mesh, G53, recon=recon)
        pg.load(U0)
        for _ in range(3):
            pg.step(0.3, 2e-3)
        outs.append(assemble(mesh, pg.current().cpu().numpy()))
        assert pg.floor_count() == 0
    assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])
