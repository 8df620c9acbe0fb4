"""GPU parity tests proper (-m gpu): the CUDA path, called through the C-ABI binding, against the
oracle on the same seeded inputs.  Tolerances are BASELINE.json's: Q14 metric <= 1e-12 after one
stage, <= 1e-9 after the config's steps, conserved totals within 1e-12, ghost fill bit-exact."""
import numpy as np
import pytest
import torch

from paper_2409_16053_b200 import inputs as I
from tests import parity as P

pytestmark = pytest.mark.gpu

TOL_STAGE, TOL_RUN, TOL_TOTALS = 1e-12, 1e-9, 1e-12


@pytest.fixture(scope="module")
def ak():
    from paper_2409_16053_b200 import ak as _ak
    _ak.lib()
    assert torch.cuda.is_available()
    return _ak


def run_lockstep(orc, ak, w, nsteps, variant=0, check_ghosts=True, rsolver=0):
    """Oracle computes dt; both sides take it.  Returns per-step Q14 and the two final states."""
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0, variant, rsolver)
    a = P.active(w.mesh)
    errs = []
    for step in range(nsteps):
        dt = po.new_dt(w.cfl)
        dt_g = pg.new_dt(w.cfl)
        assert abs(dt_g - dt) <= 4 * np.spacing(dt), (step, dt, dt_g)
        for stage in (1, 2):
            po.fill_ghosts()
            pg.fill_ghosts()
            if check_ghosts and step == 0:
                # ghosts of identical active data must be bit-identical; after the first stage the active
                # data differ by rounding, so compare the oracle's fill of the GPU's active cells instead
                ug = P.gpu_state(pg)
                chk = orc.OrcPack(w.mesh, w.gamma, w.recon, threads=P.NTHREADS)
                chk.load(ug)
                chk.fill_ghosts()
                assert np.array_equal(chk.current(), ug), f"ghost fill differs at step {step} stage {stage}"
                chk.close()
            po.hydro_stage(stage, dt)
            pg.hydro_stage(stage, dt)
            if step == 0:
                e = P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma)
                assert e <= TOL_STAGE * stage, f"stage {stage}: Q14 = {e:.3e}"
        errs.append(P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma))
    assert po.floor_count() == 0 and pg.floor_count() == 0
    # one line per parity run in the test log (pytest -s / the driver's captured tail): how far inside the bars
    P.report(f"[parity] {w.name} nmb={w.mesh.nmb} nx={tuple(w.mesh.nx)} recon={w.recon} rsolver={rsolver} variant={variant} "
          f"steps={nsteps}: worst Q14 per step {max(errs):.3e} (bar {TOL_RUN:.0e}), first step {errs[0]:.3e}")
    return errs, po, pg, U0


def check_totals(w, U0, po, pg):
    t0 = P.totals(w.mesh, U0.numpy())
    tg = P.totals(w.mesh, P.gpu_state(pg))
    to = P.totals(w.mesh, po.current())
    norm = P.momentum_norm(w.mesh, U0.numpy(), w.gamma)
    scale = np.array([t0[0], norm, norm, norm, t0[4]])
    assert (np.abs(tg - to) / scale).max() <= TOL_TOTALS
    return np.abs(tg - t0) / scale


# ------------------------------------------------------------------------------- config 0 --------
@pytest.mark.parametrize("variant", [0, 1])
def test_config0_sound_wave_every_cell(orc, ak, variant):
    w = I.config0()
    errs, po, pg, U0 = run_lockstep(orc, ak, w, w.nsteps, variant)
    assert max(errs) <= TOL_RUN, errs
    po.fill_ghosts()
    pg.fill_ghosts()
    full = (slice(None),) * 5
    assert P.q14(P.gpu_state(pg)[full], po.current()[full], w.gamma) <= TOL_RUN      # every cell, ghosts included
    drift = check_totals(w, U0, po, pg)
    assert drift.max() <= 1e-13


def test_config0_literal_reading_constant_pressure(orc, ak):
    w = I.config0(literal=True)
    errs, *_ = run_lockstep(orc, ak, w, 3)
    assert max(errs) <= TOL_RUN


# ------------------------------------------------------------------------------- config 1 --------
def test_config1_random_modes_20_steps(orc, ak):
    w = I.config1()
    errs, po, pg, U0 = run_lockstep(orc, ak, w, w.nsteps)
    assert max(errs) <= TOL_RUN, errs
    drift = check_totals(w, U0, po, pg)
    assert drift.max() <= 1e-12           # periodic single-level mesh: conservation to round-off


def test_config1_free_running_dt(orc, ak):
    w = I.config1(nrb=2)                  # 8 x 32^3
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0)
    for _ in range(10):
        po.step(w.cfl)
        pg.step(w.cfl)
    a = P.active(w.mesh)
    assert P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma) <= TOL_RUN


# ------------------------------------------------------------------------------- config 2 --------
def test_config2_sedov_32cubed_blocks(orc, ak):
    w = I.config2(nx=32, n=128)           # 64 x 32^3 crop of the 256^3 mesh, same dx-independent recipe
    errs, po, pg, U0 = run_lockstep(orc, ak, w, w.nsteps)
    assert max(errs) <= TOL_RUN, errs
    check_totals(w, U0, po, pg)


def test_config2_block_size_sweep_is_decomposition_invariant_on_gpu(ak):
    """Same 64^3 Sedov field cut into 16^3 / 32^3 / 64^3 blocks: active cells are bit-identical on the GPU as
    they are in the oracle (ghosts are exact copies, per-cell arithmetic does not know the block, and tile-edge
    faces use one instruction sequence: the stage kernels are compiled with -fmad=false)."""
    res = []
    for nx in (16, 32, 64):
        w = I.config2(nx=nx, n=64)
        w.prim_fn = I.sedov_prim(r0=0.2)
        pg = ak.Pack(w.mesh, w.gamma, w.recon)
        pg.load(w.state())
        for _ in range(5):
            pg.step(w.cfl)
        U = P.gpu_state(pg)
        ng = w.mesh.ng
        glob = np.zeros((5, 64, 64, 64))
        for m, (_, l1, l2, l3) in enumerate(w.mesh.blocks):
            glob[:, l3 * nx:(l3 + 1) * nx, l2 * nx:(l2 + 1) * nx, l1 * nx:(l1 + 1) * nx] = U[m][:, ng:-ng, ng:-ng, ng:-ng]
        res.append(glob)
    for r in res[1:]:
        assert np.array_equal(r, res[0])


# ------------------------------------------------------------------------------- config 3 --------
def test_config3_ppm_reduced_size(orc, ak):
    w = I.config3(nrb=2, nx=32)           # 8 x 32^3, PPM4, ng=3, Mach-1 modes + double shear layer
    errs, po, pg, U0 = run_lockstep(orc, ak, w, w.nsteps)
    assert max(errs) <= TOL_RUN, errs
    check_totals(w, U0, po, pg)


@pytest.mark.parametrize("variant", [0, 1])
def test_config3_ppm_noncubic_blocks(orc, ak, variant):
    w = I.config3(nrb=2, nx=32)
    w.mesh = I.uniform_mesh((2, 1, 3), (24, 40, 6), 3)
    errs, *_ = run_lockstep(orc, ak, w, 3, variant)
    assert max(errs) <= TOL_RUN, errs


# ------------------------------------------------------------------------------- config 4 --------
def test_config4_smr_sedov_20_steps(orc, ak):
    w = I.config4()
    errs, po, pg, U0 = run_lockstep(orc, ak, w, w.nsteps)
    assert max(errs) <= TOL_RUN, errs
    check_totals(w, U0, po, pg)


def test_smr_with_structure_on_level_boundaries(orc, ak):
    """SURVEY finding 3: config 4 never puts non-uniform data on a level boundary; this input does."""
    w = I.smr_parity()
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0)
    a = P.active(w.mesh)
    for step in range(w.nsteps):
        dt = po.new_dt(w.cfl)
        for stage in (1, 2):
            po.fill_ghosts()
            pg.fill_ghosts()
            ug = P.gpu_state(pg)
            chk = orc.OrcPack(w.mesh, w.gamma, w.recon, threads=P.NTHREADS)
            chk.load(ug)
            chk.fill_ghosts()
            assert np.array_equal(chk.current(), ug)          # restriction + prolongation bit-exact
            chk.close()
            po.hydro_stage(stage, dt)
            pg.hydro_stage(stage, dt)
        assert P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma) <= TOL_RUN


# ------------------------------------------------------------------------------- edge cases ------
@pytest.mark.parametrize("nrb,nx,ng,recon", [
    ((1, 1, 1), (2, 2, 2), 2, I.RECON_PLM),        # smallest legal block, self-periodic
    ((1, 1, 1), (4, 4, 4), 3, I.RECON_PPM4),
    ((1, 2, 1), (6, 2, 4), 2, I.RECON_PLM),
    ((3, 1, 2), (34, 10, 6), 2, I.RECON_PLM),      # ragged: not a multiple of any tile size
    ((1, 1, 1), (130, 18, 10), 3, I.RECON_PPM4),   # longer than one 128-wide tile row
    ((1, 1, 1), (16, 16, 16), 4, I.RECON_PPM4),    # more ghosts than the stencil needs (odd surplus: LDG-staged kernel)
    ((1, 1, 2), (16, 12, 8), 4, I.RECON_PLM),      # more ghosts than the stencil needs (even surplus: TMA-staged kernel)
])
@pytest.mark.parametrize("variant", [0, 1])
def test_ragged_and_degenerate_blocks(orc, ak, nrb, nx, ng, recon, variant):
    mesh = I.uniform_mesh(nrb, nx, ng)
    w = I.Workload("edge", mesh, recon, 2, I.modes_prim(0.5, shear=False, rho_pert=True))
    errs, *_ = run_lockstep(orc, ak, w, 2, variant)
    assert max(errs) <= TOL_RUN, errs


def test_uniform_state_preserved_bit_exactly_on_gpu(ak):
    mesh = I.uniform_mesh((2, 2, 1), (16, 8, 8), 2)
    prim = lambda X1, X2, X3: (1.3 + 0 * X1, 0.4 + 0 * X1, -0.7 + 0 * X1, 0.2 + 0 * X1, 0.9 + 0 * X1)
    for recon, mesh_ in ((I.RECON_PLM, mesh), (I.RECON_PPM4, I.uniform_mesh((2, 2, 1), (16, 8, 8), 3))):
        U0 = I.make_state(mesh_, prim)
        pg = ak.Pack(mesh_, I.GAMMA, recon)
        pg.load(U0)
        pg.step(0.3)
        a = P.active(mesh_)
        assert np.array_equal(P.gpu_state(pg)[a], U0.numpy()[a])


def test_dt_reduction_bit_exact(orc, ak):
    for w in (I.config1(nrb=2), I.smr_parity(nx=8), I.config3(nrb=1, nx=32)):
        U0 = w.state()
        po, pg = P.make_pair(orc, ak, w, U0)
        assert pg.new_dt(w.cfl) == po.new_dt(w.cfl)


def test_call_order_and_argument_errors(ak):
    w = I.config0()
    pg = ak.Pack(w.mesh, w.gamma, w.recon)
    pg.set_ghost_push(False)                         # (with the fused fill a stage leaves the ghost cells current)
    pg.load(w.state())
    with pytest.raises(ak.AkError):
        pg.hydro_stage(1, 1e-3)                      # ghosts not filled
    pg.fill_ghosts()
    with pytest.raises(ak.AkError):
        pg.hydro_stage(2, 1e-3)                      # stage 2 before stage 1
    with pytest.raises(ak.AkError):
        pg.hydro_stage(1, -1.0)
    pg.hydro_stage(1, 1e-3)
    with pytest.raises(ak.AkError):
        pg.hydro_stage(2, 1e-3)                      # ghosts stale again
    pg.fill_ghosts()
    pg.hydro_stage(2, 1e-3)
    assert pg.launch_count() >= 4


def test_upload_download_round_trip_through_c_abi(ak):
    w = I.config1(nrb=1)
    U0 = w.state()
    pg = ak.Pack(w.mesh, w.gamma, w.recon)
    host = U0.clone().pin_memory()
    pg.upload(host)
    out = torch.empty_like(host).pin_memory()
    pg.download(out)
    assert torch.equal(out, U0)


# ------------------------------------------------------------------- tiling / kernel generations --------
@pytest.mark.gpu
@pytest.mark.parametrize("recon", [0, 1])
def test_tile_shapes_give_bit_identical_results(ak, recon):
    """include/ak.h, ak_pack_set_tile: tile-edge faces are solved by both tiles sharing them with the same
    instruction sequence, so the result must not depend on the tile shape -- bit for bit, ragged tiles
    included (24 x 40 x 6 blocks: 24 = 16 + 8, 40 = 10 x 4 = 8 x 5 = 22 + 18 = 11 x 3 + 7)."""
    w = I.config3(nrb=2, nx=32) if recon else I.config1(nrb=2, nx=32)
    w.mesh = I.uniform_mesh((2, 1, 3), (24, 40, 6), 3 if recon else 2)
    ref = None
    for tile in (-1, 0, 1, 2, 3):
        pg = ak.Pack(w.mesh, w.gamma, w.recon)
        pg.set_tile(tile)
        pg.load(w.state())
        for _ in range(3):
            pg.step(w.cfl)
        U = P.gpu_state(pg)[P.active(w.mesh)]
        assert pg.floor_count() == 0
        if ref is None:
            ref = U
        else:
            assert np.array_equal(U, ref), f"tile {tile} differs from the automatic choice"


@pytest.mark.gpu
@pytest.mark.parametrize("variant", [2])
def test_ldg_staged_fallback_kernel_matches_the_oracle(orc, ak, variant):
    """Variant 2 (include/ak.h) is the kernel taken automatically when the TMA box origin would be misaligned."""
    for w in (I.config3(nrb=2, nx=32), I.config1(nrb=2, nx=32)):
        errs, *_ = run_lockstep(orc, ak, w, 2, variant, check_ghosts=False)
        assert max(errs) <= TOL_RUN, (variant, w.name, errs)


# ------------------------------------------------------- config 3 at full size, bench launch configuration --------
def _assemble(mesh, U):
    """(nmb, 5, nt3, nt2, nt1) block state -> (5, N3, N2, N1) global array of active cells (uniform mesh), on U's device."""
    g, nx = mesh.ng, mesh.nx
    G = torch.empty((5, mesh.nrb[2] * nx[2], mesh.nrb[1] * nx[1], mesh.nrb[0] * nx[0]), dtype=U.dtype, device=U.device)
    for m, (_, l1, l2, l3) in enumerate(mesh.blocks):
        G[:, l3 * nx[2]:(l3 + 1) * nx[2], l2 * nx[1]:(l2 + 1) * nx[1], l1 * nx[0]:(l1 + 1) * nx[0]] = \
            U[m][:, g:-g, g:-g, g:-g]
    return G


def _subbox(G, origin, n):
    """n^3 periodic sub-box of the global array with lower corner `origin` = (o1, o2, o3) -> host numpy (5, n, n, n)."""
    idx = [(torch.arange(n, device=G.device) + o) % G.shape[3 - d] for d, o in enumerate(origin)]
    return G.index_select(1, idx[2]).index_select(2, idx[1]).index_select(3, idx[0]).cpu().numpy()


def _dt_reference(G, gamma, dx, cfl):
    """Eq.(3) on the assembled global state with torch ops on the device (not the library's kernels)."""
    rho, mom, E = G[0], G[1:4], G[4]
    p = (gamma - 1.0) * (E - 0.5 * (mom ** 2).sum(0) / rho)
    cs = torch.sqrt(gamma * p / rho)
    return cfl * min(float((dx[d] / (mom[d].abs() / rho + cs)).min()) for d in range(3))


def test_config3_full_size_sampled(orc, ak):
    """BASELINE config 3 at its full size (64 MeshBlocks of 128^3, the launch configuration bench.py times: 16 x 10
    tiles, one k-chunk, the dt of steps 2 and 3 taken from the reduction fused into stage 2 of the step before):
    THREE RK2 steps on the GPU, checked on sampled 64^3 sub-boxes that the oracle advances one by one.  A cell's RK2
    update depends on cells within 2 x 3 of it (two PPM4 stages), so the oracle, run on a sub-box as its own small
    periodic block with the same dx and the same dt sequence, is exact on the cells >= 18 away from the sub-box
    faces after three steps (pad 20 -> 24^3 cells compared per box).  The boxes sit on a corner where 8 blocks
    meet, on the periodic wrap of the domain, on the shear layers and inside a block (every box spans several
    tiles).  Plus what holds at any size: conservation, no floors, and each step's dt against Eq.(3) evaluated with
    torch on the assembled state."""
    w = I.config3()
    dev = torch.device("cuda", 0)
    pg = ak.Pack(w.mesh, w.gamma, w.recon, device=dev)
    U0 = w.state(device=dev)
    pg.load(U0)
    G0 = _assemble(w.mesh, U0)
    del U0
    nsteps, n, pad = 3, 64, 20
    origins = [(96, 96, 96), (480, 480, 480), (300, 96, 200), (40, 352, 500), (200, 50, 60), (240, 250, 260)]
    subs0 = [_subbox(G0, o, n) for o in origins]
    tot0 = G0.sum(dim=(1, 2, 3)).cpu().numpy()
    rho, mom, E = G0[0], G0[1:4], G0[4]
    p = (w.gamma - 1.0) * (E - 0.5 * (mom ** 2).sum(0) / rho)
    mnorm = float((mom.norm(dim=0) + rho * torch.sqrt(w.gamma * p / rho)).sum())
    dx = w.mesh.dx(0)
    dt_ref = _dt_reference(G0, w.gamma, dx, w.cfl)
    del G0, rho, mom, E, p
    dts = []
    for step in range(nsteps):
        dt = pg.new_dt(w.cfl)                    # step 0: stand-alone reduction; later: from stage 2 of the step before
        assert abs(dt - dt_ref) <= 1e-13 * dt_ref, (step, dt, dt_ref)
        pg.step(w.cfl, dt)
        dts.append(dt)
        G1 = _assemble(w.mesh, pg.current())
        dt_ref = _dt_reference(G1, w.gamma, dx, w.cfl)
        if step + 1 < nsteps:
            del G1
    assert pg.floor_count() == 0
    tot1 = G1.sum(dim=(1, 2, 3)).cpu().numpy()
    scale = np.array([tot0[0], mnorm, mnorm, mnorm, tot0[4]])
    assert (np.abs(tot1 - tot0) / scale).max() <= TOL_TOTALS
    sub_mesh = I.Mesh((1, 1, 1), (n, n, n), w.mesh.ng, [(0, 0, 0, 0)], xmax=(n * dx[0], n * dx[1], n * dx[2]))
    assert sub_mesh.dx(0) == dx
    g = w.mesh.ng
    worst = 0.0
    for o, s0 in zip(origins, subs0):
        po = orc.OrcPack(sub_mesh, w.gamma, w.recon, threads=P.NTHREADS)
        u = np.zeros(sub_mesh.state_shape())
        u[0][:, g:-g, g:-g, g:-g] = s0
        po.load(u)
        for dt in dts:
            po.step(w.cfl, dt)
        ref = po.current()[0][:, g + pad:-g - pad, g + pad:-g - pad, g + pad:-g - pad]
        got = _subbox(G1, o, n)[:, pad:-pad, pad:-pad, pad:-pad]
        e = P.q14(got[None], ref[None], w.gamma)
        worst = max(worst, e)
        assert e <= 2 * nsteps * TOL_STAGE, (o, e)
        po.close()
    P.report(f"[parity] cfg3 full size (64 x 128^3, bench launch configuration): worst sampled Q14 after {nsteps} RK2 steps = {worst:.2e}")


# ------------------------------------------------------------ flux correction --------
def test_flux_correction_matches_oracle_and_conserves_on_gpu(orc, ak):
    """Config-4 mesh carrying the config-1 field (structure on the level boundaries), flux correction on both
    sides: Q14 against the oracle within the stage / run tolerances, and the GPU's own totals constant to
    round-off (they drift at 1e-6 without the correction: tests/test_oracle_fluxcorr.py)."""
    w = I.smr_parity()
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0)
    po.set_flux_correction(True)
    pg.set_flux_correction(True)
    a = P.active(w.mesh)
    errs = []
    for step in range(w.nsteps):
        dt = po.new_dt(w.cfl)
        assert pg.new_dt(w.cfl) == dt or step > 0
        for stage in (1, 2):
            po.fill_ghosts(); pg.fill_ghosts()
            po.hydro_stage(stage, dt); pg.hydro_stage(stage, dt)
            if step == 0:
                e = P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma)
                assert e <= TOL_STAGE * stage, f"stage {stage}: Q14 = {e:.3e}"
        errs.append(P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma))
    assert max(errs) <= TOL_RUN, errs
    assert po.floor_count() == 0 and pg.floor_count() == 0
    drift = check_totals(w, U0, po, pg)          # GPU totals vs oracle totals <= 1e-12 ...
    assert drift.max() <= 1e-13, drift           # ... and vs the initial totals: conservative across levels


def test_flux_correction_off_drifts_and_on_is_inert_on_uniform_mesh(ak):
    w = I.smr_parity(nx=16)
    U0 = w.state()
    pg = ak.Pack(w.mesh, w.gamma, w.recon)
    pg.load(U0)
    for _ in range(4):
        pg.step(w.cfl)
    t0, t1 = P.totals(w.mesh, U0.numpy()), P.totals(w.mesh, P.gpu_state(pg))
    assert abs(t1[0] - t0[0]) / t0[0] >= 1e-9    # without the correction mass is visibly not conserved on this input
    wu = I.config1(nrb=2, nx=16)
    res = []
    for on in (False, True):
        pu = ak.Pack(wu.mesh, wu.gamma, wu.recon)
        pu.set_flux_correction(on)
        pu.load(wu.state())
        l0 = pu.launch_count()
        for _ in range(2):
            pu.step(wu.cfl)
        # step 1: dt_init + new_dt + fill + 2 stages (stage 1 writes the ghost copies itself, so the second fill has
        # nothing to do); step 2: the dt comes from stage 2 of step 1 and both fills are already done; no correction launches
        assert pu.launch_count() - l0 == 5 + 2
        res.append(P.gpu_state(pu))
    assert np.array_equal(res[0], res[1])


def test_flux_correction_keeps_uniform_state_bit_exact_on_gpu(ak):
    mesh = I.smr_mesh((2, 2, 2), (8, 8, 8), 2, (0, 0, 0), (1, 1, 1))
    prim = lambda X1, X2, X3: (1.3 + 0 * X1, 0.4 + 0 * X1, -0.7 + 0 * X1, 0.2 + 0 * X1, 0.9 + 0 * X1)
    U0 = I.make_state(mesh, prim)
    pg = ak.Pack(mesh, I.GAMMA, I.RECON_PLM)
    pg.set_flux_correction(True)
    pg.load(U0)
    for _ in range(2):
        pg.step(0.3)
    a = P.active(mesh)
    assert np.array_equal(P.gpu_state(pg)[a], U0.numpy()[a])


# ------------------------------------------------------------ LLF / HLLE --------
@pytest.mark.parametrize("rsolver", [1, 2, 3])
def test_llf_and_hlle_match_the_oracle(orc, ak, rsolver):
    """Same kernel skeleton, other two-state solver: PLM on the config-1 recipe and on ragged blocks, PPM4 on the
    config-3 recipe, the SMR mesh with structure on the level boundaries and flux correction on."""
    for w in (I.config1(nrb=2, nx=32), I.config3(nrb=2, nx=32)):
        errs, po, pg, U0 = run_lockstep(orc, ak, w, 4, rsolver=rsolver)
        assert max(errs) <= TOL_RUN, (rsolver, w.name, errs)
        check_totals(w, U0, po, pg)
    w = I.config1(nrb=2, nx=32)
    w.mesh = I.uniform_mesh((2, 1, 3), (24, 40, 6), 2)
    errs, *_ = run_lockstep(orc, ak, w, 2, rsolver=rsolver)
    assert max(errs) <= TOL_RUN, errs
    w = I.smr_parity(nx=16)
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0, rsolver=rsolver)
    po.set_flux_correction(True); pg.set_flux_correction(True)
    for _ in range(3):
        dt = po.new_dt(w.cfl)
        po.step(w.cfl, dt); pg.step(w.cfl, dt)
    assert P.q14(P.gpu_state(pg)[P.active(w.mesh)], po.current()[P.active(w.mesh)], w.gamma) <= TOL_RUN
    assert check_totals(w, U0, po, pg).max() <= 1e-13


def test_llf_hlle_only_in_the_production_kernel(ak):
    w = I.config1(nrb=1, nx=16)
    pg = ak.Pack(w.mesh, w.gamma, w.recon, rsolver=1, variant=1)
    pg.load(w.state())
    pg.fill_ghosts()
    with pytest.raises(ak.AkError):
        pg.hydro_stage(1, 1e-3)


# ------------------------------------------------------------ in place of compute-sanitizer (closed on this pool) --------
@pytest.mark.parametrize("which", ["cfg3", "cfg1_ragged"])
def test_every_cell_is_written_and_runs_repeat_bit_identically(ak, which):
    """initcheck / racecheck stand-ins (profiles/r02_sanitizer.md): the output buffer of stage 1 and the ghost cells of
    buffer A before stage 2 are poisoned with NaN -- afterwards every active AND ghost cell must be finite, i.e. written
    by the stage kernel (fused fill) --, and two independent runs from the same input agree bit for bit, dt included
    (a shared-memory or in-place race on the TMA ring would show up as run-to-run noise)."""
    if which == "cfg3":
        w = I.config3(nrb=2, nx=32)
    else:
        w = I.config1(nrb=2, nx=32)
        w.mesh = I.uniform_mesh((2, 1, 3), (24, 40, 6), 2)
    U0 = w.state()
    g = w.mesh.ng
    finals = []
    for rep in range(2):
        pg = ak.Pack(w.mesh, w.gamma, w.recon)
        pg.load(U0)
        dts = []
        for step in range(3):
            dt = pg.new_dt(w.cfl)
            dts.append(dt)
            pg.fill_ghosts()
            pg.ub.fill_(float("nan"))                                    # stage 1 writes B
            pg.hydro_stage(1, dt)
            assert bool(torch.isfinite(pg.ub).all()), (rep, step, "stage 1 left cells of B unwritten")
            pg.fill_ghosts()
            poison = torch.full_like(pg.ua, float("nan"))
            poison[:, :, g:-g, g:-g, g:-g] = pg.ua[:, :, g:-g, g:-g, g:-g]
            pg.ua.copy_(poison)                                          # ghost cells of A only
            pg.hydro_stage(2, dt)
            assert bool(torch.isfinite(pg.ua).all()), (rep, step, "stage 2 left ghost cells of A unwritten")
        finals.append((P.gpu_state(pg), dts))
    assert finals[0][1] == finals[1][1]
    assert np.array_equal(finals[0][0], finals[1][0])


# ------------------------------------------------------------ ghost fill fused into the stage --------
@pytest.mark.parametrize("nrb,nx,ng,recon", [
    ((2, 2, 2), (16, 16, 16), 2, 0), ((2, 2, 2), (16, 16, 16), 3, 1), ((1, 1, 1), (8, 8, 8), 2, 0), ((1, 1, 1), (4, 4, 4), 3, 1),
    ((3, 1, 2), (2, 2, 2), 2, 0), ((2, 3, 1), (4, 2, 6), 2, 0), ((2, 1, 3), (24, 40, 6), 3, 1), ((1, 2, 1), (34, 10, 6), 2, 0),
])
def test_fused_ghost_push_equals_the_separate_fill(orc, ak, nrb, nx, ng, recon):
    """Uniform periodic meshes: the stage kernel writes every boundary cell also into the neighbours' ghost cells.
    After each stage -- WITHOUT calling the fill kernel -- every ghost cell must equal the oracle's fill of the GPU's
    own active cells bit for bit (blocks smaller than 2 ng, where a cell is near both faces, a single self-periodic
    block and ragged tiles included), no fill is launched after the first one, and the results are bit-identical to a
    run with the push switched off."""
    w = I.config3(nrb=1, nx=16) if recon else I.config1(nrb=1, nx=16)
    w.mesh = I.uniform_mesh(nrb, nx, ng)
    U0 = w.state()
    pg = ak.Pack(w.mesh, w.gamma, recon)
    pr = ak.Pack(w.mesh, w.gamma, recon)
    pr.set_ghost_push(False)
    pg.load(U0); pr.load(U0)
    for step in range(3):
        dt = pr.new_dt(w.cfl)
        assert pg.new_dt(w.cfl) == dt
        for stage in (1, 2):
            l0 = pg.launch_count()
            pg.fill_ghosts(); pr.fill_ghosts()
            pushing = all(n >= 2 * ng for n in nx)       # (smaller blocks keep the separate fill pass)
            assert pg.launch_count() - l0 == (1 if (step == 0 and stage == 1) or not pushing else 0)
            pg.hydro_stage(stage, dt); pr.hydro_stage(stage, dt)
            if pushing:
                ug = P.gpu_state(pg)                         # ghosts as the stage left them
                chk = orc.OrcPack(w.mesh, w.gamma, recon)
                chk.load(ug); chk.fill_ghosts()
                assert np.array_equal(chk.current(), ug), (step, stage)
                chk.close()
    pr.fill_ghosts(); pg.fill_ghosts()
    assert np.array_equal(P.gpu_state(pg), P.gpu_state(pr))


# ------------------------------------------------------------ first-order flux correction --------
@pytest.mark.parametrize("recon,ng,nst", [(I.RECON_PLM, 2, 2), (I.RECON_PPM4, 3, 2), (I.RECON_WENOZ, 3, 2), (I.RECON_PPM4, 3, 3)])
def test_fofc_matches_the_oracle_and_keeps_the_state_positive(orc, ak, recon, ng, nst):
    """Receding Mach-10 streams (colliding across the periodic boundary), where the uncorrected scheme lives on its floors:
    with FOFC on both sides the floors never fire, the same cells are flagged, the state stays positive, and GPU and
    oracle agree within the run tolerance; 3-D blocks with the interface oblique to nothing but present in x2 too."""
    import math
    c = math.sqrt(I.GAMMA)
    prim = lambda X1, X2, X3: (1.0 + 0.1 * torch.sin(6.283185307179586 * X2), torch.where(X1 < 0.5, -10.0 * c, 10.0 * c) * torch.ones_like(X1),
                               torch.where(X2 < 0.5, -2.0 * c, 2.0 * c) * torch.ones_like(X1), 0 * X1, torch.ones_like(X1))
    mesh = I.uniform_mesh((2, 2, 1), (16, 12, 8), ng)
    U0 = I.make_state(mesh, prim)
    po = orc.OrcPack(mesh, I.GAMMA, recon, threads=P.NTHREADS)
    pg = ak.Pack(mesh, I.GAMMA, recon)
    po.load(U0.numpy()); pg.load(U0)
    if nst == 3:                                             # RK3 + PPM4 + HLLC + FOFC: a combination the paper showcases
        po.set_integrator(3); pg.set_integrator(3)
    po.set_fofc(True); pg.set_fofc(True)
    a = P.active(mesh)
    worst = 0.0
    for step in range(30):
        dt = po.new_dt(0.3)
        assert abs(pg.new_dt(0.3) - dt) <= 1e-9 * dt          # (near-vacuum cells set the time step here)
        po.step(0.3, dt); pg.step(0.3, dt)
        worst = max(worst, P.q14(P.gpu_state(pg)[a], po.current()[a], I.GAMMA))
    P.report(f"[parity] FOFC receding Mach-10 streams recon={recon} stages={nst}: worst Q14 {worst:.3e}, flagged cells {pg.fofc_count()} (oracle {po.fofc_count()})")
    assert worst <= TOL_RUN
    assert pg.fofc_count() == po.fofc_count() > 0
    assert pg.floor_count() == 0 and po.floor_count() == 0
    ug = P.gpu_state(pg)[a]
    assert ug[:, 0].min() > 0 and (ug[:, 4] - 0.5 * (ug[:, 1:4] ** 2).sum(1) / ug[:, 0]).min() > 0
    t0, t1 = P.totals(mesh, U0.numpy()), P.totals(mesh, P.gpu_state(pg))
    assert abs(t1[0] - t0[0]) <= 1e-12 * t0[0] and abs(t1[4] - t0[4]) <= 1e-12 * t0[4]


def test_fofc_is_inert_on_the_configs_and_refused_where_unsupported(orc, ak):
    for w in (I.config1(nrb=2, nx=16), I.config3(nrb=2, nx=16)):
        res = []
        for on in (False, True):
            pg = ak.Pack(w.mesh, w.gamma, w.recon)
            pg.set_fofc(on)
            pg.load(w.state())
            for _ in range(3):
                pg.step(w.cfl)
            assert pg.fofc_count() == 0
            pg.fill_ghosts()
            res.append(P.gpu_state(pg))
        assert np.array_equal(res[0], res[1]), w.name
    w = I.smr_parity(nx=8)
    pg = ak.Pack(w.mesh, w.gamma, w.recon)
    pg.set_fofc(True)
    pg.load(w.state())
    pg.fill_ghosts()
    with pytest.raises(ak.AkError):
        pg.hydro_stage(1, 1e-4)                             # refined mesh


# ------------------------------------------------------------ strong collisions / non-finite states ----
@pytest.mark.parametrize("recon,ng", [(0, 2), (1, 3)])
def test_supersonic_inflow_into_a_wall_matches_the_oracle(orc, ak, recon, ng):
    """Mach-5 stream running into a reflecting wall (the mirror state makes the face a symmetric head-on collision):
    finite, floor-free, within the bar of the oracle, and the wall carries no mass flux (mass is conserved)."""
    import dataclasses
    g = 5.0 / 3.0
    mesh = dataclasses.replace(I.uniform_mesh((2, 1, 1), (16, 8, 8), ng), bc=(1, 2, 0, 0, 0, 0))   # outflow left, wall right
    c = (g * 1.0 / 1.0) ** 0.5
    prim = lambda X1, X2, X3: (1.0 + 0.1 * torch.sin(6.283185307179586 * X2), 5.0 * c + 0 * X1, 0.2 + 0 * X1, 0 * X1, 1.0 + 0 * X1)
    U0 = I.make_state(mesh, prim, gamma=g)
    po = orc.OrcPack(mesh, g, recon, threads=P.NTHREADS)
    pg = ak.Pack(mesh, g, recon)
    po.load(U0.numpy()); pg.load(U0)
    a = P.active(mesh)
    worst = 0.0
    for _ in range(8):
        dt = po.new_dt(0.3)
        assert abs(pg.new_dt(0.3) - dt) <= 1e-13 * dt              # (states differ by rounding after the first step)
        po.step(0.3, dt); pg.step(0.3, dt)
        ug = P.gpu_state(pg)[a]
        assert np.all(np.isfinite(ug))
        worst = max(worst, P.q14(ug, po.current()[a], g))
    P.report(f"[parity] wall inflow Mach 5 recon={recon}: worst Q14 {worst:.3e}")
    assert worst <= TOL_RUN
    assert po.floor_count() == 0 and pg.floor_count() == 0
    assert po.current()[a][:, 0].max() > 2.0               # the reflected shock has formed (density jump towards 4)


def test_non_finite_state_is_reported_by_new_dt(orc, ak):
    """a NaN in one active cell must not be skipped by the max / min reductions -- both the stand-alone
    reduction and the one fused into the last stage return AK_ENONFINITE (-5), as the oracle reports it."""
    w = I.config1(nrb=2, nx=16)
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0)
    dt = pg.new_dt(w.cfl)
    assert dt == po.new_dt(w.cfl)
    ng = w.mesh.ng
    bad = U0.clone()
    bad[3, 2, ng + 5, ng + 7, ng + 1] = float("nan")        # one momentum component of one cell
    pg.load(bad); po.load(bad.numpy())
    with pytest.raises(orc.OrcError):
        po.new_dt(w.cfl)
    with pytest.raises(ak.AkError) as ei:
        pg.new_dt(w.cfl)                                    # stand-alone kernel
    assert "non-finite" in str(ei.value)
    pg.step(w.cfl, dt)                                      # the NaN spreads; stage 2 reduces the speeds of its result
    with pytest.raises(ak.AkError) as ei:
        pg.new_dt(w.cfl)                                    # fused path
    assert "non-finite" in str(ei.value)
    # a healthy state afterwards works again
    pg.load(U0)
    assert pg.new_dt(w.cfl) == dt


# ------------------------------------------------------------ outflow / reflecting boundaries --------
@pytest.mark.parametrize("bc", [(1, 1, 0, 0, 2, 2), (2, 2, 2, 2, 2, 2), (0, 0, 1, 1, 0, 0), (2, 1, 1, 2, 1, 1)])
@pytest.mark.parametrize("recon,ng", [(0, 2), (1, 3)])
def test_physical_boundaries_match_the_oracle(orc, ak, bc, recon, ng):
    """Ghost cells bit-exact after every fill (run_lockstep checks them at step 0 against the oracle's fill of the
    GPU's own active cells), states within the run tolerance."""
    import dataclasses
    # the Mach-0.3 field of config 1 and the Mach-1 field of config 3, where patches of the flow run into a wall at
    # Mach > 1.9: with the round-1 pressure-based HLLC speeds that gave 0/0 on both sides (Q26); with
    # Davis's speeds (Q2, round 2) the run is finite, floor-free and within the bar
    for w in (I.config1(nrb=2, nx=16), I.config3(nrb=2, nx=16)):
        w.recon = recon
        w.mesh = dataclasses.replace(I.uniform_mesh((2, 2, 1), (16, 12, 8), ng), bc=bc)
        errs, po, pg, U0 = run_lockstep(orc, ak, w, 3)
        assert max(errs) <= TOL_RUN, (bc, errs)
        assert np.all(np.isfinite(P.gpu_state(pg)[P.active(w.mesh)]))
    po.fill_ghosts(); pg.fill_ghosts()
    chk = orc.OrcPack(w.mesh, w.gamma, w.recon)
    chk.load(P.gpu_state(pg)); chk.fill_ghosts()
    assert np.array_equal(chk.current(), P.gpu_state(pg))


def test_standard_sod_tube_on_the_gpu(orc, ak):
    """The paper's shock-tube workload shape: non-periodic x1, outflow ends, against the oracle to t = 0.1."""
    import dataclasses
    N, g = 256, 1.4
    mesh = dataclasses.replace(I.uniform_mesh((4, 1, 1), (N // 4, 4, 4), 2), bc=(1, 1, 0, 0, 0, 0))

    def prim(X1, X2, X3):
        left = X1 < 0.5
        rho = torch.where(left, 1.0, 0.125).to(torch.float64)
        pr = torch.where(left, 1.0, 0.1).to(torch.float64)
        z = torch.zeros_like(rho)
        return (rho, z, z, z, pr)

    U0 = I.make_state(mesh, prim, gamma=g)
    po = orc.OrcPack(mesh, g, I.RECON_PLM, threads=P.NTHREADS)
    pg = ak.Pack(mesh, g, I.RECON_PLM)
    po.load(U0.numpy()); pg.load(U0)
    t = 0.0
    while t < 0.1:
        dt = min(po.new_dt(0.3), 0.1 - t)
        po.step(0.3, dt); pg.step(0.3, dt)
        t += dt
    a = P.active(mesh)
    assert P.q14(P.gpu_state(pg)[a], po.current()[a], g) <= TOL_RUN
    assert pg.floor_count() == 0


@pytest.mark.parametrize("recon,nst", [(I.RECON_PLM, 2), (I.RECON_WENOZ, 3)])
def test_shu_osher_tube_on_the_gpu(orc, ak, recon, nst):
    """The paper's second shock-tube workload (Fig. 1 right): 200 cells, Mach-3 shock into a sinusoidal density,
    outflow ends, t = 0.047, with PLM + SSPRK(2,2) and with the showcased WENOZ + SSPRK(3,3): GPU against the oracle."""
    g = I.SHU_OSHER_GAMMA
    mesh = I.shu_osher_mesh(200, 3, nblocks=4)
    U0 = I.make_state(mesh, I.shu_osher_prim(), gamma=g)
    po = orc.OrcPack(mesh, g, recon, threads=P.NTHREADS)
    pg = ak.Pack(mesh, g, recon)
    if nst == 3:
        po.set_integrator(3); pg.set_integrator(3)
    po.load(U0.numpy()); pg.load(U0)
    t, n = 0.0, 0
    while t < 0.047:
        dt = min(po.new_dt(0.3), 0.047 - t)
        po.step(0.3, dt); pg.step(0.3, dt)
        t += dt; n += 1
    a = P.active(mesh)
    e = P.q14(P.gpu_state(pg)[a], po.current()[a], g)
    P.report(f"[parity] Shu-Osher tube 200 cells recon={recon} stages={nst}, {n} steps: Q14 {e:.3e}")
    assert e <= TOL_RUN
    assert pg.floor_count() == 0 and po.floor_count() == 0
    rho = P.gpu_state(pg)[:, 0][:, 3, 3, 3:-3].reshape(-1)
    assert rho.max() > 4.0                                   # the compressed entropy waves behind the shock


def test_boundary_argument_errors(ak):
    import dataclasses
    with pytest.raises(ak.AkError):
        ak.Pack(dataclasses.replace(I.uniform_mesh((1, 1, 1), (8, 8, 8), 2), bc=(1, 0, 0, 0, 0, 0)), I.GAMMA, 0)
    with pytest.raises(ak.AkError):
        ak.Pack(dataclasses.replace(I.smr_mesh((2, 2, 2), (8, 8, 8), 2, (0, 0, 0), (1, 1, 1)), bc=(1, 1, 0, 0, 0, 0)), I.GAMMA, 0)


# ------------------------------------------------------------ dt taken by stage 2 --------
@pytest.mark.parametrize("which", ["cfg1", "cfg3", "smr", "walls"])
def test_dt_from_stage2_is_bit_identical_to_the_reduction_over_the_state(orc, ak, which):
    """After a step, ak_new_dt answers from the signal speeds stage 2 left behind (no kernel launch).  It must equal,
    bit for bit, the oracle's Eq.(3) reduction over the GPU's own state -- and the stand-alone reduction kernel."""
    import dataclasses
    w = {"cfg1": lambda: I.config1(nrb=2, nx=32), "cfg3": lambda: I.config3(nrb=2, nx=32), "smr": lambda: I.smr_parity(nx=16),
         "walls": lambda: I.config1(nrb=2, nx=16)}[which]()
    if which == "walls":
        w.mesh = dataclasses.replace(w.mesh, bc=(2, 2, 1, 1, 0, 0))
    pg = ak.Pack(w.mesh, w.gamma, w.recon)
    pg.load(w.state())
    for step in range(3):
        pg.step(w.cfl)
        l0 = pg.launch_count()
        dt_fused = pg.new_dt(w.cfl)
        assert pg.launch_count() == l0                      # answered without a launch
        po = orc.OrcPack(w.mesh, w.gamma, w.recon, threads=P.NTHREADS)
        po.load(P.gpu_state(pg))
        assert po.new_dt(w.cfl) == dt_fused, (which, step)
        po.close()
        pg.upload(pg.current().cpu().contiguous())          # invalidates the cache: the reduction kernel runs
        assert pg.new_dt(w.cfl) == dt_fused and pg.launch_count() == l0 + 2


# ------------------------------------------------------------ SSPRK(3,3) --------
@pytest.mark.parametrize("which", ["cfg3", "cfg1", "smr_fc"])
def test_rk3_matches_the_oracle(orc, ak, which):
    """Three-stage integrator with the third register: the paper's showcased RK3 + PPM4 + HLLC combination on
    the config-3 recipe, PLM on config 1, and the two-level mesh with flux correction; dt from the fused reduction
    of the LAST stage is bit-identical to the oracle's reduction over the GPU state."""
    w = {"cfg3": lambda: I.config3(nrb=2, nx=32), "cfg1": lambda: I.config1(nrb=2, nx=32), "smr_fc": lambda: I.smr_parity(nx=16)}[which]()
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0)
    po.set_integrator(3); pg.set_integrator(3)
    if which == "smr_fc":
        po.set_flux_correction(True); pg.set_flux_correction(True)
    a = P.active(w.mesh)
    for step in range(4):
        dt = po.new_dt(w.cfl)
        dt_g = pg.new_dt(w.cfl)
        assert abs(dt_g - dt) <= 1e-13 * dt
        for stage in (1, 2, 3):
            po.fill_ghosts(); pg.fill_ghosts()
            po.hydro_stage(stage, dt); pg.hydro_stage(stage, dt)
            if step == 0:
                e = P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma)
                assert e <= TOL_STAGE * stage, f"stage {stage}: Q14 = {e:.3e}"
        chk = orc.OrcPack(w.mesh, w.gamma, w.recon, threads=P.NTHREADS)
        chk.load(P.gpu_state(pg))
        l0 = pg.launch_count()
        assert pg.new_dt(w.cfl) == chk.new_dt(w.cfl)
        if which != "smr_fc":
            assert pg.launch_count() == l0                  # taken from the last stage, no launch
        chk.close()
    assert P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma) <= TOL_RUN
    check_totals(w, U0, po, pg)
    assert pg.floor_count() == 0
    with pytest.raises(ak.AkError):
        pg.hydro_stage(2, 1e-3)                             # stage 1 first


# ------------------------------------------------------------ PPMX / WENOZ --------
@pytest.mark.parametrize("recon", [I.RECON_PPMX, I.RECON_WENOZ])
def test_ppmx_and_wenoz_match_the_oracle(orc, ak, recon):
    """Same kernel skeleton, other reconstruction (stencil radius 3 like PPM4): the config-3 recipe with SSPRK(2,2), ragged
    non-cubic blocks, and -- the paper's showcased combination for WENOZ -- SSPRK(3,3); every tile shape gives
    the same bits; the two-level mesh with flux correction conserves."""
    w = I.config3(nrb=2, nx=32)
    w.recon = recon
    errs, po, pg, U0 = run_lockstep(orc, ak, w, 4)
    assert max(errs) <= TOL_RUN, (recon, errs)
    check_totals(w, U0, po, pg)
    # ragged blocks, both tile shapes bit-identical
    w = I.config3(nrb=2, nx=32)
    w.recon = recon
    w.mesh = I.uniform_mesh((2, 1, 3), (24, 40, 6), 3)
    errs, po, pg, U0 = run_lockstep(orc, ak, w, 2)
    assert max(errs) <= TOL_RUN, (recon, errs)
    ref = P.gpu_state(pg)
    for tile in (0, 1):
        pt = ak.Pack(w.mesh, w.gamma, recon)
        pt.set_tile(tile)
        pt.load(U0)
        for _ in range(2):
            pt.step(w.cfl, None)
        # (free-running dt equals the lock-step one only to rounding: compare the two tile shapes with each other)
        if tile == 0:
            t0 = P.gpu_state(pt)
        else:
            assert np.array_equal(P.gpu_state(pt), t0)
    # SSPRK(3,3)
    w = I.config3(nrb=2, nx=32)
    w.recon = recon
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0)
    po.set_integrator(3); pg.set_integrator(3)
    a = P.active(w.mesh)
    for step in range(3):
        dt = po.new_dt(w.cfl)
        assert abs(pg.new_dt(w.cfl) - dt) <= 1e-13 * dt
        po.step(w.cfl, dt); pg.step(w.cfl, dt)
    e = P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma)
    P.report(f"[parity] {w.name} recon={recon} SSPRK(3,3) 3 steps: Q14 {e:.3e}")
    assert e <= TOL_RUN
    assert po.floor_count() == 0 and pg.floor_count() == 0
    # two-level mesh, flux correction on
    w = I.smr_parity(nx=16)
    w.recon = recon
    w.mesh = I.smr_mesh((4, 4, 4), (16, 16, 16), 4, (1, 1, 1), (3, 3, 3))      # ng = 4: even (SMR) and ng - 3 odd -> refused
    pg = ak.Pack(w.mesh, w.gamma, recon)
    pg.load(w.state())
    pg.fill_ghosts()
    with pytest.raises(ak.AkError):
        pg.hydro_stage(1, 1e-4)                             # TMA box origin misaligned: not offered for PPMX / WENOZ


def test_ppmx_wenoz_only_in_the_production_kernel_with_hllc(ak):
    w = I.config3(nrb=1, nx=16)
    for kw in (dict(variant=1), dict(rsolver=1)):
        pg = ak.Pack(w.mesh, w.gamma, I.RECON_WENOZ, **kw)
        pg.load(w.state())
        pg.fill_ghosts()
        with pytest.raises(ak.AkError):
            pg.hydro_stage(1, 1e-3)


def test_rk3_through_ak_step_and_integrator_errors(orc, ak):
    w = I.config1(nrb=2, nx=16)
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0)
    po.set_integrator(3); pg.set_integrator(3)
    for _ in range(3):
        dt = po.new_dt(w.cfl)
        po.step(w.cfl, dt); pg.step(w.cfl, dt)
    a = P.active(w.mesh)
    assert P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma) <= TOL_RUN
    pv = ak.Pack(w.mesh, w.gamma, w.recon, variant=1)
    pv.set_integrator(3)
    pv.load(U0)
    pv.fill_ghosts()
    with pytest.raises(ak.AkError):
        pv.hydro_stage(1, 1e-3)                             # the cross-check kernels are two-stage only
    L = ak.lib()
    assert L.ak_pack_set_integrator(pg._h, 4, None) == -1 and L.ak_pack_set_integrator(pg._h, 3, None) == -1


def test_forward_euler_matches_the_oracle(orc, ak):
    w = I.config1(nrb=2, nx=16)
    U0 = w.state()
    po, pg = P.make_pair(orc, ak, w, U0)
    po.set_integrator(1); pg.set_integrator(1)
    a = P.active(w.mesh)
    for step in range(5):
        dt = 0.5 * po.new_dt(w.cfl)
        assert abs(0.5 * pg.new_dt(w.cfl) - dt) <= 1e-13 * dt
        po.step(w.cfl, dt); pg.step(w.cfl, dt)
        assert P.q14(P.gpu_state(pg)[a], po.current()[a], w.gamma) <= TOL_STAGE * (step + 1)
    assert pg.current().data_ptr() == pg.ub.data_ptr()          # five steps: the registers alternate
    with pytest.raises(ak.AkError):
        pg.set_integrator(2)


@pytest.mark.parametrize("nx", [16, 32, 64, 128])
def test_config2_full_size_sampled(orc, ak, nx):
    """BASELINE config 2 at its full 256^3, at every block size of the sweep (4096 blocks of 16^3: every sampled box
    spans 8-27 MeshBlocks; 512 of 32^3 -- the variant BASELINE.json names for parity; 64 of 64^3; 8 blocks of 128^3),
    as bench.py runs it: two RK2 steps on the GPU against the
    oracle on 32^3 sub-boxes (PLM: a step reaches 2 x 2 cells, two steps 8 = the margin dropped on each side).  The
    boxes sit on the blast (centre, edge of the hot sphere), on a block corner and on the periodic wrap."""
    w = I.config2(nx)
    dev = torch.device("cuda", 0)
    pg = ak.Pack(w.mesh, w.gamma, w.recon, device=dev)
    U0 = w.state(device=dev)
    pg.load(U0)
    G0 = _assemble(w.mesh, U0)
    del U0
    n, pad = 32, 8
    origins = [(112, 112, 112), (100, 118, 120), (240, 240, 240), (112, 112, 121), (0, 64, 200)]
    subs0 = [_subbox(G0, o, n) for o in origins]
    tot0 = G0.sum(dim=(1, 2, 3)).cpu().numpy()
    del G0
    dts = []
    for _ in range(2):
        dts.append(pg.new_dt(w.cfl))
        pg.step(w.cfl, dts[-1])
    assert pg.floor_count() == 0
    G1 = _assemble(w.mesh, pg.current())
    tot1 = G1.sum(dim=(1, 2, 3)).cpu().numpy()
    assert abs(tot1[0] - tot0[0]) <= TOL_TOTALS * tot0[0] and abs(tot1[4] - tot0[4]) <= TOL_TOTALS * tot0[4]
    dx = w.mesh.dx(0)
    sub_mesh = I.Mesh((1, 1, 1), (n, n, n), w.mesh.ng, [(0, 0, 0, 0)], xmax=(n * dx[0], n * dx[1], n * dx[2]))
    assert sub_mesh.dx(0) == dx
    g = w.mesh.ng
    worst = 0.0
    for o, s0 in zip(origins, subs0):
        po = orc.OrcPack(sub_mesh, w.gamma, w.recon, threads=1)
        u = np.zeros(sub_mesh.state_shape())
        u[0][:, g:-g, g:-g, g:-g] = s0
        po.load(u)
        for dt in dts:
            po.step(w.cfl, dt)
        ref = po.current()[0][:, g + pad:-g - pad, g + pad:-g - pad, g + pad:-g - pad]
        got = _subbox(G1, o, n)[:, pad:-pad, pad:-pad, pad:-pad]
        e = P.q14(got[None], ref[None], w.gamma)
        worst = max(worst, e)
        assert e <= 4 * TOL_STAGE, (nx, o, e)
        po.close()
    P.report(f"[parity] cfg2 full size 256^3 in {nx}^3 blocks: worst sampled Q14 after 2 RK2 steps = {worst:.2e}")
