"""Pins for the oracle's outflow and reflecting boundaries (paper P:67 boundary functions).

  * brute force: with every active cell carrying its own global cell number, each ghost cell outside the domain must
    hold the number of the nearest active cell (outflow) or of its mirror image (reflect), and the normal momentum
    of a reflected ghost must be the negated mirror value;
  * a domain closed by reflecting walls equals one half of a periodic domain of twice the length carrying the
    mirror-symmetric initial state -- BIT FOR BIT, because the scheme is exactly mirror symmetric (pinned in
    tests/test_oracle_scheme.py); a wrong index, sign or a missed corner ghost breaks the equality;
  * the standard (non-periodic) Sod tube with outflow ends equals the corresponding half of the periodic double Sod
    problem bit for bit while the waves have not reached the ends, and therefore inherits its pin against the exact
    Riemann solution;
  * a uniform state with non-zero velocity along the wall-parallel directions is preserved bit-exactly.
"""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2409_16053_b200 import inputs as I
from tests import parity as P
from tests.test_oracle_scheme import sod_run

PER, OUT, REF = 0, 1, 2


def with_bc(mesh, bc, **kw):
    return dataclasses.replace(mesh, bc=tuple(bc), **kw)


@pytest.mark.parametrize("kind", [OUT, REF])
def test_ghosts_by_brute_force(orc, kind):
    nrb, nx, ng = (2, 1, 2), (4, 6, 4), 2
    bc = (kind, kind, PER, PER, kind, kind)
    mesh = with_bc(I.uniform_mesh(nrb, nx, ng), bc)
    N = [nrb[d] * nx[d] for d in range(3)]
    U = np.zeros(mesh.state_shape())
    for m, (_, l1, l2, l3) in enumerate(mesh.blocks):
        g1 = l1 * nx[0] + np.arange(nx[0]); g2 = l2 * nx[1] + np.arange(nx[1]); g3 = l3 * nx[2] + np.arange(nx[2])
        code = (g3[:, None, None] * N[1] + g2[None, :, None]) * N[0] + g1[None, None, :] + 1.0
        for n in range(5):
            U[m, n, ng:-ng, ng:-ng, ng:-ng] = code * (n + 1)
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    p.load(U)
    p.fill_ghosts()
    F = p.current()

    def image(g, n, k):
        if 0 <= g < n:
            return g, 1.0
        if k == PER:
            return g % n, 1.0
        if k == OUT:
            return (0 if g < 0 else n - 1), 1.0
        return (-1 - g if g < 0 else 2 * n - 1 - g), -1.0

    for m, (_, l1, l2, l3) in enumerate(mesh.blocks):
        l = (l1, l2, l3)
        for k in range(nx[2] + 2 * ng):
            for j in range(nx[1] + 2 * ng):
                for i in range(nx[0] + 2 * ng):
                    a = (i - ng, j - ng, k - ng)
                    G, s = [], [1.0] * 5
                    for d in range(3):
                        g, sg = image(l[d] * nx[d] + a[d], N[d], bc[2 * d])
                        G.append(g); s[1 + d] *= sg
                    code = (G[2] * N[1] + G[1]) * N[0] + G[0] + 1.0
                    for n in range(5):
                        assert F[m, n, k, j, i] == s[n] * code * (n + 1), (m, n, k, j, i)


@pytest.mark.parametrize("d", [0, 1, 2])
@pytest.mark.parametrize("recon,ng", [(I.RECON_PLM, 2), (I.RECON_PPM4, 3)])
def test_reflecting_walls_equal_half_of_the_mirrored_periodic_domain(orc, d, recon, ng):
    nx, nrb = [8, 8, 8], [1, 1, 1]
    nrb[d] = 2                                                   # two blocks along the wall normal: corner ghosts cross blocks
    bc = [PER] * 6
    bc[2 * d] = bc[2 * d + 1] = REF
    small = with_bc(I.uniform_mesh(tuple(nrb), tuple(nx), ng), bc)
    w = I.config1(nrb=2, nx=8)                                   # field generator only
    Us = I.make_state(small, w.prim_fn).numpy()
    # periodic domain of twice the length along d: [0, 2), second half = mirror image (normal momentum odd)
    nrb2 = list(nrb); nrb2[d] = 4
    xmax = [1.0, 1.0, 1.0]; xmax[d] = 2.0
    big = dataclasses.replace(I.uniform_mesh(tuple(nrb2), tuple(nx), ng), xmax=tuple(xmax))
    Ub = np.zeros(big.state_shape())
    loc_s = {tuple(b[1:]): m for m, b in enumerate(small.blocks)}
    ax = 4 - d                                                   # array axis of direction d in (m, n, k, j, i)
    for m, (_, *l) in enumerate(big.blocks):
        if l[d] < 2:
            Ub[m] = Us[loc_s[tuple(l)]]
        else:
            ls = list(l); ls[d] = 3 - l[d]
            src = np.flip(Us[loc_s[tuple(ls)]], axis=ax - 1).copy()
            src[1 + d] = -src[1 + d]
            Ub[m] = src
    ps, pb = orc.OrcPack(small, I.GAMMA, recon), orc.OrcPack(big, I.GAMMA, recon)
    ps.load(Us); pb.load(Ub)
    for _ in range(4):
        dt = pb.new_dt(0.3)
        assert ps.new_dt(0.3) == dt
        ps.step(0.3, dt); pb.step(0.3, dt)
    a = P.active(small)[1:]
    for m, (_, *l) in enumerate(big.blocks):
        if l[d] < 2:
            assert np.array_equal(pb.current()[m][a], ps.current()[loc_s[tuple(l)]][a]), (d, l)


def test_standard_sod_with_outflow_ends_equals_half_of_the_periodic_double_sod(orc):
    N, g, ng = 256, 1.4, 2
    U0p, Up = sod_run(orc, N, I.RECON_PLM, ng)                   # periodic line, left state on [0.25, 0.75), t = 0.1
    mesh = dataclasses.replace(I.uniform_mesh((1, 1, 1), (N // 2, 4, 4), ng), xmin=(0.5, 0.0, 0.0),
                               bc=(OUT, OUT, PER, PER, PER, PER))

    def prim(X1, X2, X3):
        left = X1 < 0.75
        rho = torch.where(left, 1.0, 0.125).to(torch.float64)
        pr = torch.where(left, 1.0, 0.1).to(torch.float64)
        z = torch.zeros_like(rho)
        return (rho, z, z, z, pr)

    U0 = I.make_state(mesh, prim, gamma=g).numpy()
    p = orc.OrcPack(mesh, g, I.RECON_PLM)
    p.load(U0)
    t = 0.0
    while t < 0.1:
        dt = p.new_dt(0.3)
        if t + dt > 0.1:
            dt = 0.1 - t
        p.step(0.3, dt)
        t += dt
    prof = p.current()[0, :, ng, ng, ng:-ng]
    assert np.array_equal(prof, Up[:, N // 2:])


def test_uniform_state_preserved_with_walls_and_outflow(orc):
    mesh = with_bc(I.uniform_mesh((2, 1, 1), (8, 8, 8), 2), (REF, REF, OUT, OUT, PER, PER))
    prim = lambda X1, X2, X3: (1.3 + 0 * X1, 0 * X1, -0.7 + 0 * X1, 0.2 + 0 * X1, 0.9 + 0 * X1)   # no flow through the walls
    U0 = I.make_state(mesh, prim).numpy()
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    p.load(U0)
    for _ in range(2):
        p.step(0.3)
    a = P.active(mesh)
    assert np.array_equal(p.current()[a], U0[a])


def test_bad_boundary_arguments_are_rejected(orc):
    mesh = with_bc(I.uniform_mesh((1, 1, 1), (8, 8, 8), 2), (OUT, PER, PER, PER, PER, PER))
    with pytest.raises(orc.OrcError):
        orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM)
    smr = with_bc(I.smr_mesh((2, 2, 2), (8, 8, 8), 2, (0, 0, 0), (1, 1, 1)), (OUT, OUT, PER, PER, PER, PER))
    with pytest.raises(orc.OrcError):
        orc.OrcPack(smr, I.GAMMA, I.RECON_PLM)
