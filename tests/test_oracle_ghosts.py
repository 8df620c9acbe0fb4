"""Pins for the oracle's ghost fill G1-G4: brute force for same-level copies, exactness
on dyadic-linear fields for restriction / prolongation, conservation of the parent mean, flatness at
extrema, and independence of the fill from the previous ghost contents."""
import numpy as np
import pytest
import torch

from paper_2409_16053_b200 import inputs as I


def fill(orc, mesh, U):
    p = orc.OrcPack(mesh, I.GAMMA, I.RECON_PLM if mesh.ng == 2 else I.RECON_PPM4)
    p.load(U)
    p.fill_ghosts()
    out = p.current().copy()
    p.close()
    return out


def global_index_arrays(mesh, m):
    """Wrapped level-local global cell index of every stored cell (ghosts included) of block m, per direction."""
    lev, *lx = mesh.blocks[m]
    out = []
    for d in range(3):
        n = mesh.nrb[d] * mesh.nx[d] * (1 << lev)
        out.append((lx[d] * mesh.nx[d] + np.arange(-mesh.ng, mesh.nx[d] + mesh.ng)) % n)
    return out


@pytest.mark.parametrize("nrb,nx,ng", [((1, 1, 1), (8, 8, 8), 2), ((2, 2, 2), (8, 8, 8), 2), ((3, 2, 1), (8, 16, 4), 3),
                                       ((2, 2, 2), (4, 4, 4), 3)])
def test_same_level_fill_brute_force(orc, nrb, nx, ng):
    mesh = I.uniform_mesh(nrb, nx, ng)
    N = [nrb[d] * nx[d] for d in range(3)]
    U = np.full(mesh.state_shape(), np.nan)
    code = lambda n, g3, g2, g1: (n + 1) * 1e6 + (g3 * N[1] + g2) * N[0] + g1        # exactly representable
    for m in range(mesh.nmb):
        g1, g2, g3 = global_index_arrays(mesh, m)
        for n in range(5):
            U[m, n, ng:-ng, ng:-ng, ng:-ng] = code(n, g3[ng:-ng, None, None], g2[None, ng:-ng, None], g1[None, None, ng:-ng])
    out = fill(orc, mesh, U)
    for m in range(mesh.nmb):
        g1, g2, g3 = global_index_arrays(mesh, m)
        for n in range(5):
            assert np.array_equal(out[m, n], code(n, g3[:, None, None], g2[None, :, None], g1[None, None, :]))


def small_smr(nx=8):
    return I.smr_mesh((4, 4, 4), (nx,) * 3, 2, (1, 1, 1), (3, 3, 3))


def linear_field(mesh, coef=(0.5, -0.25, 2.0), c0=3.0):
    """Dyadic-linear field sampled at every stored cell centre (ghost positions included, NOT wrapped)."""
    U = np.zeros(mesh.state_shape())
    for m, (lev, *lx) in enumerate(mesh.blocks):
        dx = mesh.dx(lev)
        x = [(lx[d] * mesh.nx[d] + np.arange(-mesh.ng, mesh.nx[d] + mesh.ng) + 0.5) * dx[d] for d in range(3)]
        f = c0 + coef[0] * x[0][None, None, :] + coef[1] * x[1][None, :, None] + coef[2] * x[2][:, None, None]
        for n in range(5):
            U[m, n] = (n + 1) * f
    return U


def ghost_class(mesh, m):
    """0 = active, 1 = same level, 2 = restricted (finer leaves underneath), 3 = prolonged (coarser leaf)."""
    lev, *lx = mesh.blocks[m]
    nb = [mesh.nrb[d] * (1 << lev) for d in range(3)]
    is_leaf = np.zeros((nb[2], nb[1], nb[0]), dtype=bool)
    for (l, l1, l2, l3) in mesh.blocks:
        if l == lev:
            is_leaf[l3, l2, l1] = True
    g = global_index_arrays(mesh, m)
    b = [g[d] // mesh.nx[d] for d in range(3)]
    same = is_leaf[b[2][:, None, None], b[1][None, :, None], b[0][None, None, :]]
    cls = np.where(same, 1, 2 if lev == 0 else 3)
    ng = mesh.ng
    cls[ng:-ng, ng:-ng, ng:-ng] = 0
    return cls


def test_smr_mesh_shape_and_ghost_census():
    """Counts of SURVEY 8(a) rows a2/a3 for config 4, re-derived here from the block list alone."""
    mesh = I.config4().mesh
    assert mesh.nmb == 120 and mesh.ncells_active == 3_932_160
    counts = {1: 0, 2: 0, 3: 0}
    per_block = {}
    for m in range(mesh.nmb):
        cls = ghost_class(mesh, m)
        for c in counts:
            counts[c] += int((cls == c).sum())
        per_block[m] = (int((cls == 2).sum()), int((cls == 3).sum()))
    assert counts[2] == 58_816 and counts[3] == 241_984
    assert counts[1] + counts[2] + counts[3] == 1_666_560
    assert sorted(set(v[0] for v in per_block.values())) == [0, 8, 136, 2312]
    assert sorted(set(v[1] for v in per_block.values())) == [0, 2592, 5040, 7352]


def test_restriction_and_prolongation_exact_on_dyadic_linear_field(orc):
    mesh = small_smr(8)
    exact = linear_field(mesh)
    U = exact.copy()
    ng = mesh.ng
    act = np.zeros(mesh.nt[::-1], dtype=bool)
    act[ng:-ng, ng:-ng, ng:-ng] = True
    U[:, :, ~act] = np.nan
    out = fill(orc, mesh, U)
    checked = {2: 0, 3: 0}
    for m in range(mesh.nmb):
        cls = ghost_class(mesh, m)
        for c in (2, 3):
            sel = cls == c
            if sel.any():
                # level boundaries of this mesh are far from the periodic wrap, so the linear field is valid there
                assert np.array_equal(out[m][:, sel], exact[m][:, sel]), (m, c)
                checked[c] += int(sel.sum())
        assert not np.isnan(out[m]).any()
    assert checked[2] > 0 and checked[3] > 0


def test_prolongation_preserves_parent_mean_and_is_flat_at_extrema(orc):
    mesh = small_smr(8)
    rng = np.random.default_rng(7)
    U = rng.uniform(1.0, 2.0, size=mesh.state_shape())
    out = fill(orc, mesh, U)
    # virtual coarse field at root level assembled independently from the ACTIVE data
    ng, nx = mesh.ng, 8
    C = np.zeros((5, 32, 32, 32))
    for m, (lev, l1, l2, l3) in enumerate(mesh.blocks):
        a = out[m][:, ng:-ng, ng:-ng, ng:-ng]
        if lev == 0:
            C[:, l3 * nx:(l3 + 1) * nx, l2 * nx:(l2 + 1) * nx, l1 * nx:(l1 + 1) * nx] = a
        else:
            r = a.reshape(5, 4, 2, 4, 2, 4, 2).mean(axis=(2, 4, 6))
            C[:, l3 * 4:(l3 + 1) * 4, l2 * 4:(l2 + 1) * 4, l1 * 4:(l1 + 1) * 4] = r
    n_groups = 0
    for m, (lev, *lx) in enumerate(mesh.blocks):
        if lev == 0:
            continue
        cls = ghost_class(mesh, m)
        g = global_index_arrays(mesh, m)
        # ghost depth 2 = one parent cell: stored index pairs (0,1) and (nt-2, nt-1) share a parent
        for k0 in range(0, mesh.nt[2], 2):
            for j0 in range(0, mesh.nt[1], 2):
                for i0 in range(0, mesh.nt[0], 2):
                    blk = cls[k0:k0 + 2, j0:j0 + 2, i0:i0 + 2]
                    if not (blk == 3).all():
                        continue
                    kids = out[m][:, k0:k0 + 2, j0:j0 + 2, i0:i0 + 2]
                    parent = C[:, g[2][k0] // 2, g[1][j0] // 2, g[0][i0] // 2]
                    np.testing.assert_allclose(kids.mean(axis=(1, 2, 3)), parent, rtol=4e-16)
                    # limited: children stay inside the range spanned by the parent and its 6 neighbours
                    P = [g[2][k0] // 2, g[1][j0] // 2, g[0][i0] // 2]
                    nb = [C[:, (P[0] + a) % 32, (P[1] + b) % 32, (P[2] + c) % 32]
                          for a, b, c in ((0, 0, 0), (1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1))]
                    lo, hi = np.min(nb, axis=0), np.max(nb, axis=0)
                    assert (kids >= lo[:, None, None, None] - 1e-15).all() and (kids <= hi[:, None, None, None] + 1e-15).all()
                    is_ext = np.array([all((nb[1 + 2 * d][n] - nb[0][n]) * (nb[0][n] - nb[2 + 2 * d][n]) <= 0 for d in range(3))
                                       for n in range(5)])
                    for n in np.nonzero(is_ext)[0]:
                        assert (kids[n] == parent[n]).all()
                    n_groups += 1
    assert n_groups > 100


def test_restriction_is_the_mean_of_eight_on_random_data(orc):
    mesh = small_smr(8)
    rng = np.random.default_rng(8)
    U = rng.uniform(1.0, 2.0, size=mesh.state_shape())
    out = fill(orc, mesh, U)
    ng, nx = mesh.ng, 8
    leaf = {b: m for m, b in enumerate(mesh.blocks)}
    n = 0
    for m, (lev, *lx) in enumerate(mesh.blocks):
        if lev != 0:
            continue
        cls = ghost_class(mesh, m)
        g = global_index_arrays(mesh, m)
        for k, j, i in zip(*np.nonzero(cls == 2)):
            G = (g[0][i], g[1][j], g[2][k])
            acc = np.zeros(5)
            for dk in range(2):
                for dj in range(2):
                    for di in range(2):
                        Gf = (2 * G[0] + di, 2 * G[1] + dj, 2 * G[2] + dk)
                        mf = leaf[(1, Gf[0] // nx, Gf[1] // nx, Gf[2] // nx)]
                        acc += U[mf][:, Gf[2] % nx + ng, Gf[1] % nx + ng, Gf[0] % nx + ng]
            np.testing.assert_allclose(out[m][:, k, j, i], acc / 8, rtol=4e-16)
            n += 1
    assert n == 24 * 200 + 24 * 40 + 8 * 8      # face / edge / corner sharing coarse blocks: nx^2 ng + 2 nx ng^2 + ng^3, ...


def test_fill_ignores_previous_ghost_contents_and_never_touches_active(orc):
    mesh = small_smr(8)
    rng = np.random.default_rng(9)
    U = rng.uniform(1.0, 2.0, size=mesh.state_shape())
    ng = mesh.ng
    a = (slice(None), slice(None), slice(ng, -ng), slice(ng, -ng), slice(ng, -ng))
    out1 = fill(orc, mesh, U)
    V = rng.uniform(5.0, 6.0, size=mesh.state_shape())
    V[a] = U[a]
    out2 = fill(orc, mesh, V)
    assert np.array_equal(out1, out2)
    assert np.array_equal(out1[a], U[a])
    assert np.array_equal(fill(orc, mesh, out1), out1)      # idempotent
