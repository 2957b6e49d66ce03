"""GPU gates that do NOT go through the oracle's own routines:

* the near/singular table of the CUDA path (SELF / ADJ semi-analytic entries, NEAR 19-point entries) pinned,
  entry by entry, against brute-force integrals computed here (Duffy-mapped tensor Gauss-Legendre, the Laplace SELF
  closed form of SURVEY App. A.3) by applying pb_matvec (theta = 0) to unit vectors -- an independent check of
  csrc/pb_near.cu, whose routines resemble the oracle's;
* input validation promised by the boundary (S: section 8(b), R-3);
* properties: bitwise repeatability of the reaction field with near (site, panel) pairs, independent contexts of
  different order on one device, the high-order M2P kernels at a mesh of several thousand panels.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

FOURPI = 4.0 * math.pi


def rel(a, b):
    a, b = np.asarray(a, dtype=float), np.asarray(b, dtype=float)
    d = a - b
    l2, linf = float(np.linalg.norm(d) / np.linalg.norm(b)), float(np.max(np.abs(d)) / np.max(np.abs(b)))
    return max(l2, linf if l2 < 1e-9 else 0.1 * linf)       # see tests/test_gpu_fullsize.py::rel


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test run without a CUDA device: the product has no CPU fallback")
    return torch


@pytest.fixture(scope="module")
def pbm(torch_cuda):
    from paper_1810_03698_b200 import pb
    pb.build()
    return pb


# ---- brute force, written here (no oracle/, no library routine) ---------------------------------------------------
def _duffy(v, n):
    """n x n tensor Gauss-Legendre points on the triangle v, collapsed towards v[0]: points [n*n][3], weights
    (summing to the area).  With the singular point at v[0] the Jacobian cancels a 1/R singularity."""
    xs, ws = np.polynomial.legendre.leggauss(n)
    u, wu = 0.5 * (xs + 1), 0.5 * ws
    U, V = np.meshgrid(u, u, indexing="ij")
    W = np.outer(wu, wu) * U                                   # y = v0 + U [(v1 - v0) + V (v2 - v1)]
    y = v[0] + U[..., None] * ((v[1] - v[0]) + V[..., None] * (v[2] - v[1]))
    area2 = np.linalg.norm(np.cross(v[1] - v[0], v[2] - v[0]))
    return y.reshape(-1, 3), (W * area2).reshape(-1)


def brute_entry(x, v, kappa, n=200):
    """(V_L, K_L, V_Y, K_Y) = panel integrals of Eq. (4)'s kernels with the 1/(4 pi), target x OFF the panel."""
    y, w = _duffy(v, n)
    nrm = np.cross(v[1] - v[0], v[2] - v[0])
    nrm /= np.linalg.norm(nrm)
    d = x[None, :] - y
    R = np.linalg.norm(d, axis=1)
    nd = d @ nrm
    e = np.exp(-kappa * R)
    return np.array([np.sum(w / R), np.sum(w * nd / R ** 3), np.sum(w * e / R), np.sum(w * nd * e * (1 + kappa * R) / R ** 3)]) / FOURPI


def brute_self(v, kappa, n=80):
    """SELF entries at the centroid c of the flat panel v: V_L by the closed form sum_e d_e [asinh(tan th_b) -
    asinh(tan th_a)]/(4 pi) (S: App. A.3), V_Y = V_L - int (1 - e^{-kR})/(4 pi R), the latter integrand made smooth by
    splitting the panel into three sub-triangles with the singular vertex at c (Duffy); K_L = K_Y = 0 in the plane."""
    c = v.mean(axis=0)
    nrm = np.cross(v[1] - v[0], v[2] - v[0])
    nrm /= np.linalg.norm(nrm)
    tot, smooth = 0.0, 0.0
    for e in range(3):
        a, b = v[e] - c, v[(e + 1) % 3] - c
        L = np.linalg.norm(b - a)
        t = (b - a) / L
        de = abs(np.dot(np.cross(a, b), nrm)) / L
        tot += de * (math.asinh(np.dot(b, t) / de) - math.asinh(np.dot(a, t) / de))
        y, w = _duffy(np.array([c, v[e], v[(e + 1) % 3]]), n)
        R = np.linalg.norm(y - c, axis=1)
        smooth += np.sum(w * (-np.expm1(-kappa * R)) / R)
    return np.array([tot / FOURPI, 0.0, (tot - smooth) / FOURPI, 0.0])


def tetrahedron(scale=1.0):
    v = scale * np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=float)
    t = np.array([[0, 1, 2], [0, 3, 1], [0, 2, 3], [1, 3, 2]], dtype=np.int32)
    return _outward(v, t)


def octahedron(scale=1.0):
    v = scale * np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], dtype=float)
    t = np.array([[0, 2, 4], [2, 1, 4], [1, 3, 4], [3, 0, 4], [2, 0, 5], [1, 2, 5], [3, 1, 5], [0, 3, 5]], dtype=np.int32)
    return _outward(v, t)


def _outward(v, t):
    t = t.copy()
    for k in range(t.shape[0]):
        a, b, c = v[t[k]]
        if np.dot(np.cross(b - a, c - a), (a + b + c) / 3.0) < 0:
            t[k] = t[k][[0, 2, 1]]
    return v, t


def _columns(ctx, torch, nt, cols, eps_ratio):
    """Entries (V_L, K_L, V_Y, K_Y)[i, j] of the operator the GPU applies in direct mode, for source panels j in
    `cols`, read off pb_matvec applied to unit vectors (Eq. 5)."""
    out = {}
    for j in cols:
        x = torch.zeros(2 * nt, dtype=torch.float64, device="cuda")
        x[j] = 1.0
        y = ctx.matvec(x).cpu().numpy()
        dlt = np.zeros(nt)
        dlt[j] = 0.5
        KL, KY = y[:nt] - dlt, -(y[nt:] - dlt)
        x.zero_()
        x[nt + j] = 1.0
        y = ctx.matvec(x).cpu().numpy()
        VL, VY = -y[:nt], y[nt:] / eps_ratio
        out[j] = np.stack([VL, KL, VY, KY], axis=1)            # [nt][4]
    return out


@pytest.mark.parametrize("shape,kappa", [("tet", 0.125), ("oct", 0.125), ("tet", 0.0), ("oct", 0.4)])
def test_self_and_adjacent_entries_against_brute_force(pbm, torch_cuda, shape, kappa):
    """Every pair of a regular tetrahedron is SELF or ADJ (a shared vertex); on the octahedron the pairs of opposite
    faces are NEAR (|c_i - c_j| = 1.15 < 2 sqrt(A) = 1.86).  With nq_edge = 64 the semi-analytic entries must equal
    the brute-force integrals to 2e-10; at the operator's nq_edge = 16 (D: R-16) to 5e-6 (measured 5e-8 on the
    tetrahedron, 1.5e-6 on the octahedron's vertex-sharing pairs, 2e-8 on a vdW mesh).  The NEAR (19-point) entries
    agree with the integral to the accuracy of that rule at one panel size away."""
    v, t = tetrahedron(1.3) if shape == "tet" else octahedron(1.0)
    nt = t.shape[0]
    cen = v[t].mean(axis=1)
    shared = (t[:, None, :, None] == t[None, :, None, :]).any(axis=(2, 3))
    for nq, tol in ((64, 2e-10), (16, 5e-6)):
        ctx = pbm.PB(0, theta=0.0, kappa=kappa, K_far=7, nq_edge=nq, eps_in=1.0, eps_out=80.0)
        ctx.mesh_load(v, t)
        ctx.tree_build()
        cols = _columns(ctx, torch_cuda, nt, range(nt), 1.0 / 80.0)
        for j in range(nt):
            for i in range(nt):
                got = cols[j][i]
                if i == j:
                    ref = brute_self(v[t[j]], kappa)
                    assert abs(got[0] - ref[0]) <= tol * ref[0] and abs(got[2] - ref[2]) <= tol * ref[2], (i, j, got, ref)
                    assert got[1] == 0.0 and got[3] == 0.0          # flat panel: n'.(c_i - r') == 0 (S: O-2)
                elif shared[i, j]:
                    ref = brute_entry(cen[i], v[t[j]], kappa, n=300)
                    np.testing.assert_allclose(got, ref, rtol=tol, atol=tol * abs(ref[0]), err_msg=f"ADJ {i},{j}")
                else:
                    ref = brute_entry(cen[i], v[t[j]], kappa, n=100)
                    np.testing.assert_allclose(got, ref, rtol=2e-5, atol=1e-9, err_msg=f"NEAR {i},{j}")
        ctx.close()


def test_near_table_on_a_van_der_waals_patch_against_brute_force(pbm, torch_cuda):
    """An irregular mesh (vdW union of 120 atoms, ~2,500 panels: slivers, valence 4-9 vertices): for 12 seeded source
    panels every SELF entry of their columns against brute force to 1e-8, every ADJ entry to 2e-7, every NEAR entry (19-point rule,
    |c_i - c_j| < 2 sqrt(A_i), R-8) to 2e-4, every FAR entry (7-point rule) to the rule's accuracy at that distance."""
    from paper_1810_03698_b200.workloads import random_chain_globule, seed_for, vdw_surface
    g = random_chain_globule(seed_for(2), 120)
    v, t, _ = vdw_surface(g["pos"], g["radii"], target_panels=2500)
    t = t.astype(np.int32)
    nt = t.shape[0]
    kappa = 0.125
    cen = v[t].mean(axis=1)
    area = 0.5 * np.linalg.norm(np.cross(v[t[:, 1]] - v[t[:, 0]], v[t[:, 2]] - v[t[:, 0]]), axis=1)
    ctx = pbm.PB(0, theta=0.0, kappa=kappa, K_far=7)
    ctx.mesh_load(v, t)
    ctx.tree_build()
    cols_j = np.random.Generator(np.random.PCG64(41)).choice(nt, size=12, replace=False)
    cols = _columns(ctx, torch_cuda, nt, cols_j, 1.0 / 80.0)
    n_adj = n_near = 0
    for j in cols_j:
        dist = np.linalg.norm(cen - cen[j], axis=1)
        adj = np.isin(t, t[j]).any(axis=1)
        for i in np.nonzero(dist < 6.0 * math.sqrt(area[j]))[0]:
            got = cols[j][i]
            if i == j:
                ref = brute_self(v[t[j]], kappa)
                assert abs(got[0] - ref[0]) <= 1e-8 * ref[0] and abs(got[2] - ref[2]) <= 1e-8 * ref[2]
                assert got[1] == 0.0 and got[3] == 0.0
            elif adj[i]:
                ref = brute_entry(cen[i], v[t[j]], kappa, n=300)
                np.testing.assert_allclose(got, ref, rtol=2e-7, atol=2e-7 * abs(ref[0]), err_msg=f"ADJ {i},{j}")
                n_adj += 1
            elif dist[i] < 2.0 * math.sqrt(area[i]):
                ref = brute_entry(cen[i], v[t[j]], kappa, n=100)
                np.testing.assert_allclose(got, ref, rtol=2e-4, atol=2e-4 * abs(ref[0]), err_msg=f"NEAR {i},{j}")
                n_near += 1
            else:
                ref = brute_entry(cen[i], v[t[j]], kappa, n=60)
                np.testing.assert_allclose(got, ref, rtol=5e-2, atol=5e-3 * abs(ref[0]), err_msg=f"FAR {i},{j}")
    assert n_adj >= 100 and n_near >= 8
    ctx.close()


# ---- input validation (S: section 8(b), R-3) --------------------------------------------------------------------------
def test_validation_of_mesh_and_sites(pbm, torch_cuda):
    from paper_1810_03698_b200.workloads import icosphere
    v, t = icosphere(4.0, 2)
    one = dict(pos=np.zeros((1, 3)), q=np.ones(1), dip=np.zeros((1, 3)), quad=np.zeros((1, 6)), alpha=np.zeros(1),
               group=np.zeros(1, dtype=np.int32))
    ctx = pbm.PB(0)
    with pytest.raises(pbm.PBError) as e:                       # open surface: one panel removed
        ctx.mesh_load(v, t[:-1])
    assert e.value.code == -2 and "closed" in str(e.value)
    flipped = t.copy()
    flipped[7] = flipped[7][[0, 2, 1]]
    with pytest.raises(pbm.PBError) as e:                       # one panel with the opposite orientation
        ctx.mesh_load(v, flipped)
    assert e.value.code == -2 and "orient" in str(e.value)
    with pytest.raises(pbm.PBError) as e:                       # consistently oriented, but inward
        ctx.mesh_load(v, t[:, [0, 2, 1]])
    assert e.value.code == -2 and "volume" in str(e.value)
    dup = np.concatenate([t, t[:1]])
    with pytest.raises(pbm.PBError) as e:                       # an edge shared by three panels
        ctx.mesh_load(v, dup)
    assert e.value.code == -2
    ctx.mesh_load(v, t)
    bad = dict(one, quad=np.array([[1.0, 0, 0, 0.5, 0, 0.25]]))
    with pytest.raises(pbm.PBError) as e:                       # tr Q != 0
        ctx.sites_load(**bad)
    assert e.value.code == -1 and "traceless" in str(e.value)
    with pytest.raises(pbm.PBError) as e:
        ctx.sites_load(**dict(one, alpha=np.array([-1.0])))
    assert e.value.code == -1
    with pytest.raises(pbm.PBError) as e:                       # a site in the solvent
        ctx.sites_load(**dict(one, pos=np.array([[0.0, 0.0, 4.5]])))
    assert e.value.code == -2 and "outside" in str(e.value)
    two = {k: np.concatenate([a, a]) for k, a in one.items()}
    two["pos"] = np.array([[0.0, 0.0, 3.7], [9.0, 0.0, 0.0]])   # 0.3 A inside, and far outside
    with pytest.raises(pbm.PBError) as e:
        ctx.sites_load(**two)
    assert e.value.code == -2 and "site 1 " in str(e.value)
    two["pos"][1] = [0.0, -3.7, 0.0]
    ctx.sites_load(**two)                                       # both 0.3 A inside: accepted
    # the check also runs when the mesh arrives after the sites
    with pytest.raises(pbm.PBError) as e:
        ctx.mesh_load(0.5 * v, t)
    assert e.value.code == -2 and "outside" in str(e.value)
    ctx.close()


# ---- properties --------------------------------------------------------------------------------------------------------
def test_reaction_field_with_near_pairs_is_bitwise_repeatable(pbm, torch_cuda):
    """Sites 0.45 A from the surface have several near (site, panel) pairs each (R-9); their corrections are added in a
    fixed order, so phi / grad / hess -- and with them the SCF and the energies -- repeat bit for bit."""
    from paper_1810_03698_b200.workloads import Workload, draw_sites, icosphere, make_config
    v, t = icosphere(4.0, 3)
    s = draw_sites(123, 60, 3.55, min_sep=0.5)
    w = Workload("near-sites", v, t, s, dict(eps_in=1.0, eps_out=80.0, kappa=0.125, K_far=7))
    ctx = pbm.from_workload(w, theta=0.5)
    ctx.tree_build()
    x = torch_cuda.from_numpy(np.random.Generator(np.random.PCG64(3)).normal(size=2 * t.shape[0])).cuda()
    first = [a.clone() for a in ctx.reaction_field(x)]
    for _ in range(5):
        again = ctx.reaction_field(x)
        assert all(torch_cuda.equal(a, b) for a, b in zip(first, again))
    ctx.close()
    w = make_config("C2")                                       # sites 1.2 A from a vdW mesh: near pairs, full solve
    runs = []
    for _ in range(2):
        ctx = pbm.from_workload(w)
        ctx.tree_build()
        xs, mu, res = ctx.solve()
        runs.append((xs.clone(), mu.clone(), res))
        ctx.close()
    assert torch_cuda.equal(runs[0][0], runs[1][0]) and torch_cuda.equal(runs[0][1], runs[1][1])
    assert runs[0][2]["dG_solv"] == runs[1][2]["dG_solv"]


def test_contexts_of_different_order_do_not_disturb_each_other(pbm, torch_cuda):
    """A binding triple is three live contexts on one device; the library's constant tables are the same bytes for
    every order and kappa, so a context built at P = 3, kappa = 0.3 between another's build and matvec changes nothing."""
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C1", subdiv=3)
    a = pbm.from_workload(w, theta=0.5, order_P=6)
    a.tree_build()
    x = torch_cuda.from_numpy(np.random.Generator(np.random.PCG64(1)).normal(size=2 * 1280)).cuda()
    y0 = a.matvec(x).clone()
    b = pbm.from_workload(w, theta=0.6, order_P=3, kappa=0.3)
    b.tree_build()
    yb0 = b.matvec(x).clone()
    y1 = a.matvec(x).clone()
    c = pbm.from_workload(w, theta=0.4, order_P=9, kappa=0.0)
    c.tree_build()
    c.matvec(x)
    assert torch_cuda.equal(y0, y1) and torch_cuda.equal(y0, a.matvec(x)) and torch_cuda.equal(yb0, b.matvec(x))
    for ctx in (a, b, c):
        ctx.close()


@pytest.mark.parametrize("P,bound", [(7, 4e-5), (8, 2e-5), (9, 1e-5), (10, 5e-6)])
def test_high_order_m2p_at_c2(pbm, po, torch_cuda, P, bound):
    """Orders 7-10 on BASELINE configs[2] (~9.6k panels, 150 target groups, hundreds of cells per list): against the
    oracle's direct sum, and the error must keep falling with P."""
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C2")
    nt = w.tris.shape[0]
    orc = po.Oracle(w.verts, w.tris, po.Params(K_far=w.params["K_far"]))
    x = np.random.Generator(np.random.PCG64(7)).normal(size=2 * nt)
    yref = np.concatenate(orc.matvec(x))
    ctx = pbm.from_workload(w, order_P=P)
    ctx.tree_build()
    st = ctx.stats()
    assert st["m2p_pairs"] > 0 and st["covered_pairs"] == nt * nt * w.params["K_far"]
    y = ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy()
    assert rel(y, yref) <= bound, rel(y, yref)
    ctx.close()


# ---- target sharding (S: section 8(e) / 8(f) item 4) on ONE GPU, rank after rank --------------------------------------
@pytest.mark.parametrize("name,kw,world", [("C1", dict(), 3), ("C2", dict(), 4), ("C1", dict(subdiv=1), 5)])
def test_target_sharding_is_the_same_matvec(pbm, torch_cuda, name, kw, world):
    """Every rank evaluates only its contiguous Morton range of target groups; the union of the owned rows is the
    unsharded result to rounding (a rank cuts its groups' lists into work items of its own size, so the partial sums
    of a row are grouped differently; the lists are the same), the ranks agree on the ranges, and the owned pair
    counts add up.  Then the exchange path (all-gather send buffer, un-permute kernel) with the
    collective replaced by a recorded one, against the layout of paper_1810_03698_b200/shard.py."""
    from paper_1810_03698_b200 import shard
    from paper_1810_03698_b200.workloads import make_config
    torch = torch_cuda
    w = make_config(name, **kw)
    nt = w.tris.shape[0]
    x = torch.from_numpy(np.random.Generator(np.random.PCG64(7)).normal(size=2 * nt)).cuda()
    ref = pbm.from_workload(w)
    ref.tree_build()
    y_ref = ref.matvec(x).clone()
    st_ref = ref.stats()
    ref.close()
    y = torch.full_like(x, float("nan"))
    ranges, pairs, sends = [], [0, 0], {}
    for r in range(world):
        ctx = pbm.from_workload(w)
        ctx.set_shard(r, world, exchange=False)
        ctx.tree_build()
        first = ctx.shard_ranges()
        ranges.append(first)
        before = torch.isnan(y).sum().item()
        ctx.matvec(x, out=y)                                    # writes the owned rows only
        assert before - torch.isnan(y).sum().item() == 2 * (first[r + 1] - first[r])
        st = ctx.stats()
        pairs[0] += st["p2p_pairs"]
        pairs[1] += st["m2p_pairs"]
        assert st["covered_pairs"] == st_ref["covered_pairs"]   # the lists themselves are whole on every rank
        ctx.close()
    assert all(np.array_equal(ranges[0], f) for f in ranges)
    first = ranges[0]
    assert first[0] == 0 and first[-1] == nt and np.all(np.diff(first) >= 0) and np.all(first[1:-1] % 64 == 0)
    assert pairs[0] == st_ref["p2p_pairs"] and pairs[1] == st_ref["m2p_pairs"]
    assert rel(y.cpu().numpy(), y_ref.cpu().numpy()) <= 1e-13 and not torch.isnan(y).any()
    # exchange path: pass 1 records every rank's send buffer, pass 2 hands the recorded buffers to rank 0's matvec
    for r in range(world):
        ctx = pbm.from_workload(w)

        def record(s, rbuf, r=r):
            sends[r] = s.clone()
            rbuf.zero_()
        ctx.set_shard(r, world, gather=record)
        ctx.tree_build()
        ctx.matvec(x)
        ctx.close()
    ctx = pbm.from_workload(w)

    def replay(s, rbuf):
        assert torch.equal(s, sends[0])
        rbuf.copy_(torch.cat([sends[r] for r in range(world)]))
    ctx.set_shard(0, world, gather=replay)
    ctx.tree_build()
    y_x = ctx.matvec(x).clone()
    ctx.close()
    assert torch.equal(y_x, y)                                  # exchanged result == union of the owned rows
    nmax = shard.nmax_of(first)
    assert all(sends[r].numel() == 2 * nmax for r in range(world))
    # the layout module describes the same thing: recover the Morton permutation from a matvec-free identity
    yall = torch.cat([sends[r] for r in range(world)]).cpu().numpy()
    blocks = yall.reshape(world, 2, nmax)
    got = np.sort(np.concatenate([blocks[r, 0, : first[r + 1] - first[r]] for r in range(world)]))
    assert np.array_equal(got, np.sort(y.cpu().numpy()[:nt]))   # the owned first rows, each exactly once
