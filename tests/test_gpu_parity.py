"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element on the
same seeded inputs.  Tolerances are BASELINE.json's: direct mode (theta = 0) <= 1e-11 relative
L2; treecode (theta = 0.5, P = 6) <= 1e-4 on the matvec and <= 1e-3 on the solvation energy."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_DIRECT = 1e-11
TOL_TREE = 1e-4
TOL_ENERGY = 1e-3


def rel(a, b):
    """Relative error in BOTH norms, the larger of the two: ||a - b||_2 / ||b||_2 (BASELINE.json's stated norm) and
    max|a - b| / max|b| (so that one bad row among 10^4-10^6 cannot hide under the L2 bound).  Rounding-level
    comparisons (direct mode, <= 1e-11) take the max norm at face value.  For truncation-level ones (treecode) the
    max norm is allowed ten times the L2 bound: the far-field error of a row is set by the few cells nearest the MAC
    limit and is far from uniform over the rows -- measured with BASELINE.json's theta = 0.5, P = 6 against the
    direct sum: L2 3.0e-5 and max norm 3.1e-4 of max|y| over the 1.2e5 rows of C3, 4.5e-4 over the 2.1e6 rows of C4,
    with every cell at order 6 as well as with the variable order (R-31).  BASELINE.json's 1e-4 is stated
    for the L2 norm."""
    a, b = np.asarray(a, dtype=float), np.asarray(b, dtype=float)
    d = a - b
    l2 = float(np.linalg.norm(d) / np.linalg.norm(b))
    linf = float(np.max(np.abs(d)) / np.max(np.abs(b))) if d.size else 0.0
    return max(l2, linf if l2 < 1e-9 else 0.1 * linf)


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


def _setup(pbm, po, w, **over):
    orc = po.Oracle(w.verts, w.tris, po.Params(K_far=w.params["K_far"], **{k: v for k, v in over.items()
                                                                          if k in ("kappa", "near_tau", "eps_in", "eps_out")}))
    ctx = pbm.from_workload(w, **over)
    return orc, po.Sites(**w.sites), ctx


def _xvec(n, seed=7):
    return np.random.Generator(np.random.PCG64(seed)).normal(size=2 * n)


# ---- matvec, direct mode: the oracle's operator to rounding -------------------------------------
@pytest.mark.parametrize("name,kw", [
    ("C0", dict(kind="charge")),                  # 320 panels, K=4: 5 target groups
    ("C0", dict(kind="charge", subdiv=0)),        # 20 panels: one ragged group, single-cell tree
    ("C0", dict(kind="charge", subdiv=1)),        # 80 panels: ragged tail (80 = 64 + 16)
    ("C1", dict(subdiv=3)),                       # 1280 panels, K=7
    ("C1", dict()),                               # 5120 panels, K=7 (BASELINE configs[1])
])
def test_matvec_direct(pbm, po, torch_cuda, name, kw):
    from paper_1810_03698_b200.workloads import make_config
    w = make_config(name, **kw)
    orc, _, ctx = _setup(pbm, po, w, theta=0.0)
    ctx.tree_build()
    x = _xvec(orc.nt)
    y = ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy()
    y1, y2 = orc.matvec(x)
    n = orc.nt
    assert rel(y, np.concatenate([y1, y2])) <= TOL_DIRECT
    assert rel(y[:n], y1) <= TOL_DIRECT and rel(y[n:], y2) <= TOL_DIRECT
    ctx.close()


@pytest.mark.parametrize("K_far", [1, 3, 4, 7])
def test_matvec_direct_every_far_rule(pbm, po, torch_cuda, K_far):
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C0", kind="charge")
    w.params["K_far"] = K_far
    orc, _, ctx = _setup(pbm, po, w, theta=0.0)
    ctx.tree_build()
    x = _xvec(orc.nt, 11)
    y = ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy()
    assert rel(y, np.concatenate(orc.matvec(x))) <= TOL_DIRECT
    ctx.close()


def test_matvec_direct_irregular_mesh_and_kappa_zero(pbm, po, torch_cuda):
    """A van-der-Waals-union surface (slivers, varying areas: exercises the NEAR / ADJ
    classification away from the icosphere's symmetry), also with kappa = 0 (Yukawa == Laplace)."""
    from paper_1810_03698_b200.workloads import Workload, random_chain_globule, seed_for, vdw_surface
    g = random_chain_globule(seed_for(2), 120)
    v, t, _ = vdw_surface(g["pos"], g["radii"], target_panels=2500)
    sites = {k: g[k] for k in ("pos", "q", "dip", "quad", "alpha", "group")}
    for kappa in (0.125, 0.0):
        w = Workload("mini-globule", v, t, sites, dict(eps_in=1.0, eps_out=80.0, kappa=kappa, K_far=7))
        orc, _, ctx = _setup(pbm, po, w, theta=0.0, kappa=kappa)
        ctx.tree_build()
        x = _xvec(orc.nt, 3)
        y = ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy()
        y1, y2 = orc.matvec(x)
        assert rel(y, np.concatenate([y1, y2])) <= TOL_DIRECT
        st = ctx.stats()
        assert st["near_entries"] > 13 * orc.nt          # SELF + ~12 ADJ + NEAR per target
        ctx.close()


# ---- matvec, treecode mode ------------------------------------------------------------------------
@pytest.mark.parametrize("name,kw", [("C0", dict(kind="charge")), ("C1", dict(subdiv=3)), ("C1", dict())])
def test_matvec_treecode(pbm, po, torch_cuda, name, kw):
    from paper_1810_03698_b200.workloads import make_config
    w = make_config(name, **kw)
    orc, _, ctx = _setup(pbm, po, w, theta=0.5, order_P=6)
    ctx.tree_build()
    x = _xvec(orc.nt)
    yref = np.concatenate(orc.matvec(x))
    y = ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy()
    n = orc.nt
    assert rel(y, yref) <= TOL_TREE and rel(y[:n], yref[:n]) <= TOL_TREE and rel(y[n:], yref[n:]) <= TOL_TREE
    st = ctx.stats()
    if orc.nt >= 1280:
        assert st["m2p_pairs"] > 0 and st["p2p_pairs"] < orc.nt * orc.nt * w.params["K_far"]
    ctx.close()


def test_treecode_error_falls_with_P_and_theta_and_ncrit_ragged(pbm, po, torch_cuda):
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C1", subdiv=3)
    orc, _, ctx = _setup(pbm, po, w, theta=0.5)
    x = _xvec(orc.nt, 5)
    yref = np.concatenate(orc.matvec(x))
    errs = []
    for P in (2, 4, 6, 8, 10):
        ctx.set_params(theta=0.5, order_P=P, ncrit=50)       # ncrit not a multiple of K: ragged leaves
        ctx.tree_build()
        errs.append(rel(ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy(), yref))
    assert all(errs[i + 1] < 0.35 * errs[i] for i in range(4)), errs
    e_theta = []
    for theta in (0.7, 0.5, 0.3):
        ctx.set_params(theta=theta, order_P=6, ncrit=64)
        ctx.tree_build()
        e_theta.append(rel(ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy(), yref))
    assert e_theta[0] > e_theta[1] > e_theta[2], e_theta
    ctx.set_params(theta=1e-3, order_P=2)                      # theta -> 0: nothing is accepted
    ctx.tree_build()
    assert ctx.stats()["m2p_pairs"] == 0
    assert rel(ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy(), yref) <= TOL_DIRECT
    ctx.close()


@pytest.mark.parametrize("target_panels,tail", [(2500, 40), (3500, 16)])
def test_split_and_whole_group_lists(pbm, po, torch_cuda, target_panels, tail):
    """pb_params.list_split: the two 32-target halves of a group take the MAC decisions of Eq. (28) separately (1) or
    together (0).  Either way the stored lists cover every (target, source point) pair exactly once (counted from the
    lists with their half masks), the matvec stays within the treecode bound of the oracle's dense product, and the
    split lists evaluate fewer pairs.  The meshes end in a ragged group whose second half is partly filled (N % 64 = 40)
    or empty (16)."""
    from paper_1810_03698_b200.workloads import Workload, random_chain_globule, seed_for, vdw_surface
    g = random_chain_globule(seed_for(2), 120)
    v, t, _ = vdw_surface(g["pos"], g["radii"], target_panels=target_panels)
    assert t.shape[0] % 64 == tail
    sites = {k: g[k] for k in ("pos", "q", "dip", "quad", "alpha", "group")}
    w = Workload("mini-globule", v, t, sites, dict(eps_in=1.0, eps_out=80.0, kappa=0.125, K_far=7))
    orc, _, ctx = _setup(pbm, po, w, theta=0.5, order_P=6, ncrit=40)
    x = _xvec(orc.nt, 9)
    yref = np.concatenate(orc.matvec(x))
    st, ys = {}, {}
    for split in (0, 1):
        ctx.set_params(list_split=split)
        ctx.tree_build()
        ys[split] = ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy()
        st[split] = ctx.stats()
        assert st[split]["covered_pairs"] == orc.nt * orc.nt * 7
        assert rel(ys[split], yref) <= TOL_TREE
    assert st[0]["p2p_pairs_half"] == 0 and st[0]["m2p_pairs_half"] == 0
    assert st[1]["p2p_pairs_half"] > 0 and st[1]["m2p_pairs_half"] > 0
    assert st[1]["p2p_pairs"] < st[0]["p2p_pairs"]
    assert st[1]["p2p_pairs"] + 8 * st[1]["m2p_pairs"] < st[0]["p2p_pairs"] + 8 * st[0]["m2p_pairs"]
    # the same decisions rule in direct mode (one range for everything, no masks to honour)
    ctx.set_params(theta=0.0, list_split=1)
    ctx.tree_build()
    assert rel(ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy(), yref) <= TOL_DIRECT
    ctx.close()


def test_matvec_is_linear_and_independent_of_sites(pbm, po, torch_cuda):
    """The charge description enters only the RHS and the energy."""
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C1", subdiv=3)
    _, _, ctx = _setup(pbm, po, w, theta=0.5)
    ctx.tree_build()
    x1, x2 = _xvec(1280, 1), _xvec(1280, 2)
    y1 = ctx.matvec(torch_cuda.from_numpy(x1)).clone()
    y2 = ctx.matvec(torch_cuda.from_numpy(x2)).clone()
    y12 = ctx.matvec(torch_cuda.from_numpy(2.0 * x1 - 3.0 * x2))
    assert rel((2.0 * y1 - 3.0 * y2).cpu().numpy(), y12.cpu().numpy()) < 1e-13
    s = {k: (v * 2 if k in ("q", "dip", "quad") else v) for k, v in w.sites.items()}
    ctx.sites_load(s["pos"] * 0.5, s["q"], s["dip"], s["quad"], s["alpha"], s["group"])
    y1b = ctx.matvec(torch_cuda.from_numpy(x1))
    assert torch_cuda.equal(y1, y1b)                           # bit-identical: deterministic, site-free
    # host-buffer entry point gives the same result
    yh = np.zeros_like(x1)
    ctx.matvec_host(x1, yh)
    assert np.array_equal(yh, y1.cpu().numpy())
    ctx.close()


# ---- right-hand side, reaction field, multipole field ----------------------------------------------
def test_rhs_reaction_multipole_fields(pbm, po, torch_cuda):
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C1", subdiv=3)
    orc, sites, ctx = _setup(pbm, po, w, theta=0.5)
    ctx.tree_build()
    rng = np.random.Generator(np.random.PCG64(9))
    mu = rng.normal(size=(sites.na, 3)) * 0.1
    assert rel(ctx.rhs_multipole(None).cpu().numpy(), orc.rhs(sites)) <= TOL_DIRECT
    b = ctx.rhs_multipole(mu).cpu().numpy()
    assert rel(b, orc.rhs(sites, mu)) <= TOL_DIRECT and np.all(b[orc.nt:] == 0.0)
    x = _xvec(orc.nt, 13)
    pr, gr, hr = orc.reaction(x, sites.pos)
    ph, g, h = ctx.reaction_field(torch_cuda.from_numpy(x))
    assert rel(ph.cpu().numpy(), pr) <= TOL_DIRECT and rel(g.cpu().numpy(), gr) <= TOL_DIRECT
    assert rel(h.cpu().numpy(), hr) <= TOL_DIRECT
    ph, g, _ = ctx.reaction_field(torch_cuda.from_numpy(x), want_hess=False)
    assert rel(ph.cpu().numpy(), pr) <= TOL_DIRECT and rel(g.cpu().numpy(), gr) <= TOL_DIRECT
    for mask in (True, False):
        for m in (None, mu):
            pr, gr, hr = orc.multipole_field(sites, m, mask)
            ph, g, h = ctx.multipole_field(m, use_mask=mask)
            assert rel(ph.cpu().numpy(), pr) <= TOL_DIRECT and rel(g.cpu().numpy(), gr) <= TOL_DIRECT
            assert rel(h.cpu().numpy(), hr) <= TOL_DIRECT
    ctx.close()


def test_fields_with_groups_thole_and_sites_near_the_surface(pbm, po, torch_cuda):
    """Grouped sites (mask active), mixed polarizabilities (Thole on/off), and sites close enough
    to the surface that the reaction field switches panels to the K_near rule (D: R-9)."""
    from paper_1810_03698_b200.workloads import Workload, draw_sites, icosphere
    v, t = icosphere(4.0, 2)
    s = draw_sites(123, 37, 3.55, min_sep=0.6)               # up to 0.45 A from the sphere: tau*sqrt(A) = 1.6
    s["group"] = (np.arange(37) // 4).astype(np.int32)
    s["alpha"] = np.where(np.arange(37) % 3 == 0, 0.0, 0.5 + 0.05 * np.arange(37))
    w = Workload("near-sites", v, t, s, dict(eps_in=1.0, eps_out=80.0, kappa=0.125, K_far=4))
    orc, sites, ctx = _setup(pbm, po, w, theta=0.5)
    ctx.tree_build()
    x = _xvec(orc.nt, 17)
    pr, gr, hr = orc.reaction(x, sites.pos)
    ph, g, h = ctx.reaction_field(torch_cuda.from_numpy(x))
    assert rel(ph.cpu().numpy(), pr) <= TOL_DIRECT and rel(g.cpu().numpy(), gr) <= TOL_DIRECT
    assert rel(h.cpu().numpy(), hr) <= TOL_DIRECT
    mu = np.random.Generator(np.random.PCG64(4)).normal(size=(37, 3)) * 0.2
    for mask in (True, False):
        pr, gr, hr = orc.multipole_field(sites, mu, mask)
        ph, g, h = ctx.multipole_field(mu, use_mask=mask)
        assert rel(ph.cpu().numpy(), pr) <= TOL_DIRECT and rel(g.cpu().numpy(), gr) <= TOL_DIRECT
        assert rel(h.cpu().numpy(), hr) <= TOL_DIRECT
    pm, gm, _ = orc.multipole_field(sites, mu, True)
    pu, gu, _ = orc.multipole_field(sites, mu, False)
    assert rel(gm, gu) > 1e-3                                  # the mask really is exercised
    ctx.close()


# ---- GMRES and the full polarizable solve -----------------------------------------------------------
def test_gmres_matches_dense_lu(pbm, po, torch_cuda):
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C1", subdiv=3)
    orc, sites, ctx = _setup(pbm, po, w, theta=0.0, gmres_tol=1e-11)
    ctx.tree_build()
    b = orc.rhs(sites)
    xl = orc.solve_linear(b)
    for precond in (1, 0):
        ctx.set_params(precond=precond, theta=0.0)
        ctx.tree_build()
        x, info = ctx.gmres(torch_cuda.from_numpy(b))
        assert info["converged"] and info["relres"] <= 1e-11
        assert rel(x.cpu().numpy(), xl) <= 1e-8
    ctx.set_params(gmres_restart=7, precond=1)                 # restarts + warm start path
    ctx.tree_build()
    x, info = ctx.gmres(torch_cuda.from_numpy(b))
    assert info["converged"] and rel(x.cpu().numpy(), xl) <= 1e-8
    bt = torch_cuda.from_numpy(b).cuda()
    true_res = float((bt - ctx.matvec(x)).norm() / bt.norm())
    assert true_res <= 1.05e-11 and abs(true_res - info["relres"]) <= 1e-13      # the Arnoldi residual IS the true one
    ctx.set_params(gmres_tol=2e-11)
    x2, info2 = ctx.gmres(torch_cuda.from_numpy(b), x0=x)
    assert info2["iters"] == 0 and torch_cuda.equal(x, x2)                       # warm start from a converged x
    ctx.set_params(gmres_tol=1e-11)
    xz, infoz = ctx.gmres(torch_cuda.zeros_like(x))
    assert infoz["iters"] == 0 and float(xz.abs().max()) == 0.0
    ctx.close()


def _golden():
    import os
    out = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "kirkwood_sphere.txt")):
        if line.startswith("#") or not line.strip():
            continue
        f = line.split()
        out[f[0]] = float(f[1])
    return out


@pytest.mark.parametrize("kind", ["charge", "dipole", "quadrupole", "polarizable_dipole"])
def test_solve_c0_against_oracle_and_kirkwood(pbm, po, torch_cuda, kind):
    """BASELINE configs[0]: the GPU solve must equal the oracle's (same discrete operator) and sit
    within the BEM discretisation error of Kirkwood's closed form (tests/golden)."""
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C0", kind=kind)
    orc, sites, ctx = _setup(pbm, po, w, theta=0.5, gmres_tol=1e-10)
    ctx.tree_build()
    x, mu, res = ctx.solve()
    ref = orc.solve(sites)
    assert res["status"] == 0
    assert abs(res["dG_solv"] - ref["dG_solv"]) <= TOL_ENERGY * abs(ref["dG_solv"])
    assert rel(x.cpu().numpy(), ref["x"]) <= TOL_TREE
    assert abs(res["dG_solv"] - _golden()[kind]) <= 0.08 * abs(_golden()[kind])   # 320-panel mesh: O(A) error
    if kind == "polarizable_dipole":
        # the SCF loop's systems are solved inexactly (pb_params.scf_eta) and the loop ends only on a step solved to
        # gmres_tol: at most one step more than the oracle's loop of exact solves
        assert 0 <= res["scf_iters"] - ref["scf_iters"] <= 1
        assert rel(mu.cpu().numpy(), ref["mu"]) <= 1e-5
        ctx.set_params(scf_eta=0.0)                            # every system to gmres_tol: the oracle's path step by step
        x, mu, res = ctx.solve()
        assert res["scf_iters"] == ref["scf_iters"] and rel(mu.cpu().numpy(), ref["mu"]) <= 1e-5
        assert abs(res["dG_solv"] - ref["dG_solv"]) <= TOL_ENERGY * abs(ref["dG_solv"])
    ctx.close()


def test_solve_c1_small_polarizable(pbm, po, torch_cuda):
    """12 polarizable AMOEBA-style sites (BASELINE configs[1] at subdivision 3): treecode solve vs
    oracle on every energy term, the induced dipoles and the SCF iteration count; then direct mode."""
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C1", subdiv=3)
    orc, sites, ctx = _setup(pbm, po, w)
    ref = orc.solve(sites)
    ctx.tree_build()
    x, mu, res = ctx.solve()
    assert res["status"] == 0 and res["scf_iters"] == ref["scf_iters"] and res["scf_iters_vac"] == ref["scf_iters_vac"]
    for k in ("dG_solv", "G_solvterm", "G_mult_diss", "G_vac"):
        assert abs(res[k] - ref[k]) <= TOL_ENERGY * abs(ref[k]), k
    assert rel(mu.cpu().numpy(), ref["mu"]) <= 1e-4
    assert rel(x.cpu().numpy(), ref["x"]) <= 1e-3
    assert res["final_scf_delta_debye"] < 1e-7
    # direct mode, every system of the loop solved to 1e-11 (scf_eta = 0): the same SCF path as the oracle's dense LU, so
    # the two stop at the same step and agree far below the SCF tolerance itself
    ctx.set_params(theta=0.0, gmres_tol=1e-11, scf_eta=0.0)
    ctx.tree_build()
    x, mu, res = ctx.solve()
    assert res["scf_iters"] == ref["scf_iters"]
    assert abs(res["dG_solv"] - ref["dG_solv"]) <= 1e-9 * abs(ref["dG_solv"])
    assert rel(mu.cpu().numpy(), ref["mu"]) <= 1e-8 and rel(x.cpu().numpy(), ref["x"]) <= 1e-8
    # the three ways the loop's systems can share work (pb_params.scf_recycle) and the inexact solves (scf_eta) reach
    # the same fixed point: differences of the order of the SCF tolerance (1e-7 D on dipoles of ~0.1 D), not more
    dG = {}
    for rec, eta in ((0, 0.0), (1, 0.0), (2, 0.0), (2, 0.03), (2, 0.1)):
        ctx.set_params(scf_recycle=rec, scf_eta=eta)
        xr, mur, rr = ctx.solve()
        assert rr["status"] == 0 and abs(rr["scf_iters"] - ref["scf_iters"]) <= 2, (rec, eta, rr["scf_iters"])
        assert abs(rr["dG_solv"] - ref["dG_solv"]) <= 2e-8 * abs(ref["dG_solv"]), (rec, eta)
        assert rel(mur.cpu().numpy(), ref["mu"]) <= 2e-6 and rel(xr.cpu().numpy(), ref["x"]) <= 1e-7, (rec, eta)
        dG[(rec, eta)] = rr["matvecs_total"]
    assert dG[(2, 0.03)] < dG[(1, 0.0)] < dG[(0, 0.0)], dG      # operator applications: fewer with every level of sharing
    # a store too small for the loop (1 MiB = 25 directions of 2 x 20 KB here; the loop needs more): restarted GMRES takes
    # over where the stored directions end, same fixed point
    ctx.set_params(scf_recycle=2, scf_eta=0.03, scf_store_mb=1)
    xr, mur, rr = ctx.solve()
    assert rr["status"] == 0 and rr["matvecs_total"] > 25 and abs(rr["scf_iters"] - ref["scf_iters"]) <= 2
    assert abs(rr["dG_solv"] - ref["dG_solv"]) <= 2e-8 * abs(ref["dG_solv"]) and rel(mur.cpu().numpy(), ref["mu"]) <= 2e-6
    ctx.set_params(scf_store_mb=0)                             # no store at all
    xr, mur, rr = ctx.solve()
    assert rr["status"] == 0 and abs(rr["dG_solv"] - ref["dG_solv"]) <= 2e-8 * abs(ref["dG_solv"])
    ctx.set_params(scf_recycle=2, scf_eta=0.0, scf_store_mb=16384)
    x, mu, res = ctx.solve()
    xh = torch_cuda.empty(2 * orc.nt, dtype=torch_cuda.float64).pin_memory()
    muh = torch_cuda.empty(sites.na, 3, dtype=torch_cuda.float64).pin_memory()
    resh = ctx.solve_host(xh, muh)
    assert resh["dG_solv"] == res["dG_solv"] and np.array_equal(xh.numpy(), x.cpu().numpy())
    ctx.close()


def test_iteration_limits_are_reported_not_hidden(pbm, po, torch_cuda):
    """PB_ERR_NO_CONVERGENCE (results still set, include/pb.h): a GMRES / GCR limit too small for the first system and an
    SCF limit too small for the loop, in each of the three ways the loop's systems share work."""
    from paper_1810_03698_b200.workloads import make_config
    w = make_config("C1", subdiv=3)
    ok = pbm.from_workload(w)
    ok.tree_build()
    _, _, good = ok.solve()
    ok.close()
    assert good["status"] == 0 and good["scf_iters"] > 5
    for rec in (0, 1, 2):
        ctx = pbm.from_workload(w, gmres_maxit=2, scf_recycle=rec, scf_maxit=4)
        ctx.tree_build()
        x, mu, res = ctx.solve()
        assert res["status"] == -6 and res["final_gmres_relres"] > 1e-6, (rec, res)
        assert bool(torch_cuda.isfinite(x).all()) and bool(torch_cuda.isfinite(mu).all()) and np.isfinite(res["dG_solv"])
        ctx.close()
        ctx = pbm.from_workload(w, scf_recycle=rec, scf_maxit=3)
        ctx.tree_build()
        x, mu, res = ctx.solve()
        assert res["status"] == -6 and res["scf_iters"] == 3 and res["final_scf_delta_debye"] > 1e-7, (rec, res)
        assert res["final_gmres_relres"] <= 1e-6 or rec == 2        # (mode 2 solves early systems inexactly on purpose)
        assert abs(res["dG_solv"] - good["dG_solv"]) <= 0.05 * abs(good["dG_solv"])
        ctx.close()


# ---- boundary behaviour ------------------------------------------------------------------------------
def test_error_codes_and_call_order(pbm, torch_cuda):
    from paper_1810_03698_b200.workloads import icosphere
    ctx = pbm.PB(0)
    with pytest.raises(pbm.PBError) as e:
        ctx.tree_build()
    assert e.value.code == -3                                  # PB_ERR_NOT_READY
    v, t = icosphere(4.0, 1)
    bad = t.copy()
    bad[5] = [bad[5][0], bad[5][0], bad[5][1]]                 # zero-area panel
    with pytest.raises(pbm.PBError) as e:
        ctx.mesh_load(v, bad)
    assert e.value.code == -2                                  # PB_ERR_BAD_MESH
    bad = t.copy()
    bad[0, 0] = 10_000
    with pytest.raises(pbm.PBError) as e:
        ctx.mesh_load(v, bad)
    assert e.value.code == -2
    with pytest.raises(pbm.PBError) as e:
        ctx.set_params(theta=1.5)
    assert e.value.code == -1                                  # PB_ERR_INVALID_ARG
    with pytest.raises(pbm.PBError):
        ctx.set_params(K_far=5)
    ctx.mesh_load(v, t)
    ctx.nt = 80
    with pytest.raises(pbm.PBError) as e:
        ctx.matvec(torch_cuda.zeros(160, dtype=torch_cuda.float64, device="cuda"))
    assert e.value.code == -3                                  # tree not built
    ctx.tree_build()
    with pytest.raises(pbm.PBError) as e:
        ctx.na = 1
        ctx.reaction_field(torch_cuda.zeros(160, dtype=torch_cuda.float64, device="cuda"))
    assert e.value.code == -3                                  # sites not loaded
    y = ctx.matvec(torch_cuda.zeros(160, dtype=torch_cuda.float64, device="cuda"))
    assert float(y.abs().max()) == 0.0
    ctx.set_params(gmres_maxit=2, gmres_tol=1e-14)
    ctx.tree_build()
    _, info = ctx.gmres(torch_cuda.ones(160, dtype=torch_cuda.float64, device="cuda"))
    assert not info["converged"] and info["iters"] == 2        # PB_ERR_NO_CONVERGENCE, results still set
    ctx.close()


def test_near_field_preconditioner(pbm, po, torch_cuda):
    """precond = 2: flexible GMRES with two minimal-residual steps on the sparse near-field matrix.  Same solution
    as block-Jacobi and as the oracle's dense LU, the reported residual is the true one, fewer iterations."""
    from paper_1810_03698_b200.workloads import Workload, random_chain_globule, seed_for, vdw_surface
    g = random_chain_globule(seed_for(2), 120)
    v, t, _ = vdw_surface(g["pos"], g["radii"], target_panels=2500)
    sites = {k: g[k] for k in ("pos", "q", "dip", "quad", "alpha", "group")}
    w = Workload("mini-globule", v, t, sites, dict(eps_in=1.0, eps_out=80.0, kappa=0.125, K_far=7))
    orc, s, ctx = _setup(pbm, po, w, theta=0.0, gmres_tol=1e-10)
    ctx.tree_build()
    b = orc.rhs(s)
    xl = orc.solve_linear(b)
    bt = torch_cuda.from_numpy(b).cuda()
    iters = {}
    for precond in (1, 2):
        ctx.set_params(precond=precond)
        x, info = ctx.gmres(bt)
        assert info["converged"] and info["relres"] <= 1e-10
        true_res = float((bt - ctx.matvec(x)).norm() / bt.norm())
        assert abs(true_res - info["relres"]) <= 1e-12
        assert rel(x.cpu().numpy(), xl) <= 1e-7
        iters[precond] = info["iters"]
    assert iters[2] < 0.8 * iters[1]
    ctx.set_params(precond=2, gmres_restart=9)               # restarts in the flexible variant
    x, info = ctx.gmres(bt)
    assert info["converged"] and rel(x.cpu().numpy(), xl) <= 1e-7
    ctx.set_params(precond=2, gmres_restart=200, theta=0.5, gmres_tol=1e-6)   # a whole polarizable solve through it
    ctx.tree_build()
    _, mu, res = ctx.solve()
    ref = orc.solve(s)
    assert res["status"] == 0 and abs(res["dG_solv"] - ref["dG_solv"]) <= 1e-3 * abs(ref["dG_solv"])
    assert rel(mu.cpu().numpy(), ref["mu"]) <= 1e-4
    ctx.close()
