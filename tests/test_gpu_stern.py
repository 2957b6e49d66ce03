"""Two nested surfaces / Stern layer on the GPU against oracle.SternOracle, which
tests/test_oracle_stern.py pins to the two-shell Kirkwood closed form: the block matvec in direct and treecode mode,
the right-hand side, the reaction field, and whole polarizable solves on the paper's sphere (R = 4 + 1 Angstrom Stern
layer, eps 4 / 80, kappa 0.125)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

R1, R2, E1, E2, E3, KAPPA = 4.0, 5.0, 4.0, 80.0, 80.0, 0.125


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


def _pair(po, pbm, subdiv, sites, K_far=7, eps_stern=E2, **over):
    from paper_1810_03698_b200.workloads import icosphere
    v1, t1 = icosphere(R1, subdiv)
    v2, t2 = icosphere(R2, subdiv)
    orc = po.SternOracle(v1, t1, v2, t2, po.Params(eps_in=E1, eps_out=E3, kappa=KAPPA, K_far=K_far), eps_stern=eps_stern)
    prm = dict(eps_in=E1, eps_out=E3, kappa=KAPPA, K_far=K_far, theta=0.5, order_P=6)
    prm.update(over)
    ctx = pbm.PB(0, **prm)
    ctx.mesh_load(orc.verts, orc.tris)
    ctx.sites_load(sites.pos, sites.q, sites.dip, sites.quad, sites.alpha, sites.group)
    ctx.set_stern(orc.n1, eps_stern)
    return orc, ctx


def _sites(po, n=12, seed=181003698 + 5000, alpha=1.0):
    from paper_1810_03698_b200.workloads import draw_sites
    return po.Sites(**draw_sites(seed, n, 0.7 * R1, min_sep=1.0, alpha=alpha))


def test_stern_matvec_rhs_and_reaction_field(pbm, po, torch_cuda):
    sites = _sites(po)
    orc, ctx = _pair(po, pbm, 3, sites, theta=0.0)
    n, n1 = orc.nt, orc.n1
    ctx.tree_build()
    x = np.random.Generator(np.random.PCG64(7)).normal(size=2 * n)
    y1, y2 = orc.matvec(x)
    yref = np.concatenate([y1, y2])
    y = ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy()
    for blk in (slice(0, n1), slice(n1, n), slice(n, n + n1), slice(n + n1, 2 * n)):     # every row block on its own
        assert rel(y[blk], yref[blk]) <= 1e-11
    mu = np.random.Generator(np.random.PCG64(4)).normal(0.0, 0.05, (sites.na, 3))
    b = ctx.rhs_multipole(torch_cuda.from_numpy(mu)).cpu().numpy()
    bref = orc.rhs(sites, mu)
    assert rel(b, bref) <= 1e-11 and np.all(b[n1:] == 0.0)
    got = [a.cpu().numpy() for a in ctx.reaction_field(torch_cuda.from_numpy(x))]
    for a, r in zip(got, orc.reaction(x, sites.pos)):
        assert rel(a, r) <= 1e-11
    ctx.set_params(theta=0.5, ncrit=64)
    ctx.tree_build()
    st = ctx.stats()
    assert st["m2p_pairs"] > 0 and st["covered_pairs"] == n * n * 7
    y = ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy()
    assert rel(y, yref) <= 1e-4 and rel(y[:n], yref[:n]) <= 1e-4 and rel(y[n:], yref[n:]) <= 1e-4
    assert np.array_equal(y, ctx.matvec(torch_cuda.from_numpy(x)).cpu().numpy())
    ctx.close()


@pytest.mark.parametrize("name", ["charge", "dipole", "quadrupole"])
def test_stern_sphere_against_oracle_and_two_shell_kirkwood(pbm, po, torch_cuda, name):
    """The paper's Stern-layer sphere with a centred unit multipole: GPU solve == oracle solve (same discrete system),
    both within the O(panel area) error of the two-shell closed form written out in tests/test_oracle_stern.py."""
    from test_oracle_stern import FOURPI, KCAL, SOURCES, _site, two_shell
    l, kw, s4, efac = SOURCES[name]
    dG_ref = efac * two_shell(l, s4 / (FOURPI * E1))[0] * FOURPI * KCAL
    site = _site(po, **kw)
    orc, ctx = _pair(po, pbm, 3, site, K_far=4, gmres_tol=1e-9)
    ctx.tree_build()
    x, mu, res = ctx.solve()
    ref = orc.solve(site)
    assert res["status"] == 0
    assert abs(res["dG_solv"] - ref["dG_solv"]) <= 1e-3 * abs(ref["dG_solv"])
    assert rel(x.cpu().numpy(), ref["x"]) <= 1e-3
    assert abs(res["dG_solv"] - dG_ref) <= 0.02 * abs(dG_ref)
    ctx.close()


def test_stern_polarizable_solve(pbm, po, torch_cuda):
    """12 AMOEBA-style polarizable sites (BASELINE configs[1]'s distributions) inside the Stern-layer sphere: every energy
    term, the induced dipoles and the SCF iteration count against the oracle, in treecode and in direct mode."""
    sites = _sites(po)
    orc, ctx = _pair(po, pbm, 3, sites)
    ref = orc.solve(sites)
    ctx.tree_build()
    x, mu, res = ctx.solve()
    assert res["status"] == 0 and res["scf_iters"] == ref["scf_iters"] and res["scf_iters_vac"] == ref["scf_iters_vac"]
    for k in ("dG_solv", "G_solvterm", "G_mult_diss", "G_vac"):
        assert abs(res[k] - ref[k]) <= 1e-3 * abs(ref[k]), k
    assert rel(mu.cpu().numpy(), ref["mu"]) <= 1e-4 and rel(x.cpu().numpy(), ref["x"]) <= 1e-3
    ctx.set_params(theta=0.0, gmres_tol=1e-11, scf_eta=0.0)    # every system of the loop to 1e-11: the oracle's SCF path
    ctx.tree_build()
    x, mu, res = ctx.solve()
    assert abs(res["dG_solv"] - ref["dG_solv"]) <= 1e-9 * abs(ref["dG_solv"])
    assert rel(mu.cpu().numpy(), ref["mu"]) <= 1e-8 and rel(x.cpu().numpy(), ref["x"]) <= 1e-8
    ctx.close()


def test_stern_validation(pbm, po, torch_cuda):
    from test_oracle_stern import _site
    orc, ctx = _pair(po, pbm, 2, _site(po, q=1.0))
    with pytest.raises(pbm.PBError):
        ctx.set_stern(orc.nt, E2)                              # n_inner must leave panels for Gamma_2
    with pytest.raises(pbm.PBError):
        ctx.set_stern(orc.n1, 0.0)
    ctx.set_stern(orc.n1, E2)
    s = _site(po, q=1.0, pos=(0.0, 0.0, 4.5))                  # inside Gamma_2 but in the Stern layer, not in region 1
    with pytest.raises(pbm.PBError) as e:                      # the check runs as soon as mesh, layer and sites are known
        ctx.sites_load(s.pos, s.q, s.dip, s.quad, s.alpha, s.group)
    assert e.value.code == -2 and "outside" in str(e.value)
    ctx.set_stern(0, 0.0)                                      # one surface (the union's outer sphere ... and the inner one):
    ctx.sites_load(s.pos, s.q, s.dip, s.quad, s.alpha, s.group)   # the same site is inside the closed union surface
    ctx.close()
