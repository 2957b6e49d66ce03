"""Pins for the oracle's binding cycle, Eq. (25)-(27), against closed forms that
do not depend on the mesh: the vacuum leg is plain Coulomb / induction energy of point
multipoles, and the cycle must close (Eq. 25 = Eq. 27 + Eq. 26)."""
import numpy as np
import pytest

from paper_1810_03698_b200.workloads import icosphere

KCAL = 332.0636


def _two_spheres(d, radius=2.0, subdiv=1):
    v, t = icosphere(radius, subdiv)
    va, vb = v.copy(), v + np.array([d, 0.0, 0.0])
    return (va, t), (vb, t), (np.concatenate([va, vb]), np.concatenate([t, t + va.shape[0]]))


def _site(pos, q=0.0, dip=(0, 0, 0), alpha=0.0, group=0):
    return dict(pos=np.array([pos], dtype=float), q=np.array([float(q)]), dip=np.array([dip], dtype=float),
                quad=np.zeros((1, 6)), alpha=np.array([float(alpha)]), group=np.array([group], dtype=np.int32))


def _join(a, b):
    return {k: np.concatenate([a[k], b[k]]) for k in a}


def _solve(po, mesh, sites):
    orc = po.Oracle(mesh[0], mesh[1], po.Params(K_far=4))
    return orc.solve(po.Sites(**sites))


@pytest.mark.parametrize("q1,q2,d", [(1.0, -1.0, 8.0), (0.5, 0.7, 6.0)])
def test_vacuum_leg_is_coulomb_for_two_charges(po, q1, q2, d):
    """Eq. (26) with alpha = 0: G_AB - G_A - G_B = 332.0636 q1 q2 / (eps_in d), whatever the meshes."""
    ma, mb, mab = _two_spheres(d)
    sa, sb = _site((0, 0, 0), q=q1, group=0), _site((d, 0, 0), q=q2, group=1)
    cyc = po.binding_cycle(_solve(po, mab, _join(sa, sb)), _solve(po, ma, sa), _solve(po, mb, sb))
    assert cyc["dG_bind_vac"] == pytest.approx(KCAL * q1 * q2 / d, rel=1e-12)
    assert cyc["dG_bind_diss"] == pytest.approx(cyc["ddG_bind"] + cyc["dG_bind_vac"], rel=1e-12, abs=1e-12)


def test_vacuum_leg_includes_the_polarization_energy(po):
    """A charge q and a neutral polarizable site at distance d in vacuum: the induction energy is
    -alpha q^2 / (2 d^4) (Gaussian units, eps_in = 1) -- what Eq. (26) gives with W_pol, and what
    Eq. (24)'s G gives implicitly.  Dropping W_pol or using p = d + mu in Eq. (24)
    would double it; a wrong 4 pi in mu = alpha E (R-2) changes it 12.6x."""
    q, alpha, d = 1.0, 1.0, 7.0
    ma, mb, mab = _two_spheres(d)
    sa, sb = _site((0, 0, 0), q=q, group=0), _site((d, 0, 0), alpha=alpha, group=1)
    sol_ab = _solve(po, mab, _join(sa, sb))
    cyc = po.binding_cycle(sol_ab, _solve(po, ma, sa), _solve(po, mb, sb))
    assert cyc["dG_bind_vac"] == pytest.approx(-KCAL * alpha * q * q / (2 * d ** 4), rel=1e-6)
    mu_v = sol_ab["mu_vac"][1]
    np.testing.assert_allclose(mu_v, [alpha * q / d ** 2, 0.0, 0.0], rtol=1e-6, atol=1e-12)


def test_solvent_screens_the_interaction(po):
    """Two unit charges of opposite sign in separate small cavities, eps_out = 80, kappa = 0.125: in
    solvent the attraction is the linearised-PB (DLVO-like) screened Coulomb energy between two
    spheres of radius a, 332 q1 q2 e^{-kappa (d - 2a)} / (eps_out d (1 + kappa a)^2), to the accuracy of
    that far-field formula and of 80-panel spheres; in any case it is a small fraction of the vacuum
    -41.5 kcal/mol, and ddG_bind (Eq. 27) is the (positive) desolvation penalty that removes the rest."""
    d, a = 8.0, 2.0
    ma, mb, mab = _two_spheres(d, radius=a)
    sa, sb = _site((0, 0, 0), q=1.0, group=0), _site((d, 0, 0), q=-1.0, group=1)
    cyc = po.binding_cycle(_solve(po, mab, _join(sa, sb)), _solve(po, ma, sa), _solve(po, mb, sb))
    kappa, eps_out = 0.125, 80.0
    dlvo = -KCAL * np.exp(-kappa * (d - 2 * a)) / (eps_out * d * (1 + kappa * a) ** 2)
    assert cyc["dG_bind_vac"] == pytest.approx(-KCAL / d, rel=1e-12)
    assert cyc["ddG_bind"] > 0.9 * KCAL / d
    assert cyc["dG_bind_diss"] == pytest.approx(dlvo, rel=0.25)
    assert abs(cyc["dG_bind_diss"]) < 0.02 * KCAL / d
