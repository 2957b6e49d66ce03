"""Pins 11-12 of DESIGN section 5: derivative tensors (Eq. 29-32 as corrected in App. A.2,
Thole damping App. A.5) by central finite differences, mask semantics, and the SOR
self-consistent loop against a direct linear solve."""
import numpy as np
import pytest

FOURPI = 4 * np.pi


def _random_sites(po, rng, n, alpha=1.0, spread=2.0, groups=None):
    pos = []
    while len(pos) < n:
        p = rng.uniform(-spread, spread, 3)
        if all(np.linalg.norm(p - o) > 1.0 for o in pos):
            pos.append(p)
    quad = rng.normal(0, 0.3, (n, 6))
    tr = (quad[:, 0] + quad[:, 3] + quad[:, 5]) / 3
    quad[:, [0, 3, 5]] -= tr[:, None]
    return po.Sites(pos=np.array(pos), q=rng.uniform(-0.5, 0.5, n), dip=rng.normal(0, 0.2, (n, 3)), quad=quad,
                    alpha=np.full(n, alpha), group=np.arange(n) if groups is None else groups)


def _field_at(po, o, s, mu, point, use_mask=False, probe_alpha=1.0, probe_group=-1):
    """Potential of all sites of `s` at an arbitrary point, through the oracle itself: append a
    zero-moment probe site there and read its row."""
    n = s.na
    s2 = po.Sites(pos=np.vstack([s.pos, point]), q=np.append(s.q, 0.0), dip=np.vstack([s.dip, np.zeros(3)]),
                  quad=np.vstack([s.quad, np.zeros(6)]), alpha=np.append(s.alpha, probe_alpha),
                  group=np.append(s.group, probe_group))
    mu2 = None if mu is None else np.vstack([mu, np.zeros(3)])
    phi, g, h = o.multipole_field(s2, mu2, use_mask)
    return phi[n], g[n], h[n]


def _h6(h):
    return np.array([[h[0], h[1], h[2]], [h[1], h[3], h[4]], [h[2], h[4], h[5]]])


@pytest.mark.parametrize("with_mu", [False, True])
def test_multipole_field_derivatives_by_finite_differences(po, sphere_oracles, with_mu):
    """grad and hess of Eq. (7) (+ Thole-damped induced dipoles) are the central differences
    of phi and grad (h = 1e-4, rel 1e-7): pins Eq. (31)-(32) corrections and App. A.5."""
    o = sphere_oracles(1)
    rng = np.random.default_rng(11)
    s = _random_sites(po, rng, 5)
    mu = rng.normal(0, 0.1, (5, 3)) if with_mu else None
    if with_mu:   # isolate the damped part too
        s = po.Sites(pos=s.pos, q=0 * s.q, dip=0 * s.dip, quad=0 * s.quad, alpha=s.alpha, group=s.group)
    x0 = np.array([0.35, -0.2, 0.15])      # close to the sources so damping is active
    hstep = 2e-3
    phi0, g0, h0 = _field_at(po, o, s, mu, x0)
    gfd = np.zeros(3)
    hfd = np.zeros((3, 3))
    for k in range(3):          # 4th-order central differences
        e = np.zeros(3)
        e[k] = hstep
        vals = {m: _field_at(po, o, s, mu, x0 + m * e) for m in (-2, -1, 1, 2)}
        gfd[k] = (-vals[2][0] + 8 * vals[1][0] - 8 * vals[-1][0] + vals[-2][0]) / (12 * hstep)
        hfd[:, k] = (-vals[2][1] + 8 * vals[1][1] - 8 * vals[-1][1] + vals[-2][1]) / (12 * hstep)
    np.testing.assert_allclose(g0, gfd, rtol=1e-7, atol=1e-8 * np.abs(g0).max())
    np.testing.assert_allclose(_h6(h0), hfd, rtol=1e-7, atol=1e-7 * np.abs(h0).max())
    assert abs(np.trace(_h6(h0))) < 1e-12 * np.abs(h0).max() or with_mu   # undamped Coulomb is harmonic


def test_multipole_potential_terms_against_explicit_formula(po, sphere_oracles):
    """Eq. (7): phi = (1/4 pi eps)[q/R + p.d/R^3 + Q_ij d_i d_j/(2R^5)] for one source, typed
    out with a full 3x3 Q, eps_in = 2 -> also pins the 1/eps_in and the 6-vector ordering."""
    o = po.Oracle(sphere_oracles(1).verts, sphere_oracles(1).tris, po.Params(K_far=4, eps_in=2.0))
    Qm = np.array([[0.3, -0.2, 0.5], [-0.2, 0.1, 0.7], [0.5, 0.7, -0.4]])
    s = po.Sites(pos=[[0.1, 0.2, -0.3]], q=[0.7], dip=[[0.2, -0.1, 0.4]],
                 quad=[[Qm[0, 0], Qm[0, 1], Qm[0, 2], Qm[1, 1], Qm[1, 2], Qm[2, 2]]], alpha=[0.0], group=[0])
    x = np.array([1.3, -0.8, 0.9])
    d = x - s.pos[0]
    Rr = np.linalg.norm(d)
    ref = (0.7 / Rr + s.dip[0] @ d / Rr ** 3 + d @ Qm @ d / (2 * Rr ** 5)) / (FOURPI * 2.0)
    phi, _, _ = _field_at(po, o, s, None, x)
    assert abs(phi - ref) < 1e-15 + 1e-14 * abs(ref)
    b = o.rhs(s)
    i = 3
    d = o.cen[i] - s.pos[0]
    Rr = np.linalg.norm(d)
    ref = (0.7 / Rr + s.dip[0] @ d / Rr ** 3 + d @ Qm @ d / (2 * Rr ** 5)) / (FOURPI * 2.0)
    assert abs(b[i] - ref) < 1e-14 * abs(ref)


def test_thole_limits_and_mask_semantics(po, sphere_oracles):
    """App. A.5 / R-17, R-18: damping -> 1 far away and when a polarizability is zero; the
    group mask removes permanent multipoles of the same group only, never induced dipoles;
    energies are evaluated unmasked."""
    o = sphere_oracles(1)
    rng = np.random.default_rng(3)
    s = _random_sites(po, rng, 4, groups=np.array([0, 0, 1, 1]))
    mu = rng.normal(0, 0.1, (4, 3))
    zero = po.Sites(pos=s.pos, q=0 * s.q, dip=0 * s.dip, quad=0 * s.quad, alpha=s.alpha, group=s.group)
    # induced part is identical with and without the mask
    a = o.multipole_field(zero, mu, True)
    b = o.multipole_field(zero, mu, False)
    for u, v in zip(a, b):
        np.testing.assert_array_equal(u, v)
    # permanent part, masked: site 0 sees only sites 2, 3
    sub = po.Sites(pos=s.pos[[0, 2, 3]], q=s.q[[0, 2, 3]], dip=s.dip[[0, 2, 3]], quad=s.quad[[0, 2, 3]],
                   alpha=s.alpha[[0, 2, 3]], group=np.array([5, 6, 7]))
    pm, gm, hm = o.multipole_field(s, None, True)
    pu, gu, hu = o.multipole_field(sub, None, False)
    np.testing.assert_allclose(pm[0], pu[0], rtol=1e-13)
    np.testing.assert_allclose(gm[0], gu[0], rtol=1e-13)
    np.testing.assert_allclose(hm[0], hu[0], rtol=1e-12)
    # undamped limit: alpha = 0 on the sources gives the bare dipole field = that of a permanent dipole
    bare = po.Sites(pos=s.pos, q=0 * s.q, dip=0 * s.dip, quad=0 * s.quad, alpha=0 * s.alpha, group=s.group)
    perm = po.Sites(pos=s.pos, q=0 * s.q, dip=mu, quad=0 * s.quad, alpha=0 * s.alpha, group=np.arange(4))
    for u, v in zip(o.multipole_field(bare, mu, False), o.multipole_field(perm, None, False)):
        np.testing.assert_allclose(u, v, rtol=1e-13, atol=1e-18)
    # damping reduces the close-range field and vanishes at long range
    near = po.Sites(pos=[[0, 0, 0], [0.8, 0, 0]], q=[0, 0], dip=np.zeros((2, 3)), quad=np.zeros((2, 6)), alpha=[1, 1], group=[0, 1])
    far = po.Sites(pos=[[0, 0, 0], [8.0, 0, 0]], q=[0, 0], dip=np.zeros((2, 3)), quad=np.zeros((2, 6)), alpha=[1, 1], group=[0, 1])
    m2 = np.array([[0, 0, 0], [0.0, 0.3, 0.0]])
    for st, lo, hi in ((near, 0.05, 0.5), (far, 1 - 1e-12, 1 + 1e-12)):
        gd = o.multipole_field(st, m2, False)[1][0, 1]
        st0 = po.Sites(pos=st.pos, q=st.q, dip=st.dip, quad=st.quad, alpha=[0, 0], group=st.group)
        g0 = o.multipole_field(st0, m2, False)[1][0, 1]
        assert lo < gd / g0 < hi
    # lambda_3 itself at u = 1 (R = 1, alpha = 1): 1 - exp(-a)
    one = po.Sites(pos=[[0, 0, 0], [1.0, 0, 0]], q=[0, 0], dip=np.zeros((2, 3)), quad=np.zeros((2, 6)), alpha=[1, 1], group=[0, 1])
    phi = o.multipole_field(one, np.array([[0, 0, 0], [0.5, 0, 0]]), False)[0][0]
    assert abs(phi - (1 - np.exp(-0.39)) * (0.5 * -1.0) / FOURPI) < 1e-15


def test_reaction_field_derivatives_by_finite_differences(po, sphere_oracles):
    """Eq. (13), (21) with App. A.2's kernels are the central differences of Eq. (12), for a
    random surface density (so single- and double-layer parts both matter)."""
    o = sphere_oracles(1)
    rng = np.random.default_rng(7)
    x = rng.normal(size=2 * o.nt)
    x0 = np.array([0.4, -0.3, 0.6])
    hstep = 1e-4
    phi0, g0, h0 = o.reaction(x, x0[None])
    pts = np.array([x0 + s * hstep * np.eye(3)[k] for k in range(3) for s in (1, -1)])
    phi, g, _ = o.reaction(x, pts)
    gfd = (phi[0::2] - phi[1::2]) / (2 * hstep)
    hfd = ((g[0::2] - g[1::2]) / (2 * hstep)).T
    np.testing.assert_allclose(g0[0], gfd, rtol=1e-7, atol=1e-9 * np.abs(g0).max())
    np.testing.assert_allclose(_h6(h0[0]), hfd, rtol=1e-6, atol=1e-8 * np.abs(h0).max())
    assert abs(np.trace(_h6(h0[0]))) < 1e-12 * np.abs(h0).max()          # harmonic inside


def test_reaction_field_near_rule_switch(po):
    """R-9: a site closer than tau*sqrt(A_j) to a panel centroid takes the K_near rule for that
    panel -- visible as a jump when tau crosses the distance, absent otherwise."""
    from paper_1810_03698_b200.workloads import icosphere
    v, t = icosphere(4.0, 1)
    x = np.ones(2 * 80)
    pt = np.array([[0.0, 0.0, 3.0]])
    base = po.Oracle(v, t, po.Params(K_far=1, near_tau=0.0)).reaction(x, pt)[0][0]
    same = po.Oracle(v, t, po.Params(K_far=1, near_tau=0.05)).reaction(x, pt)[0][0]
    fine = po.Oracle(v, t, po.Params(K_far=1, near_tau=5.0)).reaction(x, pt)[0][0]
    allfine = po.Oracle(v, t, po.Params(K_far=19, near_tau=0.0)).reaction(x, pt)[0][0]
    assert base == same
    assert abs(fine - allfine) < abs(base - allfine) * 0.2 and fine != base


def test_energy_formula_eq24(po):
    """Eq. (24): G = 1/2 sum [q phi + d.grad phi + (1/6) Q_ij d_i d_j phi] with the full tensor
    contraction (off-diagonals counted twice)."""
    rng = np.random.default_rng(2)
    Qm = rng.normal(size=(3, 3))
    Qm = Qm + Qm.T
    Hm = rng.normal(size=(3, 3))
    Hm = Hm + Hm.T
    s = po.Sites(pos=[[0, 0, 0]], q=[0.3], dip=[[0.1, 0.2, -0.3]],
                 quad=[[Qm[0, 0], Qm[0, 1], Qm[0, 2], Qm[1, 1], Qm[1, 2], Qm[2, 2]]], alpha=[1.0], group=[0])
    phi = np.array([0.7])
    g = np.array([[0.5, -0.4, 0.2]])
    h = np.array([[Hm[0, 0], Hm[0, 1], Hm[0, 2], Hm[1, 1], Hm[1, 2], Hm[2, 2]]])
    ref = 0.5 * (0.3 * 0.7 + s.dip[0] @ g[0] + np.sum(Qm * Hm) / 6.0)
    assert abs(po.Oracle.energy_G(s, phi, g, h) - ref) < 1e-15


def test_vacuum_scf_equals_linear_solve(po, sphere_oracles):
    """Pin 11 (vacuum): the SOR fixed point solves (alpha^-1 - T) mu = E_perm, with T the
    Thole-damped dipole field operator and E_perm the masked permanent field -- assembled here
    column by column from unit dipoles and solved with numpy.linalg.solve."""
    o = po.Oracle(sphere_oracles(1).verts, sphere_oracles(1).tris, po.Params(K_far=4, scf_tol_debye=1e-12))
    rng = np.random.default_rng(21)
    s = _random_sites(po, rng, 6, spread=2.5, groups=np.array([0, 0, 1, 1, 2, 2]))
    mu, _, its = o.scf(s, solvent=False)
    na = s.na
    zero = po.Sites(pos=s.pos, q=0 * s.q, dip=0 * s.dip, quad=0 * s.quad, alpha=s.alpha, group=s.group)
    T = np.zeros((3 * na, 3 * na))
    for c in range(3 * na):
        e = np.zeros(3 * na)
        e[c] = 1.0
        T[:, c] = (-FOURPI * o.multipole_field(zero, e.reshape(na, 3), True)[1]).reshape(-1)
    Eperm = (-FOURPI * o.multipole_field(s, None, True)[1]).reshape(-1)
    A = np.diag(np.repeat(1.0 / s.alpha, 3)) - T
    ref = np.linalg.solve(A, Eperm).reshape(na, 3)
    np.testing.assert_allclose(mu, ref, rtol=1e-9, atol=1e-12)
    assert 3 < its < 150
    np.testing.assert_allclose(T, T.T, atol=1e-14)       # dipole-dipole tensor is symmetric


def test_solvent_scf_equals_linear_solve(po, sphere_oracles):
    """Pin 11 (solvent): add the reaction-field matrix built column by column from oracle
    solves; the SOR loop (steps 1-6) lands on the same induced dipoles."""
    base = sphere_oracles(2)
    o = po.Oracle(base.verts, base.tris, po.Params(K_far=4, scf_tol_debye=1e-12))
    rng = np.random.default_rng(22)
    s = _random_sites(po, rng, 4, spread=1.8)
    mu, x, its = o.scf(s, solvent=True)
    na = s.na
    zero = po.Sites(pos=s.pos, q=0 * s.q, dip=0 * s.dip, quad=0 * s.quad, alpha=s.alpha, group=s.group)
    M = np.zeros((3 * na, 3 * na))
    for c in range(3 * na):
        e = np.zeros(3 * na)
        e[c] = 1.0
        m = e.reshape(na, 3)
        xs = o.solve_linear(o.rhs(zero, m))
        M[:, c] = (-FOURPI * (o.multipole_field(zero, m, True)[1] + o.reaction(xs, s.pos)[1])).reshape(-1)
    x0 = o.solve_linear(o.rhs(s))
    E0 = (-FOURPI * (o.multipole_field(s, None, True)[1] + o.reaction(x0, s.pos)[1])).reshape(-1)
    ref = np.linalg.solve(np.diag(np.repeat(1.0 / s.alpha, 3)) - M, E0).reshape(na, 3)
    np.testing.assert_allclose(mu, ref, rtol=1e-8, atol=1e-11)
    # the returned surface solution is the one for the converged dipoles
    np.testing.assert_allclose(o.matrix() @ x, o.rhs(s, mu), atol=1e-10)
    # and the energy assembly is Eq. (19) term by term
    r = o.solve(s)
    assert abs(r["dG_solv"] - (r["G_solvterm"] + r["G_mult_diss"] - r["G_vac"])) < 1e-12
    assert r["dG_solv"] < 0
