"""Pins 1-3 of DESIGN section 5: quadrature rules and single-panel integrals of the oracle
against things it does not compute itself (exact monomial integrals, numpy's Gauss-Legendre,
a closed form, and brute-force tensor quadrature)."""
import itertools
import math

import numpy as np
import pytest

FOURPI = 4 * math.pi


def _exact(p, q, r):
    return 2 * math.factorial(p) * math.factorial(q) * math.factorial(r) / math.factorial(p + q + r + 2)


@pytest.mark.parametrize("K,degree", [(1, 1), (3, 2), (4, 3), (7, 5), (19, 9)])
def test_triangle_rule_exactness(po, K, degree):
    """S: R-10 -- weights sum to 1 and every barycentric monomial of total degree <= the
    rule's degree is integrated exactly (and the next degree is NOT, so the degree is sharp)."""
    lam, w = po.rule(K)
    assert lam.shape == (K, 3)
    np.testing.assert_allclose(lam.sum(axis=1), 1.0, atol=1e-15)
    assert abs(w.sum() - 1.0) < 1e-15
    for deg in range(degree + 1):
        for p in range(deg + 1):
            for q in range(deg + 1 - p):
                r = deg - p - q
                got = float(np.sum(w * lam[:, 0] ** p * lam[:, 1] ** q * lam[:, 2] ** r))
                assert abs(got - _exact(p, q, r)) < 2e-16 + 1e-14 * _exact(p, q, r), (K, p, q, r)
    deg = degree + 1
    worst = max(abs(float(np.sum(w * lam[:, 0] ** p * lam[:, 1] ** (deg - p))) - _exact(p, deg - p, 0))
                for p in range(deg + 1))
    assert worst > 1e-8
    # symmetric: the node set is invariant under permutations of the barycentric coordinates
    key = sorted(tuple(np.round(sorted(l), 12)) + (round(x, 12),) for l, x in zip(lam, w))
    for perm in itertools.permutations(range(3)):
        key2 = sorted(tuple(np.round(sorted(l[list(perm)]), 12)) + (round(x, 12),) for l, x in zip(lam, w))
        assert key == key2


def test_centroid_is_a_node_for_K_1_4_7(po):
    """S: R-11 -- the far rule is singular on the self panel, hence exclusion by index."""
    for K in (1, 4, 7):
        lam, _ = po.rule(K)
        assert np.any(np.all(np.abs(lam - 1 / 3) < 1e-15, axis=1))


@pytest.mark.parametrize("n", [4, 16, 33, 64])
def test_gauss_legendre_matches_numpy(po, n):
    x, w = po.gauss_legendre(n)
    xr, wr = np.polynomial.legendre.leggauss(n)
    np.testing.assert_allclose(x, xr, atol=2e-15)
    np.testing.assert_allclose(w, wr, rtol=(1e-13 if n <= 16 else 1e-11), atol=1e-16)


# ---------------------------------------------------------------------------
# single-panel integrals

TRI = np.array([[0.1, -0.2, 0.05], [1.3, 0.1, 0.2], [0.4, 1.1, -0.1]])


def _brute(x, v, kappa, n=200):
    """Independent brute force: Duffy map of the unit square onto the triangle with an
    n x n tensor Gauss-Legendre rule (smooth integrand when x is off the panel)."""
    xs, ws = np.polynomial.legendre.leggauss(n)
    u = 0.5 * (xs + 1)
    wu = 0.5 * ws
    U, V = np.meshgrid(u, u, indexing="ij")
    W = np.outer(wu, wu) * (1 - U)                       # Jacobian of (u, v) -> (u, v(1-u))
    l1, l2 = U, V * (1 - U)
    y = (v[0][None, None, :] * (1 - l1 - l2)[..., None] + v[1][None, None, :] * l1[..., None]
         + v[2][None, None, :] * l2[..., None])
    nrm = np.cross(v[1] - v[0], v[2] - v[0])
    area2 = np.linalg.norm(nrm)
    nrm = nrm / area2
    d = x[None, None, :] - y
    R = np.linalg.norm(d, axis=2)
    nd = d @ nrm
    e = np.exp(-kappa * R)
    return np.array([np.sum(W / R), np.sum(W * nd / R ** 3), np.sum(W * e / R),
                     np.sum(W * nd * e * (1 + kappa * R) / R ** 3)]) * area2 / FOURPI


@pytest.mark.parametrize("x", [
    [0.6, 0.3, 0.35],      # above the footprint
    [0.55, 0.35, -0.2],    # below the footprint
    [2.0, 1.5, 0.4],       # outside the footprint, off plane
    [-0.6, 0.9, 0.02],     # outside, nearly in plane
])
def test_semi_analytic_matches_brute_force(po, x):
    """S: App. A.3 -- exact radial integral + Gauss-Legendre in the polar angle reproduces the
    four panel integrals.  nq=64 to machine-level, nq=16 (the operator's definition) to 1e-9."""
    x = np.array(x)
    ref = _brute(x, TRI, 0.125, n=400 if abs(x[2]) < 0.1 else 200)
    got64 = po.panel_semi(x, TRI, 64, 0.125)
    got16 = po.panel_semi(x, TRI, 16, 0.125)
    np.testing.assert_allclose(got64, ref, rtol=2e-10, atol=1e-13)
    np.testing.assert_allclose(got16, ref, rtol=1e-8, atol=1e-12)


def test_self_panel_laplace_closed_form(po):
    """Collocation at the centroid of its own panel: V_L = (1/4pi) sum_e d_e [asinh(tan th_b) -
    asinh(tan th_a)] (S: App. A.3), K = 0 in the plane."""
    v = TRI
    c = v.mean(axis=0)
    n = np.cross(v[1] - v[0], v[2] - v[0])
    n /= np.linalg.norm(n)
    tot = 0.0
    for e in range(3):
        a, b = v[e] - c, v[(e + 1) % 3] - c
        L = np.linalg.norm(b - a)
        t = (b - a) / L
        de = abs(np.dot(np.cross(a, b), n)) / L
        tot += de * (math.asinh(np.dot(b, t) / de) - math.asinh(np.dot(a, t) / de))
    ref = tot / FOURPI
    for nq, tol in ((16, 1e-9), (64, 1e-13)):
        got = po.panel_semi(c, v, nq, 0.125)
        assert abs(got[0] - ref) < tol * ref
        # (the in-plane double-layer value is the one-sided limit +-1/2 of a roundoff-signed h;
        #  the operator sets K[i,i] = 0 explicitly -- pinned in test_oracle_invariants)
        assert abs(abs(got[1]) - 0.5) < 1e-12 or abs(got[1]) < 1e-15
    # Yukawa self term is below the Laplace one and tends to it as kappa -> 0
    assert po.panel_semi(c, v, 16, 0.125)[2] < ref
    assert abs(po.panel_semi(c, v, 64, 1e-9)[2] - ref) < 1e-8 * ref


def test_kappa_to_zero_yukawa_equals_laplace(po):
    """Pin 3: kappa = 1e-12 makes V_Y, K_Y equal V_L, K_L to 1e-11 on every code path."""
    x = np.array([0.6, 0.3, 0.35])
    for K in (1, 3, 4, 7, 19):
        o = po.panel_gauss(x, TRI, K, 1e-12)
        assert abs(o[2] - o[0]) <= 1e-11 * abs(o[0]) and abs(o[3] - o[1]) <= 1e-11 * abs(o[1])
    o = po.panel_semi(x, TRI, 16, 1e-12)
    assert abs(o[2] - o[0]) <= 1e-11 * abs(o[0]) and abs(o[3] - o[1]) <= 1e-11 * abs(o[1])
    o0 = po.panel_semi(x, TRI, 16, 0.0)
    np.testing.assert_allclose(o0[2:], o0[:2], rtol=1e-14)


@pytest.mark.parametrize("K,tol", [(1, 1e-2), (3, 3e-4), (4, 3e-5), (7, 2e-7), (19, 1e-12)])
def test_gauss_rule_converges_to_the_integral_far_away(po, K, tol):
    """FAR/NEAR rules (S: O-2) approximate the same integrals: from 6 panel sizes away the
    K-point rule agrees with brute force to the accuracy its degree allows."""
    x = np.array([5.0, 4.0, 3.0])
    ref = _brute(x, TRI, 0.125, n=60)
    got = po.panel_gauss(x, TRI, K, 0.125)
    np.testing.assert_allclose(got, ref, rtol=tol)


def test_gauss_rule_is_the_weighted_sum_of_point_kernels(po):
    """The K-point rule is area * sum_g w_g kernel(x, y_g) with y_g = sum_b lam_gb v_b --
    checked for a transposed-operand / wrong-normal mistake via a mirrored panel: flipping the
    panel orientation flips the sign of the double-layer entries only."""
    x = np.array([0.7, 0.2, 0.9])
    a = po.panel_gauss(x, TRI, 7, 0.125)
    b = po.panel_gauss(x, TRI[[0, 2, 1]], 7, 0.125)
    np.testing.assert_allclose(b[[0, 2]], a[[0, 2]], rtol=1e-14)
    np.testing.assert_allclose(b[[1, 3]], -a[[1, 3]], rtol=1e-14)
    # x on the +normal side: n'.(x - r') > 0 so the double-layer entries are positive
    n = np.cross(TRI[1] - TRI[0], TRI[2] - TRI[0])
    assert np.dot(n, x - TRI[0]) > 0 and a[1] > 0 and a[3] > 0
