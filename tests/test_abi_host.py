"""CPU-side checks of the product library: it builds for sm_100a, exports every symbol that
include/pb.h declares, refuses to run without a GPU (no CPU fallback), and its own host-side
tables (quadrature rules, Gauss-Legendre nodes, the far-field M -> F conversion) are right.
No compute call is made here; nothing in the product imports the oracle."""
import ctypes
import math
import os
import re
import subprocess

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def pbmod():
    from paper_1810_03698_b200 import pb
    pb.build()
    return pb


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "pb.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:int|void|const char\s*\*)\s+\*?(pb_[a-z0-9_]+)\s*\(", src, flags=re.M)
    return sorted(set(names))


def test_library_exports_every_declared_symbol(pbmod):
    declared = _declared_functions()
    assert len(declared) >= 20
    L = ctypes.CDLL(pbmod.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), f"{name} declared in include/pb.h but not exported"
    assert sorted(pbmod.EXPORTS) == declared          # the binding covers the same set


def test_library_is_sm100a_sass(pbmod):
    out = subprocess.run(["cuobjdump", "-lelf", pbmod.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_no_cpu_fallback(pbmod):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = ctypes.c_void_p()
    rc = pbmod.lib().pb_create(ctypes.byref(h), 0, None)
    assert rc == -4 and not h.value                   # PB_ERR_CUDA, no context
    with pytest.raises(pbmod.PBError):
        pbmod.PB(0)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1810_03698_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", txt, flags=re.M), f
                assert "pb_oracle" not in txt, f


def _tri_monomial(p, q, r):
    # (1/A) int lam1^p lam2^q lam3^r dA = 2 p! q! r! / (p+q+r+2)!
    return 2.0 * math.factorial(p) * math.factorial(q) * math.factorial(r) / math.factorial(p + q + r + 2)


@pytest.mark.parametrize("K,deg", [(1, 1), (3, 2), (4, 3), (7, 5), (19, 9)])
def test_product_triangle_rules_are_exact(pbmod, K, deg):
    lam, w = pbmod.quadrature_rule(K)
    assert abs(w.sum() - 1.0) < 1e-15
    np.testing.assert_allclose(lam.sum(axis=1), 1.0, atol=1e-15)
    for n in range(deg + 1):
        for p in range(n + 1):
            for q in range(n - p + 1):
                r = n - p - q
                got = np.sum(w * lam[:, 0] ** p * lam[:, 1] ** q * lam[:, 2] ** r)
                assert abs(got - _tri_monomial(p, q, r)) < 2e-14, (K, p, q, r)


@pytest.mark.parametrize("n", [1, 2, 5, 16, 32, 64])
def test_product_gauss_legendre(pbmod, n):
    x, w = pbmod.gauss_legendre(n)
    xr, wr = np.polynomial.legendre.leggauss(n)
    np.testing.assert_allclose(x, xr, atol=2e-15)
    np.testing.assert_allclose(w, wr, rtol=1e-11, atol=1e-16)   # numpy's own nodes are the looser side at n=64
    assert abs(w.sum() - 2.0) < 1e-14 and abs(np.sum(w * x ** (2 * n - 2)) - 2.0 / (2 * n - 1)) < 1e-14


def _mom_index(a, b, c):
    n, m = a + b + c, b + c
    return n * (n + 1) * (n + 2) // 6 + m * (m + 1) // 2 + c


def _taylor_coeffs(P, d, kappa):
    """a_k = (1/k!) D_y^k G(x, y)|_{y=y_c} by the recurrences of DESIGN App. A.4 (Lindsay-Krasny /
    Li-Johnston-Krasny, P:249 refs 54-55), written out here independently of the library."""
    R = np.linalg.norm(d)
    a, b = {}, {}
    A = lambda k: a.get(k, 0.0) if min(k) >= 0 else 0.0
    B = lambda k: b.get(k, 0.0) if min(k) >= 0 else 0.0
    e = math.exp(-kappa * R)
    a[(0, 0, 0)], b[(0, 0, 0)] = e / R, e
    E = [(1, 0, 0), (0, 1, 0), (0, 0, 1)]
    sub = lambda k, u, m: (k[0] - m * u[0], k[1] - m * u[1], k[2] - m * u[2])
    for n in range(1, P + 1):
        for k0 in range(n, -1, -1):
            for k1 in range(n - k0, -1, -1):
                k = (k0, k1, n - k0 - k1)
                b[k] = kappa / n * sum(d[i] * A(sub(k, E[i], 1)) - A(sub(k, E[i], 2)) for i in range(3))
                a[k] = ((2 * n - 1) * sum(d[i] * A(sub(k, E[i], 1)) for i in range(3))
                        - (n - 1) * sum(A(sub(k, E[i], 2)) for i in range(3))
                        + kappa * sum(d[i] * B(sub(k, E[i], 1)) - B(sub(k, E[i], 2)) for i in range(3))) / (n * R * R)
    return a


@pytest.mark.parametrize("P", [0, 1, 2, 3, 4, 6, 8, 10])
def test_farfield_table_reproduces_the_taylor_sum(pbmod, P):
    """sum_k a_k M_k (the paper's order-P Cartesian Taylor far field) must equal
    sum_terms u_{|alpha|+j}(R) d^alpha F_{alpha,j} with F from the library's conversion table, for
    both kernels and both layers' moments -- to rounding, not to truncation error."""
    expo, off, idx, coef = pbmod.farfield_table(P)
    nk = (P + 1) * (P + 2) * (P + 3) // 6
    assert idx.max() == nk - 1 and expo.shape[0] == off.shape[0] - 1
    if P == 6:
        assert expo.shape[0] == 130
    rng = np.random.Generator(np.random.PCG64(P))
    h = rng.uniform(-0.4, 0.4, (25, 3))
    qV = rng.normal(size=25)
    qK = rng.normal(size=(25, 3))
    d = np.array([2.1, -1.3, 0.9])
    kappa = 0.125
    MV, MK = np.zeros(nk), np.zeros(nk)
    for a in range(P + 1):
        for b in range(P + 1 - a):
            for c in range(P + 1 - a - b):
                mono = lambda ea, eb, ec: h[:, 0] ** ea * h[:, 1] ** eb * h[:, 2] ** ec
                i = _mom_index(a, b, c)
                MV[i] = np.sum(qV * mono(a, b, c))
                MK[i] = (np.sum(qK[:, 0] * a * mono(a - 1, b, c)) if a else 0.0) \
                    + (np.sum(qK[:, 1] * b * mono(a, b - 1, c)) if b else 0.0) \
                    + (np.sum(qK[:, 2] * c * mono(a, b, c - 1)) if c else 0.0)
    R = np.linalg.norm(d)

    def u(kap):
        e = math.exp(-kap * R)
        out = [e / R, e * (1 + kap * R) / R ** 3]
        for m in range(1, P + 1):
            out.append(((2 * m + 1) * out[m] + kap * kap * out[m - 1]) / R ** 2)
        return np.array(out[:P + 1])

    for kap in (0.0, kappa):
        coeffs = _taylor_coeffs(P, d, kap)
        for M in (MV, MK):
            ref = sum(coeffs[(a, b, c)] * M[_mom_index(a, b, c)]
                      for a in range(P + 1) for b in range(P + 1 - a) for c in range(P + 1 - a - b))
            W = np.zeros(P + 1)
            for t in range(expo.shape[0]):
                a, b, c, j = expo[t]
                F = np.dot(coef[off[t]:off[t + 1]], M[idx[off[t]:off[t + 1]]])
                W[a + b + c + j] += d[0] ** a * d[1] ** b * d[2] ** c * F
            got = float(u(kap) @ W)
            assert abs(got - ref) <= 1e-12 * max(1.0, abs(ref)), (P, kap)
    # and the truncated sum converges to the direct sum as P grows (the expansion itself)
    if P >= 6:
        x = d
        Rg = np.linalg.norm(x - h, axis=1)
        exact = np.sum(qV * np.exp(-kappa * Rg) / Rg)
        coeffs = _taylor_coeffs(P, d, kappa)
        ref = sum(coeffs[(a, b, c)] * MV[_mom_index(a, b, c)]
                  for a in range(P + 1) for b in range(P + 1 - a) for c in range(P + 1 - a - b))
        assert abs(ref - exact) < 5.0 * (0.7 / R) ** (P + 1) * np.abs(qV).sum() / R
