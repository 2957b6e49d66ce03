"""CPU oracle driver -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes layer over oracle/pb_oracle.c (the per-entry arithmetic) plus the
outer algorithms of the paper written out step by step in numpy/scipy:

* the linear system of Eq. (5) assembled densely and solved by LU
  (the plain definition of x = A^{-1} b; the GPU path uses GMRES);
* the self-consistent induced-dipole loop, steps 1-6 with SOR omega = 0.7
  (P:151-160), in solvent and in vacuum;
* the solvation energy, Eq. (19) with each G from Eq. (24);
* the two-surface (Stern layer) block system of the paper's sphere test, class SternOracle.

Nothing here imports or calls the CUDA path; only tests/, __graft_entry__.smoke
and bench.py's cpu_baseline / --impl reference legs may import this module.
Readings "R-n" refer to DESIGN.md (= SURVEY.md section 8(c)).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pb_oracle.c")
_LIB = os.path.join(_HERE, "libpb_oracle.so")

KCAL = 332.0636            # e^2/Angstrom -> kcal/mol (R-1)
FOURPI = 4.0 * np.pi
DEBYE = 4.80320            # 1 e*Angstrom in Debye (R-1)


def build(force: bool = False) -> str:
    """Compile the oracle's C file with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None
_D = ctypes.POINTER(ctypes.c_double)
_I32 = ctypes.POINTER(ctypes.c_int32)
_I64 = ctypes.POINTER(ctypes.c_int64)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.orc_num_threads.restype = ctypes.c_int
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_D)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def rule(K: int):
    lam = np.zeros((K, 3))
    w = np.zeros(K)
    rc = lib().orc_rule(ctypes.c_int(K), _d(lam), _d(w))
    if rc != 0:
        raise ValueError(f"no {K}-point rule")
    return lam, w


def gauss_legendre(n: int):
    x = np.zeros(n)
    w = np.zeros(n)
    lib().orc_gauss_legendre(ctypes.c_int(n), _d(x), _d(w))
    return x, w


def panel_gauss(x, v, K, kappa):
    out = np.zeros(4)
    lib().orc_panel_gauss(_d(_f64(x)), _d(_f64(v).reshape(-1)), ctypes.c_int(K),
                          ctypes.c_double(kappa), _d(out))
    return out


def panel_semi(x, v, nq, kappa):
    out = np.zeros(4)
    lib().orc_panel_semi(_d(_f64(x)), _d(_f64(v).reshape(-1)), ctypes.c_int(nq),
                         ctypes.c_double(kappa), _d(out))
    return out


@dataclass
class Params:
    """Free parameters of the method (BASELINE.json configs)."""
    eps_in: float = 1.0
    eps_out: float = 80.0
    kappa: float = 0.125
    K_far: int = 7
    K_near: int = 19
    near_tau: float = 2.0
    nq_edge: int = 16
    thole_a: float = 0.39
    scf_omega: float = 0.7
    scf_tol_debye: float = 1e-7
    scf_maxit: int = 200


@dataclass
class Sites:
    pos: np.ndarray            # [na][3]
    q: np.ndarray              # [na]
    dip: np.ndarray            # [na][3] permanent dipole d
    quad: np.ndarray           # [na][6] xx,xy,xz,yy,yz,zz (Eq. 7 convention, traceless)
    alpha: np.ndarray          # [na] Angstrom^3
    group: np.ndarray          # [na] int32 polarization group

    def __post_init__(self):
        self.pos = _f64(self.pos).reshape(-1, 3)
        na = self.pos.shape[0]
        self.q = _f64(self.q).reshape(na)
        self.dip = _f64(self.dip).reshape(na, 3)
        self.quad = _f64(self.quad).reshape(na, 6)
        self.alpha = _f64(self.alpha).reshape(na)
        self.group = np.ascontiguousarray(self.group, dtype=np.int32).reshape(na)

    @property
    def na(self):
        return self.pos.shape[0]


class Oracle:
    """Dense-quadrature BEM on one closed triangulated surface (S: O-1 .. O-5)."""

    def __init__(self, verts, tris, params: Params | None = None):
        self.verts = _f64(verts).reshape(-1, 3)
        self.tris = np.ascontiguousarray(tris, dtype=np.int32).reshape(-1, 3)
        self.nt = self.tris.shape[0]
        self.p = params or Params()
        self.cen = np.zeros((self.nt, 3))
        self.nrm = np.zeros((self.nt, 3))
        self.area = np.zeros(self.nt)
        lib().orc_geometry(ctypes.c_int64(self.nt), _d(self.verts), self.tris.ctypes.data_as(_I32),
                           _d(self.cen), _d(self.nrm), _d(self.area))
        self._A = None
        self._lu = None

    # ---- operator -------------------------------------------------------
    def rows(self, rows=None):
        """Dense V_L, K_L, V_Y, K_Y for the listed target rows (all by default)."""
        rows = np.arange(self.nt, dtype=np.int64) if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
        nr = rows.shape[0]
        out = [np.zeros((nr, self.nt)) for _ in range(4)]
        p = self.p
        lib().orc_rows(ctypes.c_int64(self.nt), _d(self.verts), self.tris.ctypes.data_as(_I32),
                       ctypes.c_double(p.kappa), ctypes.c_double(p.near_tau), ctypes.c_int(p.K_far),
                       ctypes.c_int(p.K_near), ctypes.c_int(p.nq_edge), ctypes.c_int64(nr),
                       rows.ctypes.data_as(_I64), *[_d(o) for o in out])
        return out

    def pair_class(self, i, j):
        return int(lib().orc_pair_class(ctypes.c_int64(i), ctypes.c_int64(j), self.tris.ctypes.data_as(_I32),
                                        _d(self.cen), _d(self.area), ctypes.c_double(self.p.near_tau)))

    def matvec(self, x, rows=None):
        """y = A x by direct summation, Eq. (5).  Returns (y1[rows], y2[rows])."""
        x = _f64(x).reshape(2 * self.nt)
        rows = np.arange(self.nt, dtype=np.int64) if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
        nr = rows.shape[0]
        y1 = np.zeros(nr)
        y2 = np.zeros(nr)
        p = self.p
        lib().orc_matvec_rows(ctypes.c_int64(self.nt), _d(self.verts), self.tris.ctypes.data_as(_I32),
                              ctypes.c_double(p.kappa), ctypes.c_double(p.near_tau), ctypes.c_int(p.K_far),
                              ctypes.c_int(p.K_near), ctypes.c_int(p.nq_edge), ctypes.c_double(p.eps_in),
                              ctypes.c_double(p.eps_out), _d(x), ctypes.c_int64(nr),
                              rows.ctypes.data_as(_I64), _d(y1), _d(y2))
        return y1, y2

    def matrix(self):
        """The 2N x 2N matrix of Eq. (5): [[I/2 + K_L, -V_L], [I/2 - K_Y, (eps1/eps2) V_Y]]."""
        if self._A is None:
            VL, KL, VY, KY = self.rows()
            n = self.nt
            A = np.empty((2 * n, 2 * n))
            A[:n, :n] = KL
            A[:n, n:] = -VL
            A[n:, :n] = -KY
            A[n:, n:] = (self.p.eps_in / self.p.eps_out) * VY
            idx = np.arange(n)
            A[idx, idx] += 0.5
            A[n + idx, idx] += 0.5
            self._A = A
        return self._A

    def solve_linear(self, b):
        """x = A^{-1} b by dense LU (the definition; reused across SCF steps)."""
        import scipy.linalg as sla
        if self._lu is None:
            self._lu = sla.lu_factor(self.matrix())
        return sla.lu_solve(self._lu, _f64(b))

    # ---- right-hand side and fields -------------------------------------
    def rhs(self, s: Sites, mu=None):
        """b = [Eq. (8) at the centroids with p = d + mu ; 0]."""
        p = s.dip if mu is None else s.dip + _f64(mu).reshape(-1, 3)
        p = _f64(p)
        b = np.zeros(2 * self.nt)
        lib().orc_rhs(ctypes.c_int64(self.nt), _d(self.cen), ctypes.c_int64(s.na), _d(s.pos), _d(s.q),
                      _d(p), _d(s.quad), ctypes.c_double(self.p.eps_in), _d(b))
        return b

    def reaction(self, x, pos):
        """phi_solv, grad, hess at interior points (Eq. 12, 13, 21)."""
        pos = _f64(pos).reshape(-1, 3)
        na = pos.shape[0]
        phi = np.zeros(na)
        grad = np.zeros((na, 3))
        hess = np.zeros((na, 6))
        x = _f64(x).reshape(2 * self.nt)
        lib().orc_reaction(ctypes.c_int64(self.nt), _d(self.verts), self.tris.ctypes.data_as(_I32), _d(x),
                           ctypes.c_int64(na), _d(pos), ctypes.c_int(self.p.K_far), ctypes.c_int(self.p.K_near),
                           ctypes.c_double(self.p.near_tau), _d(phi), _d(grad), _d(hess))
        return phi, grad, hess

    def multipole_field(self, s: Sites, mu, use_mask: bool):
        """phi, grad, hess of the multipoles at the other sites (Eq. 7, 14, 31, 32)."""
        na = s.na
        phi = np.zeros(na)
        grad = np.zeros((na, 3))
        hess = np.zeros((na, 6))
        mu_c = None if mu is None else _f64(mu).reshape(na, 3)
        lib().orc_multipole_field(ctypes.c_int64(na), _d(s.pos), _d(s.q), _d(s.dip), _d(s.quad), _d(mu_c),
                                  _d(s.alpha), s.group.ctypes.data_as(_I32), ctypes.c_double(self.p.thole_a),
                                  ctypes.c_double(self.p.eps_in), ctypes.c_int(1 if use_mask else 0),
                                  _d(phi), _d(grad), _d(hess))
        return phi, grad, hess

    # ---- energies ---------------------------------------------------------
    @staticmethod
    def energy_G(s: Sites, phi, grad, hess):
        """Eq. (24): G = 1/2 sum_m [ q phi + d_i d_i phi + (1/6) Q_ij d_i d_j phi ],
        with the PERMANENT dipole d (the polarization energy is folded in)."""
        Q = s.quad
        QH = (Q[:, 0] * hess[:, 0] + Q[:, 3] * hess[:, 3] + Q[:, 5] * hess[:, 5]
              + 2.0 * (Q[:, 1] * hess[:, 1] + Q[:, 2] * hess[:, 2] + Q[:, 4] * hess[:, 4]))
        return 0.5 * float(np.sum(s.q * phi + np.sum(s.dip * grad, axis=1) + QH / 6.0))

    # ---- self-consistent induced dipoles ---------------------------------
    def scf(self, s: Sites, solvent: bool = True, history: list | None = None):
        """Steps 1-6 of P:151-160 with SOR (omega).  mu^0 = 0 (R-19).
        mu = alpha * 4 pi * E (alpha in Angstrom^3, E from 1/(4 pi eps)-normalised phi; R-2).
        Converged when sqrt(mean_m |dmu_m|^2) * 4.80320 < tol (R-19).
        Returns (mu, x, iterations)."""
        p = self.p
        mu = np.zeros((s.na, 3))
        x = None
        polarizable = bool(np.any(s.alpha != 0.0))
        for it in range(1, p.scf_maxit + 1):
            E = np.zeros((s.na, 3))
            if solvent:
                b = self.rhs(s, mu)                          # step 2: Eq. (5) with p = d + mu
                x = self.solve_linear(b)
                _, g_solv, _ = self.reaction(x, s.pos)       # step 3: Eq. (13)
                E -= g_solv
            if not polarizable:
                return mu, x, it
            _, g_mult, _ = self.multipole_field(s, mu, use_mask=True)   # step 3: Eq. (14)
            E -= g_mult                                      # step 4: Eq. (15)
            mu_new = (1.0 - p.scf_omega) * mu + p.scf_omega * s.alpha[:, None] * FOURPI * E  # step 5 + SOR
            delta = np.sqrt(np.mean(np.sum((mu_new - mu) ** 2, axis=1))) * DEBYE
            mu = mu_new
            if history is not None:
                history.append(delta)
            if delta < p.scf_tol_debye:                      # step 6
                if solvent:                                  # surface solution consistent with final mu
                    x = self.solve_linear(self.rhs(s, mu))
                return mu, x, it
        raise RuntimeError("oracle SCF did not converge")

    def solve(self, s: Sites):
        """One polarizable solve: Delta G = G[phi_solv] + G[phi_mult(mu)] - G[phi_vac(mu_v)]
        (Eq. 19 with Eq. 24), energies in kcal/mol (R-1)."""
        mu_v, _, it_v = self.scf(s, solvent=False)
        mu, x, it = self.scf(s, solvent=True)
        phi_s, g_s, h_s = self.reaction(x, s.pos)
        G_solv = self.energy_G(s, phi_s, g_s, h_s)
        G_mult = self.energy_G(s, *self.multipole_field(s, mu, use_mask=False))
        G_vac = self.energy_G(s, *self.multipole_field(s, mu_v, use_mask=False))
        c = FOURPI * KCAL
        return dict(x=x, mu=mu, mu_vac=mu_v, scf_iters=it, scf_iters_vac=it_v,
                    G_solvterm=c * G_solv, G_mult_diss=c * G_mult, G_vac=c * G_vac,
                    dG_solv=c * (G_solv + G_mult - G_vac),
                    phi_solv=phi_s, grad_solv=g_s, hess_solv=h_s)


class SternOracle(Oracle):
    """Two nested closed surfaces ("a spherical molecule ... with a 1 Angstrom Stern layer"): Gamma_1, the
    dielectric boundary enclosing the multipoles (region 1, eps_in, Laplace), and Gamma_2 around it (the ion-exclusion
    surface); between them the Stern layer (region 2, eps_stern, Laplace: no ions), outside Gamma_2 the solvent
    (region 3, eps_out, linearised Poisson-Boltzmann with kappa).  The paper uses this only in its sphere test and
    does not print the block system; it follows from Green's second identity in each region exactly as Eq. (2)/(5)
    (P:49-79), with both normals pointing away from the molecule and the interface conditions phi continuous,
    eps d(phi)/dn continuous on each surface (R-32).  Unknowns per panel: phi and q = d(phi)/dn taken on
    the INNER side of its surface (region 1 on Gamma_1, region 2 on Gamma_2).  With A = sources on Gamma_1,
    B = sources on Gamma_2, r12 = eps_in / eps_stern, r23 = eps_stern / eps_out:
      target i on Gamma_1:  y1 = phi_i/2 + K_L^A phi - V_L^A q                                   (region 1)
                            y2 = phi_i/2 - K_L^A phi + r12 V_L^A q + K_L^B phi - V_L^B q         (region 2, from outside Gamma_1)
      target i on Gamma_2:  y1 = phi_i/2 + K_L^B phi - V_L^B q - K_L^A phi + r12 V_L^A q         (region 2, from inside Gamma_2)
                            y2 = phi_i/2 - K_Y^B phi + r23 V_Y^B q                               (region 3)
    and the right-hand side is Eq. (8) in the region-1 rows only.  Both meshes are held as ONE union mesh (panels
    [0, n1) = Gamma_1), so every entry -- including the Gamma_1 <-> Gamma_2 ones, FAR or NEAR by the same distance
    rule R-8 -- comes from the same orc_rows as the single-surface operator.  The reaction potential at the sites is
    Eq. (12) over Gamma_1's layers alone; SCF loop and energies are inherited unchanged."""

    def __init__(self, verts1, tris1, verts2, tris2, params: Params | None = None, eps_stern: float | None = None):
        v1 = _f64(verts1).reshape(-1, 3)
        t1 = np.ascontiguousarray(tris1, dtype=np.int32).reshape(-1, 3)
        v2 = _f64(verts2).reshape(-1, 3)
        t2 = np.ascontiguousarray(tris2, dtype=np.int32).reshape(-1, 3)
        super().__init__(np.concatenate([v1, v2]), np.concatenate([t1, t2 + v1.shape[0]]), params)
        self.n1 = t1.shape[0]
        self.eps_stern = self.p.eps_out if eps_stern is None else float(eps_stern)

    def matrix(self):
        if self._A is None:
            VL, KL, VY, KY = self.rows()
            n, n1 = self.nt, self.n1
            r12, r23 = self.p.eps_in / self.eps_stern, self.eps_stern / self.p.eps_out
            A_, B_ = slice(0, n1), slice(n1, n)
            M = np.zeros((2 * n, 2 * n))
            phi, q = (lambda s: s), (lambda s: slice(n + s.start, n + s.stop))      # column blocks of phi and q
            row1, row2 = phi, q                                                      # row blocks y1 and y2
            # targets on Gamma_1
            M[row1(A_), phi(A_)] = KL[A_, A_]
            M[row1(A_), q(A_)] = -VL[A_, A_]
            M[row2(A_), phi(A_)] = -KL[A_, A_]
            M[row2(A_), q(A_)] = r12 * VL[A_, A_]
            M[row2(A_), phi(B_)] = KL[A_, B_]
            M[row2(A_), q(B_)] = -VL[A_, B_]
            # targets on Gamma_2
            M[row1(B_), phi(B_)] = KL[B_, B_]
            M[row1(B_), q(B_)] = -VL[B_, B_]
            M[row1(B_), phi(A_)] = -KL[B_, A_]
            M[row1(B_), q(A_)] = r12 * VL[B_, A_]
            M[row2(B_), phi(B_)] = -KY[B_, B_]
            M[row2(B_), q(B_)] = r23 * VY[B_, B_]
            idx = np.arange(n)
            M[idx, idx] += 0.5
            M[n + idx, idx] += 0.5
            self._A = M
        return self._A

    def matvec(self, x, rows=None):
        """(y1[rows], y2[rows]) of the block system above, by the dense rows."""
        x = _f64(x).reshape(2 * self.nt)
        y = self.matrix() @ x
        rows = np.arange(self.nt, dtype=np.int64) if rows is None else np.ascontiguousarray(rows, dtype=np.int64)
        return y[rows], y[self.nt + rows]

    def rhs(self, s: Sites, mu=None):
        b = super().rhs(s, mu)
        b[self.n1:self.nt] = 0.0                     # Eq. (8) stands in the region-1 rows only
        return b

    def reaction(self, x, pos):
        """Eq. (12), (13), (21) over Gamma_1's layers (the boundary of the region that holds the sites)."""
        xa = _f64(x).reshape(2 * self.nt).copy()
        xa[self.n1:self.nt] = 0.0
        xa[self.nt + self.n1:] = 0.0
        return super().reaction(xa, pos)


def binding_cycle(sol_ab: dict, sol_a: dict, sol_b: dict) -> dict:
    """The thermodynamic cycle of Fig. 3 from three `Oracle.solve` results
    (complex AB, molecule A, molecule B; kcal/mol):
      Eq. (26)  dG_bind_vac  = G_AB - G_A - G_B + W_pol, with G the vacuum Coulomb energy; using
                Eq. (24)'s G (permanent dipole d in place of p) carries W_pol implicitly;
      Eq. (27)  ddG_bind     = dG_solv,AB - dG_solv,A - dG_solv,B;
      Eq. (25)  dG_bind_diss = dG_solv,AB + dG_bind_vac - dG_solv,A - dG_solv,B."""
    dG_bind_vac = sol_ab["G_vac"] - sol_a["G_vac"] - sol_b["G_vac"]
    ddG_bind = sol_ab["dG_solv"] - sol_a["dG_solv"] - sol_b["dG_solv"]
    dG_bind_diss = sol_ab["dG_solv"] + dG_bind_vac - sol_a["dG_solv"] - sol_b["dG_solv"]
    return dict(dG_bind_vac=dG_bind_vac, ddG_bind=ddG_bind, dG_bind_diss=dG_bind_diss)
