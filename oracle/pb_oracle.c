/*
 * pb_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of what the boundary-integral
 * Poisson-Boltzmann hot path of arXiv:1810.03698 computes: a dense-quadrature
 * collocation BEM applied by direct O(N^2 K) summation.  No tree, no blocking,
 * no fusion: every function is the definition written out so it can be checked
 * against the paper by eye.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
 * code, header, table or helper with paper_1810_03698_b200/csrc/.
 *
 * Citations are "P:<line>" = /root/reference/PAPER.md line, "S:" = SURVEY.md
 * section 8(c) reading / Appendix A formula, "D:" = DESIGN.md reading.
 *
 * Pins (tests/test_oracle_*.py): quadrature exactness, brute-force panel
 * integrals, Gauss's law, sphere single-layer closed forms, Green's-identity
 * manufactured solutions, Kirkwood closed forms, finite differences of every
 * derivative tensor, SCF == linear solve.  No function here is "parity
 * unpinned"; the paper's own -65.1131 kcal/mol (Stern layer, geometry
 * in an image) is not reproduced and is listed as unpinned in DESIGN.md.
 *
 * Conventions: lengths in Angstrom, charges in e.  Potentials carry the
 * 1/(4 pi) of Eq. (4).  n' is the source-panel unit normal pointing
 * into the solvent.  Symmetric 3x3 tensors are stored as 6-vectors
 * (xx, xy, xz, yy, yz, zz).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define INV4PI 0.079577471545947667884441881686257181

enum { ORC_FAR = 0, ORC_NEAR = 1, ORC_ADJ = 2, ORC_SELF = 3 };

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* Symmetric Gauss rules on the triangle (S: R-10; "1, 3, or 4 Gauss
 * nodes", "19 Gauss nodes").  Barycentric nodes lam[K][3], weights sum to 1. */

static void orbit3(double a, double b, double w, double *lam, double *wt, int *k)
{
    /* the three permutations of (a, b, b) */
    double p[3][3] = { { a, b, b }, { b, a, b }, { b, b, a } };
    for (int i = 0; i < 3; ++i) {
        for (int d = 0; d < 3; ++d) lam[3 * (*k) + d] = p[i][d];
        wt[*k] = w;
        ++*k;
    }
}

static void orbit6(double a, double b, double c, double w, double *lam, double *wt, int *k)
{
    double p[6][3] = { { a, b, c }, { a, c, b }, { b, a, c }, { b, c, a }, { c, a, b }, { c, b, a } };
    for (int i = 0; i < 6; ++i) {
        for (int d = 0; d < 3; ++d) lam[3 * (*k) + d] = p[i][d];
        wt[*k] = w;
        ++*k;
    }
}

int orc_rule(int K, double *lam, double *w)
{
    int k = 0;
    const double t = 1.0 / 3.0;
    switch (K) {
    case 1:
        lam[0] = lam[1] = lam[2] = t; w[0] = 1.0; k = 1;
        break;
    case 3:
        orbit3(2.0 / 3.0, 1.0 / 6.0, 1.0 / 3.0, lam, w, &k);
        break;
    case 4:
        lam[0] = lam[1] = lam[2] = t; w[0] = -27.0 / 48.0; k = 1;
        orbit3(0.6, 0.2, 25.0 / 48.0, lam, w, &k);
        break;
    case 7: /* degree 5 (Radon) */
        lam[0] = lam[1] = lam[2] = t; w[0] = 0.225; k = 1;
        orbit3(0.0597158717897698, 0.4701420641051151, 0.1323941527885062, lam, w, &k);
        orbit3(0.7974269853530873, 0.1012865073234563, 0.1259391805448271, lam, w, &k);
        break;
    case 19: /* degree 9, 19 points (values polished to the moment equations by
                oracle/polish_rule19.py; exactness is pinned in tests) */
        lam[0] = lam[1] = lam[2] = t; w[0] = 0.09713579628279883382; k = 1;
        orbit3(0.02063496160252474443, 0.48968251919873762778, 0.03133470022713907054, lam, w, &k);
        orbit3(0.12582081701412672546, 0.43708959149293663727, 0.07782754100477427932, lam, w, &k);
        orbit3(0.62359292876193453952, 0.18820353561903273024, 0.07964773892721025303, lam, w, &k);
        orbit3(0.91054097321109458027, 0.04472951339445270987, 0.02557767565869803126, lam, w, &k);
        orbit6(0.03683841205473628363, 0.22196298916076569568, 0.74119859878449802069,
               0.04328353937728937729, lam, w, &k);
        break;
    default:
        return -1;
    }
    return k == K ? 0 : -1;
}

/* Gauss-Legendre nodes/weights on [-1,1] by Newton iteration on P_n. */
void orc_gauss_legendre(int n, double *x, double *w)
{
    for (int i = 0; i < n; ++i) {
        double z = cos(3.14159265358979323846 * (i + 0.75) / (n + 0.5)), pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 1; j <= n; ++j) {
                double p3 = p2;
                p2 = p1;
                p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-16) break;
        }
        /* recompute pp at the converged node */
        double p1 = 1.0, p2 = 0.0;
        for (int j = 1; j <= n; ++j) {
            double p3 = p2;
            p2 = p1;
            p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
        }
        pp = n * (z * p1 - p2) / (z * z - 1.0);
        x[n - 1 - i] = z;
        w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

/* ------------------------------------------------------------------------- */
/* Panel geometry (P:243 flat triangles, collocation at the centroid). */

static void tri_geom(const double *v, double *cen, double *nrm, double *area)
{
    double e1[3], e2[3], c[3];
    for (int d = 0; d < 3; ++d) {
        e1[d] = v[3 + d] - v[d];
        e2[d] = v[6 + d] - v[d];
        cen[d] = (v[d] + v[3 + d] + v[6 + d]) / 3.0;
    }
    c[0] = e1[1] * e2[2] - e1[2] * e2[1];
    c[1] = e1[2] * e2[0] - e1[0] * e2[2];
    c[2] = e1[0] * e2[1] - e1[1] * e2[0];
    double l = sqrt(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
    *area = 0.5 * l;
    for (int d = 0; d < 3; ++d) nrm[d] = c[d] / l;
}

static void load_tri(const double *verts, const int32_t *tris, int64_t j, double *v)
{
    for (int b = 0; b < 3; ++b)
        for (int d = 0; d < 3; ++d) v[3 * b + d] = verts[3 * (int64_t)tris[3 * j + b] + d];
}

void orc_geometry(int64_t nt, const double *verts, const int32_t *tris,
                  double *cen, double *nrm, double *area)
{
    for (int64_t j = 0; j < nt; ++j) {
        double v[9];
        load_tri(verts, tris, j, v);
        tri_geom(v, cen + 3 * j, nrm + 3 * j, area + j);
    }
}

/* ------------------------------------------------------------------------- */
/* Integrals over one flat panel of the four kernels of Eq. (3)-(4),
 * seen from the point x:
 *   out[0] = int G_L         = int 1/(4 pi R)
 *   out[1] = int dG_L/dn'    = int n'.(x-r')/(4 pi R^3)
 *   out[2] = int G_Y         = int exp(-kappa R)/(4 pi R)
 *   out[3] = int dG_Y/dn'    = int n'.(x-r') exp(-kappa R)(1+kappa R)/(4 pi R^3)
 * (normal derivatives: S: O-1, from Eq. 3-4 by grad_{r'}).                   */

/* K-point Gauss rule: area * sum_g w_g kernel(x, y_g)  (S: O-2 FAR / NEAR) */
void orc_panel_gauss(const double *x, const double *v, int K, double kappa, double *out)
{
    double lam[19 * 3], w[19], cen[3], n[3], area;
    orc_rule(K, lam, w);
    tri_geom(v, cen, n, &area);
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
    for (int g = 0; g < K; ++g) {
        double d[3], r2 = 0, nd = 0;
        for (int c = 0; c < 3; ++c) {
            double y = lam[3 * g] * v[c] + lam[3 * g + 1] * v[3 + c] + lam[3 * g + 2] * v[6 + c];
            d[c] = x[c] - y;
            r2 += d[c] * d[c];
            nd += n[c] * d[c];
        }
        double r = sqrt(r2), e = exp(-kappa * r);
        s0 += w[g] / r;
        s1 += w[g] * nd / (r2 * r);
        s2 += w[g] * e / r;
        s3 += w[g] * nd * e * (1.0 + kappa * r) / (r2 * r);
    }
    out[0] = INV4PI * area * s0;
    out[1] = INV4PI * area * s1;
    out[2] = INV4PI * area * s2;
    out[3] = INV4PI * area * s3;
}

/* Semi-analytic rule (S: App. A.3, reading of P:245 "Gauss nodes on the edges"):
 * polar coordinates about the projection x_p of x on the panel plane; the
 * radial integral is exact, the polar angle over each edge's sub-triangle is
 * an nq-point Gauss-Legendre rule.                                            */
void orc_panel_semi(const double *x, const double *v, int nq, double kappa, double *out)
{
    double gx[64], gw[64], cen[3], n[3], area;
    if (nq > 64) nq = 64;
    orc_gauss_legendre(nq, gx, gw);
    tri_geom(v, cen, n, &area);
    double h = 0;
    for (int c = 0; c < 3; ++c) h += n[c] * (x[c] - v[c]);
    double xp[3];
    for (int c = 0; c < 3; ++c) xp[c] = x[c] - h * n[c];
    double ah = fabs(h), sg = (h > 0) - (h < 0);
    double ekh = exp(-kappa * ah);
    double acc[4] = { 0, 0, 0, 0 };
    for (int e = 0; e < 3; ++e) {
        double a[3], b[3], t[3], cr[3];
        for (int c = 0; c < 3; ++c) {
            a[c] = v[3 * e + c] - xp[c];
            b[c] = v[3 * ((e + 1) % 3) + c] - xp[c];
        }
        cr[0] = a[1] * b[2] - a[2] * b[1];
        cr[1] = a[2] * b[0] - a[0] * b[2];
        cr[2] = a[0] * b[1] - a[1] * b[0];
        double sd = cr[0] * n[0] + cr[1] * n[1] + cr[2] * n[2];
        if (sd == 0.0) continue;
        double se = sd > 0 ? 1.0 : -1.0;
        double L = 0;
        for (int c = 0; c < 3; ++c) { t[c] = b[c] - a[c]; L += t[c] * t[c]; }
        L = sqrt(L);
        for (int c = 0; c < 3; ++c) t[c] /= L;
        double de = fabs(sd) / L;
        double at = a[0] * t[0] + a[1] * t[1] + a[2] * t[2];
        double bt = b[0] * t[0] + b[1] * t[1] + b[2] * t[2];
        double tha = atan2(at, de), thb = atan2(bt, de);
        double half = 0.5 * (thb - tha), mid = 0.5 * (thb + tha);
        double f[4] = { 0, 0, 0, 0 };
        for (int q = 0; q < nq; ++q) {
            double th = mid + half * gx[q];
            double rho = de / cos(th);
            double s = sqrt(rho * rho + h * h);
            double eks = exp(-kappa * s);
            f[0] += gw[q] * (s - ah);
            f[1] += gw[q] * (sg - h / s);
            /* (e^{-k|h|} - e^{-k s})/k without cancellation; k == 0 is the Laplace limit */
            f[2] += gw[q] * (kappa == 0.0 ? (s - ah) : -ekh * expm1(-kappa * (s - ah)) / kappa);
            f[3] += gw[q] * (sg * ekh - h * eks / s);
        }
        for (int m = 0; m < 4; ++m) acc[m] += se * half * f[m];
    }
    for (int m = 0; m < 4; ++m) out[m] = INV4PI * acc[m];
}

/* ------------------------------------------------------------------------- */
/* Pair classification (S: O-2, R-8, R-11): precedence SELF > ADJ > NEAR > FAR.
 * ADJ = shares at least one vertex index; NEAR = centroid distance strictly
 * below tau*sqrt(A_i), A_i the area of the TARGET's panel.            */
int orc_pair_class(int64_t i, int64_t j, const int32_t *tris, const double *cen,
                   const double *area, double tau)
{
    if (i == j) return ORC_SELF;
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b)
            if (tris[3 * i + a] == tris[3 * j + b]) return ORC_ADJ;
    double d2 = 0;
    for (int c = 0; c < 3; ++c) {
        double d = cen[3 * i + c] - cen[3 * j + c];
        d2 += d * d;
    }
    return (sqrt(d2) < tau * sqrt(area[i])) ? ORC_NEAR : ORC_FAR;
}

/* The four matrix entries V_L, K_L, V_Y, K_Y [i, j] (S: O-2). */
void orc_entry(int64_t i, int64_t j, const double *verts, const int32_t *tris,
               const double *cen, const double *area, double kappa, double tau,
               int K_far, int K_near, int nq_edge, double *out)
{
    double v[9];
    load_tri(verts, tris, j, v);
    int cls = orc_pair_class(i, j, tris, cen, area, tau);
    if (cls == ORC_FAR)
        orc_panel_gauss(cen + 3 * i, v, K_far, kappa, out);
    else if (cls == ORC_NEAR)
        orc_panel_gauss(cen + 3 * i, v, K_near, kappa, out);
    else {
        orc_panel_semi(cen + 3 * i, v, nq_edge, kappa, out);
        if (cls == ORC_SELF) { out[1] = 0.0; out[3] = 0.0; } /* flat panel: n'.(c_i - r') == 0 */
    }
}

/* Dense rows of the four operators: VL,KL,VY,KY are [nrows][nt] row-major. */
void orc_rows(int64_t nt, const double *verts, const int32_t *tris, double kappa, double tau,
              int K_far, int K_near, int nq_edge, int64_t nrows, const int64_t *rows,
              double *VL, double *KL, double *VY, double *KY)
{
    double *cen = malloc(sizeof(double) * 3 * nt), *nrm = malloc(sizeof(double) * 3 * nt);
    double *area = malloc(sizeof(double) * nt);
    orc_geometry(nt, verts, tris, cen, nrm, area);
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t r = 0; r < nrows; ++r) {
        int64_t i = rows[r];
        for (int64_t j = 0; j < nt; ++j) {
            double e[4];
            orc_entry(i, j, verts, tris, cen, area, kappa, tau, K_far, K_near, nq_edge, e);
            VL[r * nt + j] = e[0];
            KL[r * nt + j] = e[1];
            VY[r * nt + j] = e[2];
            KY[r * nt + j] = e[3];
        }
    }
    free(cen); free(nrm); free(area);
}

/* y = A x for the listed target rows, Eq. (5), x = [phi; dphi/dn]:
 *   y1_i = phi_i/2 + sum_j K_L[i,j] phi_j - sum_j V_L[i,j] dphi_j
 *   y2_i = phi_i/2 - sum_j K_Y[i,j] phi_j + (eps_in/eps_out) sum_j V_Y[i,j] dphi_j
 * by direct summation over all panels, nothing stored.                        */
void orc_matvec_rows(int64_t nt, const double *verts, const int32_t *tris, double kappa,
                     double tau, int K_far, int K_near, int nq_edge, double eps_in,
                     double eps_out, const double *x, int64_t nrows, const int64_t *rows,
                     double *y1, double *y2)
{
    double *cen = malloc(sizeof(double) * 3 * nt), *nrm = malloc(sizeof(double) * 3 * nt);
    double *area = malloc(sizeof(double) * nt);
    orc_geometry(nt, verts, tris, cen, nrm, area);
    const double *phi = x, *dphi = x + nt;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t r = 0; r < nrows; ++r) {
        int64_t i = rows[r];
        double sVL = 0, sKL = 0, sVY = 0, sKY = 0;
        for (int64_t j = 0; j < nt; ++j) {
            double e[4];
            orc_entry(i, j, verts, tris, cen, area, kappa, tau, K_far, K_near, nq_edge, e);
            sVL += e[0] * dphi[j];
            sKL += e[1] * phi[j];
            sVY += e[2] * dphi[j];
            sKY += e[3] * phi[j];
        }
        y1[r] = 0.5 * phi[i] + sKL - sVL;
        y2[r] = 0.5 * phi[i] - sKY + (eps_in / eps_out) * sVY;
    }
    free(cen); free(nrm); free(area);
}

/* ------------------------------------------------------------------------- */
/* Right-hand side, Eq. (8) at the collocation points, p = d + mu
 * (Eq. 10):  b_i = 1/(4 pi eps_in) sum_k [ q/R + p.d/R^3 + d.Q.d/(2R^5) ],
 * d = c_i - r_k.  The second block of b is zero and is not returned.   */
void orc_rhs(int64_t npt, const double *pts, int64_t na, const double *pos, const double *q,
             const double *p, const double *Q, double eps_in, double *b)
{
#pragma omp parallel for
    for (int64_t i = 0; i < npt; ++i) {
        double s = 0;
        for (int64_t k = 0; k < na; ++k) {
            double d[3], r2 = 0;
            for (int c = 0; c < 3; ++c) { d[c] = pts[3 * i + c] - pos[3 * k + c]; r2 += d[c] * d[c]; }
            double r = sqrt(r2);
            double pd = p[3 * k] * d[0] + p[3 * k + 1] * d[1] + p[3 * k + 2] * d[2];
            const double *Qk = Q + 6 * k;
            double dQd = Qk[0] * d[0] * d[0] + Qk[3] * d[1] * d[1] + Qk[5] * d[2] * d[2]
                       + 2.0 * (Qk[1] * d[0] * d[1] + Qk[2] * d[0] * d[2] + Qk[4] * d[1] * d[2]);
            s += q[k] / r + pd / (r2 * r) + dQd / (2.0 * r2 * r2 * r);
        }
        b[i] = INV4PI * s / eps_in;
    }
}

/* ------------------------------------------------------------------------- */
/* Reaction potential of the surface layers at interior points, Eq. (12)
 * (P:124): phi_solv = -K_L(phi) + V_L(dphi), with gradient (Eq. 13)
 * and Hessian (Eq. 21).  Kernel derivatives with respect to the target,
 * d = r - r' (S: App. A.2, corrected Eq. 29-30):
 *   grad   (1/R)     = -d/R^3
 *   hess   (1/R)     = 3 d d/R^5 - I/R^3
 *   D = n'.d/R^3 :  grad D = n'/R^3 - 3 (n'.d) d/R^5
 *                   hess D = -3 [n' d^T + d n'^T + (n'.d) I]/R^5 + 15 (n'.d) d d^T/R^7
 * Quadrature per panel (S: R-9): K_far rule, or K_near when
 * |r_m - c_j| < tau*sqrt(A_j).                                                */
void orc_reaction(int64_t nt, const double *verts, const int32_t *tris, const double *x,
                  int64_t na, const double *pos, int K_far, int K_near, double tau,
                  double *phi_out, double *grad_out, double *hess_out)
{
    double lamF[19 * 3], wF[19], lamN[19 * 3], wN[19];
    orc_rule(K_far, lamF, wF);
    orc_rule(K_near, lamN, wN);
    const double *phi = x, *dphi = x + nt;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t m = 0; m < na; ++m) {
        double P = 0, G[3] = { 0, 0, 0 }, H[6] = { 0, 0, 0, 0, 0, 0 };
        const double *r = pos + 3 * m;
        for (int64_t j = 0; j < nt; ++j) {
            double v[9], cen[3], n[3], area;
            load_tri(verts, tris, j, v);
            tri_geom(v, cen, n, &area);
            double dc2 = 0;
            for (int c = 0; c < 3; ++c) dc2 += (r[c] - cen[c]) * (r[c] - cen[c]);
            int near = sqrt(dc2) < tau * sqrt(area);
            int K = near ? K_near : K_far;
            const double *lam = near ? lamN : lamF, *w = near ? wN : wF;
            for (int g = 0; g < K; ++g) {
                double d[3], r2 = 0, nd = 0;
                for (int c = 0; c < 3; ++c) {
                    double y = lam[3 * g] * v[c] + lam[3 * g + 1] * v[3 + c] + lam[3 * g + 2] * v[6 + c];
                    d[c] = r[c] - y;
                    r2 += d[c] * d[c];
                    nd += n[c] * d[c];
                }
                double R = sqrt(r2), R3 = r2 * R, R5 = R3 * r2, R7 = R5 * r2;
                double wS = INV4PI * area * w[g] * dphi[j]; /* single layer, weight dphi/dn */
                double wD = -INV4PI * area * w[g] * phi[j]; /* minus double layer, weight phi */
                P += wS / R + wD * nd / R3;
                for (int c = 0; c < 3; ++c)
                    G[c] += wS * (-d[c] / R3) + wD * (n[c] / R3 - 3.0 * nd * d[c] / R5);
                int idx = 0;
                for (int a = 0; a < 3; ++a)
                    for (int b = a; b < 3; ++b, ++idx) {
                        double dl = (a == b) ? 1.0 : 0.0;
                        double hS = 3.0 * d[a] * d[b] / R5 - dl / R3;
                        double hD = -3.0 * (n[a] * d[b] + d[a] * n[b] + nd * dl) / R5
                                  + 15.0 * nd * d[a] * d[b] / R7;
                        H[idx] += wS * hS + wD * hD;
                    }
            }
        }
        if (phi_out) phi_out[m] = P;
        if (grad_out) for (int c = 0; c < 3; ++c) grad_out[3 * m + c] = G[c];
        if (hess_out) for (int c = 0; c < 6; ++c) hess_out[6 * m + c] = H[c];
    }
}

/* ------------------------------------------------------------------------- */
/* Coulomb potential of the point multipoles at the other sites, Eq. (7) with
 * p = d + mu, its gradient (Eq. 14, 31) and Hessian (Eq. 32,
 * corrected per S: App. A.2), all times 1/(4 pi eps_in):
 *   phi   = q/R + p.d/R^3 + dQd/(2 R^5),                    d = r_l - r_m
 * Permanent part (q, dperm, Q) of source m is dropped when use_mask != 0 and
 * group[m] == group[l].  The induced dipole mu_m is never masked
 * and is Thole-damped (S: App. A.5, R-17):
 *   u = R/(alpha_l alpha_m)^(1/6), E = exp(-a u^3),
 *   l3 = 1-E, l5 = 1-(1+a u^3)E, l7 = 1-(1+a u^3+(3/5)a^2 u^6)E,
 *   phi_mu = l3 mu.d/R^3 ; grad = l3 mu/R^3 - 3 l5 (mu.d) d/R^5 ;
 *   hess = -3 l5 [mu d^T + d mu^T + (mu.d) I]/R^5 + 15 l7 (mu.d) d d^T/R^7.
 * alpha_l*alpha_m == 0 -> no damping.                                         */
void orc_multipole_field(int64_t na, const double *pos, const double *q, const double *dperm,
                         const double *Q, const double *mu, const double *alpha,
                         const int32_t *group, double thole_a, double eps_in, int use_mask,
                         double *phi_out, double *grad_out, double *hess_out)
{
#pragma omp parallel for
    for (int64_t l = 0; l < na; ++l) {
        double P = 0, G[3] = { 0, 0, 0 }, H[6] = { 0, 0, 0, 0, 0, 0 };
        for (int64_t m = 0; m < na; ++m) {
            if (m == l) continue;
            double d[3], r2 = 0;
            for (int c = 0; c < 3; ++c) { d[c] = pos[3 * l + c] - pos[3 * m + c]; r2 += d[c] * d[c]; }
            double R = sqrt(r2), R3 = r2 * R, R5 = R3 * r2, R7 = R5 * r2, R9 = R7 * r2;
            int masked = use_mask && group[l] == group[m];
            if (!masked) {
                double qm = q[m];
                const double *pm = dperm + 3 * m, *Qm = Q + 6 * m;
                double pd = pm[0] * d[0] + pm[1] * d[1] + pm[2] * d[2];
                double Qd[3] = { Qm[0] * d[0] + Qm[1] * d[1] + Qm[2] * d[2],
                                 Qm[1] * d[0] + Qm[3] * d[1] + Qm[4] * d[2],
                                 Qm[2] * d[0] + Qm[4] * d[1] + Qm[5] * d[2] };
                double dQd = Qd[0] * d[0] + Qd[1] * d[1] + Qd[2] * d[2];
                double Qf[3][3] = { { Qm[0], Qm[1], Qm[2] }, { Qm[1], Qm[3], Qm[4] }, { Qm[2], Qm[4], Qm[5] } };
                P += qm / R + pd / R3 + dQd / (2.0 * R5);
                for (int k = 0; k < 3; ++k)
                    G[k] += -qm * d[k] / R3 + pm[k] / R3 - 3.0 * pd * d[k] / R5
                          + Qd[k] / R5 - 2.5 * dQd * d[k] / R7;
                int idx = 0;
                for (int j = 0; j < 3; ++j)
                    for (int k = j; k < 3; ++k, ++idx) {
                        double dl = (j == k) ? 1.0 : 0.0;
                        H[idx] += qm * (3.0 * d[j] * d[k] / R5 - dl / R3)
                                - 3.0 * (pm[k] * d[j] + pm[j] * d[k] + pd * dl) / R5
                                + 15.0 * pd * d[j] * d[k] / R7
                                + Qf[j][k] / R5 - 5.0 * (Qd[k] * d[j] + Qd[j] * d[k]) / R7
                                - 2.5 * dQd * dl / R7 + 17.5 * dQd * d[j] * d[k] / R9;
                    }
            }
            if (mu) {
                const double *um = mu + 3 * m;
                double l3 = 1.0, l5 = 1.0, l7 = 1.0;
                double aa = alpha[l] * alpha[m];
                if (aa > 0.0) {
                    double au3 = thole_a * R3 / sqrt(aa);
                    double E = exp(-au3);
                    l3 = 1.0 - E;
                    l5 = 1.0 - (1.0 + au3) * E;
                    l7 = 1.0 - (1.0 + au3 + 0.6 * au3 * au3) * E;
                }
                double ud = um[0] * d[0] + um[1] * d[1] + um[2] * d[2];
                P += l3 * ud / R3;
                for (int k = 0; k < 3; ++k) G[k] += l3 * um[k] / R3 - 3.0 * l5 * ud * d[k] / R5;
                int idx = 0;
                for (int j = 0; j < 3; ++j)
                    for (int k = j; k < 3; ++k, ++idx) {
                        double dl = (j == k) ? 1.0 : 0.0;
                        H[idx] += -3.0 * l5 * (um[k] * d[j] + um[j] * d[k] + ud * dl) / R5
                                + 15.0 * l7 * ud * d[j] * d[k] / R7;
                    }
            }
        }
        double sc = INV4PI / eps_in;
        if (phi_out) phi_out[l] = sc * P;
        if (grad_out) for (int c = 0; c < 3; ++c) grad_out[3 * l + c] = sc * G[c];
        if (hess_out) for (int c = 0; c < 6; ++c) hess_out[6 * l + c] = sc * H[c];
    }
}
