// pb_near.cu -- quadrature rules and the SELF / ADJ / NEAR correction table (D: R-8..R-12, R-16).
//
// The P2P kernel sums the K_far-point rule over EVERY panel except the target's own
// (skipped by panel index, D: R-11).  The table then holds, per target i and panel j in its
// singular / near-singular zone, (true entry) - (K_far-rule entry) for ADJ and NEAR panels and
// the true entry for SELF, so that after the table is applied the operator is exactly the
// three-zone quadrature of P:245: semi-analytic for SELF and vertex-sharing panels, K_near
// points inside tau*sqrt(A_i), K_far points elsewhere.
#include <math.h>
#include <cuda_fp16.h>
#include "pb_internal.cuh"

// ---- rules (host) -----------------------------------------------------------------------------
static void put_orbit3(pb_rule_t* r, int* k, double a, double w)
{
    double b = 0.5 * (1.0 - a);
    const double p[3][3] = {{a, b, b}, {b, a, b}, {b, b, a}};
    for (int i = 0; i < 3; ++i) {
        for (int d = 0; d < 3; ++d) r->lam[*k][d] = p[i][d];
        r->w[*k] = w;
        ++*k;
    }
}

static void put_orbit6(pb_rule_t* r, int* k, double a, double b, double w)
{
    double c = 1.0 - a - b;
    const double p[6][3] = {{a, b, c}, {b, c, a}, {c, a, b}, {a, c, b}, {c, b, a}, {b, a, c}};
    for (int i = 0; i < 6; ++i) {
        for (int d = 0; d < 3; ++d) r->lam[*k][d] = p[i][d];
        r->w[*k] = w;
        ++*k;
    }
}

// Symmetric Gauss rules on the triangle ("1, 3, or 4 Gauss nodes" far away, 19 in the
// near-singular zone; 7 = the degree-5 rule used by BASELINE.json's configs).  Published
// tables (Strang-Fix / Radon / Dunavant); weights are renormalised to sum to one.
int pb_make_rule(int K, pb_rule_t* r)
{
    memset(r, 0, sizeof(*r));
    int k = 0;
    const double third = 1.0 / 3.0;
    auto centroid = [&](double w) { r->lam[k][0] = r->lam[k][1] = r->lam[k][2] = third; r->w[k] = w; ++k; };
    switch (K) {
    case 1: centroid(1.0); break;
    case 3: put_orbit3(r, &k, 2.0 / 3.0, 1.0 / 3.0); break;
    case 4:
        centroid(-0.5625);
        put_orbit3(r, &k, 0.6, 25.0 / 48.0);
        break;
    case 7:
        centroid(0.225);
        put_orbit3(r, &k, 0.0597158717897698, 0.1323941527885062);
        put_orbit3(r, &k, 0.7974269853530873, 0.1259391805448271);
        break;
    case 19:
        centroid(0.097135796282799);
        put_orbit3(r, &k, 0.020634961602525, 0.031334700227139);
        put_orbit3(r, &k, 0.125820817014127, 0.077827541004774);
        put_orbit3(r, &k, 0.623592928761935, 0.079647738927210);
        put_orbit3(r, &k, 0.910540973211095, 0.025577675658698);
        put_orbit6(r, &k, 0.036838412054736, 0.221962989160766, 0.043283539377289);
        break;
    default: return -1;
    }
    if (k != K) return -1;
    double s = 0;
    for (int i = 0; i < K; ++i) s += r->w[i];
    for (int i = 0; i < K; ++i) r->w[i] /= s;
    r->K = K;
    return 0;
}

// Gauss-Legendre nodes on [-1, 1]: Newton on P_n in long double.
static void make_gl(int n, pb_gl_t* g)
{
    g->n = n;
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int i = 0; i < n; ++i) {
        long double z = cosl(pi * (i + 0.75L) / (n + 0.5L)), dp = 1;
        for (int it = 0; it < 60; ++it) {
            long double p0 = 1, p1 = z;
            for (int j = 2; j <= n; ++j) {
                long double p2 = ((2 * j - 1) * z * p1 - (j - 1) * p0) / j;
                p0 = p1;
                p1 = p2;
            }
            if (n == 1) { p0 = 1; p1 = z; }
            dp = n * (z * p1 - p0) / (z * z - 1);
            long double dz = p1 / dp;
            z -= dz;
            if (fabsl(dz) < 1e-19L) break;
        }
        long double p0 = 1, p1 = z;
        for (int j = 2; j <= n; ++j) {
            long double p2 = ((2 * j - 1) * z * p1 - (j - 1) * p0) / j;
            p0 = p1;
            p1 = p2;
        }
        dp = n * (z * p1 - p0) / (z * z - 1);
        g->x[n - 1 - i] = (double)z;
        g->w[n - 1 - i] = (double)(2 / ((1 - z * z) * dp * dp));
    }
}

extern "C" int pb_gauss_legendre(int n, double* x, double* w)
{
    if (n < 1 || n > 64 || !x || !w) return PB_ERR_INVALID_ARG;
    pb_gl_t g;
    make_gl(n, &g);
    for (int i = 0; i < n; ++i) { x[i] = g.x[i]; w[i] = g.w[i]; }
    return PB_OK;
}

int pb_upload_rules(pb_ctx* ctx)
{
    if (pb_make_rule(ctx->prm.K_far, &ctx->ruleF) != 0) return pb_fail(ctx, PB_ERR_INVALID_ARG, "no %d-point rule", ctx->prm.K_far);
    if (pb_make_rule(ctx->prm.K_near, &ctx->ruleN) != 0) return pb_fail(ctx, PB_ERR_INVALID_ARG, "no %d-point rule", ctx->prm.K_near);
    make_gl(ctx->prm.nq_edge, &ctx->gl);
    return PB_OK;
}

// ---- vertex -> panel incidence (Morton panel indices) --------------------------------------------
__global__ void k_vcount(int64_t N, const int32_t* __restrict__ t0, const int32_t* __restrict__ t1,
                         const int32_t* __restrict__ t2, int32_t* __restrict__ vcnt)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    atomicAdd(&vcnt[t0[i]], 1);
    atomicAdd(&vcnt[t1[i]], 1);
    atomicAdd(&vcnt[t2[i]], 1);
}

__global__ void k_vfill(int64_t N, const int32_t* __restrict__ t0, const int32_t* __restrict__ t1,
                        const int32_t* __restrict__ t2, const int32_t* __restrict__ voff, int32_t* __restrict__ vcur,
                        int32_t* __restrict__ vlist)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int32_t v[3] = {t0[i], t1[i], t2[i]};
    for (int b = 0; b < 3; ++b) vlist[voff[v[b]] + atomicAdd(&vcur[v[b]], 1)] = (int32_t)i;
}

// sort each vertex's short list so the table does not depend on atomic ordering
__global__ void k_vsort(int64_t nv, const int32_t* __restrict__ voff, int32_t* __restrict__ vlist)
{
    int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (v >= nv) return;
    int32_t a = voff[v], b = voff[v + 1];
    for (int32_t i = a + 1; i < b; ++i) {
        int32_t x = vlist[i], j = i - 1;
        while (j >= a && vlist[j] > x) { vlist[j + 1] = vlist[j]; --j; }
        vlist[j + 1] = x;
    }
}

// ---- discovery of the SELF / ADJ / NEAR pairs of each target ---------------------------------------
enum { CLS_NEAR = 1, CLS_ADJ = 2, CLS_SELF = 3 };

struct near_args {
    int64_t N;
    int K;
    double tau;
    const int32_t *t0, *t1, *t2, *voff, *vlist;
    const double *px, *py, *pz, *parea;
    const int32_t *c_first, *c_last, *c_child, *c_nchild;
    const double *cx, *cy, *cz, *crad;
    int32_t* cnt;          // pass 0 out: entries per row
    const int32_t* off;    // pass 1 in
    int32_t *col, *row;
    int8_t* cls;
};

template <int PASS>
__global__ void k_near_find(near_args a)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= a.N) return;
    const int32_t tv[3] = {a.t0[i], a.t1[i], a.t2[i]};
    int n = 0;
    int64_t o = PASS ? a.off[i] : 0;
    auto put = [&](int32_t j, int c) {
        if (PASS) { a.col[o + n] = j; a.row[o + n] = (int32_t)i; a.cls[o + n] = (int8_t)c; }
        ++n;
    };
    put((int32_t)i, CLS_SELF);
    // ADJ: shares at least one vertex (D: O-2); a panel reached through vertex b is skipped if it
    // also holds an earlier vertex of i (it was already emitted there)
    for (int b = 0; b < 3; ++b)
        for (int32_t k = a.voff[tv[b]]; k < a.voff[tv[b] + 1]; ++k) {
            int32_t j = a.vlist[k];
            if (j == i) continue;
            bool seen = false;
            for (int e = 0; e < b; ++e) seen = seen || a.t0[j] == tv[e] || a.t1[j] == tv[e] || a.t2[j] == tv[e];
            if (!seen) put(j, CLS_ADJ);
        }
    // NEAR: centroid distance strictly below tau*sqrt(A_i), A_i the TARGET's panel (D: R-8)
    const double x = a.px[i], y = a.py[i], z = a.pz[i];
    const double rho = a.tau * sqrt(a.parea[i]);
    int32_t stack[192];
    int sp = 0;
    stack[sp++] = 0;
    while (sp > 0) {
        int32_t c = stack[--sp];
        double dx = a.cx[c] - x, dy = a.cy[c] - y, dz = a.cz[c] - z;
        if (sqrt(dx * dx + dy * dy + dz * dz) - a.crad[c] >= rho) continue;   // every centroid of c is too far
        int32_t ch = a.c_child[c];
        if (ch >= 0) {
            for (int k = a.c_nchild[c] - 1; k >= 0; --k) stack[sp++] = ch + k;
            continue;
        }
        for (int32_t j = a.c_first[c]; j < a.c_last[c]; ++j) {
            if (j == i) continue;
            double ex = x - a.px[j], ey = y - a.py[j], ez = z - a.pz[j];
            if (!(sqrt(ex * ex + ey * ey + ez * ez) < rho)) continue;
            int32_t u0 = a.t0[j], u1 = a.t1[j], u2 = a.t2[j];
            bool adj = u0 == tv[0] || u0 == tv[1] || u0 == tv[2] || u1 == tv[0] || u1 == tv[1] || u1 == tv[2] ||
                       u2 == tv[0] || u2 == tv[1] || u2 == tv[2];
            if (!adj) put(j, CLS_NEAR);
        }
    }
    if (!PASS) a.cnt[i] = n;
}

// ---- panel integrals ---------------------------------------------------------------------------------
// Kernels of Eq. (3)-(4) integrated over one flat panel, seen from x:
//   out[0] = int 1/(4 pi R), out[1] = int n'.(x-r')/(4 pi R^3),
//   out[2] = int exp(-kR)/(4 pi R), out[3] = int n'.(x-r') exp(-kR)(1+kR)/(4 pi R^3).
__device__ void panel_gauss(const double x[3], const double v[9], const double n[3], double area,
                            const pb_rule_t& rule, double kappa, double out[4])
{
    double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
    for (int g = 0; g < rule.K; ++g) {
        double d[3], r2 = 0, nd = 0;
        for (int c = 0; c < 3; ++c) {
            double y = rule.lam[g][0] * v[c] + rule.lam[g][1] * v[3 + c] + rule.lam[g][2] * v[6 + c];
            d[c] = x[c] - y;
            r2 += d[c] * d[c];
            nd += n[c] * d[c];
        }
        double r = sqrt(r2), e = exp(-kappa * r), ir = 1.0 / r, ir3 = ir / r2;
        s0 += rule.w[g] * ir;
        s1 += rule.w[g] * nd * ir3;
        s2 += rule.w[g] * e * ir;
        s3 += rule.w[g] * nd * e * (1.0 + kappa * r) * ir3;
    }
    out[0] = PB_INV4PI * area * s0;
    out[1] = PB_INV4PI * area * s1;
    out[2] = PB_INV4PI * area * s2;
    out[3] = PB_INV4PI * area * s3;
}

// Semi-analytic rule ("Gauss nodes on the edges"; D: R-16 / App. A.3): polar coordinates
// about the projection x_p of x on the panel plane, radial integral in closed form, the polar
// angle over each edge's sub-triangle by Gauss-Legendre.  With rho(th) = d_e / cos(th),
// s = sqrt(rho^2 + h^2):  F_VL = s-|h|, F_KL = sgn(h) - h/s, F_VY = (e^{-k|h|} - e^{-ks})/k,
// F_KY = sgn(h) e^{-k|h|} - h e^{-ks}/s, each over 4 pi.
__device__ void panel_semi(const double x[3], const double v[9], const double n[3], const pb_gl_t& gl,
                           double kappa, double out[4])
{
    double h = 0;
    for (int c = 0; c < 3; ++c) h += n[c] * (x[c] - v[c]);
    double xp[3];
    for (int c = 0; c < 3; ++c) xp[c] = x[c] - h * n[c];
    const double ah = fabs(h), sg = (h > 0) ? 1.0 : ((h < 0) ? -1.0 : 0.0);
    const double ekh = exp(-kappa * ah);
    double acc[4] = {0, 0, 0, 0};
    for (int e = 0; e < 3; ++e) {
        const int e1 = (e + 1) % 3;
        double a[3], b[3], t[3];
        for (int c = 0; c < 3; ++c) { a[c] = v[3 * e + c] - xp[c]; b[c] = v[3 * e1 + c] - xp[c]; }
        double sd = (a[1] * b[2] - a[2] * b[1]) * n[0] + (a[2] * b[0] - a[0] * b[2]) * n[1] +
                    (a[0] * b[1] - a[1] * b[0]) * n[2];
        if (sd == 0.0) continue;
        double L = 0;
        for (int c = 0; c < 3; ++c) { t[c] = b[c] - a[c]; L += t[c] * t[c]; }
        L = sqrt(L);
        for (int c = 0; c < 3; ++c) t[c] /= L;
        const double de = fabs(sd) / L;
        const double tha = atan2(a[0] * t[0] + a[1] * t[1] + a[2] * t[2], de);
        const double thb = atan2(b[0] * t[0] + b[1] * t[1] + b[2] * t[2], de);
        const double half = 0.5 * (thb - tha), mid = 0.5 * (thb + tha);
        double f0 = 0, f1 = 0, f2 = 0, f3 = 0;
        for (int q = 0; q < gl.n; ++q) {
            double th = mid + half * gl.x[q];
            double rho = de / cos(th);
            double s = sqrt(rho * rho + h * h);
            double eks = exp(-kappa * s);
            f0 += gl.w[q] * (s - ah);
            f1 += gl.w[q] * (sg - h / s);
            f2 += gl.w[q] * (kappa == 0.0 ? (s - ah) : -ekh * expm1(-kappa * (s - ah)) / kappa);
            f3 += gl.w[q] * (sg * ekh - h * eks / s);
        }
        const double se = sd > 0 ? half : -half;
        acc[0] += se * f0; acc[1] += se * f1; acc[2] += se * f2; acc[3] += se * f3;
    }
    for (int m = 0; m < 4; ++m) out[m] = PB_INV4PI * acc[m];
}

struct entry_args {
    int64_t ne;
    int K;
    double kappa, eps_ratio;
    const int32_t *row, *col, *perm;
    const int8_t* cls;
    const double *px, *py, *pz, *nx, *ny, *nz, *parea;
    const double* pv[9];
    const double *sx, *sy, *sz, *swA;
    double* val;        // [4][ne] correction to what P2P / M2P supply (true - far rule; SELF: true)
    double* tval;       // [4][ne] the true three-zone entries (the near-field matrix of the preconditioner)
    double* precond;    // [4][N], ORIGINAL panel order
    int64_t N;
    const unsigned char* psurf;   // two surfaces (pb_set_stern): the panel's surface, else NULL
    double r12, r23;              // eps_in / eps_stern, eps_stern / eps_out
};

// One thread per table entry.
__global__ void k_near_entries(entry_args a, pb_rule_t ruleN, pb_gl_t gl)
{
    int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= a.ne) return;
    const int32_t i = a.row[e], j = a.col[e];
    const int cls = a.cls[e];
    const double x[3] = {a.px[i], a.py[i], a.pz[i]};
    double v[9];
    for (int k = 0; k < 9; ++k) v[k] = a.pv[k][j];
    const double n[3] = {a.nx[j], a.ny[j], a.nz[j]};
    double out[4];
    if (cls == CLS_NEAR) panel_gauss(x, v, n, a.parea[j], ruleN, a.kappa, out);
    else panel_semi(x, v, n, gl, a.kappa, out);
    if (cls == CLS_SELF) {
        out[1] = 0.0;   // flat panel: n'.(c_i - r') == 0 on the panel itself
        out[3] = 0.0;
        for (int m = 0; m < 4; ++m) a.tval[(int64_t)m * a.ne + e] = out[m];
        // inverse of the 2x2 diagonal block [[1/2, -V_L],[1/2, (eps1/eps2) V_Y]] (right preconditioner); with two
        // surfaces the second row of a Gamma_1 panel is the Stern layer's Laplace row, of a Gamma_2 panel the solvent's
        double m01 = -out[0], m11 = a.eps_ratio * out[2];
        if (a.psurf) m11 = a.psurf[i] == 0 ? a.r12 * out[0] : a.r23 * out[2];
        double det = 0.5 * m11 - m01 * 0.5;
        int64_t o = a.perm[i];
        a.precond[o] = m11 / det;
        a.precond[a.N + o] = -m01 / det;
        a.precond[2 * a.N + o] = -0.5 / det;
        a.precond[3 * a.N + o] = 0.5 / det;
    } else {
        for (int m = 0; m < 4; ++m) a.tval[(int64_t)m * a.ne + e] = out[m];
        // minus what P2P adds for this panel: the K_far rule over its stored Gauss points
        double s0 = 0, s1 = 0, s2 = 0, s3 = 0;
        for (int g = 0; g < a.K; ++g) {
            int64_t s = (int64_t)j * a.K + g;
            double dx = x[0] - a.sx[s], dy = x[1] - a.sy[s], dz = x[2] - a.sz[s];
            double r2 = dx * dx + dy * dy + dz * dz;
            double nd = n[0] * dx + n[1] * dy + n[2] * dz;
            double r = sqrt(r2), ir = 1.0 / r, ir3 = ir / r2, ee = exp(-a.kappa * r), w = a.swA[s];
            s0 += w * ir;
            s1 += w * nd * ir3;
            s2 += w * ee * ir;
            s3 += w * nd * ee * (1.0 + a.kappa * r) * ir3;
        }
        out[0] -= PB_INV4PI * s0;
        out[1] -= PB_INV4PI * s1;
        out[2] -= PB_INV4PI * s2;
        out[3] -= PB_INV4PI * s3;
    }
    for (int m = 0; m < 4; ++m) a.val[(int64_t)m * a.ne + e] = out[m];
}

// ---- host driver -----------------------------------------------------------------------------------
// ---- CSR -> sliced ELL: the layout k_combine streams ----------------------------------------------------------
// Slice = 32 consecutive (Morton-ordered) targets = one warp of k_combine; entry k of lane l of slice s sits at
// el_base[s] + 32 k + l, so a warp's loads are contiguous.  Rows shorter than the slice's longest are padded
// with (value 0, column = the target itself).
__global__ void k_ell_width(int64_t N, const int32_t* __restrict__ off, int32_t* __restrict__ width32)
{
    const int64_t w = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w * 32 >= N) return;
    const int64_t i = w * 32 + lane;
    int len = i < N ? off[i + 1] - off[i] : 0;
    for (int o = 16; o > 0; o >>= 1) len = max(len, __shfl_xor_sync(0xffffffffu, len, o));
    if (lane == 0) width32[w] = len * 32;
}

__global__ void k_ell_fill(int64_t N, const int32_t* __restrict__ off, const int32_t* __restrict__ col,
                           const double* __restrict__ val, const double* __restrict__ tval, int64_t ne,
                           const int32_t* __restrict__ base, int64_t ne_ell, int32_t* __restrict__ ecol,
                           double* __restrict__ eval, __half* __restrict__ etval)
{
    const int64_t w = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w * 32 >= N) return;
    const int64_t i = w * 32 + lane;
    const int32_t b0 = base[w], width = (base[w + 1] - b0) / 32;
    const int32_t e0 = i < N ? off[i] : 0, len = i < N ? off[i + 1] - e0 : 0;
    for (int k = 0; k < width; ++k) {
        const int64_t d = (int64_t)b0 + 32 * k + lane;
        const bool real = k < len;
        ecol[d] = real ? col[e0 + k] : (int32_t)(i < N ? i : N - 1);
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            eval[(int64_t)m * ne_ell + d] = real ? val[(int64_t)m * ne + e0 + k] : 0.0;
            etval[4 * d + m] = __double2half(real ? tval[(int64_t)m * ne + e0 + k] : 0.0);
        }
    }
}

int pb_near_build(pb_ctx* ctx)
{
    pb_tree& t = ctx->tree;
    cudaStream_t st = ctx->stream;
    const int64_t N = t.N, nv = ctx->nv;
    int32_t *vcnt, *voff, *vcur, *vlist;
    PB_TRY(pb_dalloc_t(ctx, &vcnt, nv + 1, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &voff, nv + 1, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &vcur, nv + 1, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &vlist, 3 * N, CAT_TMP));
    PB_CUDA(cudaMemsetAsync(vcnt, 0, sizeof(int32_t) * (nv + 1), st));
    PB_CUDA(cudaMemsetAsync(vcur, 0, sizeof(int32_t) * (nv + 1), st));
    k_vcount<<<pb_blocks(N, 256), 256, 0, st>>>(N, t.ptri[0], t.ptri[1], t.ptri[2], vcnt);
    PB_LAUNCH_CHECK();
    PB_TRY(pb_exclusive_scan_i32(ctx, vcnt, voff, nv + 1, nullptr));
    k_vfill<<<pb_blocks(N, 256), 256, 0, st>>>(N, t.ptri[0], t.ptri[1], t.ptri[2], voff, vcur, vlist);
    PB_LAUNCH_CHECK();
    k_vsort<<<pb_blocks(nv, 256), 256, 0, st>>>(nv, voff, vlist);
    PB_LAUNCH_CHECK();

    near_args a;
    a.N = N; a.K = t.K; a.tau = ctx->prm.near_tau;
    a.t0 = t.ptri[0]; a.t1 = t.ptri[1]; a.t2 = t.ptri[2]; a.voff = voff; a.vlist = vlist;
    a.px = t.pc[0]; a.py = t.pc[1]; a.pz = t.pc[2]; a.parea = t.parea;
    a.c_first = t.c_first; a.c_last = t.c_last; a.c_child = t.c_child; a.c_nchild = t.c_nchild;
    a.cx = t.c_ctr[0]; a.cy = t.c_ctr[1]; a.cz = t.c_ctr[2]; a.crad = t.c_rad;
    int32_t* cnt;
    PB_TRY(pb_dalloc_t(ctx, &cnt, N + 1, CAT_TMP));
    PB_CUDA(cudaMemsetAsync(cnt, 0, sizeof(int32_t) * (N + 1), st));
    int32_t* nr_off;
    PB_TRY(pb_dalloc_t(ctx, &nr_off, N + 1, CAT_TMP));
    a.cnt = cnt; a.off = nullptr; a.col = nullptr; a.row = nullptr; a.cls = nullptr;
    k_near_find<0><<<pb_blocks(N, 64), 64, 0, st>>>(a);
    PB_LAUNCH_CHECK();
    int64_t ne = 0;
    PB_TRY(pb_exclusive_scan_i32(ctx, cnt, nr_off, N + 1, &ne));
    t.near_entries = ne;
    int32_t* row;
    int8_t* cls;
    int32_t* nr_col;
    double* nr_val;
    PB_TRY(pb_dalloc_t(ctx, &nr_col, ne, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &nr_val, 4 * ne, CAT_TMP));
    double* nr_tval;
    PB_TRY(pb_dalloc_t(ctx, &nr_tval, 4 * ne, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &t.precond, 4 * N, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &row, ne, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &cls, ne, CAT_TMP));
    a.off = nr_off; a.col = nr_col; a.row = row; a.cls = cls;
    k_near_find<1><<<pb_blocks(N, 64), 64, 0, st>>>(a);
    PB_LAUNCH_CHECK();

    entry_args e;
    e.ne = ne; e.K = t.K; e.kappa = ctx->prm.kappa; e.eps_ratio = ctx->prm.eps_in / ctx->prm.eps_out;
    e.row = row; e.col = nr_col; e.perm = t.perm; e.cls = cls;
    e.px = t.pc[0]; e.py = t.pc[1]; e.pz = t.pc[2]; e.nx = t.pn[0]; e.ny = t.pn[1]; e.nz = t.pn[2];
    e.parea = t.parea;
    for (int k = 0; k < 9; ++k) e.pv[k] = t.pv[k];
    e.sx = t.sx[0]; e.sy = t.sx[1]; e.sz = t.sx[2]; e.swA = t.swA;
    e.val = nr_val; e.tval = nr_tval; e.precond = t.precond; e.N = N;
    e.psurf = t.psurf;
    e.r12 = t.psurf ? ctx->prm.eps_in / ctx->eps_stern : 0.0;
    e.r23 = t.psurf ? ctx->eps_stern / ctx->prm.eps_out : 0.0;
    k_near_entries<<<pb_blocks(ne, 128), 128, 0, st>>>(e, ctx->ruleN, ctx->gl);
    PB_LAUNCH_CHECK();
    // sliced ELL for the combine kernel
    {
        const int64_t nsl = (N + 31) / 32;
        int32_t* width32;
        PB_TRY(pb_dalloc_t(ctx, &width32, nsl + 1, CAT_TMP));
        PB_CUDA(cudaMemsetAsync(width32, 0, sizeof(int32_t) * (nsl + 1), st));
        k_ell_width<<<pb_blocks(nsl * 32, 128), 128, 0, st>>>(N, nr_off, width32);
        PB_LAUNCH_CHECK();
        PB_TRY(pb_dalloc_t(ctx, &t.el_base, nsl + 1, CAT_TREE));
        int64_t ne_ell = 0;
        PB_TRY(pb_exclusive_scan_i32(ctx, width32, t.el_base, nsl + 1, &ne_ell));
        if (ne_ell >= 2147483647LL) return pb_fail(ctx, PB_ERR_INVALID_ARG, "near table too large for int32 indexing");
        t.el_entries = ne_ell;
        PB_TRY(pb_dalloc_t(ctx, &t.el_col, ne_ell > 0 ? ne_ell : 1, CAT_TREE));
        PB_TRY(pb_dalloc_t(ctx, &t.el_val, ne_ell > 0 ? 4 * ne_ell : 1, CAT_TREE));
        PB_TRY(pb_dalloc_t(ctx, &t.el_tval, ne_ell > 0 ? 4 * ne_ell : 1, CAT_TREE));
        k_ell_fill<<<pb_blocks(nsl * 32, 128), 128, 0, st>>>(N, nr_off, nr_col, nr_val, nr_tval, ne, t.el_base, ne_ell, t.el_col,
                                                                 t.el_val, t.el_tval);
        PB_LAUNCH_CHECK();
    }
    PB_CUDA(cudaStreamSynchronize(st));
    pb_dfree_cat(ctx, CAT_TMP);
    return PB_OK;
}
