// pb_sites.cu -- atom-side kernels: multipole right-hand side Eq. (8), reaction
// potential / field / field gradient of the surface layers Eq. (12), (13), (21)
// and the Coulomb field of the multipoles with group mask and Thole damping Eq. (14), (31), (32)
// (derivative tensors re-derived in D: App. A.2, A.5).
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <mutex>
#include "pb_internal.cuh"

// ---- every site inside the surface (interior problem of Eq. (1); S: section 8(b)) ---------------------
// Solid angle of the closed surface seen from the site, one-point rule per panel:
//   Omega_m = sum_j (A_j n_j).(c_j - r_m) / (4 pi |c_j - r_m|^3)  = 1 inside, 0 outside.
__global__ void k_area_normals(int64_t nt, const double* __restrict__ verts, const int32_t* __restrict__ tris, double* __restrict__ an)
{
    const int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (j >= nt) return;
    const double* a = verts + 3 * (int64_t)tris[3 * j];
    const double* b = verts + 3 * (int64_t)tris[3 * j + 1];
    const double* c = verts + 3 * (int64_t)tris[3 * j + 2];
    const double e1[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]}, e2[3] = {c[0] - a[0], c[1] - a[1], c[2] - a[2]};
    an[3 * j] = 0.5 * (e1[1] * e2[2] - e1[2] * e2[1]);
    an[3 * j + 1] = 0.5 * (e1[2] * e2[0] - e1[0] * e2[2]);
    an[3 * j + 2] = 0.5 * (e1[0] * e2[1] - e1[1] * e2[0]);
}

#define IN_ST 8
__global__ void __launch_bounds__(256)
k_sites_inside(int64_t na, int64_t nt, const double* __restrict__ pos, const double* __restrict__ cen,
               const double* __restrict__ an, double thresh, int* __restrict__ first_bad)
{
    __shared__ double red[8][IN_ST];
    const int64_t m0 = (int64_t)blockIdx.x * IN_ST;
    double r[IN_ST][3], acc[IN_ST];
#pragma unroll
    for (int t = 0; t < IN_ST; ++t) {
        const int64_t m = m0 + t < na ? m0 + t : na - 1;
        r[t][0] = pos[3 * m]; r[t][1] = pos[3 * m + 1]; r[t][2] = pos[3 * m + 2];
        acc[t] = 0.0;
    }
    for (int64_t j = threadIdx.x; j < nt; j += 256) {
        const double cx = cen[3 * j], cy = cen[3 * j + 1], cz = cen[3 * j + 2];
        const double ax = an[3 * j], ay = an[3 * j + 1], az = an[3 * j + 2];
#pragma unroll
        for (int t = 0; t < IN_ST; ++t) {
            const double dx = cx - r[t][0], dy = cy - r[t][1], dz = cz - r[t][2];
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double ri = r2 > 0.0 ? rsqrt(r2) : 0.0;
            acc[t] += (ax * dx + ay * dy + az * dz) * ri * ri * ri;
        }
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int t = 0; t < IN_ST; ++t) {
        double v = acc[t];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[w][t] = v;
    }
    __syncthreads();
    if (threadIdx.x < IN_ST && m0 + threadIdx.x < na) {
        double v = 0;
        for (int k = 0; k < 8; ++k) v += red[k][threadIdx.x];
        if (!(v * PB_INV4PI > thresh)) atomicMin(first_bad, (int)(m0 + threadIdx.x));
    }
}

int pb_check_sites_inside(pb_ctx* ctx)
{
    pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    if (!ctx->mesh_loaded || !s.loaded) return PB_OK;
    double* an;
    PB_TRY(pb_dalloc_t(ctx, &an, 3 * ctx->nt, CAT_TMP));
    PB_TRY(pb_scratch(ctx, 1 << 20));
    int* bad = (int*)ctx->scratch;
    const int none = 2147483647;
    int hbad = none;
    PB_CUDA(cudaMemcpyAsync(bad, &none, sizeof(int), cudaMemcpyHostToDevice, st));
    k_area_normals<<<pb_blocks(ctx->nt, 256), 256, 0, st>>>(ctx->nt, ctx->verts, ctx->tris, an);
    PB_LAUNCH_CHECK();
    k_sites_inside<<<pb_blocks(s.na, IN_ST), 256, 0, st>>>(s.na, ctx->nt, s.pos, ctx->cen, an, ctx->stern_n1 > 0 ? 1.5 : 0.5, bad);   // inside BOTH surfaces: 2
    PB_LAUNCH_CHECK();
    PB_CUDA(cudaMemcpyAsync(&hbad, bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));
    pb_dfree_cat(ctx, CAT_TMP);
    if (hbad != none)
        return pb_fail(ctx, PB_ERR_BAD_MESH, "site %d lies outside the surface (solid angle below 2 pi): the multipoles must be inside (P:40-47)", hbad);
    s.inside_checked = true;
    return PB_OK;
}

// ---- H10: right-hand side -----------------------------------------------------------------------------
// b_i = 1/(4 pi eps_in) sum_k [ q_k/R + p_k.d/R^3 + d.Q_k.d/(2 R^5) ],  d = c_i - r_k,  p = dip + mu.
// Two collocation points per thread: every site value read from shared memory feeds two pairs.
#define RHS_TILE 64
#define RHS_TPT 2
__global__ void __launch_bounds__(128)
k_rhs(int64_t N, int64_t na, const double* __restrict__ cen, const double* __restrict__ pos,
      const double* __restrict__ q, const double* __restrict__ dip, const double* __restrict__ mu,
      const double* __restrict__ quad, double inv_eps, double* __restrict__ b)
{
    __shared__ double s[13][RHS_TILE];
    const int64_t i0 = blockIdx.x * (int64_t)(blockDim.x * RHS_TPT) + threadIdx.x;
    double x[RHS_TPT], y[RHS_TPT], z[RHS_TPT], sum[RHS_TPT];
#pragma unroll
    for (int t = 0; t < RHS_TPT; ++t) {
        const int64_t i = i0 + t * blockDim.x;
        const int64_t ic = i < N ? i : N - 1;                // padding lanes repeat the last point; never stored
        x[t] = cen[3 * ic]; y[t] = cen[3 * ic + 1]; z[t] = cen[3 * ic + 2];
        sum[t] = 0.0;
    }
    for (int64_t k0 = 0; k0 < na; k0 += RHS_TILE) {
        const int cnt = (int)(na - k0 < RHS_TILE ? na - k0 : RHS_TILE);
        __syncthreads();
        for (int k = threadIdx.x; k < cnt; k += blockDim.x) {
            const int64_t m = k0 + k;
            for (int d = 0; d < 3; ++d) {
                s[d][k] = pos[3 * m + d];
                s[4 + d][k] = dip[3 * m + d] + (mu ? mu[3 * m + d] : 0.0);
            }
            s[3][k] = q[m];
            // d.Q.d/2 = (Qxx dx^2 + Qyy dy^2 + Qzz dz^2)/2 + Qxy dx dy + Qxz dx dz + Qyz dy dz
            s[7][k] = 0.5 * quad[6 * m]; s[8][k] = quad[6 * m + 1]; s[9][k] = quad[6 * m + 2];
            s[10][k] = 0.5 * quad[6 * m + 3]; s[11][k] = quad[6 * m + 4]; s[12][k] = 0.5 * quad[6 * m + 5];
        }
        __syncthreads();
#pragma unroll 2
        for (int k = 0; k < cnt; ++k) {
            const double sx = s[0][k], sy = s[1][k], sz = s[2][k], qk = s[3][k];
            const double p0 = s[4][k], p1 = s[5][k], p2 = s[6][k];
            const double qxx = s[7][k], qxy = s[8][k], qxz = s[9][k], qyy = s[10][k], qyz = s[11][k], qzz = s[12][k];
#pragma unroll
            for (int t = 0; t < RHS_TPT; ++t) {
                const double dx = x[t] - sx, dy = y[t] - sy, dz = z[t] - sz;
                const double r2 = dx * dx + dy * dy + dz * dz;
                const double ri = pb_rsqrt(r2), ri2 = ri * ri, ri3 = ri * ri2, ri5 = ri3 * ri2;
                const double pd = p0 * dx + p1 * dy + p2 * dz;
                const double hQ = dx * (qxx * dx + qxy * dy + qxz * dz) + dy * (qyy * dy + qyz * dz) + qzz * dz * dz;
                sum[t] += qk * ri + pd * ri3 + hQ * ri5;
            }
        }
    }
#pragma unroll
    for (int t = 0; t < RHS_TPT; ++t) {
        const int64_t i = i0 + t * blockDim.x;
        if (i < N) {
            b[i] = PB_INV4PI * inv_eps * sum[t];
            b[N + i] = 0.0;   // second block of Eq. (5)'s right side
        }
    }
}

extern "C" int pb_rhs_multipole(pb_ctx* ctx, const double* mu_induced, double* b)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (!ctx->mesh_loaded || !ctx->sites.loaded) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_rhs_multipole: load mesh and sites first");
    if (!b) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_rhs_multipole: NULL output");
    const pb_sites& s = ctx->sites;
    {   // direct sum over all sites (the paper's choice) or the treecode with the sites as tree sources
        const pb_tree& t = ctx->tree;
        const int mode = ctx->prm.rhs_treecode, P = ctx->prm.order_P;
        const bool tree = t.built && ctx->prm.theta > 0.0 && P >= 1 && P <= 8 &&
                          (mode == 1 || (mode == 2 && (double)ctx->nt * (double)s.na >= 2147483648.0));
        if (tree) {
            PB_TRY(pb_rhs_tree(ctx, mu_induced, b));
            if (ctx->stern_n1 > 0)
                PB_CUDA(cudaMemsetAsync(b + ctx->stern_n1, 0, sizeof(double) * (ctx->nt - ctx->stern_n1), ctx->stream));
            return PB_OK;
        }
    }
    k_rhs<<<pb_blocks(ctx->nt, 128 * RHS_TPT), 128, 0, ctx->stream>>>(ctx->nt, s.na, ctx->cen, s.pos, s.q, s.dip, mu_induced,
                                                                    s.quad, 1.0 / ctx->prm.eps_in, b);
    PB_LAUNCH_CHECK();
    // two surfaces: Eq. (8) stands in the region-1 rows (the panels of Gamma_1) only
    if (ctx->stern_n1 > 0)
        PB_CUDA(cudaMemsetAsync(b + ctx->stern_n1, 0, sizeof(double) * (ctx->nt - ctx->stern_n1), ctx->stream));
    return PB_OK;
}

// ---- H11: reaction potential, field, field gradient at the sites ---------------------------------------
// One source point y with single-layer weight wS (= w A dphi) and double-layer vector
// wK (= w A phi n') adds, at a target with d = r - y (times 1/(4 pi), applied at the end):
//   phi  += wS/R - (wK.d)/R^3
//   grad += -wS d/R^3 - [ wK/R^3 - 3 (wK.d) d/R^5 ]
//   hess += wS (3 d d^T/R^5 - I/R^3) + 3 [wK d^T + d wK^T + (wK.d) I]/R^5 - 15 (wK.d) d d^T/R^7
template <bool HESS>
__device__ __forceinline__ void react_point(double dx, double dy, double dz, double wS, double kx, double ky,
                                            double kz, double* __restrict__ o)
{
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double ri = pb_rsqrt(r2), ri2 = ri * ri, ri3 = ri * ri2, ri5 = ri3 * ri2;
    const double kd = kx * dx + ky * dy + kz * dz;
    o[0] += wS * ri - kd * ri3;
    const double g = -wS * ri3 + 3.0 * kd * ri5;   // coefficient of d
    o[1] += g * dx - kx * ri3;
    o[2] += g * dy - ky * ri3;
    o[3] += g * dz - kz * ri3;
    if (HESS) {
        const double ri7 = ri5 * ri2;
        const double a = 3.0 * wS * ri5 - 15.0 * kd * ri7;    // coefficient of d d^T
        const double dl = -wS * ri3 + 3.0 * kd * ri5;         // coefficient of I
        const double c3 = 3.0 * ri5;
        o[4] += a * dx * dx + dl + c3 * 2.0 * kx * dx;
        o[5] += a * dx * dy + c3 * (kx * dy + ky * dx);
        o[6] += a * dx * dz + c3 * (kx * dz + kz * dx);
        o[7] += a * dy * dy + dl + c3 * 2.0 * ky * dy;
        o[8] += a * dy * dz + c3 * (ky * dz + kz * dy);
        o[9] += a * dz * dz + dl + c3 * 2.0 * kz * dz;
    }
}

#define RF_ST 4        // sites per block (register tile)
#define RF_THREADS 128
template <bool HESS>
__global__ void __launch_bounds__(RF_THREADS)
k_reaction(int64_t Ns, int64_t chunk, int64_t na, const double* __restrict__ pos, const double4* __restrict__ srec,
           double* __restrict__ partial /*[gridDim.x][na][10]*/)
{
    constexpr int NO = HESS ? 10 : 4;
    __shared__ double red[RF_THREADS / 32][RF_ST][NO];
    const int64_t m0 = (int64_t)blockIdx.y * RF_ST;
    double r[RF_ST][3];
    double acc[RF_ST][NO];
#pragma unroll
    for (int t = 0; t < RF_ST; ++t) {
        const int64_t m = m0 + t < na ? m0 + t : na - 1;   // clamp: duplicates are not written
        r[t][0] = pos[3 * m]; r[t][1] = pos[3 * m + 1]; r[t][2] = pos[3 * m + 2];
#pragma unroll
        for (int c = 0; c < NO; ++c) acc[t][c] = 0.0;
    }
    const int64_t s0 = blockIdx.x * chunk, s1 = s0 + chunk < Ns ? s0 + chunk : Ns;
    for (int64_t s = s0 + threadIdx.x; s < s1; s += RF_THREADS) {
        const double4 ra = srec[2 * s], rb = srec[2 * s + 1];
        const double yx = ra.x, yy = ra.y, yz = ra.z, wS = ra.w, kx = rb.x, ky = rb.y, kz = rb.z;
#pragma unroll
        for (int t = 0; t < RF_ST; ++t) react_point<HESS>(r[t][0] - yx, r[t][1] - yy, r[t][2] - yz, wS, kx, ky, kz, acc[t]);
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int t = 0; t < RF_ST; ++t)
#pragma unroll
        for (int c = 0; c < NO; ++c) {
            double v = acc[t][c];
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) red[w][t][c] = v;
        }
    __syncthreads();
    if (threadIdx.x < RF_ST * NO) {
        const int t = threadIdx.x / NO, c = threadIdx.x % NO;
        if (m0 + t < na) {
            double v = 0;
            for (int k = 0; k < RF_THREADS / 32; ++k) v += red[k][t][c];
            partial[((int64_t)blockIdx.x * na + (m0 + t)) * 10 + c] = v;
        }
    }
}

// sum the per-chunk partials (fixed order), apply 1/(4 pi), write phi/grad/hess
__global__ void k_reaction_finish(int64_t na, int nchunk, int NO, const double* __restrict__ partial,
                                  double* __restrict__ phi, double* __restrict__ grad, double* __restrict__ hess)
{
    int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= na * NO) return;
    int64_t m = g / NO;
    int c = (int)(g % NO);
    double v = 0;
    for (int k = 0; k < nchunk; ++k) v += partial[((int64_t)k * na + m) * 10 + c];
    v *= PB_INV4PI;
    if (c == 0) { if (phi) phi[m] = v; }
    else if (c < 4) { if (grad) grad[3 * m + c - 1] = v; }
    else if (hess) hess[6 * m + c - 4] = v;
}

// near (site, panel) pairs: |r_m - c_j| < tau*sqrt(A_j) (D: R-9).  Thread per panel.
template <int PASS>
__global__ void k_site_near_find(int64_t N, int64_t na, double tau, const double* __restrict__ px,
                                 const double* __restrict__ py, const double* __restrict__ pz,
                                 const double* __restrict__ parea, const double* __restrict__ pos,
                                 int32_t* __restrict__ cnt, const int32_t* __restrict__ off,
                                 int32_t* __restrict__ psite, int32_t* __restrict__ ppanel)
{
    int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (j >= N) return;
    const double x = px[j], y = py[j], z = pz[j], rho = tau * sqrt(parea[j]);
    int n = 0;
    int64_t o = PASS ? off[j] : 0;
    for (int64_t m = 0; m < na; ++m) {
        double dx = pos[3 * m] - x, dy = pos[3 * m + 1] - y, dz = pos[3 * m + 2] - z;
        if (sqrt(dx * dx + dy * dy + dz * dz) < rho) {
            if (PASS) { psite[o + n] = (int32_t)m; ppanel[o + n] = (int32_t)j; }
            ++n;
        }
    }
    if (!PASS) cnt[j] = n;
}

__global__ void k_near_keys(int64_t np, const int32_t* __restrict__ psite, const int32_t* __restrict__ ppanel,
                            uint64_t* __restrict__ keys, int32_t* __restrict__ vals, int32_t* __restrict__ cnt)
{
    const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= np) return;
    keys[e] = ((uint64_t)(uint32_t)psite[e] << 32) | (uint32_t)ppanel[e];
    vals[e] = (int32_t)e;
    atomicAdd(&cnt[psite[e]], 1);                     // integer counts: order does not matter
}

__global__ void k_near_unpack(int64_t np, const uint64_t* __restrict__ keys, int32_t* __restrict__ psite, int32_t* __restrict__ ppanel)
{
    const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= np) return;
    psite[e] = (int32_t)(keys[e] >> 32);
    ppanel[e] = (int32_t)(keys[e] & 0xffffffffu);
}

int pb_site_near_build(pb_ctx* ctx)
{
    pb_tree& t = ctx->tree;
    pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    pb_dfree_cat(ctx, CAT_SITE_NEAR);
    s.near_built = false;
    s.tree_built = false;
    int32_t *cnt, *off;
    PB_TRY(pb_dalloc_t(ctx, &cnt, t.N + 1, CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &off, t.N + 1, CAT_SITE_NEAR));
    PB_CUDA(cudaMemsetAsync(cnt, 0, sizeof(int32_t) * (t.N + 1), st));
    k_site_near_find<0><<<pb_blocks(t.N, 128), 128, 0, st>>>(t.N, s.na, ctx->prm.near_tau, t.pc[0], t.pc[1], t.pc[2],
                                                            t.parea, s.pos, cnt, nullptr, nullptr, nullptr);
    PB_LAUNCH_CHECK();
    int64_t np = 0;
    PB_TRY(pb_exclusive_scan_i32(ctx, cnt, off, t.N + 1, &np));
    s.n_near = np;
    PB_TRY(pb_dalloc_t(ctx, &s.near_site, np, CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &s.near_panel, np, CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &s.near_off, s.na + 1, CAT_SITE_NEAR));
    if (np > 0) {
        k_site_near_find<1><<<pb_blocks(t.N, 128), 128, 0, st>>>(t.N, s.na, ctx->prm.near_tau, t.pc[0], t.pc[1], t.pc[2],
                                                                t.parea, s.pos, cnt, off, s.near_site, s.near_panel);
        PB_LAUNCH_CHECK();
        // sort the pairs by (site, panel): each site's corrections are then added in a fixed order by one thread
        // (no floating-point atomics: the reaction field is bitwise repeatable)
        uint64_t *k0, *k1, *ks;
        int32_t *v0, *v1, *vs, *scnt;
        PB_TRY(pb_dalloc_t(ctx, &k0, np, CAT_TMP));
        PB_TRY(pb_dalloc_t(ctx, &k1, np, CAT_TMP));
        PB_TRY(pb_dalloc_t(ctx, &v0, np, CAT_TMP));
        PB_TRY(pb_dalloc_t(ctx, &v1, np, CAT_TMP));
        PB_TRY(pb_dalloc_t(ctx, &scnt, s.na + 1, CAT_TMP));
        PB_CUDA(cudaMemsetAsync(scnt, 0, sizeof(int32_t) * (s.na + 1), st));
        k_near_keys<<<pb_blocks(np, 256), 256, 0, st>>>(np, s.near_site, s.near_panel, k0, v0, scnt);
        PB_LAUNCH_CHECK();
        int abits = 1;
        while (((int64_t)1 << abits) < s.na) ++abits;
        PB_TRY(pb_radix_sort(ctx, k0, k1, v0, v1, np, 32 + abits, &ks, &vs));
        k_near_unpack<<<pb_blocks(np, 256), 256, 0, st>>>(np, ks, s.near_site, s.near_panel);
        PB_LAUNCH_CHECK();
        int64_t tot = 0;
        PB_TRY(pb_exclusive_scan_i32(ctx, scnt, s.near_off, s.na + 1, &tot));   // synchronises
    }
    s.near_built = true;
    return PB_OK;
}

// correction of one near (site, panel) pair: K_near-point rule minus the K_far-point rule
struct rf_corr_args {
    int64_t np;
    int K;
    const int32_t *psite, *ppanel;
    const double* pos;
    const double* pv[9];
    const double *nx, *ny, *nz, *parea, *xphi, *xdphi;
    const double4* srec;
    double* corr;                 // [np][10] the pairs' corrections (phi, grad, hess), pairs sorted by site
};

__global__ void k_reaction_corr(rf_corr_args a, pb_rule_t ruleN)
{
    int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= a.np) return;
    const int32_t m = a.psite[e], j = a.ppanel[e];
    const double r[3] = {a.pos[3 * m], a.pos[3 * m + 1], a.pos[3 * m + 2]};
    double v[9];
    for (int k = 0; k < 9; ++k) v[k] = a.pv[k][j];
    const double area = a.parea[j], ph = a.xphi[j], dp = a.xdphi[j];
    const double n[3] = {a.nx[j], a.ny[j], a.nz[j]};
    double fine[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0}, coarse[10] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int g = 0; g < ruleN.K; ++g) {
        double y[3];
        for (int c = 0; c < 3; ++c) y[c] = ruleN.lam[g][0] * v[c] + ruleN.lam[g][1] * v[3 + c] + ruleN.lam[g][2] * v[6 + c];
        const double wa = ruleN.w[g] * area;
        react_point<true>(r[0] - y[0], r[1] - y[1], r[2] - y[2], wa * dp, wa * ph * n[0], wa * ph * n[1], wa * ph * n[2], fine);
    }
    for (int g = 0; g < a.K; ++g) {
        const int64_t s = (int64_t)j * a.K + g;
        const double4 ra = a.srec[2 * s], rb = a.srec[2 * s + 1];
        react_point<true>(r[0] - ra.x, r[1] - ra.y, r[2] - ra.z, ra.w, rb.x, rb.y, rb.z, coarse);
    }
    for (int c = 0; c < 10; ++c) a.corr[10 * e + c] = PB_INV4PI * (fine[c] - coarse[c]);
}

// thread (site, component): the site's corrections in the order of its (panel-sorted) pair list
__global__ void k_reaction_corr_add(int64_t na, const int32_t* __restrict__ off, const double* __restrict__ corr,
                                    double* __restrict__ phi, double* __restrict__ grad, double* __restrict__ hess)
{
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= na * 10) return;
    const int64_t m = g / 10;
    const int c = (int)(g - 10 * m);
    const int32_t e0 = off[m], e1 = off[m + 1];
    if (e0 == e1) return;
    double* dst = c == 0 ? (phi ? phi + m : nullptr) : (c < 4 ? (grad ? grad + 3 * m + c - 1 : nullptr) : (hess ? hess + 6 * m + c - 4 : nullptr));
    if (!dst) return;
    double v = *dst;
    for (int32_t e = e0; e < e1; ++e) v += corr[10 * (int64_t)e + c];
    *dst = v;
}

extern "C" int pb_reaction_field(pb_ctx* ctx, const double* x, double* phi, double* grad, double* hess)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    pb_tree& t = ctx->tree;
    pb_sites& s = ctx->sites;
    if (!t.built || !s.loaded) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_reaction_field: needs pb_tree_build and pb_sites_load");
    if (!x) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_reaction_field: NULL x");
    if (!phi && !grad && !hess) return PB_OK;
    cudaStream_t st = ctx->stream;
    if (!s.near_built) PB_TRY(pb_site_near_build(ctx));
    PB_TRY(pb_weights(ctx, x, false, t.psurf ? 0 : -1));   // two surfaces: the layers of Gamma_1 only (it bounds the sites' region)
    // direct sum over every source point (the paper's choice) or the treecode over the panel tree
    const int mode = ctx->prm.site_treecode;
    const bool tree = ctx->prm.theta > 0.0 && ctx->prm.order_P <= 8 &&
                      (mode == 1 || (mode == 2 && (double)s.na * (double)t.Ns >= 2147483648.0));
    if (tree) {
        if (!s.tree_built) PB_TRY(pb_site_tree_build(ctx));
        PB_TRY(pb_reaction_field_tree(ctx, phi, grad, hess));
    } else {
        const int64_t ntile = (s.na + RF_ST - 1) / RF_ST;
        // enough source chunks to fill the GPU, each at least 4 sweeps of the block
        int64_t nchunk = (148 * 16 + ntile - 1) / ntile;
        int64_t maxchunk = (t.Ns + 4 * RF_THREADS - 1) / (4 * RF_THREADS);
        if (nchunk > maxchunk) nchunk = maxchunk;
        if (nchunk < 1) nchunk = 1;
        if (nchunk > 1024) nchunk = 1024;
        int64_t chunk = (t.Ns + nchunk - 1) / nchunk;
        nchunk = (t.Ns + chunk - 1) / chunk;
        PB_TRY(pb_scratch(ctx, (size_t)nchunk * s.na * 10 * sizeof(double) + 4096));
        double* partial = ctx->scratch;
        dim3 grid((unsigned)nchunk, (unsigned)ntile);
        const bool H = hess != nullptr;
        if (H)
            k_reaction<true><<<grid, RF_THREADS, 0, st>>>(t.Ns, chunk, s.na, s.pos, t.srec, partial);
        else
            k_reaction<false><<<grid, RF_THREADS, 0, st>>>(t.Ns, chunk, s.na, s.pos, t.srec, partial);
        PB_LAUNCH_CHECK();
        const int NO = H ? 10 : 4;
        k_reaction_finish<<<pb_blocks(s.na * NO, 128), 128, 0, st>>>(s.na, (int)nchunk, NO, partial, phi, grad, hess);
        PB_LAUNCH_CHECK();
    }
    if (s.n_near > 0) {
        rf_corr_args a;
        a.np = s.n_near; a.K = t.K; a.psite = s.near_site; a.ppanel = s.near_panel; a.pos = s.pos;
        for (int k = 0; k < 9; ++k) a.pv[k] = t.pv[k];
        a.nx = t.pn[0]; a.ny = t.pn[1]; a.nz = t.pn[2]; a.parea = t.parea; a.xphi = t.xphi; a.xdphi = t.xdphi;
        a.srec = t.srec;
        // the direct / treecode sum above is finished with the scratch area (its finish kernel is enqueued before this)
        PB_TRY(pb_scratch(ctx, (size_t)s.n_near * 10 * sizeof(double) + 4096));
        a.corr = ctx->scratch;
        k_reaction_corr<<<pb_blocks(s.n_near, 64), 64, 0, st>>>(a, ctx->ruleN);
        PB_LAUNCH_CHECK();
        k_reaction_corr_add<<<pb_blocks(s.na * 10, 128), 128, 0, st>>>(s.na, s.near_off, a.corr, phi, grad, hess);
        PB_LAUNCH_CHECK();
    }
    return PB_OK;
}

// ---- H12: Coulomb potential / field / field gradient of the multipoles at the other sites ------------------
// Block = MF_ST target sites (register tile) x one chunk of source sites swept by the block's threads;
// per-chunk partial sums are added in a fixed order by k_mfield_finish.  PERM: permanent charge, dipole,
// quadrupole of the sources (Eq. 7, 31, 32 with the corrections of App. A.2), dropped for same-group pairs
// when use_mask.  IND: induced dipoles, never masked, Thole-damped (App. A.5).
// FULL: potential, gradient and Hessian (energies, Eq. 24); otherwise the gradient alone (the SCF loop).
#define MF_ST 2
#define MF_THREADS 128

template <bool FULL, bool PERM, bool IND>
__device__ __forceinline__ void mf_pair(double dx, double dy, double dz, bool masked, double qm, const double* p,
                                        const double* Q, const double* u, double ia_l, double ia_m, double thole_a,
                                        double* o)
{
    constexpr int G0 = FULL ? 1 : 0;
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double i1 = pb_rsqrt(r2), i2 = i1 * i1, i3 = i1 * i2, i5 = i3 * i2, i7 = i5 * i2;
    const double d[3] = {dx, dy, dz};
    if (PERM && !masked) {
        const double pd = p[0] * dx + p[1] * dy + p[2] * dz;
        const double Qd[3] = {Q[0] * dx + Q[1] * dy + Q[2] * dz, Q[1] * dx + Q[3] * dy + Q[4] * dz,
                              Q[2] * dx + Q[4] * dy + Q[5] * dz};
        const double dQd = Qd[0] * dx + Qd[1] * dy + Qd[2] * dz;
        const double gd = -qm * i3 - 3.0 * pd * i5 - 2.5 * dQd * i7;        // coefficient of d in the gradient
#pragma unroll
        for (int c = 0; c < 3; ++c) o[G0 + c] += gd * d[c] + p[c] * i3 + Qd[c] * i5;
        if (FULL) {
            const double i9 = i7 * i2;
            o[0] += qm * i1 + pd * i3 + 0.5 * dQd * i5;
            const double hdd = 3.0 * qm * i5 + 15.0 * pd * i7 + 17.5 * dQd * i9;   // coefficient of d d^T
            int idx = 0;
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = a; b < 3; ++b, ++idx)
                    o[4 + idx] += hdd * d[a] * d[b] + (a == b ? gd : 0.0) - 3.0 * (p[a] * d[b] + p[b] * d[a]) * i5 +
                                  Q[idx] * i5 - 5.0 * (Qd[a] * d[b] + Qd[b] * d[a]) * i7;
        }
    }
    if (IND) {
        double l3 = 1.0, l5 = 1.0, l7 = 1.0;
        const double ia = ia_l * ia_m;                      // 1/sqrt(alpha_l alpha_m), 0 when either is 0
        const double au3 = thole_a * r2 * (r2 * i1) * ia;
        if (ia > 0.0 && au3 < 40.0) {                       // beyond: e^{-au3} < 4.3e-18, the damping factors are 1 to rounding
            const double E = exp(-au3);
            l3 = 1.0 - E;
            l5 = 1.0 - (1.0 + au3) * E;
            l7 = 1.0 - (1.0 + au3 + 0.6 * au3 * au3) * E;
        }
        const double ud = u[0] * dx + u[1] * dy + u[2] * dz;
        const double g5 = 3.0 * l5 * ud * i5;
#pragma unroll
        for (int c = 0; c < 3; ++c) o[G0 + c] += l3 * u[c] * i3 - g5 * d[c];
        if (FULL) {
            o[0] += l3 * ud * i3;
            const double h5 = 3.0 * l5 * i5, h7 = 15.0 * l7 * ud * i7;
            int idx = 0;
#pragma unroll
            for (int a = 0; a < 3; ++a)
#pragma unroll
                for (int b = a; b < 3; ++b, ++idx)
                    o[4 + idx] += -h5 * (u[a] * d[b] + u[b] * d[a] + (a == b ? ud : 0.0)) + h7 * d[a] * d[b];
        }
    }
}

template <bool FULL, bool PERM, bool IND>
__global__ void __launch_bounds__(MF_THREADS)
k_multipole_field(int64_t na, int64_t chunk, const double* __restrict__ pos, const double* __restrict__ q,
                  const double* __restrict__ dip, const double* __restrict__ quad, const double* __restrict__ mu,
                  const double* __restrict__ alpha, const int32_t* __restrict__ group, double thole_a, int use_mask,
                  double* __restrict__ partial /*[gridDim.x][na][10]*/)
{
    constexpr int NO = FULL ? 10 : 3;
    __shared__ double red[MF_THREADS / 32][MF_ST][NO];
    const int64_t l0 = (int64_t)blockIdx.y * MF_ST;
    double r[MF_ST][3], ial[MF_ST], acc[MF_ST][NO];
    int32_t gl[MF_ST];
#pragma unroll
    for (int t = 0; t < MF_ST; ++t) {
        const int64_t l = l0 + t < na ? l0 + t : na - 1;     // clamp: duplicates are not written
        r[t][0] = pos[3 * l]; r[t][1] = pos[3 * l + 1]; r[t][2] = pos[3 * l + 2];
        const double al = alpha[l];
        ial[t] = al > 0.0 ? rsqrt(al) : 0.0;
        gl[t] = group[l];
#pragma unroll
        for (int c = 0; c < NO; ++c) acc[t][c] = 0.0;
    }
    const int64_t m0 = blockIdx.x * chunk, m1 = m0 + chunk < na ? m0 + chunk : na;
    for (int64_t m = m0 + threadIdx.x; m < m1; m += MF_THREADS) {
        const double sx = pos[3 * m], sy = pos[3 * m + 1], sz = pos[3 * m + 2];
        double qm = 0.0, p[3] = {0, 0, 0}, Q[6] = {0, 0, 0, 0, 0, 0}, u[3] = {0, 0, 0}, iam = 0.0;
        if (PERM) {
            qm = q[m];
#pragma unroll
            for (int c = 0; c < 3; ++c) p[c] = dip[3 * m + c];
#pragma unroll
            for (int c = 0; c < 6; ++c) Q[c] = quad[6 * m + c];
        }
        if (IND) {
#pragma unroll
            for (int c = 0; c < 3; ++c) u[c] = mu[3 * m + c];
            const double am = alpha[m];
            iam = am > 0.0 ? rsqrt(am) : 0.0;
        }
        const int32_t gm = group[m];
#pragma unroll
        for (int t = 0; t < MF_ST; ++t) {
            if (m == l0 + t) continue;
            mf_pair<FULL, PERM, IND>(r[t][0] - sx, r[t][1] - sy, r[t][2] - sz, use_mask && gm == gl[t], qm, p, Q, u,
                                     ial[t], iam, thole_a, acc[t]);
        }
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int t = 0; t < MF_ST; ++t)
#pragma unroll
        for (int c = 0; c < NO; ++c) {
            double v = acc[t][c];
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) red[w][t][c] = v;
        }
    __syncthreads();
    if (threadIdx.x < MF_ST * NO) {
        const int t = threadIdx.x / NO, c = threadIdx.x % NO;
        if (l0 + t < na) {
            double v = 0;
            for (int k = 0; k < MF_THREADS / 32; ++k) v += red[k][t][c];
            partial[((int64_t)blockIdx.x * na + (l0 + t)) * 10 + c] = v;
        }
    }
}

// sum the per-chunk partials (fixed order), scale, write phi/grad/hess
__global__ void k_mfield_finish(int64_t na, int nchunk, int full, double scale, const double* __restrict__ partial,
                                double* __restrict__ phi, double* __restrict__ grad, double* __restrict__ hess)
{
    const int NO = full ? 10 : 3;
    int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= na * NO) return;
    int64_t m = g / NO;
    int c = (int)(g % NO);
    double v = 0;
    for (int k = 0; k < nchunk; ++k) v += partial[((int64_t)k * na + m) * 10 + c];
    v *= scale;
    if (!full) grad[3 * m + c] = v;
    else if (c == 0) { if (phi) phi[m] = v; }
    else if (c < 4) { if (grad) grad[3 * m + c - 1] = v; }
    else if (hess) hess[6 * m + c - 4] = v;
}

// parts: bit 0 = permanent multipoles, bit 1 = induced dipoles `mu`
int pb_multipole_field_impl(pb_ctx* ctx, const double* mu, int parts, int use_mask, double* phi, double* grad, double* hess)
{
    const pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    if (!mu) parts &= ~2;
    const bool full = phi || hess;
    if (!full && !grad) return PB_OK;
    const int64_t ntile = (s.na + MF_ST - 1) / MF_ST;
    int64_t nchunk = (148 * 8 + ntile - 1) / ntile;                 // enough blocks to fill the GPU ...
    const int64_t maxchunk = (s.na + MF_THREADS - 1) / MF_THREADS;  // ... but at least one source per thread
    if (nchunk > maxchunk) nchunk = maxchunk;
    if (nchunk < 1) nchunk = 1;
    int64_t chunk = (s.na + nchunk - 1) / nchunk;
    nchunk = (s.na + chunk - 1) / chunk;
    PB_TRY(pb_scratch(ctx, (size_t)nchunk * s.na * 10 * sizeof(double) + 4096));
    double* partial = ctx->scratch;
    dim3 grid((unsigned)nchunk, (unsigned)ntile);
#define MF_LAUNCH(F, PM, IN)                                                                                         \
    k_multipole_field<F, PM, IN><<<grid, MF_THREADS, 0, st>>>(s.na, chunk, s.pos, s.q, s.dip, s.quad, mu, s.alpha,    \
                                                              s.group, ctx->prm.thole_a, use_mask, partial)
    if (parts == 0) {
        PB_CUDA(cudaMemsetAsync(partial, 0, (size_t)nchunk * s.na * 10 * sizeof(double), st));
    } else if (full) {
        if (parts == 3) MF_LAUNCH(true, true, true); else if (parts == 1) MF_LAUNCH(true, true, false); else MF_LAUNCH(true, false, true);
        PB_LAUNCH_CHECK();
    } else {
        if (parts == 3) MF_LAUNCH(false, true, true); else if (parts == 1) MF_LAUNCH(false, true, false); else MF_LAUNCH(false, false, true);
        PB_LAUNCH_CHECK();
    }
#undef MF_LAUNCH
    k_mfield_finish<<<pb_blocks(s.na * (full ? 10 : 3), 128), 128, 0, st>>>(s.na, (int)nchunk, full ? 1 : 0,
                                                                            PB_INV4PI / ctx->prm.eps_in, partial, phi, grad, hess);
    PB_LAUNCH_CHECK();
    return PB_OK;
}

extern "C" int pb_multipole_field(pb_ctx* ctx, const double* mu, int use_mask, double* phi, double* grad, double* hess)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (!ctx->sites.loaded) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_multipole_field: call pb_sites_load first");
    return pb_multipole_field_impl(ctx, mu, 3, use_mask, phi, grad, hess);
}

// ---- pb_multipole_field_static: the H12 sum with NO allocation (include/pb.h) ------------------------------------------
// For callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid it).  The same two kernels as
// pb_multipole_field_impl -- k_multipole_field writes per-chunk partial sums, k_mfield_finish adds them in a fixed order --
// with the partial sums in a file-scope device array instead of the context's scratch buffer.  Every GPU that loads the
// library holds the array (PB_STATIC_MF_ROWS x 10 doubles = 510 KB) until the process exits.  All calls share it and it
// keeps the last call's contents: every element k_mfield_finish reads is written by k_multipole_field in the same call,
// so nothing has to start at zero; two calls that overlap on the GPU (different streams, no ordering) race on it.
#define PB_STATIC_MF_MAX_SITES 4096
// rows [chunk][site] of 10 doubles: n_chunk * na <= na + 148 * 8 * MF_ST + MF_ST with the chunking rule below
#define PB_STATIC_MF_ROWS (PB_STATIC_MF_MAX_SITES + 148 * 8 * MF_ST + 64)
static __device__ __align__(256) double g_mf_static_partial[(size_t)PB_STATIC_MF_ROWS * 10];

#define PB_STATIC_MAX_DEVICES 64
static double* g_mf_static_addr[PB_STATIC_MAX_DEVICES];        // device address of the array, per device (0 = not asked yet)
static std::mutex g_mf_static_mutex;
static thread_local char g_static_err[384] = {0};

static int static_fail(int code, const char* fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_static_err, sizeof(g_static_err), fmt, ap);
    va_end(ap);
    return code;
}

extern "C" const char* pb_static_last_error(void) { return g_static_err; }

extern "C" int pb_multipole_field_static_limit(int64_t* max_sites, int64_t* scratch_bytes)
{
    if (max_sites) *max_sites = PB_STATIC_MF_MAX_SITES;
    if (scratch_bytes) *scratch_bytes = (int64_t)sizeof(double) * PB_STATIC_MF_ROWS * 10;
    return PB_OK;
}

extern "C" int pb_multipole_field_static(int device, void* cuda_stream, int64_t na, const double* pos, const double* q,
                                         const double* dip, const double* quad, const double* alpha, const int32_t* group,
                                         const double* mu, double thole_a, double eps_in, int use_mask, double* phi,
                                         double* grad, double* hess)
{
    g_static_err[0] = 0;
    if (device < 0 || device >= PB_STATIC_MAX_DEVICES)
        return static_fail(PB_ERR_INVALID_ARG, "pb_multipole_field_static: device %d out of range [0, %d)", device, PB_STATIC_MAX_DEVICES);
    if (na < 1 || na > PB_STATIC_MF_MAX_SITES)
        return static_fail(PB_ERR_INVALID_ARG,
                           "pb_multipole_field_static: %lld sites, the static scratch array holds at most %d "
                           "(use pb_multipole_field, which allocates)", (long long)na, PB_STATIC_MF_MAX_SITES);
    if (!pos || !q || !dip || !quad || !alpha || !group) return static_fail(PB_ERR_INVALID_ARG, "pb_multipole_field_static: NULL site array");
    if (!(eps_in > 0.0) || !(thole_a >= 0.0)) return static_fail(PB_ERR_INVALID_ARG, "pb_multipole_field_static: eps_in > 0, thole_a >= 0 required");
    const bool full = phi || hess;
    if (!full && !grad) return PB_OK;
#define PB_STATIC_CUDA(call)                                                                                          \
    do {                                                                                                              \
        cudaError_t e__ = (call);                                                                                     \
        if (e__ != cudaSuccess) {                                                                                     \
            if (prev != device) cudaSetDevice(prev);                                                                  \
            return static_fail(PB_ERR_CUDA, "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e__));      \
        }                                                                                                             \
    } while (0)
    int prev = device;
    {
        cudaError_t e0 = cudaGetDevice(&prev);
        if (e0 != cudaSuccess) { prev = device; return static_fail(PB_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e0)); }
    }
    if (prev != device) PB_STATIC_CUDA(cudaSetDevice(device));
    // In host code the array's name is a host-side stand-in, not a device address: ask the runtime once per device,
    // with that device current
    double* partial = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_mf_static_mutex);
        if (!g_mf_static_addr[device]) {
            double* p = nullptr;
            PB_STATIC_CUDA(cudaGetSymbolAddress((void**)&p, g_mf_static_partial));
            g_mf_static_addr[device] = p;
        }
        partial = g_mf_static_addr[device];
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the chunking of pb_multipole_field_impl (same summation order, so the same bits)
    const int64_t ntile = (na + MF_ST - 1) / MF_ST;
    int64_t nchunk = (148 * 8 + ntile - 1) / ntile;
    const int64_t maxchunk = (na + MF_THREADS - 1) / MF_THREADS;
    if (nchunk > maxchunk) nchunk = maxchunk;
    if (nchunk < 1) nchunk = 1;
    const int64_t chunk = (na + nchunk - 1) / nchunk;
    nchunk = (na + chunk - 1) / chunk;
    if (nchunk * na > PB_STATIC_MF_ROWS) {
        if (prev != device) cudaSetDevice(prev);
        return static_fail(PB_ERR_INVALID_ARG, "pb_multipole_field_static: internal: %lld x %lld partial rows exceed the array",
                           (long long)nchunk, (long long)na);
    }
    dim3 grid((unsigned)nchunk, (unsigned)ntile);
#define MF_LAUNCH(F, IN) \
    k_multipole_field<F, true, IN><<<grid, MF_THREADS, 0, st>>>(na, chunk, pos, q, dip, quad, mu, alpha, group, thole_a, use_mask, partial)
    if (full) { if (mu) MF_LAUNCH(true, true); else MF_LAUNCH(true, false); }
    else { if (mu) MF_LAUNCH(false, true); else MF_LAUNCH(false, false); }
#undef MF_LAUNCH
    PB_STATIC_CUDA(cudaGetLastError());
    k_mfield_finish<<<pb_blocks(na * (full ? 10 : 3), 128), 128, 0, st>>>(na, (int)nchunk, full ? 1 : 0, PB_INV4PI / eps_in, partial, phi,
                                                                         grad, hess);
    PB_STATIC_CUDA(cudaGetLastError());
    if (prev != device) PB_STATIC_CUDA(cudaSetDevice(prev));
#undef PB_STATIC_CUDA
    return PB_OK;
}
