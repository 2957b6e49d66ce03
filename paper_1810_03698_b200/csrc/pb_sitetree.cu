// pb_sitetree.cu -- treecode for the atom-side reaction field (S: section 8(f) item 1; the paper keeps this sum
// direct): the reaction potential phi_solv = V_L(dphi) - K_L(phi) (Eq. 12), its gradient (Eq. 13) and
// Hessian (Eq. 21) at the sites, with the sites as treecode targets of the PANEL tree.
//
// Far field.  For a cell with centre y_c and moments M^V_l, M^K_l (the upward pass of pb_matvec.cu) the
// order-P Taylor sum of the potential at x is sum_{|l|<=P} a_l(x,y_c) (M^V_l - M^K_l), a_l = D_y^l (1/R) / l!
// (App. A.4).  The kernel is a function of x - y, so D_x = -D_y and the target derivatives of the SAME truncated
// sum are
//     D_x^kappa sum_l a_l M_l = (-1)^|kappa| sum_l (kappa + l)!/l! a_{kappa+l} M_l ,   |kappa| <= 2,
// which needs the coefficients a_k up to order P + 2; they come from the recurrence of App. A.4,
//     n R^2 a_k = (2n-1) sum_i d_i a_{k-e_i} - (n-1) sum_i a_{k-2e_i},  a_0 = 1/R,  n = |k|, d = x - y_c.
// Near field: the K-point rule over the group's P2P list; the 19-point correction of the few near panels
// (D: R-9) is added afterwards by k_reaction_corr exactly as in direct mode.
#include <math.h>
#include <vector>
#include "pb_internal.cuh"

#define ST_MAXP 8                 // coefficient order P + 2 <= 10
#define ST_GROUP 32               // sites per group = threads per k_site_m2p block
#define ST_SPLIT 8                // blocks per group: each takes an eighth of the group's cell list

static double st_fact(int n) { double f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }

// kappa = (0,0,0), e_x, e_y, e_z, then xx, xy, xz, yy, yz, zz  (the output order phi, grad[3], hess[6])
static const int ST_KAPPA[10][3] = {{0, 0, 0}, {1, 0, 0}, {0, 1, 0}, {0, 0, 1}, {2, 0, 0},
                                    {1, 1, 0}, {1, 0, 1}, {0, 2, 0}, {0, 1, 1}, {0, 0, 2}};

// tables for order P: neighbours of every k in the recurrence, and (index, factor) of every (kappa, l)
int pb_site_tables(pb_ctx* ctx)
{
    pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    const int P = ctx->prm.order_P, Q = P + 2;
    const int NkQ = pb_nk(Q), NkP = pb_nk(P);
    std::vector<int32_t> nb((size_t)NkQ * 8, -1);      // [k][0..2] = k - e_d, [3..5] = k - 2 e_d, [6] = n, [7] unused
    for (int a = 0; a <= Q; ++a)
        for (int b = 0; b <= Q - a; ++b)
            for (int c = 0; c <= Q - a - b; ++c) {
                const int k = mom_index(a, b, c);
                const int e[3] = {a, b, c};
                for (int d = 0; d < 3; ++d) {
                    int m1[3] = {a, b, c}, m2[3] = {a, b, c};
                    m1[d] -= 1; m2[d] -= 2;
                    if (e[d] >= 1) nb[(size_t)k * 8 + d] = mom_index(m1[0], m1[1], m1[2]);
                    if (e[d] >= 2) nb[(size_t)k * 8 + 3 + d] = mom_index(m2[0], m2[1], m2[2]);
                }
                nb[(size_t)k * 8 + 6] = a + b + c;
            }
    std::vector<int32_t> di((size_t)10 * NkP);
    std::vector<double> df((size_t)10 * NkP);
    for (int q = 0; q < 10; ++q) {
        const int* kp = ST_KAPPA[q];
        const double sgn = ((kp[0] + kp[1] + kp[2]) & 1) ? -1.0 : 1.0;
        for (int a = 0; a <= P; ++a)
            for (int b = 0; b <= P - a; ++b)
                for (int c = 0; c <= P - a - b; ++c) {
                    const int l = mom_index(a, b, c);
                    di[(size_t)q * NkP + l] = mom_index(a + kp[0], b + kp[1], c + kp[2]);
                    df[(size_t)q * NkP + l] = sgn * st_fact(a + kp[0]) / st_fact(a) * st_fact(b + kp[1]) / st_fact(b) *
                                              st_fact(c + kp[2]) / st_fact(c);
                }
    }
    PB_TRY(pb_dalloc_t(ctx, &s.nb_idx, nb.size(), CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &s.dv_idx, di.size(), CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &s.dv_fac, df.size(), CAT_SITE_NEAR));
    PB_CUDA(cudaMemcpyAsync(s.nb_idx, nb.data(), sizeof(int32_t) * nb.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(s.dv_idx, di.data(), sizeof(int32_t) * di.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(s.dv_fac, df.data(), sizeof(double) * df.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaStreamSynchronize(st));   // the host vectors go out of scope
    s.t_P = P;
    return PB_OK;
}

// ---- far field: one block per site group, one lane per site; every lane walks the group's cell list --------
// a_k of the lane's (site, cell) pair live in shared memory, [k][lane] (conflict free); the cell's moments,
// the neighbour and derivative tables are the same for all lanes (broadcast loads).
// out [ST_SPLIT][na][10] (Morton order of the sites; one slab per share of the list, added in order by
// k_site_finish): phi, grad, hess WITHOUT the 1/(4 pi); NO = 4 or 10 outputs wanted.
template <int NO>
__global__ void __launch_bounds__(ST_GROUP)
k_site_m2p(int64_t na, int P, const double* __restrict__ sx, const double* __restrict__ sy, const double* __restrict__ sz,
           const int32_t* __restrict__ m2p_off, const int32_t* __restrict__ m2p_cell, const double* __restrict__ cx,
           const double* __restrict__ cy, const double* __restrict__ cz, const double* __restrict__ M,
           const int32_t* __restrict__ nb_idx, const int32_t* __restrict__ dv_idx, const double* __restrict__ dv_fac,
           double* __restrict__ out)
{
    extern __shared__ double st_a[];                   // [NkQ][ST_GROUP]
    const int lane = threadIdx.x;
    const int64_t g = blockIdx.x;
    const int part = blockIdx.y;                       // this block's share of the group's cell list
    const int64_t i = g * ST_GROUP + lane;
    const int64_t ic = i < na ? i : na - 1;            // padding lanes repeat the last site; never stored
    const double x = sx[ic], y = sy[ic], z = sz[ic];
    const int Q = P + (NO > 4 ? 2 : 1);                // the gradient needs one order more than the sum, the Hessian two
    const int NkQ = pb_nk(Q), NkP = pb_nk(P);
    double acc[NO];
#pragma unroll
    for (int q = 0; q < NO; ++q) acc[q] = 0.0;
    double* a = st_a + lane;
    const int32_t l0 = m2p_off[g], ln = m2p_off[g + 1] - l0;
    const int32_t e_lo = l0 + (int32_t)((int64_t)ln * part / ST_SPLIT), e_hi = l0 + (int32_t)((int64_t)ln * (part + 1) / ST_SPLIT);
    for (int32_t e = e_lo; e < e_hi; ++e) {
        const int32_t c = m2p_cell[e];
        const double d[3] = {x - cx[c], y - cy[c], z - cz[c]};
        const double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
        const double ri = pb_rsqrt(r2), ri2 = ri * ri;
        a[0] = ri;
        for (int k = 1; k < NkQ; ++k) {                // graded order: every neighbour is already there
            const int4 na_ = reinterpret_cast<const int4*>(nb_idx)[2 * k], nb_ = reinterpret_cast<const int4*>(nb_idx)[2 * k + 1];
            const int32_t nb[8] = {na_.x, na_.y, na_.z, na_.w, nb_.x, nb_.y, nb_.z, nb_.w};
            const int n = nb[6];
            double s1 = 0.0, s2 = 0.0;
#pragma unroll
            for (int dd = 0; dd < 3; ++dd) {
                const int32_t k1 = nb[dd], k2 = nb[3 + dd];
                if (k1 >= 0) s1 = fma(d[dd], a[(size_t)k1 * ST_GROUP], s1);
                if (k2 >= 0) s2 += a[(size_t)k2 * ST_GROUP];
            }
            a[(size_t)k * ST_GROUP] = ((2 * n - 1) * s1 - (n - 1) * s2) * ri2 / (double)n;
        }
        const double* mv = M + (size_t)c * 2 * NkP;
        const double* mk = mv + NkP;
        for (int l = 0; l < NkP; ++l) {
            const double m = mv[l] - mk[l];            // phi_solv = V_L(dphi) - K_L(phi)
#pragma unroll
            for (int q = 0; q < NO; ++q)
                acc[q] = fma(dv_fac[(size_t)q * NkP + l] * m, a[(size_t)dv_idx[(size_t)q * NkP + l] * ST_GROUP], acc[q]);
        }
    }
    if (i < na) {
#pragma unroll
        for (int q = 0; q < NO; ++q) out[((int64_t)part * na + i) * 10 + q] = acc[q];
    }
}

// ---- near field: block = 4 sites of a group x the group's whole P2P list (source-point ranges) ---------------
// Same per-pair arithmetic as the direct kernel (k_reaction, pb_sites.cu), restated here for the list form.
template <bool HESS>
__device__ __forceinline__ void st_point(double dx, double dy, double dz, double wS, double kx, double ky, double kz,
                                         double* __restrict__ o)
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
        const double c3 = 3.0 * ri5;
        o[4] += a * dx * dx + g + c3 * 2.0 * kx * dx;
        o[5] += a * dx * dy + c3 * (kx * dy + ky * dx);
        o[6] += a * dx * dz + c3 * (kx * dz + kz * dx);
        o[7] += a * dy * dy + g + c3 * 2.0 * ky * dy;
        o[8] += a * dy * dz + c3 * (ky * dz + kz * dy);
        o[9] += a * dz * dz + g + c3 * 2.0 * kz * dz;
    }
}

#define SP_ST 4
#define SP_THREADS 128
template <bool HESS>
__global__ void __launch_bounds__(SP_THREADS)
k_site_p2p(int64_t na, const double* __restrict__ sx, const double* __restrict__ sy, const double* __restrict__ sz,
           const int32_t* __restrict__ p2p_off, const int32_t* __restrict__ p2p_lo, const int32_t* __restrict__ p2p_hi,
           const double4* __restrict__ srec, double* __restrict__ out /*[na][10]*/)
{
    constexpr int NO = HESS ? 10 : 4;
    __shared__ double red[SP_THREADS / 32][SP_ST][NO];
    const int64_t g = blockIdx.x / (ST_GROUP / SP_ST);
    const int64_t m0 = g * ST_GROUP + (blockIdx.x % (ST_GROUP / SP_ST)) * SP_ST;
    if (m0 >= na) return;
    double r[SP_ST][3], acc[SP_ST][NO];
#pragma unroll
    for (int t = 0; t < SP_ST; ++t) {
        const int64_t m = m0 + t < na ? m0 + t : na - 1;   // clamp: duplicates are not written
        r[t][0] = sx[m]; r[t][1] = sy[m]; r[t][2] = sz[m];
#pragma unroll
        for (int c = 0; c < NO; ++c) acc[t][c] = 0.0;
    }
    for (int32_t rr = p2p_off[g]; rr < p2p_off[g + 1]; ++rr) {
        const int32_t lo = p2p_lo[rr], hi = p2p_hi[rr];
        for (int32_t s = lo + threadIdx.x; s < hi; s += SP_THREADS) {
            const double4 ra = srec[2 * (int64_t)s], rb = srec[2 * (int64_t)s + 1];
#pragma unroll
            for (int t = 0; t < SP_ST; ++t)
                st_point<HESS>(r[t][0] - ra.x, r[t][1] - ra.y, r[t][2] - ra.z, ra.w, rb.x, rb.y, rb.z, acc[t]);
        }
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
    for (int t = 0; t < SP_ST; ++t)
#pragma unroll
        for (int c = 0; c < NO; ++c) {
            double v = acc[t][c];
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) red[w][t][c] = v;
        }
    __syncthreads();
    if (threadIdx.x < SP_ST * NO) {
        const int t = threadIdx.x / NO, c = threadIdx.x % NO;
        if (m0 + t < na) {
            double v = 0;
            for (int k = 0; k < SP_THREADS / 32; ++k) v += red[k][t][c];
            out[(m0 + t) * 10 + c] = v;
        }
    }
}

// near + far, 1/(4 pi), back to the caller's site order
__global__ void k_site_finish(int64_t na, int NO, const int32_t* __restrict__ perm, const double* __restrict__ nearp,
                              const double* __restrict__ farp, double* __restrict__ phi, double* __restrict__ grad,
                              double* __restrict__ hess)
{
    int64_t gidx = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (gidx >= na * NO) return;
    const int64_t i = gidx / NO;
    const int c = (int)(gidx % NO);
    const int64_t m = perm[i];
    double f = 0.0;
    for (int sp = 0; sp < ST_SPLIT; ++sp) f += farp[((int64_t)sp * na + i) * 10 + c];
    const double v = (nearp[i * 10 + c] + f) * PB_INV4PI;
    if (c == 0) { if (phi) phi[m] = v; }
    else if (c < 4) { if (grad) grad[3 * m + c - 1] = v; }
    else if (hess) hess[6 * m + c - 4] = v;
}

// lists, needed cells and tables for the current tree, sites and order (lazily, like the site-near table)
int pb_site_tree_build(pb_ctx* ctx)
{
    pb_sites& s = ctx->sites;
    PB_TRY(pb_site_lists_build(ctx));
    PB_TRY(pb_site_farfield_setup(ctx));
    PB_TRY(pb_site_tables(ctx));
    s.tree_built = true;
    return PB_OK;
}

// phi/grad/hess at the sites by the treecode; the source records of x must be in place (pb_weights)
int pb_reaction_field_tree(pb_ctx* ctx, double* phi, double* grad, double* hess)
{
    pb_tree& t = ctx->tree;
    pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    const bool H = hess != nullptr;
    const int NO = H ? 10 : 4;
    PB_TRY(pb_scratch(ctx, (size_t)(1 + ST_SPLIT) * s.na * 10 * sizeof(double) + 4096));
    double* nearp = ctx->scratch;
    double* farp = ctx->scratch + (size_t)s.na * 10;
    PB_TRY(pb_upward(ctx, st, s.t_need_leaf, s.t_n_need_leaf, s.t_up_link));
    const size_t sm = (size_t)pb_nk(t.P + 2) * ST_GROUP * sizeof(double);
    size_t* sm_set = ctx->attr_site_bytes;             // per device: remembered per context
    if (sm > 48 * 1024 && sm > sm_set[H ? 1 : 0]) {
        if (H) PB_CUDA(cudaFuncSetAttribute(k_site_m2p<10>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        else PB_CUDA(cudaFuncSetAttribute(k_site_m2p<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        sm_set[H ? 1 : 0] = sm;
    }
    const unsigned G = (unsigned)s.t_groups;
    if (H) {
        k_site_m2p<10><<<dim3(G, ST_SPLIT), ST_GROUP, sm, st>>>(s.na, t.P, s.tpos[0], s.tpos[1], s.tpos[2], s.t_m2p_off, s.t_m2p_cell, t.c_ctr[0],
                                               t.c_ctr[1], t.c_ctr[2], t.M, s.nb_idx, s.dv_idx, s.dv_fac, farp);
        PB_LAUNCH_CHECK();
        k_site_p2p<true><<<G * (ST_GROUP / SP_ST), SP_THREADS, 0, st>>>(s.na, s.tpos[0], s.tpos[1], s.tpos[2], s.t_p2p_off,
                                                                        s.t_p2p_lo, s.t_p2p_hi, t.srec, nearp);
        PB_LAUNCH_CHECK();
    } else {
        k_site_m2p<4><<<dim3(G, ST_SPLIT), ST_GROUP, sm, st>>>(s.na, t.P, s.tpos[0], s.tpos[1], s.tpos[2], s.t_m2p_off, s.t_m2p_cell, t.c_ctr[0],
                                              t.c_ctr[1], t.c_ctr[2], t.M, s.nb_idx, s.dv_idx, s.dv_fac, farp);
        PB_LAUNCH_CHECK();
        k_site_p2p<false><<<G * (ST_GROUP / SP_ST), SP_THREADS, 0, st>>>(s.na, s.tpos[0], s.tpos[1], s.tpos[2], s.t_p2p_off,
                                                                         s.t_p2p_lo, s.t_p2p_hi, t.srec, nearp);
        PB_LAUNCH_CHECK();
    }
    k_site_finish<<<pb_blocks(s.na * NO, 128), 128, 0, st>>>(s.na, NO, s.tperm, nearp, farp, phi, grad, hess);
    PB_LAUNCH_CHECK();
    return PB_OK;
}
