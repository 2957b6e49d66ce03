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

// ---- far field of the potential and its gradient in radial form (the SCF loop's call: no Hessian) ---------------------
// The order-P Taylor sum of a cell is, exactly (D: section 6),  phi(x) = sum_{|alpha| + 2j <= P} u_{|alpha|+j}(R) d^alpha F_{alpha,j},
// d = x - y_c, with the single layer F = F^V - F^K of the matvec's far-field terms (phi_solv = V_L(dphi) - K_L(phi),
// Eq. 12) and u_m = (2m-1)!! / R^(2m+1).  Because u_m'(R)/R = -u_{m+1}, its gradient in the target is
//     grad phi = sum_m [ u_m G_m - u_{m+1} d W_m ],   W_m = sum_{|alpha|+j=m} d^alpha F,   G_m = sum_{|alpha|+j=m} grad(d^alpha) F,
// the derivative of the SAME truncated sum that k_site_m2p differentiates through the coefficients a_{kappa+l}; here it
// costs four FMA per term and four products per monomial instead of an order-(P+1) coefficient recurrence in shared
// memory (C4: 64 -> see profiles).  One block per group of 32 sites (a lane per site); its 8 warps take the cells
// w, w + 8, ... of the group's list, each with its own ring of TMA-filled slots as in k_m2p2.
#define SG_W 8
#define SG_NS 4
#define SG_THREADS (32 * SG_W)

__host__ __device__ static constexpr int sg_nt(int P)
{
    int t = 0;
    for (int a = 0; a <= P; ++a)
        for (int b = 0; b <= P - a; ++b)
            for (int c = 0; c <= P - a - b; ++c) t += (P - a - b - c) / 2 + 1;
    return t;
}

template <int P> struct sg_cfg {
    static constexpr int NT = sg_nt(P);
    static constexpr size_t FF_BYTES0 = (size_t)SG_W * SG_NS * NT * sizeof(double2);
    static constexpr size_t RED_BYTES = (size_t)SG_W * 10 * ST_GROUP * sizeof(double);
    static constexpr size_t FF_BYTES = FF_BYTES0 > RED_BYTES ? FF_BYTES0 : RED_BYTES;
    static constexpr size_t SMEM = FF_BYTES + SG_W * SG_NS * sizeof(uint64_t);
};

// HESS: also the Hessian (the solve's closing call, Eq. 21/24), by differentiating once more:
//     d_i d_j phi = sum_m [ u_m H_m,ij - u_{m+1} (d_i G_m,j + d_j G_m,i + delta_ij W_m) + u_{m+2} d_i d_j W_m ],
// H_m,ij = sum_{|alpha|+j=m} d_i d_j (d^alpha) F, in a second sweep over the cell's terms (six more FMA per term; orders
// P <= 6).  At P = 5, 6 the compiler keeps the 6 (P + 1) sums of the second sweep in local memory (L1-resident; splitting
// the sweep further made it spill instead); the call is still 4.3 times faster than the coefficient recurrence (C4: 140 -> 33 ms).
template <int P, bool HESS>
__global__ void __launch_bounds__(SG_THREADS, HESS || P > 6 ? 1 : 2)
k_site_grad(int64_t na, const double* __restrict__ sx, const double* __restrict__ sy, const double* __restrict__ sz,
            const int32_t* __restrict__ m2p_off, const int32_t* __restrict__ m2p_cell, const double* __restrict__ cx,
            const double* __restrict__ cy, const double* __restrict__ cz, const double2* __restrict__ FF,
            double* __restrict__ out /*[na][10]: phi, grad, hess (Morton order of the sites), without the 1/(4 pi)*/)
{
    constexpr int NT = sg_cfg<P>::NT, NS = SG_NS, NO = HESS ? 10 : 4;
    extern __shared__ __align__(128) unsigned char sgraw[];
    const int tid = threadIdx.x, lane = tid & 31, sub = tid >> 5;
    double2* ffw = reinterpret_cast<double2*>(sgraw) + (size_t)sub * NS * NT;
    uint64_t* fullw = reinterpret_cast<uint64_t*>(sgraw + sg_cfg<P>::FF_BYTES) + sub * NS;
    const int64_t g = blockIdx.x;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) pb_mbar_init(&fullw[s], 1);
        pb_mbar_fence_init();
    }
    __syncthreads();
    const int64_t i = g * ST_GROUP + lane;
    const int64_t ic = i < na ? i : na - 1;            // padding lanes repeat the last site; never stored
    const double x = sx[ic], y = sy[ic], z = sz[ic];
    const int32_t e0 = m2p_off[g] + sub, count = m2p_off[g + 1] - m2p_off[g];
    const int nw = count > sub ? (count - sub + SG_W - 1) / SG_W : 0;
    auto issue = [&](int k, int32_t cell) {
        const int slot = k % NS;
        pb_mbar_expect_tx(&fullw[slot], (uint32_t)(NT * sizeof(double2)));
        pb_bulk_g2s(ffw + (size_t)slot * NT, FF + (int64_t)cell * NT, (uint32_t)(NT * sizeof(double2)), &fullw[slot]);
    };
    if (lane == 0)
        for (int k = 0; k < NS - 1 && k < nw; ++k) issue(k, m2p_cell[e0 + SG_W * k]);
    int32_t idn = NS - 1 < nw ? m2p_cell[e0 + SG_W * (NS - 1)] : 0;
    int32_t cn = nw > 0 ? m2p_cell[e0] : 0;
    double cxn = cx[cn], cyn = cy[cn], czn = cz[cn];
    double o[NO];
#pragma unroll
    for (int q = 0; q < NO; ++q) o[q] = 0.0;
#pragma unroll 1
    for (int k = 0; k < nw; ++k) {
        const int kn = k + NS - 1;
        if (lane == 0 && kn < nw) issue(kn, idn);
        idn = kn + 1 < nw ? m2p_cell[e0 + SG_W * (kn + 1)] : 0;
        const double dx = x - cxn, dy = y - cyn, dz = z - czn;
        if (k + 1 < nw) {
            cn = m2p_cell[e0 + SG_W * (k + 1)];
            cxn = cx[cn]; cyn = cy[cn]; czn = cz[cn];
        }
        pb_mbar_wait(&fullw[k % NS], (uint32_t)((k / NS) & 1));
        const double2* ff = ffw + (size_t)(k % NS) * NT;
        const double R2 = dx * dx + dy * dy + dz * dz;
        const double ri = pb_rsqrt(R2), ri2 = ri * ri;
        double sp = 0.0, sgx = 0.0, sgy = 0.0, sgz = 0.0, sw1 = 0.0;
        double sw2 = 0.0, g1x = 0.0, g1y = 0.0, g1z = 0.0, sh[6] = {0, 0, 0, 0, 0, 0};
        {   // first sweep over the cell's terms: W_m and G_m, then their radial sums
            double W[P + 1], GX[P + 1], GY[P + 1], GZ[P + 1];
#pragma unroll
            for (int m = 0; m <= P; ++m) { W[m] = 0.0; GX[m] = 0.0; GY[m] = 0.0; GZ[m] = 0.0; }
            int e = 0;
            double X = 1.0, X1 = 0.0;                  // x^a and a x^(a-1)
#pragma unroll
            for (int a = 0; a <= P; ++a) {
                double Y = 1.0, Y1 = 0.0;
#pragma unroll
                for (int b = 0; b <= P - a; ++b) {
                    const double XY = X * Y, X1Y = X1 * Y, XY1 = X * Y1;
                    double Z = 1.0, Z1 = 0.0;
#pragma unroll
                    for (int c = 0; c <= P - a - b; ++c) {
                        const int n = a + b + c;
                        const double mono = XY * Z, mx = X1Y * Z, my = XY1 * Z, mz = XY * Z1;
#pragma unroll
                        for (int j = 0; j <= (P - n) / 2; ++j) {
                            const double2 f2 = ff[e];
                            ++e;
                            const double f = f2.x - f2.y;      // V_L(dphi) - K_L(phi)
                            W[n + j] = fma(mono, f, W[n + j]);
                            if (a > 0) GX[n + j] = fma(mx, f, GX[n + j]);
                            if (b > 0) GY[n + j] = fma(my, f, GY[n + j]);
                            if (c > 0) GZ[n + j] = fma(mz, f, GZ[n + j]);
                        }
                        Z1 = (double)(c + 1) * Z;
                        Z *= dz;
                    }
                    Y1 = (double)(b + 1) * Y;
                    Y *= dy;
                }
                X1 = (double)(a + 1) * X;
                X *= dx;
            }
            double u = ri;
#pragma unroll
            for (int m = 0; m <= P; ++m) {
                const double un = (2 * m + 1) * u * ri2;           // u_{m+1}
                sp = fma(u, W[m], sp);
                sgx = fma(u, GX[m], sgx);
                sgy = fma(u, GY[m], sgy);
                sgz = fma(u, GZ[m], sgz);
                sw1 = fma(un, W[m], sw1);
                if (HESS) {
                    const double unn = (2 * m + 3) * un * ri2;     // u_{m+2}
                    sw2 = fma(unn, W[m], sw2);
                    g1x = fma(un, GX[m], g1x);
                    g1y = fma(un, GY[m], g1y);
                    g1z = fma(un, GZ[m], g1z);
                }
                u = un;
            }
        }
        if (HESS) {   // second sweep: H_m,ij (six sums per layer; terms of total degree < 2 do not contribute)
            double HXX[P + 1], HXY[P + 1], HXZ[P + 1], HYY[P + 1], HYZ[P + 1], HZZ[P + 1];
#pragma unroll
            for (int m = 0; m <= P; ++m) { HXX[m] = 0.0; HXY[m] = 0.0; HXZ[m] = 0.0; HYY[m] = 0.0; HYZ[m] = 0.0; HZZ[m] = 0.0; }
            int e = 0;
            double X = 1.0, X1 = 0.0, X2 = 0.0;        // x^a, a x^(a-1), a (a-1) x^(a-2)
#pragma unroll
            for (int a = 0; a <= P; ++a) {
                double Y = 1.0, Y1 = 0.0, Y2 = 0.0;
#pragma unroll
                for (int b = 0; b <= P - a; ++b) {
                    const double XY = X * Y, X1Y = X1 * Y, XY1 = X * Y1, X2Y = X2 * Y, XY2 = X * Y2, X1Y1 = X1 * Y1;
                    double Z = 1.0, Z1 = 0.0, Z2 = 0.0;
#pragma unroll
                    for (int c = 0; c <= P - a - b; ++c) {
                        const int n = a + b + c;
                        const double hxx = X2Y * Z, hxy = X1Y1 * Z, hxz = X1Y * Z1, hyy = XY2 * Z, hyz = XY1 * Z1, hzz = XY * Z2;
#pragma unroll
                        for (int j = 0; j <= (P - n) / 2; ++j) {
                            if (n >= 2) {
                                const double2 f2 = ff[e];
                                const double f = f2.x - f2.y;
                                if (a > 1) HXX[n + j] = fma(hxx, f, HXX[n + j]);
                                if (a > 0 && b > 0) HXY[n + j] = fma(hxy, f, HXY[n + j]);
                                if (a > 0 && c > 0) HXZ[n + j] = fma(hxz, f, HXZ[n + j]);
                                if (b > 1) HYY[n + j] = fma(hyy, f, HYY[n + j]);
                                if (b > 0 && c > 0) HYZ[n + j] = fma(hyz, f, HYZ[n + j]);
                                if (c > 1) HZZ[n + j] = fma(hzz, f, HZZ[n + j]);
                            }
                            ++e;
                        }
                        Z2 = (double)(c + 1) * Z1;
                        Z1 = (double)(c + 1) * Z;
                        Z *= dz;
                    }
                    Y2 = (double)(b + 1) * Y1;
                    Y1 = (double)(b + 1) * Y;
                    Y *= dy;
                }
                X2 = (double)(a + 1) * X1;
                X1 = (double)(a + 1) * X;
                X *= dx;
            }
            double u = ri;
#pragma unroll
            for (int m = 0; m <= P; ++m) {
                sh[0] = fma(u, HXX[m], sh[0]);
                sh[1] = fma(u, HXY[m], sh[1]);
                sh[2] = fma(u, HXZ[m], sh[2]);
                sh[3] = fma(u, HYY[m], sh[3]);
                sh[4] = fma(u, HYZ[m], sh[4]);
                sh[5] = fma(u, HZZ[m], sh[5]);
                u = (2 * m + 1) * u * ri2;
            }
        }
        o[0] += sp;
        o[1] += sgx - dx * sw1;
        o[2] += sgy - dy * sw1;
        o[3] += sgz - dz * sw1;
        if (HESS) {                                            // xx, xy, xz, yy, yz, zz
            o[4] += sh[0] - 2.0 * dx * g1x - sw1 + dx * dx * sw2;
            o[5] += sh[1] - (dx * g1y + dy * g1x) + dx * dy * sw2;
            o[6] += sh[2] - (dx * g1z + dz * g1x) + dx * dz * sw2;
            o[7] += sh[3] - 2.0 * dy * g1y - sw1 + dy * dy * sw2;
            o[8] += sh[4] - (dy * g1z + dz * g1y) + dy * dz * sw2;
            o[9] += sh[5] - 2.0 * dz * g1z - sw1 + dz * dz * sw2;
        }
        __syncwarp();
    }
    __syncthreads();
    double* red = reinterpret_cast<double*>(sgraw);    // [SG_W][NO][ST_GROUP]: the warps' sums, added in warp order
#pragma unroll
    for (int q = 0; q < NO; ++q) red[(sub * NO + q) * ST_GROUP + lane] = o[q];
    __syncthreads();
    for (int t = tid; t < NO * ST_GROUP; t += SG_THREADS) {
        const int m = t / ST_GROUP, l = t % ST_GROUP;
        const int64_t ii = g * ST_GROUP + l;
        if (ii < na) {
            double v = 0;
#pragma unroll
            for (int q = 0; q < SG_W; ++q) v += red[(q * NO + m) * ST_GROUP + l];
            out[ii * 10 + m] = v;
        }
    }
}

template <int P, bool HESS>
static cudaError_t launch_site_grad(pb_ctx* ctx, double* farp)
{
    pb_tree& t = ctx->tree;
    pb_sites& s = ctx->sites;
    cudaError_t e = cudaFuncSetAttribute(k_site_grad<P, HESS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sg_cfg<P>::SMEM);
    if (e != cudaSuccess) return e;
    k_site_grad<P, HESS><<<(unsigned)s.t_groups, SG_THREADS, sg_cfg<P>::SMEM, ctx->stream>>>(
        s.na, s.tpos[0], s.tpos[1], s.tpos[2], s.t_m2p_off, s.t_m2p_cell, t.c_ctr[0], t.c_ctr[1], t.c_ctr[2], t.FF, farp);
    return cudaSuccess;
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
    if (H && t.P > 6) {
        // orders 7, 8: the radial form's 10 (P + 1) partial sums per cell do not fit the register file; the coefficient
        // recurrence (k_site_m2p) differentiates the same truncated sum
        k_site_m2p<10><<<dim3(G, ST_SPLIT), ST_GROUP, sm, st>>>(s.na, t.P, s.tpos[0], s.tpos[1], s.tpos[2], s.t_m2p_off, s.t_m2p_cell, t.c_ctr[0],
                                               t.c_ctr[1], t.c_ctr[2], t.M, s.nb_idx, s.dv_idx, s.dv_fac, farp);
        PB_LAUNCH_CHECK();
    } else {
        // radial form, one slab of far-field sums; the other slabs are zero
        PB_CUDA(cudaMemsetAsync(farp + (size_t)s.na * 10, 0, (size_t)(ST_SPLIT - 1) * s.na * 10 * sizeof(double), st));
        cudaError_t e = cudaSuccess;
        if (H) {
            switch (t.P) {
            case 0: e = launch_site_grad<0, true>(ctx, farp); break;
            case 1: e = launch_site_grad<1, true>(ctx, farp); break;
            case 2: e = launch_site_grad<2, true>(ctx, farp); break;
            case 3: e = launch_site_grad<3, true>(ctx, farp); break;
            case 4: e = launch_site_grad<4, true>(ctx, farp); break;
            case 5: e = launch_site_grad<5, true>(ctx, farp); break;
            default: e = launch_site_grad<6, true>(ctx, farp); break;
            }
        } else {
            switch (t.P) {
            case 0: e = launch_site_grad<0, false>(ctx, farp); break;
            case 1: e = launch_site_grad<1, false>(ctx, farp); break;
            case 2: e = launch_site_grad<2, false>(ctx, farp); break;
            case 3: e = launch_site_grad<3, false>(ctx, farp); break;
            case 4: e = launch_site_grad<4, false>(ctx, farp); break;
            case 5: e = launch_site_grad<5, false>(ctx, farp); break;
            case 6: e = launch_site_grad<6, false>(ctx, farp); break;
            case 7: e = launch_site_grad<7, false>(ctx, farp); break;
            case 8: e = launch_site_grad<8, false>(ctx, farp); break;
            default: return pb_fail(ctx, PB_ERR_INVALID_ARG, "internal: site treecode needs order_P <= 8");
            }
        }
        PB_CUDA(e);
        PB_LAUNCH_CHECK();
    }
    if (H)
        k_site_p2p<true><<<G * (ST_GROUP / SP_ST), SP_THREADS, 0, st>>>(s.na, s.tpos[0], s.tpos[1], s.tpos[2], s.t_p2p_off,
                                                                        s.t_p2p_lo, s.t_p2p_hi, t.srec, nearp);
    else
        k_site_p2p<false><<<G * (ST_GROUP / SP_ST), SP_THREADS, 0, st>>>(s.na, s.tpos[0], s.tpos[1], s.tpos[2], s.t_p2p_off,
                                                                         s.t_p2p_lo, s.t_p2p_hi, t.srec, nearp);
    PB_LAUNCH_CHECK();
    k_site_finish<<<pb_blocks(s.na * NO, 128), 128, 0, st>>>(s.na, NO, s.tperm, nearp, farp, phi, grad, hess);
    PB_LAUNCH_CHECK();
    return PB_OK;
}
