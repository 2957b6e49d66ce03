// pb_rhstree.cu -- the multipole right-hand side Eq. (8) by a treecode with the SITES as sources in their own
// octree (S: section 8(f) item 1, second half; the paper sums it directly).
//
//   b_i = 1/(4 pi eps_1) sum_k [ q_k/R + p_k.d/R^3 + d.Q_k.d/(2 R^5) ],  d = c_i - r_k,  p = dip + mu  (Eq. 8, Eq. 10)
//
// A point multipole is a differential operator in the source variable applied to 1/|x - y|:
//   phi_k(x) = [ q + p_i d/dy_i + (1/6) Q_ij d^2/dy_i dy_j ] (1/|x - y|) at y = r_k      (Q traceless, Eq. 7's convention)
// so with the order-P Taylor expansion of the kernel about a cell centre y_c (D: App. A.4),
//   1/|x - y| ~ sum_{|k|<=P} a_k(x, y_c) (y - y_c)^k,  the cell's moments are, with h = r - y_c over its sites,
//   M_k = sum_sites [ q h^k + sum_i p_i k_i h^{k-e_i} + (1/6) sum_ij Q_ij k_i (k_j - delta_ij) h^{k-e_i-e_j} ]
// and the far field sum_k a_k M_k is evaluated in the radial form of the matvec's M2P (D: section 6; Laplace only,
// one layer): the same M -> F table, the same u_m(R) recurrence.  Near sites are summed directly with the
// arithmetic of k_rhs.  Targets are the panel centroids in Morton order in the matvec's groups of 64; a group's
// lists come from the same traversal and per-target MAC (Eq. 28) as the matvec's, against the site tree, with
// theta_rhs = 0.7 theta (the dipole and quadrupole terms are first and second source derivatives of the expansion
// and lose about one order each, like the target derivatives of the site-side treecode).
#include <algorithm>
#include <math.h>
#include "pb_internal.cuh"

#define PB_RHS_THETA_SCALE 0.7
#define RT_NCRIT 32          // sites per leaf of the site tree
#define RT_M2P_MIN 4         // cells with fewer sites are summed directly
#define RT_W 8               // warps per block (one block = one target group)
#define RT_NS 4              // cell slots per warp (TMA ring)
#define RT_THREADS (32 * RT_W)
#define RT_TILE 64           // sites per shared-memory tile of the near part
#define RT_REC 16            // doubles per packed site record

__host__ __device__ static constexpr int rt_nt(int P)
{
    int t = 0;
    for (int a = 0; a <= P; ++a)
        for (int b = 0; b <= P - a; ++b)
            for (int c = 0; c <= P - a - b; ++c) t += (P - a - b - c) / 2 + 1;
    return t;
}

// ---- per call: the sites' records in Morton order (mu changes every SCF step) ------------------------------------------
// rec[s] = x, y, z, q | p_x, p_y, p_z, Qxx/2 | Qxy, Qxz, Qyy/2, Qyz | Qzz/2, 0, 0, 0     (d.Q.d/2 as in k_rhs)
__global__ void k_rhs_pack(int64_t na, const int32_t* __restrict__ perm, const double* __restrict__ pos,
                           const double* __restrict__ q, const double* __restrict__ dip, const double* __restrict__ mu,
                           const double* __restrict__ quad, double* __restrict__ rec)
{
    const int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= na) return;
    const int64_t o = perm[s];
    double* r = rec + RT_REC * s;
    r[0] = pos[3 * o]; r[1] = pos[3 * o + 1]; r[2] = pos[3 * o + 2]; r[3] = q[o];
    for (int d = 0; d < 3; ++d) r[4 + d] = dip[3 * o + d] + (mu ? mu[3 * o + d] : 0.0);
    r[7] = 0.5 * quad[6 * o]; r[8] = quad[6 * o + 1]; r[9] = quad[6 * o + 2];
    r[10] = 0.5 * quad[6 * o + 3]; r[11] = quad[6 * o + 4]; r[12] = 0.5 * quad[6 * o + 5];
    r[13] = 0.0; r[14] = 0.0; r[15] = 0.0;
}

__global__ void k_rhs_gather_pos(int64_t na, const int32_t* __restrict__ perm, const double* __restrict__ pos,
                                 double* __restrict__ x, double* __restrict__ y, double* __restrict__ z)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= na) return;
    const int64_t o = perm[i];
    x[i] = pos[3 * o]; y[i] = pos[3 * o + 1]; z[i] = pos[3 * o + 2];
}

// ---- moments of the needed cells (directly from the cell's sites, whatever its level) and their F terms ------------------
#define RP_THREADS 128
#define RP_CH 32
#define RP_LD (PB_MAX_P + 1)
struct rp_args {
    int P, Nk, NT, NTp;
    const int32_t *need, *c_first, *c_last;
    const double *cx, *cy, *cz, *rec;
    const unsigned char *ka, *kb, *kc;      // exponents of moment index k
    const int32_t *cv_off, *cv_idx;
    const double* cv_coef;
    double* FF;
};

__global__ void __launch_bounds__(RP_THREADS) k_rhs_p2m(rp_args a)
{
    __shared__ double pw[3][RP_CH][RP_LD];
    __shared__ double cf[RP_CH][10];
    extern __shared__ double mom[];                      // [Nk]
    const int tid = threadIdx.x, Nk = a.Nk, P = a.P;
    const int32_t c = a.need[blockIdx.x];
    const int32_t f = a.c_first[c], l = a.c_last[c];
    const double ycx = a.cx[c], ycy = a.cy[c], ycz = a.cz[c];
    int ea[3], eb[3], ec[3];
    double acc[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        const int k = tid + r * RP_THREADS;
        ea[r] = k < Nk ? a.ka[k] : 0; eb[r] = k < Nk ? a.kb[k] : 0; ec[r] = k < Nk ? a.kc[k] : 0;
    }
    for (int32_t base = f; base < l; base += RP_CH) {
        const int np = l - base < RP_CH ? l - base : RP_CH;
        __syncthreads();
        if (tid < np) {
            const double* r = a.rec + RT_REC * (int64_t)(base + tid);
            const double h[3] = {r[0] - ycx, r[1] - ycy, r[2] - ycz};
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                double p = 1.0;
                for (int e = 0; e <= P; ++e) { pw[d][tid][e] = p; p *= h[d]; }
            }
            cf[tid][0] = r[3];
            cf[tid][1] = r[4]; cf[tid][2] = r[5]; cf[tid][3] = r[6];
            // (1/6) Q_ij with the record's halved diagonal: Qxx/6 = rec[7]/3, Qxy/6 (off-diagonal pairs count twice)
            cf[tid][4] = r[7] / 3.0; cf[tid][5] = r[10] / 3.0; cf[tid][6] = r[12] / 3.0;
            cf[tid][7] = r[8] / 3.0; cf[tid][8] = r[9] / 3.0; cf[tid][9] = r[11] / 3.0;
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            if (tid + r * RP_THREADS < Nk) {
                const int ax = ea[r], bx = eb[r], cc = ec[r];
                const double fa = ax, fb = bx, fc = cc;
                const double faa = ax * (ax - 1), fbb = bx * (bx - 1), fcc = cc * (cc - 1);
                for (int p = 0; p < np; ++p) {
                    const double X = pw[0][p][ax], Y = pw[1][p][bx], Z = pw[2][p][cc];
                    const double X1 = ax > 0 ? fa * pw[0][p][ax - 1] : 0.0, Y1 = bx > 0 ? fb * pw[1][p][bx - 1] : 0.0,
                                 Z1 = cc > 0 ? fc * pw[2][p][cc - 1] : 0.0;
                    const double X2 = ax > 1 ? faa * pw[0][p][ax - 2] : 0.0, Y2 = bx > 1 ? fbb * pw[1][p][bx - 2] : 0.0,
                                 Z2 = cc > 1 ? fcc * pw[2][p][cc - 2] : 0.0;
                    const double* q = cf[p];
                    double v = q[0] * X * Y * Z;                                           // charge
                    v += q[1] * X1 * Y * Z + q[2] * X * Y1 * Z + q[3] * X * Y * Z1;       // dipole
                    v += q[4] * X2 * Y * Z + q[5] * X * Y2 * Z + q[6] * X * Y * Z2;       // quadrupole, diagonal
                    v += q[7] * X1 * Y1 * Z + q[8] * X1 * Y * Z1 + q[9] * X * Y1 * Z1;    // off-diagonal (xy + yx, ...)
                    acc[r] += v;
                }
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 3; ++r)
        if (tid + r * RP_THREADS < Nk) mom[tid + r * RP_THREADS] = acc[r];
    __syncthreads();
    for (int e = tid; e < a.NTp; e += RP_THREADS) {           // M -> F (D: section 6), the matvec's table
        double v = 0;
        if (e < a.NT)
            for (int q = a.cv_off[e]; q < a.cv_off[e + 1]; ++q) v = fma(a.cv_coef[q], mom[a.cv_idx[q]], v);
        a.FF[(int64_t)c * a.NTp + e] = v;
    }
}

// ---- evaluation: one block per target group, far part (cells) then near part (sites) ------------------------------------
template <int P>
__device__ __forceinline__ void rt_terms(const double* __restrict__ ff, double dx0, double dy0, double dz0, double dx1,
                                         double dy1, double dz1, double (&W0)[P + 1], double (&W1)[P + 1])
{
    int e = 0;
    double xa0 = 1.0, xa1 = 1.0;
#pragma unroll
    for (int a = 0; a <= P; ++a) {
        double xy0 = xa0, xy1 = xa1;
#pragma unroll
        for (int b = 0; b <= P - a; ++b) {
            double m0 = xy0, m1 = xy1;
#pragma unroll
            for (int c = 0; c <= P - a - b; ++c) {
                const int n = a + b + c;
#pragma unroll
                for (int j = 0; j <= (P - n) / 2; ++j) {
                    const double f = ff[e];
                    ++e;
                    W0[n + j] = fma(m0, f, W0[n + j]);
                    W1[n + j] = fma(m1, f, W1[n + j]);
                }
                if (n < P) { m0 *= dz0; m1 *= dz1; }
            }
            if (a + b < P) { xy0 *= dy0; xy1 *= dy1; }
        }
        if (a < P) { xa0 *= dx0; xa1 *= dx1; }
    }
}

template <int P>
__device__ __forceinline__ double rt_radial(double dx, double dy, double dz, const double (&W)[P + 1])
{
    const double R2 = dx * dx + dy * dy + dz * dz;
    const double ri = pb_rsqrt(R2), ri2 = ri * ri;
    double uL = ri, s = uL * W[0];
#pragma unroll
    for (int m = 1; m <= P; ++m) {
        uL = (2 * m - 1) * uL * ri2;                      // u_m of the Laplace kernel (D: section 6)
        s = fma(uL, W[m], s);
    }
    return s;
}

__device__ __forceinline__ double rt_pair(double dx, double dy, double dz, const double* __restrict__ s, int k)
{
    // the arithmetic of k_rhs (pb_sites.cu): q/R + p.d/R^3 + (d.Q.d/2)/R^5
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double ri = pb_rsqrt(r2), ri2 = ri * ri, ri3 = ri * ri2, ri5 = ri3 * ri2;
    const double pd = s[4 * RT_TILE + k] * dx + s[5 * RT_TILE + k] * dy + s[6 * RT_TILE + k] * dz;
    const double hQ = dx * (s[7 * RT_TILE + k] * dx + s[8 * RT_TILE + k] * dy + s[9 * RT_TILE + k] * dz) +
                      dy * (s[10 * RT_TILE + k] * dy + s[11 * RT_TILE + k] * dz) + s[12 * RT_TILE + k] * dz * dz;
    return s[3 * RT_TILE + k] * ri + pd * ri3 + hQ * ri5;
}

struct rt_args {
    int64_t N;
    int NTp;
    const int32_t *m2p_off, *m2p_cell, *p2p_off, *p2p_lo, *p2p_hi, *perm;
    const double *cx, *cy, *cz, *FF, *rec, *px, *py, *pz;
    double scale;                 // 1 / (4 pi eps_1)
    double* b;
};

template <int P> struct rt_cfg {
    static constexpr int NT = rt_nt(P), NTp = NT + (NT & 1);
    static constexpr size_t FF_BYTES0 = (size_t)RT_W * RT_NS * NTp * sizeof(double);
    static constexpr size_t TILE_BYTES = (size_t)13 * RT_TILE * sizeof(double);
    static constexpr size_t RED_BYTES = (size_t)RT_W * PB_TG * sizeof(double);
    static constexpr size_t A = FF_BYTES0 > TILE_BYTES ? FF_BYTES0 : TILE_BYTES;
    static constexpr size_t FF_BYTES = A > RED_BYTES ? A : RED_BYTES;
    static constexpr size_t SMEM = FF_BYTES + RT_W * RT_NS * sizeof(uint64_t);
};

template <int P>
__global__ void __launch_bounds__(RT_THREADS, 2) k_rhs_eval(rt_args a)
{
    constexpr int NTp = rt_cfg<P>::NTp, NS = RT_NS;
    extern __shared__ __align__(128) unsigned char smraw[];
    const int tid = threadIdx.x, lane = tid & 31, sub = tid >> 5;
    double* ffw = reinterpret_cast<double*>(smraw) + (size_t)sub * NS * NTp;
    uint64_t* fullw = reinterpret_cast<uint64_t*>(smraw + rt_cfg<P>::FF_BYTES) + sub * NS;
    const int64_t g = blockIdx.x;
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) pb_mbar_init(&fullw[s], 1);
        pb_mbar_fence_init();
    }
    __syncthreads();
    const int64_t i0 = g * PB_TG + lane, i1 = i0 + 32;
    const int64_t ic0 = i0 < a.N ? i0 : a.N - 1, ic1 = i1 < a.N ? i1 : a.N - 1;
    const double tx0 = a.px[ic0], ty0 = a.py[ic0], tz0 = a.pz[ic0];
    const double tx1 = a.px[ic1], ty1 = a.py[ic1], tz1 = a.pz[ic1];
    double sum0 = 0.0, sum1 = 0.0;
    {   // ---- far part: this warp's cells are list entries e0 + 8 k; its own ring of TMA-filled slots (as in k_m2p2)
        const int32_t e0 = a.m2p_off[g] + sub, count = a.m2p_off[g + 1] - a.m2p_off[g];
        const int nw = count > sub ? (count - sub + RT_W - 1) / RT_W : 0;
        auto issue = [&](int k, int32_t cell) {
            const int slot = k % NS;
            pb_mbar_expect_tx(&fullw[slot], (uint32_t)(NTp * sizeof(double)));
            pb_bulk_g2s(ffw + (size_t)slot * NTp, a.FF + (int64_t)cell * NTp, (uint32_t)(NTp * sizeof(double)), &fullw[slot]);
        };
        if (lane == 0)
            for (int k = 0; k < NS - 1 && k < nw; ++k) issue(k, a.m2p_cell[e0 + RT_W * k]);
        int32_t idn = NS - 1 < nw ? a.m2p_cell[e0 + RT_W * (NS - 1)] : 0;
        int32_t cn = nw > 0 ? a.m2p_cell[e0] : 0;
        double cxn = a.cx[cn], cyn = a.cy[cn], czn = a.cz[cn];
#pragma unroll 1
        for (int k = 0; k < nw; ++k) {
            const int kn = k + NS - 1;
            if (lane == 0 && kn < nw) issue(kn, idn);
            idn = kn + 1 < nw ? a.m2p_cell[e0 + RT_W * (kn + 1)] : 0;
            const double ccx = cxn, ccy = cyn, ccz = czn;
            if (k + 1 < nw) {
                cn = a.m2p_cell[e0 + RT_W * (k + 1)];
                cxn = a.cx[cn]; cyn = a.cy[cn]; czn = a.cz[cn];
            }
            pb_mbar_wait(&fullw[k % NS], (uint32_t)((k / NS) & 1));
            const double dx0 = tx0 - ccx, dy0 = ty0 - ccy, dz0 = tz0 - ccz;
            const double dx1 = tx1 - ccx, dy1 = ty1 - ccy, dz1 = tz1 - ccz;
            double W0[P + 1], W1[P + 1];
#pragma unroll
            for (int m = 0; m <= P; ++m) { W0[m] = 0.0; W1[m] = 0.0; }
            rt_terms<P>(ffw + (size_t)(k % NS) * NTp, dx0, dy0, dz0, dx1, dy1, dz1, W0, W1);
            sum0 += rt_radial<P>(dx0, dy0, dz0, W0);
            sum1 += rt_radial<P>(dx1, dy1, dz1, W1);
            __syncwarp();
        }
    }
    __syncthreads();                                   // the slots are free: the near part reuses them as its site tile
    {   // ---- near part: the group's site ranges, RT_TILE sites per tile, the warps take sites sub, sub + 8, ...
        double* s = reinterpret_cast<double*>(smraw);  // [13][RT_TILE]
        for (int32_t r = a.p2p_off[g]; r < a.p2p_off[g + 1]; ++r) {
            const int32_t lo = a.p2p_lo[r], hi = a.p2p_hi[r];
            for (int32_t base = lo; base < hi; base += RT_TILE) {
                const int cnt = hi - base < RT_TILE ? hi - base : RT_TILE;
                __syncthreads();
                for (int q = tid; q < 13 * cnt; q += RT_THREADS) {
                    const int k = q / 13, f = q - 13 * k;
                    s[f * RT_TILE + k] = a.rec[RT_REC * (int64_t)(base + k) + f];
                }
                __syncthreads();
                for (int k = sub; k < cnt; k += RT_W) {
                    const double sx = s[k], sy = s[RT_TILE + k], sz = s[2 * RT_TILE + k];
                    sum0 += rt_pair(tx0 - sx, ty0 - sy, tz0 - sz, s, k);
                    sum1 += rt_pair(tx1 - sx, ty1 - sy, tz1 - sz, s, k);
                }
            }
        }
    }
    __syncthreads();
    double* red = reinterpret_cast<double*>(smraw);    // [RT_W][PB_TG]: the warps' sums, added in warp order
    red[sub * PB_TG + lane] = sum0;
    red[sub * PB_TG + lane + 32] = sum1;
    __syncthreads();
    if (tid < PB_TG) {
        const int64_t i = g * PB_TG + tid;
        if (i < a.N) {
            double v = 0;
#pragma unroll
            for (int q = 0; q < RT_W; ++q) v += red[q * PB_TG + tid];
            const int64_t o = a.perm[i];
            a.b[o] = a.scale * v;
            a.b[a.N + o] = 0.0;                          // second block of Eq. (5)'s right side
        }
    }
}

// ---- host side ---------------------------------------------------------------------------------------------------------------
int pb_rhs_tree_build(pb_ctx* ctx)
{
    pb_tree& t = ctx->tree;
    pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    pb_dfree_cat(ctx, CAT_RHS);
    s.rhs_built = false;
    const int64_t na = s.na;
    uint64_t* keys = nullptr;
    PB_TRY(pb_morton_order(ctx, s.pos, na, CAT_RHS, &s.r_perm, &keys));
    for (int d = 0; d < 3; ++d) PB_TRY(pb_dalloc_t(ctx, &s.r_pos[d], na, CAT_RHS));
    k_rhs_gather_pos<<<pb_blocks(na, 256), 256, 0, st>>>(na, s.r_perm, s.pos, s.r_pos[0], s.r_pos[1], s.r_pos[2]);
    PB_LAUNCH_CHECK();
    s.r_oc = pb_octree();
    PB_TRY(pb_octree_build(ctx, keys, na, 1, RT_NCRIT, s.r_pos[0], s.r_pos[1], s.r_pos[2], CAT_RHS, &s.r_oc));
    s.r_ls = pb_lists();
    PB_TRY(pb_lists_build(ctx, 2, t.N, t.pc[0], t.pc[1], t.pc[2], s.r_oc, 1, na, ctx->prm.theta * PB_RHS_THETA_SCALE, RT_M2P_MIN,
                          CAT_RHS, &s.r_ls));
    // the cells that appear in some list: one block of the moment kernel each
    std::vector<int32_t> lists(s.r_ls.m2p_total > 0 ? s.r_ls.m2p_total : 1);
    if (s.r_ls.m2p_total > 0)
        PB_CUDA(cudaMemcpyAsync(lists.data(), s.r_ls.m2p_cell, sizeof(int32_t) * s.r_ls.m2p_total, cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));
    std::vector<char> used(s.r_oc.n_cells, 0);
    for (int64_t e = 0; e < s.r_ls.m2p_total; ++e) used[lists[e]] = 1;
    std::vector<int32_t> need;
    for (int64_t c = 0; c < s.r_oc.n_cells; ++c)
        if (used[c]) need.push_back((int32_t)c);
    s.r_n_need = (int64_t)need.size();
    PB_TRY(pb_dalloc_t(ctx, &s.r_need, need.size() > 0 ? need.size() : 1, CAT_RHS));
    if (!need.empty())
        PB_CUDA(cudaMemcpyAsync(s.r_need, need.data(), sizeof(int32_t) * need.size(), cudaMemcpyHostToDevice, st));
    s.r_P = t.P;
    s.r_NTp = t.NT + (t.NT & 1);
    PB_TRY(pb_dalloc_t(ctx, &s.r_FF, (size_t)s.r_oc.n_cells * s.r_NTp, CAT_RHS));
    PB_CUDA(cudaStreamSynchronize(st));
    s.rhs_built = true;
    return PB_OK;
}

template <int P>
static cudaError_t launch_rhs_eval(pb_ctx* ctx, const rt_args& a, unsigned G)
{
    cudaError_t e = cudaFuncSetAttribute(k_rhs_eval<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rt_cfg<P>::SMEM);
    if (e != cudaSuccess) return e;
    k_rhs_eval<P><<<G, RT_THREADS, rt_cfg<P>::SMEM, ctx->stream>>>(a);
    return cudaSuccess;
}

int pb_rhs_tree(pb_ctx* ctx, const double* mu, double* b)
{
    pb_tree& t = ctx->tree;
    pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    if (!s.rhs_built || s.r_P != t.P) PB_TRY(pb_rhs_tree_build(ctx));
    const int64_t na = s.na;
    PB_TRY(pb_scratch(ctx, (size_t)na * RT_REC * sizeof(double) + 4096));
    double* rec = ctx->scratch;
    k_rhs_pack<<<pb_blocks(na, 128), 128, 0, st>>>(na, s.r_perm, s.pos, s.q, s.dip, mu, s.quad, rec);
    PB_LAUNCH_CHECK();
    if (s.r_n_need > 0) {
        rp_args pa;
        pa.P = t.P; pa.Nk = t.Nk; pa.NT = t.NT; pa.NTp = s.r_NTp;
        pa.need = s.r_need; pa.c_first = s.r_oc.c_first; pa.c_last = s.r_oc.c_last;
        pa.cx = s.r_oc.c_ctr[0]; pa.cy = s.r_oc.c_ctr[1]; pa.cz = s.r_oc.c_ctr[2]; pa.rec = rec;
        pa.ka = t.kexp; pa.kb = t.kexp + PB_MAX_NK_; pa.kc = t.kexp + 2 * PB_MAX_NK_;
        pa.cv_off = t.cv_off; pa.cv_idx = t.cv_idx; pa.cv_coef = t.cv_coef;
        pa.FF = s.r_FF;
        k_rhs_p2m<<<(unsigned)s.r_n_need, RP_THREADS, (size_t)t.Nk * sizeof(double), st>>>(pa);
        PB_LAUNCH_CHECK();
    }
    rt_args a;
    a.N = t.N; a.NTp = s.r_NTp;
    a.m2p_off = s.r_ls.m2p_off; a.m2p_cell = s.r_ls.m2p_cell; a.p2p_off = s.r_ls.p2p_off; a.p2p_lo = s.r_ls.p2p_lo;
    a.p2p_hi = s.r_ls.p2p_hi; a.perm = t.perm;
    a.cx = s.r_oc.c_ctr[0]; a.cy = s.r_oc.c_ctr[1]; a.cz = s.r_oc.c_ctr[2]; a.FF = s.r_FF; a.rec = rec;
    a.px = t.pc[0]; a.py = t.pc[1]; a.pz = t.pc[2];
    a.scale = PB_INV4PI / ctx->prm.eps_in;
    a.b = b;
    const unsigned G = (unsigned)t.n_groups;
    cudaError_t e = cudaSuccess;
    switch (t.P) {
    case 1: e = launch_rhs_eval<1>(ctx, a, G); break;
    case 2: e = launch_rhs_eval<2>(ctx, a, G); break;
    case 3: e = launch_rhs_eval<3>(ctx, a, G); break;
    case 4: e = launch_rhs_eval<4>(ctx, a, G); break;
    case 5: e = launch_rhs_eval<5>(ctx, a, G); break;
    case 6: e = launch_rhs_eval<6>(ctx, a, G); break;
    case 7: e = launch_rhs_eval<7>(ctx, a, G); break;
    case 8: e = launch_rhs_eval<8>(ctx, a, G); break;
    default: return pb_fail(ctx, PB_ERR_INVALID_ARG, "internal: RHS treecode needs 1 <= order_P <= 8");
    }
    PB_CUDA(e);
    PB_LAUNCH_CHECK();
    return PB_OK;
}
