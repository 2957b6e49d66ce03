// pb_matvec.cu -- the treecode matrix-vector product of Eq. (5):
// source weights, P2M / M2M Cartesian-Taylor moments, M2P far field, P2P near field,
// near/singular table and the final combine (D: sections 5-7).
//
// Far field (D: section 6).  For a cell with centre y_c and a target x, d = x - y_c, the
// order-P Taylor sum  sum_{|k|<=P} a_k(x,y_c) M_k  of P:251 (a_k = (1/k!) D_y^k G) is
// evaluated without forming the a_k.  G is radial, G = f(|d-h|^2), and
//   f(s - 2 d.h + |h|^2) = sum_m f^(m)(s)/m! (-2 d.h + |h|^2)^m ,
// so collecting total degree <= P in h gives EXACTLY the same truncated sum as
//   sum_{p+2j<=P} u_{p+j}(R) T_{p,j},   T_{p,j} = sum_{|alpha|=p} d^alpha F_{alpha,j},
//   F_{alpha,j} = (-1)^j / (2^j alpha!) sum_{|beta|=j} M_{alpha+2beta} / beta! ,
//   u_m = (-2)^m f^(m):  u_0 = G, u_1 = e^{-kR}(1+kR)/R^3, u_{m+1} = ((2m+1) u_m + k^2 u_{m-1})/R^2
// (k = 0 for the Laplace kernel).  The F (130 numbers per layer at P = 6) are kernel
// independent, so one pass over them serves V_L, K_L, V_Y and K_Y.
#include <algorithm>
#include <math.h>
#include "pb_internal.cuh"

// ---- index tables ------------------------------------------------------------------------------
__host__ __device__ static constexpr int pb_nt(int P)
{
    int t = 0;
    for (int a = 0; a <= P; ++a)
        for (int b = 0; b <= P - a; ++b)
            for (int c = 0; c <= P - a - b; ++c) t += (P - a - b - c) / 2 + 1;
    return t;
}

#define PB_MAX_NK 286   // pb_nk(10)
__constant__ unsigned char c_ka[PB_MAX_NK], c_kb[PB_MAX_NK], c_kc[PB_MAX_NK];

static double factorial(int n) { double f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }

// The M -> F conversion table for order P, terms in the order the M2P kernel consumes them
// (nested a, b, c loops, then j): F_{(a,b,c),j} = (-1)^j / (2^j a! b! c!) sum_{|beta|=j} M_{alpha+2beta}/beta!
static void farfield_table(int P, std::vector<int32_t>& expo, std::vector<int32_t>& off, std::vector<int32_t>& idx,
                           std::vector<double>& coef)
{
    off.assign(1, 0);
    for (int a = 0; a <= P; ++a)
        for (int b = 0; b <= P - a; ++b)
            for (int c = 0; c <= P - a - b; ++c) {
                int n = a + b + c;
                for (int j = 0; j <= (P - n) / 2; ++j) {
                    double pref = ((j & 1) ? -1.0 : 1.0) / (ldexp(1.0, j) * factorial(a) * factorial(b) * factorial(c));
                    for (int ba = 0; ba <= j; ++ba)
                        for (int bb = 0; bb <= j - ba; ++bb) {
                            int bc = j - ba - bb;
                            idx.push_back(mom_index(a + 2 * ba, b + 2 * bb, c + 2 * bc));
                            coef.push_back(pref / (factorial(ba) * factorial(bb) * factorial(bc)));
                        }
                    off.push_back((int32_t)idx.size());
                    expo.push_back(a); expo.push_back(b); expo.push_back(c); expo.push_back(j);
                }
            }
}

extern "C" int pb_farfield_table(int P, int32_t* expo, int32_t* off, int32_t* idx, double* coef, int64_t* nnz_out)
{
    if (P < 0 || P > PB_MAX_P) return PB_ERR_INVALID_ARG;
    std::vector<int32_t> e, o, i;
    std::vector<double> c;
    farfield_table(P, e, o, i, c);
    if (nnz_out) *nnz_out = (int64_t)i.size();
    if (expo) memcpy(expo, e.data(), sizeof(int32_t) * e.size());
    if (off) memcpy(off, o.data(), sizeof(int32_t) * o.size());
    if (idx) memcpy(idx, i.data(), sizeof(int32_t) * i.size());
    if (coef) memcpy(coef, c.data(), sizeof(double) * c.size());
    return (int)o.size() - 1;
}

int pb_farfield_setup(pb_ctx* ctx)
{
    pb_tree& t = ctx->tree;
    cudaStream_t st = ctx->stream;
    const int P = ctx->prm.order_P;
    t.P = P;
    t.Nk = pb_nk(P);
    t.NT = pb_nt(P);
    if (ctx->prm.theta <= 0.0) return PB_OK;   // direct mode: no far field
    // exponent tables.  mom_index grades by total degree, so the table of order PB_MAX_P contains the table of every
    // lower order as a prefix: the SAME bytes are uploaded whatever this context's P is, and contexts of different
    // order on one device (a binding triple) cannot disturb one another.  (Constant memory is per device; c_T256
    // below is likewise independent of kappa.)
    unsigned char ka[PB_MAX_NK], kb[PB_MAX_NK], kc[PB_MAX_NK];
    for (int a = 0; a <= PB_MAX_P; ++a)
        for (int b = 0; b <= PB_MAX_P - a; ++b)
            for (int c = 0; c <= PB_MAX_P - a - b; ++c) {
                int k = mom_index(a, b, c);
                ka[k] = (unsigned char)a; kb[k] = (unsigned char)b; kc[k] = (unsigned char)c;
            }
    PB_CUDA(cudaMemcpyToSymbolAsync(c_ka, ka, PB_MAX_NK, 0, cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyToSymbolAsync(c_kb, kb, PB_MAX_NK, 0, cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyToSymbolAsync(c_kc, kc, PB_MAX_NK, 0, cudaMemcpyHostToDevice, st));
    PB_TRY(pb_dalloc_t(ctx, &t.kexp, 3 * PB_MAX_NK_, CAT_TREE));
    PB_CUDA(cudaMemcpyAsync(t.kexp, ka, PB_MAX_NK, cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(t.kexp + PB_MAX_NK_, kb, PB_MAX_NK, cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(t.kexp + 2 * PB_MAX_NK_, kc, PB_MAX_NK, cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaStreamSynchronize(st));   // ka, kb, kc live on this stack frame
    // conversion table M -> F, entries in the order the M2P kernel consumes them
    std::vector<int32_t> off, idx, expo;
    std::vector<double> coef;
    farfield_table(P, expo, off, idx, coef);
    if ((int)off.size() - 1 != t.NT) return pb_fail(ctx, PB_ERR_INVALID_ARG, "internal: far-field term count mismatch");
    PB_TRY(pb_dalloc_t(ctx, &t.cv_off, off.size(), CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.cv_idx, idx.size(), CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.cv_coef, coef.size(), CAT_TREE));
    PB_CUDA(cudaMemcpyAsync(t.cv_off, off.data(), sizeof(int32_t) * off.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(t.cv_idx, idx.data(), sizeof(int32_t) * idx.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(t.cv_coef, coef.data(), sizeof(double) * coef.size(), cudaMemcpyHostToDevice, st));
    // the same coefficients with every term of layer m = |alpha| + j scaled by (2m-1)!!: the matvec's combined layers (m2p_radial)
    std::vector<double> coef_s(coef);
    for (int e = 0; e < t.NT; ++e) {
        const int m = expo[4 * e] + expo[4 * e + 1] + expo[4 * e + 2] + expo[4 * e + 3];
        double f = 1.0;
        for (int q = 1; q <= m; ++q) f *= 2.0 * q - 1.0;
        for (int q = off[e]; q < off[e + 1]; ++q) coef_s[q] *= f;
    }
    PB_TRY(pb_dalloc_t(ctx, &t.cv_scale, coef_s.size(), CAT_TREE));
    PB_CUDA(cudaMemcpyAsync(t.cv_scale, coef_s.data(), sizeof(double) * coef_s.size(), cudaMemcpyHostToDevice, st));
    // M2M table: for every k the triples (l, k - l, C(k,l)), l <= k componentwise; l and k - l as moment indices
    std::vector<int32_t> mo(1, 0), me;
    std::vector<double> mc;
    for (int k = 0; k < t.Nk; ++k) {
        const int a = ka[k], b = kb[k], c = kc[k];
        for (int la = 0; la <= a; ++la)
            for (int lb = 0; lb <= b; ++lb)
                for (int lc = 0; lc <= c; ++lc) {
                    me.push_back(mom_index(la, lb, lc) | (mom_index(a - la, b - lb, c - lc) << 12));
                    mc.push_back(factorial(a) / (factorial(la) * factorial(a - la)) * factorial(b) /
                                 (factorial(lb) * factorial(b - lb)) * factorial(c) / (factorial(lc) * factorial(c - lc)));
                }
        mo.push_back((int32_t)me.size());
    }
    {   // after the Nk + 1 offsets: the terms k ordered by falling row length, so that the rows a warp walks together in
        // the M2M are about equally long (lexicographic order mixes rows of 1 and of 27 entries)
        std::vector<int32_t> order(t.Nk);
        for (int k = 0; k < t.Nk; ++k) order[k] = k;
        std::stable_sort(order.begin(), order.end(), [&](int32_t x, int32_t y) { return mo[x + 1] - mo[x] > mo[y + 1] - mo[y]; });
        mo.insert(mo.end(), order.begin(), order.end());
    }
    PB_TRY(pb_dalloc_t(ctx, &t.mm_off, mo.size(), CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.mm_ent, me.size(), CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.mm_coef, mc.size(), CAT_TREE));
    PB_CUDA(cudaMemcpyAsync(t.mm_off, mo.data(), sizeof(int32_t) * mo.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(t.mm_ent, me.data(), sizeof(int32_t) * me.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(t.mm_coef, mc.data(), sizeof(double) * mc.size(), cudaMemcpyHostToDevice, st));

    // Which cells need moments: the ones in some M2P list ("used") and every descendant of a used
    // cell (M2M builds a parent from ALL its children).  Bookkeeping on the host, once per tree.
    const int64_t nc = t.n_cells;
    // (with target sharding only the cells in the OWNED groups' lists, entries [e0, e1), are needed on this rank)
    int32_t he[2] = {0, 0};
    PB_CUDA(cudaMemcpyAsync(&he[0], t.m2p_off + t.own_g0, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaMemcpyAsync(&he[1], t.m2p_off + t.own_g1, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));
    const int64_t e0 = he[0], ne = he[1] - he[0];
    std::vector<int32_t> child(nc), nchild(nc), lists(ne > 0 ? ne : 1);
    PB_CUDA(cudaMemcpyAsync(child.data(), t.c_child, sizeof(int32_t) * nc, cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaMemcpyAsync(nchild.data(), t.c_nchild, sizeof(int32_t) * nc, cudaMemcpyDeviceToHost, st));
    if (ne > 0)
        PB_CUDA(cudaMemcpyAsync(lists.data(), t.m2p_cell + e0, sizeof(int32_t) * ne, cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));   // also: the host vectors above go out of scope
    std::vector<char> used(nc, 0), need(nc, 0);
    for (int64_t e = 0; e < ne; ++e) used[lists[e]] = 1;
    std::vector<int32_t> leaf_list, parent(nc, -1), up(nc, 0);
    int64_t n_used = 0, n_internal = 0;
    for (int64_t c = 0; c < nc; ++c) {               // cells are numbered generation by generation: parents first
        need[c] = need[c] || used[c];
        if (used[c]) ++n_used;
        if (!need[c]) continue;
        if (child[c] < 0) leaf_list.push_back((int32_t)c);
        else {
            ++n_internal;
            for (int q = 0; q < nchild[c]; ++q) { need[child[c] + q] = 1; parent[child[c] + q] = (int32_t)c; }
        }
    }
    // up[c]: bit 0 = the cell's F terms are wanted (it is in an M2P list); bit 1 = its moments are stored in
    // M (a parent will read them); bits 2.. = 1 + parent when the parent's moments are needed (the block
    // finishing c then reports to it), else 0
    for (int64_t c = 0; c < nc; ++c) {
        const int32_t par = need[c] && parent[c] >= 0 ? parent[c] + 1 : 0;
        up[c] = (used[c] ? 1 : 0) | (par ? 2 : 0) | (par << 2);
    }
    t.n_used = n_used;
    t.n_need_leaf = (int64_t)leaf_list.size();
    t.n_need_internal = n_internal;
    PB_TRY(pb_dalloc_t(ctx, &t.need_leaf, leaf_list.size(), CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.up_link, (size_t)nc, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.up_count, (size_t)nc, CAT_TREE));
    if (!leaf_list.empty())
        PB_CUDA(cudaMemcpyAsync(t.need_leaf, leaf_list.data(), sizeof(int32_t) * leaf_list.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(t.up_link, up.data(), sizeof(int32_t) * nc, cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemsetAsync(t.up_count, 0, sizeof(int32_t) * nc, st));
    PB_CUDA(cudaStreamSynchronize(st));
    PB_TRY(pb_dalloc_t(ctx, &t.M, (size_t)t.n_cells * 2 * t.Nk, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.FF, (size_t)t.n_cells * t.NT, CAT_TREE));
    return PB_OK;
}

// ---- source weights (H5): q^V_g = w_g A_j dphi_j ,  q^K_g = w_g A_j phi_j n_j ------------------------
// Writes the 64-byte source records the P2P / P2M / reaction kernels stream (coordinates repeated
// so that one contiguous TMA bulk copy brings a whole tile of sources into shared memory).
// With `pc` (the right block-Jacobi preconditioner of GMRES, D: R-20) the operator is applied to
// z = Minv x, z formed on the fly: per panel the inverse 2x2 diagonal block, original panel order.
__global__ void k_weights(int64_t N, int K, const int32_t* __restrict__ perm, const double* __restrict__ x,
                          const double* __restrict__ pc, const double* __restrict__ swA,
                          const double* __restrict__ sx, const double* __restrict__ sy, const double* __restrict__ sz,
                          const double* __restrict__ nx, const double* __restrict__ ny,
                          const double* __restrict__ nz, double* __restrict__ xphi, double* __restrict__ xdphi,
                          double4* __restrict__ srec, const unsigned char* __restrict__ psurf, int keep,
                          double* __restrict__ xphi_full)
{
    // psurf != NULL (two surfaces, pb_set_stern): only the sources of surface `keep` carry weight in this pass;
    // xphi_full (first pass) receives phi of every panel for the phi_i/2 terms
    int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= N * K) return;
    int64_t i = s / K;
    int64_t o = perm[i];
    double phi = x[o], dphi = x[N + o], w = swA[s];
    if (pc) {
        const double a = phi, b = dphi;
        phi = pc[o] * a + pc[N + o] * b;
        dphi = pc[2 * N + o] * a + pc[3 * N + o] * b;
    }
    if (psurf) {
        if (xphi_full && s == i * K) xphi_full[i] = phi;
        if (psurf[i] != keep) { phi = 0.0; dphi = 0.0; }
    }
    if (s == i * K) { xphi[i] = phi; xdphi[i] = dphi; }
    double wp = w * phi;
    srec[2 * s] = make_double4(sx[s], sy[s], sz[s], w * dphi);
    srec[2 * s + 1] = make_double4(wp * nx[i], wp * ny[i], wp * nz[i], 0.0);
}

int pb_weights(pb_ctx* ctx, const double* x, bool precond, int surface)
{
    pb_tree& t = ctx->tree;
    const bool mask = surface >= 0 && t.psurf != nullptr;
    k_weights<<<pb_blocks(t.Ns, 256), 256, 0, ctx->stream>>>(t.N, t.K, t.perm, x, precond ? t.precond : nullptr, t.swA, t.sx[0],
                                                            t.sx[1], t.sx[2], t.pn[0], t.pn[1], t.pn[2], t.xphi, t.xdphi,
                                                            t.srec, mask ? t.psurf : nullptr, surface,
                                                            mask && surface == 0 ? t.xphi_full : nullptr);
    PB_LAUNCH_CHECK();
    return PB_OK;
}

// constants of pb_exp_mkr8 (pb_device.cuh); the table 2^(-j/256) does not depend on kappa and is uploaded once
__constant__ double c_T256[256];

int pb_make_expk8(pb_ctx* ctx, double kappa, pb_expk8* k)
{
    const double ln2 = 0.693147180559945309417232121458;
    k->c1 = 256.0 * kappa / ln2;
    k->Lk = kappa > 0.0 ? ln2 / (256.0 * kappa) : 0.0;
    double f = 1.0;
    for (int m = 0; m <= 4; ++m) {
        k->c[m] = f;
        f *= -kappa / (double)(m + 1);
    }
    double T[256];                                  // constant memory is per device: upload at every tree build
    for (int j = 0; j < 256; ++j) T[j] = exp2(-(double)j / 256.0);
    PB_CUDA(cudaMemcpyToSymbolAsync(c_T256, T, sizeof(T), 0, cudaMemcpyHostToDevice, ctx->stream));
    PB_CUDA(cudaStreamSynchronize(ctx->stream));
    return PB_OK;
}

// constants of pb_exp_mkr (pb_device.cuh)
void pb_make_expk(double kappa, pb_expk* k)
{
    const double ln2 = 0.693147180559945309417232121458;
    k->c1 = 32.0 * kappa / ln2;
    k->Lk = kappa > 0.0 ? ln2 / (32.0 * kappa) : 0.0;
    double f = 1.0;
    for (int m = 0; m <= 6; ++m) {
        k->c[m] = f;
        f *= -kappa / (double)(m + 1);
    }
    for (int j = 0; j < 32; ++j) k->T[j] = exp2(-(double)j / 32.0);
    k->g[0] = 0.0;
    for (int m = 1; m < 12; ++m) k->g[m] = kappa * kappa / ((2.0 * m + 1.0) * (2.0 * m - 1.0));
}

// ---- upward pass in ONE launch (H5): P2M at the leaves, M2M up the tree, M -> F conversion ---------------
// P2M: M^V_k = sum_g q^V_g h^k,  M^K_k = sum_g sum_d q^K_{g,d} k_d h^{k-e_d}.  Four plain moment
// sets per cell are accumulated, S^V, S^x, S^y, S^z (weights q^V, q^K_x, q^K_y, q^K_z), one monomial
// serving all four; then M^K_(a,b,c) = a S^x_(a-1,b,c) + b S^y_(a,b-1,c) + c S^z_(a,b,c-1).
// M2M: M'_k = sum_{l<=k} C(k,l) t^{k-l} M_l, table driven (mm_*: for every k the (l, k-l, C(k,l)) triples).
// One block per leaf whose moments are needed.  When a block has finished a cell it reports to the
// parent (if the parent's moments are needed); the block that reports LAST carries on with the
// parent's M2M, and so on upward -- nobody waits, and a parent is always formed from all its children
// in child order, so the result does not depend on the arrival order.  A cell that appears in an M2P
// list has its far-field terms F (D: section 6) written by the block that finishes it.
// Points staged per P2M chunk (<= UP_THREADS) and children per M2M round: small where the grid is many waves deep and the
// number of resident blocks counts (a leaf holds 40 points on average at C4), large where the whole grid is resident at once
// and the length of a block's own chain counts (C1, C2: 0.083 ms against 0.095 ms with the small values)
#define P2M_CH_SMALL 48
#define P2M_CH_LARGE 96
#define M2M_Q_SMALL 4
#define M2M_Q_LARGE 8
#define P2M_LD (PB_MAX_P + 1)     // 11 doubles per point: odd stride, so a warp's reads of one point do not conflict
#define UP_THREADS 128

struct up_args {
    int P, Nk, NT, K;
    int CH, MQ;      // P2M chunk, M2M round (see above)
    int comb;        // F terms as the combined layers {F^K - F^V, F^K - eps F^V} (m2p_radial) instead of {F^V, F^K}
    double eps_ratio;
    const int32_t *leaf_ids, *c_first, *c_last, *c_child, *c_nchild, *up_link;
    int32_t* up_count;
    const double *cx, *cy, *cz;
    const double4* srec;
    const int32_t *mm_off, *mm_ent;
    const double* mm_coef;
    const int32_t *cv_off, *cv_idx;
    const double* cv_coef;
    double* M;
    double2* FF;
};

static size_t up_smem_bytes(int Nk, int CH, int MQ)
{
    const size_t p2m = 3 * (size_t)CH * P2M_LD + 3 * (size_t)Nk;
    const size_t m2m = 5 * (size_t)MQ * (size_t)Nk + (size_t)MQ * 3 * P2M_LD;
    return CH * sizeof(double4) + (2 * (size_t)Nk + (p2m > m2m ? p2m : m2m)) * sizeof(double);
}

// NR = moments per thread (ceil(N_k / 128): 1 up to P = 6, 2 up to P = 8, 3 for P = 9, 10).  The pass is bound by latency
// and per-block overhead (one block per leaf), so what counts is the number of resident blocks: with NR = 1 the block
// needs 64 registers per thread and 17.5 KB of shared memory (8 blocks per SM instead of 6 with the general form): C4
// 2.94 -> 2.54 ms at P = 6, 8.09 -> 6.09 ms at P = 8.  (10 blocks at 48 registers: 2.48 ms at C4, slower at C3 -- the shared-memory
// pipe is the next limit, ncu: l1tex 70 % busy.)
template <int NR>
__global__ void __launch_bounds__(UP_THREADS, NR == 1 ? 8 : (NR == 2 ? 6 : 4)) k_upward(up_args a)
{
    extern __shared__ __align__(128) unsigned char up_raw[];
    const int Nk = a.Nk, P = a.P, tid = threadIdx.x, CH = a.CH, MQ = a.MQ;
    double4* wq = reinterpret_cast<double4*>(up_raw);          // [CH]
    double* mom = reinterpret_cast<double*>(wq + CH);      // [2][Nk] finished moments of the current cell
    double* U = mom + 2 * Nk;
    double* pw = U;                                            // P2M: [3][CH][P2M_LD] powers of h
    double* sk = pw + 3 * CH * P2M_LD;                     // P2M: [3][Nk] the S^x, S^y, S^z sets
    double* cm = U;                                            // M2M: [MQ][2][Nk] children of one round
    double* part = cm + 2 * MQ * Nk;                        // M2M: [MQ][2][Nk] shifted children
    double* tm = part + 2 * MQ * Nk;                        // M2M: [MQ][Nk] monomials of the shifts
    double* tp = tm + MQ * Nk;                              // M2M: [MQ][3][P2M_LD] powers of the shifts
    __shared__ int s_last;

    int64_t c = a.leaf_ids[blockIdx.x];
    int32_t link = a.up_link[c];                               // in flight during the P2M (one L2 round trip off the chain)
    {   // ---- P2M: thread k (and k + 128, k + 256 at high order) sweeps the leaf's points
        const int64_t s0 = (int64_t)a.c_first[c] * a.K, s1 = (int64_t)a.c_last[c] * a.K;
        const double ycx = a.cx[c], ycy = a.cy[c], ycz = a.cz[c];
        int ea[NR], eb[NR], ec[NR];
#pragma unroll
        for (int r = 0; r < NR; ++r) {
            const int k = tid + r * UP_THREADS;
            ea[r] = k < Nk ? c_ka[k] : 0; eb[r] = k < Nk ? c_kb[k] : 0; ec[r] = k < Nk ? c_kc[k] : 0;
        }
        double acc[NR][4];
#pragma unroll
        for (int r = 0; r < NR; ++r)
#pragma unroll
            for (int m = 0; m < 4; ++m) acc[r][m] = 0.0;
        // thread p stages point p of a chunk (powers of its three coordinates, its four weights); the records of the
        // next chunk are already in flight while this one is accumulated
        double4 ra = make_double4(0, 0, 0, 0), rb = ra;
        if (tid < CH && s0 + tid < s1) { ra = a.srec[2 * (s0 + tid)]; rb = a.srec[2 * (s0 + tid) + 1]; }
        for (int64_t base = s0; base < s1; base += CH) {
            const int np = (int)((s1 - base) < CH ? (s1 - base) : CH);
            __syncthreads();
            if (tid < np) {
                const double hh[3] = {ra.x - ycx, ra.y - ycy, ra.z - ycz};
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    double pwr = 1.0;
                    double* dst = pw + ((size_t)d * CH + tid) * P2M_LD;
                    for (int e = 0; e <= P; ++e) { dst[e] = pwr; pwr *= hh[d]; }
                }
                wq[tid] = make_double4(ra.w, rb.x, rb.y, rb.z);
            }
            if (tid < CH && base + CH + tid < s1) {
                ra = a.srec[2 * (base + CH + tid)];
                rb = a.srec[2 * (base + CH + tid) + 1];
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r < NR; ++r) {
                if (tid + r * UP_THREADS < Nk) {
                    const double* px = pw + ea[r];
                    const double* py = pw + (size_t)CH * P2M_LD + eb[r];
                    const double* pz = pw + (size_t)2 * CH * P2M_LD + ec[r];
#pragma unroll 4
                    for (int p = 0; p < np; ++p) {
                        const double mono = px[p * P2M_LD] * py[p * P2M_LD] * pz[p * P2M_LD];
                        const double4 w = wq[p];
                        acc[r][0] = fma(w.x, mono, acc[r][0]);
                        acc[r][1] = fma(w.y, mono, acc[r][1]);
                        acc[r][2] = fma(w.z, mono, acc[r][2]);
                        acc[r][3] = fma(w.w, mono, acc[r][3]);
                    }
                }
            }
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < NR; ++r) {
            const int k = tid + r * UP_THREADS;
            if (k < Nk) { mom[k] = acc[r][0]; sk[k] = acc[r][1]; sk[Nk + k] = acc[r][2]; sk[2 * Nk + k] = acc[r][3]; }
        }
        __syncthreads();
        for (int k = tid; k < Nk; k += UP_THREADS) {
            const int ax = c_ka[k], bx = c_kb[k], cc = c_kc[k];
            double v = 0.0;
            if (ax) v = fma((double)ax, sk[mom_index(ax - 1, bx, cc)], v);
            if (bx) v = fma((double)bx, sk[Nk + mom_index(ax, bx - 1, cc)], v);
            if (cc) v = fma((double)cc, sk[2 * Nk + mom_index(ax, bx, cc - 1)], v);
            mom[Nk + k] = v;
        }
        __syncthreads();
    }
    for (;;) {
        // mom holds the finished moments of cell c
        const int64_t parent = (int64_t)(link >> 2) - 1;
        if (link & 2)
            for (int k = tid; k < 2 * Nk; k += UP_THREADS) a.M[c * 2 * Nk + k] = mom[k];
        if (link & 1) {                                        // M -> F (cells in an M2P list)
            const double* mv = mom;
            const double* mk = mom + Nk;
            for (int e = tid; e < a.NT; e += UP_THREADS) {
                double v = 0, k = 0;
                const int q1 = __ldg(a.cv_off + e + 1);
#pragma unroll 4
                for (int q = __ldg(a.cv_off + e); q < q1; ++q) {
                    const int l = __ldg(a.cv_idx + q);
                    const double f = __ldg(a.cv_coef + q);
                    v = fma(f, mv[l], v);
                    k = fma(f, mk[l], k);
                }
                a.FF[c * a.NT + e] = a.comb ? make_double2(k - v, fma(-a.eps_ratio, v, k)) : make_double2(v, k);
            }
        }
        if (parent < 0) break;
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            const int nchild = a.c_nchild[parent];
            const int old = atomicAdd(&a.up_count[parent], 1);
            s_last = old == nchild - 1;
            if (s_last) a.up_count[parent] = 0;                // ready for the next matvec
        }
        __syncthreads();
        if (!s_last) break;
        __threadfence();
        // ---- M2M: this block reported last, it forms the parent from all the children
        c = parent;
        const int32_t ch = a.c_child[c];
        const int nc = a.c_nchild[c];
        link = a.up_link[c];                                   // the parent's own link word, in flight during its M2M
        // the children MQ at a time (they are consecutive); the parent is the sum over ALL of them in child order
        for (int q0 = 0; q0 < nc; q0 += MQ) {
            const int nq = nc - q0 < MQ ? nc - q0 : MQ;
            for (int k = tid; k < nq * 2 * Nk; k += UP_THREADS) cm[k] = __ldcg(a.M + (int64_t)(ch + q0) * 2 * Nk + k);
            if (tid < 3 * nq) {
                const int q = tid / 3, d = tid - 3 * q;
                const double* ctr = d == 0 ? a.cx : (d == 1 ? a.cy : a.cz);
                const double tt = ctr[ch + q0 + q] - ctr[c];
                double pwr = 1.0;
                for (int e = 0; e <= P; ++e) { tp[(q * 3 + d) * P2M_LD + e] = pwr; pwr *= tt; }
            }
            __syncthreads();
            for (int it = tid; it < Nk * nq; it += UP_THREADS) {   // monomials t^k of every child's shift
                const int q = it / Nk, k = it - q * Nk;
                const double* t3 = tp + q * 3 * P2M_LD;
                tm[it] = t3[c_ka[k]] * t3[P2M_LD + c_kb[k]] * t3[2 * P2M_LD + c_kc[k]];
            }
            __syncthreads();
            for (int it = tid; it < Nk * nq; it += UP_THREADS) {
                const int q = it / Nk, k = __ldg(a.mm_off + Nk + 1 + (it - q * Nk));   // rows by falling length
                const double* tq = tm + q * Nk;
                const double* cq = cm + q * 2 * Nk;
                double s0 = 0, s1 = 0;
                const int e1 = __ldg(a.mm_off + k + 1);
#pragma unroll 4
                for (int e = __ldg(a.mm_off + k); e < e1; ++e) {
                    const int32_t ent = __ldg(a.mm_ent + e);
                    const double f = __ldg(a.mm_coef + e) * tq[ent >> 12];
                    const int l = ent & 0xfff;
                    s0 = fma(f, cq[l], s0);
                    s1 = fma(f, cq[Nk + l], s1);
                }
                part[q * 2 * Nk + k] = s0;
                part[q * 2 * Nk + Nk + k] = s1;
            }
            __syncthreads();
            for (int k = tid; k < 2 * Nk; k += UP_THREADS) {
                double v = q0 ? mom[k] : 0.0;
                for (int q = 0; q < nq; ++q) v += part[q * 2 * Nk + k];
                mom[k] = v;
            }
            __syncthreads();
        }
    }
}

// ---- M2P (H6; "box-target" interactions) -----------------------------------------------------------
// PL <= P: only the terms of the order-PL sum (|alpha| + 2j <= PL), see m2p_terms2
template <int P, int PL = P>
__device__ __forceinline__ void m2p_terms(const double2* __restrict__ ff, double dx, double dy, double dz,
                                          double (&WV)[P + 1], double (&WK)[P + 1])
{
    int e = 0;
    double xa = 1.0;
#pragma unroll
    for (int a = 0; a <= P; ++a) {
        double xy = xa;
#pragma unroll
        for (int b = 0; b <= P - a; ++b) {
            double mono = xy;
#pragma unroll
            for (int c = 0; c <= P - a - b; ++c) {
                const int n = a + b + c;
#pragma unroll
                for (int j = 0; j <= (P - n) / 2; ++j) {
                    if (n + 2 * j <= PL) {
                        const double2 f = ff[e];
                        WV[n + j] = fma(mono, f.x, WV[n + j]);
                        WK[n + j] = fma(mono, f.y, WK[n + j]);
                    }
                    ++e;
                }
                if (n < PL) mono *= dz;
            }
            if (a + b < PL) xy *= dy;
        }
        if (a < PL) xa *= dx;
    }
}

// One block = one work item: a target group (PB_TG targets) x a run of its accepted cells.  The
// cells' F terms (N_T x {V,K}, contiguous per cell) and centres arrive in shared memory by TMA bulk
// copies, CT cells per stage, M2P_NS stages: a "full" mbarrier per stage (TMA completion) and an
// "empty" one (one arrival per warp) so that no warp ever waits for another warp, only for data.  The
// block's M2P_S sub-slices (2 warps each) take different cells of a stage for the same targets, so
// all shared-memory reads are warp-wide broadcasts.
#define M2P_S 4
#define M2P_NS 3
#define M2P_THREADS (PB_TG * M2P_S)
static_assert(M2P_S == 4, "the final reduction maps one of the 4 outputs to each sub-slice");

template <int P> struct m2p_cfg {
    static constexpr int NT = pb_nt(P);
    static constexpr int CT = P <= 6 ? 8 : 4;                    // cells per stage
    static constexpr size_t RED_BYTES = (size_t)M2P_S * 4 * PB_TG * sizeof(double);   // final reduction reuses the stages
    static constexpr size_t FF_BYTES0 = (size_t)M2P_NS * CT * NT * sizeof(double2);
    static constexpr size_t FF_BYTES = FF_BYTES0 > RED_BYTES ? FF_BYTES0 : RED_BYTES;
    static constexpr size_t SMEM = FF_BYTES + M2P_NS * CT * sizeof(double4) + 2 * M2P_NS * sizeof(uint64_t) + 32 * sizeof(double);
};

template <int P>
__global__ void __launch_bounds__(M2P_THREADS, 3)
k_m2p(int64_t N, double kappa, pb_expk ek, const pb_item* __restrict__ items, const int32_t* __restrict__ m2p_cell,
      const double4* __restrict__ m2p_ctr, const double2* __restrict__ FF, const double* __restrict__ px,
      const double* __restrict__ py, const double* __restrict__ pz, double* __restrict__ acc)
{
    constexpr int NT = m2p_cfg<P>::NT, CT = m2p_cfg<P>::CT, NS = M2P_NS;
    extern __shared__ __align__(128) unsigned char smraw[];
    double2* ff = reinterpret_cast<double2*>(smraw);                                  // [NS][CT][NT]
    double4* ctr = reinterpret_cast<double4*>(smraw + m2p_cfg<P>::FF_BYTES);           // [NS][CT]
    uint64_t* full = reinterpret_cast<uint64_t*>(ctr + NS * CT);                       // [NS]
    uint64_t* empty = full + NS;                                                       // [NS]
    double* Ts = reinterpret_cast<double*>(empty + NS);                                // [32]
    const int tid = threadIdx.x;
    const int tgt = tid & (PB_TG - 1), sub = tid / PB_TG;
    const pb_item item = items[blockIdx.x];
    const int64_t g = item.group;
    const int32_t e0 = item.r, count = item.count;
    if (tid < 32) Ts[tid] = ek.T[tid];
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) {
            pb_mbar_init(&full[s], 1);
            pb_mbar_init(&empty[s], M2P_THREADS / 32);
        }
        pb_mbar_fence_init();
    }
    __syncthreads();
    const int64_t i = g * PB_TG + tgt;
    const int64_t ic = i < N ? i : N - 1;
    const double tx = px[ic], ty = py[ic], tz = pz[ic];
    const int ntile = (count + CT - 1) / CT;

    // thread 0 is the producer: cell ids are fetched one tile ahead of the copies that need them
    int32_t idn[CT];
    auto load_ids = [&](int t) {
#pragma unroll
        for (int j = 0; j < CT; ++j) {
            const int32_t e = t * CT + j;
            idn[j] = e < count ? m2p_cell[e0 + e] : 0;
        }
    };
    auto issue = [&](int t, int stage) {
        const int n = count - t * CT < CT ? count - t * CT : CT;
        pb_mbar_expect_tx(&full[stage], (uint32_t)(n * (sizeof(double4) + NT * sizeof(double2))));
        pb_bulk_g2s(ctr + stage * CT, m2p_ctr + e0 + t * CT, (uint32_t)(n * sizeof(double4)), &full[stage]);
#pragma unroll
        for (int j = 0; j < CT; ++j)
            if (j < n)
                pb_bulk_g2s(ff + ((size_t)stage * CT + j) * NT, FF + (int64_t)idn[j] * NT, (uint32_t)(NT * sizeof(double2)),
                            &full[stage]);
    };
    if (tid == 0 && ntile > 0) {
        load_ids(0);
        for (int t = 0; t < NS - 1 && t < ntile; ++t) {
            issue(t, t);
            if (t + 1 < ntile) load_ids(t + 1);
        }
    }
    double VL = 0, KL = 0, VY = 0, KY = 0;
    const double k2 = kappa * kappa;
    int st = 0, ph = 0;                               // stage and phase of tile t
    for (int t = 0; t < ntile; ++t) {
        if (tid == 0) {
            const int tn = t + NS - 1;                // refill the stage tile t-1 used, once every warp has left it
            if (tn < ntile) {
                const int sn = st == 0 ? NS - 1 : st - 1;
                if (t > 0) pb_mbar_wait(&empty[sn], (uint32_t)(((t - 1) / NS) & 1));
                issue(tn, sn);
                if (tn + 1 < ntile) load_ids(tn + 1);
            }
        }
        pb_mbar_wait(&full[st], (uint32_t)ph);
        const int cnt = count - t * CT < CT ? count - t * CT : CT;
#pragma unroll 1
        for (int j = sub; j < cnt; j += M2P_S) {
            const double4 cc = ctr[st * CT + j];
            if (!(((int)cc.w >> 1) >> ((tid >> 5) & 1) & 1)) continue;   // the entry is for the other half of the group (warp-uniform)
            const double dx = tx - cc.x, dy = ty - cc.y, dz = tz - cc.z;
            double WV[P + 1], WK[P + 1];
#pragma unroll
            for (int m = 0; m <= P; ++m) { WV[m] = 0.0; WK[m] = 0.0; }
            m2p_terms<P>(ff + ((size_t)st * CT + j) * NT, dx, dy, dz, WV, WK);
            const double R2 = dx * dx + dy * dy + dz * dz;
            const double ri = pb_rsqrt(R2), R = R2 * ri, ri2 = ri * ri;
            const double ex = pb_exp_mkr(R, ek, Ts);
            double uL = ri, uY0 = ex * ri, uY1 = ex * fma(kappa, R, 1.0) * ri * ri2;
            VL = fma(uL, WV[0], VL); KL = fma(uL, WK[0], KL);
            VY = fma(uY0, WV[0], VY); KY = fma(uY0, WK[0], KY);
#pragma unroll
            for (int m = 1; m <= P; ++m) {
                uL = (2 * m - 1) * uL * ri2;
                VL = fma(uL, WV[m], VL); KL = fma(uL, WK[m], KL);
                VY = fma(uY1, WV[m], VY); KY = fma(uY1, WK[m], KY);
                const double un = ((2 * m + 1) * uY1 + k2 * uY0) * ri2;
                uY0 = uY1;
                uY1 = un;
            }
        }
        __syncwarp();
        if ((tid & 31) == 0) pb_mbar_arrive(&empty[st]);
        if (++st == NS) { st = 0; ph ^= 1; }
    }
    __syncthreads();
    // add the sub-slices in a fixed order (the stages are free: every thread passed the barrier above)
    double* red = reinterpret_cast<double*>(smraw);   // [M2P_S][4][PB_TG]
    red[(sub * 4 + 0) * PB_TG + tgt] = VL;
    red[(sub * 4 + 1) * PB_TG + tgt] = KL;
    red[(sub * 4 + 2) * PB_TG + tgt] = VY;
    red[(sub * 4 + 3) * PB_TG + tgt] = KY;
    __syncthreads();
    {
        const int m = tid / PB_TG;
        double v = 0;
#pragma unroll
        for (int q = 0; q < M2P_S; ++q) v += red[(q * 4 + m) * PB_TG + tgt];
        if (i < N) acc[((int64_t)item.slot * 4 + m) * N + i] = v;
    }
}

// ---- M2P, two targets per thread (orders P <= 8) -------------------------------------------------------------
// With one target per thread every F term costs one 16-byte shared-memory broadcast per two FMAs, and
// the shared-memory pipe, not the FP64 pipe, sets the pace (ncu: FP64 pipe 65 % busy).  Here a lane
// carries targets lane and lane + 32 of the group, so each term read feeds four FMAs; a warp covers the
// whole group, the block's 8 warps take different cells of the work item (cells sub, sub + 8, ...).
// Every warp has its OWN ring of M2Q_NS cell slots in shared memory, filled by its lane 0 with TMA bulk copies and
// its own mbarriers: no warp ever waits for another warp, only for its own data.  (The first version shared one
// ring of 8-cell tiles between the warps, refilled when all eight had left a tile; ncu at C4 showed 22 % of the warp
// samples in the wait for the next tile although the data rate needed is a few bytes per clock and SM: warp 0,
// which also ran the producer code, could never run ahead of the slowest warp, and every hiccup of one warp stalled
// the other seven at the end of the ring.)
#define M2Q_W 8
#define M2Q_NS 4
#define M2Q_THREADS (32 * M2Q_W)
static_assert(PB_TG == 64, "k_m2p2 keeps two targets per lane");

template <int P> struct m2q_cfg {
    static constexpr int NT = pb_nt(P);
    static constexpr size_t RED_BYTES = (size_t)M2Q_W * 4 * PB_TG * sizeof(double);
    static constexpr size_t FF_BYTES0 = (size_t)M2Q_W * M2Q_NS * NT * sizeof(double2);
    static constexpr size_t FF_BYTES = FF_BYTES0 > RED_BYTES ? FF_BYTES0 : RED_BYTES;
    static constexpr size_t SMEM = FF_BYTES + M2Q_W * M2Q_NS * sizeof(uint64_t) + 32 * sizeof(double);
};

// PL <= P: evaluate only the terms of the order-PL sum (|alpha| + 2j <= PL); they are a subset of the order-P terms
// with the same values F_{alpha,j}, so the same staged array serves both (the skipped entries are never read).
// The four DFMA of a term are written in a "snake" order -- (m0,f.x) (m0,f.y) (m1,f.y) (m1,f.x), the next term starting
// with the target the last one ended with -- so that consecutive instructions share a source register: a DFMA whose
// three sources are all fresh vector registers issues at 2/3 of the pipe's rate on the B200 (operand bandwidth;
// profiles/r02_fp64_pipe_probes.md), one that re-uses an operand of its predecessor at the full rate.  ptxas
// reschedules most of it (C4: 11.43 -> 11.27 ms), the summation order of every partial sum is unchanged.
template <int P, int PL>
__device__ __forceinline__ void m2p_terms2(const double2* __restrict__ ff, double dx0, double dy0, double dz0, double dx1,
                                           double dy1, double dz1, double (&WV0)[P + 1], double (&WK0)[P + 1],
                                           double (&WV1)[P + 1], double (&WK1)[P + 1])
{
    int e = 0;
    bool flip = false;
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
                    if (n + 2 * j <= PL) {
                        const double2 f = ff[e];
                        if (!flip) {
                            WV0[n + j] = fma(m0, f.x, WV0[n + j]);
                            WK0[n + j] = fma(m0, f.y, WK0[n + j]);
                            WK1[n + j] = fma(m1, f.y, WK1[n + j]);
                            WV1[n + j] = fma(m1, f.x, WV1[n + j]);
                        } else {
                            WV1[n + j] = fma(m1, f.x, WV1[n + j]);
                            WK1[n + j] = fma(m1, f.y, WK1[n + j]);
                            WK0[n + j] = fma(m0, f.y, WK0[n + j]);
                            WV0[n + j] = fma(m0, f.x, WV0[n + j]);
                        }
                        flip = !flip;
                    }
                    ++e;
                }
                if (n < PL) { m0 *= dz0; m1 *= dz1; }
            }
            if (a + b < PL) { xy0 *= dy0; xy1 *= dy1; }
        }
        if (a < PL) { xa0 *= dx0; xa1 *= dx1; }
    }
}

// radial part: u_m(R) of both kernels against the (P+1) partial sums per layer (D: section 6).
// COMB: the two layers of the cell's F terms are not {V, K} but the combinations the two rows of Eq. (5) need,
// {F^K - F^V, F^K - (eps_in / eps_out) F^V} (written so by the upward pass): the Laplace radial functions go with the first
// layer only, the Yukawa ones with the second, and the results are KL' = K_L - V_L and KY' = K_Y - eps V_Y with VL = VY = 0
// -- two FMA per layer instead of four, the combine kernel unchanged.  (Not with two surfaces, R-32: there the rows take
// V and K with per-surface factors.)
template <int P, int PL, bool COMB>
__device__ __forceinline__ void m2p_radial(double dx, double dy, double dz, const double (&WV)[P + 1], const double (&WK)[P + 1],
                                           double kappa, double k2, const pb_expk& ek, const double* __restrict__ Ts,
                                           double& VL, double& KL, double& VY, double& KY)
{
    const double R2 = dx * dx + dy * dy + dz * dz;
    const double ri = pb_rsqrt(R2), R = R2 * ri, ri2 = ri * ri;
    const double ex = pb_exp_mkr(R, ek, Ts);
    double uL = ri, uY0 = ex * ri, uY1 = ex * fma(kappa, R, 1.0) * ri * ri2;
    if (COMB) {
        // the upward pass has also multiplied layer m by (2m-1)!!, so the radial functions here are u_m / (2m-1)!!:
        // R^-(2m+1) for Laplace (one product per layer) and, for Yukawa, u~_{m+1} = (u~_m + g_m u~_{m-1}) / R^2
        KL = fma(uL, WV[0], KL);
        KY = fma(uY0, WK[0], KY);
#pragma unroll
        for (int m = 1; m <= PL; ++m) {
            uL *= ri2;
            KL = fma(uL, WV[m], KL);
            KY = fma(uY1, WK[m], KY);
            const double un = fma(ek.g[m], uY0, uY1) * ri2;
            uY0 = uY1;
            uY1 = un;
        }
        return;
    }
    VL = fma(uL, WV[0], VL); KL = fma(uL, WK[0], KL);
    VY = fma(uY0, WV[0], VY); KY = fma(uY0, WK[0], KY);
#pragma unroll
    for (int m = 1; m <= PL; ++m) {                    // p + j <= p + 2j <= PL: partial sums beyond PL are empty
        uL = (2 * m - 1) * uL * ri2;
        VL = fma(uL, WV[m], VL); KL = fma(uL, WK[m], KL);
        VY = fma(uY1, WV[m], VY); KY = fma(uY1, WK[m], KY);
        const double un = ((2 * m + 1) * uY1 + k2 * uY0) * ri2;
        uY0 = uY1;
        uY1 = un;
    }
}

// orders 7, 8: 36 partial sums per target pair leave no room for two blocks per SM (one block, up to 255 registers)
template <int P, bool COMB>
#ifndef M2Q_MINB6
#define M2Q_MINB6 2
#endif
__global__ void __launch_bounds__(M2Q_THREADS, P <= 6 ? M2Q_MINB6 : 1)
k_m2p2(int64_t N, double kappa, pb_expk ek, const pb_item* __restrict__ items, const int32_t* __restrict__ m2p_cell,
       const double4* __restrict__ m2p_ctr, const double2* __restrict__ FF, const double* __restrict__ px,
       const double* __restrict__ py, const double* __restrict__ pz, double* __restrict__ acc)
{
    constexpr int NT = m2q_cfg<P>::NT, NS = M2Q_NS;
    extern __shared__ __align__(128) unsigned char smraw[];
    const int tid = threadIdx.x;
    const int lane = tid & 31, sub = tid >> 5;
    double2* ffw = reinterpret_cast<double2*>(smraw) + (size_t)sub * NS * NT;          // this warp's slots [NS][NT]
    uint64_t* fullw = reinterpret_cast<uint64_t*>(smraw + m2q_cfg<P>::FF_BYTES) + sub * NS;   // and their barriers
    double* Ts = reinterpret_cast<double*>(smraw + m2q_cfg<P>::FF_BYTES + M2Q_W * NS * sizeof(uint64_t));   // [32]
    const pb_item item = items[blockIdx.x];
    const int64_t g = item.group;
    const int32_t e0 = item.r + sub, count = item.count;
    const int nw = count > sub ? (count - sub + M2Q_W - 1) / M2Q_W : 0;     // this warp's cells: list entries e0 + 8 k
    if (tid < 32) Ts[tid] = ek.T[tid];
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) pb_mbar_init(&fullw[s], 1);
        pb_mbar_fence_init();
    }
    __syncthreads();
    const int64_t i0 = g * PB_TG + lane, i1 = i0 + 32;
    const int64_t ic0 = i0 < N ? i0 : N - 1, ic1 = i1 < N ? i1 : N - 1;     // padding lanes repeat the last target; never stored
    const double tx0 = px[ic0], ty0 = py[ic0], tz0 = pz[ic0];
    const double tx1 = px[ic1], ty1 = py[ic1], tz1 = pz[ic1];

    auto issue = [&](int k, int32_t cell) {           // lane 0: cell k of this warp into slot k % NS
        const int slot = k % NS;
        pb_mbar_expect_tx(&fullw[slot], (uint32_t)(NT * sizeof(double2)));
        pb_bulk_g2s(ffw + (size_t)slot * NT, FF + (int64_t)cell * NT, (uint32_t)(NT * sizeof(double2)), &fullw[slot]);
    };
    if (lane == 0)
        for (int k = 0; k < NS - 1 && k < nw; ++k) issue(k, m2p_cell[e0 + M2Q_W * k]);
    int32_t idn = NS - 1 < nw ? m2p_cell[e0 + M2Q_W * (NS - 1)] : 0;        // cell of the next copy to issue
    double4 ccn = nw > 0 ? m2p_ctr[e0] : make_double4(0, 0, 0, 0);           // centre (and order flag) of the next cell to evaluate
    double VL0 = 0, KL0 = 0, VY0 = 0, KY0 = 0, VL1 = 0, KL1 = 0, VY1 = 0, KY1 = 0;
    const double k2 = kappa * kappa;
#pragma unroll 1
    for (int k = 0; k < nw; ++k) {
        // slot (k - 1) % NS was read for the last time before the __syncwarp that ended the previous iteration
        const int kn = k + NS - 1;
        if (lane == 0 && kn < nw) issue(kn, idn);
        idn = kn + 1 < nw ? m2p_cell[e0 + M2Q_W * (kn + 1)] : 0;           // in flight while cell k is evaluated
        const double4 cc = ccn;
        ccn = k + 1 < nw ? m2p_ctr[e0 + M2Q_W * (k + 1)] : cc;
        pb_mbar_wait(&fullw[k % NS], (uint32_t)((k / NS) & 1));
        const double2* ffk = ffw + (size_t)(k % NS) * NT;
        const double dx0 = tx0 - cc.x, dy0 = ty0 - cc.y, dz0 = tz0 - cc.z;
        const double dx1 = tx1 - cc.x, dy1 = ty1 - cc.y, dz1 = tz1 - cc.z;
        constexpr int PL = P >= 4 ? P - 2 : P, PM = P >= 4 ? P - 1 : P;
        // k_lists: bit 0 = order P - 2 is enough, bit 3 = order P - 1 is, bits 1-2 = half mask (all warp-uniform)
        const int code = (int)cc.w;
        const int tier = PL < P ? ((code & 1) ? 2 : ((code & 8) ? 1 : 0)) : 0;
        const int half = (code >> 1) & 3;
        if (half == 3) {                               // both targets of every lane: each term read feeds four FMAs
            double WV0[P + 1], WK0[P + 1], WV1[P + 1], WK1[P + 1];
#pragma unroll
            for (int m = 0; m <= P; ++m) { WV0[m] = 0.0; WK0[m] = 0.0; WV1[m] = 0.0; WK1[m] = 0.0; }
            if (tier == 2) {
                m2p_terms2<P, PL>(ffk, dx0, dy0, dz0, dx1, dy1, dz1, WV0, WK0, WV1, WK1);
                m2p_radial<P, PL, COMB>(dx0, dy0, dz0, WV0, WK0, kappa, k2, ek, Ts, VL0, KL0, VY0, KY0);
                m2p_radial<P, PL, COMB>(dx1, dy1, dz1, WV1, WK1, kappa, k2, ek, Ts, VL1, KL1, VY1, KY1);
            } else if (tier == 1) {
                m2p_terms2<P, PM>(ffk, dx0, dy0, dz0, dx1, dy1, dz1, WV0, WK0, WV1, WK1);
                m2p_radial<P, PM, COMB>(dx0, dy0, dz0, WV0, WK0, kappa, k2, ek, Ts, VL0, KL0, VY0, KY0);
                m2p_radial<P, PM, COMB>(dx1, dy1, dz1, WV1, WK1, kappa, k2, ek, Ts, VL1, KL1, VY1, KY1);
            } else {
                m2p_terms2<P, P>(ffk, dx0, dy0, dz0, dx1, dy1, dz1, WV0, WK0, WV1, WK1);
                m2p_radial<P, P, COMB>(dx0, dy0, dz0, WV0, WK0, kappa, k2, ek, Ts, VL0, KL0, VY0, KY0);
                m2p_radial<P, P, COMB>(dx1, dy1, dz1, WV1, WK1, kappa, k2, ek, Ts, VL1, KL1, VY1, KY1);
            }
        } else {                                       // the cell is accepted for one half of the group only
            const bool second = half == 2;
            const double dx = second ? dx1 : dx0, dy = second ? dy1 : dy0, dz = second ? dz1 : dz0;
            double vl = second ? VL1 : VL0, kl = second ? KL1 : KL0, vy = second ? VY1 : VY0, ky = second ? KY1 : KY0;
            double WV[P + 1], WK[P + 1];
#pragma unroll
            for (int m = 0; m <= P; ++m) { WV[m] = 0.0; WK[m] = 0.0; }
            if (tier == 2) {
                m2p_terms<P, PL>(ffk, dx, dy, dz, WV, WK);
                m2p_radial<P, PL, COMB>(dx, dy, dz, WV, WK, kappa, k2, ek, Ts, vl, kl, vy, ky);
            } else if (tier == 1) {
                m2p_terms<P, PM>(ffk, dx, dy, dz, WV, WK);
                m2p_radial<P, PM, COMB>(dx, dy, dz, WV, WK, kappa, k2, ek, Ts, vl, kl, vy, ky);
            } else {
                m2p_terms<P, P>(ffk, dx, dy, dz, WV, WK);
                m2p_radial<P, P, COMB>(dx, dy, dz, WV, WK, kappa, k2, ek, Ts, vl, kl, vy, ky);
            }
            if (second) { VL1 = vl; KL1 = kl; VY1 = vy; KY1 = ky; }
            else { VL0 = vl; KL0 = kl; VY0 = vy; KY0 = ky; }
        }
        __syncwarp();
    }
    __syncthreads();
    // add the warps' partial sums in a fixed order (the slots are free: every warp has consumed all its cells)
    double* red = reinterpret_cast<double*>(smraw);   // [M2Q_W][4][PB_TG]
    red[(sub * 4 + 0) * PB_TG + lane] = VL0; red[(sub * 4 + 0) * PB_TG + lane + 32] = VL1;
    red[(sub * 4 + 1) * PB_TG + lane] = KL0; red[(sub * 4 + 1) * PB_TG + lane + 32] = KL1;
    red[(sub * 4 + 2) * PB_TG + lane] = VY0; red[(sub * 4 + 2) * PB_TG + lane + 32] = VY1;
    red[(sub * 4 + 3) * PB_TG + lane] = KY0; red[(sub * 4 + 3) * PB_TG + lane + 32] = KY1;
    __syncthreads();
    {
        const int m = tid / PB_TG, tgt = tid & (PB_TG - 1);
        const int64_t i = g * PB_TG + tgt;
        double v = 0;
#pragma unroll
        for (int q = 0; q < M2Q_W; ++q) v += red[(q * 4 + m) * PB_TG + tgt];
        if (i < N) acc[((int64_t)item.slot * 4 + m) * N + i] = v;
    }
}

// ---- P2P (H7; "source-target" interactions) ---------------------------------------------------------
// Kernels of Eq. (3)-(4) without the 1/(4 pi), which the combine step applies once:
//   VL += qV/R, KL += (qK.d)/R^3, VY += qV e^{-kR}/R, KY += (qK.d) e^{-kR}(1+kR)/R^3,  d = x - y.
// One block = one target group (PB_TG consecutive Morton-ordered collocation points) x one slice of
// the group's source list.  The slice is streamed through shared memory in tiles of 64-byte source
// records by TMA bulk copies (double-buffered, mbarrier completion).  The block's P2P_S sub-slices
// (2 warps each) take interleaved sources of a tile for the same 64 targets, so every shared-memory
// read is a warp-wide broadcast; their partial sums are added in a fixed order at the end.
// Per pair: 35 FP64-pipe instructions (D: section 7).
#define P2P_S 4
#define P2P_THREADS (PB_TG * P2P_S)
#define P2P_TILE 256
static_assert(P2P_S == 4, "the final reduction maps one of the 4 outputs to each sub-slice");

__device__ __forceinline__ void p2p_pair(const double4& a, const double4& b, double tx, double ty, double tz, double kappa,
                                         const pb_expk8& ek, const double* __restrict__ Ts, double& VL, double& KL,
                                         double& VY, double& KY)
{
    const double dx = tx - a.x, dy = ty - a.y, dz = tz - a.z;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double nd = fma(b.z, dz, fma(b.y, dy, b.x * dx));
    const double ri = pb_rsqrt(r2);
    const double r = r2 * ri, ri2 = ri * ri;
    const double ex = pb_exp_mkr8(r, ek, Ts);
    const double qr = a.w * ri;
    const double kl = nd * (ri2 * ri);
    VL += qr;
    KL += kl;
    VY = fma(qr, ex, VY);
    KY = fma(kl * ex, fma(kappa, r, 1.0), KY);
}

// Two targets per lane (lane and lane + 32 of the group): every source record read from shared memory feeds two pairs,
// and the loop / address arithmetic is shared; the block's eight warps take interleaved sources of a tile.
#define P2Q_W 8
template <bool CHECK_SELF>
__device__ __forceinline__ void p2p_tile2(const double4* __restrict__ buf, int cnt, int sub, int32_t s0, int32_t self0,
                                          int32_t self1, int K, double kappa, const pb_expk8& ek,
                                          const double* __restrict__ Ts, const double (&t0)[3], const double (&t1)[3],
                                          double (&o0)[4], double (&o1)[4])
{
#pragma unroll 2
    for (int k = sub; k < cnt; k += P2Q_W) {
        const double4 a = buf[2 * k], b = buf[2 * k + 1];
        if (!CHECK_SELF || (unsigned)(s0 + k - self0) >= (unsigned)K)          // own panel: by index (D: R-11)
            p2p_pair(a, b, t0[0], t0[1], t0[2], kappa, ek, Ts, o0[0], o0[1], o0[2], o0[3]);
        if (!CHECK_SELF || (unsigned)(s0 + k - self1) >= (unsigned)K)
            p2p_pair(a, b, t1[0], t1[1], t1[2], kappa, ek, Ts, o1[0], o1[1], o1[2], o1[3]);
    }
}

// a tile of a range listed for one half of the group only (k_lists): one target per lane
template <bool CHECK_SELF>
__device__ __forceinline__ void p2p_tile1(const double4* __restrict__ buf, int cnt, int sub, int32_t s0, int32_t self, int K,
                                          double kappa, const pb_expk8& ek, const double* __restrict__ Ts,
                                          const double (&t)[3], double (&o)[4])
{
#pragma unroll 4
    for (int k = sub; k < cnt; k += P2Q_W) {
        const double4 a = buf[2 * k], b = buf[2 * k + 1];
        if (!CHECK_SELF || (unsigned)(s0 + k - self) >= (unsigned)K)
            p2p_pair(a, b, t[0], t[1], t[2], kappa, ek, Ts, o[0], o[1], o[2], o[3]);
    }
}

template <bool CHECK_SELF>
__device__ __forceinline__ void p2p_tile(const double4* __restrict__ buf, int cnt, int sub, int32_t s0, int32_t selfLo,
                                         int K, double kappa, const pb_expk8& ek, const double* __restrict__ Ts,
                                         double tx, double ty, double tz, double& VL, double& KL, double& VY,
                                         double& KY)
{
#pragma unroll 4
    for (int k = sub; k < cnt; k += P2P_S) {
        if (CHECK_SELF && (unsigned)(s0 + k - selfLo) < (unsigned)K) continue;   // own panel: by index (D: R-11)
        const double4 a = buf[2 * k], b = buf[2 * k + 1];
        const double dx = tx - a.x, dy = ty - a.y, dz = tz - a.z;
        const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        const double nd = fma(b.z, dz, fma(b.y, dy, b.x * dx));
        const double ri = pb_rsqrt(r2);
        const double r = r2 * ri, ri2 = ri * ri;
        const double ex = pb_exp_mkr8(r, ek, Ts);
        const double qr = a.w * ri;
        const double kl = nd * (ri2 * ri);
        VL += qr;
        KL += kl;
        VY = fma(qr, ex, VY);
        KY = fma(kl * ex, fma(kappa, r, 1.0), KY);
    }
}

__global__ void __launch_bounds__(P2P_THREADS)
k_p2p(int64_t N, int K, double kappa, pb_expk8 ek, const pb_item* __restrict__ items,
      const int32_t* __restrict__ p2p_lo, const int32_t* __restrict__ p2p_hi, const int8_t* __restrict__ p2p_mask,
      const double4* __restrict__ srec, const double* __restrict__ px, const double* __restrict__ py, const double* __restrict__ pz,
      double* __restrict__ acc)
{
    __shared__ __align__(128) double4 tile[2][2 * P2P_TILE];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ double Ts[256];
    const int tid = threadIdx.x;
    const int tgt = tid & (PB_TG - 1), sub = tid / PB_TG;
    const pb_item item = items[blockIdx.x];
    const int64_t g = item.group;
    const int slice = item.slot;
    static_assert(P2P_THREADS == 256, "one table entry per thread");
    Ts[tid] = c_T256[tid];
    if (tid == 0) {
        pb_mbar_init(&bar[0], 1);
        pb_mbar_init(&bar[1], 1);
        pb_mbar_fence_init();
    }
    __syncthreads();
    const int64_t i = g * PB_TG + tgt;
    const int64_t ic = i < N ? i : N - 1;            // padding lanes repeat the last target; never stored
    const double tx = px[ic], ty = py[ic], tz = pz[ic];
    const int32_t selfLo = (int32_t)(ic * K);
    const int64_t i1 = (g + 1) * PB_TG < N ? (g + 1) * PB_TG : N;
    const int32_t grpLo = (int32_t)(g * PB_TG * K), grpHi = (int32_t)(i1 * K);

    // this item's share of the group's source list: `count` points from point `a` of range `r` on
    int32_t r = item.r, a = item.a;
    int32_t hi = p2p_hi[r];
    int64_t remaining = item.count;
    int rmask = p2p_mask[r];                          // which half of the group range r is for (k_lists)
    auto next_tile = [&](int32_t& s0, int& cnt, int& mk) -> bool {
        while (remaining > 0) {
            if (a >= hi) { ++r; a = p2p_lo[r]; hi = p2p_hi[r]; rmask = p2p_mask[r]; continue; }
            int64_t c = hi - a;
            if (c > P2P_TILE) c = P2P_TILE;
            if (c > remaining) c = remaining;
            s0 = a; cnt = (int)c; mk = rmask;
            a += (int32_t)c; remaining -= c;
            return true;
        }
        return false;
    };

    double VL = 0, KL = 0, VY = 0, KY = 0;
    int32_t cs0 = 0, ns0 = 0;
    int ccnt = 0, ncnt = 0, cmk = 0, nmk = 0;
    const int half = (tid >> 5) & 1;                  // this warp's targets: 0..31 or 32..63 of the group
    bool have = next_tile(cs0, ccnt, cmk);
    if (have && tid == 0) {
        pb_mbar_expect_tx(&bar[0], (uint32_t)ccnt * 64u);
        pb_bulk_g2s(tile[0], srec + 2 * (int64_t)cs0, (uint32_t)ccnt * 64u, &bar[0]);
    }
    for (uint32_t it = 0; have; ++it) {
        const int st = it & 1;
        const bool more = next_tile(ns0, ncnt, nmk);
        if (more && tid == 0) {                       // the other buffer was released by the barrier below
            pb_mbar_expect_tx(&bar[st ^ 1], (uint32_t)ncnt * 64u);
            pb_bulk_g2s(tile[st ^ 1], srec + 2 * (int64_t)ns0, (uint32_t)ncnt * 64u, &bar[st ^ 1]);
        }
        pb_mbar_wait(&bar[st], (it >> 1) & 1u);
        if (!((cmk >> half) & 1)) {
            // the range is for the other half of the group
        } else if (cs0 < grpHi && cs0 + ccnt > grpLo)
            p2p_tile<true>(tile[st], ccnt, sub, cs0, selfLo, K, kappa, ek, Ts, tx, ty, tz, VL, KL, VY, KY);
        else
            p2p_tile<false>(tile[st], ccnt, sub, cs0, selfLo, K, kappa, ek, Ts, tx, ty, tz, VL, KL, VY, KY);
        __syncthreads();
        have = more;
        cs0 = ns0;
        ccnt = ncnt;
        cmk = nmk;
    }
    // add the sub-slices in a fixed order (tile[0] is free: every thread passed the last barrier)
    double* red = reinterpret_cast<double*>(tile[0]);   // [P2P_S][4][PB_TG]
    red[(sub * 4 + 0) * PB_TG + tgt] = VL;
    red[(sub * 4 + 1) * PB_TG + tgt] = KL;
    red[(sub * 4 + 2) * PB_TG + tgt] = VY;
    red[(sub * 4 + 3) * PB_TG + tgt] = KY;
    __syncthreads();
    {
        const int m = tid / PB_TG;                     // 0..3 (P2P_S == 4 outputs per target)
        double v = 0;
#pragma unroll
        for (int q = 0; q < P2P_S; ++q) v += red[(q * 4 + m) * PB_TG + tgt];
        if (i < N) acc[((int64_t)slice * 4 + m) * N + i] = v;
    }
}

// A ring of P2Q_NS tiles: a leaf holds about 40 Gauss points at C4 and a range is a run of adjacent leaves for the same
// half of the group, often a single one, so a tile is short (the eight warps get five sources each) and one tile of
// look-ahead did not cover the latency of the next copy plus that of the range descriptor it starts from (ncu source
// page, C4: 14 % of the kernel's samples before the first pair and in the descriptor loads).  Descriptors are one
// 16-byte load each and are fetched one range ahead.
#define P2Q_NS 3
#define P2Q_SMEM (P2Q_NS * 2 * P2P_TILE * sizeof(double4) + 256 * sizeof(double) + P2Q_NS * sizeof(uint64_t))
__global__ void __launch_bounds__(P2P_THREADS, 2)
k_p2p2(int64_t N, int K, double kappa, pb_expk8 ek, const pb_item* __restrict__ items, const int4* __restrict__ p2p_rng,
       const double4* __restrict__ srec, const double* __restrict__ px, const double* __restrict__ py, const double* __restrict__ pz,
       double* __restrict__ acc)
{
    extern __shared__ __align__(128) unsigned char p2q_raw[];
    double4* tiles = reinterpret_cast<double4*>(p2q_raw);                                  // [P2Q_NS][2 * P2P_TILE]
    double* Ts = reinterpret_cast<double*>(p2q_raw + P2Q_NS * 2 * P2P_TILE * sizeof(double4));   // [256]
    uint64_t* bar = reinterpret_cast<uint64_t*>(Ts + 256);                                 // [P2Q_NS]
    static_assert(PB_TG == 64 && P2P_THREADS == 32 * P2Q_W, "two targets per lane, eight warps");
    const int tid = threadIdx.x;
    const int lane = tid & 31, sub = tid >> 5;
    const pb_item item = items[blockIdx.x];
    const int64_t g = item.group;
    const int slice = item.slot;
    int32_t r = item.r;
    int4 rc = p2p_rng[r], rn = p2p_rng[r + 1];           // this range and the next one {lo, hi, mask}
    Ts[tid] = c_T256[tid];
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < P2Q_NS; ++s) pb_mbar_init(&bar[s], 1);
        pb_mbar_fence_init();
    }
    __syncthreads();
    const int64_t ia = g * PB_TG + lane, ib = ia + 32;
    const int64_t ica = ia < N ? ia : N - 1, icb = ib < N ? ib : N - 1;   // padding lanes repeat the last target; never stored
    const double t0[3] = {px[ica], py[ica], pz[ica]}, t1[3] = {px[icb], py[icb], pz[icb]};
    const int32_t self0 = (int32_t)(ica * K), self1 = (int32_t)(icb * K);
    const int64_t i1 = (g + 1) * PB_TG < N ? (g + 1) * PB_TG : N;
    const int32_t grpLo = (int32_t)(g * PB_TG * K), grpHi = (int32_t)(i1 * K);

    // this item's share of the group's source list: `count` points from point `a` of range `r` on
    int32_t a = item.a;
    int64_t remaining = item.count;
    struct tile_t { int32_t s0; int cnt, mk; };
    auto next_tile = [&](tile_t& tl, int buf) -> bool {   // the next tile, its copy started into buffer `buf` (thread 0)
        while (remaining > 0) {
            if (a >= rc.y) { ++r; rc = rn; rn = p2p_rng[r + 1]; a = rc.x; continue; }
            int64_t c = rc.y - a;
            if (c > P2P_TILE) c = P2P_TILE;
            if (c > remaining) c = remaining;
            tl.s0 = a; tl.cnt = (int)c; tl.mk = rc.z;
            if (tid == 0) {
                pb_mbar_expect_tx(&bar[buf], (uint32_t)c * 64u);
                pb_bulk_g2s(tiles + (size_t)buf * 2 * P2P_TILE, srec + 2 * (int64_t)a, (uint32_t)c * 64u, &bar[buf]);
            }
            a += (int32_t)c; remaining -= c;
            return true;
        }
        tl.cnt = 0;
        return false;
    };

    double o0[4] = {0, 0, 0, 0}, o1[4] = {0, 0, 0, 0};
    static_assert(P2Q_NS == 3, "the tiles in flight are kept in three registers sets");
    tile_t tc, tn, tnn;                                   // tile it, it + 1, it + 2
    next_tile(tc, 0);
    next_tile(tn, 1);
    for (uint32_t it = 0; tc.cnt > 0; ++it) {
        const int st = it % P2Q_NS;
        next_tile(tnn, (it + 2) % P2Q_NS);                // its buffer held tile it - 1: released by the barrier below
        pb_mbar_wait(&bar[st], (it / P2Q_NS) & 1u);
        const double4* tile = tiles + (size_t)st * 2 * P2P_TILE;
        const bool own = tc.s0 < grpHi && tc.s0 + tc.cnt > grpLo;   // the tile holds points of the group's own panels
        if (tc.mk == 3) {
            if (own) p2p_tile2<true>(tile, tc.cnt, sub, tc.s0, self0, self1, K, kappa, ek, Ts, t0, t1, o0, o1);
            else p2p_tile2<false>(tile, tc.cnt, sub, tc.s0, self0, self1, K, kappa, ek, Ts, t0, t1, o0, o1);
        } else if (tc.mk == 1) {
            if (own) p2p_tile1<true>(tile, tc.cnt, sub, tc.s0, self0, K, kappa, ek, Ts, t0, o0);
            else p2p_tile1<false>(tile, tc.cnt, sub, tc.s0, self0, K, kappa, ek, Ts, t0, o0);
        } else {
            if (own) p2p_tile1<true>(tile, tc.cnt, sub, tc.s0, self1, K, kappa, ek, Ts, t1, o1);
            else p2p_tile1<false>(tile, tc.cnt, sub, tc.s0, self1, K, kappa, ek, Ts, t1, o1);
        }
        __syncthreads();
        tc = tn;
        tn = tnn;
    }
    // add the warps' partial sums in a fixed order (tile[0] is free: every thread passed the last barrier)
    double* red = reinterpret_cast<double*>(tiles);   // [P2Q_W][4][PB_TG] = 16 KB = tile[0]
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        red[(sub * 4 + m) * PB_TG + lane] = o0[m];
        red[(sub * 4 + m) * PB_TG + lane + 32] = o1[m];
    }
    __syncthreads();
    {
        const int m = tid / PB_TG, tgt = tid & (PB_TG - 1);
        const int64_t i = g * PB_TG + tgt;
        double v = 0;
#pragma unroll
        for (int q = 0; q < P2Q_W; ++q) v += red[(q * 4 + m) * PB_TG + tgt];
        if (i < N) acc[((int64_t)slice * 4 + m) * N + i] = v;
    }
}

// ---- near/singular table + Eq. (5) combine + un-permute (H8) ------------------------------------------------
// Block = 32 targets x 4 outputs: thread (tgt, m) adds output m of its target over the group's slots
// and over its row of the near table, then thread m == 0 forms the two rows of Eq. (5).  The kernel is
// latency bound (a few dozen dependent loads per thread), so loads are issued eight at a time and
// added in their fixed order afterwards: same sum, an eighth of the round trips.
__device__ __forceinline__ double sum_slots(const double* __restrict__ acc, int ns, int64_t stride, double s)
{
    int q = 0;
    for (; q + 8 <= ns; q += 8) {
        double v[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = acc[(int64_t)(q + k) * stride];
#pragma unroll
        for (int k = 0; k < 8; ++k) s += v[k];
    }
    double v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = q + k < ns ? acc[(int64_t)(q + k) * stride] : 0.0;
#pragma unroll
    for (int k = 0; k < 8; ++k) s += v[k];
    return s;
}

__global__ void __launch_bounds__(128)
k_combine(int64_t N, const int32_t* __restrict__ itemP_off, const int32_t* __restrict__ itemM_off, double eps_ratio,
          const double* __restrict__ accP, const double* __restrict__ accM, const int32_t* __restrict__ el_base,
          const int32_t* __restrict__ el_col, const double* __restrict__ el_val, int64_t ne,
          const double* __restrict__ xphi, const double* __restrict__ xdphi, const int32_t* __restrict__ perm,
          double* __restrict__ y, int64_t blk0, int64_t i1, double* __restrict__ ymort, int64_t nmax,
          double* __restrict__ raw)
{
    // raw != NULL (two surfaces): the four sums V_L, K_L, V_Y, K_Y of this pass go to raw[m N + i] (Morton order)
    // instead of being combined into the rows of Eq. (5)
    // blk0, i1: the launch covers the Morton panels [32 blk0, i1) (target sharding; 0, N otherwise).  ymort != NULL:
    // the two rows go to ymort[k], ymort[nmax + k], k = i - 32 blk0 (Morton order, the all-gather send buffer)
    __shared__ double sm[4][32];
    const int tgt = threadIdx.x & 31, m = threadIdx.x >> 5;
    const int64_t blk = blk0 + blockIdx.x;
    const int64_t i = blk * 32LL + tgt;
    double s = 0.0;
    {
        const int64_t ic = i < N ? i : N - 1;                      // padding lanes: same loads, nothing stored
        const int64_t g = ic / PB_TG;
        const int nsP = itemP_off[g + 1] - itemP_off[g];
        const int nsM = itemM_off ? itemM_off[g + 1] - itemM_off[g] : 0;
        s = sum_slots(accP + (int64_t)m * N + ic, nsP, 4 * N, s);
        if (nsM > 0) s = sum_slots(accM + (int64_t)m * N + ic, nsM, 4 * N, s);
        s *= PB_INV4PI;
        const double* __restrict__ xv = (m & 1) ? xphi : xdphi;     // V_L, V_Y act on dphi; K_L, K_Y on phi
        // the slice's rows of the near table (sliced ELL: the warp reads 32 consecutive entries per step)
        const int32_t b0 = el_base[blk], width = (el_base[blk + 1] - b0) / 32;
        const double* __restrict__ val = el_val + (int64_t)m * ne + b0 + tgt;
        const int32_t* __restrict__ col = el_col + b0 + tgt;
        int k = 0;
        for (; k + 4 <= width; k += 4) {
            double a[4], b[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) { a[q] = val[32 * (k + q)]; b[q] = xv[col[32 * (k + q)]]; }
#pragma unroll
            for (int q = 0; q < 4; ++q) s = fma(a[q], b[q], s);
        }
        for (; k < width; ++k) s = fma(val[32 * k], xv[col[32 * k]], s);
    }
    if (raw) {
        if (i < i1) raw[(int64_t)m * N + i] = s;
        return;
    }
    sm[m][tgt] = s;
    __syncthreads();
    if (m == 0 && i < i1) {
        const double VL = sm[0][tgt], KL = sm[1][tgt], VY = sm[2][tgt], KY = sm[3][tgt];
        const double phi = xphi[i];
        const double r1 = 0.5 * phi + KL - VL;                    // Eq. (5), first row
        const double r2 = 0.5 * phi - KY + eps_ratio * VY;        // Eq. (5), second row
        if (ymort) {
            const int64_t k = i - 32 * blk0;
            ymort[k] = r1;
            ymort[nmax + k] = r2;
        } else {
            const int64_t o = perm[i];
            y[o] = r1;
            y[N + o] = r2;
        }
    }
}

// after the all-gather: rank r's rows [2][nmax] hold the Morton panels first[r] .. first[r + 1]; un-permute into y
__global__ void k_shard_scatter(int64_t N, int world, const int64_t* __restrict__ first, int64_t nmax,
                                const double* __restrict__ yall, const int32_t* __restrict__ perm, double* __restrict__ y)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int r = 0;
    while (r + 1 < world && i >= first[r + 1]) ++r;
    const int64_t k = i - first[r];
    const double* src = yall + (int64_t)r * 2 * nmax;
    const int64_t o = perm[i];
    y[o] = src[k];
    y[N + o] = src[nmax + k];
}

// Two surfaces (pb_set_stern; D: R-32): the rows of the block system from the per-surface sums.
// sA = sums over Gamma_1's sources, sB = over Gamma_2's; [4][N] each: V_L, K_L, V_Y, K_Y (1/(4 pi) and near table included)
__global__ void k_stern_combine(int64_t N, const unsigned char* __restrict__ psurf, const double* __restrict__ sA,
                                const double* __restrict__ sB, const double* __restrict__ xphi_full, double r12, double r23,
                                const int32_t* __restrict__ perm, double* __restrict__ y)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double h = 0.5 * xphi_full[i];
    const double VLA = sA[i], KLA = sA[N + i], VLB = sB[i], KLB = sB[N + i];
    double r1, r2;
    if (psurf[i] == 0) {
        r1 = h + KLA - VLA;                               // region 1 (inside Gamma_1)
        r2 = h - KLA + r12 * VLA + KLB - VLB;             // Stern layer, from outside Gamma_1
    } else {
        r1 = h + KLB - VLB - KLA + r12 * VLA;             // Stern layer, from inside Gamma_2
        r2 = h - sB[3 * N + i] + r23 * sB[2 * N + i];     // solvent (Yukawa), outside Gamma_2
    }
    const int64_t o = perm[i];
    y[o] = r1;
    y[N + o] = r2;
}

// the matvec's far field with the two layers combined (m2p_radial): the two-target kernel's orders, one surface
static bool pb_layers_combined(const pb_ctx* ctx) { return ctx->tree.P <= 8 && !ctx->tree.psurf; }

// ---- host driver ----------------------------------------------------------------------------------------------
template <int P, bool COMB>
static cudaError_t launch_m2p2c(pb_ctx* ctx, cudaStream_t fs)
{
    pb_tree& t = ctx->tree;
    const unsigned bit = 1u << (P + (COMB ? 16 : 0));
    if (!(ctx->attr_m2p_mask & bit)) {   // per device and function: remembered per context (D: section 1)
        cudaError_t e = cudaFuncSetAttribute(k_m2p2<P, COMB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)m2q_cfg<P>::SMEM);
        if (e != cudaSuccess) return e;
        ctx->attr_m2p_mask |= bit;
    }
    k_m2p2<P, COMB><<<(unsigned)t.n_itemM_own, M2Q_THREADS, m2q_cfg<P>::SMEM, fs>>>(
        t.N, ctx->prm.kappa, t.ek, t.itemM + t.itemM0, t.m2p_cell, t.m2p_ctr, t.FF, t.pc[0], t.pc[1], t.pc[2], t.accM);
    return cudaSuccess;
}

// one surface: combined layers (m2p_radial); two surfaces (R-32): V and K apart
template <int P>
static cudaError_t launch_m2p2(pb_ctx* ctx, cudaStream_t fs)
{
    return pb_layers_combined(ctx) ? launch_m2p2c<P, true>(ctx, fs) : launch_m2p2c<P, false>(ctx, fs);
}

template <int P>
static cudaError_t launch_m2p(pb_ctx* ctx, cudaStream_t fs)
{
    pb_tree& t = ctx->tree;
    if (!(ctx->attr_m2p_mask & (1u << P))) {
        cudaError_t e = cudaFuncSetAttribute(k_m2p<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)m2p_cfg<P>::SMEM);
        if (e != cudaSuccess) return e;
        ctx->attr_m2p_mask |= 1u << P;
    }
    k_m2p<P><<<(unsigned)t.n_itemM_own, M2P_THREADS, m2p_cfg<P>::SMEM, fs>>>(
        t.N, ctx->prm.kappa, t.ek, t.itemM + t.itemM0, t.m2p_cell, t.m2p_ctr, t.FF, t.pc[0], t.pc[1], t.pc[2], t.accM);
    return cudaSuccess;
}

// The upward pass for one set of needed cells: `leaf_ids` (one block each) and the per-cell `up_link` words.
// The panel matvec and the site-side treecode (pb_sitetree.cu) each have their own set; both write t.M.
int pb_upward(pb_ctx* ctx, cudaStream_t fs, const int32_t* leaf_ids, int64_t n_leaf, const int32_t* up_link, bool comb)
{
    pb_tree& t = ctx->tree;
    if (n_leaf <= 0) return PB_OK;
    up_args ua;
    ua.P = t.P; ua.Nk = t.Nk; ua.NT = t.NT; ua.K = t.K;
    ua.leaf_ids = leaf_ids; ua.c_first = t.c_first; ua.c_last = t.c_last; ua.c_child = t.c_child;
    ua.c_nchild = t.c_nchild; ua.up_link = up_link; ua.up_count = t.up_count;
    ua.cx = t.c_ctr[0]; ua.cy = t.c_ctr[1]; ua.cz = t.c_ctr[2];
    ua.srec = t.srec;
    ua.mm_off = t.mm_off; ua.mm_ent = t.mm_ent; ua.mm_coef = t.mm_coef;
    ua.cv_off = t.cv_off; ua.cv_idx = t.cv_idx; ua.cv_coef = comb ? t.cv_scale : t.cv_coef;   // comb: layers scaled by (2m-1)!!
    ua.M = t.M; ua.FF = t.FF;
    ua.comb = comb ? 1 : 0;
    ua.eps_ratio = ctx->prm.eps_in / ctx->prm.eps_out;
    const int nr = (t.Nk + UP_THREADS - 1) / UP_THREADS;
    const bool deep = n_leaf >= 148 * 8 * 2;          // more than two waves of blocks even at the highest occupancy
    ua.CH = deep ? P2M_CH_SMALL : P2M_CH_LARGE;
    ua.MQ = deep ? M2M_Q_SMALL : M2M_Q_LARGE;
    const size_t sm = up_smem_bytes(t.Nk, ua.CH, ua.MQ);
    if (sm > 48 * 1024 && sm > ctx->attr_up_bytes) {   // per device: remembered per context
        PB_CUDA(cudaFuncSetAttribute(k_upward<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        PB_CUDA(cudaFuncSetAttribute(k_upward<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        PB_CUDA(cudaFuncSetAttribute(k_upward<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
        ctx->attr_up_bytes = sm;
    }
    if (nr == 1) k_upward<1><<<(unsigned)n_leaf, UP_THREADS, sm, fs>>>(ua);
    else if (nr == 2) k_upward<2><<<(unsigned)n_leaf, UP_THREADS, sm, fs>>>(ua);
    else k_upward<3><<<(unsigned)n_leaf, UP_THREADS, sm, fs>>>(ua);
    PB_LAUNCH_CHECK();
    return PB_OK;
}

// Which cells the SITE lists need (S: section 8(f) item 1): same bookkeeping as in pb_farfield_setup, but every
// needed cell stores its moments (the site kernel reads M, not the F terms).
int pb_site_farfield_setup(pb_ctx* ctx)
{
    pb_tree& t = ctx->tree;
    pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    const int64_t nc = t.n_cells;
    std::vector<int32_t> child(nc), nchild(nc), lists(s.t_m2p_total > 0 ? s.t_m2p_total : 1);
    PB_CUDA(cudaMemcpyAsync(child.data(), t.c_child, sizeof(int32_t) * nc, cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaMemcpyAsync(nchild.data(), t.c_nchild, sizeof(int32_t) * nc, cudaMemcpyDeviceToHost, st));
    if (s.t_m2p_total > 0)
        PB_CUDA(cudaMemcpyAsync(lists.data(), s.t_m2p_cell, sizeof(int32_t) * s.t_m2p_total, cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));
    std::vector<char> need(nc, 0);
    for (int64_t e = 0; e < s.t_m2p_total; ++e) need[lists[e]] = 1;
    std::vector<int32_t> leaf_list, parent(nc, -1), up(nc, 0);
    for (int64_t c = 0; c < nc; ++c) {               // parents come before their children
        if (!need[c]) continue;
        if (child[c] < 0) leaf_list.push_back((int32_t)c);
        else
            for (int q = 0; q < nchild[c]; ++q) { need[child[c] + q] = 1; parent[child[c] + q] = (int32_t)c; }
    }
    std::vector<char> listed(nc, 0);
    for (int64_t e = 0; e < s.t_m2p_total; ++e) listed[lists[e]] = 1;
    // bit 0: the cell's far-field terms F are wanted (k_site_grad reads them), bit 1: its moments are stored (k_site_m2p)
    for (int64_t c = 0; c < nc; ++c)
        if (need[c]) up[c] = (listed[c] ? 1 : 0) | 2 | ((parent[c] >= 0 ? parent[c] + 1 : 0) << 2);
    s.t_n_need_leaf = (int64_t)leaf_list.size();
    PB_TRY(pb_dalloc_t(ctx, &s.t_need_leaf, leaf_list.size() > 0 ? leaf_list.size() : 1, CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &s.t_up_link, (size_t)nc, CAT_SITE_NEAR));
    if (!leaf_list.empty())
        PB_CUDA(cudaMemcpyAsync(s.t_need_leaf, leaf_list.data(), sizeof(int32_t) * leaf_list.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyAsync(s.t_up_link, up.data(), sizeof(int32_t) * nc, cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaStreamSynchronize(st));
    return PB_OK;
}

// Far-field branch: the upward pass (P2M, M2M, M -> F) in one launch, then M2P.  `fs` is the stream it
// is enqueued on: the context's side stream (concurrent with P2P) or, when per-kernel event timing
// is wanted, the main stream.
static int pb_far_branch(pb_ctx* ctx, cudaStream_t fs, bool timed)
{
    pb_tree& t = ctx->tree;
    PB_TRY(pb_upward(ctx, fs, t.need_leaf, t.n_need_leaf, t.up_link, pb_layers_combined(ctx)));
    if (timed) PB_CUDA(cudaEventRecord(ctx->ev[2], fs));
    if (t.n_itemM_own > 0) {
        PB_TRY(pb_prof_begin(ctx, 1));
        cudaError_t e = cudaSuccess;
        switch (t.P) {
        case 0: e = launch_m2p2<0>(ctx, fs); break;
        case 1: e = launch_m2p2<1>(ctx, fs); break;
        case 2: e = launch_m2p2<2>(ctx, fs); break;
        case 3: e = launch_m2p2<3>(ctx, fs); break;
        case 4: e = launch_m2p2<4>(ctx, fs); break;
        case 5: e = launch_m2p2<5>(ctx, fs); break;
        case 6: e = launch_m2p2<6>(ctx, fs); break;
        case 7: e = launch_m2p2<7>(ctx, fs); break;
        case 8: e = launch_m2p2<8>(ctx, fs); break;
        case 9: e = launch_m2p<9>(ctx, fs); break;
        case 10: e = launch_m2p<10>(ctx, fs); break;
        default: return pb_fail(ctx, PB_ERR_INVALID_ARG, "unsupported order_P %d", t.P);
        }
        PB_CUDA(e);
        PB_LAUNCH_CHECK();
        PB_TRY(pb_prof_end(ctx, 1));
    }
    return PB_OK;
}

// y = A x (or A Minv x with `precond`).  Normal operation: the near field (P2P) runs on the context's
// stream while the far-field branch runs on the side stream; both join before the combine.  With
// `timed` or pb_set_profiling the two branches run back to back on the context's stream so that
// every CUDA-event pair brackets exactly one kernel.
int pb_matvec_impl(pb_ctx* ctx, const double* x, double* y, bool timed, bool precond)
{
    pb_tree& t = ctx->tree;
    cudaStream_t st = ctx->stream;
    if (!t.built) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_matvec: call pb_tree_build first");
    if (!x || !y || x == y) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_matvec: x and y must be distinct non-NULL device arrays");
    if (timed && !ctx->ev_made) {
        for (int k = 0; k < 8; ++k) PB_CUDA(cudaEventCreate(&ctx->ev[k]));
        ctx->ev_made = true;
    }
    const bool stern = t.psurf != nullptr;
    // two surfaces: the same kernels twice, once with the sources of Gamma_1 and once with those of Gamma_2 (the
    // sums are linear in the source weights), then the rows of the block system from the two sets of sums
    for (int surface = stern ? 0 : -1; surface < (stern ? 2 : 0); ++surface) {
        const bool far = ctx->prm.theta > 0.0;
        const bool serial = timed || ctx->profiling;
        if (timed) PB_CUDA(cudaEventRecord(ctx->ev[0], st));
        PB_TRY(pb_weights(ctx, x, precond, surface));
        if (timed) PB_CUDA(cudaEventRecord(ctx->ev[1], st));
        if (far && serial) PB_TRY(pb_far_branch(ctx, st, timed));
        if (far && !serial) {
            // the far-field branch is the longer one on small meshes (a latency chain): enqueue it first
            PB_CUDA(cudaEventRecord(ctx->ev_fork, st));
            PB_CUDA(cudaStreamWaitEvent(ctx->side, ctx->ev_fork, 0));
            PB_TRY(pb_far_branch(ctx, ctx->side, false));
            PB_CUDA(cudaEventRecord(ctx->ev_join, ctx->side));
        }
        if (timed) {
            if (!far) PB_CUDA(cudaEventRecord(ctx->ev[2], st));
            PB_CUDA(cudaEventRecord(ctx->ev[3], st));
        }
        {
            PB_TRY(pb_prof_begin(ctx, 0));
            // two targets per lane pays once the kernel is throughput-bound (measured: C3 529 -> 516 us, C4 8.43 -> 8.24 ms;
            // C1 / C2, a few waves of short blocks, are 2-4 % faster with one target per thread and twice the resident warps)
            if (t.n_itemP_own > 0) {
                if (t.N >= 30000) {
                    if (!ctx->attr_p2p_set) {     // per device and function: remembered per context
                        PB_CUDA(cudaFuncSetAttribute(k_p2p2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P2Q_SMEM));
                        ctx->attr_p2p_set = true;
                    }
                    k_p2p2<<<(unsigned)t.n_itemP_own, P2P_THREADS, P2Q_SMEM, st>>>(t.N, t.K, ctx->prm.kappa, t.ek8, t.itemP + t.itemP0, t.p2p_rng,
                                                                                 t.srec, t.pc[0], t.pc[1], t.pc[2], t.accP);
                }
                else
                    k_p2p<<<(unsigned)t.n_itemP_own, P2P_THREADS, 0, st>>>(t.N, t.K, ctx->prm.kappa, t.ek8, t.itemP + t.itemP0, t.p2p_lo,
                                                                         t.p2p_hi, t.p2p_mask, t.srec, t.pc[0], t.pc[1], t.pc[2], t.accP);
                PB_LAUNCH_CHECK();
            }
            PB_TRY(pb_prof_end(ctx, 0));
            pb_prof_next(ctx);
        }
        if (far && !serial) PB_CUDA(cudaStreamWaitEvent(st, ctx->ev_join, 0));
        if (timed) PB_CUDA(cudaEventRecord(ctx->ev[4], st));
        {
            // the owned Morton panels [own_i0, own_i1) (all of them without sharding); own_i0 is a multiple of PB_TG = 2 x 32
            const bool exchange = ctx->shard_world > 1 && ctx->allgather != nullptr;
            const int64_t nown = t.own_i1 - t.own_i0;
            if (nown > 0) {
                k_combine<<<pb_blocks(nown, 32), 128, 0, st>>>(t.N, t.itemP_off, far ? t.itemM_off : nullptr,
                                                              ctx->prm.eps_in / ctx->prm.eps_out, t.accP, t.accM, t.el_base, t.el_col,
                                                              t.el_val, t.el_entries, t.xphi, t.xdphi, t.perm, y, t.own_i0 / 32,
                                                              t.own_i1, exchange ? t.ysend : nullptr, t.shard_nmax,
                                                              surface >= 0 ? t.sraw + (size_t)surface * 4 * t.N : nullptr);
                PB_LAUNCH_CHECK();
            }
            if (exchange && surface < 0) {
                // the ONE exchange step of a sharded matvec: all-gather of the owned rows (enqueued on this stream by the callback)
                if (ctx->allgather(ctx->allgather_user, t.ysend, t.yall, (size_t)2 * t.shard_nmax * sizeof(double)) != 0)
                    return pb_fail(ctx, PB_ERR_CUDA, "pb_matvec: the all-gather callback failed");
                k_shard_scatter<<<pb_blocks(t.N, 256), 256, 0, st>>>(t.N, ctx->shard_world, t.shard_first_dev, t.shard_nmax, t.yall,
                                                                    t.perm, y);
                PB_LAUNCH_CHECK();
            }
        }
    }
    if (stern) {
        k_stern_combine<<<pb_blocks(t.N, 256), 256, 0, st>>>(t.N, t.psurf, t.sraw, t.sraw + (size_t)4 * t.N, t.xphi_full,
                                                            ctx->prm.eps_in / ctx->eps_stern, ctx->eps_stern / ctx->prm.eps_out,
                                                            t.perm, y);
        PB_LAUNCH_CHECK();
    }
    ctx->matvec_calls++;
    if (timed) {
        PB_CUDA(cudaEventRecord(ctx->ev[5], st));
        PB_CUDA(cudaEventSynchronize(ctx->ev[5]));
        float ms;
        for (int k = 0; k < 5; ++k) {
            PB_CUDA(cudaEventElapsedTime(&ms, ctx->ev[k], ctx->ev[k + 1]));
            ctx->last_ms[k] = ms;
        }
        PB_CUDA(cudaEventElapsedTime(&ms, ctx->ev[0], ctx->ev[5]));
        ctx->last_ms[5] = ms;
    }
    return PB_OK;
}

extern "C" int pb_matvec(pb_ctx* ctx, const double* x, double* y)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    return pb_matvec_impl(ctx, x, y, false, false);
}

extern "C" int pb_matvec_timed(pb_ctx* ctx, const double* x, double* y)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    return pb_matvec_impl(ctx, x, y, true, false);
}

extern "C" int pb_matvec_host(pb_ctx* ctx, const double* x_host, double* y_host)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (!ctx->tree.built) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_matvec_host: call pb_tree_build first");
    if (!x_host || !y_host) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_matvec_host: NULL buffer");
    const size_t n = 2 * (size_t)ctx->nt;
    PB_TRY(pb_scratch(ctx, 2 * n * sizeof(double) + 4096));
    double* dx = ctx->scratch;
    double* dy = ctx->scratch + n;
    PB_CUDA(cudaMemcpyAsync(dx, x_host, n * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    PB_TRY(pb_matvec_impl(ctx, dx, dy, false, false));
    PB_CUDA(cudaMemcpyAsync(y_host, dy, n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    PB_CUDA(cudaStreamSynchronize(ctx->stream));
    return PB_OK;
}
