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
#include <math.h>
#include "pb_internal.cuh"

// ---- index tables ------------------------------------------------------------------------------
__host__ __device__ static inline int mom_index(int a, int b, int c)
{
    int n = a + b + c, m = b + c;
    return n * (n + 1) * (n + 2) / 6 + m * (m + 1) / 2 + c;
}

__host__ __device__ static constexpr int pb_nk(int P) { return (P + 1) * (P + 2) * (P + 3) / 6; }
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
    // exponent tables
    unsigned char ka[PB_MAX_NK], kb[PB_MAX_NK], kc[PB_MAX_NK];
    for (int a = 0; a <= P; ++a)
        for (int b = 0; b <= P - a; ++b)
            for (int c = 0; c <= P - a - b; ++c) {
                int k = mom_index(a, b, c);
                ka[k] = (unsigned char)a; kb[k] = (unsigned char)b; kc[k] = (unsigned char)c;
            }
    PB_CUDA(cudaMemcpyToSymbolAsync(c_ka, ka, t.Nk, 0, cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyToSymbolAsync(c_kb, kb, t.Nk, 0, cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaMemcpyToSymbolAsync(c_kc, kc, t.Nk, 0, cudaMemcpyHostToDevice, st));
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
    // M2M table: for every k the triples (l, k - l, C(k,l)), l <= k componentwise
    std::vector<int32_t> mo(1, 0), me;
    std::vector<double> mc;
    for (int k = 0; k < t.Nk; ++k) {
        const int a = ka[k], b = kb[k], c = kc[k];
        for (int la = 0; la <= a; ++la)
            for (int lb = 0; lb <= b; ++lb)
                for (int lc = 0; lc <= c; ++lc) {
                    me.push_back(mom_index(la, lb, lc) | ((a - la) << 12) | ((b - lb) << 16) | ((c - lc) << 20));
                    mc.push_back(factorial(a) / (factorial(la) * factorial(a - la)) * factorial(b) /
                                 (factorial(lb) * factorial(b - lb)) * factorial(c) / (factorial(lc) * factorial(c - lc)));
                }
        mo.push_back((int32_t)me.size());
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
    std::vector<int32_t> child(nc), nchild(nc), lists(t.m2p_total > 0 ? t.m2p_total : 1);
    PB_CUDA(cudaMemcpyAsync(child.data(), t.c_child, sizeof(int32_t) * nc, cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaMemcpyAsync(nchild.data(), t.c_nchild, sizeof(int32_t) * nc, cudaMemcpyDeviceToHost, st));
    if (t.m2p_total > 0)
        PB_CUDA(cudaMemcpyAsync(lists.data(), t.m2p_cell, sizeof(int32_t) * t.m2p_total, cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));   // also: the host vectors above go out of scope
    std::vector<char> used(nc, 0), need(nc, 0);
    for (int64_t e = 0; e < t.m2p_total; ++e) used[lists[e]] = 1;
    std::vector<int32_t> used_list, leaf_list, m2m_list;
    t.m2m_start.assign(1, 0);
    for (size_t g = 0; g + 1 < t.gen_start.size(); ++g) {     // cells are numbered generation by generation
        for (int64_t c = t.gen_start[g]; c < t.gen_start[g + 1]; ++c) {
            need[c] = need[c] || used[c];
            if (used[c]) used_list.push_back((int32_t)c);
            if (!need[c]) continue;
            if (child[c] < 0) leaf_list.push_back((int32_t)c);
            else {
                m2m_list.push_back((int32_t)c);
                for (int q = 0; q < nchild[c]; ++q) need[child[c] + q] = 1;
            }
        }
        t.m2m_start.push_back((int64_t)m2m_list.size());
    }
    t.n_used = (int64_t)used_list.size();
    t.n_need_leaf = (int64_t)leaf_list.size();
    PB_TRY(pb_dalloc_t(ctx, &t.used_cells, used_list.size(), CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.need_leaf, leaf_list.size(), CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.m2m_cells, m2m_list.size(), CAT_TREE));
    if (!used_list.empty())
        PB_CUDA(cudaMemcpyAsync(t.used_cells, used_list.data(), sizeof(int32_t) * used_list.size(), cudaMemcpyHostToDevice, st));
    if (!leaf_list.empty())
        PB_CUDA(cudaMemcpyAsync(t.need_leaf, leaf_list.data(), sizeof(int32_t) * leaf_list.size(), cudaMemcpyHostToDevice, st));
    if (!m2m_list.empty())
        PB_CUDA(cudaMemcpyAsync(t.m2m_cells, m2m_list.data(), sizeof(int32_t) * m2m_list.size(), cudaMemcpyHostToDevice, st));
    PB_CUDA(cudaStreamSynchronize(st));
    PB_TRY(pb_dalloc_t(ctx, &t.M, (size_t)t.n_cells * 2 * t.Nk, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.FF, (size_t)t.n_cells * t.NT, CAT_TREE));
    return PB_OK;
}

// ---- source weights (H5): q^V_g = w_g A_j dphi_j ,  q^K_g = w_g A_j phi_j n_j ------------------------
// Writes the 64-byte source records the P2P / P2M / reaction kernels stream (coordinates repeated
// so that one contiguous TMA bulk copy brings a whole tile of sources into shared memory).
__global__ void k_weights(int64_t N, int K, const int32_t* __restrict__ perm, const double* __restrict__ x,
                          const double* __restrict__ swA, const double* __restrict__ sx,
                          const double* __restrict__ sy, const double* __restrict__ sz,
                          const double* __restrict__ nx, const double* __restrict__ ny,
                          const double* __restrict__ nz, double* __restrict__ xphi, double* __restrict__ xdphi,
                          double4* __restrict__ srec)
{
    int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= N * K) return;
    int64_t i = s / K;
    int64_t o = perm[i];
    double phi = x[o], dphi = x[N + o], w = swA[s];
    if (s == i * K) { xphi[i] = phi; xdphi[i] = dphi; }
    double wp = w * phi;
    srec[2 * s] = make_double4(sx[s], sy[s], sz[s], w * dphi);
    srec[2 * s + 1] = make_double4(wp * nx[i], wp * ny[i], wp * nz[i], 0.0);
}

int pb_weights(pb_ctx* ctx, const double* x)
{
    pb_tree& t = ctx->tree;
    k_weights<<<pb_blocks(t.Ns, 256), 256, 0, ctx->stream>>>(t.N, t.K, t.perm, x, t.swA, t.sx[0], t.sx[1], t.sx[2], t.pn[0],
                                                            t.pn[1], t.pn[2], t.xphi, t.xdphi, t.srec);
    PB_LAUNCH_CHECK();
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
}

// ---- P2M at the leaves: M^V_k = sum_g q^V_g h^k,  M^K_k = sum_g sum_d q^K_{g,d} k_d h^{k-e_d} ---
// Four plain moment sets per cell are accumulated, S^V, S^x, S^y, S^z (weights q^V, q^K_x, q^K_y,
// q^K_z), one monomial serving all four; then M^K_(a,b,c) = a S^x_(a-1,b,c) + b S^y_(a,b-1,c) + c S^z_(a,b,c-1).
#define P2M_CH 32
#define P2M_LD (PB_MAX_P + 1)     // 11 doubles per point: odd stride, so a warp's reads of one point do not conflict
__global__ void __launch_bounds__(128)
k_p2m_leaf(int P, int Nk, int K, const int32_t* __restrict__ leaf_ids, const int32_t* __restrict__ c_first,
           const int32_t* __restrict__ c_last, const double* __restrict__ cx, const double* __restrict__ cy,
           const double* __restrict__ cz, const double4* __restrict__ srec, double* __restrict__ M)
{
    __shared__ double pw[3][P2M_CH][P2M_LD];
    __shared__ double4 wq[P2M_CH];
    __shared__ double sk[3][PB_MAX_NK];
    const int nth = blockDim.x;
    const int32_t c = leaf_ids[blockIdx.x];
    const int64_t s0 = (int64_t)c_first[c] * K, s1 = (int64_t)c_last[c] * K;
    const double yc[3] = {cx[c], cy[c], cz[c]};
    int ea[3], eb[3], ec[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        const int k = threadIdx.x + r * nth;
        ea[r] = k < Nk ? c_ka[k] : 0; eb[r] = k < Nk ? c_kb[k] : 0; ec[r] = k < Nk ? c_kc[k] : 0;
    }
    double acc[3][4];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int m = 0; m < 4; ++m) acc[r][m] = 0.0;
    for (int64_t base = s0; base < s1; base += P2M_CH) {
        const int np = (int)((s1 - base) < P2M_CH ? (s1 - base) : P2M_CH);
        __syncthreads();
        if (threadIdx.x < np) {
            const int64_t s = base + threadIdx.x;
            const double4 ra = srec[2 * s], rb = srec[2 * s + 1];
            const double h[3] = {ra.x - yc[0], ra.y - yc[1], ra.z - yc[2]};
            for (int d = 0; d < 3; ++d) {
                double p = 1.0;
                for (int e = 0; e <= P; ++e) { pw[d][threadIdx.x][e] = p; p *= h[d]; }
            }
            wq[threadIdx.x] = make_double4(ra.w, rb.x, rb.y, rb.z);
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            if (threadIdx.x + r * nth < Nk) {
#pragma unroll 4
                for (int p = 0; p < np; ++p) {
                    const double mono = pw[0][p][ea[r]] * pw[1][p][eb[r]] * pw[2][p][ec[r]];
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
    for (int r = 0; r < 3; ++r) {
        const int k = threadIdx.x + r * nth;
        if (k < Nk) {
            M[((int64_t)c * 2 + 0) * Nk + k] = acc[r][0];
            sk[0][k] = acc[r][1]; sk[1][k] = acc[r][2]; sk[2][k] = acc[r][3];
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        const int k = threadIdx.x + r * nth;
        if (k < Nk) {
            const int a = ea[r], b = eb[r], cc = ec[r];
            double v = 0.0;
            if (a) v = fma((double)a, sk[0][mom_index(a - 1, b, cc)], v);
            if (b) v = fma((double)b, sk[1][mom_index(a, b - 1, cc)], v);
            if (cc) v = fma((double)cc, sk[2][mom_index(a, b, cc - 1)], v);
            M[((int64_t)c * 2 + 1) * Nk + k] = v;
        }
    }
}

// ---- M2M: moments of a parent from its children, M'_k = sum_{l<=k} C(k,l) t^{k-l} M_l -------------
// Table driven: for every k the (l, k-l, C(k,l)) triples are listed once on the host (mm_*), so a
// thread does no index arithmetic.  Only cells some M2P list needs (directly or through an accepted
// ancestor) are visited: `cells` is the compacted list for one BFS generation.  All children are
// staged in shared memory at once (one global-memory latency per cell).
__global__ void __launch_bounds__(128)
k_m2m(const int32_t* __restrict__ cells, int P, int Nk, const int32_t* __restrict__ c_child,
      const int32_t* __restrict__ c_nchild, const double* __restrict__ cx, const double* __restrict__ cy,
      const double* __restrict__ cz, const int32_t* __restrict__ mm_off, const int32_t* __restrict__ mm_ent,
      const double* __restrict__ mm_coef, double* __restrict__ M)
{
    extern __shared__ double m2m_sm[];                 // cm[8][2*Nk], tp[8][3][PB_MAX_P+1]
    double* cm = m2m_sm;
    double* tp = m2m_sm + 8 * 2 * Nk;
    const int nth = blockDim.x;
    const int64_t c = cells[blockIdx.x];
    const int32_t ch = c_child[c];
    const int nc = c_nchild[c];
    for (int k = threadIdx.x; k < nc * 2 * Nk; k += nth) cm[k] = M[(int64_t)ch * 2 * Nk + k];   // children are consecutive
    if (threadIdx.x < 3 * nc) {
        const int q = threadIdx.x / 3, d = threadIdx.x % 3;
        const double* ctr = d == 0 ? cx : (d == 1 ? cy : cz);
        double tt = ctr[ch + q] - ctr[c], p = 1.0;
        for (int e = 0; e <= P; ++e) { tp[(q * 3 + d) * (PB_MAX_P + 1) + e] = p; p *= tt; }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < Nk; k += nth) {
        double s0 = 0, s1 = 0;
        const int e0 = mm_off[k], e1 = mm_off[k + 1];
        for (int e = e0; e < e1; ++e) {
            const int32_t ent = mm_ent[e];
            const double cf = mm_coef[e];
            const int l = ent & 0xfff, dx = (ent >> 12) & 15, dy = (ent >> 16) & 15, dz = (ent >> 20) & 15;
            for (int q = 0; q < nc; ++q) {
                const double* t3 = tp + q * 3 * (PB_MAX_P + 1);
                const double f = cf * t3[dx] * t3[(PB_MAX_P + 1) + dy] * t3[2 * (PB_MAX_P + 1) + dz];
                s0 = fma(f, cm[q * 2 * Nk + l], s0);
                s1 = fma(f, cm[q * 2 * Nk + Nk + l], s1);
            }
        }
        M[(c * 2 + 0) * Nk + k] = s0;
        M[(c * 2 + 1) * Nk + k] = s1;
    }
}

// ---- M -> F conversion (cells that appear in an M2P list only) ---------------------------------------
__global__ void k_convert(int64_t nused, const int32_t* __restrict__ used, int Nk, int NT,
                          const int32_t* __restrict__ cv_off, const int32_t* __restrict__ cv_idx,
                          const double* __restrict__ cv_coef, const double* __restrict__ M, double2* __restrict__ FF)
{
    int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= nused * NT) return;
    const int64_t c = used[g / NT];
    const int e = (int)(g % NT);
    const double* mv = M + c * 2 * Nk;
    const double* mk = mv + Nk;
    double v = 0, k = 0;
    for (int q = cv_off[e]; q < cv_off[e + 1]; ++q) {
        int l = cv_idx[q];
        double f = cv_coef[q];
        v += f * mv[l];
        k += f * mk[l];
    }
    FF[c * NT + e] = make_double2(v, k);
}

// ---- M2P (H6; "box-target" interactions) -----------------------------------------------------------
template <int P>
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
                    const double2 f = ff[e];
                    ++e;
                    WV[n + j] = fma(mono, f.x, WV[n + j]);
                    WK[n + j] = fma(mono, f.y, WK[n + j]);
                }
                mono *= dz;
            }
            xy *= dy;
        }
        xa *= dx;
    }
}

// One block = one work item: a target group (PB_TG targets) x a run of its accepted cells.  The
// cells' F terms (N_T x {V,K}, contiguous per cell) and centres arrive in shared memory by TMA bulk
// copies, CT cells per stage, two stages; the block's M2P_S sub-slices (2 warps each) take different
// cells of a stage for the same targets, so all shared-memory reads are warp-wide broadcasts.
#define M2P_S 4
#define M2P_THREADS (PB_TG * M2P_S)
static_assert(M2P_S == 4, "the final reduction maps one of the 4 outputs to each sub-slice");

template <int P> struct m2p_cfg {
    static constexpr int NT = pb_nt(P);
    static constexpr int CT = P <= 6 ? 8 : 4;                    // cells per stage
    static constexpr size_t RED_BYTES = (size_t)M2P_S * 4 * PB_TG * sizeof(double);   // final reduction reuses the stages
    static constexpr size_t FF_BYTES0 = (size_t)2 * CT * NT * sizeof(double2);
    static constexpr size_t FF_BYTES = FF_BYTES0 > RED_BYTES ? FF_BYTES0 : RED_BYTES;
    static constexpr size_t SMEM = FF_BYTES + 2 * CT * sizeof(double4) + 2 * sizeof(uint64_t) + 32 * sizeof(double);
};

template <int P>
__global__ void __launch_bounds__(M2P_THREADS)
k_m2p(int64_t N, double kappa, pb_expk ek, const pb_item* __restrict__ items, const int32_t* __restrict__ m2p_cell,
      const double4* __restrict__ m2p_ctr, const double2* __restrict__ FF, const double* __restrict__ px,
      const double* __restrict__ py, const double* __restrict__ pz, double* __restrict__ acc)
{
    constexpr int NT = m2p_cfg<P>::NT, CT = m2p_cfg<P>::CT;
    extern __shared__ __align__(128) unsigned char smraw[];
    double2* ff = reinterpret_cast<double2*>(smraw);                                  // [2][CT][NT]
    double4* ctr = reinterpret_cast<double4*>(smraw + m2p_cfg<P>::FF_BYTES);           // [2][CT]
    uint64_t* bar = reinterpret_cast<uint64_t*>(ctr + 2 * CT);                         // [2]
    double* Ts = reinterpret_cast<double*>(bar + 2);                                   // [32]
    const int tid = threadIdx.x;
    const int tgt = tid & (PB_TG - 1), sub = tid / PB_TG;
    const pb_item item = items[blockIdx.x];
    const int64_t g = item.group;
    const int32_t e0 = item.r, count = item.count;
    if (tid < 32) Ts[tid] = ek.T[tid];
    if (tid == 0) {
        pb_mbar_init(&bar[0], 1);
        pb_mbar_init(&bar[1], 1);
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
        pb_mbar_expect_tx(&bar[stage], (uint32_t)(n * (sizeof(double4) + NT * sizeof(double2))));
        pb_bulk_g2s(ctr + stage * CT, m2p_ctr + e0 + t * CT, (uint32_t)(n * sizeof(double4)), &bar[stage]);
#pragma unroll
        for (int j = 0; j < CT; ++j)
            if (j < n)
                pb_bulk_g2s(ff + ((size_t)stage * CT + j) * NT, FF + (int64_t)idn[j] * NT, (uint32_t)(NT * sizeof(double2)),
                            &bar[stage]);
    };
    if (tid == 0 && ntile > 0) {
        load_ids(0);
        issue(0, 0);
        if (ntile > 1) load_ids(1);
    }
    double VL = 0, KL = 0, VY = 0, KY = 0;
    const double k2 = kappa * kappa;
    for (int t = 0; t < ntile; ++t) {
        const int st = t & 1;
        if (tid == 0 && t + 1 < ntile) {              // the other stage was released by the barrier below
            issue(t + 1, st ^ 1);
            if (t + 2 < ntile) load_ids(t + 2);
        }
        pb_mbar_wait(&bar[st], (t >> 1) & 1u);
        const int cnt = count - t * CT < CT ? count - t * CT : CT;
#pragma unroll 1
        for (int j = sub; j < cnt; j += M2P_S) {
            const double4 cc = ctr[st * CT + j];
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
        __syncthreads();
    }
    // add the sub-slices in a fixed order (the stages are free: every thread passed the last barrier)
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

template <bool CHECK_SELF>
__device__ __forceinline__ void p2p_tile(const double4* __restrict__ buf, int cnt, int sub, int32_t s0, int32_t selfLo,
                                         int K, double kappa, const pb_expk& ek, const double* __restrict__ Ts,
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
        const double ex = pb_exp_mkr(r, ek, Ts);
        const double qr = a.w * ri;
        const double kl = nd * (ri2 * ri);
        VL += qr;
        KL += kl;
        VY = fma(qr, ex, VY);
        KY = fma(kl * ex, fma(kappa, r, 1.0), KY);
    }
}

__global__ void __launch_bounds__(P2P_THREADS)
k_p2p(int64_t N, int K, double kappa, pb_expk ek, const pb_item* __restrict__ items,
      const int32_t* __restrict__ p2p_lo, const int32_t* __restrict__ p2p_hi, const double4* __restrict__ srec,
      const double* __restrict__ px, const double* __restrict__ py, const double* __restrict__ pz,
      double* __restrict__ acc)
{
    __shared__ __align__(128) double4 tile[2][2 * P2P_TILE];
    __shared__ __align__(8) uint64_t bar[2];
    __shared__ double Ts[32];
    const int tid = threadIdx.x;
    const int tgt = tid & (PB_TG - 1), sub = tid / PB_TG;
    const pb_item item = items[blockIdx.x];
    const int64_t g = item.group;
    const int slice = item.slot;
    if (tid < 32) Ts[tid] = ek.T[tid];
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
    auto next_tile = [&](int32_t& s0, int& cnt) -> bool {
        while (remaining > 0) {
            if (a >= hi) { ++r; a = p2p_lo[r]; hi = p2p_hi[r]; continue; }
            int64_t c = hi - a;
            if (c > P2P_TILE) c = P2P_TILE;
            if (c > remaining) c = remaining;
            s0 = a; cnt = (int)c;
            a += (int32_t)c; remaining -= c;
            return true;
        }
        return false;
    };

    double VL = 0, KL = 0, VY = 0, KY = 0;
    int32_t cs0 = 0, ns0 = 0;
    int ccnt = 0, ncnt = 0;
    bool have = next_tile(cs0, ccnt);
    if (have && tid == 0) {
        pb_mbar_expect_tx(&bar[0], (uint32_t)ccnt * 64u);
        pb_bulk_g2s(tile[0], srec + 2 * (int64_t)cs0, (uint32_t)ccnt * 64u, &bar[0]);
    }
    for (uint32_t it = 0; have; ++it) {
        const int st = it & 1;
        const bool more = next_tile(ns0, ncnt);
        if (more && tid == 0) {                       // the other buffer was released by the barrier below
            pb_mbar_expect_tx(&bar[st ^ 1], (uint32_t)ncnt * 64u);
            pb_bulk_g2s(tile[st ^ 1], srec + 2 * (int64_t)ns0, (uint32_t)ncnt * 64u, &bar[st ^ 1]);
        }
        pb_mbar_wait(&bar[st], (it >> 1) & 1u);
        if (cs0 < grpHi && cs0 + ccnt > grpLo)
            p2p_tile<true>(tile[st], ccnt, sub, cs0, selfLo, K, kappa, ek, Ts, tx, ty, tz, VL, KL, VY, KY);
        else
            p2p_tile<false>(tile[st], ccnt, sub, cs0, selfLo, K, kappa, ek, Ts, tx, ty, tz, VL, KL, VY, KY);
        __syncthreads();
        have = more;
        cs0 = ns0;
        ccnt = ncnt;
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

// ---- near/singular table + Eq. (5) combine + un-permute (H8) ------------------------------------------------
// Block = 32 targets x 4 outputs: thread (tgt, m) adds output m of its target over the group's slots
// and over its row of the near table, then thread m == 0 forms the two rows of Eq. (5).
__global__ void __launch_bounds__(128)
k_combine(int64_t N, const int32_t* __restrict__ itemP_off, const int32_t* __restrict__ itemM_off, double eps_ratio,
          const double* __restrict__ accP, const double* __restrict__ accM, const int32_t* __restrict__ nr_off,
          const int32_t* __restrict__ nr_col, const double* __restrict__ nr_val, int64_t ne,
          const double* __restrict__ xphi, const double* __restrict__ xdphi, const int32_t* __restrict__ perm,
          double* __restrict__ y)
{
    __shared__ double sm[4][32];
    const int tgt = threadIdx.x & 31, m = threadIdx.x >> 5;
    const int64_t i = blockIdx.x * 32LL + tgt;
    double s = 0.0;
    if (i < N) {
        const int64_t g = i / PB_TG;
        const int nsP = itemP_off[g + 1] - itemP_off[g];
        const int nsM = itemM_off ? itemM_off[g + 1] - itemM_off[g] : 0;
        for (int q = 0; q < nsP; ++q) s += accP[((int64_t)q * 4 + m) * N + i];
        for (int q = 0; q < nsM; ++q) s += accM[((int64_t)q * 4 + m) * N + i];
        s *= PB_INV4PI;
        const double* __restrict__ xv = (m & 1) ? xphi : xdphi;     // V_L, V_Y act on dphi; K_L, K_Y on phi
        const double* __restrict__ val = nr_val + (int64_t)m * ne;
        for (int32_t e = nr_off[i]; e < nr_off[i + 1]; ++e) s = fma(val[e], xv[nr_col[e]], s);
    }
    sm[m][tgt] = s;
    __syncthreads();
    if (m == 0 && i < N) {
        const double VL = sm[0][tgt], KL = sm[1][tgt], VY = sm[2][tgt], KY = sm[3][tgt];
        const double phi = xphi[i];
        const int64_t o = perm[i];
        y[o] = 0.5 * phi + KL - VL;                    // Eq. (5), first row
        y[N + o] = 0.5 * phi - KY + eps_ratio * VY;    // Eq. (5), second row
    }
}

// ---- host driver ----------------------------------------------------------------------------------------------
template <int P>
static cudaError_t launch_m2p(pb_ctx* ctx)
{
    pb_tree& t = ctx->tree;
    static bool attr_set = false;   // per instantiation; the attribute belongs to the function, not the context
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(k_m2p<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)m2p_cfg<P>::SMEM);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    k_m2p<P><<<(unsigned)t.n_itemM, M2P_THREADS, m2p_cfg<P>::SMEM, ctx->stream>>>(
        t.N, ctx->prm.kappa, t.ek, t.itemM, t.m2p_cell, t.m2p_ctr, t.FF, t.pc[0], t.pc[1], t.pc[2], t.accM);
    return cudaSuccess;
}

int pb_matvec_impl(pb_ctx* ctx, const double* x, double* y, bool timed)
{
    pb_tree& t = ctx->tree;
    cudaStream_t st = ctx->stream;
    if (!t.built) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_matvec: call pb_tree_build first");
    if (!x || !y || x == y) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_matvec: x and y must be distinct non-NULL device arrays");
    if (timed && !ctx->ev_made) {
        for (int k = 0; k < 8; ++k) PB_CUDA(cudaEventCreate(&ctx->ev[k]));
        ctx->ev_made = true;
    }
    const bool far = ctx->prm.theta > 0.0;
    if (timed) PB_CUDA(cudaEventRecord(ctx->ev[0], st));
    PB_TRY(pb_weights(ctx, x));
    if (timed) PB_CUDA(cudaEventRecord(ctx->ev[1], st));
    if (far) {
        if (t.n_need_leaf > 0) {
            k_p2m_leaf<<<(unsigned)t.n_need_leaf, t.Nk <= 96 ? 96 : 128, 0, st>>>(t.P, t.Nk, t.K, t.need_leaf, t.c_first, t.c_last, t.c_ctr[0],
                                                               t.c_ctr[1], t.c_ctr[2], t.srec, t.M);
            PB_LAUNCH_CHECK();
        }
        for (int g = (int)t.m2m_start.size() - 2; g >= 0; --g) {   // deepest generation first
            const int64_t n = t.m2m_start[g + 1] - t.m2m_start[g];
            if (n == 0) continue;
            k_m2m<<<(unsigned)n, t.Nk <= 96 ? 96 : 128, (size_t)(16 * t.Nk + 24 * (PB_MAX_P + 1)) * sizeof(double), st>>>(t.m2m_cells + t.m2m_start[g], t.P, t.Nk, t.c_child, t.c_nchild, t.c_ctr[0],
                                               t.c_ctr[1], t.c_ctr[2], t.mm_off, t.mm_ent, t.mm_coef, t.M);
            PB_LAUNCH_CHECK();
        }
        if (t.n_used > 0) {
            k_convert<<<pb_blocks(t.n_used * t.NT, 256), 256, 0, st>>>(t.n_used, t.used_cells, t.Nk, t.NT, t.cv_off, t.cv_idx,
                                                                      t.cv_coef, t.M, t.FF);
            PB_LAUNCH_CHECK();
        }
    }
    if (timed) PB_CUDA(cudaEventRecord(ctx->ev[2], st));
    if (far && t.n_itemM > 0) {
        PB_TRY(pb_prof_begin(ctx, 1));
        switch (t.P) {
        case 0: PB_CUDA(launch_m2p<0>(ctx)); break;
        case 1: PB_CUDA(launch_m2p<1>(ctx)); break;
        case 2: PB_CUDA(launch_m2p<2>(ctx)); break;
        case 3: PB_CUDA(launch_m2p<3>(ctx)); break;
        case 4: PB_CUDA(launch_m2p<4>(ctx)); break;
        case 5: PB_CUDA(launch_m2p<5>(ctx)); break;
        case 6: PB_CUDA(launch_m2p<6>(ctx)); break;
        case 7: PB_CUDA(launch_m2p<7>(ctx)); break;
        case 8: PB_CUDA(launch_m2p<8>(ctx)); break;
        case 9: PB_CUDA(launch_m2p<9>(ctx)); break;
        case 10: PB_CUDA(launch_m2p<10>(ctx)); break;
        default: return pb_fail(ctx, PB_ERR_INVALID_ARG, "unsupported order_P %d", t.P);
        }
        PB_LAUNCH_CHECK();
        PB_TRY(pb_prof_end(ctx, 1));
    }
    if (timed) PB_CUDA(cudaEventRecord(ctx->ev[3], st));
    {
        PB_TRY(pb_prof_begin(ctx, 0));
        k_p2p<<<(unsigned)t.n_itemP, P2P_THREADS, 0, st>>>(t.N, t.K, ctx->prm.kappa, t.ek, t.itemP, t.p2p_lo, t.p2p_hi, t.srec,
                                                         t.pc[0], t.pc[1], t.pc[2], t.accP);
        PB_LAUNCH_CHECK();
        PB_TRY(pb_prof_end(ctx, 0));
        pb_prof_next(ctx);
    }
    if (timed) PB_CUDA(cudaEventRecord(ctx->ev[4], st));
    k_combine<<<pb_blocks(t.N, 32), 128, 0, st>>>(t.N, t.itemP_off, far ? t.itemM_off : nullptr,
                                                  ctx->prm.eps_in / ctx->prm.eps_out, t.accP, t.accM, t.nr_off,
                                                  t.nr_col, t.nr_val, t.near_entries, t.xphi, t.xdphi, t.perm, y);
    PB_LAUNCH_CHECK();
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
    return pb_matvec_impl(ctx, x, y, false);
}

extern "C" int pb_matvec_timed(pb_ctx* ctx, const double* x, double* y)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    return pb_matvec_impl(ctx, x, y, true);
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
    PB_TRY(pb_matvec_impl(ctx, dx, dy, false));
    PB_CUDA(cudaMemcpyAsync(y_host, dy, n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    PB_CUDA(cudaStreamSynchronize(ctx->stream));
    return PB_OK;
}
