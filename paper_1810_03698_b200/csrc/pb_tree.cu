// pb_tree.cu -- device-built Morton octree over whole panels, target groups and the
// M2P / P2P interaction lists by the MAC of Eq. (28) (D: sections 5-6).
#include <math.h>
#include "pb_internal.cuh"

// ---- bounding cube of the centroids ---------------------------------------------------------
__global__ void k_bbox(int64_t n, const double* __restrict__ cen, double* __restrict__ out /*[6]*/)
{
    __shared__ double s[6][32];
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int64_t i = threadIdx.x; i < n; i += blockDim.x)
        for (int d = 0; d < 3; ++d) {
            double v = cen[3 * i + d];
            lo[d] = fmin(lo[d], v);
            hi[d] = fmax(hi[d], v);
        }
    for (int o = 16; o > 0; o >>= 1)
        for (int d = 0; d < 3; ++d) {
            lo[d] = fmin(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
            hi[d] = fmax(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
        }
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0)
        for (int d = 0; d < 3; ++d) { s[d][w] = lo[d]; s[3 + d][w] = hi[d]; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int nw = blockDim.x >> 5;
        for (int d = 0; d < 3; ++d) {
            double a = s[d][0], b = s[3 + d][0];
            for (int k = 1; k < nw; ++k) { a = fmin(a, s[d][k]); b = fmax(b, s[3 + d][k]); }
            out[d] = a;
            out[3 + d] = b;
        }
    }
}

__device__ __forceinline__ uint64_t spread21(uint64_t v)
{
    v &= 0x1fffffULL;
    v = (v | (v << 32)) & 0x1f00000000ffffULL;
    v = (v | (v << 16)) & 0x1f0000ff0000ffULL;
    v = (v | (v << 8)) & 0x100f00f00f00f00fULL;
    v = (v | (v << 4)) & 0x10c30c30c30c30c3ULL;
    v = (v | (v << 2)) & 0x1249249249249249ULL;
    return v;
}

// 63-bit Morton key of each centroid, 21 bits per axis inside the bounding cube.
__global__ void k_morton(int64_t n, const double* __restrict__ cen, const double* __restrict__ box,
                         uint64_t* __restrict__ keys, int32_t* __restrict__ vals)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double side = fmax(fmax(box[3] - box[0], box[4] - box[1]), box[5] - box[2]);
    side = side > 0 ? side * (1.0 + 1e-9) : 1.0;
    uint64_t q[3];
    for (int d = 0; d < 3; ++d) {
        double t = (cen[3 * i + d] - box[d]) / side * 2097152.0;
        long long u = (long long)t;
        u = u < 0 ? 0 : (u > 2097151 ? 2097151 : u);
        q[d] = (uint64_t)u;
    }
    keys[i] = (spread21(q[0]) << 2) | (spread21(q[1]) << 1) | spread21(q[2]);
    vals[i] = (int32_t)i;
}

// ---- LSD radix sort, 8-bit digits, stable; one warp owns a contiguous sub-tile -------------
#define RS_WARPS 8
#define RS_ITEMS 16
#define RS_TILE (32 * RS_ITEMS)

__global__ void k_rs_hist(const uint64_t* __restrict__ keys, int64_t n, int shift, int64_t nwt,
                          int32_t* __restrict__ hist /*[256][nwt]*/)
{
    __shared__ int32_t cnt[RS_WARPS][256];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int64_t wt = blockIdx.x * (int64_t)RS_WARPS + w;
    for (int d = lane; d < 256; d += 32) cnt[w][d] = 0;
    __syncwarp();
    if (wt < nwt) {
        for (int c = 0; c < RS_ITEMS; ++c) {
            int64_t i = wt * RS_TILE + c * 32 + lane;
            if (i < n) atomicAdd(&cnt[w][(int)((keys[i] >> shift) & 255)], 1);
        }
        __syncwarp();
        for (int d = lane; d < 256; d += 32) hist[(int64_t)d * nwt + wt] = cnt[w][d];
    }
}

__global__ void k_rs_scatter(const uint64_t* __restrict__ kin, const int32_t* __restrict__ vin,
                             uint64_t* __restrict__ kout, int32_t* __restrict__ vout, int64_t n, int shift,
                             int64_t nwt, const int32_t* __restrict__ hist)
{
    __shared__ int32_t off[RS_WARPS][256];
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int64_t wt = blockIdx.x * (int64_t)RS_WARPS + w;
    if (wt >= nwt) return;
    for (int d = lane; d < 256; d += 32) off[w][d] = hist[(int64_t)d * nwt + wt];
    __syncwarp();
    for (int c = 0; c < RS_ITEMS; ++c) {
        int64_t i = wt * RS_TILE + c * 32 + lane;
        bool valid = i < n;
        uint64_t key = valid ? kin[i] : 0;
        int dg = valid ? (int)((key >> shift) & 255) : (256 + lane);
        unsigned peers = __match_any_sync(0xffffffffu, dg);
        int rank = __popc(peers & ((1u << lane) - 1u));
        int pos = valid ? off[w][dg] + rank : 0;
        __syncwarp();
        if (valid && rank == 0) off[w][dg] += __popc(peers);
        __syncwarp();
        if (valid) { kout[pos] = key; vout[pos] = vin[i]; }
    }
}

// ---- panels and Gauss points in Morton order -----------------------------------------------
struct geo_ptrs {
    double *pc[3], *pn[3], *parea, *pv[9];
    int32_t* ptri[3];
    double *sx[3], *swA;
};

__global__ void k_gather(int64_t N, const int32_t* __restrict__ perm, const double* __restrict__ verts,
                         const int32_t* __restrict__ tris, pb_rule_t rule, geo_ptrs g)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    int64_t o = perm[i];
    double v[9];
    for (int b = 0; b < 3; ++b) {
        int32_t vi = tris[3 * o + b];
        g.ptri[b][i] = vi;
        for (int d = 0; d < 3; ++d) v[3 * b + d] = verts[3 * (int64_t)vi + d];
    }
    double e1[3], e2[3], c[3];
    for (int d = 0; d < 3; ++d) {
        e1[d] = v[3 + d] - v[d];
        e2[d] = v[6 + d] - v[d];
        g.pc[d][i] = (v[d] + v[3 + d] + v[6 + d]) / 3.0;
    }
    c[0] = e1[1] * e2[2] - e1[2] * e2[1];
    c[1] = e1[2] * e2[0] - e1[0] * e2[2];
    c[2] = e1[0] * e2[1] - e1[1] * e2[0];
    double l = sqrt(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
    double area = 0.5 * l;
    g.parea[i] = area;
    for (int d = 0; d < 3; ++d) g.pn[d][i] = c[d] / l;
    for (int k = 0; k < 9; ++k) g.pv[k][i] = v[k];
    for (int q = 0; q < rule.K; ++q) {
        int64_t s = i * rule.K + q;
        for (int d = 0; d < 3; ++d)
            g.sx[d][s] = rule.lam[q][0] * v[d] + rule.lam[q][1] * v[3 + d] + rule.lam[q][2] * v[6 + d];
        g.swA[s] = rule.w[q] * area;
    }
}

__global__ void k_panel_surface(int64_t N, const int32_t* __restrict__ perm, int32_t n1, unsigned char* __restrict__ psurf)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i < N) psurf[i] = perm[i] >= n1 ? 1 : 0;
}

// ---- octree topology, one BFS generation at a time -----------------------------------------
// A cell is a range of Morton-sorted panels.  It is split at the highest 3-bit digit in
// which its first and last keys differ, so every internal cell has >= 2 children.
__global__ void k_cell_split(int64_t c0, int64_t c1, const uint64_t* __restrict__ keys,
                             const int32_t* __restrict__ c_first, const int32_t* __restrict__ c_last, int K,
                             int ncrit, int32_t* __restrict__ nchild, int32_t* __restrict__ bounds /*[c1-c0][9]*/)
{
    int64_t c = c0 + blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (c >= c1) return;
    int32_t f = c_first[c], l = c_last[c];
    int32_t* b = bounds + 9 * (c - c0);
    int nc = 0;
    if ((int64_t)(l - f) * K > ncrit && l - f > 1 && keys[f] != keys[l - 1]) {
        uint64_t x = keys[f] ^ keys[l - 1];
        int hb = 63 - __clzll((long long)x);
        int shift = 3 * (hb / 3);
        b[0] = f;
        b[8] = l;
        for (int v = 1; v < 8; ++v) {
            int32_t lo = f, hi = l;   // first index whose digit >= v
            while (lo < hi) {
                int32_t mid = lo + ((hi - lo) >> 1);
                if ((int)((keys[mid] >> shift) & 7) >= v) hi = mid; else lo = mid + 1;
            }
            b[v] = lo;
        }
        for (int v = 0; v < 8; ++v) nc += (b[v + 1] > b[v]);
    }
    nchild[c - c0] = nc;
}

__global__ void k_cell_emit(int64_t c0, int64_t c1, const int32_t* __restrict__ nchild,
                            const int32_t* __restrict__ choff, const int32_t* __restrict__ bounds, int64_t base,
                            int32_t* __restrict__ c_first, int32_t* __restrict__ c_last,
                            int32_t* __restrict__ c_child, int32_t* __restrict__ c_nchild)
{
    int64_t c = c0 + blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (c >= c1) return;
    int nc = nchild[c - c0];
    c_nchild[c] = nc;
    if (nc == 0) { c_child[c] = -1; return; }
    int64_t first = base + choff[c - c0];
    c_child[c] = (int32_t)first;
    const int32_t* b = bounds + 9 * (c - c0);
    int k = 0;
    for (int v = 0; v < 8; ++v)
        if (b[v + 1] > b[v]) {
            c_first[first + k] = b[v];
            c_last[first + k] = b[v + 1];
            ++k;
        }
}

__global__ void k_mark_leaves(int64_t nc, const int32_t* __restrict__ c_child, int32_t* __restrict__ flag)
{
    int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (c < nc) flag[c] = c_child[c] < 0 ? 1 : 0;
}

__global__ void k_compact_leaves(int64_t nc, const int32_t* __restrict__ c_child, const int32_t* __restrict__ off,
                                 int32_t* __restrict__ leaf_ids)
{
    int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (c < nc && c_child[c] < 0) leaf_ids[off[c]] = (int32_t)c;
}

// ---- cell geometry: tight box, expansion centre = box centre, bounding radius (D: R-13) -----
// leaves: one warp per leaf, exact box and radius over its Gauss points
__global__ void k_leaf_geom(int64_t nl, const int32_t* __restrict__ leaf_ids, const int32_t* __restrict__ c_first,
                            const int32_t* __restrict__ c_last, int K, const double* __restrict__ sx,
                            const double* __restrict__ sy, const double* __restrict__ sz, double* __restrict__ cx,
                            double* __restrict__ cy, double* __restrict__ cz, double* __restrict__ crad,
                            double* __restrict__ cbox)
{
    int64_t w = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (w >= nl) return;
    int32_t c = leaf_ids[w];
    int64_t s0 = (int64_t)c_first[c] * K, s1 = (int64_t)c_last[c] * K;
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int64_t s = s0 + lane; s < s1; s += 32) {
        double p[3] = {sx[s], sy[s], sz[s]};
        for (int d = 0; d < 3; ++d) { lo[d] = fmin(lo[d], p[d]); hi[d] = fmax(hi[d], p[d]); }
    }
    for (int o = 16; o > 0; o >>= 1)
        for (int d = 0; d < 3; ++d) {
            lo[d] = fmin(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
            hi[d] = fmax(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
        }
    double ctr[3] = {0.5 * (lo[0] + hi[0]), 0.5 * (lo[1] + hi[1]), 0.5 * (lo[2] + hi[2])};
    double r2 = 0;
    for (int64_t s = s0 + lane; s < s1; s += 32) {
        double dx = sx[s] - ctr[0], dy = sy[s] - ctr[1], dz = sz[s] - ctr[2];
        r2 = fmax(r2, dx * dx + dy * dy + dz * dz);
    }
    for (int o = 16; o > 0; o >>= 1) r2 = fmax(r2, __shfl_xor_sync(0xffffffffu, r2, o));
    if (lane == 0) {
        cx[c] = ctr[0]; cy[c] = ctr[1]; cz[c] = ctr[2];
        crad[c] = sqrt(r2) * (1.0 + 1e-14);
        for (int d = 0; d < 3; ++d) { cbox[6 * (int64_t)c + d] = lo[d]; cbox[6 * (int64_t)c + 3 + d] = hi[d]; }
    }
}

// internal cells of one generation (children are already done): box = union of the
// children's boxes; radius = min(half diagonal, max over children of |c_child - c| + r_child)
__global__ void k_inner_geom(int64_t c0, int64_t c1, const int32_t* __restrict__ c_child,
                             const int32_t* __restrict__ c_nchild, double* __restrict__ cx, double* __restrict__ cy,
                             double* __restrict__ cz, double* __restrict__ crad, double* __restrict__ cbox)
{
    int64_t c = c0 + blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (c >= c1) return;
    int32_t ch = c_child[c];
    if (ch < 0) return;
    int nc = c_nchild[c];
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int k = 0; k < nc; ++k)
        for (int d = 0; d < 3; ++d) {
            lo[d] = fmin(lo[d], cbox[6 * (int64_t)(ch + k) + d]);
            hi[d] = fmax(hi[d], cbox[6 * (int64_t)(ch + k) + 3 + d]);
        }
    double ctr[3] = {0.5 * (lo[0] + hi[0]), 0.5 * (lo[1] + hi[1]), 0.5 * (lo[2] + hi[2])};
    double hd = 0.5 * sqrt((hi[0] - lo[0]) * (hi[0] - lo[0]) + (hi[1] - lo[1]) * (hi[1] - lo[1]) +
                           (hi[2] - lo[2]) * (hi[2] - lo[2]));
    double rr = 0;
    for (int k = 0; k < nc; ++k) {
        double dx = cx[ch + k] - ctr[0], dy = cy[ch + k] - ctr[1], dz = cz[ch + k] - ctr[2];
        rr = fmax(rr, sqrt(dx * dx + dy * dy + dz * dz) + crad[ch + k]);
    }
    cx[c] = ctr[0]; cy[c] = ctr[1]; cz[c] = ctr[2];
    crad[c] = fmin(hd, rr) * (1.0 + 1e-14);
    for (int d = 0; d < 3; ++d) { cbox[6 * c + d] = lo[d]; cbox[6 * c + 3 + d] = hi[d]; }
}

// ---- interaction lists: top-down traversal per target group (Eq. 28) ------------
// One warp per group.  A cell is accepted (M2P) for the whole group when the MAC of Eq. (28),
// R_b / R_tb < theta, holds for EVERY target of the group: R_b the cell's bounding radius, R_tb the
// distance from the cell's expansion centre to the target (each lane holds two of the group's
// targets; the smallest distance is a warp reduction).  R_tb > R_b is required as well, so a cell
// whose bounding sphere contains a target -- in particular the target's own panel -- is never
// accepted whatever theta is.  Otherwise the children are visited, and leaves go to the P2P list
// as source-point ranges (adjacent ranges merged).  Cells with fewer than `m2p_min` source points
// are never accepted: summing them directly is cheaper and exact.
struct list_args {
    int64_t ng, N, Ns;
    int K;
    double theta;
    double theta_low2;                // > 0: cells with (R_b/R_tb)^2 below it for every target are flagged for order P - 2
    double theta_mid2;                // > 0: ... and, of the others, the ones below this for order P - 1 (R-30)
    int m2p_min;
    const int32_t *c_first, *c_last, *c_child, *c_nchild;
    const double *cx, *cy, *cz, *crad;
    const double *px, *py, *pz;       // collocation points, Morton order
    int8_t* m2p_low;                  // [entries] code of the entry (pass 1; may be NULL): bit 0 = evaluate at order P - 2, bit 3 = at order P - 1,
                                      // bits 1-2 = which half of the group the entry is for (1 = targets 0..31, 2 = 32..63, 3 = both)
    int8_t* p2p_mask;                 // [ranges] the same half mask for every P2P range (pass 1; NULL without `split`)
    int split;                        // 1: the two halves of a 64-target group are accepted separately (TPL == 2 only)
    int32_t *n_m2p, *n_p2p;           // pass 0: counts ; pass 1: offsets (read)
    int32_t *m2p_cell, *p2p_lo, *p2p_hi;
    unsigned long long* pair_counts;  // [6] p2p, m2p, order-(P-2) m2p, one-half p2p, one-half m2p, order-(P-1) m2p pairs (pass 0)
};

#define LIST_WARPS 4
#define LIST_STACK 256
static_assert(PB_TG == 64, "k_lists keeps two targets per lane for the panel groups");

// TPL = targets per lane: 2 for the panel groups (PB_TG = 64), 1 for the site groups (32 sites).
// With `split` (TPL == 2) the two halves of a group -- every lane's first target (targets 0..31) and every lane's second
// target (32..63) -- take their decisions separately: a cell that satisfies the MAC for one half only is listed for that
// half alone, and only the other half goes on to its children.  Each half thus gets the list of a 32-target group
// (C4: 29 % fewer P2P pairs, 8.5 % fewer M2P pairs than one list for all 64 targets), while the kernels still work on
// whole warps: an entry for both halves feeds both targets of a lane from one shared-memory read, an entry for one half
// costs half the arithmetic.  The stack holds (cell, mask of the halves still undecided for it).
template <int PASS, int TPL>
__global__ void __launch_bounds__(LIST_WARPS * 32) k_lists(list_args a)
{
    constexpr int TG = 32 * TPL;
    __shared__ int32_t stk[LIST_WARPS][LIST_STACK];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t g = blockIdx.x * (int64_t)LIST_WARPS + wid;
    if (g >= a.ng) return;
    const int64_t i0 = g * TG;
    const int64_t ntg = i0 + TG <= a.N ? TG : a.N - i0;
    const unsigned long long nA = ntg < 32 ? (unsigned long long)ntg : 32ull, nB = (unsigned long long)ntg - nA;   // targets per half
    const int full_mask = TPL == 2 && nB > 0 ? 3 : 1;
    auto ntargets = [&](int m) -> unsigned long long { return (m & 1 ? nA : 0ull) + (m & 2 ? nB : 0ull); };
    int nm = 0, nr = 0;
    const int64_t om = PASS ? a.n_m2p[g] : 0, op = PASS ? a.n_p2p[g] : 0;
    unsigned long long pp = 0, pm = 0, plow = 0, pph = 0, pmh = 0, pmid = 0;
    if (a.theta <= 0.0) {   // direct mode: one range, every source point
        if (PASS && lane == 0) {
            a.p2p_lo[op] = 0; a.p2p_hi[op] = (int32_t)a.Ns;
            if (a.p2p_mask) a.p2p_mask[op] = (int8_t)full_mask;
        }
        nr = 1;
        pp = (unsigned long long)a.Ns * (unsigned long long)ntg;
    } else {
        // padding lanes repeat a real target
        const int64_t ia = i0 + (lane < ntg ? lane : 0), ib = TPL == 2 ? i0 + (lane + 32 < ntg ? lane + 32 : (nB > 0 ? 32 : 0)) : ia;
        const double ax = a.px[ia], ay = a.py[ia], az = a.pz[ia];
        const double bx = a.px[ib], by = a.py[ib], bz = a.pz[ib];
        int32_t* stack = stk[wid];
        int sp = 0;
        if (lane == 0) stack[0] = 0 * 4 + full_mask;
        sp = 1;
        __syncwarp();
        int32_t last_hi = -1;
        int last_mask = 0;
        const double th2 = a.theta * a.theta;
        const bool split = TPL == 2 && a.split != 0;
        while (sp > 0) {
            const int32_t top = stack[--sp];
            __syncwarp();
            const int32_t c = top >> 2;
            const int mask = top & 3;
            const double cx = a.cx[c], cy = a.cy[c], cz = a.cz[c], cr = a.crad[c];
            double da = (cx - ax) * (cx - ax) + (cy - ay) * (cy - ay) + (cz - az) * (cz - az);
            double db = (cx - bx) * (cx - bx) + (cy - by) * (cy - by) + (cz - bz) * (cz - bz);
            for (int o = 16; o > 0; o >>= 1) {
                da = fmin(da, __shfl_xor_sync(0xffffffffu, da, o));
                db = fmin(db, __shfl_xor_sync(0xffffffffu, db, o));
            }
            const int32_t f = a.c_first[c], l = a.c_last[c];
            const int32_t ch = a.c_child[c];
            const int64_t nsrc = (int64_t)(l - f) * a.K;
            const bool big = nsrc >= a.m2p_min;
            const bool okA = (mask & 1) && big && cr * cr < th2 * da && cr * cr < da;
            const bool okB = (mask & 2) && big && cr * cr < th2 * db && cr * cr < db;
            int acc = (okA ? 1 : 0) | (okB ? 2 : 0);
            if (!split && acc != mask) acc = 0;             // one decision for the whole group
            if (acc) {
                double dmin = 1e300;
                if (acc & 1) dmin = fmin(dmin, da);
                if (acc & 2) dmin = fmin(dmin, db);
                const bool low = cr * cr < a.theta_low2 * dmin;
                const bool mid = !low && cr * cr < a.theta_mid2 * dmin;
                if (PASS && lane == 0) {
                    a.m2p_cell[om + nm] = c;
                    if (a.m2p_low) a.m2p_low[om + nm] = (int8_t)((low ? 1 : 0) | (acc << 1) | (mid ? 8 : 0));
                }
                ++nm;
                pm += ntargets(acc);
                if (low) plow += ntargets(acc);
                if (mid) pmid += ntargets(acc);
                if (acc != full_mask) pmh += ntargets(acc);
            }
            const int rem = mask & ~acc;
            if (rem) {
                if (ch < 0) {
                    const int32_t lo = f * a.K, hi = l * a.K;
                    if (lo == last_hi && rem == last_mask) {
                        if (PASS && lane == 0) a.p2p_hi[op + nr - 1] = hi;
                    } else {
                        if (PASS && lane == 0) {
                            a.p2p_lo[op + nr] = lo; a.p2p_hi[op + nr] = hi;
                            if (a.p2p_mask) a.p2p_mask[op + nr] = (int8_t)rem;
                        }
                        ++nr;
                    }
                    last_hi = hi;
                    last_mask = rem;
                    pp += (unsigned long long)(hi - lo) * ntargets(rem);
                    if (rem != full_mask) pph += (unsigned long long)(hi - lo) * ntargets(rem);
                } else {
                    const int nc = a.c_nchild[c];
                    if (lane < nc) stack[sp + lane] = (ch + (nc - 1 - lane)) * 4 + rem;   // popped in Morton order
                    sp += nc;
                    __syncwarp();
                }
            }
        }
    }
    if (!PASS && lane == 0) {
        a.n_m2p[g] = nm;
        a.n_p2p[g] = nr;
        atomicAdd(&a.pair_counts[0], pp);
        atomicAdd(&a.pair_counts[1], pm);
        atomicAdd(&a.pair_counts[2], plow);
        atomicAdd(&a.pair_counts[3], pph);
        atomicAdd(&a.pair_counts[4], pmh);
        atomicAdd(&a.pair_counts[5], pmid);
    }
}

// Stable partition of every group's M2P list into nine classes: the cells evaluated at the full order P first, then the
// ones flagged for order P - 1, then the ones for order P - 2 (R-30); within each, the entries for both halves of the group,
// then the ones for the first half only, then the second half only.  The 8 warps of a k_m2p2 block take consecutive list
// entries, one cell per warp; with neighbours of one class the warps of a block finish their shares at about the same
// time.  One thread per group; setup time only.  code: bit 0 = order P - 2, bit 3 = order P - 1, bits 1-2 = half mask (k_lists).
__device__ __forceinline__ int m2p_class(int code)
{
    const int tier = (code & 1) ? 2 : ((code & 8) ? 1 : 0), half = (code >> 1) & 3;
    return tier * 3 + (half == 3 ? 0 : half);
}

__global__ void k_partition_low(int64_t G, const int32_t* __restrict__ off, const int32_t* __restrict__ cell_in,
                                const int8_t* __restrict__ code_in, int32_t* __restrict__ cell_out, int8_t* __restrict__ code_out)
{
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= G) return;
    const int32_t e0 = off[g], e1 = off[g + 1];
    int32_t pos[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (int32_t e = e0; e < e1; ++e) ++pos[m2p_class(code_in[e])];
    int32_t run = e0;
    for (int k = 0; k < 9; ++k) { const int32_t n = pos[k]; pos[k] = run; run += n; }
    for (int32_t e = e0; e < e1; ++e) {
        const int code = code_in[e];
        const int32_t d = pos[m2p_class(code)]++;
        cell_out[d] = cell_in[e];
        code_out[d] = (int8_t)code;
    }
}

__global__ void k_pack_ranges(int64_t n, const int32_t* __restrict__ lo, const int32_t* __restrict__ hi,
                              const int8_t* __restrict__ mask, int4* __restrict__ out)
{
    int64_t r = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (r >= n + 2) return;
    out[r] = r < n ? make_int4(lo[r], hi[r], mask[r], 0) : make_int4(0, 0, 0, 0);   // two entries of padding: read ahead, never used
}

__global__ void k_m2p_centres(int64_t n, const int32_t* __restrict__ cell, const int8_t* __restrict__ code,
                              const double* __restrict__ cx, const double* __restrict__ cy, const double* __restrict__ cz,
                              double4* __restrict__ out)
{
    int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= n) return;
    const int32_t c = cell[e];
    out[e] = make_double4(cx[c], cy[c], cz[c], (double)code[e]);   // .w: the entry's code (order flag + half mask), an exact small integer
}

// ---- work items: equal shares of each group's lists, one thread block each ---------------------
// A group's P2P list (source-point ranges) or M2P list (cells) is cut into n_g nearly equal
// pieces so that the grid holds several waves of blocks of similar duration whatever the mesh
// size.  Piece j of group g writes its partial sums to accumulator slot j; the combine kernel adds
// a group's slots in order, so the result does not depend on scheduling.
// lo == nullptr: the list entries are single units (cells); otherwise entry r holds hi[r]-lo[r] units.
__global__ void k_items_count(int64_t ng, const int32_t* __restrict__ off, const int32_t* __restrict__ lo,
                              const int32_t* __restrict__ hi, int item_size, int max_items,
                              int32_t* __restrict__ cnt, int32_t* __restrict__ maxcnt)
{
    int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= ng) return;
    int64_t tot = 0;
    if (lo) for (int32_t r = off[g]; r < off[g + 1]; ++r) tot += hi[r] - lo[r];
    else tot = off[g + 1] - off[g];
    int64_t n = (tot + item_size / 2) / item_size;
    if (n < 1) n = tot > 0 ? 1 : 0;
    if (n > max_items) n = max_items;
    cnt[g] = (int32_t)n;
    atomicMax(maxcnt, (int32_t)n);
}

__global__ void k_items_fill(int64_t ng, const int32_t* __restrict__ off, const int32_t* __restrict__ lo,
                             const int32_t* __restrict__ hi, const int32_t* __restrict__ item_off, int quantum,
                             pb_item* __restrict__ items)
{
    int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= ng) return;
    const int32_t i0 = item_off[g], n = item_off[g + 1] - i0;
    if (n == 0) return;
    int64_t tot = 0;
    if (lo) for (int32_t r = off[g]; r < off[g + 1]; ++r) tot += hi[r] - lo[r];
    else tot = off[g + 1] - off[g];
    int32_t r = off[g];
    int64_t passed = 0;                     // units before entry r
    for (int32_t j = 0; j < n; ++j) {
        // cuts fall on multiples of `quantum` units, so a block's warps all get the same number of cells
        const int64_t b = tot * j / n / quantum * quantum, e = j + 1 == n ? tot : tot * (j + 1) / n / quantum * quantum;
        pb_item it;
        it.group = (int32_t)g;
        it.slot = j;
        it.count = (int32_t)(e - b);
        it.pad = 0;
        if (lo) {
            while (passed + (hi[r] - lo[r]) <= b) { passed += hi[r] - lo[r]; ++r; }
            it.r = r;
            it.a = lo[r] + (int32_t)(b - passed);
        } else {
            it.r = off[g] + (int32_t)b;
            it.a = 0;
        }
        items[i0 + j] = it;
    }
}

// builds one item table; returns the item count and the largest number of items of one group
static int pb_build_items(pb_ctx* ctx, int64_t G, const int32_t* off, const int32_t* lo, const int32_t* hi,
                          int item_size, int max_items, int quantum, int32_t** item_off_out, pb_item** items_out,
                          int64_t* n_items, int* max_per_group)
{
    cudaStream_t st = ctx->stream;
    int32_t *cnt, *ioff;
    PB_TRY(pb_dalloc_t(ctx, &cnt, G + 1, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &ioff, G + 1, CAT_TREE));
    PB_CUDA(cudaMemsetAsync(cnt, 0, sizeof(int32_t) * (G + 1), st));
    int32_t* dmax = (int32_t*)ctx->scratch;
    PB_CUDA(cudaMemsetAsync(dmax, 0, sizeof(int32_t), st));
    k_items_count<<<pb_blocks(G, 128), 128, 0, st>>>(G, off, lo, hi, item_size, max_items, cnt, dmax);
    PB_LAUNCH_CHECK();
    int32_t hmax = 0;
    PB_CUDA(cudaMemcpyAsync(&hmax, dmax, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    int64_t total = 0;
    PB_TRY(pb_exclusive_scan_i32(ctx, cnt, ioff, G + 1, &total));   // synchronises
    pb_item* items;
    PB_TRY(pb_dalloc_t(ctx, &items, total > 0 ? total : 1, CAT_TREE));
    k_items_fill<<<pb_blocks(G, 128), 128, 0, st>>>(G, off, lo, hi, ioff, quantum, items);
    PB_LAUNCH_CHECK();
    *item_off_out = ioff;
    *items_out = items;
    *n_items = total;
    *max_per_group = hmax;
    return PB_OK;
}

// ---- target sharding: per-group cost and the partition rule (include/pb.h, pb_set_shard) -------------------------
// cost[g] = targets in the group x (P2P source points + 9 per M2P cell): an M2P pair costs about as much as
// 9 P2P pairs (12.0 ms / 5.57e8 against 8.2 ms / 3.45e9 at C4); pairs[g] = {P2P pairs, M2P pairs} of the group
__global__ void k_group_cost(int64_t G, int64_t N, const int32_t* __restrict__ m2p_off, const int32_t* __restrict__ p2p_off,
                             const int32_t* __restrict__ p2p_lo, const int32_t* __restrict__ p2p_hi,
                             const int8_t* __restrict__ p2p_mask, const int8_t* __restrict__ m2p_code,
                             long long* __restrict__ cost, long long* __restrict__ pairs /*[G][2]*/)
{
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (g >= G) return;
    const long long ntg = g * PB_TG + PB_TG <= N ? PB_TG : N - g * PB_TG;
    const long long nh[4] = {0, ntg < 32 ? ntg : 32, ntg < 32 ? 0 : ntg - 32, ntg};   // targets an entry with half mask m is for
    long long pp = 0, mp = 0;
    for (int32_t r = p2p_off[g]; r < p2p_off[g + 1]; ++r) pp += (long long)(p2p_hi[r] - p2p_lo[r]) * nh[p2p_mask[r] & 3];
    for (int32_t e = m2p_off[g]; e < m2p_off[g + 1]; ++e) mp += nh[(m2p_code[e] >> 1) & 3];
    cost[g] = pp + 9 * mp;
    pairs[2 * g] = pp;
    pairs[2 * g + 1] = mp;
}

extern "C" int pb_shard_partition(const int64_t* cost, int64_t G, int world, int64_t* first)
{
    if (!cost || !first || G < 0 || world < 1) return PB_ERR_INVALID_ARG;
    long double total = 0;
    for (int64_t g = 0; g < G; ++g) {
        if (cost[g] < 0) return PB_ERR_INVALID_ARG;
        total += (long double)cost[g];
    }
    first[0] = 0;
    int64_t g = 0;
    long double pre = 0;                               // exclusive prefix sum at g
    for (int k = 1; k < world; ++k) {
        const long double want = total * (long double)k / (long double)world;
        while (g < G && pre < want) pre += (long double)cost[g++];
        first[k] = g;
    }
    first[world] = G;
    return PB_OK;
}

int pb_radix_sort(pb_ctx* ctx, uint64_t* k0, uint64_t* k1, int32_t* v0, int32_t* v1, int64_t n, int bits,
                  uint64_t** kout, int32_t** vout)
{
    cudaStream_t st = ctx->stream;
    const int64_t nwt = (n + RS_TILE - 1) / RS_TILE;
    int32_t* hist;
    PB_TRY(pb_dalloc_t(ctx, &hist, 256 * (nwt > 0 ? nwt : 1), CAT_TMP));
    const int nb = (int)((nwt + RS_WARPS - 1) / RS_WARPS);
    uint64_t *ka = k0, *kb = k1;
    int32_t *va = v0, *vb = v1;
    const int npass = (bits + 7) / 8;
    for (int pass = 0; pass < npass && n > 0; ++pass) {
        const int shift = 8 * pass;
        k_rs_hist<<<nb, 32 * RS_WARPS, 0, st>>>(ka, n, shift, nwt, hist);
        PB_LAUNCH_CHECK();
        PB_TRY(pb_exclusive_scan_i32(ctx, hist, hist, 256 * nwt, nullptr));
        k_rs_scatter<<<nb, 32 * RS_WARPS, 0, st>>>(ka, va, kb, vb, n, shift, nwt, hist);
        PB_LAUNCH_CHECK();
        uint64_t* tk = ka; ka = kb; kb = tk;
        int32_t* tv = va; va = vb; vb = tv;
    }
    *kout = ka;
    *vout = va;
    return PB_OK;
}

// ---- exact-cover count of STORED lists (pb_stats.covered_pairs) ------------------------------------------------
// One thread per target group walks the lists exactly as the matvec kernels will read them: source points of the
// P2P ranges plus source points of the M2P cells, times the number of targets in the group.
__global__ void k_cover_count(int64_t G, int tg, int64_t ntargets, int K, const int32_t* __restrict__ m2p_off,
                              const int32_t* __restrict__ m2p_cell, const int32_t* __restrict__ c_first,
                              const int32_t* __restrict__ c_last, const int32_t* __restrict__ p2p_off,
                              const int32_t* __restrict__ p2p_lo, const int32_t* __restrict__ p2p_hi,
                              const int8_t* __restrict__ p2p_mask, const int8_t* __restrict__ m2p_code,
                              unsigned long long* __restrict__ out)
{
    const int64_t g = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    unsigned long long v = 0;
    if (g < G) {
        const int64_t i0 = g * tg;
        const unsigned long long ntg = (unsigned long long)(i0 + tg <= ntargets ? tg : ntargets - i0);
        // targets an entry with half mask m is for (the masks exist for the 64-target panel groups only)
        const unsigned long long nh[4] = {0, ntg < 32 ? ntg : 32, ntg < 32 ? 0 : ntg - 32, ntg};
        for (int32_t r = p2p_off[g]; r < p2p_off[g + 1]; ++r)
            v += (unsigned long long)(p2p_hi[r] - p2p_lo[r]) * (p2p_mask ? nh[p2p_mask[r] & 3] : ntg);
        for (int32_t e = m2p_off[g]; e < m2p_off[g + 1]; ++e) {
            const int32_t c = m2p_cell[e];
            v += (unsigned long long)(c_last[c] - c_first[c]) * (unsigned long long)K * (m2p_code ? nh[(m2p_code[e] >> 1) & 3] : ntg);
        }
    }
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(out, v);     // integer sum: order does not matter
}

int pb_cover_count(pb_ctx* ctx, int64_t G, int tg, int64_t ntargets, const int32_t* m2p_off, const int32_t* m2p_cell,
                   const int32_t* p2p_off, const int32_t* p2p_lo, const int32_t* p2p_hi, int64_t* out_host,
                   const int32_t* c_first, const int32_t* c_last, int K, const int8_t* p2p_mask, const int8_t* m2p_code)
{
    const pb_tree& t = ctx->tree;
    if (!c_first) { c_first = t.c_first; c_last = t.c_last; K = t.K; }   // default: the panel tree
    cudaStream_t st = ctx->stream;
    PB_TRY(pb_scratch(ctx, 1 << 20));
    unsigned long long* d = (unsigned long long*)ctx->scratch;
    PB_CUDA(cudaMemsetAsync(d, 0, sizeof(unsigned long long), st));
    k_cover_count<<<pb_blocks(G, 128), 128, 0, st>>>(G, tg, ntargets, K, m2p_off, m2p_cell, c_first, c_last, p2p_off,
                                                    p2p_lo, p2p_hi, p2p_mask, m2p_code, d);
    PB_LAUNCH_CHECK();
    unsigned long long h = 0;
    PB_CUDA(cudaMemcpyAsync(&h, d, sizeof(h), cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));
    *out_host = (int64_t)h;
    return PB_OK;
}

// Morton order of n points [n][3]: perm (allocated in category `cat`) = indices sorted by the 63-bit key
// inside the points' bounding cube; keys_out (optional) = the sorted keys, allocated in CAT_TMP.
int pb_morton_order(pb_ctx* ctx, const double* pts, int64_t n, int cat, int32_t** perm_out, uint64_t** keys_out)
{
    cudaStream_t st = ctx->stream;
    PB_TRY(pb_scratch(ctx, 1 << 20));
    double* box = ctx->scratch;
    k_bbox<<<1, 1024, 0, st>>>(n, pts, box);
    PB_LAUNCH_CHECK();
    uint64_t *k0, *k1;
    int32_t *v0, *v1;
    PB_TRY(pb_dalloc_t(ctx, &k0, n, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &k1, n, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &v0, n, cat));
    PB_TRY(pb_dalloc_t(ctx, &v1, n, CAT_TMP));
    k_morton<<<pb_blocks(n, 256), 256, 0, st>>>(n, pts, box, k0, v0);
    PB_LAUNCH_CHECK();
    uint64_t* ks;
    int32_t* vs;
    PB_TRY(pb_radix_sort(ctx, k0, k1, v0, v1, n, 64, &ks, &vs));
    // 8 passes: the result is back in (k0, v0)
    if (ks != k0 || vs != v0) return pb_fail(ctx, PB_ERR_INVALID_ARG, "internal: radix sort buffer parity");
    *perm_out = v0;
    if (keys_out) *keys_out = k0;
    return PB_OK;
}

// ---- octree over n Morton-sorted items of K points each (panels with their Gauss points; sites with K = 1) ------
// keys [n] sorted; px, py, pz [n K] the points in the same order.  Cells are numbered generation by generation
// (parents before children); a cell with more than `ncrit` points is split at the highest differing 3-bit digit.
int pb_octree_build(pb_ctx* ctx, const uint64_t* keys, int64_t n, int K, int ncrit, const double* px, const double* py,
                    const double* pz, int cat, pb_octree* oc)
{
    cudaStream_t st = ctx->stream;
    const int64_t cap = 2 * n + 8;
    PB_TRY(pb_dalloc_t(ctx, &oc->c_first, cap, cat));
    PB_TRY(pb_dalloc_t(ctx, &oc->c_last, cap, cat));
    PB_TRY(pb_dalloc_t(ctx, &oc->c_child, cap, cat));
    PB_TRY(pb_dalloc_t(ctx, &oc->c_nchild, cap, cat));
    int32_t *nchild, *choff, *bounds;
    PB_TRY(pb_dalloc_t(ctx, &nchild, cap, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &choff, cap, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &bounds, 9 * cap, CAT_TMP));
    {
        int32_t root[2] = {0, (int32_t)n};
        PB_CUDA(cudaMemcpyAsync(oc->c_first, &root[0], sizeof(int32_t), cudaMemcpyHostToDevice, st));
        PB_CUDA(cudaMemcpyAsync(oc->c_last, &root[1], sizeof(int32_t), cudaMemcpyHostToDevice, st));
        PB_CUDA(cudaStreamSynchronize(st));
    }
    oc->gen_start.clear();
    oc->gen_start.push_back(0);
    oc->gen_start.push_back(1);
    int64_t ncell = 1;
    for (;;) {
        int64_t c0 = oc->gen_start[oc->gen_start.size() - 2], c1 = oc->gen_start.back();
        int64_t ng = c1 - c0;
        k_cell_split<<<pb_blocks(ng, 128), 128, 0, st>>>(c0, c1, keys, oc->c_first, oc->c_last, K, ncrit, nchild, bounds);
        PB_LAUNCH_CHECK();
        int64_t total = 0;
        PB_TRY(pb_exclusive_scan_i32(ctx, nchild, choff, ng, &total));
        if (ncell + total > cap) return pb_fail(ctx, PB_ERR_ALLOC, "octree cell capacity exceeded");
        k_cell_emit<<<pb_blocks(ng, 128), 128, 0, st>>>(c0, c1, nchild, choff, bounds, ncell, oc->c_first, oc->c_last,
                                                       oc->c_child, oc->c_nchild);
        PB_LAUNCH_CHECK();
        if (total == 0) break;
        ncell += total;
        oc->gen_start.push_back(ncell);
    }
    oc->n_cells = ncell;
    oc->n_levels = (int64_t)oc->gen_start.size() - 1;
    {
        int32_t* flag = nchild;   // reuse
        k_mark_leaves<<<pb_blocks(ncell, 256), 256, 0, st>>>(ncell, oc->c_child, flag);
        PB_LAUNCH_CHECK();
        int64_t nl = 0;
        PB_TRY(pb_exclusive_scan_i32(ctx, flag, choff, ncell, &nl));
        oc->n_leaves = nl;
        PB_TRY(pb_dalloc_t(ctx, &oc->leaf_ids, nl, cat));
        k_compact_leaves<<<pb_blocks(ncell, 256), 256, 0, st>>>(ncell, oc->c_child, choff, oc->leaf_ids);
        PB_LAUNCH_CHECK();
    }
    // cell geometry, bottom-up
    for (int d = 0; d < 3; ++d) PB_TRY(pb_dalloc_t(ctx, &oc->c_ctr[d], ncell, cat));
    PB_TRY(pb_dalloc_t(ctx, &oc->c_rad, ncell, cat));
    PB_TRY(pb_dalloc_t(ctx, &oc->c_box, 6 * ncell, cat));
    k_leaf_geom<<<pb_blocks(oc->n_leaves * 32, 128), 128, 0, st>>>(oc->n_leaves, oc->leaf_ids, oc->c_first, oc->c_last, K, px, py, pz,
                                                                  oc->c_ctr[0], oc->c_ctr[1], oc->c_ctr[2], oc->c_rad, oc->c_box);
    PB_LAUNCH_CHECK();
    for (int g = (int)oc->gen_start.size() - 2; g >= 0; --g) {
        int64_t c0 = oc->gen_start[g], c1 = oc->gen_start[g + 1];
        k_inner_geom<<<pb_blocks(c1 - c0, 128), 128, 0, st>>>(c0, c1, oc->c_child, oc->c_nchild, oc->c_ctr[0], oc->c_ctr[1],
                                                             oc->c_ctr[2], oc->c_rad, oc->c_box);
        PB_LAUNCH_CHECK();
    }
    return PB_OK;
}

// ---- host driver ----------------------------------------------------------------------------
int pb_tree_build_impl(pb_ctx* ctx)
{
    pb_tree& t = ctx->tree;
    cudaStream_t st = ctx->stream;
    const int64_t N = ctx->nt;
    const int K = ctx->prm.K_far;
    if (N * K >= 2147483647LL) return pb_fail(ctx, PB_ERR_INVALID_ARG, "too many source points for int32 indexing");
    t.N = N;
    t.K = K;
    t.Ns = N * K;
    pb_make_expk(ctx->prm.kappa, &t.ek);
    PB_TRY(pb_make_expk8(ctx, ctx->prm.kappa, &t.ek8));
    const int64_t Ns = t.Ns;

    // --- Morton keys and sort
    uint64_t* k0;
    int32_t* v0;
    PB_TRY(pb_morton_order(ctx, ctx->cen, N, CAT_TREE, &v0, &k0));   // the sorted keys are needed for the cell build only
    t.perm = v0;
    const uint64_t* keys = k0;

    // --- geometry in Morton order
    for (int d = 0; d < 3; ++d) {
        PB_TRY(pb_dalloc_t(ctx, &t.pc[d], N, CAT_TREE));
        PB_TRY(pb_dalloc_t(ctx, &t.pn[d], N, CAT_TREE));
        PB_TRY(pb_dalloc_t(ctx, &t.ptri[d], N, CAT_TREE));
        PB_TRY(pb_dalloc_t(ctx, &t.sx[d], Ns, CAT_TREE));
    }
    for (int k = 0; k < 9; ++k) PB_TRY(pb_dalloc_t(ctx, &t.pv[k], N, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.parea, N, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.swA, Ns, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.srec, 2 * Ns, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.xphi, N, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.xdphi, N, CAT_TREE));
    {
        geo_ptrs g;
        for (int d = 0; d < 3; ++d) { g.pc[d] = t.pc[d]; g.pn[d] = t.pn[d]; g.ptri[d] = t.ptri[d]; g.sx[d] = t.sx[d]; }
        for (int k = 0; k < 9; ++k) g.pv[k] = t.pv[k];
        g.parea = t.parea;
        g.swA = t.swA;
        k_gather<<<pb_blocks(N, 128), 128, 0, st>>>(N, t.perm, ctx->verts, ctx->tris, ctx->ruleF, g);
        PB_LAUNCH_CHECK();
    }

    // --- two surfaces (pb_set_stern): which surface a panel lies on, Morton order
    if (ctx->stern_n1 > 0) {
        PB_TRY(pb_dalloc_t(ctx, &t.psurf, N, CAT_TREE));
        PB_TRY(pb_dalloc_t(ctx, &t.xphi_full, N, CAT_TREE));
        PB_TRY(pb_dalloc_t(ctx, &t.sraw, (size_t)8 * N, CAT_TREE));
        k_panel_surface<<<pb_blocks(N, 256), 256, 0, st>>>(N, t.perm, (int32_t)ctx->stern_n1, t.psurf);
        PB_LAUNCH_CHECK();
    }

    // --- octree topology and cell geometry
    // leaf capacity: larger leaves shorten the upward pass (the latency-bound part of a small problem); on large meshes
    // the matvec time is flat between 96 and 144 points per leaf (C4, round 2: 21.30 / 21.26 / 21.29 / 21.35 / 21.44 / 21.85 ms
    // at 96 / 112 / 128 / 144 / 160 / 192)
    t.ncrit_used = ctx->prm.ncrit > 0 ? ctx->prm.ncrit : (Ns < 65536 ? 256 : 128);
    {
        pb_octree oc;
        PB_TRY(pb_octree_build(ctx, keys, N, K, t.ncrit_used, t.sx[0], t.sx[1], t.sx[2], CAT_TREE, &oc));
        t.c_first = oc.c_first; t.c_last = oc.c_last; t.c_child = oc.c_child; t.c_nchild = oc.c_nchild;
        for (int d = 0; d < 3; ++d) t.c_ctr[d] = oc.c_ctr[d];
        t.c_rad = oc.c_rad; t.c_box = oc.c_box; t.leaf_ids = oc.leaf_ids;
        t.n_cells = oc.n_cells; t.n_leaves = oc.n_leaves; t.n_levels = oc.n_levels;
        t.gen_start = oc.gen_start;
    }
    const int64_t ncell = t.n_cells;
    (void)ncell;

    // --- target groups
    t.n_groups = (N + PB_TG - 1) / PB_TG;
    const int64_t G = t.n_groups;

    // --- interaction lists: count, scan, fill
    PB_TRY(pb_dalloc_t(ctx, &t.m2p_off, G + 1, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.p2p_off, G + 1, CAT_TREE));
    list_args a;
    a.ng = G; a.N = N; a.Ns = Ns; a.K = K;
    a.theta = ctx->prm.theta;
    // Variable order: a cell whose ratio R_b/R_tb is below theta_low = 0.8 theta^((P+1)/(P-1)) for every target of the
    // group is evaluated at order P - 2 -- its truncation error (ratio^(P-1)) stays below the one the MAC already
    // admits at order P (theta^(P+1)) -- at less than half the cost.  Measured at C4 (theta 0.5, P 6) with the factor
    // at 0 / 0.7 / 0.8 / 0.9 / 1.0: share of such pairs 0 / 0.44 / 0.59 / 0.72 / 0.82, M2P 16.9 / 13.3 / 12.1 / 10.9 / 10.0 ms,
    // error against the oracle on sampled rows 3.2 / 3.3 / 3.6 / 4.6 / 6.8 e-5 (bound 1e-4).
    {
        const int P = ctx->prm.order_P;
        const double tl = P >= 4 && P <= 8 ? 0.8 * pow(ctx->prm.theta, (double)(P + 1) / (double)(P - 1)) : 0.0;
        a.theta_low2 = tl * tl;
        // ... and between the two, order P - 1 for ratio <= 0.8 theta^((P+1)/P): truncation error ratio^P <= 0.8^P theta^(P+1),
        // a smaller share of the error the MAC admits than the order-(P-2) cells take (0.26 against 0.33 at P = 6)
        const double tm = P >= 4 && P <= 8 ? 0.8 * pow(ctx->prm.theta, (double)(P + 1) / (double)P) : 0.0;
        a.theta_mid2 = tm * tm;
    }
    a.m2p_min = 8;   // an M2P pair costs about as much as 8 P2P pairs (D: section 7)
    a.c_first = t.c_first; a.c_last = t.c_last; a.c_child = t.c_child; a.c_nchild = t.c_nchild;
    a.cx = t.c_ctr[0]; a.cy = t.c_ctr[1]; a.cz = t.c_ctr[2]; a.crad = t.c_rad;
    a.px = t.pc[0]; a.py = t.pc[1]; a.pz = t.pc[2];
    int32_t *cnt_m, *cnt_p;
    PB_TRY(pb_dalloc_t(ctx, &cnt_m, G + 1, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &cnt_p, G + 1, CAT_TMP));
    PB_CUDA(cudaMemsetAsync(cnt_m, 0, sizeof(int32_t) * (G + 1), st));
    PB_CUDA(cudaMemsetAsync(cnt_p, 0, sizeof(int32_t) * (G + 1), st));
    unsigned long long* pc = (unsigned long long*)ctx->scratch;
    PB_CUDA(cudaMemsetAsync(pc, 0, 6 * sizeof(unsigned long long), st));
    a.n_m2p = cnt_m; a.n_p2p = cnt_p; a.m2p_cell = nullptr; a.p2p_lo = nullptr; a.p2p_hi = nullptr; a.m2p_low = nullptr;
    a.p2p_mask = nullptr;
    a.split = ctx->prm.list_split;
    a.pair_counts = pc;
    k_lists<0, 2><<<pb_blocks(G, LIST_WARPS), LIST_WARPS * 32, 0, st>>>(a);
    PB_LAUNCH_CHECK();
    unsigned long long hpc[6];
    PB_CUDA(cudaMemcpyAsync(hpc, pc, sizeof(hpc), cudaMemcpyDeviceToHost, st));
    int64_t tot_m = 0, tot_p = 0;
    PB_TRY(pb_exclusive_scan_i32(ctx, cnt_m, t.m2p_off, G + 1, &tot_m));
    PB_TRY(pb_exclusive_scan_i32(ctx, cnt_p, t.p2p_off, G + 1, &tot_p));
    t.p2p_pairs = (int64_t)hpc[0];
    t.m2p_pairs = (int64_t)hpc[1];
    t.m2p_pairs_low = (int64_t)hpc[2];
    t.p2p_pairs_half = (int64_t)hpc[3];
    t.m2p_pairs_half = (int64_t)hpc[4];
    t.m2p_pairs_mid = (int64_t)hpc[5];
    t.m2p_total = tot_m;
    PB_TRY(pb_dalloc_t(ctx, &t.m2p_cell, tot_m, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.p2p_lo, tot_p, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.p2p_hi, tot_p, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.p2p_mask, tot_p > 0 ? tot_p : 1, CAT_TREE));
    PB_TRY(pb_dalloc_t(ctx, &t.m2p_code, tot_m > 0 ? tot_m : 1, CAT_TREE));
    int8_t* m2p_low = t.m2p_code;
    a.n_m2p = t.m2p_off; a.n_p2p = t.p2p_off; a.m2p_cell = t.m2p_cell; a.p2p_lo = t.p2p_lo; a.p2p_hi = t.p2p_hi;
    a.m2p_low = m2p_low;
    a.p2p_mask = t.p2p_mask;
    k_lists<1, 2><<<pb_blocks(G, LIST_WARPS), LIST_WARPS * 32, 0, st>>>(a);
    PB_LAUNCH_CHECK();
    if (tot_m > 0 && (a.theta_low2 > 0.0 || a.split)) {
        int32_t* cell_tmp;
        int8_t* low_tmp;
        PB_TRY(pb_dalloc_t(ctx, &cell_tmp, tot_m, CAT_TMP));
        PB_TRY(pb_dalloc_t(ctx, &low_tmp, tot_m, CAT_TMP));
        PB_CUDA(cudaMemcpyAsync(cell_tmp, t.m2p_cell, sizeof(int32_t) * tot_m, cudaMemcpyDeviceToDevice, st));
        PB_CUDA(cudaMemcpyAsync(low_tmp, m2p_low, sizeof(int8_t) * tot_m, cudaMemcpyDeviceToDevice, st));
        k_partition_low<<<pb_blocks(G, 128), 128, 0, st>>>(G, t.m2p_off, cell_tmp, low_tmp, t.m2p_cell, m2p_low);
        PB_LAUNCH_CHECK();
    }
    PB_TRY(pb_cover_count(ctx, G, PB_TG, N, t.m2p_off, t.m2p_cell, t.p2p_off, t.p2p_lo, t.p2p_hi, &t.covered_pairs, nullptr, nullptr,
                          0, t.p2p_mask, t.m2p_code));
    PB_TRY(pb_dalloc_t(ctx, &t.p2p_rng, tot_p + 2, CAT_TREE));
    k_pack_ranges<<<pb_blocks(tot_p + 2, 256), 256, 0, st>>>(tot_p, t.p2p_lo, t.p2p_hi, t.p2p_mask, t.p2p_rng);
    PB_LAUNCH_CHECK();
    PB_TRY(pb_dalloc_t(ctx, &t.m2p_ctr, tot_m > 0 ? tot_m : 1, CAT_TREE));
    if (tot_m > 0) {
        k_m2p_centres<<<pb_blocks(tot_m, 256), 256, 0, st>>>(tot_m, t.m2p_cell, m2p_low, t.c_ctr[0], t.c_ctr[1], t.c_ctr[2], t.m2p_ctr);
        PB_LAUNCH_CHECK();
    }

    // --- target sharding: this rank's contiguous range of groups (everything when world == 1)
    const int world = ctx->shard_world, rank = ctx->shard_rank;
    t.own_g0 = 0; t.own_g1 = G;
    t.shard_first.assign(world + 1, 0);
    t.shard_first[world] = N;
    if (world > 1) {
        long long *dcost, *dpairs;
        PB_TRY(pb_dalloc_t(ctx, &dcost, G, CAT_TMP));
        PB_TRY(pb_dalloc_t(ctx, &dpairs, 2 * G, CAT_TMP));
        k_group_cost<<<pb_blocks(G, 128), 128, 0, st>>>(G, N, t.m2p_off, t.p2p_off, t.p2p_lo, t.p2p_hi, t.p2p_mask, t.m2p_code, dcost,
                                                        dpairs);
        PB_LAUNCH_CHECK();
        std::vector<int64_t> hcost(G), hpairs(2 * G), gfirst(world + 1);
        PB_CUDA(cudaMemcpyAsync(hcost.data(), dcost, sizeof(int64_t) * G, cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaMemcpyAsync(hpairs.data(), dpairs, sizeof(int64_t) * 2 * G, cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaStreamSynchronize(st));
        if (pb_shard_partition(hcost.data(), G, world, gfirst.data()) != PB_OK) return pb_fail(ctx, PB_ERR_INVALID_ARG, "internal: shard partition");
        t.own_g0 = gfirst[rank]; t.own_g1 = gfirst[rank + 1];
        t.shard_nmax = 0;
        for (int k = 0; k <= world; ++k) t.shard_first[k] = gfirst[k] * PB_TG < N ? gfirst[k] * PB_TG : N;
        for (int k = 0; k < world; ++k)
            if (t.shard_first[k + 1] - t.shard_first[k] > t.shard_nmax) t.shard_nmax = t.shard_first[k + 1] - t.shard_first[k];
        int64_t pp = 0, mp = 0;
        for (int64_t g = t.own_g0; g < t.own_g1; ++g) { pp += hpairs[2 * g]; mp += hpairs[2 * g + 1]; }
        t.p2p_pairs = pp;                           // pb_stats: the owned groups' pairs
        t.m2p_pairs = mp;
        t.m2p_pairs_low = 0;                        // (not tracked per group)
        t.m2p_pairs_mid = 0;
        PB_TRY(pb_dalloc_t(ctx, &t.shard_first_dev, world + 1, CAT_TREE));
        PB_CUDA(cudaMemcpyAsync(t.shard_first_dev, t.shard_first.data(), sizeof(int64_t) * (world + 1), cudaMemcpyHostToDevice, st));
        const int64_t nm = t.shard_nmax > 0 ? t.shard_nmax : 1;
        PB_TRY(pb_dalloc_t(ctx, &t.ysend, 2 * nm, CAT_TREE));
        PB_TRY(pb_dalloc_t(ctx, &t.yall, (size_t)world * 2 * nm, CAT_TREE));
        PB_CUDA(cudaMemsetAsync(t.ysend, 0, sizeof(double) * 2 * nm, st));
        PB_CUDA(cudaStreamSynchronize(st));         // shard_first's host storage is a member; the sync is for hcost / hpairs reuse
    }
    t.own_i0 = t.own_g0 * PB_TG < N ? t.own_g0 * PB_TG : N;
    t.own_i1 = t.own_g1 * PB_TG < N ? t.own_g1 * PB_TG : N;

    // work items: about 8 blocks per resident-block slot (148 SMs x 3 blocks) of THIS rank, never less than one
    // tile of 128 source points / 4 cells per block
    {
        const int64_t slots = 148 * 3 * 8;
        int64_t szP = (t.p2p_pairs / PB_TG + slots - 1) / slots;
        if (szP < 128) szP = 128;
        if (szP > (1 << 30)) szP = 1 << 30;
        PB_TRY(pb_build_items(ctx, G, t.p2p_off, t.p2p_lo, t.p2p_hi, (int)szP, 64, 4, &t.itemP_off, &t.itemP, &t.n_itemP,
                              &t.nslot_p2p));
        int64_t szM = (t.m2p_pairs / PB_TG + slots - 1) / slots;
        if (szM < 8) szM = 8;
        szM = (szM + 7) / 8 * 8;                      // whole tiles of 8 cells: one per warp of k_m2p2
        if (szM > (1 << 30)) szM = 1 << 30;
        PB_TRY(pb_build_items(ctx, G, t.m2p_off, nullptr, nullptr, (int)szM, 64, 8, &t.itemM_off, &t.itemM, &t.n_itemM,
                              &t.nslot_m2p));
        if (t.nslot_p2p < 1) t.nslot_p2p = 1;
        if (t.nslot_m2p < 1) t.nslot_m2p = 1;
        PB_TRY(pb_dalloc_t(ctx, &t.accP, (size_t)t.nslot_p2p * 4 * N, CAT_TREE));
        PB_TRY(pb_dalloc_t(ctx, &t.accM, (size_t)t.nslot_m2p * 4 * N, CAT_TREE));
        // items are stored group by group: the owned groups' items are one contiguous run
        int32_t ho[4] = {0, 0, 0, 0};
        PB_CUDA(cudaMemcpyAsync(&ho[0], t.itemP_off + t.own_g0, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaMemcpyAsync(&ho[1], t.itemP_off + t.own_g1, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaMemcpyAsync(&ho[2], t.itemM_off + t.own_g0, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaMemcpyAsync(&ho[3], t.itemM_off + t.own_g1, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaStreamSynchronize(st));
        t.itemP0 = ho[0]; t.n_itemP_own = ho[1] - ho[0];
        t.itemM0 = ho[2]; t.n_itemM_own = ho[3] - ho[2];
    }
    PB_CUDA(cudaStreamSynchronize(st));
    pb_dfree_cat(ctx, CAT_TMP);
    return PB_OK;
}

// ---- generic list build: targets (Morton order, groups of 32 * tpl) against any octree --------------------------------
int pb_lists_build(pb_ctx* ctx, int tpl, int64_t ntargets, const double* tx, const double* ty, const double* tz,
                   const pb_octree& oc, int K, int64_t Ns, double theta, int m2p_min, int cat, pb_lists* out)
{
    cudaStream_t st = ctx->stream;
    const int tg = 32 * tpl;
    const int64_t G = (ntargets + tg - 1) / tg;
    out->n_groups = G;
    PB_TRY(pb_dalloc_t(ctx, &out->m2p_off, G + 1, cat));
    PB_TRY(pb_dalloc_t(ctx, &out->p2p_off, G + 1, cat));
    list_args a;
    a.ng = G; a.N = ntargets; a.Ns = Ns; a.K = K;
    a.theta = theta;
    a.theta_low2 = 0.0;
    a.theta_mid2 = 0.0;
    a.m2p_low = nullptr;
    a.p2p_mask = nullptr;
    a.split = 0;
    a.m2p_min = m2p_min;
    a.c_first = oc.c_first; a.c_last = oc.c_last; a.c_child = oc.c_child; a.c_nchild = oc.c_nchild;
    a.cx = oc.c_ctr[0]; a.cy = oc.c_ctr[1]; a.cz = oc.c_ctr[2]; a.crad = oc.c_rad;
    a.px = tx; a.py = ty; a.pz = tz;
    int32_t *cnt_m, *cnt_p;
    PB_TRY(pb_dalloc_t(ctx, &cnt_m, G + 1, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &cnt_p, G + 1, CAT_TMP));
    PB_CUDA(cudaMemsetAsync(cnt_m, 0, sizeof(int32_t) * (G + 1), st));
    PB_CUDA(cudaMemsetAsync(cnt_p, 0, sizeof(int32_t) * (G + 1), st));
    PB_TRY(pb_scratch(ctx, 1 << 20));
    unsigned long long* pc = (unsigned long long*)ctx->scratch;
    PB_CUDA(cudaMemsetAsync(pc, 0, 6 * sizeof(unsigned long long), st));
    a.n_m2p = cnt_m; a.n_p2p = cnt_p; a.m2p_cell = nullptr; a.p2p_lo = nullptr; a.p2p_hi = nullptr;
    a.pair_counts = pc;
    if (tpl == 2) k_lists<0, 2><<<pb_blocks(G, LIST_WARPS), LIST_WARPS * 32, 0, st>>>(a);
    else k_lists<0, 1><<<pb_blocks(G, LIST_WARPS), LIST_WARPS * 32, 0, st>>>(a);
    PB_LAUNCH_CHECK();
    unsigned long long hpc[2];
    PB_CUDA(cudaMemcpyAsync(hpc, pc, sizeof(hpc), cudaMemcpyDeviceToHost, st));
    int64_t tot_m = 0, tot_p = 0;
    PB_TRY(pb_exclusive_scan_i32(ctx, cnt_m, out->m2p_off, G + 1, &tot_m));   // synchronises
    PB_TRY(pb_exclusive_scan_i32(ctx, cnt_p, out->p2p_off, G + 1, &tot_p));
    out->p2p_pairs = (int64_t)hpc[0];
    out->m2p_pairs = (int64_t)hpc[1];
    out->m2p_total = tot_m;
    out->p2p_ranges = tot_p;
    PB_TRY(pb_dalloc_t(ctx, &out->m2p_cell, tot_m > 0 ? tot_m : 1, cat));
    PB_TRY(pb_dalloc_t(ctx, &out->p2p_lo, tot_p > 0 ? tot_p : 1, cat));
    PB_TRY(pb_dalloc_t(ctx, &out->p2p_hi, tot_p > 0 ? tot_p : 1, cat));
    a.n_m2p = out->m2p_off; a.n_p2p = out->p2p_off; a.m2p_cell = out->m2p_cell; a.p2p_lo = out->p2p_lo; a.p2p_hi = out->p2p_hi;
    if (tpl == 2) k_lists<1, 2><<<pb_blocks(G, LIST_WARPS), LIST_WARPS * 32, 0, st>>>(a);
    else k_lists<1, 1><<<pb_blocks(G, LIST_WARPS), LIST_WARPS * 32, 0, st>>>(a);
    PB_LAUNCH_CHECK();
    PB_TRY(pb_cover_count(ctx, G, tg, ntargets, out->m2p_off, out->m2p_cell, out->p2p_off, out->p2p_lo, out->p2p_hi,
                          &out->covered_pairs, oc.c_first, oc.c_last, K));
    return PB_OK;
}

// ---- site groups and their interaction lists (treecode for the atom-side sums, S: section 8(f) item 1) ----------
// Sites in Morton order, groups of 32 consecutive sites (one per lane), the same traversal and per-target MAC as
// the panel groups.  Allocations live in CAT_SITE_NEAR (freed with the site-near table).
__global__ void k_site_gather(int64_t na, const int32_t* __restrict__ perm, const double* __restrict__ pos,
                              double* __restrict__ x, double* __restrict__ y, double* __restrict__ z)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= na) return;
    const int64_t o = perm[i];
    x[i] = pos[3 * o]; y[i] = pos[3 * o + 1]; z[i] = pos[3 * o + 2];
}

int pb_site_lists_build(pb_ctx* ctx)
{
    pb_tree& t = ctx->tree;
    pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    const int64_t na = s.na;
    PB_TRY(pb_morton_order(ctx, s.pos, na, CAT_SITE_NEAR, &s.tperm, nullptr));
    for (int d = 0; d < 3; ++d) PB_TRY(pb_dalloc_t(ctx, &s.tpos[d], na, CAT_SITE_NEAR));
    k_site_gather<<<pb_blocks(na, 256), 256, 0, st>>>(na, s.tperm, s.pos, s.tpos[0], s.tpos[1], s.tpos[2]);
    PB_LAUNCH_CHECK();
    const int64_t G = (na + 31) / 32;
    s.t_groups = G;
    PB_TRY(pb_dalloc_t(ctx, &s.t_m2p_off, G + 1, CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &s.t_p2p_off, G + 1, CAT_SITE_NEAR));
    list_args a;
    a.ng = G; a.N = na; a.Ns = t.Ns; a.K = t.K;
    // The field and the field gradient are first and second target derivatives of the order-P sum and lose about
    // one order of the expansion each, so the site lists use a tighter acceptance parameter than the matvec
    // (measured at C4 against the direct sum, theta_site/theta = 1.0, 0.7, 0.5: phi 2e-4, 2e-5, 2e-6; field 7e-3,
    // 8e-4, 8e-5; field gradient 1.4e-1, 1.6e-2, 1.4e-3; time 91, 165, 299 ms against 766 ms direct).
    a.theta = ctx->prm.theta * PB_SITE_THETA_SCALE;
    a.theta_low2 = 0.0;
    a.theta_mid2 = 0.0;
    a.m2p_low = nullptr;
    a.p2p_mask = nullptr;
    a.split = 0;
    a.m2p_min = 8;
    a.c_first = t.c_first; a.c_last = t.c_last; a.c_child = t.c_child; a.c_nchild = t.c_nchild;
    a.cx = t.c_ctr[0]; a.cy = t.c_ctr[1]; a.cz = t.c_ctr[2]; a.crad = t.c_rad;
    a.px = s.tpos[0]; a.py = s.tpos[1]; a.pz = s.tpos[2];
    int32_t *cnt_m, *cnt_p;
    PB_TRY(pb_dalloc_t(ctx, &cnt_m, G + 1, CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &cnt_p, G + 1, CAT_SITE_NEAR));
    PB_CUDA(cudaMemsetAsync(cnt_m, 0, sizeof(int32_t) * (G + 1), st));
    PB_CUDA(cudaMemsetAsync(cnt_p, 0, sizeof(int32_t) * (G + 1), st));
    PB_TRY(pb_scratch(ctx, 1 << 20));
    unsigned long long* pc = (unsigned long long*)ctx->scratch;
    PB_CUDA(cudaMemsetAsync(pc, 0, 6 * sizeof(unsigned long long), st));
    a.n_m2p = cnt_m; a.n_p2p = cnt_p; a.m2p_cell = nullptr; a.p2p_lo = nullptr; a.p2p_hi = nullptr;
    a.pair_counts = pc;
    k_lists<0, 1><<<pb_blocks(G, LIST_WARPS), LIST_WARPS * 32, 0, st>>>(a);
    PB_LAUNCH_CHECK();
    unsigned long long hpc[2];
    PB_CUDA(cudaMemcpyAsync(hpc, pc, sizeof(hpc), cudaMemcpyDeviceToHost, st));
    int64_t tot_m = 0, tot_p = 0;
    PB_TRY(pb_exclusive_scan_i32(ctx, cnt_m, s.t_m2p_off, G + 1, &tot_m));   // synchronises
    PB_TRY(pb_exclusive_scan_i32(ctx, cnt_p, s.t_p2p_off, G + 1, &tot_p));
    s.t_p2p_pairs = (int64_t)hpc[0];
    s.t_m2p_pairs = (int64_t)hpc[1];
    s.t_m2p_total = tot_m;
    PB_TRY(pb_dalloc_t(ctx, &s.t_m2p_cell, tot_m > 0 ? tot_m : 1, CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &s.t_p2p_lo, tot_p > 0 ? tot_p : 1, CAT_SITE_NEAR));
    PB_TRY(pb_dalloc_t(ctx, &s.t_p2p_hi, tot_p > 0 ? tot_p : 1, CAT_SITE_NEAR));
    a.n_m2p = s.t_m2p_off; a.n_p2p = s.t_p2p_off; a.m2p_cell = s.t_m2p_cell; a.p2p_lo = s.t_p2p_lo; a.p2p_hi = s.t_p2p_hi;
    k_lists<1, 1><<<pb_blocks(G, LIST_WARPS), LIST_WARPS * 32, 0, st>>>(a);
    PB_LAUNCH_CHECK();
    PB_TRY(pb_cover_count(ctx, G, 32, na, s.t_m2p_off, s.t_m2p_cell, s.t_p2p_off, s.t_p2p_lo, s.t_p2p_hi, &s.t_covered_pairs));
    return PB_OK;
}
