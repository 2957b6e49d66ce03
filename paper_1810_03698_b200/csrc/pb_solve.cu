// pb_solve.cu -- GMRES on Eq. (5) with device dot products / Arnoldi updates (H9), the
// self-consistent induced-dipole loop with SOR (H13) and the energies of Eq. (19)/(24)
// (H14).  Host code only steers: Givens rotations on the (m+1) x m Hessenberg matrix
// and the convergence tests; every vector operation is a kernel.
#include <math.h>
#include <vector>
#include <cooperative_groups.h>
#include "pb_internal.cuh"
namespace cg = cooperative_groups;

#define DOT_CHUNK 512
#define DOT_THREADS 256
#define DOT_WARPS (DOT_THREADS / 32)
#define DOT_MAXBLK 1184         // 8 blocks per SM: enough loads in flight to stream V at HBM speed

// h[j] = V_j . w for j < nv and, with `self`, h[nv] = w . w.  Block (bx, by) takes the chunks bx,
// bx + gridDim.x, ... of w through shared memory and the vectors by*8R + {warp, warp + 8, ...}; the
// per-block partial sums are added by the LAST block to finish, in a fixed order, so the result does
// not depend on which block that is.  R = 1 spreads a short vector over many blocks (latency), R = 4
// re-reads w less often on long ones (bandwidth).
template <int R>
__global__ void __launch_bounds__(DOT_THREADS)
k_dots(int64_t n, int nv, const double* __restrict__ V, int64_t ld, const double* __restrict__ w, int self,
       double* __restrict__ partial, unsigned int* __restrict__ counter, double* __restrict__ hout)
{
    __shared__ bool last;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int nvt = nv + (self ? 1 : 0);
    const int64_t nchunk = (n + DOT_CHUNK - 1) / DOT_CHUNK;
    const int j0 = blockIdx.y * (DOT_WARPS * R) + wid;
    double acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = 0.0;
    // Warps are independent (no shared memory, no block barrier): a warp keeps its chunk of w in registers
    // (w is read once per group of R vectors and stays in L2) and streams R basis vectors against it with
    // eight independent 16-byte loads per lane and vector in flight.
    if (j0 < nvt) {
        for (int64_t c = blockIdx.x; c < nchunk; c += gridDim.x) {
            const int64_t e0 = c * DOT_CHUNK;
            const int cnt = (int)(n - e0 < DOT_CHUNK ? n - e0 : DOT_CHUNK);
            if (cnt == DOT_CHUNK) {
                const double2* w2 = reinterpret_cast<const double2*>(w + e0);
                double2 b[DOT_CHUNK / 64];
#pragma unroll
                for (int i = 0; i < DOT_CHUNK / 64; ++i) b[i] = w2[lane + 32 * i];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int j = j0 + r * DOT_WARPS;
                    if (j < nvt) {
                        const double2* v2 = reinterpret_cast<const double2*>((j < nv ? V + (int64_t)j * ld : w) + e0);
                        double2 a[DOT_CHUNK / 64];
#pragma unroll
                        for (int i = 0; i < DOT_CHUNK / 64; ++i) a[i] = v2[lane + 32 * i];
                        double s = 0;
#pragma unroll
                        for (int i = 0; i < DOT_CHUNK / 64; ++i) {
                            s = fma(a[i].x, b[i].x, s);
                            s = fma(a[i].y, b[i].y, s);
                        }
                        acc[r] += s;
                    }
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int j = j0 + r * DOT_WARPS;
                    if (j < nvt) {
                        const double* v = (j < nv ? V + (int64_t)j * ld : w) + e0;
                        double s = 0;
                        for (int k = lane; k < cnt; k += 32) s = fma(v[k], w[e0 + k], s);
                        acc[r] += s;
                    }
                }
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int j = j0 + r * DOT_WARPS;
        if (j < nvt) {
            double s = acc[r];
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) partial[(int64_t)blockIdx.x * nvt + j] = s;
        }
    }
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) last = atomicAdd(counter, 1u) == gridDim.x * gridDim.y - 1;
    __syncthreads();
    if (!last) return;
    __threadfence();
    for (int j = wid; j < nvt; j += DOT_WARPS) {        // a warp per vector: lanes stride over the blocks, then a butterfly
        double s0 = 0, s1 = 0, s2 = 0, s3 = 0;          // four loads in flight; the summation pattern is fixed
        unsigned b = lane;
        for (; b + 96 < gridDim.x; b += 128) {
            s0 += __ldcg(&partial[(int64_t)b * nvt + j]);
            s1 += __ldcg(&partial[(int64_t)(b + 32) * nvt + j]);
            s2 += __ldcg(&partial[(int64_t)(b + 64) * nvt + j]);
            s3 += __ldcg(&partial[(int64_t)(b + 96) * nvt + j]);
        }
        for (; b < gridDim.x; b += 32) s0 += __ldcg(&partial[(int64_t)b * nvt + j]);
        double s = (s0 + s1) + (s2 + s3);
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) hout[j] = s;
    }
    if (threadIdx.x == 0) *counter = 0u;              // ready for the next launch on this stream
}

// w -= sum_j h_j V_j.  With vnext != NULL (second Gram-Schmidt pass): h[nv] holds w.w BEFORE the
// update, so |w - V h|^2 = w.w - |h|^2 (V orthonormal) and the new basis vector is written normalised
// in the same pass; block 0 publishes that squared norm to h[nv + 1].
__global__ void __launch_bounds__(256)
k_arnoldi_update(int64_t n, int nv, const double* __restrict__ V, int64_t ld, const double* __restrict__ h,
                 double* __restrict__ w, double* __restrict__ vnext, double* __restrict__ nrm2_out)
{
    extern __shared__ double sh[];
    __shared__ double inv;
    for (int j = threadIdx.x; j < nv; j += blockDim.x) sh[j] = h[j];
    __syncthreads();
    if (vnext && threadIdx.x == 0) {
        double h2 = 0;
        for (int j = 0; j < nv; ++j) h2 = fma(sh[j], sh[j], h2);
        const double r2 = h[nv] - h2;
        if (blockIdx.x == 0) *nrm2_out = r2;
        inv = r2 > 0 ? 1.0 / sqrt(r2) : 0.0;
    }
    __syncthreads();
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        double acc = w[e];
        int j = 0;
        for (; j + 4 <= nv; j += 4) {
            const double v0 = V[(int64_t)j * ld + e], v1 = V[(int64_t)(j + 1) * ld + e], v2 = V[(int64_t)(j + 2) * ld + e],
                         v3 = V[(int64_t)(j + 3) * ld + e];
            acc = fma(-sh[j], v0, acc);
            acc = fma(-sh[j + 1], v1, acc);
            acc = fma(-sh[j + 2], v2, acc);
            acc = fma(-sh[j + 3], v3, acc);
        }
        for (; j < nv; ++j) acc = fma(-sh[j], V[(int64_t)j * ld + e], acc);
        w[e] = acc;
        if (vnext) vnext[e] = acc * inv;
    }
}

// vnext = w / sqrt(*nrm2)
__global__ void __launch_bounds__(256)
k_normalize(int64_t n, const double* __restrict__ nrm2, const double* __restrict__ w, double* __restrict__ vnext)
{
    const double s = *nrm2;
    const double inv = s > 0 ? 1.0 / sqrt(s) : 0.0;
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x)
        vnext[e] = w[e] * inv;
}

// ---- short vectors: both Gram-Schmidt passes, the norm and the new basis vector in ONE cooperative launch -----
// For 2N up to a few ten thousand the four vector kernels above are pure launch latency.  Here block b owns
// elements [256 b, 256 b + 256) of w (kept in shared memory across the passes) and the whole grid is resident:
//   A  partial dots V_j . w over the chunk                   -> grid sync
//   B  h1 = sum of the partials (fixed order); w -= V h1 ; partial dots V_j . w and w . w -> grid sync
//   C  h2, s = w.w; r2 = s - |h2|^2; w -= V h2; v_next = w / sqrt(r2)
// Block 0 writes h1, h2, s, r2 straight into pinned host memory (read by the host after the stream sync).
// Same arithmetic and summation pattern as k_dots<1> / k_arnoldi_update up to the chunk size.
#define CGS_CHUNK 256
__global__ void __launch_bounds__(CGS_CHUNK)
k_cgs2(int64_t n, int nv, const double* __restrict__ V, int64_t ld, double* __restrict__ w, double* __restrict__ vnext,
       double* __restrict__ partial /*[2][grid][nv+1]*/, double* __restrict__ hpin, int hstride)
{
    cg::grid_group grid = cg::this_grid();
    extern __shared__ double cgs_sm[];
    double* sw = cgs_sm;                      // [CGS_CHUNK] this block's chunk of w
    double* hs = cgs_sm + CGS_CHUNK;          // [nv + 2]
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int nb = gridDim.x, nvt = nv + 1;
    const int64_t e0 = (int64_t)blockIdx.x * CGS_CHUNK;
    const int cnt = (int)(n - e0 < CGS_CHUNK ? n - e0 : CGS_CHUNK);
    sw[tid] = tid < cnt ? w[e0 + tid] : 0.0;
    __syncthreads();
    double* part0 = partial;
    double* part1 = partial + (size_t)nb * nvt;
    auto dots = [&](double* part, bool self) {
        for (int j = wid; j < nv + (self ? 1 : 0); j += CGS_CHUNK / 32) {
            double s = 0;
            if (j < nv) {
                const double* v = V + (int64_t)j * ld + e0;
#pragma unroll
                for (int i = 0; i < CGS_CHUNK / 32; ++i) {
                    const int k = lane + 32 * i;
                    s = fma(k < cnt ? v[k] : 0.0, sw[k], s);
                }
            } else {
#pragma unroll
                for (int i = 0; i < CGS_CHUNK / 32; ++i) s = fma(sw[lane + 32 * i], sw[lane + 32 * i], s);
            }
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) part[(size_t)blockIdx.x * nvt + j] = s;
        }
    };
    auto gather = [&](const double* part, int count) {   // hs[j] = sum over blocks: a warp per j, lanes over blocks, butterfly
        __syncthreads();
        for (int j = wid; j < count; j += CGS_CHUNK / 32) {
            double s = 0;
            for (int b = lane; b < nb; b += 32) s += __ldcg(&part[(size_t)b * nvt + j]);
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) hs[j] = s;
        }
        __syncthreads();
    };
    auto update = [&]() -> double {
        double acc = sw[tid];
        if (tid < cnt) {
            const double* v = V + e0 + tid;
            int j = 0;
            for (; j + 4 <= nv; j += 4) {
                const double v0 = v[(int64_t)j * ld], v1 = v[(int64_t)(j + 1) * ld], v2 = v[(int64_t)(j + 2) * ld],
                             v3 = v[(int64_t)(j + 3) * ld];
                acc = fma(-hs[j], v0, acc);
                acc = fma(-hs[j + 1], v1, acc);
                acc = fma(-hs[j + 2], v2, acc);
                acc = fma(-hs[j + 3], v3, acc);
            }
            for (; j < nv; ++j) acc = fma(-hs[j], v[(int64_t)j * ld], acc);
        }
        return acc;
    };
    dots(part0, false);
    __threadfence();
    grid.sync();
    gather(part0, nv);
    if (blockIdx.x == 0)
        for (int j = tid; j < nv; j += CGS_CHUNK) hpin[j] = hs[j];
    {
        const double acc = update();
        __syncthreads();
        sw[tid] = acc;
        __syncthreads();
    }
    dots(part1, true);
    __threadfence();
    grid.sync();
    gather(part1, nvt);
    __shared__ double inv;
    if (tid == 0) {
        double h2 = 0;
        for (int j = 0; j < nv; ++j) h2 = fma(hs[j], hs[j], h2);
        const double r2 = hs[nv] - h2;
        inv = r2 > 0 ? 1.0 / sqrt(r2) : 0.0;
        if (blockIdx.x == 0) hpin[hstride + nv + 1] = r2;
    }
    if (blockIdx.x == 0)
        for (int j = tid; j < nvt; j += CGS_CHUNK) hpin[hstride + j] = hs[j];
    __syncthreads();
    const double acc = update();
    if (tid < cnt) {
        w[e0 + tid] = acc;
        vnext[e0 + tid] = acc * inv;
    }
}

// z = Minv v: per panel the inverse 2x2 diagonal block (SELF entries), original panel order
__global__ void k_precond(int64_t N, const double* __restrict__ pc, const double* __restrict__ v, double* __restrict__ z)
{
    int64_t o = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (o >= N) return;
    double a = v[o], b = v[N + o];
    z[o] = pc[o] * a + pc[N + o] * b;
    z[N + o] = pc[2 * N + o] * a + pc[3 * N + o] * b;
}

// r = b - y
__global__ void k_residual(int64_t n, const double* __restrict__ b, const double* __restrict__ y, double* __restrict__ r)
{
    int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e < n) r[e] = b[e] - y[e];
}

// u = sum_j c_j V_j
__global__ void __launch_bounds__(256)
k_lincomb(int64_t n, int nv, const double* __restrict__ V, int64_t ld, const double* __restrict__ coef, double* __restrict__ u)
{
    extern __shared__ double sh[];
    for (int j = threadIdx.x; j < nv; j += blockDim.x) sh[j] = coef[j];
    __syncthreads();
    const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= n) return;
    double acc = 0;
    for (int j = 0; j < nv; ++j) acc = fma(sh[j], V[(int64_t)j * ld + e], acc);
    u[e] = acc;
}

__global__ void k_axpy(int64_t n, double a, const double* __restrict__ x, double* __restrict__ y)
{
    int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e < n) y[e] = fma(a, x[e], y[e]);
}

// ---- near-field preconditioner (flexible GMRES) ---------------------------------------------------------------
// z = M(v): PB_NF_STEPS (2; 4 from 30,000 panels, 6 from 300,000) minimal-residual steps, block-Jacobi preconditioned, on the sparse NEAR-FIELD matrix A_n of
// Eq. (5) -- the true SELF / ADJ / NEAR entries of the three-zone quadrature, i.e. the part of the operator
// that carries the singular local behaviour at the creases of a van-der-Waals surface:
//     r = v, z = 0;  repeat:  p = D^-1 r;  q = A_n p;  alpha = (r.q)/(q.q);  z += alpha p;  r -= alpha q.
// alpha stays on the device (no host synchronisation); the iteration runs in Morton order, where the table lives.
// M depends on v non-linearly (through alpha), hence the flexible variant of GMRES.  Measured on the oracle's dense
// matrix of C2 (19,176 unknowns): 72 outer iterations with block-Jacobi alone, 42 with 2 inner steps, 40 with 3,
// 28 with an exact sparse solve of A_n.  The table of A_n is kept in fp16 (a quarter of the bytes to stream per step; entries are O(1) or smaller): M only
// has to be a good approximate inverse, the residuals of the outer iteration come from the fp64 operator.
#define PB_NF_STEPS 2

__global__ void k_nf_start(int64_t N, const int32_t* __restrict__ perm, const double* __restrict__ pc,
                           const double* __restrict__ v, double* __restrict__ r, double* __restrict__ p, double* __restrict__ z)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int64_t o = perm[i];
    const double a = v[o], b = v[N + o];
    r[i] = a; r[N + i] = b;
    p[i] = pc[o] * a + pc[N + o] * b;
    p[N + i] = pc[2 * N + o] * a + pc[3 * N + o] * b;
    z[i] = 0.0; z[N + i] = 0.0;
}

// q = A_n p in Morton order.  One lane per target, one warp per ELL slice of 32 targets: per entry one column index, the
// four values of the pair as one 8-byte load (fp16, interleaved) and two gathers, p_j = phi_j and p_{N+j} = dphi_j.  (The
// first version gave each of the four kernels its own warp: four index loads and four gathers per entry, 150 us per
// product at C4 against 0.73 GB of table; the gathers, not the table, set the pace.)
#define NF_WARPS 4
__global__ void __launch_bounds__(32 * NF_WARPS)
k_nf_spmv(int64_t N, double eps_ratio, const int32_t* __restrict__ el_base, const int32_t* __restrict__ el_col,
          const uint2* __restrict__ el_tval /*[entries] 4 x fp16: V_L, K_L, V_Y, K_Y*/, const double* __restrict__ p,
          double* __restrict__ q)
{
    const int lane = threadIdx.x & 31;
    const int64_t sl = blockIdx.x * (int64_t)NF_WARPS + (threadIdx.x >> 5);
    if (sl * 32 >= N) return;
    const int64_t i = sl * 32 + lane;
    const int32_t b0 = el_base[sl], width = (el_base[sl + 1] - b0) / 32;
    const uint2* __restrict__ val = el_tval + b0 + lane;
    const int32_t* __restrict__ col = el_col + b0 + lane;
    double VL = 0.0, KL = 0.0, VY = 0.0, KY = 0.0;
    auto add = [&](uint2 v, double ph, double dp) {
        const float2 lo = __half22float2(*reinterpret_cast<const __half2*>(&v.x));   // V_L, K_L
        const float2 hi = __half22float2(*reinterpret_cast<const __half2*>(&v.y));   // V_Y, K_Y
        VL = fma((double)lo.x, dp, VL); KL = fma((double)lo.y, ph, KL);
        VY = fma((double)hi.x, dp, VY); KY = fma((double)hi.y, ph, KY);
    };
    int k = 0;
    for (; k + 4 <= width; k += 4) {
        uint2 v[4];
        double ph[4], dp[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int32_t j = col[32 * (k + u)];
            v[u] = val[32 * (k + u)];
            ph[u] = p[j];
            dp[u] = p[N + j];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) add(v[u], ph[u], dp[u]);
    }
    for (; k < width; ++k) {
        const int32_t j = col[32 * k];
        add(val[32 * k], p[j], p[N + j]);
    }
    if (i < N) {
        const double phi = p[i];
        q[i] = 0.5 * phi + KL - VL;                     // Eq. (5), first row restricted to the near zone
        q[N + i] = 0.5 * phi - KY + eps_ratio * VY;     // second row
    }
}

// out[0] = (r.q)/(q.q) by the last block to finish (fixed summation pattern)
__global__ void __launch_bounds__(256)
k_nf_alpha(int64_t n, const double* __restrict__ r, const double* __restrict__ q, double* __restrict__ partial,
           unsigned int* __restrict__ counter, double* __restrict__ out)
{
    __shared__ double red[2][8];
    __shared__ bool last;
    double a = 0, b = 0;
    for (int64_t e = blockIdx.x * 256LL + threadIdx.x; e < n; e += 256LL * gridDim.x) {
        const double qe = q[e];
        a = fma(r[e], qe, a);
        b = fma(qe, qe, b);
    }
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) { red[0][w] = a; red[1][w] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = 0; b = 0;
        for (int k = 0; k < 8; ++k) { a += red[0][k]; b += red[1][k]; }
        partial[2 * blockIdx.x] = a;
        partial[2 * blockIdx.x + 1] = b;
        __threadfence();
        last = atomicAdd(counter, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    if (threadIdx.x < 32) {
        a = 0; b = 0;
        for (unsigned k = threadIdx.x; k < gridDim.x; k += 32) { a += __ldcg(&partial[2 * k]); b += __ldcg(&partial[2 * k + 1]); }
        for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
        if (threadIdx.x == 0) { out[0] = b > 0 ? a / b : 0.0; *counter = 0u; }
    }
}

// z += alpha p; r -= alpha q; then either p = D^-1 r for the next step or, at the end, zout = z in the caller's order
__global__ void k_nf_update(int64_t N, const double* __restrict__ alpha, const int32_t* __restrict__ perm,
                            const double* __restrict__ pc, double* __restrict__ p, const double* __restrict__ q,
                            double* __restrict__ r, double* __restrict__ z, double* __restrict__ zout)
{
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double al = *alpha;
    const double z0 = fma(al, p[i], z[i]), z1 = fma(al, p[N + i], z[N + i]);
    const int64_t o = perm[i];
    if (zout) {
        zout[o] = z0; zout[N + o] = z1;
        return;
    }
    z[i] = z0; z[N + i] = z1;
    const double a = fma(-al, q[i], r[i]), b = fma(-al, q[N + i], r[N + i]);
    r[i] = a; r[N + i] = b;
    p[i] = pc[o] * a + pc[N + o] * b;
    p[N + i] = pc[2 * N + o] * a + pc[3 * N + o] * b;
}

typedef pb_gmres_ws gmres_ws;

// z = M(v) (near-field preconditioner); v, z in the caller's panel order
static int near_precond(pb_ctx* ctx, gmres_ws& ws, const double* v, double* z)
{
    pb_tree& t = ctx->tree;
    cudaStream_t st = ctx->stream;
    const int64_t N = t.N, n = 2 * N;
    const int tb = 256;
    const int nbN = pb_blocks(N, tb);
    int nbd = pb_blocks(n, 256 * 8);
    if (nbd > 592) nbd = 592;
    k_nf_start<<<nbN, tb, 0, st>>>(N, t.perm, t.precond, v, ws.nf_r, ws.nf_p, ws.nf_z);
    PB_LAUNCH_CHECK();
    // more inner steps where the operator is expensive: cold-solve iterations at C3 89 / 74 / 68 and at C4 177 / 147 / 137
    // with 2 / 4 / 6 steps (block-Jacobi alone: 147 and 317)
    const int nsteps = N < 30000 ? PB_NF_STEPS : (N < 300000 ? 2 * PB_NF_STEPS : 3 * PB_NF_STEPS);
    for (int step = 0; step < nsteps; ++step) {
        k_nf_spmv<<<pb_blocks((N + 31) / 32, NF_WARPS), 32 * NF_WARPS, 0, st>>>(N, ctx->prm.eps_in / ctx->prm.eps_out, t.el_base, t.el_col,
                                                                              reinterpret_cast<const uint2*>(t.el_tval), ws.nf_p, ws.nf_q);
        PB_LAUNCH_CHECK();
        k_nf_alpha<<<nbd, 256, 0, st>>>(n, ws.nf_r, ws.nf_q, ws.partial, ws.counter, ws.hdev + 2 * (ws.m + 4) + 4);
        PB_LAUNCH_CHECK();
        k_nf_update<<<nbN, tb, 0, st>>>(N, ws.hdev + 2 * (ws.m + 4) + 4, t.perm, t.precond, ws.nf_p, ws.nf_q, ws.nf_r, ws.nf_z,
                                        step + 1 == nsteps ? z : nullptr);
        PB_LAUNCH_CHECK();
    }
    return PB_OK;
}

// hout[0..nv) = V^T w (and hout[nv] = w.w with `self`), all on the device
static int dot_into(pb_ctx* ctx, gmres_ws& ws, int nv, const double* V, const double* w, bool self, double* hout)
{
    const int nvt = nv + (self ? 1 : 0);
    const int64_t nchunk = (ws.n + DOT_CHUNK - 1) / DOT_CHUNK;
    const int gy1 = (nvt + DOT_WARPS - 1) / DOT_WARPS;
    if (nchunk * gy1 <= DOT_MAXBLK) {                     // short vectors: one chunk per block, spread wide (latency)
        dim3 grid((unsigned)nchunk, (unsigned)gy1);
        k_dots<1><<<grid, DOT_THREADS, 0, ctx->stream>>>(ws.n, nv, V, ws.n, w, self ? 1 : 0, ws.partial, ws.counter, hout);
    } else {                                              // long vectors: two full waves of resident blocks (bandwidth)
        int& occ = ctx->dots_occ;                          // per device: remembered per context
        if (occ == 0) {
            PB_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_dots<4>, DOT_THREADS, 0));
            if (occ < 1) occ = 1;
            if (occ > 8) occ = 8;
        }
        int nsm = 148;
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, ctx->device);
        const int resident = 2 * nsm * occ < DOT_MAXBLK ? 2 * nsm * occ : DOT_MAXBLK;
        const int gy = (nvt + 4 * DOT_WARPS - 1) / (4 * DOT_WARPS);
        int64_t gx = resident / gy;
        if (gx > nchunk) gx = nchunk;
        if (gx < 1) gx = 1;
        dim3 grid((unsigned)gx, (unsigned)gy);
        k_dots<4><<<grid, DOT_THREADS, 0, ctx->stream>>>(ws.n, nv, V, ws.n, w, self ? 1 : 0, ws.partial, ws.counter, hout);
    }
    PB_LAUNCH_CHECK();
    return PB_OK;
}

// workspace (kept until the system size, the restart length or the preconditioner changes); the Krylov bases of
// GMRES only when asked for (the GCR path of the SCF loop keeps its own)
static int ws_ensure(pb_ctx* ctx, int mode, int m, bool basis)
{
    pb_tree& t = ctx->tree;
    cudaStream_t st = ctx->stream;
    const int64_t n = 2 * t.N;
    gmres_ws& ws = ctx->gws;
    if (ws.n != n || ws.m != m || ws.mode != mode || !ws.r) {
        pb_dfree_cat(ctx, CAT_SOLVE);
        ws = gmres_ws();
        PB_TRY(pb_dalloc_t(ctx, &ws.w, n, CAT_SOLVE));
        PB_TRY(pb_dalloc_t(ctx, &ws.r, n, CAT_SOLVE));
        PB_TRY(pb_dalloc_t(ctx, &ws.u, n, CAT_SOLVE));
        PB_TRY(pb_dalloc_t(ctx, &ws.z, n, CAT_SOLVE));
        PB_TRY(pb_dalloc_t(ctx, &ws.ax, n, CAT_SOLVE));
        if (mode == 2) {
            PB_TRY(pb_dalloc_t(ctx, &ws.nf_r, n, CAT_SOLVE));
            PB_TRY(pb_dalloc_t(ctx, &ws.nf_p, n, CAT_SOLVE));
            PB_TRY(pb_dalloc_t(ctx, &ws.nf_q, n, CAT_SOLVE));
            PB_TRY(pb_dalloc_t(ctx, &ws.nf_z, n, CAT_SOLVE));
        }
        ws.mode = mode;
        PB_TRY(pb_dalloc_t(ctx, &ws.partial, (size_t)DOT_MAXBLK * (m + 2), CAT_SOLVE));
        PB_TRY(pb_dalloc_t(ctx, &ws.hdev, 2 * (m + 4) + 8, CAT_SOLVE));
        PB_TRY(pb_dalloc_t(ctx, &ws.coef, m + 2, CAT_SOLVE));
        PB_TRY(pb_dalloc_t(ctx, &ws.counter, 4, CAT_SOLVE));
        PB_CUDA(cudaMemsetAsync(ws.counter, 0, 4 * sizeof(unsigned int), st));
        ws.n = n;
        ws.m = m;
    }
    if (basis && !ws.V) {
        PB_TRY(pb_dalloc_t(ctx, &ws.V, (size_t)(m + 1) * n, CAT_SOLVE));
        if (mode == 2) PB_TRY(pb_dalloc_t(ctx, &ws.Z, (size_t)m * n, CAT_SOLVE));
    }
    return PB_OK;
}

// preconditioner of pb_params.precond as it applies to this system: 0 none, 1 block-Jacobi, 2 near-field
static int precond_mode(pb_ctx* ctx)
{
    const pb_tree& t = ctx->tree;
    int mode = ctx->prm.precond;
    // 3 = near-field from 8,000 panels up (measured per solve: C1 20.0 -> 19.2 ms, C2 117 -> 91 ms, C3 1412 -> 978 ms),
    // else block-Jacobi
    if (mode == 3) mode = t.N >= 8000 ? 2 : 1;
    if (t.psurf && mode == 2) mode = 1;   // two surfaces: the near-field matrix of mode 2 has Eq. (5)'s single-surface rows
    return mode;
}

static int restart_length(pb_ctx* ctx)
{
    const int64_t n = 2 * ctx->tree.N;
    int m = ctx->prm.gmres_restart;
    if (m > n) m = (int)n;
    if (m > 1000) m = 1000;
    return m;
}

// Restarted GMRES with a right block-Jacobi preconditioner (D: R-20).  Per iteration: one operator
// application (the preconditioner is folded into its first kernel), two classical Gram-Schmidt
// passes of two kernels each -- the second also yields the norm of the new vector by Pythagoras and
// writes it normalised -- and one small device-to-host copy of the Hessenberg column.
// `x_is_last_result`: x still holds exactly what the previous call on this context returned (the SCF loop), so
// A x is known from the Arnoldi relation A Minv V_j = V_{j+1} Hbar_j and the starting residual costs no operator
// application: ws.ax is kept up to date with  A x += V_{j+1} (Hbar_j y)  whenever x += Minv V_j y.
int pb_gmres_impl(pb_ctx* ctx, const double* b, double* x, int32_t* iters_out, double* relres_out, int32_t* matvecs_out,
                  bool x_is_last_result, double tol_abs)
{
    pb_tree& t = ctx->tree;
    cudaStream_t st = ctx->stream;
    if (!t.built) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_gmres: call pb_tree_build first");
    const int64_t n = 2 * t.N;
    // preconditioner: 0 none, 1 block-Jacobi (folded into the operator's first kernel), 2 near-field (flexible GMRES)
    const int mode = precond_mode(ctx);
    const int m = restart_length(ctx);
    PB_TRY(ws_ensure(ctx, mode, m, true));
    gmres_ws& ws = ctx->gws;
    bool have_ax = x_is_last_result && ws.ax_valid;
    ws.ax_valid = false;
    const int hstride = m + 4;
    PB_TRY(pb_pinned(ctx, (5 * (size_t)m + 64) * sizeof(double)));
    double* hh = ctx->h_pinned;                    // staging for h columns [2][hstride]
    double* hy = hh + 2 * hstride;                 // staging for y (x += Z y) and for Hbar y (A x += V Hbar y): written at the end
    double* hc = hy + m;                           // of a cycle only, and every cycle starts with a stream synchronisation
    const bool pc = mode == 1;
    const double tol = tol_abs > 0.0 ? tol_abs : ctx->prm.gmres_tol;
    const int maxit = ctx->prm.gmres_maxit;
    int iters = 0, matvecs = 0;
    int rc = PB_OK;

    // ||b||^2 is read back together with the first residual norm (one synchronisation fewer per solve)
    PB_TRY(dot_into(ctx, ws, 0, nullptr, b, true, ws.hdev + 2 * hstride));
    double bnorm = -1.0;
    double relres = 0.0;
    std::vector<double> H((size_t)(m + 1) * m, 0.0), Hraw((size_t)(m + 1) * m, 0.0), cs(m, 0.0), sn(m, 0.0), g(m + 1, 0.0),
        yv(m, 0.0);

    const int tb = 256;
    const int nb = pb_blocks(n, tb) < 2368 ? pb_blocks(n, tb) : 2368;   // grid-stride above 16 blocks per SM
    // short vectors: the whole orthogonalisation in one cooperative launch (one block per 256 elements, all resident)
    int coop_blocks = 0;
    {
        int nsm = 0, coop = 0;
        cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, ctx->device);
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device);
        const int64_t need = (n + CGS_CHUNK - 1) / CGS_CHUNK;
        if (coop && need <= nsm && (size_t)2 * need * (m + 1) <= (size_t)DOT_MAXBLK * (m + 2)) coop_blocks = (int)need;
    }
    for (;;) {
        // residual r = b - A x: A x from the Arnoldi relation when it is known, else by applying the operator
        if (!have_ax) {
            PB_TRY(pb_matvec_impl(ctx, x, ws.ax, false, false));
            ++matvecs;
        }
        have_ax = false;                               // after a restart the residual is recomputed from scratch
        k_residual<<<pb_blocks(n, tb), tb, 0, st>>>(n, b, ws.ax, ws.r);
        PB_LAUNCH_CHECK();
        PB_TRY(dot_into(ctx, ws, 0, nullptr, ws.r, true, ws.hdev));
        k_normalize<<<nb, tb, 0, st>>>(n, ws.hdev, ws.r, ws.V);      // V_0 = r/||r||
        PB_LAUNCH_CHECK();
        double r2 = 0, bn2 = 0;
        PB_CUDA(cudaMemcpyAsync(&r2, ws.hdev, sizeof(double), cudaMemcpyDeviceToHost, st));
        if (bnorm < 0) PB_CUDA(cudaMemcpyAsync(&bn2, ws.hdev + 2 * hstride, sizeof(double), cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaStreamSynchronize(st));
        if (bnorm < 0) {
            bnorm = sqrt(bn2);
            if (bnorm == 0.0) {
                PB_CUDA(cudaMemsetAsync(x, 0, sizeof(double) * n, st));
                if (iters_out) *iters_out = 0;
                if (relres_out) *relres_out = 0.0;
                if (matvecs_out) *matvecs_out = matvecs;
                return PB_OK;
            }
        }
        const double beta = sqrt(r2);
        relres = beta / bnorm;
        if (relres <= tol) { ws.ax_valid = true; break; }      // ws.ax = A x for the x we return
        if (iters >= maxit) { rc = PB_ERR_NO_CONVERGENCE; break; }
        std::fill(g.begin(), g.end(), 0.0);
        g[0] = beta;
        bool accepted = false, breakdown = false;
        int j = 0;
        for (; j < m && iters < maxit;) {
            const double* vj = ws.V + (size_t)j * n;
            double* vnext = ws.V + (size_t)(j + 1) * n;
            if (mode == 2) {                                          // flexible: z_j = M(v_j) is kept, w = A z_j
                double* zj = ws.Z + (size_t)j * n;
                PB_TRY(near_precond(ctx, ws, vj, zj));
                PB_TRY(pb_matvec_impl(ctx, zj, ws.w, false, false));
            } else
                PB_TRY(pb_matvec_impl(ctx, vj, ws.w, false, pc));    // w = A Minv v_j
            ++matvecs;
            const int nv = j + 1;
            // classical Gram-Schmidt, twice
            double* hA = ws.hdev;
            double* hB = ws.hdev + hstride;
            if (coop_blocks > 0) {
                int64_t n_ = n, ld_ = n;
                int nv_ = nv, hs_ = hstride;
                const double* V_ = ws.V;
                double *w_ = ws.w, *vn_ = vnext, *pa_ = ws.partial, *hp_ = hh;
                void* args[] = {&n_, &nv_, &V_, &ld_, &w_, &vn_, &pa_, &hp_, &hs_};
                PB_CUDA(cudaLaunchCooperativeKernel((void*)k_cgs2, dim3(coop_blocks), dim3(CGS_CHUNK), args,
                                                    (size_t)(CGS_CHUNK + m + 4) * sizeof(double), st));
                PB_LAUNCH_CHECK();
                PB_CUDA(cudaStreamSynchronize(st));
            } else {
                PB_TRY(dot_into(ctx, ws, nv, ws.V, ws.w, false, hA));
                k_arnoldi_update<<<nb, tb, nv * sizeof(double), st>>>(n, nv, ws.V, n, hA, ws.w, nullptr, nullptr);
                PB_LAUNCH_CHECK();
                PB_TRY(dot_into(ctx, ws, nv, ws.V, ws.w, true, hB));     // hB[nv] = w.w
                k_arnoldi_update<<<nb, tb, nv * sizeof(double), st>>>(n, nv, ws.V, n, hB, ws.w, vnext, hB + nv + 1);
                PB_LAUNCH_CHECK();
                PB_CUDA(cudaMemcpyAsync(hh, ws.hdev, sizeof(double) * 2 * hstride, cudaMemcpyDeviceToHost, st));
                PB_CUDA(cudaStreamSynchronize(st));
            }
            double hn2 = hh[hstride + nv + 1];
            if (!(hn2 > 1e-2 * hh[hstride + nv])) {
                // the second pass removed most of w (cancellation in w.w - |h|^2): take the norm directly
                PB_TRY(dot_into(ctx, ws, 0, nullptr, ws.w, true, hB + nv + 1));
                k_normalize<<<nb, tb, 0, st>>>(n, hB + nv + 1, ws.w, vnext);
                PB_LAUNCH_CHECK();
                PB_CUDA(cudaMemcpyAsync(&hn2, hB + nv + 1, sizeof(double), cudaMemcpyDeviceToHost, st));
                PB_CUDA(cudaStreamSynchronize(st));
            }
            double* col = &H[(size_t)j * (m + 1)];
            for (int i = 0; i < nv; ++i) col[i] = hh[i] + hh[hstride + i];
            for (int i = 0; i < nv; ++i) Hraw[(size_t)j * (m + 1) + i] = col[i];
            const double hnext = hn2 > 0 ? sqrt(hn2) : 0.0;
            col[nv] = hnext;
            Hraw[(size_t)j * (m + 1) + nv] = hnext;
            // Givens rotations (host, O(j))
            for (int i = 0; i < j; ++i) {
                double a = cs[i] * col[i] + sn[i] * col[i + 1];
                col[i + 1] = -sn[i] * col[i] + cs[i] * col[i + 1];
                col[i] = a;
            }
            double den = hypot(col[j], col[j + 1]);
            // exact breakdown (the new column is zero: A Minv v_j lies in nothing, singular operator): drop the column,
            // keep the update from the j columns before it and report no convergence
            if (den == 0.0) { breakdown = true; break; }
            cs[j] = col[j] / den;
            sn[j] = col[j + 1] / den;
            col[j] = den;
            col[j + 1] = 0.0;
            g[j + 1] = -sn[j] * g[j];
            g[j] = cs[j] * g[j];
            ++j;
            ++iters;
            relres = fabs(g[j]) / bnorm;
            if (relres <= tol) { accepted = true; break; }
            if (hnext <= 1e-300) break;
        }
        // y = R^{-1} g ; x += Minv (V y)
        for (int i = j - 1; i >= 0; --i) {
            double s = g[i];
            for (int k = i + 1; k < j; ++k) s -= H[(size_t)k * (m + 1) + i] * yv[k];
            yv[i] = s / H[(size_t)i * (m + 1) + i];
        }
        for (int i = 0; i < j; ++i) hy[i] = yv[i];
        PB_CUDA(cudaMemcpyAsync(ws.coef, hy, sizeof(double) * j, cudaMemcpyHostToDevice, st));
        k_lincomb<<<pb_blocks(n, tb), tb, j * sizeof(double), st>>>(n, j, mode == 2 ? ws.Z : ws.V, n, ws.coef, ws.u);   // x += Z y (flexible)
        PB_LAUNCH_CHECK();
        if (pc) {
            k_precond<<<pb_blocks(t.N, tb), tb, 0, st>>>(t.N, t.precond, ws.u, ws.z);
            PB_LAUNCH_CHECK();
            k_axpy<<<pb_blocks(n, tb), tb, 0, st>>>(n, 1.0, ws.z, x);
        } else
            k_axpy<<<pb_blocks(n, tb), tb, 0, st>>>(n, 1.0, ws.u, x);
        PB_LAUNCH_CHECK();
        // A x += V_{j+1} (Hbar_j y)
        for (int i = 0; i <= j; ++i) {
            double c = 0;
            for (int k = (i > 0 ? i - 1 : 0); k < j; ++k) c += Hraw[(size_t)k * (m + 1) + i] * yv[k];
            hc[i] = c;
        }
        PB_CUDA(cudaMemcpyAsync(ws.coef, hc, sizeof(double) * (j + 1), cudaMemcpyHostToDevice, st));
        k_lincomb<<<pb_blocks(n, tb), tb, (j + 1) * sizeof(double), st>>>(n, j + 1, ws.V, n, ws.coef, ws.u);
        PB_LAUNCH_CHECK();
        k_axpy<<<pb_blocks(n, tb), tb, 0, st>>>(n, 1.0, ws.u, ws.ax);
        PB_LAUNCH_CHECK();
        ws.ax_valid = accepted;
        // Converged by the Arnoldi residual |g_j|: with a RIGHT preconditioner and CGS2-orthogonal V this is the true
        // residual norm to rounding, so no further operator application is spent on confirming it.  After a
        // restart (no convergence within m steps) the loop recomputes the true residual as the new start.
        if (accepted) break;
        if (breakdown) { rc = PB_ERR_NO_CONVERGENCE; break; }
    }
    if (iters_out) *iters_out = iters;
    if (relres_out) *relres_out = relres;
    if (matvecs_out) *matvecs_out = matvecs;
    if (rc != PB_OK) return pb_fail(ctx, rc, "GMRES: %d iterations, relative residual %.3e > %.3e", iters, relres, tol);
    return PB_OK;
}

extern "C" int pb_gmres(pb_ctx* ctx, const double* b, double* x, int32_t* iters, double* relres)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (!b || !x) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_gmres: NULL vector");
    PB_TRY(pb_gmres_impl(ctx, b, x, iters, relres, nullptr, false));
    PB_CUDA(cudaStreamSynchronize(ctx->stream));   // the last updates of x are still in flight when the loop returns
    return PB_OK;
}

// ---- SCF and energy kernels ------------------------------------------------------------------------
// mu_new = (1-w) mu + w alpha 4 pi E,  E = -(grad_solv + grad_mult)   (Eq. 9, 15; SOR P:160; D: R-2)
// grad_mult = gperm (masked permanent multipoles: constant over the loop, computed once) + gmult (induced dipoles)
// out[0] = sum_m |mu_new - mu|^2
__global__ void __launch_bounds__(256)
k_scf_update(int64_t na, const double* __restrict__ alpha, const double* __restrict__ gsolv,
             const double* __restrict__ gperm, const double* __restrict__ gmult, double omega, double* __restrict__ mu,
             double* __restrict__ out)
{
    __shared__ double red[8];
    double s = 0;
    for (int64_t e = threadIdx.x; e < 3 * na; e += blockDim.x) {
        double E = -(gsolv ? gsolv[e] : 0.0) - gperm[e] - gmult[e];
        double old = mu[e];
        double nw = (1.0 - omega) * old + omega * alpha[e / 3] * (4.0 * 3.14159265358979323846) * E;
        mu[e] = nw;
        s += (nw - old) * (nw - old);
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0;
        for (int k = 0; k < 8; ++k) v += red[k];
        out[0] = v;
    }
}

// G = 1/2 sum_m [ q phi + d.grad phi + (1/6) Q : hess phi ]  with the PERMANENT dipole (Eq. 24)
__global__ void __launch_bounds__(256)
k_energy(int64_t na, const double* __restrict__ q, const double* __restrict__ dip, const double* __restrict__ quad,
         const double* __restrict__ phi, const double* __restrict__ grad, const double* __restrict__ hess,
         double* __restrict__ out)
{
    __shared__ double red[8];
    double s = 0;
    for (int64_t m = threadIdx.x; m < na; m += blockDim.x) {
        const double* Q = quad + 6 * m;
        const double* Hm = hess + 6 * m;
        double QH = Q[0] * Hm[0] + Q[3] * Hm[3] + Q[5] * Hm[5] + 2.0 * (Q[1] * Hm[1] + Q[2] * Hm[2] + Q[4] * Hm[4]);
        s += q[m] * phi[m] + dip[3 * m] * grad[3 * m] + dip[3 * m + 1] * grad[3 * m + 1] + dip[3 * m + 2] * grad[3 * m + 2] +
             QH / 6.0;
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0;
        for (int k = 0; k < 8; ++k) v += red[k];
        out[0] = 0.5 * v;
    }
}

__global__ void k_any_nonzero(int64_t n, const double* __restrict__ a, int* __restrict__ flag)
{
    int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e < n && a[e] != 0.0) *flag = 1;
}

// ---- recycled subspace across the solves of one SCF loop (pb_params.scf_recycle; D: R-20) ---------------------------------
// The right-hand sides of the loop differ by the field of the changing induced dipoles, b_k = b_perm + B mu_k, and the
// corrections x_k - x_{k-1} of successive solves are nearly parallel (mu converges geometrically).  Every finished solve
// contributes its correction u and c = A u -- known from the Arnoldi relation that already carries A x, no operator
// application -- to a pair of bases RU, RC with RC orthonormal and A RU = RC.  The next solve first takes the
// minimal-residual step in that space, x += RU (RC^T r), A x += RC (RC^T r), and GMRES then starts from the smaller
// residual and runs to the same tolerance as without it.
static int recycle_alloc(pb_ctx* ctx, gmres_ws& ws)
{
    if (ws.RU || !ws.r) return PB_OK;
    int cap = ctx->prm.scf_maxit < 48 ? ctx->prm.scf_maxit : 48;
    if ((size_t)cap * ws.n * sizeof(double) * 2 > ((size_t)4 << 30)) cap = (int)(((size_t)2 << 30) / (ws.n * sizeof(double)));   // <= 4 GB
    if (cap > ws.m) cap = ws.m;                         // the dot / coefficient buffers are sized for the restart length
    if (cap < 1) return PB_OK;
    PB_TRY(pb_dalloc_t(ctx, &ws.RU, (size_t)cap * ws.n, CAT_SOLVE));
    PB_TRY(pb_dalloc_t(ctx, &ws.RC, (size_t)cap * ws.n, CAT_SOLVE));
    PB_TRY(pb_dalloc_t(ctx, &ws.xb, ws.n, CAT_SOLVE));
    PB_TRY(pb_dalloc_t(ctx, &ws.axb, ws.n, CAT_SOLVE));
    ws.rec_cap = cap;
    ws.nrec = 0;
    return PB_OK;
}

// x += RU a, A x += RC a with a = RC^T (b - A x); needs ws.ax = A x
static int recycle_project(pb_ctx* ctx, gmres_ws& ws, const double* b, double* x)
{
    cudaStream_t st = ctx->stream;
    const int64_t n = ws.n;
    const int k = ws.nrec, tb = 256;
    if (k == 0 || !ws.ax_valid) return PB_OK;
    k_residual<<<pb_blocks(n, tb), tb, 0, st>>>(n, b, ws.ax, ws.r);
    PB_LAUNCH_CHECK();
    PB_TRY(dot_into(ctx, ws, k, ws.RC, ws.r, false, ws.hdev));
    k_lincomb<<<pb_blocks(n, tb), tb, k * sizeof(double), st>>>(n, k, ws.RU, n, ws.hdev, ws.u);
    PB_LAUNCH_CHECK();
    k_axpy<<<pb_blocks(n, tb), tb, 0, st>>>(n, 1.0, ws.u, x);
    PB_LAUNCH_CHECK();
    k_lincomb<<<pb_blocks(n, tb), tb, k * sizeof(double), st>>>(n, k, ws.RC, n, ws.hdev, ws.u);
    PB_LAUNCH_CHECK();
    k_axpy<<<pb_blocks(n, tb), tb, 0, st>>>(n, 1.0, ws.u, ws.ax);
    PB_LAUNCH_CHECK();
    return PB_OK;
}

// after a solve that moved x from ws.xb (with A x = ws.axb) to x (with A x = ws.ax): append the correction
static int recycle_append(pb_ctx* ctx, gmres_ws& ws, const double* x)
{
    cudaStream_t st = ctx->stream;
    const int64_t n = ws.n;
    const int k = ws.nrec, tb = 256;
    if (k >= ws.rec_cap || !ws.ax_valid) return PB_OK;
    const int nb = pb_blocks(n, tb) < 2368 ? pb_blocks(n, tb) : 2368;
    double* u = ws.RU + (size_t)k * n;
    double* c = ws.RC + (size_t)k * n;
    k_residual<<<pb_blocks(n, tb), tb, 0, st>>>(n, x, ws.xb, u);          // u = x - xb
    PB_LAUNCH_CHECK();
    k_residual<<<pb_blocks(n, tb), tb, 0, st>>>(n, ws.ax, ws.axb, c);     // c = A u
    PB_LAUNCH_CHECK();
    for (int pass = 0; pass < 2 && k > 0; ++pass) {                        // Gram-Schmidt twice against the older RC
        PB_TRY(dot_into(ctx, ws, k, ws.RC, c, false, ws.hdev));
        k_arnoldi_update<<<nb, tb, k * sizeof(double), st>>>(n, k, ws.RC, n, ws.hdev, c, nullptr, nullptr);
        PB_LAUNCH_CHECK();
        k_arnoldi_update<<<nb, tb, k * sizeof(double), st>>>(n, k, ws.RU, n, ws.hdev, u, nullptr, nullptr);
        PB_LAUNCH_CHECK();
    }
    PB_TRY(dot_into(ctx, ws, 0, nullptr, c, true, ws.hdev));               // c.c
    k_normalize<<<nb, tb, 0, st>>>(n, ws.hdev, c, c);
    PB_LAUNCH_CHECK();
    k_normalize<<<nb, tb, 0, st>>>(n, ws.hdev, u, u);
    PB_LAUNCH_CHECK();
    ws.nrec = k + 1;
    return PB_OK;
}

// ---- GCR over the whole SCF loop (pb_params.scf_recycle = 2; D: R-20) --------------------------------------------------
// The systems of the loop, A x_k = b_perm + B mu_k, share the operator.  GMRES started afresh for every one of them
// rebuilds the same slowly converging part of the Krylov space every time (measured at C4: 22 iterations per SCF step
// on average although the right-hand side changes by a factor 0.6 per step).  Here every search direction ever used is
// kept: GU[k] and GC[k] = A GU[k], the GC orthonormal (generalised conjugate residuals, Eisenstat / Elman / Schultz
// 1983, with the preconditioned residual as the new direction; flexible: the preconditioner may change from step to
// step).  A solve first takes the minimal-residual step in the stored space (one batch of dot products, no operator
// application), then adds directions until the residual is small enough:
//     z = M(r);  c = A z;  (c, z) orthogonalised against all (GC, GU) by classical Gram-Schmidt, twice, normalised;
//     alpha = c . r;  x += alpha u;  A x += alpha c;  r -= alpha c.
// A x is carried along (linearity of the operator with its fixed lists), so a solve costs exactly one operator
// application per new direction.  When the store is full the remaining work goes to restarted GMRES.
__global__ void __launch_bounds__(256)
k_gcr_orth(int64_t n, int nv, const double* __restrict__ C, const double* __restrict__ U, int64_t ld,
           const double* __restrict__ h, double* __restrict__ c, double* __restrict__ u, double* __restrict__ h2_out)
{
    extern __shared__ double sh[];
    for (int j = threadIdx.x; j < nv; j += blockDim.x) sh[j] = h[j];
    __syncthreads();
    if (h2_out && blockIdx.x == 0 && threadIdx.x == 0) {   // |h|^2: how much of c this pass removes (fixed order)
        double h2 = 0;
        for (int j = 0; j < nv; ++j) h2 = fma(sh[j], sh[j], h2);
        *h2_out = h2;
    }
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        double ac = c[e], au = u[e];
        int j = 0;
        for (; j + 4 <= nv; j += 4) {
            const double c0 = C[(int64_t)j * ld + e], c1 = C[(int64_t)(j + 1) * ld + e], c2 = C[(int64_t)(j + 2) * ld + e],
                         c3 = C[(int64_t)(j + 3) * ld + e];
            const double u0 = U[(int64_t)j * ld + e], u1 = U[(int64_t)(j + 1) * ld + e], u2 = U[(int64_t)(j + 2) * ld + e],
                         u3 = U[(int64_t)(j + 3) * ld + e];
            ac = fma(-sh[j], c0, ac); au = fma(-sh[j], u0, au);
            ac = fma(-sh[j + 1], c1, ac); au = fma(-sh[j + 1], u1, au);
            ac = fma(-sh[j + 2], c2, ac); au = fma(-sh[j + 2], u2, au);
            ac = fma(-sh[j + 3], c3, ac); au = fma(-sh[j + 3], u3, au);
        }
        for (; j < nv; ++j) { ac = fma(-sh[j], C[(int64_t)j * ld + e], ac); au = fma(-sh[j], U[(int64_t)j * ld + e], au); }
        c[e] = ac;
        u[e] = au;
    }
}

// the minimal-residual step in the stored space: x += GU a, A x += GC a, r -= GC a with a = GC^T r
__global__ void __launch_bounds__(256)
k_gcr_project(int64_t n, int nv, const double* __restrict__ C, const double* __restrict__ U, int64_t ld,
              const double* __restrict__ a, double* __restrict__ x, double* __restrict__ ax, double* __restrict__ r)
{
    extern __shared__ double sh[];
    for (int j = threadIdx.x; j < nv; j += blockDim.x) sh[j] = a[j];
    __syncthreads();
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        double sc = 0, su = 0;
        for (int j = 0; j < nv; ++j) {
            sc = fma(sh[j], C[(int64_t)j * ld + e], sc);
            su = fma(sh[j], U[(int64_t)j * ld + e], su);
        }
        x[e] += su;
        ax[e] += sc;
        r[e] -= sc;
    }
}

// d = {r . c, c . c} of the orthogonalised, not yet normalised pair: normalise (c, u), then the step along them
__global__ void __launch_bounds__(256)
k_gcr_step(int64_t n, const double* __restrict__ d, double* __restrict__ c, double* __restrict__ u, double* __restrict__ x,
           double* __restrict__ ax, double* __restrict__ r)
{
    const double cc = d[1];
    const double inv = cc > 0 ? 1.0 / sqrt(cc) : 0.0;
    const double alpha = d[0] * inv;                    // (c / |c|) . r
    for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.x * blockDim.x) {
        const double ce = c[e] * inv, ue = u[e] * inv;
        c[e] = ce;
        u[e] = ue;
        x[e] = fma(alpha, ue, x[e]);
        ax[e] = fma(alpha, ce, ax[e]);
        r[e] = fma(-alpha, ce, r[e]);
    }
}

static int gcr_alloc(pb_ctx* ctx, gmres_ws& ws)
{
    if (ws.gh || !ws.r) return PB_OK;
    // room for a few hundred directions: pb_params.scf_store_mb, 16 GB by default (C4: 493 directions of 2 x 16.6 MB); with no
    // room at all (cap 0) gcr_solve hands every system to restarted GMRES
    size_t budget = (size_t)ctx->prm.scf_store_mb << 20;
    {
        size_t free_b = 0, total_b = 0;                 // never more than half of what the device has left
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && free_b / 2 < budget) budget = free_b / 2;
    }
    size_t cap = budget / (2 * (size_t)ws.n * sizeof(double));
    if (cap > 1024) cap = 1024;
    if (cap > (size_t)ws.n) cap = (size_t)ws.n;
    PB_TRY(pb_dalloc_t(ctx, &ws.gh, cap + 16, CAT_SOLVE));
    if (cap >= 1) {
        PB_TRY(pb_dalloc_t(ctx, &ws.GU, cap * ws.n, CAT_SOLVE));
        PB_TRY(pb_dalloc_t(ctx, &ws.GC, cap * ws.n, CAT_SOLVE));
    }
    ws.gcap = (int)cap;
    ws.ngc = 0;
    return PB_OK;
}

// gh[0..k) = GC^T w, in batches of at most ws.m vectors (the size the reduction buffers were made for)
static int gcr_dots(pb_ctx* ctx, gmres_ws& ws, int k, const double* w)
{
    for (int c0 = 0; c0 < k; c0 += ws.m) {
        const int nv = k - c0 < ws.m ? k - c0 : ws.m;
        PB_TRY(dot_into(ctx, ws, nv, ws.GC + (size_t)c0 * ws.n, w, false, ws.gh + c0));
    }
    return PB_OK;
}

// One system of the SCF loop.  Needs ws.ax = A x on entry (x = 0, A x = 0 before the first one) and keeps it.
// tol_factor > 0: stop at max(gmres_tol, tol_factor * the relative residual the system starts with).
static int gcr_solve(pb_ctx* ctx, const double* b, double* x, double tol_factor, int32_t* iters_out, double* relres_out,
                     int32_t* matvecs_out, double* tol_out)
{
    pb_tree& t = ctx->tree;
    cudaStream_t st = ctx->stream;
    const int64_t n = 2 * t.N;
    const int mode = precond_mode(ctx);
    PB_TRY(ws_ensure(ctx, mode, restart_length(ctx), false));
    gmres_ws& ws = ctx->gws;
    PB_TRY(gcr_alloc(ctx, ws));
    const int tb = 256;
    const int nb = pb_blocks(n, tb) < 2368 ? pb_blocks(n, tb) : 2368;
    double* dsc = ws.gh + ws.gcap;                       // device scalars: [0] b.b, [1] r.r, [2] r.c, [3] c.c, [4] |h|^2 of the first Gram-Schmidt pass
    int iters = 0, matvecs = 0;
    k_residual<<<pb_blocks(n, tb), tb, 0, st>>>(n, b, ws.ax, ws.r);
    PB_LAUNCH_CHECK();
    PB_TRY(dot_into(ctx, ws, 0, nullptr, b, true, dsc));
    PB_TRY(dot_into(ctx, ws, 0, nullptr, ws.r, true, dsc + 1));
    double h[5] = {0, 0, 0, 0, 0};
    bool two_pass = false;
    PB_CUDA(cudaMemcpyAsync(h, dsc, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));
    const double bnorm = sqrt(h[0]);
    *iters_out = 0; *matvecs_out = 0; *tol_out = ctx->prm.gmres_tol;
    if (bnorm == 0.0) {
        PB_CUDA(cudaMemsetAsync(x, 0, sizeof(double) * n, st));
        PB_CUDA(cudaMemsetAsync(ws.ax, 0, sizeof(double) * n, st));
        ws.ax_valid = true;
        *relres_out = 0.0;
        return PB_OK;
    }
    double relres = sqrt(h[1]) / bnorm;
    // The x of the previous system already solves this one to gmres_tol: keep it.  (Late in the loop the right-hand side
    // changes by less than gmres_tol * |b|; a step in the stored space would then follow a change it cannot resolve --
    // measured at C2 with every system solved to 1e-6: the dipole change stops falling at 5e-6 D and oscillates.)
    if (relres <= ctx->prm.gmres_tol) {
        ws.ax_valid = true;
        *relres_out = relres;
        return PB_OK;
    }
    // ... and a system that does need work is solved to a quarter of gmres_tol, so that the small changes of the next
    // right-hand sides leave its x valid for them (with the target at gmres_tol itself every late step took another
    // step in the stored space: C3 needed 95 SCF steps instead of 31)
    double tol = 0.25 * ctx->prm.gmres_tol;
    if (tol_factor > 0.0 && tol_factor * relres > tol) tol = tol_factor * relres;
    if (ws.ngc > 0) {
        PB_TRY(gcr_dots(ctx, ws, ws.ngc, ws.r));
        k_gcr_project<<<nb, tb, ws.ngc * sizeof(double), st>>>(n, ws.ngc, ws.GC, ws.GU, n, ws.gh, x, ws.ax, ws.r);
        PB_LAUNCH_CHECK();
        PB_TRY(dot_into(ctx, ws, 0, nullptr, ws.r, true, dsc + 1));
        PB_CUDA(cudaMemcpyAsync(h + 1, dsc + 1, sizeof(double), cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaStreamSynchronize(st));
        relres = sqrt(h[1]) / bnorm;
    }
    int rc = PB_OK;
    while (relres > tol) {
        if (ws.ngc >= ws.gcap || iters >= ctx->prm.gmres_maxit) {
            // the store is full: restarted GMRES finishes this system from the x and A x reached so far
            int32_t gi = 0, mv = 0;
            ws.ax_valid = true;
            rc = pb_gmres_impl(ctx, b, x, &gi, &relres, &mv, true, tol);
            iters += gi;
            matvecs += mv;
            break;
        }
        double* u = ws.GU + (size_t)ws.ngc * n;
        double* c = ws.GC + (size_t)ws.ngc * n;
        if (mode == 2) PB_TRY(near_precond(ctx, ws, ws.r, u));
        else if (mode == 1) {
            k_precond<<<pb_blocks(t.N, tb), tb, 0, st>>>(t.N, t.precond, ws.r, u);
            PB_LAUNCH_CHECK();
        } else
            PB_CUDA(cudaMemcpyAsync(u, ws.r, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
        PB_TRY(pb_matvec_impl(ctx, u, c, false, false));
        ++matvecs;
        // Classical Gram-Schmidt against the stored pairs.  One pass leaves |C^T c| / |c| of the order of
        // eps |c before| / |c after| (the cancellation is what costs orthogonality; Daniel / Gragg / Kaufman / Stewart), and the
        // process needs orthogonality far below gmres_tol, not to rounding: a second pass only while the first one takes
        // c down by more than 10^4 in norm, judged from the previous direction.  Measured at C4: the first pass removes
        // between a fifth and most of |c|^2, the second changes neither iteration counts nor residuals in 9 digits and costs
        // 0.19 s of a 5.25 s solve.  x, A x and r stay consistent whatever the orthogonality: c = A u holds by linearity.
        const int npass = ws.ngc > 0 ? (two_pass ? 2 : 1) : 0;
        for (int pass = 0; pass < npass; ++pass) {
            PB_TRY(gcr_dots(ctx, ws, ws.ngc, c));
            k_gcr_orth<<<nb, tb, ws.ngc * sizeof(double), st>>>(n, ws.ngc, ws.GC, ws.GU, n, ws.gh, c, u, pass == 0 ? dsc + 4 : nullptr);
            PB_LAUNCH_CHECK();
        }
        PB_TRY(dot_into(ctx, ws, 1, ws.r, c, true, dsc + 2));              // r . c and c . c
        k_gcr_step<<<nb, tb, 0, st>>>(n, dsc + 2, c, u, x, ws.ax, ws.r);
        PB_LAUNCH_CHECK();
        PB_TRY(dot_into(ctx, ws, 0, nullptr, ws.r, true, dsc + 1));
        PB_CUDA(cudaMemcpyAsync(h, dsc, 5 * sizeof(double), cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaStreamSynchronize(st));
        ++iters;
        if (!(h[3] > 0.0)) {                            // A M(r) lies in the stored space: nothing new to add (singular operator)
            rc = pb_fail(ctx, PB_ERR_NO_CONVERGENCE, "GCR: breakdown at relative residual %.3e", relres);
            break;
        }
        two_pass = npass > 0 && h[4] > 1e8 * h[3];
        ++ws.ngc;
        relres = sqrt(h[1]) / bnorm;
    }
    if (rc == PB_OK) ws.ax_valid = true;
    *iters_out = iters;
    *relres_out = relres;
    *matvecs_out = matvecs;
    *tol_out = tol;
    return rc;
}

static int pb_solve_core(pb_ctx* ctx, double* x_out, double* mu_out, pb_result* res, bool host_out)
{
    pb_tree& t = ctx->tree;
    pb_sites& s = ctx->sites;
    cudaStream_t st = ctx->stream;
    if (!t.built || !s.loaded) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_solve: needs pb_mesh_load, pb_sites_load, pb_tree_build");
    if (!res) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_solve: NULL result");
    memset(res, 0, sizeof(*res));
    const int64_t n = 2 * t.N, na = s.na;
    // solve-scoped buffers from the scratch category (GMRES re-allocates CAT_SOLVE, so use CAT_TMP here)
    pb_dfree_cat(ctx, CAT_TMP);
    double *b, *x, *mu, *muv, *gs, *gm, *gp, *phi, *hess, *dscal;
    PB_TRY(pb_dalloc_t(ctx, &b, n, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &x, n, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &mu, 3 * na, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &muv, 3 * na, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &gs, 3 * na, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &gm, 3 * na, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &gp, 3 * na, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &phi, na, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &hess, 6 * na, CAT_TMP));
    PB_TRY(pb_dalloc_t(ctx, &dscal, 8, CAT_TMP));
    PB_CUDA(cudaMemsetAsync(x, 0, sizeof(double) * n, st));
    PB_CUDA(cudaMemsetAsync(mu, 0, sizeof(double) * 3 * na, st));
    PB_CUDA(cudaMemsetAsync(muv, 0, sizeof(double) * 3 * na, st));
    PB_CUDA(cudaMemsetAsync(dscal, 0, sizeof(double) * 8, st));
    int hflag = 0;
    k_any_nonzero<<<pb_blocks(na, 256), 256, 0, st>>>(na, s.alpha, (int*)dscal);
    PB_LAUNCH_CHECK();
    PB_CUDA(cudaMemcpyAsync(&hflag, dscal, sizeof(int), cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));
    const bool polarizable = hflag != 0;
    ctx->gws.nrec = 0;                                   // the recycled subspace belongs to one SCF loop
    const double tol = ctx->prm.scf_tol_debye, omega = ctx->prm.scf_omega;
    int status = PB_OK;
    double h[2];

    // --- vacuum SCF: mu^v from the multipole field alone
    int it_v = 0;
    if (polarizable) {
        PB_TRY(pb_multipole_field_impl(ctx, nullptr, 1, 1, nullptr, gp, nullptr));   // masked permanent field, once
        bool conv = false;
        for (it_v = 1; it_v <= ctx->prm.scf_maxit; ++it_v) {
            PB_TRY(pb_multipole_field_impl(ctx, muv, 2, 1, nullptr, gm, nullptr));
            k_scf_update<<<1, 256, 0, st>>>(na, s.alpha, nullptr, gp, gm, omega, muv, dscal);
            PB_LAUNCH_CHECK();
            PB_CUDA(cudaMemcpyAsync(h, dscal, sizeof(double), cudaMemcpyDeviceToHost, st));
            PB_CUDA(cudaStreamSynchronize(st));
            if (sqrt(h[0] / (double)na) * PB_DEBYE < tol) { conv = true; break; }
        }
        if (!conv) { status = PB_ERR_NO_CONVERGENCE; it_v = ctx->prm.scf_maxit; }
    }
    res->scf_iters_vac = it_v;

    // --- solvent SCF (steps 1-6)
    int it = 0, gm_total = 0, mv_total = 0;
    double delta = 0, relres = 0;
    bool conv = false;
    // scf_recycle = 2: one GCR process over all the systems of the loop, each solved only as far as the loop needs it
    // (a fixed reduction scf_eta of its starting residual, never below gmres_tol); the loop ends on a step that was
    // solved to gmres_tol.  1: GMRES per system, started from the stored corrections of the earlier ones.  0: plain.
    const int recycle_mode = polarizable ? ctx->prm.scf_recycle : 0;
    bool full_tol = !(ctx->prm.scf_eta > 0.0);
    if (recycle_mode == 2) {
        PB_TRY(ws_ensure(ctx, precond_mode(ctx), restart_length(ctx), false));
        ctx->gws.ngc = 0;                                            // the stored directions belong to one SCF loop
        PB_CUDA(cudaMemsetAsync(ctx->gws.ax, 0, sizeof(double) * n, st));   // x = 0, A x = 0
        ctx->gws.ax_valid = true;
    }
    for (it = 1; it <= ctx->prm.scf_maxit; ++it) {
        int32_t gi = 0, mv = 0;
        double tol_used = ctx->prm.gmres_tol;
        PB_TRY(pb_rhs_multipole(ctx, mu, b));                        // step 2: Eq. (5) with p = d + mu
        int rc = PB_OK;
        if (recycle_mode == 2) {
            rc = gcr_solve(ctx, b, x, full_tol ? 0.0 : ctx->prm.scf_eta, &gi, &relres, &mv, &tol_used);
        } else {
            const bool recycle = recycle_mode == 1;
            gmres_ws& ws = ctx->gws;
            if (recycle && it > 1) {
                PB_TRY(recycle_alloc(ctx, ws));
                PB_TRY(recycle_project(ctx, ws, b, x));              // minimal-residual step in the recycled subspace
                if (ws.xb && ws.ax_valid) {
                    PB_CUDA(cudaMemcpyAsync(ws.xb, x, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
                    PB_CUDA(cudaMemcpyAsync(ws.axb, ws.ax, sizeof(double) * n, cudaMemcpyDeviceToDevice, st));
                }
            }
            const bool had_ax = it > 1 && ws.ax_valid;
            rc = pb_gmres_impl(ctx, b, x, &gi, &relres, &mv, it > 1);
            if (rc == PB_OK && recycle && gi > 0) {
                if (it == 1) {                                       // the cold solve: x_b = 0, A x_b = 0
                    PB_TRY(recycle_alloc(ctx, ws));
                    if (ws.xb) {
                        PB_CUDA(cudaMemsetAsync(ws.xb, 0, sizeof(double) * n, st));
                        PB_CUDA(cudaMemsetAsync(ws.axb, 0, sizeof(double) * n, st));
                        PB_TRY(recycle_append(ctx, ws, x));
                    }
                } else if (ws.xb && had_ax)
                    PB_TRY(recycle_append(ctx, ws, x));
            }
        }
        if (rc == PB_ERR_NO_CONVERGENCE) status = rc; else if (rc != PB_OK) return rc;
        gm_total += gi;
        mv_total += mv;
        if (!polarizable) { conv = true; break; }
        PB_TRY(pb_reaction_field(ctx, x, nullptr, gs, nullptr));      // step 3: Eq. (13)
        PB_TRY(pb_multipole_field_impl(ctx, mu, 2, 1, nullptr, gm, nullptr));   // step 3: Eq. (14), induced part
        k_scf_update<<<1, 256, 0, st>>>(na, s.alpha, gs, gp, gm, omega, mu, dscal);   // steps 4-5 + SOR
        PB_LAUNCH_CHECK();
        PB_CUDA(cudaMemcpyAsync(h, dscal, sizeof(double), cudaMemcpyDeviceToHost, st));
        PB_CUDA(cudaStreamSynchronize(st));
        delta = sqrt(h[0] / (double)na) * PB_DEBYE;
        if (delta < tol && tol_used > ctx->prm.gmres_tol) {           // small change after an inexact solve: confirm it
            full_tol = true;                                          // with systems solved to gmres_tol from here on
            continue;
        }
        if (delta < tol) {                                            // step 6
            // surface solution consistent with the final mu
            PB_TRY(pb_rhs_multipole(ctx, mu, b));
            if (recycle_mode == 2)
                rc = gcr_solve(ctx, b, x, 0.0, &gi, &relres, &mv, &tol_used);
            else {
                if (recycle_mode == 1) PB_TRY(recycle_project(ctx, ctx->gws, b, x));
                rc = pb_gmres_impl(ctx, b, x, &gi, &relres, &mv, true);
            }
            if (rc == PB_ERR_NO_CONVERGENCE) status = rc; else if (rc != PB_OK) return rc;
            gm_total += gi;
            mv_total += mv;
            conv = true;
            break;
        }
    }
    if (!conv) { status = PB_ERR_NO_CONVERGENCE; it = ctx->prm.scf_maxit; }
    res->scf_iters = it;
    res->gmres_iters_total = gm_total;
    res->matvecs_total = mv_total;
    res->final_scf_delta_debye = delta;
    res->final_gmres_relres = relres;

    // --- energies: Delta G = G[phi_solv] + G[phi_mult(mu)] - G[phi_vac(mu^v)]   (Eq. 19, 24)
    PB_TRY(pb_reaction_field(ctx, x, phi, gs, hess));
    k_energy<<<1, 256, 0, st>>>(na, s.q, s.dip, s.quad, phi, gs, hess, dscal + 1);
    PB_LAUNCH_CHECK();
    PB_TRY(pb_multipole_field(ctx, mu, 0, phi, gm, hess));
    k_energy<<<1, 256, 0, st>>>(na, s.q, s.dip, s.quad, phi, gm, hess, dscal + 2);
    PB_LAUNCH_CHECK();
    PB_TRY(pb_multipole_field(ctx, muv, 0, phi, gm, hess));
    k_energy<<<1, 256, 0, st>>>(na, s.q, s.dip, s.quad, phi, gm, hess, dscal + 3);
    PB_LAUNCH_CHECK();
    double G[3];
    PB_CUDA(cudaMemcpyAsync(G, dscal + 1, 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (x_out)
        PB_CUDA(cudaMemcpyAsync(x_out, x, sizeof(double) * n, host_out ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, st));
    if (mu_out)
        PB_CUDA(cudaMemcpyAsync(mu_out, mu, sizeof(double) * 3 * na, host_out ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice, st));
    PB_CUDA(cudaStreamSynchronize(st));
    const double c = 4.0 * 3.14159265358979323846 * PB_KCAL;
    res->G_solvterm = c * G[0];
    res->G_mult_diss = c * G[1];
    res->G_vac = c * G[2];
    res->dG_solv = c * (G[0] + G[1] - G[2]);
    res->status = status;
    pb_dfree_cat(ctx, CAT_TMP);
    if (status != PB_OK) return pb_fail(ctx, status, "pb_solve: iteration limit reached (scf %d, gmres relres %.3e)", it, relres);
    return PB_OK;
}

extern "C" int pb_solve(pb_ctx* ctx, double* x_out, double* mu_out, pb_result* result)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    return pb_solve_core(ctx, x_out, mu_out, result, false);
}

extern "C" int pb_solve_host(pb_ctx* ctx, double* x_host, double* mu_host, pb_result* result)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    return pb_solve_core(ctx, x_host, mu_host, result, true);
}
