// pb_api.cu -- context lifetime, memory, parameters, mesh and site loading (include/pb.h).
#include <stdarg.h>
#include <math.h>
#include "pb_internal.cuh"

int pb_fail(pb_ctx* ctx, int code, const char* fmt, ...)
{
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

// ---- memory -----------------------------------------------------------------------------
int pb_dalloc(pb_ctx* ctx, void** out, size_t bytes, int cat)
{
    *out = nullptr;
    if (bytes == 0) bytes = 256;
    bytes = (bytes + 255) & ~(size_t)255;
    void* p = nullptr;
    if (ctx->alloc) {
        p = ctx->alloc(ctx->user, bytes);
        if (!p) return pb_fail(ctx, PB_ERR_ALLOC, "allocator callback returned NULL for %zu bytes", bytes);
    } else {
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e != cudaSuccess)
            return pb_fail(ctx, PB_ERR_ALLOC, "cudaMalloc(%zu) failed: %s", bytes, cudaGetErrorString(e));
    }
    ctx->allocs.push_back({p, bytes, cat});
    ctx->bytes_held += bytes;
    *out = p;
    return PB_OK;
}

void pb_dfree_cat(pb_ctx* ctx, int cat)
{
    bool any = false;
    for (auto& a : ctx->allocs) any = any || (a.cat == cat || cat < 0);
    if (any) cudaStreamSynchronize(ctx->stream);   // nothing in flight may still use the memory
    std::vector<pb_allocation> keep;
    for (auto& a : ctx->allocs) {
        if (a.cat == cat || cat < 0) {
            if (ctx->free_) ctx->free_(ctx->user, a.ptr);
            else if (!ctx->alloc) cudaFree(a.ptr);
            ctx->bytes_held -= a.bytes;
        } else
            keep.push_back(a);
    }
    ctx->allocs.swap(keep);
}

int pb_scratch(pb_ctx* ctx, size_t bytes)
{
    if (ctx->scratch_bytes >= bytes) return PB_OK;
    // scratch is allocated once, generously, outside the categories (freed at destroy)
    size_t want = bytes < ((size_t)1 << 20) ? ((size_t)1 << 20) : bytes;
    void* p;
    PB_TRY(pb_dalloc(ctx, &p, want, -2));
    ctx->scratch = (double*)p;
    ctx->scratch_bytes = want;
    return PB_OK;
}

int pb_pinned(pb_ctx* ctx, size_t bytes)
{
    if (ctx->h_pinned_bytes >= bytes) return PB_OK;
    if (ctx->h_pinned) cudaFreeHost(ctx->h_pinned);
    ctx->h_pinned = nullptr;
    ctx->h_pinned_bytes = 0;
    size_t want = bytes < 4096 ? 4096 : bytes;
    PB_CUDA(cudaMallocHost((void**)&ctx->h_pinned, want));
    ctx->h_pinned_bytes = want;
    return PB_OK;
}

// ---- lifetime -----------------------------------------------------------------------------
extern "C" void pb_default_params(pb_params* p)
{
    memset(p, 0, sizeof(*p));
    p->eps_in = 1.0;
    p->eps_out = 80.0;
    p->kappa = 0.125;
    p->theta = 0.5;
    p->order_P = 6;
    p->ncrit = 0;
    p->K_far = 7;
    p->K_near = 19;
    p->near_tau = 2.0;
    p->nq_edge = 16;
    p->precond = 3;
    p->gmres_tol = 1e-6;
    p->gmres_restart = 200;
    p->gmres_maxit = 1000;
    p->scf_tol_debye = 1e-7;
    p->scf_omega = 0.7;
    p->scf_maxit = 200;
    p->site_treecode = 2;
    p->thole_a = 0.39;
    p->rhs_treecode = 2;
    p->scf_recycle = 2;
    p->scf_eta = 0.03;
    p->scf_store_mb = 16384;
    p->list_split = 1;
}

extern "C" int pb_create(pb_ctx** out, int device, void* cuda_stream)
{
    if (!out) return PB_ERR_INVALID_ARG;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev)
        return PB_ERR_CUDA;   // no CPU fallback: without a CUDA device there is no library
    if (cudaSetDevice(device) != cudaSuccess) return PB_ERR_CUDA;
    pb_ctx* ctx = new pb_ctx();
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    pb_default_params(&ctx->prm);
    int lo = 0, hi = 0;
    bool ok = cudaDeviceGetStreamPriorityRange(&lo, &hi) == cudaSuccess &&
              cudaStreamCreateWithPriority(&ctx->side, cudaStreamNonBlocking, hi) == cudaSuccess &&
              cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) { delete ctx; return PB_ERR_CUDA; }
    *out = ctx;
    return PB_OK;
}

extern "C" int pb_destroy(pb_ctx* ctx)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    cudaStreamSynchronize(ctx->side);
    cudaStreamDestroy(ctx->side);
    cudaEventDestroy(ctx->ev_fork);
    cudaEventDestroy(ctx->ev_join);
    pb_dfree_cat(ctx, -1);
    if (ctx->h_pinned) cudaFreeHost(ctx->h_pinned);
    if (ctx->ev_made)
        for (int i = 0; i < 8; ++i) cudaEventDestroy(ctx->ev[i]);
    for (auto e : ctx->prof_ev) cudaEventDestroy(e);
    delete ctx;
    return PB_OK;
}

extern "C" const char* pb_last_error(const pb_ctx* ctx) { return ctx ? ctx->err : "null context"; }

extern "C" int pb_set_allocator(pb_ctx* ctx, pb_alloc_fn alloc, pb_free_fn free_, void* user)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (!ctx->allocs.empty())
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_set_allocator must be called before any allocation");
    ctx->alloc = alloc;
    ctx->free_ = free_;
    ctx->user = user;
    return PB_OK;
}

extern "C" int pb_get_params(const pb_ctx* ctx, pb_params* out)
{
    if (!ctx || !out) return PB_ERR_INVALID_ARG;
    *out = ctx->prm;
    return PB_OK;
}

extern "C" int pb_set_params(pb_ctx* ctx, const pb_params* p)
{
    if (!ctx || !p) return PB_ERR_INVALID_ARG;
    if (!(p->eps_in > 0) || !(p->eps_out > 0) || !(p->kappa >= 0))
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "eps_in, eps_out must be > 0 and kappa >= 0");
    if (!(p->theta >= 0) || !(p->theta < 1))
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "theta must be in [0, 1)");
    if (p->order_P < 0 || p->order_P > PB_MAX_P)
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "order_P must be in [0, %d]", PB_MAX_P);
    if (!(p->K_far == 1 || p->K_far == 3 || p->K_far == 4 || p->K_far == 7))
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "K_far must be 1, 3, 4 or 7");
    if (!(p->K_near == 1 || p->K_near == 3 || p->K_near == 4 || p->K_near == 7 || p->K_near == 19))
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "K_near must be 1, 3, 4, 7 or 19");
    if (p->ncrit < 0 || p->nq_edge < 1 || p->nq_edge > 64 || !(p->near_tau >= 0))
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "ncrit >= 0, 1 <= nq_edge <= 64, near_tau >= 0 required");
    if (p->gmres_restart < 1 || p->gmres_maxit < 1 || p->scf_maxit < 1 || !(p->gmres_tol > 0) ||
        !(p->scf_tol_debye > 0) || !(p->scf_omega > 0))
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "solver limits/tolerances must be positive");
    if (p->precond < 0 || p->precond > 3) return pb_fail(ctx, PB_ERR_INVALID_ARG, "precond must be 0, 1, 2 or 3");
    if (p->site_treecode < 0 || p->site_treecode > 2) return pb_fail(ctx, PB_ERR_INVALID_ARG, "site_treecode must be 0, 1 or 2");
    if (p->rhs_treecode < 0 || p->rhs_treecode > 2) return pb_fail(ctx, PB_ERR_INVALID_ARG, "rhs_treecode must be 0, 1 or 2");
    if (p->scf_recycle < 0 || p->scf_recycle > 2) return pb_fail(ctx, PB_ERR_INVALID_ARG, "scf_recycle must be 0, 1 or 2");
    if (!(p->scf_eta >= 0.0 && p->scf_eta < 1.0)) return pb_fail(ctx, PB_ERR_INVALID_ARG, "0 <= scf_eta < 1 required");
    if (p->scf_store_mb < 0) return pb_fail(ctx, PB_ERR_INVALID_ARG, "scf_store_mb >= 0 required");
    if (p->list_split < 0 || p->list_split > 1) return pb_fail(ctx, PB_ERR_INVALID_ARG, "list_split must be 0 or 1");
    const pb_params& o = ctx->prm;
    bool shape = o.kappa != p->kappa || o.theta != p->theta || o.order_P != p->order_P ||
                 o.ncrit != p->ncrit || o.K_far != p->K_far || o.K_near != p->K_near ||
                 o.near_tau != p->near_tau || o.nq_edge != p->nq_edge || o.eps_in != p->eps_in ||
                 o.eps_out != p->eps_out || o.list_split != p->list_split;
    const bool store = o.scf_store_mb != p->scf_store_mb;       // the solver workspace is sized by it: rebuilt on the next solve
    ctx->prm = *p;
    if (store && !(shape && ctx->tree.built)) {
        pb_dfree_cat(ctx, CAT_SOLVE);
        ctx->gws = pb_gmres_ws();
    }
    if (shape && ctx->tree.built) {
        pb_dfree_cat(ctx, CAT_TREE);
        pb_dfree_cat(ctx, CAT_SITE_NEAR);
    pb_dfree_cat(ctx, CAT_RHS);
        pb_dfree_cat(ctx, CAT_SOLVE);
        ctx->gws = pb_gmres_ws();
        ctx->tree = pb_tree();
        ctx->sites.near_built = false;
        ctx->sites.tree_built = false;
        ctx->sites.rhs_built = false;
    }
    return PB_OK;
}

// ---- target sharding (include/pb.h) ---------------------------------------------------------
extern "C" int pb_set_shard(pb_ctx* ctx, int rank, int world, pb_allgather_fn allgather, void* user)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (world < 1 || rank < 0 || rank >= world) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_set_shard: need 0 <= rank < world");
    if (world > 4096) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_set_shard: world too large");
    ctx->shard_rank = rank;
    ctx->shard_world = world;
    ctx->allgather = world > 1 ? allgather : nullptr;
    ctx->allgather_user = user;
    if (ctx->tree.built) {                      // the work items and needed cells depend on the owned range
        pb_dfree_cat(ctx, CAT_TREE);
        pb_dfree_cat(ctx, CAT_SITE_NEAR);
    pb_dfree_cat(ctx, CAT_RHS);
        pb_dfree_cat(ctx, CAT_SOLVE);
        ctx->gws = pb_gmres_ws();
        ctx->tree = pb_tree();
        ctx->sites.near_built = false;
        ctx->sites.tree_built = false;
        ctx->sites.rhs_built = false;
    }
    return PB_OK;
}

extern "C" int pb_set_stern(pb_ctx* ctx, int64_t n_inner, double eps_stern)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (!ctx->mesh_loaded) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_set_stern: call pb_mesh_load first");
    if (n_inner < 0 || n_inner >= ctx->nt) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_set_stern: need 0 <= n_inner < panels");
    if (n_inner > 0 && !(eps_stern > 0)) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_set_stern: eps_stern must be > 0");
    ctx->stern_n1 = n_inner;
    ctx->eps_stern = eps_stern;
    ctx->sites.inside_checked = false;   // with two surfaces the sites must lie inside both
    if (ctx->tree.built) {
        pb_dfree_cat(ctx, CAT_TREE);
        pb_dfree_cat(ctx, CAT_SITE_NEAR);
        pb_dfree_cat(ctx, CAT_RHS);
        pb_dfree_cat(ctx, CAT_SOLVE);
        ctx->gws = pb_gmres_ws();
        ctx->tree = pb_tree();
        ctx->sites.near_built = false;
        ctx->sites.tree_built = false;
        ctx->sites.rhs_built = false;
    }
    return PB_OK;
}

extern "C" int pb_get_shard(const pb_ctx* ctx, int64_t* first)
{
    if (!ctx || !first) return PB_ERR_INVALID_ARG;
    if (!ctx->tree.built) return PB_ERR_NOT_READY;
    for (int k = 0; k <= ctx->shard_world; ++k) first[k] = ctx->tree.shard_first[k];
    return PB_OK;
}

// ---- mesh ---------------------------------------------------------------------------------
// Per panel: centroid (v0+v1+v2)/3 = collocation point; flags degenerate panels.
__global__ void k_mesh_check(int64_t nt, int64_t nv, const double* __restrict__ verts,
                             const int32_t* __restrict__ tris, double* __restrict__ cen, int* __restrict__ bad)
{
    int64_t j = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (j >= nt) return;
    int32_t a = tris[3 * j], b = tris[3 * j + 1], c = tris[3 * j + 2];
    if (a < 0 || b < 0 || c < 0 || a >= nv || b >= nv || c >= nv) { atomicOr(bad, 1); return; }
    double v[9];
    for (int d = 0; d < 3; ++d) { v[d] = verts[3 * (int64_t)a + d]; v[3 + d] = verts[3 * (int64_t)b + d]; v[6 + d] = verts[3 * (int64_t)c + d]; }
    double e1[3], e2[3];
    for (int d = 0; d < 3; ++d) {
        e1[d] = v[3 + d] - v[d];
        e2[d] = v[6 + d] - v[d];
        cen[3 * j + d] = (v[d] + v[3 + d] + v[6 + d]) / 3.0;
    }
    double cx = e1[1] * e2[2] - e1[2] * e2[1], cy = e1[2] * e2[0] - e1[0] * e2[2], cz = e1[0] * e2[1] - e1[1] * e2[0];
    double l = sqrt(cx * cx + cy * cy + cz * cz);
    if (!(l > 0.0) || !isfinite(l)) atomicOr(bad, 2);
}

// Closedness and orientation: the 3 nt directed edges a->b as keys (min << 32 | max) with the
// direction as value; after sorting, every key must occur exactly twice, once in each direction.
__global__ void k_edge_keys(int64_t nt, const int32_t* __restrict__ tris, uint64_t* __restrict__ keys, int32_t* __restrict__ dir)
{
    const int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (e >= 3 * nt) return;
    const int64_t j = e / 3;
    const int k = (int)(e - 3 * j);
    const uint32_t a = (uint32_t)tris[3 * j + k], b = (uint32_t)tris[3 * j + (k + 1) % 3];
    keys[e] = a < b ? ((uint64_t)a << 32 | b) : ((uint64_t)b << 32 | a);
    dir[e] = a < b ? 0 : 1;
}

__global__ void k_edge_check(int64_t ne, const uint64_t* __restrict__ keys, const int32_t* __restrict__ dir, int* __restrict__ bad)
{
    const int64_t i = 2 * (blockIdx.x * (int64_t)blockDim.x + threadIdx.x);
    if (i >= ne) return;
    if (i + 1 >= ne || keys[i] != keys[i + 1] || (i > 0 && keys[i - 1] == keys[i])) { atomicOr(bad, 4); return; }   // open / non-manifold edge
    if (dir[i] == dir[i + 1]) atomicOr(bad, 8);                                                                      // inconsistent orientation
}

// enclosed volume sum_j v0.(v1 x v2)/6 (block partials, then one thread adds them in order)
__global__ void __launch_bounds__(256)
k_mesh_volume(int64_t nt, const double* __restrict__ verts, const int32_t* __restrict__ tris, double* __restrict__ partial)
{
    __shared__ double red[8];
    double s = 0;
    for (int64_t j = blockIdx.x * 256LL + threadIdx.x; j < nt; j += 256LL * gridDim.x) {
        const double* a = verts + 3 * (int64_t)tris[3 * j];
        const double* b = verts + 3 * (int64_t)tris[3 * j + 1];
        const double* c = verts + 3 * (int64_t)tris[3 * j + 2];
        s += a[0] * (b[1] * c[2] - b[2] * c[1]) + a[1] * (b[2] * c[0] - b[0] * c[2]) + a[2] * (b[0] * c[1] - b[1] * c[0]);
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0;
        for (int k = 0; k < 8; ++k) v += red[k];
        partial[blockIdx.x] = v / 6.0;
    }
}

extern "C" int pb_mesh_load(pb_ctx* ctx, const double* verts, int64_t nv, const int32_t* tris, int64_t nt)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (!verts || !tris || nv < 3 || nt < 1) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_mesh_load: empty mesh or NULL pointer");
    if (nt > (int64_t)200000000 || nv > (int64_t)2000000000) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_mesh_load: mesh too large for int32 indexing");
    PB_CUDA(cudaSetDevice(ctx->device));
    pb_dfree_cat(ctx, CAT_TREE);
    pb_dfree_cat(ctx, CAT_SITE_NEAR);
    pb_dfree_cat(ctx, CAT_RHS);
    pb_dfree_cat(ctx, CAT_SOLVE);
    ctx->gws = pb_gmres_ws();
    pb_dfree_cat(ctx, CAT_MESH);
    ctx->tree = pb_tree();
    ctx->sites.near_built = false;
        ctx->sites.tree_built = false;
        ctx->sites.rhs_built = false;
    ctx->mesh_loaded = false;
    ctx->stern_n1 = 0;             // a new mesh is one surface until pb_set_stern says otherwise
    ctx->nv = nv;
    ctx->nt = nt;
    PB_TRY(pb_dalloc_t(ctx, &ctx->verts, 3 * nv, CAT_MESH));
    PB_TRY(pb_dalloc_t(ctx, &ctx->tris, 3 * nt, CAT_MESH));
    PB_TRY(pb_dalloc_t(ctx, &ctx->cen, 3 * nt, CAT_MESH));
    PB_CUDA(cudaMemcpyAsync(ctx->verts, verts, sizeof(double) * 3 * nv, cudaMemcpyDeviceToDevice, ctx->stream));
    PB_CUDA(cudaMemcpyAsync(ctx->tris, tris, sizeof(int32_t) * 3 * nt, cudaMemcpyDeviceToDevice, ctx->stream));
    PB_TRY(pb_scratch(ctx, 1 << 20));
    int* bad = (int*)ctx->scratch;
    PB_CUDA(cudaMemsetAsync(bad, 0, sizeof(int), ctx->stream));
    k_mesh_check<<<pb_blocks(nt, 256), 256, 0, ctx->stream>>>(nt, nv, ctx->verts, ctx->tris, ctx->cen, bad);
    PB_LAUNCH_CHECK();
    int hbad = 0;
    PB_CUDA(cudaMemcpyAsync(&hbad, bad, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    PB_CUDA(cudaStreamSynchronize(ctx->stream));
    if (hbad & 1) return pb_fail(ctx, PB_ERR_BAD_MESH, "pb_mesh_load: triangle vertex index out of range");
    if (hbad & 2) return pb_fail(ctx, PB_ERR_BAD_MESH, "pb_mesh_load: degenerate (zero-area or non-finite) panel");
    {   // closed, consistently and outward oriented (S: section 8(b))
        const int64_t ne = 3 * nt;
        uint64_t *k0, *k1, *ks;
        int32_t *d0, *d1, *ds;
        PB_TRY(pb_dalloc_t(ctx, &k0, ne, CAT_TMP));
        PB_TRY(pb_dalloc_t(ctx, &k1, ne, CAT_TMP));
        PB_TRY(pb_dalloc_t(ctx, &d0, ne, CAT_TMP));
        PB_TRY(pb_dalloc_t(ctx, &d1, ne, CAT_TMP));
        k_edge_keys<<<pb_blocks(ne, 256), 256, 0, ctx->stream>>>(nt, ctx->tris, k0, d0);
        PB_LAUNCH_CHECK();
        int vbits = 1;
        while (((int64_t)1 << vbits) < nv) ++vbits;
        PB_TRY(pb_radix_sort(ctx, k0, k1, d0, d1, ne, 32 + vbits, &ks, &ds));
        PB_CUDA(cudaMemsetAsync(bad, 0, sizeof(int), ctx->stream));
        k_edge_check<<<pb_blocks((ne + 1) / 2, 256), 256, 0, ctx->stream>>>(ne, ks, ds, bad);
        PB_LAUNCH_CHECK();
        const int nvb = 256;
        double* vpart = ctx->scratch + 64;
        k_mesh_volume<<<nvb, 256, 0, ctx->stream>>>(nt, ctx->verts, ctx->tris, vpart);
        PB_LAUNCH_CHECK();
        double hv[256];
        PB_CUDA(cudaMemcpyAsync(&hbad, bad, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        PB_CUDA(cudaMemcpyAsync(hv, vpart, sizeof(hv), cudaMemcpyDeviceToHost, ctx->stream));
        PB_CUDA(cudaStreamSynchronize(ctx->stream));
        pb_dfree_cat(ctx, CAT_TMP);
        if (hbad & 4) return pb_fail(ctx, PB_ERR_BAD_MESH, "pb_mesh_load: surface not closed (an edge is not shared by exactly two panels)");
        if (hbad & 8) return pb_fail(ctx, PB_ERR_BAD_MESH, "pb_mesh_load: panels not consistently oriented (an edge is traversed twice in the same direction)");
        double vol = 0;
        for (int k = 0; k < nvb; ++k) vol += hv[k];
        if (!(vol > 0.0)) return pb_fail(ctx, PB_ERR_BAD_MESH, "pb_mesh_load: enclosed volume %.6g <= 0 (normals must point into the solvent, P:49)", vol);
    }
    ctx->mesh_loaded = true;
    ctx->sites.inside_checked = false;
    if (ctx->sites.loaded) PB_TRY(pb_check_sites_inside(ctx));
    return PB_OK;
}

// ---- sites --------------------------------------------------------------------------------
// traceless quadrupoles (Eq. 20's factor 1/6 assumes them, D: R-3) and non-negative polarizabilities
__global__ void k_sites_check(int64_t na, const double* __restrict__ quad, const double* __restrict__ alpha, int* __restrict__ bad)
{
    const int64_t m = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (m >= na) return;
    const double* Q = quad + 6 * m;
    double mx = 0;
    for (int c = 0; c < 6; ++c) mx = fmax(mx, fabs(Q[c]));
    const double tr = Q[0] + Q[3] + Q[5];
    if (!(fabs(tr) <= 1e-10 * mx)) atomicOr(bad, 1);           // also catches NaN
    if (!(alpha[m] >= 0.0)) atomicOr(bad, 2);
}

extern "C" int pb_sites_load(pb_ctx* ctx, int64_t na, const double* pos, const double* q, const double* dip,
                             const double* quad, const double* alpha, const int32_t* group)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (na < 1 || !pos || !q || !dip || !quad || !alpha || !group)
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_sites_load: na >= 1 and non-NULL arrays required");
    PB_CUDA(cudaSetDevice(ctx->device));
    pb_dfree_cat(ctx, CAT_SITE_NEAR);
    pb_dfree_cat(ctx, CAT_RHS);
    pb_dfree_cat(ctx, CAT_SITES);
    pb_sites& s = ctx->sites;
    s = pb_sites();
    s.na = na;
    PB_TRY(pb_dalloc_t(ctx, &s.pos, 3 * na, CAT_SITES));
    PB_TRY(pb_dalloc_t(ctx, &s.q, na, CAT_SITES));
    PB_TRY(pb_dalloc_t(ctx, &s.dip, 3 * na, CAT_SITES));
    PB_TRY(pb_dalloc_t(ctx, &s.quad, 6 * na, CAT_SITES));
    PB_TRY(pb_dalloc_t(ctx, &s.alpha, na, CAT_SITES));
    PB_TRY(pb_dalloc_t(ctx, &s.group, na, CAT_SITES));
    cudaStream_t st = ctx->stream;
    PB_CUDA(cudaMemcpyAsync(s.pos, pos, sizeof(double) * 3 * na, cudaMemcpyDeviceToDevice, st));
    PB_CUDA(cudaMemcpyAsync(s.q, q, sizeof(double) * na, cudaMemcpyDeviceToDevice, st));
    PB_CUDA(cudaMemcpyAsync(s.dip, dip, sizeof(double) * 3 * na, cudaMemcpyDeviceToDevice, st));
    PB_CUDA(cudaMemcpyAsync(s.quad, quad, sizeof(double) * 6 * na, cudaMemcpyDeviceToDevice, st));
    PB_CUDA(cudaMemcpyAsync(s.alpha, alpha, sizeof(double) * na, cudaMemcpyDeviceToDevice, st));
    PB_CUDA(cudaMemcpyAsync(s.group, group, sizeof(int32_t) * na, cudaMemcpyDeviceToDevice, st));
    PB_TRY(pb_scratch(ctx, 1 << 20));
    int* bad = (int*)ctx->scratch;
    int hbad = 0;
    PB_CUDA(cudaMemsetAsync(bad, 0, sizeof(int), st));
    k_sites_check<<<pb_blocks(na, 256), 256, 0, st>>>(na, s.quad, s.alpha, bad);
    PB_LAUNCH_CHECK();
    PB_CUDA(cudaMemcpyAsync(&hbad, bad, sizeof(int), cudaMemcpyDeviceToHost, st));
    PB_CUDA(cudaStreamSynchronize(st));
    if (hbad & 1) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_sites_load: a quadrupole is not traceless (Eq. 7 / Eq. 20 convention, D: R-3)");
    if (hbad & 2) return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_sites_load: negative or non-finite polarizability");
    s.loaded = true;
    if (ctx->mesh_loaded) PB_TRY(pb_check_sites_inside(ctx));
    return PB_OK;
}

// ---- setup -------------------------------------------------------------------------------
extern "C" int pb_tree_build(pb_ctx* ctx)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    if (!ctx->mesh_loaded) return pb_fail(ctx, PB_ERR_NOT_READY, "pb_tree_build: call pb_mesh_load first");
    PB_CUDA(cudaSetDevice(ctx->device));
    pb_dfree_cat(ctx, CAT_TREE);
    pb_dfree_cat(ctx, CAT_SITE_NEAR);
    pb_dfree_cat(ctx, CAT_RHS);
    pb_dfree_cat(ctx, CAT_SOLVE);
    ctx->gws = pb_gmres_ws();
    ctx->tree = pb_tree();
    ctx->sites.near_built = false;
        ctx->sites.tree_built = false;
        ctx->sites.rhs_built = false;
    ctx->attr_m2p_mask = 0;
    ctx->attr_p2p_set = false;
    ctx->attr_up_bytes = 0;
    ctx->attr_site_bytes[0] = ctx->attr_site_bytes[1] = 0;
    if (ctx->stern_n1 > 0 && ctx->shard_world > 1)
        return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_tree_build: the two-surface (Stern) system is not combined with target sharding");
    if (ctx->sites.loaded && !ctx->sites.inside_checked) PB_TRY(pb_check_sites_inside(ctx));
    PB_TRY(pb_upload_rules(ctx));
    PB_TRY(pb_tree_build_impl(ctx));
    PB_TRY(pb_farfield_setup(ctx));
    PB_TRY(pb_near_build(ctx));
    PB_CUDA(cudaStreamSynchronize(ctx->stream));
    ctx->tree.built = true;
    return PB_OK;
}

// Eq. (25)-(27): the binding cycle from three solves (host arithmetic on result structs)
extern "C" int pb_binding_cycle(const pb_result* ab, const pb_result* a, const pb_result* b, pb_binding* out)
{
    if (!ab || !a || !b || !out) return PB_ERR_INVALID_ARG;
    out->dG_bind_vac = ab->G_vac - a->G_vac - b->G_vac;          // Eq. (26), W_pol implicit in Eq. (24)
    out->ddG_bind = ab->dG_solv - a->dG_solv - b->dG_solv;       // Eq. (27)
    out->dG_bind_diss = out->ddG_bind + out->dG_bind_vac;        // Eq. (25)
    if (ab->status != PB_OK || a->status != PB_OK || b->status != PB_OK) return PB_ERR_NO_CONVERGENCE;
    return PB_OK;
}

extern "C" int pb_get_stats(pb_ctx* ctx, pb_stats* out)
{
    if (!ctx || !out) return PB_ERR_INVALID_ARG;
    memset(out, 0, sizeof(*out));
    const pb_tree& t = ctx->tree;
    out->n_panels = ctx->nt;
    out->n_sources = t.Ns;
    out->n_sites = ctx->sites.na;
    out->n_cells = t.n_cells;
    out->n_leaves = t.n_leaves;
    out->n_levels = t.n_levels;
    out->n_groups = t.n_groups;
    out->p2p_pairs = t.p2p_pairs;
    out->m2p_pairs = t.m2p_pairs;
    out->near_entries = t.near_entries;
    out->n_terms = t.NT;
    out->matvec_calls = ctx->matvec_calls;
    out->device_bytes = (int64_t)ctx->bytes_held;
    out->kernel_launches = ctx->launches;
    PB_TRY(pb_prof_drain(ctx));
    out->prof_p2p_launches = ctx->prof_launches[0];
    out->prof_m2p_launches = ctx->prof_launches[1];
    out->prof_p2p_ms = ctx->prof_ms[0];
    out->prof_m2p_ms = ctx->prof_ms[1];
    for (int i = 0; i < 8; ++i) out->last_matvec_ms[i] = ctx->last_ms[i];
    out->ncrit_used = t.ncrit_used;
    out->m2p_pairs_low = t.m2p_pairs_low;
    out->covered_pairs = t.covered_pairs;
    out->p2p_pairs_half = t.p2p_pairs_half;
    out->m2p_pairs_half = t.m2p_pairs_half;
    out->m2p_pairs_mid = t.m2p_pairs_mid;
    if (ctx->sites.rhs_built) {
        out->rhs_p2p_pairs = ctx->sites.r_ls.p2p_pairs;
        out->rhs_m2p_pairs = ctx->sites.r_ls.m2p_pairs;
        out->rhs_covered_pairs = ctx->sites.r_ls.covered_pairs;
    }
    if (ctx->sites.tree_built) {
        out->site_p2p_pairs = ctx->sites.t_p2p_pairs;
        out->site_m2p_pairs = ctx->sites.t_m2p_pairs;
        out->site_covered_pairs = ctx->sites.t_covered_pairs;
    }
    return PB_OK;
}

// ---- exclusive scan of int32 (single block, chunked; setup-time only) ---------------------
__global__ void k_scan_i32(const int32_t* __restrict__ in, int32_t* __restrict__ out, int64_t n, int64_t* total)
{
    __shared__ int32_t warp_sums[32];
    __shared__ int64_t carry_s;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (int64_t base = 0; base < n; base += blockDim.x) {
        int64_t i = base + tid;
        int32_t v = (i < n) ? in[i] : 0;
        int32_t incl = v;
        for (int o = 1; o < 32; o <<= 1) {
            int32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) warp_sums[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            int32_t w = (lane < (int)(blockDim.x >> 5)) ? warp_sums[lane] : 0;
            int32_t wi = w;
            for (int o = 1; o < 32; o <<= 1) {
                int32_t t = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += t;
            }
            warp_sums[lane] = wi - w;   // exclusive warp offsets
        }
        __syncthreads();
        int64_t carry = carry_s;
        int64_t excl = carry + warp_sums[wid] + (incl - v);
        if (i < n) out[i] = (int32_t)excl;
        __syncthreads();
        if (tid == blockDim.x - 1) carry_s = excl + v;
        __syncthreads();
    }
    if (tid == 0 && total) *total = carry_s;
}

int pb_exclusive_scan_i32(pb_ctx* ctx, const int32_t* in, int32_t* out, int64_t n, int64_t* total_host)
{
    PB_TRY(pb_scratch(ctx, 1 << 20));
    // the total lives at the END of the scratch area so callers may use its start
    int64_t* dtotal = (int64_t*)((char*)ctx->scratch + ctx->scratch_bytes - 256);
    k_scan_i32<<<1, 1024, 0, ctx->stream>>>(in, out, n, dtotal);
    PB_LAUNCH_CHECK();
    if (total_host) {
        PB_CUDA(cudaMemcpyAsync(total_host, dtotal, sizeof(int64_t), cudaMemcpyDeviceToHost, ctx->stream));
        PB_CUDA(cudaStreamSynchronize(ctx->stream));
        if (*total_host > 2147483647LL)
            return pb_fail(ctx, PB_ERR_ALLOC, "list too long for int32 offsets (%lld entries)", (long long)*total_host);
    }
    return PB_OK;
}

// ---- FP64 peak probe: independent DFMA chains, no memory traffic (roofline denominator check) --------
__global__ void __launch_bounds__(256) k_dfma_probe(int iters, double a, double b, double* __restrict__ out)
{
    double x0 = threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == 123.456) out[0] = s;   // never true; keeps the chains alive
}

extern "C" int pb_fp64_peak_probe(pb_ctx* ctx, double* tflops_out)
{
    if (!ctx || !tflops_out) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(ctx->device));
    PB_TRY(pb_scratch(ctx, 1 << 20));
    cudaEvent_t e0, e1;
    PB_CUDA(cudaEventCreate(&e0));
    PB_CUDA(cudaEventCreate(&e1));
    const int iters = 20000, blocks = 148 * 8, threads = 256;
    double best = 0;
    for (int rep = 0; rep < 4; ++rep) {
        PB_CUDA(cudaEventRecord(e0, ctx->stream));
        k_dfma_probe<<<blocks, threads, 0, ctx->stream>>>(iters, 0.999999, 1e-6, ctx->scratch);
        PB_CUDA(cudaEventRecord(e1, ctx->stream));
        PB_CUDA(cudaEventSynchronize(e1));
        float ms = 0;
        PB_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        double tf = 2.0 * 8.0 * (double)iters * blocks * threads / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *tflops_out = best;
    return PB_OK;
}

// ---- FP64 pipe probe: what the pipe sustains with few resident warps, little instruction-level parallelism, and with
// integer instructions mixed into the stream (D: section 7; profiles/r02_fp64_pipe_probes.md) ----------------------------
template <int ILP, int NI, int KIND>
__global__ void __launch_bounds__(128) k_pipe_probe(int iters, double a, double b, int c, double* __restrict__ out)
{
    double x[8], u[8], v[8];
    int y[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x * 1e-3 + i; y[i] = threadIdx.x + i; u[i] = a + 1e-9 * (threadIdx.x + i); v[i] = b * (1 + i) + 1e-15 * threadIdx.x; }   // per-thread values: vector registers, not uniform ones
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8 / ILP; ++r)
#pragma unroll
            for (int i = 0; i < ILP; ++i) {
                if (KIND == 2) x[i] = fma(x[i], u[i], v[i]);                // three DISTINCT vector registers per DFMA
                else x[i] = fma(x[i], a, b);                                // ILP independent chains, 8 DFMA per iteration; a, b shared
                if (r * ILP + i < NI) {
                    if (KIND == 0) y[i] = y[i] * c + it;                    // IMAD (FMA-heavy / integer-multiply pipe)
                    else y[i] = (y[i] ^ c) & 0x7fffffff;                    // LOP3 (ALU pipe)
                }
            }
    }
    double s = 0;
    int t = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { s += x[i] + u[i] + v[i]; t += y[i]; }
    if (s == 123.456 || t == 77) out[0] = s + t;   // never true; keeps the chains alive
}

template <int ILP, int NI, int KIND>
static cudaError_t pipe_probe_launch(int blocks, size_t smem, int iters, double* out, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(k_pipe_probe<ILP, NI, KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    k_pipe_probe<ILP, NI, KIND><<<blocks, 128, smem, st>>>(iters, 0.999999, 1e-6, 3, out);
    return cudaGetLastError();
}

extern "C" int pb_fp64_pipe_probe(pb_ctx* ctx, int warps_per_sm, int ilp, int other_per_8, int other_kind, double* pct_out)
{
    if (!ctx || !pct_out) return PB_ERR_INVALID_ARG;
    if (warps_per_sm < 4 || warps_per_sm > 64 || warps_per_sm % 4) return pb_fail(ctx, PB_ERR_INVALID_ARG, "warps_per_sm: 4 .. 64, a multiple of 4");
    PB_CUDA(cudaSetDevice(ctx->device));
    PB_TRY(pb_scratch(ctx, 1 << 20));
    int nsm = 148, mhz = 1965000;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, ctx->device);
    cudaDeviceGetAttribute(&mhz, cudaDevAttrClockRate, ctx->device);      // kHz
    const int bps = warps_per_sm / 4;                                      // blocks of 4 warps; residency limited by dynamic shared memory
    const size_t smem = (size_t)200 * 1024 / bps - 1024;
    const int iters = 20000, blocks = nsm * bps;
    cudaEvent_t e0, e1;
    PB_CUDA(cudaEventCreate(&e0));
    PB_CUDA(cudaEventCreate(&e1));
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        PB_CUDA(cudaEventRecord(e0, ctx->stream));
        cudaError_t e = cudaErrorInvalidValue;
#define PROBE_CASE(I, N, K) if (ilp == I && other_per_8 == N && other_kind == K) e = pipe_probe_launch<I, N, K>(blocks, smem, iters, ctx->scratch, ctx->stream);
        PROBE_CASE(1, 0, 0) PROBE_CASE(2, 0, 0) PROBE_CASE(4, 0, 0) PROBE_CASE(8, 0, 0)
        PROBE_CASE(8, 2, 0) PROBE_CASE(8, 4, 0) PROBE_CASE(8, 8, 0) PROBE_CASE(8, 2, 1) PROBE_CASE(8, 4, 1) PROBE_CASE(8, 8, 1)
        PROBE_CASE(8, 0, 2)
#undef PROBE_CASE
        if (e != cudaSuccess) {
            cudaEventDestroy(e0); cudaEventDestroy(e1);
            return pb_fail(ctx, PB_ERR_INVALID_ARG, "pb_fp64_pipe_probe: ilp in {1,2,4,8} with other_per_8 = 0 and kind 0, ilp = 8 with other_per_8 in {2,4,8} and kind 0|1, or (8, 0, 2)");
        }
        PB_CUDA(cudaEventRecord(e1, ctx->stream));
        PB_CUDA(cudaEventSynchronize(e1));
        float ms = 0;
        PB_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    const double inst = 8.0 * iters * (double)blocks * 128.0;
    *pct_out = 100.0 * inst / (best * 1e-3) / ((double)nsm * 64.0 * (double)mhz * 1e3);
    return PB_OK;
}

// ---- profiling ring: event pairs around the P2P / M2P launches ------------------------------------------
#define PROF_SLOTS 512
extern "C" int pb_set_profiling(pb_ctx* ctx, int on)
{
    if (!ctx) return PB_ERR_INVALID_ARG;
    PB_CUDA(cudaSetDevice(ctx->device));
    if (on && ctx->prof_ev.empty()) {
        ctx->prof_ev.resize(PROF_SLOTS * 4);
        ctx->prof_mask.assign(PROF_SLOTS, 0);
        for (auto& e : ctx->prof_ev) PB_CUDA(cudaEventCreate(&e));
    }
    PB_CUDA(cudaStreamSynchronize(ctx->stream));
    ctx->prof_head = 0;
    ctx->prof_pending = 0;
    if (on) { ctx->prof_ms[0] = ctx->prof_ms[1] = 0; ctx->prof_launches[0] = ctx->prof_launches[1] = 0; }
    ctx->profiling = on != 0;
    return PB_OK;
}

// one slot per matvec; a full ring is drained (stream sync) before it wraps
int pb_prof_drain(pb_ctx* ctx)
{
    if (ctx->prof_pending == 0) return PB_OK;
    PB_CUDA(cudaStreamSynchronize(ctx->stream));
    for (int slot = 0; slot < ctx->prof_pending; ++slot)
        for (int kern = 0; kern < 2; ++kern) {
            if (!(ctx->prof_mask[slot] & (1 << kern))) continue;
            float ms = 0;
            PB_CUDA(cudaEventElapsedTime(&ms, ctx->prof_ev[(slot * 2 + kern) * 2], ctx->prof_ev[(slot * 2 + kern) * 2 + 1]));
            ctx->prof_ms[kern] += ms;
            ctx->prof_launches[kern] += 1;
        }
    ctx->prof_pending = 0;
    ctx->prof_head = 0;
    return PB_OK;
}

int pb_prof_begin(pb_ctx* ctx, int kernel)
{
    if (!ctx->profiling) return PB_OK;
    if (ctx->prof_head >= PROF_SLOTS) PB_TRY(pb_prof_drain(ctx));
    if (ctx->prof_pending <= ctx->prof_head) { ctx->prof_mask[ctx->prof_head] = 0; ctx->prof_pending = ctx->prof_head + 1; }
    PB_CUDA(cudaEventRecord(ctx->prof_ev[(ctx->prof_head * 2 + kernel) * 2], ctx->stream));
    return PB_OK;
}

int pb_prof_end(pb_ctx* ctx, int kernel)
{
    if (!ctx->profiling) return PB_OK;
    PB_CUDA(cudaEventRecord(ctx->prof_ev[(ctx->prof_head * 2 + kernel) * 2 + 1], ctx->stream));
    ctx->prof_mask[ctx->prof_head] |= (unsigned char)(1 << kernel);
    return PB_OK;
}

void pb_prof_next(pb_ctx* ctx)
{
    if (ctx->profiling && ctx->prof_pending > ctx->prof_head) ctx->prof_head++;
}

extern "C" int pb_quadrature_rule(int K, double* lam, double* w)
{
    pb_rule_t r;
    if (!lam || !w || pb_make_rule(K, &r) != 0) return PB_ERR_INVALID_ARG;
    for (int i = 0; i < K; ++i) {
        for (int d = 0; d < 3; ++d) lam[3 * i + d] = r.lam[i][d];
        w[i] = r.w[i];
    }
    return PB_OK;
}
