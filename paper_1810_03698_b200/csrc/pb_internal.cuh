// pb_internal.cuh -- shared declarations of the CUDA library behind include/pb.h.
// Product code.  Nothing here includes, links or calls anything under oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <vector>
#include <utility>

#include "../../include/pb.h"
#include "pb_device.cuh"

#define PB_INV4PI 0.079577471545947667884
#define PB_MAX_P 10
#define PB_MAX_NK_ 286   // pb_nk(PB_MAX_P)
#define PB_SITE_THETA_SCALE 0.7   // site lists: theta_site = 0.7 theta (pb_tree.cu, pb_site_lists_build)
#define PB_TG 64            // targets (panels) per target group = threads per M2P/P2P block
#define PB_KCAL 332.0636    // e^2/Angstrom -> kcal/mol (D: R-1)
#define PB_DEBYE 4.80320    // 1 e*Angstrom in Debye (D: R-1)

// Cartesian multi-index (a,b,c) -> position in a moment / coefficient array, graded by n = a+b+c
__host__ __device__ static inline int mom_index(int a, int b, int c)
{
    int n = a + b + c, m = b + c;
    return n * (n + 1) * (n + 2) / 6 + m * (m + 1) / 2 + c;
}
__host__ __device__ static constexpr int pb_nk(int P) { return (P + 1) * (P + 2) * (P + 3) / 6; }

enum pb_mem_cat { CAT_MESH = 0, CAT_SITES = 1, CAT_TREE = 2, CAT_SOLVE = 3, CAT_SITE_NEAR = 4, CAT_TMP = 5, CAT_RHS = 6, CAT_COUNT = 7 };

// Symmetric Gauss rule on the triangle (barycentric nodes, weights summing to 1) and a
// Gauss-Legendre rule on [-1,1]; passed to kernels by value.
struct pb_rule_t { int K; double lam[19][3]; double w[19]; };
struct pb_gl_t { int n; double x[64]; double w[64]; };

// One thread block's share of a target group's P2P or M2P list (pb_tree.cu).
// P2P: r = index of the first source range, a = first source point, count = source points.
// M2P: r = index of the first list entry (cell), count = cells.
struct __align__(16) pb_item { int32_t group, slot, r, a; int32_t count, pad; };

struct pb_allocation { void* ptr; size_t bytes; int cat; };

// Source-point and panel arrays in MORTON order (built by pb_tree_build).
struct pb_tree {
    bool built = false;
    int64_t N = 0, Ns = 0;
    int K = 0;
    int32_t* perm = nullptr;      // [N] Morton position -> original panel index
    // panels (SoA)
    double* pc[3] = {0, 0, 0};    // centroid
    double* pn[3] = {0, 0, 0};    // unit normal
    double* parea = nullptr;
    double* pv[9] = {0};          // vertices v0x v0y v0z v1x ...
    int32_t* ptri[3] = {0, 0, 0}; // vertex indices
    // source Gauss points (SoA), s = panel*K + g
    double* sx[3] = {0, 0, 0};
    double* swA = nullptr;        // w_g * A_j
    // per-matvec source records, 64 B per Gauss point: srec[2s] = (y_x, y_y, y_z, w A dphi),
    // srec[2s+1] = (w A phi n_x, w A phi n_y, w A phi n_z, 0)   (written by k_weights)
    double4* srec = nullptr;
    pb_expk ek;                   // constants of exp(-kappa r) for this kappa (M2P)
    pb_expk8 ek8;                 // ... with the 256-entry table (P2P)
    unsigned char* psurf = nullptr; // [N] Stern mode: 0 = the panel lies on Gamma_1, 1 = on Gamma_2 (Morton order)
    double* xphi_full = nullptr;  // [N] Stern mode: phi of every panel (xphi holds one surface's at a time)
    double* sraw = nullptr;       // [2][4][N] Stern mode: V_L, K_L, V_Y, K_Y sums over the sources of Gamma_1 / Gamma_2
    double* xphi = nullptr;       // [N] phi in Morton order
    double* xdphi = nullptr;      // [N]
    // cells
    int64_t n_cells = 0, n_leaves = 0, n_levels = 0;
    int ncrit_used = 0;           // leaf capacity in source points this tree was built with
    int32_t* c_first = nullptr;   // [cells] first panel
    int32_t* c_last = nullptr;    // one past last panel
    int32_t* c_child = nullptr;   // first child cell (-1 for leaves)
    int32_t* c_nchild = nullptr;
    double* c_ctr[3] = {0, 0, 0};
    double* c_rad = nullptr;
    double* c_box = nullptr;      // [cells][6] lo, hi
    std::vector<int64_t> gen_start; // BFS generations: cells [gen_start[g], gen_start[g+1])
    int32_t* leaf_ids = nullptr;  // [n_leaves]
    // target groups: PB_TG consecutive Morton-ordered collocation points
    int64_t n_groups = 0;
    // lists (CSR per group)
    int32_t* m2p_off = nullptr;   // [groups+1]
    int32_t* m2p_cell = nullptr;
    double4* m2p_ctr = nullptr;   // [entries] centre of m2p_cell[e] (one contiguous TMA copy per tile of cells)
    int32_t* p2p_off = nullptr;   // [groups+1]
    int32_t* p2p_lo = nullptr;    // source-point ranges [lo, hi)
    int32_t* p2p_hi = nullptr;
    int4* p2p_rng = nullptr;      // [ranges + 2] {lo, hi, mask, 0}: one 16-byte load per range for k_p2p2
    int8_t* p2p_mask = nullptr;   // [ranges] which half of the group the range is for: 1 = targets 0..31, 2 = 32..63, 3 = both (k_lists)
    int8_t* m2p_code = nullptr;   // [entries] bit 0: order P - 2; bit 3: order P - 1; bits 1-2: the same half mask (also in m2p_ctr[e].w)
    int64_t p2p_pairs = 0, m2p_pairs = 0, m2p_pairs_low = 0;   // m2p_pairs_low: those evaluated at order P - 2
    int64_t m2p_pairs_mid = 0;                                  // ... at order P - 1
    int64_t p2p_pairs_half = 0, m2p_pairs_half = 0;            // of those: pairs of entries listed for one half only
    int64_t covered_pairs = 0;    // (target, source point) pairs the STORED lists cover (k_cover_count); == N * Ns
    // far-field data
    int P = 0, Nk = 0, NT = 0;
    double* M = nullptr;          // [cells][2][Nk] Cartesian moments (V, K)
    double2* FF = nullptr;        // [cells][NT] converted far-field terms {V, K}
    int32_t* mm_off = nullptr;    // [Nk+1] M2M table (CSR over k), then [Nk] the terms by falling row length: packed (l | dx<<12 | dy<<16 | dz<<20), binomials
    int32_t* mm_ent = nullptr;
    double* mm_coef = nullptr;
    int64_t m2p_total = 0;        // entries of m2p_cell
    int64_t n_used = 0, n_need_leaf = 0, n_need_internal = 0;
    int32_t* need_leaf = nullptr;    // leaves whose moments are needed (one k_upward block each)
    int32_t* up_link = nullptr;      // [cells] bit 0: F terms wanted; bits 1..: 1 + parent if the parent needs moments
    int32_t* up_count = nullptr;     // [cells] children finished so far (self-resetting)
    unsigned char* kexp = nullptr; // [3][PB_MAX_NK_] exponents (a, b, c) of moment index k (device copy for kernels outside pb_matvec.cu)
    int32_t* cv_off = nullptr;    // [NT+1] conversion table (CSR over source moment indices)
    int32_t* cv_idx = nullptr;
    double* cv_coef = nullptr;
    double* cv_scale = nullptr;   // cv_coef with every term of layer m scaled by (2m-1)!! (combined layers of the matvec)
    // near / singular correction table (CSR per target, Morton order)
    int64_t near_entries = 0;
    // ... stored as sliced ELL: slice = 32 consecutive targets, entry k of lane l at el_base[slice] + 32 k + l
    int64_t el_entries = 0;       // padded entries
    int32_t* el_base = nullptr;   // [slices + 1]
    int32_t* el_col = nullptr;    // [el_entries] source panel (Morton); padding: the target itself
    double* el_val = nullptr;     // [4][el_entries] VL, KL, VY, KY corrections; padding: 0
    __half* el_tval = nullptr;    // [el_entries][4] (V_L, K_L, V_Y, K_Y interleaved) the true near-zone entries, rounded to fp16 (all are O(1) or smaller; 11 bits): they
                                  // only feed the near-field preconditioner, whose SpMV streams this table (a quarter of the
                                  // bytes of fp64); padding: 0
    double* precond = nullptr;    // [N][4] inverse 2x2 diagonal blocks
    // partial accumulators
    // work items (one thread block each) and their accumulator slots
    pb_item* itemP = nullptr;     // [n_itemP]
    pb_item* itemM = nullptr;     // [n_itemM]
    int32_t* itemP_off = nullptr; // [groups+1]: group g owns items/slots itemP_off[g] .. itemP_off[g+1]
    int32_t* itemM_off = nullptr;
    int64_t n_itemP = 0, n_itemM = 0;
    int nslot_p2p = 1, nslot_m2p = 1;   // largest number of items of one group
    double* accP = nullptr;       // [nslot_p2p][4][N]
    double* accM = nullptr;       // [nslot_m2p][4][N]
    // target sharding (S: section 8(e)/(f)4): this context evaluates the rows of the target groups [own_g0, own_g1)
    // = Morton panels [own_i0, own_i1); without sharding that is every group
    int64_t own_g0 = 0, own_g1 = 0, own_i0 = 0, own_i1 = 0;
    int64_t itemP0 = 0, n_itemP_own = 0, itemM0 = 0, n_itemM_own = 0;   // the owned groups' work items
    std::vector<int64_t> shard_first;   // [world + 1] first Morton panel of every rank's range
    int64_t shard_nmax = 0;             // largest number of owned panels over the ranks
    int64_t* shard_first_dev = nullptr; // device copy of shard_first
    double* ysend = nullptr;            // [2][shard_nmax] owned rows of y, Morton order (all-gather send buffer)
    double* yall = nullptr;             // [world][2][shard_nmax] gathered rows
};

// an octree over Morton-sorted items (pb_octree_build) and interaction lists against one (pb_lists_build)
struct pb_octree {
    int32_t *c_first = nullptr, *c_last = nullptr, *c_child = nullptr, *c_nchild = nullptr, *leaf_ids = nullptr;
    double *c_ctr[3] = {0, 0, 0}, *c_rad = nullptr, *c_box = nullptr;
    int64_t n_cells = 0, n_leaves = 0, n_levels = 0;
    std::vector<int64_t> gen_start;
};
struct pb_lists {
    int64_t n_groups = 0, m2p_total = 0, p2p_ranges = 0, p2p_pairs = 0, m2p_pairs = 0, covered_pairs = 0;
    int32_t *m2p_off = nullptr, *m2p_cell = nullptr, *p2p_off = nullptr, *p2p_lo = nullptr, *p2p_hi = nullptr;
};

struct pb_sites {
    bool loaded = false;
    int64_t na = 0;
    double* pos = nullptr;        // [na][3]
    double* q = nullptr;
    double* dip = nullptr;        // [na][3]
    double* quad = nullptr;       // [na][6]
    double* alpha = nullptr;
    int32_t* group = nullptr;
    // near (site, panel) pairs for the reaction field (D: R-9); built lazily
    bool near_built = false;
    int64_t n_near = 0;
    int32_t* near_site = nullptr;  // pairs sorted by (site, panel): a site's corrections are added in a fixed order
    int32_t* near_panel = nullptr; // Morton index
    int32_t* near_off = nullptr;   // [na + 1] a site's pairs are near_off[m] .. near_off[m + 1]
    // treecode for the reaction field (S: section 8(f) item 1): sites in Morton order, groups of 32, their lists,
    // and the cells whose moments those lists need (a second configuration of the upward pass)
    bool tree_built = false;
    int32_t* tperm = nullptr;      // [na] Morton position -> original site index
    double* tpos[3] = {0, 0, 0};   // [na] sorted positions (SoA)
    int64_t t_groups = 0, t_m2p_total = 0, t_p2p_pairs = 0, t_m2p_pairs = 0, t_covered_pairs = 0;
    bool inside_checked = false;   // every site has been found inside the loaded surface
    int32_t *t_m2p_off = nullptr, *t_m2p_cell = nullptr, *t_p2p_off = nullptr, *t_p2p_lo = nullptr, *t_p2p_hi = nullptr;
    int32_t* t_need_leaf = nullptr;
    int32_t* t_up_link = nullptr;
    int64_t t_n_need_leaf = 0;
    int32_t* nb_idx = nullptr;     // [Nk(P+2)][6] indices of k - e_d, k - 2 e_d (or -1) for the coefficient recurrence
    int32_t* dv_idx = nullptr;     // [10][Nk(P)] index of kappa + l
    double* dv_fac = nullptr;      // [10][Nk(P)] (-1)^|kappa| (kappa + l)! / l!
    int t_P = -1;
    // treecode for the right-hand side Eq. (8) with the SITES as sources in their own octree (S: section 8(f) item 1,
    // second half): sites in Morton order, cells, the panel groups' lists against that tree, moments and far-field terms
    bool rhs_built = false;
    int32_t* r_perm = nullptr;     // [na] Morton position -> original site index
    double* r_pos[3] = {0, 0, 0};  // [na] sorted positions (SoA)
    pb_octree r_oc;
    pb_lists r_ls;
    int32_t* r_need = nullptr;     // cells that appear in some list (one block of the moment kernel each)
    int64_t r_n_need = 0;
    double* r_FF = nullptr;        // [cells][NTp] far-field terms of the site multipoles (one layer)
    int r_NTp = 0;                 // row stride: NT rounded up to even (16-byte rows for the TMA copies)
    int r_P = -1;
};

// GMRES workspace, kept between solves while the system size and restart length are unchanged
struct pb_gmres_ws {
    int64_t n = 0;
    int m = 0;
    double *V = nullptr, *w = nullptr, *z = nullptr, *r = nullptr, *u = nullptr;
    double* ax = nullptr;         // A x of the x last returned (Arnoldi relation), valid while ax_valid
    double* Z = nullptr;          // [m][n] preconditioned basis of flexible GMRES (near-field preconditioner only)
    double *nf_r = nullptr, *nf_p = nullptr, *nf_q = nullptr, *nf_z = nullptr;   // [n] inner iteration, Morton order
    int mode = -1;                // preconditioner the workspace was sized for
    bool ax_valid = false;
    double *partial = nullptr, *hdev = nullptr, *coef = nullptr;
    unsigned int* counter = nullptr;   // arrival counter of k_dots' last-block reduction (self-resetting)
    // recycled subspace of the SCF loop (pb_params.scf_recycle): RU[k] = a past solve's correction, RC[k] = A RU[k],
    // the RC orthonormal; xb / axb = x and A x before the current solve
    double *RU = nullptr, *RC = nullptr, *xb = nullptr, *axb = nullptr;
    int nrec = 0, rec_cap = 0;
    // scf_recycle = 2: GCR with every search direction of the SCF loop kept: GU[k], GC[k] = A GU[k], the GC orthonormal;
    // gh = device scalars of the orthogonalisation (coefficients [gcap], then a few dot products)
    double *GU = nullptr, *GC = nullptr, *gh = nullptr;
    int ngc = 0, gcap = 0;
};

struct pb_ctx {
    int device = 0;
    cudaStream_t stream = 0;
    // far-field branch of the matvec (P2M, M2M, M -> F, M2P) runs here, concurrently with P2P on `stream`
    cudaStream_t side = 0;
    cudaEvent_t ev_fork = 0, ev_join = 0;
    char err[512] = {0};
    pb_alloc_fn alloc = nullptr;
    pb_free_fn free_ = nullptr;
    void* user = nullptr;
    std::vector<pb_allocation> allocs;
    size_t bytes_held = 0;
    pb_params prm;
    pb_rule_t ruleF, ruleN;       // far and near-singular rules
    pb_gl_t gl;                   // edge rule of the semi-analytic integrals (D: R-16)
    // mesh, original order
    bool mesh_loaded = false;
    int64_t nv = 0, nt = 0;
    double* verts = nullptr;      // [nv][3]
    int32_t* tris = nullptr;      // [nt][3]
    double* cen = nullptr;        // [nt][3] centroids, original order (RHS targets)
    pb_tree tree;
    pb_sites sites;
    pb_gmres_ws gws;
    // target sharding: rank / world and the exchange callback (NULL: no exchange, only the owned rows of y are written)
    int64_t stern_n1 = 0;         // > 0: panels [0, stern_n1) of the loaded mesh are Gamma_1, the rest Gamma_2 (pb_set_stern)
    double eps_stern = 0.0;
    int shard_rank = 0, shard_world = 1;
    pb_allgather_fn allgather = nullptr;
    void* allgather_user = nullptr;
    // scratch
    double* scratch = nullptr;    // small device scratch for reductions
    size_t scratch_bytes = 0;
    double* h_pinned = nullptr;   // pinned host staging
    size_t h_pinned_bytes = 0;
    int64_t matvec_calls = 0;
    int64_t launches = 0;         // kernels launched by this context
    // cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device and per function: remembered per context
    // (a context lives on one device), bit P for k_m2p2<P> / k_m2p<P>, byte counts for the others
    uint32_t attr_m2p_mask = 0;
    bool attr_p2p_set = false;
    size_t attr_up_bytes = 0, attr_site_bytes[2] = {0, 0};
    int dots_occ = 0;
    // profiling: CUDA-event pairs around every P2P and M2P launch (pb_set_profiling)
    bool profiling = false;
    std::vector<cudaEvent_t> prof_ev;   // ring: [slot][kernel 0=p2p,1=m2p][begin,end]
    std::vector<unsigned char> prof_mask;
    int prof_head = 0, prof_pending = 0;
    double prof_ms[2] = {0, 0};
    int64_t prof_launches[2] = {0, 0};
    double last_ms[8] = {0};
    cudaEvent_t ev[8] = {0};
    bool ev_made = false;
};

// ---- error handling ---------------------------------------------------------------------
int pb_fail(pb_ctx* ctx, int code, const char* fmt, ...);

#define PB_CUDA(call)                                                                          \
    do {                                                                                       \
        cudaError_t e__ = (call);                                                              \
        if (e__ != cudaSuccess)                                                                \
            return pb_fail(ctx, PB_ERR_CUDA, "%s:%d %s: %s", __FILE__, __LINE__, #call,        \
                           cudaGetErrorString(e__));                                           \
    } while (0)

#define PB_LAUNCH_CHECK()                                                                      \
    do {                                                                                       \
        ++ctx->launches;                                                                       \
        PB_CUDA(cudaGetLastError());                                                           \
    } while (0)

#define PB_TRY(call)                                                                           \
    do {                                                                                       \
        int rc__ = (call);                                                                     \
        if (rc__ != PB_OK) return rc__;                                                        \
    } while (0)

// ---- memory -----------------------------------------------------------------------------
int pb_dalloc(pb_ctx* ctx, void** out, size_t bytes, int cat);
void pb_dfree_cat(pb_ctx* ctx, int cat);
int pb_scratch(pb_ctx* ctx, size_t bytes);           // ensures ctx->scratch >= bytes
int pb_pinned(pb_ctx* ctx, size_t bytes);            // ensures ctx->h_pinned >= bytes

template <typename T>
static inline int pb_dalloc_t(pb_ctx* ctx, T** out, size_t count, int cat)
{
    return pb_dalloc(ctx, (void**)out, count * sizeof(T), cat);
}

static inline int pb_blocks(int64_t n, int threads) { return (int)((n + threads - 1) / threads); }

// ---- cross-file entry points -------------------------------------------------------------
// pb_scan.cu
int pb_exclusive_scan_i32(pb_ctx* ctx, const int32_t* in, int32_t* out, int64_t n, int64_t* total_host);
// pb_tree.cu
int pb_tree_build_impl(pb_ctx* ctx);
int pb_morton_order(pb_ctx* ctx, const double* pts, int64_t n, int cat, int32_t** perm_out, uint64_t** keys_out);
// stable LSD radix sort of n (64-bit key, int32 value) pairs on the context's stream; `bits` key bits are sorted
// (rounded up to whole bytes); k1 / v1 are scratch of the same size; the result is in (*kout, *vout) = (k0, v0) or (k1, v1)
int pb_radix_sort(pb_ctx* ctx, uint64_t* k0, uint64_t* k1, int32_t* v0, int32_t* v1, int64_t n, int bits,
                  uint64_t** kout, int32_t** vout);
int pb_cover_count(pb_ctx* ctx, int64_t G, int tg, int64_t ntargets, const int32_t* m2p_off, const int32_t* m2p_cell,
                   const int32_t* p2p_off, const int32_t* p2p_lo, const int32_t* p2p_hi, int64_t* out_host,
                   const int32_t* c_first = nullptr, const int32_t* c_last = nullptr, int K = 0,
                   const int8_t* p2p_mask = nullptr, const int8_t* m2p_code = nullptr);
int pb_lists_build(pb_ctx* ctx, int tpl, int64_t ntargets, const double* tx, const double* ty, const double* tz,
                   const pb_octree& oc, int K, int64_t Ns, double theta, int m2p_min, int cat, pb_lists* out);
int pb_octree_build(pb_ctx* ctx, const uint64_t* keys, int64_t n, int K, int ncrit, const double* px, const double* py,
                    const double* pz, int cat, pb_octree* oc);
int pb_site_lists_build(pb_ctx* ctx);
// pb_rhstree.cu
int pb_rhs_tree_build(pb_ctx* ctx);
int pb_rhs_tree(pb_ctx* ctx, const double* mu, double* b);
// pb_sitetree.cu
int pb_site_tree_build(pb_ctx* ctx);
int pb_reaction_field_tree(pb_ctx* ctx, double* phi, double* grad, double* hess);
// pb_near.cu
int pb_near_build(pb_ctx* ctx);
int pb_make_rule(int K, pb_rule_t* r);
int pb_upload_rules(pb_ctx* ctx);   // fills ctx->ruleF, ruleN, gl from the parameters
// pb_matvec.cu
int pb_farfield_setup(pb_ctx* ctx);
int pb_site_farfield_setup(pb_ctx* ctx);
// comb: the F terms as the matvec's combined layers (pb_matvec.cu, m2p_radial); the site kernels want {F^V, F^K}
int pb_upward(pb_ctx* ctx, cudaStream_t fs, const int32_t* leaf_ids, int64_t n_leaf, const int32_t* up_link, bool comb = false);
int pb_matvec_impl(pb_ctx* ctx, const double* x, double* y, bool timed, bool precond);
int pb_weights(pb_ctx* ctx, const double* x, bool precond, int surface = -1);   // surface 0 / 1: only that surface's sources
void pb_make_expk(double kappa, pb_expk* out);
int pb_make_expk8(pb_ctx* ctx, double kappa, pb_expk8* out);
// pb_sites.cu
int pb_site_near_build(pb_ctx* ctx);
int pb_check_sites_inside(pb_ctx* ctx);   // PB_ERR_BAD_MESH when a site lies outside the loaded surface
int pb_multipole_field_impl(pb_ctx* ctx, const double* mu, int parts, int use_mask, double* phi, double* grad, double* hess);
// pb_api.cu: profiling ring
int pb_prof_begin(pb_ctx* ctx, int kernel);
int pb_prof_end(pb_ctx* ctx, int kernel);
int pb_prof_drain(pb_ctx* ctx);
void pb_prof_next(pb_ctx* ctx);
// pb_solve.cu
// tol_abs > 0 replaces pb_params.gmres_tol (the inexact solves of the SCF loop)
int pb_gmres_impl(pb_ctx* ctx, const double* b, double* x, int32_t* iters, double* relres, int32_t* matvecs,
                  bool x_is_last_result, double tol_abs = 0.0);
