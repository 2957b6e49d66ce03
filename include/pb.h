/*
 * pb.h -- C ABI of the B200-native treecode-BEM Poisson-Boltzmann hot path
 *         (arXiv:1810.03698; citations "P:<line>" = PAPER.md line, "D:" = DESIGN.md section).
 *
 * One closed triangulated molecular surface, piecewise-constant collocation BEM,
 * Yoon-Lenhoff system Eq. (5), point multipoles up to quadrupoles with induced
 * dipoles, solvation energy Eq. (19)/(24).
 *
 * Conventions
 *  - Every function returns PB_OK (0) or a negative pb_status; pb_last_error() gives a
 *    library-owned, NUL-terminated message for the last failure on that context.
 *  - Unless a parameter is marked HOST, every array argument is a DEVICE pointer owned by
 *    the caller (e.g. a torch tensor), fp64 / int32, row-major, in the caller's ORIGINAL
 *    panel and site order.  The internal Morton permutation never leaks.
 *  - Work is enqueued on the context's cudaStream_t.  Calls that return host values
 *    (pb_solve, pb_gmres, pb_get_stats, the *_host variants) synchronise that stream;
 *    pb_matvec, pb_rhs_multipole, pb_reaction_field and pb_multipole_field do not.  pb_matvec runs
 *    its far-field branch on a library-owned second stream that forks from and joins back into the
 *    context's stream, so stream order as seen by the caller is unchanged.
 *  - Device memory for internal state is obtained through the allocator callbacks
 *    (pb_set_allocator: the Python binding hands out torch tensors); with no allocator set
 *    the library falls back to cudaMalloc/cudaFree.  Memory is released by pb_destroy or
 *    when the state it belongs to is rebuilt.
 *  - Units: Angstrom, e.  Potentials carry the 1/(4 pi) of Eq. (4).  Energies in
 *    pb_result are kcal/mol: 4 pi * 332.0636 * G, G from Eq. (24) (D: R-1).
 *  - There is no CPU fallback anywhere: without a CUDA device pb_create fails.
 */
#ifndef PB_B200_H
#define PB_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pb_ctx pb_ctx;

typedef enum pb_status {
    PB_OK = 0,
    PB_ERR_INVALID_ARG = -1,
    PB_ERR_BAD_MESH = -2,       /* degenerate panel, too many panels around one vertex, surface not closed or not
                                   consistently / outward oriented, a site outside the surface (S: section 8(b)) */
    PB_ERR_NOT_READY = -3,      /* call order: mesh -> (sites) -> tree -> operators          */
    PB_ERR_CUDA = -4,
    PB_ERR_ALLOC = -5,
    PB_ERR_NO_CONVERGENCE = -6  /* GMRES or SCF hit its iteration limit (results still set)  */
} pb_status;

/* Free parameters of the method.  pb_default_params() fills the values used for
 * BASELINE.json configs[1]: eps 1/80, kappa 0.125, theta 0.5, P 6, K 7/19, tau 2. */
typedef struct pb_params {
    double eps_in;          /* eps_1, solute                                        */
    double eps_out;         /* eps_2, solvent                                                 */
    double kappa;           /* inverse Debye length, 1/Angstrom                        */
    double theta;           /* multipole acceptance parameter, Eq. (28);
                               0 => direct mode: every pair by P2P (the oracle's operator)   */
    int32_t order_P;        /* Taylor order, 0..10                                    */
    int32_t ncrit;          /* max source Gauss points per leaf cell;
                               0 (default) => built-in choice: 256 below 65,536 source points, else 128
                               (measured optimum on B200)                 */
    int32_t K_far;          /* Gauss points per panel, far rule: 1, 3, 4 or 7         */
    int32_t K_near;         /* near-singular rule: 19                                 */
    double near_tau;        /* near-singular zone |c_i-c_j| < tau*sqrt(A_i)    */
    int32_t nq_edge;        /* Gauss-Legendre points per edge, semi-analytic rule (D: R-16)   */
    int32_t precond;        /* GMRES right preconditioner: 0 none; 1 block-Jacobi (2x2 per panel from the SELF
                               entries); 2 near-field: two block-Jacobi-preconditioned minimal-residual steps on
                               the sparse matrix of the true SELF/ADJ/NEAR entries, inside flexible GMRES;
                               3 (default) = 2 from 8,000 panels up, else 1                                    */
    double gmres_tol;       /* relative residual ||b-Ax||/||b||                       */
    int32_t gmres_restart;
    int32_t gmres_maxit;
    double scf_tol_debye;   /* RMS change of induced dipoles, Debye (D: R-19)          */
    double scf_omega;       /* SOR factor, 0.7                                        */
    int32_t scf_maxit;
    int32_t site_treecode;  /* reaction field at the sites (Eq. 12, 13, 21): 0 = direct sum over all source
                               points (the paper's choice), 1 = treecode over the panel tree when
                               theta > 0 and order_P <= 8, 2 (default) = treecode when N_a * N_s >= 2^31   */
    double thole_a;         /* Thole damping constant, 0.39 (D: R-17)                  */
    int32_t rhs_treecode;   /* right-hand side Eq. (8): 0 = direct sum over all sites (the paper's choice),
                               1 = treecode with the sites as sources in their own octree (Cartesian multipole
                               moments of q, p, Q per site cell, Laplace far field at the collocation points) when
                               theta > 0, 2 (default) = treecode when N * N_a >= 2^31                          */
    int32_t scf_recycle;    /* pb_solve, how the systems A x_k = b(mu_k) of the SCF loop share work (they have one operator;
                               D: R-20).  2 (default) = one GCR process over the whole loop: every search direction u
                               with A u is kept (orthonormal A u), each system first takes the minimal-residual step in
                               the stored space and then adds directions, one operator application each, until its
                               residual has fallen by scf_eta (never below gmres_tol); up to 16 GB of directions, then
                               restarted GMRES.  1 = flexible GMRES per system, started from the minimal-residual
                               combination of the earlier systems' net corrections.  0 = GMRES per system, warm start
                               from the previous x.  Non-polarizable solves (one system) always use GMRES.          */
    int32_t list_split;     /* interaction lists of the matvec: 1 (default) = the two halves (32 consecutive
                               Morton-ordered targets each) of a 64-target group take the MAC decisions of Eq. (28)
                               separately -- a cell accepted for one half only is listed for that half alone and only the
                               other half descends to its children; 0 = one decision per group (accepted only when the
                               MAC holds for all 64 targets).  Both cover every (target, source) pair exactly once and
                               satisfy the MAC per target; 1 evaluates fewer pairs (D: section 7)                     */
    double scf_eta;         /* scf_recycle = 2: every system of the SCF loop is solved until its relative residual is
                               max(gmres_tol, scf_eta * the residual it starts with, b(mu_k) - A x_{k-1}) -- the induced
                               dipoles still change by a factor ~0.6 per step, so early systems need not be solved to
                               gmres_tol.  The loop only ends on a step whose system was solved to gmres_tol, and the
                               closing system is, too.  0 = every system to gmres_tol.  Default 0.03.               */
    int32_t scf_store_mb;   /* scf_recycle = 2: device memory for the stored directions (u and A u, 2 x 16 N bytes per
                               direction), in MiB; never more than half of the device's free memory.  When the store is
                               full the rest of the loop's work goes to restarted GMRES.  Default 16384; 0 = no store. */
} pb_params;

/* Result of one polarizable solve (HOST struct). */
typedef struct pb_result {
    double dG_solv;             /* Eq. (19): G_solvterm + G_mult_diss - G_vac, kcal/mol        */
    double G_solvterm;          /* Eq. (24) on phi_solv (reaction potential)                   */
    double G_mult_diss;         /* Eq. (24) on the multipole potential with dissolved mu       */
    double G_vac;               /* Eq. (24) on the multipole potential with vacuum mu^v        */
    double final_scf_delta_debye;
    double final_gmres_relres;
    int32_t scf_iters;
    int32_t scf_iters_vac;
    int32_t gmres_iters_total;
    int32_t matvecs_total;
    int32_t status;             /* PB_OK or PB_ERR_NO_CONVERGENCE                              */
    int32_t reserved;
} pb_result;

/* Counters and sizes of the built tree and lists (HOST struct). */
typedef struct pb_stats {
    int64_t n_panels, n_sources, n_sites;
    int64_t n_cells, n_leaves, n_levels;
    int64_t n_groups;           /* target groups (blocks of consecutive Morton-ordered panels) */
    int64_t p2p_pairs;          /* (target, source Gauss point) pairs per matvec (sharded: of the owned groups) */
    int64_t m2p_pairs;          /* (target, cell) pairs per matvec (sharded: of the owned groups)               */
    int64_t near_entries;       /* SELF+ADJ+NEAR correction-table entries                      */
    int64_t n_terms;            /* far-field terms per cell and layer (130 at P=6)             */
    int64_t matvec_calls;
    int64_t device_bytes;       /* bytes currently held through the allocator                  */
    int64_t kernel_launches;    /* kernels launched by this context so far                     */
    int64_t prof_p2p_launches;  /* with pb_set_profiling(ctx, 1): P2P launches timed so far     */
    int64_t prof_m2p_launches;
    double prof_p2p_ms;         /* ... and their summed CUDA-event durations                   */
    double prof_m2p_ms;
    double last_matvec_ms[8];   /* CUDA-event times of the last pb_matvec_timed call:
                                   0 weights, 1 P2M+M2M+convert, 2 M2P, 3 P2P, 4 near table +
                                   combine, 5 total                                            */
    int64_t ncrit_used;         /* leaf capacity the tree was built with (see pb_params.ncrit)  */
    int64_t m2p_pairs_low;      /* of m2p_pairs: those evaluated at order P - 2 (cells far inside the MAC) */
    /* Exact-cover check of the stored interaction lists: counted by a kernel that walks the lists the
     * matvec kernels read -- sum over groups of (targets in the group) x (source points in its P2P ranges + source
     * points of its M2P cells).  Every (target, source point) pair is covered exactly once iff this equals
     * n_panels * n_sources; the traversal cannot double-count (a cell is either accepted, listed as a leaf, or
     * replaced by ALL its children), so equality rules out a missed cell. */
    int64_t covered_pairs;
    int64_t site_p2p_pairs;     /* the same three counters for the site lists of the treecode reaction field       */
    int64_t site_m2p_pairs;     /* (0 until that path has been used: pb_params.site_treecode)                      */
    int64_t site_covered_pairs; /* == n_sites * n_sources when the site lists are complete                         */
    int64_t rhs_p2p_pairs;      /* RHS by the site tree (pb_params.rhs_treecode): (panel, site) pairs summed directly */
    int64_t rhs_m2p_pairs;      /* (panel, site cell) pairs through a multipole expansion                          */
    int64_t rhs_covered_pairs;  /* == n_panels * n_sites when those lists are complete                             */
    int64_t p2p_pairs_half;     /* of p2p_pairs / m2p_pairs: pairs of list entries that serve one half (32 targets) of a   */
    int64_t m2p_pairs_half;     /* 64-target group only (the two halves of a group are accepted separately)               */
    int64_t m2p_pairs_mid;      /* of m2p_pairs: those evaluated at order P - 1 (D: R-30)                                  */
} pb_stats;

typedef void* (*pb_alloc_fn)(void* user, size_t bytes);     /* returns a 256-byte aligned device pointer or NULL */
typedef void (*pb_free_fn)(void* user, void* ptr);

/* ---- lifetime ---------------------------------------------------------------------- */
int pb_create(pb_ctx** out, int device, void* cuda_stream /* cudaStream_t, may be NULL */);
int pb_destroy(pb_ctx* ctx);
const char* pb_last_error(const pb_ctx* ctx);
int pb_set_allocator(pb_ctx* ctx, pb_alloc_fn alloc, pb_free_fn free_, void* user);
void pb_default_params(pb_params* out /* HOST */);
/* Changing a parameter that shapes the operator (kappa, theta, P, ncrit, K, tau, nq_edge)
 * invalidates the tree: pb_tree_build must be called again. */
int pb_set_params(pb_ctx* ctx, const pb_params* p /* HOST */);
int pb_get_params(const pb_ctx* ctx, pb_params* out /* HOST */);

/* ---- inputs ------------------------------------------------------------------------ */
/* Closed, outward-oriented triangulated surface.  Computes per panel the
 * area, unit normal (pointing into the solvent) and centroid = collocation point.
 * verts [nv][3] fp64, tris [nt][3] int32.  The arrays are copied.  PB_ERR_BAD_MESH if an index is out of
 * range, a panel has zero area, the surface is not closed and consistently oriented (every directed edge
 * a->b must occur exactly once and be matched by exactly one b->a: checked on the device by sorting the
 * 3 nt edge keys), or its enclosed volume sum v0.(v1 x v2)/6 is not positive (normals must point into the
 * solvent).  Synchronises. */
int pb_mesh_load(pb_ctx* ctx, const double* verts, int64_t nv, const int32_t* tris, int64_t nt);

/* Point multipoles of Eq. (7): charge q [na], permanent dipole dip [na][3],
 * traceless quadrupole quad [na][6] = xx,xy,xz,yy,yz,zz in the convention of Eq. (7)
 * (potential term Q_ij d_i d_j / (2 R^5)), isotropic polarizability alpha [na] in
 * Angstrom^3 (D: R-2), polarization group [na].  Copied.  Synchronises.
 * PB_ERR_INVALID_ARG if a quadrupole is not traceless (|tr Q| > 1e-10 max|Q_ij|: Eq. (20)'s factor 1/6 assumes
 * it, D: R-3) or alpha < 0.  Every site must lie inside the surface (the interior problem of Eq. (1)):
 * checked as soon as both the mesh and the sites are loaded (here or in pb_mesh_load / pb_tree_build) through the
 * solid angle sum_j A_j n_j.(c_j - r_m)/(4 pi |c_j - r_m|^3), which is 1 inside and 0 outside a closed
 * surface; a site with less than 1/2 gives PB_ERR_BAD_MESH. */
int pb_sites_load(pb_ctx* ctx, int64_t na, const double* pos, const double* q, const double* dip,
                  const double* quad, const double* alpha, const int32_t* group);

/* Two nested surfaces / Stern layer (S: section 8(f) item 3; D: R-32).  The mesh loaded by pb_mesh_load is
 * the UNION of two closed, outward-oriented surfaces: panels [0, n_inner) form Gamma_1, the dielectric boundary that
 * encloses every site (region 1: eps_in, Laplace), the others Gamma_2 around it (the ion-exclusion surface); between
 * them lies the Stern layer (eps_stern, Laplace), outside Gamma_2 the solvent (eps_out, kappa).  x and y keep their
 * layout [phi (nt); q (nt)] over the union's panels, q being dphi/dn on the INNER side of the panel's surface, and the
 * rows become (A = sources on Gamma_1, B = on Gamma_2, r12 = eps_in/eps_stern, r23 = eps_stern/eps_out)
 *   i on Gamma_1:  y[i]      = phi_i/2 + K_L^A phi - V_L^A q
 *                  y[nt + i] = phi_i/2 - K_L^A phi + r12 V_L^A q + K_L^B phi - V_L^B q
 *   i on Gamma_2:  y[i]      = phi_i/2 + K_L^B phi - V_L^B q - K_L^A phi + r12 V_L^A q
 *                  y[nt + i] = phi_i/2 - K_Y^B phi + r23 V_Y^B q
 * (Green's second identity per region, as Eq. (2)/(5)).  pb_rhs_multipole puts Eq. (8) in the Gamma_1 rows of
 * the first block only; pb_reaction_field sums Gamma_1's layers only; pb_gmres / pb_solve work unchanged on the
 * 2 nt system (right block-Jacobi preconditioner from the SELF entries of the region pair of each surface).
 * pb_matvec evaluates the union's near and far field twice, once per source surface, through the same kernels.
 * Call after pb_mesh_load and before pb_tree_build; n_inner = 0 switches back to one surface.  Not combined with
 * pb_set_shard (PB_ERR_INVALID_ARG at pb_tree_build). */
int pb_set_stern(pb_ctx* ctx, int64_t n_inner, double eps_stern);

/* ---- setup: octree, interaction lists, near/singular table --------------- */
/* Morton-sorts the panels (63-bit key of the centroid), builds the octree over the K_far
 * Gauss points of whole panels (leaf <= ncrit points), the M2P / P2P lists of every group of 64
 * consecutive targets (a cell is accepted when the MAC of Eq. (28) holds for each target of the group),
 * and the SELF/ADJ/NEAR table (semi-analytic and K_near-point entries; both the corrections to the far
 * rule that the matvec adds and the true entries that the near-field preconditioner uses).  Needs
 * pb_mesh_load. */
int pb_tree_build(pb_ctx* ctx);

/* ---- multi-GPU: target sharding (S: section 8(e), 8(f) item 4) --------------------------------------------------
 * One process per GPU, every process with its own context holding the WHOLE problem (mesh, sites, tree, moments and
 * near table are replicated: < 5 GB at 10^6 panels) but evaluating only the rows of a contiguous Morton range of
 * target groups: the P2P / M2P work items, the needed cells of the upward pass and the combine step are restricted
 * to the owned groups.  The ranges are cut where the prefix sum of the per-group cost (P2P source points + 9 per
 * M2P cell, times the targets of the group) crosses k/world of the total, identically on every rank.
 * The ONE exchange step per matvec is an all-gather of the owned rows of y (2 x 8 bytes per owned panel; 16.6 MB in
 * total at C4) through the callback, which must enqueue the collective on the context's stream (the Python binding
 * calls torch.distributed.all_gather_into_tensor: NCCL over NVLink): `send` holds bytes_per_rank bytes, `recv`
 * world x bytes_per_rank, both device pointers owned by the library.  After it every rank holds the full y, so
 * GMRES, the SCF loop and the site-side operators run replicated and unchanged, and all ranks take identical
 * decisions (the kernels are bitwise repeatable).  With allgather == NULL nothing is exchanged and pb_matvec writes
 * ONLY the owned rows of y (original panel order), leaving the others untouched -- used to test the partition on one
 * GPU, rank after rank.  Call before pb_tree_build (it invalidates a built tree); rank 0 / world 1 switches it off. */
typedef int (*pb_allgather_fn)(void* user, const void* send, void* recv, size_t bytes_per_rank);
int pb_set_shard(pb_ctx* ctx, int rank, int world, pb_allgather_fn allgather, void* user);
/* After pb_tree_build: first [world + 1] (HOST) = first owned panel, in Morton order, of every rank. */
int pb_get_shard(const pb_ctx* ctx, int64_t* first);
/* HOST-only: the partition rule itself.  cost [G] >= 0; first [world + 1] with first[0] = 0, first[world] = G,
 * first[k] = the smallest g whose exclusive prefix sum reaches k/world of the total (ranges may be empty). */
int pb_shard_partition(const int64_t* cost, int64_t G, int world, int64_t* first);

/* ---- operators --------------------------------------------------------------------- */
/* b [2 nt]: b[0:nt] = Eq. (8) at the collocation points with p = dip + mu_induced
 * (Eq. 10; mu_induced [na][3] or NULL), b[nt:2nt] = 0. */
int pb_rhs_multipole(pb_ctx* ctx, const double* mu_induced, double* b);

/* y = A x, the left side of Eq. (5), x = [phi (nt); dphi/dn (nt)]:
 *   y[i]      = phi_i/2 + K_L phi - V_L dphi
 *   y[nt + i] = phi_i/2 - K_Y phi + (eps_in/eps_out) V_Y dphi
 * by the treecode (theta > 0) or by direct summation (theta == 0).  x != y. */
int pb_matvec(pb_ctx* ctx, const double* x, double* y);
/* Same, with CUDA events around each phase; times land in pb_stats.last_matvec_ms.  Synchronises. */
int pb_matvec_timed(pb_ctx* ctx, const double* x, double* y);
/* Same operation with HOST buffers: copies x in, runs, copies y out, synchronises. */
int pb_matvec_host(pb_ctx* ctx, const double* x_host, double* y_host);

/* Reaction potential of the surface layers at the sites, Eq. (12)
 * phi_solv = -K_L(phi) + V_L(dphi), its gradient (Eq. 13) and Hessian (Eq. 21,
 * P:195; 6-vector xx,xy,xz,yy,yz,zz).  phi [na], grad [na][3], hess [na][6]; NULL outputs
 * are skipped.  Far rule over all source points -- summed directly or, per pb_params.site_treecode, by
 * the treecode over the panel tree (the same order-P Taylor sum and MAC as the matvec, with
 * theta_site = 0.7 theta) -- and the K_near rule for panels with |r_m - c_j| < tau*sqrt(A_j) (D: R-9). */
int pb_reaction_field(pb_ctx* ctx, const double* x, double* phi, double* grad, double* hess);

/* Coulomb potential, gradient, Hessian at each site of the multipoles on all OTHER sites,
 * Eq. (7), (14), (31), (32) times 1/(4 pi eps_in), with p = dip (permanent part, dropped for
 * same-group pairs when use_mask != 0) and the induced dipoles mu [na][3] (or
 * NULL), Thole-damped, never masked. */
int pb_multipole_field(pb_ctx* ctx, const double* mu, int use_mask, double* phi, double* grad,
                       double* hess);

/* ---- solvers ----------------------------------------------------------------------- */
/* Restarted GMRES on A x = b, initial guess = x on entry.  iters/relres are HOST
 * outputs (may be NULL).  relres is ||b - A x|| / ||b||: computed explicitly at the start and at every
 * restart, and on exit taken from the Arnoldi recurrence (equal to it to rounding: right preconditioning,
 * twice-orthogonalised basis), which saves one operator application per solve. */
int pb_gmres(pb_ctx* ctx, const double* b, double* x, int32_t* iters, double* relres);

/* One polarizable solve: vacuum SCF for mu^v, then the solvent SCF
 * (rhs -> GMRES -> reaction field + multipole field -> SOR update) to scf_tol_debye, then
 * the energies.  x_out [2 nt] and mu_out [na][3] may be NULL.  result is HOST. */
int pb_solve(pb_ctx* ctx, double* x_out, double* mu_out, pb_result* result);
/* Same with HOST outputs (x_host [2 nt], mu_host [na][3], either may be NULL). */
int pb_solve_host(pb_ctx* ctx, double* x_host, double* mu_host, pb_result* result);

/* Binding thermodynamic cycle of Fig. 3 from three finished solves -- the complex AB
 * and the separate molecules A and B, each its own context / mesh / sites (HOST structs, no GPU work):
 *   dG_bind_vac  = G_vac,AB - G_vac,A - G_vac,B                        Eq. (26), the polarization energy
 *                  being implicit in Eq. (24)'s G
 *   ddG_bind     = dG_solv,AB - dG_solv,A - dG_solv,B                  Eq. (27)
 *   dG_bind_diss = ddG_bind + dG_bind_vac                              Eq. (25)
 * all in kcal/mol.  Returns PB_ERR_INVALID_ARG on NULL, PB_ERR_NO_CONVERGENCE if any of the three
 * solves carries that status (the numbers are still filled in). */
typedef struct pb_binding {
    double dG_bind_vac;
    double ddG_bind;
    double dG_bind_diss;
} pb_binding;
int pb_binding_cycle(const pb_result* ab, const pb_result* a, const pb_result* b, pb_binding* out);

int pb_get_stats(pb_ctx* ctx, pb_stats* out /* HOST */);

/* Profiling: when on, every P2P and M2P launch is bracketed by a CUDA-event pair on the
 * context's stream; pb_get_stats drains the pairs and reports summed durations and counts.
 * Turning it on resets the sums. */
int pb_set_profiling(pb_ctx* ctx, int on);

/* HOST-only helpers (no GPU needed): the library's own tables, exported so they can be tested.
 * pb_quadrature_rule: K in {1,3,4,7,19}; lam [K][3] barycentric nodes, w [K] weights (sum 1).
 * pb_gauss_legendre: n <= 64 nodes x and weights w on [-1,1].
 * pb_farfield_table: the M -> F conversion of the far field (D: section 6) for order P <= 10:
 *   returns the number of terms NT (or a negative pb_status); expo [NT][4] = (a,b,c,j) of each
 *   term; off [NT+1], idx/coef [off[NT]] the CSR combination of Cartesian moments, moment
 *   (a,b,c) living at index n(n+1)(n+2)/6 + (b+c)(b+c+1)/2 + c, n=a+b+c.  Arrays may be NULL to
 *   query sizes: *nnz_out receives off[NT]. */
int pb_quadrature_rule(int K, double* lam, double* w);
int pb_gauss_legendre(int n, double* x, double* w);
int pb_farfield_table(int P, int32_t* expo, int32_t* off, int32_t* idx, double* coef, int64_t* nnz_out);

/* Measured FP64 FMA throughput of the device in TFLOP/s (independent DFMA chains, no memory
 * traffic): the denominator check for the ALU roofline of the P2P / M2P kernels.  Synchronises. */
int pb_fp64_peak_probe(pb_ctx* ctx, double* tflops_out /* HOST */);
/* The same pipe under conditions a real kernel meets: `warps_per_sm` resident warps (4 .. 64), `ilp` independent DFMA
 * chains per thread (1, 2, 4, 8) and, with ilp = 8, `other_per_8` (0, 2, 4, 8) integer instructions per 8 DFMA of
 * `other_kind` 0 = IMAD (FMA-heavy pipe) or 1 = LOP3 (ALU pipe); (ilp 8, other_per_8 0, other_kind 2) = every DFMA with
 * three DISTINCT vector-register sources instead of two shared ones (operand bandwidth).  *pct_out = DFMA lane-instructions per second as a
 * percentage of SMs x 64 lanes x SM clock (D: section 7).  Synchronises. */
int pb_fp64_pipe_probe(pb_ctx* ctx, int warps_per_sm, int ilp, int other_per_8, int other_kind, double* pct_out /* HOST */);

/* ---- an entry point that allocates nothing -------------------------------------------------------------------------
 * pb_multipole_field (Eq. (7), (14), (31), (32)) for callers that cannot allocate: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc.  No context: every input and output is the caller's
 * DEVICE array on `device` -- pos [na][3], q [na], dip [na][3], quad [na][6] (xx,xy,xz,yy,yz,zz), alpha [na], group [na]
 * (int32), mu [na][3] or NULL, outputs phi [na], grad [na][3], hess [na][6] (each may be NULL) -- and the kernels run on
 * `cuda_stream` (a cudaStream_t of that device, NULL = the default stream) without synchronising.  Same kernels, chunking
 * and summation order as pb_multipole_field, hence the same bits.  The per-chunk partial sums live in a file-scope
 * device array of the library (510 KB, held by every GPU that loads the library until the process exits) instead of an
 * allocated scratch buffer; the call makes no cudaMalloc / cudaFree and calls no allocating routine (the array's device
 * address is looked up once per device).  Limits and sharing: na <= 4,096 sites (pb_multipole_field_static_limit),
 * more gives PB_ERR_INVALID_ARG with a message in pb_static_last_error(); ALL calls share the one array, which keeps the
 * last call's contents (nothing needs to start at zero: every element read is written first in the same call), so two
 * calls that may overlap on the GPU -- different streams without an ordering between them, or two processes' threads on
 * one device through the same library instance -- race: order them. */
int pb_multipole_field_static(int device, void* cuda_stream, int64_t na, const double* pos, const double* q,
                              const double* dip, const double* quad, const double* alpha, const int32_t* group,
                              const double* mu, double thole_a, double eps_in, int use_mask, double* phi, double* grad,
                              double* hess);
/* max_sites, scratch_bytes: HOST outputs (may be NULL) */
int pb_multipole_field_static_limit(int64_t* max_sites, int64_t* scratch_bytes);
/* message of the last failed pb_multipole_field_static call of this thread ("" if it succeeded) */
const char* pb_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PB_B200_H */
