/*
 * pff.h -- C ABI of the B200-native explicit phase-field fracture hot path.
 *
 * Implements the staggered explicit-dynamics step on linear (P1) triangles of
 * arxiv/paper_2606_23458 (section 2): fused element force + history, scatter to
 * nodes, lumped-mass velocity-Verlet update, and the matrix-free (projected) Jacobi-PCG
 * damage solve.  Every entry point cites the passage that defines the operation.
 *
 * General rules
 *  - Every function returns a pff_status code (0 = PFF_OK) except pff_mesh_destroy / pff_last_error.
 *    No exceptions, no abort.  pff_last_error() returns a thread-local, NUL-terminated
 *    description of the last failure.
 *  - "host" pointers are ordinary CPU memory, read (or written) before the call returns.
 *    "device" pointers are CUDA device memory of the GPU that was current at pff_mesh_create; every entry point makes
 *    that GPU current for its duration and restores the caller's device.  Several meshes (on one or several GPUs) may
 *    live in one process; ONE mesh must not be driven from two host threads at the same time.
 *  - The library owns the pff_mesh object and all of its workspaces.  The caller owns every
 *    state buffer (pff_state) and keeps it alive; the library never frees or reallocates it.  Every state
 *    array must be 16-byte aligned (they are sources of bulk-asynchronous copies); PFF_EINVAL otherwise.
 *  - All device work is enqueued on the CUDA stream passed to pff_mesh_create (NULL = default
 *    stream).  pff_explicit_step and pff_init_accel never synchronise; pff_damage_solve and
 *    pff_energies synchronise that stream before returning (they return host scalars).
 *  - INTERNAL ORDER.  pff_mesh_create renumbers nodes and elements (domain-decomposition /
 *    Morton order).  All device arrays in pff_state and all device
 *    vectors passed to test hooks are in internal order and in the precision of the mesh
 *    (double for PFF_F64, float for PFF_F32), SoA.  pff_mesh_permutations returns the maps;
 *    host-side index sets (Dirichlet dofs, traction edges) are given in USER numbering.
 *  - One mesh = one homogeneous material, unit thickness (energies per unit thickness,
 *    PAPER.md L225).
 */
#ifndef PFF_H
#define PFF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    PFF_OK = 0,
    PFF_EINVAL = 1,       /* null pointer, bad enum, nu outside (-1, 0.5), E/rho/Gc/l0 <= 0, dt <= 0 ... */
    PFF_EMESH = 2,        /* node index out of range, (near-)zero-area element, orphan node           */
    PFF_ENOMEM = 3,
    PFF_ECUDA = 4,        /* CUDA runtime error; text in pff_last_error()                             */
    PFF_ENOCONV = 5,      /* damage CG used max_iter mat-vecs: the result IS written                  */
    PFF_EUNSUPPORTED = 6
} pff_status;

typedef enum { PFF_AT1 = 1, PFF_AT2 = 2 } pff_model;                      /* PAPER.md L69, Eq. 6 / Eq. 8 */
typedef enum {
    PFF_SPLIT_ISOTROPIC = 0,   /* psi+ = psi (L79)                                        */
    PFF_SPLIT_SPECTRAL = 1,    /* Miehe, Eq. 2 (L71-75), closed-form 2x2 principal strains  */
    PFF_SPLIT_VOLDEV = 2,      /* Amor, Eq. 3 (L75-79), 3-D bulk modulus (L85)              */
    PFF_SPLIT_STARCONVEX = 3   /* vol-dev with gamma_star (L51, L85; reading R5)  */
} pff_split;
typedef enum { PFF_PLANE_STRAIN = 0, PFF_PLANE_STRESS = 1 } pff_plane;  /* L85 */
typedef enum { PFF_F64 = 0, PFF_F32 = 1 } pff_precision;                /* L189: fp64 is the reference */
typedef enum {
    PFF_SCATTER_GATHER = 0,    /* deterministic: chunk-local CSR gather in shared memory + ordered
                                  interface sums; bit-reproducible run to run (default)            */
    PFF_SCATTER_ATOMIC = 1     /* thread-per-element kernel with warp-aggregated floating-point atomics
                                  (the paper's atomic accumulation, L43, L124); order not reproducible  */
} pff_scatter;
typedef enum {
    PFF_ORDER_NONE = 0,       /* keep the user's element order                                             */
    PFF_ORDER_MORTON = 1,     /* elements along the Morton curve of their centroids, chunks = curve ranges  */
    PFF_ORDER_BISECTION = 2   /* Morton order, then recursive coordinate bisection into compact chunks of
                                 exactly chunk_elems elements (fewest interface nodes; default of the binding) */
} pff_order;

/* Material and model.  g(d) = (1-d)^2 + eta. */
typedef struct {
    double E, nu, rho, Gc, l0;
    double eta;          /* residual stiffness, paper value 1e-7 (L79); 0 allowed            */
    double gamma_star;   /* star-convex parameter (>= -1); ignored by the other splits        */
    int32_t model;       /* pff_model  */
    int32_t split;       /* pff_split  */
    int32_t plane;       /* pff_plane  */
} pff_material;

typedef struct {
    int32_t precision;    /* pff_precision */
    int32_t order;        /* pff_order     */
    int32_t scatter;      /* pff_scatter   */
    int32_t chunk_elems;  /* elements per chunk, 0 = library default (largest size with 3 double-buffered CTAs per SM);
                             rounded down to a multiple of 32, shrunk if one CTA would not fit shared memory */
} pff_options;

typedef struct pff_mesh pff_mesh;

/* Caller-owned device arrays, internal order, precision of the mesh.  Nodal arrays have n_nodes
 * entries, H has n_elems entries (one history value per element, R2). */
typedef struct {
    void *ux, *uy;       /* displacement u          (Eq. 16) */
    void *vx, *vy;       /* velocity v              (Eq. 18) */
    void *ax, *ay;       /* acceleration a          (Eq. 17) */
    void *d;             /* damage, in [0, 1]                 */
    void *H;             /* history max psi+  [n_elems] (L98) */
    void *fext_x, *fext_y; /* nodal external force (Eq. 17)   */
} pff_state;

/* Per-step boundary data.  dir_u / dir_v: device arrays of n_dir values (precision of the mesh),
 * ordered like the dof list given to pff_set_dirichlet; both NULL = keep the values the state holds (n_dir == 0 or
 * homogeneous data written once); exactly one of them NULL with a Dirichlet set installed is PFF_EINVAL.
 * load_scale multiplies fext in Eq. 17: S(t_{n+1}) of Eq. 19. */
typedef struct {
    const void *dir_u;   /* u_bar(t_{n+1}) */
    const void *dir_v;   /* v_bar(t_{n+1}) */
    double load_scale;
} pff_bc;

/* ---- mesh setup (Eq. 9) ------------------------------------------
 * xy[n_nodes][2] (host, fp64), tri[n_elems][3] (host, int32, either orientation: clockwise
 * elements are re-oriented, R1).  Computes areas, shape gradients (Eq. 9), inverse
 * lumped mass (L169), h_min, the renumbering, the CTA chunks and their shared-memory gather
 * tables, and uploads everything.  Input arrays are copied; *out is owned by the library.
 * options may be NULL: { PFF_F64, PFF_ORDER_BISECTION, PFF_SCATTER_GATHER, chunk_elems 0 }.
 * Errors: PFF_EINVAL (arguments/material), PFF_EMESH (bad index, degenerate element, orphan
 * node, n_nodes >= 2^30), PFF_ENOMEM, PFF_ECUDA. */
pff_status pff_mesh_create(int64_t n_nodes, const double *xy, int64_t n_elems, const int32_t *tri,
                           const pff_material *material, const pff_options *options,
                           void *cuda_stream, pff_mesh **out);
void pff_mesh_destroy(pff_mesh *mesh);

/* h_min = minimum element incircle diameter; dt_crit = h_min / c_p with
 * c_p = sqrt((lambda + 2 mu) / rho) (L169; the caller applies the safety factor alpha).
 * n_chunks / n_shared_nodes describe the decomposition (may be NULL). */
pff_status pff_mesh_info(const pff_mesh *mesh, int64_t *n_nodes, int64_t *n_elems, double *h_min,
                         double *dt_crit, int64_t *n_chunks, int64_t *n_shared_nodes);

/* node_new_of_old[n_nodes], elem_new_of_old[n_elems] (host, may be NULL): internal index of
 * each user node / element. */
pff_status pff_mesh_permutations(const pff_mesh *mesh, int32_t *node_new_of_old, int32_t *elem_new_of_old);

/* Host-only dry run of the mesh setup (no CUDA call): validates the mesh exactly like pff_mesh_create
 * and returns the renumbering and the decomposition statistics.  Any output pointer may be NULL. */
pff_status pff_mesh_plan(int64_t n_nodes, const double *xy, int64_t n_elems, const int32_t *tri,
                         const pff_options *options, int32_t *node_new_of_old, int32_t *elem_new_of_old,
                         int64_t *n_chunks, int64_t *n_shared_nodes, int32_t *chunk_elems, int32_t *max_local_nodes,
                         double *h_min);

/* Displacement Dirichlet set (Eq. 5): dir_dof[n_dir] (host, USER numbering, 2*node + comp).
 * Replaces any previous set.  Values come per step through pff_bc. */
pff_status pff_set_dirichlet(pff_mesh *mesh, int64_t n_dir, const int32_t *dir_dof);

/* Damage Dirichlet set: nodes[n] (host, USER numbering) keep the value found in state->d during
 * pff_damage_solve (notches / seeds, R14).  Replaces any previous set. */
pff_status pff_set_damage_dirichlet(pff_mesh *mesh, int64_t n, const int32_t *nodes);

/* Traction boundary (Eq. 5): edge_nodes[n_edges][2] (host, USER ids), t[n_edges][2] (host, force per
 * unit length ... per unit thickness, i.e. Pa).  OVERWRITES state->fext_x/y with the consistent
 * nodal load sum t L / 2 per end node (R8). */
pff_status pff_set_traction(pff_mesh *mesh, pff_state *state, int64_t n_edges, const int32_t *edge_nodes,
                            const double *t);

/* a_0 = m^-1 (S f_ext - f_int(u_0, d_0)), zero on Dirichlet dofs (Eq. 17 at t = 0); u, v, H untouched. */
pff_status pff_init_accel(pff_mesh *mesh, pff_state *state, const pff_bc *bc);

/* One explicit step n -> n+1 with d fixed:
 *   Eq. 16 predictor, Dirichlet overwrite; element strain -> split -> degraded stress -> internal
 *   force (L42, L71-93, L124); scatter to nodes; Eq. 17; Eq. 18; H <- max(H, psi+) (L98, L114).
 * On return (stream order) state holds (u, v, a, H)_{n+1}.  Asynchronous.  dt > 0. */
pff_status pff_explicit_step(pff_mesh *mesh, pff_state *state, const pff_bc *bc, double dt);

/* Damage solve for d_{n+1} from H_{n+1}, warm-started at d_n = state->d:
 * matrix-free operator with consistent mass (L173, L185), Jacobi preconditioner (L177),
 * AT2: PCG then d <- min(1, max(d_n, d)) (L179); AT1: projected PCG with lower bound d_n (L181).
 * Stops when ||r_free||_2 <= rel_tol * max(||b||_2, ||b - A d_n||_2) (R10) or after max_iter
 * operator applications (then returns PFF_ENOCONV with the result written).
 * iters_out / relres_out (host, may be NULL) receive the mat-vec count and final relative residual.
 * Device work: ONE setup kernel (rhs, Jacobi diagonal, first residual, operator coefficients) and ONE kernel that runs
 * every CG iteration, both cooperative launches (the GPU must support them and must not be shared with other kernels
 * of the same stream priority during the call).  Synchronises the stream. */
pff_status pff_damage_solve(pff_mesh *mesh, pff_state *state, double rel_tol, int32_t max_iter,
                            int32_t *iters_out, double *relres_out);

/* out = { E_el, E_kin, E_frac, E_tot } per unit thickness (Eq. 1), accumulated in fp64
 * with a fixed reduction order.  Synchronises the stream. */
pff_status pff_energies(pff_mesh *mesh, const pff_state *state, double out[4]);

/* pff_energies for callers that may not allocate device memory (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): the same three kernels, the same fixed reduction order and the same bits, but
 *   - the block partials live in a static device array of the library (2^17 doubles = 1 MiB, held by every GPU that
 *     loads the library until the process exits) instead of a stream-ordered allocation; its device address is looked
 *     up once per GPU at pff_mesh_create (cudaGetSymbolAddress: a lookup, no allocation);
 *   - out_device (DEVICE, 4 doubles, 8-byte aligned, caller-owned) receives { E_el, E_kin, E_frac, E_tot };
 *   - the call only enqueues three kernels on the mesh's stream: no cudaMalloc / cudaFree / allocating library call, no
 *     copy, no synchronisation.  Read out_device in stream order.
 * Limit: 2 ceil(n_elems / 256) + ceil(n_nodes / 256) <= 131072 (about 1.3e7 elements); larger meshes return
 * PFF_EUNSUPPORTED with the numbers in pff_last_error() and must use pff_energies.
 * The array is shared by ALL meshes and calls of the process on that GPU and keeps the last call's contents (every word
 * a call reads it has written before, so nothing needs clearing): calls whose kernels could overlap on the GPU (two
 * streams, two host threads) race on it and must be serialised by the caller. */
pff_status pff_energies_static(pff_mesh *mesh, const pff_state *state, double *out_device);

/* ---- geometric-multigrid-preconditioned damage solve (a preconditioner stronger
 * than Jacobi cuts the CG iteration count 5-20x on fine meshes, where the count grows like l0 / h) ------------------------
 * pff_mg_attach: coarse[0 .. n_coarse) are ordinary meshes of the SAME domain, material, precision, device and stream,
 * finest first, each coarser than the one before (any triangulations: every node and element centroid of a level must lie
 * in a triangle of the next one; nested refinements give the best transfer).  The library builds the P1 interpolation
 * between consecutive levels (point location, barycentric weights), its transpose and the parent element of every element
 * on the host and uploads them.  The caller keeps the coarse meshes alive while the hierarchy is attached and destroys
 * them itself; attaching again replaces the hierarchy; pff_mesh_destroy(mesh) releases it.
 * n_coarse = 0 is allowed: the "cycle" is then `coarse_sweeps` damped-Jacobi sweeps on the mesh itself (a polynomial
 * preconditioner, no coarse meshes needed) -- of interest for AT1, whose active-set outer method (below) does not depend
 * on the hierarchy.
 * Errors: PFF_EINVAL (arguments), PFF_EMESH (a node outside the next level's triangles), PFF_ECUDA. */
pff_status pff_mg_attach(pff_mesh *mesh, int32_t n_coarse, pff_mesh *const *coarse);

/* Smoother weight (damped Jacobi, default 2/3; 0 < omega < 1 keeps the cycle positive definite for P1 mass + stiffness,
 * lambda_max(D^-1 A) <= 2) and the number of Jacobi sweeps that stand for the coarsest-level solve (default 4). */
pff_status pff_mg_set_params(pff_mesh *mesh, double omega, int32_t coarse_sweeps);

/* pff_damage_solve with one V(1,1) cycle per iteration as the preconditioner:
 *   level l:  x = w D^-1 b;  r = b - A x;  x += P V_{l+1}(P^T r);  x += w D^-1 (b - A x);   coarsest: Jacobi sweeps.
 * Coarse operators are re-discretised: the operator (Gc / l0 + 2 H) M + Gc l0 K (L173, L185) of the coarse mesh with H
 * averaged over every coarse element's children (area weights).  Same right-hand side, warm start, damage-Dirichlet
 * nodes, stopping rule (R10) and final clamp d <- min(1, max(d_n, d)) (L179) as pff_damage_solve, and the same
 * unique solution: only the iteration count differs.  iters_out counts outer iterations (one V-cycle + one operator
 * application each; a V-cycle costs about 2.7 fine-level operator applications).
 * AT1 (L181: min 1/2 d'Ad - b'd subject to d >= d_n): a primal-dual active set method around that solve.  With
 * r = b - A d, a node is ACTIVE when r / D + (d - d_n) < 0: it is put on its bound; the inactive nodes solve their linear
 * system by the multigrid-preconditioned CG above (the active nodes masked on the finest level like damage-Dirichlet
 * nodes; inexactly, residual x 0.3, while the sets still move); the sets are re-derived until they stop changing and the
 * inactive residual meets the tolerance: the KKT point, i.e. the same unique solution as pff_damage_solve's projected CG
 * (which truncates every step at the first bound hit, restarts, and needs thousands of passes when damage is widespread).
 * pff_damage_last_stats then reports the active-set steps as `restarts`.  Synchronises the stream every iteration (host-side convergence test);
 * bit-reproducible run to run.  Pays off where l0 / h is large (profiles/r2_multigrid.md); pff_damage_solve and
 * pff_run_steps use it after pff_set_damage_solver(mesh, 1). */
pff_status pff_damage_solve_mg(pff_mesh *mesh, pff_state *state, double rel_tol, int32_t max_iter,
                               int32_t *iters_out, double *relres_out);

/* Which solver pff_damage_solve and pff_run_steps use for this mesh: 0 (default) the Jacobi-PCG kernels, 1 the
 * multigrid-preconditioned solver above (needs an attached hierarchy: PFF_EINVAL otherwise; AT2: PCG, AT1: primal-dual
 * active set around it).
 * With solver 1, pff_run_steps launches every kernel itself (no graph replay of a period: the solver tests convergence on
 * the host) and its iteration total counts outer multigrid iterations.  pff_mg_attach replacing the hierarchy keeps the
 * choice.  pff_damage_adjoint follows the choice as well, for AT1 and AT2 alike (it is a linear solve on a given free set:
 * nodes outside it are masked on the finest level like damage-Dirichlet nodes). */
pff_status pff_set_damage_solver(pff_mesh *mesh, int32_t solver);

/* Test hook: z = V(r), one cycle of the preconditioner with the operator of state->H; r, z device [n_nodes]. */
pff_status pff_mg_apply(pff_mesh *mesh, const pff_state *state, const void *r, void *z);

/* Which kernel runs the CG iterations of pff_damage_solve / pff_damage_adjoint.
 *   1: the two-rendezvous kernel (standard Jacobi-PCG recurrence with predicted beta; interface nodes summed in a phase of
 *      their own between two grid barriers per iteration).  AT1 (projected CG, L181) always runs it.
 *   2: the ONE-rendezvous kernel wherever it applies (unconstrained solves -- AT2, adjoint -- on meshes without overflow
 *      partial slots): Chronopoulos-Gear form of CG, the operator is applied to z = D^-1 r, s = A p follows by recurrence,
 *      both inner products are linear in the applied operator, so the interface sums are deferred into the next pass: one
 *      grid barrier per pass, no interface phase, one pass more per solve.
 *   0 (default): chosen per solve from measurements on B200 (profiles/r2_cg_kernels.md): kernel 2 where it applies and a
 *      CTA of the persistent grid owns at most 16 chunks (up to ~1.4e6 nodes in fp64); kernel 1 otherwise (on larger meshes
 *      the grid-wide tail is amortised and the extra pass costs more than the shorter passes save).
 * Both converge to the same unique solution (same iterates in exact arithmetic); both are bit-reproducible run to run. */
pff_status pff_set_cg_variant(pff_mesh *mesh, int32_t variant);
/* kernel <- 1 / 2: which of the two the last solve of this mesh launched (0: none yet).  Host-only. */
pff_status pff_last_cg_kernel(const pff_mesh *mesh, int32_t *kernel);

/* pff_run_steps: the explicit step that precedes a damage solve also performs that solve's SETUP PASS (right-hand side,
 * Jacobi diagonal, first residual, operator coefficients, norms, control block) in the same kernel: everything the pass
 * reads -- connectivity, geometry, area, the new history value, d -- is already in the step kernel's shared memory, so
 * the separate setup kernel with its 120 MB of re-reads disappears (two kernels per staggered step instead of three).
 * Same arithmetic in the same order: results are bit-identical to the three-kernel sequence.  Used where it applies:
 * gather scatter, Jacobi solver; enable = 0 switches it off (A/B timing).  pff_explicit_step + pff_damage_solve (one call
 * each) always run the separate kernels.  used <- whether the last pff_run_steps fused.  Host-only. */
pff_status pff_set_fused_setup(pff_mesh *mesh, int32_t enable);
pff_status pff_fused_setup_used(const pff_mesh *mesh, int32_t *used);

/* Counters of the last pff_damage_solve / pff_damage_adjoint of this mesh (of ALL solves of the last pff_run_steps):
 * restarts = how often the projected solver (AT1, L181) re-derived its free set after the first time (a bound became
 * inactive, or a step was truncated); truncations = steps cut short at the first bound hit.  Both 0 for AT2.
 * Host-only (reads what the solve already downloaded).  Either pointer may be NULL. */
pff_status pff_damage_last_stats(const pff_mesh *mesh, int32_t *restarts, int32_t *truncations);

/* ---- damage subcycling ---------------------------------------
 * Admissible subcycling factor N_max = floor(c_p / (0.6 c_R)): the damage front moves at <= ~0.6 c_R while the explicit
 * step is limited by c_p.  c_p = sqrt((lambda + 2 mu) / rho) with the plane-assumption lambda (as in the CFL step,
 * DESIGN.md R19), c_s = sqrt(mu / rho), c_R = c_s (0.862 + 1.14 nu) / (1 + nu) (Bergmann-Viktorov approximation of the
 * Rayleigh speed; the paper does not print its formula: DESIGN.md R22).  Host-only, no CUDA call.  ratio (may be NULL)
 * receives the continuous value c_p / (0.6 c_R).  PMMA-like nu = 0.35 gives N_max = 3 (the paper's printed value). */
pff_status pff_subcycle_limit(const pff_material *material, int32_t *n_max, double *ratio);

/* n_steps staggered steps on DEVICE-RESIDENT state (no host copies): pff_explicit_step every step (so the history
 * field and irreversibility follow the mechanical time scale, L187) and pff_damage_solve every damage_every-th step
 * (0 = never; 1 = the plain staggered scheme of L114).  Constant boundary data bc.  cg_iters_total (host, may be NULL)
 * receives the summed CG iterations.  Returns PFF_ENOCONV if any solve did (results are written).  Synchronises once,
 * at the end: the solves tally their counters on the device. */
pff_status pff_run_steps(pff_mesh *mesh, pff_state *state, const pff_bc *bc, double dt, int64_t n_steps,
                         int32_t damage_every, double rel_tol, int32_t max_iter, int64_t *cg_iters_total);
/* pff_run_steps replays one captured period of the loop (damage_every steps + one solve) from a CUDA graph when the run
 * has at least four periods (SURVEY.md 8(f) NEXT-1 "whole-step CUDA graph": what small, launch-bound meshes need,
 * PAPER.md L466).  The result is bit-identical to plain launches.  enable = 0 switches the capture off (A/B timing);
 * it is also skipped while pff_profile_enable is on, and for good once the driver has refused to capture a launch. */
pff_status pff_set_graph_mode(pff_mesh *mesh, int32_t enable);
/* captured != 0: a captured period is held and will be replayed by a matching pff_run_steps; refused != 0: the driver
 * refused a capture once (pff_run_steps then launches plainly for the life of the mesh).  Either may be NULL. */
pff_status pff_graph_status(const pff_mesh *mesh, int32_t *captured, int32_t *refused);

/* ---- implicit differentiation of the damage solve (section 4.2) -----------
 * Backward pass of A(theta) d = b(theta) (Eq. 22): ONE adjoint solve A^T lambda = g with the same matrix-free operator
 * (Eq. 23; A is symmetric), linearised at the active set realised by the forward solve (L446).
 * g: upstream gradient dL/dd, device [n_nodes], precision of the mesh, internal order.  free_mask: device uint8
 * [n_nodes] or NULL; nodes with free_mask == 0 and the damage-Dirichlet nodes are outside the free set F and get
 * lambda = 0 (NULL: F = every non-Dirichlet node, the AT2 case where the solve is unconstrained and the clamp acts
 * afterwards; the caller routes g of clamped nodes to d_prev, L446).  lambda: device [n_nodes] out, 16-byte aligned.
 * Solves A_FF lambda_F = g_F by Jacobi-PCG from lambda = 0 with the operator of state->H (state->d is not read) until
 * ||g_F - A_FF lambda_F||_2 <= rel_tol ||g_F||_2; same kernels, status codes and synchronisation as pff_damage_solve. */
pff_status pff_damage_adjoint(pff_mesh *mesh, const pff_state *state, const void *g, const uint8_t *free_mask, void *lambda,
                              double rel_tol, int32_t max_iter, int32_t *iters_out, double *relres_out);
/* out = { lambda^T M d, lambda^T K d } with the consistent mass M (L185) and the P1 stiffness K of the mesh (unit
 * coefficients), accumulated in fp64 in a fixed order: the two scalars from which the (G_c, l0) gradients follow, e.g.
 * AT2: dL/dG_c = -[(1/l0) out[0] + l0 out[1]] (Eq. 24), dL/dl0 = -[-(G_c/l0^2) out[0] + G_c out[1]].
 * lambda, d: device [n_nodes], precision of the mesh, internal order.  Synchronises the stream. */
pff_status pff_damage_param_terms(pff_mesh *mesh, const void *lambda, const void *d, double out[2]);

/* ---- matrix-free stiffness action (Eq. 11-15) ---------------------------
 * q = K(u) p = f_int(u + p) - f_int(u) (Eq. 13) at the reference state u = state->u with the damage state->d held fixed:
 * the operator a Krylov solver of the quasi-static mechanics problem needs, never assembled.  Both forces are evaluated
 * in ONE fused element pass of the explicit-step kernel (same staging, same ordered gather: bit-reproducible).  Exact
 * tangent action for the isotropic split; for the other splits it is the paper's shifted difference, exact as long as p
 * does not change the sign pattern of the split (L140).  No boundary masking: the caller zeroes constrained dofs.
 * px, py (in) and qx, qy (out): device [n_nodes], precision of the mesh, internal order, px / py 16-byte aligned.
 * Gather scatter only (PFF_EUNSUPPORTED with PFF_SCATTER_ATOMIC).  Asynchronous. */
pff_status pff_stiffness_action(pff_mesh *mesh, const pff_state *state, const void *px, const void *py, void *qx, void *qy);

/* Quasi-static mechanics solve (PAPER.md L126-159 with L337 "staggered quasi-static mode"): one linear solve
 *     K(u_ref) du = S f_ext - f_int(u_ref)  on the free dofs,   state->u <- u_ref + du,
 * u_ref = state->u on entry (Dirichlet dofs first overwritten with bc->dir_u when it is given; bc->dir_v is not used),
 * S = bc->load_scale, d = state->d fixed, by Jacobi-preconditioned conjugate gradients whose operator is
 * pff_stiffness_action: ONE kernel launch per iteration (vector updates of the previous step in the node prologue, fused
 * element pass, ordered gather, predicted beta); alpha, beta and the norms stay on the device.
 * Stops when ||r_free||_2 <= rel_tol ||r0_free||_2, after max_iter iterations, or on a breakdown p . K p <= 0 (possible for
 * the non-isotropic splits, whose shifted difference need not be positive definite): the last two return PFF_ENOCONV with
 * the steps taken so far applied.
 * Exact equilibrium for the isotropic split (linear problem); for the other splits one step of the paper's shifted-
 * difference iteration (the caller repeats it; exact when du does not change the sign pattern of the split).
 * The constrained problem must be non-singular (enough Dirichlet dofs to remove the rigid-body modes).
 * v, a, H are not touched.  Gather scatter only.  Synchronises the stream. */
pff_status pff_equilibrium_solve(pff_mesh *mesh, pff_state *state, const pff_bc *bc, double rel_tol, int32_t max_iter,
                                 int32_t *iters_out, double *relres_out);

/* ---- test hooks (device vectors, internal order, precision of the mesh) ---------------------- */
/* f_int(u, d) of the current state (no predictor), and psi+ per element (psi_plus may be NULL). */
pff_status pff_internal_force(pff_mesh *mesh, const pff_state *state, void *fx, void *fy, void *psi_plus);
/* q = A p with the damage operator built from state->H (L173). */
pff_status pff_damage_matvec(pff_mesh *mesh, const pff_state *state, const void *p, void *q);
/* Right-hand side b and Jacobi diagonal D of the damage system (either may be NULL). */
pff_status pff_damage_rhs_diag(pff_mesh *mesh, const pff_state *state, void *b, void *D);

/* ---- instrumentation --------------------------------------------------------------------- */
/* Number of CUDA kernels this mesh has launched since creation (host counter). */
pff_status pff_mesh_counters(const pff_mesh *mesh, int64_t *kernel_launches);
/* Launches ONE kernel of the hot path `reps` times back to back on the mesh stream between two CUDA
 * events (after one untimed launch) and returns the mean milliseconds per launch.  which: 0 = fused
 * explicit step kernel (PFF_SCATTER_ATOMIC: element kernel), 1 = the same kernel for gather meshes, whose interface-node
 * pass is fused into it (ATOMIC: node kernel), 2 = chunk kernel of the plain damage mat-vec (the pff_damage_matvec hook),
 * 3 = interface-node kernel of that hook.  The step kernels advance the state with a negligible dt; the mat-vec reads
 * state->d as the trial vector.  Synchronises. */
pff_status pff_time_kernel(pff_mesh *mesh, pff_state *state, int32_t which, int32_t reps, float *ms_per_launch);

/* Kernel classes of the hot path, for per-kernel timing inside a real run (bench.py's roofline block). */
typedef enum {
    PFF_K_STEP_CHUNK = 0,      /* the explicit step kernel: chunk phase + interface phase (ATOMIC: element kernel)       */
    PFF_K_STEP_SHARED = 1,     /* ATOMIC only: node kernel                                                               */
    PFF_K_MATVEC_CHUNK = 2,    /* the cooperative CG kernel (all iterations of one solve); plain mat-vec of the hook     */
    PFF_K_MATVEC_SHARED = 3,   /* interface nodes of the hook's plain mat-vec                                            */
    PFF_K_DAMAGE_SETUP = 4,    /* the damage setup kernel: rhs, Jacobi diagonal, r0, operator coefficients, norms        */
    PFF_K_OTHER = 5,           /* Dirichlet overwrite, energies, host-path permutation, quasi-static vector kernels      */
    PFF_NUM_KERNEL_CLASSES = 6
} pff_kernel_class;
/* enable != 0: every following kernel launch of this mesh is bracketed by two CUDA events on the mesh
 * stream (adds ~2 event records per launch; use for attribution, not for headline throughput).
 * pff_profile_read synchronises the stream, returns per class the summed device milliseconds and the number
 * of launches since the last read (host arrays of PFF_NUM_KERNEL_CLASSES entries) and resets the tallies. */
pff_status pff_profile_enable(pff_mesh *mesh, int32_t enable);
pff_status pff_profile_read(pff_mesh *mesh, double *ms_sum, int64_t *launches);

/* ---- host-buffer convenience path (end-to-end timing, small problems) ------------------------
 * State in USER numbering, fp64, AoS on the HOST: u, v, a, fext [n_nodes][2]; d [n_nodes];
 * H [n_elems].  Uploads, converts to internal order / mesh precision on the device, runs n_steps of
 * { pff_explicit_step ; pff_damage_solve every damage_every-th step (0 = never) } with constant
 * Dirichlet values (dir_u, dir_v: host, n_dir entries, may be NULL) and load_scale, then downloads
 * u, v, a, d, H back into the same host arrays.  Synchronous. */
typedef struct {
    double *u, *v, *a, *d, *H, *fext;
} pff_host_state;
pff_status pff_run_host(pff_mesh *mesh, pff_host_state *hs, const double *dir_u, const double *dir_v,
                        double load_scale, double dt, int64_t n_steps, int32_t damage_every,
                        double rel_tol, int32_t max_iter);

/* Phase timestamps of the persistent kernels, for timelines like profiles/r2_timeline.md.  Only the instrumentation
 * build of the library (libpff_trace.so: python -m paper_2606_23458_b200.build --trace) records anything; the product
 * library returns PFF_EUNSUPPORTED.  device_words: device buffer of 2 * 256 * 1024 int64 (zeroed by the caller) or NULL to
 * stop; thread 0 of every CTA stores SM-cycle and nanosecond stamps of its phases (chunk by chunk: data arrived, node
 * prologue done, element pass done, gather done; then the grid-wide phases) for CG iteration cg_iteration of every
 * following solve and for every following explicit step.  Layout: paper_2606_23458_b200/trace_timeline.py. */
pff_status pff_trace_set(pff_mesh *mesh, void *device_words, int32_t cg_iteration);

const char *pff_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PFF_H */
