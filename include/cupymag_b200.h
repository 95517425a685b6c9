/*
 * cupymag_b200.h -- C ABI of the B200-native GSPM hot path of CuPyMag (arXiv 2510.09812).
 *
 * One GPU, one process.  Plain pointers and sizes only; no torch / C++ types cross this
 * boundary.  "P:n" cites /root/reference/PAPER.md line n; "R#" the readings in DESIGN.md.
 *
 * Conventions
 *  - Every function returns CM_OK (0) or a negative cm_status; it never throws or exits.
 *    cm_last_error() gives a thread-local message for the last failure.
 *  - "host" pointers are read (or written) only during the call.  "dev" pointers are CUDA
 *    device pointers owned by the CALLER (e.g. torch tensors' data_ptr()); `stream` is a
 *    cudaStream_t passed as void* (NULL = default stream).
 *  - The library owns cm_mesh / cm_system and every internal device buffer; nothing is
 *    allocated inside cm_spmv / cm_cg_solve* / cm_field_rhs / cm_gspm_step.  Two calls may allocate:
 *    cm_hysteresis_run (a capture stream, the graph, logs grown to max_fields) and cm_volume_average
 *    (a library-order staging copy kept in the mesh, grown on demand).  cm_volume_average_noalloc is the variant of the latter that
 *    allocates nothing (fixed scratch inside the library, see its declaration).
 *  - Calls on one cm_system share its scratch buffers: they must not run concurrently (one stream at a
 *    time per system).  cm_volume_average calls on one cm_mesh are serialised inside the library.
 *  - All field vectors are in USER node order, interleaved [node][component], of the
 *    system's dtype (double for CM_F64, float for CM_F32).  The locality reordering is
 *    internal; cm_mesh_get exposes it for bit-exact structure parity.
 *  - Quantities are nondimensional as in P:131: lengths x/l_d, fields H/m_s,
 *    potential U/(m_s l_d), displacement u/l_d, stiffness C/(mu0 m_s^2), time gamma m_s t.
 *  - Calls are asynchronous on `stream` except those that return host scalars
 *    (cm_cg_solve, cm_volume_average, cm_gspm_step with info != NULL, the *_host calls,
 *    the getters), which synchronise that stream before returning.
 *  - There is no CPU fallback: without a CUDA device every compute call fails with CM_E_CUDA.
 */
#ifndef CUPYMAG_B200_H
#define CUPYMAG_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cm_mesh cm_mesh;     /* opaque: reordered connectivity, node->element lists, CSR pattern */
typedef struct cm_system cm_system; /* opaque: geometry, assembled matrices, masks, work vectors (one dtype) */

typedef enum { CM_F64 = 0, CM_F32 = 1 } cm_dtype;
/* Locality reordering of the nodes (R21).  MORTON_SORTED: Morton order, then within every window of 256
 * consecutive positions the nodes in descending order of row length (ties keep their Morton order): the slices of the
 * SELL layouts then hold rows of nearly equal length on meshes of irregular valence (unstructured meshes). */
typedef enum { CM_REORDER_NONE = 0, CM_REORDER_MORTON = 1, CM_REORDER_RCM = 2, CM_REORDER_MORTON_SORTED = 3 } cm_reorder;

/* Matrices of Eq. 12 on the shared sparsity pattern; constraints applied as the symmetric
 * projection P A P + (I - P).  K_MS: all tets, one pinned node.  K_GS1/2 = M_m + eps K_m over
 * magnetic tets with eps1 = A* dtau (Alg. B.1 Step 1), eps2 = alpha A* dtau (Step 3),
 * identity rows on non-magnetic ("dead") nodes.  MASS = M_m = F^GS of Eq. 13.
 * K_MECH: 3x3 blocks, clamped DOFs. */
typedef enum { CM_MAT_K_MS = 0, CM_MAT_K_GS1 = 1, CM_MAT_K_GS2 = 2, CM_MAT_MASS = 3, CM_MAT_K_MECH = 4 } cm_matrix_id;

/* Preconditioner of the CG solves.  The paper runs plain CG ("no preconditioner") and names preconditioning as
 * future work; CM_PC_JACOBI is z = r / diag(A) with the diagonal of the constrained matrix as stored. */
typedef enum { CM_PC_NONE = 0, CM_PC_JACOBI = 1 } cm_precond;

/* Outputs of cm_field_rhs (Eq. 14; Eq. 15). */
typedef enum {
    CM_RHS_MS = 0,    /* b (N):    sum_e V_e grad phi_i . (mean_e m - mbar), 0 at the pin (R9)              */
    CM_RHS_MECH = 1,  /* b (N x 3): sum_{e magnetic} V_e [C*_e : mean_e E0(m)] grad phi_i, 0 at clamped DOFs  */
    CM_RHS_GS = 2,    /* b (N x 3): M_m (m + coeff * h(m; U, u))                                              */
    CM_OUT_HD = 3,    /* h_d (N x 3): -recovered grad U + <grad U> - N_d mbar (Eq. 4; R8, R10)         */
    CM_OUT_SIGMA = 4, /* sigma_hat (N x 6, Voigt xx,yy,zz,yz,xz,xy): recovered C*:(E(u) - E0(m))             */
    CM_OUT_FIELD = 5  /* h(m) (N x 3): anisotropy + Zeeman + demag + magnetoelastic (no exchange)     */
} cm_rhs_id;

enum { CM_TERM_ANIS = 1, CM_TERM_ZEEMAN = 2, CM_TERM_DEMAG = 4, CM_TERM_FARFIELD = 8, CM_TERM_MAGEL = 16 };

typedef enum {
    CM_OK = 0,
    CM_E_BADARG = -1,
    CM_E_DEGENERATE_TET = -2, /* V_e <= 1e-14 * (bounding-box diagonal)^3 */
    CM_E_INDEX_RANGE = -3,
    CM_E_ALLOC = -4,
    CM_E_CUDA = -5,
    CM_E_CG_BREAKDOWN = -6,   /* p^T A p <= 0 */
    CM_E_CG_MAXITER = -7      /* warning: the iterate is still written */
} cm_status;

/* what-codes of cm_mesh_get (all int32 arrays except COUNTS) */
enum {
    CM_GET_COUNTS = 0,    /* long[3]: n_nodes, n_tets, nnz                                   */
    CM_GET_ORDER = 1,     /* order[new] = user node                                          */
    CM_GET_IPERM = 2,     /* iperm[user] = new node                                          */
    CM_GET_TETS = 3,      /* n_tets x 4, relabelled, sorted by (min new node id, user tet)   */
    CM_GET_TET_ORDER = 4, /* tet_order[new] = user tet                                       */
    CM_GET_ROWPTR = 5,    /* n_nodes + 1                                                     */
    CM_GET_COLIDX = 6,    /* nnz, ascending in each row, diagonal present                    */
    CM_GET_N2E_PTR = 7,   /* n_nodes + 1                                                     */
    CM_GET_N2E = 8,       /* 4 n_tets entries element*4 + local index, ascending per node    */
    CM_GET_LAYOUT = 9     /* long[6]: stored elements (padding included) of the SELL-16 scalar and the SELL-8 block
                             layout, element chunks, chunk slots, chunk capacity in elements and in nodes */
};

/* Material constants of Eq. 1 and Appendix A; SI units. */
typedef struct {
    double Ms;           /* saturation magnetisation m_s, A/m */
    double Aex;          /* exchange coefficient A, J/m */
    double K1;           /* cubic anisotropy kappa_1, J/m^3 */
    double lambda100, lambda111; /* magnetostriction constants (E0(m)) */
    double alpha;        /* damping constant (Eq. 7) */
    double gamma;        /* gyromagnetic ratio in m/(A s): tau = gamma m_s t (R4) */
    double length_scale; /* l_d, metres */
    double Nd[9];        /* demagnetisation tensor of the ellipsoid, row-major (Eq. 4) */
    int n_elastic;       /* number of elastic materials; 0 = no mechanics */
    const double *C_voigt; /* host, n_elastic x 36 row-major, Pa; Voigt order xx,yy,zz,yz,xz,xy, engineering shears; CRYSTAL axes */
    double R[9];         /* Appendix D (R25): rotation crystal -> simulation frame, v_sim = R v_crystal
                            (Eq. D.2), row-major; all zeros = identity.  The library forms C_sim = M C M^T (Eq. D.3-D.4) and
                            evaluates E0(m), the anisotropy and the magnetoelastic field in crystal axes (Alg. D.1).
                            Not a proper rotation: CM_E_BADARG. */
    double sigma_ext[6]; /* uniform external stress of Eq. 1 (energy term -sigma_ext : E), Pa, simulation frame, tensor
                            components xx,yy,zz,yz,xz,xy.  DESIGN.md R17: with E = sym grad u it is one more mechanical
                            right-hand-side term, sum_e V_e sigma_ext,ab d_b phi_i over ALL elements; the homogeneous-strain
                            treatment of periodic domains (defined in the paper's ref. [2] only) is not built. */
} cm_material;

typedef struct {
    double dt;            /* s; must equal the dt given to cm_assemble_csr */
    double Hext[3];       /* A/m */
    unsigned terms;       /* CM_TERM_* bitmask; exchange is always on */
    int gspm_variant;     /* 0: Alg. B.1 as printed; 1: fully Gauss-Seidel second component (R1) */
    double cg_tol;        /* stop when ||r||_2 < cg_tol ||b||_2 */
    int cg_maxiter;
    int cg_fixed_iters;   /* >= 0: run exactly this many iterations in every solve; < 0: off */
    int cg_precond;       /* cm_precond of every solve of the step; CM_PC_NONE = the paper's unpreconditioned CG */
    int mech_matfree;     /* != 0: the mechanical solve applies K^mech matrix-free (cm_cg_solve_matfree); tetrahedra only */
} cm_step_params;

/* it_gs / res_gs slots: 0-2 g^n components, 3-4 g*_1, g*_2, 5-7 m** components. */
typedef struct {
    int it_ms, it_mech, it_gs[8];
    double res_ms, res_mech, res_gs[8];
    double mbar[3];       /* volume average of m^n (Eq. 17) */
    double mean_dm;       /* mean over magnetic nodes of ||m^{n+1}_i - m^n_i||_2 */
    double energy;        /* NaN (not computed on the device) */
} cm_step_info;

/* Kernel-class timers (CUDA events on the caller's stream) and launch counters. */
enum { CM_PROF_CG_MS = 0, CM_PROF_CG_MECH = 1, CM_PROF_CG_GS = 2, CM_PROF_SPMV = 3, CM_PROF_ELEMENT = 4,
       CM_PROF_POINTWISE = 5, CM_PROF_NCLASS = 6 };
typedef struct {
    double ms[CM_PROF_NCLASS];        /* accumulated device time per class, milliseconds */
    long launches[CM_PROF_NCLASS];    /* kernel launches per class */
    long cg_iters[CM_PROF_NCLASS];    /* CG iterations summed over right-hand sides (CG classes only) */
    long cg_matrix_passes[CM_PROF_NCLASS]; /* passes over the matrix inside CG: one per iteration (a 3-RHS solve reads it once per
                                              iteration) plus the r0 = b - A x0 pass of every launch */
} cm_profile;

/* S0: validate, reorder (R21), relabel, node->element lists, CSR pattern.
 * xyz: host, n_nodes x 3, metres.  tets: host, n_tets x 4, 0-based user node ids.
 * magnetic: host, n_tets, 1 = ferromagnet (NULL = all magnetic).  elastic_id: host, n_tets, index
 * into cm_material.C_voigt (NULL = all 0).  Errors: BADARG, INDEX_RANGE, DEGENERATE_TET, ALLOC, CUDA. */
int cm_mesh_create(const double *xyz, long n_nodes, const int *tets, long n_tets, const unsigned char *magnetic,
                   const int *elastic_id, cm_reorder reorder, void *stream, cm_mesh **out);
/* Periodic boundary conditions by node wrapping (R23).
 * cm_periodic_wrap: "wrapping any node whose coordinate in a given direction lies at the domain's maximum extent to the
 * corresponding node at the domain's minimum extent in that direction", each wrapped pair getting one unified index.
 * axes: bit d set = direction d periodic.  A node is wrapped along d when x_d >= max_d - rel_tol * span_d; nodes wrapped
 * along no direction are the representatives, numbered 0.. in ascending node index; a wrapped node takes the number of the
 * one representative within rel_tol * span of its image x - span_d e_d.  dof_of_node: host out, n_nodes; *n_dof: host out.
 * Host-only (no device needed).  Errors: BADARG (no or several partners: faces do not match).
 * cm_mesh_create_wrapped: as cm_mesh_create, with dof_of_node (host, n_nodes, values in [0, n_dof); NULL = identity).
 * Element geometry comes from the element's own corner coordinates; every nodal quantity is indexed by DOF: the mesh then
 * has n_dof "nodes" (cm_mesh_get counts, field vectors, clamp_dof, pin_node are all in DOF numbering).  A tet with two
 * corners on one DOF (domain one cell wide in a periodic direction) is rejected with BADARG. */
int cm_periodic_wrap(const double *xyz, long n_nodes, unsigned axes, double rel_tol, int *dof_of_node, long *n_dof);
int cm_mesh_create_wrapped(const double *xyz, long n_nodes, const int *tets, long n_tets, const unsigned char *magnetic,
                           const int *elastic_id, const int *dof_of_node, long n_dof, cm_reorder reorder, void *stream,
                           cm_mesh **out);
/* Linear hexahedral (Q1) meshes (R26): the paper's structured Fig. 2-3
 * workloads.  hexes: host, n_hexes x 8, local node a = i + 2 j + 4 k at corner (i, j, k) of the cell; trilinear shape
 * functions; every element integral (matrices, right-hand sides, recovered fields, lumped masses, Eq. 17) by the
 * 2 x 2 x 2 Gauss rule.  Every call of this header works on a hexahedral mesh (cm_assemble_csr, cm_spmv, cm_cg_solve*,
 * cm_field_rhs, cm_gspm_step*, cm_hysteresis_run, cm_volume_average) except cm_system_get_geometry(what = 0, 1), whose
 * per-element V_e / grad phi are stored for tetrahedra only (CM_E_BADARG).  cm_mesh_create_hex_wrapped: periodic node
 * wrapping exactly as cm_mesh_create_wrapped (dof_of_node from cm_periodic_wrap) -- the paper's own setting.  cm_mesh_get:
 * CM_GET_TETS has 8 ids per element, CM_GET_N2E entries are element*8 + local index.  Errors as cm_mesh_create
 * (DEGENERATE_TET: det J <= 0 at a Gauss point, i.e. an inverted or collapsed cell). */
int cm_mesh_create_hex(const double *xyz, long n_nodes, const int *hexes, long n_hexes, const unsigned char *magnetic,
                       const int *elastic_id, cm_reorder reorder, void *stream, cm_mesh **out);
int cm_mesh_create_hex_wrapped(const double *xyz, long n_nodes, const int *hexes, long n_hexes, const unsigned char *magnetic,
                               const int *elastic_id, const int *dof_of_node, long n_dof, cm_reorder reorder, void *stream,
                               cm_mesh **out);
int cm_mesh_destroy(cm_mesh *mesh);
/* Copies structure arrays to host_out (capacity in elements); returns BADARG if capacity is too small. */
int cm_mesh_get(const cm_mesh *mesh, int what, void *host_out, long capacity);

/* S1: geometry (V_e, grad phi SoA, lumped masses) and matrix values on the device (Eq. 12), for one
 * dtype and one dt (which fixes eps1, eps2).  clamp_dof: host, 3 n_nodes flags in user order or NULL.
 * pin_node: user index of the pinned node of K^ms.  The mesh must outlive the system. */
int cm_assemble_csr(cm_mesh *mesh, const cm_material *material, cm_dtype dtype, double dt,
                    const unsigned char *clamp_dof, long pin_node, void *stream, cm_system **out);
int cm_system_destroy(cm_system *sys);
/* Matrix values in LIBRARY node order, plain CSR (nnz) or block-CSR (nnz x 3 x 3 row-major), system dtype. */
int cm_system_get_values(const cm_system *sys, cm_matrix_id id, void *host_out, long capacity);
/* Geometry in library order: what = 0 V_e (n_tets), 1 grad phi (n_tets x 4 x 3), 2 mL (n_nodes), 3 mLm (n_nodes);
 * system dtype. */
int cm_system_get_geometry(const cm_system *sys, int what, void *host_out, long capacity);

/* y = A x.  x_dev, y_dev: N (scalar matrices) or N x 3 (K_MECH), user order. */
int cm_spmv(cm_system *sys, cm_matrix_id id, const void *x_dev, void *y_dev, void *stream);
/* Mass product for three interleaved components: y (N x 3) = M_m x (N x 3)  (b^GS of Eq. 14). */
int cm_spmv3(cm_system *sys, cm_matrix_id id, const void *x_dev, void *y_dev, void *stream);

/* Unpreconditioned CG (O-4): x_dev holds x0 on entry and x on exit.  Stops when the recurrence
 * residual satisfies ||r|| < tol ||b|| (tested before each iteration), after maxiter iterations
 * (CM_E_CG_MAXITER), or after exactly fixed_iters iterations when fixed_iters >= 0.  ||b|| = 0 gives x = 0
 * and 0 iterations.  One persistent cooperative kernel; the stopping test runs on the device. */
int cm_cg_solve(cm_system *sys, cm_matrix_id id, const void *b_dev, void *x_dev, double tol, int maxiter,
                int fixed_iters, int *iters_out, double *relres_out, void *stream);
/* Three independent CG solves with one scalar matrix (b, x: N x 3 interleaved), the matrix read once per
 * iteration; iters_out / relres_out have 3 entries. */
int cm_cg_solve3(cm_system *sys, cm_matrix_id id, const void *b_dev, void *x_dev, double tol, int maxiter,
                 int fixed_iters, int *iters_out, double *relres_out, void *stream);

/* The same solves with a preconditioner (cm_precond).  The stopping rule is unchanged (||r||_2 < tol ||b||_2 on the
 * unpreconditioned recurrence residual); CM_PC_NONE gives cm_cg_solve / cm_cg_solve3 bit for bit.  CM_MAT_MASS has no
 * Jacobi preconditioner (it is singular on non-magnetic nodes): BADARG. */
int cm_cg_solve_pc(cm_system *sys, cm_matrix_id id, const void *b_dev, void *x_dev, double tol, int maxiter,
                   int fixed_iters, int precond, int *iters_out, double *relres_out, void *stream);
int cm_cg_solve3_pc(cm_system *sys, cm_matrix_id id, const void *b_dev, void *x_dev, double tol, int maxiter,
                    int fixed_iters, int precond, int *iters_out, double *relres_out, void *stream);
/* Residual history of the solves that follow (on != 0): the kernel records ||r_k|| / ||b|| before iteration k,
 * k = 0 .. iters, per right-hand side (up to 65536 iterations).  cm_cg_history copies the history of the LAST solve to
 * host_out ([k][n_rhs] doubles, n_rhs = 1, or 3 for cm_cg_solve3*), at most `capacity` doubles; *n_out = entries written.
 * Only cm_cg_solve, cm_cg_solve3 and their _pc forms record.  *n_out = 0 when the last solve ran with the history off, and
 * after cm_cg_solve_matfree, cm_gspm_step, cm_gspm_step_host or cm_hysteresis_run (their solves are not recorded as a
 * history; a step with the history on reuses the buffer). */
int cm_cg_history_enable(cm_system *sys, int on);
int cm_cg_history(cm_system *sys, double *host_out, long capacity, long *n_out);

/* Matrix-free K^mech (the paper's future work: it "assembles and stores sparse matrices explicitly").
 * cm_spmv_matfree: y = (P K^mech P + (I - P)) x, the same operator as cm_spmv(CM_MAT_K_MECH), applied as an element pass
 * (strain of x, stress C*_e : E, nodal forces V_e sigma grad phi_k per chunk slot) and a node pass; nothing of the stored
 * matrix is read.  cm_cg_solve_matfree: CG (optionally Jacobi, with the stored diagonal) on that operator, same stopping
 * rule and outputs as cm_cg_solve_pc; four launches per iteration, the stream is synchronised once per 16 iterations.
 * Linear tetrahedra only (hexahedral meshes: BADARG).  x, y, b: N x 3, user order. */
int cm_spmv_matfree(cm_system *sys, const void *x_dev, void *y_dev, void *stream);
int cm_cg_solve_matfree(cm_system *sys, const void *b_dev, void *x_dev, double tol, int maxiter, int fixed_iters,
                        int precond, int *iters_out, double *relres_out, void *stream);

/* Element-wise gather / compute / deterministic gather-scatter assembly (see cm_rhs_id).  m_dev: N x 3;
 * U_dev: N (may be NULL when DEMAG is off); u_dev: N x 3 (may be NULL when MAGEL is off); coeff: dtau or
 * alpha dtau for CM_RHS_GS.  b_dev: output of the size listed at cm_rhs_id. */
int cm_field_rhs(cm_system *sys, cm_rhs_id id, const void *m_dev, const void *U_dev, const void *u_dev,
                 const cm_step_params *params, double coeff, void *b_dev, void *stream);

/* Volume average (Eq. 16-17) of an ncomp-component nodal field (user order): out_host[c]. */
int cm_volume_average(const cm_mesh *mesh, cm_dtype dtype, const void *g_dev, int ncomp, double *out_host,
                      void *stream);

/* The same volume average for callers that must not allocate device memory: a host program that gave the whole
 * device to its own memory pool at start-up (cudaMalloc then fails), or a time loop that monitors <m> while other
 * streams work (cudaMalloc / cudaFree may synchronise the whole device).  cm_volume_average grows a staging copy
 * inside the mesh with cudaFree + cudaMalloc; this call allocates and frees nothing, calls no allocating library
 * routine and does not synchronise: it is asynchronous on `stream`.
 *   g_dev    device, N x ncomp, user order, of `dtype`            (input, caller's)
 *   out_dev  DEVICE pointer to ncomp doubles, written on `stream`  (output, caller's; read it after the stream
 *            has reached this point)
 * Its scratch memory (one partial sum per tile of 8192 nodes) is a fixed device array inside the library, 96 KiB
 * that every GPU which loads the library holds until the process exits.  Consequences:
 *   - limits: mesh nodes <= CM_NOALLOC_MAX_NODES and ncomp in {1, 3, 6}; beyond them CM_E_BADARG with a message and
 *     nothing is launched (cm_volume_average has no node limit);
 *   - every call on a GPU shares that one array, whatever mesh or stream it is given: calls that can overlap on the
 *     GPU race and give garbage.  Keep them on one stream or order them with events.  The array keeps the previous
 *     call's partial sums; no part of it has to start at zero (each call writes every row it reads), so back-to-back
 *     calls of different sizes need nothing cleared;
 *   - the first call on each GPU looks up the array's device address (cudaGetSymbolAddress, that GPU current) and
 *     caches it; make that first call once per GPU at set-up, before any stream capture begins.  Call with the
 *     mesh's GPU current.
 * Result: the same sum as cm_volume_average in another (fixed, run-to-run reproducible) order; they agree to
 * rounding (<= 1e-13 fp64 / 1e-7 fp32 on O(1) fields, tests/test_zz_no_alloc.py). */
#define CM_NOALLOC_MAX_NODES 16777216L
int cm_volume_average_noalloc(const cm_mesh *mesh, cm_dtype dtype, const void *g_dev, int ncomp, double *out_dev,
                              void *stream);

/* One Gauss-Seidel projection step (Alg. B.1; SURVEY O-3).  m_dev (N x 3), U_dev (N), u_dev
 * (N x 3) are updated in place (U, u are the warm starts of the magnetostatic / mechanical CG).
 * info may be NULL (then the call does not synchronise).  Returns the worst CG status. */
int cm_gspm_step(cm_system *sys, const cm_step_params *params, void *m_dev, void *U_dev, void *u_dev,
                 cm_step_info *info, void *stream);
/* Same with HOST buffers: copies m, U, u to the device, steps, copies them back (end-to-end path). */
int cm_gspm_step_host(cm_system *sys, const cm_step_params *params, void *m_host, void *U_host, void *u_host,
                      cm_step_info *info, void *stream);

/* Hysteresis driver (Fig. 1; R24).  Field k is H0 + k dH.  At each field GSPM
 * steps run until <||m^{n+1} - m^n||_2> over magnetic nodes < conv_tol (5e-10) or max_steps steps; then the volume
 * average of the converged m (Eq. 17), H and the step count are logged ("written at convergence").  The run ends
 * when that average has a negative component along H0/|H0| ("the magnetization field in the domain reverses") or
 * after max_fields fields. */
typedef struct {
    double H0[3], dH[3]; /* A/m; 200 A/m e1, -20 A/m e1 */
    double conv_tol;
    int max_fields, max_steps;
} cm_hyst_params;
typedef struct {
    int n_fields, reversed;
    long total_steps;
    long cg_iters_ms, cg_iters_mech, cg_passes_gs; /* summed over all steps */
    int worst_cg_status;                           /* CM_OK, CM_E_CG_MAXITER or CM_E_CG_BREAKDOWN */
    double device_ms;                              /* CUDA-event time of the whole loop */
} cm_hyst_result;
/* The WHOLE loop runs on the device: one CUDA graph whose body (one GSPM step with the applied field read from device
 * memory, the average of the new m, a one-thread controller that tests convergence, logs, decrements the field and
 * detects reversal) sits in a conditional WHILE node; the host launches it once and synchronises once.
 * base: step parameters (Hext ignored).  m_dev, U_dev, u_dev: in/out as in cm_gspm_step.  H_log, mbar_log (host,
 * max_fields x 3) and steps_log (host, max_fields): filled for the first result->n_fields fields.
 * Returns CM_OK, or the worst CG status.  Errors: BADARG (H0 = 0, non-positive caps, null pointers), CUDA. */
int cm_hysteresis_run(cm_system *sys, const cm_step_params *base, const cm_hyst_params *hp, void *m_dev, void *U_dev, void *u_dev,
                      double *H_log, double *mbar_log, int *steps_log, cm_hyst_result *result, void *stream);

/* Tuning / measurement switches of a system (value 0 = default).
 * CM_OPT_STORED_GEOMETRY: how the element passes S3/S5/S6/S8 of a plain (not wrapped) tetrahedral mesh get V_e and grad phi.
 * 0: per pass, whichever kernel is faster -- the fp64 passes S3 and S5 recompute them in fp64 from the chunk's staged node
 * coordinates, the others stream the stored values (ten words per tetrahedron); 1: every pass streams; 2: every pass
 * recomputes.  All three give the same bits.  Other values: BADARG.
 * CM_OPT_NO_FUSED_S5S8: 1 = cm_gspm_step runs gradient recovery (S5) and the first stress recovery (S8) as separate element
 * passes; by default, with DEMAG and MAGEL on a tetrahedral mesh, one pass computes both (same bits). */
enum { CM_OPT_STORED_GEOMETRY = 0, CM_OPT_NO_FUSED_S5S8 = 1 };
int cm_system_set_option(cm_system *sys, int option, int value);

int cm_profile_enable(cm_system *sys, int on);
int cm_profile_get(cm_system *sys, cm_profile *out); /* synchronises outstanding timers */
int cm_profile_reset(cm_system *sys);

const char *cm_last_error(void);
const char *cm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CUPYMAG_B200_H */
