/*
 * cm_oracle.c -- CPU ORACLE for the GSPM hot path of CuPyMag (arXiv 2510.09812).
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg may load this library.  It shares no code, header,
 * table or helper with the CUDA library (paper_2510_09812_b200/csrc); neither includes
 * the other.  It is written from the paper, plainly: loops over elements and rows in
 * index order, no blocking, no fusion, no reordering, so it can be checked against the
 * paper by eye.  "P:n" = /root/reference/PAPER.md line n.  "R#" = reading # listed in
 * DESIGN.md (the points where the paper is silent or ambiguous).
 *
 * Compiled twice: -DORC_F32 gives the single-precision twin (R20: matrices, geometry and
 * vectors stored in fp32; set-up quantities computed in fp64 then rounded; every
 * reduction accumulated in fp64).  OpenMP pragmas sit on independent row loops only; the
 * dot products use fixed-order chunk partials, so results are bit-reproducible run to run.
 *
 * Pins (tests/test_oracle_pins.py): element volumes sum to the box volume; grad(phi)
 * duality; K symmetric, zero row sums, patch test, u^T K u = |a|^2 vol for linear u;
 * M row sums = lumped mass, u^T M u = int (a.x+b)^2; K^mech rigid-body null space and
 * u^T K u = vol * symG:C:symG; volume average of a linear field = value at centroid;
 * uniform m => b^ms = 0 and h_d = -N_d mbar (sphere: -mbar/3); gradient/stress recovery
 * exact on linear fields; fields h_an, h_d, h_me = -(1/mass) dEnergy/dm by central finite
 * differences; closed-form energies of uniform states; CG against dense solves; the GSPM
 * step against the analytic macrospin solution (first order in dtau), fixed points,
 * |m| = 1 and energy decay.  Later rows have their own pin files: periodic node wrapping
 * (tests/test_oracle_periodic.py: brute-force wrap, Fourier symbol of the periodic 7-point
 * operator, Eq. 20, literal = adjoint Eq. 14 right-hand side), the hysteresis driver
 * (tests/test_oracle_hysteresis.py: macrospin switching field), the rotated crystal frame
 * (tests/test_oracle_rotation.py: numpy tensor rotations, <111> modulus) and linear
 * hexahedra (tests/test_oracle_hex.py: 27-point stiffness and tensor-product mass in closed
 * form, exactness of the 2 x 2 x 2 rule, energy gradients), Jacobi-preconditioned CG
 * (tests/test_oracle_pcg.py: plain CG on the symmetrically scaled system iterate by iterate,
 * dense solves, precond 0 bitwise the plain solver), the external stress
 * (tests/test_oracle_sigma_ext.py: homogeneous Hooke state, energy stationarity, traction
 * moment) and the row-length-sorted Morton order (tests/test_oracle_pins.py, brute force).
 * The two readings of Alg. B.1 Step 2 (gspm_variant 0 and 1, R1) are pinned by the 2 x 2
 * maps they reduce to for an undamped macrospin (alpha = 0, h || z: forward Euler with
 * determinant 1 + a^2 as printed, symplectic Euler with determinant 1 for Gauss-Seidel) and
 * by the conservation of m . h that Eq. 7 demands there.  The adjoint magnetostatic RHS
 * (R9) is pinned against the paper's literal form on periodic domains, where they agree.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORC_F32
typedef float real;
#else
typedef double real;
#endif

typedef unsigned char uchar;

#define ORC_OK 0
#define ORC_E_BADARG (-1)
#define ORC_E_DEGENERATE (-2)
#define ORC_E_RANGE (-3)
#define ORC_E_ALLOC (-4)
#define ORC_E_BREAKDOWN (-6)
#define ORC_W_MAXITER (-7)

#define T_ANIS 1u
#define T_ZEEMAN 2u
#define T_DEMAG 4u
#define T_FARFIELD 8u
#define T_MAGEL 16u

enum { MAT_K_MS = 0, MAT_K_GS1 = 1, MAT_K_GS2 = 2, MAT_MASS = 3, MAT_K_MECH = 4,
       MAT_K_FREE = 5, MAT_K_M = 6, MAT_K_MECH_FREE = 7 };

typedef struct {
    double Ms, Aex, K1, lambda100, lambda111, alpha, gamma, length_scale;
    double Nd[9];
    int n_elastic;
    const double *C_voigt; /* n_elastic x 36, Pa; in CRYSTAL axes */
    double R[9];           /* App. D: crystal -> simulation frame, v_sim = R v_crystal (Eq. D.2), row-major; all zeros = identity */
    double sigma_ext[6];   /* uniform external stress of Eq. 1 (term -sigma_ext : E), Pa, simulation frame,
                              tensor components (xx,yy,zz,yz,xz,xy); R17: the homogeneous-strain part of ref. [2] stays out */
} orc_material;

typedef struct {
    double dt;
    double Hext[3];
    unsigned terms;
    int gspm_variant;
    double cg_tol;
    int cg_maxiter;
    int cg_fixed_iters;
    int cg_precond;        /* 0: none (the paper); 1: Jacobi in every solve */
} orc_step_params;

typedef struct {
    int it_ms, it_mech, it_gs[8];
    double res_ms, res_mech, res_gs[8];
    double mbar[3];
    double mean_dm;
    double energy;
} orc_step_info;

typedef struct {
    long N, Ne, nnz;
    double *x;      /* N x 3, nondimensional x/l_d (O-0) */
    int *tet;       /* Ne x 4 */
    uchar *mag;     /* Ne */
    int *eid;       /* Ne */
    real *V;        /* Ne          element volumes (|J|/6) */
    real *G;        /* Ne x 4 x 3  grad phi_k of each element */
    real *mL, *mLm; /* N lumped masses (all tets / magnetic tets) */
    uchar *live;    /* N: touched by a magnetic tet */
    int *n2e_ptr, *n2e; /* node -> (element*4 + local) */
    int *rowptr, *col;
    /* scalar matrices on the shared pattern */
    real *K, *Kms, *Km, *Mm, *Kgs1, *Kgs2;
    /* 3x3 block matrices [nnz][3][3] */
    real *Kmech, *Kmech_free;
    uchar *clamp; long pin;
    double dt, Astar, Kstar, dtau, eps1, eps2, alpha, lam100, lam111, Ms, Nd[9];
    int n_elastic; double *Cstar; /* n_elastic x 36, C/(mu0 Ms^2) */
    double Vtot, Vmag;
    double R[9]; int rot; /* App. D rotation (identity: rot = 0) */
    double sext[6];       /* sigma_ext / (mu0 Ms^2) */
    int nen; int *hex;    /* nen = 8: linear hexahedra; hex = Ne x 8 connectivity in DOF numbering; 0 / 4: tetrahedra */
    int *ghex;            /* hexahedra: Ne x 8 geometric node ids (coordinates); differs from hex on a wrapped (periodic) mesh */
} oracle;

static const double MU0 = 4.0e-7 * 3.14159265358979323846;
static int hex_rhs_ms(const oracle *o, const real *m, const double *mbar, real *b);
static int hex_demag_field(const oracle *o, const real *U, const double *mbar, unsigned terms, real *hd, double *gradU_mean);
static int hex_rhs_mech(const oracle *o, const real *m, real *b);
static int hex_stress_recover(const oracle *o, const real *u, const real *w, real *sig);
static double hex_elastic_energy(const oracle *o, const real *m, const real *u);

/* ------------------------------------------------------------------------------------ */
/* S0: reordering, relabelling, node->element lists, sparsity pattern (R21)              */
/* ------------------------------------------------------------------------------------ */

static int build_n2e(long N, long Ne, const int *tet, int **ptr_out, int **lst_out)
{
    int *ptr = (int *)calloc((size_t)N + 1, sizeof(int));
    int *lst = (int *)malloc((size_t)Ne * 4 * sizeof(int));
    if (!ptr || !lst) return ORC_E_ALLOC;
    for (long e = 0; e < Ne; e++)
        for (int k = 0; k < 4; k++) ptr[tet[4 * e + k] + 1]++;
    for (long i = 0; i < N; i++) ptr[i + 1] += ptr[i];
    int *fill = (int *)malloc((size_t)N * sizeof(int));
    memcpy(fill, ptr, (size_t)N * sizeof(int));
    for (long e = 0; e < Ne; e++) /* ascending e => each list is ascending in e */
        for (int k = 0; k < 4; k++) lst[fill[tet[4 * e + k]]++] = (int)(4 * e + k);
    free(fill);
    *ptr_out = ptr; *lst_out = lst;
    return ORC_OK;
}

static int cmp_int(const void *a, const void *b)
{
    int x = *(const int *)a, y = *(const int *)b;
    return (x > y) - (x < y);
}

/* Row pattern of node i = { j : i and j share a tet } U { i }, columns ascending. */
static int build_pattern(long N, const int *tet, const int *ptr, const int *lst,
                         int **rowptr_out, int **col_out, long *nnz_out)
{
    int *rowptr = (int *)calloc((size_t)N + 1, sizeof(int));
    int cap = 4096; int *tmp = (int *)malloc(cap * sizeof(int));
    if (!rowptr || !tmp) return ORC_E_ALLOC;
    for (int pass = 0; pass < 2; pass++) {
        int *col = pass ? *col_out : NULL;
        for (long i = 0; i < N; i++) {
            int m = 0, cnt = ptr[i + 1] - ptr[i];
            if (4 * cnt + 1 > cap) { cap = 8 * cnt + 1; tmp = (int *)realloc(tmp, cap * sizeof(int)); }
            tmp[m++] = (int)i;
            for (int s = ptr[i]; s < ptr[i + 1]; s++) {
                int e = lst[s] >> 2;
                for (int k = 0; k < 4; k++) tmp[m++] = tet[4 * e + k];
            }
            qsort(tmp, m, sizeof(int), cmp_int);
            int u = 0;
            for (int q = 0; q < m; q++) if (q == 0 || tmp[q] != tmp[q - 1]) tmp[u++] = tmp[q];
            if (!pass) rowptr[i + 1] = u;
            else memcpy(col + rowptr[i], tmp, u * sizeof(int));
        }
        if (!pass) {
            for (long i = 0; i < N; i++) rowptr[i + 1] += rowptr[i];
            *col_out = (int *)malloc((size_t)rowptr[N] * sizeof(int));
            if (!*col_out) return ORC_E_ALLOC;
        }
    }
    free(tmp);
    *rowptr_out = rowptr; *nnz_out = rowptr[N];
    return ORC_OK;
}

/* the same two builders for elements with nen nodes (list entries nen * e + k) */
static int build_n2e_n(long N, long Ne, const int *conn, int nen, int **ptr_out, int **lst_out)
{
    int *ptr = (int *)calloc((size_t)N + 1, sizeof(int));
    int *lst = (int *)malloc((size_t)Ne * nen * sizeof(int));
    int *fill = (int *)malloc((size_t)N * sizeof(int));
    if (!ptr || !lst || !fill) return ORC_E_ALLOC;
    for (long q = 0; q < nen * Ne; q++) ptr[conn[q] + 1]++;
    for (long i = 0; i < N; i++) ptr[i + 1] += ptr[i];
    memcpy(fill, ptr, (size_t)N * sizeof(int));
    for (long q = 0; q < nen * Ne; q++) lst[fill[conn[q]]++] = (int)q;
    free(fill);
    *ptr_out = ptr; *lst_out = lst;
    return ORC_OK;
}

static int build_pattern_n(long N, const int *conn, int nen, const int *ptr, const int *lst, int **rowptr_out, int **col_out, long *nnz_out)
{
    int *rowptr = (int *)calloc((size_t)N + 1, sizeof(int));
    if (!rowptr) return ORC_E_ALLOC;
    int *col = NULL;
    for (int pass = 0; pass < 2; pass++) {
        for (long i = 0; i < N; i++) {
            int cnt = ptr[i + 1] - ptr[i], m = 0;
            int *tmp = (int *)malloc(((size_t)nen * cnt + 1) * sizeof(int));
            tmp[m++] = (int)i;
            for (int s = ptr[i]; s < ptr[i + 1]; s++) {
                long e = lst[s] / nen;
                for (int k = 0; k < nen; k++) tmp[m++] = conn[nen * e + k];
            }
            qsort(tmp, m, sizeof(int), cmp_int);
            int u = 0;
            for (int q = 0; q < m; q++) if (q == 0 || tmp[q] != tmp[q - 1]) tmp[u++] = tmp[q];
            if (!pass) rowptr[i + 1] = u; else memcpy(col + rowptr[i], tmp, u * sizeof(int));
            free(tmp);
        }
        if (!pass) {
            for (long i = 0; i < N; i++) rowptr[i + 1] += rowptr[i];
            col = (int *)malloc((size_t)rowptr[N] * sizeof(int));
            if (!col) return ORC_E_ALLOC;
        }
    }
    *rowptr_out = rowptr; *col_out = col; *nnz_out = rowptr[N];
    return ORC_OK;
}

typedef struct { unsigned long long key; int idx; } keyidx;
static int cmp_keyidx(const void *a, const void *b)
{
    const keyidx *x = (const keyidx *)a, *y = (const keyidx *)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return (x->idx > y->idx) - (x->idx < y->idx);
}

/* Morton order (R21): q_d = floor((x_d-min_d)/(max_d-min_d)*(2^21-1)) in fp64; 63-bit
 * interleave with x in the least significant lane; stable sort by (code, user index). */
static void order_morton(long N, const double *xyz, int *order)
{
    double lo[3], hi[3];
    for (int d = 0; d < 3; d++) { lo[d] = xyz[d]; hi[d] = xyz[d]; }
    for (long i = 0; i < N; i++)
        for (int d = 0; d < 3; d++) {
            if (xyz[3 * i + d] < lo[d]) lo[d] = xyz[3 * i + d];
            if (xyz[3 * i + d] > hi[d]) hi[d] = xyz[3 * i + d];
        }
    keyidx *k = (keyidx *)malloc((size_t)N * sizeof(keyidx));
    for (long i = 0; i < N; i++) {
        unsigned long long code = 0, q[3];
        for (int d = 0; d < 3; d++) {
            double span = hi[d] - lo[d];
            double t = span > 0 ? (xyz[3 * i + d] - lo[d]) / span * 2097151.0 : 0.0;
            q[d] = (unsigned long long)floor(t);
        }
        for (int b = 0; b < 21; b++)
            for (int d = 0; d < 3; d++) code |= ((q[d] >> b) & 1ull) << (3 * b + d);
        k[i].key = code; k[i].idx = (int)i;
    }
    qsort(k, N, sizeof(keyidx), cmp_keyidx);
    for (long i = 0; i < N; i++) order[i] = k[i].idx;
    free(k);
}

/* Reverse Cuthill-McKee (R21): per component start at the unvisited node of minimum
 * degree (lowest index on ties); BFS, appending the unvisited neighbours of each node by
 * (degree, index) ascending; reverse the final order. */
static void order_rcm(long N, const int *rowptr, const int *col, int *order)
{
    keyidx *bydeg = (keyidx *)malloc((size_t)N * sizeof(keyidx));
    uchar *seen = (uchar *)calloc((size_t)N, 1);
    int *cm = (int *)malloc((size_t)N * sizeof(int));
    for (long i = 0; i < N; i++) { bydeg[i].key = (unsigned long long)(rowptr[i + 1] - rowptr[i] - 1); bydeg[i].idx = (int)i; }
    qsort(bydeg, N, sizeof(keyidx), cmp_keyidx);
    long head = 0, tail = 0, scan = 0;
    int cap = 64; keyidx *nb = (keyidx *)malloc(cap * sizeof(keyidx));
    while (tail < N) {
        while (seen[bydeg[scan].idx]) scan++;
        int s = bydeg[scan].idx;
        seen[s] = 1; cm[tail++] = s;
        while (head < tail) {
            int v = cm[head++], m = 0;
            if (rowptr[v + 1] - rowptr[v] > cap) { cap = 2 * (rowptr[v + 1] - rowptr[v]); nb = (keyidx *)realloc(nb, cap * sizeof(keyidx)); }
            for (int q = rowptr[v]; q < rowptr[v + 1]; q++) {
                int j = col[q];
                if (j != v && !seen[j]) { nb[m].key = (unsigned long long)(rowptr[j + 1] - rowptr[j] - 1); nb[m].idx = j; m++; seen[j] = 1; }
            }
            qsort(nb, m, sizeof(keyidx), cmp_keyidx);
            for (int q = 0; q < m; q++) cm[tail++] = nb[q].idx;
        }
    }
    for (long i = 0; i < N; i++) order[i] = cm[N - 1 - i];
    free(bydeg); free(seen); free(cm); free(nb);
}

/* Public: compute the locality permutation and the relabelled, sorted connectivity.
 * method: 0 none, 1 Morton, 2 RCM, 3 Morton followed by a windowed row-length sort (R21: within every window
 * of 256 consecutive Morton positions the nodes are put in descending order of their row length, i.e. number of distinct
 * neighbours, ties keeping their Morton order -- the sigma-window of a SELL-C-sigma layout written into the node order).
 * order[new] = old node; iperm[old] = new node.
 * Tets keep their local node order and are sorted by (min new node id, user tet index);
 * tet_order[new_tet] = old tet. */
int orc_reorder(const double *xyz, long N, const int *tets, long Ne, int method,
                int *order, int *iperm, int *tets_new, int *tet_order)
{
    if (method == 0) for (long i = 0; i < N; i++) order[i] = (int)i;
    else if (method == 1) order_morton(N, xyz, order);
    else if (method == 2) {
        int *ptr, *lst, *rowptr, *col; long nnz;
        int rc = build_n2e(N, Ne, tets, &ptr, &lst); if (rc) return rc;
        rc = build_pattern(N, tets, ptr, lst, &rowptr, &col, &nnz); if (rc) return rc;
        order_rcm(N, rowptr, col, order);
        free(ptr); free(lst); free(rowptr); free(col);
    } else if (method == 3) {
        int *ptr, *lst, *rowptr, *col; long nnz;
        order_morton(N, xyz, order);
        int rc = build_n2e(N, Ne, tets, &ptr, &lst); if (rc) return rc;
        rc = build_pattern(N, tets, ptr, lst, &rowptr, &col, &nnz); if (rc) return rc;
        int *tmp = (int *)malloc(256 * sizeof(int));
        for (long w0 = 0; w0 < N; w0 += 256) {
            long w1 = w0 + 256 < N ? w0 + 256 : N;
            /* insertion sort: stable, descending row length */
            for (long i = w0; i < w1; i++) tmp[i - w0] = order[i];
            for (long i = 1; i < w1 - w0; i++) {
                int v = tmp[i], lv = rowptr[v + 1] - rowptr[v];
                long j = i - 1;
                while (j >= 0 && rowptr[tmp[j] + 1] - rowptr[tmp[j]] < lv) { tmp[j + 1] = tmp[j]; j--; }
                tmp[j + 1] = v;
            }
            for (long i = w0; i < w1; i++) order[i] = tmp[i - w0];
        }
        free(tmp); free(ptr); free(lst); free(rowptr); free(col);
    } else return ORC_E_BADARG;
    for (long i = 0; i < N; i++) iperm[order[i]] = (int)i;
    keyidx *k = (keyidx *)malloc((size_t)Ne * sizeof(keyidx));
    for (long e = 0; e < Ne; e++) {
        int mn = iperm[tets[4 * e]];
        for (int q = 1; q < 4; q++) if (iperm[tets[4 * e + q]] < mn) mn = iperm[tets[4 * e + q]];
        k[e].key = (unsigned long long)mn; k[e].idx = (int)e;
    }
    qsort(k, Ne, sizeof(keyidx), cmp_keyidx);
    for (long e = 0; e < Ne; e++) {
        tet_order[e] = k[e].idx;
        for (int q = 0; q < 4; q++) tets_new[4 * e + q] = iperm[tets[4 * k[e].idx + q]];
    }
    free(k);
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------ */
/* Periodic boundary conditions by node wrapping (R23)               */
/* ------------------------------------------------------------------------------------ */
/* "wrapping any node whose coordinate in a given direction lies at the domain's maximum extent to the corresponding
 * node at the domain's minimum extent in that direction.  Then [...] inserts each wrapped node pair into a hash map
 * and assigns a unique global index."
 * axes: bit d set = direction d periodic.  A node is wrapped along d when x_d >= hi_d - tol_d (tol_d = rel_tol * span_d);
 * its image is x - span_d e_d for every such d.  Nodes wrapped along no direction are the representatives and are
 * numbered 0.. in ascending node index; a wrapped node takes the number of the one representative within tol of its
 * image (none or several: ORC_E_BADARG, "only works for [...] perfectly matched node distributions"). */
static unsigned long long cell_hash(long long cx, long long cy, long long cz)
{
    unsigned long long h = (unsigned long long)cx * 0x9E3779B97F4A7C15ull;
    h ^= (unsigned long long)cy * 0xC2B2AE3D27D4EB4Full + (h << 6) + (h >> 2);
    h ^= (unsigned long long)cz * 0x165667B19E3779F9ull + (h << 6) + (h >> 2);
    return h;
}

int orc_periodic_wrap(const double *xyz, long N, unsigned axes, double rel_tol, int *dof, long *ndof_out)
{
    if (!xyz || !dof || !ndof_out || N <= 0 || !(rel_tol > 0) || rel_tol > 1e-3) return ORC_E_BADARG;
    double lo[3], hi[3], span[3], tol[3], h[3];
    for (int d = 0; d < 3; d++) { lo[d] = 1e300; hi[d] = -1e300; }
    for (long i = 0; i < N; i++) for (int d = 0; d < 3; d++) {
        if (xyz[3 * i + d] < lo[d]) lo[d] = xyz[3 * i + d];
        if (xyz[3 * i + d] > hi[d]) hi[d] = xyz[3 * i + d];
    }
    for (int d = 0; d < 3; d++) {
        span[d] = hi[d] - lo[d];
        if (((axes >> d) & 1u) && !(span[d] > 0)) return ORC_E_BADARG;
        tol[d] = rel_tol * span[d];
        h[d] = span[d] > 0 ? 4.0 * tol[d] : 1.0;
    }
    /* pass 1: representatives, numbered in ascending node index */
    long nrep = 0;
    for (long i = 0; i < N; i++) {
        int wrapped = 0;
        for (int d = 0; d < 3; d++) if (((axes >> d) & 1u) && xyz[3 * i + d] >= hi[d] - tol[d]) wrapped = 1;
        dof[i] = wrapped ? -1 : (int)nrep++;
    }
    *ndof_out = nrep;
    if (nrep == N) return ORC_OK;
    /* hash map: cell of side 4 tol -> chain of representatives */
    long nb = 1; while (nb < 2 * nrep) nb <<= 1;
    int *head = (int *)malloc((size_t)nb * sizeof(int)), *next = (int *)malloc((size_t)N * sizeof(int));
    if (!head || !next) { free(head); free(next); return ORC_E_ALLOC; }
    for (long b = 0; b < nb; b++) head[b] = -1;
    for (long i = 0; i < N; i++) {
        if (dof[i] < 0) continue;
        long long c[3];
        for (int d = 0; d < 3; d++) c[d] = (long long)floor((xyz[3 * i + d] - lo[d]) / h[d]);
        unsigned long long b = cell_hash(c[0], c[1], c[2]) & (unsigned long long)(nb - 1);
        next[i] = head[b]; head[b] = (int)i;
    }
    int rc = ORC_OK;
    for (long i = 0; i < N && rc == ORC_OK; i++) {
        if (dof[i] >= 0) continue;
        double w[3]; long long c[3];
        for (int d = 0; d < 3; d++) {
            w[d] = xyz[3 * i + d];
            if (((axes >> d) & 1u) && w[d] >= hi[d] - tol[d]) w[d] -= span[d];
            c[d] = (long long)floor((w[d] - lo[d]) / h[d]);
        }
        int found = -1, count = 0;
        for (int a = -1; a <= 1; a++) for (int bq = -1; bq <= 1; bq++) for (int cq = -1; cq <= 1; cq++) {
            long long cx = c[0] + a, cy = c[1] + bq, cz = c[2] + cq;
            unsigned long long b = cell_hash(cx, cy, cz) & (unsigned long long)(nb - 1);
            for (int j = head[b]; j >= 0; j = next[j]) {
                /* the chain of a bucket may hold other cells (hash collisions): test the cell, then the distance */
                if ((long long)floor((xyz[3 * j] - lo[0]) / h[0]) != cx || (long long)floor((xyz[3 * j + 1] - lo[1]) / h[1]) != cy ||
                    (long long)floor((xyz[3 * j + 2] - lo[2]) / h[2]) != cz) continue;
                if (fabs(xyz[3 * j] - w[0]) <= tol[0] && fabs(xyz[3 * j + 1] - w[1]) <= tol[1] && fabs(xyz[3 * j + 2] - w[2]) <= tol[2]) {
                    found = j; count++;
                }
            }
        }
        if (count != 1) rc = ORC_E_BADARG; else dof[i] = dof[found];
    }
    free(head); free(next);
    return rc;
}

/* ------------------------------------------------------------------------------------ */
/* O-1 geometry, O-2 matrices                                                            */
/* ------------------------------------------------------------------------------------ */

/* B_i^T C B_j for Voigt order xx,yy,zz,yz,xz,xy with engineering shears (P:476 order). */
static void strain_disp(const double g[3], double B[6][3])
{
    memset(B, 0, 18 * sizeof(double));
    B[0][0] = g[0]; B[1][1] = g[1]; B[2][2] = g[2];
    B[3][1] = g[2]; B[3][2] = g[1];
    B[4][0] = g[2]; B[4][2] = g[0];
    B[5][0] = g[1]; B[5][1] = g[0];
}

static long find_col(const oracle *o, long i, int j)
{
    for (long q = o->rowptr[i]; q < o->rowptr[i + 1]; q++) if (o->col[q] == j) return q;
    return -1;
}

void orc_destroy(oracle *o);
void orc_voigt_rotation(const double *R, double *M);

static int finish_matrices(oracle *o, const double *K, const double *Km, const double *Mm, const double *Kme);

/* O-0 nondimensionalisation and Appendix D (R25): R (all zeros = identity) must be a
 * proper rotation; C_sim = M C_crystal M^T (Eq. D.4, Alg. D.1 line 1).  Shared by tetrahedra and hexahedra. */
static int setup_material(oracle *o, const orc_material *mat, double dt)
{
    double ld = mat->length_scale, mu0Ms2 = MU0 * mat->Ms * mat->Ms;
    o->Ms = mat->Ms; o->dt = dt;
    o->Astar = 2.0 * mat->Aex / (mu0Ms2 * ld * ld);
    o->Kstar = mat->K1 / mu0Ms2;
    o->dtau = mat->gamma * mat->Ms * dt;
    o->alpha = mat->alpha;
    o->eps1 = o->Astar * o->dtau;              /* Step 1 */
    o->eps2 = o->alpha * o->Astar * o->dtau;   /* Step 3 */
    o->lam100 = mat->lambda100; o->lam111 = mat->lambda111;
    memcpy(o->Nd, mat->Nd, sizeof(o->Nd));
    for (int q = 0; q < 6; q++) o->sext[q] = mat->sigma_ext[q] / mu0Ms2;
    o->n_elastic = mat->n_elastic > 0 ? mat->n_elastic : 0;
    o->Cstar = (double *)calloc((size_t)(o->n_elastic > 0 ? o->n_elastic : 1) * 36, sizeof(double));
    double nrm = 0; for (int q = 0; q < 9; q++) nrm += mat->R[q] * mat->R[q];
    for (int q = 0; q < 9; q++) o->R[q] = nrm == 0 ? (q % 4 == 0 ? 1.0 : 0.0) : mat->R[q];
    double dev = 0;
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) {
        double acc = 0; for (int k = 0; k < 3; k++) acc += o->R[3 * i + k] * o->R[3 * j + k];
        dev = fmax(dev, fabs(acc - (i == j)));
    }
    const double *r = o->R;
    double det = r[0] * (r[4] * r[8] - r[5] * r[7]) - r[1] * (r[3] * r[8] - r[5] * r[6]) + r[2] * (r[3] * r[7] - r[4] * r[6]);
    if (dev > 1e-10 || det < 0) return ORC_E_BADARG;
    o->rot = 0;
    for (int q = 0; q < 9; q++) if (o->R[q] != (q % 4 == 0 ? 1.0 : 0.0)) o->rot = 1;
    for (int k = 0; k < o->n_elastic; k++) {
        const double *C = mat->C_voigt + 36 * k;
        double M[36], MC[36];
        if (!o->rot) { for (int q = 0; q < 36; q++) o->Cstar[36 * k + q] = C[q] / mu0Ms2; continue; }
        orc_voigt_rotation(o->R, M);
        for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) { double acc = 0; for (int c = 0; c < 6; c++) acc += M[6 * a + c] * C[6 * c + b]; MC[6 * a + b] = acc; }
        for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) { double acc = 0; for (int c = 0; c < 6; c++) acc += MC[6 * a + c] * M[6 * b + c]; o->Cstar[36 * k + 6 * a + b] = acc / mu0Ms2; }
    }
    return ORC_OK;
}

/* Periodic boundary conditions: `dof` (NULL = identity) maps each of the Ng geometric nodes to one of N
 * unified degrees of freedom ("the two nodes in the pair are treated as one unified node").  Element geometry is
 * computed from the element's own corner coordinates; every nodal quantity (matrix rows, lumped masses, fields)
 * is indexed by DOF. */
int orc_create_wrapped(const double *xyz_m, long Ng, const int *gtets, long Ne, const uchar *magnetic,
                       const int *elastic_id, const int *dof, long N, const orc_material *mat, double dt,
                       const uchar *clamp_dof, long pin_node, oracle **out)
{
    if (!xyz_m || !gtets || !mat || !out || N <= 0 || Ng <= 0 || Ne <= 0) return ORC_E_BADARG;
    if (!dof && N != Ng) return ORC_E_BADARG;
    oracle *o = (oracle *)calloc(1, sizeof(oracle));
    if (!o) return ORC_E_ALLOC;
    o->N = N; o->Ne = Ne;
    int *tets = (int *)malloc((size_t)Ne * 4 * sizeof(int));   /* DOF connectivity */
    if (!tets) { free(o); return ORC_E_ALLOC; }
    for (long q = 0; q < 4 * Ne; q++) {
        if (gtets[q] < 0 || gtets[q] >= Ng) { free(tets); free(o); return ORC_E_RANGE; }
        tets[q] = dof ? dof[gtets[q]] : gtets[q];
        if (tets[q] < 0 || tets[q] >= N) { free(tets); free(o); return ORC_E_RANGE; }
    }
    if (dof) for (long e = 0; e < Ne; e++) /* two corners on one DOF: the domain is a single cell wide in a periodic direction */
        for (int i = 0; i < 4; i++) for (int j = i + 1; j < 4; j++)
            if (tets[4 * e + i] == tets[4 * e + j]) { free(tets); free(o); return ORC_E_BADARG; }
    double ld = mat->length_scale;
    if (setup_material(o, mat, dt)) { free(tets); free(o->Cstar); free(o); return ORC_E_BADARG; }

    o->x = (double *)malloc((size_t)Ng * 3 * sizeof(double));
    o->tet = tets;
    o->mag = (uchar *)malloc((size_t)Ne);
    o->eid = (int *)calloc((size_t)Ne, sizeof(int));
    o->V = (real *)malloc((size_t)Ne * sizeof(real));
    o->G = (real *)malloc((size_t)Ne * 12 * sizeof(real));
    o->mL = (real *)malloc((size_t)N * sizeof(real));
    o->mLm = (real *)malloc((size_t)N * sizeof(real));
    o->live = (uchar *)calloc((size_t)N, 1);
    o->clamp = (uchar *)calloc((size_t)N * 3, 1);
    if (!o->x || !o->tet || !o->mag || !o->eid || !o->V || !o->G || !o->mL || !o->mLm || !o->live || !o->clamp) { orc_destroy(o); return ORC_E_ALLOC; }
    for (long i = 0; i < 3 * Ng; i++) o->x[i] = xyz_m[i] / ld;
    for (long e = 0; e < Ne; e++) o->mag[e] = magnetic ? (magnetic[e] != 0) : 1;
    if (elastic_id) memcpy(o->eid, elastic_id, (size_t)Ne * sizeof(int));
    if (clamp_dof) for (long i = 0; i < 3 * N; i++) o->clamp[i] = clamp_dof[i] != 0;
    o->pin = pin_node;
    for (long e = 0; e < Ne; e++) {
        if (o->n_elastic && (o->eid[e] < 0 || o->eid[e] >= o->n_elastic)) { orc_destroy(o); return ORC_E_RANGE; }
    }
    if (pin_node < 0 || pin_node >= N) { orc_destroy(o); return ORC_E_BADARG; }

    /* O-1: V_e = |det J|/6, grad phi_k = k-th row of J^-1 (k=1..3), grad phi_0 = -sum */
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (long i = 0; i < Ng; i++) for (int d = 0; d < 3; d++) {
        if (o->x[3 * i + d] < lo[d]) lo[d] = o->x[3 * i + d];
        if (o->x[3 * i + d] > hi[d]) hi[d] = o->x[3 * i + d];
    }
    double diag = sqrt((hi[0] - lo[0]) * (hi[0] - lo[0]) + (hi[1] - lo[1]) * (hi[1] - lo[1]) + (hi[2] - lo[2]) * (hi[2] - lo[2]));
    double Vmin = 1e-14 * diag * diag * diag;
    double *mL = (double *)calloc((size_t)N, sizeof(double)), *mLm = (double *)calloc((size_t)N, sizeof(double));
    o->Vtot = 0; o->Vmag = 0;
    for (long e = 0; e < Ne; e++) {
        const double *x0 = o->x + 3 * gtets[4 * e], *x1 = o->x + 3 * gtets[4 * e + 1],
                     *x2 = o->x + 3 * gtets[4 * e + 2], *x3 = o->x + 3 * gtets[4 * e + 3];
        double a[3], b[3], c[3];
        for (int d = 0; d < 3; d++) { a[d] = x1[d] - x0[d]; b[d] = x2[d] - x0[d]; c[d] = x3[d] - x0[d]; }
        double bc[3] = {b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0]};
        double ca[3] = {c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0]};
        double ab[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
        double det = a[0] * bc[0] + a[1] * bc[1] + a[2] * bc[2];
        double V = fabs(det) / 6.0;
        if (!(V > Vmin)) { free(mL); free(mLm); orc_destroy(o); return ORC_E_DEGENERATE; }
        double g[4][3];
        for (int d = 0; d < 3; d++) {
            g[1][d] = bc[d] / det; g[2][d] = ca[d] / det; g[3][d] = ab[d] / det;
            g[0][d] = -(g[1][d] + g[2][d] + g[3][d]);
        }
        o->V[e] = (real)V;
        for (int k = 0; k < 4; k++) for (int d = 0; d < 3; d++) o->G[12 * e + 3 * k + d] = (real)g[k][d];
        o->Vtot += V;
        if (o->mag[e]) o->Vmag += V;
        for (int k = 0; k < 4; k++) {
            mL[tets[4 * e + k]] += V / 4.0;            /* int_e phi_i = V_e/4 */
            if (o->mag[e]) { mLm[tets[4 * e + k]] += V / 4.0; o->live[tets[4 * e + k]] = 1; }
        }
    }
    for (long i = 0; i < N; i++) { o->mL[i] = (real)mL[i]; o->mLm[i] = (real)mLm[i]; }
    free(mL); free(mLm);

    int rc = build_n2e(N, Ne, o->tet, &o->n2e_ptr, &o->n2e); if (rc) { orc_destroy(o); return rc; }
    rc = build_pattern(N, o->tet, o->n2e_ptr, o->n2e, &o->rowptr, &o->col, &o->nnz); if (rc) { orc_destroy(o); return rc; }

    /* O-2 (Eq. 12): accumulate in fp64 in element order, round once (R20). */
    long nnz = o->nnz;
    double *K = (double *)calloc((size_t)nnz, sizeof(double)), *Km = (double *)calloc((size_t)nnz, sizeof(double)),
           *Mm = (double *)calloc((size_t)nnz, sizeof(double));
    double *Kme = o->n_elastic ? (double *)calloc((size_t)nnz * 9, sizeof(double)) : NULL;
    if (!K || !Km || !Mm || (o->n_elastic && !Kme)) { orc_destroy(o); return ORC_E_ALLOC; }
    for (long e = 0; e < Ne; e++) {
        /* recompute the fp64 geometry of this element (not the rounded copy) */
        const int *t = tets + 4 * e, *tg = gtets + 4 * e;
        const double *x0 = o->x + 3 * tg[0], *x1 = o->x + 3 * tg[1], *x2 = o->x + 3 * tg[2], *x3 = o->x + 3 * tg[3];
        double a[3], b[3], c[3];
        for (int d = 0; d < 3; d++) { a[d] = x1[d] - x0[d]; b[d] = x2[d] - x0[d]; c[d] = x3[d] - x0[d]; }
        double bc[3] = {b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0]};
        double ca[3] = {c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0]};
        double ab[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
        double det = a[0] * bc[0] + a[1] * bc[1] + a[2] * bc[2];
        double V = fabs(det) / 6.0, g[4][3];
        for (int d = 0; d < 3; d++) {
            g[1][d] = bc[d] / det; g[2][d] = ca[d] / det; g[3][d] = ab[d] / det;
            g[0][d] = -(g[1][d] + g[2][d] + g[3][d]);
        }
        const double *C = o->n_elastic ? o->Cstar + 36 * o->eid[e] : NULL;
        for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) {
            long q = find_col(o, t[i], t[j]);
            double kij = V * (g[i][0] * g[j][0] + g[i][1] * g[j][1] + g[i][2] * g[j][2]); /* int grad.grad */
            double mij = V * (i == j ? 2.0 : 1.0) / 20.0;                                 /* int phi phi  */
            K[q] += kij;
            if (o->mag[e]) { Km[q] += kij; Mm[q] += mij; }
            if (C) {
                double Bi[6][3], Bj[6][3], CB[6][3];
                strain_disp(g[i], Bi); strain_disp(g[j], Bj);
                for (int r = 0; r < 6; r++) for (int s = 0; s < 3; s++) {
                    double acc = 0; for (int w = 0; w < 6; w++) acc += C[6 * r + w] * Bj[w][s];
                    CB[r][s] = acc;
                }
                for (int r = 0; r < 3; r++) for (int s = 0; s < 3; s++) {
                    double acc = 0; for (int w = 0; w < 6; w++) acc += Bi[w][r] * CB[w][s];
                    Kme[9 * q + 3 * r + s] += V * acc;
                }
            }
        }
    }
    rc = finish_matrices(o, K, Km, Mm, Kme);
    if (rc) { free(K); free(Km); free(Mm); free(Kme); orc_destroy(o); return rc; }
    free(K); free(Km); free(Mm); free(Kme);
    *out = o;
    return ORC_OK;
}

int orc_create(const double *xyz_m, long N, const int *tets, long Ne, const uchar *magnetic,
               const int *elastic_id, const orc_material *mat, double dt, const uchar *clamp_dof,
               long pin_node, oracle **out)
{
    return orc_create_wrapped(xyz_m, N, tets, Ne, magnetic, elastic_id, NULL, N, mat, dt, clamp_dof, pin_node, out);
}

/* round the fp64 sums once (R20); constraints as the symmetric projection P A P + (I - P) (R11);
 * K^GS(eps) = M_m + eps K_m with identity rows on dead nodes (R12) */
static int finish_matrices(oracle *o, const double *K, const double *Km, const double *Mm, const double *Kme)
{
    long N = o->N, nnz = o->nnz;
    o->K = (real *)malloc((size_t)nnz * sizeof(real)); o->Kms = (real *)malloc((size_t)nnz * sizeof(real));
    o->Km = (real *)malloc((size_t)nnz * sizeof(real)); o->Mm = (real *)malloc((size_t)nnz * sizeof(real));
    o->Kgs1 = (real *)malloc((size_t)nnz * sizeof(real)); o->Kgs2 = (real *)malloc((size_t)nnz * sizeof(real));
    if (Kme) { o->Kmech = (real *)malloc((size_t)nnz * 9 * sizeof(real)); o->Kmech_free = (real *)malloc((size_t)nnz * 9 * sizeof(real)); }
    if (!o->K || !o->Kms || !o->Km || !o->Mm || !o->Kgs1 || !o->Kgs2 || (Kme && (!o->Kmech || !o->Kmech_free))) return ORC_E_ALLOC;
    for (long i = 0; i < N; i++)
        for (long q = o->rowptr[i]; q < o->rowptr[i + 1]; q++) {
            long j = o->col[q];
            o->K[q] = (real)K[q]; o->Km[q] = (real)Km[q]; o->Mm[q] = (real)Mm[q];
            double kms = K[q];
            if (i == o->pin || j == o->pin) kms = (i == j) ? 1.0 : 0.0;
            o->Kms[q] = (real)kms;
            double dead = (i == j && !o->live[i]) ? 1.0 : 0.0;
            o->Kgs1[q] = (real)(Mm[q] + o->eps1 * Km[q] + dead);
            o->Kgs2[q] = (real)(Mm[q] + o->eps2 * Km[q] + dead);
            if (Kme) for (int r = 0; r < 3; r++) for (int s = 0; s < 3; s++) {
                double v = Kme[9 * q + 3 * r + s];
                o->Kmech_free[9 * q + 3 * r + s] = (real)v;
                if (o->clamp[3 * i + r] || o->clamp[3 * j + s]) v = (i == j && r == s) ? 1.0 : 0.0;
                o->Kmech[9 * q + 3 * r + s] = (real)v;
            }
        }
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------ */
/* Linear hexahedral (Q1) elements (R26) */
/* ------------------------------------------------------------------------------------ */
/* "Currently, only linear hexahedral and tetrahedral Lagrange elements are supported"; the paper's Fig. 2-3
 * workloads are structured hexahedral meshes.  Trilinear shape functions on the reference cube
 * [-1,1]^3, local node a = i + 2 j + 4 k <-> (xi, eta, zeta) = (2i-1, 2j-1, 2k-1):
 *   phi_a = (1 + xi_a xi)(1 + eta_a eta)(1 + zeta_a zeta) / 8,
 * integrated with the 2 x 2 x 2 Gauss rule (points +-1/sqrt 3, unit weights; Eq. 17's |J(e,p)| w_p):
 *   K_ab = sum_p |J_p| grad phi_a . grad phi_b,  M_ab = sum_p |J_p| phi_a phi_b,  K^mech_ab = sum_p |J_p| B_a^T C B_b,
 *   grad phi_a = J^-T grad_xi phi_a,  J = sum_a x_a (x) grad_xi phi_a.
 * Covered: the matrices of Eq. 12 (K^ms, K^GS, M, K^mech with their constraints), the lumped masses int phi_a, the
 * volume average of Eq. 17, and every element-wise right-hand side and recovered field of the GSPM step (hex_* below). */
static void hex_gauss_point(const double *X /* 8 x 3 */, int p, double *detJ, double phi[8], double g[8][3])
{
    const double q = 0.57735026918962576451; /* 1/sqrt(3) */
    double xi[3] = {(p & 1) ? q : -q, (p & 2) ? q : -q, (p & 4) ? q : -q};
    double dN[8][3], J[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    for (int a = 0; a < 8; a++) {
        double s[3] = {(a & 1) ? 1.0 : -1.0, (a & 2) ? 1.0 : -1.0, (a & 4) ? 1.0 : -1.0};
        double f[3] = {1 + s[0] * xi[0], 1 + s[1] * xi[1], 1 + s[2] * xi[2]};
        phi[a] = f[0] * f[1] * f[2] / 8;
        dN[a][0] = s[0] * f[1] * f[2] / 8; dN[a][1] = f[0] * s[1] * f[2] / 8; dN[a][2] = f[0] * f[1] * s[2] / 8;
        for (int r = 0; r < 3; r++) for (int c = 0; c < 3; c++) J[r][c] += X[3 * a + r] * dN[a][c]; /* J_rc = d x_r / d xi_c */
    }
    double cof[3][3];
    cof[0][0] = J[1][1] * J[2][2] - J[1][2] * J[2][1]; cof[0][1] = J[1][2] * J[2][0] - J[1][0] * J[2][2]; cof[0][2] = J[1][0] * J[2][1] - J[1][1] * J[2][0];
    cof[1][0] = J[0][2] * J[2][1] - J[0][1] * J[2][2]; cof[1][1] = J[0][0] * J[2][2] - J[0][2] * J[2][0]; cof[1][2] = J[0][1] * J[2][0] - J[0][0] * J[2][1];
    cof[2][0] = J[0][1] * J[1][2] - J[0][2] * J[1][1]; cof[2][1] = J[0][2] * J[1][0] - J[0][0] * J[1][2]; cof[2][2] = J[0][0] * J[1][1] - J[0][1] * J[1][0];
    double det = J[0][0] * cof[0][0] + J[0][1] * cof[0][1] + J[0][2] * cof[0][2];
    *detJ = det;
    /* grad phi_a = J^-T grad_xi phi_a;  (J^-1)_cr = cof_rc / det  =>  (grad phi_a)_r = sum_c cof_rc dN_ac / det */
    for (int a = 0; a < 8; a++)
        for (int r = 0; r < 3; r++) g[a][r] = (cof[r][0] * dN[a][0] + cof[r][1] * dN[a][1] + cof[r][2] * dN[a][2]) / det;
}

/* dof (NULL = identity): periodic node wrapping as for tetrahedra: geometry from the cell's own corners, every
 * nodal quantity indexed by DOF. */
int orc_create_hex(const double *xyz_m, long Ng, const int *hexes, long Ne, const uchar *magnetic, const int *elastic_id,
                   const int *dof, long N, const orc_material *mat, double dt, const uchar *clamp_dof, long pin_node, oracle **out)
{
    if (!xyz_m || !hexes || !mat || !out || N <= 0 || Ng <= 0 || Ne <= 0 || pin_node < 0 || pin_node >= N) return ORC_E_BADARG;
    if (!dof && N != Ng) return ORC_E_BADARG;
    for (long q = 0; q < 8 * Ne; q++) if (hexes[q] < 0 || hexes[q] >= Ng) return ORC_E_RANGE;
    if (dof) {
        for (long i = 0; i < Ng; i++) if (dof[i] < 0 || dof[i] >= N) return ORC_E_RANGE;
        for (long e = 0; e < Ne; e++)
            for (int a = 0; a < 8; a++) for (int b = a + 1; b < 8; b++)
                if (dof[hexes[8 * e + a]] == dof[hexes[8 * e + b]]) return ORC_E_BADARG; /* one cell wide in a periodic direction */
    }
    oracle *o = (oracle *)calloc(1, sizeof(oracle));
    if (!o) return ORC_E_ALLOC;
    o->N = N; o->Ne = Ne; o->nen = 8;
    double ld = mat->length_scale;
    if (setup_material(o, mat, dt)) { free(o->Cstar); free(o); return ORC_E_BADARG; }   /* App. D applies to hexahedra too */
    o->x = (double *)malloc((size_t)Ng * 3 * sizeof(double));
    o->hex = (int *)malloc((size_t)Ne * 8 * sizeof(int));
    o->ghex = (int *)malloc((size_t)Ne * 8 * sizeof(int));
    o->mag = (uchar *)malloc((size_t)Ne);
    o->eid = (int *)calloc((size_t)Ne, sizeof(int));
    o->V = (real *)malloc((size_t)Ne * sizeof(real));
    o->mL = (real *)malloc((size_t)N * sizeof(real)); o->mLm = (real *)malloc((size_t)N * sizeof(real));
    o->live = (uchar *)calloc((size_t)N, 1);
    o->clamp = (uchar *)calloc((size_t)N * 3, 1);
    for (long i = 0; i < 3 * Ng; i++) o->x[i] = xyz_m[i] / ld;
    memcpy(o->ghex, hexes, (size_t)Ne * 8 * sizeof(int));
    for (long q = 0; q < 8 * Ne; q++) o->hex[q] = dof ? dof[hexes[q]] : hexes[q];
    for (long e = 0; e < Ne; e++) o->mag[e] = magnetic ? (magnetic[e] != 0) : 1;
    if (elastic_id) memcpy(o->eid, elastic_id, (size_t)Ne * sizeof(int));
    if (clamp_dof) for (long i = 0; i < 3 * N; i++) o->clamp[i] = clamp_dof[i] != 0;
    o->pin = pin_node;
    for (long e = 0; e < Ne; e++) if (o->n_elastic && (o->eid[e] < 0 || o->eid[e] >= o->n_elastic)) { orc_destroy(o); return ORC_E_RANGE; }

    /* pattern: { j : i, j share a hexahedron } U { i }, ascending */
    int rc = build_n2e_n(N, Ne, o->hex, 8, &o->n2e_ptr, &o->n2e); if (rc) { orc_destroy(o); return rc; }
    rc = build_pattern_n(N, o->hex, 8, o->n2e_ptr, o->n2e, &o->rowptr, &o->col, &o->nnz); if (rc) { orc_destroy(o); return rc; }
    long nnz = o->nnz;
    double *K = (double *)calloc((size_t)nnz, sizeof(double)), *Km = (double *)calloc((size_t)nnz, sizeof(double)),
           *Mm = (double *)calloc((size_t)nnz, sizeof(double)), *mL = (double *)calloc((size_t)N, sizeof(double)),
           *mLm = (double *)calloc((size_t)N, sizeof(double));
    double *Kme = o->n_elastic ? (double *)calloc((size_t)nnz * 9, sizeof(double)) : NULL;
    if (!K || !Km || !Mm || !mL || !mLm || (o->n_elastic && !Kme)) { orc_destroy(o); return ORC_E_ALLOC; }
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (long i = 0; i < Ng; i++) for (int d = 0; d < 3; d++) {
        if (o->x[3 * i + d] < lo[d]) lo[d] = o->x[3 * i + d];
        if (o->x[3 * i + d] > hi[d]) hi[d] = o->x[3 * i + d];
    }
    double diag = sqrt((hi[0] - lo[0]) * (hi[0] - lo[0]) + (hi[1] - lo[1]) * (hi[1] - lo[1]) + (hi[2] - lo[2]) * (hi[2] - lo[2]));
    double Jmin = 1e-14 * diag * diag * diag;
    o->Vtot = 0; o->Vmag = 0;
    for (long e = 0; e < Ne; e++) {
        const int *t = o->hex + 8 * e, *tg = o->ghex + 8 * e;
        double X[24];
        for (int a = 0; a < 8; a++) for (int d = 0; d < 3; d++) X[3 * a + d] = o->x[3 * (long)tg[a] + d];
        const double *C = o->n_elastic ? o->Cstar + 36 * o->eid[e] : NULL;
        double Ve = 0;
        for (int p = 0; p < 8; p++) {
            double det, phi[8], g[8][3];
            hex_gauss_point(X, p, &det, phi, g);
            if (!(det > Jmin)) { free(K); free(Km); free(Mm); free(mL); free(mLm); free(Kme); orc_destroy(o); return ORC_E_DEGENERATE; }
            Ve += det;
            for (int a = 0; a < 8; a++) {
                mL[t[a]] += det * phi[a];
                if (o->mag[e]) { mLm[t[a]] += det * phi[a]; o->live[t[a]] = 1; }
                for (int b = 0; b < 8; b++) {
                    long q = find_col(o, t[a], t[b]);
                    double kab = det * (g[a][0] * g[b][0] + g[a][1] * g[b][1] + g[a][2] * g[b][2]);
                    double mab = det * phi[a] * phi[b];
                    K[q] += kab;
                    if (o->mag[e]) { Km[q] += kab; Mm[q] += mab; }
                    if (C) {
                        double Ba[6][3], Bb[6][3], CB[6][3];
                        strain_disp(g[a], Ba); strain_disp(g[b], Bb);
                        for (int r = 0; r < 6; r++) for (int s = 0; s < 3; s++) {
                            double acc = 0; for (int w = 0; w < 6; w++) acc += C[6 * r + w] * Bb[w][s];
                            CB[r][s] = acc;
                        }
                        for (int r = 0; r < 3; r++) for (int s = 0; s < 3; s++) {
                            double acc = 0; for (int w = 0; w < 6; w++) acc += Ba[w][r] * CB[w][s];
                            Kme[9 * q + 3 * r + s] += det * acc;
                        }
                    }
                }
            }
        }
        o->V[e] = (real)Ve;
        o->Vtot += Ve;
        if (o->mag[e]) o->Vmag += Ve;
    }
    for (long i = 0; i < N; i++) { o->mL[i] = (real)mL[i]; o->mLm[i] = (real)mLm[i]; }
    rc = finish_matrices(o, K, Km, Mm, Kme);
    free(K); free(Km); free(Mm); free(mL); free(mLm); free(Kme);
    if (rc) { orc_destroy(o); return rc; }
    *out = o;
    return ORC_OK;
}

void orc_destroy(oracle *o)
{
    if (!o) return;
    free(o->hex); free(o->ghex);
    free(o->x); free(o->tet); free(o->mag); free(o->eid); free(o->V); free(o->G); free(o->mL); free(o->mLm);
    free(o->live); free(o->n2e_ptr); free(o->n2e); free(o->rowptr); free(o->col); free(o->K); free(o->Kms);
    free(o->Km); free(o->Mm); free(o->Kgs1); free(o->Kgs2); free(o->Kmech); free(o->Kmech_free); free(o->clamp);
    free(o->Cstar); free(o);
}

/* accessors: sizes, then copies */
long orc_nnz(const oracle *o) { return o->nnz; }
double orc_scalar(const oracle *o, int what)
{
    switch (what) {
    case 0: return o->Vtot; case 1: return o->Vmag; case 2: return o->Astar; case 3: return o->Kstar;
    case 4: return o->dtau; case 5: return o->eps1; case 6: return o->eps2;
    } return NAN;
}
/* what: 0 rowptr(int N+1) 1 col(int nnz) 2 n2e_ptr(int N+1) 3 n2e(int 4Ne) 4 V(real Ne) 5 G(real 12Ne)
 *       6 mL(real N) 7 mLm(real N) 8 live(uchar N) */
int orc_get(const oracle *o, int what, void *dst)
{
    switch (what) {
    case 0: memcpy(dst, o->rowptr, (size_t)(o->N + 1) * sizeof(int)); break;
    case 1: memcpy(dst, o->col, (size_t)o->nnz * sizeof(int)); break;
    case 2: memcpy(dst, o->n2e_ptr, (size_t)(o->N + 1) * sizeof(int)); break;
    case 3: memcpy(dst, o->n2e, (size_t)o->Ne * (o->nen == 8 ? 8 : 4) * sizeof(int)); break;
    case 4: memcpy(dst, o->V, (size_t)o->Ne * sizeof(real)); break;
    case 5: if (o->nen == 8) return ORC_E_BADARG; memcpy(dst, o->G, (size_t)o->Ne * 12 * sizeof(real)); break;
    case 6: memcpy(dst, o->mL, (size_t)o->N * sizeof(real)); break;
    case 7: memcpy(dst, o->mLm, (size_t)o->N * sizeof(real)); break;
    case 8: memcpy(dst, o->live, (size_t)o->N); break;
    default: return ORC_E_BADARG;
    }
    return ORC_OK;
}

static const real *mat_values(const oracle *o, int id, int *bs)
{
    *bs = 1;
    switch (id) {
    case MAT_K_MS: return o->Kms; case MAT_K_GS1: return o->Kgs1; case MAT_K_GS2: return o->Kgs2;
    case MAT_MASS: return o->Mm; case MAT_K_FREE: return o->K; case MAT_K_M: return o->Km;
    case MAT_K_MECH: *bs = 3; return o->Kmech; case MAT_K_MECH_FREE: *bs = 3; return o->Kmech_free;
    } return NULL;
}

int orc_get_values(const oracle *o, int id, void *dst)
{
    int bs; const real *v = mat_values(o, id, &bs);
    if (!v) return ORC_E_BADARG;
    memcpy(dst, v, (size_t)o->nnz * bs * bs * sizeof(real));
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------ */
/* SpMV and O-4 CG                                                                       */
/* ------------------------------------------------------------------------------------ */

/* y = A x.  Scalar matrices: x, y have `stride` interleaved components and component
 * `comp` is used (stride 1 for plain vectors).  Block matrices: x, y are N x 3. */
static void spmv(const oracle *o, int id, const real *x, real *y, int stride, int comp)
{
    int bs; const real *v = mat_values(o, id, &bs);
    long N = o->N;
    if (bs == 1) {
#pragma omp parallel for schedule(static)
        for (long i = 0; i < N; i++) {
            real acc = 0;
            for (long q = o->rowptr[i]; q < o->rowptr[i + 1]; q++) acc += v[q] * x[(long)o->col[q] * stride + comp];
            y[i * stride + comp] = acc;
        }
    } else {
#pragma omp parallel for schedule(static)
        for (long i = 0; i < N; i++) {
            real acc[3] = {0, 0, 0};
            for (long q = o->rowptr[i]; q < o->rowptr[i + 1]; q++) {
                const real *xb = x + 3 * (long)o->col[q], *a = v + 9 * q;
                for (int r = 0; r < 3; r++) acc[r] += a[3 * r] * xb[0] + a[3 * r + 1] * xb[1] + a[3 * r + 2] * xb[2];
            }
            y[3 * i] = acc[0]; y[3 * i + 1] = acc[1]; y[3 * i + 2] = acc[2];
        }
    }
}

int orc_spmv(const oracle *o, int id, const void *x, void *y)
{
    int bs; if (!mat_values(o, id, &bs)) return ORC_E_BADARG;
    spmv(o, id, (const real *)x, (real *)y, 1, 0);
    return ORC_OK;
}

/* Fixed-order dot product: partial sums over chunks of DOT_CHUNK consecutive entries (each summed in index order),
 * then the partials added in index order.  The result does not depend on the number of threads or on scheduling,
 * so two runs of the oracle are bit-identical. */
#define DOT_CHUNK 4096
static double dot(long n, const real *a, const real *b, int stride, int comp)
{
    long nch = (n + DOT_CHUNK - 1) / DOT_CHUNK;
    double *part = (double *)malloc((size_t)(nch > 0 ? nch : 1) * sizeof(double));
#pragma omp parallel for schedule(static)
    for (long c = 0; c < nch; c++) {
        long i1 = (c + 1) * DOT_CHUNK < n ? (c + 1) * DOT_CHUNK : n;
        double s = 0;
        for (long i = c * DOT_CHUNK; i < i1; i++) s += (double)a[i * stride + comp] * (double)b[i * stride + comp];
        part[c] = s;
    }
    double s = 0;
    for (long c = 0; c < nch; c++) s += part[c];
    free(part);
    return s;
}

/* Optional residual history of the solves that follow: hist[k] = ||r_k|| / ||b|| of the recurrence residual before
 * iteration k (k = 0 .. iters), for at most cap entries; *n = entries written by the LAST solve.  NULL switches it off. */
static double *g_hist = NULL; static int g_hist_cap = 0; static int *g_hist_n = NULL;
void orc_set_cg_history(double *hist, int cap, int *n) { g_hist = hist; g_hist_cap = cap; g_hist_n = n; }

/* z = D^-1 r with D = diag(A) (Jacobi; the paper's "future work" row: "no preconditioner by choice") */
static void apply_jacobi(const oracle *o, int id, const real *r, real *z, int stride, int comp)
{
    int bs; const real *v = mat_values(o, id, &bs);
    long N = o->N;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < N; i++) {
        long q = o->rowptr[i];
        while (o->col[q] != i) q++;                       /* the diagonal is always present (R21) */
        if (bs == 1) z[i * stride + comp] = r[i * stride + comp] / v[q];
        else for (int c = 0; c < 3; c++) z[3 * i + c] = r[3 * i + c] / v[9 * q + 4 * c];
    }
}

/* Textbook conjugate gradients (O-4).  precond = 0: unpreconditioned, as the paper runs it;
 * precond = 1: Jacobi-preconditioned (z = D^-1 r, beta = r.z ratios; SURVEY 8f unranked row).  Stop when
 * ||r|| < tol ||b|| (recurrence residual, the true 2-norm in both variants), tested before each iteration; fixed >= 0
 * runs exactly `fixed` iterations.  Dots in fp64; alpha, beta formed in fp64 and cast to the vector type. */
static int cg_pc(const oracle *o, int id, const real *b, real *x, int stride, int comp, double tol, int maxiter,
                 int fixed, int precond, int *iters, double *relres)
{
    int bs; mat_values(o, id, &bs);
    long N = o->N, n = (bs == 3) ? 3 * N : N;   /* entries visited through (stride, comp) */
    if (bs == 3) { stride = 1; comp = 0; }
    long len = (bs == 3) ? 3 * N : N * stride;
    real *r = (real *)calloc((size_t)len, sizeof(real)), *p = (real *)calloc((size_t)len, sizeof(real)),
         *Ap = (real *)calloc((size_t)len, sizeof(real)), *z = precond ? (real *)calloc((size_t)len, sizeof(real)) : NULL;
    int status = ORC_OK, k = 0;
    if (g_hist_n) *g_hist_n = 0;
    double bb = dot(n, b, b, stride, comp);
    if (bb == 0.0 && fixed < 0) {       /* ||b|| = 0 -> x = 0, 0 iterations */
        for (long i = 0; i < n; i++) x[i * stride + comp] = 0;
        *iters = 0; *relres = 0; free(r); free(p); free(Ap); free(z); return ORC_OK;
    }
    spmv(o, id, x, Ap, stride, comp);
    for (long i = 0; i < n; i++) r[i * stride + comp] = b[i * stride + comp] - Ap[i * stride + comp];
    if (precond) apply_jacobi(o, id, r, z, stride, comp);
    const real *zz = precond ? z : r;
    for (long i = 0; i < n; i++) p[i * stride + comp] = zz[i * stride + comp];
    double rr = dot(n, r, r, stride, comp);
    double rz = precond ? dot(n, r, z, stride, comp) : rr;
    for (;;) {
        if (g_hist && k < g_hist_cap) { g_hist[k] = bb > 0 ? sqrt(rr / bb) : 0.0; if (g_hist_n) *g_hist_n = k + 1; }
        if (rr == 0.0) break;
        if (fixed >= 0) { if (k == fixed) break; }
        else { if (rr < tol * tol * bb) break; if (k >= maxiter) { status = ORC_W_MAXITER; break; } }
        spmv(o, id, p, Ap, stride, comp);
        double pAp = dot(n, p, Ap, stride, comp);
        if (!(pAp > 0.0)) { status = ORC_E_BREAKDOWN; break; }
        real alpha = (real)(rz / pAp);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) {
            x[i * stride + comp] += alpha * p[i * stride + comp];
            r[i * stride + comp] -= alpha * Ap[i * stride + comp];
        }
        double rr_new = dot(n, r, r, stride, comp), rz_new = rr_new;
        if (precond) { apply_jacobi(o, id, r, z, stride, comp); rz_new = dot(n, r, z, stride, comp); }
        real beta = (real)(rz_new / rz);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; i++) p[i * stride + comp] = zz[i * stride + comp] + beta * p[i * stride + comp];
        rr = rr_new; rz = rz_new; k++;
    }
    *iters = k; *relres = bb > 0 ? sqrt(rr / bb) : 0.0;
    free(r); free(p); free(Ap); free(z);
    return status;
}

static int cg(const oracle *o, int id, const real *b, real *x, int stride, int comp, double tol, int maxiter,
              int fixed, int *iters, double *relres)
{
    return cg_pc(o, id, b, x, stride, comp, tol, maxiter, fixed, 0, iters, relres);
}

int orc_cg(const oracle *o, int id, const void *b, void *x, double tol, int maxiter, int fixed, int *iters, double *relres)
{
    int bs; if (!mat_values(o, id, &bs)) return ORC_E_BADARG;
    return cg(o, id, (const real *)b, (real *)x, 1, 0, tol, maxiter, fixed, iters, relres);
}

int orc_cg_pc(const oracle *o, int id, const void *b, void *x, double tol, int maxiter, int fixed, int precond, int *iters, double *relres)
{
    int bs; if (!mat_values(o, id, &bs) || precond < 0 || precond > 1) return ORC_E_BADARG;
    return cg_pc(o, id, (const real *)b, (real *)x, 1, 0, tol, maxiter, fixed, precond, iters, relres);
}

/* ------------------------------------------------------------------------------------ */
/* S2 volume average (Eq. 16-17).  For P1 tets the Gauss sum is exact:        */
/* int_e g = V_e * mean of the 4 nodal values.                                           */
/* ------------------------------------------------------------------------------------ */
int orc_volume_average(const oracle *o, const void *g_, int ncomp, double *out)
{
    const real *g = (const real *)g_;
    double den = 0; double num[16];
    if (ncomp < 1 || ncomp > 16) return ORC_E_BADARG;
    for (int c = 0; c < ncomp; c++) num[c] = 0;
    if (o->nen == 8) { /* Eq. 17 with the 2 x 2 x 2 Gauss rule: sum_e sum_p g_e(r_p) |J(e,p)| w_p */
        for (long e = 0; e < o->Ne; e++) {
            const int *t = o->hex + 8 * e, *tg = o->ghex + 8 * e;
            double X[24];
            for (int a = 0; a < 8; a++) for (int d = 0; d < 3; d++) X[3 * a + d] = o->x[3 * (long)tg[a] + d];
            for (int p = 0; p < 8; p++) {
                double det, phi[8], gr[8][3];
                hex_gauss_point(X, p, &det, phi, gr);
                for (int c = 0; c < ncomp; c++) {
                    double ge = 0;
                    for (int a = 0; a < 8; a++) ge += phi[a] * (double)g[(long)t[a] * ncomp + c];
                    num[c] += ge * det;
                }
                den += det;
            }
        }
        for (int c = 0; c < ncomp; c++) out[c] = num[c] / den;
        return ORC_OK;
    }
    for (long e = 0; e < o->Ne; e++) {
        const int *t = o->tet + 4 * e;
        for (int c = 0; c < ncomp; c++) {
            double ge = ((double)g[(long)t[0] * ncomp + c] + (double)g[(long)t[1] * ncomp + c] +
                         (double)g[(long)t[2] * ncomp + c] + (double)g[(long)t[3] * ncomp + c]) / 4.0;
            num[c] += ge * (double)o->V[e];
        }
        den += (double)o->V[e];
    }
    for (int c = 0; c < ncomp; c++) out[c] = num[c] / den;
    return ORC_OK;
}

/* ------------------------------------------------------------------------------------ */
/* S3 magnetostatic RHS (Eq. 9, 13, 14; R9 adjoint form):                                */
/* b_i = sum_{e contains i} V_e grad phi_i . (mean_e(m) - mbar); b[pin] = 0.             */
/* ------------------------------------------------------------------------------------ */
int orc_rhs_ms(const oracle *o, const void *m_, const double *mbar, void *b_)
{
    if (o->nen == 8) return hex_rhs_ms(o, (const real *)m_, mbar, (real *)b_);
    const real *m = (const real *)m_; real *b = (real *)b_;
    for (long i = 0; i < o->N; i++) b[i] = 0;
    for (long e = 0; e < o->Ne; e++) {
        const int *t = o->tet + 4 * e; const real *G = o->G + 12 * e;
        real mt[3];
        for (int d = 0; d < 3; d++)
            mt[d] = (m[3 * (long)t[0] + d] + m[3 * (long)t[1] + d] + m[3 * (long)t[2] + d] + m[3 * (long)t[3] + d]) / (real)4 - (real)mbar[d];
        for (int k = 0; k < 4; k++)
            b[t[k]] += o->V[e] * (G[3 * k] * mt[0] + G[3 * k + 1] * mt[1] + G[3 * k + 2] * mt[2]);
    }
    b[o->pin] = 0;
    return ORC_OK;
}

/* S5 gradient recovery and demagnetising field (Eq. 4, 15; R8, R10):
 * grad U_e = sum_k U_k grad phi_k;  <grad U> = sum_e V_e grad U_e / V;
 * h_d,i = -sum_{e contains i} V_e grad U_e/(4 mL_i) [+ <grad U>] (DEMAG)  - N_d mbar (FARFIELD). */
int orc_demag_field(const oracle *o, const void *U_, const double *mbar, unsigned terms, void *hd_, double *gradU_mean)
{
    if (o->nen == 8) return hex_demag_field(o, (const real *)U_, mbar, terms, (real *)hd_, gradU_mean);
    const real *U = (const real *)U_; real *hd = (real *)hd_;
    long N = o->N;
    for (long i = 0; i < 3 * N; i++) hd[i] = 0;
    double gm[3] = {0, 0, 0};
    if (terms & T_DEMAG) {
        double acc[3] = {0, 0, 0};
        for (long e = 0; e < o->Ne; e++) {
            const int *t = o->tet + 4 * e; const real *G = o->G + 12 * e;
            real gU[3];
            for (int d = 0; d < 3; d++) gU[d] = U[t[0]] * G[d] + U[t[1]] * G[3 + d] + U[t[2]] * G[6 + d] + U[t[3]] * G[9 + d];
            for (int d = 0; d < 3; d++) acc[d] += (double)o->V[e] * (double)gU[d];
            for (int k = 0; k < 4; k++) for (int d = 0; d < 3; d++) hd[3 * (long)t[k] + d] += o->V[e] * gU[d];
        }
        for (int d = 0; d < 3; d++) gm[d] = acc[d] / o->Vtot;
        for (long i = 0; i < N; i++) for (int d = 0; d < 3; d++)
            hd[3 * i + d] = -hd[3 * i + d] / ((real)4 * o->mL[i]) + (real)gm[d];
    }
    if (terms & T_FARFIELD)
        for (long i = 0; i < N; i++) for (int d = 0; d < 3; d++)
            hd[3 * i + d] -= (real)(o->Nd[3 * d] * mbar[0] + o->Nd[3 * d + 1] * mbar[1] + o->Nd[3 * d + 2] * mbar[2]);
    if (gradU_mean) for (int d = 0; d < 3; d++) gradU_mean[d] = gm[d];
    return ORC_OK;
}

/* E0(m), Table A.1, Voigt engineering vector (E11,E22,E33,2E23,2E13,2E12). */
/* ------------------------------------------------------------------------------------ */
/* Appendix D: rotated coordinate system (R25)                       */
/* ------------------------------------------------------------------------------------ */
/* Eq. D.3: the 6x6 matrix M with sigma_sim = M sigma_crystal for Voigt vectors (xx,yy,zz,yz,xz,xy) of tensor
 * components, so that C_sim = M C_crystal M^T (Eq. D.4) for a stiffness acting on engineering shears. */
void orc_voigt_rotation(const double *R, double *M)
{
    static const int I[6] = {0, 1, 2, 1, 0, 0}, J[6] = {0, 1, 2, 2, 2, 1};
    for (int a = 0; a < 6; a++) for (int b = 0; b < 6; b++) {
        int i = I[a], j = J[a], k = I[b], l = J[b];
        /* (R S R^T)_ij = sum_kl R_ik R_jl S_kl; S symmetric: off-diagonal (k,l) appears twice */
        M[6 * a + b] = (b < 3) ? R[3 * i + k] * R[3 * j + k] : R[3 * i + k] * R[3 * j + l] + R[3 * i + l] * R[3 * j + k];
    }
}

/* v_c = R^T v (m_100 = R^-1 m_111, Alg. D.1 Step 1) and v = R v_c (h_111 = R h_100, Step 4) */
static void to_crystal(const oracle *o, const real *v, real *vc)
{
    for (int a = 0; a < 3; a++) vc[a] = (real)o->R[a] * v[0] + (real)o->R[3 + a] * v[1] + (real)o->R[6 + a] * v[2];
}
static void to_sim(const oracle *o, const real *vc, real *v)
{
    for (int a = 0; a < 3; a++) v[a] = (real)o->R[3 * a] * vc[0] + (real)o->R[3 * a + 1] * vc[1] + (real)o->R[3 * a + 2] * vc[2];
}
/* symmetric tensor given as (xx,yy,zz,yz,xz,xy) tensor components: t_out = Q t Q^T with Q = R (inv = 0) or R^T (inv = 1) */
static void rotate_sym(const oracle *o, const real t[6], int inv, real out[6])
{
    real A[3][3] = {{t[0], t[5], t[4]}, {t[5], t[1], t[3]}, {t[4], t[3], t[2]}}, B[3][3], Q[3][3];
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) Q[i][j] = (real)(inv ? o->R[3 * j + i] : o->R[3 * i + j]);
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) { real acc = 0; for (int k = 0; k < 3; k++) acc += Q[i][k] * A[k][j]; B[i][j] = acc; }
    for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) { real acc = 0; for (int k = 0; k < 3; k++) acc += B[i][k] * Q[j][k]; A[i][j] = acc; }
    out[0] = A[0][0]; out[1] = A[1][1]; out[2] = A[2][2]; out[3] = A[1][2]; out[4] = A[0][2]; out[5] = A[0][1];
}

/* Table A.1 in crystal axes; engineering-shear Voigt vector */
static void E0_crystal(const oracle *o, const real *m, real e0[6])
{
    real l1 = (real)o->lam100, l2 = (real)o->lam111, th = (real)1.5;
    e0[0] = th * l1 * (m[0] * m[0] - (real)(1.0 / 3.0));
    e0[1] = th * l1 * (m[1] * m[1] - (real)(1.0 / 3.0));
    e0[2] = th * l1 * (m[2] * m[2] - (real)(1.0 / 3.0));
    e0[3] = (real)2 * th * l2 * m[1] * m[2];
    e0[4] = (real)2 * th * l2 * m[0] * m[2];
    e0[5] = (real)2 * th * l2 * m[0] * m[1];
}

/* E0 in the simulation frame: Alg. D.1 Step 1, E0_sim(m) = R E0_crystal(R^T m) R^T as a tensor (Eq. D.2) */
static void E0_voigt(const oracle *o, const real *m, real e0[6])
{
    if (!o->rot) { E0_crystal(o, m, e0); return; }
    real mc[3], ec[6], t[6];
    to_crystal(o, m, mc);
    E0_crystal(o, mc, ec);
    for (int q = 3; q < 6; q++) ec[q] /= (real)2;   /* engineering -> tensor shears */
    rotate_sym(o, ec, 0, t);
    for (int q = 0; q < 3; q++) { e0[q] = t[q]; e0[3 + q] = (real)2 * t[3 + q]; }
}

/* mean over the 4 nodes of a magnetic tet of E0(m_k) (R13) */
static void mean_E0(const oracle *o, const real *m, const int *t, real e0[6])
{
    for (int q = 0; q < 6; q++) e0[q] = 0;
    for (int k = 0; k < 4; k++) {
        real ek[6]; E0_voigt(o, m + 3 * (long)t[k], ek);
        for (int q = 0; q < 6; q++) e0[q] += ek[q];
    }
    for (int q = 0; q < 6; q++) e0[q] /= (real)4;
}

static void C_times(const oracle *o, long e, const real eps[6], real sig[6])
{
    const double *C = o->Cstar + 36 * o->eid[e];
    for (int r = 0; r < 6; r++) {
        real acc = 0;
        for (int s = 0; s < 6; s++) acc += (real)C[6 * r + s] * eps[s];
        sig[r] = acc;
    }
}

/* ------------------------------------------------------------------------------------ */
/* Element-wise right-hand sides on linear hexahedra (R26): the tetrahedral definitions   */
/* of O-3 with every element integral taken by the 2 x 2 x 2 Gauss rule:                  */
/*   b^ms_i     = sum_e sum_p |J_p| grad phi_i(p) . (m_h(p) - mbar),   m_h = sum_a phi_a m_a */
/*   h_d,i      = -[sum_e sum_p |J_p| phi_i(p) grad U_h(p)] / mL_i + <grad U> - N_d mbar    */
/*   b^mech_ia  = sum_{e mag} sum_p |J_p| [C_e : E0_h(p)]_ab d_b phi_i(p), E0_h = sum_a phi_a E0(m_a) */
/*   sigma^_i   = [sum_{e mag} sum_p |J_p| phi_i(p) C_e : (E_h(p) - E0_h(p))] / mLm_i        */
/* (for a one-point rule on a tetrahedron these are the formulas above them in this file) */
/* Geometry (|J|, phi, grad phi) is fp64 and rounded once to `real` (R20).                */
/* ------------------------------------------------------------------------------------ */
static void hex_coords(const oracle *o, long e, double X[24])
{
    const int *t = o->ghex + 8 * e;
    for (int a = 0; a < 8; a++) for (int d = 0; d < 3; d++) X[3 * a + d] = o->x[3 * (long)t[a] + d];
}

static int hex_rhs_ms(const oracle *o, const real *m, const double *mbar, real *b)
{
    for (long i = 0; i < o->N; i++) b[i] = 0;
    for (long e = 0; e < o->Ne; e++) {
        const int *t = o->hex + 8 * e;
        double X[24]; hex_coords(o, e, X);
        for (int p = 0; p < 8; p++) {
            double det, phi[8], g[8][3];
            hex_gauss_point(X, p, &det, phi, g);
            real mt[3] = {0, 0, 0};
            for (int a = 0; a < 8; a++) for (int d = 0; d < 3; d++) mt[d] += (real)phi[a] * m[3 * (long)t[a] + d];
            for (int d = 0; d < 3; d++) mt[d] -= (real)mbar[d];
            for (int a = 0; a < 8; a++)
                b[t[a]] += (real)det * ((real)g[a][0] * mt[0] + (real)g[a][1] * mt[1] + (real)g[a][2] * mt[2]);
        }
    }
    b[o->pin] = 0;
    return ORC_OK;
}

static int hex_demag_field(const oracle *o, const real *U, const double *mbar, unsigned terms, real *hd, double *gradU_mean)
{
    long N = o->N;
    for (long i = 0; i < 3 * N; i++) hd[i] = 0;
    double gm[3] = {0, 0, 0};
    if (terms & T_DEMAG) {
        double acc[3] = {0, 0, 0};
        for (long e = 0; e < o->Ne; e++) {
            const int *t = o->hex + 8 * e;
            double X[24]; hex_coords(o, e, X);
            for (int p = 0; p < 8; p++) {
                double det, phi[8], g[8][3];
                hex_gauss_point(X, p, &det, phi, g);
                real gU[3] = {0, 0, 0};
                for (int a = 0; a < 8; a++) for (int d = 0; d < 3; d++) gU[d] += U[t[a]] * (real)g[a][d];
                for (int d = 0; d < 3; d++) acc[d] += det * (double)gU[d];
                for (int a = 0; a < 8; a++) for (int d = 0; d < 3; d++) hd[3 * (long)t[a] + d] += (real)det * (real)phi[a] * gU[d];
            }
        }
        for (int d = 0; d < 3; d++) gm[d] = acc[d] / o->Vtot;
        for (long i = 0; i < N; i++) for (int d = 0; d < 3; d++) hd[3 * i + d] = -hd[3 * i + d] / o->mL[i] + (real)gm[d];
    }
    if (terms & T_FARFIELD)
        for (long i = 0; i < N; i++) for (int d = 0; d < 3; d++)
            hd[3 * i + d] -= (real)(o->Nd[3 * d] * mbar[0] + o->Nd[3 * d + 1] * mbar[1] + o->Nd[3 * d + 2] * mbar[2]);
    if (gradU_mean) for (int d = 0; d < 3; d++) gradU_mean[d] = gm[d];
    return ORC_OK;
}

/* E0_h(p) = sum_a phi_a(p) E0(w_a) and, if u != NULL, eps = E_h(p)(u) - E0_h(p); else eps = E0_h(p) */
static void hex_point_strain(const oracle *o, const int *t, const double phi[8], double g[8][3], const real *u, const real *w, real eps[6])
{
    real e0[6] = {0, 0, 0, 0, 0, 0};
    for (int a = 0; a < 8; a++) {
        real ek[6]; E0_voigt(o, w + 3 * (long)t[a], ek);
        for (int q = 0; q < 6; q++) e0[q] += (real)phi[a] * ek[q];
    }
    if (!u) { for (int q = 0; q < 6; q++) eps[q] = e0[q]; return; }
    real H[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}}; /* H[a][b] = d_b u_a */
    for (int k = 0; k < 8; k++) for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) H[a][b] += u[3 * (long)t[k] + a] * (real)g[k][b];
    eps[0] = H[0][0] - e0[0]; eps[1] = H[1][1] - e0[1]; eps[2] = H[2][2] - e0[2];
    eps[3] = H[1][2] + H[2][1] - e0[3]; eps[4] = H[0][2] + H[2][0] - e0[4]; eps[5] = H[0][1] + H[1][0] - e0[5];
}

static int hex_rhs_mech(const oracle *o, const real *m, real *b)
{
    for (long i = 0; i < 3 * o->N; i++) b[i] = 0;
    for (long e = 0; e < o->Ne; e++) {
        const int *t = o->hex + 8 * e;
        double X[24]; hex_coords(o, e, X);
        for (int p = 0; p < 8; p++) {
            double det, phi[8], g[8][3];
            hex_gauss_point(X, p, &det, phi, g);
            real e0[6], s[6] = {0, 0, 0, 0, 0, 0};
            if (o->mag[e]) {
                hex_point_strain(o, t, phi, g, NULL, m, e0);
                C_times(o, e, e0, s);
            }
            for (int q = 0; q < 6; q++) s[q] += (real)o->sext[q];   /* uniform external stress (R17), all cells */
            for (int a = 0; a < 8; a++) {
                real gx = (real)g[a][0], gy = (real)g[a][1], gz = (real)g[a][2], w = (real)det;
                b[3 * (long)t[a] + 0] += w * (s[0] * gx + s[5] * gy + s[4] * gz);
                b[3 * (long)t[a] + 1] += w * (s[5] * gx + s[1] * gy + s[3] * gz);
                b[3 * (long)t[a] + 2] += w * (s[4] * gx + s[3] * gy + s[2] * gz);
            }
        }
    }
    for (long i = 0; i < 3 * o->N; i++) if (o->clamp[i]) b[i] = 0;
    return ORC_OK;
}

static int hex_stress_recover(const oracle *o, const real *u, const real *w, real *sig)
{
    for (long i = 0; i < 6 * o->N; i++) sig[i] = 0;
    for (long e = 0; e < o->Ne; e++) {
        if (!o->mag[e]) continue;
        const int *t = o->hex + 8 * e;
        double X[24]; hex_coords(o, e, X);
        for (int p = 0; p < 8; p++) {
            double det, phi[8], g[8][3];
            hex_gauss_point(X, p, &det, phi, g);
            real eps[6], s[6];
            hex_point_strain(o, t, phi, g, u, w, eps);
            C_times(o, e, eps, s);
            for (int a = 0; a < 8; a++) for (int q = 0; q < 6; q++) sig[6 * (long)t[a] + q] += (real)det * (real)phi[a] * s[q];
        }
    }
    for (long i = 0; i < o->N; i++)
        for (int q = 0; q < 6; q++) sig[6 * i + q] = o->live[i] ? sig[6 * i + q] / o->mLm[i] : (real)0;
    return ORC_OK;
}

static double hex_elastic_energy(const oracle *o, const real *m, const real *u)
{
    double E = 0;
    for (long e = 0; e < o->Ne; e++) {
        const int *t = o->hex + 8 * e;
        double X[24]; hex_coords(o, e, X);
        for (int p = 0; p < 8; p++) {
            double det, phi[8], g[8][3];
            hex_gauss_point(X, p, &det, phi, g);
            real eps[6], s[6];
            if (o->mag[e]) hex_point_strain(o, t, phi, g, u, m, eps);
            else {
                real zero[24] = {0};
                (void)zero;
                real H[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
                for (int k = 0; k < 8; k++) for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) H[a][b] += u[3 * (long)t[k] + a] * (real)g[k][b];
                eps[0] = H[0][0]; eps[1] = H[1][1]; eps[2] = H[2][2];
                eps[3] = H[1][2] + H[2][1]; eps[4] = H[0][2] + H[2][0]; eps[5] = H[0][1] + H[1][0];
            }
            C_times(o, e, eps, s);
            double w = 0; for (int q = 0; q < 6; q++) w += (double)eps[q] * (double)s[q];
            E += 0.5 * det * w;
            real H[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};   /* - sigma_ext : E_h(p), total strain */
            for (int k = 0; k < 8; k++) for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) H[a][b] += u[3 * (long)t[k] + a] * (real)g[k][b];
            real et[6] = {H[0][0], H[1][1], H[2][2], H[1][2] + H[2][1], H[0][2] + H[2][0], H[0][1] + H[1][0]};
            for (int q = 0; q < 6; q++) E -= det * o->sext[q] * (double)et[q];
        }
    }
    return E;
}

/* S6 mechanical RHS (Eq. 10, 13, 14):
 * b_(i,a) = sum_{e contains i, magnetic} V_e [C*_e : mean_e E0(m)]_ab d_b phi_i
 *         + sum_{e contains i}           V_e sigma_ext,ab d_b phi_i          (the -sigma_ext : E term of Eq. 1; R17)
 * clamped DOFs zeroed. */
int orc_rhs_mech(const oracle *o, const void *m_, void *b_)
{
    if (o->nen == 8) return hex_rhs_mech(o, (const real *)m_, (real *)b_);
    const real *m = (const real *)m_; real *b = (real *)b_;
    if (!o->n_elastic) return ORC_E_BADARG;
    for (long i = 0; i < 3 * o->N; i++) b[i] = 0;
    for (long e = 0; e < o->Ne; e++) {
        const int *t = o->tet + 4 * e; const real *G = o->G + 12 * e;
        real e0[6], s[6] = {0, 0, 0, 0, 0, 0};
        if (o->mag[e]) {
            mean_E0(o, m, t, e0);
            C_times(o, e, e0, s);   /* Voigt stress xx,yy,zz,yz,xz,xy */
        }
        for (int q = 0; q < 6; q++) s[q] += (real)o->sext[q];
        for (int k = 0; k < 4; k++) {
            const real *g = G + 3 * k;
            b[3 * (long)t[k] + 0] += o->V[e] * (s[0] * g[0] + s[5] * g[1] + s[4] * g[2]);
            b[3 * (long)t[k] + 1] += o->V[e] * (s[5] * g[0] + s[1] * g[1] + s[3] * g[2]);
            b[3 * (long)t[k] + 2] += o->V[e] * (s[4] * g[0] + s[3] * g[1] + s[2] * g[2]);
        }
    }
    for (long i = 0; i < 3 * o->N; i++) if (o->clamp[i]) b[i] = 0;
    return ORC_OK;
}

/* element strain E_e = sym(sum_k u_k (x) grad phi_k), Voigt engineering vector */
static void elem_strain(const oracle *o, long e, const real *u, real eps[6])
{
    const int *t = o->tet + 4 * e; const real *G = o->G + 12 * e;
    real H[3][3];  /* H[a][b] = d_b u_a */
    for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) {
        real acc = 0;
        for (int k = 0; k < 4; k++) acc += u[3 * (long)t[k] + a] * G[3 * k + b];
        H[a][b] = acc;
    }
    eps[0] = H[0][0]; eps[1] = H[1][1]; eps[2] = H[2][2];
    eps[3] = H[1][2] + H[2][1]; eps[4] = H[0][2] + H[2][0]; eps[5] = H[0][1] + H[1][0];
}

/* S8 stress recovery (O-3 item 5): sigma_e = C*_e:(E_e(u) - mean_e E0(w)) on magnetic tets;
 * sigma_hat_i = sum_{e contains i, magnetic} V_e sigma_e/(4 mLm_i).  Output N x 6 Voigt. */
int orc_stress_recover(const oracle *o, const void *u_, const void *w_, void *sig_)
{
    if (o->nen == 8) return hex_stress_recover(o, (const real *)u_, (const real *)w_, (real *)sig_);
    const real *u = (const real *)u_, *w = (const real *)w_; real *sg = (real *)sig_;
    if (!o->n_elastic) return ORC_E_BADARG;
    for (long i = 0; i < 6 * o->N; i++) sg[i] = 0;
    for (long e = 0; e < o->Ne; e++) {
        if (!o->mag[e]) continue;
        const int *t = o->tet + 4 * e;
        real eps[6], e0[6], s[6];
        elem_strain(o, e, u, eps);
        mean_E0(o, w, t, e0);
        for (int q = 0; q < 6; q++) eps[q] -= e0[q];
        C_times(o, e, eps, s);
        for (int k = 0; k < 4; k++) for (int q = 0; q < 6; q++) sg[6 * (long)t[k] + q] += o->V[e] * s[q];
    }
    for (long i = 0; i < o->N; i++)
        for (int q = 0; q < 6; q++) sg[6 * i + q] = o->live[i] ? sg[6 * i + q] / ((real)4 * o->mLm[i]) : (real)0;
    return ORC_OK;
}

/* O-3 item 5: h(w)_i = h_an + h_ext + h_d,i + h_me on live nodes, 0 on dead nodes.
 * h_an,1 = -2K* w1 (w2^2 + w3^2) and cyclic (kappa_1 term of Eq. 1);
 * h_me,1 = 3 [lam100 w1 s11 + lam111 (w2 s12 + w3 s13)] and cyclic (R14). */
int orc_field(const oracle *o, const void *w_, const void *hd_, const void *sig_, const double *hext, unsigned terms, void *h_)
{
    const real *w = (const real *)w_, *hd = (const real *)hd_, *sg = (const real *)sig_; real *h = (real *)h_;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < o->N; i++) {
        real hi[3] = {0, 0, 0};
        if (o->live[i]) {
            /* Alg. D.1 Step 4: the m-dependent terms are evaluated in crystal axes (m_c = R^T m, sigma_c = R^T sigma R) and
             * rotated back, h = R h_c; the applied and demagnetising fields are already in the simulation frame */
            real mcv[3], scv[6], hc[3] = {0, 0, 0};
            const real *m = w + 3 * i;
            if (o->rot) { to_crystal(o, w + 3 * i, mcv); m = mcv; }
            if (terms & T_ANIS) {
                real k2 = (real)(2.0 * o->Kstar);
                hc[0] -= k2 * m[0] * (m[1] * m[1] + m[2] * m[2]);
                hc[1] -= k2 * m[1] * (m[2] * m[2] + m[0] * m[0]);
                hc[2] -= k2 * m[2] * (m[0] * m[0] + m[1] * m[1]);
            }
            if (terms & T_MAGEL) {
                const real *s = sg + 6 * i; /* xx,yy,zz,yz,xz,xy */
                if (o->rot) { rotate_sym(o, s, 1, scv); s = scv; }
                real l1 = (real)o->lam100, l2 = (real)o->lam111;
                hc[0] += (real)3 * (l1 * m[0] * s[0] + l2 * (m[1] * s[5] + m[2] * s[4]));
                hc[1] += (real)3 * (l1 * m[1] * s[1] + l2 * (m[0] * s[5] + m[2] * s[3]));
                hc[2] += (real)3 * (l1 * m[2] * s[2] + l2 * (m[0] * s[4] + m[1] * s[3]));
            }
            if (o->rot) to_sim(o, hc, hi); else for (int d = 0; d < 3; d++) hi[d] = hc[d];
            if (terms & T_ZEEMAN) for (int d = 0; d < 3; d++) hi[d] += (real)hext[d];
            if (terms & (T_DEMAG | T_FARFIELD)) for (int d = 0; d < 3; d++) hi[d] += hd[3 * i + d];
        }
        h[3 * i] = hi[0]; h[3 * i + 1] = hi[1]; h[3 * i + 2] = hi[2];
    }
    return ORC_OK;
}

/* discrete energy / (mu0 Ms^2 l_d^3)  (O-3 item 10); used by tests only */
double orc_energy(const oracle *o, const void *m_, const void *U_, const void *u_, const double *hext, unsigned terms)
{
    const real *m = (const real *)m_, *U = (const real *)U_, *u = (const real *)u_;
    long N = o->N;
    double E = 0;

    real *y = (real *)malloc((size_t)3 * N * sizeof(real));
    for (int c = 0; c < 3; c++) { /* exchange 1/2 A* m_a^T K_m m_a */
        spmv(o, MAT_K_M, m, y, 3, c);
        E += 0.5 * o->Astar * dot(N, m, y, 3, c);
    }
    for (long i = 0; i < N; i++) {
        double a = m[3 * i], b = m[3 * i + 1], c = m[3 * i + 2];
        real mcv[3] = {m[3 * i], m[3 * i + 1], m[3 * i + 2]};
        if (o->rot) to_crystal(o, m + 3 * i, mcv);
        double ac = mcv[0], bc = mcv[1], cc = mcv[2];
        if (terms & T_ANIS) E += o->Kstar * (double)o->mLm[i] * (ac * ac * bc * bc + bc * bc * cc * cc + cc * cc * ac * ac);
        if (terms & T_ZEEMAN) E -= (double)o->mLm[i] * (hext[0] * a + hext[1] * b + hext[2] * c);
    }
    double mbar[3]; orc_volume_average(o, m, 3, mbar);
    if (terms & T_DEMAG) { spmv(o, MAT_K_FREE, U, y, 1, 0); E += 0.5 * dot(N, U, y, 1, 0); }
    if (terms & T_FARFIELD)
        for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) E += 0.5 * o->Vtot * mbar[a] * o->Nd[3 * a + b] * mbar[b];
    if ((terms & T_MAGEL) && o->n_elastic && o->nen == 8) E += hex_elastic_energy(o, m, u);
    else if ((terms & T_MAGEL) && o->n_elastic)
        for (long e = 0; e < o->Ne; e++) {
            real eps[6], e0[6], s[6];
            elem_strain(o, e, u, eps);
            if (o->mag[e]) { mean_E0(o, m, o->tet + 4 * e, e0); for (int q = 0; q < 6; q++) eps[q] -= e0[q]; }
            C_times(o, e, eps, s);
            double w = 0; for (int q = 0; q < 6; q++) w += (double)eps[q] * (double)s[q];
            E += 0.5 * (double)o->V[e] * w;
            real et[6]; elem_strain(o, e, u, et);           /* - sigma_ext : E (Eq. 1), total strain */
            for (int q = 0; q < 6; q++) E -= (double)o->V[e] * o->sext[q] * (double)et[q];
        }
    free(y);
    return E;
}

/* ------------------------------------------------------------------------------------ */
/* O-3: one GSPM step (Alg. B.1)                                              */
/* ------------------------------------------------------------------------------------ */

/* Helmholtz solve (M_m + eps K_m) g_a = M_m f_a, x0 = f_a (R15), for component a */
static int helmholtz(const oracle *o, int id, const real *f, real *g, int a, const orc_step_params *p, int *it, double *res, real *b)
{
    spmv(o, MAT_MASS, f, b, 3, a);                                  /* b = M_m f (Eq. 14) */
    for (long i = 0; i < o->N; i++) g[3 * i + a] = f[3 * i + a];
    return cg_pc(o, id, b, g, 3, a, p->cg_tol, p->cg_maxiter, p->cg_fixed_iters, p->cg_precond, it, res);
}

int orc_gspm_step(const oracle *o, const orc_step_params *p, void *m_, void *U_, void *u_, orc_step_info *info)
{
    real *m = (real *)m_, *U = (real *)U_, *u = (real *)u_;
    long N = o->N; unsigned terms = p->terms;
    int worst = ORC_OK, rc;
    if (p->dt != o->dt || p->cg_precond < 0 || p->cg_precond > 1) return ORC_E_BADARG; /* K^GS was assembled for the dt given at create */
    real *b = (real *)calloc((size_t)3 * N, sizeof(real)), *hd = (real *)calloc((size_t)3 * N, sizeof(real)),
         *sg = (real *)calloc((size_t)6 * N, sizeof(real)), *hn = (real *)calloc((size_t)3 * N, sizeof(real)),
         *f = (real *)calloc((size_t)3 * N, sizeof(real)), *gn = (real *)calloc((size_t)3 * N, sizeof(real)),
         *gs = (real *)calloc((size_t)3 * N, sizeof(real)), *ms = (real *)calloc((size_t)3 * N, sizeof(real)),
         *mss = (real *)calloc((size_t)3 * N, sizeof(real));
    double hext[3] = {p->Hext[0] / o->Ms, p->Hext[1] / o->Ms, p->Hext[2] / o->Ms};
    real dtau = (real)o->dtau, adtau = (real)(o->alpha * o->dtau);
    memset(info, 0, sizeof(*info)); info->energy = NAN;

    /* 1. mbar over all of Omega_c (Eq. 17) */
    double mbar[3]; orc_volume_average(o, m, 3, mbar);
    for (int d = 0; d < 3; d++) info->mbar[d] = mbar[d];
    /* 2. magnetostatic solve, warm start (Eq. 5, 9) */
    if (terms & T_DEMAG) {
        orc_rhs_ms(o, m, mbar, b);
        rc = cg_pc(o, MAT_K_MS, b, U, 1, 0, p->cg_tol, p->cg_maxiter, p->cg_fixed_iters, p->cg_precond, &info->it_ms, &info->res_ms);
        if (rc < worst) worst = rc;
    }
    /* 3. demagnetising field (Eq. 4) */
    orc_demag_field(o, U, mbar, terms, hd, NULL);
    /* 4. mechanical equilibrium (Eq. 6, 10), warm start */
    if (terms & T_MAGEL) {
        orc_rhs_mech(o, m, b);
        rc = cg_pc(o, MAT_K_MECH, b, u, 1, 0, p->cg_tol, p->cg_maxiter, p->cg_fixed_iters, p->cg_precond, &info->it_mech, &info->res_mech);
        if (rc < worst) worst = rc;
        orc_stress_recover(o, u, m, sg);
    }
    /* 5. h[m^n] */
    orc_field(o, m, hd, sg, hext, terms, hn);
    /* 6. Step 1: g^n */
    for (long i = 0; i < 3 * N; i++) f[i] = m[i] + dtau * hn[i];
    for (int a = 0; a < 3; a++) {
        if (p->gspm_variant == 1 && a == 0) continue;  /* g_1^n unused in the Gauss-Seidel variant (R1) */
        rc = helmholtz(o, MAT_K_GS1, f, gn, a, p, &info->it_gs[a], &info->res_gs[a], b);
        if (rc < worst) worst = rc;
    }
    /* 7. Step 2 interleaved with the g* solves (g* uses m* and h[m^n]) */
    for (long i = 0; i < N; i++) ms[3 * i] = m[3 * i] + (gn[3 * i + 1] * m[3 * i + 2] - gn[3 * i + 2] * m[3 * i + 1]);
    if (p->gspm_variant == 0) {
        for (long i = 0; i < N; i++) ms[3 * i + 1] = m[3 * i + 1] + (gn[3 * i + 2] * m[3 * i] - gn[3 * i] * m[3 * i + 2]);
        for (long i = 0; i < N; i++) for (int a = 0; a < 2; a++) f[3 * i + a] = ms[3 * i + a] + dtau * hn[3 * i + a];
        for (int a = 0; a < 2; a++) {
            rc = helmholtz(o, MAT_K_GS1, f, gs, a, p, &info->it_gs[3 + a], &info->res_gs[3 + a], b);
            if (rc < worst) worst = rc;
        }
    } else {
        for (long i = 0; i < N; i++) f[3 * i] = ms[3 * i] + dtau * hn[3 * i];
        rc = helmholtz(o, MAT_K_GS1, f, gs, 0, p, &info->it_gs[3], &info->res_gs[3], b); if (rc < worst) worst = rc;
        for (long i = 0; i < N; i++) ms[3 * i + 1] = m[3 * i + 1] + (gn[3 * i + 2] * ms[3 * i] - gs[3 * i] * m[3 * i + 2]);
        for (long i = 0; i < N; i++) f[3 * i + 1] = ms[3 * i + 1] + dtau * hn[3 * i + 1];
        rc = helmholtz(o, MAT_K_GS1, f, gs, 1, p, &info->it_gs[4], &info->res_gs[4], b); if (rc < worst) worst = rc;
    }
    for (long i = 0; i < N; i++) ms[3 * i + 2] = m[3 * i + 2] + (gs[3 * i] * ms[3 * i + 1] - gs[3 * i + 1] * ms[3 * i]);
    /* 8. Step 3: h* = h[m*] with U, u frozen (R3) */
    if (terms & T_MAGEL) orc_stress_recover(o, u, ms, sg);
    orc_field(o, ms, hd, sg, hext, terms, hn);
    for (long i = 0; i < 3 * N; i++) f[i] = ms[i] + adtau * hn[i];
    for (int a = 0; a < 3; a++) {
        rc = helmholtz(o, MAT_K_GS2, f, mss, a, p, &info->it_gs[5 + a], &info->res_gs[5 + a], b);
        if (rc < worst) worst = rc;
    }
    /* 9. Step 4 projection on live nodes; 10. mean |dm| over live nodes */
    double sdm = 0; long nlive = 0;
    for (long i = 0; i < N; i++) {
        if (!o->live[i]) { m[3 * i] = m[3 * i + 1] = m[3 * i + 2] = 0; continue; }
        real *v = mss + 3 * i;
        real nrm = (real)sqrt((double)(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));
        real nw[3] = {m[3 * i], m[3 * i + 1], m[3 * i + 2]};
        if (nrm > 0) for (int d = 0; d < 3; d++) nw[d] = v[d] / nrm;
        double d0 = (double)nw[0] - (double)m[3 * i], d1 = (double)nw[1] - (double)m[3 * i + 1], d2 = (double)nw[2] - (double)m[3 * i + 2];
        sdm += sqrt(d0 * d0 + d1 * d1 + d2 * d2); nlive++;
        m[3 * i] = nw[0]; m[3 * i + 1] = nw[1]; m[3 * i + 2] = nw[2];
    }
    info->mean_dm = nlive ? sdm / (double)nlive : 0.0;
    free(b); free(hd); free(sg); free(hn); free(f); free(gn); free(gs); free(ms); free(mss);
    return worst;
}

/* Helmholtz right-hand side b = M_m f for all three components (Eq. 14) */
/* ------------------------------------------------------------------------------------ */
/* Hysteresis driver (R24)               */
/* ------------------------------------------------------------------------------------ */
/* "The external field H_ext is decreased in increments up to a critical coercive field H_c, at which the magnetization
 * field in the domain reverses"; at each field "the LLG equation is solved iteratively by GSPM until
 * <||m^n - m^{n-1}||_2>_DOF < 5e-10"; "the external field is reduced in intervals of dH = -20 A/m";
 * the average magnetisation and H_ext are written at convergence (Fig. 1).
 * Field k is H0 + k dH.  At each field: GSPM steps until mean_dm < conv_tol (or max_steps at that field); then the
 * volume average of the converged m (Eq. 17) is logged with H and the step count.  The run ends when that average has
 * a negative component along e0 = H0/|H0| (reversal), or after max_fields fields. */
typedef struct {
    double H0[3], dH[3];   /* A/m */
    double conv_tol;       /* on <||dm||_2> */
    int max_fields, max_steps;
} orc_hyst_params;

typedef struct {
    int n_fields, reversed;
    long total_steps;
} orc_hyst_result;

int orc_hysteresis_run(const oracle *o, const orc_step_params *base, const orc_hyst_params *hp, void *m, void *U, void *u,
                       double *H_log, double *mbar_log, int *steps_log, orc_hyst_result *res)
{
    if (!o || !base || !hp || !m || !H_log || !mbar_log || !steps_log || !res || hp->max_fields < 1 || hp->max_steps < 1)
        return ORC_E_BADARG;
    double n0 = sqrt(hp->H0[0] * hp->H0[0] + hp->H0[1] * hp->H0[1] + hp->H0[2] * hp->H0[2]);
    if (!(n0 > 0)) return ORC_E_BADARG;
    double e0[3] = {hp->H0[0] / n0, hp->H0[1] / n0, hp->H0[2] / n0};
    res->n_fields = 0; res->reversed = 0; res->total_steps = 0;
    int worst = ORC_OK;
    for (int k = 0; k < hp->max_fields; k++) {
        orc_step_params p = *base;
        for (int d = 0; d < 3; d++) p.Hext[d] = hp->H0[d] + (double)k * hp->dH[d];
        int steps = 0;
        for (;;) {
            orc_step_info info;
            int rc = orc_gspm_step(o, &p, m, U, u, &info);
            if (rc == ORC_E_BADARG || rc == ORC_E_ALLOC) return rc;
            if (rc < worst) worst = rc;
            steps++; res->total_steps++;
            if (info.mean_dm < hp->conv_tol || steps >= hp->max_steps) break;
        }
        double mbar[3];
        orc_volume_average(o, m, 3, mbar);
        for (int d = 0; d < 3; d++) { H_log[3 * k + d] = p.Hext[d]; mbar_log[3 * k + d] = mbar[d]; }
        steps_log[k] = steps;
        res->n_fields = k + 1;
        if (mbar[0] * e0[0] + mbar[1] * e0[1] + mbar[2] * e0[2] < 0) { res->reversed = 1; break; }
    }
    return worst;
}

int orc_rhs_gs(const oracle *o, const void *f_, void *b_)
{
    for (int a = 0; a < 3; a++) spmv(o, MAT_MASS, (const real *)f_, (real *)b_, 3, a);
    return ORC_OK;
}

int orc_sizeof_real(void) { return (int)sizeof(real); }
