// Internal declarations of the CuPyMag-B200 library (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/cupymag_b200.h"

typedef unsigned char uchar;

void cm_set_error(const char *fmt, ...);

#define CM_CUDA(call)                                                                          \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            cm_set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            return CM_E_CUDA;                                                                  \
        }                                                                                      \
    } while (0)

#define CM_TRY(call)             \
    do {                         \
        int rc_ = (call);        \
        if (rc_ < 0) return rc_; \
    } while (0)

// Persistent-kernel launch shape: NT threads per CTA everywhere in the SpMV / CG path.
// NT is a multiple of 3 so that thread t always serves the same vector component in the streaming phases.
constexpr int CM_NT = 384;
// Sliced storage (SELL-C): rows are grouped into slices of C consecutive rows, every row of a slice is padded to the
// slice's longest row and the slice is stored column-major, so element (row i, j-th nonzero) sits at
// sp[i / C] + j * C + i % C.  One warp works on one slice with all 32 lanes: lane -> (row i % C, column phase
// lane / C).  Scalar matrices use C = 16, the 3x3-block matrix C = 8.
constexpr int CM_C_SCALAR = 16;
constexpr int CM_C_BLOCK = 8;

enum SpmvMode { MODE_CSR1 = 0, MODE_CSR3 = 1, MODE_BSR3 = 2 };

// One sliced pattern (shared by every matrix with that slice height).
struct Sell {
    int C = 0;
    int nslices = 0;
    long E = 0;                 // stored elements including padding = sp[nslices]
    std::vector<int> sp, col;   // host copies: nslices + 1 offsets, E column indices (padding: the row itself)
    int *d_sp = nullptr, *d_col = nullptr;
};

// Element chunks for the assembly passes (S3, S5, S6, S8): consecutive elements are cut into chunks of at most
// CM_EC_MAX elements that reference at most CM_NL_MAX distinct nodes; every chunk starts at a multiple of 8 elements
// (16-byte aligned rows for the bulk copies), so only the last chunk has a ragged size.  A chunk numbers its nodes locally (sorted by
// global id); "slot" nptr[c] + l is local node l of chunk c, and every slot owns one partial sum per pass.
//   eptr[c]            first element of chunk c
//   nptr[c]            first slot of chunk c;  nodes[slot] = global node id
//   lid[4 e + k]       local id of node k of element e within its chunk
//   lptr[slot + c]     start of the slot's run in the chunk's incidence list (runs of chunk c end at lptr[nptr[c+1] + c])
//   lent[4 eptr[c] + q] incidence q of chunk c: 4 * (e - eptr[c]) + k, ascending inside every run
//   ns_ptr / ns_slot   node -> its slots, ascending (so ascending chunk = ascending element order)
constexpr int CM_EC_MAX = 768;
constexpr int CM_NL_MAX = 384; // a full chunk of 768 Kuhn tets touches ~260 nodes
constexpr int CM_HC_MAX = 128; // hexahedral cells per chunk (8 threads per cell, one per Gauss point)
struct Chunks {
    int nchunks = 0;
    long nslots = 0;
    std::vector<int> eptr, nptr, nodes, ns_ptr, ns_slot;
    std::vector<unsigned short> lid, lptr, lent;
    int *d_eptr = nullptr, *d_nptr = nullptr, *d_nodes = nullptr, *d_ns_ptr = nullptr, *d_ns_slot = nullptr;
    unsigned short *d_lid = nullptr, *d_lptr = nullptr, *d_lent = nullptr;
};

struct cm_mesh {
    long N = 0, Ne = 0, nnz = 0;
    int nen = 4;               // nodes per element: 4 = linear tetrahedra, 8 = linear hexahedra (matrices and averages only, R26)
    double vtot_m3 = 0, vmag_m3 = 0; // hexahedra: volumes summed on the host (metres^3)
    bool identity = true;
    // host copies, library order
    std::vector<int> order, iperm, tets, tet_order, rowptr, col, n2e_ptr, n2e, eid;
    std::vector<uchar> mag;
    std::vector<double> xyz;   // N x 3 metres, library order (wrapped mesh: coordinates of the DOF's representative node)
    // geometric connectivity: corner k of tet e has coordinates gxyz[gtets[4 e + k]].  Plain mesh: the same arrays as
    // tets / xyz.  Wrapped (periodic): gtets holds the caller's node ids (library tet order), gxyz its xyz.
    bool wrapped = false;
    long Ng = 0;
    std::vector<int> gtets;
    std::vector<double> gxyz;
    int *d_gtets = nullptr;    // == d_tets when !wrapped
    double *d_gxyz = nullptr;  // == d_xyz when !wrapped
    std::vector<double> wvol;  // N: lumped volume fraction mL_i / V (sums to 1)
    // device
    int *d_order = nullptr, *d_tets = nullptr, *d_rowptr = nullptr, *d_col = nullptr, *d_n2e_ptr = nullptr, *d_n2e = nullptr,
        *d_eid = nullptr;
    uchar *d_mag = nullptr;
    double *d_xyz = nullptr, *d_wvol = nullptr;
    Sell sell[2];              // [0]: C = CM_C_SCALAR, [1]: C = CM_C_BLOCK
    Chunks ck;
    std::vector<unsigned short> emat; // per element: elastic id << 1 | magnetic flag
    unsigned short *d_emat = nullptr;
    // scratch for cm_volume_average; calls on one mesh are serialised by avg_lock (they synchronise their stream before returning)
    std::mutex avg_lock;
    double *d_red = nullptr;   // partials
    void *d_tmp = nullptr;     // library-order copy of the averaged field (grown on demand by cm_volume_average)
    long tmp_bytes = 0;
    double *h_red = nullptr;   // pinned, 16 doubles
};

// App. D rotation as a kernel argument (by value); on == 0: identity, nothing is rotated
template <typename T>
struct Rot {
    T r[9];
    int on;
};
struct SystemBase;
template <typename T>
inline Rot<T> make_rot(const SystemBase *S);

constexpr int CM_HIST_CAP = 3 << 16;
struct CgResult {
    int iters[3];
    double relres[3];
    int status;
    int pad;
};

struct Profiler {
    bool on = false;
    struct Rec { cudaEvent_t a, b; int cls; };
    std::vector<Rec> pending;
    std::vector<cudaEvent_t> pool;
    double ms[CM_PROF_NCLASS] = {0};
    long launches[CM_PROF_NCLASS] = {0};
    long cg_iters[CM_PROF_NCLASS] = {0};
    long cg_passes[CM_PROF_NCLASS] = {0};
    cudaEvent_t get();
    void begin(int cls, cudaStream_t s, int nlaunch = 1); // counts launches always, times them when `on`
    void end(cudaStream_t s);
    int flush();
    ~Profiler();
};

struct SystemBase {
    cm_mesh *mesh = nullptr;
    cm_dtype dtype = CM_F64;
    long N = 0, Ne = 0, nnz = 0;
    double dt = 0, Astar = 0, Kstar = 0, dtau = 0, eps1 = 0, eps2 = 0, alpha = 0, lam100 = 0, lam111 = 0, Ms = 0;
    double Nd[9] = {0};
    double R[9] = {1, 0, 0, 0, 1, 0, 0, 0, 1}; // App. D: crystal -> simulation frame
    bool rot = false;
    double sext[6] = {0}; // sigma_ext / (mu0 Ms^2), tensor components xx,yy,zz,yz,xz,xy (Eq. 1; R17)
    bool has_sext = false;
    int n_elastic = 0;
    double Vtot = 0, Vmag = 0;
    double ld = 1;  // length scale l_d, metres
    long nlive = 0;
    int pin = 0; // library index
    int num_sms = 0;
    Profiler prof;
    bool no_fuse = false;  // CM_OPT_NO_FUSED_S5S8: the step runs S5 and S8 as separate element passes (A/B measurement)
    int sig_hs = 6, sig_ho = 0; // where the stress partials of the last stress pass sit in hpart: words per slot, first word
    int geometry_mode = 0; // CM_OPT_STORED_GEOMETRY: 0 per-pass choice, 1 every pass streams the stored geometry, 2 every pass recomputes it
    double *d_hist = nullptr;  // residual history of the last solve (cm_cg_history), CM_HIST_CAP doubles
    bool hist_on = false;
    long hist_len = 0;
    int hist_nr = 1;
    virtual ~SystemBase() {}
};

template <typename T>
inline Rot<T> make_rot(const SystemBase *S)
{
    Rot<T> q;
    for (int k = 0; k < 9; k++) q.r[k] = (T)S->R[k];
    q.on = S->rot ? 1 : 0;
    return q;
}

template <typename T>
struct System : SystemBase {
    // geometry
    // element geometry, chunk-blocked: chunk c owns 10 planes of ne8 = round_up(ne_c, 8) values at EG + 10 eptr[c]:
    // plane 0 = V_e, plane 3 (k - 1) + d + 1 = d-th component of grad phi_k, k = 1..3 (grad phi_0 = -sum, O-1)
    T *EG = nullptr;
    // nondimensional fp64 coordinates for the passes that recompute the geometry with the set-up's own arithmetic
    // (tet_geometry_x / hex_point).  Plain tetrahedral meshes: of every chunk slot, [slot][4] (x/l_d, y/l_d, z/l_d, 0),
    // contiguous per chunk, staged by one coalesced read.  Hexahedral meshes (plain and wrapped): the cell's own eight
    // corners, [cell][8][3], staged by one bulk copy.  Wrapped tetrahedral meshes: none (they stream the stored geometry EG).
    double *CX = nullptr;
    T *mL = nullptr, *mLm = nullptr;
    T *Cstar = nullptr; // n_elastic x 36
    T *Ccub = nullptr;  // n_elastic x 12 (C11 C12 C13 C21 .. C33, C44 C55 C66) when every C* is zero outside that pattern
    bool cubic_pattern = false;
    uchar *live = nullptr, *clamp = nullptr;
    // matrices
    T *Kms = nullptr, *Kgs1 = nullptr, *Kgs2 = nullptr, *Mm = nullptr;
    T *Kmech = nullptr; // sliced, 9 planes per slice: [slice][3 r + c][L_slice]
    // diagonals of the constrained matrices (Jacobi preconditioner): N entries each, Dmech 3N
    T *Dms = nullptr, *Dgs1 = nullptr, *Dgs2 = nullptr, *Dmech = nullptr;
    // CG work
    T *r = nullptr, *p = nullptr, *p2 = nullptr, *Ap = nullptr, *bvec = nullptr;
    double *partial = nullptr;
    int grid_cap = 0;
    CgResult *d_res = nullptr, *h_res = nullptr; // 8 slots
    // step state (library order)
    T *m = nullptr, *U = nullptr, *u = nullptr, *hd = nullptr, *hn = nullptr, *f = nullptr, *gn = nullptr, *gs = nullptr,
      *ms = nullptr, *mss = nullptr, *xin = nullptr, *xout = nullptr;
    T *sig = nullptr;                                        // N x 6 parity output of CM_OUT_SIGMA
    T *stg_m = nullptr, *stg_U = nullptr, *stg_u = nullptr;  // device staging of the host-buffer step
    T *hpart = nullptr;    // per-slot partial sums of the element passes, 6 per slot
    double *red = nullptr; // reduction partials
    double *dscal = nullptr, *h_scal = nullptr; // device / pinned scalars: mbar[3], gradU mean[3], dm sum, ...
    // hysteresis driver (cm_hysteresis_run): device-resident controller state and logs, grown on demand
    void *mf_state = nullptr, *h_mf = nullptr; // matrix-free CG: two device states, pinned host copy
    void *hyst_ctl = nullptr;
    double *hyst_log = nullptr; // [cap][3] H, [cap][3] mbar
    int *hyst_steps = nullptr;  // [cap]
    int hyst_cap = 0;
    ~System();
};

// O-1: volume and shape-function gradients of a tetrahedron from its four (nondimensional) corner coordinates, fp64.
// One reciprocal instead of nine divisions; every user (matrix assembly, stored geometry, element passes) calls this
// one function, so the recomputed and the stored geometry are the same bits.
struct TetGeom {
    double V;
    double g[4][3];
};
__device__ __forceinline__ void tet_geometry_x(const double x[4][3], TetGeom &G)
{
    double a[3], b[3], c[3];
#pragma unroll
    for (int d = 0; d < 3; d++) { a[d] = x[1][d] - x[0][d]; b[d] = x[2][d] - x[0][d]; c[d] = x[3][d] - x[0][d]; }
    const double bc[3] = {b[1] * c[2] - b[2] * c[1], b[2] * c[0] - b[0] * c[2], b[0] * c[1] - b[1] * c[0]};
    const double ca[3] = {c[1] * a[2] - c[2] * a[1], c[2] * a[0] - c[0] * a[2], c[0] * a[1] - c[1] * a[0]};
    const double ab[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
    const double det = a[0] * bc[0] + a[1] * bc[1] + a[2] * bc[2];
    const double idet = 1.0 / det;
    G.V = fabs(det) / 6.0;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        G.g[1][d] = bc[d] * idet; G.g[2][d] = ca[d] * idet; G.g[3][d] = ab[d] * idet;
        G.g[0][d] = -(G.g[1][d] + G.g[2][d] + G.g[3][d]);
    }
}

// Linear hexahedron (R26): |J|, phi_a and grad phi_a (fp64) at Gauss point p of the 2 x 2 x 2 rule; local node
// a = i + 2 j + 4 k <-> reference corner (2i-1, 2j-1, 2k-1)
__device__ __forceinline__ double hex_point(const double X[8][3], int p, double phi[8], double g[8][3])
{
    const double q = 0.57735026918962576451;
    const double xi[3] = {(p & 1) ? q : -q, (p & 2) ? q : -q, (p & 4) ? q : -q};
    double dN[8][3], J[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
    for (int a = 0; a < 8; a++) {
        const double s[3] = {(a & 1) ? 1.0 : -1.0, (a & 2) ? 1.0 : -1.0, (a & 4) ? 1.0 : -1.0};
        const double f[3] = {1 + s[0] * xi[0], 1 + s[1] * xi[1], 1 + s[2] * xi[2]};
        phi[a] = f[0] * f[1] * f[2] / 8;
        dN[a][0] = s[0] * f[1] * f[2] / 8; dN[a][1] = f[0] * s[1] * f[2] / 8; dN[a][2] = f[0] * f[1] * s[2] / 8;
#pragma unroll
        for (int r = 0; r < 3; r++)
#pragma unroll
            for (int c = 0; c < 3; c++) J[r][c] += X[a][r] * dN[a][c];
    }
    double cof[3][3];
    cof[0][0] = J[1][1] * J[2][2] - J[1][2] * J[2][1]; cof[0][1] = J[1][2] * J[2][0] - J[1][0] * J[2][2]; cof[0][2] = J[1][0] * J[2][1] - J[1][1] * J[2][0];
    cof[1][0] = J[0][2] * J[2][1] - J[0][1] * J[2][2]; cof[1][1] = J[0][0] * J[2][2] - J[0][2] * J[2][0]; cof[1][2] = J[0][1] * J[2][0] - J[0][0] * J[2][1];
    cof[2][0] = J[0][1] * J[1][2] - J[0][2] * J[1][1]; cof[2][1] = J[0][2] * J[1][0] - J[0][0] * J[1][2]; cof[2][2] = J[0][0] * J[1][1] - J[0][1] * J[1][0];
    const double det = J[0][0] * cof[0][0] + J[0][1] * cof[0][1] + J[0][2] * cof[0][2];
    const double idet = 1.0 / det; // one division per Gauss point instead of 24 (fp64 divisions dominate these passes)
#pragma unroll
    for (int a = 0; a < 8; a++)
#pragma unroll
        for (int r = 0; r < 3; r++) g[a][r] = (cof[r][0] * dN[a][0] + cof[r][1] * dN[a][1] + cof[r][2] * dN[a][2]) * idet;
    return det;
}

// ---- cm_mesh.cu ----
int mesh_build_host(cm_mesh *M, const double *xyz, long Ng, const int *gtets, long Ne, const uchar *mag, const int *eid,
                    const int *dof, long N, cm_reorder reorder);
int mesh_build_host_hex(cm_mesh *M, const double *xyz, long Ng, const int *ghexes, long Ne, const uchar *mag, const int *eid,
                        const int *dof, long N, cm_reorder reorder);
int build_sell(long N, const std::vector<int> &rowptr, const std::vector<int> &col, int C, Sell *out);
int build_chunks(long N, long Ne, const int *conn, int nen, int ecmax, Chunks *out);

// ---- kernels (templated launchers; defined in the .cu files, instantiated for float and double) ----
template <typename T> int sys_assemble(System<T> *S, const cm_material *mat, const uchar *clamp_user, long pin_user, cudaStream_t st);
template <typename T> int sys_spmv(System<T> *S, cm_matrix_id id, int mode, const T *x, T *y, cudaStream_t st);
template <typename T> int sys_cg(System<T> *S, cm_matrix_id id, int mode, const T *b, T *x, double tol, int maxiter, int fixed,
                                 unsigned mask, int slot, int prof_cls, int precond, cudaStream_t st);
template <typename T> int sys_helmholtz(System<T> *S, cm_matrix_id id, const T *f4, T *x, double tol, int maxiter, int fixed, unsigned mask,
                                        int slot, int precond, cudaStream_t st);
template <typename T> int sys_get_values(const System<T> *S, cm_matrix_id id, void *host_out, long capacity);
template <typename T> int sys_permute_in(System<T> *S, const T *user, T *lib, int ncomp, cudaStream_t st); // ncomp = -3: [node][3] -> padded [node][4]
template <typename T> int sys_permute_out(System<T> *S, const T *lib, T *user, int ncomp, cudaStream_t st);
template <typename T> int sys_mbar(System<T> *S, const T *m_lib, cudaStream_t st);                         // -> dscal[0..2]
template <typename T> int sys_rhs_ms(System<T> *S, const T *m_lib, T *b, cudaStream_t st);                 // uses dscal[0..2]
template <typename T> int sys_demag_field(System<T> *S, const T *U_lib, unsigned terms, T *hd, cudaStream_t st);
template <typename T> int sys_rhs_mech(System<T> *S, const T *m_lib, T *b, cudaStream_t st);
template <typename T> int sys_stress(System<T> *S, const T *u_lib, const T *w_lib, cudaStream_t st);       // -> hpart (V sigma per slot)
template <typename T> int sys_field(System<T> *S, const T *w_lib, const T *hd, const double hext[3], unsigned terms, T *h,
                                    T *sig_out, cudaStream_t st, const double *hext_dev = nullptr);                                          // gathers hpart when MAGEL
template <typename T> int sys_step(System<T> *S, const cm_step_params *p, T *m_user, T *U_user, T *u_user, cm_step_info *info,
                                   cudaStream_t st);
template <typename T> int sys_hysteresis(System<T> *S, const cm_step_params *base, const cm_hyst_params *hp, T *m_user, T *U_user,
                                         T *u_user, double *H_log, double *mbar_log, int *steps_log, cm_hyst_result *res, cudaStream_t st);
template <typename T> int sys_spmv_matfree(System<T> *S, const T *x_lib, T *y_lib, cudaStream_t st);
template <typename T> int sys_cg_matfree(System<T> *S, const T *b_lib, T *x_lib, double tol, int maxiter, int fixed, int precond, int slot,
                                         cudaStream_t st);
template <typename T> int sys_axpby3(System<T> *S, const T *base, const T *h, T c, T *f, cudaStream_t st);
