// S4 / S7 / S10: sparse matrix-vector products and the fused, persistent, unpreconditioned
// conjugate-gradient solver (O-4).
//
// Layout.  All scalar matrices share rowptr / colidx; values are plain CSR arrays.  The 3x3-block
// elasticity matrix is stored "tile-SoA": blocks are grouped by 32 and inside a group the 9 block
// entries are 9 contiguous planes of 32 values, [nnz/32][9][32], so that a warp reading 32 consecutive
// blocks issues 9 fully coalesced 256-byte (fp64) loads and the whole matrix is one sequential stream.
//
// Work decomposition.  Rows are cut once, on the host, into "tiles" of consecutive rows holding at most
// TILE nonzeros (blocks).  A CTA owns a contiguous range of tiles for the whole solve.  Per tile:
//   phase 1  one thread per nonzero: stream value(s) + column index, gather x[col] (1 or 3 components,
//            L1/L2 hits thanks to the locality ordering), write the product(s) to shared memory;
//   phase 2  one thread per (row, component): sum the row's segment of products in column order
//            (deterministic, same order as the definition), write y, accumulate the dot p.Ap.
// The CG kernel is ONE cooperative launch per solve: SpMV, both dot products, the three vector updates
// and the convergence test run on the device with grid-wide barriers in between; every CTA reduces the
// per-CTA partial sums in the same fixed order, so all CTAs take the same decision and the result is
// bit-reproducible run to run.  No float atomics anywhere.
#include <cooperative_groups.h>

#include <algorithm>

#include "cm_internal.h"

namespace cg = cooperative_groups;

template <typename T>
struct MatView {
    const int *rowptr;
    const int *col;
    const T *val;
    const int *tile_row;
    int ntiles;
    int tile;
    long N;
};

template <int MODE> struct ModeTraits;
template <> struct ModeTraits<MODE_CSR1> { static constexpr int NC = 1, NR = 1, TILE = CM_TILE_S1; };
template <> struct ModeTraits<MODE_CSR3> { static constexpr int NC = 3, NR = 3, TILE = CM_TILE_3; };
template <> struct ModeTraits<MODE_BSR3> { static constexpr int NC = 3, NR = 1, TILE = CM_TILE_3; };

// Contiguous tile range of CTA `b` out of `nb`.
__device__ __forceinline__ void cta_tiles(int ntiles, int b, int nb, int &t0, int &t1)
{
    int q = ntiles / nb, r = ntiles % nb;
    t0 = b * q + min(b, r);
    t1 = t0 + q + (b < r ? 1 : 0);
}

// Deterministic block-wide sum of NV doubles per thread; result broadcast to all threads.
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double *sh /* >= NV * 32 doubles */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; k++) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
    }
    __syncthreads(); // protect sh from a previous use
    if (lane == 0)
#pragma unroll
        for (int k = 0; k < NV; k++) sh[k * 32 + warp] = v[k];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NV; k++) {
        double s = 0;
        for (int w = 0; w < nwarp; w++) s += sh[k * 32 + w]; // fixed order, identical in every thread
        v[k] = s;
    }
}

// y = A x on the tiles [t0, t1); optionally accumulates dot[c] += y.x over the rows written (own rows).
// `prod` is shared memory of NC * TILE elements of T.
template <typename T, int MODE, bool DOT>
__device__ __forceinline__ void spmv_tiles(const MatView<T> &A, const T *x, T *y, int t0, int t1, T *prod, double *dot)
{
    constexpr int NC = ModeTraits<MODE>::NC, TILE = ModeTraits<MODE>::TILE;
    const int tid = threadIdx.x, nt = blockDim.x;
    for (int t = t0; t < t1; t++) {
        const int r0 = A.tile_row[t], r1 = A.tile_row[t + 1];
        const int q0 = A.rowptr[r0], q1 = A.rowptr[r1];
        if (q1 - q0 <= TILE) {
            // ---- phase 1
            for (int q = q0 + tid; q < q1; q += nt) {
                const int c = __ldg(A.col + q);
                if (MODE == MODE_CSR1) {
                    prod[q - q0] = __ldg(A.val + q) * x[c];
                } else if (MODE == MODE_CSR3) {
                    const T a = __ldg(A.val + q);
                    const T *xc = x + 3 * (long)c;
                    prod[q - q0] = a * xc[0];
                    prod[TILE + q - q0] = a * xc[1];
                    prod[2 * TILE + q - q0] = a * xc[2];
                } else {
                    const T *v = A.val + (long)(q >> 5) * 288 + (q & 31);
                    const T *xc = x + 3 * (long)c;
                    const T x0 = xc[0], x1 = xc[1], x2 = xc[2];
                    prod[q - q0] = __ldg(v) * x0 + __ldg(v + 32) * x1 + __ldg(v + 64) * x2;
                    prod[TILE + q - q0] = __ldg(v + 96) * x0 + __ldg(v + 128) * x1 + __ldg(v + 160) * x2;
                    prod[2 * TILE + q - q0] = __ldg(v + 192) * x0 + __ldg(v + 224) * x1 + __ldg(v + 256) * x2;
                }
            }
            __syncthreads();
            // ---- phase 2: thread -> (row, component); component = tid % NC is fixed because nt % 3 == 0
            const int ntask = (r1 - r0) * NC;
            for (int k = tid; k < ntask; k += nt) {
                const int row = r0 + k / NC, c = k % NC;
                const int a = A.rowptr[row] - q0, b = A.rowptr[row + 1] - q0;
                T acc = 0;
                for (int j = a; j < b; j++) acc += prod[c * TILE + j];
                const long o = (long)row * NC + c;
                y[o] = acc;
                if (DOT) dot[MODE == MODE_CSR3 ? c : 0] += (double)acc * (double)x[o];
            }
            __syncthreads();
        } else {
            // a single row longer than a tile (r1 == r0 + 1): block-wide strided accumulation
            double acc[3] = {0, 0, 0};
            for (int q = q0 + tid; q < q1; q += nt) {
                const int c = __ldg(A.col + q);
                if (MODE == MODE_CSR1) {
                    acc[0] += (double)(__ldg(A.val + q) * x[c]);
                } else if (MODE == MODE_CSR3) {
                    const T a = __ldg(A.val + q);
                    const T *xc = x + 3 * (long)c;
                    acc[0] += (double)(a * xc[0]); acc[1] += (double)(a * xc[1]); acc[2] += (double)(a * xc[2]);
                } else {
                    const T *v = A.val + (long)(q >> 5) * 288 + (q & 31);
                    const T *xc = x + 3 * (long)c;
                    const T x0 = xc[0], x1 = xc[1], x2 = xc[2];
                    acc[0] += (double)(__ldg(v) * x0 + __ldg(v + 32) * x1 + __ldg(v + 64) * x2);
                    acc[1] += (double)(__ldg(v + 96) * x0 + __ldg(v + 128) * x1 + __ldg(v + 160) * x2);
                    acc[2] += (double)(__ldg(v + 192) * x0 + __ldg(v + 224) * x1 + __ldg(v + 256) * x2);
                }
            }
            block_sum<3>(acc, reinterpret_cast<double *>(prod));
            if (tid < NC) {
                const long o = (long)r0 * NC + tid;
                const T yv = (T)acc[tid];
                y[o] = yv;
                if (DOT) dot[MODE == MODE_CSR3 ? tid : 0] += (double)yv * (double)x[o];
            }
            __syncthreads();
        }
    }
}

template <typename T, int MODE>
__global__ void __launch_bounds__(CM_NT) spmv_kernel(MatView<T> A, const T *x, T *y)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *prod = reinterpret_cast<T *>(smem_raw);
    int t0, t1;
    cta_tiles(A.ntiles, blockIdx.x, gridDim.x, t0, t1);
    spmv_tiles<T, MODE, false>(A, x, y, t0, t1, prod, nullptr);
}

// --------------------------------------------------------------------------------------------------
// persistent CG
// --------------------------------------------------------------------------------------------------
template <typename T>
struct CgArgs {
    MatView<T> A;
    const T *b;
    T *x, *r, *p, *Ap;
    double *partial; // [2][grid][3]
    double tol;
    int maxiter, fixed;
    unsigned mask;
    CgResult *out;
};

// Sum over CTAs of partial[slot][cta][c] (fixed order; every CTA computes the same bits).
template <int NR>
__device__ __forceinline__ void grid_sum(const double *partial, int slot, double (&out)[NR], double *sh)
{
    const int nb = gridDim.x;
    double v[NR];
#pragma unroll
    for (int c = 0; c < NR; c++) v[c] = 0;
    for (int j = threadIdx.x; j < nb; j += blockDim.x)
#pragma unroll
        for (int c = 0; c < NR; c++) v[c] += __ldcg(partial + ((long)slot * nb + j) * 3 + c);
    block_sum<NR>(v, sh);
#pragma unroll
    for (int c = 0; c < NR; c++) out[c] = v[c];
}

template <typename T, int MODE>
__global__ void __launch_bounds__(CM_NT) cg_kernel(CgArgs<T> a)
{
    constexpr int NC = ModeTraits<MODE>::NC, NR = ModeTraits<MODE>::NR;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    T *prod = reinterpret_cast<T *>(smem_raw);
    __shared__ double red[3 * 32];
    cg::grid_group grid = cg::this_grid();
    const int tid = threadIdx.x, nt = blockDim.x, nb = gridDim.x, bid = blockIdx.x;
    int t0, t1;
    cta_tiles(a.A.ntiles, bid, nb, t0, t1);
    // own entries: [e0, e1) of the interleaved vectors
    const long e0 = (long)a.A.tile_row[t0] * NC, e1 = (long)a.A.tile_row[t1] * NC;
    double *part0 = a.partial + ((long)0 * nb + bid) * 3, *part1 = a.partial + ((long)1 * nb + bid) * 3;
    // component served by this thread in the vector phases: e0 % 3 == 0 and nt % 3 == 0, so it is fixed
    const int c = (NR == 3) ? tid % 3 : 0;

    // ---- r = b - A x0, p = r, rr, bb
    spmv_tiles<T, MODE, false>(a.A, a.x, a.Ap, t0, t1, prod, nullptr);
    double s_rr[3] = {0, 0, 0}, s_bb[3] = {0, 0, 0};
    for (long i = e0 + tid; i < e1; i += nt) {
        const T bi = a.b[i], ri = bi - a.Ap[i];
        a.r[i] = ri;
        a.p[i] = ri;
        s_rr[c] += (double)ri * (double)ri;
        s_bb[c] += (double)bi * (double)bi;
    }
    block_sum<3>(s_rr, red);
    block_sum<3>(s_bb, red);
    if (tid == 0)
        for (int c = 0; c < 3; c++) { part0[c] = s_rr[c]; part1[c] = s_bb[c]; }
    grid.sync();
    double rr[NR], bb[NR];
    grid_sum<NR>(a.partial, 0, rr, red);
    grid_sum<NR>(a.partial, 1, bb, red);
    grid.sync(); // partial slots are reused below

    bool active[NR];
    int iters[NR], status = CM_OK;
    bool zero_rhs[NR];
#pragma unroll
    for (int c = 0; c < NR; c++) {
        iters[c] = 0;
        active[c] = (a.mask >> c) & 1u;
        zero_rhs[c] = active[c] && bb[c] == 0.0 && a.fixed < 0; // ||b|| = 0 -> x = 0, 0 iterations
        if (zero_rhs[c]) { active[c] = false; rr[c] = 0; }
    }
    bool anyzero = false;
#pragma unroll
    for (int c = 0; c < NR; c++) anyzero |= zero_rhs[c];
    if (anyzero)
        for (long i = e0 + tid; i < e1; i += nt) {
            if (zero_rhs[c]) a.x[i] = 0;
        }

    for (int k = 0;; k++) {
        bool any = false;
#pragma unroll
        for (int c = 0; c < NR; c++) {
            if (!active[c]) continue;
            if (rr[c] == 0.0) active[c] = false;
            else if (a.fixed >= 0) { if (k == a.fixed) active[c] = false; }
            else if (rr[c] < a.tol * a.tol * bb[c]) active[c] = false;
            else if (k >= a.maxiter) { active[c] = false; if (status == CM_OK) status = CM_E_CG_MAXITER; }
            any |= active[c];
        }
        if (!any) break;
        // ---- A: Ap = A p, pAp
        double s_pap[3] = {0, 0, 0};
        spmv_tiles<T, MODE, true>(a.A, a.p, a.Ap, t0, t1, prod, s_pap);
        block_sum<3>(s_pap, red);
        if (tid == 0)
            for (int c = 0; c < 3; c++) part0[c] = s_pap[c];
        grid.sync();
        double pap[NR];
        grid_sum<NR>(a.partial, 0, pap, red);
        T alpha[NR];
#pragma unroll
        for (int c = 0; c < NR; c++) {
            alpha[c] = 0;
            if (!active[c]) continue;
            if (!(pap[c] > 0.0)) { active[c] = false; status = CM_E_CG_BREAKDOWN; continue; }
            alpha[c] = (T)(rr[c] / pap[c]);
        }
        // ---- B: x += alpha p, r -= alpha Ap, rr_new
        double s_new[3] = {0, 0, 0};
        for (long i = e0 + tid; i < e1; i += nt) {
            if (!active[c]) continue;
            a.x[i] += alpha[c] * a.p[i];
            const T ri = a.r[i] - alpha[c] * a.Ap[i];
            a.r[i] = ri;
            s_new[c] += (double)ri * (double)ri;
        }
        block_sum<3>(s_new, red);
        if (tid == 0)
            for (int c = 0; c < 3; c++) part1[c] = s_new[c];
        grid.sync();
        double rr_new[NR];
        grid_sum<NR>(a.partial, 1, rr_new, red);
        // ---- C: p = r + beta p
        T beta[NR];
#pragma unroll
        for (int c = 0; c < NR; c++) beta[c] = active[c] ? (T)(rr_new[c] / rr[c]) : (T)0;
        for (long i = e0 + tid; i < e1; i += nt) {
            if (!active[c]) continue;
            a.p[i] = a.r[i] + beta[c] * a.p[i];
        }
#pragma unroll
        for (int c = 0; c < NR; c++)
            if (active[c]) { rr[c] = rr_new[c]; iters[c]++; }
        grid.sync();
    }
    if (bid == 0 && tid == 0) {
        for (int c = 0; c < 3; c++) { a.out->iters[c] = 0; a.out->relres[c] = 0; }
        for (int c = 0; c < NR; c++) {
            a.out->iters[c] = iters[c];
            a.out->relres[c] = bb[c] > 0 ? sqrt(rr[c] / bb[c]) : 0.0;
        }
        a.out->status = status;
    }
}

// --------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------
int build_tiling(const std::vector<int> &rowptr, long N, int tile, Tiling *out, cudaStream_t st)
{
    std::vector<int> tr;
    tr.push_back(0);
    long r = 0;
    while (r < N) {
        long r1 = r + 1; // always at least one row (a single over-long row forms its own tile)
        while (r1 < N && rowptr[r1 + 1] - rowptr[r] <= tile) r1++;
        tr.push_back((int)r1);
        r = r1;
    }
    out->tile = tile;
    out->ntiles = (int)tr.size() - 1;
    CM_CUDA(cudaMalloc((void **)&out->d_tile_row, tr.size() * sizeof(int)));
    CM_CUDA(cudaMemcpyAsync(out->d_tile_row, tr.data(), tr.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    CM_CUDA(cudaStreamSynchronize(st));
    return CM_OK;
}

template <typename T>
static const T *mat_values(const System<T> *S, cm_matrix_id id)
{
    switch (id) {
    case CM_MAT_K_MS: return S->Kms;
    case CM_MAT_K_GS1: return S->Kgs1;
    case CM_MAT_K_GS2: return S->Kgs2;
    case CM_MAT_MASS: return S->Mm;
    case CM_MAT_K_MECH: return S->Kmech;
    }
    return nullptr;
}

template <typename T>
static int make_view(const System<T> *S, cm_matrix_id id, int mode, MatView<T> *A)
{
    const T *v = mat_values(S, id);
    if (!v) { cm_set_error("matrix %d is not assembled (no elastic material?)", (int)id); return CM_E_BADARG; }
    if ((id == CM_MAT_K_MECH) != (mode == MODE_BSR3)) { cm_set_error("matrix %d does not match mode %d", (int)id, mode); return CM_E_BADARG; }
    const Tiling &tl = (mode == MODE_CSR1) ? S->til1 : S->til3;
    A->rowptr = S->mesh->d_rowptr; A->col = S->mesh->d_col; A->val = v;
    A->tile_row = tl.d_tile_row; A->ntiles = tl.ntiles; A->tile = tl.tile; A->N = S->N;
    return CM_OK;
}

template <typename T, int MODE>
static size_t smem_bytes() { return (size_t)ModeTraits<MODE>::NC * ModeTraits<MODE>::TILE * sizeof(T); }

template <typename T, int MODE>
static int launch_spmv(System<T> *S, const MatView<T> &A, const T *x, T *y, cudaStream_t st)
{
    int occ = 0;
    CM_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, spmv_kernel<T, MODE>, CM_NT, smem_bytes<T, MODE>()));
    int grid = std::max(1, std::min(A.ntiles, occ * S->num_sms));
    S->prof.begin(CM_PROF_SPMV, st);
    spmv_kernel<T, MODE><<<grid, CM_NT, smem_bytes<T, MODE>(), st>>>(A, x, y);
    S->prof.end(st);
    CM_CUDA(cudaGetLastError());
    return CM_OK;
}

template <typename T>
int sys_spmv(System<T> *S, cm_matrix_id id, int mode, const T *x, T *y, cudaStream_t st)
{
    MatView<T> A;
    CM_TRY(make_view(S, id, mode, &A));
    switch (mode) {
    case MODE_CSR1: return launch_spmv<T, MODE_CSR1>(S, A, x, y, st);
    case MODE_CSR3: return launch_spmv<T, MODE_CSR3>(S, A, x, y, st);
    case MODE_BSR3: return launch_spmv<T, MODE_BSR3>(S, A, x, y, st);
    }
    return CM_E_BADARG;
}

template <typename T, int MODE>
static int launch_cg(System<T> *S, CgArgs<T> &a, int prof_cls, cudaStream_t st)
{
    int occ = 0;
    CM_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, cg_kernel<T, MODE>, CM_NT, smem_bytes<T, MODE>()));
    if (occ < 1) { cm_set_error("cg kernel does not fit on an SM"); return CM_E_CUDA; }
    int grid = std::max(1, std::min({a.A.ntiles, occ * S->num_sms, S->grid_cap}));
    void *args[] = {&a};
    S->prof.begin(prof_cls, st);
    cudaError_t e = cudaLaunchCooperativeKernel((void *)cg_kernel<T, MODE>, dim3(grid), dim3(CM_NT), args, smem_bytes<T, MODE>(), st);
    S->prof.end(st);
    if (e != cudaSuccess) { cm_set_error("cudaLaunchCooperativeKernel: %s", cudaGetErrorString(e)); return CM_E_CUDA; }
    return CM_OK;
}

// Enqueue one CG solve; the result lands in S->d_res[slot].
template <typename T>
int sys_cg(System<T> *S, cm_matrix_id id, int mode, const T *b, T *x, double tol, int maxiter, int fixed, unsigned mask, int slot,
           int prof_cls, cudaStream_t st)
{
    CgArgs<T> a;
    CM_TRY(make_view(S, id, mode, &a.A));
    a.b = b; a.x = x; a.r = S->r; a.p = S->p; a.Ap = S->Ap; a.partial = S->partial;
    a.tol = tol; a.maxiter = maxiter; a.fixed = fixed; a.mask = mask; a.out = S->d_res + slot;
    switch (mode) {
    case MODE_CSR1: return launch_cg<T, MODE_CSR1>(S, a, prof_cls, st);
    case MODE_CSR3: return launch_cg<T, MODE_CSR3>(S, a, prof_cls, st);
    case MODE_BSR3: return launch_cg<T, MODE_BSR3>(S, a, prof_cls, st);
    }
    return CM_E_BADARG;
}

template int sys_spmv<double>(System<double> *, cm_matrix_id, int, const double *, double *, cudaStream_t);
template int sys_spmv<float>(System<float> *, cm_matrix_id, int, const float *, float *, cudaStream_t);
template int sys_cg<double>(System<double> *, cm_matrix_id, int, const double *, double *, double, int, int, unsigned, int, int, cudaStream_t);
template int sys_cg<float>(System<float> *, cm_matrix_id, int, const float *, float *, double, int, int, unsigned, int, int, cudaStream_t);
