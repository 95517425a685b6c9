// S4 / S7 / S10: sparse matrix-vector products and the fused, persistent, unpreconditioned
// conjugate-gradient solver (O-4).
//
// Layout.  All scalar matrices share rowptr / colidx; values are plain CSR arrays.  The 3x3-block
// elasticity matrix is stored "tile-SoA": blocks are grouped by 32 and inside a group the 9 block
// entries are 9 contiguous planes of 32 values, [nnz/32][9][32], so that a warp reading 32 consecutive
// blocks issues 9 fully coalesced 256-byte (fp64) loads and the whole matrix is one sequential stream.
//
// Work decomposition.  Rows are cut once, on the host, into "warp tiles" of consecutive rows holding at most
// WT = 32 U nonzeros (blocks).  A CTA owns a contiguous range of tiles for the whole solve and its warps take
// them round-robin, each warp on its own -- there is no block-wide barrier inside the SpMV.  Per tile:
//   phase 1  one lane per nonzero, U in flight per lane: stream value(s) + column index, gather x[col] (1 or 3
//            components, L1/L2 hits thanks to the locality ordering), write the product(s) to the warp's
//            private shared-memory slots;
//   phase 2  one lane per (row, component): sum the row's segment of products in column order
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
    const int2 *tile; // ntiles + 1 descriptors {first row, first nonzero}
    int ntiles;
    long N;
};

// WT = nonzeros (blocks) per warp tile = 32 * U, U loads in flight per lane.
template <int MODE> struct ModeTraits;
template <> struct ModeTraits<MODE_CSR1> { static constexpr int NC = 1, NR = 1, NV = 1, WT = CM_WT_CSR1; };
template <> struct ModeTraits<MODE_CSR3> { static constexpr int NC = 3, NR = 3, NV = 1, WT = CM_WT_CSR3; };
template <> struct ModeTraits<MODE_BSR3> { static constexpr int NC = 3, NR = 1, NV = 9, WT = CM_WT_BSR3; };

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

// y = A x on the warp tiles [t0, t1) of this CTA (warp w takes t0 + w, t0 + w + nwarps, ...); optionally
// accumulates dot[c] += y.x over the rows written.  `prod` = this warp's private NC * WT shared-memory slots.
// No block-wide barrier: warps stream independently, so DRAM latency is hidden by the other warps of the SM.
template <typename T, int MODE, bool DOT>
__device__ __forceinline__ void spmv_warp_tiles(const MatView<T> &A, const T *x, T *y, int t0, int t1, T *prod, double (&dot)[3])
{
    constexpr int NC = ModeTraits<MODE>::NC, NV = ModeTraits<MODE>::NV, WT = ModeTraits<MODE>::WT, U = WT / 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    int t = t0 + warp;
    if (t >= t1) return;
    int2 d0 = __ldg(A.tile + t), d1 = __ldg(A.tile + t + 1);
    for (;;) {
        const int r0 = d0.x, q0 = d0.y, r1 = d1.x, q1 = d1.y;
        const int tn = t + nw;
        if (tn < t1) { d0 = __ldg(A.tile + tn); d1 = __ldg(A.tile + tn + 1); } // prefetch the next descriptors
        if (q1 - q0 <= WT) {
            // ---- phase 1: all streaming loads first (U per lane in flight), then the dependent gathers
            int col[U];
            T v[U][NV];
#pragma unroll
            for (int j = 0; j < U; j++) {
                const int q = q0 + lane + 32 * j;
                col[j] = 0;
#pragma unroll
                for (int k = 0; k < NV; k++) v[j][k] = 0;
                if (q < q1) {
                    col[j] = __ldg(A.col + q);
                    if (MODE == MODE_BSR3) {
                        const T *vp = A.val + (long)(q >> 5) * 288 + (q & 31);
#pragma unroll
                        for (int k = 0; k < NV; k++) v[j][k] = __ldg(vp + 32 * k);
                    } else {
                        v[j][0] = __ldg(A.val + q);
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < U; j++) {
                const int q = q0 + lane + 32 * j;
                if (q < q1) {
                    const int o = q - q0;
                    if (MODE == MODE_CSR1) {
                        prod[o] = v[j][0] * x[col[j]];
                    } else {
                        const T *xc = x + 3 * (long)col[j];
                        const T x0 = xc[0], x1 = xc[1], x2 = xc[2];
                        if (MODE == MODE_CSR3) {
                            prod[o] = v[j][0] * x0; prod[WT + o] = v[j][0] * x1; prod[2 * WT + o] = v[j][0] * x2;
                        } else {
                            prod[o] = v[j][0] * x0 + v[j][1] * x1 + v[j][2] * x2;
                            prod[WT + o] = v[j][3] * x0 + v[j][4] * x1 + v[j][5] * x2;
                            prod[2 * WT + o] = v[j][6] * x0 + v[j][7] * x1 + v[j][8] * x2;
                        }
                    }
                }
            }
            __syncwarp();
            // ---- phase 2: lane -> (row, component); sum the row's products in column order
            const int ntask = (r1 - r0) * NC;
            for (int k = lane; k < ntask; k += 32) {
                const int row = r0 + k / NC, c = k % NC;
                const int a = __ldg(A.rowptr + row) - q0, b = __ldg(A.rowptr + row + 1) - q0;
                T acc = 0;
                for (int j = a; j < b; j++) acc += prod[c * WT + j];
                const long o = (long)row * NC + c;
                y[o] = acc;
                if (DOT) {
                    const double d = (double)acc * (double)x[o];
                    if (MODE != MODE_CSR3 || c == 0) dot[0] += d;
                    else if (c == 1) dot[1] += d;
                    else dot[2] += d;
                }
            }
            __syncwarp();
        } else {
            // a single row longer than a warp tile (r1 == r0 + 1): lane-strided accumulation, shuffle reduction
            double acc[3] = {0, 0, 0};
            for (int q = q0 + lane; q < q1; q += 32) {
                const int c = __ldg(A.col + q);
                if (MODE == MODE_CSR1) {
                    acc[0] += (double)(__ldg(A.val + q) * x[c]);
                } else if (MODE == MODE_CSR3) {
                    const T a = __ldg(A.val + q);
                    const T *xc = x + 3 * (long)c;
                    acc[0] += (double)(a * xc[0]); acc[1] += (double)(a * xc[1]); acc[2] += (double)(a * xc[2]);
                } else {
                    const T *vp = A.val + (long)(q >> 5) * 288 + (q & 31);
                    const T *xc = x + 3 * (long)c;
                    const T x0 = xc[0], x1 = xc[1], x2 = xc[2];
                    acc[0] += (double)(__ldg(vp) * x0 + __ldg(vp + 32) * x1 + __ldg(vp + 64) * x2);
                    acc[1] += (double)(__ldg(vp + 96) * x0 + __ldg(vp + 128) * x1 + __ldg(vp + 160) * x2);
                    acc[2] += (double)(__ldg(vp + 192) * x0 + __ldg(vp + 224) * x1 + __ldg(vp + 256) * x2);
                }
            }
#pragma unroll
            for (int k = 0; k < 3; k++)
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], o);
            if (lane == 0) {
#pragma unroll
                for (int c = 0; c < NC; c++) {
                    const long o = (long)r0 * NC + c;
                    const T yv = (T)acc[c];
                    y[o] = yv;
                    if (DOT) dot[MODE == MODE_CSR3 ? c : 0] += (double)yv * (double)x[o];
                }
            }
        }
        if (tn >= t1) break;
        t = tn;
    }
}

template <typename T, int MODE>
__global__ void __launch_bounds__(CM_NT) spmv_kernel(MatView<T> A, const T *x, T *y)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int PW = ModeTraits<MODE>::NC * ModeTraits<MODE>::WT;
    T *prod = reinterpret_cast<T *>(smem_raw) + (threadIdx.x >> 5) * PW;
    int t0, t1;
    cta_tiles(A.ntiles, blockIdx.x, gridDim.x, t0, t1);
    double dot[3] = {0, 0, 0};
    spmv_warp_tiles<T, MODE, false>(A, x, y, t0, t1, prod, dot);
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

template <int NR, typename V>
__device__ __forceinline__ V pick(const V (&a)[NR], int c)
{
    V r = a[0];
    if (NR == 3) { if (c == 1) r = a[1]; else if (c == 2) r = a[2]; }
    return r;
}

template <typename T, int MODE>
__global__ void __launch_bounds__(CM_NT, 2) cg_kernel(CgArgs<T> a)
{
    constexpr int NC = ModeTraits<MODE>::NC, NR = ModeTraits<MODE>::NR, VU = 2;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int PW = NC * ModeTraits<MODE>::WT;
    T *prod = reinterpret_cast<T *>(smem_raw) + (threadIdx.x >> 5) * PW;
    __shared__ double red[6 * 32];
    cg::grid_group grid = cg::this_grid();
    const int tid = threadIdx.x, nt = blockDim.x, nb = gridDim.x, bid = blockIdx.x;
    int t0, t1;
    cta_tiles(a.A.ntiles, bid, nb, t0, t1);
    // own entries: [e0, e1) of the interleaved vectors
    const long e0 = (long)a.A.tile[t0].x * NC, e1 = (long)a.A.tile[t1].x * NC;
    double *part0 = a.partial + ((long)0 * nb + bid) * 3, *part1 = a.partial + ((long)1 * nb + bid) * 3;
    // component served by this thread in the vector phases: e0 % 3 == 0 and nt % 3 == 0, so it is fixed
    const int c = (NR == 3) ? tid % 3 : 0;
    double nodot[3] = {0, 0, 0};

    // ---- r = b - A x0, p = r, rr, bb
    spmv_warp_tiles<T, MODE, false>(a.A, a.x, a.Ap, t0, t1, prod, nodot);
    __syncthreads(); // Ap of the CTA's rows was written by other warps
    {
        double srr = 0, sbb = 0;
        for (long i = e0 + tid; i < e1; i += nt) {
            const T bi = a.b[i], ri = bi - a.Ap[i];
            a.r[i] = ri;
            a.p[i] = ri;
            srr += (double)ri * (double)ri;
            sbb += (double)bi * (double)bi;
        }
        double v[6];
#pragma unroll
        for (int k = 0; k < 3; k++) { v[k] = (k == c) ? srr : 0.0; v[3 + k] = (k == c) ? sbb : 0.0; }
        block_sum<6>(v, red);
        if (tid == 0)
            for (int k = 0; k < 3; k++) { part0[k] = v[k]; part1[k] = v[3 + k]; }
    }
    grid.sync();
    double rr[NR], bb[NR];
    grid_sum<NR>(a.partial, 0, rr, red);
    grid_sum<NR>(a.partial, 1, bb, red);
    grid.sync(); // partial slots are reused below

    bool active[NR];
    int iters[NR], status = CM_OK;
    bool zero_rhs[NR];
#pragma unroll
    for (int k = 0; k < NR; k++) {
        iters[k] = 0;
        active[k] = (a.mask >> k) & 1u;
        zero_rhs[k] = active[k] && bb[k] == 0.0 && a.fixed < 0; // ||b|| = 0 -> x = 0, 0 iterations
        if (zero_rhs[k]) { active[k] = false; rr[k] = 0; }
    }
    if (pick<NR>(zero_rhs, c))
        for (long i = e0 + tid; i < e1; i += nt) a.x[i] = 0;

    for (int k = 0;; k++) {
        bool any = false;
#pragma unroll
        for (int q = 0; q < NR; q++) {
            if (!active[q]) continue;
            if (rr[q] == 0.0) active[q] = false;
            else if (a.fixed >= 0) { if (k == a.fixed) active[q] = false; }
            else if (rr[q] < a.tol * a.tol * bb[q]) active[q] = false;
            else if (k >= a.maxiter) { active[q] = false; if (status == CM_OK) status = CM_E_CG_MAXITER; }
            any |= active[q];
        }
        if (!any) break;
        // ---- A: Ap = A p, pAp
        double s_pap[3] = {0, 0, 0};
        spmv_warp_tiles<T, MODE, true>(a.A, a.p, a.Ap, t0, t1, prod, s_pap);
        block_sum<3>(s_pap, red);
        if (tid == 0)
            for (int q = 0; q < 3; q++) part0[q] = s_pap[q];
        grid.sync();
        double pap[NR];
        grid_sum<NR>(a.partial, 0, pap, red);
        T alpha[NR];
#pragma unroll
        for (int q = 0; q < NR; q++) {
            alpha[q] = 0;
            if (!active[q]) continue;
            if (!(pap[q] > 0.0)) { active[q] = false; status = CM_E_CG_BREAKDOWN; continue; }
            alpha[q] = (T)(rr[q] / pap[q]);
        }
        // ---- B: x += alpha p, r -= alpha Ap, rr_new   (VU independent elements per thread in flight)
        const bool my_active = pick<NR>(active, c);
        double snew = 0;
        if (my_active) {
            const T al = pick<NR>(alpha, c);
            for (long i = e0 + tid; i < e1; i += (long)nt * VU) {
                T pv[VU], av[VU], xv[VU], rv[VU];
#pragma unroll
                for (int q = 0; q < VU; q++) {
                    const long ii = i + (long)q * nt;
                    if (ii < e1) { pv[q] = a.p[ii]; av[q] = a.Ap[ii]; xv[q] = a.x[ii]; rv[q] = a.r[ii]; }
                }
#pragma unroll
                for (int q = 0; q < VU; q++) {
                    const long ii = i + (long)q * nt;
                    if (ii < e1) {
                        a.x[ii] = xv[q] + al * pv[q];
                        const T ri = rv[q] - al * av[q];
                        a.r[ii] = ri;
                        snew += (double)ri * (double)ri;
                    }
                }
            }
        }
        {
            double v[3];
#pragma unroll
            for (int q = 0; q < 3; q++) v[q] = (q == c) ? snew : 0.0;
            block_sum<3>(v, red);
            if (tid == 0)
                for (int q = 0; q < 3; q++) part1[q] = v[q];
        }
        grid.sync();
        double rr_new[NR];
        grid_sum<NR>(a.partial, 1, rr_new, red);
        // ---- C: p = r + beta p
        T beta[NR];
#pragma unroll
        for (int q = 0; q < NR; q++) beta[q] = active[q] ? (T)(rr_new[q] / rr[q]) : (T)0;
        if (my_active) {
            const T be = pick<NR>(beta, c);
            for (long i = e0 + tid; i < e1; i += (long)nt * VU) {
                T pv[VU], rv[VU];
#pragma unroll
                for (int q = 0; q < VU; q++) {
                    const long ii = i + (long)q * nt;
                    if (ii < e1) { pv[q] = a.p[ii]; rv[q] = a.r[ii]; }
                }
#pragma unroll
                for (int q = 0; q < VU; q++) {
                    const long ii = i + (long)q * nt;
                    if (ii < e1) a.p[ii] = rv[q] + be * pv[q];
                }
            }
        }
#pragma unroll
        for (int q = 0; q < NR; q++)
            if (active[q]) { rr[q] = rr_new[q]; iters[q]++; }
        grid.sync();
    }
    if (bid == 0 && tid == 0) {
        for (int q = 0; q < 3; q++) { a.out->iters[q] = 0; a.out->relres[q] = 0; }
        for (int q = 0; q < NR; q++) {
            a.out->iters[q] = iters[q];
            a.out->relres[q] = bb[q] > 0 ? sqrt(rr[q] / bb[q]) : 0.0;
        }
        a.out->status = status;
    }
}

// --------------------------------------------------------------------------------------------------
// host side
// --------------------------------------------------------------------------------------------------
int build_tiling(const std::vector<int> &rowptr, long N, int tile, Tiling *out, cudaStream_t st)
{
    std::vector<int2> td;
    long r = 0;
    while (r < N) {
        td.push_back(make_int2((int)r, rowptr[r]));
        long r1 = r + 1; // always at least one row (a single over-long row forms its own tile)
        while (r1 < N && rowptr[r1 + 1] - rowptr[r] <= tile) r1++;
        r = r1;
    }
    td.push_back(make_int2((int)N, rowptr[N]));
    out->tile = tile;
    out->ntiles = (int)td.size() - 1;
    CM_CUDA(cudaMalloc((void **)&out->d_tile, td.size() * sizeof(int2)));
    CM_CUDA(cudaMemcpyAsync(out->d_tile, td.data(), td.size() * sizeof(int2), cudaMemcpyHostToDevice, st));
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
    const Tiling &tl = S->til[mode];
    A->rowptr = S->mesh->d_rowptr; A->col = S->mesh->d_col; A->val = v;
    A->tile = tl.d_tile; A->ntiles = tl.ntiles; A->N = S->N;
    return CM_OK;
}

template <typename T, int MODE>
static size_t smem_bytes() { return (size_t)(CM_NT / 32) * ModeTraits<MODE>::NC * ModeTraits<MODE>::WT * sizeof(T); }

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
