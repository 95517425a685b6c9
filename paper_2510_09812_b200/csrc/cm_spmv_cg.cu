// S4 / S7 / S10: sparse matrix-vector products and the fused, persistent, unpreconditioned
// conjugate-gradient solver (O-4).
//
// Layout.  Matrices are stored sliced (SELL-C, cm_internal.h): C consecutive rows form a slice, padded to the
// slice's longest row and stored column-major, so that the 32 lanes of a warp read 32 consecutive elements of
// every array.  The 3x3-block elasticity matrix keeps its 9 block entries in 9 planes per slice
// ([slice][3r + c][L_slice]): each plane is one coalesced stream.  On the paper's tetrahedral meshes almost every
// row has 15 entries, so the padding is about 1.5 % (config 3).
//
// SpMV.  One warp per slice, all 32 lanes busy: lane -> (row i % C of the slice, column phase lane / C).  A lane
// streams its elements (value(s) + column index, U iterations in flight, L1 bypassed, L2 evict-first), gathers
// x[col] (L1 / L2 hits thanks to the locality ordering) and accumulates in registers in column order; the
// 32 / C column phases of a row are combined with a fixed shuffle butterfly.  No shared memory, no atomics.
//
// CG.  ONE cooperative launch per solve; a CTA owns a contiguous range of slices, hence of rows, for the whole
// solve.  Per iteration k (three grid-wide barriers, the two dot products ride on two of them):
//   C   x += alpha_{k-1} p_{k-1} (deferred: p_{k-1} is read here anyway), p_k = r_k + beta p_{k-1} on the own rows;  -> barrier
//   A   Ap = A p_k, dot p.Ap;                                                              -> barrier, alpha
//   B   r -= alpha Ap, dot r.r;                                                            -> barrier, beta
// Every CTA reduces the per-CTA partial sums in the same fixed order, so all CTAs take the same decisions and the
// result is bit-reproducible run to run.  Dot products accumulate in fp64 in both precisions (R20).
#include <cooperative_groups.h>

#include <algorithm>

#include "cm_internal.h"

namespace cg = cooperative_groups;

template <typename T>
struct MatView {
    const int *sp;  // nslices + 1 element offsets
    const int *col; // E column indices, sliced order
    const T *val;   // E values (scalar) or 9 E (block: 9 planes per slice)
    int nslices;
    long N;
};

// NC vector components per node, NR independent right-hand sides, NV stored values per element, C rows per slice,
// U 32-element iterations in flight per warp.
template <int MODE> struct ModeTraits;
#ifndef CM_U_CSR1
#define CM_U_CSR1 8
#endif
#ifndef CM_U_CSR3
#define CM_U_CSR3 8
#endif
#ifndef CM_U_BSR3
#define CM_U_BSR3 2
#endif
template <> struct ModeTraits<MODE_CSR1> { static constexpr int NC = 1, NR = 1, NV = 1, C = CM_C_SCALAR, U = CM_U_CSR1; };
template <> struct ModeTraits<MODE_CSR3> { static constexpr int NC = 3, NR = 3, NV = 1, C = CM_C_SCALAR, U = CM_U_CSR3; };
template <> struct ModeTraits<MODE_BSR3> { static constexpr int NC = 3, NR = 1, NV = 9, C = CM_C_BLOCK, U = CM_U_BSR3; };

// ---- streaming loads of the matrix: read once per pass, so keep them out of L1 and first in line for L2 eviction
__device__ __forceinline__ unsigned long long policy_evict_first()
{
    unsigned long long p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ double ld_stream(const double *p, unsigned long long pol)
{
    double v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ float ld_stream(const float *p, unsigned long long pol)
{
    float v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ int ld_stream(const int *p, unsigned long long pol)
{
    int v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.s32 %0, [%1], %2;" : "=r"(v) : "l"(p), "l"(pol));
    return v;
}

__device__ __forceinline__ double fma_t(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_t(float a, float b, float c) { return fmaf(a, b, c); }

// Contiguous slice range of CTA `b` out of `nb`.
__device__ __forceinline__ void cta_units(int n, int b, int nb, int &u0, int &u1)
{
    int q = n / nb, r = n % nb;
    u0 = b * q + min(b, r);
    u1 = u0 + q + (b < r ? 1 : 0);
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

template <int NR, typename V>
__device__ __forceinline__ V pick(const V (&a)[NR], int c)
{
    V r = a[0];
    if (NR == 3) { if (c == 1) r = a[1]; else if (c == 2) r = a[2]; }
    return r;
}

// x[col] for all NC components of a node
template <typename T, int MODE>
__device__ __forceinline__ void fetch(const T *__restrict__ x, int col, T (&out)[ModeTraits<MODE>::NC])
{
    constexpr int NC = ModeTraits<MODE>::NC;
    const long o = (long)col * NC;
#pragma unroll
    for (int c = 0; c < NC; c++) out[c] = x[o + c];
}

// Batches in flight per warp.  The fp32 block matrix streams half the bytes per element, so it takes twice the batches
// (measured on B200, config 3 fp32: mechanical CG 88 % -> 94 % of the measured HBM peak with 4 instead of 2).
#ifndef CM_U_BSR3_F32
#define CM_U_BSR3_F32 4
#endif
template <typename T, int MODE>
constexpr int batch_u() { return (MODE == MODE_BSR3 && sizeof(T) == 4) ? CM_U_BSR3_F32 : ModeTraits<MODE>::U; }

// One batch = U consecutive 32-element groups of one slice: the unit of the load pipeline.
template <typename T, int MODE>
struct Batch {
    int col[batch_u<T, MODE>()];
    T v[batch_u<T, MODE>()][ModeTraits<MODE>::NV];
};

// position in the stream of batches of a warp: slice s with extent [b0, b0 + L), batch offset it
struct Cursor {
    int s, b0, L, it;
};

template <typename T, int MODE>
__device__ __forceinline__ void load_batch(const MatView<T> &A, const Cursor &c, int lane, unsigned long long pol, Batch<T, MODE> &B)
{
    constexpr int NV = ModeTraits<MODE>::NV, U = batch_u<T, MODE>();
    const int *colp = A.col + c.b0;
    const T *valp = A.val + (long)NV * c.b0; // plane k at valp + k * L
#pragma unroll
    for (int u = 0; u < U; u++) {
        const int e = c.it + 32 * u + lane;
        B.col[u] = 0;
#pragma unroll
        for (int k = 0; k < NV; k++) B.v[u][k] = 0;
        if (e < c.L) {
            B.col[u] = ld_stream(colp + e, pol);
#pragma unroll
            for (int k = 0; k < NV; k++) B.v[u][k] = ld_stream(valp + (long)k * c.L + e, pol);
        }
    }
}

// y = A x on the slices [u0, u1) of this CTA (warp w takes u0 + w, u0 + w + nwarps, ...); optionally accumulates
// dot[c] += y.x over the rows written.
template <typename T, int MODE, bool DOT>
__device__ __forceinline__ void spmv_units(const MatView<T> &A, const T *__restrict__ x, T *y, int u0, int u1, double (&dot)[3])
{
    constexpr int NC = ModeTraits<MODE>::NC, C = ModeTraits<MODE>::C, U = batch_u<T, MODE>();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int rl = lane % C, jl = lane / C;
    const unsigned long long pol = policy_evict_first();
    Cursor cur;
    cur.s = u0 + warp;
    if (cur.s >= u1) return;
    cur.b0 = __ldg(A.sp + cur.s);
    cur.L = __ldg(A.sp + cur.s + 1) - cur.b0;
    cur.it = 0;
    // extent of the slice after the current one, fetched one slice ahead
    int n0 = 0, n1 = 0;
    if (cur.s + nw < u1) { n0 = __ldg(A.sp + cur.s + nw); n1 = __ldg(A.sp + cur.s + nw + 1); }
    Batch<T, MODE> Bc;
    load_batch<T, MODE>(A, cur, lane, pol, Bc);
    T acc[NC];
#pragma unroll
    for (int c = 0; c < NC; c++) acc[c] = 0;
    for (;;) {
        // ---- advance the cursor and issue the next batch's streaming loads
        Cursor nxt = cur;
        nxt.it += 32 * U;
        const bool last_of_slice = nxt.it >= cur.L;
        if (last_of_slice) {
            nxt.s = cur.s + nw; nxt.b0 = n0; nxt.L = n1 - n0; nxt.it = 0;
            if (nxt.s + nw < u1) { n0 = __ldg(A.sp + nxt.s + nw); n1 = __ldg(A.sp + nxt.s + nw + 1); }
        }
        const bool more = nxt.s < u1;
        // ---- current batch: dependent gathers, multiply-accumulate in column order
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int e = cur.it + 32 * u + lane;
            if (e < cur.L) {
                T xv[NC];
                fetch<T, MODE>(x, Bc.col[u], xv);
                if (MODE == MODE_BSR3) {
                    acc[0] += Bc.v[u][0] * xv[0] + Bc.v[u][1] * xv[1] + Bc.v[u][2] * xv[2];
                    acc[1] += Bc.v[u][3] * xv[0] + Bc.v[u][4] * xv[1] + Bc.v[u][5] * xv[2];
                    acc[2] += Bc.v[u][6] * xv[0] + Bc.v[u][7] * xv[1] + Bc.v[u][8] * xv[2];
                } else {
#pragma unroll
                    for (int c = 0; c < NC; c++) acc[c] += Bc.v[u][0] * xv[c];
                }
            }
        }
        if (last_of_slice) {
            // combine the 32 / C column phases of each row (fixed butterfly: every lane ends with the same sum)
#pragma unroll
            for (int o = C; o < 32; o <<= 1)
#pragma unroll
                for (int c = 0; c < NC; c++) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
            const long row = (long)cur.s * C + rl;
            if (row < A.N) {
                if (MODE == MODE_BSR3) {
                    // 32 / C = 4 >= 3 phases: phase jl writes component jl
                    if (jl < 3) {
                        const T a = jl == 0 ? acc[0] : (jl == 1 ? acc[1] : acc[2]);
                        y[3 * row + jl] = a;
                        if (DOT) dot[0] += (double)a * (double)x[3 * row + jl];
                    }
                } else if (jl == 0) {
#pragma unroll
                    for (int c = 0; c < NC; c++) {
                        y[NC * row + c] = acc[c];
                        if (DOT) dot[c] += (double)acc[c] * (double)x[NC * row + c];
                    }
                }
            }
#pragma unroll
            for (int c = 0; c < NC; c++) acc[c] = 0;
        }
        if (!more) break;
        cur = nxt;
        load_batch<T, MODE>(A, cur, lane, pol, Bc);
    }
}

template <typename T, int MODE>
__global__ void __launch_bounds__(CM_NT, 2) spmv_kernel(MatView<T> A, const T *x, T *y)
{
    int u0, u1;
    cta_units(A.nslices, blockIdx.x, gridDim.x, u0, u1);
    double dot[3] = {0, 0, 0};
    spmv_units<T, MODE, false>(A, x, y, u0, u1, dot);
}

// --------------------------------------------------------------------------------------------------
// streaming vector phases of CG: 128-bit accesses, UN vectors per array per thread in flight
// --------------------------------------------------------------------------------------------------
template <typename T> struct VecOf;
template <> struct VecOf<double> { typedef double2 V; static constexpr int W = 2; };
template <> struct VecOf<float> { typedef float4 V; static constexpr int W = 4; };

// lane-wise c[j] * a[j] + b[j]
__device__ __forceinline__ double2 vfma(const double (&c)[2], double2 a, double2 b) { return make_double2(fma(c[0], a.x, b.x), fma(c[1], a.y, b.y)); }
__device__ __forceinline__ float4 vfma(const float (&c)[4], float4 a, float4 b)
{
    return make_float4(fmaf(c[0], a.x, b.x), fmaf(c[1], a.y, b.y), fmaf(c[2], a.z, b.z), fmaf(c[3], a.w, b.w));
}
// lane-wise acc[j] += v[j]^2 in fp64
__device__ __forceinline__ void vsq(double (&acc)[2], double2 v) { acc[0] += v.x * v.x; acc[1] += v.y * v.y; }
__device__ __forceinline__ void vsq(double (&acc)[4], float4 v)
{
    acc[0] += (double)v.x * (double)v.x; acc[1] += (double)v.y * (double)v.y;
    acc[2] += (double)v.z * (double)v.z; acc[3] += (double)v.w * (double)v.w;
}

// The streaming phases run over the CTA's own entries [e0, e1): a 16-byte aligned vector body (e0 is a multiple
// of 8 entries because slices hold 8 or 16 rows) plus a scalar tail.  e0 % 3 == 0 and blockDim.x * W % 3 == 0, so
// the component served by lane j of a thread's vectors is the same in every trip: (tid * W + j) % 3.

// C': x += alpha_prev pold (the x update of the PREVIOUS iteration, deferred to here because pold is read anyway: one
// vector stream less per iteration than updating x in phase B; the fma is the same, so x is bit-identical), then
// pnew = r + beta pold
template <typename T, int NR>
__device__ __forceinline__ void phase_p(T *pnew, const T *pold, const T *r, T *x, long e0, long e1, const T (&beta)[NR],
                                        const T (&aprev)[NR], bool upd_x)
{
    constexpr int W = VecOf<T>::W, UN = 2;
    typedef typename VecOf<T>::V V;
    const int tid = threadIdx.x, nt = blockDim.x;
    const long a1 = e0 + (e1 - e0) / W * W, nv = (a1 - e0) / W;
    T be[W], al[W];
#pragma unroll
    for (int j = 0; j < W; j++) {
        const int cj = NR == 3 ? (tid * W + j) % 3 : 0;
        be[j] = pick<NR>(beta, cj); al[j] = pick<NR>(aprev, cj);
    }
    V *pn = reinterpret_cast<V *>(pnew + e0), *xv = reinterpret_cast<V *>(x + e0);
    const V *po = reinterpret_cast<const V *>(pold + e0), *rv = reinterpret_cast<const V *>(r + e0);
    long v = tid;
    if (upd_x) {
        for (; v + (long)(UN - 1) * nt < nv; v += (long)nt * UN) {
            V a[UN], b[UN], c[UN];
#pragma unroll
            for (int q = 0; q < UN; q++) { a[q] = po[v + (long)q * nt]; b[q] = rv[v + (long)q * nt]; c[q] = xv[v + (long)q * nt]; }
#pragma unroll
            for (int q = 0; q < UN; q++) { xv[v + (long)q * nt] = vfma(al, a[q], c[q]); pn[v + (long)q * nt] = vfma(be, a[q], b[q]); }
        }
        for (; v < nv; v += nt) { const V a = po[v]; xv[v] = vfma(al, a, xv[v]); pn[v] = vfma(be, a, rv[v]); }
        for (long i = a1 + tid; i < e1; i += nt) {
            const int c = NR == 3 ? (int)(i % 3) : 0;
            const T pv = pold[i];
            x[i] = fma_t(pick<NR>(aprev, c), pv, x[i]);
            pnew[i] = fma_t(pick<NR>(beta, c), pv, r[i]);
        }
    } else {
        for (; v + (long)(UN - 1) * nt < nv; v += (long)nt * UN) {
            V a[UN], b[UN];
#pragma unroll
            for (int q = 0; q < UN; q++) { a[q] = po[v + (long)q * nt]; b[q] = rv[v + (long)q * nt]; }
#pragma unroll
            for (int q = 0; q < UN; q++) pn[v + (long)q * nt] = vfma(be, a[q], b[q]);
        }
        for (; v < nv; v += nt) pn[v] = vfma(be, po[v], rv[v]);
        for (long i = a1 + tid; i < e1; i += nt) pnew[i] = fma_t(pick<NR>(beta, NR == 3 ? (int)(i % 3) : 0), pold[i], r[i]);
    }
}

// the x update still pending when the loop ends: x += alpha_last p_last
template <typename T, int NR>
__device__ __forceinline__ void phase_x_final(T *x, const T *p, long e0, long e1, const T (&alpha)[NR])
{
    const int tid = threadIdx.x, nt = blockDim.x;
    for (long i = e0 + tid; i < e1; i += nt) x[i] = fma_t(pick<NR>(alpha, NR == 3 ? (int)(i % 3) : 0), p[i], x[i]);
}

// B: r -= alpha Ap; s[c] += sum of r_new^2 per component
template <typename T, int NR>
__device__ __forceinline__ void phase_xr(T *r, const T *Ap, long e0, long e1, const T (&alpha)[NR], double (&s)[3])
{
    constexpr int W = VecOf<T>::W, UN = 4;
    typedef typename VecOf<T>::V V;
    const int tid = threadIdx.x, nt = blockDim.x;
    const long a1 = e0 + (e1 - e0) / W * W, nv = (a1 - e0) / W;
    T nal[W];
    int cj[W];
    double acc[W];
#pragma unroll
    for (int j = 0; j < W; j++) { cj[j] = NR == 3 ? (tid * W + j) % 3 : 0; nal[j] = -pick<NR>(alpha, cj[j]); acc[j] = 0; }
    V *rv = reinterpret_cast<V *>(r + e0);
    const V *av = reinterpret_cast<const V *>(Ap + e0);
    long v = tid;
    for (; v + (long)(UN - 1) * nt < nv; v += (long)nt * UN) {
        V b[UN], d[UN];
#pragma unroll
        for (int q = 0; q < UN; q++) { b[q] = av[v + (long)q * nt]; d[q] = rv[v + (long)q * nt]; }
#pragma unroll
        for (int q = 0; q < UN; q++) {
            const V rn = vfma(nal, b[q], d[q]);
            rv[v + (long)q * nt] = rn;
            vsq(acc, rn);
        }
    }
    for (; v < nv; v += nt) {
        const V rn = vfma(nal, av[v], rv[v]);
        rv[v] = rn;
        vsq(acc, rn);
    }
#pragma unroll
    for (int j = 0; j < W; j++)
#pragma unroll
        for (int q = 0; q < 3; q++) s[q] += (cj[j] == q) ? acc[j] : 0.0;
    for (long i = a1 + tid; i < e1; i += nt) {
        const int c = NR == 3 ? (int)(i % 3) : 0;
        const T ri = fma_t(-pick<NR>(alpha, c), Ap[i], r[i]);
        r[i] = ri;
        s[c] += (double)ri * (double)ri;
    }
}

// --------------------------------------------------------------------------------------------------
// persistent CG
// --------------------------------------------------------------------------------------------------
template <typename T>
struct CgArgs {
    MatView<T> A;
    const T *b;
    T *x, *r, *p, *p2, *Ap;
    double *partial; // [4][grid][3]
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
__global__ void __launch_bounds__(CM_NT, 2) cg_kernel(CgArgs<T> a)
{
    constexpr int NC = ModeTraits<MODE>::NC, NR = ModeTraits<MODE>::NR, C = ModeTraits<MODE>::C;
    __shared__ double red[6 * 32];
    cg::grid_group grid = cg::this_grid();
    const int tid = threadIdx.x, nt = blockDim.x, nb = gridDim.x, bid = blockIdx.x;
    int u0, u1;
    cta_units(a.A.nslices, bid, nb, u0, u1);
    // own rows [own0, own1) and own entries [e0, e1) of the interleaved vectors
    const int own0 = (int)min((long)u0 * C, a.A.N), own1 = (int)min((long)u1 * C, a.A.N);
    const long e0 = (long)own0 * NC, e1 = (long)own1 * NC;
    auto part = [&](int slot) { return a.partial + ((long)slot * nb + bid) * 3; };
    // component served by this thread in the scalar loops below: e0 % 3 == 0 and nt % 3 == 0, so it is fixed
    const int c = (NR == 3) ? tid % 3 : 0;
    double nodot[3] = {0, 0, 0};

    // ---- r = b - A x0, rr, bb
    spmv_units<T, MODE, false>(a.A, a.x, a.Ap, u0, u1, nodot);
    __syncthreads(); // Ap of the CTA's rows was written by other warps
    {
        double srr = 0, sbb = 0;
        for (long i = e0 + tid; i < e1; i += nt) {
            const T bi = a.b[i], ri = bi - a.Ap[i];
            a.r[i] = ri;
            srr += (double)ri * (double)ri;
            sbb += (double)bi * (double)bi;
        }
        double v[6];
#pragma unroll
        for (int k = 0; k < 3; k++) { v[k] = (k == c) ? srr : 0.0; v[3 + k] = (k == c) ? sbb : 0.0; }
        block_sum<6>(v, red);
        if (tid == 0)
            for (int k = 0; k < 3; k++) { part(2)[k] = v[k]; part(3)[k] = v[3 + k]; }
    }
    grid.sync();
    double rr[NR], bb[NR];
    grid_sum<NR>(a.partial, 2, rr, red);
    grid_sum<NR>(a.partial, 3, bb, red);

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

    // p_0 = r_0: beta = 0 and "p_{-1}" = r (any finite vector)
    T beta[NR];
#pragma unroll
    for (int q = 0; q < NR; q++) beta[q] = 0;
    const T *pold = a.r;
    T *pnew = a.p, *pother = a.p2;
    T aprev[NR]; // alpha of the previous iteration: its x update is applied in the next phase C' (or after the loop)
#pragma unroll
    for (int q = 0; q < NR; q++) aprev[q] = 0;

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
        // ---- C': p_k on the own rows
        phase_p<T, NR>(pnew, pold, a.r, a.x, e0, e1, beta, aprev, k > 0);
        double s_pap[3] = {0, 0, 0};
        grid.sync(); // textbook loop: p_k visible everywhere before the product
        spmv_units<T, MODE, true>(a.A, pnew, a.Ap, u0, u1, s_pap);
        block_sum<3>(s_pap, red);
        if (tid == 0)
            for (int q = 0; q < 3; q++) part(0)[q] = s_pap[q];
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
        // ---- B: r -= alpha Ap, rr_new (alpha = 0 freezes a finished component; x += alpha p is deferred to phase C')
        double snew[3] = {0, 0, 0};
        phase_xr<T, NR>(a.r, a.Ap, e0, e1, alpha, snew);
        block_sum<3>(snew, red);
        if (tid == 0)
            for (int q = 0; q < 3; q++) part(1)[q] = snew[q];
        grid.sync();
        double rr_new[NR];
        grid_sum<NR>(a.partial, 1, rr_new, red);
#pragma unroll
        for (int q = 0; q < NR; q++) {
            beta[q] = active[q] ? (T)(rr_new[q] / rr[q]) : (T)0;
            if (active[q]) { rr[q] = rr_new[q]; iters[q]++; }
            aprev[q] = alpha[q];
        }
        // rotate the p buffers: p_k becomes p_{k-1}
        T *t = (pold == a.r) ? pother : const_cast<T *>(pold);
        pold = pnew;
        pnew = t;
    }
    {
        bool pending = false;
#pragma unroll
        for (int q = 0; q < NR; q++) pending |= aprev[q] != (T)0;
        if (pending) phase_x_final<T, NR>(a.x, pold, e0, e1, aprev);
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
    const Sell &L = S->mesh->sell[mode == MODE_BSR3 ? 1 : 0];
    A->sp = L.d_sp; A->col = L.d_col; A->val = v;
    A->nslices = L.nslices; A->N = S->N;
    return CM_OK;
}

template <typename T, int MODE>
static int launch_spmv(System<T> *S, const MatView<T> &A, const T *x, T *y, cudaStream_t st)
{
    int occ = 0;
    CM_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, spmv_kernel<T, MODE>, CM_NT, 0));
    int grid = std::max(1, std::min(A.nslices, occ * S->num_sms));
    S->prof.begin(CM_PROF_SPMV, st);
    spmv_kernel<T, MODE><<<grid, CM_NT, 0, st>>>(A, x, y);
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
    CM_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, cg_kernel<T, MODE>, CM_NT, 0));
    if (occ < 1) { cm_set_error("cg kernel does not fit on an SM"); return CM_E_CUDA; }
    int grid = std::max(1, std::min({a.A.nslices, occ * S->num_sms, S->grid_cap}));
    void *args[] = {&a};
    S->prof.begin(prof_cls, st);
    cudaError_t e = cudaLaunchCooperativeKernel((void *)cg_kernel<T, MODE>, dim3(grid), dim3(CM_NT), args, 0, st);
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
    a.b = b; a.x = x; a.r = S->r; a.p = S->p; a.p2 = S->p2; a.Ap = S->Ap; a.partial = S->partial;
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
