// S4 / S7 / S10: sparse matrix-vector products and the fused, persistent conjugate-gradient solver
// (O-4), unpreconditioned as the paper runs it or Jacobi-preconditioned (the paper's future work).
//
// Layout.  Matrices are stored sliced (SELL-C, cm_internal.h): C consecutive rows form a slice, padded to the
// slice's longest row and stored column-major, so that the 32 lanes of a warp read 32 consecutive elements of
// every array.  The 3x3-block elasticity matrix keeps its 9 block entries in 9 planes per slice
// ([slice][3r + c][L_slice]): each plane is one coalesced stream.
//
// SpMV.  One warp per slice, all 32 lanes busy: lane -> (row i % C of the slice, column phase lane / C).  A lane
// streams its elements (value(s) + column index, U iterations in flight, L1 bypassed, L2 evict-first), gathers
// x[col] (L1 / L2 hits thanks to the locality ordering) and accumulates in registers in column order; the
// 32 / C column phases of a row are combined with a fixed shuffle butterfly.  No shared memory, no atomics.
// The three-right-hand-side product (MODE_CSR3) gathers its vector from a PADDED copy, four words per node: one
// aligned 32-byte (fp64: ld.global.v4.f64, a 256-bit load) or 16-byte (fp32) request per nonzero touches exactly
// one sector, where three scalar gathers from [node][3] cost three requests and ~2.4 sectors (the L1 bound
// measured in round 1, a round-1 ncu capture).
//
// CG.  ONE cooperative launch per solve; a CTA owns a contiguous range of slices, hence of rows, for the whole
// solve.  Per iteration k (three grid-wide barriers, the dot products ride on two of them):
//   C   x += alpha_{k-1} p_{k-1} (deferred: p_{k-1} is read here anyway), p_k = z_k + beta p_{k-1} on the own rows;  -> barrier
//   A   Ap = A p_k, dot p.Ap;                                                              -> barrier, alpha
//   B   r -= alpha Ap, dots r.r (stopping test) and r.z;                                   -> barrier, beta
// with z = r (plain CG) or z = r / diag(A) (Jacobi).  Every CTA reduces the per-CTA partial sums in the same fixed
// order, so all CTAs take the same decisions and the result is bit-reproducible run to run.  Dot products
// accumulate in fp64 in both precisions (R20).
// A Helmholtz solve of the GSPM step (Alg. B.1 Steps 1 and 3: (M_m + eps K_m) g = M_m f from x0 = f) is
// one launch: its first pass streams both value arrays on the shared pattern, forms b = M_m f and A f in
// registers, writes r0 = b - A f and x0 = f and sums |b|^2 -- no separate mass product, no copy of f.
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

// ---- one padded node (four words, the fourth unused): a single aligned vector access
__device__ __forceinline__ void ld_node4(const double *p, double (&o)[3])
{
    double w;
    asm volatile("ld.global.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(o[0]), "=d"(o[1]), "=d"(o[2]), "=d"(w) : "l"(p));
}
__device__ __forceinline__ void ld_node4(const float *p, float (&o)[3])
{
    const float4 v = *reinterpret_cast<const float4 *>(p);
    o[0] = v.x; o[1] = v.y; o[2] = v.z;
}
__device__ __forceinline__ void st_node4(double *p, const double (&v)[3])
{
    asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(p), "d"(v[0]), "d"(v[1]), "d"(v[2]), "d"(0.0) : "memory");
}
__device__ __forceinline__ void st_node4(float *p, const float (&v)[3]) { *reinterpret_cast<float4 *>(p) = make_float4(v[0], v[1], v[2], 0.f); }

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

// x[col] for all NC components of a node; XS = words per node of x in memory (NC, or 4 for the padded 3-vector)
template <typename T, int NC, int XS>
__device__ __forceinline__ void fetch(const T *x, int col, T (&out)[NC])
{
    if (NC == 3 && XS == 4) {
        T v[3];
        ld_node4(x + 4L * col, v);
#pragma unroll
        for (int c = 0; c < NC; c++) out[c] = v[c < 3 ? c : 0];
    } else {
        const long o = (long)col * XS;
#pragma unroll
        for (int c = 0; c < NC; c++) out[c] = x[o + c];
    }
}

// Batches in flight per warp.  The fp32 block matrix streams half the bytes per element, so it takes twice the batches
// (measured on B200, config 3 fp32: mechanical CG 88 % -> 94 % of the measured HBM peak with 4 instead of 2).
#ifndef CM_F32_CSR3_CTAS
#define CM_F32_CSR3_CTAS 2 // resident CTAs per SM asked for the fp32 three-right-hand-side CG (3: 56 registers; measured)
#endif
#ifndef CM_U_CSR3_F32
#define CM_U_CSR3_F32 CM_U_CSR3
#endif
#ifndef CM_U_BSR3_F32
#define CM_U_BSR3_F32 4
#endif
template <typename T, int MODE>
constexpr int batch_u() { return (MODE == MODE_BSR3 && sizeof(T) == 4) ? CM_U_BSR3_F32 : ((MODE == MODE_CSR3 && sizeof(T) == 4) ? CM_U_CSR3_F32 : ModeTraits<MODE>::U); }

// One batch = U consecutive 32-element groups of one slice: the unit of the load pipeline.  NV2 = 2: a second
// scalar value array on the same pattern (the Helmholtz first pass streams K^GS and M_m together).
template <typename T, int MODE, int NV2 = 1>
struct Batch {
    int col[batch_u<T, MODE>()];
    T v[batch_u<T, MODE>()][ModeTraits<MODE>::NV * NV2];
};

// position in the stream of batches of a warp: slice s with extent [b0, b0 + L), batch offset it
struct Cursor {
    int s, b0, L, it;
};

template <typename T, int MODE, int NV2>
__device__ __forceinline__ void load_batch(const MatView<T> &A, const T *val2, const Cursor &c, int lane, unsigned long long pol,
                                           Batch<T, MODE, NV2> &B)
{
    constexpr int NV = ModeTraits<MODE>::NV, U = batch_u<T, MODE>();
    const int *colp = A.col + c.b0;
    const T *valp = A.val + (long)NV * c.b0; // plane k at valp + k * L
#pragma unroll
    for (int u = 0; u < U; u++) {
        const int e = c.it + 32 * u + lane;
        B.col[u] = 0;
#pragma unroll
        for (int k = 0; k < NV * NV2; k++) B.v[u][k] = 0;
        if (e < c.L) {
            B.col[u] = ld_stream(colp + e, pol);
#pragma unroll
            for (int k = 0; k < NV; k++) B.v[u][k] = ld_stream(valp + (long)k * c.L + e, pol);
            if (NV2 == 2) B.v[u][NV] = ld_stream(val2 + c.b0 + e, pol);
        }
    }
}

// What a warp does with a finished row of the product.
//   SpmvStore: y = A x, optionally dot[c] += y.x over the rows written (x valid on those rows).
template <typename T, int MODE, int XS, bool DOT>
struct SpmvStore {
    T *y;
    const T *x;
    __device__ __forceinline__ void row(long row, int jl, const T (&acc)[ModeTraits<MODE>::NC], const T (&)[ModeTraits<MODE>::NC], double (&dot)[9]) const
    {
        constexpr int NC = ModeTraits<MODE>::NC;
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
                if (DOT) dot[c] += (double)acc[c] * (double)x[(long)XS * row + c];
            }
        }
    }
};
//   HelmStore (MODE_CSR3, two value arrays): acc = A f, acc2 = M f = b;  r0 = b - A f, x0 = f on the masked
//   components, dot[0..2] += r0^2, dot[3..5] += b^2, dot[6..8] += r0 z0 (Jacobi).
template <typename T, bool PRE>
struct HelmStore {
    T *r, *x;
    const T *f4, *diag;
    unsigned mask;
    __device__ __forceinline__ void row(long row, int jl, const T (&acc)[3], const T (&acc2)[3], double (&dot)[9]) const
    {
        if (jl != 0) return;
        T fv[3];
        ld_node4(f4 + 4 * row, fv);
        T d = 1;
        if (PRE) d = diag[row];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const T bi = acc2[c], ri = bi - acc[c];
            r[3 * row + c] = ri;
            if ((mask >> c) & 1u) x[3 * row + c] = fv[c];
            dot[c] += (double)ri * (double)ri;
            dot[3 + c] += (double)bi * (double)bi;
            if (PRE) dot[6 + c] += (double)ri * (double)(ri / d);
        }
    }
};

// The product on the slices [u0, u1) of this CTA (warp w takes u0 + w, u0 + w + nwarps, ...).
template <typename T, int MODE, int XS, int NV2, typename STORE>
__device__ __forceinline__ void spmv_units(const MatView<T> &A, const T *val2, const T *x, const STORE &st, int u0, int u1, double (&dot)[9])
{
    constexpr int NC = ModeTraits<MODE>::NC, C = ModeTraits<MODE>::C, U = batch_u<T, MODE>(), NV = ModeTraits<MODE>::NV;
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
    Batch<T, MODE, NV2> Bc;
    load_batch<T, MODE, NV2>(A, val2, cur, lane, pol, Bc);
    T acc[NC], acc2[NC];
#pragma unroll
    for (int c = 0; c < NC; c++) { acc[c] = 0; acc2[c] = 0; }
    for (;;) {
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
                fetch<T, NC, XS>(x, Bc.col[u], xv);
                if (MODE == MODE_BSR3) {
                    acc[0] += Bc.v[u][0] * xv[0] + Bc.v[u][1] * xv[1] + Bc.v[u][2] * xv[2];
                    acc[1] += Bc.v[u][3] * xv[0] + Bc.v[u][4] * xv[1] + Bc.v[u][5] * xv[2];
                    acc[2] += Bc.v[u][6] * xv[0] + Bc.v[u][7] * xv[1] + Bc.v[u][8] * xv[2];
                } else {
#pragma unroll
                    for (int c = 0; c < NC; c++) acc[c] += Bc.v[u][0] * xv[c];
                    if (NV2 == 2)
#pragma unroll
                        for (int c = 0; c < NC; c++) acc2[c] += Bc.v[u][NV] * xv[c];
                }
            }
        }
        if (last_of_slice) {
            // combine the 32 / C column phases of each row (fixed butterfly: every lane ends with the same sum)
#pragma unroll
            for (int o = C; o < 32; o <<= 1)
#pragma unroll
                for (int c = 0; c < NC; c++) {
                    acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
                    if (NV2 == 2) acc2[c] += __shfl_xor_sync(0xffffffffu, acc2[c], o);
                }
            const long row = (long)cur.s * C + rl;
            if (row < A.N) st.row(row, jl, acc, acc2, dot);
#pragma unroll
            for (int c = 0; c < NC; c++) { acc[c] = 0; acc2[c] = 0; }
        }
        if (!more) break;
        cur = nxt;
        load_batch<T, MODE, NV2>(A, val2, cur, lane, pol, Bc);
    }
}

// standalone product; the 3-vector of MODE_CSR3 is read from a padded copy (four words per node)
template <typename T, int MODE>
__global__ void __launch_bounds__(CM_NT, 2) spmv_kernel(MatView<T> A, const T *x, T *y)
{
    constexpr int XS = MODE == MODE_CSR3 ? 4 : ModeTraits<MODE>::NC;
    int u0, u1;
    cta_units(A.nslices, blockIdx.x, gridDim.x, u0, u1);
    double dot[9];
    SpmvStore<T, MODE, XS, false> st{y, x};
    spmv_units<T, MODE, XS, 1>(A, (const T *)nullptr, x, st, u0, u1, dot);
}

// --------------------------------------------------------------------------------------------------
// streaming vector phases of CG, one right-hand side (MODE_CSR1, MODE_BSR3): 128-bit accesses over the CTA's own
// entries [e0, e1): a 16-byte aligned vector body (e0 is a multiple of 8 entries because slices hold 8 or 16 rows)
// plus a scalar tail
// --------------------------------------------------------------------------------------------------
template <typename T> struct VecOf;
template <> struct VecOf<double> { typedef double2 V; static constexpr int W = 2; };
template <> struct VecOf<float> { typedef float4 V; static constexpr int W = 4; };

__device__ __forceinline__ double2 vfma(double c, double2 a, double2 b) { return make_double2(fma(c, a.x, b.x), fma(c, a.y, b.y)); }
__device__ __forceinline__ float4 vfma(float c, float4 a, float4 b)
{
    return make_float4(fmaf(c, a.x, b.x), fmaf(c, a.y, b.y), fmaf(c, a.z, b.z), fmaf(c, a.w, b.w));
}
__device__ __forceinline__ double2 vdiv(double2 a, double2 d) { return make_double2(a.x / d.x, a.y / d.y); }
__device__ __forceinline__ float4 vdiv(float4 a, float4 d) { return make_float4(a.x / d.x, a.y / d.y, a.z / d.z, a.w / d.w); }
// acc += sum_j a[j] b[j] in fp64
__device__ __forceinline__ void vdot(double &acc, double2 a, double2 b) { acc += a.x * b.x; acc += a.y * b.y; }
__device__ __forceinline__ void vdot(double &acc, float4 a, float4 b)
{
    acc += (double)a.x * (double)b.x; acc += (double)a.y * (double)b.y; acc += (double)a.z * (double)b.z; acc += (double)a.w * (double)b.w;
}

// C': x += alpha_prev pold (the x update of the PREVIOUS iteration, deferred to here because pold is read anyway: one
// vector stream less per iteration than updating x in phase B; the fma is the same, so x is bit-identical), then
// pnew = z + beta pold with z = r or r / diag
template <typename T, bool PRE>
__device__ __forceinline__ void phase_p(T *pnew, const T *pold, const T *r, T *x, const T *diag, long e0, long e1, T beta, T aprev, bool upd_x)
{
    constexpr int W = VecOf<T>::W, UN = 2;
    typedef typename VecOf<T>::V V;
    const int tid = threadIdx.x, nt = blockDim.x;
    const long a1 = e0 + (e1 - e0) / W * W, nv = (a1 - e0) / W;
    V *pn = reinterpret_cast<V *>(pnew + e0), *xv = reinterpret_cast<V *>(x + e0);
    const V *po = reinterpret_cast<const V *>(pold + e0), *rv = reinterpret_cast<const V *>(r + e0);
    const V *dv = PRE ? reinterpret_cast<const V *>(diag + e0) : nullptr;
    long v = tid;
    for (; v + (long)(UN - 1) * nt < nv; v += (long)nt * UN) {
        V a[UN], b[UN], c[UN], d[UN];
#pragma unroll
        for (int q = 0; q < UN; q++) {
            a[q] = po[v + (long)q * nt]; b[q] = rv[v + (long)q * nt];
            if (upd_x) c[q] = xv[v + (long)q * nt];
            if (PRE) d[q] = dv[v + (long)q * nt];
        }
#pragma unroll
        for (int q = 0; q < UN; q++) {
            if (upd_x) xv[v + (long)q * nt] = vfma(aprev, a[q], c[q]);
            pn[v + (long)q * nt] = vfma(beta, a[q], PRE ? vdiv(b[q], d[q]) : b[q]);
        }
    }
    for (; v < nv; v += nt) {
        const V a = po[v];
        if (upd_x) xv[v] = vfma(aprev, a, xv[v]);
        pn[v] = vfma(beta, a, PRE ? vdiv(rv[v], dv[v]) : rv[v]);
    }
    for (long i = a1 + tid; i < e1; i += nt) {
        const T pv = pold[i];
        if (upd_x) x[i] = fma_t(aprev, pv, x[i]);
        pnew[i] = fma_t(beta, pv, PRE ? r[i] / diag[i] : r[i]);
    }
}

// B: r -= alpha Ap; srr += sum r_new^2, srz += sum r_new z_new
template <typename T, bool PRE>
__device__ __forceinline__ void phase_r(T *r, const T *Ap, const T *diag, long e0, long e1, T alpha, double &srr, double &srz)
{
    constexpr int W = VecOf<T>::W, UN = 4;
    typedef typename VecOf<T>::V V;
    const int tid = threadIdx.x, nt = blockDim.x;
    const long a1 = e0 + (e1 - e0) / W * W, nv = (a1 - e0) / W;
    V *rv = reinterpret_cast<V *>(r + e0);
    const V *av = reinterpret_cast<const V *>(Ap + e0), *dv = PRE ? reinterpret_cast<const V *>(diag + e0) : nullptr;
    long v = tid;
    for (; v + (long)(UN - 1) * nt < nv; v += (long)nt * UN) {
        V b[UN], d[UN], g[UN];
#pragma unroll
        for (int q = 0; q < UN; q++) {
            b[q] = av[v + (long)q * nt]; d[q] = rv[v + (long)q * nt];
            if (PRE) g[q] = dv[v + (long)q * nt];
        }
#pragma unroll
        for (int q = 0; q < UN; q++) {
            const V rn = vfma(-alpha, b[q], d[q]);
            rv[v + (long)q * nt] = rn;
            vdot(srr, rn, rn);
            if (PRE) vdot(srz, rn, vdiv(rn, g[q]));
        }
    }
    for (; v < nv; v += nt) {
        const V rn = vfma(-alpha, av[v], rv[v]);
        rv[v] = rn;
        vdot(srr, rn, rn);
        if (PRE) vdot(srz, rn, vdiv(rn, dv[v]));
    }
    for (long i = a1 + tid; i < e1; i += nt) {
        const T ri = fma_t(-alpha, Ap[i], r[i]);
        r[i] = ri;
        srr += (double)ri * (double)ri;
        if (PRE) srz += (double)ri * (double)(ri / diag[i]);
    }
}

// --------------------------------------------------------------------------------------------------
// vector phases of the three-right-hand-side CG (MODE_CSR3): one thread per node of the own range [n0, n1); r, x, Ap
// are [node][3], the search directions are padded [node][4] (they are what the product gathers); diag has one
// entry per node (the three systems share the matrix)
// --------------------------------------------------------------------------------------------------
// G = 128 bits / sizeof(T) nodes per thread: the 3 G words of a [node][3] array are three aligned 128-bit accesses, the 4 G
// words of a padded array four, G diagonal entries one; every load of a group is issued before the first use (13 in flight)
template <typename T>
__device__ __forceinline__ void ldv(const T *p, T *out, int nvec)
{
    typedef typename VecOf<T>::V V;
    constexpr int W = VecOf<T>::W;
    for (int q = 0; q < nvec; q++) *reinterpret_cast<V *>(out + W * q) = reinterpret_cast<const V *>(p)[q];
}
template <typename T>
__device__ __forceinline__ void stv(T *p, const T *in, int nvec)
{
    typedef typename VecOf<T>::V V;
    constexpr int W = VecOf<T>::W;
    for (int q = 0; q < nvec; q++) reinterpret_cast<V *>(p)[q] = *reinterpret_cast<const V *>(in + W * q);
}

template <typename T, bool PRE>
__device__ __forceinline__ void phase_p3(T *pnew4, const T *pold4, const T *r, T *x, const T *diag, int n0, int n1, const T (&beta)[3],
                                         const T (&aprev)[3], bool first)
{
    constexpr int G = VecOf<T>::W;
    // fp32 only: in fp64 the group's 20 live doubles do not fit beside the solver's state in 80 registers (measured with the
    // spills: 3-iteration solve 1.03 -> 1.18 ms at 144^3; fp32: 0.70 -> 0.66 ms)
    const int ng = sizeof(T) == 4 ? (n1 - n0) / G : 0; // n0 is a multiple of the slice height
    if constexpr (sizeof(T) == 4)
    for (int g = threadIdx.x; g < ng; g += blockDim.x) {
        const long i0 = n0 + (long)g * G;
        __align__(16) T rv[3 * G], xv[3 * G], po[4 * G], dv[G]; // po becomes the new p in place
#pragma unroll
        for (int q = 0; q < 3; q++) ldv(r + 3 * i0 + q * G, rv + q * G, 1);
        if (!first) {
#pragma unroll
            for (int q = 0; q < 3; q++) ldv(x + 3 * i0 + q * G, xv + q * G, 1);
#pragma unroll
            for (int q = 0; q < 4; q++) ldv(pold4 + 4 * i0 + q * G, po + q * G, 1);
        }
        if (PRE) ldv(diag + i0, dv, 1);
#pragma unroll
        for (int j = 0; j < 3 * G; j++) {
            const int q = j / 3, c = j % 3;
            T z = PRE ? rv[j] / dv[q] : rv[j];
            if (!first) {
                xv[j] = fma_t(aprev[c], po[4 * q + c], xv[j]);
                z = fma_t(beta[c], po[4 * q + c], z);
            }
            po[4 * q + c] = z;
        }
#pragma unroll
        for (int q = 0; q < G; q++) po[4 * q + 3] = 0;
        if (!first)
#pragma unroll
            for (int q = 0; q < 3; q++) stv(x + 3 * i0 + q * G, xv + q * G, 1);
#pragma unroll
        for (int q = 0; q < 4; q++) stv(pnew4 + 4 * i0 + q * G, po + q * G, 1);
    }
    for (int i = n0 + ng * G + threadIdx.x; i < n1; i += blockDim.x) {
        T z[3] = {r[3L * i], r[3L * i + 1], r[3L * i + 2]};
        if (PRE) {
            const T d = diag[i];
#pragma unroll
            for (int c = 0; c < 3; c++) z[c] = z[c] / d;
        }
        if (!first) {
            T po[3];
            ld_node4(pold4 + 4L * i, po);
#pragma unroll
            for (int c = 0; c < 3; c++) {
                x[3L * i + c] = fma_t(aprev[c], po[c], x[3L * i + c]);
                z[c] = fma_t(beta[c], po[c], z[c]);
            }
        }
        st_node4(pnew4 + 4L * i, z);
    }
}

template <typename T, bool PRE>
__device__ __forceinline__ void phase_r3(T *r, const T *Ap, const T *diag, int n0, int n1, const T (&alpha)[3], double (&srr)[3], double (&srz)[3])
{
    constexpr int G = VecOf<T>::W;
    const int ng = sizeof(T) == 4 ? (n1 - n0) / G : 0; // fp32 only, as in phase_p3
    if constexpr (sizeof(T) == 4)
    for (int g = threadIdx.x; g < ng; g += blockDim.x) {
        const long i0 = n0 + (long)g * G;
        __align__(16) T rv[3 * G], av[3 * G], dv[G];
#pragma unroll
        for (int q = 0; q < 3; q++) { ldv(r + 3 * i0 + q * G, rv + q * G, 1); ldv(Ap + 3 * i0 + q * G, av + q * G, 1); }
        if (PRE) ldv(diag + i0, dv, 1);
#pragma unroll
        for (int j = 0; j < 3 * G; j++) {
            const int q = j / 3, c = j % 3;
            const T ri = fma_t(-alpha[c], av[j], rv[j]);
            rv[j] = ri;
            srr[c] += (double)ri * (double)ri;
            if (PRE) srz[c] += (double)ri * (double)(ri / dv[q]);
        }
#pragma unroll
        for (int q = 0; q < 3; q++) stv(r + 3 * i0 + q * G, rv + q * G, 1);
    }
    for (int i = n0 + ng * G + threadIdx.x; i < n1; i += blockDim.x) {
        T d = 1;
        if (PRE) d = diag[i];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const T ri = fma_t(-alpha[c], Ap[3L * i + c], r[3L * i + c]);
            r[3L * i + c] = ri;
            srr[c] += (double)ri * (double)ri;
            if (PRE) srz[c] += (double)ri * (double)(ri / d);
        }
    }
}

// --------------------------------------------------------------------------------------------------
// persistent CG
// --------------------------------------------------------------------------------------------------
template <typename T>
struct CgArgs {
    MatView<T> A;
    const T *Mval;   // HELM: values of M_m on the same sliced pattern
    const T *f4;     // HELM: f, padded [node][4]; right-hand side b = M_m f, start vector x0 = f
    const T *b;      // otherwise: right-hand side
    T *x, *r, *p, *p2, *Ap; // MODE_CSR3: p, p2 are padded [node][4]
    const T *diag;   // PRE: diag(A), N (scalar matrices) or 3N (block matrix) entries
    double *partial; // [5][grid][3]
    double tol;
    int maxiter, fixed;
    unsigned mask;
    CgResult *out;
    double *hist;    // optional: hist[k NR + q] = ||r_k|| / ||b|| of right-hand side q before iteration k
    int hist_cap;
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

// (three resident CTAs for the fp32 scalar solve, which fits 56 registers: 81 % -> 87 % of the measured HBM peak at 144^3)
template <typename T, int MODE, bool PRE, bool HELM>
__global__ void __launch_bounds__(CM_NT, (sizeof(T) == 4 && ((MODE == MODE_CSR1 && !PRE) || (MODE == MODE_CSR3 && !PRE && CM_F32_CSR3_CTAS == 3))) ? 3 : 2) cg_kernel(CgArgs<T> a)
{
    constexpr int NC = ModeTraits<MODE>::NC, NR = ModeTraits<MODE>::NR, C = ModeTraits<MODE>::C;
    constexpr int PS = MODE == MODE_CSR3 ? 4 : NC; // words per node of the search directions in memory
    static_assert(!HELM || MODE == MODE_CSR3, "the fused Helmholtz start is a three-right-hand-side solve");
    __shared__ double red[9 * 32];
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

    // ---- r0 = b - A x0, rr, bb, rz
    {
        double v[9];
#pragma unroll
        for (int k = 0; k < 9; k++) v[k] = 0;
        if constexpr (HELM) {
            HelmStore<T, PRE> st{a.r, a.x, a.f4, a.diag, a.mask};
            spmv_units<T, MODE, 4, 2>(a.A, a.Mval, a.f4, st, u0, u1, v);
        } else {
            double nodot[9];
            SpmvStore<T, MODE, NC, false> st{a.Ap, a.x};
            spmv_units<T, MODE, NC, 1>(a.A, (const T *)nullptr, a.x, st, u0, u1, nodot);
            __syncthreads(); // Ap of the CTA's rows was written by other warps
            double srr = 0, sbb = 0, srz = 0;
            for (long i = e0 + tid; i < e1; i += nt) {
                const T bi = a.b[i], ri = bi - a.Ap[i];
                a.r[i] = ri;
                srr += (double)ri * (double)ri;
                sbb += (double)bi * (double)bi;
                if (PRE) srz += (double)ri * (double)(ri / a.diag[NR == 3 ? i / 3 : i]);
            }
#pragma unroll
            for (int k = 0; k < 3; k++) { v[k] = (k == c) ? srr : 0.0; v[3 + k] = (k == c) ? sbb : 0.0; v[6 + k] = (k == c) ? srz : 0.0; }
        }
        block_sum<9>(v, red);
        if (tid == 0)
            for (int k = 0; k < 3; k++) { part(2)[k] = v[k]; part(3)[k] = v[3 + k]; part(4)[k] = v[6 + k]; }
    }
    grid.sync();
    double rr[NR], bb[NR], rz[NR];
    grid_sum<NR>(a.partial, 2, rr, red);
    grid_sum<NR>(a.partial, 3, bb, red);
    if (PRE) grid_sum<NR>(a.partial, 4, rz, red);
    else
#pragma unroll
        for (int q = 0; q < NR; q++) rz[q] = rr[q];

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
    {
        bool zc = false;
#pragma unroll
        for (int q = 0; q < NR; q++) zc |= (q == c) && zero_rhs[q];
        if (zc)
            for (long i = e0 + tid; i < e1; i += nt) a.x[i] = 0;
    }

    // p_0 = z_0: beta = 0 and "p_{-1}" = r (any finite vector) for the one-right-hand-side modes; the
    // three-right-hand-side mode writes its first padded p from z directly
    T beta[NR], aprev[NR]; // aprev: alpha of the previous iteration, its x update is applied in the next phase C' (or after the loop)
#pragma unroll
    for (int q = 0; q < NR; q++) { beta[q] = 0; aprev[q] = 0; }
    const T *pold = (MODE == MODE_CSR3) ? a.p2 : a.r;
    T *pnew = a.p, *pother = a.p2;

    for (int k = 0;; k++) {
        if (a.hist && bid == 0 && tid == 0 && (long)(k + 1) * NR <= a.hist_cap)
#pragma unroll
            for (int q = 0; q < NR; q++) a.hist[(long)k * NR + q] = bb[q] > 0 ? sqrt(rr[q] / bb[q]) : 0.0;
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
        if (MODE == MODE_CSR3) {
            T be3[3], ap3[3];
#pragma unroll
            for (int q = 0; q < 3; q++) { be3[q] = beta[q < NR ? q : 0]; ap3[q] = aprev[q < NR ? q : 0]; }
            phase_p3<T, PRE>(pnew, pold, a.r, a.x, a.diag, own0, own1, be3, ap3, k == 0);
        } else {
            phase_p<T, PRE>(pnew, pold, a.r, a.x, a.diag, e0, e1, beta[0], aprev[0], k > 0);
        }
        grid.sync(); // textbook loop: p_k visible everywhere before the product
        // ---- A: Ap = A p_k, pAp
        double s_pap[9];
#pragma unroll
        for (int q = 0; q < 9; q++) s_pap[q] = 0;
        {
            SpmvStore<T, MODE, PS, true> st{a.Ap, pnew};
            spmv_units<T, MODE, PS, 1>(a.A, (const T *)nullptr, pnew, st, u0, u1, s_pap);
        }
        double s3[3] = {s_pap[0], s_pap[1], s_pap[2]};
        block_sum<3>(s3, red);
        if (tid == 0)
            for (int q = 0; q < 3; q++) part(0)[q] = s3[q];
        grid.sync();
        double pap[NR];
        grid_sum<NR>(a.partial, 0, pap, red);
        T alpha[NR];
#pragma unroll
        for (int q = 0; q < NR; q++) {
            alpha[q] = 0;
            if (!active[q]) continue;
            if (!(pap[q] > 0.0)) { active[q] = false; status = CM_E_CG_BREAKDOWN; continue; }
            alpha[q] = (T)(rz[q] / pap[q]);
        }
        // ---- B: r -= alpha Ap, rr_new, rz_new (alpha = 0 freezes a finished component; x += alpha p is deferred to phase C')
        double snew[6] = {0, 0, 0, 0, 0, 0};
        if (MODE == MODE_CSR3) {
            T al3[3];
#pragma unroll
            for (int q = 0; q < 3; q++) al3[q] = alpha[q < NR ? q : 0];
            double srr[3] = {0, 0, 0}, srz[3] = {0, 0, 0};
            phase_r3<T, PRE>(a.r, a.Ap, a.diag, own0, own1, al3, srr, srz);
#pragma unroll
            for (int q = 0; q < 3; q++) { snew[q] = srr[q]; snew[3 + q] = srz[q]; }
        } else {
            phase_r<T, PRE>(a.r, a.Ap, a.diag, e0, e1, alpha[0], snew[0], snew[3]);
        }
        block_sum<6>(snew, red);
        if (tid == 0)
            for (int q = 0; q < 3; q++) { part(1)[q] = snew[q]; part(4)[q] = snew[3 + q]; }
        grid.sync();
        double rr_new[NR], rz_new[NR];
        grid_sum<NR>(a.partial, 1, rr_new, red);
        if (PRE) grid_sum<NR>(a.partial, 4, rz_new, red);
        else
#pragma unroll
            for (int q = 0; q < NR; q++) rz_new[q] = rr_new[q];
#pragma unroll
        for (int q = 0; q < NR; q++) {
            beta[q] = active[q] ? (T)(rz_new[q] / rz[q]) : (T)0;
            if (active[q]) { rr[q] = rr_new[q]; rz[q] = rz_new[q]; iters[q]++; }
            aprev[q] = alpha[q];
        }
        // rotate the p buffers: p_k becomes p_{k-1}
        T *t = (pold == a.r) ? pother : const_cast<T *>(pold);
        pold = pnew;
        pnew = t;
    }
    {
        // the x update still pending when the loop ends: x += alpha_last p_last
        bool pending = false;
#pragma unroll
        for (int q = 0; q < NR; q++) pending |= aprev[q] != (T)0;
        if (pending) {
            if (MODE == MODE_CSR3) {
                for (int i = own0 + tid; i < own1; i += nt) {
                    T po[3];
                    ld_node4(pold + 4L * i, po);
#pragma unroll
                    for (int q = 0; q < 3; q++) a.x[3L * i + q] = fma_t(aprev[q < NR ? q : 0], po[q], a.x[3L * i + q]);
                }
            } else {
                for (long i = e0 + tid; i < e1; i += nt) a.x[i] = fma_t(aprev[0], pold[i], a.x[i]);
            }
        }
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
static const T *mat_diag(const System<T> *S, cm_matrix_id id)
{
    switch (id) {
    case CM_MAT_K_MS: return S->Dms;
    case CM_MAT_K_GS1: return S->Dgs1;
    case CM_MAT_K_GS2: return S->Dgs2;
    case CM_MAT_MASS: return nullptr; // singular on dead nodes: never solved with
    case CM_MAT_K_MECH: return S->Dmech;
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

// x: N (MODE_CSR1), N x 3 (MODE_BSR3) or the PADDED N x 4 copy of a 3-vector (MODE_CSR3)
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

template <typename T, int MODE, bool PRE, bool HELM>
static int launch_cg(System<T> *S, CgArgs<T> &a, int prof_cls, cudaStream_t st)
{
    int occ = 0;
    CM_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, cg_kernel<T, MODE, PRE, HELM>, CM_NT, 0));
    if (occ < 1) { cm_set_error("cg kernel does not fit on an SM"); return CM_E_CUDA; }
    int grid = std::max(1, std::min({a.A.nslices, occ * S->num_sms, S->grid_cap}));
    void *args[] = {&a};
    S->prof.begin(prof_cls, st);
    cudaError_t e = cudaLaunchCooperativeKernel((void *)cg_kernel<T, MODE, PRE, HELM>, dim3(grid), dim3(CM_NT), args, 0, st);
    S->prof.end(st);
    if (e != cudaSuccess) { cm_set_error("cudaLaunchCooperativeKernel: %s", cudaGetErrorString(e)); return CM_E_CUDA; }
    return CM_OK;
}

template <typename T>
static int fill_args(System<T> *S, cm_matrix_id id, int mode, T *x, double tol, int maxiter, int fixed, unsigned mask, int slot, int precond,
                     CgArgs<T> *a)
{
    CM_TRY(make_view(S, id, mode, &a->A));
    if (precond != CM_PC_NONE && precond != CM_PC_JACOBI) { cm_set_error("unknown preconditioner %d", precond); return CM_E_BADARG; }
    a->Mval = nullptr; a->f4 = nullptr; a->b = nullptr;
    a->x = x; a->r = S->r; a->p = S->p; a->p2 = S->p2; a->Ap = S->Ap; a->partial = S->partial;
    a->diag = precond == CM_PC_JACOBI ? mat_diag(S, id) : nullptr;
    if (precond == CM_PC_JACOBI && !a->diag) { cm_set_error("matrix %d has no Jacobi preconditioner", (int)id); return CM_E_BADARG; }
    a->tol = tol; a->maxiter = maxiter; a->fixed = fixed; a->mask = mask; a->out = S->d_res + slot;
    a->hist = S->hist_on ? S->d_hist : nullptr; a->hist_cap = S->hist_on ? CM_HIST_CAP : 0;
    return CM_OK;
}

// Enqueue one CG solve; the result lands in S->d_res[slot].
template <typename T>
int sys_cg(System<T> *S, cm_matrix_id id, int mode, const T *b, T *x, double tol, int maxiter, int fixed, unsigned mask, int slot,
           int prof_cls, int precond, cudaStream_t st)
{
    CgArgs<T> a;
    CM_TRY(fill_args(S, id, mode, x, tol, maxiter, fixed, mask, slot, precond, &a));
    a.b = b;
    const bool pre = precond == CM_PC_JACOBI;
    switch (mode) {
    case MODE_CSR1: return pre ? launch_cg<T, MODE_CSR1, true, false>(S, a, prof_cls, st) : launch_cg<T, MODE_CSR1, false, false>(S, a, prof_cls, st);
    case MODE_CSR3: return pre ? launch_cg<T, MODE_CSR3, true, false>(S, a, prof_cls, st) : launch_cg<T, MODE_CSR3, false, false>(S, a, prof_cls, st);
    case MODE_BSR3: return pre ? launch_cg<T, MODE_BSR3, true, false>(S, a, prof_cls, st) : launch_cg<T, MODE_BSR3, false, false>(S, a, prof_cls, st);
    }
    return CM_E_BADARG;
}

// Helmholtz solve of Alg. B.1: (M_m + eps K_m) x = M_m f from x0 = f, three components, one launch.
// f4: f padded [node][4]; x: [node][3], written for the components in `mask` only.
template <typename T>
int sys_helmholtz(System<T> *S, cm_matrix_id id, const T *f4, T *x, double tol, int maxiter, int fixed, unsigned mask, int slot, int precond,
                  cudaStream_t st)
{
    if (id != CM_MAT_K_GS1 && id != CM_MAT_K_GS2) { cm_set_error("sys_helmholtz: matrix %d is not a Helmholtz matrix", (int)id); return CM_E_BADARG; }
    CgArgs<T> a;
    CM_TRY(fill_args(S, id, MODE_CSR3, x, tol, maxiter, fixed, mask, slot, precond, &a));
    a.Mval = S->Mm; a.f4 = f4;
    return precond == CM_PC_JACOBI ? launch_cg<T, MODE_CSR3, true, true>(S, a, CM_PROF_CG_GS, st)
                                   : launch_cg<T, MODE_CSR3, false, true>(S, a, CM_PROF_CG_GS, st);
}

template int sys_spmv<double>(System<double> *, cm_matrix_id, int, const double *, double *, cudaStream_t);
template int sys_spmv<float>(System<float> *, cm_matrix_id, int, const float *, float *, cudaStream_t);
template int sys_cg<double>(System<double> *, cm_matrix_id, int, const double *, double *, double, int, int, unsigned, int, int, int, cudaStream_t);
template int sys_cg<float>(System<float> *, cm_matrix_id, int, const float *, float *, double, int, int, unsigned, int, int, int, cudaStream_t);
template int sys_helmholtz<double>(System<double> *, cm_matrix_id, const double *, double *, double, int, int, unsigned, int, int, cudaStream_t);
template int sys_helmholtz<float>(System<float> *, cm_matrix_id, const float *, float *, double, int, int, unsigned, int, int, cudaStream_t);
