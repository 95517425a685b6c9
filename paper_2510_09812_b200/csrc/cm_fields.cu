// S2, S3, S5, S6, S8, S9, S11, S12: volume averages, element-wise gather / compute /
// deterministic gather-scatter right-hand sides, field recovery, the pointwise Gauss-Seidel algebra and the
// projection; and the orchestration of one GSPM step (Alg. B.1).
//
// Scatter is deterministic: a chunk pass (one CTA per element chunk; nodal inputs and per-element contributions
// staged in shared memory) reduces every chunk to one partial per local node ("slot"); a node pass sums a node's
// slots in ascending chunk order.  No float atomics, no per-element scratch in HBM.
#include <cmath>
#include <cstring>
#include <limits>

#include "cm_internal.h"

namespace {

constexpr int BS = 256;
inline unsigned nblk(long n, int b = BS) { return (unsigned)((n + b - 1) / b); }

// ---------------------------------------------------------------- reductions (deterministic, two-stage)
template <int NV>
__device__ __forceinline__ void block_reduce_write(double (&v)[NV], double *out /* [gridDim][NV] */)
{
    __shared__ double sh[NV * 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; k++)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
    if (lane == 0)
#pragma unroll
        for (int k = 0; k < NV; k++) sh[k * 32 + warp] = v[k];
    __syncthreads();
    if (threadIdx.x == 0)
#pragma unroll
        for (int k = 0; k < NV; k++) {
            double s = 0;
            for (int w = 0; w < nwarp; w++) s += sh[k * 32 + w];
            out[(long)blockIdx.x * NV + k] = s;
        }
}

// single block: out[k] = scale * sum_j partial[j][k]
__global__ void reduce_final_kernel(int nparts, int nv, const double *__restrict__ partial, double scale, double *out)
{
    __shared__ double sh[1024];
    for (int k = 0; k < nv; k++) {
        double s = 0;
        for (int j = threadIdx.x; j < nparts; j += blockDim.x) s += partial[(long)j * nv + k];
        sh[threadIdx.x] = s;
        __syncthreads();
        for (int o = blockDim.x / 2; o > 0; o >>= 1) {
            if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) out[k] = scale * sh[0];
        __syncthreads();
    }
}

constexpr int RED_BLOCKS = 2048; // partial blocks of the node-parallel reductions

// S2: sum_i w_i g[i][c]  (w = lumped volume fraction; algebraically Eq. 17 for P1 elements)
template <typename T, int NC>
__global__ void wsum_kernel(long N, const double *__restrict__ w, const T *__restrict__ g, double *partial)
{
    double acc[NC];
#pragma unroll
    for (int c = 0; c < NC; c++) acc[c] = 0;
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < N; i += (long)gridDim.x * blockDim.x) {
        const double wi = w[i];
#pragma unroll
        for (int c = 0; c < NC; c++) acc[c] += wi * (double)g[i * NC + c];
    }
    block_reduce_write<NC>(acc, partial);
}

// ---------------------------------------------------------------- permutation
template <typename T>
__global__ void permute_in_kernel(long N, int nc, const int *__restrict__ order, const T *__restrict__ user, T *lib)
{
    long k = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (k >= N * nc) return;
    long i = k / nc;
    int c = (int)(k - i * nc);
    lib[k] = user[(long)order[i] * nc + c];
}
// user [node][3] -> library PADDED [node][4] (order == NULL: identity)
template <typename T>
__global__ void permute_in4_kernel(long N, const int *__restrict__ order, const T *__restrict__ user, T *lib4)
{
    long k = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (k >= 3 * N) return;
    const long i = k / 3;
    const int c = (int)(k - 3 * i);
    lib4[4 * i + c] = user[(order ? (long)order[i] : i) * 3 + c];
}
template <typename T>
__global__ void permute_out_kernel(long N, int nc, const int *__restrict__ order, const T *__restrict__ lib, T *user)
{
    long k = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (k >= N * nc) return;
    long i = k / nc;
    int c = (int)(k - i * nc);
    user[(long)order[i] * nc + c] = lib[k];
}

// ---------------------------------------------------------------- element passes (S3, S5, S6, S8)
// One CTA per element chunk (cm_internal.h).  At entry one thread issues four TMA bulk copies (cp.async.bulk) that
// stream the chunk's element data -- the chunk-blocked geometry (V_e and nine gradient words per tetrahedron;
// grad phi_0 = -sum of the others, O-1), local node ids, incidence list, material flags -- into shared memory, all
// bytes in flight at once and landing on an mbarrier.  Meanwhile phase 0 stages the chunk's nodal inputs (one global
// gather per local node instead of one per element corner).  Phase 1, one thread per tetrahedron: compute from shared
// memory; the contributions overwrite the element's own column of the staged planes.  Phase 2, one thread per local
// node: sums the node's incidences inside the chunk in ascending element order and writes ONE partial per slot.  A
// node pass then adds a node's slots in ascending chunk order -- a deterministic gather end to end, no float
// atomics, and no per-element scratch in HBM.
enum ElemKind { EK_MS = 0, EK_GRADU = 1, EK_MECH = 2, EK_STRESS = 3, EK_KMECH = 4, EK_GRADU_STRESS = 5 };
// NIN staged words per node, NOUT shared-memory words per element, NC words per slot, PERK: contribution depends on
// the local node index k (NOUT = 4 NC) or is the same for the 4 nodes (NOUT = NC).
template <int KIND> struct KindTraits;
template <> struct KindTraits<EK_MS> { static constexpr int NIN = 3, NOUT = 4, NC = 1; static constexpr bool PERK = true; };
template <> struct KindTraits<EK_GRADU> { static constexpr int NIN = 1, NOUT = 3, NC = 3; static constexpr bool PERK = false; };
template <> struct KindTraits<EK_MECH> { static constexpr int NIN = 3, NOUT = 12, NC = 3; static constexpr bool PERK = true; };
template <> struct KindTraits<EK_STRESS> { static constexpr int NIN = 6, NOUT = 6, NC = 6; static constexpr bool PERK = false; };
// S5 and S8 of the same state in ONE pass (both follow the two solves of a step and read the same geometry, ids and
// incidences): in U, u, w; out V_e grad U_e (3) and V_e C*_e : (E_e(u) - mean_e E0(w)) (6) per slot
template <> struct KindTraits<EK_GRADU_STRESS> { static constexpr int NIN = 7, NOUT = 9, NC = 9; static constexpr bool PERK = false; };
// matrix-free K^mech x (Eq. 12): in x (projected: clamped DOFs read as 0), out sum_e V_e B_k^T C_e B x per slot
template <> struct KindTraits<EK_KMECH> { static constexpr int NIN = 3, NOUT = 12, NC = 3; static constexpr bool PERK = true; };

#ifndef CM_EK_NT
#define CM_EK_NT 384
#endif
constexpr int EK_NT = CM_EK_NT;

template <typename T>
struct ChunkArgs {
    const int *eptr, *nptr, *nodes;
    long N;
    const unsigned short *lid, *lptr, *lent, *emat;
    const T *EG;          // chunk-blocked geometry, 10 planes per chunk (cm_internal.h)
    const double *CX;     // tetrahedra: slot coordinates [slot][4] (GEOM kernels: geometry recomputed, EG not read); hexahedra: [cell][8][3]
    const T *in0, *in1;   // MS, MECH: m;  GRADU: U;  STRESS: u, w;  GRADU_STRESS: u, w and U in in2
    const T *in2;
    const uchar *clamp;   // KMECH: clamped DOFs of the input read as zero (the projection P of P A P + (I - P))
    const int *skip;      // KMECH inside CG: the solve has finished, the launch is a no-op
    const double *mbar;   // MS
    const T *Cstar;       // MECH, STRESS: 36 words per material, or the 12 of the cubic pattern
    T l1, l2;
    T sext[6];            // MECH: sigma_ext / (mu0 Ms^2), added to the stress of EVERY element (R17)
    int has_sext;
    Rot<T> rot;           // App. D: crystal -> simulation frame
    T *hpart;             // [slot][NC]
    double *partial;      // GRADU: per-chunk sums of V_e grad U_e (fp64)
};

// shared-memory layout (every region a multiple of 16 bytes):
//   GEOM = false (stored geometry; wrapped meshes):
//     planes [max(10, NOUT)][EC] T    staged geometry, overwritten in place by the contributions (fixed plane stride EC: the
//                                     plane offsets are immediates)
//   GEOM = true (geometry recomputed from the staged slot coordinates):
//     scx    [CM_NL_MAX][3] double    nondimensional coordinates of the local nodes (region sized for 4 words per node)
//     planes [NOUT][EC] T             contributions
//   sin    [CM_NL_MAX][NIN] T       nodal inputs
//   slid   [EC] ushort4, sle [4 EC] ushort, sem [EC] ushort, slp [CM_NL_MAX + 8] ushort, mbarrier
// node stride of the staged inputs: dense.  Measured at 144^3: records padded to a power-of-two stride for 128-bit loads put the
// random corner gathers on 2-4 bank groups (S8 +17 %); an odd stride of 7 words for the 6-word records of S8: no change (fp64), +3 % (fp32)
constexpr int nin_padded(int nin) { return nin; }
template <int KIND, bool GEOM> constexpr int chunk_planes() { return (GEOM || KindTraits<KIND>::NOUT > 10) ? KindTraits<KIND>::NOUT : 10; }
template <int KIND, typename T, bool GEOM>
constexpr size_t chunk_smem_bytes()
{
    return (GEOM ? (size_t)CM_NL_MAX * 4 * sizeof(double) : 0) +
           (size_t)(chunk_planes<KIND, GEOM>() * CM_EC_MAX + CM_NL_MAX * nin_padded(KindTraits<KIND>::NIN)) * sizeof(T) +
           (size_t)(4 * CM_EC_MAX + 4 * CM_EC_MAX + CM_EC_MAX + CM_NL_MAX + 8) * sizeof(unsigned short) + 16;
}
// resident CTAs per SM the launch bounds ask for (register cap): what the shared-memory footprint allows, at most 4
// (40 registers per thread: enough for every fp32 kernel that streams the stored geometry) or 3 (56 registers) when the
// fp64 geometry is recomputed in the kernel
template <int KIND, typename T, bool GEOM>
constexpr int chunk_minb()
{
    const size_t per = chunk_smem_bytes<KIND, T, GEOM>() + 1024, cap = 227 * 1024;
    const int n = (int)(cap / per), most = GEOM ? 3 : 4;
    return n < 1 ? 1 : (n > most ? most : n);
}
// Which passes recompute the geometry (measured on B200, 144^3 nodes, profiles/r02_microbench_elem.txt): the passes are bound
// by the LSU data pipe that serves shared memory (ncu: 80-88 % of its peak, profiles/r02_elem_ncu.md), not by DRAM, so
// trading ten streamed words per element for twelve more shared-memory gathers and ~100 fp64 instructions pays only where
// the rest of the pass is light: fp64 S3 (0.43 -> 0.36 ms) and S5 (0.61 -> 0.50 ms).  fp64 S6 / S8 and every fp32 pass
// stream the stored geometry.
template <int KIND, typename T>
constexpr bool chunk_recompute() { return sizeof(T) == 8 && (KIND == EK_MS || KIND == EK_GRADU); }

// ---- TMA bulk copy global -> shared, completion on an mbarrier
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile("{\n"
                 ".reg .pred p;\n"
                 "WAIT_%=:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                 "@p bra DONE_%=;\n"
                 "bra WAIT_%=;\n"
                 "DONE_%=:\n"
                 "}" ::"r"(smem_u32(bar)), "r"(parity)
                 : "memory");
}

// E0(m), Table A.1, Voigt engineering vector (E11, E22, E33, 2 E23, 2 E13, 2 E12)
template <typename T>
__device__ __forceinline__ void E0_voigt(const T *m, T l1, T l2, T e0[6])
{
    const T th = (T)1.5, third = (T)(1.0 / 3.0);
    e0[0] = th * l1 * (m[0] * m[0] - third);
    e0[1] = th * l1 * (m[1] * m[1] - third);
    e0[2] = th * l1 * (m[2] * m[2] - third);
    e0[3] = (T)2 * th * l2 * m[1] * m[2];
    e0[4] = (T)2 * th * l2 * m[0] * m[2];
    e0[5] = (T)2 * th * l2 * m[0] * m[1];
}

// ---- App. D helpers: v_c = R^T v, v = R v_c, and Q t Q^T for a symmetric tensor given by its 6 tensor components
template <typename T>
__device__ __forceinline__ void rot_to_crystal(const Rot<T> &R, const T v[3], T vc[3])
{
#pragma unroll
    for (int a = 0; a < 3; a++) vc[a] = R.r[a] * v[0] + R.r[3 + a] * v[1] + R.r[6 + a] * v[2];
}
template <typename T>
__device__ __forceinline__ void rot_to_sim(const Rot<T> &R, const T vc[3], T v[3])
{
#pragma unroll
    for (int a = 0; a < 3; a++) v[a] = R.r[3 * a] * vc[0] + R.r[3 * a + 1] * vc[1] + R.r[3 * a + 2] * vc[2];
}
template <typename T, bool INV>
__device__ __forceinline__ void rot_sym(const Rot<T> &R, const T t[6], T out[6])
{
    const T A[3][3] = {{t[0], t[5], t[4]}, {t[5], t[1], t[3]}, {t[4], t[3], t[2]}};
    T B[3][3], Cm[3][3];
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            T acc = 0;
#pragma unroll
            for (int k = 0; k < 3; k++) acc += (INV ? R.r[3 * k + i] : R.r[3 * i + k]) * A[k][j];
            B[i][j] = acc;
        }
#pragma unroll
    for (int i = 0; i < 3; i++)
#pragma unroll
        for (int j = 0; j < 3; j++) {
            T acc = 0;
#pragma unroll
            for (int k = 0; k < 3; k++) acc += B[i][k] * (INV ? R.r[3 * k + j] : R.r[3 * j + k]);
            Cm[i][j] = acc;
        }
    out[0] = Cm[0][0]; out[1] = Cm[1][1]; out[2] = Cm[2][2]; out[3] = Cm[1][2]; out[4] = Cm[0][2]; out[5] = Cm[0][1];
}

// E0 in the simulation frame (Alg. D.1 Step 1): R E0_crystal(R^T m) R^T, engineering-shear Voigt vector
template <typename T>
__device__ __forceinline__ void E0_sim(const Rot<T> &R, const T *m, T l1, T l2, T e0[6])
{
    if (!R.on) { E0_voigt(m, l1, l2, e0); return; }
    T mc[3], ec[6], t[6];
    rot_to_crystal(R, m, mc);
    E0_voigt(mc, l1, l2, ec);
#pragma unroll
    for (int q = 3; q < 6; q++) ec[q] /= (T)2;
    rot_sym<T, false>(R, ec, t);
#pragma unroll
    for (int q = 0; q < 3; q++) { e0[q] = t[q]; e0[3 + q] = (T)2 * t[3 + q]; }
}

// a staged 3-vector
template <typename T>
__device__ __forceinline__ void ld3(const T *p, T (&o)[3]) { o[0] = p[0]; o[1] = p[1]; o[2] = p[2]; }

// H[a][b] = d_b x_a = sum_k x_k[a] grad phi_k[b], x_k = sx[ST * l[k] ..]
template <typename T, int ST>
__device__ __forceinline__ void strain_H(const T *sx, const int *l, const T (&g)[4][3], T (&H)[3][3])
{
#pragma unroll
    for (int x = 0; x < 3; x++)
#pragma unroll
        for (int y = 0; y < 3; y++) H[x][y] = 0;
#pragma unroll
    for (int k = 0; k < 4; k++) {
        T xk[3];
        ld3(sx + ST * l[k], xk);
#pragma unroll
        for (int x = 0; x < 3; x++)
#pragma unroll
            for (int y = 0; y < 3; y++) H[x][y] += xk[x] * g[k][y];
    }
}

// mean over the 4 corners of E0(w); w_k = sw[ST * l[k] + OFF ..]
template <typename T, int ST, int OFF>
__device__ __forceinline__ void mean_E0(const Rot<T> &R, const T *sw, const int *l, T l1, T l2, T e0[6])
{
#pragma unroll
    for (int q = 0; q < 6; q++) e0[q] = 0;
#pragma unroll
    for (int k = 0; k < 4; k++) {
        T mk[3], ek[6];
        ld3(sw + ST * l[k] + OFF, mk);
        E0_sim(R, mk, l1, l2, ek);
#pragma unroll
        for (int q = 0; q < 6; q++) e0[q] += ek[q];
    }
#pragma unroll
    for (int q = 0; q < 6; q++) e0[q] /= (T)4;
}

template <typename T>
__device__ __forceinline__ void C_times(const T *__restrict__ C, const T eps[6], T sig[6])
{
#pragma unroll
    for (int r = 0; r < 6; r++) {
        T acc = 0;
#pragma unroll
        for (int s = 0; s < 6; s++) acc += __ldg(C + 6 * r + s) * eps[s];
        sig[r] = acc;
    }
}

// same product when C* has the cubic pattern; Cc = (C11 C12 C13 C21 C22 C23 C31 C32 C33 C44 C55 C66)
template <typename T>
__device__ __forceinline__ void C_times_cubic(const T *__restrict__ Cc, const T eps[6], T sig[6])
{
    T c[12];
    if (sizeof(T) == 8) {
#pragma unroll
        for (int q = 0; q < 6; q++) *reinterpret_cast<double2 *>(c + 2 * q) = __ldg(reinterpret_cast<const double2 *>(Cc) + q);
    } else {
#pragma unroll
        for (int q = 0; q < 3; q++) *reinterpret_cast<float4 *>(c + 4 * q) = __ldg(reinterpret_cast<const float4 *>(Cc) + q);
    }
#pragma unroll
    for (int r = 0; r < 3; r++) {
        T acc = 0;
#pragma unroll
        for (int s = 0; s < 3; s++) acc += c[3 * r + s] * eps[s];
        sig[r] = acc;
    }
#pragma unroll
    for (int r = 3; r < 6; r++) sig[r] = c[6 + r] * eps[r];
}

template <typename T, int KIND, bool CUBIC, bool GEOM>
__global__ void __launch_bounds__(EK_NT, (chunk_minb<KIND, T, GEOM>())) elem_chunk_kernel(ChunkArgs<T> a)
{
    typedef KindTraits<KIND> K;
    constexpr int NIN = K::NIN, NOUT = K::NOUT, NC = K::NC, EC = CM_EC_MAX, NP = chunk_planes<KIND, GEOM>(), NINP = nin_padded(NIN);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *scx = reinterpret_cast<double *>(smem_raw);                          // [nl][4] (GEOM)
    T *scr = reinterpret_cast<T *>(smem_raw + (GEOM ? (size_t)CM_NL_MAX * 4 * sizeof(double) : 0)); // [NP][EC]
    T *sin = scr + NP * EC;                                                     // [nl][NIN]
    ushort4 *slid = reinterpret_cast<ushort4 *>(sin + CM_NL_MAX * NINP);        // [ne]
    unsigned short *sle = reinterpret_cast<unsigned short *>(slid + EC);        // [4 ne]
    unsigned short *sem = sle + 4 * EC;                                         // [ne]
    unsigned short *slp = sem + EC;                                             // [nl + 1]
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(slp + CM_NL_MAX + 8);
    const int c = blockIdx.x, tid = threadIdx.x;
    if (KIND == EK_KMECH && a.skip && *a.skip) return;
    const int e0 = a.eptr[c], ne = a.eptr[c + 1] - e0, ne8 = (ne + 7) & ~7, s0 = a.nptr[c], nl = a.nptr[c + 1] - s0;

    // ---- element data: bulk copies, all of the chunk's streaming bytes in flight at once
    if (tid == 0) {
        mbar_init(bar, 1);
        const unsigned bg = GEOM ? 0u : 10u * ne8 * (unsigned)sizeof(T), bl = 8u * ne8, be = 2u * ne8;
        mbar_expect_tx(bar, bg + 2 * bl + be);
        if (!GEOM)
            for (int q = 0; q < 10; q++) bulk_g2s(scr + q * EC, a.EG + 10L * e0 + (long)q * ne8, bg / 10, bar);
        bulk_g2s(slid, a.lid + 4L * e0, bl, bar);
        bulk_g2s(sle, a.lent + 4L * e0, bl, bar);
        bulk_g2s(sem, a.emat + e0, be, bar);
    }
    // ---- phase 0: nodal inputs, incidence runs; slot coordinates at a dense 3-word stride (coalesced read of the 32-byte
    // slot records; the dense stride spreads the corner gathers of phase 1 over all bank pairs, the records' own stride over 4)
    for (int l = tid; l < nl; l += EK_NT) {
        if (GEOM) {
            const double2 c0 = *reinterpret_cast<const double2 *>(a.CX + 4L * (s0 + l));
            scx[3 * l] = c0.x; scx[3 * l + 1] = c0.y; scx[3 * l + 2] = a.CX[4L * (s0 + l) + 2];
        }
        const long g = a.nodes[s0 + l];
        if (KIND == EK_GRADU) {
            sin[l] = a.in0[g];
        } else if (KIND == EK_KMECH) {
#pragma unroll
            for (int d = 0; d < 3; d++) sin[NINP * l + d] = a.clamp[3 * g + d] ? (T)0 : a.in0[3 * g + d];
        } else if (KIND == EK_GRADU_STRESS) {
            sin[NINP * l] = a.in2[g];
#pragma unroll
            for (int d = 0; d < 3; d++) { sin[NINP * l + 1 + d] = a.in0[3 * g + d]; sin[NINP * l + 4 + d] = a.in1[3 * g + d]; }
        } else {
#pragma unroll
            for (int d = 0; d < 3; d++) sin[NINP * l + d] = a.in0[3 * g + d];
            if (KIND == EK_STRESS)
#pragma unroll
                for (int d = 0; d < 3; d++) sin[NINP * l + 3 + d] = a.in1[3 * g + d];
        }
    }
    for (int l = tid; l <= nl; l += EK_NT) slp[l] = a.lptr[s0 + c + l];
    __syncthreads(); // also orders the mbarrier initialisation before the waits
    mbar_wait(bar, 0);

    // ---- phase 1: one thread per tetrahedron; its contributions go to its own column of the planes
    double gsum[3] = {0, 0, 0};
    for (int el = tid; el < ne; el += EK_NT) {
        const ushort4 lq = slid[el];
        const int l[4] = {lq.x, lq.y, lq.z, lq.w};
        T V, g[4][3];
        if (GEOM) {
            // O-1 in fp64 from the staged coordinates, rounded once to T: the bits the stored geometry holds (R20)
            double x[4][3];
#pragma unroll
            for (int k = 0; k < 4; k++) {
                x[k][0] = scx[3 * l[k]]; x[k][1] = scx[3 * l[k] + 1]; x[k][2] = scx[3 * l[k] + 2];
            }
            TetGeom G;
            tet_geometry_x(x, G);
            V = (T)G.V;
#pragma unroll
            for (int k = 1; k < 4; k++)
#pragma unroll
                for (int d = 0; d < 3; d++) g[k][d] = (T)G.g[k][d];
        } else {
            V = scr[el];
#pragma unroll
            for (int k = 1; k < 4; k++)
#pragma unroll
                for (int d = 0; d < 3; d++) g[k][d] = scr[(3 * (k - 1) + d + 1) * EC + el];
        }
#pragma unroll
        for (int d = 0; d < 3; d++) g[0][d] = -(g[1][d] + g[2][d] + g[3][d]);

        if (KIND == EK_MS) {
            // c_k = V_e grad phi_k . (mean_e m - mbar)
            T mt[3], w0[3], w1[3], w2[3], w3[3];
            ld3(sin + NINP * l[0], w0); ld3(sin + NINP * l[1], w1); ld3(sin + NINP * l[2], w2); ld3(sin + NINP * l[3], w3);
#pragma unroll
            for (int d = 0; d < 3; d++) mt[d] = (w0[d] + w1[d] + w2[d] + w3[d]) / (T)4 - (T)a.mbar[d];
#pragma unroll
            for (int k = 0; k < 4; k++) scr[k * EC + el] = V * (g[k][0] * mt[0] + g[k][1] * mt[1] + g[k][2] * mt[2]);
        } else if (KIND == EK_GRADU) {
            // V_e grad U_e, and its fp64 sum for <grad U>
            const T u0 = sin[l[0]], u1 = sin[l[1]], u2 = sin[l[2]], u3 = sin[l[3]];
#pragma unroll
            for (int d = 0; d < 3; d++) {
                const T gU = u0 * g[0][d] + u1 * g[1][d] + u2 * g[2][d] + u3 * g[3][d];
                scr[d * EC + el] = V * gU;
                gsum[d] += (double)V * (double)gU;
            }
        } else if (KIND == EK_GRADU_STRESS) {
            const T u0 = sin[NINP * l[0]], u1 = sin[NINP * l[1]], u2 = sin[NINP * l[2]], u3 = sin[NINP * l[3]];
#pragma unroll
            for (int d = 0; d < 3; d++) {
                const T gU = u0 * g[0][d] + u1 * g[1][d] + u2 * g[2][d] + u3 * g[3][d];
                scr[d * EC + el] = V * gU;
                gsum[d] += (double)V * (double)gU;
            }
            const unsigned em = sem[el];
            if (!(em & 1u)) {
#pragma unroll
                for (int q = 0; q < 6; q++) scr[(3 + q) * EC + el] = 0;
            } else {
                T H[3][3];
                strain_H<T, NINP>(sin + 1, l, g, H);
                T eps[6] = {H[0][0], H[1][1], H[2][2], H[1][2] + H[2][1], H[0][2] + H[2][0], H[0][1] + H[1][0]}, e0v[6], sg[6];
                mean_E0<T, NINP, 4>(a.rot, sin, l, a.l1, a.l2, e0v);
#pragma unroll
                for (int q = 0; q < 6; q++) eps[q] -= e0v[q];
                if (CUBIC) C_times_cubic(a.Cstar + 12 * (em >> 1), eps, sg);
                else C_times(a.Cstar + 36 * (em >> 1), eps, sg);
#pragma unroll
                for (int q = 0; q < 6; q++) scr[(3 + q) * EC + el] = V * sg[q];
            }
        } else if (KIND == EK_KMECH) {
            // sigma = C*_e : E_e(x), H[a][b] = d_b x_a;  c_(k,a) = V_e (sigma grad phi_k)_a   (every element is elastic)
            T H[3][3];
            strain_H<T, NINP>(sin, l, g, H);
            const T eps[6] = {H[0][0], H[1][1], H[2][2], H[1][2] + H[2][1], H[0][2] + H[2][0], H[0][1] + H[1][0]};
            T sg[6];
            const unsigned em = sem[el];
            if (CUBIC) C_times_cubic(a.Cstar + 12 * (em >> 1), eps, sg);
            else C_times(a.Cstar + 36 * (em >> 1), eps, sg);
#pragma unroll
            for (int k = 0; k < 4; k++) {
                scr[(3 * k + 0) * EC + el] = V * (sg[0] * g[k][0] + sg[5] * g[k][1] + sg[4] * g[k][2]);
                scr[(3 * k + 1) * EC + el] = V * (sg[5] * g[k][0] + sg[1] * g[k][1] + sg[3] * g[k][2]);
                scr[(3 * k + 2) * EC + el] = V * (sg[4] * g[k][0] + sg[3] * g[k][1] + sg[2] * g[k][2]);
            }
        } else {
            const unsigned em = sem[el];
            if (!(em & 1u) && !(KIND == EK_MECH && a.has_sext)) {
#pragma unroll
                for (int q = 0; q < NOUT; q++) scr[q * EC + el] = 0;
            } else if (KIND == EK_MECH) {
                // S = C*_e : mean_e E0(m) (magnetic elements) + sigma_ext (all elements);  c_(k,a) = V_e (S grad phi_k)_a
                T e0v[6], sg[6] = {0, 0, 0, 0, 0, 0};
                if (em & 1u) {
                    mean_E0<T, NINP, 0>(a.rot, sin, l, a.l1, a.l2, e0v);
                    if (CUBIC) C_times_cubic(a.Cstar + 12 * (em >> 1), e0v, sg);
                    else C_times(a.Cstar + 36 * (em >> 1), e0v, sg);
                }
                if (a.has_sext)
#pragma unroll
                    for (int q = 0; q < 6; q++) sg[q] += a.sext[q];
#pragma unroll
                for (int k = 0; k < 4; k++) {
                    scr[(3 * k + 0) * EC + el] = V * (sg[0] * g[k][0] + sg[5] * g[k][1] + sg[4] * g[k][2]);
                    scr[(3 * k + 1) * EC + el] = V * (sg[5] * g[k][0] + sg[1] * g[k][1] + sg[3] * g[k][2]);
                    scr[(3 * k + 2) * EC + el] = V * (sg[4] * g[k][0] + sg[3] * g[k][1] + sg[2] * g[k][2]);
                }
            } else {
                // V_e C*_e : (E_e(u) - mean_e E0(w)),  H[a][b] = d_b u_a
                T H[3][3];
                strain_H<T, NINP>(sin, l, g, H);
                T eps[6] = {H[0][0], H[1][1], H[2][2], H[1][2] + H[2][1], H[0][2] + H[2][0], H[0][1] + H[1][0]}, e0v[6], sg[6];
                mean_E0<T, NINP, 3>(a.rot, sin, l, a.l1, a.l2, e0v);
#pragma unroll
                for (int q = 0; q < 6; q++) eps[q] -= e0v[q];
                if (CUBIC) C_times_cubic(a.Cstar + 12 * (em >> 1), eps, sg);
                else C_times(a.Cstar + 36 * (em >> 1), eps, sg);
#pragma unroll
                for (int q = 0; q < 6; q++) scr[q * EC + el] = V * sg[q];
            }
        }
    }
    __syncthreads();

    // ---- phase 2: one thread per local node, incidences in ascending element order
    for (int l = tid; l < nl; l += EK_NT) {
        T acc[NC];
#pragma unroll
        for (int q = 0; q < NC; q++) acc[q] = 0;
        for (int q = slp[l]; q < slp[l + 1]; q++) {
            const int ent = sle[q], el = ent >> 2, k = ent & 3;
#pragma unroll
            for (int x = 0; x < NC; x++) acc[x] += scr[(K::PERK ? NC * k + x : x) * EC + el];
        }
#pragma unroll
        for (int x = 0; x < NC; x++) a.hpart[(long)(s0 + l) * NC + x] = acc[x];
    }
    if (KIND == EK_GRADU || KIND == EK_GRADU_STRESS) block_reduce_write<3>(gsum, a.partial);
}

// node pass: b_i = sum of the node's slot partials (ascending chunk order); zero where the mask says so
template <typename T, int NC>
__global__ void node_gather_kernel(long N, const int *__restrict__ ns_ptr, const int *__restrict__ ns_slot, const T *__restrict__ hpart,
                                   const uchar *__restrict__ zero_mask /* N*NC or NULL */, int zero_node, T *b)
{
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    T acc[NC];
#pragma unroll
    for (int c = 0; c < NC; c++) acc[c] = 0;
    for (int s = ns_ptr[i]; s < ns_ptr[i + 1]; s++) {
        const long q = __ldg(ns_slot + s);
#pragma unroll
        for (int c = 0; c < NC; c++) acc[c] += hpart[q * NC + c];
    }
#pragma unroll
    for (int c = 0; c < NC; c++) {
        if (zero_mask && zero_mask[i * NC + c]) acc[c] = 0;
        if (i == zero_node) acc[c] = 0;
        b[i * NC + c] = acc[c];
    }
}

// node pass of S5: h_d,i = -sum_{e} V_e grad U_e / (4 mL_i) + <grad U>   (DEMAG)   - N_d mbar   (FARFIELD)
template <typename T>
__global__ void node_hd_kernel(long N, const int *__restrict__ ns_ptr, const int *__restrict__ ns_slot, const T *__restrict__ hpart,
                               const T *__restrict__ mL, const double *__restrict__ scal /* mbar[0..2], gradU mean[3..5] */,
                               unsigned terms, double n00, double n01, double n02, double n10, double n11,
                               double n12, double n20, double n21, double n22, T dscale /* 4: tets (V_e / 4 weights), 1: hexahedra */,
                               int hs /* words per slot in hpart */, T *hd)
{
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    T h[3] = {0, 0, 0};
    if (terms & CM_TERM_DEMAG) {
        T acc[3] = {0, 0, 0};
        for (int s = ns_ptr[i]; s < ns_ptr[i + 1]; s++) {
            const long q = __ldg(ns_slot + s);
#pragma unroll
            for (int d = 0; d < 3; d++) acc[d] += hpart[hs * q + d];
        }
        const T den = dscale * mL[i];
#pragma unroll
        for (int d = 0; d < 3; d++) h[d] = -acc[d] / den + (T)scal[3 + d];
    }
    if (terms & CM_TERM_FARFIELD) {
        const double m0 = scal[0], m1 = scal[1], m2 = scal[2];
        h[0] -= (T)(n00 * m0 + n01 * m1 + n02 * m2);
        h[1] -= (T)(n10 * m0 + n11 * m1 + n12 * m2);
        h[2] -= (T)(n20 * m0 + n21 * m1 + n22 * m2);
    }
    hd[3 * i] = h[0]; hd[3 * i + 1] = h[1]; hd[3 * i + 2] = h[2];
}

// ---------------------------------------------------------------- S9 nodal field
// node pass: sigma_hat_i (from the slot partials of the stress pass when MAGEL), h = h_an + h_ext + h_d + h_me on
// live nodes; optionally also writes sigma_hat (parity output).
template <typename T>
__global__ void node_field_kernel(long N, const int *__restrict__ ns_ptr, const int *__restrict__ ns_slot, const T *__restrict__ hpart,
                                  const T *__restrict__ mLm, const uchar *__restrict__ live, const T *__restrict__ w,
                                  const T *__restrict__ hd, unsigned terms, T Kstar2, T hx, T hy, T hz, const double *__restrict__ hext_dev,
                                  T l1, T l2, Rot<T> rot, T dscale, int hs /* words per slot in hpart */, T *h, T *sig_out)
{
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    if (hext_dev) { hx = (T)hext_dev[0]; hy = (T)hext_dev[1]; hz = (T)hext_dev[2]; } // device-resident field (hysteresis driver)
    T hi[3] = {0, 0, 0}, s[6] = {0, 0, 0, 0, 0, 0};
    if (live[i]) {
        // Alg. D.1 Step 4: m-dependent terms in crystal axes (m_c = R^T m, sigma_c = R^T sigma R), then h = R h_c
        const T ms_[3] = {w[3 * i], w[3 * i + 1], w[3 * i + 2]};
        T m[3] = {ms_[0], ms_[1], ms_[2]}, hc[3] = {0, 0, 0};
        if (rot.on) rot_to_crystal(rot, ms_, m);
        if (terms & CM_TERM_ANIS) {
            hc[0] -= Kstar2 * m[0] * (m[1] * m[1] + m[2] * m[2]);
            hc[1] -= Kstar2 * m[1] * (m[2] * m[2] + m[0] * m[0]);
            hc[2] -= Kstar2 * m[2] * (m[0] * m[0] + m[1] * m[1]);
        }
        if (terms & CM_TERM_MAGEL) {
            for (int q = ns_ptr[i]; q < ns_ptr[i + 1]; q++) {
                const long sl = __ldg(ns_slot + q);
#pragma unroll
                for (int c = 0; c < 6; c++) s[c] += hpart[hs * sl + c];
            }
            const T den = dscale * mLm[i];
#pragma unroll
            for (int c = 0; c < 6; c++) s[c] /= den;
            T sc[6] = {s[0], s[1], s[2], s[3], s[4], s[5]};
            if (rot.on) rot_sym<T, true>(rot, s, sc);
            hc[0] += (T)3 * (l1 * m[0] * sc[0] + l2 * (m[1] * sc[5] + m[2] * sc[4]));
            hc[1] += (T)3 * (l1 * m[1] * sc[1] + l2 * (m[0] * sc[5] + m[2] * sc[3]));
            hc[2] += (T)3 * (l1 * m[2] * sc[2] + l2 * (m[0] * sc[4] + m[1] * sc[3]));
        }
        if (rot.on) rot_to_sim(rot, hc, hi);
        else { hi[0] = hc[0]; hi[1] = hc[1]; hi[2] = hc[2]; }
        if (terms & CM_TERM_ZEEMAN) { hi[0] += hx; hi[1] += hy; hi[2] += hz; }
        if (terms & (CM_TERM_DEMAG | CM_TERM_FARFIELD)) { hi[0] += hd[3 * i]; hi[1] += hd[3 * i + 1]; hi[2] += hd[3 * i + 2]; }
    }
    if (h) { h[3 * i] = hi[0]; h[3 * i + 1] = hi[1]; h[3 * i + 2] = hi[2]; }
    if (sig_out)
#pragma unroll
        for (int c = 0; c < 6; c++) sig_out[6 * i + c] = s[c];
}

// ---------------------------------------------------------------- pointwise GSPM algebra (S9, S11, S12)
// f = base + c h per node; f is PADDED, four words per node (what the three-right-hand-side products gather)
template <typename T>
__global__ void axpby_kernel(long N, const T *__restrict__ base, const T *__restrict__ h, T c, T *f4)
{
    long k = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (k >= 3 * N) return;
    const long i = k / 3;
    f4[4 * i + (k - 3 * i)] = base[k] + c * h[k];
}

// Step 2, first part.  variant 0: m*_1, m*_2 from level-n values; f_a = m*_a + dtau h_a[m^n], a = 1, 2.
// variant 1, stage 0: m*_1 and f_1 only; stage 1: m*_2 = m_2 + (g^n_3 m*_1 - g*_1 m_3) and f_2.  f is padded [node][4].
template <typename T>
__global__ void gs_step2_kernel(long N, int variant, int stage, const T *__restrict__ m, const T *__restrict__ gn,
                                const T *__restrict__ gs, const T *__restrict__ hn, T dtau, T *ms, T *f)
{
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const T m0 = m[3 * i], m1 = m[3 * i + 1], m2 = m[3 * i + 2];
    if (variant == 0 || stage == 0) {
        const T s0 = m0 + (gn[3 * i + 1] * m2 - gn[3 * i + 2] * m1);
        ms[3 * i] = s0;
        f[4 * i] = s0 + dtau * hn[3 * i];
    }
    if (variant == 0) {
        const T s1 = m1 + (gn[3 * i + 2] * m0 - gn[3 * i] * m2);
        ms[3 * i + 1] = s1;
        f[4 * i + 1] = s1 + dtau * hn[3 * i + 1];
    } else if (stage == 1) {
        const T s1 = m1 + (gn[3 * i + 2] * ms[3 * i] - gs[3 * i] * m2);
        ms[3 * i + 1] = s1;
        f[4 * i + 1] = s1 + dtau * hn[3 * i + 1];
    }
}

// m*_3 = m_3 + (g*_1 m*_2 - g*_2 m*_1)
template <typename T>
__global__ void gs_step2c_kernel(long N, const T *__restrict__ m, const T *__restrict__ gs, T *ms)
{
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    ms[3 * i + 2] = m[3 * i + 2] + (gs[3 * i] * ms[3 * i + 1] - gs[3 * i + 1] * ms[3 * i]);
}

// Step 4: projection on live nodes, dead nodes zero; partial sums of ||m_new - m_old||_2
template <typename T>
__global__ void project_kernel(long N, const uchar *__restrict__ live, const T *__restrict__ mss, T *m, double *partial)
{
    double acc[1] = {0};
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < N; i += (long)gridDim.x * blockDim.x) {
        if (!live[i]) { m[3 * i] = 0; m[3 * i + 1] = 0; m[3 * i + 2] = 0; continue; }
        const T v0 = mss[3 * i], v1 = mss[3 * i + 1], v2 = mss[3 * i + 2];
        const T nrm = (T)sqrt((double)(v0 * v0 + v1 * v1 + v2 * v2));
        const T o0 = m[3 * i], o1 = m[3 * i + 1], o2 = m[3 * i + 2];
        T n0 = o0, n1 = o1, n2 = o2;
        if (nrm > 0) { n0 = v0 / nrm; n1 = v1 / nrm; n2 = v2 / nrm; }
        const double d0 = (double)n0 - (double)o0, d1 = (double)n1 - (double)o1, d2 = (double)n2 - (double)o2;
        acc[0] += sqrt(d0 * d0 + d1 * d1 + d2 * d2);
        m[3 * i] = n0; m[3 * i + 1] = n1; m[3 * i + 2] = n2;
    }
    block_reduce_write<1>(acc, partial);
}

} // namespace

// ------------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------------
#define LAUNCH_CHECK() CM_CUDA(cudaGetLastError())

template <typename T>
int sys_permute_in(System<T> *S, const T *user, T *lib, int nc, cudaStream_t st)
{
    if (nc == -3) { // three components into the padded layout
        S->prof.begin(CM_PROF_POINTWISE, st);
        permute_in4_kernel<T><<<nblk(3 * S->N), BS, 0, st>>>(S->N, S->mesh->identity ? nullptr : S->mesh->d_order, user, lib);
        S->prof.end(st);
        LAUNCH_CHECK();
        return CM_OK;
    }
    const long n = S->N * nc;
    if (S->mesh->identity) { CM_CUDA(cudaMemcpyAsync(lib, user, n * sizeof(T), cudaMemcpyDeviceToDevice, st)); return CM_OK; }
    S->prof.begin(CM_PROF_POINTWISE, st);
    permute_in_kernel<T><<<nblk(n), BS, 0, st>>>(S->N, nc, S->mesh->d_order, user, lib);
    S->prof.end(st);
    LAUNCH_CHECK();
    return CM_OK;
}
template <typename T>
int sys_permute_out(System<T> *S, const T *lib, T *user, int nc, cudaStream_t st)
{
    const long n = S->N * nc;
    if (S->mesh->identity) { CM_CUDA(cudaMemcpyAsync(user, lib, n * sizeof(T), cudaMemcpyDeviceToDevice, st)); return CM_OK; }
    S->prof.begin(CM_PROF_POINTWISE, st);
    permute_out_kernel<T><<<nblk(n), BS, 0, st>>>(S->N, nc, S->mesh->d_order, lib, user);
    S->prof.end(st);
    LAUNCH_CHECK();
    return CM_OK;
}

// volume average of an NC-component library-order field into dst[0..NC) (device)
template <typename T>
static int wavg(const cm_mesh *M, const T *g_lib, int nc, double *red, double *dst, cudaStream_t st)
{
    const int nb = (int)std::min<long>(RED_BLOCKS, nblk(M->N));
    switch (nc) {
    case 1: wsum_kernel<T, 1><<<nb, BS, 0, st>>>(M->N, M->d_wvol, g_lib, red); break;
    case 3: wsum_kernel<T, 3><<<nb, BS, 0, st>>>(M->N, M->d_wvol, g_lib, red); break;
    case 6: wsum_kernel<T, 6><<<nb, BS, 0, st>>>(M->N, M->d_wvol, g_lib, red); break;
    default: cm_set_error("volume average: ncomp must be 1, 3 or 6"); return CM_E_BADARG;
    }
    reduce_final_kernel<<<1, 1024, 0, st>>>(nb, nc, red, 1.0, dst);
    LAUNCH_CHECK();
    return CM_OK;
}

template <typename T>
int sys_mbar(System<T> *S, const T *m_lib, cudaStream_t st)
{
    S->prof.begin(CM_PROF_POINTWISE, st, 2);
    int rc = wavg<T>(S->mesh, m_lib, 3, S->red, S->dscal, st);
    S->prof.end(st);
    return rc;
}

template <typename T>
static ChunkArgs<T> chunk_args(System<T> *S)
{
    const cm_mesh *M = S->mesh;
    const Chunks &K = M->ck;
    ChunkArgs<T> a;
    a.eptr = K.d_eptr; a.nptr = K.d_nptr; a.nodes = K.d_nodes; a.lid = K.d_lid; a.lptr = K.d_lptr; a.lent = K.d_lent;
    a.emat = M->d_emat; a.EG = S->EG; a.CX = S->CX;
    a.N = S->N;
    a.in0 = nullptr; a.in1 = nullptr; a.in2 = nullptr; a.clamp = S->clamp; a.skip = nullptr; a.mbar = S->dscal; a.Cstar = S->Cstar; a.l1 = (T)S->lam100; a.l2 = (T)S->lam111;
    a.rot = make_rot<T>(S);
    for (int q = 0; q < 6; q++) a.sext[q] = (T)S->sext[q];
    a.has_sext = S->has_sext ? 1 : 0;
    a.hpart = S->hpart; a.partial = S->red;
    return a;
}

template <typename T, int KIND, bool CUBIC, bool GEOM>
static int launch_chunk_kernel(System<T> *S, const ChunkArgs<T> &a, cudaStream_t st)
{
    constexpr size_t smem = chunk_smem_bytes<KIND, T, GEOM>();
    // per device and per function; a host-side table lookup, set on every launch so that any device / context works
    CM_CUDA(cudaFuncSetAttribute(elem_chunk_kernel<T, KIND, CUBIC, GEOM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    elem_chunk_kernel<T, KIND, CUBIC, GEOM><<<S->mesh->ck.nchunks, EK_NT, smem, st>>>(a);
    return CM_OK;
}

// geometry recomputed from the slot coordinates where that is the faster kernel (chunk_recompute; geometry_mode 0), never
// (mode 1) or in every pass (mode 2: the A/B measurement); wrapped meshes have no slot coordinates and always stream EG
template <typename T, int KIND>
static int launch_chunks(System<T> *S, const ChunkArgs<T> &a, cudaStream_t st)
{
    constexpr bool USES_C = KIND == EK_MECH || KIND == EK_STRESS || KIND == EK_KMECH || KIND == EK_GRADU_STRESS;
    const bool geom = S->CX != nullptr && (S->geometry_mode == 2 || (S->geometry_mode == 0 && chunk_recompute<KIND, T>()));
    if (USES_C && S->cubic_pattern) {
        ChunkArgs<T> b = a;
        b.Cstar = S->Ccub;
        return geom ? launch_chunk_kernel<T, KIND, USES_C, true>(S, b, st) : launch_chunk_kernel<T, KIND, USES_C, false>(S, b, st);
    }
    return geom ? launch_chunk_kernel<T, KIND, false, true>(S, a, st) : launch_chunk_kernel<T, KIND, false, false>(S, a, st);
}

// ---------------------------------------------------------------- element passes on linear hexahedra (R26)
// Element-centric: one CTA per chunk of at most CM_HC_MAX cells, EIGHT lanes per cell, one per Gauss point.  A lane recomputes
// the fp64 geometry at its point from the cell's own corner coordinates (staged per cell, 24 words: a wrapped -- periodic --
// cell takes its corners from its own images, so coordinates cannot be shared per node, R23), evaluates the
// integrand there and its contribution to the cell's eight corners; a three-step exchange
// inside the 8-lane group (halving the corners kept at every step) leaves lane p with the cell's total for corner p,
// which goes to the contribution planes.  Phase 2 and the node passes are those of the tetrahedral kernels.  Each cell is
// integrated once (round 1's node-centric kernel integrated it eight times, once per corner: 1.3-3.0 ms per pass at 10^6
// nodes against 0.23-0.61 ms).
constexpr int HK_NT = 256;

__device__ __forceinline__ double shfl_x(unsigned mask, double v, int o) { return __shfl_xor_sync(mask, v, o); }
__device__ __forceinline__ float shfl_x(unsigned mask, float v, int o) { return __shfl_xor_sync(mask, v, o); }

// lane p holds the contribution ph[a] * w[x] (RANK1) or c[a][x] of its Gauss point to corner a; out[x] = sum over the 8
// lanes of the contributions to corner p (fixed order)
template <typename T, int NC, bool RANK1>
__device__ __forceinline__ void cell_exchange(unsigned mask, int p, const T (&ph)[8], const T (&w)[NC], const T (&c)[8][NC], T (&out)[NC])
{
    const bool h4 = p & 4, h2 = p & 2, h1 = p & 1;
    T k1[4][NC];
#pragma unroll
    for (int j = 0; j < 4; j++)
#pragma unroll
        for (int x = 0; x < NC; x++) {
            const T lo = RANK1 ? ph[j] * w[x] : c[j][x], hi = RANK1 ? ph[4 + j] * w[x] : c[4 + j][x];
            k1[j][x] = (h4 ? hi : lo) + shfl_x(mask, h4 ? lo : hi, 4);
        }
    T k2[2][NC];
#pragma unroll
    for (int i = 0; i < 2; i++)
#pragma unroll
        for (int x = 0; x < NC; x++) k2[i][x] = (h2 ? k1[2 + i][x] : k1[i][x]) + shfl_x(mask, h2 ? k1[i][x] : k1[2 + i][x], 2);
#pragma unroll
    for (int x = 0; x < NC; x++) out[x] = (h1 ? k2[1][x] : k2[0][x]) + shfl_x(mask, h1 ? k2[0][x] : k2[1][x], 1);
}

template <int KIND, typename T>
constexpr size_t hex_smem_bytes()
{
    return (size_t)CM_HC_MAX * 24 * sizeof(double) + (size_t)(8 * KindTraits<KIND>::NC * CM_HC_MAX + CM_NL_MAX * KindTraits<KIND>::NIN) * sizeof(T) +
           (size_t)(8 * CM_HC_MAX + 8 * CM_HC_MAX + CM_HC_MAX + CM_NL_MAX + 8) * sizeof(unsigned short) + 16;
}

template <typename T, int KIND>
__global__ void __launch_bounds__(HK_NT, 2) hex_chunk_kernel(ChunkArgs<T> a)
{
    typedef KindTraits<KIND> K;
    constexpr int NIN = K::NIN, NC = K::NC, HC = CM_HC_MAX;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double *scx = reinterpret_cast<double *>(smem_raw);                          // [ne][8][3] corner coordinates of the cells
    T *scr = reinterpret_cast<T *>(scx + (size_t)CM_HC_MAX * 24);                // [8 NC][HC]
    T *sin = scr + 8 * NC * HC;                                                 // [nl][NIN]
    unsigned short *slid = reinterpret_cast<unsigned short *>(sin + CM_NL_MAX * NIN); // [ne][8]
    unsigned short *sle = slid + 8 * HC;                                        // [8 ne]
    unsigned short *sem = sle + 8 * HC;                                         // [ne]
    unsigned short *slp = sem + HC;                                             // [nl + 1]
    unsigned long long *bar = reinterpret_cast<unsigned long long *>(slp + CM_NL_MAX + 8);
    const int c = blockIdx.x, tid = threadIdx.x;
    const int e0 = a.eptr[c], ne = a.eptr[c + 1] - e0, ne8 = (ne + 7) & ~7, s0 = a.nptr[c], nl = a.nptr[c + 1] - s0;
    if (tid == 0) {
        mbar_init(bar, 1);
        const unsigned bg = 192u * ne, bl = 16u * ne8, be = 2u * ne8;
        mbar_expect_tx(bar, bg + 2 * bl + be);
        bulk_g2s(scx, a.CX + 24L * e0, bg, bar);
        bulk_g2s(slid, a.lid + 8L * e0, bl, bar);
        bulk_g2s(sle, a.lent + 8L * e0, bl, bar);
        bulk_g2s(sem, a.emat + e0, be, bar);
    }
    for (int l = tid; l < nl; l += HK_NT) {
        const long g = a.nodes[s0 + l];
        if (KIND == EK_GRADU) {
            sin[l] = a.in0[g];
        } else {
#pragma unroll
            for (int d = 0; d < 3; d++) sin[NIN * l + d] = a.in0[3 * g + d];
            if (KIND == EK_STRESS)
#pragma unroll
                for (int d = 0; d < 3; d++) sin[NIN * l + 3 + d] = a.in1[3 * g + d];
        }
    }
    for (int l = tid; l <= nl; l += HK_NT) slp[l] = a.lptr[s0 + c + l];
    __syncthreads();
    mbar_wait(bar, 0);

    // ---- phase 1: lane (cell, Gauss point)
    double gsum[3] = {0, 0, 0};
    for (int base = 0; base < 8 * ne; base += HK_NT) {
        const int pair = base + tid, el = pair >> 3, p = pair & 7;
        const bool active = pair < 8 * ne;
        const unsigned mask = __ballot_sync(0xffffffffu, active);
        if (!active) continue;
        int l[8];
        {
            const uint4 q = *reinterpret_cast<const uint4 *>(slid + 8 * el);
            l[0] = q.x & 0xffff; l[1] = q.x >> 16; l[2] = q.y & 0xffff; l[3] = q.y >> 16;
            l[4] = q.z & 0xffff; l[5] = q.z >> 16; l[6] = q.w & 0xffff; l[7] = q.w >> 16;
        }
        double X[8][3], phid[8], gd[8][3];
#pragma unroll
        for (int k = 0; k < 4; k++) { // the cell's 24 words as twelve 128-bit loads, the same addresses in its eight lanes
            const double2 q0 = *reinterpret_cast<const double2 *>(scx + 24 * el + 6 * k);
            const double2 q1 = *reinterpret_cast<const double2 *>(scx + 24 * el + 6 * k + 2);
            const double2 q2 = *reinterpret_cast<const double2 *>(scx + 24 * el + 6 * k + 4);
            X[2 * k][0] = q0.x; X[2 * k][1] = q0.y; X[2 * k][2] = q1.x;
            X[2 * k + 1][0] = q1.y; X[2 * k + 1][1] = q2.x; X[2 * k + 1][2] = q2.y;
        }
        const T det = (T)hex_point(X, p, phid, gd);
        const unsigned em = sem[el];
        T ph[8], w[NC], cc[8][NC], out[NC];
#pragma unroll
        for (int k = 0; k < 8; k++) ph[k] = (T)phid[k];
        constexpr bool RANK1 = KIND == EK_GRADU || KIND == EK_STRESS;
        if (KIND == EK_MS) {
            T mt[3] = {0, 0, 0};
#pragma unroll
            for (int k = 0; k < 8; k++)
#pragma unroll
                for (int d = 0; d < 3; d++) mt[d] += ph[k] * sin[3 * l[k] + d];
#pragma unroll
            for (int d = 0; d < 3; d++) mt[d] -= (T)a.mbar[d];
#pragma unroll
            for (int k = 0; k < 8; k++) cc[k][0] = det * ((T)gd[k][0] * mt[0] + (T)gd[k][1] * mt[1] + (T)gd[k][2] * mt[2]);
        } else if (KIND == EK_GRADU) {
            T gU[3] = {0, 0, 0};
#pragma unroll
            for (int k = 0; k < 8; k++)
#pragma unroll
                for (int d = 0; d < 3; d++) gU[d] += sin[l[k]] * (T)gd[k][d];
#pragma unroll
            for (int d = 0; d < 3; d++) {
                w[d < NC ? d : 0] = det * gU[d];
                gsum[d] += (double)(det * gU[d]);   // sum_a phi_a = 1: the cell's share of int grad U_h
            }
        } else {
            T eps[6] = {0, 0, 0, 0, 0, 0}, sg[6] = {0, 0, 0, 0, 0, 0};
            if (em & 1u) {
#pragma unroll
                for (int k = 0; k < 8; k++) {
                    const T *wk = sin + NIN * l[k] + (KIND == EK_STRESS ? 3 : 0);
                    const T mk[3] = {wk[0], wk[1], wk[2]};
                    T ek[6];
                    E0_sim(a.rot, mk, a.l1, a.l2, ek);
#pragma unroll
                    for (int q = 0; q < 6; q++) eps[q] += ph[k] * ek[q];
                }
                if (KIND == EK_STRESS) {
                    T H[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
#pragma unroll
                    for (int k = 0; k < 8; k++)
#pragma unroll
                        for (int x = 0; x < 3; x++)
#pragma unroll
                            for (int y = 0; y < 3; y++) H[x][y] += sin[NIN * l[k] + x] * (T)gd[k][y];
                    const T E[6] = {H[0][0], H[1][1], H[2][2], H[1][2] + H[2][1], H[0][2] + H[2][0], H[0][1] + H[1][0]};
#pragma unroll
                    for (int q = 0; q < 6; q++) eps[q] = E[q] - eps[q];
                }
                C_times(a.Cstar + 36 * (em >> 1), eps, sg);
            }
            if (KIND == EK_MECH) {
                if (a.has_sext)
#pragma unroll
                    for (int q = 0; q < 6; q++) sg[q] += a.sext[q];
#pragma unroll
                for (int k = 0; k < 8; k++) {
                    const T gx = (T)gd[k][0], gy = (T)gd[k][1], gz = (T)gd[k][2];
                    cc[k][0] = det * (sg[0] * gx + sg[5] * gy + sg[4] * gz);
                    cc[k][1 < NC ? 1 : 0] = det * (sg[5] * gx + sg[1] * gy + sg[3] * gz);
                    cc[k][2 < NC ? 2 : 0] = det * (sg[4] * gx + sg[3] * gy + sg[2] * gz);
                }
            } else {
#pragma unroll
                for (int q = 0; q < NC; q++) w[q] = det * sg[q < 6 ? q : 0];
            }
        }
        cell_exchange<T, NC, RANK1>(mask, p, ph, w, cc, out);
#pragma unroll
        for (int x = 0; x < NC; x++) scr[(NC * p + x) * HC + el] = out[x];
    }
    __syncthreads();

    // ---- phase 2: one thread per local node, incidences in ascending cell order
    for (int l = tid; l < nl; l += HK_NT) {
        T acc[NC];
#pragma unroll
        for (int q = 0; q < NC; q++) acc[q] = 0;
        for (int q = slp[l]; q < slp[l + 1]; q++) {
            const int ent = sle[q], el = ent >> 3, k = ent & 7;
#pragma unroll
            for (int x = 0; x < NC; x++) acc[x] += scr[(NC * k + x) * HC + el];
        }
#pragma unroll
        for (int x = 0; x < NC; x++) a.hpart[(long)(s0 + l) * NC + x] = acc[x];
    }
    if (KIND == EK_GRADU) block_reduce_write<3>(gsum, a.partial);
}

template <typename T, int KIND>
static int launch_hex(System<T> *S, const ChunkArgs<T> &a, cudaStream_t st, int *grid_out = nullptr)
{
    constexpr size_t smem = hex_smem_bytes<KIND, T>();
    CM_CUDA(cudaFuncSetAttribute(hex_chunk_kernel<T, KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    hex_chunk_kernel<T, KIND><<<S->mesh->ck.nchunks, HK_NT, smem, st>>>(a);
    if (grid_out) *grid_out = S->mesh->ck.nchunks;
    return CM_OK;
}

template <typename T>
int sys_rhs_ms(System<T> *S, const T *m_lib, T *b, cudaStream_t st)
{
    const Chunks &K = S->mesh->ck;
    ChunkArgs<T> a = chunk_args(S);
    a.in0 = m_lib;
    S->prof.begin(CM_PROF_ELEMENT, st, 2);
    if (S->mesh->nen == 8) CM_TRY((launch_hex<T, EK_MS>(S, a, st)));
    else CM_TRY((launch_chunks<T, EK_MS>(S, a, st)));
    node_gather_kernel<T, 1><<<nblk(S->N), BS, 0, st>>>(S->N, K.d_ns_ptr, K.d_ns_slot, S->hpart, nullptr, S->pin, b);
    S->prof.end(st);
    LAUNCH_CHECK();
    return CM_OK;
}

// node pass of S5 (and the mean of grad U) from slot partials of `hs` words per slot; nparts per-block sums of V grad U in S->red
template <typename T>
static int demag_node_pass(System<T> *S, unsigned terms, int nparts, int hs, T *hd, cudaStream_t st)
{
    const Chunks &K = S->mesh->ck;
    if (terms & CM_TERM_DEMAG) reduce_final_kernel<<<1, 1024, 0, st>>>(nparts, 3, S->red, 1.0 / S->Vtot, S->dscal + 3);
    const double *n = S->Nd;
    node_hd_kernel<T><<<nblk(S->N), BS, 0, st>>>(S->N, K.d_ns_ptr, K.d_ns_slot, S->hpart, S->mL, S->dscal, terms, n[0], n[1], n[2], n[3],
                                                 n[4], n[5], n[6], n[7], n[8], (T)(S->mesh->nen == 8 ? 1 : 4), hs, hd);
    return CM_OK;
}

template <typename T>
int sys_demag_field(System<T> *S, const T *U_lib, unsigned terms, T *hd, cudaStream_t st)
{
    const Chunks &K = S->mesh->ck;
    S->prof.begin(CM_PROF_ELEMENT, st, (terms & CM_TERM_DEMAG) ? 3 : 1);
    int nparts = K.nchunks;
    if (terms & CM_TERM_DEMAG) {
        ChunkArgs<T> a = chunk_args(S);
        a.in0 = U_lib;
        if (S->mesh->nen == 8) CM_TRY((launch_hex<T, EK_GRADU>(S, a, st, &nparts)));
        else CM_TRY((launch_chunks<T, EK_GRADU>(S, a, st)));
    }
    CM_TRY(demag_node_pass(S, terms, nparts, 3, hd, st));
    S->prof.end(st);
    LAUNCH_CHECK();
    return CM_OK;
}

// S5 and S8 of the state (U, u, w) in one element pass (tetrahedra): h_d into hd, the stress partials stay in S->hpart
// (9 words per slot, the stress in words 3..8) for the sys_field call that follows
template <typename T>
int sys_demag_stress(System<T> *S, const T *U_lib, const T *u_lib, const T *w_lib, unsigned terms, T *hd, cudaStream_t st)
{
    ChunkArgs<T> a = chunk_args(S);
    a.in0 = u_lib; a.in1 = w_lib; a.in2 = U_lib;
    S->prof.begin(CM_PROF_ELEMENT, st, 3);
    CM_TRY((launch_chunks<T, EK_GRADU_STRESS>(S, a, st)));
    CM_TRY(demag_node_pass(S, terms, S->mesh->ck.nchunks, 9, hd, st));
    S->prof.end(st);
    LAUNCH_CHECK();
    S->sig_hs = 9; S->sig_ho = 3;
    return CM_OK;
}

template <typename T>
int sys_rhs_mech(System<T> *S, const T *m_lib, T *b, cudaStream_t st)
{
    const Chunks &K = S->mesh->ck;
    if (!S->n_elastic) { cm_set_error("mechanics requested but the material has no elastic constants"); return CM_E_BADARG; }
    ChunkArgs<T> a = chunk_args(S);
    a.in0 = m_lib;
    S->prof.begin(CM_PROF_ELEMENT, st, 2);
    if (S->mesh->nen == 8) CM_TRY((launch_hex<T, EK_MECH>(S, a, st)));
    else CM_TRY((launch_chunks<T, EK_MECH>(S, a, st)));
    node_gather_kernel<T, 3><<<nblk(S->N), BS, 0, st>>>(S->N, K.d_ns_ptr, K.d_ns_slot, S->hpart, S->clamp, -1, b);
    S->prof.end(st);
    LAUNCH_CHECK();
    return CM_OK;
}

template <typename T>
int sys_stress(System<T> *S, const T *u_lib, const T *w_lib, cudaStream_t st)
{
    if (!S->n_elastic) { cm_set_error("mechanics requested but the material has no elastic constants"); return CM_E_BADARG; }
    ChunkArgs<T> a = chunk_args(S);
    a.in0 = u_lib; a.in1 = w_lib;
    S->prof.begin(CM_PROF_ELEMENT, st);
    if (S->mesh->nen == 8) CM_TRY((launch_hex<T, EK_STRESS>(S, a, st)));
    else CM_TRY((launch_chunks<T, EK_STRESS>(S, a, st)));
    S->prof.end(st);
    LAUNCH_CHECK();
    S->sig_hs = 6; S->sig_ho = 0;
    return CM_OK;
}

template <typename T>
int sys_field(System<T> *S, const T *w_lib, const T *hd, const double hext[3], unsigned terms, T *h, T *sig_out, cudaStream_t st,
              const double *hext_dev)
{
    const Chunks &K = S->mesh->ck;
    S->prof.begin(CM_PROF_ELEMENT, st);
    node_field_kernel<T><<<nblk(S->N), BS, 0, st>>>(S->N, K.d_ns_ptr, K.d_ns_slot, S->hpart + S->sig_ho, S->mLm, S->live, w_lib, hd, terms,
                                                   (T)(2.0 * S->Kstar), (T)hext[0], (T)hext[1], (T)hext[2], hext_dev, (T)S->lam100,
                                                   (T)S->lam111, make_rot<T>(S), (T)(S->mesh->nen == 8 ? 1 : 4), S->sig_hs, h, sig_out);
    S->prof.end(st);
    LAUNCH_CHECK();
    return CM_OK;
}

template <typename T>
int sys_axpby3(System<T> *S, const T *base, const T *h, T c, T *f, cudaStream_t st)
{
    S->prof.begin(CM_PROF_POINTWISE, st);
    axpby_kernel<T><<<nblk(3 * S->N), BS, 0, st>>>(S->N, base, h, c, f);
    S->prof.end(st);
    LAUNCH_CHECK();
    return CM_OK;
}

// ------------------------------------------------------------------------------------------------
// one GSPM step (O-3)
// ------------------------------------------------------------------------------------------------
template <typename T>
static int step_check(System<T> *S, const cm_step_params *p, const T *m_user, const T *U_user, const T *u_user, const char *fn)
{
    const unsigned terms = p->terms;
    if (p->dt != S->dt) { cm_set_error("%s: params->dt differs from the dt given to cm_assemble_csr", fn); return CM_E_BADARG; }
    if ((terms & CM_TERM_MAGEL) && !S->n_elastic) { cm_set_error("%s: MAGEL needs elastic constants", fn); return CM_E_BADARG; }
    if (p->mech_matfree && (terms & CM_TERM_MAGEL) && S->mesh->nen != 4) { cm_set_error("%s: mech_matfree is built for tetrahedra", fn); return CM_E_BADARG; }
    if (p->cg_precond != CM_PC_NONE && p->cg_precond != CM_PC_JACOBI) { cm_set_error("%s: unknown cg_precond %d", fn, p->cg_precond); return CM_E_BADARG; }
    if (((terms & CM_TERM_DEMAG) && !U_user) || ((terms & CM_TERM_MAGEL) && !u_user) || !m_user) {
        cm_set_error("%s: null field pointer", fn);
        return CM_E_BADARG;
    }
    return CM_OK;
}

// Items 1-10 of O-3 on the library-order state S->m, S->U, S->u.  hext_dev != NULL: the nondimensional applied field is
// read from device memory (3 doubles) by the field kernels instead of params->Hext, so that the same enqueued work --
// or a captured graph of it -- follows a field that changes on the device.  Ends with <||dm||> in S->dscal[6].
template <typename T>
static int step_core(System<T> *S, const cm_step_params *p, const double *hext_dev, cudaStream_t st)
{
    const long N = S->N;
    const unsigned terms = p->terms;
    const double hext[3] = {p->Hext[0] / S->Ms, p->Hext[1] / S->Ms, p->Hext[2] / S->Ms};
    const T dtau = (T)S->dtau, adtau = (T)(S->alpha * S->dtau);
    const double tol = p->cg_tol;
    const int mx = p->cg_maxiter, fx = p->cg_fixed_iters, pc = p->cg_precond;
    CM_CUDA(cudaMemsetAsync(S->d_res, 0, 8 * sizeof(CgResult), st));
    // 1. mbar (Eq. 17)
    CM_TRY(sys_mbar(S, S->m, st));
    // 2. magnetostatic solve, warm start (Eq. 5, 9)
    if (terms & CM_TERM_DEMAG) {
        CM_TRY(sys_rhs_ms(S, S->m, S->bvec, st));
        CM_TRY(sys_cg(S, CM_MAT_K_MS, MODE_CSR1, S->bvec, S->U, tol, mx, fx, 1u, 0, CM_PROF_CG_MS, pc, st));
    }
    // 3. demagnetising field (Eq. 4); with mechanics on a tetrahedral mesh S5 waits for S8 and shares its element pass
    const bool fuse = (terms & CM_TERM_DEMAG) && (terms & CM_TERM_MAGEL) && S->mesh->nen == 4 && !S->no_fuse;
    if ((terms & (CM_TERM_DEMAG | CM_TERM_FARFIELD)) && !fuse) CM_TRY(sys_demag_field(S, S->U, terms, S->hd, st));
    // 4. mechanical equilibrium (Eq. 6, 10), warm start; stress at m^n
    if (terms & CM_TERM_MAGEL) {
        CM_TRY(sys_rhs_mech(S, S->m, S->bvec, st));
        if (p->mech_matfree) CM_TRY(sys_cg_matfree(S, S->bvec, S->u, tol, mx, fx, pc, 1, st));
        else CM_TRY(sys_cg(S, CM_MAT_K_MECH, MODE_BSR3, S->bvec, S->u, tol, mx, fx, 1u, 1, CM_PROF_CG_MECH, pc, st));
        if (fuse) CM_TRY(sys_demag_stress(S, S->U, S->u, S->m, terms, S->hd, st));
        else CM_TRY(sys_stress(S, S->u, S->m, st));
    }
    // 5. h[m^n];  6. Step 1: g^n.  A Helmholtz solve is ONE launch: b = M_m f, x0 = f, r0 = b - A f in its first pass
    CM_TRY(sys_field(S, S->m, S->hd, hext, terms, S->hn, (T *)nullptr, st, hext_dev));
    CM_TRY(sys_axpby3(S, S->m, S->hn, dtau, S->f, st));
    CM_TRY(sys_helmholtz(S, CM_MAT_K_GS1, S->f, S->gn, tol, mx, fx, p->gspm_variant == 1 ? 6u : 7u, 2, pc, st));
    // 7. Step 2 interleaved with the g* solves
    S->prof.begin(CM_PROF_POINTWISE, st);
    gs_step2_kernel<T><<<nblk(N), BS, 0, st>>>(N, p->gspm_variant, 0, S->m, S->gn, S->gs, S->hn, dtau, S->ms, S->f);
    S->prof.end(st);
    LAUNCH_CHECK();
    if (p->gspm_variant == 0) {
        CM_TRY(sys_helmholtz(S, CM_MAT_K_GS1, S->f, S->gs, tol, mx, fx, 3u, 3, pc, st));
    } else {
        CM_TRY(sys_helmholtz(S, CM_MAT_K_GS1, S->f, S->gs, tol, mx, fx, 1u, 3, pc, st));
        S->prof.begin(CM_PROF_POINTWISE, st);
        gs_step2_kernel<T><<<nblk(N), BS, 0, st>>>(N, 1, 1, S->m, S->gn, S->gs, S->hn, dtau, S->ms, S->f);
        S->prof.end(st);
        LAUNCH_CHECK();
        // x0 = f for component 2 only (component 1 already holds g*_1): the solve writes the masked components
        CM_TRY(sys_helmholtz(S, CM_MAT_K_GS1, S->f, S->gs, tol, mx, fx, 2u, 4, pc, st));
    }
    S->prof.begin(CM_PROF_POINTWISE, st);
    gs_step2c_kernel<T><<<nblk(N), BS, 0, st>>>(N, S->m, S->gs, S->ms);
    S->prof.end(st);
    LAUNCH_CHECK();
    // 8. Step 3: h* = h[m*] with U, u frozen (R3)
    if (terms & CM_TERM_MAGEL) CM_TRY(sys_stress(S, S->u, S->ms, st));
    CM_TRY(sys_field(S, S->ms, S->hd, hext, terms, S->hn, (T *)nullptr, st, hext_dev));
    CM_TRY(sys_axpby3(S, S->ms, S->hn, adtau, S->f, st));
    CM_TRY(sys_helmholtz(S, CM_MAT_K_GS2, S->f, S->mss, tol, mx, fx, 7u, 5, pc, st));
    // 9. Step 4 projection; 10. diagnostics
    {
        const int nb = (int)std::min<long>(RED_BLOCKS, nblk(N));
        S->prof.begin(CM_PROF_POINTWISE, st, 2);
        project_kernel<T><<<nb, BS, 0, st>>>(N, S->live, S->mss, S->m, S->red);
        reduce_final_kernel<<<1, 1024, 0, st>>>(nb, 1, S->red, S->nlive ? 1.0 / (double)S->nlive : 0.0, S->dscal + 6);
        S->prof.end(st);
        LAUNCH_CHECK();
    }
    return CM_OK;
}

template <typename T>
int sys_step(System<T> *S, const cm_step_params *p, T *m_user, T *U_user, T *u_user, cm_step_info *info, cudaStream_t st)
{
    const unsigned terms = p->terms;
    CM_TRY(step_check(S, p, m_user, U_user, u_user, "cm_gspm_step"));
    CM_TRY(sys_permute_in(S, m_user, S->m, 3, st));
    if (terms & CM_TERM_DEMAG) CM_TRY(sys_permute_in(S, U_user, S->U, 1, st));
    if (terms & CM_TERM_MAGEL) CM_TRY(sys_permute_in(S, u_user, S->u, 3, st));
    CM_TRY(step_core(S, p, (const double *)nullptr, st));
    CM_TRY(sys_permute_out(S, S->m, m_user, 3, st));
    if (terms & CM_TERM_DEMAG) CM_TRY(sys_permute_out(S, S->U, U_user, 1, st));
    if (terms & CM_TERM_MAGEL) CM_TRY(sys_permute_out(S, S->u, u_user, 3, st));

    int worst = CM_OK;
    if (info) {
        CM_CUDA(cudaMemcpyAsync(S->h_res, S->d_res, 8 * sizeof(CgResult), cudaMemcpyDeviceToHost, st));
        CM_CUDA(cudaMemcpyAsync(S->h_scal, S->dscal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CM_CUDA(cudaStreamSynchronize(st));
        std::memset(info, 0, sizeof(*info));
        const CgResult *R = S->h_res;
        info->it_ms = R[0].iters[0]; info->res_ms = R[0].relres[0];
        info->it_mech = R[1].iters[0]; info->res_mech = R[1].relres[0];
        for (int a = 0; a < 3; a++) { info->it_gs[a] = R[2].iters[a]; info->res_gs[a] = R[2].relres[a]; }
        if (p->gspm_variant == 0) {
            for (int a = 0; a < 2; a++) { info->it_gs[3 + a] = R[3].iters[a]; info->res_gs[3 + a] = R[3].relres[a]; }
        } else {
            info->it_gs[3] = R[3].iters[0]; info->res_gs[3] = R[3].relres[0];
            info->it_gs[4] = R[4].iters[1]; info->res_gs[4] = R[4].relres[1];
        }
        for (int a = 0; a < 3; a++) { info->it_gs[5 + a] = R[5].iters[a]; info->res_gs[5 + a] = R[5].relres[a]; }
        for (int d = 0; d < 3; d++) info->mbar[d] = S->h_scal[d];
        info->mean_dm = S->h_scal[6];
        info->energy = std::numeric_limits<double>::quiet_NaN();
        for (int s = 0; s < 6; s++) worst = std::min(worst, R[s].status);
        // profiler bookkeeping of CG work
        // (a launch makes one matrix pass per iteration plus the r0 = b - A x0 pass)
        S->prof.cg_iters[CM_PROF_CG_MS] += R[0].iters[0];
        if (terms & CM_TERM_DEMAG) S->prof.cg_passes[CM_PROF_CG_MS] += R[0].iters[0] + 1;
        S->prof.cg_iters[CM_PROF_CG_MECH] += R[1].iters[0];
        if (terms & CM_TERM_MAGEL) S->prof.cg_passes[CM_PROF_CG_MECH] += R[1].iters[0] + 1;
        for (int s = 2; s < 6; s++) {
            if (s == 4 && p->gspm_variant == 0) continue; // slot 4 is used by variant 1 only
            int mxit = 0;
            for (int a = 0; a < 3; a++) { S->prof.cg_iters[CM_PROF_CG_GS] += R[s].iters[a]; mxit = std::max(mxit, R[s].iters[a]); }
            S->prof.cg_passes[CM_PROF_CG_GS] += mxit + 1;
        }
    }
    return worst;
}

// ------------------------------------------------------------------------------------------------
// hysteresis driver (R24): the whole loop on the device
// ------------------------------------------------------------------------------------------------
struct HystCtl {
    double H[3], hnd[3];      // current field (A/m) and H / Ms, read by the field kernels
    double H0[3], dH[3], e0[3], Ms, conv_tol;
    int k, steps, done, reversed, max_fields, max_steps, worst, variant;
    long total, it_ms, it_mech, gs_passes;
};

// One thread, after every step: dscal[0..2] = volume average of the NEW m, dscal[6] = <||dm||>.
__global__ void hyst_control_kernel(HystCtl *c, const double *__restrict__ dscal, const CgResult *__restrict__ R, double *log, int *slog,
                                    int cap, cudaGraphConditionalHandle handle)
{
    if (threadIdx.x || blockIdx.x) return;
    c->steps++;
    c->total++;
    c->it_ms += R[0].iters[0];
    c->it_mech += R[1].iters[0];
    for (int s = 2; s < 6; s++) c->gs_passes += max(R[s].iters[0], max(R[s].iters[1], R[s].iters[2]));
    for (int s = 0; s < 6; s++) c->worst = min(c->worst, R[s].status);
    if (dscal[6] < c->conv_tol || c->steps >= c->max_steps) {
        const int k = c->k;
        for (int d = 0; d < 3; d++) { log[3 * k + d] = c->H[d]; log[3 * (cap + k) + d] = dscal[d]; }
        slog[k] = c->steps;
        const double proj = dscal[0] * c->e0[0] + dscal[1] * c->e0[1] + dscal[2] * c->e0[2];
        if (proj < 0) { c->reversed = 1; c->done = 1; }
        else if (k + 1 >= c->max_fields) c->done = 1;
        c->k = k + 1;
        if (!c->done) {
            c->steps = 0;
            for (int d = 0; d < 3; d++) {
                c->H[d] = __dadd_rn(c->H0[d], __dmul_rn((double)(k + 1), c->dH[d])); // H0 + k dH, product rounded first (no FMA)
                c->hnd[d] = c->H[d] / c->Ms;
            }
        }
    }
    cudaGraphSetConditional(handle, c->done ? 0u : 1u);
}

template <typename T>
int sys_hysteresis(System<T> *S, const cm_step_params *base, const cm_hyst_params *hp, T *m_user, T *U_user, T *u_user, double *H_log,
                   double *mbar_log, int *steps_log, cm_hyst_result *res, cudaStream_t st)
{
    const unsigned terms = base->terms;
    CM_TRY(step_check(S, base, m_user, U_user, u_user, "cm_hysteresis_run"));
    if (base->mech_matfree) { cm_set_error("cm_hysteresis_run: the matrix-free mechanical solve synchronises the stream and cannot be captured"); return CM_E_BADARG; }
    const double n0 = std::sqrt(hp->H0[0] * hp->H0[0] + hp->H0[1] * hp->H0[1] + hp->H0[2] * hp->H0[2]);
    if (!(n0 > 0) || hp->max_fields < 1 || hp->max_steps < 1 || !H_log || !mbar_log || !steps_log || !res) {
        cm_set_error("cm_hysteresis_run: H0 must be non-zero, max_fields and max_steps positive, outputs non-null");
        return CM_E_BADARG;
    }
    const int cap = hp->max_fields;
    if (!S->hyst_ctl) CM_CUDA(cudaMalloc(&S->hyst_ctl, sizeof(HystCtl)));
    if (S->hyst_cap < cap) {
        cudaFree(S->hyst_log); cudaFree(S->hyst_steps);
        S->hyst_log = nullptr; S->hyst_steps = nullptr; S->hyst_cap = 0;
        CM_CUDA(cudaMalloc((void **)&S->hyst_log, (size_t)cap * 6 * sizeof(double)));
        CM_CUDA(cudaMalloc((void **)&S->hyst_steps, (size_t)cap * sizeof(int)));
        S->hyst_cap = cap;
    }
    HystCtl h0;
    std::memset(&h0, 0, sizeof(h0));
    for (int d = 0; d < 3; d++) {
        h0.H[d] = h0.H0[d] = hp->H0[d]; h0.dH[d] = hp->dH[d]; h0.e0[d] = hp->H0[d] / n0; h0.hnd[d] = hp->H0[d] / S->Ms;
    }
    h0.Ms = S->Ms; h0.conv_tol = hp->conv_tol; h0.max_fields = hp->max_fields; h0.max_steps = hp->max_steps; h0.worst = CM_OK;
    HystCtl *ctl = (HystCtl *)S->hyst_ctl;
    CM_CUDA(cudaMemcpyAsync(ctl, &h0, sizeof(h0), cudaMemcpyHostToDevice, st));
    CM_CUDA(cudaMemsetAsync(S->hyst_log, 0, (size_t)cap * 6 * sizeof(double), st));
    CM_CUDA(cudaMemsetAsync(S->hyst_steps, 0, (size_t)cap * sizeof(int), st));
    CM_TRY(sys_permute_in(S, m_user, S->m, 3, st));
    if (terms & CM_TERM_DEMAG) CM_TRY(sys_permute_in(S, U_user, S->U, 1, st));
    if (terms & CM_TERM_MAGEL) CM_TRY(sys_permute_in(S, u_user, S->u, 3, st));
    CM_CUDA(cudaStreamSynchronize(st)); // h0 is on this stack frame

    // ---- graph: WHILE (not done) { one GSPM step; average of the new m; controller }
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    const bool prof_on = S->prof.on;
    S->prof.on = false; // no event records inside a conditional body
    cudaStream_t cs = nullptr; // capture stream: the caller's may be the legacy default stream, which cannot capture
    auto build = [&]() -> int {
        CM_CUDA(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
        CM_CUDA(cudaGraphCreate(&graph, 0));
        cudaGraphConditionalHandle handle;
        CM_CUDA(cudaGraphConditionalHandleCreate(&handle, graph, 1, cudaGraphCondAssignDefault));
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = handle;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        cudaGraphNode_t node;
        CM_CUDA(cudaGraphAddNode(&node, graph, nullptr, 0, &np));
        cudaGraph_t body = np.conditional.phGraph_out[0];
        CM_CUDA(cudaStreamBeginCaptureToGraph(cs, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
        int rc = step_core(S, base, ctl->hnd, cs);
        if (rc == CM_OK) rc = sys_mbar(S, S->m, cs);
        if (rc == CM_OK) {
            hyst_control_kernel<<<1, 32, 0, cs>>>(ctl, S->dscal, S->d_res, S->hyst_log, S->hyst_steps, cap, handle);
            if (cudaGetLastError() != cudaSuccess) rc = CM_E_CUDA;
        }
        cudaGraph_t captured = nullptr;
        cudaError_t e = cudaStreamEndCapture(cs, &captured);
        if (rc != CM_OK) return rc;
        if (e != cudaSuccess) { cm_set_error("cm_hysteresis_run: stream capture failed: %s", cudaGetErrorString(e)); return CM_E_CUDA; }
        CM_CUDA(cudaGraphInstantiate(&exec, graph, 0));
        return CM_OK;
    };
    int rc = build();
    S->prof.on = prof_on;
    cudaEvent_t ea = nullptr, eb = nullptr;
    auto run = [&]() -> int {
        CM_CUDA(cudaEventCreate(&ea));
        CM_CUDA(cudaEventCreate(&eb));
        CM_CUDA(cudaEventRecord(ea, st));
        CM_CUDA(cudaGraphLaunch(exec, st));
        CM_CUDA(cudaEventRecord(eb, st));
        CM_TRY(sys_permute_out(S, S->m, m_user, 3, st));
        if (terms & CM_TERM_DEMAG) CM_TRY(sys_permute_out(S, S->U, U_user, 1, st));
        if (terms & CM_TERM_MAGEL) CM_TRY(sys_permute_out(S, S->u, u_user, 3, st));
        HystCtl hr;
        std::vector<double> lg((size_t)cap * 6);
        CM_CUDA(cudaMemcpyAsync(&hr, ctl, sizeof(hr), cudaMemcpyDeviceToHost, st));
        CM_CUDA(cudaMemcpyAsync(lg.data(), S->hyst_log, lg.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
        CM_CUDA(cudaMemcpyAsync(steps_log, S->hyst_steps, (size_t)cap * sizeof(int), cudaMemcpyDeviceToHost, st));
        CM_CUDA(cudaStreamSynchronize(st));
        float ms = 0;
        CM_CUDA(cudaEventElapsedTime(&ms, ea, eb));
        std::memcpy(H_log, lg.data(), (size_t)cap * 3 * sizeof(double));
        std::memcpy(mbar_log, lg.data() + (size_t)cap * 3, (size_t)cap * 3 * sizeof(double));
        res->n_fields = hr.k; res->reversed = hr.reversed; res->total_steps = hr.total;
        res->cg_iters_ms = hr.it_ms; res->cg_iters_mech = hr.it_mech; res->cg_passes_gs = hr.gs_passes;
        res->worst_cg_status = hr.worst; res->device_ms = ms;
        return hr.worst;
    };
    if (rc == CM_OK) rc = run();
    if (ea) cudaEventDestroy(ea);
    if (eb) cudaEventDestroy(eb);
    if (exec) cudaGraphExecDestroy(exec);
    if (cs) cudaStreamDestroy(cs);
    if (graph) cudaGraphDestroy(graph);
    return rc;
}

// ------------------------------------------------------------------------------------------------
// matrix-free K^mech (the paper's future work: "assembles and stores sparse matrices explicitly")
// ------------------------------------------------------------------------------------------------
// y = (P K P + (I - P)) x applied as an element pass (EK_KMECH: strain of x, stress, nodal forces per chunk slot) and a node
// pass (slots summed in ascending chunk order; a clamped DOF returns x).  The CG around it is a sequence of four launches per
// iteration on one stream; the scalars live in a double-buffered device state that every block re-reduces from per-block
// partials in a fixed order (bit-reproducible), and a finished solve turns the remaining launches of a batch into no-ops.
namespace {

constexpr int MF_GRID = 1024, MF_BS = 256, MF_BATCH = 16;

struct MfState {
    double rr, bb, rz;
    int iters, done, status, zero_rhs;
};

// sum over the MF_GRID per-block partials of component c (fixed order, the same bits in every block)
template <int NV>
__device__ __forceinline__ void mf_reduce(const double *partial, double (&out)[NV])
{
    __shared__ double sh[NV * 32];
    double v[NV];
#pragma unroll
    for (int c = 0; c < NV; c++) v[c] = 0;
    for (int j = threadIdx.x; j < MF_GRID; j += blockDim.x)
#pragma unroll
        for (int c = 0; c < NV; c++) v[c] += __ldcg(partial + (long)j * NV + c);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int c = 0; c < NV; c++)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    __syncthreads();
    if (lane == 0)
#pragma unroll
        for (int c = 0; c < NV; c++) sh[c * 32 + warp] = v[c];
    __syncthreads();
#pragma unroll
    for (int c = 0; c < NV; c++) {
        double t = 0;
        for (int w = 0; w < nwarp; w++) t += sh[c * 32 + w];
        out[c] = t;
    }
    __syncthreads();
}

template <int NV>
__device__ __forceinline__ void mf_block_partial(double (&v)[NV], double *partial)
{
    __shared__ double sh[NV * 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
#pragma unroll
    for (int c = 0; c < NV; c++)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    __syncthreads();
    if (lane == 0)
#pragma unroll
        for (int c = 0; c < NV; c++) sh[c * 32 + warp] = v[c];
    __syncthreads();
    if (threadIdx.x == 0)
#pragma unroll
        for (int c = 0; c < NV; c++) {
            double t = 0;
            for (int w = 0; w < nwarp; w++) t += sh[c * 32 + w];
            partial[(long)blockIdx.x * NV + c] = t;
        }
}

// node pass of the operator.  MODE 0: y = A x.  MODE 1 (start of a solve): r = b - A x, p = z = r or r / D, partials
// (rr, bb, rz).  MODE 2 (iteration): y = A x with partial x . y.
template <typename T, int MODE, bool PRE>
__global__ void __launch_bounds__(MF_BS) mf_apply_kernel(long N, const int *__restrict__ ns_ptr, const int *__restrict__ ns_slot,
                                                          const T *__restrict__ hpart, const uchar *__restrict__ clamp, const T *__restrict__ x,
                                                          T *y, const T *__restrict__ b, const T *__restrict__ D, T *r, double *partial,
                                                          const MfState *st)
{
    if (MODE == 2 && st->done) return;
    double acc3[3] = {0, 0, 0};
    for (long i = blockIdx.x * (long)blockDim.x + threadIdx.x; i < N; i += (long)gridDim.x * blockDim.x) {
        T a[3] = {0, 0, 0};
        for (int s = ns_ptr[i]; s < ns_ptr[i + 1]; s++) {
            const long q = __ldg(ns_slot + s);
#pragma unroll
            for (int d = 0; d < 3; d++) a[d] += hpart[3 * q + d];
        }
#pragma unroll
        for (int d = 0; d < 3; d++) {
            const long k = 3 * i + d;
            const T xv = x[k];
            if (clamp[k]) a[d] = xv;
            if (MODE == 0) y[k] = a[d];
            if (MODE == 2) { y[k] = a[d]; acc3[0] += (double)xv * (double)a[d]; }
            if (MODE == 1) {
                const T bi = b[k], ri = bi - a[d], zi = PRE ? ri / D[k] : ri;
                r[k] = ri; y[k] = zi;
                acc3[0] += (double)ri * (double)ri; acc3[1] += (double)bi * (double)bi; acc3[2] += (double)ri * (double)zi;
            }
        }
    }
    if (MODE == 1) mf_block_partial<3>(acc3, partial);
    if (MODE == 2) { double v[1] = {acc3[0]}; mf_block_partial<1>(v, partial); }
}

// state before iteration 0: the stopping test of the textbook loop (O-4), zero right-hand side
__global__ void mf_init_state_kernel(const double *partial, double tol, int maxiter, int fixed, MfState *st)
{
    double v[3];
    mf_reduce<3>(partial, v);
    if (threadIdx.x) return;
    MfState s;
    s.rr = v[0]; s.bb = v[1]; s.rz = v[2]; s.iters = 0; s.done = 0; s.status = CM_OK; s.zero_rhs = 0;
    if (s.bb == 0.0 && fixed < 0) { s.zero_rhs = 1; s.rr = 0; s.done = 1; }
    else if (s.rr == 0.0) s.done = 1;
    else if (fixed >= 0) { if (fixed == 0) s.done = 1; }
    else if (s.rr < tol * tol * s.bb) s.done = 1;
    else if (maxiter <= 0) { s.done = 1; s.status = CM_E_CG_MAXITER; }
    st[0] = s;
}

template <typename T>
__global__ void mf_zero_x_kernel(long n, T *x, const MfState *st)
{
    if (!st->zero_rhs) return;
    for (long k = blockIdx.x * (long)blockDim.x + threadIdx.x; k < n; k += (long)gridDim.x * blockDim.x) x[k] = 0;
}

// alpha = rz / pAp; x += alpha p; r -= alpha Ap; partials (rr, rz) of the new residual
template <typename T, bool PRE>
__global__ void __launch_bounds__(MF_BS) mf_update_kernel(long n, const T *__restrict__ p, const T *__restrict__ Ap, const T *__restrict__ D, T *x,
                                                           T *r, const double *pap_partial, double *partial, const MfState *st)
{
    if (st->done) return;
    double pap[1];
    mf_reduce<1>(pap_partial, pap);
    double acc[2] = {0, 0};
    if (pap[0] > 0.0) {
        const T alpha = (T)(st->rz / pap[0]);
        for (long k = blockIdx.x * (long)blockDim.x + threadIdx.x; k < n; k += (long)gridDim.x * blockDim.x) {
            x[k] = fma(alpha, p[k], x[k]);
            const T ri = fma(-alpha, Ap[k], r[k]);
            r[k] = ri;
            acc[0] += (double)ri * (double)ri;
            acc[1] += (double)ri * (double)(PRE ? ri / D[k] : ri);
        }
    }
    mf_block_partial<2>(acc, partial);
}

// beta = rz_new / rz; p = z + beta p; next state with the stopping test before the next iteration
template <typename T, bool PRE>
__global__ void __launch_bounds__(MF_BS) mf_p_kernel(long n, const T *__restrict__ r, const T *__restrict__ D, T *p, const double *pap_partial,
                                                      const double *partial, double tol, int maxiter, int fixed, const MfState *st, MfState *nxt)
{
    if (st->done) {
        if (blockIdx.x == 0 && threadIdx.x == 0) *nxt = *st;
        return;
    }
    double pap[1], v[2];
    mf_reduce<1>(pap_partial, pap);
    mf_reduce<2>(partial, v);
    const bool breakdown = !(pap[0] > 0.0);
    MfState s = *st;
    if (breakdown) { s.done = 1; s.status = CM_E_CG_BREAKDOWN; }
    else {
        const T beta = (T)(v[1] / s.rz);
        s.rr = v[0]; s.rz = v[1]; s.iters += 1;
        if (s.rr == 0.0) s.done = 1;
        else if (fixed >= 0) { if (s.iters == fixed) s.done = 1; }
        else if (s.rr < tol * tol * s.bb) s.done = 1;
        else if (s.iters >= maxiter) { s.done = 1; s.status = CM_E_CG_MAXITER; }
        if (!s.done)
            for (long k = blockIdx.x * (long)blockDim.x + threadIdx.x; k < n; k += (long)gridDim.x * blockDim.x)
                p[k] = fma(beta, p[k], PRE ? r[k] / D[k] : r[k]);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) *nxt = s;
}

__global__ void mf_result_kernel(const MfState *st, CgResult *out)
{
    if (threadIdx.x || blockIdx.x) return;
    for (int q = 0; q < 3; q++) { out->iters[q] = 0; out->relres[q] = 0; }
    out->iters[0] = st->iters;
    out->relres[0] = st->bb > 0 ? sqrt(st->rr / st->bb) : 0.0;
    out->status = st->status;
}

} // namespace

template <typename T>
static int mf_check(System<T> *S, const char *fn)
{
    if (!S->n_elastic) { cm_set_error("%s: the material has no elastic constants", fn); return CM_E_BADARG; }
    if (S->mesh->nen != 4) { cm_set_error("%s: the matrix-free operator is built for tetrahedra", fn); return CM_E_BADARG; }
    return CM_OK;
}

// element pass of the operator on library-order x -> S->hpart
template <typename T>
static int mf_elements(System<T> *S, const T *x, const int *skip, int prof_cls, cudaStream_t st)
{
    ChunkArgs<T> a = chunk_args(S);
    a.in0 = x; a.skip = skip;
    S->prof.begin(prof_cls, st);
    CM_TRY((launch_chunks<T, EK_KMECH>(S, a, st)));
    S->prof.end(st);
    LAUNCH_CHECK();
    return CM_OK;
}

template <typename T>
int sys_spmv_matfree(System<T> *S, const T *x, T *y, cudaStream_t st)
{
    CM_TRY(mf_check(S, "cm_spmv_matfree"));
    const Chunks &K = S->mesh->ck;
    CM_TRY(mf_elements(S, x, nullptr, CM_PROF_SPMV, st));
    S->prof.begin(CM_PROF_SPMV, st);
    mf_apply_kernel<T, 0, false><<<MF_GRID, MF_BS, 0, st>>>(S->N, K.d_ns_ptr, K.d_ns_slot, S->hpart, S->clamp, x, y, nullptr, nullptr, nullptr, nullptr, nullptr);
    S->prof.end(st);
    LAUNCH_CHECK();
    return CM_OK;
}

// CG on the matrix-free operator; b, x in library order; result in S->d_res[slot].  Synchronises the stream once per
// MF_BATCH iterations (the host has to know when to stop enqueueing).
template <typename T>
int sys_cg_matfree(System<T> *S, const T *b, T *x, double tol, int maxiter, int fixed, int precond, int slot, cudaStream_t st)
{
    CM_TRY(mf_check(S, "cm_cg_solve_matfree"));
    if (precond != CM_PC_NONE && precond != CM_PC_JACOBI) { cm_set_error("unknown preconditioner %d", precond); return CM_E_BADARG; }
    const bool pre = precond == CM_PC_JACOBI;
    const Chunks &K = S->mesh->ck;
    const long N = S->N, n = 3 * N;
    MfState *ms = (MfState *)S->mf_state;
    double *part_pap = S->red, *part2 = S->red + MF_GRID, *part3 = S->red + 3 * MF_GRID;
    const T *D = S->Dmech;
    // ---- r0 = b - A x0, p0 = z0
    CM_TRY(mf_elements(S, x, nullptr, CM_PROF_CG_MECH, st));
    S->prof.begin(CM_PROF_CG_MECH, st, 3);
    if (pre) mf_apply_kernel<T, 1, true><<<MF_GRID, MF_BS, 0, st>>>(N, K.d_ns_ptr, K.d_ns_slot, S->hpart, S->clamp, x, S->p, b, D, S->r, part3, nullptr);
    else mf_apply_kernel<T, 1, false><<<MF_GRID, MF_BS, 0, st>>>(N, K.d_ns_ptr, K.d_ns_slot, S->hpart, S->clamp, x, S->p, b, D, S->r, part3, nullptr);
    mf_init_state_kernel<<<1, MF_BS, 0, st>>>(part3, tol, maxiter, fixed, ms);
    mf_zero_x_kernel<T><<<MF_GRID, MF_BS, 0, st>>>(n, x, ms);
    S->prof.end(st);
    LAUNCH_CHECK();
    MfState *hs = (MfState *)S->h_mf;
    const int cap = fixed >= 0 ? fixed : maxiter;
    int k = 0; // iterations enqueued so far: iteration j reads ms[j & 1] and writes ms[(j + 1) & 1]
    while (k < cap) {
        const int kend = std::min(cap, k + MF_BATCH);
        for (; k < kend; k++) {
            const MfState *cur = ms + (k & 1);
            MfState *nxt = ms + ((k + 1) & 1);
            CM_TRY(mf_elements(S, S->p, &cur->done, CM_PROF_CG_MECH, st));
            S->prof.begin(CM_PROF_CG_MECH, st, 3);
            mf_apply_kernel<T, 2, false><<<MF_GRID, MF_BS, 0, st>>>(N, K.d_ns_ptr, K.d_ns_slot, S->hpart, S->clamp, S->p, S->Ap, nullptr, nullptr, nullptr, part_pap, cur);
            if (pre) {
                mf_update_kernel<T, true><<<MF_GRID, MF_BS, 0, st>>>(n, S->p, S->Ap, D, x, S->r, part_pap, part2, cur);
                mf_p_kernel<T, true><<<MF_GRID, MF_BS, 0, st>>>(n, S->r, D, S->p, part_pap, part2, tol, maxiter, fixed, cur, nxt);
            } else {
                mf_update_kernel<T, false><<<MF_GRID, MF_BS, 0, st>>>(n, S->p, S->Ap, D, x, S->r, part_pap, part2, cur);
                mf_p_kernel<T, false><<<MF_GRID, MF_BS, 0, st>>>(n, S->r, D, S->p, part_pap, part2, tol, maxiter, fixed, cur, nxt);
            }
            S->prof.end(st);
            LAUNCH_CHECK();
        }
        CM_CUDA(cudaMemcpyAsync(hs, ms + (k & 1), sizeof(MfState), cudaMemcpyDeviceToHost, st));
        CM_CUDA(cudaStreamSynchronize(st));
        if (S->prof.on) CM_TRY(S->prof.flush()); // the stream is idle here: fold this batch's event pairs in, so `pending` stays bounded by one batch
        if (hs->done) break;
    }
    const int kfin = k & 1;
    mf_result_kernel<<<1, 32, 0, st>>>(ms + kfin, S->d_res + slot);
    LAUNCH_CHECK();
    return CM_OK;
}

#define INST(T)                                                                                                       \
    template int sys_permute_in<T>(System<T> *, const T *, T *, int, cudaStream_t);                                   \
    template int sys_permute_out<T>(System<T> *, const T *, T *, int, cudaStream_t);                                  \
    template int sys_mbar<T>(System<T> *, const T *, cudaStream_t);                                                   \
    template int sys_rhs_ms<T>(System<T> *, const T *, T *, cudaStream_t);                                            \
    template int sys_demag_field<T>(System<T> *, const T *, unsigned, T *, cudaStream_t);                             \
    template int sys_rhs_mech<T>(System<T> *, const T *, T *, cudaStream_t);                                          \
    template int sys_stress<T>(System<T> *, const T *, const T *, cudaStream_t);                                      \
    template int sys_field<T>(System<T> *, const T *, const T *, const double *, unsigned, T *, T *, cudaStream_t, const double *); \
    template int sys_axpby3<T>(System<T> *, const T *, const T *, T, T *, cudaStream_t);                              \
    template int sys_spmv_matfree<T>(System<T> *, const T *, T *, cudaStream_t);                                      \
    template int sys_cg_matfree<T>(System<T> *, const T *, T *, double, int, int, int, int, cudaStream_t);            \
    template int sys_step<T>(System<T> *, const cm_step_params *, T *, T *, T *, cm_step_info *, cudaStream_t);        \
    template int sys_hysteresis<T>(System<T> *, const cm_step_params *, const cm_hyst_params *, T *, T *, T *, double *, double *, int *, \
                                   cm_hyst_result *, cudaStream_t);
INST(double)
INST(float)

// volume average entry used by cm_volume_average (user-order input)
template <typename T>
int mesh_volume_average(cm_mesh *M, const T *g_user, int nc, double *out_host, cudaStream_t st)
{
    std::lock_guard<std::mutex> hold(M->avg_lock); // the mesh's scratch is shared by every system built on it
    const long n = M->N * nc;
    const T *g_lib = g_user;
    if (!M->identity) {
        if (M->tmp_bytes < (long)(n * sizeof(T))) {
            cudaFree(M->d_tmp);
            M->d_tmp = nullptr;
            M->tmp_bytes = 0;
            CM_CUDA(cudaMalloc(&M->d_tmp, n * sizeof(T)));
            M->tmp_bytes = n * sizeof(T);
        }
        permute_in_kernel<T><<<nblk(n), BS, 0, st>>>(M->N, nc, M->d_order, g_user, (T *)M->d_tmp);
        g_lib = (const T *)M->d_tmp;
    }
    CM_TRY(wavg<T>(M, g_lib, nc, M->d_red, M->d_red + RED_BLOCKS * 8, st));
    CM_CUDA(cudaMemcpyAsync(M->h_red, M->d_red + RED_BLOCKS * 8, nc * sizeof(double), cudaMemcpyDeviceToHost, st));
    CM_CUDA(cudaStreamSynchronize(st));
    for (int c = 0; c < nc; c++) out_host[c] = M->h_red[c];
    return CM_OK;
}
template int mesh_volume_average<double>(cm_mesh *, const double *, int, double *, cudaStream_t);
template int mesh_volume_average<float>(cm_mesh *, const float *, int, double *, cudaStream_t);
