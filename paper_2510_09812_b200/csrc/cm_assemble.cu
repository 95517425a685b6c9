// S1: geometry (O-1) and matrix values (O-2; Eq. 12) on the device.
// All set-up arithmetic is fp64 and rounded once to the system dtype (R20).  Matrix entries
// are accumulated by one thread per row over the row's incident elements in ascending element order
// (deterministic; no atomics), each element's 4x4 local matrix being recomputed from the coordinates.
#include <algorithm>
#include <cmath>
#include <cstring>

#include "cm_internal.h"

static const double MU0 = 4.0e-7 * 3.14159265358979323846;

__device__ __forceinline__ void tet_geometry(const double *__restrict__ xyz, const int *t, double ld, TetGeom &G)
{
    double x[4][3];
#pragma unroll
    for (int k = 0; k < 4; k++)
#pragma unroll
        for (int d = 0; d < 3; d++) x[k][d] = xyz[3 * (long)t[k] + d] / ld;
    tet_geometry_x(x, G);
}

// nondimensional corner coordinates of every hexahedral cell, [cell][8][3] (System::CX on hexahedral meshes)
__global__ void cell_xyz_kernel(long ncorners, const int *__restrict__ gconn, const double *__restrict__ gxyz, double ld, double *CX)
{
    const long q = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (q >= ncorners) return;
    const long i = gconn[q];
    CX[3 * q] = gxyz[3 * i] / ld; CX[3 * q + 1] = gxyz[3 * i + 1] / ld; CX[3 * q + 2] = gxyz[3 * i + 2] / ld;
}

// nondimensional coordinates of every chunk slot, [slot][4] (System::CX on tetrahedral meshes)
__global__ void slot_xyz_kernel(long nslots, const int *__restrict__ nodes, const double *__restrict__ xyz, double ld, double *CX)
{
    const long s = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (s >= nslots) return;
    const long i = nodes[s];
    CX[4 * s] = xyz[3 * i] / ld; CX[4 * s + 1] = xyz[3 * i + 1] / ld; CX[4 * s + 2] = xyz[3 * i + 2] / ld; CX[4 * s + 3] = 0.0;
}

// one CTA per element chunk: V_e and grad phi_1..3 (rounded to T) into the chunk-blocked geometry array
// (cm_internal.h), fp64 volume copy for the lumped masses
template <typename T>
__global__ void geom_kernel(const int *__restrict__ eptr, const int *__restrict__ gtets, const double *__restrict__ xyz, double ld, T *EG,
                            double *Vd)
{
    const int c = blockIdx.x, e0 = eptr[c], ne = eptr[c + 1] - e0, ne8 = (ne + 7) & ~7;
    T *blk = EG + 10L * e0;
    for (int el = threadIdx.x; el < ne; el += blockDim.x) {
        const long e = e0 + el;
        int t[4];
        *reinterpret_cast<int4 *>(t) = reinterpret_cast<const int4 *>(gtets)[e];
        TetGeom g;
        tet_geometry(xyz, t, ld, g);
        Vd[e] = g.V;
        blk[el] = (T)g.V;
#pragma unroll
        for (int k = 1; k < 4; k++)
#pragma unroll
            for (int d = 0; d < 3; d++) blk[(long)(3 * (k - 1) + d + 1) * ne8 + el] = (T)g.g[k][d];
    }
}

// one thread per node: lumped masses over all / magnetic incident tets, live flag
template <typename T>
__global__ void lump_kernel(long N, const int *__restrict__ n2e_ptr, const int *__restrict__ n2e, const double *__restrict__ Vd,
                            const uchar *__restrict__ mag, T *mL, T *mLm, uchar *live)
{
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    double a = 0, am = 0;
    bool lv = false;
    for (int s = n2e_ptr[i]; s < n2e_ptr[i + 1]; s++) {
        int e = n2e[s] >> 2;
        double v = Vd[e] / 4.0;
        a += v;
        if (mag[e]) { am += v; lv = true; }
    }
    mL[i] = (T)a; mLm[i] = (T)am; live[i] = lv;
}

// deterministic sum of Vd (all, magnetic): one block
__global__ void volume_sum_kernel(long Ne, const double *__restrict__ Vd, const uchar *__restrict__ mag, double *out)
{
    __shared__ double sa[1024], sm[1024];
    double a = 0, m = 0;
    for (long e = threadIdx.x; e < Ne; e += blockDim.x) { a += Vd[e]; if (mag[e]) m += Vd[e]; }
    sa[threadIdx.x] = a; sm[threadIdx.x] = m;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) { sa[threadIdx.x] += sa[threadIdx.x + o]; sm[threadIdx.x] += sm[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) { out[0] = sa[0]; out[1] = sm[0]; }
}

__device__ __forceinline__ void strain_disp(const double g[3], double B[6][3])
{
#pragma unroll
    for (int r = 0; r < 6; r++)
#pragma unroll
        for (int s = 0; s < 3; s++) B[r][s] = 0;
    B[0][0] = g[0]; B[1][1] = g[1]; B[2][2] = g[2];
    B[3][1] = g[2]; B[3][2] = g[1];
    B[4][0] = g[2]; B[4][2] = g[0];
    B[5][0] = g[1]; B[5][1] = g[0];
}

// one thread per row i: accumulate scalar entries K (all tets), K_m, M_m (magnetic tets) and, if
// Cstar != NULL, the 3x3 blocks of K^mech into fp64 scratch arrays laid out on the CSR pattern.
__global__ void assemble_rows_kernel(long N, const int *__restrict__ tets, const int *__restrict__ gtets, const double *__restrict__ xyz,
                                     double ld,
                                     const int *__restrict__ n2e_ptr, const int *__restrict__ n2e, const uchar *__restrict__ mag,
                                     const int *__restrict__ eid, const double *__restrict__ Cstar, const int *__restrict__ rowptr,
                                     const int *__restrict__ col, double *K, double *Km, double *Mm, double *Kme)
{
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int q0 = rowptr[i], q1 = rowptr[i + 1];
    for (int s = n2e_ptr[i]; s < n2e_ptr[i + 1]; s++) {
        const int e = n2e[s] >> 2, k = n2e[s] & 3;
        int t[4], tg[4]; // DOF ids (matrix columns) and geometric node ids (coordinates; the same unless the mesh is wrapped)
        *reinterpret_cast<int4 *>(t) = reinterpret_cast<const int4 *>(tets)[e];
        *reinterpret_cast<int4 *>(tg) = reinterpret_cast<const int4 *>(gtets)[e];
        TetGeom g;
        tet_geometry(xyz, tg, ld, g);
        const bool m = mag[e];
        double CBt[3][6]; // (B_k^T C): row r, Voigt column w
        if (Cstar) {
            const double *C = Cstar + 36 * eid[e];
            double Bk[6][3];
            strain_disp(g.g[k], Bk);
            for (int r = 0; r < 3; r++)
                for (int w = 0; w < 6; w++) {
                    double acc = 0;
                    for (int v = 0; v < 6; v++) acc += Bk[v][r] * C[6 * v + w];
                    CBt[r][w] = acc;
                }
        }
        for (int l = 0; l < 4; l++) {
            const int j = t[l];
            int lo = q0, hi = q1 - 1; // binary search of j in the sorted row
            while (lo < hi) {
                int mid = (lo + hi) >> 1;
                if (col[mid] < j) lo = mid + 1; else hi = mid;
            }
            const double kij = g.V * (g.g[k][0] * g.g[l][0] + g.g[k][1] * g.g[l][1] + g.g[k][2] * g.g[l][2]);
            const double mij = g.V * (k == l ? 2.0 : 1.0) / 20.0;
            K[lo] += kij;
            if (m) { Km[lo] += kij; Mm[lo] += mij; }
            if (Cstar) {
                double Bl[6][3];
                strain_disp(g.g[l], Bl);
                for (int r = 0; r < 3; r++)
                    for (int c = 0; c < 3; c++) {
                        double acc = 0;
                        for (int w = 0; w < 6; w++) acc += CBt[r][w] * Bl[w][c];
                        Kme[9 * (long)lo + 3 * r + c] += g.V * acc;
                    }
            }
        }
    }
}

// ---- linear hexahedra (R26): one thread per row i accumulates, over the incident elements in ascending order and the
// 2 x 2 x 2 Gauss points in order, row i of K, K_m, M_m, K^mech and the lumped masses int phi_i.
template <typename T>
__global__ void hex_rows_kernel(long N, const int *__restrict__ hexes, const int *__restrict__ ghexes, const double *__restrict__ xyz, double ld,
                                const int *__restrict__ n2e_ptr, const int *__restrict__ n2e, const uchar *__restrict__ mag,
                                const int *__restrict__ eid, const double *__restrict__ Cstar, const int *__restrict__ rowptr,
                                const int *__restrict__ col, double *K, double *Km, double *Mm, double *Kme, T *mL, T *mLm, uchar *live)
{
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int q0 = rowptr[i], q1 = rowptr[i + 1];
    double ml = 0, mlm = 0;
    bool lv = false;
    for (int s = n2e_ptr[i]; s < n2e_ptr[i + 1]; s++) {
        const int e = n2e[s] >> 3, k = n2e[s] & 7;
        int t[8], pos[8];
        double X[8][3];
        for (int a = 0; a < 8; a++) {
            t[a] = hexes[8 * (long)e + a];
            const long ga = ghexes[8 * (long)e + a]; // coordinates come from the cell's own corner (wrapped meshes: != DOF)
            for (int d = 0; d < 3; d++) X[a][d] = xyz[3 * ga + d] / ld;
            int lo = q0, hi = q1 - 1; // position of column t[a] in the sorted row
            while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (col[mid] < t[a]) lo = mid + 1; else hi = mid;
            }
            pos[a] = lo;
        }
        const bool m = mag[e];
        const double *C = Cstar ? Cstar + 36 * eid[e] : nullptr;
        for (int p = 0; p < 8; p++) {
            double phi[8], g[8][3];
            const double det = hex_point(X, p, phi, g);
            ml += det * phi[k];
            if (m) { mlm += det * phi[k]; lv = true; }
            double CBt[3][6];
            if (C) {
                double Bk[6][3];
                strain_disp(g[k], Bk);
                for (int r = 0; r < 3; r++)
                    for (int w = 0; w < 6; w++) {
                        double acc = 0;
                        for (int v = 0; v < 6; v++) acc += Bk[v][r] * C[6 * v + w];
                        CBt[r][w] = acc;
                    }
            }
            for (int b = 0; b < 8; b++) {
                const double kab = det * (g[k][0] * g[b][0] + g[k][1] * g[b][1] + g[k][2] * g[b][2]);
                const double mab = det * phi[k] * phi[b];
                K[pos[b]] += kab;
                if (m) { Km[pos[b]] += kab; Mm[pos[b]] += mab; }
                if (C) {
                    double Bb[6][3];
                    strain_disp(g[b], Bb);
                    for (int r = 0; r < 3; r++)
                        for (int c = 0; c < 3; c++) {
                            double acc = 0;
                            for (int w = 0; w < 6; w++) acc += CBt[r][w] * Bb[w][c];
                            Kme[9 * (long)pos[b] + 3 * r + c] += det * acc;
                        }
                }
            }
        }
    }
    mL[i] = (T)ml; mLm[i] = (T)mlm; live[i] = lv;
}

// one thread per row: apply constraints (P A P + (I - P)), form K^GS(eps), round to T and store in the sliced
// layouts (cm_internal.h): scalar matrices at spS[i / CS] + j * CS + i % CS, the 9 entries of a K^mech block in
// the 9 planes of its slice, plane k at 9 * spB[s] + k * L_s + (j * CB + i % CB).
template <typename T>
__global__ void finalize_kernel(long N, long nnz, const int *__restrict__ rowptr, const int *__restrict__ col, const double *K,
                                const double *Km, const double *Mm, const double *Kme, const uchar *__restrict__ live,
                                const uchar *__restrict__ clamp, int pin, double eps1, double eps2, const int *__restrict__ spS,
                                const int *__restrict__ spB, T *Kms, T *Kgs1, T *Kgs2, T *MmT, T *Kmech, T *Dms, T *Dgs1, T *Dgs2, T *Dmech)
{
    constexpr int CS = CM_C_SCALAR, CB = CM_C_BLOCK;
    long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
    if (i >= N) return;
    const long baseS = spS[i / CS] + i % CS;
    const long bB = spB[i / CB], LB = spB[i / CB + 1] - bB;
    const int q0 = rowptr[i];
    for (int q = q0; q < rowptr[i + 1]; q++) {
        const int j = col[q];
        const long dS = baseS + (long)(q - q0) * CS;
        double kms = K[q];
        if (i == pin || j == pin) kms = (i == j) ? 1.0 : 0.0;
        Kms[dS] = (T)kms;
        const double dead = (i == j && !live[i]) ? 1.0 : 0.0;
        Kgs1[dS] = (T)(Mm[q] + eps1 * Km[q] + dead);
        Kgs2[dS] = (T)(Mm[q] + eps2 * Km[q] + dead);
        MmT[dS] = (T)Mm[q];
        if (i == j) { Dms[i] = Kms[dS]; Dgs1[i] = Kgs1[dS]; Dgs2[i] = Kgs2[dS]; } // diagonals as stored (Jacobi)
        if (Kme) {
            T *dst = Kmech + 9 * bB + (long)(q - q0) * CB + i % CB;
            for (int r = 0; r < 3; r++)
                for (int c = 0; c < 3; c++) {
                    double v = Kme[9 * (long)q + 3 * r + c];
                    if (clamp[3 * i + r] || clamp[3 * (long)j + c]) v = (i == j && r == c) ? 1.0 : 0.0;
                    dst[LB * (3 * r + c)] = (T)v;
                    if (i == j && r == c) Dmech[3 * i + r] = (T)v;
                }
        }
    }
}

template <typename T>
System<T>::~System()
{
    T *ptrs[] = {EG, mL, mLm, Cstar, Ccub, Kms, Kgs1, Kgs2, Mm, Kmech, Dms, Dgs1, Dgs2, Dmech, r, p, p2, Ap, bvec, m, U, u, hd, hn, f, gn, gs, ms, mss, xin, xout, hpart, sig, stg_m, stg_U, stg_u};
    for (T *q : ptrs) cudaFree(q);
    cudaFree(CX); cudaFree(live); cudaFree(clamp); cudaFree(partial); cudaFree(d_res); cudaFree(red); cudaFree(dscal);
    cudaFree(hyst_ctl); cudaFree(hyst_log); cudaFree(hyst_steps); cudaFree(d_hist); cudaFree(mf_state);
    if (h_mf) cudaFreeHost(h_mf);
    if (h_res) cudaFreeHost(h_res);
    if (h_scal) cudaFreeHost(h_scal);
}
template struct System<double>;
template struct System<float>;

template <typename T>
int sys_assemble(System<T> *S, const cm_material *mat, const uchar *clamp_user, long pin_user, cudaStream_t st)
{
    cm_mesh *M = S->mesh;
    const long N = S->N, Ne = S->Ne, nnz = S->nnz;
    const double ld = mat->length_scale, mu0Ms2 = MU0 * mat->Ms * mat->Ms;
    // O-0 nondimensionalisation
    S->Ms = mat->Ms;
    S->ld = ld;
    S->Astar = 2.0 * mat->Aex / (mu0Ms2 * ld * ld);
    S->Kstar = mat->K1 / mu0Ms2;
    S->dtau = mat->gamma * mat->Ms * S->dt;
    S->alpha = mat->alpha;
    S->eps1 = S->Astar * S->dtau;
    S->eps2 = S->alpha * S->Astar * S->dtau;
    S->lam100 = mat->lambda100; S->lam111 = mat->lambda111;
    std::memcpy(S->Nd, mat->Nd, sizeof(S->Nd));
    {   // App. D: all zeros = identity; otherwise R R^T = I and det R = +1 are required
        bool zero = true, ident = true;
        for (int q = 0; q < 9; q++) zero = zero && mat->R[q] == 0.0;
        for (int q = 0; q < 9; q++) S->R[q] = zero ? (q % 4 == 0 ? 1.0 : 0.0) : mat->R[q];
        const double *r = S->R;
        double worst = 0;
        for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++)
                worst = std::max(worst, std::fabs(r[3 * a] * r[3 * b] + r[3 * a + 1] * r[3 * b + 1] + r[3 * a + 2] * r[3 * b + 2] - (a == b ? 1.0 : 0.0)));
        const double det = r[0] * (r[4] * r[8] - r[5] * r[7]) - r[1] * (r[3] * r[8] - r[5] * r[6]) + r[2] * (r[3] * r[7] - r[4] * r[6]);
        if (!(worst <= 1e-10) || !(det > 0)) { cm_set_error("cm_assemble_csr: material R is not a proper rotation (|R R^T - I| = %.2e, det = %.3f)", worst, det); return CM_E_BADARG; }
        for (int q = 0; q < 9; q++) ident = ident && S->R[q] == (q % 4 == 0 ? 1.0 : 0.0);
        S->rot = !ident;
    }
    S->n_elastic = mat->n_elastic > 0 ? mat->n_elastic : 0;
    S->has_sext = false;
    for (int q = 0; q < 6; q++) { S->sext[q] = mat->sigma_ext[q] / mu0Ms2; S->has_sext = S->has_sext || mat->sigma_ext[q] != 0.0; }
    S->pin = M->iperm[pin_user];
    int dev = 0;
    CM_CUDA(cudaGetDevice(&dev));
    CM_CUDA(cudaDeviceGetAttribute(&S->num_sms, cudaDevAttrMultiProcessorCount, dev));

    auto alloc = [&](auto **p, size_t n) -> int {
        CM_CUDA(cudaMalloc((void **)p, std::max<size_t>(n, 1) * sizeof(**p) + 256));
        CM_CUDA(cudaMemsetAsync(*p, 0, std::max<size_t>(n, 1) * sizeof(**p) + 256, st));
        return CM_OK;
    };
    CM_TRY(alloc(&S->EG, 10 * (Ne + 8))); CM_TRY(alloc(&S->mL, N)); CM_TRY(alloc(&S->mLm, N));
    CM_TRY(alloc(&S->live, N)); CM_TRY(alloc(&S->clamp, 3 * N));
    const long ES = M->sell[0].E, EB = M->sell[1].E; // stored elements of the sliced layouts (padding is zero)
    CM_TRY(alloc(&S->Kms, ES)); CM_TRY(alloc(&S->Kgs1, ES)); CM_TRY(alloc(&S->Kgs2, ES)); CM_TRY(alloc(&S->Mm, ES));
    if (S->n_elastic) CM_TRY(alloc(&S->Kmech, 9 * EB));
    CM_TRY(alloc(&S->Dms, N)); CM_TRY(alloc(&S->Dgs1, N)); CM_TRY(alloc(&S->Dgs2, N));
    if (S->n_elastic) CM_TRY(alloc(&S->Dmech, 3 * N));

    // elastic constants C* = C / (mu0 Ms^2): fp64 for assembly, T for the element kernels
    // set-up scratch (fp64 matrices on the CSR pattern, volumes, C*): freed on every exit path
    struct Scratch {
        double *Cd = nullptr, *Vd = nullptr, *vsum = nullptr, *K = nullptr, *Km = nullptr, *Mm = nullptr, *Kme = nullptr;
        ~Scratch() { cudaFree(Cd); cudaFree(Vd); cudaFree(vsum); cudaFree(K); cudaFree(Km); cudaFree(Mm); cudaFree(Kme); }
    } scr;
    double *&Cd = scr.Cd;
    if (S->n_elastic) {
        std::vector<double> Cs(36 * S->n_elastic);
        std::vector<T> Ct(36 * S->n_elastic);
        // Eq. D.3-D.4: stiffness in the simulation frame, C_sim = M C_crystal M^T, where row (ij), column (kl)
        // of M holds the coefficient of sigma_kl in (R sigma R^T)_ij
        double Mv[6][6];
        {
            const int vi[6] = {0, 1, 2, 1, 0, 0}, vj[6] = {0, 1, 2, 2, 2, 1};
            auto Rm = [&](int a, int b) { return S->R[3 * a + b]; };
            for (int p = 0; p < 6; p++)
                for (int q = 0; q < 6; q++) {
                    const int i = vi[p], j = vj[p], k = vi[q], l = vj[q];
                    Mv[p][q] = k == l ? Rm(i, k) * Rm(j, k) : Rm(i, k) * Rm(j, l) + Rm(i, l) * Rm(j, k);
                }
        }
        for (int e = 0; e < S->n_elastic; e++) {
            const double *C = mat->C_voigt + 36 * e;
            double *out = Cs.data() + 36 * e;
            if (!S->rot) {
                for (int q = 0; q < 36; q++) out[q] = C[q] / mu0Ms2;
                continue;
            }
            double MC[6][6];
            for (int p = 0; p < 6; p++)
                for (int q = 0; q < 6; q++) {
                    double acc = 0;
                    for (int w = 0; w < 6; w++) acc += Mv[p][w] * C[6 * w + q];
                    MC[p][q] = acc;
                }
            for (int p = 0; p < 6; p++)
                for (int q = 0; q < 6; q++) {
                    double acc = 0;
                    for (int w = 0; w < 6; w++) acc += MC[p][w] * Mv[q][w];
                    out[6 * p + q] = acc / mu0Ms2;
                }
        }
        for (size_t q = 0; q < Cs.size(); q++) Ct[q] = (T)Cs[q];
        CM_CUDA(cudaMalloc((void **)&Cd, Cs.size() * sizeof(double)));
        CM_CUDA(cudaMemcpyAsync(Cd, Cs.data(), Cs.size() * sizeof(double), cudaMemcpyHostToDevice, st));
        CM_TRY(alloc(&S->Cstar, Ct.size()));
        CM_CUDA(cudaMemcpyAsync(S->Cstar, Ct.data(), Ct.size() * sizeof(T), cudaMemcpyHostToDevice, st));
        // cubic / isotropic / orthotropic stiffness in the crystal frame: only the normal 3x3 block and the three shear
        // diagonals are non-zero.  Skipping exact zeros leaves every product C : eps unchanged, so the element
        // kernels then read 12 words per material instead of 36.
        S->cubic_pattern = true;
        std::vector<T> Cc(12 * S->n_elastic);
        for (int q = 0; q < S->n_elastic; q++)
            for (int r = 0; r < 6; r++)
                for (int c = 0; c < 6; c++) {
                    const bool in = (r < 3 && c < 3) || r == c;
                    if (!in && Cs[36 * q + 6 * r + c] != 0.0) S->cubic_pattern = false;
                    if (r < 3 && c < 3) Cc[12 * q + 3 * r + c] = Ct[36 * q + 6 * r + c];
                    if (r >= 3 && r == c) Cc[12 * q + 9 + (r - 3)] = Ct[36 * q + 6 * r + c];
                }
        CM_TRY(alloc(&S->Ccub, Cc.size()));
        CM_CUDA(cudaMemcpyAsync(S->Ccub, Cc.data(), Cc.size() * sizeof(T), cudaMemcpyHostToDevice, st));
        CM_CUDA(cudaStreamSynchronize(st));
    }
    // clamp flags to library order
    {
        std::vector<uchar> cl(3 * N, 0);
        if (clamp_user)
            for (long i = 0; i < N; i++)
                for (int d = 0; d < 3; d++) cl[3 * i + d] = clamp_user[3 * (long)M->order[i] + d] != 0;
        CM_CUDA(cudaMemcpyAsync(S->clamp, cl.data(), cl.size(), cudaMemcpyHostToDevice, st));
        CM_CUDA(cudaStreamSynchronize(st));
    }
    // geometry
    const bool hex = M->nen == 8;
    double *&Vd = scr.Vd, *&vsum = scr.vsum;
    const int B = 256;
    if (!hex) {
        CM_CUDA(cudaMalloc((void **)&Vd, Ne * sizeof(double)));
        CM_CUDA(cudaMalloc((void **)&vsum, 2 * sizeof(double)));
        geom_kernel<T><<<M->ck.nchunks, B, 0, st>>>(M->ck.d_eptr, M->d_gtets, M->d_gxyz, ld, S->EG, Vd);
        lump_kernel<T><<<(unsigned)((N + B - 1) / B), B, 0, st>>>(N, M->d_n2e_ptr, M->d_n2e, Vd, M->d_mag, S->mL, S->mLm, S->live);
        volume_sum_kernel<<<1, 1024, 0, st>>>(Ne, Vd, M->d_mag, vsum);
        if (!M->wrapped) { // a wrapped element takes its corners from its own images, not from the DOFs' representatives
            CM_TRY(alloc(&S->CX, (size_t)4 * M->ck.nslots + 8));
            slot_xyz_kernel<<<(unsigned)((M->ck.nslots + B - 1) / B), B, 0, st>>>(M->ck.nslots, M->ck.d_nodes, M->d_xyz, ld, S->CX);
        }
        CM_CUDA(cudaGetLastError());
        double hv[2];
        CM_CUDA(cudaMemcpyAsync(hv, vsum, sizeof(hv), cudaMemcpyDeviceToHost, st));
        CM_CUDA(cudaStreamSynchronize(st));
        S->Vtot = hv[0]; S->Vmag = hv[1];
    } else {
        S->Vtot = M->vtot_m3 / (ld * ld * ld); S->Vmag = M->vmag_m3 / (ld * ld * ld);
        // corner coordinates per CELL (a wrapped cell takes them from its own images): [cell][8][3]
        CM_TRY(alloc(&S->CX, (size_t)24 * Ne + 32));
        cell_xyz_kernel<<<(unsigned)((8 * Ne + B - 1) / B), B, 0, st>>>(8 * Ne, M->d_gtets, M->d_gxyz, ld, S->CX);
    }
    // matrices: fp64 scratch on the pattern
    double *&K = scr.K, *&Km = scr.Km, *&Mm = scr.Mm, *&Kme = scr.Kme;
    CM_TRY(alloc(&K, nnz)); CM_TRY(alloc(&Km, nnz)); CM_TRY(alloc(&Mm, nnz));
    if (S->n_elastic) CM_TRY(alloc(&Kme, 9 * nnz));
    const int BA = 128;
    if (hex)
        hex_rows_kernel<T><<<(unsigned)((N + 63) / 64), 64, 0, st>>>(N, M->d_tets, M->d_gtets, M->d_gxyz, ld, M->d_n2e_ptr, M->d_n2e, M->d_mag, M->d_eid, Cd,
                                                                    M->d_rowptr, M->d_col, K, Km, Mm, Kme, S->mL, S->mLm, S->live);
    else
        assemble_rows_kernel<<<(unsigned)((N + BA - 1) / BA), BA, 0, st>>>(N, M->d_tets, M->d_gtets, M->d_gxyz, ld, M->d_n2e_ptr, M->d_n2e,
                                                                          M->d_mag, M->d_eid, Cd, M->d_rowptr, M->d_col, K, Km, Mm, Kme);
    CM_CUDA(cudaGetLastError());
    CM_CUDA(cudaStreamSynchronize(st));
    {
        std::vector<uchar> lv(N);
        CM_CUDA(cudaMemcpy(lv.data(), S->live, N, cudaMemcpyDeviceToHost));
        S->nlive = 0;
        for (long i = 0; i < N; i++) S->nlive += lv[i];
    }
    finalize_kernel<T><<<(unsigned)((N + B - 1) / B), B, 0, st>>>(N, nnz, M->d_rowptr, M->d_col, K, Km, Mm, Kme, S->live, S->clamp, S->pin,
                                                                 S->eps1, S->eps2, M->sell[0].d_sp, M->sell[1].d_sp, S->Kms, S->Kgs1, S->Kgs2,
                                                                 S->Mm, S->Kmech, S->Dms, S->Dgs1, S->Dgs2, S->Dmech);
    CM_CUDA(cudaGetLastError());
    CM_CUDA(cudaStreamSynchronize(st));
    for (double **q : {&K, &Km, &Mm, &Kme, &Vd, &vsum, &Cd}) { cudaFree(*q); *q = nullptr; } // before the work vectors are allocated

    // work vectors
    T **vecs3[] = {&S->r, &S->Ap, &S->bvec, &S->m, &S->u, &S->hd, &S->hn, &S->gn, &S->gs, &S->ms, &S->mss, &S->xout, &S->stg_m, &S->stg_u};
    for (T **v : vecs3) CM_TRY(alloc(v, 3 * N));
    T **vecs4[] = {&S->p, &S->p2, &S->f, &S->xin}; // padded [node][4] when they hold a 3-vector that a product gathers
    for (T **v : vecs4) CM_TRY(alloc(v, 4 * N));
    CM_TRY(alloc(&S->U, N)); CM_TRY(alloc(&S->stg_U, N)); CM_TRY(alloc(&S->sig, 6 * N));
    CM_TRY(alloc(&S->hpart, (size_t)9 * M->ck.nslots));
    S->grid_cap = S->num_sms * 8;
    CM_TRY(alloc(&S->partial, (size_t)5 * S->grid_cap * 3));
    CM_TRY(alloc(&S->d_hist, (size_t)CM_HIST_CAP));
    CM_TRY(alloc(&S->d_res, 8));
    CM_TRY(alloc(&S->red, std::max<size_t>({(size_t)4096 * 16, (size_t)8 * M->ck.nchunks, (size_t)3 * ((N + 127) / 128) + 64})));
    CM_TRY(alloc(&S->dscal, 32));
    CM_CUDA(cudaMalloc(&S->mf_state, 256));
    CM_CUDA(cudaMemsetAsync(S->mf_state, 0, 256, st));
    CM_CUDA(cudaMallocHost(&S->h_mf, 256));
    CM_CUDA(cudaMallocHost((void **)&S->h_res, 8 * sizeof(CgResult)));
    CM_CUDA(cudaMallocHost((void **)&S->h_scal, 32 * sizeof(double)));
    CM_CUDA(cudaStreamSynchronize(st));
    return CM_OK;
}

// values back to the host in standard CSR / BSR order (for parity tests)
template <typename T>
int sys_get_values(const System<T> *S, cm_matrix_id id, void *host_out, long capacity)
{
    const long nnz = S->nnz;
    const T *src = nullptr;
    switch (id) {
    case CM_MAT_K_MS: src = S->Kms; break;
    case CM_MAT_K_GS1: src = S->Kgs1; break;
    case CM_MAT_K_GS2: src = S->Kgs2; break;
    case CM_MAT_MASS: src = S->Mm; break;
    case CM_MAT_K_MECH: src = S->Kmech; break;
    }
    if (!src) { cm_set_error("cm_system_get_values: matrix %d not assembled", (int)id); return CM_E_BADARG; }
    const cm_mesh *M = S->mesh;
    const std::vector<int> &rp = M->rowptr;
    T *out = (T *)host_out;
    if (id != CM_MAT_K_MECH) {
        if (capacity < nnz) { cm_set_error("cm_system_get_values: capacity"); return CM_E_BADARG; }
        const Sell &L = M->sell[0];
        std::vector<T> tmp(L.E);
        CM_CUDA(cudaMemcpy(tmp.data(), src, tmp.size() * sizeof(T), cudaMemcpyDeviceToHost));
        for (long i = 0; i < S->N; i++)
            for (int q = rp[i]; q < rp[i + 1]; q++) out[q] = tmp[L.sp[i / L.C] + (long)(q - rp[i]) * L.C + i % L.C];
        return CM_OK;
    }
    if (capacity < 9 * nnz) { cm_set_error("cm_system_get_values: capacity"); return CM_E_BADARG; }
    const Sell &L = M->sell[1];
    std::vector<T> tmp(9 * L.E);
    CM_CUDA(cudaMemcpy(tmp.data(), src, tmp.size() * sizeof(T), cudaMemcpyDeviceToHost));
    for (long i = 0; i < S->N; i++) {
        const long b = L.sp[i / L.C], len = L.sp[i / L.C + 1] - b;
        for (int q = rp[i]; q < rp[i + 1]; q++)
            for (int k = 0; k < 9; k++) out[9 * (long)q + k] = tmp[9 * b + k * len + (long)(q - rp[i]) * L.C + i % L.C];
    }
    return CM_OK;
}

template int sys_assemble<double>(System<double> *, const cm_material *, const uchar *, long, cudaStream_t);
template int sys_assemble<float>(System<float> *, const cm_material *, const uchar *, long, cudaStream_t);
template int sys_get_values<double>(const System<double> *, cm_matrix_id, void *, long);
template int sys_get_values<float>(const System<float> *, cm_matrix_id, void *, long);
