// S0: mesh preprocessing -- validation, locality reordering (Morton / RCM, R21),
// relabelled + sorted connectivity, node->element CSR, sparsity pattern, lumped volume fractions.
// Host C++ (set-up, once per mesh; not in the timed step), results uploaded to the device.
#include <algorithm>
#include <limits>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <numeric>

#include "cm_internal.h"

static thread_local char g_err[512] = "";
void cm_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}
extern "C" const char *cm_last_error(void) { return g_err; }
extern "C" const char *cm_version(void) { return "cupymag-b200 0.1 (sm_100a)"; }

namespace {

// Spread the low 21 bits of v so that bit b lands at position 3b.
inline uint64_t spread3(uint64_t v)
{
    v &= 0x1fffffull;
    v = (v | v << 32) & 0x1f00000000ffffull;
    v = (v | v << 16) & 0x1f0000ff0000ffull;
    v = (v | v << 8) & 0x100f00f00f00f00full;
    v = (v | v << 4) & 0x10c30c30c30c30c3ull;
    v = (v | v << 2) & 0x1249249249249249ull;
    return v;
}

void morton_order(long N, const double *xyz, std::vector<int> &order)
{
    double lo[3], hi[3];
    for (int d = 0; d < 3; d++) lo[d] = hi[d] = xyz[d];
    for (long i = 0; i < N; i++)
        for (int d = 0; d < 3; d++) {
            lo[d] = std::min(lo[d], xyz[3 * i + d]);
            hi[d] = std::max(hi[d], xyz[3 * i + d]);
        }
    std::vector<std::pair<uint64_t, int>> key(N);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < N; i++) {
        uint64_t q[3];
        for (int d = 0; d < 3; d++) {
            double span = hi[d] - lo[d];
            double t = span > 0 ? (xyz[3 * i + d] - lo[d]) / span * 2097151.0 : 0.0;
            q[d] = (uint64_t)std::floor(t);
        }
        key[i] = {spread3(q[0]) | spread3(q[1]) << 1 | spread3(q[2]) << 2, (int)i};
    }
    std::sort(key.begin(), key.end()); // (code, user index): unique keys, so equal to a stable sort by code
    order.resize(N);
    for (long i = 0; i < N; i++) order[i] = key[i].second;
}

void build_n2e(long N, long Ne, const int *tets, std::vector<int> &ptr, std::vector<int> &lst, int nen = 4)
{
    ptr.assign(N + 1, 0);
    lst.resize((long)nen * Ne);
    for (long q = 0; q < (long)nen * Ne; q++) ptr[tets[q] + 1]++;
    for (long i = 0; i < N; i++) ptr[i + 1] += ptr[i];
    std::vector<int> fill(ptr.begin(), ptr.end() - 1);
    for (long q = 0; q < (long)nen * Ne; q++) lst[fill[tets[q]]++] = (int)q; // q = nen e + k, ascending
}

void build_pattern(long N, const int *tets, const std::vector<int> &ptr, const std::vector<int> &lst, std::vector<int> &rowptr,
                   std::vector<int> &col, int nen = 4)
{
    rowptr.assign(N + 1, 0);
    std::vector<int> cnt(N);
#pragma omp parallel
    {
        std::vector<int> tmp;
#pragma omp for schedule(dynamic, 4096)
        for (long i = 0; i < N; i++) {
            tmp.clear();
            tmp.push_back((int)i);
            for (int s = ptr[i]; s < ptr[i + 1]; s++) {
                const int *t = tets + (long)nen * (lst[s] / nen);
                tmp.insert(tmp.end(), t, t + nen);
            }
            std::sort(tmp.begin(), tmp.end());
            cnt[i] = (int)(std::unique(tmp.begin(), tmp.end()) - tmp.begin());
        }
    }
    for (long i = 0; i < N; i++) rowptr[i + 1] = rowptr[i] + cnt[i];
    col.resize(rowptr[N]);
#pragma omp parallel
    {
        std::vector<int> tmp;
#pragma omp for schedule(dynamic, 4096)
        for (long i = 0; i < N; i++) {
            tmp.clear();
            tmp.push_back((int)i);
            for (int s = ptr[i]; s < ptr[i + 1]; s++) {
                const int *t = tets + (long)nen * (lst[s] / nen);
                tmp.insert(tmp.end(), t, t + nen);
            }
            std::sort(tmp.begin(), tmp.end());
            auto e = std::unique(tmp.begin(), tmp.end());
            std::copy(tmp.begin(), e, col.begin() + rowptr[i]);
        }
    }
}

// Reverse Cuthill-McKee as specified in DESIGN.md R21.
void rcm_order(long N, const std::vector<int> &rowptr, const std::vector<int> &col, std::vector<int> &order)
{
    auto deg = [&](int i) { return rowptr[i + 1] - rowptr[i] - 1; };
    std::vector<int> bydeg(N);
    std::iota(bydeg.begin(), bydeg.end(), 0);
    std::sort(bydeg.begin(), bydeg.end(), [&](int a, int b) { return deg(a) != deg(b) ? deg(a) < deg(b) : a < b; });
    std::vector<uchar> seen(N, 0);
    std::vector<int> cm;
    cm.reserve(N);
    std::vector<int> nb;
    size_t head = 0;
    long scan = 0;
    while ((long)cm.size() < N) {
        while (seen[bydeg[scan]]) scan++;
        int s = bydeg[scan];
        seen[s] = 1;
        cm.push_back(s);
        while (head < cm.size()) {
            int v = cm[head++];
            nb.clear();
            for (int q = rowptr[v]; q < rowptr[v + 1]; q++) {
                int j = col[q];
                if (j != v && !seen[j]) { seen[j] = 1; nb.push_back(j); }
            }
            std::sort(nb.begin(), nb.end(), [&](int a, int b) { return deg(a) != deg(b) ? deg(a) < deg(b) : a < b; });
            cm.insert(cm.end(), nb.begin(), nb.end());
        }
    }
    order.assign(cm.rbegin(), cm.rend());
}

} // namespace

// R21, CM_REORDER_MORTON_SORTED: within every window of CM_SORT_WINDOW consecutive positions of `order`, nodes in
// descending order of their row length (rowptr in USER numbering), ties keeping their order -- the sigma-window of a
// SELL-C-sigma layout folded into the node permutation, so that the slices of 8 / 16 consecutive rows hold rows of
// nearly equal length on meshes of irregular valence and no kernel needs a row indirection
constexpr long CM_SORT_WINDOW = 256;
static void window_sort(long N, const std::vector<int> &rowptr, std::vector<int> &order)
{
#pragma omp parallel for schedule(static)
    for (long w0 = 0; w0 < N; w0 += CM_SORT_WINDOW) {
        const long w1 = std::min(N, w0 + CM_SORT_WINDOW);
        std::stable_sort(order.begin() + w0, order.begin() + w1,
                         [&](int a, int b) { return rowptr[a + 1] - rowptr[a] > rowptr[b + 1] - rowptr[b]; });
    }
}

int mesh_build_host(cm_mesh *M, const double *gx, long Ng, const int *gtets, long Ne, const uchar *mag, const int *eid,
                    const int *dof, long N, cm_reorder reorder)
{
    M->N = N;
    M->Ne = Ne;
    M->Ng = Ng;
    M->wrapped = dof != nullptr;
    for (long q = 0; q < 4 * Ne; q++)
        if (gtets[q] < 0 || gtets[q] >= Ng) {
            cm_set_error("cm_mesh_create: tet %ld references node %d outside [0, %ld)", q / 4, gtets[q], Ng);
            return CM_E_INDEX_RANGE;
        }
    // DOF connectivity and DOF coordinates (wrapped mesh: componentwise minimum over the nodes of a DOF = its
    // representative on the minimum faces)
    std::vector<int> tets_v;
    std::vector<double> xyz_v;
    const int *tets = gtets;
    const double *xyz = gx;
    if (dof) {
        for (long i = 0; i < Ng; i++)
            if (dof[i] < 0 || dof[i] >= N) {
                cm_set_error("cm_mesh_create_wrapped: dof_of_node[%ld] = %d outside [0, %ld)", i, dof[i], N);
                return CM_E_INDEX_RANGE;
            }
        tets_v.resize(4 * Ne);
        for (long q = 0; q < 4 * Ne; q++) tets_v[q] = dof[gtets[q]];
        for (long e = 0; e < Ne; e++)
            for (int a = 0; a < 4; a++)
                for (int b2 = a + 1; b2 < 4; b2++)
                    if (tets_v[4 * e + a] == tets_v[4 * e + b2]) {
                        cm_set_error("cm_mesh_create_wrapped: tet %ld has two corners on DOF %d (domain one cell wide in a periodic direction)",
                                     e, tets_v[4 * e + a]);
                        return CM_E_BADARG;
                    }
        xyz_v.assign(3 * N, std::numeric_limits<double>::infinity());
        for (long i = 0; i < Ng; i++)
            for (int d = 0; d < 3; d++) xyz_v[3 * (long)dof[i] + d] = std::min(xyz_v[3 * (long)dof[i] + d], gx[3 * i + d]);
        for (long i = 0; i < 3 * N; i++)
            if (!std::isfinite(xyz_v[i])) { cm_set_error("cm_mesh_create_wrapped: DOF %ld has no node", i / 3); return CM_E_BADARG; }
        tets = tets_v.data();
        xyz = xyz_v.data();
    }
    // geometry validation + lumped volume fractions (fp64, metres), user order
    double lo[3], hi[3];
    for (int d = 0; d < 3; d++) lo[d] = hi[d] = gx[d];
    for (long i = 0; i < Ng; i++)
        for (int d = 0; d < 3; d++) {
            lo[d] = std::min(lo[d], gx[3 * i + d]);
            hi[d] = std::max(hi[d], gx[3 * i + d]);
        }
    double diag = std::sqrt((hi[0] - lo[0]) * (hi[0] - lo[0]) + (hi[1] - lo[1]) * (hi[1] - lo[1]) + (hi[2] - lo[2]) * (hi[2] - lo[2]));
    double vmin = 1e-14 * diag * diag * diag, vtot = 0;
    std::vector<double> w_user(N, 0.0);
    for (long e = 0; e < Ne; e++) {
        const double *x0 = gx + 3 * (long)gtets[4 * e], *x1 = gx + 3 * (long)gtets[4 * e + 1], *x2 = gx + 3 * (long)gtets[4 * e + 2],
                     *x3 = gx + 3 * (long)gtets[4 * e + 3];
        double a[3], b[3], c[3];
        for (int d = 0; d < 3; d++) { a[d] = x1[d] - x0[d]; b[d] = x2[d] - x0[d]; c[d] = x3[d] - x0[d]; }
        double det = a[0] * (b[1] * c[2] - b[2] * c[1]) + a[1] * (b[2] * c[0] - b[0] * c[2]) + a[2] * (b[0] * c[1] - b[1] * c[0]);
        double V = std::fabs(det) / 6.0;
        if (!(V > vmin)) {
            cm_set_error("cm_mesh_create: tet %ld is degenerate (V = %.3e <= %.3e)", e, V, vmin);
            return CM_E_DEGENERATE_TET;
        }
        vtot += V;
        for (int k = 0; k < 4; k++) w_user[tets[4 * e + k]] += V * 0.25;
    }

    // ordering
    std::vector<int> ptr_u, lst_u;
    if (reorder == CM_REORDER_NONE) {
        M->order.resize(N);
        std::iota(M->order.begin(), M->order.end(), 0);
    } else if (reorder == CM_REORDER_MORTON) {
        morton_order(N, xyz, M->order);
    } else if (reorder == CM_REORDER_RCM) {
        std::vector<int> rp, cl;
        build_n2e(N, Ne, tets, ptr_u, lst_u);
        build_pattern(N, tets, ptr_u, lst_u, rp, cl);
        rcm_order(N, rp, cl, M->order);
    } else if (reorder == CM_REORDER_MORTON_SORTED) {
        std::vector<int> rp, cl;
        morton_order(N, xyz, M->order);
        build_n2e(N, Ne, tets, ptr_u, lst_u);
        build_pattern(N, tets, ptr_u, lst_u, rp, cl);
        window_sort(N, rp, M->order);
    } else {
        cm_set_error("cm_mesh_create: unknown reorder %d", (int)reorder);
        return CM_E_BADARG;
    }
    M->identity = true;
    M->iperm.resize(N);
    for (long i = 0; i < N; i++) {
        M->iperm[M->order[i]] = (int)i;
        if (M->order[i] != i) M->identity = false;
    }
    // tets: relabel, keep local order, sort by (min new id, user tet index)
    std::vector<std::pair<int, int>> key(Ne);
#pragma omp parallel for schedule(static)
    for (long e = 0; e < Ne; e++) {
        int mn = M->iperm[tets[4 * e]];
        for (int k = 1; k < 4; k++) mn = std::min(mn, M->iperm[tets[4 * e + k]]);
        key[e] = {mn, (int)e};
    }
    std::sort(key.begin(), key.end());
    M->tets.resize(4 * Ne);
    M->tet_order.resize(Ne);
    M->mag.resize(Ne);
    M->eid.resize(Ne);
#pragma omp parallel for schedule(static)
    for (long e = 0; e < Ne; e++) {
        int old = key[e].second;
        M->tet_order[e] = old;
        for (int k = 0; k < 4; k++) M->tets[4 * e + k] = M->iperm[tets[4 * old + k]];
        M->mag[e] = mag ? (mag[old] != 0) : 1;
        M->eid[e] = eid ? eid[old] : 0;
    }
    if (M->wrapped) {
        M->gtets.resize(4 * Ne);
#pragma omp parallel for schedule(static)
        for (long e = 0; e < Ne; e++)
            for (int k = 0; k < 4; k++) M->gtets[4 * e + k] = gtets[4 * (long)M->tet_order[e] + k];
        M->gxyz.assign(gx, gx + 3 * Ng);
    }
    M->xyz.resize(3 * N);
    M->wvol.resize(N);
    for (long i = 0; i < N; i++) {
        for (int d = 0; d < 3; d++) M->xyz[3 * i + d] = xyz[3 * (long)M->order[i] + d];
        M->wvol[i] = w_user[M->order[i]] / vtot;
    }
    build_n2e(N, Ne, M->tets.data(), M->n2e_ptr, M->n2e);
    build_pattern(N, M->tets.data(), M->n2e_ptr, M->n2e, M->rowptr, M->col);
    M->nnz = M->rowptr[N];
    if (build_sell(N, M->rowptr, M->col, CM_C_SCALAR, &M->sell[0]) != CM_OK) return CM_E_BADARG;
    if (build_sell(N, M->rowptr, M->col, CM_C_BLOCK, &M->sell[1]) != CM_OK) return CM_E_BADARG;
    CM_TRY(build_chunks(N, Ne, M->tets.data(), 4, CM_EC_MAX, &M->ck));
    M->emat.resize(Ne);
    for (long e = 0; e < Ne; e++) {
        if (M->eid[e] < 0 || M->eid[e] > 0x7ffe) { cm_set_error("cm_mesh_create: elastic_id %d outside [0, 32766]", M->eid[e]); return CM_E_INDEX_RANGE; }
        M->emat[e] = (unsigned short)(M->eid[e] << 1 | (M->mag[e] ? 1 : 0));
    }
    return CM_OK;
}

// ---- linear hexahedra (R26): host-side Gauss quadrature used for validation, volumes and lumped volume fractions
// local node a = i + 2 j + 4 k <-> (xi, eta, zeta) = (2i-1, 2j-1, 2k-1); 2 x 2 x 2 Gauss points, unit weights
static double hex_detJ_phi(const double X[8][3], int p, double phi[8])
{
    const double g = 0.57735026918962576451;
    const double xi[3] = {(p & 1) ? g : -g, (p & 2) ? g : -g, (p & 4) ? g : -g};
    double J[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    for (int a = 0; a < 8; a++) {
        const double s[3] = {(a & 1) ? 1.0 : -1.0, (a & 2) ? 1.0 : -1.0, (a & 4) ? 1.0 : -1.0};
        const double f[3] = {1 + s[0] * xi[0], 1 + s[1] * xi[1], 1 + s[2] * xi[2]};
        phi[a] = f[0] * f[1] * f[2] / 8;
        const double dN[3] = {s[0] * f[1] * f[2] / 8, f[0] * s[1] * f[2] / 8, f[0] * f[1] * s[2] / 8};
        for (int r = 0; r < 3; r++)
            for (int c = 0; c < 3; c++) J[r][c] += X[a][r] * dN[c];
    }
    return J[0][0] * (J[1][1] * J[2][2] - J[1][2] * J[2][1]) - J[0][1] * (J[1][0] * J[2][2] - J[1][2] * J[2][0]) +
           J[0][2] * (J[1][0] * J[2][1] - J[1][1] * J[2][0]);
}

int mesh_build_host_hex(cm_mesh *M, const double *gx, long Ng, const int *ghexes, long Ne, const uchar *mag, const int *eid,
                        const int *dof, long N, cm_reorder reorder)
{
    M->N = N; M->Ne = Ne; M->Ng = Ng; M->nen = 8; M->wrapped = dof != nullptr;
    for (long q = 0; q < 8 * Ne; q++)
        if (ghexes[q] < 0 || ghexes[q] >= Ng) {
            cm_set_error("cm_mesh_create_hex: element %ld references node %d outside [0, %ld)", q / 8, ghexes[q], Ng);
            return CM_E_INDEX_RANGE;
        }
    // DOF connectivity and DOF coordinates (wrapped mesh: as for tetrahedra)
    std::vector<int> hex_v;
    std::vector<double> xyz_v;
    const int *hexes = ghexes;
    const double *xyz = gx;
    if (dof) {
        for (long i = 0; i < Ng; i++)
            if (dof[i] < 0 || dof[i] >= N) { cm_set_error("cm_mesh_create_hex_wrapped: dof_of_node[%ld] = %d outside [0, %ld)", i, dof[i], N); return CM_E_INDEX_RANGE; }
        hex_v.resize(8 * Ne);
        for (long q = 0; q < 8 * Ne; q++) hex_v[q] = dof[ghexes[q]];
        for (long e = 0; e < Ne; e++)
            for (int a = 0; a < 8; a++)
                for (int b = a + 1; b < 8; b++)
                    if (hex_v[8 * e + a] == hex_v[8 * e + b]) {
                        cm_set_error("cm_mesh_create_hex_wrapped: element %ld has two corners on DOF %d (domain one cell wide in a periodic direction)", e, hex_v[8 * e + a]);
                        return CM_E_BADARG;
                    }
        xyz_v.assign(3 * N, std::numeric_limits<double>::infinity());
        for (long i = 0; i < Ng; i++)
            for (int d = 0; d < 3; d++) xyz_v[3 * (long)dof[i] + d] = std::min(xyz_v[3 * (long)dof[i] + d], gx[3 * i + d]);
        for (long i = 0; i < 3 * N; i++)
            if (!std::isfinite(xyz_v[i])) { cm_set_error("cm_mesh_create_hex_wrapped: DOF %ld has no node", i / 3); return CM_E_BADARG; }
        hexes = hex_v.data();
        xyz = xyz_v.data();
    }
    double lo[3], hi[3];
    for (int d = 0; d < 3; d++) lo[d] = hi[d] = gx[d];
    for (long i = 0; i < Ng; i++)
        for (int d = 0; d < 3; d++) { lo[d] = std::min(lo[d], gx[3 * i + d]); hi[d] = std::max(hi[d], gx[3 * i + d]); }
    const double diag = std::sqrt((hi[0] - lo[0]) * (hi[0] - lo[0]) + (hi[1] - lo[1]) * (hi[1] - lo[1]) + (hi[2] - lo[2]) * (hi[2] - lo[2]));
    const double jmin = 1e-14 * diag * diag * diag;
    std::vector<double> w_user(N, 0.0);
    double vtot = 0, vmag = 0;
    for (long e = 0; e < Ne; e++) {
        double X[8][3], phi[8];
        for (int a = 0; a < 8; a++)
            for (int d = 0; d < 3; d++) X[a][d] = gx[3 * (long)ghexes[8 * e + a] + d];
        double ve = 0;
        for (int p = 0; p < 8; p++) {
            const double det = hex_detJ_phi(X, p, phi);
            if (!(det > jmin)) {
                cm_set_error("cm_mesh_create_hex: element %ld is degenerate or inverted (det J = %.3e at Gauss point %d)", e, det, p);
                return CM_E_DEGENERATE_TET;
            }
            ve += det;
            for (int a = 0; a < 8; a++) w_user[hexes[8 * e + a]] += det * phi[a];
        }
        vtot += ve;
        if (!mag || mag[e]) vmag += ve;
    }
    M->vtot_m3 = vtot; M->vmag_m3 = vmag;
    std::vector<int> ptr_u, lst_u;
    if (reorder == CM_REORDER_NONE) {
        M->order.resize(N);
        std::iota(M->order.begin(), M->order.end(), 0);
    } else if (reorder == CM_REORDER_MORTON) {
        morton_order(N, xyz, M->order);
    } else if (reorder == CM_REORDER_RCM) {
        std::vector<int> rp, cl;
        build_n2e(N, Ne, hexes, ptr_u, lst_u, 8);
        build_pattern(N, hexes, ptr_u, lst_u, rp, cl, 8);
        rcm_order(N, rp, cl, M->order);
    } else if (reorder == CM_REORDER_MORTON_SORTED) {
        std::vector<int> rp, cl;
        morton_order(N, xyz, M->order);
        build_n2e(N, Ne, hexes, ptr_u, lst_u, 8);
        build_pattern(N, hexes, ptr_u, lst_u, rp, cl, 8);
        window_sort(N, rp, M->order);
    } else {
        cm_set_error("cm_mesh_create_hex: unknown reorder %d", (int)reorder);
        return CM_E_BADARG;
    }
    M->identity = true;
    M->iperm.resize(N);
    for (long i = 0; i < N; i++) { M->iperm[M->order[i]] = (int)i; if (M->order[i] != i) M->identity = false; }
    // elements: relabel, keep the local node order, sort by (min new id, user index)
    std::vector<std::pair<int, int>> key(Ne);
    for (long e = 0; e < Ne; e++) {
        int mn = M->iperm[hexes[8 * e]];
        for (int k = 1; k < 8; k++) mn = std::min(mn, M->iperm[hexes[8 * e + k]]);
        key[e] = {mn, (int)e};
    }
    std::sort(key.begin(), key.end());
    M->tets.resize(8 * Ne); M->tet_order.resize(Ne); M->mag.resize(Ne); M->eid.resize(Ne); M->emat.resize(Ne);
    for (long e = 0; e < Ne; e++) {
        const int old = key[e].second;
        M->tet_order[e] = old;
        for (int k = 0; k < 8; k++) M->tets[8 * e + k] = M->iperm[hexes[8 * (long)old + k]];
        M->mag[e] = mag ? (mag[old] != 0) : 1;
        M->eid[e] = eid ? eid[old] : 0;
        if (M->eid[e] < 0 || M->eid[e] > 0x7ffe) { cm_set_error("cm_mesh_create_hex: elastic_id %d outside [0, 32766]", M->eid[e]); return CM_E_INDEX_RANGE; }
        M->emat[e] = (unsigned short)(M->eid[e] << 1 | (M->mag[e] ? 1 : 0));
    }
    if (M->wrapped) {
        M->gtets.resize(8 * Ne);
        for (long e = 0; e < Ne; e++)
            for (int k = 0; k < 8; k++) M->gtets[8 * e + k] = ghexes[8 * (long)M->tet_order[e] + k];
        M->gxyz.assign(gx, gx + 3 * Ng);
    }
    M->xyz.resize(3 * N); M->wvol.resize(N);
    for (long i = 0; i < N; i++) {
        for (int d = 0; d < 3; d++) M->xyz[3 * i + d] = xyz[3 * (long)M->order[i] + d];
        M->wvol[i] = w_user[M->order[i]] / vtot;
    }
    build_n2e(N, Ne, M->tets.data(), M->n2e_ptr, M->n2e, 8);
    build_pattern(N, M->tets.data(), M->n2e_ptr, M->n2e, M->rowptr, M->col, 8);
    M->nnz = M->rowptr[N];
    if (build_sell(N, M->rowptr, M->col, CM_C_SCALAR, &M->sell[0]) != CM_OK) return CM_E_BADARG;
    if (build_sell(N, M->rowptr, M->col, CM_C_BLOCK, &M->sell[1]) != CM_OK) return CM_E_BADARG;
    // element-centric passes: chunks of at most CM_HC_MAX cells, as for tetrahedra (DOF connectivity; the cells' own corner
    // coordinates are staged per cell, so wrapped meshes need nothing else)
    CM_TRY(build_chunks(N, Ne, M->tets.data(), 8, CM_HC_MAX, &M->ck));
    return CM_OK;
}

// Sliced (SELL-C) copy of the CSR pattern: element (i, j) -> sp[i / C] + j * C + i % C; padding entries point at the
// row itself (clamped to N - 1 in the ragged last slice) and carry zero values.
int build_sell(long N, const std::vector<int> &rowptr, const std::vector<int> &col, int C, Sell *out)
{
    const long ns = (N + C - 1) / C;
    out->C = C;
    out->nslices = (int)ns;
    out->sp.assign(ns + 1, 0);
    long E = 0;
    for (long s = 0; s < ns; s++) {
        int w = 0;
        for (long i = s * C; i < std::min(N, (s + 1) * C); i++) w = std::max(w, rowptr[i + 1] - rowptr[i]);
        out->sp[s] = (int)E;
        E += (long)w * C;
        if (E > 0x7fffffffL / 9) { cm_set_error("cm_mesh_create: sliced matrix too large for 32-bit offsets"); return CM_E_BADARG; }
    }
    out->sp[ns] = (int)E;
    out->E = E;
    out->col.resize(E);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < ns; s++) {
        const int b = out->sp[s], w = (out->sp[s + 1] - b) / C;
        for (int rl = 0; rl < C; rl++) {
            const long i = s * C + rl;
            const long ic = std::min(i, N - 1);
            const int len = i < N ? rowptr[i + 1] - rowptr[i] : 0;
            for (int j = 0; j < w; j++) out->col[b + (long)j * C + rl] = j < len ? col[rowptr[i] + j] : (int)ic;
        }
    }
    return CM_OK;
}

// Element chunks (cm_internal.h): greedy cut of the element sequence, local numbering, per-chunk incidence lists and
// the node -> slot transpose.  Elements are sorted by their smallest node id, so with a locality ordering a chunk
// touches a compact node set (about 230 nodes per 768 elements on the paper's meshes).
int build_chunks(long N, long Ne, const int *conn, int nen, int ecmax, Chunks *out)
{
    Chunks &K = *out;
    K.eptr.assign(1, 0);
    K.nptr.assign(1, 0);
    K.nodes.clear();
    K.nodes.reserve(Ne / 2 + 16);
    // pass 1 (sequential): chunk boundaries and the nodes of every chunk in first-seen order; elements are taken in
    // groups of 8 so that chunks start at multiples of 8
    std::vector<int> stamp(N, -1);
    int cur = 0, ne = 0, nl = 0;
    std::vector<int> grp;
    for (long g0 = 0; g0 < Ne; g0 += 8) {
        const long g1 = std::min(Ne, g0 + 8);
        grp.clear();
        for (long q = nen * g0; q < nen * g1; q++)
            if (stamp[conn[q]] != cur) grp.push_back(conn[q]);
        std::sort(grp.begin(), grp.end());
        const int fresh = (int)(std::unique(grp.begin(), grp.end()) - grp.begin());
        if (ne > 0 && (ne + 8 > ecmax || nl + fresh > CM_NL_MAX)) {
            K.eptr.push_back((int)g0);
            K.nptr.push_back((int)K.nodes.size());
            cur++; ne = 0; nl = 0;
        }
        for (long q = nen * g0; q < nen * g1; q++) {
            const int v = conn[q];
            if (stamp[v] != cur) { stamp[v] = cur; K.nodes.push_back(v); nl++; }
        }
        ne += (int)(g1 - g0);
    }
    K.eptr.push_back((int)Ne);
    K.nptr.push_back((int)K.nodes.size());
    K.nchunks = (int)K.eptr.size() - 1;
    K.nslots = (long)K.nodes.size();
    if (K.nslots > 0x7fffffffL / 8) { cm_set_error("cm_mesh_create: too many chunk slots for 32-bit offsets"); return CM_E_BADARG; }
    // pass 2 (parallel over chunks): sort the local nodes, local ids, incidence runs
    K.lid.resize((size_t)nen * Ne);
    K.lent.resize((size_t)nen * Ne);
    K.lptr.assign(K.nslots + K.nchunks, 0);
#pragma omp parallel
    {
        std::vector<int> cnt;
#pragma omp for schedule(dynamic, 64)
        for (int c = 0; c < K.nchunks; c++) {
            const int s0 = K.nptr[c], n = K.nptr[c + 1] - s0, e0 = K.eptr[c], m = K.eptr[c + 1] - e0;
            int *nd = K.nodes.data() + s0;
            std::sort(nd, nd + n);
            cnt.assign(n + 1, 0);
            for (long q = (long)nen * e0; q < (long)nen * (e0 + m); q++) {
                const int l = (int)(std::lower_bound(nd, nd + n, conn[q]) - nd);
                K.lid[q] = (unsigned short)l;
                cnt[l + 1]++;
            }
            for (int l = 0; l < n; l++) cnt[l + 1] += cnt[l];
            unsigned short *lp = K.lptr.data() + s0 + c;
            for (int l = 0; l <= n; l++) lp[l] = (unsigned short)cnt[l];
            unsigned short *le = K.lent.data() + (long)nen * e0;
            for (int q = 0; q < nen * m; q++) le[cnt[K.lid[(long)nen * e0 + q]]++] = (unsigned short)q; // q = nen (e - e0) + k ascending
        }
    }
    // pass 3: node -> slots, ascending
    K.ns_ptr.assign(N + 1, 0);
    for (long s = 0; s < K.nslots; s++) K.ns_ptr[K.nodes[s] + 1]++;
    for (long i = 0; i < N; i++) K.ns_ptr[i + 1] += K.ns_ptr[i];
    K.ns_slot.resize(K.nslots);
    std::vector<int> fill(K.ns_ptr.begin(), K.ns_ptr.end() - 1);
    for (long s = 0; s < K.nslots; s++) K.ns_slot[fill[K.nodes[s]]++] = (int)s;
    return CM_OK;
}

// (256 bytes of slack: the bulk copies of a ragged last chunk read its arrays up to the next multiple of 8 elements)
template <typename U>
static int upload(U **dst, const std::vector<U> &src, cudaStream_t st)
{
    CM_CUDA(cudaMalloc((void **)dst, std::max<size_t>(src.size(), 1) * sizeof(U) + 256));
    CM_CUDA(cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(U), cudaMemcpyHostToDevice, st));
    return CM_OK;
}

// P:233-235 (R23): sort-based pairing.  Representatives are sorted by their cell (side 4 tol) in lexicographic
// order; the image of a wrapped node is looked up in its cell and the 26 neighbours by binary search.
extern "C" int cm_periodic_wrap(const double *xyz, long n_nodes, unsigned axes, double rel_tol, int *dof_of_node, long *n_dof)
{
    if (!xyz || !dof_of_node || !n_dof || n_nodes <= 0 || n_nodes > 0x7fffffffL / 4 || !(rel_tol > 0) || rel_tol > 1e-3 || axes > 7u) {
        cm_set_error("cm_periodic_wrap: bad argument");
        return CM_E_BADARG;
    }
    const long N = n_nodes;
    double lo[3], hi[3], span[3], tol[3], cell[3];
    for (int d = 0; d < 3; d++) lo[d] = hi[d] = xyz[d];
    for (long i = 0; i < N; i++)
        for (int d = 0; d < 3; d++) {
            lo[d] = std::min(lo[d], xyz[3 * i + d]);
            hi[d] = std::max(hi[d], xyz[3 * i + d]);
        }
    for (int d = 0; d < 3; d++) {
        span[d] = hi[d] - lo[d];
        if (((axes >> d) & 1u) && !(span[d] > 0)) { cm_set_error("cm_periodic_wrap: zero extent along periodic direction %d", d); return CM_E_BADARG; }
        tol[d] = rel_tol * span[d];
        cell[d] = span[d] > 0 ? 4.0 * tol[d] : 1.0;
    }
    struct Rep { long long c[3]; int node; };
    auto less = [](const Rep &a, const Rep &b) {
        if (a.c[0] != b.c[0]) return a.c[0] < b.c[0];
        if (a.c[1] != b.c[1]) return a.c[1] < b.c[1];
        return a.c[2] < b.c[2];
    };
    try {
        std::vector<Rep> reps;
        std::vector<int> wrapped;
        long nrep = 0;
        for (long i = 0; i < N; i++) {
            bool w = false;
            for (int d = 0; d < 3; d++) w |= ((axes >> d) & 1u) && xyz[3 * i + d] >= hi[d] - tol[d];
            if (w) { dof_of_node[i] = -1; wrapped.push_back((int)i); continue; }
            dof_of_node[i] = (int)nrep++;
            Rep r;
            for (int d = 0; d < 3; d++) r.c[d] = (long long)std::floor((xyz[3 * i + d] - lo[d]) / cell[d]);
            r.node = (int)i;
            reps.push_back(r);
        }
        *n_dof = nrep;
        std::sort(reps.begin(), reps.end(), less);
        int bad = -1;
#pragma omp parallel for schedule(static)
        for (long q = 0; q < (long)wrapped.size(); q++) {
            const int i = wrapped[q];
            double w[3];
            long long c[3];
            for (int d = 0; d < 3; d++) {
                w[d] = xyz[3 * (long)i + d];
                if (((axes >> d) & 1u) && w[d] >= hi[d] - tol[d]) w[d] -= span[d];
                c[d] = (long long)std::floor((w[d] - lo[d]) / cell[d]);
            }
            int found = -1, count = 0;
            for (int a = -1; a <= 1; a++)
                for (int b = -1; b <= 1; b++)
                    for (int g = -1; g <= 1; g++) {
                        Rep key;
                        key.c[0] = c[0] + a; key.c[1] = c[1] + b; key.c[2] = c[2] + g; key.node = 0;
                        for (auto it = std::lower_bound(reps.begin(), reps.end(), key, less); it != reps.end() && !less(key, *it); ++it) {
                            const double *x = xyz + 3 * (long)it->node;
                            if (std::fabs(x[0] - w[0]) <= tol[0] && std::fabs(x[1] - w[1]) <= tol[1] && std::fabs(x[2] - w[2]) <= tol[2]) {
                                found = it->node;
                                count++;
                            }
                        }
                    }
            if (count == 1) dof_of_node[i] = dof_of_node[found];
            else {
#pragma omp critical
                bad = i;
            }
        }
        if (bad >= 0) {
            cm_set_error("cm_periodic_wrap: node %d on a periodic maximum face has no unique partner on the minimum face (P:235: matched faces required)", bad);
            return CM_E_BADARG;
        }
    } catch (const std::bad_alloc &) {
        cm_set_error("cm_periodic_wrap: out of host memory");
        return CM_E_ALLOC;
    }
    return CM_OK;
}

extern "C" int cm_mesh_create(const double *xyz, long n_nodes, const int *tets, long n_tets, const unsigned char *magnetic,
                              const int *elastic_id, cm_reorder reorder, void *stream, cm_mesh **out)
{
    return cm_mesh_create_wrapped(xyz, n_nodes, tets, n_tets, magnetic, elastic_id, nullptr, n_nodes, reorder, stream, out);
}

static int mesh_create_any(const double *xyz, long n_nodes, const int *tets, long n_tets, const unsigned char *magnetic,
                           const int *elastic_id, const int *dof_of_node, long n_dof, cm_reorder reorder, void *stream, cm_mesh **out,
                           int nen);

extern "C" int cm_mesh_create_wrapped(const double *xyz, long n_nodes, const int *tets, long n_tets, const unsigned char *magnetic,
                                      const int *elastic_id, const int *dof_of_node, long n_dof, cm_reorder reorder, void *stream,
                                      cm_mesh **out)
{
    return mesh_create_any(xyz, n_nodes, tets, n_tets, magnetic, elastic_id, dof_of_node, n_dof, reorder, stream, out, 4);
}

extern "C" int cm_mesh_create_hex(const double *xyz, long n_nodes, const int *hexes, long n_hexes, const unsigned char *magnetic,
                                  const int *elastic_id, cm_reorder reorder, void *stream, cm_mesh **out)
{
    return mesh_create_any(xyz, n_nodes, hexes, n_hexes, magnetic, elastic_id, nullptr, n_nodes, reorder, stream, out, 8);
}

extern "C" int cm_mesh_create_hex_wrapped(const double *xyz, long n_nodes, const int *hexes, long n_hexes, const unsigned char *magnetic,
                                          const int *elastic_id, const int *dof_of_node, long n_dof, cm_reorder reorder, void *stream,
                                          cm_mesh **out)
{
    return mesh_create_any(xyz, n_nodes, hexes, n_hexes, magnetic, elastic_id, dof_of_node, n_dof, reorder, stream, out, 8);
}

static int mesh_create_any(const double *xyz, long n_nodes, const int *tets, long n_tets, const unsigned char *magnetic,
                           const int *elastic_id, const int *dof_of_node, long n_dof, cm_reorder reorder, void *stream, cm_mesh **out,
                           int nen)
{
    if (!xyz || !tets || !out || n_nodes <= 0 || n_tets <= 0 || n_nodes > 0x7fffffffL / 4 || n_tets > 0x7fffffffL / 16 || n_dof <= 0 ||
        n_dof > n_nodes || (!dof_of_node && n_dof != n_nodes)) {
        cm_set_error("cm_mesh_create: bad argument");
        return CM_E_BADARG;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cm_set_error("cm_mesh_create: no CUDA device (this library has no CPU fallback)");
        return CM_E_CUDA;
    }
    cudaStream_t st = (cudaStream_t)stream;
    cm_mesh *M = new (std::nothrow) cm_mesh();
    if (!M) return CM_E_ALLOC;
    int rc;
    try {
        rc = nen == 8 ? mesh_build_host_hex(M, xyz, n_nodes, tets, n_tets, magnetic, elastic_id, dof_of_node, n_dof, reorder)
                      : mesh_build_host(M, xyz, n_nodes, tets, n_tets, magnetic, elastic_id, dof_of_node, n_dof, reorder);
    } catch (const std::bad_alloc &) {
        cm_set_error("cm_mesh_create: out of host memory");
        rc = CM_E_ALLOC;
    }
    if (rc == CM_OK) {
        auto up = [&]() -> int {
            CM_TRY(upload(&M->d_order, M->order, st));
            CM_TRY(upload(&M->d_tets, M->tets, st));
            CM_TRY(upload(&M->d_rowptr, M->rowptr, st));
            CM_TRY(upload(&M->d_col, M->col, st));
            CM_TRY(upload(&M->d_n2e_ptr, M->n2e_ptr, st));
            CM_TRY(upload(&M->d_n2e, M->n2e, st));
            CM_TRY(upload(&M->d_eid, M->eid, st));
            CM_TRY(upload(&M->d_mag, M->mag, st));
            CM_TRY(upload(&M->d_xyz, M->xyz, st));
            CM_TRY(upload(&M->d_wvol, M->wvol, st));
            if (M->wrapped) {
                CM_TRY(upload(&M->d_gtets, M->gtets, st));
                CM_TRY(upload(&M->d_gxyz, M->gxyz, st));
            } else {
                M->d_gtets = M->d_tets;
                M->d_gxyz = M->d_xyz;
            }
            for (Sell &L : M->sell) {
                CM_TRY(upload(&L.d_sp, L.sp, st));
                CM_TRY(upload(&L.d_col, L.col, st));
            }
            Chunks &K = M->ck;
            CM_TRY(upload(&K.d_eptr, K.eptr, st)); CM_TRY(upload(&K.d_nptr, K.nptr, st)); CM_TRY(upload(&K.d_nodes, K.nodes, st));
            CM_TRY(upload(&K.d_ns_ptr, K.ns_ptr, st)); CM_TRY(upload(&K.d_ns_slot, K.ns_slot, st));
            CM_TRY(upload(&K.d_lid, K.lid, st)); CM_TRY(upload(&K.d_lptr, K.lptr, st)); CM_TRY(upload(&K.d_lent, K.lent, st));
            CM_TRY(upload(&M->d_emat, M->emat, st));
            CM_CUDA(cudaMalloc((void **)&M->d_red, 4096 * 16 * sizeof(double)));
            CM_CUDA(cudaMallocHost((void **)&M->h_red, 16 * sizeof(double)));
            CM_CUDA(cudaStreamSynchronize(st));
            return CM_OK;
        };
        rc = up();
    }
    if (rc != CM_OK) {
        cm_mesh_destroy(M);
        return rc;
    }
    *out = M;
    return CM_OK;
}

extern "C" int cm_mesh_destroy(cm_mesh *M)
{
    if (!M) return CM_OK;
    cudaFree(M->d_order); cudaFree(M->d_tets); cudaFree(M->d_rowptr); cudaFree(M->d_col); cudaFree(M->d_n2e_ptr);
    cudaFree(M->d_n2e); cudaFree(M->d_eid); cudaFree(M->d_mag); cudaFree(M->d_xyz); cudaFree(M->d_wvol);
    cudaFree(M->d_red); cudaFree(M->d_tmp);
    if (M->wrapped) { cudaFree(M->d_gtets); cudaFree(M->d_gxyz); }
    for (Sell &L : M->sell) { cudaFree(L.d_sp); cudaFree(L.d_col); }
    Chunks &K = M->ck;
    cudaFree(K.d_eptr); cudaFree(K.d_nptr); cudaFree(K.d_nodes); cudaFree(K.d_ns_ptr); cudaFree(K.d_ns_slot);
    cudaFree(K.d_lid); cudaFree(K.d_lptr); cudaFree(K.d_lent); cudaFree(M->d_emat);
    if (M->h_red) cudaFreeHost(M->h_red);
    delete M;
    return CM_OK;
}

extern "C" int cm_mesh_get(const cm_mesh *M, int what, void *host_out, long capacity)
{
    if (!M || !host_out) { cm_set_error("cm_mesh_get: null argument"); return CM_E_BADARG; }
    const std::vector<int> *v = nullptr;
    switch (what) {
    case CM_GET_COUNTS:
        if (capacity < 3) { cm_set_error("cm_mesh_get: capacity"); return CM_E_BADARG; }
        ((long *)host_out)[0] = M->N; ((long *)host_out)[1] = M->Ne; ((long *)host_out)[2] = M->nnz;
        return CM_OK;
    case CM_GET_LAYOUT: {
        if (capacity < 6) { cm_set_error("cm_mesh_get: capacity"); return CM_E_BADARG; }
        long *o = (long *)host_out;
        o[0] = M->sell[0].E; o[1] = M->sell[1].E; o[2] = M->ck.nchunks; o[3] = M->ck.nslots; o[4] = M->nen == 8 ? CM_HC_MAX : CM_EC_MAX; o[5] = CM_NL_MAX;
        return CM_OK;
    }
    case CM_GET_ORDER: v = &M->order; break;
    case CM_GET_IPERM: v = &M->iperm; break;
    case CM_GET_TETS: v = &M->tets; break;
    case CM_GET_TET_ORDER: v = &M->tet_order; break;
    case CM_GET_ROWPTR: v = &M->rowptr; break;
    case CM_GET_COLIDX: v = &M->col; break;
    case CM_GET_N2E_PTR: v = &M->n2e_ptr; break;
    case CM_GET_N2E: v = &M->n2e; break;
    default: cm_set_error("cm_mesh_get: unknown what=%d", what); return CM_E_BADARG;
    }
    if (capacity < (long)v->size()) { cm_set_error("cm_mesh_get: capacity %ld < %zu", capacity, v->size()); return CM_E_BADARG; }
    std::memcpy(host_out, v->data(), v->size() * sizeof(int));
    return CM_OK;
}
