// C-ABI entry points (include/cupymag_b200.h): argument checks, dtype dispatch, user<->library node order.
#include <algorithm>
#include <cstring>
#include <new>

#include "cm_internal.h"

template <typename T> int mesh_volume_average(cm_mesh *M, const T *g_user, int nc, double *out_host, cudaStream_t st);

struct cm_system {
    SystemBase *impl = nullptr;
};

// ---------------------------------------------------------------- profiler
cudaEvent_t Profiler::get()
{
    if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
void Profiler::begin(int cls, cudaStream_t s, int nlaunch)
{
    launches[cls] += nlaunch;
    if (!on) return;
    Rec r;
    r.a = get(); r.b = get(); r.cls = cls;
    cudaEventRecord(r.a, s);
    pending.push_back(r);
}
void Profiler::end(cudaStream_t s)
{
    if (!on || pending.empty()) return;
    cudaEventRecord(pending.back().b, s);
}
int Profiler::flush()
{
    for (Rec &r : pending) {
        CM_CUDA(cudaEventSynchronize(r.b));
        float t = 0;
        CM_CUDA(cudaEventElapsedTime(&t, r.a, r.b));
        ms[r.cls] += t;
        pool.push_back(r.a);
        pool.push_back(r.b);
    }
    pending.clear();
    return CM_OK;
}
Profiler::~Profiler()
{
    for (Rec &r : pending) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (cudaEvent_t e : pool) cudaEventDestroy(e);
}

// ---------------------------------------------------------------- helpers
#define SYS_DISPATCH(sys, expr_d, expr_f)                                        \
    ((sys)->impl->dtype == CM_F64 ? [&]() -> int { auto *S = static_cast<System<double> *>((sys)->impl); (void)S; return (expr_d); }() \
                                  : [&]() -> int { auto *S = static_cast<System<float> *>((sys)->impl); (void)S; return (expr_f); }())

static int check_sys(const cm_system *sys, const char *fn)
{
    if (!sys || !sys->impl) { cm_set_error("%s: null system", fn); return CM_E_BADARG; }
    return CM_OK;
}

static int mode_of(cm_matrix_id id) { return id == CM_MAT_K_MECH ? MODE_BSR3 : MODE_CSR1; }

// ---------------------------------------------------------------- assemble / destroy / getters
template <typename T>
static int create_system(cm_mesh *mesh, const cm_material *mat, cm_dtype dtype, double dt, const uchar *clamp, long pin, cudaStream_t st,
                         cm_system **out)
{
    System<T> *S = new (std::nothrow) System<T>();
    if (!S) return CM_E_ALLOC;
    S->mesh = mesh; S->dtype = dtype; S->N = mesh->N; S->Ne = mesh->Ne; S->nnz = mesh->nnz; S->dt = dt;
    int rc = sys_assemble<T>(S, mat, clamp, pin, st);
    if (rc != CM_OK) { delete S; return rc; }
    cm_system *h = new (std::nothrow) cm_system();
    if (!h) { delete S; return CM_E_ALLOC; }
    h->impl = S;
    *out = h;
    return CM_OK;
}

extern "C" int cm_assemble_csr(cm_mesh *mesh, const cm_material *material, cm_dtype dtype, double dt, const unsigned char *clamp_dof,
                               long pin_node, void *stream, cm_system **out)
{
    if (!mesh || !material || !out) { cm_set_error("cm_assemble_csr: null argument"); return CM_E_BADARG; }
    if (pin_node < 0 || pin_node >= mesh->N) { cm_set_error("cm_assemble_csr: pin_node out of range"); return CM_E_BADARG; }
    if (!(material->Ms > 0) || !(material->length_scale > 0) || !(dt > 0)) { cm_set_error("cm_assemble_csr: Ms, length_scale, dt must be > 0"); return CM_E_BADARG; }
    if (material->n_elastic > 0) {
        if (!material->C_voigt) { cm_set_error("cm_assemble_csr: C_voigt is null"); return CM_E_BADARG; }
        for (long e = 0; e < mesh->Ne; e++)
            if (mesh->eid[e] < 0 || mesh->eid[e] >= material->n_elastic) {
                cm_set_error("cm_assemble_csr: elastic_id %d out of range", mesh->eid[e]);
                return CM_E_INDEX_RANGE;
            }
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == CM_F64) return create_system<double>(mesh, material, dtype, dt, clamp_dof, pin_node, st, out);
    if (dtype == CM_F32) return create_system<float>(mesh, material, dtype, dt, clamp_dof, pin_node, st, out);
    cm_set_error("cm_assemble_csr: unknown dtype");
    return CM_E_BADARG;
}

extern "C" int cm_system_destroy(cm_system *sys)
{
    if (!sys) return CM_OK;
    cudaDeviceSynchronize();
    delete sys->impl;
    delete sys;
    return CM_OK;
}

extern "C" int cm_system_get_values(const cm_system *sys, cm_matrix_id id, void *host_out, long capacity)
{
    CM_TRY(check_sys(sys, "cm_system_get_values"));
    if (!host_out) { cm_set_error("cm_system_get_values: null output"); return CM_E_BADARG; }
    cudaDeviceSynchronize();
    return SYS_DISPATCH(sys, sys_get_values<double>(S, id, host_out, capacity), sys_get_values<float>(S, id, host_out, capacity));
}

template <typename T>
static int get_geometry(const System<T> *S, int what, void *host_out, long capacity)
{
    const long Ne = S->Ne, N = S->N;
    T *out = (T *)host_out;
    switch (what) {
    case 0:
    case 1: {
        if (S->mesh->nen != 4) { cm_set_error("cm_system_get_geometry: element geometry is stored for tetrahedra only"); return CM_E_BADARG; }
        if (capacity < (what == 0 ? Ne : 12 * Ne)) break;
        std::vector<T> tmp(10 * (Ne + 8));
        CM_CUDA(cudaMemcpy(tmp.data(), S->EG, tmp.size() * sizeof(T), cudaMemcpyDeviceToHost));
        const Chunks &K = S->mesh->ck;
        for (int c = 0; c < K.nchunks; c++) {
            const long e0 = K.eptr[c], ne = K.eptr[c + 1] - e0, ne8 = (ne + 7) & ~7L;
            const T *blk = tmp.data() + 10 * e0;
            for (long el = 0; el < ne; el++) {
                if (what == 0) { out[e0 + el] = blk[el]; continue; }
                T *g = out + 12 * (e0 + el);
                for (int q = 0; q < 9; q++) g[3 + q] = blk[(q + 1) * ne8 + el];
                for (int d = 0; d < 3; d++) g[d] = -(g[3 + d] + g[6 + d] + g[9 + d]); // grad phi_0 (O-1)
            }
        }
        return CM_OK;
    }
    case 2:
        if (capacity < N) break;
        CM_CUDA(cudaMemcpy(out, S->mL, N * sizeof(T), cudaMemcpyDeviceToHost));
        return CM_OK;
    case 3:
        if (capacity < N) break;
        CM_CUDA(cudaMemcpy(out, S->mLm, N * sizeof(T), cudaMemcpyDeviceToHost));
        return CM_OK;
    default: cm_set_error("cm_system_get_geometry: unknown what=%d", what); return CM_E_BADARG;
    }
    cm_set_error("cm_system_get_geometry: capacity too small");
    return CM_E_BADARG;
}

extern "C" int cm_system_get_geometry(const cm_system *sys, int what, void *host_out, long capacity)
{
    CM_TRY(check_sys(sys, "cm_system_get_geometry"));
    if (!host_out) { cm_set_error("cm_system_get_geometry: null output"); return CM_E_BADARG; }
    cudaDeviceSynchronize();
    return SYS_DISPATCH(sys, get_geometry<double>(S, what, host_out, capacity), get_geometry<float>(S, what, host_out, capacity));
}

// ---------------------------------------------------------------- SpMV
template <typename T>
static int api_spmv(System<T> *S, cm_matrix_id id, int mode, const void *x, void *y, cudaStream_t st)
{
    const int nc = (mode == MODE_CSR1) ? 1 : 3;
    // the three-right-hand-side product gathers from a padded copy, four words per node
    CM_TRY(sys_permute_in<T>(S, (const T *)x, S->xin, mode == MODE_CSR3 ? -3 : nc, st));
    CM_TRY(sys_spmv<T>(S, id, mode, S->xin, S->xout, st));
    CM_TRY(sys_permute_out<T>(S, S->xout, (T *)y, nc, st));
    return CM_OK;
}

extern "C" int cm_spmv(cm_system *sys, cm_matrix_id id, const void *x_dev, void *y_dev, void *stream)
{
    CM_TRY(check_sys(sys, "cm_spmv"));
    if (!x_dev || !y_dev || (int)id < 0 || (int)id > CM_MAT_K_MECH) { cm_set_error("cm_spmv: bad argument"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    const int mode = mode_of(id);
    return SYS_DISPATCH(sys, api_spmv<double>(S, id, mode, x_dev, y_dev, st), api_spmv<float>(S, id, mode, x_dev, y_dev, st));
}

extern "C" int cm_spmv3(cm_system *sys, cm_matrix_id id, const void *x_dev, void *y_dev, void *stream)
{
    CM_TRY(check_sys(sys, "cm_spmv3"));
    if (!x_dev || !y_dev || (int)id < 0 || (int)id >= CM_MAT_K_MECH) { cm_set_error("cm_spmv3: bad argument (scalar matrices only)"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    return SYS_DISPATCH(sys, api_spmv<double>(S, id, MODE_CSR3, x_dev, y_dev, st), api_spmv<float>(S, id, MODE_CSR3, x_dev, y_dev, st));
}

// ---------------------------------------------------------------- CG
template <typename T>
static int api_cg(System<T> *S, cm_matrix_id id, int mode, const void *b, void *x, double tol, int maxiter, int fixed, int precond,
                  int *iters, double *relres, cudaStream_t st)
{
    const int nc = (mode == MODE_CSR1) ? 1 : 3, nr = (mode == MODE_CSR3) ? 3 : 1;
    const int cls = id == CM_MAT_K_MS ? CM_PROF_CG_MS : (id == CM_MAT_K_MECH ? CM_PROF_CG_MECH : CM_PROF_CG_GS);
    CM_TRY(sys_permute_in<T>(S, (const T *)b, S->bvec, nc, st));
    CM_TRY(sys_permute_in<T>(S, (const T *)x, S->xin, nc, st));
    CM_TRY(sys_cg<T>(S, id, mode, S->bvec, S->xin, tol, maxiter, fixed, nr == 3 ? 7u : 1u, 7, cls, precond, st));
    S->hist_nr = nr;
    CM_TRY(sys_permute_out<T>(S, S->xin, (T *)x, nc, st));
    CM_CUDA(cudaMemcpyAsync(S->h_res + 7, S->d_res + 7, sizeof(CgResult), cudaMemcpyDeviceToHost, st));
    CM_CUDA(cudaStreamSynchronize(st));
    const CgResult &R = S->h_res[7];
    int mxit = 0;
    for (int c = 0; c < nr; c++) {
        if (iters) iters[c] = R.iters[c];
        if (relres) relres[c] = R.relres[c];
        S->prof.cg_iters[cls] += R.iters[c];
        mxit = std::max(mxit, R.iters[c]);
    }
    S->prof.cg_passes[cls] += mxit + 1; // one matrix pass per iteration plus the r0 = b - A x0 pass
    S->hist_len = S->hist_on ? (long)std::min<long>((long)(mxit + 1) * nr, CM_HIST_CAP / nr * nr) : 0; // nothing was recorded otherwise
    return R.status;
}

extern "C" int cm_cg_solve_pc(cm_system *sys, cm_matrix_id id, const void *b_dev, void *x_dev, double tol, int maxiter, int fixed_iters,
                              int precond, int *iters_out, double *relres_out, void *stream)
{
    CM_TRY(check_sys(sys, "cm_cg_solve"));
    if (!b_dev || !x_dev || (int)id < 0 || (int)id > CM_MAT_K_MECH) { cm_set_error("cm_cg_solve: bad argument"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    const int mode = mode_of(id);
    return SYS_DISPATCH(sys, api_cg<double>(S, id, mode, b_dev, x_dev, tol, maxiter, fixed_iters, precond, iters_out, relres_out, st),
                        api_cg<float>(S, id, mode, b_dev, x_dev, tol, maxiter, fixed_iters, precond, iters_out, relres_out, st));
}

extern "C" int cm_cg_solve3_pc(cm_system *sys, cm_matrix_id id, const void *b_dev, void *x_dev, double tol, int maxiter, int fixed_iters,
                               int precond, int *iters_out, double *relres_out, void *stream)
{
    CM_TRY(check_sys(sys, "cm_cg_solve3"));
    if (!b_dev || !x_dev || (int)id < 0 || (int)id >= CM_MAT_K_MECH) { cm_set_error("cm_cg_solve3: bad argument (scalar matrices only)"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    return SYS_DISPATCH(sys, api_cg<double>(S, id, MODE_CSR3, b_dev, x_dev, tol, maxiter, fixed_iters, precond, iters_out, relres_out, st),
                        api_cg<float>(S, id, MODE_CSR3, b_dev, x_dev, tol, maxiter, fixed_iters, precond, iters_out, relres_out, st));
}

extern "C" int cm_cg_solve(cm_system *sys, cm_matrix_id id, const void *b_dev, void *x_dev, double tol, int maxiter, int fixed_iters,
                           int *iters_out, double *relres_out, void *stream)
{
    return cm_cg_solve_pc(sys, id, b_dev, x_dev, tol, maxiter, fixed_iters, CM_PC_NONE, iters_out, relres_out, stream);
}

extern "C" int cm_cg_solve3(cm_system *sys, cm_matrix_id id, const void *b_dev, void *x_dev, double tol, int maxiter, int fixed_iters,
                            int *iters_out, double *relres_out, void *stream)
{
    return cm_cg_solve3_pc(sys, id, b_dev, x_dev, tol, maxiter, fixed_iters, CM_PC_NONE, iters_out, relres_out, stream);
}

template <typename T>
static int api_spmv_matfree(System<T> *S, const void *x, void *y, cudaStream_t st)
{
    CM_TRY(sys_permute_in<T>(S, (const T *)x, S->xin, 3, st));
    CM_TRY(sys_spmv_matfree<T>(S, S->xin, S->xout, st));
    return sys_permute_out<T>(S, S->xout, (T *)y, 3, st);
}

extern "C" int cm_spmv_matfree(cm_system *sys, const void *x_dev, void *y_dev, void *stream)
{
    CM_TRY(check_sys(sys, "cm_spmv_matfree"));
    if (!x_dev || !y_dev) { cm_set_error("cm_spmv_matfree: null argument"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    return SYS_DISPATCH(sys, api_spmv_matfree<double>(S, x_dev, y_dev, st), api_spmv_matfree<float>(S, x_dev, y_dev, st));
}

template <typename T>
static int api_cg_matfree(System<T> *S, const void *b, void *x, double tol, int maxiter, int fixed, int precond, int *iters, double *relres,
                          cudaStream_t st)
{
    CM_TRY(sys_permute_in<T>(S, (const T *)b, S->bvec, 3, st));
    CM_TRY(sys_permute_in<T>(S, (const T *)x, S->xin, 3, st));
    CM_TRY(sys_cg_matfree<T>(S, S->bvec, S->xin, tol, maxiter, fixed, precond, 7, st));
    CM_TRY(sys_permute_out<T>(S, S->xin, (T *)x, 3, st));
    CM_CUDA(cudaMemcpyAsync(S->h_res + 7, S->d_res + 7, sizeof(CgResult), cudaMemcpyDeviceToHost, st));
    CM_CUDA(cudaStreamSynchronize(st));
    const CgResult &R = S->h_res[7];
    if (iters) *iters = R.iters[0];
    if (relres) *relres = R.relres[0];
    S->prof.cg_iters[CM_PROF_CG_MECH] += R.iters[0];
    S->prof.cg_passes[CM_PROF_CG_MECH] += R.iters[0] + 1;
    return R.status;
}

extern "C" int cm_cg_solve_matfree(cm_system *sys, const void *b_dev, void *x_dev, double tol, int maxiter, int fixed_iters, int precond,
                                   int *iters_out, double *relres_out, void *stream)
{
    CM_TRY(check_sys(sys, "cm_cg_solve_matfree"));
    if (!b_dev || !x_dev) { cm_set_error("cm_cg_solve_matfree: null argument"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    sys->impl->hist_len = 0; // cm_cg_history covers cm_cg_solve* only: after this call it reads empty, not an earlier solve's curve
    return SYS_DISPATCH(sys, api_cg_matfree<double>(S, b_dev, x_dev, tol, maxiter, fixed_iters, precond, iters_out, relres_out, st),
                        api_cg_matfree<float>(S, b_dev, x_dev, tol, maxiter, fixed_iters, precond, iters_out, relres_out, st));
}

extern "C" int cm_cg_history_enable(cm_system *sys, int on)
{
    CM_TRY(check_sys(sys, "cm_cg_history_enable"));
    sys->impl->hist_on = on != 0;
    sys->impl->hist_len = 0;
    return CM_OK;
}

extern "C" int cm_cg_history(cm_system *sys, double *host_out, long capacity, long *n_out)
{
    CM_TRY(check_sys(sys, "cm_cg_history"));
    if (!host_out || !n_out || capacity < 0) { cm_set_error("cm_cg_history: bad argument"); return CM_E_BADARG; }
    const long n = std::min(capacity, sys->impl->hist_len);
    if (n > 0) CM_CUDA(cudaMemcpy(host_out, sys->impl->d_hist, n * sizeof(double), cudaMemcpyDeviceToHost));
    *n_out = n;
    return CM_OK;
}

// ---------------------------------------------------------------- field / RHS
template <typename T>
static int api_field_rhs(System<T> *S, cm_rhs_id id, const void *m, const void *U, const void *u, const cm_step_params *p, double coeff,
                         void *b, cudaStream_t st)
{
    const unsigned terms = p ? p->terms : 0u;
    double hext[3] = {0, 0, 0};
    if (p) for (int d = 0; d < 3; d++) hext[d] = p->Hext[d] / S->Ms;
    CM_TRY(sys_permute_in<T>(S, (const T *)m, S->m, 3, st));
    const bool need_hd = (id == CM_OUT_HD) || ((id == CM_RHS_GS || id == CM_OUT_FIELD) && (terms & (CM_TERM_DEMAG | CM_TERM_FARFIELD)));
    const bool need_sig = (id == CM_OUT_SIGMA) || ((id == CM_RHS_GS || id == CM_OUT_FIELD) && (terms & CM_TERM_MAGEL));
    if (id == CM_RHS_MS || need_hd) CM_TRY(sys_mbar<T>(S, S->m, st));
    if (id == CM_RHS_MS) {
        CM_TRY(sys_rhs_ms<T>(S, S->m, S->xout, st));
        return sys_permute_out<T>(S, S->xout, (T *)b, 1, st);
    }
    if (id == CM_RHS_MECH) {
        CM_TRY(sys_rhs_mech<T>(S, S->m, S->xout, st));
        return sys_permute_out<T>(S, S->xout, (T *)b, 3, st);
    }
    if (need_hd) {
        const unsigned t = (id == CM_OUT_HD && !p) ? (CM_TERM_DEMAG | CM_TERM_FARFIELD) : terms;
        if ((t & CM_TERM_DEMAG)) {
            if (!U) { cm_set_error("cm_field_rhs: U_dev is null but DEMAG is on"); return CM_E_BADARG; }
            CM_TRY(sys_permute_in<T>(S, (const T *)U, S->U, 1, st));
        }
        CM_TRY(sys_demag_field<T>(S, S->U, t, S->hd, st));
        if (id == CM_OUT_HD) return sys_permute_out<T>(S, S->hd, (T *)b, 3, st);
    }
    if (need_sig) {
        if (!u) { cm_set_error("cm_field_rhs: u_dev is null but MAGEL is on"); return CM_E_BADARG; }
        CM_TRY(sys_permute_in<T>(S, (const T *)u, S->u, 3, st));
        CM_TRY(sys_stress<T>(S, S->u, S->m, st));
    }
    if (id == CM_OUT_SIGMA) {
        CM_TRY(sys_field<T>(S, S->m, S->hd, hext, CM_TERM_MAGEL, (T *)nullptr, S->sig, st));
        return sys_permute_out<T>(S, S->sig, (T *)b, 6, st);
    }
    CM_TRY(sys_field<T>(S, S->m, S->hd, hext, terms, S->hn, (T *)nullptr, st));
    if (id == CM_OUT_FIELD) return sys_permute_out<T>(S, S->hn, (T *)b, 3, st);
    if (id == CM_RHS_GS) {
        CM_TRY(sys_axpby3<T>(S, S->m, S->hn, (T)coeff, S->f, st));
        CM_TRY(sys_spmv<T>(S, CM_MAT_MASS, MODE_CSR3, S->f, S->xout, st));
        return sys_permute_out<T>(S, S->xout, (T *)b, 3, st);
    }
    cm_set_error("cm_field_rhs: unknown id %d", (int)id);
    return CM_E_BADARG;
}

extern "C" int cm_field_rhs(cm_system *sys, cm_rhs_id id, const void *m_dev, const void *U_dev, const void *u_dev,
                            const cm_step_params *params, double coeff, void *b_dev, void *stream)
{
    CM_TRY(check_sys(sys, "cm_field_rhs"));
    if (!m_dev || !b_dev) { cm_set_error("cm_field_rhs: null m_dev / b_dev"); return CM_E_BADARG; }
    if ((id == CM_RHS_GS || id == CM_OUT_FIELD) && !params) { cm_set_error("cm_field_rhs: params required"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    return SYS_DISPATCH(sys, api_field_rhs<double>(S, id, m_dev, U_dev, u_dev, params, coeff, b_dev, st),
                        api_field_rhs<float>(S, id, m_dev, U_dev, u_dev, params, coeff, b_dev, st));
}

// ---------------------------------------------------------------- volume average
extern "C" int cm_volume_average(const cm_mesh *mesh, cm_dtype dtype, const void *g_dev, int ncomp, double *out_host, void *stream)
{
    if (!mesh || !g_dev || !out_host) { cm_set_error("cm_volume_average: null argument"); return CM_E_BADARG; }
    cm_mesh *M = const_cast<cm_mesh *>(mesh); // scratch buffers only
    cudaStream_t st = (cudaStream_t)stream;
    if (dtype == CM_F64) return mesh_volume_average<double>(M, (const double *)g_dev, ncomp, out_host, st);
    if (dtype == CM_F32) return mesh_volume_average<float>(M, (const float *)g_dev, ncomp, out_host, st);
    cm_set_error("cm_volume_average: unknown dtype");
    return CM_E_BADARG;
}

// ---------------------------------------------------------------- GSPM step
extern "C" int cm_gspm_step(cm_system *sys, const cm_step_params *params, void *m_dev, void *U_dev, void *u_dev, cm_step_info *info,
                            void *stream)
{
    CM_TRY(check_sys(sys, "cm_gspm_step"));
    if (!params) { cm_set_error("cm_gspm_step: null params"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    sys->impl->hist_len = 0; // cm_cg_history covers cm_cg_solve* only: after this call it reads empty, not an earlier solve's curve
    return SYS_DISPATCH(sys, sys_step<double>(S, params, (double *)m_dev, (double *)U_dev, (double *)u_dev, info, st),
                        sys_step<float>(S, params, (float *)m_dev, (float *)U_dev, (float *)u_dev, info, st));
}

template <typename T>
static int api_step_host(System<T> *S, const cm_step_params *p, void *m_h, void *U_h, void *u_h, cm_step_info *info, cudaStream_t st)
{
    const long N = S->N;
    const bool demag = p->terms & CM_TERM_DEMAG, magel = p->terms & CM_TERM_MAGEL;
    if (!m_h || (demag && !U_h) || (magel && !u_h)) { cm_set_error("cm_gspm_step_host: null field pointer"); return CM_E_BADARG; }
    CM_CUDA(cudaMemcpyAsync(S->stg_m, m_h, 3 * N * sizeof(T), cudaMemcpyHostToDevice, st));
    if (demag) CM_CUDA(cudaMemcpyAsync(S->stg_U, U_h, N * sizeof(T), cudaMemcpyHostToDevice, st));
    if (magel) CM_CUDA(cudaMemcpyAsync(S->stg_u, u_h, 3 * N * sizeof(T), cudaMemcpyHostToDevice, st));
    cm_step_info local;
    int rc = sys_step<T>(S, p, S->stg_m, S->stg_U, S->stg_u, info ? info : &local, st);
    if (rc < 0 && rc != CM_E_CG_MAXITER && rc != CM_E_CG_BREAKDOWN) return rc;
    CM_CUDA(cudaMemcpyAsync(m_h, S->stg_m, 3 * N * sizeof(T), cudaMemcpyDeviceToHost, st));
    if (demag) CM_CUDA(cudaMemcpyAsync(U_h, S->stg_U, N * sizeof(T), cudaMemcpyDeviceToHost, st));
    if (magel) CM_CUDA(cudaMemcpyAsync(u_h, S->stg_u, 3 * N * sizeof(T), cudaMemcpyDeviceToHost, st));
    CM_CUDA(cudaStreamSynchronize(st));
    return rc;
}

extern "C" int cm_gspm_step_host(cm_system *sys, const cm_step_params *params, void *m_host, void *U_host, void *u_host,
                                 cm_step_info *info, void *stream)
{
    CM_TRY(check_sys(sys, "cm_gspm_step_host"));
    if (!params) { cm_set_error("cm_gspm_step_host: null params"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    sys->impl->hist_len = 0; // cm_cg_history covers cm_cg_solve* only: after this call it reads empty, not an earlier solve's curve
    return SYS_DISPATCH(sys, api_step_host<double>(S, params, m_host, U_host, u_host, info, st),
                        api_step_host<float>(S, params, m_host, U_host, u_host, info, st));
}

// ---------------------------------------------------------------- hysteresis driver
extern "C" int cm_hysteresis_run(cm_system *sys, const cm_step_params *base, const cm_hyst_params *hp, void *m_dev, void *U_dev,
                                 void *u_dev, double *H_log, double *mbar_log, int *steps_log, cm_hyst_result *result, void *stream)
{
    CM_TRY(check_sys(sys, "cm_hysteresis_run"));
    if (!base || !hp) { cm_set_error("cm_hysteresis_run: null params"); return CM_E_BADARG; }
    cudaStream_t st = (cudaStream_t)stream;
    sys->impl->hist_len = 0; // cm_cg_history covers cm_cg_solve* only: after this call it reads empty, not an earlier solve's curve
    return SYS_DISPATCH(sys, sys_hysteresis<double>(S, base, hp, (double *)m_dev, (double *)U_dev, (double *)u_dev, H_log, mbar_log, steps_log, result, st),
                        sys_hysteresis<float>(S, base, hp, (float *)m_dev, (float *)U_dev, (float *)u_dev, H_log, mbar_log, steps_log, result, st));
}

// ---------------------------------------------------------------- options
extern "C" int cm_system_set_option(cm_system *sys, int option, int value)
{
    CM_TRY(check_sys(sys, "cm_system_set_option"));
    switch (option) {
    case CM_OPT_STORED_GEOMETRY:
        if (value < 0 || value > 2) break;
        sys->impl->geometry_mode = value;
        return CM_OK;
    case CM_OPT_NO_FUSED_S5S8:
        if (value < 0 || value > 1) break;
        sys->impl->no_fuse = value != 0;
        return CM_OK;
    }
    cm_set_error("cm_system_set_option: unknown option %d or value %d out of range", option, value);
    return CM_E_BADARG;
}

// ---------------------------------------------------------------- profile
extern "C" int cm_profile_enable(cm_system *sys, int on)
{
    CM_TRY(check_sys(sys, "cm_profile_enable"));
    sys->impl->prof.on = on != 0;
    return CM_OK;
}
extern "C" int cm_profile_get(cm_system *sys, cm_profile *out)
{
    CM_TRY(check_sys(sys, "cm_profile_get"));
    if (!out) { cm_set_error("cm_profile_get: null output"); return CM_E_BADARG; }
    Profiler &P = sys->impl->prof;
    CM_TRY(P.flush());
    for (int c = 0; c < CM_PROF_NCLASS; c++) {
        out->ms[c] = P.ms[c]; out->launches[c] = P.launches[c]; out->cg_iters[c] = P.cg_iters[c];
        out->cg_matrix_passes[c] = P.cg_passes[c];
    }
    return CM_OK;
}
extern "C" int cm_profile_reset(cm_system *sys)
{
    CM_TRY(check_sys(sys, "cm_profile_reset"));
    Profiler &P = sys->impl->prof;
    CM_TRY(P.flush());
    for (int c = 0; c < CM_PROF_NCLASS; c++) { P.ms[c] = 0; P.launches[c] = 0; P.cg_iters[c] = 0; P.cg_passes[c] = 0; }
    return CM_OK;
}
