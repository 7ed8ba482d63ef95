// ovl.cu -- the extern "C" entry points declared in include/ovl.h.  Argument checking, pointer staging
// (host <-> device) and precision dispatch only; the arithmetic lives in ovl_wilson.cuh / ovl_blas.cuh.
#include "ovl_engine.cuh"
#include "ovl_eigsolve.cuh"

using namespace ovl;

#define DISPATCH(c, fn, ...) ((c)->prec == OVL_F64 ? fn<double>(__VA_ARGS__) : fn<float>(__VA_ARGS__))

namespace {

int check_cfg(const int dims[4], int prec, int recon) {
    if (!dims) return OVL_EINVAL;
    long long v = 1;
    for (int i = 0; i < 4; ++i) {
        if (dims[i] < 2) return OVL_EINVAL;
        v *= dims[i];
        if (v > (1ll << 30)) return OVL_EINVAL;
    }
    if (prec != OVL_F64 && prec != OVL_F32) return OVL_EINVAL;
    if (recon != OVL_RECON18 && recon != OVL_RECON12) return OVL_EINVAL;
    return OVL_OK;
}

// bring `bytes` of caller memory to the device: in place if it already is device memory, else through *stage
int stage_to_device(ovl_ctx *c, const void *p, size_t bytes, void **stage, const void **dev) {
    if (is_device_ptr(p)) { *dev = p; return OVL_OK; }
    OVL_TRY(dev_alloc(c, stage, c->n() * sizeof(double2)));
    OVL_CUDA(c, cudaMemcpyAsync(*stage, p, bytes, cudaMemcpyHostToDevice, c->st));
    *dev = *stage;
    return OVL_OK;
}

template <typename T> int import_t(ovl_ctx *c, const void *canon_dev, void *native) {
    k_import_spinor<T, T><<<grid_for(c->n(), BLAS_THREADS), BLAS_THREADS, 0, c->st>>>(c->g.V, (const cx<T> *)canon_dev, (cx<T> *)native);
    OVL_LAUNCH_CHECK(c);
    return OVL_OK;
}
template <typename T> int export_t(ovl_ctx *c, const void *native, void *canon_dev) {
    k_export_spinor<T, T><<<grid_for(c->n(), BLAS_THREADS), BLAS_THREADS, 0, c->st>>>(c->g.V, (const cx<T> *)native, (cx<T> *)canon_dev);
    OVL_LAUNCH_CHECK(c);
    return OVL_OK;
}

int import_any(ovl_ctx *c, const void *canon, void *native) {
    const void *d = nullptr;
    OVL_TRY(stage_to_device(c, canon, c->canon_bytes(), &c->stage_in, &d));
    return DISPATCH(c, import_t, c, d, native);
}
int export_any(ovl_ctx *c, const void *native, void *canon) {
    if (is_device_ptr(canon)) return DISPATCH(c, export_t, c, native, canon);
    OVL_TRY(dev_alloc(c, &c->stage_out, c->n() * sizeof(double2)));
    OVL_TRY(DISPATCH(c, export_t, c, native, c->stage_out));
    OVL_CUDA(c, cudaMemcpyAsync(canon, c->stage_out, c->canon_bytes(), cudaMemcpyDeviceToHost, c->st));
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    return OVL_OK;
}

template <typename T> int import_links_t(ovl_ctx *c, const double2 *src_dev) {
    const size_t n = (size_t)4 * c->nrow() * 3 * c->g.V;
    k_import_links<T><<<grid_for(n, BLAS_THREADS), BLAS_THREADS, 0, c->st>>>(c->g.V, c->nrow(), src_dev, (cx<T> *)c->U);
    OVL_LAUNCH_CHECK(c);
    return OVL_OK;
}
template <typename T> int import_phi_t(ovl_ctx *c, const double2 *src_dev, int i) {
    k_import_spinor<double, T><<<grid_for(c->n(), BLAS_THREADS), BLAS_THREADS, 0, c->st>>>(
        c->g.V, src_dev, (cx<T> *)c->phi + (size_t)i * c->n());
    OVL_LAUNCH_CHECK(c);
    return OVL_OK;
}

// canonical in -> native psi_n, run `body(psi_n, out_n)`, native out_n -> canonical out
template <typename F> int with_canonical(ovl_ctx *c, const void *psi, void *out, F body) {
    if (!c) return OVL_EINVAL;
    if (!psi || !out || psi == out) return fail(c, OVL_EINVAL, "null or aliased spinor pointers");
    OVL_TRY(import_any(c, psi, c->psi_n));
    OVL_TRY(body(c->psi_n, c->out_n));
    return export_any(c, c->out_n, out);
}

}  // namespace

extern "C" {

const char *ovl_version(void) { return "ovl-b200 0.2 (sm_100a)"; }

size_t ovl_device_bytes(const int dims[4], int prec, int recon, int max_nev) {
    if (check_cfg(dims, prec, recon) != OVL_OK || max_nev < 0) return 0;
    const size_t V = (size_t)dims[0] * dims[1] * dims[2] * dims[3];
    const size_t ts = prec == OVL_F64 ? 8 : 4;
    const size_t field = V * 12 * 2 * ts;
    const size_t links = V * 4 * (recon == OVL_RECON18 ? 9 : 6) * 2 * ts;
    return links + field * (6 + 4 + (size_t)max_nev) + 2 * V * 12 * 16;
}

int ovl_create(ovl_ctx **out, const int dims[4], const void *links_c128, int prec, int recon, void *cuda_stream) {
    if (!out) return OVL_EINVAL;
    *out = nullptr;
    if (!links_c128 || check_cfg(dims, prec, recon) != OVL_OK) return OVL_EINVAL;
    ovl_ctx *c = new (std::nothrow) ovl_ctx();
    if (!c) return OVL_ENOMEM;
    for (int i = 0; i < 4; ++i) c->g.L[i] = dims[i];
    c->g.V = dims[0] * dims[1] * dims[2] * dims[3];
    c->g.sxy = dims[0] * dims[1];
    c->g.sxyz = c->g.sxy * dims[2];
    c->prec = prec;
    c->recon = recon;
    c->st = (cudaStream_t)cuda_stream;
    auto body = [&]() -> int {
        const size_t fb = c->field_bytes();
        OVL_TRY(dev_alloc(c, &c->U, c->link_bytes()));
        void **bufs[] = {&c->psi_n, &c->out_n, &c->tA, &c->tB, &c->acc, &c->g5b};
        for (void **b : bufs) OVL_TRY(dev_alloc(c, b, fb));
        c->red_nblk = grid_for(c->n(), BLAS_THREADS * 4, 148 * 8);
        OVL_CUDA(c, cudaMalloc((void **)&c->red_partial, sizeof(double) * c->red_nblk * OVL_MAX_RHS));
        OVL_CUDA(c, cudaMalloc((void **)&c->sc_dev, sizeof(double) * SC_N * OVL_MAX_RHS));
        OVL_CUDA(c, cudaMemsetAsync(c->sc_dev, 0, sizeof(double) * SC_N * OVL_MAX_RHS, c->st));
        OVL_CUDA(c, cudaMallocHost((void **)&c->sc_host, sizeof(double) * SC_N * OVL_MAX_RHS));
        OVL_CUDA(c, cudaMalloc((void **)&c->w_dev, sizeof(double2)));
        for (int i = 0; i < ovl_ctx::NPROF; ++i) {
            OVL_CUDA(c, cudaEventCreate(&c->pev0[i]));
            OVL_CUDA(c, cudaEventCreate(&c->pev1[i]));
        }
        // links: host pointers go through a temporary device copy of the canonical array
        const size_t cb = (size_t)c->g.V * 36 * sizeof(double2);
        const double2 *src = (const double2 *)links_c128;
        void *tmp = nullptr;
        if (!is_device_ptr(links_c128)) {
            OVL_CUDA(c, cudaMalloc(&tmp, cb));
            cudaError_t e = cudaMemcpyAsync(tmp, links_c128, cb, cudaMemcpyHostToDevice, c->st);
            if (e != cudaSuccess) { cudaFree(tmp); return fail(c, OVL_ECUDA, "link upload: %s", cudaGetErrorString(e)); }
            src = (const double2 *)tmp;
        }
        int rc = DISPATCH(c, import_links_t, c, src);
        cudaError_t e = cudaStreamSynchronize(c->st);
        if (tmp) cudaFree(tmp);
        if (rc != OVL_OK) return rc;
        if (e != cudaSuccess) return fail(c, OVL_ECUDA, "link import: %s", cudaGetErrorString(e));
        return OVL_OK;
    };
    int rc = body();
    if (rc != OVL_OK) { ovl_destroy(c); return rc; }
    *out = c;
    return OVL_OK;
}

int ovl_destroy(ovl_ctx *c) {
    if (!c) return OVL_EINVAL;
    cudaStreamSynchronize(c->st);
    void *bufs[] = {c->U, c->phi, c->psi_n, c->out_n, c->tA, c->tB, c->acc, c->g5b, c->cg_r, c->cg_p, c->cg_q, c->cg_Ap,
                    c->stage_in, c->stage_out, c->proj_partial, c->w_dev, c->coef_dev, c->red_partial, c->sc_dev,
                    c->multi_in, c->multi_out};
    for (void *b : bufs)
        if (b) cudaFree(b);
    for (auto &e : c->graphs)
        if (e.exec) cudaGraphExecDestroy(e.exec);
    if (c->sc_host) cudaFreeHost(c->sc_host);
    for (int i = 0; i < ovl_ctx::NPROF; ++i) {
        if (c->pev0[i]) cudaEventDestroy(c->pev0[i]);
        if (c->pev1[i]) cudaEventDestroy(c->pev1[i]);
    }
    cudaGetLastError();
    delete c;
    return OVL_OK;
}

int ovl_set_kernel(ovl_ctx *c, double m_w, double lambda_max) {
    if (!c) return OVL_EINVAL;
    if (!(lambda_max > 0) || !std::isfinite(m_w) || !std::isfinite(lambda_max)) return fail(c, OVL_EINVAL, "lambda_max must be > 0 and finite");
    c->m_w = m_w;
    c->lambda_max = lambda_max;
    c->coef_stale = true;
    ++c->poly_gen;
    return OVL_OK;
}

int ovl_set_chebyshev(ovl_ctx *c, int N, const double *alpha) {
    if (!c) return OVL_EINVAL;
    if (N < 1 || !alpha) return fail(c, OVL_EINVAL, "degree_N >= 1 and a non-null alpha are required");
    for (int m = 0; m <= N; ++m)
        if (!std::isfinite(alpha[m])) return fail(c, OVL_EINVAL, "alpha[%d] is not finite", m);
    c->alpha.assign(alpha, alpha + N + 1);
    int last = 1;
    for (int m = 1; m <= N; ++m)
        if (alpha[m] != 0.0) last = m;
    c->norders = last;
    c->coef_stale = true;
    ++c->poly_gen;
    return OVL_OK;
}

int ovl_poly_orders(const ovl_ctx *c) { return c ? c->norders : 0; }

int ovl_set_recurrence(ovl_ctx *c, int mode) {
    if (!c) return OVL_EINVAL;
    if (mode != OVL_REC_CLENSHAW && mode != OVL_REC_FORWARD) return fail(c, OVL_EINVAL, "unknown recurrence mode %d", mode);
    c->recurrence = mode;
    ++c->poly_gen;
    return OVL_OK;
}
int ovl_get_recurrence(const ovl_ctx *c) { return c ? c->recurrence : -1; }

int ovl_set_graphs(ovl_ctx *c, int on) {
    if (!c) return OVL_EINVAL;
    c->use_graphs = on != 0;
    return OVL_OK;
}

int ovl_set_deflation(ovl_ctx *c, int nev, const void *phi, const double *lambda) {
    if (!c) return OVL_EINVAL;
    if (nev < 0 || (nev > 0 && (!phi || !lambda))) return fail(c, OVL_EINVAL, "nev >= 0 and non-null phi, lambda are required");
    for (int i = 0; i < nev; ++i)
        if (!std::isfinite(lambda[i]) || std::fabs(lambda[i]) < 1e-14 * c->lambda_max)
            return fail(c, OVL_EINVAL, "lambda[%d] = %g is zero or not finite (reading R9)", i, lambda[i]);
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    c->nev = 0;
    if (nev == 0) return OVL_OK;
    if (nev > c->proj_cap) {
        if (c->phi) cudaFree(c->phi);
        if (c->proj_partial) cudaFree(c->proj_partial);
        if (c->w_dev) cudaFree(c->w_dev);
        if (c->coef_dev) cudaFree(c->coef_dev);
        c->phi = nullptr; c->proj_partial = nullptr; c->w_dev = nullptr; c->coef_dev = nullptr;
        c->proj_cap = 0;
        c->proj_nblk = (int)((c->n() + BLAS_THREADS * PROJ_EPT - 1) / (BLAS_THREADS * PROJ_EPT));
        OVL_CUDA(c, cudaMalloc(&c->phi, c->field_bytes() * nev));
        OVL_CUDA(c, cudaMalloc((void **)&c->proj_partial, sizeof(double2) * (size_t)c->proj_nblk * nev));
        OVL_CUDA(c, cudaMalloc((void **)&c->w_dev, sizeof(double2) * nev * OVL_MAX_RHS));
        OVL_CUDA(c, cudaMalloc((void **)&c->coef_dev, sizeof(double) * nev));
        c->proj_cap = nev;
    }
    const size_t vb = c->n() * sizeof(double2);  // one canonical complex128 vector
    const bool dev = is_device_ptr(phi);
    if (!dev) OVL_TRY(dev_alloc(c, &c->stage_in, vb));
    for (int i = 0; i < nev; ++i) {
        const double2 *src = (const double2 *)((const char *)phi + (size_t)i * vb);
        if (!dev) {
            OVL_CUDA(c, cudaMemcpyAsync(c->stage_in, src, vb, cudaMemcpyHostToDevice, c->st));
            src = (const double2 *)c->stage_in;
        }
        OVL_TRY(DISPATCH(c, import_phi_t, c, src, i));
    }
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    c->lambda.assign(lambda, lambda + nev);
    c->nev = nev;
    c->coef_stale = true;
    return OVL_OK;
}

int ovl_dw(ovl_ctx *c, const void *psi, void *out) {
    return with_canonical(c, psi, out, [&](const void *i, void *o) { return DISPATCH(c, dw_native, c, i, o); });
}
int ovl_khat(ovl_ctx *c, const void *psi, void *out) {
    return with_canonical(c, psi, out, [&](const void *i, void *o) { return DISPATCH(c, khat_native, c, i, o); });
}
int ovl_sign(ovl_ctx *c, const void *psi, void *out) {
    return with_canonical(c, psi, out, [&](const void *i, void *o) { return DISPATCH(c, sign_combine_native, c, 1, 0.0, 1.0, 0, 0, i, o); });
}
int ovl_overlap(ovl_ctx *c, double mu, int dagger, const void *psi, void *out) {
    return with_canonical(c, psi, out, [&](const void *i, void *o) { return DISPATCH(c, overlap_native, c, mu, dagger ? 1 : 0, i, o); });
}

int ovl_cg(ovl_ctx *c, double mu, const void *b, void *x, double tol, int maxiter, int *iters_out, double *relres_out) {
    if (!c) return OVL_EINVAL;
    if (!b || !x || b == x || !iters_out || !relres_out || maxiter < 0) return fail(c, OVL_EINVAL, "bad ovl_cg arguments");
    if (c->alpha.empty()) return fail(c, OVL_ESTATE, "ovl_set_chebyshev has not been called");
    OVL_TRY(import_any(c, b, c->psi_n));
    int rc = DISPATCH(c, cg_native, c, mu, c->psi_n, c->out_n, tol, maxiter, iters_out, relres_out);
    if (rc != OVL_OK && rc != OVL_ENOTCONV) return rc;
    int rc2 = export_any(c, c->out_n, x);
    if (rc2 != OVL_OK) return rc2;
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    return rc;
}

int ovl_cg_multi(ovl_ctx *c, int nrhs, double mu, const void *b, void *x, double tol, int maxiter, int *iters_out, double *relres_out) {
    if (!c) return OVL_EINVAL;
    if (!b || !x || b == x || !iters_out || !relres_out || maxiter < 0) return fail(c, OVL_EINVAL, "bad ovl_cg_multi arguments");
    if (nrhs < 1 || nrhs > OVL_MAX_RHS) return fail(c, OVL_EINVAL, "nrhs must be in 1..%d", OVL_MAX_RHS);
    if (c->alpha.empty()) return fail(c, OVL_ESTATE, "ovl_set_chebyshev has not been called");
    if (nrhs > c->multi_cap) {
        OVL_CUDA(c, cudaStreamSynchronize(c->st));
        if (c->multi_in) cudaFree(c->multi_in);
        if (c->multi_out) cudaFree(c->multi_out);
        c->multi_in = c->multi_out = nullptr;
        c->multi_cap = 0;
        OVL_TRY(dev_alloc(c, &c->multi_in, c->field_bytes() * nrhs));
        OVL_TRY(dev_alloc(c, &c->multi_out, c->field_bytes() * nrhs));
        c->multi_cap = nrhs;
    }
    const size_t cb = c->canon_bytes(), fb = c->field_bytes();
    for (int r = 0; r < nrhs; ++r) OVL_TRY(import_any(c, (const char *)b + r * cb, (char *)c->multi_in + r * fb));
    int rc = DISPATCH(c, cg_native, c, mu, c->multi_in, c->multi_out, tol, maxiter, iters_out, relres_out, nrhs);
    if (rc != OVL_OK && rc != OVL_ENOTCONV) return rc;
    for (int r = 0; r < nrhs; ++r) {
        int rc2 = export_any(c, (const char *)c->multi_out + r * fb, (char *)x + r * cb);
        if (rc2 != OVL_OK) return rc2;
    }
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    return rc;
}

int ovl_cg_mixed(ovl_ctx *c, ovl_ctx *c32, double mu, const void *b, void *x, double tol, double inner_tol, int max_outer,
                 int max_inner, int *outer_out, int *inner_out, double *relres_out) {
    if (!c || !c32) return OVL_EINVAL;
    if (!b || !x || b == x || !outer_out || !inner_out || !relres_out || max_outer < 0 || max_inner < 1 || !(tol > 0) || !(inner_tol > 0))
        return fail(c, OVL_EINVAL, "bad ovl_cg_mixed arguments");
    if (c->prec != OVL_F64 || c32->prec != OVL_F32) return fail(c, OVL_EINVAL, "ovl_cg_mixed needs an OVL_F64 and an OVL_F32 context");
    if (c->g.V != c32->g.V || memcmp(c->g.L, c32->g.L, sizeof c->g.L) != 0) return fail(c, OVL_EINVAL, "contexts differ in lattice size");
    if (c->st != c32->st) return fail(c, OVL_EINVAL, "both contexts must have been created on the same stream");
    if (c->alpha.empty() || c32->alpha.empty()) return fail(c, OVL_ESTATE, "ovl_set_chebyshev has not been called on both contexts");
    OVL_TRY(import_any(c, b, c->psi_n));
    int rc = cg_mixed_native(c, c32, mu, c->psi_n, c->out_n, tol, inner_tol, max_outer, max_inner, outer_out, inner_out, relres_out);
    if (rc != OVL_OK && rc != OVL_ENOTCONV) return rc;
    int rc2 = export_any(c, c->out_n, x);
    if (rc2 != OVL_OK) return rc2;
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    return rc;
}

int ovl_lowest_eigenpairs(ovl_ctx *c, int nev, double tol, int max_cycles, int filter_degree, int block, void *phi_out,
                          double *lambda_out, double *resid_out, int *cycles_out) {
    if (!c) return OVL_EINVAL;
    if (nev < 1 || !(tol > 0) || max_cycles < 0 || !phi_out || !lambda_out || !cycles_out || block < 0)
        return fail(c, OVL_EINVAL, "bad ovl_lowest_eigenpairs arguments");
    if (c->prec != OVL_F64) return fail(c, OVL_EINVAL, "the eigensolver needs an OVL_F64 context");
    return eig_lowest(c, nev, tol, max_cycles, filter_degree > 0 ? filter_degree : 100, block, 1510068970ull, phi_out, lambda_out,
                      resid_out, cycles_out);
}

const char *ovl_last_error(const ovl_ctx *c) { return c ? c->err : "null context"; }

size_t ovl_field_bytes(const ovl_ctx *c) { return c ? c->field_bytes() : 0; }
int ovl_field_import(ovl_ctx *c, const void *canonical, void *native) {
    if (!c || !canonical || !native) return OVL_EINVAL;
    return import_any(c, canonical, native);
}
int ovl_field_export(ovl_ctx *c, const void *native, void *canonical) {
    if (!c || !canonical || !native) return OVL_EINVAL;
    return export_any(c, native, canonical);
}
int ovl_dw_native(ovl_ctx *c, const void *in, void *out) {
    if (!c || !in || !out || in == out) return OVL_EINVAL;
    return DISPATCH(c, dw_native, c, in, out);
}
int ovl_overlap_native(ovl_ctx *c, double mu, int dagger, const void *in, void *out) {
    if (!c || !in || !out || in == out) return OVL_EINVAL;
    return DISPATCH(c, overlap_native, c, mu, dagger ? 1 : 0, in, out);
}

int ovl_overlap_multi_native(ovl_ctx *c, int nrhs, double mu, int dagger, const void *in, void *out) {
    if (!c || !in || !out || in == out) return OVL_EINVAL;
    if (nrhs < 1 || nrhs > OVL_MAX_RHS) return fail(c, OVL_EINVAL, "nrhs must be in 1..%d", OVL_MAX_RHS);
    return DISPATCH(c, overlap_native, c, mu, dagger ? 1 : 0, in, out, nrhs);
}

int ovl_overlap_multi(ovl_ctx *c, int nrhs, double mu, int dagger, const void *psi, void *out) {
    if (!c) return OVL_EINVAL;
    if (!psi || !out || psi == out) return fail(c, OVL_EINVAL, "null or aliased spinor pointers");
    if (nrhs < 1 || nrhs > OVL_MAX_RHS) return fail(c, OVL_EINVAL, "nrhs must be in 1..%d", OVL_MAX_RHS);
    if (nrhs > c->multi_cap) {
        OVL_CUDA(c, cudaStreamSynchronize(c->st));
        if (c->multi_in) cudaFree(c->multi_in);
        if (c->multi_out) cudaFree(c->multi_out);
        c->multi_in = c->multi_out = nullptr;
        c->multi_cap = 0;
        OVL_TRY(dev_alloc(c, &c->multi_in, c->field_bytes() * nrhs));
        OVL_TRY(dev_alloc(c, &c->multi_out, c->field_bytes() * nrhs));
        c->multi_cap = nrhs;
    }
    const size_t cb = c->canon_bytes(), fb = c->field_bytes();
    for (int r = 0; r < nrhs; ++r)
        OVL_TRY(import_any(c, (const char *)psi + r * cb, (char *)c->multi_in + r * fb));
    OVL_TRY(DISPATCH(c, overlap_native, c, mu, dagger ? 1 : 0, c->multi_in, c->multi_out, nrhs));
    for (int r = 0; r < nrhs; ++r)
        OVL_TRY(export_any(c, (const char *)c->multi_out + r * fb, (char *)out + r * cb));
    return OVL_OK;
}

int ovl_set_profiling(ovl_ctx *c, int on) {
    if (!c) return OVL_EINVAL;
    c->profiling = on != 0;
    c->prof_count = 0;
    return OVL_OK;
}
int ovl_last_poly_timing(ovl_ctx *c, float *ms, int *launches) {
    if (!c || !ms || !launches) return OVL_EINVAL;
    int n = 0;
    OVL_TRY(ovl_poly_timings(c, 1, ms, &n));
    *launches = c->last_poly_launches;
    return OVL_OK;
}
int ovl_poly_timings(ovl_ctx *c, int max_n, float *ms_out, int *n_out) {
    if (!c || !ms_out || !n_out || max_n < 1) return OVL_EINVAL;
    if (c->prof_count == 0) return fail(c, OVL_ESTATE, "no profiled polynomial loop yet");
    long long n = c->prof_count < ovl_ctx::NPROF ? c->prof_count : ovl_ctx::NPROF;
    if (n > max_n) n = max_n;
    for (long long i = 0; i < n; ++i) {  // oldest of the last n first
        const int slot = (int)((c->prof_count - n + i) % ovl_ctx::NPROF);
        OVL_CUDA(c, cudaEventSynchronize(c->pev1[slot]));
        OVL_CUDA(c, cudaEventElapsedTime(&ms_out[i], c->pev0[slot], c->pev1[slot]));
    }
    *n_out = (int)n;
    return OVL_OK;
}
long long ovl_launch_count(const ovl_ctx *c) { return c ? c->launches : 0; }

}  // extern "C"
