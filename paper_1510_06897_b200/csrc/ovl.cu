// ovl.cu -- the extern "C" entry points declared in include/ovl.h.  Argument checking, pointer staging
// (host <-> device) and precision dispatch only; the arithmetic lives in ovl_wilson.cuh / ovl_blas.cuh.
#include "ovl_engine.cuh"
#include "ovl_eigsolve.cuh"
#include "ovl_group.cuh"

#include <fcntl.h>
#include <sys/mman.h>
#include <sys/stat.h>
#include <unistd.h>

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

// native staging of the multi-right-hand-side calls with canonical arguments
int ensure_multi_staging(ovl_ctx *c, int nrhs) {
    if (nrhs <= c->multi_cap) return OVL_OK;
    if (c->ws_mode) return fail(c, OVL_EINVAL, "%d right-hand sides exceed the workspace capacity max_rhs = %d", nrhs, c->max_rhs);
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    dev_release(c, &c->multi_in);
    dev_release(c, &c->multi_out);
    c->multi_cap = 0;
    OVL_TRY(dev_alloc(c, &c->multi_in, c->field_bytes() * nrhs));
    OVL_TRY(dev_alloc(c, &c->multi_out, c->field_bytes() * nrhs));
    c->multi_cap = nrhs;
    return OVL_OK;
}

int set_deflation_strided(ovl_ctx *c, int nev, const void *phi, const double *lambda, size_t vec_stride);

// canonical in -> native psi_n, run `body(psi_n, out_n)`, native out_n -> canonical out
template <typename F> int with_canonical(ovl_ctx *c, const void *psi, void *out, F body) {
    if (!c) return OVL_EINVAL;
    if (!psi || !out || psi == out) return fail(c, OVL_EINVAL, "null or aliased spinor pointers");
    OVL_TRY(import_any(c, psi, c->psi_n));
    OVL_TRY(body(c->psi_n, c->out_n));
    return export_any(c, c->out_n, out);
}


// ---- the device-memory plan of a context (the caller owns the workspace).  One routine enumerates every
// buffer in a fixed order; ovl_workspace_bytes sums it and create_impl carves it, so the two cannot disagree.
struct WsGeom { size_t V; };
WsGeom ws_geom(const int dims[4]) { return WsGeom{(size_t)dims[0] * dims[1] * dims[2] * dims[3]}; }
enum WsId { WS_U, WS_PSI, WS_OUT, WS_TA, WS_TB, WS_ACC, WS_G5B, WS_RED, WS_SC, WS_W, WS_CG_R, WS_CG_P, WS_CG_Q, WS_CG_AP,
            WS_MULTI_IN, WS_MULTI_OUT, WS_PHI, WS_PROJ, WS_COEF, WS_STAGE_IN, WS_STAGE_OUT, WS_EIG };
size_t eig_ws_bytes(size_t V, int cap) { return eig_ws_total(V, cap); }  // ovl_eigsolve.cuh's work block for `cap` vectors
template <typename F> void ws_visit(WsGeom g, int prec, int recon, int max_nev, int max_rhs, int eig_cap, F f) {
    const size_t ts = prec == OVL_F64 ? 8 : 4, n = 12 * g.V, fb = n * 2 * ts;
    const size_t red_nblk = grid_for(n, BLAS_THREADS * 4, 148 * 8), proj_nblk = (n + BLAS_THREADS * PROJ_EPT - 1) / (BLAS_THREADS * PROJ_EPT);
    f(WS_U, g.V * 4 * (recon == OVL_RECON18 ? 9 : 6) * 2 * ts);
    // psi_n .. g5b are contiguous and come first after the links: the canonical link array (36 V complex128) is staged there
    // during ovl_create when the links are passed as a host pointer
    f(WS_PSI, fb); f(WS_OUT, fb);
    f(WS_TA, fb * max_rhs); f(WS_TB, fb * max_rhs); f(WS_ACC, fb * max_rhs); f(WS_G5B, fb * max_rhs);
    f(WS_RED, sizeof(double) * red_nblk * OVL_MAX_RHS);
    f(WS_SC, sizeof(double) * SC_N * OVL_MAX_RHS);
    f(WS_W, sizeof(double2) * (max_nev > 0 ? max_nev : 1) * OVL_MAX_RHS);
    // everything below is optional for a library-owned context (allocated on first use); a workspace holds all of it
    f(WS_CG_R, fb * max_rhs); f(WS_CG_P, fb * max_rhs); f(WS_CG_Q, fb * max_rhs); f(WS_CG_AP, fb * max_rhs);
    if (max_rhs > 1) { f(WS_MULTI_IN, fb * max_rhs); f(WS_MULTI_OUT, fb * max_rhs); }
    if (max_nev > 0) {
        f(WS_PHI, fb * max_nev);
        f(WS_PROJ, sizeof(double2) * proj_nblk * max_nev * max_rhs);
        f(WS_COEF, sizeof(double) * max_nev);
    }
    f(WS_STAGE_IN, n * sizeof(double2)); f(WS_STAGE_OUT, n * sizeof(double2));
    if (eig_cap > 0) f(WS_EIG, eig_ws_bytes(g.V, eig_cap));
}

int create_impl(ovl_ctx **out, const int dims[4], const void *links_c128, int prec, int recon, void *cuda_stream, void *ws,
                size_t ws_bytes, int max_nev, int max_rhs, int eig_cap) {
    ovl_ctx *c = new (std::nothrow) ovl_ctx();
    if (!c) return OVL_ENOMEM;
    for (int i = 0; i < 4; ++i) c->g.L[i] = dims[i];
    c->g.V = dims[0] * dims[1] * dims[2] * dims[3];
    c->g.sxy = dims[0] * dims[1];
    c->g.sxyz = c->g.sxy * dims[2];
    {   // L2-aware sweep (ovl_types.cuh): only when two time slices of a spinor plus one of the links no longer fit half the
        // L2 (48^3 x 96 class), and only when z-slabs of whole 128-site tiles exist
        const size_t ts = prec == OVL_F64 ? 8 : 4;
        const size_t slice_bytes = (size_t)c->g.sxyz * (2 * 24 + 4 * (size_t)(recon == OVL_RECON18 ? 18 : 12)) * ts;
        if (slice_bytes > (size_t)40 << 20) {
            int best = 0;
            for (int zw = 1; zw <= dims[2]; ++zw)
                if (dims[2] % zw == 0 && ((size_t)c->g.sxy * zw) % 128 == 0 && (size_t)c->g.sxy * zw <= 32768) best = zw;
            if (best > 0 && best < dims[2]) { c->sweep.tpc = c->g.sxy * best / 128; c->sweep.nzs = dims[2] / best; }
        }
    }
    // brick order (ovl_types.cuh): possible whenever Lz and Lt are even (brick_geom); chosen by default for 2^15 <= V <= 2^17
    // (12^3 x 24 ... 16^3 x 32: -2 ... -5 % per order; smaller lattices are faster in plain order, 8^3 x 32 4.6 against 5.0 us,
    // from 16^3 x 48 on there is no difference)
    if (dims[2] % 2 == 0 && dims[3] % 2 == 0) {
        c->brick_geom.half = c->g.sxyz / 2;
        c->brick_geom.nchunk = (c->brick_geom.half + ovl::BRICK_GS - 1) / ovl::BRICK_GS;
    }
    if (c->g.V >= (1 << 15) && c->g.V <= (1 << 17)) c->brick = c->brick_geom;
    c->brick_auto = c->brick;
    c->prec = prec;
    c->recon = recon;
    c->st = (cudaStream_t)cuda_stream;
    {
        int dv = 0, sms = 0;
        if (cudaGetDevice(&dv) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dv) == cudaSuccess && sms > 0) c->sm_count = sms;
        cudaGetLastError();
    }
    c->red_nblk = grid_for(c->n(), BLAS_THREADS * 4, 148 * 8);
    c->proj_nblk = (int)((c->n() + BLAS_THREADS * PROJ_EPT - 1) / (BLAS_THREADS * PROJ_EPT));
    auto body = [&]() -> int {
        const WsGeom wg = ws_geom(dims);
        if (ws) {  // caller-owned: carve everything now, never allocate again
            c->ws_mode = true;
            c->arena.base = (char *)ws; c->arena.size = ws_bytes;
            c->max_nev = max_nev; c->max_rhs = max_rhs; c->eig_cap = eig_cap;
        } else {   // library-owned: ONE cudaMalloc for the base set (links + recurrence vectors + reduction scratch)
            size_t base = 0;
            ws_visit(wg, prec, recon, 0, 1, 0, [&](int id, size_t b) { if (id <= WS_W) base += ws_round(b ? b : 16); });
            void *p = nullptr;
            OVL_CUDA(c, cudaMalloc(&p, base));
            c->owned.push_back(p);
            c->arena.base = (char *)p; c->arena.size = base;
        }
        int rc = OVL_OK;
        ws_visit(wg, prec, recon, max_nev, max_rhs, eig_cap, [&](int id, size_t b) {
            if (rc != OVL_OK || (!ws && id > WS_W)) return;
            void **slot = nullptr;
            switch (id) {
                case WS_U: slot = &c->U; break;
                case WS_PSI: slot = &c->psi_n; break;
                case WS_OUT: slot = &c->out_n; break;
                case WS_TA: slot = &c->tA; break;
                case WS_TB: slot = &c->tB; break;
                case WS_ACC: slot = &c->acc; break;
                case WS_G5B: slot = &c->g5b; break;
                case WS_RED: slot = (void **)&c->red_partial; break;
                case WS_SC: slot = (void **)&c->sc_dev; break;
                case WS_W: slot = (void **)&c->w_dev; break;
                case WS_CG_R: slot = &c->cg_r; break;
                case WS_CG_P: slot = &c->cg_p; break;
                case WS_CG_Q: slot = &c->cg_q; break;
                case WS_CG_AP: slot = &c->cg_Ap; break;
                case WS_MULTI_IN: slot = &c->multi_in; break;
                case WS_MULTI_OUT: slot = &c->multi_out; break;
                case WS_PHI: slot = &c->phi; break;
                case WS_PROJ: slot = (void **)&c->proj_partial; break;
                case WS_COEF: slot = (void **)&c->coef_dev; break;
                case WS_STAGE_IN: slot = &c->stage_in; break;
                case WS_STAGE_OUT: slot = &c->stage_out; break;
                case WS_EIG: slot = &c->eig_ws; c->eig_ws_bytes = b; break;
            }
            rc = dev_alloc(c, slot, b);
        });
        if (rc != OVL_OK) return rc;
        c->work_nrhs = max_rhs;
        if (ws) {
            c->cg_nrhs = max_rhs;
            c->multi_cap = max_rhs > 1 ? max_rhs : 0;
            c->proj_cap = max_nev;
            c->proj_rhs = max_rhs;
        }
        OVL_CUDA(c, cudaMemsetAsync(c->sc_dev, 0, sizeof(double) * SC_N * OVL_MAX_RHS, c->st));
        OVL_CUDA(c, cudaMallocHost((void **)&c->sc_host, sizeof(double) * 2 * SC_N * OVL_MAX_RHS));
        for (int i = 0; i < 2; ++i) OVL_CUDA(c, cudaEventCreateWithFlags(&c->cg_ev[i], cudaEventDisableTiming));
        for (int i = 0; i < ovl_ctx::NPROF; ++i) {
            OVL_CUDA(c, cudaEventCreate(&c->pev0[i]));
            OVL_CUDA(c, cudaEventCreate(&c->pev1[i]));
        }
        // links: a host array is staged through the (still unused) recurrence vectors, which start at psi_n and are
        // contiguous: 6 fields >= 576 V bytes = the canonical link array in either precision
        const size_t cb = (size_t)c->g.V * 36 * sizeof(double2);
        const double2 *src = (const double2 *)links_c128;
        if (!is_device_ptr(links_c128)) {
            if ((size_t)((char *)c->g5b + c->field_bytes() * max_rhs - (char *)c->psi_n) < cb)
                return fail(c, OVL_ENOMEM, "internal: link staging area too small");
            OVL_CUDA(c, cudaMemcpyAsync(c->psi_n, links_c128, cb, cudaMemcpyHostToDevice, c->st));
            src = (const double2 *)c->psi_n;
        }
        rc = DISPATCH(c, import_links_t, c, src);
        cudaError_t e = cudaStreamSynchronize(c->st);
        if (rc != OVL_OK) return rc;
        if (e != cudaSuccess) return fail(c, OVL_ECUDA, "link import: %s", cudaGetErrorString(e));
        return OVL_OK;
    };
    int rc = body();
    if (rc != OVL_OK) { ovl_destroy(c); return rc; }
    *out = c;
    return OVL_OK;
}

}  // namespace

extern "C" {

const char *ovl_version(void) { return "ovl-b200 0.2 (sm_100a)"; }

size_t ovl_workspace_bytes(const int dims[4], int prec, int recon, int max_nev, int max_rhs, int eig_block) {
    if (check_cfg(dims, prec, recon) != OVL_OK || max_nev < 0 || max_rhs < 1 || max_rhs > OVL_MAX_RHS || eig_block < 0 || eig_block > 128) return 0;
    size_t total = 0;
    ws_visit(ws_geom(dims), prec, recon, max_nev, max_rhs, eig_block, [&](int, size_t b) { total += ws_round(b ? b : 16); });
    return total;
}

size_t ovl_device_bytes(const int dims[4], int prec, int recon, int max_nev) {
    return ovl_workspace_bytes(dims, prec, recon, max_nev, 1, 0);
}

int ovl_create_ws(ovl_ctx **out, const int dims[4], const void *links_c128, int prec, int recon, int max_nev, int max_rhs,
                  int eig_block, void *workspace, size_t workspace_bytes, void *cuda_stream) {
    if (!out) return OVL_EINVAL;
    *out = nullptr;
    if (!links_c128 || !workspace || check_cfg(dims, prec, recon) != OVL_OK) return OVL_EINVAL;
    const size_t need = ovl_workspace_bytes(dims, prec, recon, max_nev, max_rhs, eig_block);
    if (need == 0 || workspace_bytes < need || ((uintptr_t)workspace % WS_ALIGN) != 0 || !is_device_ptr(workspace)) return OVL_EINVAL;
    return create_impl(out, dims, links_c128, prec, recon, cuda_stream, workspace, workspace_bytes, max_nev, max_rhs, eig_block);
}

int ovl_create(ovl_ctx **out, const int dims[4], const void *links_c128, int prec, int recon, void *cuda_stream) {
    if (!out) return OVL_EINVAL;
    *out = nullptr;
    if (!links_c128 || check_cfg(dims, prec, recon) != OVL_OK) return OVL_EINVAL;
    return create_impl(out, dims, links_c128, prec, recon, cuda_stream, nullptr, 0, 0, 1, 0);
}

int ovl_destroy(ovl_ctx *c) {
    if (!c) return OVL_EINVAL;
    cudaStreamSynchronize(c->st);
    for (void *b : c->owned)   // library-owned allocations only: a caller-owned workspace is never freed
        if (b) cudaFree(b);
    for (auto &e : c->graphs)
        if (e.exec) cudaGraphExecDestroy(e.exec);
    if (c->sc_host) cudaFreeHost(c->sc_host);
    for (int i = 0; i < 2; ++i)
        if (c->cg_ev[i]) cudaEventDestroy(c->cg_ev[i]);
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

int ovl_set_fused_variant(ovl_ctx *c, int variant) {
    if (!c) return OVL_EINVAL;
    if (variant != OVL_FUSED_REGISTER && variant != OVL_FUSED_BULK && variant != OVL_FUSED_PLAIN && variant != OVL_FUSED_BRICK)
        return fail(c, OVL_EINVAL, "unknown fused-kernel variant %d", variant);
    if (variant == OVL_FUSED_BRICK && c->brick_geom.nchunk == 0) return fail(c, OVL_EINVAL, "brick order needs Lz and Lt even");
    c->fused_variant = variant;
    c->brick = variant == OVL_FUSED_PLAIN ? ovl::Brick{0, 0} : variant == OVL_FUSED_BRICK ? c->brick_geom : c->brick_auto;
    ++c->poly_gen;  // captured graphs hold the other kernel
    return OVL_OK;
}

int ovl_set_graphs(ovl_ctx *c, int on) {
    if (!c) return OVL_EINVAL;
    c->use_graphs = on != 0;
    return OVL_OK;
}

int ovl_set_deflation(ovl_ctx *c, int nev, const void *phi, const double *lambda) {
    return c ? set_deflation_strided(c, nev, phi, lambda, c->n() * sizeof(double2)) : OVL_EINVAL;
}

}  // extern "C"

namespace {
// the deflation space from vectors that start `vec_stride` bytes apart (a slab's part of global eigenvectors)
int set_deflation_strided(ovl_ctx *c, int nev, const void *phi, const double *lambda, size_t vec_stride) {
    if (nev < 0 || (nev > 0 && (!phi || !lambda))) return fail(c, OVL_EINVAL, "nev >= 0 and non-null phi, lambda are required");
    for (int i = 0; i < nev; ++i)
        if (!std::isfinite(lambda[i]) || std::fabs(lambda[i]) < 1e-14 * c->lambda_max)
            return fail(c, OVL_EINVAL, "lambda[%d] = %g is zero or not finite (reading R9)", i, lambda[i]);
    if (nev > c->proj_cap && c->ws_mode)  // refused before any state changes: the current deflation space stays in force
        return fail(c, OVL_EINVAL, "%d eigenvectors exceed the workspace capacity max_nev = %d", nev, c->max_nev);
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    c->nev = 0;
    if (nev == 0) return OVL_OK;
    if (nev > c->proj_cap) {
        dev_release(c, &c->phi);
        dev_release(c, (void **)&c->proj_partial);
        dev_release(c, (void **)&c->w_dev);
        dev_release(c, (void **)&c->coef_dev);
        c->proj_cap = 0;
        OVL_TRY(dev_alloc(c, &c->phi, c->field_bytes() * nev));
        c->proj_rhs = c->work_nrhs;
        OVL_TRY(dev_alloc(c, (void **)&c->proj_partial, sizeof(double2) * (size_t)c->proj_nblk * nev * c->proj_rhs));
        OVL_TRY(dev_alloc(c, (void **)&c->w_dev, sizeof(double2) * nev * OVL_MAX_RHS));
        OVL_TRY(dev_alloc(c, (void **)&c->coef_dev, sizeof(double) * nev));
        c->proj_cap = nev;
    }
    const size_t vb = c->n() * sizeof(double2);  // one canonical complex128 vector
    const bool dev = is_device_ptr(phi);
    if (!dev) OVL_TRY(dev_alloc(c, &c->stage_in, vb));
    for (int i = 0; i < nev; ++i) {
        const double2 *src = (const double2 *)((const char *)phi + (size_t)i * vec_stride);
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
}  // namespace

extern "C" {

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

int ovl_cg_chiral(ovl_ctx *c, double mu, int chirality, const void *b, void *x, double tol, int maxiter, int *iters_out,
                  double *relres_out) {
    if (!c) return OVL_EINVAL;
    if (!b || !x || b == x || !iters_out || !relres_out || maxiter < 0 || (chirality != 1 && chirality != -1))
        return fail(c, OVL_EINVAL, "bad ovl_cg_chiral arguments (chirality must be +1 or -1)");
    if (c->alpha.empty()) return fail(c, OVL_ESTATE, "ovl_set_chebyshev has not been called");
    OVL_TRY(import_any(c, b, c->psi_n));
    int rc = DISPATCH(c, cg_native, c, mu, c->psi_n, c->out_n, tol, maxiter, iters_out, relres_out, 1, chirality);
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
    OVL_TRY(ensure_multi_staging(c, nrhs));
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

int ovl_cg_multi_chiral(ovl_ctx *c, int nrhs, double mu, int chirality, const void *b, void *x, double tol, int maxiter, int *iters_out,
                        double *relres_out) {
    if (!c) return OVL_EINVAL;
    if (!b || !x || b == x || !iters_out || !relres_out || maxiter < 0 || (chirality != 1 && chirality != -1))
        return fail(c, OVL_EINVAL, "bad ovl_cg_multi_chiral arguments (chirality must be +1 or -1)");
    if (nrhs < 1 || nrhs > OVL_MAX_RHS) return fail(c, OVL_EINVAL, "nrhs must be in 1..%d", OVL_MAX_RHS);
    if (c->alpha.empty()) return fail(c, OVL_ESTATE, "ovl_set_chebyshev has not been called");
    OVL_TRY(ensure_multi_staging(c, nrhs));
    const size_t cb = c->canon_bytes(), fb = c->field_bytes();
    for (int r = 0; r < nrhs; ++r) OVL_TRY(import_any(c, (const char *)b + r * cb, (char *)c->multi_in + r * fb));
    int rc = DISPATCH(c, cg_native, c, mu, c->multi_in, c->multi_out, tol, maxiter, iters_out, relres_out, nrhs, chirality);
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

int ovl_cg_mixed_chiral(ovl_ctx *c, ovl_ctx *c32, double mu, int chirality, const void *b, void *x, double tol, double inner_tol,
                        int max_outer, int max_inner, int *outer_out, int *inner_out, double *relres_out) {
    if (!c || !c32) return OVL_EINVAL;
    if (!b || !x || b == x || !outer_out || !inner_out || !relres_out || max_outer < 0 || max_inner < 1 || !(tol > 0) || !(inner_tol > 0) ||
        (chirality != 1 && chirality != -1))
        return fail(c, OVL_EINVAL, "bad ovl_cg_mixed_chiral arguments (chirality must be +1 or -1)");
    if (c->prec != OVL_F64 || c32->prec != OVL_F32) return fail(c, OVL_EINVAL, "ovl_cg_mixed_chiral needs an OVL_F64 and an OVL_F32 context");
    if (c->g.V != c32->g.V || memcmp(c->g.L, c32->g.L, sizeof c->g.L) != 0) return fail(c, OVL_EINVAL, "contexts differ in lattice size");
    if (c->st != c32->st) return fail(c, OVL_EINVAL, "both contexts must have been created on the same stream");
    if (c->alpha.empty() || c32->alpha.empty()) return fail(c, OVL_ESTATE, "ovl_set_chebyshev has not been called on both contexts");
    OVL_TRY(import_any(c, b, c->psi_n));
    int rc = cg_mixed_native(c, c32, mu, c->psi_n, c->out_n, tol, inner_tol, max_outer, max_inner, outer_out, inner_out, relres_out, chirality);
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
    return eig_lowest(c, nullptr, nev, tol, max_cycles, filter_degree > 0 ? filter_degree : 100, block, 1510068970ull, phi_out, lambda_out,
                      resid_out, cycles_out);
}

int ovl_lowest_eigenpairs_mixed(ovl_ctx *c, ovl_ctx *c32, int nev, double tol, int max_cycles, int filter_degree, int block,
                                void *phi_out, double *lambda_out, double *resid_out, int *cycles_out, int *f32_cycles_out) {
    if (!c || !c32) return OVL_EINVAL;
    if (nev < 1 || !(tol > 0) || max_cycles < 0 || !phi_out || !lambda_out || !cycles_out || block < 0)
        return fail(c, OVL_EINVAL, "bad ovl_lowest_eigenpairs_mixed arguments");
    if (c->prec != OVL_F64 || c32->prec != OVL_F32) return fail(c, OVL_EINVAL, "ovl_lowest_eigenpairs_mixed needs an OVL_F64 and an OVL_F32 context");
    if (c->g.V != c32->g.V || memcmp(c->g.L, c32->g.L, sizeof c->g.L) != 0) return fail(c, OVL_EINVAL, "contexts differ in lattice size");
    if (c->st != c32->st) return fail(c, OVL_EINVAL, "both contexts must have been created on the same stream");
    if (c->m_w != c32->m_w || c->lambda_max != c32->lambda_max) return fail(c, OVL_EINVAL, "contexts differ in m_w or lambda_max (ovl_set_kernel)");
    return eig_lowest(c, c32, nev, tol, max_cycles, filter_degree > 0 ? filter_degree : 100, block, 1510068970ull, phi_out, lambda_out,
                      resid_out, cycles_out, f32_cycles_out);
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
    OVL_TRY(ensure_multi_staging(c, nrhs));
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


// ---------------------------------------------------------------------------------------------- t-split lattice (ovl_group)

}  // extern "C"

namespace {
// one slab context + its wire block (one device allocation: halos, ghost U_t slice, reduction scratch) + its two events
int group_add_slab(ovl_group *g, int r, const int ldims[4], const void *links_local, void *stream, bool ipc) {
    ovl_ctx *c = nullptr;
    const int rc = create_impl(&c, ldims, links_local, g->prec, g->recon, stream, nullptr, 0, 0, 1, 0);
    if (rc != OVL_OK) return gfail(g, rc, "slab %d: context creation failed", r);
    g->s[r] = c;
    c->use_graphs = false;  // the launch sequence of a slab is interleaved with event waits on its neighbours
    const WireLayout L = wire_layout((size_t)c->g.sxyz, c->nrow(), c->tsize());
    void *base = nullptr;
    GRP_CUDA(g, cudaMalloc(&base, L.total));  // its own allocation: exported as ONE IPC handle when the slabs are processes
    c->owned.push_back(base);
    wire_point(g->w[r], L, base);
    for (int b = 0; b < 2; ++b)
        GRP_CUDA(g, cudaEventCreateWithFlags(&g->w[r].ev[b], cudaEventDisableTiming | (ipc ? cudaEventInterprocess : 0)));
    return OVL_OK;
}
// U_t of slab lo's last time slice -> the ghost slice of slab `to` (a peer or IPC pointer), on lo's stream
int group_send_ghost_links(ovl_group *g, int lo, int to) {
    ovl_ctx *cl = g->s[lo];
    DevGuard dg(g->dev[lo]);
    const int npl = cl->nrow() * 3;
    const size_t ne = (size_t)npl * cl->g.sxyz;
    if (g->prec == OVL_F64)
        k_pack_ut_last<double><<<(unsigned)((ne + 255) / 256), 256, 0, cl->st>>>(
            cl->g.V, cl->g.sxyz, npl, (const double2 *)cl->U + (size_t)3 * npl * cl->g.V, (double2 *)g->w[to].u_lo);
    else
        k_pack_ut_last<float><<<(unsigned)((ne + 255) / 256), 256, 0, cl->st>>>(
            cl->g.V, cl->g.sxyz, npl, (const float2 *)cl->U + (size_t)3 * npl * cl->g.V, (float2 *)g->w[to].u_lo);
    GRP_CUDA(g, cudaGetLastError());
    GRP_CUDA(g, cudaStreamSynchronize(cl->st));
    return OVL_OK;
}
int group_check(const int dims[4], int nslabs, int prec, int recon) {
    if (check_cfg(dims, prec, recon) != OVL_OK) return OVL_EINVAL;
    if (nslabs < 1 || nslabs > MAX_SLABS || dims[3] % nslabs != 0 || dims[3] / nslabs < 2) return OVL_EINVAL;
    return OVL_OK;
}
struct SlabBlob {  // what ovl_slab_export hands to the other processes (fits OVL_SLAB_BLOB_BYTES)
    int magic, rank;
    cudaIpcMemHandle_t mem;
    cudaIpcEventHandle_t ev[2];
};
static_assert(sizeof(SlabBlob) <= OVL_SLAB_BLOB_BYTES, "blob too large");
}  // namespace

extern "C" {

int ovl_group_create(ovl_group **out, const int dims[4], int nslabs, const void *links_c128, int prec, int recon,
                     void *const *cuda_streams, const int *devices) {
    if (!out) return OVL_EINVAL;
    *out = nullptr;
    if (!links_c128 || !cuda_streams || group_check(dims, nslabs, prec, recon) != OVL_OK) return OVL_EINVAL;
    ovl_group *g = new (std::nothrow) ovl_group();
    if (!g) return OVL_ENOMEM;
    g->n = nslabs; g->prec = prec; g->recon = recon;
    for (int i = 0; i < 4; ++i) g->gdims[i] = dims[i];
    const int ldims[4] = {dims[0], dims[1], dims[2], dims[3] / nslabs};
    g->Vloc = (size_t)ldims[0] * ldims[1] * ldims[2] * ldims[3];
    g->w.resize(nslabs);
    g->s.assign(nslabs, nullptr);
    int cur = 0;
    cudaGetDevice(&cur);
    for (int r = 0; r < nslabs; ++r) { g->dev.push_back(devices ? devices[r] : cur); g->mine.push_back(r); }
    for (int r = 1; r < nslabs; ++r)
        if (g->dev[r] != g->dev[0]) g->split_launch = true;
    auto body = [&]() -> int {
        for (int r = 0; r < nslabs; ++r)  // every slab reads its neighbours' halos and every slab's reduction scratch
            for (int q = 0; q < nslabs; ++q)
                if (g->dev[r] != g->dev[q]) {
                    DevGuard dg(g->dev[r]);
                    cudaError_t e = cudaDeviceEnablePeerAccess(g->dev[q], 0);
                    if (e != cudaSuccess && e != cudaErrorPeerAccessAlreadyEnabled)
                        return gfail(g, OVL_ECUDA, "no peer access from device %d to %d: %s", g->dev[r], g->dev[q], cudaGetErrorString(e));
                    cudaGetLastError();
                }
        for (int r = 0; r < nslabs; ++r) {
            DevGuard dg(g->dev[r]);
            const char *lk = (const char *)links_c128 + (size_t)r * g->Vloc * 36 * sizeof(double2);
            OVL_TRY(group_add_slab(g, r, ldims, lk, cuda_streams[r], false));
        }
        // the backward t hop of a slab's first time slice needs U_t of the lower neighbour's last slice: sent once, here
        for (int r = 0; r < nslabs; ++r) OVL_TRY(group_send_ghost_links(g, lo_of(g, r), r));
        return OVL_OK;
    };
    const int rc = body();
    if (rc != OVL_OK) { ovl_group_destroy(g); return rc; }
    *out = g;
    return OVL_OK;
}

/* ---- one process per GPU: the same slabs, wired through CUDA IPC ---- */
int ovl_slab_create(ovl_group **out, const int dims[4], int rank, int nranks, const void *links_local_c128, int prec, int recon,
                    void *cuda_stream, const char *shm_name) {
    if (!out) return OVL_EINVAL;
    *out = nullptr;
    if (!links_local_c128 || !shm_name || group_check(dims, nranks, prec, recon) != OVL_OK || rank < 0 || rank >= nranks) return OVL_EINVAL;
    if (strlen(shm_name) == 0 || strlen(shm_name) >= sizeof(((ovl_group *)0)->shm_name)) return OVL_EINVAL;
    ovl_group *g = new (std::nothrow) ovl_group();
    if (!g) return OVL_ENOMEM;
    g->n = nranks; g->prec = prec; g->recon = recon; g->distributed = true; g->rank = rank;
    g->split_launch = nranks > 1;
    for (int i = 0; i < 4; ++i) g->gdims[i] = dims[i];
    const int ldims[4] = {dims[0], dims[1], dims[2], dims[3] / nranks};
    g->Vloc = (size_t)ldims[0] * ldims[1] * ldims[2] * ldims[3];
    g->w.resize(nranks);
    g->s.assign(nranks, nullptr);
    int cur = 0;
    cudaGetDevice(&cur);
    g->dev.assign(nranks, cur);
    g->mine.push_back(rank);
    strcpy(g->shm_name, shm_name);
    auto body = [&]() -> int {
        // "rounds issued" counters shared by the processes of the group (a record must have been issued before a wait on it)
        const size_t bytes = sizeof(unsigned long long) * MAX_SLABS;
        const int fd = shm_open(shm_name, O_CREAT | O_RDWR, 0600);
        if (fd < 0) return gfail(g, OVL_ECUDA, "shm_open(%s) failed", shm_name);
        if (ftruncate(fd, (off_t)bytes) != 0) { close(fd); return gfail(g, OVL_ECUDA, "ftruncate on %s failed", shm_name); }
        void *m = mmap(nullptr, bytes, PROT_READ | PROT_WRITE, MAP_SHARED, fd, 0);
        close(fd);
        if (m == MAP_FAILED) return gfail(g, OVL_ECUDA, "mmap of %s failed", shm_name);
        g->issued = (volatile unsigned long long *)m;
        __atomic_store_n(&g->issued[rank], 0ull, __ATOMIC_RELEASE);
        return group_add_slab(g, rank, ldims, links_local_c128, cuda_stream, true);
    };
    const int rc = body();
    if (rc != OVL_OK) { ovl_group_destroy(g); return rc; }
    *out = g;
    return OVL_OK;
}

int ovl_slab_export(ovl_group *g, void *blob) {
    if (!g || !blob || !g->distributed) return OVL_EINVAL;
    SlabBlob b;
    memset(&b, 0, sizeof b);
    b.magic = 0x0516a5b; b.rank = g->rank;
    DevGuard dg(g->dev[g->rank]);
    GRP_CUDA(g, cudaIpcGetMemHandle(&b.mem, g->w[g->rank].base));
    for (int i = 0; i < 2; ++i) GRP_CUDA(g, cudaIpcGetEventHandle(&b.ev[i], g->w[g->rank].ev[i]));
    memset(blob, 0, OVL_SLAB_BLOB_BYTES);
    memcpy(blob, &b, sizeof b);
    return OVL_OK;
}

int ovl_slab_connect(ovl_group *g, const void *blobs) {
    if (!g || !blobs || !g->distributed) return OVL_EINVAL;
    ovl_ctx *c = g->s[g->rank];
    DevGuard dg(g->dev[g->rank]);
    const WireLayout L = wire_layout((size_t)c->g.sxyz, c->nrow(), c->tsize());
    for (int q = 0; q < g->n; ++q) {
        if (q == g->rank) continue;
        SlabBlob b;
        memcpy(&b, (const char *)blobs + (size_t)q * OVL_SLAB_BLOB_BYTES, sizeof b);
        if (b.magic != 0x0516a5b || b.rank != q) return gfail(g, OVL_EINVAL, "blob %d is not the export of slab %d", q, q);
        void *base = nullptr;
        GRP_CUDA(g, cudaIpcOpenMemHandle(&base, b.mem, cudaIpcMemLazyEnablePeerAccess));
        wire_point(g->w[q], L, base);
        g->w[q].remote = true;
        for (int i = 0; i < 2; ++i) GRP_CUDA(g, cudaIpcOpenEventHandle(&g->w[q].ev[i], b.ev[i]));
    }
    // my last U_t slice is the upper neighbour's ghost slice (the caller runs a barrier across the processes after this call)
    return group_send_ghost_links(g, g->rank, hi_of(g, g->rank));
}

int ovl_group_destroy(ovl_group *g) {
    if (!g) return OVL_EINVAL;
    for (int r : g->mine)
        if (g->s[r]) {
            DevGuard dg(g->dev[r]);
            cudaStreamSynchronize(g->s[r]->st);
        }
    for (size_t q = 0; q < g->w.size(); ++q) {
        if (g->w[q].remote) {
            if (g->w[q].base) cudaIpcCloseMemHandle(g->w[q].base);
            for (int b = 0; b < 2; ++b)
                if (g->w[q].ev[b]) cudaEventDestroy(g->w[q].ev[b]);
        }
    }
    for (int r : g->mine) {
        DevGuard dg(g->dev[r]);
        for (int b = 0; b < 2; ++b)
            if (g->w[r].ev[b]) cudaEventDestroy(g->w[r].ev[b]);
        if (g->s[r]) ovl_destroy(g->s[r]);
    }
    if (g->issued) {
        munmap((void *)g->issued, sizeof(unsigned long long) * MAX_SLABS);
        if (g->rank == 0) shm_unlink(g->shm_name);
    }
    cudaGetLastError();
    delete g;
    return OVL_OK;
}

int ovl_group_slabs(const ovl_group *g) { return g ? g->n : 0; }
int ovl_group_set_split_launch(ovl_group *g, int on) {
    if (!g) return OVL_EINVAL;
    g->split_launch = on != 0;
    return OVL_OK;
}
const char *ovl_group_last_error(const ovl_group *g) { return g ? g->err : "null group"; }
long long ovl_group_launch_count(const ovl_group *g) {
    long long t = 0;
    if (g) for (int r : g->mine) t += g->s[r]->launches;
    return t;
}

int ovl_group_set_kernel(ovl_group *g, double m_w, double lambda_max) {
    if (!g) return OVL_EINVAL;
    for (int r : g->mine) GRP_TRY(g, r, ovl_set_kernel(g->s[r], m_w, lambda_max));
    return OVL_OK;
}
int ovl_group_set_chebyshev(ovl_group *g, int N, const double *alpha) {
    if (!g) return OVL_EINVAL;
    for (int r : g->mine) GRP_TRY(g, r, ovl_set_chebyshev(g->s[r], N, alpha));
    return OVL_OK;
}
int ovl_group_set_deflation(ovl_group *g, int nev, const void *phi, const double *lambda) {
    if (!g) return OVL_EINVAL;
    if (nev > WIRE_MAX_NEV) return gfail(g, OVL_EINVAL, "at most %d deflation vectors on a split lattice", WIRE_MAX_NEV);
    // phi holds, per eigenvector, the parts of this process's slabs back to back (all slabs: the global vector)
    const size_t vstride = g->mine.size() * g->Vloc * 12 * sizeof(double2);
    for (size_t li = 0; li < g->mine.size(); ++li) {
        const int r = g->mine[li];
        DevGuard dg(g->dev[r]);
        const char *p = phi ? (const char *)phi + li * g->Vloc * 12 * sizeof(double2) : nullptr;
        GRP_TRY(g, r, set_deflation_strided(g->s[r], nev, p, lambda, vstride));
    }
    g->nev = nev;
    return OVL_OK;
}

}  // extern "C"

namespace {
// canonical GLOBAL field -> every slab's psi_n, body on the slabs' native fields, every slab's out_n -> canonical GLOBAL field
template <typename F> int group_with_canonical(ovl_group *g, const void *psi, void *out, F body) {
    if (!g) return OVL_EINVAL;
    if (!psi || !out || psi == out) return gfail(g, OVL_EINVAL, "null or aliased spinor pointers");
    std::vector<void *> in(g->n, nullptr), o(g->n, nullptr);
    for (size_t li = 0; li < g->mine.size(); ++li) {  // this process's slabs lie back to back in psi / out
        const int r = g->mine[li];
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        GRP_TRY(g, r, import_any(c, (const char *)psi + li * c->canon_bytes(), c->psi_n));
        in[r] = c->psi_n; o[r] = c->out_n;
    }
    const int rc = body(in.data(), o.data());
    if (rc != OVL_OK && rc != OVL_ENOTCONV) return rc;
    for (size_t li = 0; li < g->mine.size(); ++li) {
        const int r = g->mine[li];
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        GRP_TRY(g, r, export_any(c, c->out_n, (char *)out + li * c->canon_bytes()));
    }
    for (int r : g->mine) {  // the group calls synchronise: their result spans several streams
        DevGuard dg(g->dev[r]);
        GRP_CUDA(g, cudaStreamSynchronize(g->s[r]->st));
    }
    return rc;
}
#define GDISPATCH(g, fn, ...) ((g)->prec == OVL_F64 ? fn<double>(__VA_ARGS__) : fn<float>(__VA_ARGS__))
}  // namespace

extern "C" {

int ovl_group_dw(ovl_group *g, const void *psi, void *out) {
    return group_with_canonical(g, psi, out, [&](void *const *i, void *const *o) { return GDISPATCH(g, group_stencil, g, 0, i, o); });
}
int ovl_group_khat(ovl_group *g, const void *psi, void *out) {
    return group_with_canonical(g, psi, out, [&](void *const *i, void *const *o) { return GDISPATCH(g, group_stencil, g, 1, i, o); });
}
int ovl_group_sign(ovl_group *g, const void *psi, void *out) {
    return group_with_canonical(g, psi, out, [&](void *const *i, void *const *o) { return GDISPATCH(g, group_sign_combine, g, 0.0, 1.0, 0, 0, i, o); });
}
int ovl_group_overlap(ovl_group *g, double mu, int dagger, const void *psi, void *out) {
    return group_with_canonical(g, psi, out, [&](void *const *i, void *const *o) { return GDISPATCH(g, group_overlap, g, mu, dagger ? 1 : 0, i, o); });
}
int ovl_group_cg(ovl_group *g, double mu, const void *b, void *x, double tol, int maxiter, int *iters_out, double *relres_out) {
    if (!g) return OVL_EINVAL;
    if (!iters_out || !relres_out || maxiter < 0) return gfail(g, OVL_EINVAL, "bad ovl_group_cg arguments");
    if (g->s[g->mine[0]]->alpha.empty()) return gfail(g, OVL_ESTATE, "ovl_group_set_chebyshev has not been called");
    return group_with_canonical(g, b, x, [&](void *const *i, void *const *o) { return GDISPATCH(g, group_cg, g, mu, i, o, tol, maxiter, iters_out, relres_out); });
}

}  // extern "C"
