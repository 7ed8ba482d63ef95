// ovl_engine.cuh -- host-side drivers: kernel launches for one stencil pass, the Chebyshev loop (a4),
// deflation (a5-a7), overlap assembly (a8) and CG on D^dag D (a9).  Everything here only enqueues kernels.
#pragma once
#include "ovl_blas.cuh"
#include "ovl_ctx.cuh"
#include "ovl_wilson.cuh"
#include "ovl_wilson_tp.cuh"

namespace ovl {

#define OVL_LAUNCH_CHECK(c)                                                                      \
    do {                                                                                         \
        ++(c)->launches;                                                                         \
        cudaError_t e_ = cudaGetLastError();                                                     \
        if (e_ != cudaSuccess) return fail((c), OVL_ECUDA, "kernel launch: %s", cudaGetErrorString(e_)); \
    } while (0)

// launch shape of the fused kernel: 128-thread CTAs (tiles of 128 consecutive sites).  Several right-hand sides, the L2-aware
// sweep and the t-split slabs: fp64 3 CTAs/SM at up to 168 registers, fp32 4 CTAs/SM.  The single-right-hand-side fp64 kernel
// (MINB_SINGLE): 2 CTAs/SM, up to 255 registers, no spills -- at boost clocks the same speed as 3 CTAs/SM (ptxas turns the
// registers into deeper load batches), under the power cap of a long run and together with the evict-first loads of the
// single-use streams 3 % faster (A/B on one box: 130.1 -> 126.0 us/order)
template <typename T> struct WilsonCfg;
template <> struct WilsonCfg<double> { static constexpr int THREADS = 128, MINB = 3, MINB_SINGLE = 2; };
template <> struct WilsonCfg<float> { static constexpr int THREADS = 128, MINB = 4, MINB_SINGLE = 4; };

struct WilsonArgs {
    const void *in = nullptr, *prev = nullptr, *psi = nullptr;
    void *out = nullptr, *acc = nullptr;
    double c_diag = 0, c_hop = 0, a_psi = 0, a_acc = 0, a_init = 0;
    double c_prev = 1.0;  // out = ... - c_prev * prev (1 everywhere except the eigensolver's scaled filter recurrence)
    int flip = 0, nrhs = 1;
};

// The bulk-copy variant (ovl_wilson_tp.cuh; ovl_set_fused_variant): persistent warps, the warp's own links landed in shared
// memory by cp.async.bulk + mbarrier.  4 warps per CTA; 2 (fp64) / 4 (fp32) CTAs per SM keep 147 KB of landing zone and
// leave 81 KB of L1 for the neighbour reuse -- the best staged configuration measured on B200, and still
// slower than the register-landing kernel, which therefore stays the default.
template <typename T, int RECON, int FLAGS> inline void launch_wilson_tp(ovl_ctx *c, const WilsonArgs &a, const StepParams<T> &sp) {
    constexpr int NW = 4, MINB = sizeof(T) == 8 ? 2 : 4, OPT = STG_LINKS;
    using SM = TpSmem<T, RECON, FLAGS, OPT>;
    auto kern = k_wilson_tp<T, RECON, FLAGS, OPT, NW, MINB>;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SM::total(NW));
        attr_set = true;
    }
    const int nsub = c->g.V / 32;
    int grid = c->sm_count * MINB;
    if (grid * NW > nsub) grid = (nsub + NW - 1) / NW;
    kern<<<grid, NW * 32, SM::total(NW), c->st>>>(c->g, (const cx<T> *)c->U, (const cx<T> *)a.in, (const cx<T> *)a.prev, (const cx<T> *)a.psi,
                                                  (cx<T> *)a.out, sp, nsub);
}

template <typename T, int RECON, int FLAGS> inline void launch_wilson_t(ovl_ctx *c, const WilsonArgs &a) {
    constexpr int TH = WilsonCfg<T>::THREADS;
    const int grid = ((c->g.V + TH - 1) / TH) * a.nrhs;
    StepParams<T> sp{(T)a.c_hop, (T)(a.c_diag / a.c_hop), (T)(a.c_prev / a.c_hop), (T)(a.a_psi / a.c_hop), (T)a.a_acc, (T)a.a_init, a.flip};
    if constexpr (!(FLAGS & (K_ACC | K_ACCI | K_NOWRITE))) {
        if (c->fused_variant == OVL_FUSED_BULK && a.nrhs == 1 && c->g.V % 32 == 0 && c->g.sxyz % 32 == 0) {
            launch_wilson_tp<T, RECON, FLAGS>(c, a, sp);
            return;
        }
    }
    if (c->brick.nchunk > 0 && a.nrhs == 1) {
        static_assert(TH == 4 * BRICK_GS, "brick CTAs are 4 groups of BRICK_GS sites");
        k_wilson_fused_brick<T, RECON, FLAGS><<<c->brick.nchunk * (c->g.L[3] / 2), TH, 0, c->st>>>(
            c->g, (const cx<T> *)c->U, (const cx<T> *)a.in, (const cx<T> *)a.prev, (const cx<T> *)a.psi, (cx<T> *)a.out, (cx<T> *)a.acc, sp, c->brick);
        return;
    }
    if (a.nrhs > 1)
        k_wilson_fused_multi<T, RECON, FLAGS, TH, WilsonCfg<T>::MINB><<<grid, TH, 0, c->st>>>(
            c->g, (const cx<T> *)c->U, (const cx<T> *)a.in, (const cx<T> *)a.prev, (const cx<T> *)a.psi, (cx<T> *)a.out, (cx<T> *)a.acc, sp,
            a.nrhs, c->n());
    else if (c->sweep.tpc > 0)
        k_wilson_fused_swept<T, RECON, FLAGS, TH, WilsonCfg<T>::MINB><<<grid, TH, 0, c->st>>>(
            c->g, (const cx<T> *)c->U, (const cx<T> *)a.in, (const cx<T> *)a.prev, (const cx<T> *)a.psi, (cx<T> *)a.out, (cx<T> *)a.acc, sp, c->sweep);
    else if ((FLAGS & K_PREV) || c->g.V <= (1 << 18))
        k_wilson_fused<T, RECON, FLAGS, TH, WilsonCfg<T>::MINB_SINGLE><<<grid, TH, 0, c->st>>>(
            c->g, (const cx<T> *)c->U, (const cx<T> *)a.in, (const cx<T> *)a.prev, (const cx<T> *)a.psi, (cx<T> *)a.out, (cx<T> *)a.acc, sp);
    else  // no b_{k+2} stream (D_W, K^, the first two Clenshaw launches) on a large lattice: 3 CTAs/SM is 3 % faster at boost clocks
        k_wilson_fused<T, RECON, FLAGS, TH, WilsonCfg<T>::MINB><<<grid, TH, 0, c->st>>>(
            c->g, (const cx<T> *)c->U, (const cx<T> *)a.in, (const cx<T> *)a.prev, (const cx<T> *)a.psi, (cx<T> *)a.out, (cx<T> *)a.acc, sp);
}

template <typename T, int FLAGS> inline int launch_wilson(ovl_ctx *c, const WilsonArgs &a) {
    if (c->recon == OVL_RECON18) launch_wilson_t<T, 18, FLAGS>(c, a);
    else launch_wilson_t<T, 12, FLAGS>(c, a);
    OVL_LAUNCH_CHECK(c);
    return OVL_OK;
}

// out = D_W in
template <typename T> int dw_native(ovl_ctx *c, const void *in, void *out) {
    WilsonArgs a;
    a.in = in; a.out = out; a.c_diag = 4.0; a.c_hop = -0.5;
    return launch_wilson<T, 0>(c, a);
}
// out = K^ in
template <typename T> int khat_native(ovl_ctx *c, const void *in, void *out) {
    WilsonArgs a;
    a.in = in; a.out = out; a.c_diag = (4.0 - c->m_w) / c->lambda_max; a.c_hop = -0.5 / c->lambda_max;
    return launch_wilson<T, K_G5>(c, a);
}

// acc = sum_{m=0}^{N} alpha_m T_m(K^) src by the forward recurrence exactly as printed:
// t_0 = src, t_1 = K^ src, t_{m+1} = 2 K^ t_m - t_{m-1}, acc = sum alpha_m t_m.  N launches.
template <typename T> int cheb_forward(ovl_ctx *c, const void *src, int nrhs) {
    const double cd = (4.0 - c->m_w) / c->lambda_max, ch = -0.5 / c->lambda_max;
    const std::vector<double> &al = c->alpha;
    const int N = c->norders;
    WilsonArgs a;
    a.nrhs = nrhs;
    a.in = src; a.out = c->tA; a.acc = c->acc; a.c_diag = cd; a.c_hop = ch; a.a_init = al[0]; a.a_acc = al[1];
    if (N == 1) OVL_TRY((launch_wilson<T, K_G5 | K_ACCI | K_NOWRITE>(c, a)));
    else OVL_TRY((launch_wilson<T, K_G5 | K_ACCI>(c, a)));
    for (int m = 1; m < N; ++m) {  // produces t_{m+1}
        WilsonArgs b;
        b.nrhs = nrhs;
        b.in = (m & 1) ? c->tA : c->tB;
        b.out = (m & 1) ? c->tB : c->tA;
        b.prev = (m == 1) ? src : b.out;
        b.acc = c->acc;
        b.c_diag = 2 * cd; b.c_hop = 2 * ch; b.a_acc = al[m + 1]; b.flip = m & 1;
        if (m + 1 == N) OVL_TRY((launch_wilson<T, K_G5 | K_PREV | K_ACC | K_NOWRITE>(c, b)));
        else if (b.a_acc != 0.0) OVL_TRY((launch_wilson<T, K_G5 | K_PREV | K_ACC>(c, b)));
        else OVL_TRY((launch_wilson<T, K_G5 | K_PREV>(c, b)));
    }
    return OVL_OK;
}

// The same sum by Clenshaw's backward recurrence (the adjoint of the three-term recurrence; SURVEY.md §8(c) O4,
// §8(d) "Clenshaw form"):  b_{N+1} = b_{N+2} = 0,  b_k = alpha_k src + 2 K^ b_{k+1} - b_{k+2}  (k = N..1),
// acc = alpha_0 src + K^ b_1 - b_2.  It has no read-modify-write accumulator stream: one order reads b_{k+1} (stencil),
// b_{k+2} and - when alpha_k != 0 - src, and writes b_k over b_{k+2}.  b_N = alpha_N src is never formed: the first
// launch applies 2 alpha_N K^ to src directly and the second one carries the (- alpha_N src) term.  N launches.
template <typename T> int cheb_clenshaw(ovl_ctx *c, const void *src, int nrhs) {
    const double cd = (4.0 - c->m_w) / c->lambda_max, ch = -0.5 / c->lambda_max;
    const std::vector<double> &al = c->alpha;
    const int N = c->norders;
    int nl = 0;
    auto step = [&](const void *in, const void *prev, void *out, double scale, double a_psi) -> int {
        WilsonArgs a;
        a.nrhs = nrhs;
        a.in = in; a.prev = prev; a.psi = src; a.out = out;
        a.c_diag = scale * cd; a.c_hop = scale * ch; a.a_psi = a_psi; a.flip = (nl++) & 1;
        if (prev) return a_psi != 0.0 ? launch_wilson<T, K_G5 | K_PREV | K_PSI>(c, a) : launch_wilson<T, K_G5 | K_PREV>(c, a);
        return a_psi != 0.0 ? launch_wilson<T, K_G5 | K_PSI>(c, a) : launch_wilson<T, K_G5>(c, a);
    };
    if (N == 1) return step(src, nullptr, c->acc, al[1], al[0]);
    OVL_TRY(step(src, nullptr, c->tA, 2 * al[N], al[N - 1]));                  // b_{N-1}
    if (N == 2) return step(c->tA, nullptr, c->acc, 1.0, al[0] - al[2]);      // acc = alpha_0 src + K^ b_1 - alpha_2 src
    OVL_TRY(step(c->tA, nullptr, c->tB, 2.0, al[N - 2] - al[N]));              // b_{N-2}
    void *cur = c->tB, *oth = c->tA;                                          // cur = b_{k+1}, oth = b_{k+2}
    for (int k = N - 3; k >= 1; --k) {
        OVL_TRY(step(cur, oth, oth, 2.0, al[k]));
        void *t = cur; cur = oth; oth = t;
    }
    return step(cur, oth, c->acc, 1.0, al[0]);
}

template <typename T> int cheb_launches(ovl_ctx *c, const void *src, int nrhs) {
    // a table with alpha_m = 0 for all m >= 1 (reading R8: alpha_0 is honoured) has no K^ term to scale the Clenshaw
    // launch by; the forward launch evaluates acc = alpha_0 src + 0 * K^ src without dividing by the hop coefficient
    if (c->norders == 1 && c->alpha[1] == 0.0) return cheb_forward<T>(c, src, nrhs);
    return c->recurrence == OVL_REC_FORWARD ? cheb_forward<T>(c, src, nrhs) : cheb_clenshaw<T>(c, src, nrhs);
}

// The loop is a fixed sequence of launches for a given source field, so it is captured once into a CUDA graph and
// replayed (0.5 us instead of 2 us of launch overhead per order on B200: 20 % of an order at 8^3x32).  Capture needs a
// real stream: on the legacy default stream (handle 0), or if capture fails (the caller is itself capturing), the
// launches are issued directly.  Returns OVL_OK with *done = false when the caller has to launch directly.
template <typename T> int cheb_graph(ovl_ctx *c, const void *src, int nrhs, bool *done) {
    *done = false;
    if (!c->use_graphs || c->st == nullptr || c->st == cudaStreamLegacy || c->st == cudaStreamPerThread) return OVL_OK;
    ovl_ctx::PolyGraph *hit = nullptr, *victim = nullptr;
    for (auto &e : c->graphs) {
        const bool valid = e.exec && e.gen == c->poly_gen;
        if (valid && e.src == src && e.nrhs == nrhs) hit = &e;
        if (!valid) { if (!victim || (victim->exec && victim->gen == c->poly_gen)) victim = &e; }
        else if (!victim || (victim->exec && victim->gen == c->poly_gen && e.last_use < victim->last_use)) victim = &e;
    }
    if (!hit) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(c->st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); return OVL_OK; }
        if (cudaStreamBeginCapture(c->st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return OVL_OK; }
        const long long l0 = c->launches;
        const int rc = cheb_launches<T>(c, src, nrhs);
        c->launches = l0;  // counted per replay below
        cudaGraph_t gr = nullptr;
        const cudaError_t e = cudaStreamEndCapture(c->st, &gr);
        if (rc != OVL_OK || e != cudaSuccess || !gr) {
            if (gr) cudaGraphDestroy(gr);
            cudaGetLastError();
            return rc;
        }
        cudaGraphExec_t ex = nullptr;
        const cudaError_t ei = cudaGraphInstantiate(&ex, gr, 0);
        cudaGraphDestroy(gr);
        if (ei != cudaSuccess) { cudaGetLastError(); return OVL_OK; }
        if (victim->exec) cudaGraphExecDestroy(victim->exec);
        victim->exec = ex; victim->src = src; victim->gen = c->poly_gen; victim->nrhs = nrhs;
        hit = victim;
    }
    hit->last_use = ++c->use_clock;
    OVL_CUDA(c, cudaGraphLaunch(hit->exec, c->st));
    c->launches += c->norders;
    *done = true;
    return OVL_OK;
}

// acc = sum_{m=0}^{norders} alpha_m T_m(K^) src    (first sum of eq. 2.3; src is not modified)
template <typename T> int cheb_native(ovl_ctx *c, const void *src, int nrhs) {
    const int pslot = (int)(c->prof_count % ovl_ctx::NPROF);
    if (c->profiling) OVL_CUDA(c, cudaEventRecord(c->pev0[pslot], c->st));
    bool done = false;
    OVL_TRY(cheb_graph<T>(c, src, nrhs, &done));
    if (!done) OVL_TRY(cheb_launches<T>(c, src, nrhs));
    if (c->profiling) {
        OVL_CUDA(c, cudaEventRecord(c->pev1[pslot], c->st));
        c->last_poly_launches = c->norders;
        ++c->prof_count;
    }
    return OVL_OK;
}

inline int refresh_coef(ovl_ctx *c) {
    if (!c->coef_stale || c->nev == 0) return OVL_OK;
    c->coef.resize(c->nev);
    for (int i = 0; i < c->nev; ++i) {
        const double l = c->lambda[i];
        const double sg = (l > 0) - (l < 0);
        c->coef[i] = sg - cheb_scalar(c->alpha, l / c->lambda_max);
    }
    OVL_CUDA(c, cudaMemcpyAsync(c->coef_dev, c->coef.data(), sizeof(double) * c->nev, cudaMemcpyHostToDevice, c->st));
    OVL_CUDA(c, cudaStreamSynchronize(c->st));  // coef.data() is pageable host memory
    c->coef_stale = false;
    return OVL_OK;
}

// work vectors of the recurrence (t_A, t_B, acc, gamma5 psi) for `nrhs` right-hand sides; grown on demand when the library
// owns the memory, fixed at max_rhs in a caller-owned workspace
inline int ensure_work(ovl_ctx *c, int nrhs) {
    if (nrhs <= c->work_nrhs) return OVL_OK;
    if (c->ws_mode) return fail(c, OVL_EINVAL, "%d right-hand sides exceed the workspace capacity max_rhs = %d", nrhs, c->max_rhs);
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    void **bufs[] = {&c->tA, &c->tB, &c->acc, &c->g5b};
    void *fresh[4] = {nullptr, nullptr, nullptr, nullptr};
    for (int i = 0; i < 4; ++i) {
        const int rc = dev_alloc(c, &fresh[i], c->field_bytes() * nrhs);
        if (rc != OVL_OK) {  // keep the old (smaller) workspace usable
            for (int j = 0; j < i; ++j) dev_release(c, &fresh[j]);
            return rc;
        }
    }
    for (int i = 0; i < 4; ++i) {
        dev_release(c, bufs[i]);
        *bufs[i] = fresh[i];
    }
    c->work_nrhs = nrhs;
    ++c->poly_gen;  // captured graphs point at the old buffers
    return OVL_OK;
}

// scratch of the projection for nrhs right-hand sides (library-owned contexts grow it; a workspace holds max_rhs)
inline int ensure_proj(ovl_ctx *c, int nrhs) {
    if (nrhs <= c->proj_rhs) return OVL_OK;
    if (c->ws_mode) return fail(c, OVL_EINVAL, "%d right-hand sides exceed the workspace capacity max_rhs = %d", nrhs, c->max_rhs);
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    dev_release(c, (void **)&c->proj_partial);
    c->proj_rhs = 0;
    OVL_TRY(dev_alloc(c, (void **)&c->proj_partial, sizeof(double2) * (size_t)c->proj_nblk * c->proj_cap * nrhs));
    c->proj_rhs = nrhs;
    return OVL_OK;
}

// out_r = a*in_r + b*[gamma5]( sign(K) src_r ) for r < nrhs consecutive native fields;  src = in (dagger = 0) or gamma5 in
// (dagger = 1, gamma5 not applied on the way out).  ovl_sign uses a = 0, b = 1, g5out = 0.  The polynomial loop handles
// all right-hand sides in every launch (links amortised); the two deflation passes read every phi_i once per group of
// DEFL_RB right-hand sides.
template <typename T> int sign_combine_native(ovl_ctx *c, int nrhs, double a, double b, int dagger, int g5out, const void *in, void *out, int chir = 0) {
    if (c->alpha.empty()) return fail(c, OVL_ESTATE, "ovl_set_chebyshev has not been called");
    OVL_TRY(ensure_work(c, nrhs));
    const size_t n = c->n(), n_upper = (size_t)6 * c->g.V;
    const void *src = in;
    if (dagger) {
        k_gamma5<T><<<dim3(grid_for(n, BLAS_THREADS, 1 << 30), nrhs), BLAS_THREADS, 0, c->st>>>(n, n_upper, (const cx<T> *)in, (cx<T> *)c->g5b);
        OVL_LAUNCH_CHECK(c);
        src = c->g5b;
    }
    const int ngrp = (nrhs + DEFL_RB - 1) / DEFL_RB;
    if (c->nev > 0) {
        OVL_TRY(refresh_coef(c));
        OVL_TRY(ensure_proj(c, nrhs));
        // phi_i is streamed once per group of DEFL_RB right-hand sides (projection) ...
        k_project<T><<<dim3(c->proj_nblk, ngrp), BLAS_THREADS, 0, c->st>>>(n, c->nev, nrhs, (const cx<T> *)c->phi, (const cx<T> *)src, c->proj_partial);
        OVL_LAUNCH_CHECK(c);
        k_project_final<<<dim3(c->nev, nrhs), BLAS_THREADS, 0, c->st>>>(c->proj_nblk, c->nev, c->proj_cap, c->proj_partial, c->coef_dev, c->w_dev);
        OVL_LAUNCH_CHECK(c);
    }
    OVL_TRY(cheb_native<T>(c, src, nrhs));
    // ... and once more per group in the update + assembly pass
    k_deflate_assemble<T><<<dim3(grid_for(n, BLAS_THREADS, 1 << 30), ngrp), BLAS_THREADS, 0, c->st>>>(
        n, n_upper, c->nev, nrhs, c->proj_cap > 0 ? c->proj_cap : 1, (const cx<T> *)c->phi, c->w_dev, (const cx<T> *)in, (const cx<T> *)c->acc, (T)a,
        (T)b, g5out, chir, (cx<T> *)out);
    OVL_LAUNCH_CHECK(c);
    return OVL_OK;
}

template <typename T> int overlap_native(ovl_ctx *c, double mu, int dagger, const void *in, void *out, int nrhs = 1) {
    return sign_combine_native<T>(c, nrhs, 0.5 * (1.0 + mu), 0.5 * (1.0 - mu), dagger, dagger ? 0 : 1, in, out);
}

// ---- CG on A = D^dag D (a9), nrhs independent systems in lockstep (nrhs = 1: the plain CG).  b_n, x_n: nrhs
// consecutive native fields; x0 = 0.  Every operator application handles all systems at once (multi-right-hand-side
// kernel launches); the vector kernels are batched over blockIdx.y with per-system alpha, beta, rr on the device.  A
// system that reaches the tolerance is frozen (alpha = beta = 0: x and r stop changing) while the others go on.
template <typename T> int reduce_redot(ovl_ctx *c, const void *x, const void *y, int what, int nrhs) {
    k_redot<T><<<dim3(c->red_nblk, nrhs), BLAS_THREADS, 0, c->st>>>(c->n(), (const cx<T> *)x, (const cx<T> *)y, c->red_partial);
    OVL_LAUNCH_CHECK(c);
    k_cg_scalars<<<nrhs, BLAS_THREADS, 0, c->st>>>(c->red_nblk, c->red_partial, c->sc_dev, what, 0.0);
    OVL_LAUNCH_CHECK(c);
    return OVL_OK;
}
inline int fetch_scalars(ovl_ctx *c, int nrhs) {  // synchronous read-out into slot 0 (start-up and final residual only)
    OVL_CUDA(c, cudaMemcpyAsync(c->sc_host, c->sc_dev, sizeof(double) * SC_N * nrhs, cudaMemcpyDeviceToHost, c->st));
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    return OVL_OK;
}
inline int ensure_cg(ovl_ctx *c, int nrhs) {
    if (nrhs <= c->cg_nrhs) return OVL_OK;
    if (c->ws_mode) return fail(c, OVL_EINVAL, "%d systems exceed the workspace capacity max_rhs = %d", nrhs, c->max_rhs);
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    void **bufs[] = {&c->cg_r, &c->cg_p, &c->cg_q, &c->cg_Ap};
    for (void **b : bufs) dev_release(c, b);
    c->cg_nrhs = 0;
    for (void **b : bufs) OVL_TRY(dev_alloc(c, b, c->field_bytes() * nrhs));
    c->cg_nrhs = nrhs;
    return OVL_OK;
}

// chir = 0: A = D^dag D (two sign applications per operator application).  chir = +1 / -1: the chiral-sector system
// A_c x = P_c b,  A_c = 1/2 (1+mu^2) + c/2 (1-mu^2) P_c sign(K) P_c  (reading R23; = P_c D^dag D P_c for sign(K)^2 = 1):
// ONE sign application per operator application; every CG vector stays in the chirality sector.
template <typename T>
int cg_native(ovl_ctx *c, double mu, const void *b_n, void *x_n, double tol, int maxiter, int *iters, double *relres, int nrhs = 1,
              int chir = 0) {
    const size_t n = c->n(), fb = c->field_bytes() * nrhs, n_upper = (size_t)6 * c->g.V;
    OVL_TRY(ensure_cg(c, nrhs));
    const dim3 gride(grid_for(n, BLAS_THREADS, 1 << 30), nrhs);
    auto apply_A = [&](const void *in, void *out) -> int {
        if (chir) return sign_combine_native<T>(c, nrhs, 0.5 * (1.0 + mu * mu), 0.5 * chir * (1.0 - mu * mu), 0, 0, in, out, chir);
        OVL_TRY(overlap_native<T>(c, mu, 0, in, c->cg_q, nrhs));
        return overlap_native<T>(c, mu, 1, c->cg_q, out, nrhs);
    };
    OVL_CUDA(c, cudaMemsetAsync(x_n, 0, fb, c->st));
    if (chir) {
        k_chiral_project<T><<<gride, BLAS_THREADS, 0, c->st>>>(n, n_upper, chir, (const cx<T> *)b_n, (cx<T> *)c->cg_r);
        OVL_LAUNCH_CHECK(c);
    } else {
        OVL_CUDA(c, cudaMemcpyAsync(c->cg_r, b_n, fb, cudaMemcpyDeviceToDevice, c->st));
    }
    OVL_CUDA(c, cudaMemcpyAsync(c->cg_p, c->cg_r, fb, cudaMemcpyDeviceToDevice, c->st));
    OVL_TRY(reduce_redot<T>(c, c->cg_r, c->cg_r, 0, nrhs));
    OVL_TRY(fetch_scalars(c, nrhs));
    double bb[OVL_MAX_RHS], rr[OVL_MAX_RHS];
    bool conv[OVL_MAX_RHS];
    const double tol2 = tol > 0 ? tol * tol : 0.0;
    int nconv = 0;
    for (int r = 0; r < nrhs; ++r) {
        bb[r] = rr[r] = c->sc_host[r * SC_N + SC_BB];
        iters[r] = 0;
        conv[r] = tol > 0 && rr[r] <= tol2 * bb[r];  // b = 0
        nconv += conv[r];
    }
    const dim3 gridv(grid_for(n, BLAS_THREADS), nrhs), gridr(c->red_nblk, nrhs);
    // The host never stalls the device between iterations: iteration `it` is enqueued BEFORE the convergence scalars of
    // iteration it-1 are read (asynchronous copy into one of two pinned slots + an event).  A system that has reached the
    // tolerance is frozen on the device in the same kernel that forms beta (alpha = beta = 0 from then on: x and r stop
    // changing), so the one iteration that may run past convergence leaves the solution bit-identical.
    int enq = 0, seen = 0;
    auto check = [&](int j) -> int {  // consume the scalars of iteration j (0-based)
        OVL_CUDA(c, cudaEventSynchronize(c->cg_ev[j & 1]));
        const double *h = c->sc_host + (size_t)(j & 1) * SC_N * OVL_MAX_RHS;
        for (int r = 0; r < nrhs; ++r) {
            if (conv[r]) continue;
            rr[r] = h[r * SC_N + SC_RR];
            iters[r] = j + 1;
            if (!(rr[r] == rr[r])) return fail(c, OVL_ECUDA, "CG broke down (NaN residual) at iteration %d, system %d", j + 1, r);
            if (tol > 0 && rr[r] <= tol2 * bb[r]) { conv[r] = true; ++nconv; }  // same test as the device-side freeze
        }
        return OVL_OK;
    };
    while (enq < maxiter && nconv < nrhs) {
        OVL_TRY(apply_A(c->cg_p, c->cg_Ap));
        OVL_TRY(reduce_redot<T>(c, c->cg_p, c->cg_Ap, 1, nrhs));  // alpha = rr / Re(p^dag A p)
        k_cg_update<T><<<gridr, BLAS_THREADS, 0, c->st>>>(n, c->sc_dev, (const cx<T> *)c->cg_p, (const cx<T> *)c->cg_Ap,
                                                        (cx<T> *)x_n, (cx<T> *)c->cg_r, c->red_partial);
        OVL_LAUNCH_CHECK(c);
        k_cg_scalars<<<nrhs, BLAS_THREADS, 0, c->st>>>(c->red_nblk, c->red_partial, c->sc_dev, 2, tol2);  // beta, rr, freeze
        OVL_LAUNCH_CHECK(c);
        k_xpay<T><<<gridv, BLAS_THREADS, 0, c->st>>>(n, c->sc_dev, (const cx<T> *)c->cg_r, (cx<T> *)c->cg_p);
        OVL_LAUNCH_CHECK(c);
        OVL_CUDA(c, cudaMemcpyAsync(c->sc_host + (size_t)(enq & 1) * SC_N * OVL_MAX_RHS, c->sc_dev, sizeof(double) * SC_N * nrhs,
                                    cudaMemcpyDeviceToHost, c->st));
        OVL_CUDA(c, cudaEventRecord(c->cg_ev[enq & 1], c->st));
        ++enq;
        if (enq - seen == 2) OVL_TRY(check(seen++));  // one iteration behind the device
    }
    while (seen < enq && nconv < nrhs) OVL_TRY(check(seen++));
    const int it = enq;
    // true residuals ||b - A x|| / ||b||   (chiral: || P_c (b - A_c x) || / || P_c b ||)
    OVL_TRY(apply_A(x_n, c->cg_Ap));
    k_sub<T><<<gridv, BLAS_THREADS, 0, c->st>>>(n, (const cx<T> *)b_n, (const cx<T> *)c->cg_Ap, (cx<T> *)c->cg_q);
    OVL_LAUNCH_CHECK(c);
    if (chir) {
        k_chiral_project<T><<<gride, BLAS_THREADS, 0, c->st>>>(n, n_upper, chir, (const cx<T> *)c->cg_q, (cx<T> *)c->cg_q);
        OVL_LAUNCH_CHECK(c);
    }
    OVL_TRY(reduce_redot<T>(c, c->cg_q, c->cg_q, 3, nrhs));
    OVL_TRY(fetch_scalars(c, nrhs));
    for (int r = 0; r < nrhs; ++r) relres[r] = bb[r] > 0 ? std::sqrt(c->sc_host[r * SC_N + SC_PAP] / bb[r]) : 0.0;
    if (tol > 0 && nconv < nrhs) {
        int worst = 0;
        for (int r = 1; r < nrhs; ++r)
            if (rr[r] / bb[r] > rr[worst] / bb[worst]) worst = r;
        return fail(c, OVL_ENOTCONV, "CG: %d iterations, %d of %d systems above tol (worst ||r||/||b|| = %.3e, system %d)", it,
                    nrhs - nconv, nrhs, std::sqrt(rr[worst] / bb[worst]), worst);
    }
    return OVL_OK;
}

// ---- mixed-precision CG ("10^-13 for overlap fermions (using mixed precision)"):
// defect correction x <- x + A32^{-1} (b - A64 x).  Outer residuals and the solution are fp64 (context c), the inner
// solves run the whole fp32 path (context c32: fp32 links, eigenvectors, stencil arithmetic; its own Chebyshev table, which
// may be of lower degree) on the residual normalised to unit length.  b_n, x_n: native fp64 fields of c.
// chir = +1 / -1: the chiral-sector system A_c x = P_c b of cg_native (one sign application per operator application in
// both precisions); the outer residual is P_c b - A_c x.
inline int cg_mixed_native(ovl_ctx *c, ovl_ctx *c32, double mu, const void *b_n, void *x_n, double tol, double inner_tol,
                           int max_outer, int max_inner, int *outer_out, int *inner_out, double *relres, int chir = 0) {
    const size_t n = c->n(), fb = c->field_bytes(), n_upper = (size_t)6 * c->g.V;
    OVL_TRY(ensure_cg(c, 1));
    const int gridv = grid_for(n, BLAS_THREADS);
    OVL_CUDA(c, cudaMemsetAsync(x_n, 0, fb, c->st));
    if (chir) {  // P_c b lives in cg_p (the outer iteration has no search direction of its own)
        k_chiral_project<double><<<dim3(grid_for(n, BLAS_THREADS, 1 << 30), 1), BLAS_THREADS, 0, c->st>>>(n, n_upper, chir, (const double2 *)b_n, (double2 *)c->cg_p);
        OVL_LAUNCH_CHECK(c);
        b_n = c->cg_p;
    }
    OVL_CUDA(c, cudaMemcpyAsync(c->cg_r, b_n, fb, cudaMemcpyDeviceToDevice, c->st));
    OVL_TRY(reduce_redot<double>(c, b_n, b_n, 0, 1));
    OVL_TRY(fetch_scalars(c, 1));
    const double bb = c->sc_host[SC_BB];
    double rr = bb;
    int outer = 0, inner_total = 0;
    while (outer < max_outer && bb > 0 && !(rr <= tol * tol * bb)) {
        const double rn = std::sqrt(rr);
        k_convert_scaled<double, float><<<gridv, BLAS_THREADS, 0, c->st>>>(n, 1.0 / rn, (const double2 *)c->cg_r, (float2 *)c32->psi_n);
        OVL_LAUNCH_CHECK(c);
        int it = 0;
        double rel32 = 0;
        const int rc = cg_native<float>(c32, mu, c32->psi_n, c32->out_n, inner_tol, max_inner, &it, &rel32, 1, chir);
        if (rc != OVL_OK && rc != OVL_ENOTCONV) return fail(c, rc, "inner fp32 CG: %s", c32->err);
        inner_total += it;
        k_axpy_mixed<float, double><<<gridv, BLAS_THREADS, 0, c->st>>>(n, rn, (const float2 *)c32->out_n, (double2 *)x_n);
        OVL_LAUNCH_CHECK(c);
        // r = b - A64 x
        if (chir) {
            OVL_TRY(sign_combine_native<double>(c, 1, 0.5 * (1.0 + mu * mu), 0.5 * chir * (1.0 - mu * mu), 0, 0, x_n, c->cg_Ap, chir));
        } else {
            OVL_TRY(overlap_native<double>(c, mu, 0, x_n, c->cg_q));
            OVL_TRY(overlap_native<double>(c, mu, 1, c->cg_q, c->cg_Ap));
        }
        k_sub<double><<<gridv, BLAS_THREADS, 0, c->st>>>(n, (const double2 *)b_n, (const double2 *)c->cg_Ap, (double2 *)c->cg_r);
        OVL_LAUNCH_CHECK(c);
        OVL_TRY(reduce_redot<double>(c, c->cg_r, c->cg_r, 3, 1));
        OVL_TRY(fetch_scalars(c, 1));
        const double rr_new = c->sc_host[SC_PAP];
        ++outer;
        if (!(rr_new == rr_new)) return fail(c, OVL_ECUDA, "mixed CG broke down (NaN residual) in outer iteration %d", outer);
        if (it == 0 || rr_new >= rr) {  // no progress: the fp32 operator cannot improve this residual any further
            rr = rr_new < rr ? rr_new : rr;
            break;
        }
        rr = rr_new;
    }
    *outer_out = outer;
    *inner_out = inner_total;
    *relres = bb > 0 ? std::sqrt(rr / bb) : 0.0;  // rr is the TRUE fp64 residual of the returned x
    if (bb > 0 && !(rr <= tol * tol * bb))
        return fail(c, OVL_ENOTCONV, "mixed CG: %d outer / %d inner iterations, ||r||/||b|| = %.3e > tol", outer, inner_total, std::sqrt(rr / bb));
    return OVL_OK;
}

}  // namespace ovl
