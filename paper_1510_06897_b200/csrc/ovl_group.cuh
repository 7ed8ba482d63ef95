// ovl_group.cuh -- host side of the t-split lattice (ovl_slab.cuh has the kernels and the design): a group of slab contexts
// living in this process, each on its own stream and (optionally) its own GPU, wired to its two t-neighbours by peer
// pointers and events.  Included by ovl.cu after its canonical import / export helpers.
#pragma once
#include "ovl_engine.cuh"
#include "ovl_slab.cuh"

#include <chrono>

struct ovl_group {
    int n = 0;                 // slabs of the lattice
    int gdims[4] = {0, 0, 0, 0};
    int prec = OVL_F64, recon = OVL_RECON18;
    size_t Vloc = 0;
    std::vector<ovl_ctx *> s;  // slab contexts (local lattice Lx x Ly x Lz x (Lt / n)); null for slabs of other processes
    std::vector<int> mine;     // the slabs this process runs: all of them (in-process group) or one (one process per GPU)
    std::vector<int> dev;      // device ordinal per local slab (index = slab)
    struct Wire {              // what a slab exposes to the others: all of it lives in ONE device allocation (one IPC handle)
        void *base = nullptr;
        void *halo[3][2] = {{nullptr, nullptr}, {nullptr, nullptr}, {nullptr, nullptr}};  // [slot][lo / hi], one time slice each
        void *u_lo = nullptr;                                                            // ghost U_t slice
        // this slab's share of the deflation coefficients (2 nev doubles) / of a CG scalar; two buffers used alternately, so a
        // slab that runs ahead never overwrites what a slower slab is still summing
        double *w_loc[2] = {nullptr, nullptr};
        double *red_loc[2] = {nullptr, nullptr};
        cudaEvent_t ev[2] = {nullptr, nullptr};
        bool remote = false;   // opened through CUDA IPC (another process)
    };
    std::vector<Wire> w;
    unsigned long long round = 0;  // launch rounds so far: round k waits on the neighbours' events of round k-1
    // split every stencil round into a boundary launch (the two edge time slices: all halo reads and pushes), after which the
    // round's event is recorded, and an interior launch: the neighbours' next round then overlaps this slab's interior, which
    // hides the cross-GPU event latency.  Default: on when the slabs sit on different devices.
    bool split_launch = false;
    int nev = 0;
    unsigned defl_par = 0, red_par = 0;
    // one process per GPU: a record must have been ISSUED by the neighbour's host thread before this process may wait on
    // the (IPC) event, so every process publishes "rounds issued so far" in a small POSIX shared-memory segment
    bool distributed = false;
    int rank = 0;
    volatile unsigned long long *issued = nullptr;  // [n], shared between the processes of the group
    char shm_name[96] = {0};
    char err[256] = {0};
};

namespace ovl {

enum { SLOT_SRC = 0, SLOT_A = 1, SLOT_B = 2 };

struct DevGuard {
    int prev = 0;
    explicit DevGuard(int d) {
        cudaGetDevice(&prev);
        if (d != prev) cudaSetDevice(d);
    }
    ~DevGuard() { cudaSetDevice(prev); }
};

inline int gfail(ovl_group *g, int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g->err, sizeof g->err, fmt, ap);
    va_end(ap);
    return code;
}
#define GRP_CUDA(g, call)                                                                        \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess) {                                                                 \
            cudaGetLastError();                                                                  \
            return ovl::gfail((g), OVL_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));          \
        }                                                                                        \
    } while (0)
#define GRP_TRY(g, r, expr)                                                                      \
    do {                                                                                         \
        int rc_ = (expr);                                                                        \
        if (rc_ != OVL_OK) return ovl::gfail((g), rc_, "slab %d: %s", (r), (g)->s[(r)]->err);    \
    } while (0)

constexpr int WIRE_MAX_NEV = 512;  // capacity of the deflation-coefficient scratch (fixed so the layout never changes)
struct WireLayout { size_t halo[3][2], u_lo, w_loc[2], red_loc[2], total; };
inline WireLayout wire_layout(size_t sxyz, int nrow, size_t ts) {
    WireLayout L;
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t o = off; off += ws_round(bytes); return o; };
    for (int sl = 0; sl < 3; ++sl)
        for (int side = 0; side < 2; ++side) L.halo[sl][side] = take(12 * sxyz * 2 * ts);
    L.u_lo = take((size_t)nrow * 3 * sxyz * 2 * ts);
    for (int b = 0; b < 2; ++b) L.w_loc[b] = take(sizeof(double2) * WIRE_MAX_NEV);
    for (int b = 0; b < 2; ++b) L.red_loc[b] = take(sizeof(double) * 8);
    L.total = off;
    return L;
}
inline void wire_point(ovl_group::Wire &w, const WireLayout &L, void *base) {
    char *p = (char *)base;
    w.base = base;
    for (int sl = 0; sl < 3; ++sl)
        for (int side = 0; side < 2; ++side) w.halo[sl][side] = p + L.halo[sl][side];
    w.u_lo = p + L.u_lo;
    for (int b = 0; b < 2; ++b) { w.w_loc[b] = (double *)(p + L.w_loc[b]); w.red_loc[b] = (double *)(p + L.red_loc[b]); }
}

// one process per GPU: block (on the host) until slab q's process has issued the record of round `need - 1`
inline int wait_issued(ovl_group *g, int q, unsigned long long need) {
    if (!g->distributed || g->s[q] != nullptr) return OVL_OK;
    const auto t0 = std::chrono::steady_clock::now();
    unsigned spins = 0;
    while (__atomic_load_n(&g->issued[q], __ATOMIC_ACQUIRE) < need) {
        if ((++spins & 0xfff) == 0 && std::chrono::steady_clock::now() - t0 > std::chrono::seconds(60))
            return gfail(g, OVL_ECUDA, "slab %d did not issue round %llu within 60 s", q, need - 1);
    }
    return OVL_OK;
}

inline int lo_of(const ovl_group *g, int r) { return (r + g->n - 1) % g->n; }
inline int hi_of(const ovl_group *g, int r) { return (r + 1) % g->n; }

// Start a launch round on slab r: its stream waits for what the two t-neighbours did in the previous round (their pushes into
// this slab's halos are complete, and they no longer read the halos this round is about to overwrite).
inline int round_begin(ovl_group *g, int r) {
    if (g->round == 0) return OVL_OK;
    const int p = (int)((g->round - 1) & 1);
    OVL_TRY(wait_issued(g, lo_of(g, r), g->round));
    GRP_CUDA(g, cudaStreamWaitEvent(g->s[r]->st, g->w[lo_of(g, r)].ev[p], 0));
    if (hi_of(g, r) != lo_of(g, r)) {
        OVL_TRY(wait_issued(g, hi_of(g, r), g->round));
        GRP_CUDA(g, cudaStreamWaitEvent(g->s[r]->st, g->w[hi_of(g, r)].ev[p], 0));
    }
    return OVL_OK;
}
inline int round_end(ovl_group *g, int r) {
    GRP_CUDA(g, cudaEventRecord(g->w[r].ev[g->round & 1], g->s[r]->st));
    if (g->distributed) __atomic_store_n(&g->issued[r], g->round + 1, __ATOMIC_RELEASE);
    return OVL_OK;
}
// a round in which every slab waits for EVERY slab's previous round (reductions over slabs)
inline int round_begin_all(ovl_group *g, int r) {
    if (g->round == 0) return OVL_OK;
    const int p = (int)((g->round - 1) & 1);
    for (int q = 0; q < g->n; ++q)
        if (q != r) {
            OVL_TRY(wait_issued(g, q, g->round));
            GRP_CUDA(g, cudaStreamWaitEvent(g->s[r]->st, g->w[q].ev[p], 0));
        }
    return OVL_OK;
}

template <typename T> SlabArgs<T> slab_args(ovl_group *g, int r, int in_slot, int out_slot) {
    SlabArgs<T> a;
    a.h_lo = (const cx<T> *)g->w[r].halo[in_slot][0];
    a.h_hi = (const cx<T> *)g->w[r].halo[in_slot][1];
    // my first time slice is the lower neighbour's UPPER halo, my last one the upper neighbour's LOWER halo
    a.p_lo = out_slot >= 0 ? (cx<T> *)g->w[lo_of(g, r)].halo[out_slot][1] : nullptr;
    a.p_hi = out_slot >= 0 ? (cx<T> *)g->w[hi_of(g, r)].halo[out_slot][0] : nullptr;
    a.u_lo = (const cx<T> *)g->w[r].u_lo;
    a.s_lo = r == 0 ? T(-1) : T(1);          // the hop from global t = 0 backwards crosses the antiperiodic boundary
    a.s_hi = r == g->n - 1 ? T(-1) : T(1);   // the hop from global t = Lt - 1 forwards does
    return a;
}

// one fused stencil launch (or a boundary + an interior launch) on every slab = one round
template <typename T, int RECON, int FLAGS>
int slab_step_t(ovl_group *g, const WilsonArgs *args, int in_slot, int out_slot) {
    constexpr int TH = WilsonCfg<T>::THREADS;
    for (int r : g->mine) {
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        OVL_TRY(round_begin(g, r));
        const WilsonArgs &a = args[r];
        StepParams<T> sp{(T)a.c_hop, (T)(a.c_diag / a.c_hop), (T)(1.0 / a.c_hop), (T)(a.a_psi / a.c_hop), (T)0, (T)0, a.flip};
        const SlabArgs<T> sl = slab_args<T>(g, r, in_slot, out_slot);
        const int ntile = (c->g.V + TH - 1) / TH, tps = c->g.sxyz / TH;  // tiles per time slice (when they align)
        auto launch = [&](int grid, TileRange tr) {
            k_wilson_slab<T, RECON, FLAGS, TH, WilsonCfg<T>::MINB><<<grid, TH, 0, c->st>>>(
                c->g, (const cx<T> *)c->U, (const cx<T> *)a.in, (const cx<T> *)a.prev, (const cx<T> *)a.psi, (cx<T> *)a.out, sp, sl, tr);
            ++c->launches;
        };
        const bool split = g->split_launch && c->g.sxyz % TH == 0 && c->g.L[3] >= 3;
        if (split) {
            launch(2 * tps, TileRange{0, tps, ntile - tps});         // time slices 0 and Lt-1: halo reads + pushes
            GRP_CUDA(g, cudaGetLastError());
            OVL_TRY(round_end(g, r));                                 // the neighbours may start their next round now
            launch(ntile - 2 * tps, TileRange{tps, ntile, 0});        // interior
        } else {
            launch(ntile, TileRange{0, ntile, 0});
            GRP_CUDA(g, cudaGetLastError());
            OVL_TRY(round_end(g, r));
        }
        GRP_CUDA(g, cudaGetLastError());
    }
    ++g->round;
    return OVL_OK;
}
template <typename T, int FLAGS> int slab_step(ovl_group *g, const WilsonArgs *args, int in_slot, int out_slot) {
    return g->recon == OVL_RECON18 ? slab_step_t<T, 18, FLAGS>(g, args, in_slot, out_slot) : slab_step_t<T, 12, FLAGS>(g, args, in_slot, out_slot);
}

// push the faces of field f_r (one per slab) into the neighbours' halo slot: one round
template <typename T> int push_faces(ovl_group *g, void *const *f, int slot) {
    for (int r : g->mine) {
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        OVL_TRY(round_begin(g, r));
        const size_t ne = (size_t)12 * c->g.sxyz;
        k_push_faces<T><<<(unsigned)((ne + 255) / 256), 256, 0, c->st>>>(c->g.V, c->g.sxyz, (const cx<T> *)f[r],
                                                                        (cx<T> *)g->w[lo_of(g, r)].halo[slot][1],
                                                                        (cx<T> *)g->w[hi_of(g, r)].halo[slot][0]);
        ++c->launches;
        GRP_CUDA(g, cudaGetLastError());
        OVL_TRY(round_end(g, r));
    }
    ++g->round;
    return OVL_OK;
}

// out_r = sigma (c_diag in_r + c_hop hop(in))_r: D_W (g5 = 0) or K^ (g5 = 1) of a field given slab by slab
template <typename T> int group_stencil(ovl_group *g, int g5, void *const *in, void *const *out) {
    OVL_TRY(push_faces<T>(g, in, SLOT_SRC));
    std::vector<WilsonArgs> a(g->n);
    for (int r : g->mine) {
        a[r].in = in[r]; a[r].out = out[r];
        a[r].c_diag = g5 ? (4.0 - g->s[r]->m_w) / g->s[r]->lambda_max : 4.0;
        a[r].c_hop = g5 ? -0.5 / g->s[r]->lambda_max : -0.5;
    }
    return g5 ? slab_step<T, K_G5>(g, a.data(), SLOT_SRC, -1) : slab_step<T, 0>(g, a.data(), SLOT_SRC, -1);
}

// acc_r = sum_m alpha_m T_m(K^) src_r by Clenshaw's recurrence, the launch sequence of cheb_clenshaw() on every slab
template <typename T> int group_cheb(ovl_group *g, void *const *src) {
    ovl_ctx *c0 = g->s[g->mine[0]];
    const double cd = (4.0 - c0->m_w) / c0->lambda_max, ch = -0.5 / c0->lambda_max;
    const std::vector<double> &al = c0->alpha;
    const int N = c0->norders, n = g->n;
    if (N == 1 && al[1] == 0.0) return gfail(g, OVL_EINVAL, "a table without a K^ term is not supported on a split lattice");
    OVL_TRY(push_faces<T>(g, src, SLOT_SRC));
    int nl = 0;
    std::vector<WilsonArgs> a(n);
    // in / prev / out given as: 0 = src, 1 = tA, 2 = tB, 3 = acc
    auto buf = [&](int r, int which) -> void * {
        ovl_ctx *c = g->s[r];
        return which == 0 ? src[r] : which == 1 ? c->tA : which == 2 ? c->tB : c->acc;
    };
    auto step = [&](int in, int prev, int out, double scale, double a_psi) -> int {
        for (int r : g->mine) {
            a[r] = WilsonArgs();
            a[r].in = buf(r, in); a[r].prev = prev >= 0 ? buf(r, prev) : nullptr; a[r].psi = src[r]; a[r].out = buf(r, out);
            a[r].c_diag = scale * cd; a[r].c_hop = scale * ch; a[r].a_psi = a_psi; a[r].flip = nl & 1;
        }
        ++nl;
        const int in_slot = in, out_slot = (out == 1 || out == 2) ? out : -1;
        if (prev >= 0) return a_psi != 0.0 ? slab_step<T, K_G5 | K_PREV | K_PSI>(g, a.data(), in_slot, out_slot)
                                           : slab_step<T, K_G5 | K_PREV>(g, a.data(), in_slot, out_slot);
        return a_psi != 0.0 ? slab_step<T, K_G5 | K_PSI>(g, a.data(), in_slot, out_slot) : slab_step<T, K_G5>(g, a.data(), in_slot, out_slot);
    };
    if (N == 1) return step(0, -1, 3, al[1], al[0]);
    OVL_TRY(step(0, -1, 1, 2 * al[N], al[N - 1]));
    if (N == 2) return step(1, -1, 3, 1.0, al[0] - al[2]);
    OVL_TRY(step(1, -1, 2, 2.0, al[N - 2] - al[N]));
    int cur = 2, oth = 1;
    for (int k = N - 3; k >= 1; --k) {
        OVL_TRY(step(cur, oth, oth, 2.0, al[k]));
        std::swap(cur, oth);
    }
    return step(cur, oth, 3, 1.0, al[0]);
}

// out_r = a in_r + b [gamma5] sign(K) src_r on the split lattice (see sign_combine_native); chir as there
template <typename T> int group_sign_combine(ovl_group *g, double a, double b, int dagger, int g5out, void *const *in, void *const *out, int chir = 0) {
    const int n = g->n;
    if (g->s[g->mine[0]]->alpha.empty()) return gfail(g, OVL_ESTATE, "ovl_group_set_chebyshev has not been called");
    std::vector<void *> src(n);
    for (int r : g->mine) {
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        const size_t ne = c->n(), n_upper = (size_t)6 * c->g.V;
        src[r] = in[r];
        if (dagger) {
            k_gamma5<T><<<grid_for(ne, BLAS_THREADS, 1 << 30), BLAS_THREADS, 0, c->st>>>(ne, n_upper, (const cx<T> *)in[r], (cx<T> *)c->g5b);
            ++c->launches;
            src[r] = c->g5b;
        }
        if (g->nev > 0) {  // this slab's share of c_i = phi_i^dag src, times the scalar correction (a5, a6)
            GRP_TRY(g, r, refresh_coef(c));
            GRP_TRY(g, r, ensure_proj(c, 1));
            k_project<T><<<dim3(c->proj_nblk, 1), BLAS_THREADS, 0, c->st>>>(ne, c->nev, 1, (const cx<T> *)c->phi, (const cx<T> *)src[r], c->proj_partial);
            k_project_final<<<dim3(c->nev, 1), BLAS_THREADS, 0, c->st>>>(c->proj_nblk, c->nev, c->proj_cap, c->proj_partial, c->coef_dev, (double2 *)g->w[r].w_loc[g->defl_par & 1]);
            c->launches += 2;
            GRP_CUDA(g, cudaGetLastError());
        }
    }
    OVL_TRY(group_cheb<T>(g, src.data()));
    if (g->nev > 0) {  // w_i = sum over slabs, in slab order, on every slab (the tiny all-reduce of SURVEY §8(e))
        for (int r : g->mine) { DevGuard dg(g->dev[r]); OVL_TRY(round_end(g, r)); }
        ++g->round;
        SlabPtrs parts;
        for (int q = 0; q < n; ++q) parts.p[q] = g->w[q].w_loc[g->defl_par & 1];
        ++g->defl_par;
        for (int r : g->mine) {
            ovl_ctx *c = g->s[r];
            DevGuard dg(g->dev[r]);
            OVL_TRY(round_begin_all(g, r));
            k_sum_over_slabs<<<(2 * g->nev + 127) / 128, 128, 0, c->st>>>(n, parts, 2 * g->nev, (double *)c->w_dev);
            ++c->launches;
            OVL_TRY(round_end(g, r));
        }
        ++g->round;
    }
    for (int r : g->mine) {
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        const size_t ne = c->n(), n_upper = (size_t)6 * c->g.V;
        k_deflate_assemble<T><<<dim3(grid_for(ne, BLAS_THREADS, 1 << 30), 1), BLAS_THREADS, 0, c->st>>>(
            ne, n_upper, c->nev, 1, c->proj_cap > 0 ? c->proj_cap : 1, (const cx<T> *)c->phi, c->w_dev, (const cx<T> *)in[r],
            (const cx<T> *)c->acc, (T)a, (T)b, g5out, chir, (cx<T> *)out[r]);
        ++c->launches;
        GRP_CUDA(g, cudaGetLastError());
    }
    return OVL_OK;
}

template <typename T> int group_overlap(ovl_group *g, double mu, int dagger, void *const *in, void *const *out) {
    return group_sign_combine<T>(g, 0.5 * (1.0 + mu), 0.5 * (1.0 - mu), dagger, dagger ? 0 : 1, in, out);
}

// One CG scalar over the whole lattice: every slab reduces its part (k_redot / k_cg_update left it in red_partial), then
// every slab sums the slab totals in slab order and updates its own copy of the CG scalars -- all copies stay bit-identical.
__global__ void __launch_bounds__(BLAS_THREADS) k_slab_total(int nblk, const double *__restrict__ partial, double *__restrict__ out) {
    __shared__ double sm[BLAS_THREADS / 32];
    double r = 0;
    for (int b = threadIdx.x; b < nblk; b += blockDim.x) r += partial[b];
    r = block_sum(r, sm);
    if (threadIdx.x == 0) out[0] = r;
}
__global__ void k_cg_scalars_slabs(int nslabs, SlabPtrs locs, double *sc, int what, double tol2) {
    double r = 0;
    for (int q = 0; q < nslabs; ++q) r += locs.p[q][0];
    cg_scalar_update(sc, r, what, tol2);
}
inline int group_scalar(ovl_group *g, int what, double tol2) {
    const int n = g->n;
    for (int r : g->mine) {
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        k_slab_total<<<1, BLAS_THREADS, 0, c->st>>>(c->red_nblk, c->red_partial, g->w[r].red_loc[g->red_par & 1]);
        ++c->launches;
        OVL_TRY(round_end(g, r));
    }
    ++g->round;
    SlabPtrs locs;
    for (int q = 0; q < n; ++q) locs.p[q] = g->w[q].red_loc[g->red_par & 1];
    ++g->red_par;
    for (int r : g->mine) {
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        OVL_TRY(round_begin_all(g, r));
        k_cg_scalars_slabs<<<1, 1, 0, c->st>>>(n, locs, c->sc_dev, what, tol2);
        ++c->launches;
        GRP_CUDA(g, cudaGetLastError());
        OVL_TRY(round_end(g, r));
    }
    ++g->round;
    return OVL_OK;
}

// CG on D^dag D x = b over the split lattice (x0 = 0; same recurrences, same stopping rule as cg_native).  b_r, x_r: the
// slabs' native fields.  The convergence scalar is read from slab 0 (all slabs hold the same bits).
template <typename T>
int group_cg(ovl_group *g, double mu, void *const *b, void *const *x, double tol, int maxiter, int *iters, double *relres) {
    const int n = g->n;
    std::vector<void *> r_(n), p_(n), q_(n), Ap_(n);
    for (int r : g->mine) {
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        GRP_TRY(g, r, ensure_cg(c, 1));
        r_[r] = c->cg_r; p_[r] = c->cg_p; q_[r] = c->cg_q; Ap_[r] = c->cg_Ap;
        const size_t fb = c->field_bytes();
        GRP_CUDA(g, cudaMemsetAsync(x[r], 0, fb, c->st));
        GRP_CUDA(g, cudaMemcpyAsync(c->cg_r, b[r], fb, cudaMemcpyDeviceToDevice, c->st));
        GRP_CUDA(g, cudaMemcpyAsync(c->cg_p, b[r], fb, cudaMemcpyDeviceToDevice, c->st));
        k_redot<T><<<dim3(c->red_nblk, 1), BLAS_THREADS, 0, c->st>>>(c->n(), (const cx<T> *)b[r], (const cx<T> *)b[r], c->red_partial);
        ++c->launches;
    }
    OVL_TRY(group_scalar(g, 0, 0.0));
    ovl_ctx *c0 = g->s[g->mine[0]];
    auto fetch0 = [&]() -> int {
        DevGuard dg(g->dev[g->mine[0]]);
        GRP_CUDA(g, cudaMemcpyAsync(c0->sc_host, c0->sc_dev, sizeof(double) * SC_N, cudaMemcpyDeviceToHost, c0->st));
        GRP_CUDA(g, cudaStreamSynchronize(c0->st));
        return OVL_OK;
    };
    OVL_TRY(fetch0());
    const double bb = c0->sc_host[SC_BB], tol2 = tol > 0 ? tol * tol : 0.0;
    double rr = bb;
    int it = 0;
    bool conv = tol > 0 && rr <= tol2 * bb;
    while (it < maxiter && !conv) {
        OVL_TRY(group_overlap<T>(g, mu, 0, p_.data(), q_.data()));
        OVL_TRY(group_overlap<T>(g, mu, 1, q_.data(), Ap_.data()));
        for (int r : g->mine) {
            ovl_ctx *c = g->s[r];
            DevGuard dg(g->dev[r]);
            k_redot<T><<<dim3(c->red_nblk, 1), BLAS_THREADS, 0, c->st>>>(c->n(), (const cx<T> *)c->cg_p, (const cx<T> *)c->cg_Ap, c->red_partial);
            ++c->launches;
        }
        OVL_TRY(group_scalar(g, 1, 0.0));
        for (int r : g->mine) {
            ovl_ctx *c = g->s[r];
            DevGuard dg(g->dev[r]);
            k_cg_update<T><<<dim3(c->red_nblk, 1), BLAS_THREADS, 0, c->st>>>(c->n(), c->sc_dev, (const cx<T> *)c->cg_p, (const cx<T> *)c->cg_Ap,
                                                                          (cx<T> *)x[r], (cx<T> *)c->cg_r, c->red_partial);
            ++c->launches;
        }
        OVL_TRY(group_scalar(g, 2, tol2));
        for (int r : g->mine) {
            ovl_ctx *c = g->s[r];
            DevGuard dg(g->dev[r]);
            k_xpay<T><<<dim3(grid_for(c->n(), BLAS_THREADS), 1), BLAS_THREADS, 0, c->st>>>(c->n(), c->sc_dev, (const cx<T> *)c->cg_r, (cx<T> *)c->cg_p);
            ++c->launches;
        }
        OVL_TRY(fetch0());
        ++it;
        rr = c0->sc_host[SC_RR];
        if (!(rr == rr)) return gfail(g, OVL_ECUDA, "CG broke down (NaN residual) at iteration %d", it);
        if (tol > 0 && rr <= tol2 * bb) conv = true;
    }
    *iters = it;
    OVL_TRY(group_overlap<T>(g, mu, 0, x, q_.data()));
    OVL_TRY(group_overlap<T>(g, mu, 1, q_.data(), Ap_.data()));
    for (int r : g->mine) {
        ovl_ctx *c = g->s[r];
        DevGuard dg(g->dev[r]);
        k_sub<T><<<dim3(grid_for(c->n(), BLAS_THREADS), 1), BLAS_THREADS, 0, c->st>>>(c->n(), (const cx<T> *)b[r], (const cx<T> *)c->cg_Ap, (cx<T> *)c->cg_q);
        k_redot<T><<<dim3(c->red_nblk, 1), BLAS_THREADS, 0, c->st>>>(c->n(), (const cx<T> *)c->cg_q, (const cx<T> *)c->cg_q, c->red_partial);
        c->launches += 2;
    }
    OVL_TRY(group_scalar(g, 3, 0.0));
    OVL_TRY(fetch0());
    *relres = bb > 0 ? std::sqrt(c0->sc_host[SC_PAP] / bb) : 0.0;
    if (tol > 0 && !conv) return gfail(g, OVL_ENOTCONV, "CG: %d iterations, ||r||/||b|| = %.3e > tol", it, std::sqrt(rr / bb));
    return OVL_OK;
}

}  // namespace ovl
