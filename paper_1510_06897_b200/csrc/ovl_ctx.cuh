// ovl_ctx.cuh -- the context behind the opaque ovl_ctx of include/ovl.h, and small host helpers.
#pragma once
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <vector>

#include "../../include/ovl.h"
#include "ovl_types.cuh"

struct ovl_ctx {
    ovl::Geom g{};
    ovl::Sweep sweep{0, 0};  // L2-aware tile order (tpc = 0: plain order)
    ovl::Brick brick{0, 0};  // brick order for small lattices (nchunk = 0: plain order)
    ovl::Brick brick_auto{0, 0};  // what create chose (OVL_FUSED_PLAIN switches `brick` off, OVL_FUSED_REGISTER restores it)
    ovl::Brick brick_geom{0, 0};  // the brick decomposition of this lattice if it has one (OVL_FUSED_BRICK forces it)
    int prec = OVL_F64, recon = OVL_RECON18, recurrence = OVL_REC_CLENSHAW, fused_variant = OVL_FUSED_REGISTER;
    int sm_count = 148;
    cudaStream_t st = nullptr;
    double m_w = 1.5, lambda_max = 6.5;

    // eq. 2.3 inputs
    std::vector<double> alpha;  // alpha[0..N]
    int norders = 0;            // K^ applications actually run (last non-zero alpha, >= 1)
    int nev = 0;
    std::vector<double> lambda, coef;  // coef_i = sign(lambda_i) - p(lambda_i / lambda_max)
    bool coef_stale = true;

    // device memory owned by the context (all native layout unless said otherwise)
    void *U = nullptr;    // links
    void *phi = nullptr;  // eigenvectors [nev][12][V]
    void *psi_n = nullptr, *out_n = nullptr, *tA = nullptr, *tB = nullptr, *acc = nullptr, *g5b = nullptr;
    int work_nrhs = 1;                               // right-hand sides tA, tB, acc, g5b are sized for
    void *multi_in = nullptr, *multi_out = nullptr;  // native staging of ovl_overlap_multi (multi_cap fields each)
    int multi_cap = 0;
    void *cg_r = nullptr, *cg_p = nullptr, *cg_q = nullptr, *cg_Ap = nullptr;
    int cg_nrhs = 0;  // systems the CG vectors are sized for
    void *stage_in = nullptr, *stage_out = nullptr;  // canonical staging for host pointers (12V complex128 each)
    double2 *proj_partial = nullptr, *w_dev = nullptr;
    double *coef_dev = nullptr;
    int proj_nblk = 0, proj_cap = 0, proj_rhs = 0;  // blocks of the projection grid; eigenvector / right-hand-side capacity of its scratch
    double *red_partial = nullptr, *sc_dev = nullptr, *sc_host = nullptr;  // sc_host: two pinned slots of SC_N * OVL_MAX_RHS
    cudaEvent_t cg_ev[2] = {nullptr, nullptr};                             // read-back events of the pipelined CG check
    int red_nblk = 0;

    // CUDA graphs of the polynomial loop (one per source field), replayed instead of re-issuing norders launches
    struct PolyGraph {
        const void *src = nullptr;
        unsigned long long gen = 0, last_use = 0;
        int nrhs = 1;
        cudaGraphExec_t exec = nullptr;
    };
    static constexpr int NGRAPH = 8;
    PolyGraph graphs[NGRAPH];
    unsigned long long poly_gen = 1, use_clock = 0;  // poly_gen changes whenever the launch sequence would
    bool use_graphs = true;

    // measurement
    bool profiling = false;
    static constexpr int NPROF = 64;  // ring of event pairs: one per profiled polynomial loop
    cudaEvent_t pev0[NPROF] = {}, pev1[NPROF] = {};
    long long prof_count = 0;         // profiled loops since ovl_set_profiling(on)
    int last_poly_launches = 0;
    long long launches = 0;

    // memory: either one caller-owned workspace (ovl_create_ws: everything below is carved from it at create time and
    // nothing is allocated afterwards) or library-owned allocations (ovl_create: one cudaMalloc for the base set, more
    // only when a capacity grows: eigenvector store, multi-rhs workspaces, eigensolver block)
    struct Arena { char *base = nullptr; size_t size = 0, off = 0; } arena;
    bool ws_mode = false;            // caller-owned workspace: never cudaMalloc / cudaFree
    std::vector<void *> owned;       // library-owned device allocations (freed by ovl_destroy)
    int max_nev = 0, max_rhs = 1, eig_cap = 0;   // capacities of a caller-owned workspace
    void *eig_ws = nullptr;          // eigensolver block inside a caller-owned workspace
    size_t eig_ws_bytes = 0;

    char err[256] = {0};

    size_t n() const { return (size_t)12 * g.V; }                       // complex elements per spinor
    size_t tsize() const { return prec == OVL_F64 ? sizeof(double) : sizeof(float); }
    size_t field_bytes() const { return n() * 2 * tsize(); }
    size_t canon_bytes() const { return n() * 2 * tsize(); }            // canonical spinor at the boundary
    int nrow() const { return recon == OVL_RECON18 ? 3 : 2; }
    size_t link_bytes() const { return (size_t)4 * nrow() * 3 * g.V * 2 * tsize(); }
};

namespace ovl {

inline int fail(ovl_ctx *c, int code, const char *fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof c->err, fmt, ap);
        va_end(ap);
    }
    return code;
}

#define OVL_CUDA(c, call)                                                                              \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess) {                                                                       \
            cudaGetLastError();                                                                        \
            return ovl::fail((c), e_ == cudaErrorMemoryAllocation ? OVL_ENOMEM : OVL_ECUDA, "%s: %s", #call, \
                             cudaGetErrorString(e_));                                                  \
        }                                                                                              \
    } while (0)

#define OVL_TRY(expr)                  \
    do {                               \
        int rc_ = (expr);              \
        if (rc_ != OVL_OK) return rc_; \
    } while (0)

// device (or managed) pointer -> usable by kernels in place; anything else is treated as host memory
inline bool is_device_ptr(const void *p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

constexpr size_t WS_ALIGN = 256;
inline size_t ws_round(size_t b) { return (b + WS_ALIGN - 1) / WS_ALIGN * WS_ALIGN; }

// Device memory for the context: carved from the arena while it has room; otherwise cudaMalloc -- unless the context
// lives in a caller-owned workspace, where running out is an error (the capacity was fixed by ovl_workspace_bytes).
inline int dev_alloc(ovl_ctx *c, void **p, size_t bytes) {
    if (*p) return OVL_OK;
    const size_t b = ws_round(bytes ? bytes : 16);
    if (c->arena.base && c->arena.off + b <= c->arena.size) {
        *p = c->arena.base + c->arena.off;
        c->arena.off += b;
        return OVL_OK;
    }
    if (c->ws_mode) return fail(c, OVL_ENOMEM, "the caller-owned workspace is exhausted (%zu more bytes needed)", b);
    OVL_CUDA(c, cudaMalloc(p, b));
    c->owned.push_back(*p);
    return OVL_OK;
}
// give a buffer back: only library-owned allocations are freed (arena memory lives until ovl_destroy)
inline void dev_release(ovl_ctx *c, void **p) {
    if (!*p) return;
    for (size_t i = 0; i < c->owned.size(); ++i)
        if (c->owned[i] == *p) {
            cudaFree(*p);
            c->owned.erase(c->owned.begin() + i);
            break;
        }
    *p = nullptr;
}

inline int grid_for(size_t n, int threads, int cap = 148 * 16) {
    size_t b = (n + threads - 1) / threads;
    if (b > (size_t)cap) b = cap;
    if (b < 1) b = 1;
    return (int)b;
}

// p(x) = sum_m alpha_m T_m(x) for a real scalar (a6), Clenshaw's backward recurrence in fp64
inline double cheb_scalar(const std::vector<double> &alpha, double x) {
    double b1 = 0, b2 = 0;
    for (int k = (int)alpha.size() - 1; k >= 1; --k) {
        const double b0 = alpha[k] + 2.0 * x * b1 - b2;
        b2 = b1;
        b1 = b0;
    }
    return alpha[0] + x * b1 - b2;
}

}  // namespace ovl
