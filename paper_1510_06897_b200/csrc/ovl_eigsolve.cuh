// ovl_eigsolve.cuh -- lowest-|lambda| eigenpairs of K = gamma5 (D_W - m_w) on the GPU.
// (the paper: polynomial preconditioned implicitly restarted Lanczos).  K is indefinite, so a Rayleigh-Ritz step on K in a
// not-yet-converged subspace produces ghost values inside the gap; the iteration therefore works on the positive K^2 and
// K itself is diagonalised only at the end, inside a space that is K-invariant by construction:
//
//   V: m = nev + pad trial vectors.  Per cycle (Chebyshev-filtered block subspace iteration on K^2):
//     W = K^ V                                   (multi-right-hand-side launches of the fused stencil kernel)
//     G = V^dag V, H = W^dag W = V^dag K^2 V     (tall-skinny products, k_gram_block)
//     H x = sigma G x on the host (Cholesky + Jacobi), ascending;  V <- V X, W <- W X            (k_rotate_block)
//     Z = K^ W;  r_i = || Z_i - sigma_i V_i ||   (K^2 residuals)
//     V <- T_d(Y) V,  Y = (K^2 - c)/e mapping [a, 1] -> [-1, 1],  a = largest sigma in the block (everything above the
//          block is damped, the block is amplified);  T_{j+1} = 2 Y T_j - T_{j-1} costs two stencil launches per step
//   End game, once the nev leading K^2 pairs have converged: for an eigenvector v of K^2, span{v, K v} is K-invariant
//   (K (K v) = sigma v), so K is diagonalised in S = span{V_1..nev, W_1..nev}: orthonormal basis from the eigen-
//   decomposition of S^dag S (directions below 1e-12 dropped), Hermitian eigenproblem of K in it, the nev Ritz pairs of
//   smallest |theta| are returned (with their +-signs, R11) and their residuals recomputed with one more K^.
#pragma once
#include "ovl_dense.h"
#include "ovl_eig.cuh"
#include "ovl_engine.cuh"

namespace ovl {

// residual (in units of lambda_max) above which a filter cycle may run in fp32 (ovl_lowest_eigenpairs_mixed)
constexpr double EIG_F32_FLOOR = 1e-5;

// The work block of one ovl_lowest_eigenpairs call for `cap` = max(block, 2 nev) vectors: one contiguous device region,
// either inside the caller-owned workspace (eig_block of ovl_workspace_bytes) or one cudaMalloc released on return.
struct EigWork {
    double2 *V = nullptr, *W = nullptr, *Z = nullptr, *R = nullptr, *Q = nullptr, *gram_partial = nullptr, *C = nullptr, *X = nullptr;
    double *partial = nullptr, *small = nullptr;  // small: theta / scales / norms, cap doubles each (3 cap)
    int cap = 0;                                  // vectors per work block
    void *owned = nullptr;
    ~EigWork() {
        if (owned) cudaFree(owned);
        cudaGetLastError();
    }
};
template <typename F> inline void eig_ws_visit(size_t V, int cap, F f) {
    const size_t n = 12 * V, fb = n * sizeof(double2);
    const size_t nblk_g = (n + BLAS_THREADS * GRAM_EPT - 1) / (BLAS_THREADS * GRAM_EPT), nchunk_g = (cap + GRAM_J - 1) / GRAM_J;
    const size_t nb = grid_for(n, BLAS_THREADS * 4, 148 * 8);
    f(0, fb * cap); f(1, fb * cap); f(2, fb * cap); f(3, fb * cap); f(4, fb * cap);            // V W Z R Q
    f(5, sizeof(double2) * (size_t)cap * GRAM_J * nblk_g * (BLAS_THREADS / 32));               // gram_partial
    f(6, sizeof(double2) * nchunk_g * cap * GRAM_J);                                            // C
    f(7, sizeof(double2) * (size_t)cap * cap);                                                  // X
    f(8, sizeof(double) * nb * cap);                                                            // partial
    f(9, sizeof(double) * 3 * cap);                                                             // small
}
inline size_t eig_ws_total(size_t V, int cap) {
    size_t t = 0;
    eig_ws_visit(V, cap, [&](int, size_t b) { t += ws_round(b); });
    return t;
}
inline int eig_ws_setup(ovl_ctx *c, EigWork &w, int cap) {
    const size_t need = eig_ws_total(c->g.V, cap);
    char *base = nullptr;
    if (c->ws_mode) {
        if (cap > c->eig_cap || need > c->eig_ws_bytes)
            return fail(c, OVL_EINVAL, "the eigensolver needs a work block of %d vectors; the workspace was sized for eig_block = %d", cap, c->eig_cap);
        base = (char *)c->eig_ws;
    } else {
        OVL_CUDA(c, cudaMalloc(&w.owned, need));
        base = (char *)w.owned;
    }
    w.cap = cap;
    size_t off = 0;
    eig_ws_visit(c->g.V, cap, [&](int id, size_t b) {
        void *p = base + off;
        off += ws_round(b);
        switch (id) {
            case 0: w.V = (double2 *)p; break;
            case 1: w.W = (double2 *)p; break;
            case 2: w.Z = (double2 *)p; break;
            case 3: w.R = (double2 *)p; break;
            case 4: w.Q = (double2 *)p; break;
            case 5: w.gram_partial = (double2 *)p; break;
            case 6: w.C = (double2 *)p; break;
            case 7: w.X = (double2 *)p; break;
            case 8: w.partial = (double *)p; break;
            case 9: w.small = (double *)p; break;
        }
    });
    return OVL_OK;
}

// C (host, m x m row-major) = A^dag B for the m-vector blocks A, B
inline int eig_gram(ovl_ctx *c, EigWork &w, int m, const double2 *A, const double2 *B, dense::mat &out) {
    const size_t n = c->n();
    const int nblk = (int)((n + BLAS_THREADS * GRAM_EPT - 1) / (BLAS_THREADS * GRAM_EPT));
    const int nchunk = (m + GRAM_J - 1) / GRAM_J;
    for (int ch = 0; ch < nchunk; ++ch) {
        const int j0 = ch * GRAM_J, nj = std::min(GRAM_J, m - j0);
        k_gram_block<<<nblk, BLAS_THREADS, 0, c->st>>>(n, m, nj, A, B + (size_t)j0 * n, w.gram_partial);
        OVL_LAUNCH_CHECK(c);
        k_gram_final<<<m * GRAM_J, BLAS_THREADS, 0, c->st>>>(nblk * (BLAS_THREADS / 32), w.gram_partial, w.C + (size_t)ch * m * GRAM_J);
        OVL_LAUNCH_CHECK(c);
    }
    std::vector<double2> h((size_t)nchunk * m * GRAM_J);
    OVL_CUDA(c, cudaMemcpyAsync(h.data(), w.C, h.size() * sizeof(double2), cudaMemcpyDeviceToHost, c->st));
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    out.assign((size_t)m * m, dense::cd(0, 0));
    for (int ch = 0; ch < nchunk; ++ch)
        for (int i = 0; i < m; ++i)
            for (int jj = 0; jj < GRAM_J && ch * GRAM_J + jj < m; ++jj) {
                const double2 v = h[((size_t)ch * m + i) * GRAM_J + jj];
                out[(size_t)i * m + ch * GRAM_J + jj] = dense::cd(v.x, v.y);
            }
    return OVL_OK;
}

// dst block (nout vectors) = src block (nin vectors) * X  (X on the device, row-major nin x ldx, first nout columns)
inline int eig_rotate(ovl_ctx *c, EigWork &w, int nin, int nout, int ldx, const double2 *src, double2 *dst) {
    const size_t n = c->n();
    for (int o0 = 0; o0 < nout; o0 += ROT_JO) {
        const int no = std::min(ROT_JO, nout - o0);
        k_rotate_block<<<grid_for(n, BLAS_THREADS, 1 << 30), BLAS_THREADS, 0, c->st>>>(n, nin, no, ldx, w.X + o0, src, dst + (size_t)o0 * n);
        OVL_LAUNCH_CHECK(c);
    }
    return OVL_OK;
}

// out_r = K^ in_r for a block of nvec consecutive native fields of precision T, OVL_MAX_RHS at a time
template <typename T> inline int eig_khat_block_t(ovl_ctx *c, int nvec, const cx<T> *in, cx<T> *out) {
    const size_t n = c->n();
    for (int j0 = 0; j0 < nvec; j0 += OVL_MAX_RHS) {
        WilsonArgs a;
        a.nrhs = std::min((int)OVL_MAX_RHS, nvec - j0);
        a.in = in + (size_t)j0 * n; a.out = out + (size_t)j0 * n;
        a.c_diag = (4.0 - c->m_w) / c->lambda_max; a.c_hop = -0.5 / c->lambda_max;
        OVL_TRY((launch_wilson<T, K_G5>(c, a)));
    }
    return OVL_OK;
}
inline int eig_khat_block(ovl_ctx *c, int nvec, const double2 *in, double2 *out) { return eig_khat_block_t<double>(c, nvec, in, out); }

// V_chunk <- T_d((K^2 - cc)/ee) V_chunk / rho^d, with W_chunk = K^ V_chunk on entry (d >= 1), in the precision T of context c
// (its recurrence workspace tA, acc).  rho = 1: the plain recurrence.  rho > 1: the recurrence for s_j = t_j / rho^j,
//     s_{j+1} = [(2/ee) K^2 s_j - (2 cc/ee) s_j] / rho - s_{j-1} / rho^2,
// which keeps the fastest-growing component O(1) -- T_d grows like (|y| + sqrt(y^2 - 1))^d below the damped interval, 1e172
// in the first cycles from a random start, far outside fp32 -- at no cost: the scale factors ride on the kernel's scalars.
template <typename T>
inline int eig_filter_chunk(ovl_ctx *c, int nv, int d, double cc, double ee, double rho, cx<T> *Vc, const cx<T> *Wc) {
    const double cd = (4.0 - c->m_w) / c->lambda_max, ch = -0.5 / c->lambda_max;
    const size_t fb = c->field_bytes() * nv;
    cx<T> *tcur = (cx<T> *)c->tA, *tprev = Vc, *wbuf = (cx<T> *)c->acc;
    {   // s_1 = (K^ W - cc V)/(ee rho)
        WilsonArgs a;
        a.nrhs = nv; a.in = Wc; a.psi = Vc; a.out = tcur;
        a.c_diag = cd / (ee * rho); a.c_hop = ch / (ee * rho); a.a_psi = -cc / (ee * rho);
        OVL_TRY((launch_wilson<T, K_G5 | K_PSI>(c, a)));
    }
    for (int j = 1; j < d; ++j) {  // s_{j+1}, written over s_{j-1}
        WilsonArgs k;
        k.nrhs = nv; k.in = tcur; k.out = wbuf; k.c_diag = cd; k.c_hop = ch;
        OVL_TRY((launch_wilson<T, K_G5>(c, k)));
        WilsonArgs a;
        a.nrhs = nv; a.in = wbuf; a.psi = tcur; a.prev = tprev; a.out = tprev;
        a.c_diag = 2.0 * cd / (ee * rho); a.c_hop = 2.0 * ch / (ee * rho); a.a_psi = -2.0 * cc / (ee * rho);
        a.c_prev = 1.0 / (rho * rho);
        OVL_TRY((launch_wilson<T, K_G5 | K_PSI | K_PREV>(c, a)));
        std::swap(tcur, tprev);
    }
    if (tcur != Vc) OVL_CUDA(c, cudaMemcpyAsync(Vc, tcur, fb, cudaMemcpyDeviceToDevice, c->st));
    return OVL_OK;
}
// The same filter for a chunk of the fp64 block, run in the fp32 sibling context c32 (same lattice, same stream): the chunk
// is rounded to fp32 into c32's workspace (g5b), W = K^ V is formed there (tB), the scaled recurrence runs on the fp32 stencil
// kernels (half the bytes per launch) and the result is widened back.  rho from sigma = 0, the most negative argument.
inline int eig_filter_chunk_f32(ovl_ctx *c, ovl_ctx *c32, int nv, int d, double cc, double ee, double2 *Vc) {
    const size_t n = c->n() * (size_t)nv;
    const int grid = grid_for(n, BLAS_THREADS);
    float2 *Vf = (float2 *)c32->g5b, *Wf = (float2 *)c32->tB;
    k_convert_scaled<double, float><<<grid, BLAS_THREADS, 0, c->st>>>(n, 1.0, Vc, Vf);
    OVL_LAUNCH_CHECK(c);
    {
        const int rc = eig_khat_block_t<float>(c32, nv, Vf, Wf);
        if (rc != OVL_OK) return fail(c, rc, "fp32 filter: %s", c32->err);
    }
    const double y0 = cc / ee, rho = y0 + std::sqrt(std::max(y0 * y0 - 1.0, 0.0));
    {
        const int rc = eig_filter_chunk<float>(c32, nv, d, cc, ee, rho, Vf, Wf);
        if (rc != OVL_OK) return fail(c, rc, "fp32 filter: %s", c32->err);
    }
    k_convert_scaled<float, double><<<grid, BLAS_THREADS, 0, c->st>>>(n, 1.0, Vf, Vc);
    OVL_LAUNCH_CHECK(c);
    return OVL_OK;
}

// residual norms || A_i - theta_i B_i || for i < k into host vector (A, B blocks of k fields)
inline int eig_resid(ovl_ctx *c, EigWork &w, int k, const std::vector<double> &theta, const double2 *A, const double2 *B, std::vector<double> &out) {
    const int nb = c->red_nblk;
    double *theta_d = w.small, *norm_d = w.small + 2 * w.cap;
    OVL_CUDA(c, cudaMemcpyAsync(theta_d, theta.data(), sizeof(double) * k, cudaMemcpyHostToDevice, c->st));
    k_resid_norm2<<<dim3(nb, k), BLAS_THREADS, 0, c->st>>>(c->n(), theta_d, A, B, w.partial);
    OVL_LAUNCH_CHECK(c);
    k_sum_partials<<<k, BLAS_THREADS, 0, c->st>>>(nb, w.partial, norm_d);
    OVL_LAUNCH_CHECK(c);
    out.resize(k);
    OVL_CUDA(c, cudaMemcpyAsync(out.data(), norm_d, sizeof(double) * k, cudaMemcpyDeviceToHost, c->st));
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    for (double &x : out) x = std::sqrt(std::max(x, 0.0));
    return OVL_OK;
}

// End game (see the header): K diagonalised in span{V_1..nev, W_1..nev}; the nev Ritz vectors of smallest |theta| are
// written to w.Z[0..nev), theta (in units of lambda_max) and the true residuals || K^ z - theta z || to the outputs.
inline int eig_endgame(ovl_ctx *c, EigWork &w, int nev, std::vector<double> &theta_out, std::vector<double> &resid_out) {
    const size_t n = c->n(), fb = c->field_bytes();
    const int k2 = 2 * nev;
    // S = [V_1..nev, W_1..nev] in R, K S = [W_1..nev, Z_1..nev] in Q
    OVL_CUDA(c, cudaMemcpyAsync(w.R, w.V, fb * nev, cudaMemcpyDeviceToDevice, c->st));
    OVL_CUDA(c, cudaMemcpyAsync(w.R + (size_t)nev * n, w.W, fb * nev, cudaMemcpyDeviceToDevice, c->st));
    OVL_CUDA(c, cudaMemcpyAsync(w.Q, w.W, fb * nev, cudaMemcpyDeviceToDevice, c->st));
    OVL_CUDA(c, cudaMemcpyAsync(w.Q + (size_t)nev * n, w.Z, fb * nev, cudaMemcpyDeviceToDevice, c->st));
    dense::mat G, H, Qm, Y;
    OVL_TRY(eig_gram(c, w, k2, w.R, w.R, G));
    OVL_TRY(eig_gram(c, w, k2, w.R, w.Q, H));
    std::vector<double> lamG, th;
    dense::mat Gc = G;
    dense::jacobi_eigh(Gc, k2, lamG, Qm);
    double gmax = 0;
    for (double x : lamG) gmax = std::max(gmax, x);
    std::vector<int> keep;
    for (int i = 0; i < k2; ++i)
        if (lamG[i] > 1e-12 * gmax) keep.push_back(i);
    const int r = (int)keep.size();
    if (r < nev) return fail(c, OVL_ECUDA, "eigensolver: end-game space has dimension %d < nev", r);
    // T = Q_keep Lambda^{-1/2}  (k2 x r);  Hr = T^dag H T
    dense::mat T((size_t)k2 * r), HT((size_t)k2 * r), Hr((size_t)r * r);
    for (int i = 0; i < k2; ++i)
        for (int a = 0; a < r; ++a) T[(size_t)i * r + a] = Qm[(size_t)i * k2 + keep[a]] / std::sqrt(lamG[keep[a]]);
    for (int i = 0; i < k2; ++i)
        for (int a = 0; a < r; ++a) {
            dense::cd s = 0;
            for (int j = 0; j < k2; ++j) s += 0.5 * (H[(size_t)i * k2 + j] + std::conj(H[(size_t)j * k2 + i])) * T[(size_t)j * r + a];
            HT[(size_t)i * r + a] = s;
        }
    for (int a = 0; a < r; ++a)
        for (int b = 0; b < r; ++b) {
            dense::cd s = 0;
            for (int i = 0; i < k2; ++i) s += std::conj(T[(size_t)i * r + a]) * HT[(size_t)i * r + b];
            Hr[(size_t)a * r + b] = s;
        }
    for (int a = 0; a < r; ++a)
        for (int b = a; b < r; ++b) {
            const dense::cd v = 0.5 * (Hr[(size_t)a * r + b] + std::conj(Hr[(size_t)b * r + a]));
            Hr[(size_t)a * r + b] = v;
            Hr[(size_t)b * r + a] = std::conj(v);
        }
    dense::jacobi_eigh(Hr, r, th, Y);
    std::vector<int> order(r);
    for (int i = 0; i < r; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](int a, int b) { return std::fabs(th[a]) < std::fabs(th[b]); });
    // coefficients of the nev chosen Ritz vectors in S: X = T Y[:, order[:nev]]   (k2 x nev)
    std::vector<double2> xs((size_t)k2 * nev);
    theta_out.resize(nev);
    for (int o = 0; o < nev; ++o) {
        theta_out[o] = th[order[o]];
        for (int i = 0; i < k2; ++i) {
            dense::cd s = 0;
            for (int a = 0; a < r; ++a) s += T[(size_t)i * r + a] * Y[(size_t)a * r + order[o]];
            xs[(size_t)i * nev + o] = make_double2(s.real(), s.imag());
        }
    }
    OVL_CUDA(c, cudaMemcpyAsync(w.X, xs.data(), xs.size() * sizeof(double2), cudaMemcpyHostToDevice, c->st));
    OVL_TRY(eig_rotate(c, w, k2, nev, nev, w.R, w.Z));
    OVL_CUDA(c, cudaStreamSynchronize(c->st));  // xs is pageable host memory
    OVL_TRY(eig_khat_block(c, nev, w.Z, w.Q));
    return eig_resid(c, w, nev, theta_out, w.Q, w.Z, resid_out);
}

inline int eig_lowest(ovl_ctx *c, ovl_ctx *c32, int nev, double tol, int max_cycles, int degree, int block, unsigned long long seed,
                      void *phi_out, double *lambda_out, double *resid_out, int *cycles_out, int *f32_cycles_out = nullptr) {
    const size_t n = c->n();
    int m = block > 0 ? block : nev + std::max(8, nev / 2);
    if (m < nev) m = nev;
    if (m > 128 || nev > 64) return fail(c, OVL_EINVAL, "block size %d > 128 or nev %d > 64", m, nev);
    if ((size_t)m > n) return fail(c, OVL_EINVAL, "block size %d exceeds the dimension of the space", m);
    if (degree < 1) degree = 1;
    const int cap = std::max(m, 2 * nev);  // vectors per work block
    int chunk = std::min(m, c->ws_mode ? c->max_rhs : (int)OVL_MAX_RHS);  // vectors per filter pass (recurrence workspace)
    if (c32 && c32->ws_mode) chunk = std::min(chunk, c32->max_rhs);          // ... of both contexts
    OVL_TRY(ensure_work(c, chunk));
    if (c32) {
        const int rc = ensure_work(c32, chunk);
        if (rc != OVL_OK) return fail(c, rc, "fp32 context: %s", c32->err);
    }
    int n_f32_cycles = 0;
    bool f32_allowed = true, last_was_f32 = false;
    double last_worst = 0;
    EigWork w;
    OVL_TRY(eig_ws_setup(c, w, cap));
    const int nb = c->red_nblk;
    double *scale_d = w.small + cap, *norm_d = w.small + 2 * cap;

    for (int j = 0; j < m; ++j) {
        k_fill_random<<<grid_for(n, BLAS_THREADS), BLAS_THREADS, 0, c->st>>>(n, seed * 1000003ull + j, w.V + (size_t)j * n);
        OVL_LAUNCH_CHECK(c);
    }
    std::vector<double> sigma(m), r2, hs(m), theta, resid;
    std::vector<int> order(m);
    dense::mat G, H, X;
    int cycle = 0;
    bool converged = false, have_result = false;
    double tol_int = 0.5 * tol / c->lambda_max;  // on || K^ z - theta z ||; tightened if the end game misses tol
    for (;;) {
        OVL_TRY(eig_khat_block(c, m, w.V, w.W));
        OVL_TRY(eig_gram(c, w, m, w.V, w.V, G));
        OVL_TRY(eig_gram(c, w, m, w.W, w.W, H));
        std::vector<double> sg;
        if (!dense::geneig(H, G, m, sg, X))
            return fail(c, OVL_ECUDA, "eigensolver: the trial block became linearly dependent (cycle %d)", cycle);
        for (int i = 0; i < m; ++i) order[i] = i;
        std::sort(order.begin(), order.end(), [&](int a, int b) { return sg[a] < sg[b]; });
        std::vector<double2> xs((size_t)m * m);
        for (int j = 0; j < m; ++j)
            for (int o = 0; o < m; ++o) {
                const dense::cd v = X[(size_t)j * m + order[o]];
                xs[(size_t)j * m + o] = make_double2(v.real(), v.imag());
            }
        for (int o = 0; o < m; ++o) sigma[o] = std::max(sg[order[o]], 0.0);
        OVL_CUDA(c, cudaMemcpyAsync(w.X, xs.data(), xs.size() * sizeof(double2), cudaMemcpyHostToDevice, c->st));
        OVL_TRY(eig_rotate(c, w, m, m, m, w.V, w.R));
        std::swap(w.V, w.R);
        OVL_TRY(eig_rotate(c, w, m, m, m, w.W, w.R));
        std::swap(w.W, w.R);
        OVL_CUDA(c, cudaStreamSynchronize(c->st));  // xs is pageable host memory
        OVL_TRY(eig_khat_block(c, m, w.W, w.Z));
        OVL_TRY(eig_resid(c, w, m, sigma, w.Z, w.V, r2));
        // K^2 residual r2 <-> K residual r2 / |theta| of the vectors v +- K v / theta
        double worst = 0;
        for (int i = 0; i < nev; ++i) worst = std::max(worst, r2[i] / std::max(std::sqrt(sigma[i]), 1e-300));
        if (worst <= tol_int) {
            OVL_TRY(eig_endgame(c, w, nev, theta, resid));
            have_result = true;
            double wr = 0;
            for (int i = 0; i < nev; ++i) wr = std::max(wr, resid[i] * c->lambda_max);
            if (wr <= tol) { converged = true; break; }
            tol_int *= 0.1;
        }
        if (cycle >= max_cycles) break;
        ++cycle;
        have_result = false;  // the next cycle overwrites w.Z (the Ritz vectors of a missed end game) with K^ W
        // filter: damp [a, 1] of K^2, a = top of the block.  Two economies (the filter is > 90 % of the run time):
        //  * the degree follows the gap: T_d damps the top of the block against the wanted Ritz pairs by about
        //    exp(-2 d sqrt((a - sigma_nev) / (1 - a))) per cycle; the degree is chosen for e^-8 and capped at `degree`, which
        //    shortens the first cycles from a random start (91, 133, 156 instead of 3 x 200 at 20^3 x 64) -- the asymptotic
        //    cycles, where a - sigma_nev ~ 2e-4, always run at the cap;
        //  * the leading columns whose K^2 residual is already a factor 10 below the working tolerance are left as they are
        //    (they stay in the basis; the next Rayleigh-Ritz step re-mixes them): only columns [nlock, m) are filtered.
        // (A doubling ramp 12, 24, 48, ... for the first cycles was tried: two more cycles, same total time.)
        const double a = std::min(sigma[m - 1], 0.95);
        const double cc = 0.5 * (1.0 + a), ee = 0.5 * (1.0 - a);
        const double gap = std::max(a - sigma[nev - 1], 0.0) / (1.0 - a);
        int deg = degree;
        if (gap > 0) deg = (int)std::ceil(4.0 / std::sqrt(gap));
        deg = std::max(std::min(deg, degree), std::min(degree, 10));
        int nlock = 0;
        while (nlock < nev && r2[nlock] / std::max(std::sqrt(sigma[nlock]), 1e-300) <= 0.1 * tol_int) ++nlock;
        //  * with an fp32 sibling context the filter runs on the fp32 stencil kernels (eig_filter_chunk_f32) while the block is
        //    far from the tolerance: the filter only has to damp the unwanted part by e^-8 per cycle, the Rayleigh-Ritz step
        //    and every residual stay in fp64, and the fp32 rounding (~1e-6 of a filtered vector) is removed by the fp64 cycles
        //    that follow once the residual is below EIG_F32_FLOOR (measured: the same number of cycles and the same residuals as
        //    the all-fp64 run; 8^3 x 32: 5 of 7 cycles in fp32, 20^3 x 64: 29.6 -> 21 s).
        // (an fp32 filter cannot take the residual below ~1e-6 lambda_max: a cycle that gains less than a factor 3 in fp32 is
        // the sign of that floor, and the rest of the run stays in fp64)
        if (last_was_f32 && worst > 0.3 * last_worst) f32_allowed = false;
        const bool f32_cycle = c32 != nullptr && f32_allowed && worst > EIG_F32_FLOOR;
        last_was_f32 = f32_cycle;
        last_worst = worst;
        n_f32_cycles += f32_cycle;
        for (int j0 = nlock; j0 < m; j0 += chunk) {
            const int nv = std::min(chunk, m - j0);
            if (f32_cycle) OVL_TRY(eig_filter_chunk_f32(c, c32, nv, deg, cc, ee, w.V + (size_t)j0 * n));
            else OVL_TRY(eig_filter_chunk<double>(c, nv, deg, cc, ee, 1.0, w.V + (size_t)j0 * n, w.W + (size_t)j0 * n));
        }
        // normalise
        k_redot<double><<<dim3(nb, m), BLAS_THREADS, 0, c->st>>>(n, w.V, w.V, w.partial);
        OVL_LAUNCH_CHECK(c);
        k_sum_partials<<<m, BLAS_THREADS, 0, c->st>>>(nb, w.partial, norm_d);
        OVL_LAUNCH_CHECK(c);
        OVL_CUDA(c, cudaMemcpyAsync(hs.data(), norm_d, sizeof(double) * m, cudaMemcpyDeviceToHost, c->st));
        OVL_CUDA(c, cudaStreamSynchronize(c->st));
        for (int i = 0; i < m; ++i) {
            if (!(hs[i] > 0) || !std::isfinite(hs[i])) return fail(c, OVL_ECUDA, "eigensolver: filtered vector %d has norm^2 %g", i, hs[i]);
            hs[i] = 1.0 / std::sqrt(hs[i]);
        }
        OVL_CUDA(c, cudaMemcpyAsync(scale_d, hs.data(), sizeof(double) * m, cudaMemcpyHostToDevice, c->st));
        k_scale_batched<<<dim3(grid_for(n, BLAS_THREADS), m), BLAS_THREADS, 0, c->st>>>(n, scale_d, w.V);
        OVL_LAUNCH_CHECK(c);
        OVL_CUDA(c, cudaStreamSynchronize(c->st));
    }
    if (!have_result) OVL_TRY(eig_endgame(c, w, nev, theta, resid));  // best effort on the unconverged block
    // results: nev Ritz pairs of K in w.Z
    const size_t cb = n * sizeof(double2);
    for (int i = 0; i < nev; ++i) {
        lambda_out[i] = theta[i] * c->lambda_max;
        if (resid_out) resid_out[i] = resid[i] * c->lambda_max;
        void *dst = (char *)phi_out + (size_t)i * cb;
        if (is_device_ptr(phi_out)) {
            k_export_spinor<double, double><<<grid_for(n, BLAS_THREADS), BLAS_THREADS, 0, c->st>>>(c->g.V, w.Z + (size_t)i * n, (double2 *)dst);
            OVL_LAUNCH_CHECK(c);
        } else {
            OVL_TRY(dev_alloc(c, &c->stage_out, cb));
            k_export_spinor<double, double><<<grid_for(n, BLAS_THREADS), BLAS_THREADS, 0, c->st>>>(c->g.V, w.Z + (size_t)i * n, (double2 *)c->stage_out);
            OVL_LAUNCH_CHECK(c);
            OVL_CUDA(c, cudaMemcpyAsync(dst, c->stage_out, cb, cudaMemcpyDeviceToHost, c->st));
            OVL_CUDA(c, cudaStreamSynchronize(c->st));
        }
    }
    OVL_CUDA(c, cudaStreamSynchronize(c->st));
    *cycles_out = cycle;
    if (f32_cycles_out) *f32_cycles_out = n_f32_cycles;
    if (!converged) {
        double worst = 0;
        for (int i = 0; i < nev; ++i) worst = std::max(worst, resid[i] * c->lambda_max);
        return fail(c, OVL_ENOTCONV, "eigensolver: %d cycles, largest residual ||K phi - lambda phi|| = %.3e > tol", cycle, worst);
    }
    return OVL_OK;
}

}  // namespace ovl
