/*
 * ovl_oracle.c -- CPU ORACLE for the overlap Dirac operator hot path of arXiv 1510.06897.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the plain, slow, obviously-correct fp64 statement of what the
 * hot path computes, written from the paper's equations.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code, header,
 * table or layout with the CUDA path under paper_1510_06897_b200/csrc/ and neither includes the other.
 *
 * What follows the paper, passage by passage (PAPER.md = /root/reference/PAPER.md):
 *   orc_dw        eq. 2.2, read as 4 psi(x) - 1/2 sum_mu [...]           (R1)
 *   orc_khat      K = gamma5 (D_W - m_w); K^ = K / lambda_max               (R5)
 *   orc_cheb      first sum of eq. 2.3: sum_m alpha_m T_m(K^) psi by the
 *                 three-term recurrence T_{m+1} = 2x T_m - T_{m-1}
 *   orc_clenshaw  the same polynomial by Clenshaw's backward recurrence (self-check only)
 *   orc_deflate   second sum of eq. 2.3
 *   orc_sign      eq. 2.3 complete
 *   orc_overlap   eq. 2.1 and its adjoint                               (R12)
 *   orc_cg        textbook Hestenes-Stiefel CG on D^dag D (north_star (d); R13, R14)
 *   orc_chiral_op, orc_cg_chiral
 *                 the chiral-sector form of D^dag D ("[D^dag D, gamma5] = 0": one sign
 *                 application per operator application) and the same textbook CG on it          (R23)
 *
 * Conventions: dims = {Lx,Ly,Lz,Lt}; site s = x + Lx (y + Ly (z + Lz t));
 * links U[s][mu][row][col], mu = x,y,z,t, U_mu(x) is the matrix multiplying psi(x + mu) in eq. 2.2;
 * spinor psi[s][spin][colour]; periodic in x,y,z, antiperiodic in t (R3): a hop across the t boundary
 * carries -1.  Gamma matrices: Euclidean Hermitian chiral basis fixed in GAMMA below (R2),
 * gamma5 = gamma_x gamma_y gamma_z gamma_t = diag(1,1,-1,-1).
 *
 * Parity pins: tests/test_oracle_*.py (closed-form free spectrum, gamma5-hermiticity, gauge covariance,
 * dense eigendecomposition on 2^4/4^4, sign^2 = 1, Ginsparg-Wilson, dense CG solve; the chiral-sector
 * operator against P_c D^dag D P_c built from the dense exact sign function).  Nothing here is
 * "parity unpinned" except what is tied to the paper's ensembles and timings (unavailable).
 *
 * Loops over sites are OpenMP-parallel; there is no blocking, fusion or reordering beyond that.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

/* gamma_mu[row][col], rows top to bottom (R2) */
static const cplx GAMMA[4][4][4] = {
    /* gamma_x */ {{0, 0, 0, I}, {0, 0, I, 0}, {0, -I, 0, 0}, {-I, 0, 0, 0}},
    /* gamma_y */ {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    /* gamma_z */ {{0, 0, I, 0}, {0, 0, 0, -I}, {-I, 0, 0, 0}, {0, I, 0, 0}},
    /* gamma_t */ {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}},
};
static const double GAMMA5[4] = {1.0, 1.0, -1.0, -1.0};

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_gamma(int mu, cplx *out16) { /* expose the basis to the pins (Clifford algebra test) */
    for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b) out16[4 * a + b] = GAMMA[mu][a][b];
}

static long vol(const int *d) { return (long)d[0] * d[1] * d[2] * d[3]; }

/* (D_W psi)(x) = 4 psi(x) - 1/2 sum_mu [ (1 - gamma_mu) U_mu(x) psi(x+mu) + (1 + gamma_mu) U_mu(x-mu)^dag psi(x-mu) ] */
void orc_dw(const int *dims, const cplx *U, const cplx *psi, cplx *out) {
    const long V = vol(dims);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s) {
        int x[4];
        long r = s;
        for (int mu = 0; mu < 4; ++mu) { x[mu] = (int)(r % dims[mu]); r /= dims[mu]; }
        cplx hop[4][3];
        memset(hop, 0, sizeof hop);
        long stride = 1;
        for (int mu = 0; mu < 4; ++mu) {
            const int L = dims[mu];
            /* forward neighbour x + mu */
            long sf = s + ((x[mu] == L - 1) ? -(long)(L - 1) * stride : stride);
            double bf = (mu == 3 && x[mu] == L - 1) ? -1.0 : 1.0;
            /* backward neighbour x - mu */
            long sb = s + ((x[mu] == 0) ? (long)(L - 1) * stride : -stride);
            double bb = (mu == 3 && x[mu] == 0) ? -1.0 : 1.0;
            const cplx *Uf = U + (s * 4 + mu) * 9;   /* U_mu(x)      */
            const cplx *Ub = U + (sb * 4 + mu) * 9;  /* U_mu(x - mu) */
            cplx cf[4][3], cb[4][3]; /* colour-multiplied neighbours */
            for (int a = 0; a < 4; ++a)
                for (int c = 0; c < 3; ++c) {
                    cplx f = 0, b = 0;
                    for (int k = 0; k < 3; ++k) {
                        f += Uf[3 * c + k] * psi[(sf * 4 + a) * 3 + k];
                        b += conj(Ub[3 * k + c]) * psi[(sb * 4 + a) * 3 + k];
                    }
                    cf[a][c] = bf * f;
                    cb[a][c] = bb * b;
                }
            for (int a = 0; a < 4; ++a)
                for (int c = 0; c < 3; ++c) {
                    cplx acc = cf[a][c] + cb[a][c]; /* the "1" of (1 -+ gamma_mu) */
                    for (int b = 0; b < 4; ++b) acc += GAMMA[mu][a][b] * (cb[b][c] - cf[b][c]);
                    hop[a][c] += acc;
                }
            stride *= L;
        }
        for (int a = 0; a < 4; ++a)
            for (int c = 0; c < 3; ++c) out[(s * 4 + a) * 3 + c] = 4.0 * psi[(s * 4 + a) * 3 + c] - 0.5 * hop[a][c];
    }
}

/* out = K^ psi = gamma5 (D_W - m_w) psi / lambda_max */
void orc_khat(const int *dims, const cplx *U, double m_w, double lambda_max, const cplx *psi, cplx *out) {
    const long V = vol(dims);
    orc_dw(dims, U, psi, out);
#pragma omp parallel for schedule(static)
    for (long s = 0; s < V; ++s)
        for (int a = 0; a < 4; ++a)
            for (int c = 0; c < 3; ++c) {
                long i = (s * 4 + a) * 3 + c;
                out[i] = GAMMA5[a] * (out[i] - m_w * psi[i]) / lambda_max;
            }
}

/* s = sum_{m=0}^{N} alpha_m T_m(K^) psi;  t_0 = psi, t_1 = K^ psi, t_{m+1} = 2 K^ t_m - t_{m-1} */
void orc_cheb(const int *dims, const cplx *U, double m_w, double lambda_max, int N, const double *alpha,
              const cplx *psi, cplx *out) {
    const long n = vol(dims) * 12;
    cplx *tm1 = malloc(sizeof(cplx) * n), *tm = malloc(sizeof(cplx) * n), *tp = malloc(sizeof(cplx) * n);
    memcpy(tm1, psi, sizeof(cplx) * n);
    for (long i = 0; i < n; ++i) out[i] = alpha[0] * psi[i];
    if (N >= 1) {
        orc_khat(dims, U, m_w, lambda_max, psi, tm);
        for (long i = 0; i < n; ++i) out[i] += alpha[1] * tm[i];
    }
    for (int m = 1; m < N; ++m) {
        orc_khat(dims, U, m_w, lambda_max, tm, tp);
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) {
            tp[i] = 2.0 * tp[i] - tm1[i];
            out[i] += alpha[m + 1] * tp[i];
        }
        cplx *t = tm1; tm1 = tm; tm = tp; tp = t;
    }
    free(tm1); free(tm); free(tp);
}

/* Clenshaw: b_k = alpha_k psi + 2 K^ b_{k+1} - b_{k+2} (k = N..1), s = alpha_0 psi + K^ b_1 - b_2.  Self-check. */
void orc_clenshaw(const int *dims, const cplx *U, double m_w, double lambda_max, int N, const double *alpha,
                  const cplx *psi, cplx *out) {
    const long n = vol(dims) * 12;
    cplx *b1 = calloc(n, sizeof(cplx)), *b2 = calloc(n, sizeof(cplx)), *w = malloc(sizeof(cplx) * n);
    for (int k = N; k >= 1; --k) {
        orc_khat(dims, U, m_w, lambda_max, b1, w);
        for (long i = 0; i < n; ++i) w[i] = alpha[k] * psi[i] + 2.0 * w[i] - b2[i];
        cplx *t = b2; b2 = b1; b1 = w; w = t;
    }
    orc_khat(dims, U, m_w, lambda_max, b1, w);
    for (long i = 0; i < n; ++i) out[i] = alpha[0] * psi[i] + w[i] - b2[i];
    free(b1); free(b2); free(w);
}

/* p(x) = sum_m alpha_m T_m(x) for a real scalar, same forward recurrence */
double orc_cheb_scalar(int N, const double *alpha, double x) {
    double tm1 = 1.0, tm = x, p = alpha[0];
    if (N >= 1) p += alpha[1] * x;
    for (int m = 1; m < N; ++m) {
        double tp = 2.0 * x * tm - tm1;
        p += alpha[m + 1] * tp;
        tm1 = tm; tm = tp;
    }
    return p;
}

/* s += sum_i phi_i (phi_i^dag psi) [ sign(lambda_i) - sum_m alpha_m T_m(lambda_i / lambda_max) ] */
void orc_deflate(const int *dims, double lambda_max, int N, const double *alpha, int nev, const cplx *phi,
                 const double *lambda, const cplx *psi, cplx *s) {
    const long n = vol(dims) * 12;
    for (int i = 0; i < nev; ++i) {
        const cplx *ph = phi + (long)i * n;
        cplx c = 0;
        for (long j = 0; j < n; ++j) c += conj(ph[j]) * psi[j];
        double sg = (lambda[i] > 0) - (lambda[i] < 0);
        cplx w = c * (sg - orc_cheb_scalar(N, alpha, lambda[i] / lambda_max));
        for (long j = 0; j < n; ++j) s[j] += w * ph[j];
    }
}

void orc_sign(const int *dims, const cplx *U, double m_w, double lambda_max, int N, const double *alpha, int nev,
              const cplx *phi, const double *lambda, const cplx *psi, cplx *out) {
    orc_cheb(dims, U, m_w, lambda_max, N, alpha, psi, out);
    if (nev > 0) orc_deflate(dims, lambda_max, N, alpha, nev, phi, lambda, psi, out);
}

/* dagger = 0:  y = 1/2 [ (1+mu) psi + (1-mu) gamma5 sign(K) psi ]          (eq. 2.1)
 * dagger = 1:  y = 1/2 [ (1+mu) psi + (1-mu) sign(K) gamma5 psi ]          (adjoint, sign(K) Hermitian) */
void orc_overlap(const int *dims, const cplx *U, double m_w, double lambda_max, int N, const double *alpha, int nev,
                 const cplx *phi, const double *lambda, double mu, int dagger, const cplx *psi, cplx *out) {
    const long V = vol(dims), n = V * 12;
    cplx *in = malloc(sizeof(cplx) * n), *sg = malloc(sizeof(cplx) * n);
    for (long s = 0; s < V; ++s)
        for (int a = 0; a < 4; ++a)
            for (int c = 0; c < 3; ++c) {
                long i = (s * 4 + a) * 3 + c;
                in[i] = dagger ? GAMMA5[a] * psi[i] : psi[i];
            }
    orc_sign(dims, U, m_w, lambda_max, N, alpha, nev, phi, lambda, in, sg);
    for (long s = 0; s < V; ++s)
        for (int a = 0; a < 4; ++a)
            for (int c = 0; c < 3; ++c) {
                long i = (s * 4 + a) * 3 + c;
                cplx g = dagger ? sg[i] : GAMMA5[a] * sg[i];
                out[i] = 0.5 * ((1.0 + mu) * psi[i] + (1.0 - mu) * g);
            }
    free(in); free(sg);
}

static double norm2(long n, const cplx *a) {
    double r = 0;
    for (long i = 0; i < n; ++i) r += creal(a[i]) * creal(a[i]) + cimag(a[i]) * cimag(a[i]);
    return r;
}

/* CG on A = D^dag D, x0 = 0, stop when ||r_k|| <= tol ||b|| (recursive residual) or after maxiter iterations
 * (tol <= 0: run exactly maxiter iterations).  Returns iterations; *true_relres = ||b - A x|| / ||b||. */
int orc_cg(const int *dims, const cplx *U, double m_w, double lambda_max, int N, const double *alpha, int nev,
           const cplx *phi, const double *lambda, double mu, const cplx *b, cplx *x, double tol, int maxiter,
           double *true_relres) {
    const long n = vol(dims) * 12;
    cplx *r = malloc(sizeof(cplx) * n), *p = malloc(sizeof(cplx) * n), *q = malloc(sizeof(cplx) * n),
         *Ap = malloc(sizeof(cplx) * n);
    memset(x, 0, sizeof(cplx) * n);
    memcpy(r, b, sizeof(cplx) * n);
    memcpy(p, b, sizeof(cplx) * n);
    const double bb = norm2(n, b);
    double rr = bb;
    int it = 0;
    while (it < maxiter && !(tol > 0 && sqrt(rr) <= tol * sqrt(bb))) {
        orc_overlap(dims, U, m_w, lambda_max, N, alpha, nev, phi, lambda, mu, 0, p, q);
        orc_overlap(dims, U, m_w, lambda_max, N, alpha, nev, phi, lambda, mu, 1, q, Ap);
        cplx pAp = 0;
        for (long i = 0; i < n; ++i) pAp += conj(p[i]) * Ap[i];
        const double a = rr / creal(pAp);
        for (long i = 0; i < n; ++i) { x[i] += a * p[i]; r[i] -= a * Ap[i]; }
        const double rr_new = norm2(n, r);
        const double beta = rr_new / rr;
        for (long i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
        rr = rr_new;
        ++it;
    }
    orc_overlap(dims, U, m_w, lambda_max, N, alpha, nev, phi, lambda, mu, 0, x, q);
    orc_overlap(dims, U, m_w, lambda_max, N, alpha, nev, phi, lambda, mu, 1, q, Ap);
    for (long i = 0; i < n; ++i) Ap[i] = b[i] - Ap[i];
    *true_relres = sqrt(norm2(n, Ap) / bb);
    free(r); free(p); free(q); free(Ap);
    return it;
}

/* Chiral-sector operator (reading R23).  With P_c = (1 + c gamma5)/2, c = +1 or -1, and s = sign(K):
 *   D^dag D = 1/4 [ (1+mu)^2 + (1-mu)^2 s^2 + (1-mu^2) (gamma5 s + s gamma5) ]           from eq. 2.1 and its adjoint,
 *   s^2 = 1  =>  D^dag D = 1/2 (1+mu^2) + 1/4 (1-mu^2) {gamma5, s},  which commutes with gamma5, and
 *   P_c D^dag D P_c = [ 1/2 (1+mu^2) + c/2 (1-mu^2) P_c s P_c ] P_c .
 * This routine applies  A_c v = 1/2 (1+mu^2) P_c v + c/2 (1-mu^2) P_c s P_c v   with ONE evaluation of eq. 2.3
 * (the full D^dag D needs two).  For the polynomial s of eq. 2.3, A_c differs from P_c D^dag D P_c by
 * 1/4 (1-mu)^2 P_c (s^2 - 1) P_c.  `v` need not be chiral: it is projected first. */
void orc_chiral_op(const int *dims, const cplx *U, double m_w, double lambda_max, int N, const double *alpha, int nev,
                   const cplx *phi, const double *lambda, double mu, int chirality, const cplx *v, cplx *out) {
    const long V = vol(dims), n = V * 12;
    const double c = chirality >= 0 ? 1.0 : -1.0;
    cplx *pv = malloc(sizeof(cplx) * n), *sg = malloc(sizeof(cplx) * n);
    for (long s = 0; s < V; ++s)
        for (int a = 0; a < 4; ++a)
            for (int k = 0; k < 3; ++k) {
                long i = (s * 4 + a) * 3 + k;
                pv[i] = 0.5 * (1.0 + c * GAMMA5[a]) * v[i];          /* P_c v */
            }
    orc_sign(dims, U, m_w, lambda_max, N, alpha, nev, phi, lambda, pv, sg);
    for (long s = 0; s < V; ++s)
        for (int a = 0; a < 4; ++a)
            for (int k = 0; k < 3; ++k) {
                long i = (s * 4 + a) * 3 + k;
                cplx ps = 0.5 * (1.0 + c * GAMMA5[a]) * sg[i];       /* P_c s P_c v */
                out[i] = 0.5 * (1.0 + mu * mu) * pv[i] + 0.5 * c * (1.0 - mu * mu) * ps;
            }
    free(pv); free(sg);
}

/* CG on A_c x = P_c b in the chirality-c subspace, x0 = 0; same stopping rule as orc_cg.  Returns iterations;
 * *true_relres = || P_c b - A_c x || / || P_c b ||.  (P_c b = 0: x = 0, zero iterations.) */
int orc_cg_chiral(const int *dims, const cplx *U, double m_w, double lambda_max, int N, const double *alpha, int nev,
                  const cplx *phi, const double *lambda, double mu, int chirality, const cplx *b, cplx *x, double tol,
                  int maxiter, double *true_relres) {
    const long V = vol(dims), n = V * 12;
    const double c = chirality >= 0 ? 1.0 : -1.0;
    cplx *bc = malloc(sizeof(cplx) * n), *r = malloc(sizeof(cplx) * n), *p = malloc(sizeof(cplx) * n),
         *Ap = malloc(sizeof(cplx) * n);
    for (long s = 0; s < V; ++s)
        for (int a = 0; a < 4; ++a)
            for (int k = 0; k < 3; ++k) {
                long i = (s * 4 + a) * 3 + k;
                bc[i] = 0.5 * (1.0 + c * GAMMA5[a]) * b[i];
            }
    memset(x, 0, sizeof(cplx) * n);
    memcpy(r, bc, sizeof(cplx) * n);
    memcpy(p, bc, sizeof(cplx) * n);
    const double bb = norm2(n, bc);
    double rr = bb;
    int it = 0;
    while (bb > 0 && it < maxiter && !(tol > 0 && sqrt(rr) <= tol * sqrt(bb))) {
        orc_chiral_op(dims, U, m_w, lambda_max, N, alpha, nev, phi, lambda, mu, chirality, p, Ap);
        cplx pAp = 0;
        for (long i = 0; i < n; ++i) pAp += conj(p[i]) * Ap[i];
        const double a = rr / creal(pAp);
        for (long i = 0; i < n; ++i) { x[i] += a * p[i]; r[i] -= a * Ap[i]; }
        const double rr_new = norm2(n, r);
        const double beta = rr_new / rr;
        for (long i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
        rr = rr_new;
        ++it;
    }
    orc_chiral_op(dims, U, m_w, lambda_max, N, alpha, nev, phi, lambda, mu, chirality, x, Ap);
    for (long i = 0; i < n; ++i) Ap[i] = bc[i] - Ap[i];
    *true_relres = bb > 0 ? sqrt(norm2(n, Ap) / bb) : 0.0;
    free(bc); free(r); free(p); free(Ap);
    return it;
}
