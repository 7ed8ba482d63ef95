// ovl_dense.h -- small dense complex Hermitian linear algebra on the host (m <= ~128) for the Rayleigh-Ritz step of the
// eigensolver: Cholesky, triangular solves, cyclic Jacobi.  Plain C++, column-major-free: matrices are row-major
// std::vector<std::complex<double>> of size m*m, element (i, j) at i*m + j.
#pragma once
#include <algorithm>
#include <cmath>
#include <complex>
#include <vector>

namespace ovl {
namespace dense {

using cd = std::complex<double>;
using mat = std::vector<cd>;

// G = L L^dag, L lower triangular (returned in the lower triangle of a fresh matrix, upper = 0). false if G is not
// numerically positive definite.
inline bool cholesky(const mat &G, int m, mat &L) {
    L.assign((size_t)m * m, cd(0, 0));
    for (int j = 0; j < m; ++j) {
        double d = G[(size_t)j * m + j].real();
        for (int k = 0; k < j; ++k) d -= std::norm(L[(size_t)j * m + k]);
        if (!(d > 0)) return false;
        const double ljj = std::sqrt(d);
        L[(size_t)j * m + j] = ljj;
        for (int i = j + 1; i < m; ++i) {
            cd s = G[(size_t)i * m + j];
            for (int k = 0; k < j; ++k) s -= L[(size_t)i * m + k] * std::conj(L[(size_t)j * m + k]);
            L[(size_t)i * m + j] = s / ljj;
        }
    }
    return true;
}
// B <- L^{-1} B   (forward substitution on every column of the m x m matrix B)
inline void solve_lower(const mat &L, int m, mat &B) {
    for (int c = 0; c < m; ++c)
        for (int i = 0; i < m; ++i) {
            cd s = B[(size_t)i * m + c];
            for (int k = 0; k < i; ++k) s -= L[(size_t)i * m + k] * B[(size_t)k * m + c];
            B[(size_t)i * m + c] = s / L[(size_t)i * m + i];
        }
}
// B <- L^{-dag} B  (back substitution with the upper triangular L^dag)
inline void solve_lower_dag(const mat &L, int m, mat &B) {
    for (int c = 0; c < m; ++c)
        for (int i = m - 1; i >= 0; --i) {
            cd s = B[(size_t)i * m + c];
            for (int k = i + 1; k < m; ++k) s -= std::conj(L[(size_t)k * m + i]) * B[(size_t)k * m + c];
            B[(size_t)i * m + c] = s / L[(size_t)i * m + i];
        }
}
inline mat dagger(const mat &A, int m) {
    mat R((size_t)m * m);
    for (int i = 0; i < m; ++i)
        for (int j = 0; j < m; ++j) R[(size_t)j * m + i] = std::conj(A[(size_t)i * m + j]);
    return R;
}

// Hermitian M = Y diag(w) Y^dag by cyclic Jacobi rotations; M is destroyed, columns of Y are the eigenvectors.
// Rotation in the (p, q) plane: U = [[c, s e^{i phi}], [-s e^{-i phi}, c]], phi = arg M_pq,
// t = s/c = sign(tau) / (|tau| + sqrt(1 + tau^2)), tau = (M_qq - M_pp) / (2 |M_pq|).
inline void jacobi_eigh(mat &M, int m, std::vector<double> &w, mat &Y) {
    Y.assign((size_t)m * m, cd(0, 0));
    for (int i = 0; i < m; ++i) Y[(size_t)i * m + i] = 1.0;
    double scale = 0;
    for (const cd &x : M) scale = std::max(scale, std::abs(x));
    for (int sweep = 0; sweep < 60; ++sweep) {
        double off = 0;
        for (int p = 0; p < m; ++p)
            for (int q = p + 1; q < m; ++q) off = std::max(off, std::abs(M[(size_t)p * m + q]));
        if (off <= 1e-15 * scale) break;
        for (int p = 0; p < m; ++p)
            for (int q = p + 1; q < m; ++q) {
                const cd g = M[(size_t)p * m + q];
                const double ag = std::abs(g);
                if (ag <= 1e-300 || ag <= 1e-17 * scale) continue;
                const cd ph = g / ag;  // e^{i phi}
                const double tau = (M[(size_t)q * m + q].real() - M[(size_t)p * m + p].real()) / (2.0 * ag);
                const double t = (tau >= 0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
                const double c = 1.0 / std::sqrt(1.0 + t * t), s = t * c;
                const cd se = s * ph, sec = s * std::conj(ph);
                for (int k = 0; k < m; ++k) {  // M <- M U, Y <- Y U
                    const cd mp = M[(size_t)k * m + p], mq = M[(size_t)k * m + q];
                    M[(size_t)k * m + p] = c * mp - sec * mq;
                    M[(size_t)k * m + q] = se * mp + c * mq;
                    const cd yp = Y[(size_t)k * m + p], yq = Y[(size_t)k * m + q];
                    Y[(size_t)k * m + p] = c * yp - sec * yq;
                    Y[(size_t)k * m + q] = se * yp + c * yq;
                }
                for (int k = 0; k < m; ++k) {  // M <- U^dag M
                    const cd mp = M[(size_t)p * m + k], mq = M[(size_t)q * m + k];
                    M[(size_t)p * m + k] = c * mp - se * mq;
                    M[(size_t)q * m + k] = sec * mp + c * mq;
                }
                M[(size_t)p * m + q] = 0.0;
                M[(size_t)q * m + p] = 0.0;
            }
    }
    w.resize(m);
    for (int i = 0; i < m; ++i) w[i] = M[(size_t)i * m + i].real();
}

// Generalised Hermitian problem H x = theta G x (G positive definite): X with X^dag G X = 1, X^dag H X = diag(theta).
// Returns false if G is not positive definite.
inline bool geneig(const mat &H, const mat &G, int m, std::vector<double> &theta, mat &X) {
    mat L;
    if (!cholesky(G, m, L)) return false;
    mat Z = H;
    solve_lower(L, m, Z);       // Z = L^{-1} H
    mat Zd = dagger(Z, m);
    solve_lower(L, m, Zd);      // L^{-1} Z^dag = (Z L^{-dag})^dag
    mat M = dagger(Zd, m);      // M = L^{-1} H L^{-dag}
    for (int i = 0; i < m; ++i)  // symmetrise against rounding
        for (int j = i; j < m; ++j) {
            const cd a = 0.5 * (M[(size_t)i * m + j] + std::conj(M[(size_t)j * m + i]));
            M[(size_t)i * m + j] = a;
            M[(size_t)j * m + i] = std::conj(a);
        }
    jacobi_eigh(M, m, theta, X);
    solve_lower_dag(L, m, X);   // X = L^{-dag} Y
    return true;
}

}  // namespace dense
}  // namespace ovl
