// ovl_eig.cuh -- kernels of the GPU eigensolver for the deflation space of eq. 2.3 (the paper
// computes the lowest eigenpairs of K with "a polynomial preconditioned implicitly restarted Lanczos routine",
// here a Chebyshev-filtered block subspace iteration, which needs only the fused stencil kernel, two
// tall-skinny products and a small dense eigenproblem on the host).  fp64 only.  All reductions use fixed trees.
#pragma once
#include "ovl_blas.cuh"

namespace ovl {

// v[e] = uniform in [-1/2, 1/2) from a counter hash (start block of the subspace iteration)
__global__ void k_fill_random(size_t n, unsigned long long seed, double2 *__restrict__ v) {
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        double r[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            unsigned long long z = (2 * e + h + 1) * 0x9E3779B97F4A7C15ull + seed * 0xD1B54A32D192ED03ull;
            z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull; z ^= z >> 27; z *= 0x94D049BB133111EBull; z ^= z >> 31;
            r[h] = (double)(z >> 11) * (1.0 / 9007199254740992.0) - 0.5;
        }
        v[e] = make_double2(r[0], r[1]);
    }
}

// field r (blockIdx.y) *= s[r]
__global__ void k_scale_batched(size_t n, const double *__restrict__ s, double2 *__restrict__ v) {
    v += blockIdx.y * n;
    const double f = s[blockIdx.y];
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        double2 x = v[e];
        x.x *= f; x.y *= f;
        v[e] = x;
    }
}

// Tall-skinny product, J columns at a time:  C[i][jj] = a_i^dag b_{j0+jj},  i < m, jj < J (unused columns: pass nj < J).
// A block owns GRAM_EPT * BLAS_THREADS consecutive elements: its chunk of the J columns stays in registers while every
// row a_i is streamed once.  partial[((i * J + jj) * nslot) + slot], slot = block * 8 + warp (warp shuffle only).
constexpr int GRAM_J = 6;
constexpr int GRAM_EPT = 2;
__global__ void __launch_bounds__(BLAS_THREADS)
k_gram_block(size_t n, int m, int nj, const double2 *__restrict__ A, const double2 *__restrict__ B, double2 *__restrict__ partial) {
    const size_t base = (size_t)blockIdx.x * (BLAS_THREADS * GRAM_EPT) + threadIdx.x;
    const int nslot = gridDim.x * (BLAS_THREADS / 32);
    const int slot = blockIdx.x * (BLAS_THREADS / 32) + (threadIdx.x >> 5);
    double2 b[GRAM_J][GRAM_EPT];
#pragma unroll
    for (int jj = 0; jj < GRAM_J; ++jj)
#pragma unroll
        for (int q = 0; q < GRAM_EPT; ++q) {
            const size_t e = base + (size_t)q * BLAS_THREADS;
            b[jj][q] = (jj < nj && e < n) ? B[(size_t)jj * n + e] : make_double2(0.0, 0.0);
        }
    for (int i = 0; i < m; ++i) {
        double2 a[GRAM_EPT];
#pragma unroll
        for (int q = 0; q < GRAM_EPT; ++q) {
            const size_t e = base + (size_t)q * BLAS_THREADS;
            a[q] = e < n ? __ldg(A + (size_t)i * n + e) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int jj = 0; jj < GRAM_J; ++jj) {
            double re = 0, im = 0;
#pragma unroll
            for (int q = 0; q < GRAM_EPT; ++q) {
                re += a[q].x * b[jj][q].x + a[q].y * b[jj][q].y;
                im += a[q].x * b[jj][q].y - a[q].y * b[jj][q].x;
            }
            re = warp_sum(re);
            im = warp_sum(im);
            if ((threadIdx.x & 31) == 0) partial[((size_t)i * GRAM_J + jj) * nslot + slot] = make_double2(re, im);
        }
    }
}
// C[i * J + jj] = sum over slots (one block per entry)
__global__ void __launch_bounds__(BLAS_THREADS) k_gram_final(int nslot, const double2 *__restrict__ partial, double2 *__restrict__ C) {
    __shared__ double sm[2 * (BLAS_THREADS / 32)];
    const double2 *p = partial + (size_t)blockIdx.x * nslot;
    double re = 0, im = 0;
    for (int s = threadIdx.x; s < nslot; s += blockDim.x) { re += p[s].x; im += p[s].y; }
    const double r0 = block_sum(re, sm);
    const double r1 = block_sum(im, sm + BLAS_THREADS / 32);
    if (threadIdx.x == 0) C[blockIdx.x] = make_double2(r0, r1);
}

// Basis rotation, JO output vectors at a time:  out_o = sum_{j < m} X[j * ldx + o0 + o] v_j,  o < no <= ROT_JO
constexpr int ROT_JO = 8;
__global__ void __launch_bounds__(BLAS_THREADS)
k_rotate_block(size_t n, int m, int no, int ldx, const double2 *__restrict__ X, const double2 *__restrict__ V, double2 *__restrict__ out) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    double2 acc[ROT_JO];
#pragma unroll
    for (int o = 0; o < ROT_JO; ++o) acc[o] = make_double2(0.0, 0.0);
    for (int j = 0; j < m; ++j) {
        const double2 v = __ldg(V + (size_t)j * n + e);
#pragma unroll
        for (int o = 0; o < ROT_JO; ++o) {
            if (o < no) {
                const double2 x = __ldg(X + (size_t)j * ldx + o);
                acc[o].x = fma(x.x, v.x, fma(-x.y, v.y, acc[o].x));
                acc[o].y = fma(x.x, v.y, fma(x.y, v.x, acc[o].y));
            }
        }
    }
#pragma unroll
    for (int o = 0; o < ROT_JO; ++o)
        if (o < no) out[(size_t)o * n + e] = acc[o];
}

// partial[b] of || w_r - theta[r] v_r ||^2  (blockIdx.y = r)
__global__ void __launch_bounds__(BLAS_THREADS)
k_resid_norm2(size_t n, const double *__restrict__ theta, const double2 *__restrict__ W, const double2 *__restrict__ V, double *__restrict__ partial) {
    __shared__ double sm[BLAS_THREADS / 32];
    W += blockIdx.y * n; V += blockIdx.y * n; partial += blockIdx.y * gridDim.x;
    const double th = theta[blockIdx.y];
    double r = 0;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const double2 w = W[e], v = V[e];
        const double dx = w.x - th * v.x, dy = w.y - th * v.y;
        r += dx * dx + dy * dy;
    }
    r = block_sum(r, sm);
    if (threadIdx.x == 0) partial[blockIdx.x] = r;
}
// out[r] = sum_b partial[r][b]  (one block per r)
__global__ void __launch_bounds__(BLAS_THREADS) k_sum_partials(int nblk, const double *__restrict__ partial, double *__restrict__ out) {
    __shared__ double sm[BLAS_THREADS / 32];
    double r = 0;
    for (int b = threadIdx.x; b < nblk; b += blockDim.x) r += partial[(size_t)blockIdx.x * nblk + b];
    r = block_sum(r, sm);
    if (threadIdx.x == 0) out[blockIdx.x] = r;
}

}  // namespace ovl
