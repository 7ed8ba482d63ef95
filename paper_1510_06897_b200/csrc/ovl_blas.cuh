// ovl_blas.cuh -- layout import/export (a1), deflation projection / update (a5-a8), CG vector kernels (a9).
// All reductions accumulate in fp64 with a fixed tree (thread-serial, warp shuffle, smem across warps, then a
// single-block second stage), so results are bit-identical run to run (no float atomics).
#pragma once
#include "ovl_types.cuh"

namespace ovl {

constexpr int BLAS_THREADS = 256;

// ---------------------------------------------------------------- a1: canonical AoS <-> native SoA
// canonical spinor [V][12] complex (TS = double or float) -> native planes [12][V] of T
template <typename TS, typename T>
__global__ void k_import_spinor(int V, const cx<TS> *__restrict__ src, cx<T> *__restrict__ dst) {
    const size_t n = (size_t)12 * V;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int k = (int)(e / V);
        const int s = (int)(e - (size_t)k * V);
        const cx<TS> v = src[(size_t)s * 12 + k];
        dst[e] = mk<T>((T)v.x, (T)v.y);
    }
}
template <typename T, typename TD>
__global__ void k_export_spinor(int V, const cx<T> *__restrict__ src, cx<TD> *__restrict__ dst) {
    const size_t n = (size_t)12 * V;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int s = (int)(e / 12);
        const int k = (int)(e - (size_t)s * 12);
        const cx<T> v = src[(size_t)k * V + s];
        dst[e] = mk<TD>((TD)v.x, (TD)v.y);
    }
}
// canonical links [V][4][3][3] complex128 -> native [mu][row < NROW][col][V] of T (round to nearest for fp32)
template <typename T>
__global__ void k_import_links(int V, int nrow, const double2 *__restrict__ src, cx<T> *__restrict__ dst) {
    const size_t n = (size_t)4 * nrow * 3 * V;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int pl = (int)(e / V);  // (mu*nrow + r)*3 + c
        const int s = (int)(e - (size_t)pl * V);
        const int c = pl % 3, r = (pl / 3) % nrow, mu = pl / (3 * nrow);
        const double2 v = src[((size_t)s * 4 + mu) * 9 + r * 3 + c];
        dst[e] = mk<T>((T)v.x, (T)v.y);
    }
}

// ---------------------------------------------------------------- block reduction of NV fp64 values (fixed tree)
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// returns the block total in thread 0 (other threads: garbage). smem: BLAS_THREADS/32 doubles.
__device__ __forceinline__ double block_sum(double v, double *sm) {
    v = warp_sum(v);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sm[w] = v;
    __syncthreads();
    double r = 0;
    if (threadIdx.x == 0)
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) r += sm[i];
    return r;
}

// ---------------------------------------------------------------- a5: c_{r,i} = phi_i^dag psi_r, i < nev, r < nrhs
// grid = (nblk, ceil(nrhs / DEFL_RB)); block b owns the elements [b*CH, (b+1)*CH) of the flat 12V-complex field for ALL i
// and for a group of DEFL_RB right-hand sides: the psi chunks of the group stay in registers and every phi_i is streamed
// ONCE per group (not once per right-hand side).  partial[((r * nev) + i) * nblk + b]  (complex fp64).
// The reduction tree per (r, i) -- thread-serial over the chunk, warp shuffle, warps 0..7 in order -- does not depend on
// the group size, so a right-hand side gets bit-identical coefficients whether it is projected alone or in a batch.
constexpr int PROJ_EPT = 4;   // elements per thread
constexpr int PROJ_IB = 4;    // eigenvectors per pass of the loop: PROJ_IB * PROJ_EPT loads in flight per thread, one barrier
constexpr int DEFL_RB = 4;    // right-hand sides per group
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS, 2)
k_project(size_t n, int nev, int nrhs, const cx<T> *__restrict__ phi, const cx<T> *__restrict__ psi, double2 *__restrict__ partial) {
    __shared__ double sm[2][PROJ_IB][BLAS_THREADS / 32][2 * DEFL_RB];
    const size_t base = (size_t)blockIdx.x * (BLAS_THREADS * PROJ_EPT) + threadIdx.x;
    const int r0 = blockIdx.y * DEFL_RB;
    const int nr = min(DEFL_RB, nrhs - r0);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    cx<T> p[DEFL_RB][PROJ_EPT];
#pragma unroll
    for (int r = 0; r < DEFL_RB; ++r)
#pragma unroll
        for (int j = 0; j < PROJ_EPT; ++j) {
            const size_t e = base + (size_t)j * BLAS_THREADS;
            p[r][j] = (r < nr && e < n) ? psi[(size_t)(r0 + r) * n + e] : mk<T>(0, 0);
        }
    for (int i0 = 0, pass = 0; i0 < nev; i0 += PROJ_IB, ++pass) {
        // all loads of the pass first (the eigenvector stream is the whole traffic of this kernel) ...
        cx<T> f[PROJ_IB][PROJ_EPT];
#pragma unroll
        for (int q = 0; q < PROJ_IB; ++q) {
            const cx<T> *ph = phi + (size_t)min(i0 + q, nev - 1) * n;
#pragma unroll
            for (int j = 0; j < PROJ_EPT; ++j) {
                const size_t e = base + (size_t)j * BLAS_THREADS;
                f[q][j] = e < n ? ldg(ph + e) : mk<T>(0, 0);
            }
        }
        // ... then, per eigenvector, exactly the tree of the one-vector-per-pass version: thread-serial over j, warp
        // shuffle, warps in order
#pragma unroll
        for (int q = 0; q < PROJ_IB; ++q) {
            double (*buf)[2 * DEFL_RB] = sm[pass & 1][q];
#pragma unroll
            for (int r = 0; r < DEFL_RB; ++r) {
                if (r < nr) {
                    double re = 0, im = 0;
#pragma unroll
                    for (int j = 0; j < PROJ_EPT; ++j) {
                        if (base + (size_t)j * BLAS_THREADS < n) {
                            re += (double)f[q][j].x * (double)p[r][j].x + (double)f[q][j].y * (double)p[r][j].y;
                            im += (double)f[q][j].x * (double)p[r][j].y - (double)f[q][j].y * (double)p[r][j].x;
                        }
                    }
                    re = warp_sum(re);
                    im = warp_sum(im);
                    if (l == 0) { buf[w][2 * r] = re; buf[w][2 * r + 1] = im; }
                }
            }
        }
        __syncthreads();  // (the other half of sm is rewritten only after the next barrier)
        if (threadIdx.x < nr * PROJ_IB) {
            const int q = threadIdx.x / nr, r = threadIdx.x - q * nr;
            if (i0 + q < nev) {
                double (*buf)[2 * DEFL_RB] = sm[pass & 1][q];
                double re = 0, im = 0;
                for (int k = 0; k < BLAS_THREADS / 32; ++k) { re += buf[k][2 * r]; im += buf[k][2 * r + 1]; }
                partial[((size_t)(r0 + r) * nev + i0 + q) * gridDim.x + blockIdx.x] = make_double2(re, im);
            }
        }
    }
}
// second stage: one block per (i, r); w[r * wstride + i] = coef_i * sum_b partial[r][i][b]   (a6: coef_i = sign(lambda_i) - p(lambda^_i))
__global__ void __launch_bounds__(BLAS_THREADS)
k_project_final(int nblk, int nev, int wstride, const double2 *__restrict__ partial, const double *__restrict__ coef, double2 *__restrict__ w) {
    __shared__ double sm[2 * (BLAS_THREADS / 32)];
    const int i = blockIdx.x, r = blockIdx.y;
    const double2 *p = partial + ((size_t)r * nev + i) * nblk;
    double re = 0, im = 0;
    for (int b = threadIdx.x; b < nblk; b += blockDim.x) {
        const double2 v = p[b];
        re += v.x; im += v.y;
    }
    const double q0 = block_sum(re, sm);
    const double q1 = block_sum(im, sm + BLAS_THREADS / 32);
    if (threadIdx.x == 0) w[(size_t)r * wstride + i] = make_double2(coef[i] * q0, coef[i] * q1);
}

// ---------------------------------------------------------------- a7 + a8: s_r = acc_r + sum_i w_{r,i} phi_i;  out_r = a psi_r + b [gamma5] s_r
// flat element e = k*V + s: gamma5 is -1 for e >= 6V (planes of spin 2,3).  grid.y = groups of DEFL_RB right-hand sides:
// every phi_i[e] is loaded once per group.  The deflation sum is carried in fp64 and added to the polynomial part once.
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS)
k_deflate_assemble(size_t n, size_t n_upper, int nev, int nrhs, int wstride, const cx<T> *__restrict__ phi, const double2 *__restrict__ w,
                   const cx<T> *__restrict__ psi, const cx<T> *__restrict__ acc, T a, T b, int g5, int chir, cx<T> *__restrict__ out) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    // chir = +1 / -1: the result is projected with P_c = (1 + c gamma5)/2, i.e. the planes of the other chirality are zero
    const bool dead = (chir > 0 && e >= n_upper) || (chir < 0 && e < n_upper);
    const int r0 = blockIdx.y * DEFL_RB;
    const int nr = min(DEFL_RB, nrhs - r0);
    double re[DEFL_RB], im[DEFL_RB];
#pragma unroll
    for (int r = 0; r < DEFL_RB; ++r) re[r] = im[r] = 0.0;
    for (int i = 0; i < nev; ++i) {
        const cx<T> f = ldg(phi + (size_t)i * n + e);
#pragma unroll
        for (int r = 0; r < DEFL_RB; ++r) {
            if (r < nr) {
                const double2 wi = w[(size_t)(r0 + r) * wstride + i];
                re[r] += wi.x * (double)f.x - wi.y * (double)f.y;
                im[r] += wi.x * (double)f.y + wi.y * (double)f.x;
            }
        }
    }
#pragma unroll
    for (int r = 0; r < DEFL_RB; ++r) {
        if (r < nr) {
            const size_t o = (size_t)(r0 + r) * n + e;
            const cx<T> s0 = acc[o];
            T sx = (T)((double)s0.x + re[r]), sy = (T)((double)s0.y + im[r]);
            if (g5 && e >= n_upper) { sx = -sx; sy = -sy; }
            cx<T> q;
            if (a != T(0)) {
                const cx<T> pp = psi[o];
                q.x = fma(a, pp.x, b * sx);
                q.y = fma(a, pp.y, b * sy);
            } else {
                q.x = b * sx; q.y = b * sy;
            }
            if (dead) q = mk<T>(0, 0);
            out[o] = q;
        }
    }
}

// out = P_c in, P_c = (1 + c gamma5)/2: zero the planes of the other chirality (blockIdx.y = right-hand side)
template <typename T>
__global__ void k_chiral_project(size_t n, size_t n_upper, int chir, const cx<T> *__restrict__ in, cx<T> *__restrict__ out) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    in += blockIdx.y * n; out += blockIdx.y * n;
    const bool dead = (chir > 0 && e >= n_upper) || (chir < 0 && e < n_upper);
    out[e] = dead ? mk<T>(0, 0) : in[e];
}

// out = gamma5 in (only used to form the input of sign() in D^dag)
template <typename T>
__global__ void k_gamma5(size_t n, size_t n_upper, const cx<T> *__restrict__ in, cx<T> *__restrict__ out) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    in += blockIdx.y * n; out += blockIdx.y * n;  // blockIdx.y = right-hand side
    cx<T> v = in[e];
    if (e >= n_upper) { v.x = -v.x; v.y = -v.y; }
    out[e] = v;
}

// ---------------------------------------------------------------- a9: CG vector kernels (device-side scalars)
// sc[]: 0 rr, 1 pAp, 2 alpha, 3 beta, 4 bb, 5 frozen (system reached the tolerance: alpha = beta = 0 from then on)
// Batched over right-hand sides with blockIdx.y = rhs: field r starts at r*n, its scalars at r*SC_N, its partial sums
// at r*gridDim.x (gridDim.y = 1 is the single-system CG).
enum { SC_RR = 0, SC_PAP = 1, SC_ALPHA = 2, SC_BETA = 3, SC_BB = 4, SC_FROZEN = 5, SC_N = 8 };

// partial[b] = sum Re(conj(x) y) over the block's grid-stride elements
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS)
k_redot(size_t n, const cx<T> *__restrict__ x, const cx<T> *__restrict__ y, double *__restrict__ partial) {
    __shared__ double sm[BLAS_THREADS / 32];
    x += blockIdx.y * n; y += blockIdx.y * n; partial += blockIdx.y * gridDim.x;
    double r = 0;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const cx<T> a = x[e], b = y[e];
        r += (double)a.x * (double)b.x + (double)a.y * (double)b.y;
    }
    r = block_sum(r, sm);
    if (threadIdx.x == 0) partial[blockIdx.x] = r;
}
// x += alpha p, r -= alpha q, partial[b] = |r|^2      (alpha = sc[SC_ALPHA])
template <typename T>
__global__ void __launch_bounds__(BLAS_THREADS)
k_cg_update(size_t n, const double *__restrict__ sc, const cx<T> *__restrict__ p, const cx<T> *__restrict__ q,
            cx<T> *__restrict__ x, cx<T> *__restrict__ r, double *__restrict__ partial) {
    __shared__ double sm[BLAS_THREADS / 32];
    p += blockIdx.y * n; q += blockIdx.y * n; x += blockIdx.y * n; r += blockIdx.y * n;
    sc += blockIdx.y * SC_N; partial += blockIdx.y * gridDim.x;
    const T al = (T)sc[SC_ALPHA];
    double acc = 0;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const cx<T> pe = p[e], qe = q[e];
        cx<T> xe = x[e], re = r[e];
        xe.x = fma(al, pe.x, xe.x); xe.y = fma(al, pe.y, xe.y);
        re.x = fma(-al, qe.x, re.x); re.y = fma(-al, qe.y, re.y);
        x[e] = xe; r[e] = re;
        acc += (double)re.x * (double)re.x + (double)re.y * (double)re.y;
    }
    acc = block_sum(acc, sm);
    if (threadIdx.x == 0) partial[blockIdx.x] = acc;
}
// p = r + beta p   (beta = sc[SC_BETA])
template <typename T>
__global__ void k_xpay(size_t n, const double *__restrict__ sc, const cx<T> *__restrict__ r, cx<T> *__restrict__ p) {
    r += blockIdx.y * n; p += blockIdx.y * n; sc += blockIdx.y * SC_N;
    const T be = (T)sc[SC_BETA];
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const cx<T> re = r[e];
        cx<T> pe = p[e];
        pe.x = fma(be, pe.x, re.x); pe.y = fma(be, pe.y, re.y);
        p[e] = pe;
    }
}
// out = x - y  (true residual)
template <typename T>
__global__ void k_sub(size_t n, const cx<T> *__restrict__ x, const cx<T> *__restrict__ y, cx<T> *__restrict__ out) {
    x += blockIdx.y * n; y += blockIdx.y * n; out += blockIdx.y * n;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const cx<T> a = x[e], b = y[e];
        out[e] = mk<T>(a.x - b.x, a.y - b.y);
    }
}
// mixed precision (fp32 inner / fp64 outer defect correction): dst = scale * src across precisions, x += scale * e
template <typename TS, typename TD>
__global__ void k_convert_scaled(size_t n, double scale, const cx<TS> *__restrict__ src, cx<TD> *__restrict__ dst) {
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const cx<TS> v = src[e];
        dst[e] = mk<TD>((TD)(scale * (double)v.x), (TD)(scale * (double)v.y));
    }
}
template <typename TE, typename TX>
__global__ void k_axpy_mixed(size_t n, double scale, const cx<TE> *__restrict__ e_, cx<TX> *__restrict__ x) {
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const cx<TE> v = e_[e];
        cx<TX> xe = x[e];
        xe.x = (TX)((double)xe.x + scale * (double)v.x);
        xe.y = (TX)((double)xe.y + scale * (double)v.y);
        x[e] = xe;
    }
}

// second stage of the CG reductions, one block per system (blockIdx.x = rhs).  what: 0 -> bb = rr = sum (start),
// 1 -> pAp = sum, alpha = rr / pAp (0 if frozen), 2 -> rr_new = sum, beta = rr_new / rr, rr = rr_new; the system is
// frozen once rr_new <= tol2 * bb (tol2 = 0: never), 3 -> sc[SC_PAP] = sum (generic norm^2 read-out)
// the scalar recurrences of CG given a freshly reduced sum r (see k_cg_scalars)
__device__ __forceinline__ void cg_scalar_update(double *sc, double r, int what, double tol2) {
    const bool frozen = sc[SC_FROZEN] != 0.0;
    // a zero right-hand side is frozen from the start (x = 0 is its solution; 0/0 must not reach the vectors)
    if (what == 0) { sc[SC_BB] = r; sc[SC_RR] = r; sc[SC_FROZEN] = r == 0.0 ? 1.0 : 0.0; sc[SC_ALPHA] = 0.0; sc[SC_BETA] = 0.0; }
    else if (what == 1) { sc[SC_PAP] = r; sc[SC_ALPHA] = (frozen || r == 0.0) ? 0.0 : sc[SC_RR] / r; }
    else if (what == 2) {
        if (frozen) sc[SC_BETA] = 0.0;
        else {
            sc[SC_BETA] = r / sc[SC_RR];
            sc[SC_RR] = r;
            if (tol2 > 0.0 && r <= tol2 * sc[SC_BB]) { sc[SC_FROZEN] = 1.0; sc[SC_BETA] = 0.0; }
        }
    } else { sc[SC_PAP] = r; }
}
__global__ void __launch_bounds__(BLAS_THREADS)
k_cg_scalars(int nblk, const double *__restrict__ partial, double *sc, int what, double tol2) {
    __shared__ double sm[BLAS_THREADS / 32];
    partial += (size_t)blockIdx.x * nblk;
    sc += blockIdx.x * SC_N;
    double r = 0;
    for (int b = threadIdx.x; b < nblk; b += blockDim.x) r += partial[b];
    r = block_sum(r, sm);
    if (threadIdx.x == 0) cg_scalar_update(sc, r, what, tol2);
}

}  // namespace ovl
