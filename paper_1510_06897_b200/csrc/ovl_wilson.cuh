// ovl_wilson.cuh -- the fused Wilson-stencil / Chebyshev-step kernel.
//
// One launch = one polynomial order of eq. 2.3, i.e. one pass over HBM:
//     hop(x) = sum_mu [ (1 - gamma_mu) U_mu(x) in(x+mu) + (1 + gamma_mu) U_mu(x-mu)^dag in(x-mu) ]   eq. 2.2
//     w(x)   = c_diag * in(x) + c_hop * hop(x)            (D_W: c_diag = 4, c_hop = -1/2;
//                                                          K^ : (4 - m_w)/lambda_max, -1/(2 lambda_max); x2 for m >= 1)
//     w      = gamma5 w                     [F_G5]        (K = gamma5 (D_W - m_w); sign flip of spins 2,3)
//     w     -= prev(x)                      [F_PREV]      (t_{m+1} = 2 K^ t_m - t_{m-1})
//     out(x) = w                            [F_WRITE]     (may alias prev: the ONLY aliasing pair is prev[k,x] / out[k,x], read then
//                                                          written by the same thread with a true data dependency, so declaring
//                                                          both __restrict__ is safe and lets the loads be batched before the stores)
//     acc(x) = a0 * in(x) + a1 * w          [F_ACC_INIT]  (alpha_0 t_0 + alpha_1 t_1)
//     acc(x)+= a1 * w                       [F_ACC_ADD]   (alpha_{m+1} t_{m+1})
// This is the paper's "merging together the Wilson matrix and polynomial algebra ... into a single GPU kernel"
// (PAPER.md:72), re-derived for sm_100a: thread per site, SoA planes so that every load of a warp is one
// contiguous segment, spin projection before the colour multiply (2 x 3 complex per hop instead of 4 x 3),
// antiperiodic t phase applied in-kernel (reading R3), optional 12-real links (third row = conj(r0 x r1)).
//
// Spin projectors in the basis of reading R2 (gamma5 = diag(1,1,-1,-1)); s = +1 for (1 + gamma_mu), -1 for (1 - gamma_mu):
//   x: h0 = p0 + s i p3, h1 = p1 + s i p2;  r2 = -s i h1, r3 = -s i h0
//   y: h0 = p0 - s p3,   h1 = p1 + s p2;    r2 =  s h1,   r3 = -s h0
//   z: h0 = p0 + s i p2, h1 = p1 - s i p3;  r2 = -s i h0, r3 =  s i h1
//   t: h0 = p0 + s p2,   h1 = p1 + s p3;    r2 =  s h0,   r3 =  s h1
// (r0 = h0, r1 = h1 always.)
#pragma once
#include "ovl_types.cuh"

namespace ovl {

enum : int { F_G5 = 1, F_PREV = 2, F_WRITE = 4, F_ACC_INIT = 8, F_ACC_ADD = 16 };

template <typename T> struct StepParams {
    T c_diag, c_hop, a0, a1;
};

// Load the 3x3 link U_mu(su) (rows r, cols c) from the native planes; rebuild row 2 for 12-real storage.
template <typename T, int RECON>
__device__ __forceinline__ void load_link(cx<T> (&u)[3][3], const cx<T> *__restrict__ Umu, int V, int su) {
    constexpr int NROW = RECON == 18 ? 3 : 2;
#pragma unroll
    for (int r = 0; r < NROW; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) u[r][c] = ldg(Umu + (size_t)(r * 3 + c) * V + su);
    if (RECON == 12) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
            cx<T> a = cmul(u[0][c1], u[1][c2]);
            cx<T> b = cmul(u[0][c2], u[1][c1]);
            u[2][c].x = a.x - b.x;
            u[2][c].y = -(a.y - b.y);
        }
    }
}

// One hop: MU direction, FWD = 1: (1 - gamma_mu) U_mu(x) in(x+mu);  FWD = 0: (1 + gamma_mu) U_mu(x-mu)^dag in(x-mu).
// sn = neighbour site, su = site that owns the link, bs = boundary phase (+1 / -1).
template <typename T, int RECON, int MU, int FWD>
__device__ __forceinline__ void hop_dir(cx<T> (&hop)[12], const cx<T> *__restrict__ in, const cx<T> *__restrict__ U,
                                        int V, int sn, int su, T bs) {
    constexpr int NROW = RECON == 18 ? 3 : 2;
    cx<T> p[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) p[k] = ldg(in + (size_t)k * V + sn);
    cx<T> u[3][3];
    load_link<T, RECON>(u, U + (size_t)MU * NROW * 3 * V, V, su);

    cx<T> h0[3], h1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const cx<T> p0 = p[c], p1 = p[3 + c], p2 = p[6 + c], p3 = p[9 + c];
        if (MU == 0) {
            h0[c] = FWD ? csubi(p0, p3) : caddi(p0, p3);
            h1[c] = FWD ? csubi(p1, p2) : caddi(p1, p2);
        } else if (MU == 1) {
            h0[c] = FWD ? cadd(p0, p3) : csub(p0, p3);
            h1[c] = FWD ? csub(p1, p2) : cadd(p1, p2);
        } else if (MU == 2) {
            h0[c] = FWD ? csubi(p0, p2) : caddi(p0, p2);
            h1[c] = FWD ? caddi(p1, p3) : csubi(p1, p3);
        } else {
            h0[c] = FWD ? csub(p0, p2) : cadd(p0, p2);
            h1[c] = FWD ? csub(p1, p3) : cadd(p1, p3);
        }
        h0[c].x *= bs; h0[c].y *= bs;
        h1[c].x *= bs; h1[c].y *= bs;
    }
    cx<T> g0[3], g1[3];
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        g0[i] = mk<T>(0, 0);
        g1[i] = mk<T>(0, 0);
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            if (FWD) {
                cfma(g0[i], u[i][j], h0[j]);
                cfma(g1[i], u[i][j], h1[j]);
            } else {
                cfmac(g0[i], u[j][i], h0[j]);
                cfmac(g1[i], u[j][i], h1[j]);
            }
        }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        hop[c] = cadd(hop[c], g0[c]);
        hop[3 + c] = cadd(hop[3 + c], g1[c]);
        // s = -1 for FWD, +1 for backward
        if (MU == 0) {  // r2 = -s i h1, r3 = -s i h0
            hop[6 + c] = FWD ? caddi(hop[6 + c], g1[c]) : csubi(hop[6 + c], g1[c]);
            hop[9 + c] = FWD ? caddi(hop[9 + c], g0[c]) : csubi(hop[9 + c], g0[c]);
        } else if (MU == 1) {  // r2 = s h1, r3 = -s h0
            hop[6 + c] = FWD ? csub(hop[6 + c], g1[c]) : cadd(hop[6 + c], g1[c]);
            hop[9 + c] = FWD ? cadd(hop[9 + c], g0[c]) : csub(hop[9 + c], g0[c]);
        } else if (MU == 2) {  // r2 = -s i h0, r3 = s i h1
            hop[6 + c] = FWD ? caddi(hop[6 + c], g0[c]) : csubi(hop[6 + c], g0[c]);
            hop[9 + c] = FWD ? csubi(hop[9 + c], g1[c]) : caddi(hop[9 + c], g1[c]);
        } else {  // r2 = s h0, r3 = s h1
            hop[6 + c] = FWD ? csub(hop[6 + c], g0[c]) : cadd(hop[6 + c], g0[c]);
            hop[9 + c] = FWD ? csub(hop[9 + c], g1[c]) : cadd(hop[9 + c], g1[c]);
        }
    }
}

template <typename T, int RECON, int MU>
__device__ __forceinline__ void hop_pair(cx<T> (&hop)[12], const cx<T> *__restrict__ in, const cx<T> *__restrict__ U,
                                         const Geom &g, int s, int xmu, int stride) {
    const int L = g.L[MU];
    const int sf = s + (xmu == L - 1 ? -(L - 1) * stride : stride);
    const int sb = s + (xmu == 0 ? (L - 1) * stride : -stride);
    const T bf = (MU == 3 && xmu == L - 1) ? T(-1) : T(1);
    const T bb = (MU == 3 && xmu == 0) ? T(-1) : T(1);
    hop_dir<T, RECON, MU, 1>(hop, in, U, g.V, sf, s, bf);
    hop_dir<T, RECON, MU, 0>(hop, in, U, g.V, sb, sb, bb);
}

constexpr int WILSON_THREADS = 128;

template <typename T, int RECON, int FLAGS>
__global__ void __launch_bounds__(WILSON_THREADS)
k_wilson_fused(const Geom g, const cx<T> *__restrict__ U, const cx<T> *__restrict__ in, const cx<T> *__restrict__ prev,
               cx<T> *__restrict__ out,
               cx<T> *__restrict__ acc, const StepParams<T> sp) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.V) return;
    const int x = s % g.L[0];
    const int y = (s / g.L[0]) % g.L[1];
    const int z = (s / g.sxy) % g.L[2];
    const int t = s / g.sxyz;

    cx<T> hop[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) hop[k] = mk<T>(0, 0);
    hop_pair<T, RECON, 0>(hop, in, U, g, s, x, 1);
    hop_pair<T, RECON, 1>(hop, in, U, g, s, y, g.L[0]);
    hop_pair<T, RECON, 2>(hop, in, U, g, s, z, g.sxy);
    hop_pair<T, RECON, 3>(hop, in, U, g, s, t, g.sxyz);

    const size_t V = g.V;
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        const cx<T> c = ldg(in + k * V + s);
        cx<T> w;
        w.x = fma(sp.c_diag, c.x, sp.c_hop * hop[k].x);
        w.y = fma(sp.c_diag, c.y, sp.c_hop * hop[k].y);
        if ((FLAGS & F_G5) && k >= 6) { w.x = -w.x; w.y = -w.y; }
        if (FLAGS & F_PREV) {
            const cx<T> pv = prev[k * V + s];
            w.x -= pv.x; w.y -= pv.y;
        }
        if (FLAGS & F_WRITE) out[k * V + s] = w;
        if (FLAGS & F_ACC_INIT) {
            cx<T> a;
            a.x = fma(sp.a0, c.x, sp.a1 * w.x);
            a.y = fma(sp.a0, c.y, sp.a1 * w.y);
            acc[k * V + s] = a;
        }
        if (FLAGS & F_ACC_ADD) {
            cx<T> a = acc[k * V + s];
            a.x = fma(sp.a1, w.x, a.x);
            a.y = fma(sp.a1, w.y, a.y);
            acc[k * V + s] = a;
        }
    }
}

}  // namespace ovl
