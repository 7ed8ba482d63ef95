// ovl_wilson.cuh -- the fused Wilson-stencil / Chebyshev-step kernel.
//
// One launch = one polynomial order of eq. 2.3, i.e. one pass over HBM:
//     hop(x) = sum_mu [ (1 - gamma_mu) U_mu(x) in(x+mu) + (1 + gamma_mu) U_mu(x-mu)^dag in(x-mu) ]   eq. 2.2
//     w(x)   = sigma (c_diag in(x) + c_hop hop(x))        D_W: c_diag = 4, c_hop = -1/2, sigma = 1;
//                                                         K^ : (4 - m_w)/lambda_max, -1/(2 lambda_max), sigma = gamma5 [K_G5]
//                                                         (K = gamma5 (D_W - m_w); gamma5 = sign flip of spins 2,3)
//     w     -= prev(x)                      [K_PREV]      three-term recurrence, forward t_{m+1} = 2 K^ t_m - t_{m-1}
//                                                         or Clenshaw b_k = alpha_k psi + 2 K^ b_{k+1} - b_{k+2}
//     w     += a_psi psi(x)                 [K_PSI]       the alpha_k psi term of the Clenshaw form
//     out(x) = w                            [unless K_NOWRITE]  (may alias prev: prev[k,x] / out[k,x] are read then written by
//                                                         the same thread with a true data dependency; prev is therefore read
//                                                         with plain coherent loads and neither pointer is __restrict__)
//     acc(x)+= a_acc w                      [K_ACC]       forward form: + alpha_{m+1} t_{m+1}
//     acc(x) = a_init in(x) + a_acc w       [K_ACCI]      forward form, first order: alpha_0 t_0 + alpha_1 t_1
// This is the paper's "merging together the Wilson matrix and polynomial algebra ... into a single GPU kernel"
// (PAPER.md:72), re-derived for sm_100a: thread per site, SoA planes so that every load of a warp is one
// contiguous segment, spin projection before the colour multiply (2 x 3 complex per hop instead of 4 x 3),
// antiperiodic t phase applied in-kernel (reading R3), optional 12-real links (third row = conj(r0 x r1)).
//
// Latency structure: the site-local operands (in(x), prev(x), psi(x)) are folded into the INITIAL value of
// the 12 hop accumulators at the top of the kernel,
//     h_k := (c_diag/c_hop) in_k + sigma_k (a_psi psi_k - prev_k)/c_hop ,   w_k = sigma_k c_hop (h_k + hop_k) ,
// so their first-touch (DRAM) loads are in flight together with the first hop's and the epilogue is store-only:
// no load of the kernel waits behind the whole stencil.  Measured on B200 at 20^3x64 fp64 this (with the Clenshaw form,
// which has no read-modify-write stream) took one order from 171 us to 125 us.
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

enum : int { K_G5 = 1, K_PREV = 2, K_PSI = 4, K_ACC = 8, K_ACCI = 16, K_NOWRITE = 32 };

// c_hop and the ratios r_c = c_diag/c_hop, r_p = 1/c_hop, r_a = a_psi/c_hop (see the header); flip = sweep the lattice
// from the last CTA tile to the first (consecutive orders alternate, so an order starts on what the previous one left in L2)
template <typename T> struct StepParams {
    T c_hop, r_c, r_p, r_a, a_acc, a_init;
    int flip;
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

// The arithmetic of one hop given the neighbour spinor p and the link u (already in registers), in two halves:
//   hop_half   spin projection to a half spinor and the 3x3 colour multiply (U for FWD = 1, U^dag for FWD = 0): g0, g1;
//   hop_accum  reconstruction of the four spin rows from (g0, g1), added to the 12 accumulators (one addition each).
// MU direction, FWD = 1: (1 - gamma_mu) U_mu(x) in(x+mu);  FWD = 0: (1 + gamma_mu) U_mu(x-mu)^dag in(x-mu); bs = boundary phase.
template <typename T, int MU, int FWD>
__device__ __forceinline__ void hop_half(cx<T> (&g0)[3], cx<T> (&g1)[3], const cx<T> (&p)[12], const cx<T> (&u)[3][3], T bs) {
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
        if (MU == 3) {  // only the t hops can cross the antiperiodic boundary (bs = +-1; elsewhere it is exactly 1)
            h0[c].x *= bs; h0[c].y *= bs;
            h1[c].x *= bs; h1[c].y *= bs;
        }
    }
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
}
// row r (0..3) of the reconstructed hop for colour c, added to acc:  rows 0, 1 are g0, g1; rows 2, 3 follow the table in the
// file header (s = -1 for FWD, +1 for backward)
template <typename T, int MU, int FWD, int ROW>
__device__ __forceinline__ cx<T> hop_row_add(cx<T> acc, cx<T> g0c, cx<T> g1c) {
    if (ROW == 0) return cadd(acc, g0c);
    if (ROW == 1) return cadd(acc, g1c);
    if (MU == 0) {  // r2 = -s i h1, r3 = -s i h0
        if (ROW == 2) return FWD ? caddi(acc, g1c) : csubi(acc, g1c);
        return FWD ? caddi(acc, g0c) : csubi(acc, g0c);
    } else if (MU == 1) {  // r2 = s h1, r3 = -s h0
        if (ROW == 2) return FWD ? csub(acc, g1c) : cadd(acc, g1c);
        return FWD ? cadd(acc, g0c) : csub(acc, g0c);
    } else if (MU == 2) {  // r2 = -s i h0, r3 = s i h1
        if (ROW == 2) return FWD ? caddi(acc, g0c) : csubi(acc, g0c);
        return FWD ? csubi(acc, g1c) : caddi(acc, g1c);
    } else {  // r2 = s h0, r3 = s h1
        if (ROW == 2) return FWD ? csub(acc, g0c) : cadd(acc, g0c);
        return FWD ? csub(acc, g1c) : cadd(acc, g1c);
    }
}
template <typename T, int MU, int FWD>
__device__ __forceinline__ void hop_accum(cx<T> (&hop)[12], const cx<T> (&g0)[3], const cx<T> (&g1)[3]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        hop[c] = hop_row_add<T, MU, FWD, 0>(hop[c], g0[c], g1[c]);
        hop[3 + c] = hop_row_add<T, MU, FWD, 1>(hop[3 + c], g0[c], g1[c]);
        hop[6 + c] = hop_row_add<T, MU, FWD, 2>(hop[6 + c], g0[c], g1[c]);
        hop[9 + c] = hop_row_add<T, MU, FWD, 3>(hop[9 + c], g0[c], g1[c]);
    }
}
template <typename T, int MU, int FWD>
__device__ __forceinline__ void hop_math(cx<T> (&hop)[12], const cx<T> (&p)[12], const cx<T> (&u)[3][3], T bs) {
    cx<T> g0[3], g1[3];
    hop_half<T, MU, FWD>(g0, g1, p, u, bs);
    hop_accum<T, MU, FWD>(hop, g0, g1);
}

// One hop with both operands loaded from global memory: sn = neighbour site, su = site that owns the link.
template <typename T, int RECON, int MU, int FWD>
__device__ __forceinline__ void hop_dir(cx<T> (&hop)[12], const cx<T> *__restrict__ in, const cx<T> *__restrict__ U,
                                        int V, int sn, int su, T bs) {
    constexpr int NROW = RECON == 18 ? 3 : 2;
    cx<T> p[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) p[k] = ldg(in + (size_t)k * V + sn);
    cx<T> u[3][3];
    load_link<T, RECON>(u, U + (size_t)MU * NROW * 3 * V, V, su);
    hop_math<T, MU, FWD>(hop, p, u, bs);
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

// Forward recurrence only: landing buffer of the accumulator stream.  acc(x) is needed after the whole stencil; loading it
// there exposes a DRAM round trip per thread, loading it into registers at the top costs 48 registers.  It is copied
// global -> shared with cp.async at the top instead (each thread its own 12 elements, so no barrier) and read back in the
// epilogue: 24 KB per CTA in fp64.
template <typename T, int THREADS, bool ENABLE> __device__ __forceinline__ cx<T> *acc_stage() {
    if constexpr (ENABLE) {
        __shared__ cx<T> buf[12 * THREADS];
        return buf;
    } else {
        return nullptr;
    }
}

// The kernel body for site s of one right-hand side (THREADS = CTA size: the accumulator staging is indexed by thread).
template <typename T, int RECON, int FLAGS, int THREADS>
__device__ __forceinline__ void wilson_site(const Geom &g, const cx<T> *__restrict__ U, const cx<T> *__restrict__ in,
                                            const cx<T> *prev, const cx<T> *__restrict__ psi, cx<T> *out,
                                            cx<T> *__restrict__ acc, const StepParams<T> &sp, const int s) {
    const int x = s % g.L[0];
    const int y = (s / g.L[0]) % g.L[1];
    const int z = (s / g.sxy) % g.L[2];
    const int t = s / g.sxyz;
    const size_t V = g.V;
    cx<T> *const acc_sm = acc_stage<T, THREADS, (FLAGS & K_ACC) != 0>();
    if (FLAGS & K_ACC) {
#pragma unroll
        for (int k = 0; k < 12; ++k) cp_async_cx(acc_sm + k * THREADS + threadIdx.x, acc + k * V + s);
        asm volatile("cp.async.commit_group;" ::: "memory");
    }

    // accumulators start from the site-local terms (no loads are left for the epilogue)
    cx<T> hop[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        const cx<T> c = ldg(in + k * V + s);
        hop[k].x = sp.r_c * c.x;
        hop[k].y = sp.r_c * c.y;
    }
    if (FLAGS & K_PREV) {
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const cx<T> pv = ld_once(prev + k * V + s);  // coherent load (not .nc): out may alias prev
            const T r = ((FLAGS & K_G5) && k >= 6) ? sp.r_p : -sp.r_p;
            hop[k].x = fma(r, pv.x, hop[k].x);
            hop[k].y = fma(r, pv.y, hop[k].y);
        }
    }
    if (FLAGS & K_PSI) {
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const cx<T> ps = ldg_once(psi + k * V + s);
            const T r = ((FLAGS & K_G5) && k >= 6) ? -sp.r_a : sp.r_a;
            hop[k].x = fma(r, ps.x, hop[k].x);
            hop[k].y = fma(r, ps.y, hop[k].y);
        }
    }
    // t first: in(x + t^) and U_t(x) are the first touches of the sweep (DRAM), everything after is mostly cache
    hop_pair<T, RECON, 3>(hop, in, U, g, s, t, g.sxyz);
    hop_pair<T, RECON, 2>(hop, in, U, g, s, z, g.sxy);
    hop_pair<T, RECON, 1>(hop, in, U, g, s, y, g.L[0]);
    hop_pair<T, RECON, 0>(hop, in, U, g, s, x, 1);

#pragma unroll
    for (int k = 0; k < 12; ++k) {
        const T f = ((FLAGS & K_G5) && k >= 6) ? -sp.c_hop : sp.c_hop;
        cx<T> w;
        w.x = f * hop[k].x;
        w.y = f * hop[k].y;
        if (!(FLAGS & K_NOWRITE)) out[k * V + s] = w;
        if (FLAGS & K_ACCI) {
            const cx<T> c = ldg(in + k * V + s);
            cx<T> a;
            a.x = fma(sp.a_init, c.x, sp.a_acc * w.x);
            a.y = fma(sp.a_init, c.y, sp.a_acc * w.y);
            acc[k * V + s] = a;
        }
        if (FLAGS & K_ACC) {
            if (k == 0) cp_async_wait_all();
            cx<T> a = acc_sm[k * THREADS + threadIdx.x];
            a.x = fma(sp.a_acc, w.x, a.x);
            a.y = fma(sp.a_acc, w.y, a.y);
            acc[k * V + s] = a;
        }
    }
}

// ... for one tile of THREADS consecutive sites
template <typename T, int RECON, int FLAGS, int THREADS>
__device__ __forceinline__ void wilson_tile(const Geom &g, const cx<T> *__restrict__ U, const cx<T> *__restrict__ in,
                                            const cx<T> *prev, const cx<T> *__restrict__ psi, cx<T> *out,
                                            cx<T> *__restrict__ acc, const StepParams<T> &sp, int tile) {
    const int s = tile * THREADS + threadIdx.x;
    if (s >= g.V) return;
    wilson_site<T, RECON, FLAGS, THREADS>(g, U, in, prev, psi, out, acc, sp, s);
}

// Single right-hand side: the field pointers stay kernel parameters (constant bank).
template <typename T, int RECON, int FLAGS, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
k_wilson_fused(const Geom g, const cx<T> *__restrict__ U, const cx<T> *__restrict__ in, const cx<T> *prev,
               const cx<T> *__restrict__ psi, cx<T> *out, cx<T> *__restrict__ acc, const StepParams<T> sp) {
    const int tile = sp.flip ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
    wilson_tile<T, RECON, FLAGS, THREADS>(g, U, in, prev, psi, out, acc, sp, tile);
}

// The same kernel visiting the tiles in the L2-aware z-slab order (Sweep, ovl_types.cuh).  A kernel of its own with its own
// parameter list: the register allocation of the plain-order kernel at the 168-register cap is fragile, and it stays
// exactly as it was.
template <typename T, int RECON, int FLAGS, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
k_wilson_fused_swept(const Geom g, const cx<T> *__restrict__ U, const cx<T> *__restrict__ in, const cx<T> *prev,
                     const cx<T> *__restrict__ psi, cx<T> *out, cx<T> *__restrict__ acc, const StepParams<T> sp, const Sweep sw) {
    const int tile = sweep_tile(sw, g.L[3], sp.flip ? gridDim.x - 1 - blockIdx.x : blockIdx.x);
    wilson_tile<T, RECON, FLAGS, THREADS>(g, U, in, prev, psi, out, acc, sp, tile);
}

// Several right-hand sides: blockIdx.x = rhs + nrhs * tile, so the CTAs that work on the same
// tile for different right-hand sides are adjacent in launch order, run at the same time, and the tile's links come from
// DRAM once and from L2 after that.  Field r starts r * fstride complex elements after field 0.
template <typename T, int RECON, int FLAGS, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
k_wilson_fused_multi(const Geom g, const cx<T> *__restrict__ U, const cx<T> *in, const cx<T> *prev, const cx<T> *psi, cx<T> *out,
                     cx<T> *acc, const StepParams<T> sp, int nrhs, size_t fstride) {
    const int ntile = gridDim.x / nrhs, btile = blockIdx.x / nrhs;
    const int tile = sp.flip ? ntile - 1 - btile : btile;
    const size_t off = (size_t)(blockIdx.x % nrhs) * fstride;
    wilson_tile<T, RECON, FLAGS, THREADS>(g, U, in + off, (FLAGS & K_PREV) ? prev + off : prev, (FLAGS & K_PSI) ? psi + off : psi,
                                          (FLAGS & K_NOWRITE) ? out : out + off, (FLAGS & (K_ACC | K_ACCI)) ? acc + off : acc, sp, tile);
}

// The single-right-hand-side kernel in brick order (Brick, ovl_types.cuh) for small lattices: same arithmetic per site, so
// the results are bit-identical to the plain order.  4 * BRICK_GS = 128 threads per CTA; such a lattice is at most a few CTAs
// per SM, so the kernel is compiled without an occupancy target (up to 255 registers, no spills, deeper load batches).
// (Several right-hand sides stay on k_wilson_fused_multi: with nrhs CTAs per tile the plain order measured faster.)
template <typename T, int RECON, int FLAGS>
__global__ void __launch_bounds__(4 * BRICK_GS, 1)
k_wilson_fused_brick(const Geom g, const cx<T> *__restrict__ U, const cx<T> *__restrict__ in, const cx<T> *prev,
                     const cx<T> *__restrict__ psi, cx<T> *out, cx<T> *__restrict__ acc, const StepParams<T> sp, const Brick bk) {
    const int s = brick_site(bk, g, sp.flip ? gridDim.x - 1 - blockIdx.x : blockIdx.x, threadIdx.x);
    if (s < 0) return;
    wilson_site<T, RECON, FLAGS, 4 * BRICK_GS>(g, U, in, prev, psi, out, acc, sp, s);
}
}  // namespace ovl
