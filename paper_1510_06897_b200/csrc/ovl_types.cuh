// ovl_types.cuh -- complex helpers, lattice geometry and the native (SoA, site-coalesced) field layout.
//
// Native layout (north_star (a)):
//   spinor:  12 planes of V complex, plane k = 3*spin + colour:   f[k*V + s]
//   links:   4 directions x NROW*3 planes of V complex (NROW = 3 for 18-real, 2 for 12-real storage):
//            U[((mu*NROW + row)*3 + col)*V + s]
// so a warp of consecutive sites reads one contiguous 512 B (fp64) / 256 B (fp32) segment per plane.
// This file shares nothing with oracle/ (AoS, explicit 4x4 gamma matrices).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ovl {

template <typename T> struct cx_of;
template <> struct cx_of<double> { using type = double2; };
template <> struct cx_of<float> { using type = float2; };
template <typename T> using cx = typename cx_of<T>::type;

template <typename T> __host__ __device__ __forceinline__ cx<T> mk(T re, T im) {
    cx<T> r; r.x = re; r.y = im; return r;
}
// a + b, a - b
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { a.x += b.x; a.y += b.y; return a; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { a.x -= b.x; a.y -= b.y; return a; }
// a + i b, a - i b
template <typename C> __device__ __forceinline__ C caddi(C a, C b) { a.x -= b.y; a.y += b.x; return a; }
template <typename C> __device__ __forceinline__ C csubi(C a, C b) { a.x += b.y; a.y -= b.x; return a; }
// acc += a * b
template <typename C> __device__ __forceinline__ void cfma(C &acc, C a, C b) {
    acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a) * b
template <typename C> __device__ __forceinline__ void cfmac(C &acc, C a, C b) {
    acc.x = fma(a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y); acc.y = fma(-a.y, b.x, acc.y);
}
// a * b, conj(a * b)
template <typename C> __device__ __forceinline__ C cmul(C a, C b) {
    C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}

struct Geom {
    int L[4];      // Lx, Ly, Lz, Lt
    int V;         // sites
    int sxy, sxyz; // Lx*Ly, Lx*Ly*Lz
};
// L2-aware sweep order for lattices whose time slices outgrow the L2: the 128-site tiles are visited z-slab by z-slab
// (nzs slabs of tpc tiles per time slice), all time slices of a slab before the next slab, so the reuse distance of the t
// neighbours and of U_t(x - t^) is one slab of one time slice instead of a whole time slice.  Position in the sweep -> tile
// (a permutation of whole tiles).
struct Sweep { int tpc, nzs; };
__device__ __forceinline__ int sweep_tile(const Sweep &sw, int Lt, int pos) {
    const int c = pos / sw.tpc, w = pos - c * sw.tpc;
    const int zs = c / Lt, t = c - zs * Lt;
    return (t * sw.nzs + zs) * sw.tpc + w;
}

// Brick order for lattices small enough that a launch is bound by what every SM pulls out of the L2 (L1 is cold at every
// launch): a 128-thread CTA handles a 2 x 2 stack in (z, t) of chunks of 32 sites that are consecutive in the half volume
// u = x + Lx (y + Ly (z / 2)), so the z and t neighbours (and backward links) of half of the hops are the centre sites of
// another warp of the same CTA and are found in its L1.  Needs Lz and Lt even.  nchunk = 0: plain order.
struct Brick { int nchunk, half; };
constexpr int BRICK_GS = 32;
// CTA index, thread -> site (or -1 for the ragged end of the last chunk of a time-slice pair)
__device__ __forceinline__ int brick_site(const Brick &bk, const Geom &g, int cta, int thread) {
    const int grp = thread / BRICK_GS, li = thread - grp * BRICK_GS;
    const int th = cta / bk.nchunk, ch = cta - th * bk.nchunk;
    const int u = ch * BRICK_GS + li;
    if (u >= bk.half) return -1;
    const int zh = u / g.sxy, r = u - zh * g.sxy;
    return r + g.sxy * (2 * zh + (grp & 1)) + g.sxyz * (2 * th + (grp >> 1));
}

// read-only (non-coherent) loads, for the fields a kernel never writes (links, the stencil operand, psi, eigenvectors);
// `prev` of the fused kernel may alias its output and is NOT read through this path
__device__ __forceinline__ double2 ldg(const double2 *p) { return __ldg(p); }
__device__ __forceinline__ float2 ldg(const float2 *p) { return __ldg(p); }

// loads of single-use streams (b_{k+2}, psi: read once per launch, no neighbour reuse): L2 evict-first, so that they do not
// displace the stencil operand and the links, which the neighbouring sites and the backward hops find in L2
__device__ __forceinline__ unsigned long long l2_evict_first_policy() {
    unsigned long long p;
    asm("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ double2 ldg_once(const double2 *p) {
    double2 v;
    asm("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(l2_evict_first_policy()));
    return v;
}
__device__ __forceinline__ float2 ldg_once(const float2 *p) {
    float2 v;
    asm("ld.global.nc.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(l2_evict_first_policy()));
    return v;
}
// the same for a field the kernel also writes (coherent load, ordered against the store of the same thread)
__device__ __forceinline__ double2 ld_once(const double2 *p) {
    double2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(p), "l"(l2_evict_first_policy()) : "memory");
    return v;
}
__device__ __forceinline__ float2 ld_once(const float2 *p) {
    float2 v;
    asm volatile("ld.global.L2::cache_hint.v2.f32 {%0,%1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(l2_evict_first_policy()) : "memory");
    return v;
}

// 16- or 8-byte asynchronous global -> shared copy of one complex (LDGSTS), and its completion wait
template <typename C> __device__ __forceinline__ void cp_async_cx(C *smem, const C *gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    if (sizeof(C) == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

}  // namespace ovl
