// ovl_slab.cuh -- the lattice split along t over several GPUs (the paper ran this
// decomposition on 2 GPUs over MPI: PAPER.md:82-88 Table 3, :99-102 Table 4, :108 "MPI communication between processors").
//
// Slab r of nslabs owns the time slices [r Lt/nslabs, (r+1) Lt/nslabs) of every field: its sites, its 4 links per site, the
// matching part of every eigenvector.  One stencil application needs, per slab, the neighbour slabs' boundary time slices
// of the stencil operand (and, once, the lower neighbour's U_t on its last slice for the backward hop).  B200-first design:
// there is NO separate exchange step --
//   * the fused kernel of order m STORES the two boundary time slices of its output straight into the neighbours' halo
//     buffers (peer pointers: NVLink stores when the slabs sit on different GPUs) in the same epilogue that writes the
//     field, so the transfer is spread over the kernel's run time tile by tile;
//   * the kernel of order m+1 READS the t-neighbours of its boundary sites from its own halo buffers;
//   * the only synchronisation is stream-ordered: slab r's order m+1 waits (cudaStreamWaitEvent) on the events its two
//     neighbours recorded after their order m.  No kernel ever spins on a flag.
// The antiperiodic phase (reading R3) is applied where a hop crosses the GLOBAL t boundary: by the slab that owns t = Lt-1
// (forward) and the one that owns t = 0 (backward).  The arithmetic per site is that of k_wilson_fused, operand by operand,
// so D_W, K^ and the polynomial part of eq. 2.3 are bit-identical to the undivided lattice; reductions (deflation
// coefficients, CG scalars) are summed over slabs in a fixed order and agree to rounding.
#pragma once
#include "ovl_wilson.cuh"

namespace ovl {

// halo wiring of one launch: lo / hi = towards smaller / larger t.  Halo buffers hold one time slice, 12 planes of sxyz.
template <typename T> struct SlabArgs {
    const cx<T> *h_lo, *h_hi;  // operand's halos: the lower neighbour's last slice, the upper neighbour's first slice
    cx<T> *p_lo, *p_hi;        // where this launch's output boundary slices go (neighbours' halo buffers), or null
    const cx<T> *u_lo;         // U_t of the lower neighbour's last slice, NROW*3 planes of sxyz
    T s_lo, s_hi;              // boundary phase of the hop across the lower / upper slab edge (-1 on the global boundary)
};

// Which tiles a launch covers: the whole slab (n1 = all tiles), or -- when the launch is split so that the neighbours can go
// on as soon as the halo traffic is done -- the tiles of the two boundary time slices (first n1 tiles from off1, the rest
// from off2) or the interior (one range).  Position p of the launch -> tile.
struct TileRange {
    int off1, n1, off2;
    __host__ __device__ int tile(int p) const { return p < n1 ? off1 + p : off2 + (p - n1); }
};

// one hop with explicit plane strides (halo buffers and the ghost link slice are time-slice sized)
template <typename T, int RECON, int MU, int FWD>
__device__ __forceinline__ void hop_dir_strided(cx<T> (&hop)[12], const cx<T> *__restrict__ in, size_t in_stride, int sn,
                                                const cx<T> *__restrict__ Umu, size_t u_stride, int su, T bs) {
    cx<T> p[12];
#pragma unroll
    for (int k = 0; k < 12; ++k) p[k] = ldg(in + (size_t)k * in_stride + sn);
    cx<T> u[3][3];
    load_link<T, RECON>(u, Umu, (int)u_stride, su);
    hop_math<T, MU, FWD>(hop, p, u, bs);
}

template <typename T, int RECON, int FLAGS, int THREADS, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
k_wilson_slab(const Geom g, const cx<T> *__restrict__ U, const cx<T> *__restrict__ in, const cx<T> *prev,
              const cx<T> *__restrict__ psi, cx<T> *out, const StepParams<T> sp, const SlabArgs<T> sl, const TileRange tr) {
    constexpr int NROW = RECON == 18 ? 3 : 2;
    const int tile = tr.tile((int)(sp.flip ? gridDim.x - 1 - blockIdx.x : blockIdx.x));
    const int s = tile * THREADS + threadIdx.x;
    if (s >= g.V) return;
    const int x = s % g.L[0];
    const int y = (s / g.L[0]) % g.L[1];
    const int z = (s / g.sxy) % g.L[2];
    const int t = s / g.sxyz;
    const int s3 = s - t * g.sxyz;  // index inside the time slice
    const size_t V = g.V;
    const int Lt = g.L[3];

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
            const cx<T> pv = prev[k * V + s];
            const T r = ((FLAGS & K_G5) && k >= 6) ? sp.r_p : -sp.r_p;
            hop[k].x = fma(r, pv.x, hop[k].x);
            hop[k].y = fma(r, pv.y, hop[k].y);
        }
    }
    if (FLAGS & K_PSI) {
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const cx<T> ps = ldg(psi + k * V + s);
            const T r = ((FLAGS & K_G5) && k >= 6) ? -sp.r_a : sp.r_a;
            hop[k].x = fma(r, ps.x, hop[k].x);
            hop[k].y = fma(r, ps.y, hop[k].y);
        }
    }
    // t hops (same order as k_wilson_fused: forward, then backward); slab edges read the halos
    const cx<T> *Ut = U + (size_t)3 * NROW * 3 * V;
    if (t == Lt - 1) hop_dir_strided<T, RECON, 3, 1>(hop, sl.h_hi, (size_t)g.sxyz, s3, Ut, V, s, sl.s_hi);
    else hop_dir_strided<T, RECON, 3, 1>(hop, in, V, s + g.sxyz, Ut, V, s, T(1));
    if (t == 0) hop_dir_strided<T, RECON, 3, 0>(hop, sl.h_lo, (size_t)g.sxyz, s3, sl.u_lo, (size_t)g.sxyz, s3, sl.s_lo);
    else hop_dir_strided<T, RECON, 3, 0>(hop, in, V, s - g.sxyz, Ut, V, s - g.sxyz, T(1));
    hop_pair<T, RECON, 2>(hop, in, U, g, s, z, g.sxy);
    hop_pair<T, RECON, 1>(hop, in, U, g, s, y, g.L[0]);
    hop_pair<T, RECON, 0>(hop, in, U, g, s, x, 1);

#pragma unroll
    for (int k = 0; k < 12; ++k) {
        const T f = ((FLAGS & K_G5) && k >= 6) ? -sp.c_hop : sp.c_hop;
        cx<T> w;
        w.x = f * hop[k].x;
        w.y = f * hop[k].y;
        out[k * V + s] = w;
        // fused halo push: the boundary slices of the output land in the neighbours' halo buffers (peer stores)
        if (t == 0 && sl.p_lo) sl.p_lo[(size_t)k * g.sxyz + s3] = w;
        if (t == Lt - 1 && sl.p_hi) sl.p_hi[(size_t)k * g.sxyz + s3] = w;
    }
}

// faces of a field that was not produced by the fused kernel (the source of a polynomial, a CG vector): copy the first
// and the last time slice into the neighbours' halo buffers.  grid covers 12 * sxyz elements.
template <typename T>
__global__ void k_push_faces(int V, int sxyz, const cx<T> *__restrict__ f, cx<T> *p_lo, cx<T> *p_hi) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (size_t)12 * sxyz) return;
    const int k = (int)(e / sxyz), s3 = (int)(e - (size_t)k * sxyz);
    if (p_lo) p_lo[e] = f[(size_t)k * V + s3];
    if (p_hi) p_hi[e] = f[(size_t)k * V + (V - sxyz) + s3];
}
// the last time slice of the native U_t planes -> a contiguous ghost slice (sent to the upper neighbour once, at create)
template <typename T>
__global__ void k_pack_ut_last(int V, int sxyz, int nplanes, const cx<T> *__restrict__ Ut, cx<T> *__restrict__ dst) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (size_t)nplanes * sxyz) return;
    const int k = (int)(e / sxyz), s3 = (int)(e - (size_t)k * sxyz);
    dst[e] = Ut[(size_t)k * V + (V - sxyz) + s3];
}

// reductions over slabs: out[j] = sum_{slab} parts[slab][j], fixed order (every slab runs this and gets the same bits)
constexpr int MAX_SLABS = 16;
struct SlabPtrs { const double *p[MAX_SLABS]; };
__global__ void k_sum_over_slabs(int nslabs, SlabPtrs parts, int n, double *__restrict__ out) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    double r = 0;
    for (int q = 0; q < nslabs; ++q) r += parts.p[q][j];
    out[j] = r;
}

}  // namespace ovl
