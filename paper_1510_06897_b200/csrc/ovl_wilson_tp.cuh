// ovl_wilson_tp.cuh -- the fused Wilson-stencil / Chebyshev-step kernel
// as a persistent, warp-pipelined kernel with a shared-memory landing zone fed by bulk asynchronous copies.
//
// Same arithmetic, operand order and flags as k_wilson_fused (ovl_wilson.cuh) -- results are bit-identical -- but:
//   * persistent warps: warp w of CTA b walks the 32-site sub-tiles  b*NW + w, + gridDim.x*NW, ...  of the lattice;
//   * the first-touch (DRAM) streams of a sub-tile land in shared memory by cp.async.bulk (1-D bulk copies: a plane segment
//     of 32 consecutive sites is one contiguous 512 B / 256 B block of the SoA layout, so no tensor map is needed and the
//     periodic wrap never cuts a copy) with mbarrier complete_tx: the warp's own links U_mu(x) per direction [STG_LINKS],
//     optionally in(x + t^) [STG_TFW] and prev(x), psi(x) [STG_SITE];
//   * every staged buffer is refilled for the warp's NEXT sub-tile the moment its last reader is done (direction by
//     direction), so the DRAM fetch of sub-tile i+1 overlaps the rest of the arithmetic of sub-tile i and the bytes in
//     flight per SM are no longer bounded by the register file ("transfer from global memory to the
//     registers (very important)");
//   * the streams that are not staged can be pulled into L2 ahead of use by cp.async.bulk.prefetch.L2 [PF_L2].
// Neighbour spinors in x, y, z, t- and the backward links U_mu(x - mu) were touched by earlier sites and come through
// L1/L2 with ordinary loads.  Requires V % 32 == 0 and Lx*Ly*Lz % 32 == 0 (a sub-tile never straddles a time slice); the
// library falls back to k_wilson_fused otherwise.
#pragma once
#include "ovl_wilson.cuh"

namespace ovl {

enum : int { STG_LINKS = 1, PF_L2 = 2, STG_TFW = 4, STG_SITE = 8, STG_TZ_ONLY = 16 };

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
// global -> shared bulk copy, completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void *src, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}

// Shared-memory bytes of one warp's landing zone
template <typename T, int RECON, int FLAGS, int OPT> struct TpSmem {
    static constexpr int NPL = (RECON == 18 ? 3 : 2) * 3;            // planes per link direction
    static constexpr int SEG = 32 * (int)sizeof(cx<T>);              // one plane segment of a sub-tile
    static constexpr int LINKS = (OPT & STG_LINKS) ? 4 * NPL * SEG : 0;  // (all four slots are kept even with STG_TZ_ONLY)
    static constexpr int TFW = (OPT & STG_TFW) ? 12 * SEG : 0;
    static constexpr int PREV = ((OPT & STG_SITE) && (FLAGS & K_PREV)) ? 12 * SEG : 0;
    static constexpr int PSI = ((OPT & STG_SITE) && (FLAGS & K_PSI)) ? 12 * SEG : 0;
    static constexpr int PER_WARP = LINKS + TFW + PREV + PSI;
    static constexpr int NBAR = 8;                                    // links x4, tfw, prev, psi (+1 pad)
    static constexpr size_t total(int nw) { return (size_t)nw * (PER_WARP + NBAR * 8); }
};

template <typename T, int RECON, int FLAGS, int OPT, int NW, int MINB>
__global__ void __launch_bounds__(NW * 32, MINB)
k_wilson_tp(const Geom g, const cx<T> *__restrict__ U, const cx<T> *__restrict__ in, const cx<T> *prev,
            const cx<T> *__restrict__ psi, cx<T> *out, const StepParams<T> sp, int nsub) {
    static_assert(!(FLAGS & (K_ACC | K_ACCI | K_NOWRITE)), "the forward-recurrence accumulator modes stay on k_wilson_fused");
    using SM = TpSmem<T, RECON, FLAGS, OPT>;
    constexpr int NPL = SM::NPL, NROW = RECON == 18 ? 3 : 2;
    extern __shared__ __align__(128) unsigned char tp_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char *my = tp_smem + (size_t)warp * SM::PER_WARP;
    cx<T> *const sm_lk = (cx<T> *)my;
    cx<T> *const sm_tfw = (cx<T> *)(my + SM::LINKS);
    cx<T> *const sm_prev = (cx<T> *)(my + SM::LINKS + SM::TFW);
    cx<T> *const sm_psi = (cx<T> *)(my + SM::LINKS + SM::TFW + SM::PREV);
    uint64_t *const bars = (uint64_t *)(tp_smem + (size_t)NW * SM::PER_WARP) + warp * SM::NBAR;
    enum { B_TFW = 4, B_PREV = 5, B_PSI = 6 };
    const size_t V = g.V;

    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < SM::NBAR; ++i) mbar_init(&bars[i], 1);
        mbar_fence_init();
    }
    __syncwarp();

    const int stride = gridDim.x * NW;
    int sub = blockIdx.x * NW + warp;
    auto site0 = [&](int sb) { return (sp.flip ? nsub - 1 - sb : sb) * 32; };
    // t-forward neighbour block of a sub-tile (a sub-tile lies inside one time slice)
    auto tfw0 = [&](int s0) {
        const int t = s0 / g.sxyz;
        return t == g.L[3] - 1 ? s0 - (g.L[3] - 1) * g.sxyz : s0 + g.sxyz;
    };
    // refill one staged buffer for sub-tile sb: lane 0 arms the barrier, lanes < nplanes copy one plane segment each
    auto fill = [&](uint64_t *bar, cx<T> *dst, const cx<T> *src_plane0, int nplanes, int s0) {
        if (lane == 0) {
            mbar_expect_tx(bar, (uint32_t)(nplanes * SM::SEG));
#pragma unroll
            for (int pl = 0; pl < 12; ++pl)
                if (pl < nplanes) bulk_g2s(dst + pl * 32, src_plane0 + (size_t)pl * V + s0, SM::SEG, bar);
        }
    };
    auto fill_links = [&](int mu, int sb) { fill(&bars[mu], sm_lk + mu * NPL * 32, U + (size_t)mu * NPL * V, NPL, site0(sb)); };
    auto prefetch = [&](int sb) {  // L2 prefetch of the un-staged first-touch streams of sub-tile sb
        const int s0 = site0(sb), sf = tfw0(s0);
        if (!(OPT & STG_TFW) && lane < 12) bulk_prefetch_l2(in + (size_t)lane * V + sf, SM::SEG);
        if (!(OPT & STG_SITE)) {
            if ((FLAGS & K_PREV) && lane >= 12 && lane < 24) bulk_prefetch_l2(prev + (size_t)(lane - 12) * V + s0, SM::SEG);
            if ((FLAGS & K_PSI) && lane >= 20) bulk_prefetch_l2(psi + (size_t)(lane - 20) * V + s0, SM::SEG);
        }
        if (!(OPT & STG_LINKS)) {
#pragma unroll
            for (int j = 0; j < (4 * NPL + 31) / 32; ++j)
                if (lane + 32 * j < 4 * NPL) bulk_prefetch_l2(U + (size_t)(lane + 32 * j) * V + s0, SM::SEG);
        }
    };

    if (sub < nsub) {  // prologue: everything for the first sub-tile
        if (OPT & STG_LINKS) {
#pragma unroll
            for (int mu = 3; mu >= ((OPT & STG_TZ_ONLY) ? 2 : 0); --mu) fill_links(mu, sub);
        }
        if (OPT & STG_TFW) fill(&bars[B_TFW], sm_tfw, in, 12, tfw0(site0(sub)));
        if ((OPT & STG_SITE) && (FLAGS & K_PREV)) fill(&bars[B_PREV], sm_prev, prev, 12, site0(sub));
        if ((OPT & STG_SITE) && (FLAGS & K_PSI)) fill(&bars[B_PSI], sm_psi, psi, 12, site0(sub));
    }
    uint32_t phase = 0;
    for (; sub < nsub; sub += stride, phase ^= 1) {
        const int s = site0(sub) + lane;
        const int nxt = sub + stride;
        const bool more = nxt < nsub;
        const int x = s % g.L[0];
        const int y = (s / g.L[0]) % g.L[1];
        const int z = (s / g.sxy) % g.L[2];
        const int t = s / g.sxyz;
        if ((OPT & PF_L2) && more) prefetch(nxt);

        // accumulators start from the site-local terms (as k_wilson_fused)
        cx<T> hop[12];
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const cx<T> c = ldg(in + k * V + s);
            hop[k].x = sp.r_c * c.x;
            hop[k].y = sp.r_c * c.y;
        }
        if (FLAGS & K_PREV) {
            if (OPT & STG_SITE) mbar_wait(&bars[B_PREV], phase);
#pragma unroll
            for (int k = 0; k < 12; ++k) {
                const cx<T> pv = (OPT & STG_SITE) ? sm_prev[k * 32 + lane] : prev[k * V + s];
                const T r = ((FLAGS & K_G5) && k >= 6) ? sp.r_p : -sp.r_p;
                hop[k].x = fma(r, pv.x, hop[k].x);
                hop[k].y = fma(r, pv.y, hop[k].y);
            }
            if ((OPT & STG_SITE) && more) { __syncwarp(); fill(&bars[B_PREV], sm_prev, prev, 12, site0(nxt)); }
        }
        if (FLAGS & K_PSI) {
            if (OPT & STG_SITE) mbar_wait(&bars[B_PSI], phase);
#pragma unroll
            for (int k = 0; k < 12; ++k) {
                const cx<T> ps = (OPT & STG_SITE) ? sm_psi[k * 32 + lane] : ldg(psi + k * V + s);
                const T r = ((FLAGS & K_G5) && k >= 6) ? -sp.r_a : sp.r_a;
                hop[k].x = fma(r, ps.x, hop[k].x);
                hop[k].y = fma(r, ps.y, hop[k].y);
            }
            if ((OPT & STG_SITE) && more) { __syncwarp(); fill(&bars[B_PSI], sm_psi, psi, 12, site0(nxt)); }
        }

        // forward hop in direction MU with the staged own link (and, for t, the staged neighbour), then the backward hop
        auto pair = [&](auto mu_c, int xmu, int strd) {
            constexpr int MU = decltype(mu_c)::value;
            const int L = g.L[MU];
            const int sf = s + (xmu == L - 1 ? -(L - 1) * strd : strd);
            const int sb = s + (xmu == 0 ? (L - 1) * strd : -strd);
            const T bf = (MU == 3 && xmu == L - 1) ? T(-1) : T(1);
            const T bb = (MU == 3 && xmu == 0) ? T(-1) : T(1);
            if ((OPT & STG_LINKS) && (!(OPT & STG_TZ_ONLY) || MU >= 2)) {
                cx<T> p[12];
                if (MU == 3 && (OPT & STG_TFW)) {
                    mbar_wait(&bars[B_TFW], phase);
#pragma unroll
                    for (int k = 0; k < 12; ++k) p[k] = sm_tfw[k * 32 + lane];
                } else {
#pragma unroll
                    for (int k = 0; k < 12; ++k) p[k] = ldg(in + (size_t)k * V + sf);
                }
                mbar_wait(&bars[MU], phase);
                cx<T> u[3][3];
                const cx<T> *lk = sm_lk + MU * NPL * 32 + lane;
#pragma unroll
                for (int r = 0; r < NROW; ++r)
#pragma unroll
                    for (int c = 0; c < 3; ++c) u[r][c] = lk[(r * 3 + c) * 32];
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
                hop_math<T, MU, 1>(hop, p, u, bf);
                if (more) {
                    __syncwarp();
                    fill_links(MU, nxt);
                    if (MU == 3 && (OPT & STG_TFW)) fill(&bars[B_TFW], sm_tfw, in, 12, tfw0(site0(nxt)));
                }
            } else {
                hop_dir<T, RECON, MU, 1>(hop, in, U, g.V, sf, s, bf);
            }
            hop_dir<T, RECON, MU, 0>(hop, in, U, g.V, sb, sb, bb);
        };
        pair(std::integral_constant<int, 3>{}, t, g.sxyz);
        pair(std::integral_constant<int, 2>{}, z, g.sxy);
        pair(std::integral_constant<int, 1>{}, y, g.L[0]);
        pair(std::integral_constant<int, 0>{}, x, 1);

#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const T f = ((FLAGS & K_G5) && k >= 6) ? -sp.c_hop : sp.c_hop;
            cx<T> w;
            w.x = f * hop[k].x;
            w.y = f * hop[k].y;
            out[k * V + s] = w;
        }
    }
}

}  // namespace ovl
