/*
 * ovl.h -- C-ABI boundary of the B200-native overlap Dirac operator hot path of arXiv 1510.06897
 *          (Cundy & Lee, "Overlap fermions on GPUs").  PAPER.md = /root/reference/PAPER.md.
 *
 * What the library computes (every step runs in hand-written sm_100a kernels; there is no CPU fallback):
 *     y = D[mu] psi = 1/2 (1 + mu + (1 - mu) gamma5 sign(K)) psi                    eq. 2.1
 *     K = gamma5 (D_W - m_w),  m_w = 1.5
 *     (D_W psi)(x) = 4 psi(x) - 1/2 sum_mu [ (1 - gamma_mu) U_mu(x) psi(x + mu)
 *                                          + (1 + gamma_mu) U_mu(x - mu)^dag psi(x - mu) ]
 *                                                                 eq. 2.2, PAPER.md:41 (reading R1)
 *     sign(K) psi ~= sum_{m=0}^{N} alpha_m T_m(K^) psi
 *                    + sum_i phi_i (phi_i^dag psi) [ sign(lambda_i) - sum_m alpha_m T_m(lambda_i / lambda_max) ]
 *                    with K^ = K / lambda_max                     eq. 2.3, PAPER.md:62-64 (reading R5)
 *     CG on D[mu]^dag D[mu] x = b                                 BASELINE.json north_star (d) (R13, R14)
 *
 * Conventions:
 *   dims = {Lx, Ly, Lz, Lt}, every extent >= 2; V = Lx Ly Lz Lt; site index s = x + Lx (y + Ly (z + Lz t)).
 *   Canonical spinor:  [V][spin 4][colour 3] complex, interleaved (re, im).  complex128 when the context was
 *                      created with OVL_F64, complex64 with OVL_F32.
 *   Canonical links:   [V][mu = x,y,z,t][row 3][col 3] complex128, U_mu(x) being exactly the matrix that multiplies
 *                      psi(x + mu) in eq. 2.2.  NO boundary phase folded in: the library applies periodic x,y,z and
 *                      antiperiodic t (the hop across the t boundary carries -1, reading R3).
 *   Eigenvectors:      [nev][V][4][3] complex128 (always fp64 at the boundary; rounded to fp32 inside for OVL_F32).
 *   gamma basis:       Euclidean Hermitian chiral (DeGrand-Rossi), gamma5 = diag(+1,+1,-1,-1) (reading R2,
 *                      tests/golden/gamma_basis.txt).
 *
 * Pointers.  Every `const void *` / `void *` data argument marked [H|D] may be a device pointer (used in place) or
 *   a host pointer (pageable or pinned; the library stages it through its own device buffer with cudaMemcpyAsync on
 *   the context stream and, for outputs, synchronises before returning).  The kind is detected with
 *   cudaPointerGetAttributes.  `alpha`, `lambda`, `dims` and the scalar out-parameters are host memory.
 *
 * Ownership.  The caller owns everything it passes in; the library never frees or keeps caller pointers.  Links and
 *   eigenvectors are re-laid-out into the context's device memory -- the caller's workspace (ovl_create_ws) or
 *   library allocations (ovl_create) -- at create / set time, so the caller may release them afterwards.  `out` must
 *   not alias `psi`.
 *
 * Execution.  All work is enqueued on the stream given to ovl_create.  Calls with device outputs return without
 *   synchronising; ovl_cg, ovl_destroy and any call with a host output synchronise the stream.  A context is
 *   not thread-safe.  Same inputs => bit-identical outputs run to run (fixed reduction trees, no float atomics).
 *
 * Errors.  Every function returns an OVL_* status; nothing throws or prints.  ovl_last_error gives a
 *   human-readable message for the last non-OK status of that context.
 */
#ifndef OVL_H
#define OVL_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ovl_ctx ovl_ctx; /* opaque */

enum { OVL_OK = 0, OVL_EINVAL = 1, OVL_ENOMEM = 2, OVL_ECUDA = 3, OVL_ESTATE = 4, OVL_ENOTCONV = 5 };
enum { OVL_F64 = 0, OVL_F32 = 1 };        /* storage + stencil arithmetic precision (reading R18) */
enum { OVL_RECON18 = 18, OVL_RECON12 = 12 }; /* reals stored per link; 12: third row rebuilt as conj(r0 x r1) */
#define OVL_MAX_RHS 12                        /* right-hand sides per multi call (12 = one propagator's spin-colour sources) */
enum { OVL_REC_CLENSHAW = 0, OVL_REC_FORWARD = 1 }; /* how sum_m alpha_m T_m(K^) psi of eq. 2.3 is evaluated */
enum { OVL_FUSED_REGISTER = 0, OVL_FUSED_BULK = 1, OVL_FUSED_PLAIN = 2, OVL_FUSED_BRICK = 3 }; /* implementation of the fused Wilson / Chebyshev launch */

/* Library version string, e.g. "ovl-b200 0.1 (sm_100a)". */
const char *ovl_version(void);

/* Device bytes of the workspace a context needs for: this lattice / precision / link storage, up to max_nev deflation
 * vectors, up to max_rhs right-hand sides per ovl_overlap_multi / ovl_cg_multi call (1..OVL_MAX_RHS) and an
 * ovl_lowest_eigenpairs work block of eig_block = max(block, 2 nev) vectors (0: the eigensolver is not used; <= 128).
 * It holds the re-laid-out links, the recurrence vectors (S4: "short three vector recurrence"), the CG vectors,
 * the multi-right-hand-side staging, the eigenvector store (S5), the canonical staging for host pointers, the reduction
 * scratch and the eigensolver block.  0 for invalid arguments. */
size_t ovl_workspace_bytes(const int dims[4], int prec, int recon, int max_nev, int max_rhs, int eig_block);
/* = ovl_workspace_bytes(dims, prec, recon, max_nev, 1, 0). */
size_t ovl_device_bytes(const int dims[4], int prec, int recon, int max_nev);

/* Create a context inside a CALLER-OWNED workspace (PyTorch owns device memory): `workspace` is device
 * memory of at least ovl_workspace_bytes(...) bytes for the same capacities, 256-byte aligned, and must stay valid until
 * ovl_destroy, which does not free it.  Every device buffer of the context is carved from it here; NO later call
 * allocates or frees device memory (calls that exceed a capacity -- nev > max_nev, nrhs > max_rhs, an eigensolver block
 * above eig_block -- return OVL_EINVAL), so no call hides a device-wide synchronisation behind an allocation.
 * Links are re-laid-out (S2; SoA site-coalesced planes, optional 12-real compression) before the call returns.
 *   links_c128 [H|D]  canonical links, V*4*9 complex128 (a host array is staged through the workspace).
 *   cuda_stream       a cudaStream_t (0 = legacy default stream); all later work is enqueued there.
 * Defaults: m_w = 1.5, lambda_max = 8 - m_w = 6.5 (reading R5); no polynomial, no deflation.
 * Errors: OVL_EINVAL (null / misaligned / non-device / too small workspace, extent < 2, unknown prec/recon, capacities
 * out of range), OVL_ECUDA. */
int ovl_create_ws(ovl_ctx **out, const int dims[4], const void *links_c128, int prec, int recon, int max_nev, int max_rhs,
                  int eig_block, void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Convenience: the same context with LIBRARY-owned memory.  One cudaMalloc here for the base set (links, recurrence
 * vectors, reduction scratch = ovl_device_bytes(dims, prec, recon, 0) minus the optional parts); further allocations
 * happen only when a capacity is first needed or grows: ovl_set_deflation (eigenvector store), the first ovl_cg*, the
 * first multi-right-hand-side call with a larger nrhs, the first host-pointer call (staging), ovl_lowest_eigenpairs
 * (work block, released on return).  Use ovl_create_ws when allocations inside calls are not acceptable.
 * Errors: OVL_EINVAL (null pointer, extent < 2, unknown prec/recon), OVL_ENOMEM, OVL_ECUDA. */
int ovl_create(ovl_ctx **out, const int dims[4], const void *links_c128, int prec, int recon, void *cuda_stream);

/* Synchronise the stream and free everything the library allocated (never the caller's workspace). */
int ovl_destroy(ovl_ctx *ctx);

/* K = gamma5 (D_W - m_w), K^ = K / lambda_max (R5).  lambda_max > 0. */
int ovl_set_kernel(ovl_ctx *ctx, double m_w, double lambda_max);

/* Chebyshev table of eq. 2.3: alpha[0..degree_N] (host, fp64), degree_N >= 1.  The recurrence is run up to the
 * last non-zero alpha (reading R7); ovl_poly_orders reports that number of K^ applications. */
int ovl_set_chebyshev(ovl_ctx *ctx, int degree_N, const double *alpha);
int ovl_poly_orders(const ovl_ctx *ctx);

/* Evaluation order of the polynomial sum of eq. 2.3 ("a short three vector recurrence").  Both run
 * exactly ovl_poly_orders fused stencil launches and give the same polynomial (they differ by rounding only):
 *   OVL_REC_FORWARD   t_0 = psi, t_1 = K^ psi, t_{m+1} = 2 K^ t_m - t_{m-1}, s = sum_m alpha_m t_m, as printed;
 *   OVL_REC_CLENSHAW  b_k = alpha_k psi + 2 K^ b_{k+1} - b_{k+2} (k = N..1), s = alpha_0 psi + K^ b_1 - b_2: the
 *                     adjoint recurrence, which has no read-modify-write accumulator stream (default).
 * Errors: OVL_EINVAL for an unknown mode. */
int ovl_set_recurrence(ovl_ctx *ctx, int mode);
int ovl_get_recurrence(const ovl_ctx *ctx);

/* Implementation of the fused Wilson-stencil / Chebyshev-step launch ("merging ... into a single GPU kernel";
 * :70-72 on the transfer "from global memory to the registers").  All give bit-identical results.
 *   OVL_FUSED_REGISTER  one thread per site, every operand lands in registers through coalesced 128-bit loads (default:
 *                       the faster one on B200 at every size measured);
 *   OVL_FUSED_BULK      persistent warps; the first-touch stream of a warp's own links lands in shared memory by
 *                       cp.async.bulk with mbarrier completion and is refilled for the warp's next 32 sites while the
 *                       current ones are computed.  Used for single-right-hand-side launches of D_W, K^ and the Clenshaw
 *                       recurrence when V and Lx*Ly*Lz are multiples of 32; other launches use the default kernel.
 *   OVL_FUSED_PLAIN     the register kernel with the CTAs always in plain site order;
 *   OVL_FUSED_BRICK     the register kernel with the CTAs in "brick" order on any lattice with Lz and Lt even (OVL_EINVAL
 *                       otherwise): a CTA takes a 2 x 2 stack in (z, t) of 32-site chunks, so half of the z / t neighbours
 *                       come out of its own L1.  Single-right-hand-side launches only.  Under OVL_FUSED_REGISTER the library
 *                       picks brick order for 2^15 <= V <= 2^17 sites (12^3 x 24 ... 16^3 x 32: 2-5 % faster per order) and
 *                       plain order elsewhere.  Same arithmetic per site, same bits.
 * Kept selectable so that the comparisons (bench.py extras) can be re-measured and the tests can hold every
 * variant against the others. */
int ovl_set_fused_variant(ovl_ctx *ctx, int variant);

/* The polynomial loop is a fixed launch sequence per source field; by default it is captured once into a CUDA graph and
 * replayed (launch overhead 0.5 us instead of 2 us per order).  Graphs need a real stream: a context created on the
 * legacy default stream (cuda_stream = 0) always launches directly.  on = 0 forces direct launches. */
int ovl_set_graphs(ovl_ctx *ctx, int on);

/* Deflation space of eq. 2.3: nev >= 0 vectors phi_c128 [H|D] and eigenvalues lambda (host).
 * nev = 0 switches deflation off.  |lambda_i| < 1e-14 lambda_max is rejected with OVL_EINVAL (reading R9).
 * The vectors are used exactly as given (no re-orthonormalisation; reading R10). */
int ovl_set_deflation(ovl_ctx *ctx, int nev, const void *phi_c128, const double *lambda);

/* out = D_W psi, eq. 2.2 (no m_w shift, no gamma5).  psi, out [H|D] canonical spinors. */
int ovl_dw(ovl_ctx *ctx, const void *psi, void *out);

/* out = K^ psi = gamma5 (D_W - m_w) psi / lambda_max (one fused stencil pass). */
int ovl_khat(ovl_ctx *ctx, const void *psi, void *out);

/* out = sign(K) psi by eq. 2.3 (needs ovl_set_chebyshev; OVL_ESTATE otherwise). */
int ovl_sign(ovl_ctx *ctx, const void *psi, void *out);

/* out = D[mu] psi (dagger = 0, eq. 2.1) or D[mu]^dag psi = 1/2 [(1+mu) psi + (1-mu) sign(K) gamma5 psi]
 * (dagger = 1, reading R12). */
int ovl_overlap(ovl_ctx *ctx, double mu, int dagger, const void *psi, void *out);

/* out_r = D[mu] psi_r (or D[mu]^dag psi_r) for r < nrhs right-hand sides in one call, 1 <= nrhs <= OVL_MAX_RHS
 * (the paper's end use is propagators, i.e. 12 sources per configuration).
 * psi, out [H|D]: nrhs consecutive canonical spinors, [nrhs][V][4][3].  Every launch of the fused Wilson/Chebyshev
 * kernel works on all right-hand sides, so the links (576 of the 1248 B/site/order in fp64) are read from HBM once per
 * tile instead of once per right-hand side; each out_r is bit-identical to what ovl_overlap returns for psi_r.
 * The recurrence workspace grows to 4 * nrhs fields on first use.  Errors: OVL_EINVAL (nrhs out of range, null or
 * aliased pointers), OVL_ESTATE (no polynomial), OVL_ENOMEM. */
int ovl_overlap_multi(ovl_ctx *ctx, int nrhs, double mu, int dagger, const void *psi, void *out);

/* Conjugate gradient on D[mu]^dag D[mu] x = b, x0 = 0, stop when the recursive residual ||r_k|| <= tol ||b||
 * or after maxiter iterations (tol <= 0: exactly maxiter iterations, status OVL_OK).  b, x [H|D] canonical.
 * *iters_out = iterations done, *true_relres_out = ||b - A x|| / ||b|| recomputed at the end.
 * Returns OVL_ENOTCONV (x = last iterate) if tol > 0 was not reached.  Synchronises. */
int ovl_cg(ovl_ctx *ctx, double mu, const void *b, void *x, double tol, int maxiter, int *iters_out,
           double *true_relres_out);

/* CG in one chirality sector ("[D^dag D, gamma5] = 0", one sign application per operator
 * application instead of two; reading R23).  With P_c = (1 + c gamma5)/2, c = chirality = +1 or -1, solves
 *     A_c x = P_c b,   A_c = 1/2 (1 + mu^2) + c/2 (1 - mu^2) P_c sign(K) P_c     ( = P_c D^dag D P_c when sign(K)^2 = 1;
 * for the polynomial of eq. 2.3 the two differ by 1/4 (1-mu)^2 P_c (sign(K)^2 - 1) P_c ),  x0 = 0, same stopping rule and
 * outputs as ovl_cg; x = P_c x.  *true_relres_out = ||P_c b - A_c x|| / ||P_c b||.  b need not be chiral (it is projected);
 * P_c b = 0 returns x = 0 after 0 iterations.  Errors as ovl_cg; OVL_EINVAL for chirality not +-1.  Synchronises. */
int ovl_cg_chiral(ovl_ctx *ctx, double mu, int chirality, const void *b, void *x, double tol, int maxiter, int *iters_out,
                  double *true_relres_out);

/* nrhs independent systems D^dag D x_r = b_r solved in lockstep (1 <= nrhs <= OVL_MAX_RHS): every operator application
 * is one multi-right-hand-side call (see ovl_overlap_multi), alpha, beta and the residual norms are kept per system; a
 * system that has reached tol is frozen while the others iterate.  b, x [H|D]: [nrhs][V][4][3]; iters_out, true_relres_out:
 * host arrays of nrhs entries.  Returns OVL_ENOTCONV if any system is above tol after maxiter iterations.  Synchronises. */
int ovl_cg_multi(ovl_ctx *ctx, int nrhs, double mu, const void *b, void *x, double tol, int maxiter, int *iters_out,
                 double *true_relres_out);

/* ovl_cg_multi in one chirality sector: nrhs systems A_c x_r = P_c b_r (ovl_cg_chiral) in lockstep, one multi-right-hand-
 * side sign application per iteration.  The spin-colour point sources of a propagator are chirality
 * eigenstates: six of the twelve go through chirality +1, six through -1.  Arguments, outputs and errors as ovl_cg_multi;
 * OVL_EINVAL for chirality not +-1.  Synchronises. */
int ovl_cg_multi_chiral(ovl_ctx *ctx, int nrhs, double mu, int chirality, const void *b, void *x, double tol, int maxiter,
                        int *iters_out, double *true_relres_out);

/* Mixed-precision CG on D^dag D x = b ("10^-13 for overlap fermions (using mixed precision)"; SURVEY.md
 * §8(f) rank 2): defect correction x <- x + A32^{-1}(b - A64 x).  ctx64 is an OVL_F64 context and carries b, x (canonical
 * complex128 [H|D]), the outer fp64 residuals and the final accuracy; ctx32 is an OVL_F32 context on the same lattice and
 * the same stream, with its own links / Chebyshev table / deflation set (the table may be of lower degree: the paper's
 * relaxed inner sign function).  Each outer step solves for the unit-normalised residual with the fp32 CG to the relative
 * tolerance inner_tol (at most max_inner iterations) and recomputes the residual in fp64 (two fp64 applies).  Stops when
 * ||b - A64 x|| <= tol ||b||, after max_outer steps, or when an outer step no longer lowers the residual.
 * *outer_out / *inner_total_out = outer steps / fp32 iterations done; *true_relres_out = fp64 ||b - A x|| / ||b||.
 * Returns OVL_ENOTCONV (x = best iterate) if tol was not reached; OVL_EINVAL for mismatched contexts.  Synchronises. */
int ovl_cg_mixed(ovl_ctx *ctx64, ovl_ctx *ctx32, double mu, const void *b, void *x, double tol, double inner_tol,
                 int max_outer, int max_inner, int *outer_out, int *inner_total_out, double *true_relres_out);

/* ovl_cg_mixed in one chirality sector: the system A_c x = P_c b of ovl_cg_chiral (reading R23; SURVEY.md §8(f)
 * ranks 2 and 4 combined) by defect correction with fp32 inner solves -- one sign application per operator application in
 * both precisions.  The outer residual is P_c b - A_c x in fp64.  Arguments, outputs and errors as ovl_cg_mixed;
 * OVL_EINVAL for chirality not +-1.  x = P_c x.  Synchronises. */
int ovl_cg_mixed_chiral(ovl_ctx *ctx64, ovl_ctx *ctx32, double mu, int chirality, const void *b, void *x, double tol,
                        double inner_tol, int max_outer, int max_inner, int *outer_out, int *inner_total_out,
                        double *true_relres_out);

/* The nev eigenpairs of K = gamma5 (D_W - m_w) of smallest |lambda| -- the deflation space of eq. 2.3 (PAPER.md:62, :66:
 * "a polynomial preconditioned implicitly restarted Lanczos routine"; here a Chebyshev-filtered block subspace iteration on
 * K^2 with a Rayleigh-Ritz step on K, which separates +lambda from -lambda).  OVL_F64 contexts.
 *   tol            stop when ||K phi_i - lambda_i phi_i|| <= tol for all i < nev (phi_i normalised)
 *   max_cycles     filter + Rayleigh-Ritz cycles at most;  filter_degree: Chebyshev degree in K^2 per cycle (0 = 100)
 *   block          trial vectors (0 = nev + max(8, nev/2); at most 128).  A block that ends inside a cluster of
 *                  (near-)degenerate eigenvalues converges slowly: choose it to reach past the cluster.
 *   phi_out [H|D]  nev canonical complex128 spinors [nev][V][4][3], orthonormal; lambda_out, resid_out (may be NULL):
 *                  host arrays of nev entries, sorted by |lambda|; *cycles_out = cycles done.
 * Device memory: 3 * block fields on top of the context, released on return.  Deterministic (fixed start vectors).
 * Returns OVL_ENOTCONV (best Ritz pairs returned) if tol was not reached.  Synchronises. */
int ovl_lowest_eigenpairs(ovl_ctx *ctx, int nev, double tol, int max_cycles, int filter_degree, int block, void *phi_out,
                          double *lambda_out, double *resid_out, int *cycles_out);

/* The same eigensolver with the Chebyshev filter -- more than 90 % of its run time -- on the fp32 stencil kernels of a sibling
 * context while the block is far from the tolerance (PAPER.md:66 names the polynomial preconditioning, :110 the mixed
 * precision).  ctx32 is an OVL_F32 context on the same lattice, stream, m_w and lambda_max
 * (its links are the same links rounded to fp32).  A filter cycle runs in fp32 while the largest residual of the wanted
 * pairs is above 1e-5 lambda_max (and fp32 cycles keep gaining at least a factor 3): the filter only has to damp the unwanted part of the spectrum by e^-8 per cycle; the
 * trial block, the Rayleigh-Ritz steps, the residuals and the final diagonalisation of K stay in fp64, and the cycles below
 * that threshold run entirely in fp64, so the returned pairs meet the same tol.  The fp32 recurrence is rescaled step by
 * step (T_d grows like 1e172 in the first cycles from a random start), at no extra cost.
 * Arguments and results as ovl_lowest_eigenpairs; *f32_cycles_out (may be NULL) = cycles whose filter ran in fp32.
 * Errors: additionally OVL_EINVAL for mismatched contexts.  Synchronises. */
int ovl_lowest_eigenpairs_mixed(ovl_ctx *ctx64, ovl_ctx *ctx32, int nev, double tol, int max_cycles, int filter_degree,
                                int block, void *phi_out, double *lambda_out, double *resid_out, int *cycles_out,
                                int *f32_cycles_out);

const char *ovl_last_error(const ovl_ctx *ctx);

/* ---- the lattice split along t over several GPUs --------------------------------------
 * The paper ran this decomposition on 2 GPUs over MPI (PAPER.md:82-88 Table 3, :99-102 Table 4, :108).  An ovl_group is
 * nslabs slab contexts in THIS process: slab r owns the time slices [r Lt/nslabs, (r+1) Lt/nslabs) of every field, runs
 * on cuda_streams[r] and on device devices[r] (NULL: all on the current device -- several slabs on one GPU is the
 * single-GPU test configuration).  There is no separate exchange step: each fused stencil launch stores the boundary
 * time slices of its output straight into the neighbour slabs' halo buffers (peer stores over NVLink when the slabs are
 * on different GPUs; peer access is enabled here), reads the t-neighbours of its own boundary sites from its halos, and is
 * ordered against its two neighbours by events only (no kernel spins on a flag).  The antiperiodic t phase (reading R3)
 * is applied by the slabs that own t = 0 and t = Lt-1.  Deflation coefficients and CG scalars are summed over slabs in slab
 * order by every slab (peer reads).
 * Results: D_W, K^ and the polynomial part of eq. 2.3 are BIT-IDENTICAL to the undivided lattice (same arithmetic per
 * site); with deflation or in CG the reductions are partitioned differently and agree to rounding (~1e-15 relative).
 * Arguments are GLOBAL canonical arrays [H|D] exactly as for the ovl_* calls of the undivided lattice (device pointers
 * must be readable from every slab's device); slab r works on its contiguous t-range of them.  Every group call that
 * produces a field synchronises all slab streams before returning.  Only the Clenshaw evaluation order is offered.
 * Requirements: 1 <= nslabs <= 16, Lt % nslabs == 0, Lt / nslabs >= 2.  Errors as the corresponding ovl_* calls;
 * ovl_group_last_error names the slab. */
typedef struct ovl_group ovl_group;
int ovl_group_create(ovl_group **out, const int dims[4], int nslabs, const void *links_c128, int prec, int recon,
                     void *const *cuda_streams, const int *devices);
int ovl_group_destroy(ovl_group *g);
int ovl_group_slabs(const ovl_group *g);
/* Split every stencil round of a slab into a boundary launch (its first and last time slice: every halo read and every
 * push to the neighbours) and an interior launch, with the round's event recorded in between: the neighbours' next round
 * then overlaps this slab's interior, which hides the cross-GPU event latency.  Same results bit for bit.  Default: on
 * when the slabs sit on different devices, off when they share one. */
int ovl_group_set_split_launch(ovl_group *g, int on);
int ovl_group_set_kernel(ovl_group *g, double m_w, double lambda_max);
int ovl_group_set_chebyshev(ovl_group *g, int degree_N, const double *alpha);
int ovl_group_set_deflation(ovl_group *g, int nev, const void *phi_c128, const double *lambda);
int ovl_group_dw(ovl_group *g, const void *psi, void *out);
int ovl_group_khat(ovl_group *g, const void *psi, void *out);
int ovl_group_sign(ovl_group *g, const void *psi, void *out);
int ovl_group_overlap(ovl_group *g, double mu, int dagger, const void *psi, void *out);
int ovl_group_cg(ovl_group *g, double mu, const void *b, void *x, double tol, int maxiter, int *iters_out, double *true_relres_out);
/* ONE PROCESS PER GPU (the torchrun model): each process creates the group object of ITS slab, the processes swap the
 * export blobs (OVL_SLAB_BLOB_BYTES each; e.g. torch.distributed.all_gather) and connect.  After that the ovl_group_* calls
 * above work unchanged, with LOCAL arguments: this rank's contiguous t-range of every canonical field / eigenvector, and
 * every rank must make the same calls in the same order (they are collective).  The wiring is the in-process one moved
 * behind CUDA IPC: the neighbours' halo buffers and every rank's reduction scratch are opened with cudaIpcOpenMemHandle
 * (the fused kernels then store into / read from them directly over NVLink), the round events are interprocess events,
 * and because a wait on an IPC event only covers records ISSUED before it, every process publishes the number of rounds it
 * has issued in a small POSIX shared-memory segment (`shm_name`, the same string on every rank, unique per group) which
 * the neighbours' host threads poll before they enqueue their wait.  No kernel spins; NCCL is not on the data path.
 *   ovl_slab_create   links_local_c128 [H|D]: this rank's [V/nranks][4][3][3] complex128 links; cuda_stream: a real stream.
 *   ovl_slab_export   fills `blob` (OVL_SLAB_BLOB_BYTES) with this rank's IPC handles.
 *   ovl_slab_connect  `blobs`: nranks blobs in rank order; opens the other ranks' memory and events and sends this rank's
 *                     last U_t time slice to its upper neighbour.  The caller must run a barrier across the processes
 *                     after ovl_slab_connect and before the first collective call, and before ovl_group_destroy.
 * Single node (CUDA IPC + POSIX shm).  Tested as two processes sharing one GPU; unmeasured across GPUs. */
#define OVL_SLAB_BLOB_BYTES 256
int ovl_slab_create(ovl_group **out, const int dims[4], int rank, int nranks, const void *links_local_c128, int prec, int recon,
                    void *cuda_stream, const char *shm_name);
int ovl_slab_export(ovl_group *g, void *blob);
int ovl_slab_connect(ovl_group *g, const void *blobs);
const char *ovl_group_last_error(const ovl_group *g);
long long ovl_group_launch_count(const ovl_group *g);

/* ---- native-layout fields (benchmark / solver plumbing: no relayout passes inside the timed calls) -------------
 * A native field is an opaque device buffer of ovl_field_bytes(ctx) bytes owned by the caller (device memory). */
size_t ovl_field_bytes(const ovl_ctx *ctx);
int ovl_field_import(ovl_ctx *ctx, const void *canonical /*[H|D]*/, void *native /*D*/);
int ovl_field_export(ovl_ctx *ctx, const void *native /*D*/, void *canonical /*[H|D]*/);
int ovl_dw_native(ovl_ctx *ctx, const void *in_native, void *out_native);
int ovl_overlap_native(ovl_ctx *ctx, double mu, int dagger, const void *in_native, void *out_native);
/* nrhs consecutive native fields (nrhs * ovl_field_bytes bytes each side), see ovl_overlap_multi */
int ovl_overlap_multi_native(ovl_ctx *ctx, int nrhs, double mu, int dagger, const void *in_native, void *out_native);

/* ---- measurement hooks ------------------------------------------------------------------------------------------
 * With profiling on, ovl_sign / ovl_overlap(_native) bracket the polynomial loop (the launches of the fused
 * Wilson+Chebyshev kernel) with CUDA events on the context stream.  ovl_last_poly_timing synchronises
 * those events and returns the loop's device time in ms and the number of fused-kernel launches in it. */
int ovl_set_profiling(ovl_ctx *ctx, int on);
int ovl_last_poly_timing(ovl_ctx *ctx, float *ms_out, int *launches_out);
/* Loop times of the last min(max_n, 64, loops profiled since ovl_set_profiling) profiled polynomial loops, oldest first
 * (one event pair per loop, kept in a ring of 64): ms_out[0..*n_out).  Synchronises those events.  OVL_ESTATE if no loop
 * has been profiled yet. */
int ovl_poly_timings(ovl_ctx *ctx, int max_n, float *ms_out, int *n_out);
/* Total kernels this context has launched since creation (bench.py's gpu_launches). */
long long ovl_launch_count(const ovl_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* OVL_H */
