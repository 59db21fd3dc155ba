/* =====================================================================================
 * qxd.h -- C ABI of the B200-native clover-Wilson QCD+QED Dirac solver with C* boundaries.
 *
 * The library solves D_w psi = eta for the O(a)-improved Wilson-Dirac operator
 * with U(3) hopping links e^{i q A_mu(x)} U_mu(x), the
 * SU(3)+U(1) Sheikholeslami-Wohlert (clover) term and C* spatial boundary
 * conditions realised as a lattice doubled in direction 1 with shifted boundaries
 * (PAPER.md:137).  The operator itself is never written in the paper; the definition used is
 * recorded in DESIGN.md "Readings" (R1..R18).  The paper's own boundary is
 * invertQuda(void* h_x, void* h_b, param) on host arrays in application order
 * (PAPER.md:73-79); this ABI keeps that spirit ("interfacing only a minimal set of
 * parameters"): plain pointers and sizes, no C++/torch types.
 *
 * Conventions common to all calls
 *  - Every function returns a qxd_status (0 = QXD_OK).  No exceptions, no abort, no stdout.
 *    qxd_last_error(ctx) gives a human-readable message for the last failing call.
 *  - Pointers marked DEVICE are CUDA device pointers owned by the caller (PyTorch tensors);
 *    pointers marked HOST are host pointers.  The library never allocates device memory: the
 *    caller provides one workspace (qxd_workspace_bytes / qxd_workspace_bind).
 *  - Calls enqueue work on the bound CUDA stream (qxd_set_stream; default stream 0).  Only
 *    qxd_solve*, the *_host variants and the qxd_blas_* reductions synchronise that stream.
 *  - A context is not thread-safe: use it from one host thread at a time (different contexts are independent).
 *  - Natural ("application") order, used by every non-packed entry point:
 *      site index  Lambda(x) = L3 L2 X1 x0 + L3 L2 x1 + L3 x2 + x3        (Eq. (1))
 *      with x = (t,x,y,z) and X1 = 2*L1 if C* is on (extended lattice) else L1;
 *      spinor  [V][4 spin][3 colour] complex fp64 (re,im), colour fastest;
 *      links   [V_phys][4 mu][3][3] complex fp64 row-major, the 4 FORWARD links of every site
 *              of the PHYSICAL lattice T x L1 x L2 x L3 (the "common convention" of
 *              PAPER.md:51; row-major a,b as PAPER.md:133);
 *      A       [V_phys][4 mu] real fp64;
 *      clover  [V][2 chirality][36] real fp64: 6 diagonal reals, then (re,im) of the 15
 *              strictly-upper-triangular entries in row-major order;
 *      even-sublattice fields [V/2][4][3]: the even sites (sum of coordinates even,
 *              PAPER.md:97) in increasing Lambda order.
 *  - Packed order is the library's device layout: even-odd,
 *    tiled, structure-of-arrays in 16-byte chunks.  Packed buffers are opaque; their sizes
 *    come from qxd_packed_spinor_bytes.
 * ===================================================================================== */
#ifndef QXD_H
#define QXD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qxd_ctx qxd_ctx; /* opaque, host-side; holds borrowed device pointers only */

typedef enum {
  QXD_OK = 0,
  QXD_EINVAL = -1,     /* bad argument (odd extent, extent < 2, null pointer, unknown enum ...) */
  QXD_ESTATE = -2,     /* call out of order (e.g. apply before clover_build)                    */
  QXD_EWORKSPACE = -3, /* workspace missing, misaligned or too small                            */
  QXD_ECUDA = -4,      /* a CUDA runtime call or kernel launch failed                            */
  QXD_ENOCONV = -5     /* solver hit maxiter or broke down; psi and info still hold the best iterate */
} qxd_status;

typedef enum { QXD_F64 = 0, QXD_F32 = 1, QXD_F16 = 2 } qxd_prec;
#define QXD_PREC_MASK(p) (1 << (p))

typedef enum { QXD_CGNE = 0, QXD_BICGSTAB = 1, QXD_GCR = 2, QXD_DFL_GCR = 3 } qxd_algo;

/* Solver controls (in) and report (out).  Zero-initialise for defaults. */
typedef struct {
  /* in */
  int algo;          /* qxd_algo; CG on the normal equations of D-hat, BiCGstab on D-hat, or SAP-preconditioned
                        flexible GCR on the full-lattice D_w (needs qxd_set_gcr before qxd_workspace_bind)      */
  int sloppy;        /* qxd_prec of the inner iteration; QXD_F64 = plain double-precision solver   */
  double delta;      /* reliable-update threshold: true residual recomputed in fp64 whenever the
                        iterated residual has dropped below delta * (max since last update);
                        0 -> default 0.1 (ref [4])                                    */
  int maxiter;       /* 0 -> 10000                                                                  */
  /* out */
  int iters;         /* inner iterations done                                                       */
  int n_reliable;    /* reliable updates done                                                       */
  double true_res;   /* final fp64 ||eta-hat_e - D-hat psi_e|| / ||eta||  (= ||eta - D_w psi||/||eta||) */
  double seconds;    /* wall time of the call measured with CUDA events on the bound stream         */
} qxd_solve_info;

/* ---- geometry --------------------------------
 * T,L1,L2,L3: PHYSICAL extents, all even and >= 2.  bc = cstar | (antiperiodic_time << 2), with
 * cstar in 0..3 = number of spatial directions 1..cstar with C* boundary conditions (direction 1
 * is doubled when cstar > 0; directions 2..cstar wrap with the shift x1 -> x1 + L1 mod 2 L1).
 * All site indices are computed on the fly by pure inlined functions. */
int qxd_geometry_create(int T, int L1, int L2, int L3, int bc, qxd_ctx** out);
int qxd_geometry_destroy(qxd_ctx* ctx);
/* Optional: the device site order (the paper's host code orders sites in cache
 * blocks).  Tile extents b (powers of two dividing the extended extents, b3 >= 2): the
 * sites one CTA works on.  Block extents B (powers of two, multiples of b, dividing the extents): tiles
 * are visited block by block, blocks lexicographically with direction 0 slowest.  qxd_set_tile keeps the
 * current block where it is still a multiple of the tile, else sets B = b.  Both must precede
 * qxd_workspace_bind.  Default: chosen by the library.  The order only permutes sites in memory.  In the C*-paired
 * layout (the default for C* geometries, see qxd_set_cstar_pairing) the site order runs over the PHYSICAL lattice, so
 * b1 and B1 must divide L1; qxd_set_cstar_pairing resets tile and block to the defaults of the layout it selects. */
int qxd_set_tile(qxd_ctx* ctx, int b0, int b1, int b2, int b3);
int qxd_set_block(qxd_ctx* ctx, int B0, int B1, int B2, int B3);
/* Number of sites of the extended lattice (V). */
/* C*-paired device layout: the DEFAULT for C* geometries (on = 0 selects the extended-lattice layout; call before
 * qxd_workspace_bind; on = 1 without a C* direction -> QXD_EINVAL).  A site of the extended lattice and its mirror
 * image x + L1 e1 carry the same gauge information (U^*, -A, R8), so links and clover blocks are stored
 * once per PHYSICAL site and the two sites are processed by neighbouring threads that share every link and clover load: the
 * traffic of the even-odd operator drops from 488 to 248 reals per even site (14-real links).  Results are unchanged (same
 * arithmetic per site up to the conjugations); the natural-order ABI is unchanged. */
int qxd_set_cstar_pairing(qxd_ctx* ctx, int on);
long qxd_volume(const qxd_ctx* ctx);
/* Introspection of the device site order (host-only, no GPU needed; used by the CPU tests of row a1).
 * qxd_site_index: extended coordinates x[4] -> checkerboard index cb in [0,V/2) and parity (sum of coordinates mod 2).
 * qxd_site_coords: the inverse.  qxd_site_neighbour: checkerboard index (of the opposite parity) of x + dir*mu-hat,
 * dir = +1/-1, with the boundary rules of reading R8 (shifted C* boundaries); the same inlined
 * function the kernels use.  All return QXD_EINVAL on out-of-range arguments. */
int qxd_site_index(const qxd_ctx* ctx, const int x[4], int* cb, int* parity);
int qxd_site_coords(const qxd_ctx* ctx, int cb, int parity, int x[4]);
int qxd_site_neighbour(const qxd_ctx* ctx, int cb, int parity, int mu, int dir, int* cb_nb);

/* ---- workspace and stream --------------------------------------------------------------------
 * prec_mask: OR of QXD_PREC_MASK(p) for every precision that will be used (QXD_F64 is always
 * included).  nrhs >= 1: right-hand sides of qxd_solve_multi.  The buffer must be 256-byte aligned
 * DEVICE memory and stay alive until qxd_geometry_destroy. */
size_t qxd_workspace_bytes(const qxd_ctx* ctx, int prec_mask, int nrhs);
int qxd_workspace_bind(qxd_ctx* ctx, void* dev /*DEVICE*/, size_t bytes, int prec_mask, int nrhs);
int qxd_set_stream(qxd_ctx* ctx, void* cuda_stream /* cudaStream_t, e.g. torch stream .cuda_stream */);

/* ---- gauge field (row a2) -------------------------------------------------
 * U_su3: DEVICE, natural order on the physical lattice; A_u1: DEVICE or NULL (QCD only);
 * qel: elementary charge unit of the compact U(1) clover term (reading R5), ignored if A_u1 NULL.
 * The library builds the mirror half (U^*, -A) itself. */
int qxd_gauge_load(qxd_ctx* ctx, const double* U_su3, const double* A_u1, double qel);
/* Quark parameters (reading R6): m0 = 1/(2 kappa) - 4, charge q in the hop phase e^{i q A}.
 * Builds the hopping links W = e^{iqA} U (time-boundary sign folded in) in every bound precision. */
int qxd_set_quark(qxd_ctx* ctx, double kappa, double q);

/* ---- field-status manager --------------------------------------
 * Inside an HMC trajectory the gauge field changes while kappa, q, c_sw stay: the hopping links and the clover term
 * (with its inverse) are DERIVED fields that must follow it.  By default every setter regenerates (qxd_set_quark) or
 * invalidates (qxd_gauge_load: set_quark and clover_build must be called again, else QXD_ESTATE) what depends on it.
 * With lazy refresh ON the setters only record their parameters and mark the derived fields stale; the first call that
 * reads them (any apply, solve, qxd_clover_export, or qxd_refresh) regenerates them on the bound stream, once, from the
 * recorded parameters -- a trajectory is then  qxd_gauge_load; qxd_solve; qxd_gauge_load; qxd_solve; ...
 * Turning it OFF regenerates whatever is stale.  qxd_field_status: *status = OR of QXD_FS_*; counts (may be NULL):
 * [0] hopping-link regenerations, [1] clover build+inversion passes since qxd_geometry_create. */
enum { QXD_FS_GAUGE = 1, QXD_FS_HOPLINKS = 2, QXD_FS_CLOVER = 4, QXD_FS_HOPLINKS_STALE = 8, QXD_FS_CLOVER_STALE = 16, QXD_FS_LAZY = 32 };
int qxd_set_lazy_refresh(qxd_ctx* ctx, int on);
int qxd_refresh(qxd_ctx* ctx);
int qxd_field_status(const qxd_ctx* ctx, int* status /*HOST*/, long counts[2] /*HOST or NULL*/);

/* ---- clover term (row a3) -----------------------------------------
 * Builds M(x) = (4+m0) + c_sw (i/4) sigma.F-hat + q c_sw_qed (i/4) sigma.A-hat as two Hermitian
 * 6x6 blocks per site and inverts both blocks, on the device.  Needs gauge + quark. */
int qxd_clover_build(qxd_ctx* ctx, double csw, double csw_qed);
/* How the 6x6 block inverses were obtained so far (HOST counts[2]): [0] parity passes of the unpivoted in-register
 * Gauss-Jordan (the fast path: the blocks are (4 + m0) + O(c_sw F), diagonally dominant for every sensible field),
 * [1] parity passes redone with the partially pivoted kernel because a pivot fell below 1e-6 of the largest diagonal entry. */
int qxd_clover_stats(const qxd_ctx* ctx, long counts[2] /*HOST*/);
/* Storage format of the hopping links W = e^{iqA} U (north_star "12-real SU(3) reconstruct and the U(1)
 * phase fused into the link multiply").  QXD_RECON_NONE: all 18 reals of W.  QXD_RECON_12: rows 0 and 1 of W (12 reals)
 * plus det W = e^{3iqA} det U (x -1 on the antiperiodic time boundary) as (re, im) = 14 reals per link; the dslash rebuilds
 * row 2 = det W * conj(row0 x row1), which holds for every unitary W, so the phase costs no separate multiply.  Traffic per
 * D_w site drops from 192 to 176 reals.  The input links must be unitary to the working precision (they are only used
 * through this identity); det U is computed, not assumed to be 1.  May be called at any time; if a quark is set the links
 * of every bound precision are rewritten in the new format.  Other values -> QXD_EINVAL.  The _prec form sets the
 * format of one storage precision only (measured on B200: the 14-real format is faster in fp64 and fp32, where the
 * dslash is bandwidth bound, and slower in fp16, where it is bound by instruction issue). */
enum { QXD_RECON_NONE = 18, QXD_RECON_12 = 12 };
int qxd_set_gauge_reconstruct(qxd_ctx* ctx, int recon);
int qxd_set_gauge_reconstruct_prec(qxd_ctx* ctx, int prec, int recon);
/* Copy the fp64 clover field (inverse != 0: the block inverses) to natural order, out: DEVICE
 * [V][2][36] doubles, packing of PAPER.md:117. */
int qxd_clover_export(qxd_ctx* ctx, double* out, int inverse);

/* ---- operator applications, natural order (rows a4, a5) -----------------------------------------
 * psi/out: DEVICE fp64 natural-order spinors on the extended lattice; prec selects the storage
 * precision of the fields the kernel streams (fp64 arithmetic for QXD_F64, fp32 otherwise). */
int qxd_apply_Dw(qxd_ctx* ctx, int prec, const double* psi, double* out);
/* D-hat = A_ee - D_eo A_oo^{-1} D_oe on the even sublattice; dagger != 0 applies D-hat^dagger. */
int qxd_apply_Dhat_eo(qxd_ctx* ctx, int prec, const double* psi_e, double* out_e, int dagger);
/* Same as qxd_apply_Dw but psi/out are HOST arrays (pinned memory for full speed; the paper's boundary).
 * The lattice is processed in time slabs of one tile thickness: copy-in, pack, apply, unpack and copy-out of different
 * slabs overlap on three streams, so the two PCIe directions run at the same time.  Synchronises before returning. */
int qxd_apply_Dw_host(qxd_ctx* ctx, int prec, const double* psi_host, double* out_host);

/* ---- solver (rows a7, a8) --------------------------------------------------------
 * Solves D_w psi = eta to ||eta - D_w psi|| <= tol ||eta|| (checked in fp64 on the even-odd system).
 * eta, psi: DEVICE natural order (qxd_solve) or HOST (qxd_solve_host).  info may be NULL (defaults).
 * On QXD_ENOCONV psi holds the best iterate and info->true_res its residual. */
int qxd_solve(qxd_ctx* ctx, const double* eta, double* psi, double tol, qxd_solve_info* info);
int qxd_solve_host(qxd_ctx* ctx, const double* eta_host, double* psi_host, double tol, qxd_solve_info* info);

/* ---- SAP-preconditioned GCR ("heavily preconditioned GCR ... Schwarz alternating
 * procedure"; precisions PAPER.md:168-170) ---------------------------------------------------------------------------
 * qxd_solve with algo = QXD_GCR solves the full-lattice system D_w psi = eta by a flexible, restarted GCR(nkv):
 *   per step  z_k = M_sap r ;  w_k = D_w z_k  (fp32) ;  w_k orthonormalised against w_0..w_{k-1} ;  r -= <w_k, r> w_k
 *   restart   psi += sum_k y_k z_k in fp64 (y from the triangular system of the orthogonalisation coefficients), and the
 *             true residual eta - D_w psi is recomputed in fp64 (after nkv steps, or when the fp32 residual has dropped by
 *             1e-4 within the cycle, or looks converged); convergence is only ever declared on that fp64 residual.
 * M_sap = ncy cycles of the multiplicative Schwarz alternating procedure over a two-colouring of blocks: a block is one
 * 128-index tile of both parities (256 sites: 4x4x4x4, or 2x4x4x4 with both C* mirror images in the paired layout) with
 * Dirichlet boundaries; on each block nmr minimal-residual steps on D_w restricted to the block, run by ONE thread block
 * entirely out of shared memory (links and clover blocks of the block staged once per visit, storage precision
 * info->sloppy = QXD_F16 or QXD_F32; residual and correction in fp32); the residual of the neighbouring blocks is
 * corrected lazily from the stored corrections when they are visited.  info->delta is ignored; info->iters counts GCR
 * steps, info->n_reliable the fp64 restarts.
 * qxd_set_gcr: nkv = 0 releases the Krylov space (default; QXD_GCR then returns QXD_EWORKSPACE), else 1 <= nkv <= 32,
 * ncy >= 1, nmr >= 1 (0 = defaults ncy 4, nmr 4).  Must precede qxd_workspace_bind (the 2 nkv + 3 fp32 full-lattice
 * vectors are part of the workspace).  Geometries whose tiles admit no two-colouring (an odd number of blocks in a
 * direction) are rejected with QXD_EINVAL by qxd_solve.
 * qxd_apply_sap: out = M_sap in on fp32 packed full-lattice spinors (test and bench entry point of the preconditioner). */
int qxd_set_gcr(qxd_ctx* ctx, int nkv, int ncy, int nmr);
/* Second level (deflated SAP-GCR on the CPU, multigrid GCR on the GPU): local-coherence deflation on the SAP blocks.
 *   qxd_set_deflation    ns null vectors (even, <= 32; 0 = off), ninv smoothing passes in the setup (0 = default 4), nkc GCR steps of
 *                        every coarse-grid solve (0 = default 16), nref rounds of adaptive refinement in the setup (every null
 *                        vector replaced by the current two-level preconditioner applied to it, space and coarse operator rebuilt;
 *                        needs ns <= 2 nkv); before qxd_workspace_bind; needs qxd_set_gcr too.
 *   qxd_set_deflation_chirality   on = 1: every null vector is split into its two chirality components (upper / lower two spin
 *                        components in the chiral basis of reading R3), the aggregation of the multigrid solvers the paper's GPU runs
 *                        use: the deflation space is span{P_b P_chi phi_i}, 2 ns complex dimensions per block for ns smoothed
 *                        vectors (ns <= 16), and gamma5 maps it onto itself.  Before qxd_workspace_bind.  Default 0.  With the split
 *                        qxd_deflation_info reports 2 ns and the coarse vectors of qxd_deflation_op are [nblocks][2 ns], index
 *                        2 i + chi.
 *   qxd_set_deflation_refine   nref refinement rounds (replaces the nref of qxd_set_deflation) and what a round does to every null
 *                        vector: steps = 1 (default) applies the current two-level preconditioner once; steps > 1 is an inverse
 *                        iteration, phi_i <- `steps` steps of the deflated flexible GCR on D_w x = phi_i in fp32 (no convergence
 *                        test, no host round trip); after every round the space is re-orthonormalised and the coarse operator
 *                        rebuilt.  Needs ns <= 2 (nkv - steps) (checked by qxd_deflation_setup, QXD_EWORKSPACE).  May be called at
 *                        any time; takes effect at the next qxd_deflation_setup.  Pays where D_w is close to singular with a
 *                        well-defined sign of the real parts of its spectrum; off by default.
 *   qxd_deflation_setup  random_vectors: DEVICE, ns packed fp32 full-lattice spinors back to back (the caller draws them; any
 *                        linearly independent set works).  Each is smoothed by ninv applications of M_sap (block operator in storage
 *                        precision prec = QXD_F32 / QXD_F16), the set is orthonormalised block by block, and the coarse operator
 *                        A_c = R D_w P (nine-point stencil of ns x ns complex matrices per block) is built.  Must be repeated after
 *                        every change of the gauge field, the quark or the clover coefficients (else QXD_ESTATE).
 *   qxd_solve            with algo = QXD_DFL_GCR: the flexible GCR of QXD_GCR with the two-level preconditioner
 *                            z = P A_c^{-1} R r + M_sap (r - D_w P A_c^{-1} R r),   A_c^{-1} ~ nkc GCR steps on the even-odd
 *                        (Schur) form of the coarse system: the blocks are two-coloured and the nine-point operator only joins
 *                        opposite colours, so x_e solves (1 - Dinv_e H_eo Dinv_o H_oe) x_e = Dinv_e (b_e - H_eo Dinv_o b_o) and
 *                        x_o = Dinv_o (b_o - H_oe x_e); the hop matrices and the inverses Dinv of the diagonal blocks are read
 *                        from a binary16 copy (a preconditioner: the outer flexible GCR absorbs the rounding).
 *   qxd_deflation_info   number of blocks, ns, and whether the setup is valid.
 *   qxd_deflation_op     test entry: op 0  coarse = R fine;  1  fine = P coarse;  2  coarse_out = A_c coarse_in (fp32 operator);
 *                        3  fine_out = two-level preconditioner applied to fine_in;  4  coarse_out = the coarse solver applied to
 *                        coarse_in (~ A_c^{-1} coarse_in).  fine: DEVICE packed fp32 full-lattice spinor; coarse: DEVICE [nblocks][ns]
 *                        complex fp32 (block index = checkerboard index >> 7). */
int qxd_set_deflation(qxd_ctx* ctx, int ns, int ninv, int nkc, int nref);
int qxd_set_deflation_chirality(qxd_ctx* ctx, int on);
int qxd_set_deflation_refine(qxd_ctx* ctx, int nref, int steps);
int qxd_deflation_setup(qxd_ctx* ctx, int prec, const void* random_vectors /*DEVICE*/);
int qxd_deflation_info(const qxd_ctx* ctx, int* nblocks, int* ns, int* ready);
int qxd_deflation_op(qxd_ctx* ctx, int op, const void* in, void* out);
/* Host-only introspection of the SAP block decomposition (no GPU needed; CPU tests of reading R21): block index (= cb >> 7) and
 * colour (0 / 1) of the site (cb, parity).  QXD_EINVAL if the geometry admits no two-colouring (qxd_last_error says why). */
int qxd_sap_block_of(qxd_ctx* ctx, int cb, int parity, int* block, int* colour);
int qxd_apply_sap(qxd_ctx* ctx, int prec, const void* in /*DEVICE, packed fp32*/, void* out /*DEVICE, packed fp32*/);

/* ---- batched solve (rows a7 + a10; "for many right-hand sides"; BASELINE config 4) -------------------
 * nrhs (<= the nrhs the workspace was bound with, <= 64) systems with the same operator: eta, psi are DEVICE arrays
 * [nrhs][V][4][3] complex fp64 in natural order (psi may be the same buffer as eta).  The CG iterations on the normal
 * equations run in lockstep so that every sloppy operator application is ONE multi-RHS dslash launch that reads each
 * link and clover block once for all right-hand sides; each system has its own scalars and reliable updates and is
 * frozen once its fp64 residual meets tol.  info: array of nrhs entries; algo (QXD_CGNE only), sloppy, delta, maxiter
 * are read from info[0]; every entry receives that system's iters, n_reliable, true_res (seconds = whole call).
 * Returns QXD_ENOCONV if any system missed tol (its best iterate and true residual are still returned). */
int qxd_solve_multi(qxd_ctx* ctx, int nrhs, const double* eta, double* psi, double tol, qxd_solve_info* info);

/* ---- packed-layout entry points (row a9; benchmark and building blocks) ---------------------------
 * Packed spinors: parity 0 (even) half followed by the parity 1 half; `half_only` != 0 gives the size
 * of one parity.  For QXD_F16 each half is 24 binary16 per site plus one fp32 scale per site. */
size_t qxd_packed_spinor_bytes(const qxd_ctx* ctx, int prec, int half_only);
int qxd_spinor_pack(qxd_ctx* ctx, int prec, const double* nat /*DEVICE [V][4][3]*/, void* packed /*DEVICE*/);
int qxd_spinor_unpack(qxd_ctx* ctx, int prec, const void* packed, double* nat);
int qxd_apply_Dw_packed(qxd_ctx* ctx, int prec, const void* in, void* out);
int qxd_apply_Dhat_packed(qxd_ctx* ctx, int prec, const void* in_e, void* out_e, int dagger);
/* Alternative kernel for qxd_apply_Dw_packed in fp32 (18-real links, extended-lattice layout, 4^4 tiles, extents multiples of
 * (4, 8, 8, 4)): a CTA owns an 8 x 8 x 4 spatial footprint and sweeps tseg time slices, keeping the slices t-1, t, t+1 of its
 * footprint in a shared-memory ring filled by cp.async two slices ahead, so that time neighbours and in-footprint spatial
 * neighbours never go back to L2 / DRAM.  tseg = 0 (default): the tile kernel; tseg >= 2: the sweep kernel where
 * it applies (silently the tile kernel elsewhere).  Same results up to the summation order of nothing: identical arithmetic. */
int qxd_set_dw_sweep(qxd_ctx* ctx, int tseg);
/* Multi-RHS D_w (row a10): in/out hold nrhs packed full-lattice spinors back to back, qxd_packed_spinor_bytes(prec,0)
 * apart.  One launch: the CTAs working on the same tile for different right-hand sides are consecutive, so the links
 * and clover blocks of a tile come from DRAM once and from L2 afterwards; every thread applies its site's links and
 * clover blocks to r right-hand sides (qxd_set_rhs_per_thread: 0 = library default (1), 1..3; fp64 always 1). */
int qxd_apply_Dw_multi_packed(qxd_ctx* ctx, int prec, int nrhs, const void* in, void* out);
int qxd_set_rhs_per_thread(qxd_ctx* ctx, int r);
/* EXPERIMENTAL variant of qxd_apply_Dw_multi_packed with the right-hand sides ACROSS LANES (csrc/dslash_ilv.cu): nrhs (a
 * multiple of 4) spinors are stored in groups of four, chunk c of site cb of right-hand side j of a group at vector index
 * (c Vh + cb) 4 + j, so that the four lanes of a site share every link and clover load.  qxd_multi_interleave converts between
 * nrhs plain packed spinors (back to back) and that layout (to_interleaved != 0) or back; same total size.  Same arithmetic per
 * site and right-hand side as the plain batch: identical results. */
int qxd_multi_interleave(qxd_ctx* ctx, int prec, int nrhs, void* plain /*DEVICE*/, void* interleaved /*DEVICE*/, int to_interleaved);
int qxd_apply_Dw_multi_interleaved(qxd_ctx* ctx, int prec, int nrhs, const void* in, void* out);

/* ---- openQxD field orders (§2, §4.1) ---------------------------------
 * The paper's host code keeps its fields in its own order; these calls convert between that order and the natural
 * order of this header, so that its arrays can be passed as they are (the load()/save() pair of PAPER.md:107).
 *   site index  xhat = floor((V_B Lambda(n,N_B) + Lambda(b,B)) / 2) + P(x) V/2     (Eq. (2); R14)
 *               for cache blocks of extent block[mu], even points first, on the EXTENDED
 *               lattice; computed on the fly, no ipt[] table.  block[mu] must divide the extent, block[3] even.
 *   qxd_openqxd_index    xs: DEVICE [n][4] int coordinates (t,x,y,z) -> out: DEVICE [n] long xhat.
 *   qxd_openqxd_reorder  records of reals_per_site doubles per site (24 = spinor (x,alpha,a), PAPER.md:49,111;
 *                        72 = clover (x,+-,i)): to_openqxd != 0: out[xhat] = in[Lambda(x)], else the
 *                        inverse.  in, out: DEVICE [V][reals_per_site], must not alias.
 *   qxd_openqxd_gauge    reals_per_link = 18: SU(3) links, = 1: U(1) field A.  openQxD side: DEVICE [V/2][8][reals], the 8
 *                        links of every odd point of the extended lattice in the order +0,-0,+1,-1,+2,-2,+3,-3, entry +mu =
 *                        U_mu(x), entry -mu = U_mu(x-mu) (R20).  Natural side: DEVICE
 *                        [V_phys][4][reals] as qxd_gauge_load takes it.  to_openqxd != 0 builds the mirror half
 *                        (conjugate links, -A) and applies the shifted boundaries; the inverse reads the physical half only.
 * All three enqueue on the bound stream and return QXD_EINVAL for a bad block, reals count or null / aliased pointers. */
int qxd_openqxd_index(qxd_ctx* ctx, const int block[4], const int* xs, long n, long* out);
int qxd_openqxd_reorder(qxd_ctx* ctx, const int block[4], int reals_per_site, int to_openqxd, const double* in, double* out);
int qxd_openqxd_gauge(qxd_ctx* ctx, const int block[4], int reals_per_link, int to_openqxd, const double* in, double* out);

/* ---- domain decomposition: device-side halo and building blocks ----
 * A rank works on a LOCAL lattice = its own sites plus ghost layers in the cut directions (the geometry is created with the
 * local extents; time ghosts are one tile thick so that owned sites are whole time slabs).  The calls below are what a
 * distributed operator or solver is assembled from (paper_2502_02490_b200/domain.py drives them and moves the face buffers
 * between ranks with torch.distributed: NCCL over NVLink between GPUs); they all enqueue on the bound stream.
 *   qxd_time_slabs     number of time slabs of the site order and their thickness (the tile extent b0); QXD_EINVAL if the order
 *                      has no such slabs (tile volume != 256 sites, fewer than 3 or more than 64 slabs).
 *   qxd_dslash_packed  one dslash-shaped pass on packed FULL-lattice buffers (even half followed by odd half), restricted to the
 *                      time slabs [slab_lo, slab_hi) -- interior and boundary slabs are separate launches, so the halo exchange
 *                      overlaps the interior.  mode: QXD_DS_*; flags: QXD_DSF_*; the hop reads `in` on parity 1 - parity_out,
 *                      `phi` and `out` live on parity_out (QXD_DS_DW: both parities, phi ignored).  phi may be NULL if unused.
 *   qxd_clover_apply_packed   out = M in (inverse != 0: M^{-1} in) on one parity of packed full-lattice buffers.
 *   qxd_face_gather    buf[f][12] = upper two spin components of (1 - sign gamma_mu) psi(x) on the layer x_mu = coord, face sites f
 *                      in lexicographic order of the other three extended coordinates; reals of type double (QXD_F64) or float;
 *                      parity_mask 1 / 2: only that parity, compact index f >> 1; 3: both.  Size: qxd_face_bytes.
 *   qxd_face_scatter   ghost layer x_mu = coord <- (h, 0): the spinor whose projection has the upper components h; shift1 != 0
 *                      (even, mu != 1) reads the face site displaced by shift1 in direction 1: a message that crossed a C*
 *                      boundary lands shifted by L1.
 *   qxd_halo_zero      psi(x) = 0 on the layers lo <= x_mu < hi.
 *   qxd_blas_*_dev     BLAS-1 with device-resident scalars (a distributed solver all-reduces them with NCCL in place):
 *                      norm2_dev: *out = |x|^2;  cg_xr: alpha = *num / *den, x += alpha p, r -= alpha t, *rr = |r|^2;
 *                      cg_p: beta = *num / *den, p = s + beta p;  copy: y = x;  zero: x = 0;  convert / acc_hi / sub_norm_dev: the steps of
 *                      a reliable update (fp64 solution accumulation and true residual).  Half-lattice packed vectors. */
enum { QXD_DS_DW = 0, QXD_DS_HOP_AINV = 1, QXD_DS_A_XMHOP = 2, QXD_DS_X_MHOP = 3, QXD_DS_AINV_X_MHOP = 4 };
enum { QXD_DSF_G5IN = 1, QXD_DSF_G5HOP = 2 };
int qxd_time_slabs(const qxd_ctx* ctx, int* nslabs, int* thickness);
int qxd_dslash_packed(qxd_ctx* ctx, int prec, int mode, int flags, int parity_out, const void* in, const void* phi, void* out, int slab_lo, int slab_hi);
int qxd_clover_apply_packed(qxd_ctx* ctx, int prec, int inverse, int parity, const void* in, void* out);
size_t qxd_face_bytes(const qxd_ctx* ctx, int prec, int mu);
int qxd_face_gather(qxd_ctx* ctx, int prec, const void* packed, int parity_mask, int mu, int coord, int sign, void* buf);
int qxd_face_scatter(qxd_ctx* ctx, int prec, void* packed, int parity_mask, int mu, int coord, int shift1, const void* buf);
int qxd_halo_zero(qxd_ctx* ctx, int prec, void* packed, int parity_mask, int mu, int lo, int hi);
int qxd_blas_norm2_dev(qxd_ctx* ctx, int prec, const void* x, double* out /*DEVICE*/);
int qxd_blas_cg_xr(qxd_ctx* ctx, int prec, const double* num, const double* den, const void* p, const void* t, void* x, void* r, double* rr /*all scalars DEVICE*/);
int qxd_blas_cg_p(qxd_ctx* ctx, int prec, const double* num, const double* den, const void* s, void* p);
/* binary16 operator with fp32 Krylov vectors (the form the single-GPU solver uses, reading R12): x32 += alpha p16, r32 -= alpha t16,
 * r16 = half(r32), *rr = |r32|^2   and   p32 = s16 + beta p32, p16 = half(p32);  alpha, beta = *num / *den (DEVICE scalars). */
int qxd_blas_cg_xr_h(qxd_ctx* ctx, const double* num, const double* den, const void* p16, const void* t16, void* x32, void* r32, void* r16, double* rr);
int qxd_blas_cg_p_h(qxd_ctx* ctx, const double* num, const double* den, const void* s16, void* p32, void* p16);
int qxd_blas_copy(qxd_ctx* ctx, int prec, const void* x, void* y);
int qxd_blas_zero(qxd_ctx* ctx, int prec, void* x);
/* reliable-update building blocks: y (prec_to) = x (prec_from);  x_hi (fp64) += x_lo (prec), x_lo = 0;  r = b - t, *rr = |r|^2 */
int qxd_blas_convert(qxd_ctx* ctx, int prec_from, const void* x, int prec_to, void* y);
int qxd_blas_acc_hi(qxd_ctx* ctx, int prec, void* x_lo, void* x_hi);
int qxd_blas_sub_norm_dev(qxd_ctx* ctx, int prec, const void* b, const void* t, void* r, double* rr /*DEVICE*/);

/* ---- BLAS-1 on packed half-lattice spinors (row a6) ---------------------------------------------
 * y <- a*x + y ;  returns <x,y> = sum conj(x) y  and  |x|^2 (fp64 accumulation, HOST results). */
int qxd_blas_axpy(qxd_ctx* ctx, int prec, double a, const void* x, void* y);
int qxd_blas_cdot(qxd_ctx* ctx, int prec, const void* x, const void* y, double* re_im /*HOST [2]*/);
int qxd_blas_norm2(qxd_ctx* ctx, int prec, const void* x, double* out /*HOST*/);

/* ---- allocation-free entry point (noalloc.cu) -------------------------------------------------------------------------
 * For callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the norm reduction of the solvers (row a6, the |r|^2 of every iteration: PAPER.md:45) on a flat array, with
 * its per-CTA partial sums in a file-scope __device__ array of the library instead of the caller's workspace.  Needs no
 * context and no workspace, and calls no cudaMalloc / cudaFree / allocating library routine.
 *   qxd_norm2_noalloc      *out = sum_{k < nreals} x[k]^2, accumulated in fp64.  prec: QXD_F64 (x: const double*) or QXD_F32
 *                          (x: const float*); QXD_F16 -> QXD_EINVAL.  x: DEVICE, nreals reals (any packed fp64 / fp32 spinor of
 *                          this library is such an array: 24 Vh reals per half lattice); out: DEVICE, one double, written by
 *                          the GPU in stream order (no host synchronisation); stream: a cudaStream_t, NULL = the default
 *                          stream.  nreals = 0 gives 0 (x may then be NULL).  nreals > qxd_noalloc_max_reals() = 268 435 456 (65 536 partial sums
 *                          of 4096 reals, 512 KB of static device memory per GPU that loads the library) -> QXD_EINVAL, with
 *                          the limit in qxd_noalloc_last_error().  The result is independent of the launch configuration
 *                          (fixed chunks, fixed order).  All calls on a device share the one scratch array, which keeps the
 *                          last call's partial sums (none of them is read again: every call overwrites what it uses): calls
 *                          in one stream are safe, calls that OVERLAP on the GPU (different streams, no ordering) race.
 *   qxd_noalloc_init       set-up of the current device (looks up the device address of the scratch array); once per device,
 *                          with that device current, outside any graph capture.  qxd_norm2_noalloc does it on its first call
 *                          on a device if it was not done.
 *   qxd_noalloc_last_error message of the last failure of these calls in this thread. */
int qxd_noalloc_init(void);
size_t qxd_noalloc_max_reals(void);
const char* qxd_noalloc_last_error(void);
int qxd_norm2_noalloc(int prec, const void* x /*DEVICE*/, size_t nreals, double* out /*DEVICE*/, void* stream);

/* Number of kernel launches issued by this context so far (bench.py's gpu_launches). */
long qxd_launch_count(const qxd_ctx* ctx);
const char* qxd_last_error(const qxd_ctx* ctx);
const char* qxd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QXD_H */
