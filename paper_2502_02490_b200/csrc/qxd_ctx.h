// qxd_ctx.h -- host-side context of the C-ABI library and the internal launcher prototypes.
#pragma once
#include <cuda_runtime.h>
#include <string>
#include <cstdio>
#include "../../include/qxd.h"
#include "qxd_common.cuh"

namespace qxd {

enum { NPREC = 3 };
inline size_t prec_size(int p) { return p == 0 ? 8 : (p == 1 ? 4 : 2); }

// dslash epilogue selection:  tmp = PHI-term + (NEG ? -1 : +1) * hop(in);
// out = POST applied to tmp, where hop(in) = -1/2 sum_mu [...] is the off-diagonal part of D_w.
enum DslashMode {
  DS_DW_FULL = 0,   // out = M in(x) + hop(in)                      both parities in one launch   (row a4)
  DS_HOP_AINV,      // out_p = M^{-1} hop(in)                       pass 1 of D-hat               (row a5)
  DS_A_XMHOP,       // out_p = M phi - hop(in)                      pass 2 of D-hat               (row a5)
  DS_X_MHOP,        // out_p = phi - hop(in)                        source preparation            (row a8)
  DS_AINV_X_MHOP,   // out_p = M^{-1} (phi - hop(in))               odd-site reconstruction       (row a8)
  DS_NMODES
};
enum { DSF_G5IN = 1, DSF_G5HOP = 2, DSF_NORM = 4, DSF_DOT = 8 };

struct Scalars;  // device-resident solver scalars (solver.cu)

}  // namespace qxd

struct qxd_ctx {
  qxd::Geom g;
  int T, L1, L2, L3, bc;
  int tile[4] = {1, 1, 1, 2}, block[4] = {1, 1, 1, 2};
  long V;
  cudaStream_t stream = 0;
  // workspace
  char* ws = nullptr;
  size_t ws_bytes = 0, ws_used = 0;
  int prec_mask = 0, nrhs = 1;
  int link_reals[qxd::NPREC] = {18, 18, 18};     // per storage precision: stored reals per hopping link, 18 or 14 = rows 0,1 + det (qxd_set_gauge_reconstruct)
  int rhs_per_thread = 0;                        // multi-RHS dslash: right-hand sides per thread (0 = default)
  int dw_sweep_tseg = 0;                         // > 0: the fp32 full-lattice D_w uses the time-sweep kernel with this segment length (qxd_set_dw_sweep)
  // state
  bool have_gauge = false, have_qed = false, have_quark = false, have_clover = false;
  // field-status manager (row f4): derived fields marked stale by a setter and regenerated at their first use
  bool lazy = false, hop_stale = false, clover_stale = false;
  long n_hop_refresh = 0, n_clover_refresh = 0;
  long n_inv_fast = 0, n_inv_pivoted = 0;          // block-inversion passes: unpivoted fast path / pivoted fallback (qxd_clover_stats)
  double qel = 1.0, kappa = 0, q = 0, m0 = 0, csw = 0, csw_qed = 0;
  // fields (device, carved from the workspace); [parity]
  void* Ug[2] = {nullptr, nullptr};              // fp64 SU(3) links, record of 72 reals (4 links x 18)
  void* Ag[2] = {nullptr, nullptr};              // fp64 U(1) field, record of 4 reals
  void* W[qxd::NPREC][2] = {};                   // hopping links e^{iqA} U (time-BC sign folded in), 4 x link_reals (buffer: 72 reals)
  void* M[qxd::NPREC][2] = {};                   // clover blocks, 72 reals (PAPER.md:117 order)
  void* Mi[qxd::NPREC][2] = {};                  // inverse blocks
  // scratch spinors
  void* sp64[12] = {};                           // fp64 half-lattice spinors
  void* splo[8] = {};                            // sloppy half-lattice spinors (sized for fp32)
  void* full_a = nullptr;                        // packed full-lattice spinors (sized for fp64)
  void* full_b = nullptr;
  double* nat_a = nullptr;                       // natural-order staging (host-pointer entry points)
  double* nat_b = nullptr;
  // batch (multi-RHS) vectors, present when the workspace was bound with nrhs > 1: nrhs half-lattice spinors each
  void* mhi[2] = {};                             // fp64: b, x
  void* mlo[7] = {};                             // sloppy: x, r, p, t(=s), odd-site scratch, r16, p16 (fp16 operator with fp32 vectors); mlo_size bytes per real
  size_t mlo_size = 0;
  double* mscal = nullptr;                       // device scalars [64 systems][8]
  double* mact = nullptr;                        // device activity mask [64]
  double* h_mscal = nullptr;                     // pinned host mirrors
  double* h_mact = nullptr;
  // SAP-preconditioned GCR (row f3): Krylov space z_k, w_k and the preconditioner's residual / correction fields, fp32 full lattice
  int gcr_nkv = 0, gcr_ncy = 4, gcr_nmr = 4;
  void* gz[32] = {};
  void* gw[32] = {};
  void* g_r = nullptr;                           // fp32 residual of the GCR cycle
  void* g_res = nullptr;                         // SAP: block residuals
  void* g_corr = nullptr;                        // SAP: latest block corrections
  void* g_r64 = nullptr;                         // fp64 full-lattice residual / scratch
  void* g_t64 = nullptr;
  int sap_ok = -1, sap_boxsh[4] = {}, sap_colmask[4] = {};   // two-colouring of the SAP blocks (-1: not yet checked for the current site order)
  double* gscal = nullptr;                       // device scalars of the GCR cycle: coefficient matrix b[32][32] (complex), c[32], y[32], norms
  // two-level (deflated) preconditioner of the GCR (dfl.cu): null vectors, coarse operator, coarse-grid vectors
  int dfl_ns = 0, dfl_ninv = 4, dfl_nkc = 16, dfl_nref = 0, dfl_prec = 1;
  int dfl_refk = 1;                              // GCR steps of every inverse-iteration solve of the refinement rounds (1 = one preconditioner application)
  int dfl_chiral = 0;                            // 1: null vectors split by chirality, coarse dimension per block = 2 ns (qxd_set_deflation_chirality)
  bool dfl_ready = false;
  void* dphi[32] = {};                           // fp32 packed full-lattice null vectors, block-orthonormal
  void* d_t1 = nullptr;                          // fp32 fine-grid temporaries
  void* d_t2 = nullptr;
  void* dAc = nullptr;                           // coarse operator [nblocks][9][ns][ns] complex fp32
  int* dnbr = nullptr;                           // neighbour blocks [nblocks][8]
  void* dDinv = nullptr;                         // inverses of the diagonal coarse blocks [nblocks][ns][ns] (block-Jacobi preconditioner)
  void* dAh = nullptr;                           // binary16 transposed copy for the even-odd coarse solver: [nblocks][9][ns][ns] half2, slot d < 8 = (A_c[1+d])^T, slot 8 = Dinv^T
  int* dcol = nullptr;                           // colour (0 / 1) of every block
  void* dcs = nullptr;                           // coarse scratch vectors of the even-odd solver
  void* dct = nullptr;
  void* dcb = nullptr;                           // coarse vectors [nblocks][ns] complex fp32: right-hand side / scratch,
  void* dcx = nullptr;                           //   solution,
  void* dcr = nullptr;                           //   residual,
  void* dcz[32] = {};                            //   Krylov vectors of the coarse GCR
  void* dcw[32] = {};
  double* dscal = nullptr;                       // device scalars of the coarse GCR (layout of gcr_kernels.cuh)
  // reductions
  double* partials = nullptr;
  double* scal = nullptr;                        // device scalars [64]
  double* h_scal = nullptr;                      // pinned host mirror [64]
  int max_blocks = 0;
  long launches = 0;
  std::string err;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  cudaStream_t s_in = nullptr, s_out = nullptr;  // copy streams of the pipelined host-pointer apply (created on first use)
  cudaEvent_t ev_slab[2][64] = {};               // [in/out][slab]
  cudaEvent_t ev_scal = nullptr;                 // marks the device->host copy of solver scalars (solver.cu: post_scal / wait_scal)
};

namespace qxd {

inline int fail(qxd_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}
#define QXD_CUDA_OK(ctx, expr)                                                                   \
  do {                                                                                           \
    cudaError_t e__ = (expr);                                                                    \
    if (e__ != cudaSuccess) return qxd::fail(ctx, QXD_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e__)); \
  } while (0)

#define QXD_LAUNCH_CHECK(c)                                                                                    \
  do {                                                                                                         \
    (c)->launches++;                                                                                           \
    cudaError_t e__ = cudaGetLastError();                                                                      \
    if (e__ != cudaSuccess) return qxd::fail((c), QXD_ECUDA, std::string(__func__) + ": " + cudaGetErrorString(e__)); \
  } while (0)

inline SpinorPtr half_view(int prec, void* base, int Vh, int parity) {
  return prec == 0 ? spinor_view<double>(base, Vh, parity) : prec == 1 ? spinor_view<float>(base, Vh, parity) : spinor_view<__half>(base, Vh, parity);
}
inline size_t half_bytes(int prec, int Vh) {
  return prec == 0 ? spinor_half_bytes<double>(Vh) : prec == 1 ? spinor_half_bytes<float>(Vh) : spinor_half_bytes<__half>(Vh);
}

// ---- launchers (each returns a qxd_status and bumps ctx->launches) ----
// pack.cu
int launch_gauge_pack(qxd_ctx* c, const double* U, const double* A);
int launch_hoplinks(qxd_ctx* c, int prec);
int launch_spinor_pack(qxd_ctx* c, int prec, const double* nat, void* packed, int parity_mask /*1 even,2 odd,3 both*/, int compact_even,
                       const TileMap& tm = TileMap());
int launch_spinor_unpack(qxd_ctx* c, int prec, const void* packed, double* nat, int parity_mask, int compact_even,
                         const TileMap& tm = TileMap());
int launch_convert_spinor(qxd_ctx* c, int prec_from, const SpinorPtr& from, int prec_to, const SpinorPtr& to, int n = 1, size_t rs_from = 0,
                          size_t rs_to = 0);
int launch_convert_record72(qxd_ctx* c, const void* from64, int prec_to, void* to);
int launch_clover_export(qxd_ctx* c, double* out, int inverse);
// clover.cu
int launch_clover_build(qxd_ctx* c);
// dslash.cu
struct DslashCall {
  int prec;
  int mode;         // DslashMode
  int flags;        // DSF_*
  int parity_out;   // parity of the output sites (ignored for DS_DW_FULL)
  SpinorPtr in[2];  // input spinor per parity (hop reads in[1-p]; DS_DW_FULL also in[p])
  SpinorPtr phi;    // PHI-term input on the output parity (modes with phi)
  SpinorPtr out[2]; // output per parity (only [parity_out] used unless DS_DW_FULL)
  double* norm_result;  // DSF_NORM: device slot receiving |out|^2 (right-hand side r: norm_result[r * norm_stride]);
                        // DSF_DOT: three slots receiving Re <phi,out>, Im <phi,out>, |out|^2
  // multi-RHS launches (row a10): nrhs > 1 right-hand sides, rs_* bytes apart in in / phi / out
  int nrhs;
  size_t rs_in, rs_phi, rs_out;
  int norm_stride;
  TileMap tm;       // launch on a subset of the tiles (time slab); default: whole lattice
  int t_lo, t_hi;   // t_hi > 0: compute only the sites with t_lo <= x0 < t_hi (CTAs outside the range retire at once)
};
int launch_dslash(qxd_ctx* c, const DslashCall& d);
int launch_clover_apply(qxd_ctx* c, int prec, int inverse, int parity, const SpinorPtr& in, const SpinorPtr& out);
// blas.cu
// A batch of right-hand sides (row a10): n vectors rs bytes apart, per-system scalars ss doubles apart, optional
// activity mask act[n] (1.0 = iterate, 0.0 = frozen).  The default is a single vector.
struct Batch {
  int n = 1;
  size_t rs = 0;
  int ss = 0;
  const double* act = nullptr;
};
int blas_axpy(qxd_ctx* c, int prec, double a, const SpinorPtr& x, const SpinorPtr& y);            // y += a x
// exact: every product and sum in fp64; default: per-site sums in the arithmetic type, fp64 across sites (solver calls)
int blas_cdot(qxd_ctx* c, int prec, const SpinorPtr& x, const SpinorPtr& y, double* dev_result3, bool exact = false);  // Re<x,y>, Im<x,y>, |y|^2
int blas_norm2(qxd_ctx* c, int prec, const SpinorPtr& x, double* dev_result, const Batch& b = Batch(), bool exact = false);
int blas_zero(qxd_ctx* c, int prec, const SpinorPtr& x, const Batch& b = Batch());
// z = x + a*y + b*w with complex scalars by value (w may be unused when b == 0); BiCGstab building block
int blas_cxpaypbw(qxd_ctx* c, int prec, const SpinorPtr& x, double ar, double ai, const SpinorPtr& y, double br, double bi,
                  const SpinorPtr& w, const SpinorPtr& z);
// BiCGstab: x += alpha p + omega s ; r = s - omega t ; res3 = (Re<r0,r>, Im<r0,r>, |r|^2)
int blas_bicg_s(qxd_ctx* c, int prec, double rho_re, double rho_im, const double* r0v, const SpinorPtr& r, const SpinorPtr& v, const SpinorPtr& s);
int blas_bicg_xr(qxd_ctx* c, int prec, double rho_re, double rho_im, const double* r0v, const double* dst, const SpinorPtr& p, const SpinorPtr& s,
                 const SpinorPtr& t, const SpinorPtr& r0, const SpinorPtr& x, const SpinorPtr& r, double* res3);
// alpha = *num / *den (device scalars): x += alpha p ; r -= alpha t ; *rr = |r|^2
int blas_cg_xr(qxd_ctx* c, int prec, const double* num, const double* den, const SpinorPtr& p, const SpinorPtr& t, const SpinorPtr& x,
               const SpinorPtr& r, double* rr, const Batch& b = Batch());
// beta = *num / *den : p = s + beta p
int blas_cg_p(qxd_ctx* c, int prec, const double* num, const double* den, const SpinorPtr& s, const SpinorPtr& p, const Batch& b = Batch());
// fp16 operator with fp32 vectors: x, r, p in float; t, s and the operator inputs r16, p16 in binary16
// (batch b: fp32 vectors b.rs bytes apart, binary16 vectors rs_o bytes apart)
int blas_cg_xr_h(qxd_ctx* c, const double* num, const double* den, const SpinorPtr& p, const SpinorPtr& t, const SpinorPtr& x,
                 const SpinorPtr& r, const SpinorPtr& r16, double* rr, const Batch& b = Batch(), size_t rs_o = 0);
int blas_cg_p_h(qxd_ctx* c, const double* num, const double* den, const SpinorPtr& s, const SpinorPtr& p, const SpinorPtr& p16,
                const Batch& b = Batch(), size_t rs_o = 0);
int blas_acc_hi(qxd_ctx* c, int prec, const SpinorPtr& xlo, const SpinorPtr& xhi);                  // x_hi += x_lo ; x_lo = 0
int blas_sub_norm(qxd_ctx* c, int prec, const SpinorPtr& b, const SpinorPtr& t, const SpinorPtr& r, double* res);  // r = b - t
int blas_copy(qxd_ctx* c, int prec, const SpinorPtr& x, const SpinorPtr& y, const Batch& b = Batch());   // y = x
// solver.cu
int solve_eo(qxd_ctx* c, const double* eta_nat, double* psi_nat, double tol, qxd_solve_info* info);
int solve_eo_multi(qxd_ctx* c, int nrhs, const double* eta_nat, double* psi_nat, double tol, qxd_solve_info* info);
// dslash_ilv.cu
int launch_dw_ilv(qxd_ctx* c, int prec, int nrhs, const void* in, void* out);
int launch_ilv_convert(qxd_ctx* c, int prec, int nrhs, void* plain, void* ilv, int to_ilv);
// dslash_sweep.cu
int launch_dw_sweep(qxd_ctx* c, const SpinorPtr in[2], const SpinorPtr out[2]);
// halo.cu (row f2)
size_t face_bytes(const qxd_ctx* c, int prec, int mu);
int launch_face_gather(qxd_ctx* c, int prec, void* packed, int pmask, int mu, int coord, int sign, void* buf);
int launch_face_scatter(qxd_ctx* c, int prec, void* packed, int pmask, int mu, int coord, int shift1, const void* buf);
int launch_halo_zero(qxd_ctx* c, int prec, void* packed, int pmask, int mu, int lo, int hi);
// sap.cu / gcr.cu (row f3)
int sap_check_geometry(qxd_ctx* c);
int launch_sap(qxd_ctx* c, int prec, const void* in_full32, void* out_full32);   // out = M_sap in (fp32 packed full-lattice vectors)
int solve_gcr(qxd_ctx* c, const double* eta_nat, double* psi_nat, double tol, qxd_solve_info* info);
int launch_coarse_build(qxd_ctx* c, int prec, int ns, void* const* phi, void* A, int* nbr);
// dfl.cu (row f3, second level)
int launch_dfl_precond(qxd_ctx* c, int prec, const void* r, void* z);
int gcr_cycle32(qxd_ctx* c, int pprec, bool use_dfl, int K, void* x);
int dfl_setup(qxd_ctx* c, int prec, const void* random_vectors);
int dfl_restrict(qxd_ctx* c, const void* fine, void* coarse);
int dfl_prolong(qxd_ctx* c, const void* coarse, void* fine);
int dfl_coarse_apply(qxd_ctx* c, const void* x, void* y);
int dfl_coarse_solve(qxd_ctx* c, const void* b, void* x);

}  // namespace qxd
