// solver.cu -- SURVEY.md §8 rows a7 (mixed-precision even-odd CGNE / BiCGstab with reliable updates) and a8
// (even-odd source preparation and reconstruction).  The paper offloads "the solution of a large linear
// system D_w psi = eta" with a mixed half/single/double precision solver
// and checks the result a posteriori; this file does the same with the solvers named in
// BASELINE.json north_star: the inner iteration runs in the sloppy precision, the solution is accumulated
// and the true residual recomputed in fp64 ("reliable updates", ref [4] of the paper), and the
// call only reports convergence on the fp64 residual.
//
//   eta-hat_e = eta_e - D_eo A_oo^{-1} eta_o ;  D-hat psi_e = eta-hat_e ;  psi_o = A_oo^{-1}(eta_o - D_oe psi_e)
//   D-hat = A_ee - D_eo A_oo^{-1} D_oe (reading R10), D-hat^dag = gamma5 D-hat gamma5.
#include "qxd_ctx.h"
#include <cmath>

namespace qxd {

namespace {

enum { SC_GAM0 = 0, SC_GAM1 = 1, SC_TT = 2, SC_RR = 3, SC_RRT = 4, SC_NE = 5, SC_NO = 6, SC_DOT = 8 /* 9 slots: <r0,v>, <s,t> and |t|^2, <r0,r> and |r|^2 of a BiCGstab iteration */ };

struct Ws {
  int Vh;
  SpinorPtr eta_e, eta_o, b, xhi, rhi, thi, tmp_o_hi, out_e, out_o, xbest;
  SpinorPtr xlo, rlo, p, t, s, tmp_o_lo, v, r0;
};

SpinorPtr hv(int prec, void* base, int Vh) { return half_view(prec, base, Vh, 0); }

int read_scal(qxd_ctx* c, int idx, int n, double* out) {
  QXD_CUDA_OK(c, cudaMemcpyAsync(c->h_scal + idx, c->scal + idx, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
  QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
  for (int i = 0; i < n; i++) out[i] = c->h_scal[idx + i];
  return QXD_OK;
}

// Split form of read_scal: post_scal enqueues the copy and marks it with an event; work enqueued afterwards keeps the GPU
// busy while wait_scal blocks the host on that event only (not on the whole stream).
int post_scal(qxd_ctx* c, int idx, int n) {
  QXD_CUDA_OK(c, cudaMemcpyAsync(c->h_scal + idx, c->scal + idx, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
  QXD_CUDA_OK(c, cudaEventRecord(c->ev_scal, c->stream));
  return QXD_OK;
}
int wait_scal(qxd_ctx* c, int idx, int n, double* out) {
  QXD_CUDA_OK(c, cudaEventSynchronize(c->ev_scal));
  for (int i = 0; i < n; i++) out[i] = c->h_scal[idx + i];
  return QXD_OK;
}

#define QXD_TRY(expr)        \
  do {                       \
    int rc__ = (expr);       \
    if (rc__) return rc__;   \
  } while (0)

}  // namespace

// out_e = D-hat in_e (dagger: D-hat^dag in_e); tmp_o: odd-site scratch of the same precision.  A batch b applies the
// operator to b.n right-hand sides b.rs bytes apart with the multi-RHS kernels (row a10); norms go to norm_slot[k * b.ss].
int apply_dhat(qxd_ctx* c, int prec, const SpinorPtr& in_e, const SpinorPtr& out_e, const SpinorPtr& tmp_o, int dagger, double* norm_slot,
               const Batch& b) {
  DslashCall d1{};
  d1.prec = prec; d1.mode = DS_HOP_AINV; d1.flags = dagger ? DSF_G5IN : 0; d1.parity_out = 1;
  d1.in[0] = in_e; d1.out[1] = tmp_o;
  d1.nrhs = b.n; d1.rs_in = d1.rs_phi = d1.rs_out = b.rs;
  QXD_TRY(launch_dslash(c, d1));
  DslashCall d2{};
  d2.prec = prec; d2.mode = DS_A_XMHOP; d2.flags = (dagger ? DSF_G5HOP : 0) | (norm_slot ? DSF_NORM : 0); d2.parity_out = 0;
  d2.in[1] = tmp_o; d2.phi = in_e; d2.out[0] = out_e; d2.norm_result = norm_slot; d2.norm_stride = b.ss;
  d2.nrhs = b.n; d2.rs_in = d2.rs_phi = d2.rs_out = b.rs;
  QXD_TRY(launch_dslash(c, d2));
  return QXD_OK;
}
// out_e = D-hat in_e with the fused reduction dot_slot[0..2] = (Re <in,out>, Im <in,out>, |out|^2)
int apply_dhat_dot(qxd_ctx* c, int prec, const SpinorPtr& in_e, const SpinorPtr& out_e, const SpinorPtr& tmp_o, double* dot_slot) {
  DslashCall d1{};
  d1.prec = prec; d1.mode = DS_HOP_AINV; d1.flags = 0; d1.parity_out = 1;
  d1.in[0] = in_e; d1.out[1] = tmp_o;
  d1.nrhs = 1;
  QXD_TRY(launch_dslash(c, d1));
  DslashCall d2{};
  d2.prec = prec; d2.mode = DS_A_XMHOP; d2.flags = DSF_DOT; d2.parity_out = 0;
  d2.in[1] = tmp_o; d2.phi = in_e; d2.out[0] = out_e; d2.norm_result = dot_slot; d2.norm_stride = 0;
  d2.nrhs = 1;
  QXD_TRY(launch_dslash(c, d2));
  return QXD_OK;
}
int apply_dhat(qxd_ctx* c, int prec, const SpinorPtr& in_e, const SpinorPtr& out_e, const SpinorPtr& tmp_o, int dagger, double* norm_slot) {
  return apply_dhat(c, prec, in_e, out_e, tmp_o, dagger, norm_slot, Batch());
}

namespace {

// fp64 true residual: x_hi += x_lo; x_lo = 0; r_hi = b - D-hat x_hi; r_lo = r_hi; returns |r_hi|^2
int reliable_update(qxd_ctx* c, int plo, Ws& w, double* rr_true, const SpinorPtr* r16 = nullptr) {
  QXD_TRY(blas_acc_hi(c, plo, w.xlo, w.xhi));
  QXD_TRY(apply_dhat(c, 0, w.xhi, w.thi, w.tmp_o_hi, 0, nullptr));
  QXD_TRY(blas_sub_norm(c, 0, w.b, w.thi, w.rhi, c->scal + SC_RRT));
  QXD_TRY(launch_convert_spinor(c, 0, w.rhi, plo, w.rlo));
  if (r16) QXD_TRY(launch_convert_spinor(c, 0, w.rhi, 2, *r16));
  QXD_TRY(read_scal(c, SC_RRT, 1, rr_true));
  return QXD_OK;
}

// CG on the normal equations of D-hat keeping the system residual (reading R11):
//   s = A^dag r, p = s, gam = |s|^2; loop: t = A p; al = gam/|t|^2; x += al p; r -= al t; s = A^dag r;
//   gam' = |s|^2; p = s + (gam'/gam) p.
int cgne(qxd_ctx* c, int pop, Ws& w0, double stop2, double delta, int maxiter, qxd_solve_info* info) {
  // pop: precision of the sloppy operator; plo: precision of the Krylov vectors x, r, p.  With a binary16 operator the
  // vectors stay in float and the operator reads binary16 copies r16 (slot v) and p16 (slot r0), see blas.cu.
  const bool h16 = (pop == 2);
  const int plo = h16 ? 1 : pop;
  Ws w = w0;
  SpinorPtr r16 = w0.v, p16 = w0.r0;
  if (h16) { w.xlo.scale = nullptr; w.rlo.scale = nullptr; w.p.scale = nullptr; }
  const SpinorPtr& rin = h16 ? r16 : w.rlo;   // operator inputs
  const SpinorPtr& pin = h16 ? p16 : w.p;
  double rr = 0;
  QXD_TRY(blas_zero(c, 0, w.xhi));
  QXD_TRY(blas_zero(c, plo, w.xlo));
  QXD_TRY(blas_copy(c, 0, w.b, w.rhi));
  QXD_TRY(blas_norm2(c, 0, w.rhi, c->scal + SC_RRT));
  QXD_TRY(read_scal(c, SC_RRT, 1, &rr));
  QXD_TRY(launch_convert_spinor(c, 0, w.rhi, plo, w.rlo));
  if (h16) QXD_TRY(launch_convert_spinor(c, 0, w.rhi, 2, r16));
  int it = 0, nrel = 0, status = QXD_ENOCONV;
  double maxr = std::sqrt(rr), rr_true = rr;
  if (rr <= stop2) status = QXD_OK;
  if (status != QXD_OK) {
    QXD_TRY(apply_dhat(c, pop, rin, w.s, w.tmp_o_lo, 1, c->scal + SC_GAM0));
    QXD_TRY(launch_convert_spinor(c, pop, w.s, plo, w.p));
    if (h16) QXD_TRY(blas_copy(c, 2, w.s, p16));
  }
  while (status != QXD_OK && it < maxiter) {
    double* gam = c->scal + SC_GAM0 + (it & 1);
    double* gam_next = c->scal + SC_GAM0 + ((it + 1) & 1);
    QXD_TRY(apply_dhat(c, pop, pin, w.t, w.tmp_o_lo, 0, c->scal + SC_TT));
    if (h16) QXD_TRY(blas_cg_xr_h(c, gam, c->scal + SC_TT, p16, w.t, w.xlo, w.rlo, r16, c->scal + SC_RR));
    else QXD_TRY(blas_cg_xr(c, plo, gam, c->scal + SC_TT, w.p, w.t, w.xlo, w.rlo, c->scal + SC_RR));
    // |r|^2 decides on the host whether to stop or to do a reliable update.  s = A^dag r is enqueued BEFORE the host waits
    // for it, so the GPU never idles on the round trip; it is only wasted (recomputed from the corrected r) in the
    // iterations that do a reliable update.
    QXD_TRY(post_scal(c, SC_RR, 1));
    QXD_TRY(apply_dhat(c, pop, rin, w.s, w.tmp_o_lo, 1, gam_next));
    QXD_TRY(wait_scal(c, SC_RR, 1, &rr));
    it++;
    if (!(rr == rr)) {  // NaN: breakdown.  x_lo is poisoned: drop it, so that x_hi (the last reliable update) is what is returned
      QXD_TRY(blas_zero(c, plo, w.xlo));
      break;
    }
    double rn = std::sqrt(rr);
    if (rn > maxr) maxr = rn;
    if (rn < delta * maxr || rr <= stop2) {
      QXD_TRY(reliable_update(c, plo, w, &rr_true, h16 ? &r16 : nullptr));
      nrel++;
      maxr = std::sqrt(rr_true);
      if (rr_true <= stop2) { status = QXD_OK; break; }
      QXD_TRY(apply_dhat(c, pop, rin, w.s, w.tmp_o_lo, 1, gam_next));
    }
    if (h16) QXD_TRY(blas_cg_p_h(c, gam_next, gam, w.s, w.p, p16));
    else QXD_TRY(blas_cg_p(c, plo, gam_next, gam, w.s, w.p));
  }
  if (status != QXD_OK) {  // leave the best iterate in x_hi with its true residual
    QXD_TRY(reliable_update(c, plo, w, &rr_true));
    nrel++;
    if (rr_true <= stop2) status = QXD_OK;
  }
  info->iters = it; info->n_reliable = nrel; info->true_res = rr_true;  // |r|^2 for now; caller normalises
  return status;
}

struct cplx { double re, im; };
inline cplx cdiv(cplx a, cplx b) { double d = b.re * b.re + b.im * b.im; return {(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d}; }
inline cplx cmul(cplx a, cplx b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
inline double cabs2(cplx a) { return a.re * a.re + a.im * a.im; }

// BiCGstab on D-hat (van der Vorst recurrences) with the same reliable-update wrapper.  Breakdown
// (rho ~ 0 or omega ~ 0) is reported as QXD_ENOCONV with the best iterate (reading R11).
int bicgstab(qxd_ctx* c, int plo, Ws& w, double stop2, double delta, int maxiter, qxd_solve_info* info) {
  double rr = 0, d3[3];
  QXD_TRY(blas_zero(c, 0, w.xhi));
  QXD_TRY(blas_zero(c, plo, w.xlo));
  QXD_TRY(blas_copy(c, 0, w.b, w.rhi));
  QXD_TRY(blas_norm2(c, 0, w.rhi, c->scal + SC_RRT));
  QXD_TRY(read_scal(c, SC_RRT, 1, &rr));
  QXD_TRY(launch_convert_spinor(c, 0, w.rhi, plo, w.rlo));
  QXD_TRY(blas_copy(c, plo, w.rlo, w.r0));
  QXD_TRY(blas_copy(c, plo, w.rlo, w.p));
  int it = 0, nrel = 0, status = QXD_ENOCONV;
  double maxr = std::sqrt(rr), rr_true = rr;
  if (rr <= stop2) status = QXD_OK;
  cplx rho = {rr, 0.0};
  const double tiny = 1e-290;
  // stagnation guard: BiCGstab on D-hat can stall near / beyond the critical kappa (it did at config c4); if the iterated
  // residual has not improved on its best value for 500 iterations the solve is reported as not converged (R11)
  double best_rr = rr;
  int since_best = 0;
  // BiCGstab's residual is not monotonic: keep the fp64 iterate with the smallest TRUE residual seen at a reliable update
  // (x = 0 to begin with), so that a solve that fails still returns its best iterate (include/qxd.h, QXD_ENOCONV)
  double best_true = rr;
  QXD_TRY(blas_zero(c, 0, w.xbest));
  while (status != QXD_OK && it < maxiter) {
    if (cabs2(rho) < tiny) break;
    // alpha and omega are formed on the device from the reduction results (blas.cu: bicg_alpha, bicg_omega), so the six
    // kernels of an iteration are enqueued back to back; the host reads all nine scalars once, at the end
    QXD_TRY(apply_dhat(c, plo, w.p, w.v, w.tmp_o_lo, 0, nullptr));                 // v = A p
    QXD_TRY(blas_cdot(c, plo, w.r0, w.v, c->scal + SC_DOT));                        // <r0,v>
    QXD_TRY(blas_bicg_s(c, plo, rho.re, rho.im, c->scal + SC_DOT, w.rlo, w.v, w.s));   // s = r - alpha v
    QXD_TRY(apply_dhat_dot(c, plo, w.s, w.t, w.tmp_o_lo, c->scal + SC_DOT + 3));   // t = A s with <s,t> = conj <t,s> and |t|^2 fused
    // x += alpha p + omega s ; r = s - omega t ; rho' = <r0,r>, |r|^2 -- one kernel
    QXD_TRY(blas_bicg_xr(c, plo, rho.re, rho.im, c->scal + SC_DOT, c->scal + SC_DOT + 3, w.p, w.s, w.t, w.r0, w.xlo, w.rlo, c->scal + SC_DOT + 6));
    double d9[9];
    QXD_TRY(read_scal(c, SC_DOT, 9, d9));
    cplx r0v = {d9[0], d9[1]};
    cplx ts = {d9[3], -d9[4]};
    const double tt = d9[5];
    d3[0] = d9[6]; d3[1] = d9[7]; d3[2] = d9[8];
    // the degenerate steps the device took with alpha = 0 or omega = 0 (x and r consistent either way) end the iteration
    if (cabs2(r0v) < tiny) { it++; break; }
    cplx alpha = cdiv(rho, r0v);
    if (!(tt > tiny)) { it++; break; }   // t = 0: s was already the exact residual update (the device used omega = 0)
    cplx omega = {ts.re / tt, ts.im / tt};
    it++;
    cplx rho_new = {d3[0], d3[1]};
    rr = d3[2];
    if (!(rr == rr)) { QXD_TRY(blas_zero(c, plo, w.xlo)); break; }   // NaN: drop the poisoned x_lo (x_hi / xbest are returned)
    if (rr < best_rr) { best_rr = rr; since_best = 0; } else if (++since_best >= 500) break;
    double rn = std::sqrt(rr);
    if (rn > maxr) maxr = rn;
    bool updated = false;
    if (rn < delta * maxr || rr <= stop2) {
      QXD_TRY(reliable_update(c, plo, w, &rr_true));
      nrel++; updated = true;
      if (rr_true < best_true) { best_true = rr_true; QXD_TRY(blas_copy(c, 0, w.xhi, w.xbest)); }
      maxr = std::sqrt(rr_true);
      if (rr_true <= stop2) { status = QXD_OK; break; }
    }
    if (updated) {  // rho' must refer to the replaced residual
      QXD_TRY(blas_cdot(c, plo, w.r0, w.rlo, c->scal + SC_DOT));
      QXD_TRY(read_scal(c, SC_DOT, 3, d3));
      rho_new = {d3[0], d3[1]};
    }
    if (cabs2(omega) < tiny) break;
    cplx beta = cmul(cdiv(rho_new, rho), cdiv(alpha, omega));
    cplx bo = cmul(beta, omega);
    QXD_TRY(blas_cxpaypbw(c, plo, w.rlo, beta.re, beta.im, w.p, -bo.re, -bo.im, w.v, w.p));          // p = r + beta (p - omega v)
    rho = rho_new;
  }
  if (status != QXD_OK) {
    QXD_TRY(reliable_update(c, plo, w, &rr_true));
    nrel++;
    if (rr_true <= stop2) status = QXD_OK;
    else if (rr_true > best_true) { QXD_TRY(blas_copy(c, 0, w.xbest, w.xhi)); rr_true = best_true; }
  }
  info->iters = it; info->n_reliable = nrel; info->true_res = rr_true;
  return status;
}

}  // namespace

int solve_eo(qxd_ctx* c, const double* eta_nat, double* psi_nat, double tol, qxd_solve_info* info) {
  const int Vh = c->g.Vh;
  const int plo = info->sloppy;
  if (plo < 0 || plo >= NPREC || !((c->prec_mask >> plo) & 1)) return fail(c, QXD_EINVAL, "solve: sloppy precision not bound");
  if (!(tol > 0.0)) return fail(c, QXD_EINVAL, "solve: tol must be > 0");
  const double delta = info->delta > 0.0 ? info->delta : 0.1;
  const int maxiter = info->maxiter > 0 ? info->maxiter : 10000;
  Ws w;
  w.Vh = Vh;
  w.eta_e = half_view(0, c->full_a, Vh, 0); w.eta_o = half_view(0, c->full_a, Vh, 1);
  w.out_e = half_view(0, c->full_b, Vh, 0); w.out_o = half_view(0, c->full_b, Vh, 1);
  w.b = hv(0, c->sp64[0], Vh); w.xhi = hv(0, c->sp64[1], Vh); w.rhi = hv(0, c->sp64[2], Vh); w.thi = hv(0, c->sp64[3], Vh);
  w.tmp_o_hi = hv(0, c->sp64[4], Vh); w.xbest = hv(0, c->sp64[5], Vh);
  w.xlo = hv(plo, c->splo[0], Vh); w.rlo = hv(plo, c->splo[1], Vh); w.p = hv(plo, c->splo[2], Vh); w.t = hv(plo, c->splo[3], Vh);
  w.s = hv(plo, c->splo[4], Vh); w.tmp_o_lo = hv(plo, c->splo[5], Vh); w.v = hv(plo, c->splo[6], Vh); w.r0 = hv(plo, c->splo[7], Vh);

  QXD_CUDA_OK(c, cudaEventRecord(c->ev0, c->stream));
  QXD_TRY(launch_spinor_pack(c, 0, eta_nat, c->full_a, 3, 0));
  QXD_TRY(blas_norm2(c, 0, w.eta_e, c->scal + SC_NE));
  QXD_TRY(blas_norm2(c, 0, w.eta_o, c->scal + SC_NO));
  double nn[2];
  QXD_TRY(read_scal(c, SC_NE, 2, nn));
  const double eta2 = nn[0] + nn[1];
  int status;
  if (eta2 == 0.0) {
    QXD_TRY(blas_zero(c, 0, w.out_e));
    QXD_TRY(blas_zero(c, 0, w.out_o));
    info->iters = 0; info->n_reliable = 0; info->true_res = 0.0;
    status = QXD_OK;
  } else {
    // source preparation (row a8): b = eta_e - D_eo A_oo^{-1} eta_o
    QXD_TRY(launch_clover_apply(c, 0, 1, 1, w.eta_o, w.tmp_o_hi));
    DslashCall d{};
    d.prec = 0; d.mode = DS_X_MHOP; d.parity_out = 0; d.in[1] = w.tmp_o_hi; d.phi = w.eta_e; d.out[0] = w.b;
    QXD_TRY(launch_dslash(c, d));
    const double stop2 = tol * tol * eta2;
    status = (info->algo == QXD_BICGSTAB) ? bicgstab(c, plo, w, stop2, delta, maxiter, info) : cgne(c, plo, w, stop2, delta, maxiter, info);
    if (status != QXD_OK && status != QXD_ENOCONV) return status;
    info->true_res = std::sqrt(info->true_res / eta2);
    // reconstruction (row a8): psi_o = A_oo^{-1}(eta_o - D_oe psi_e)
    DslashCall r{};
    r.prec = 0; r.mode = DS_AINV_X_MHOP; r.parity_out = 1; r.in[0] = w.xhi; r.phi = w.eta_o; r.out[1] = w.out_o;
    QXD_TRY(launch_dslash(c, r));
    QXD_TRY(blas_copy(c, 0, w.xhi, w.out_e));
  }
  QXD_TRY(launch_spinor_unpack(c, 0, c->full_b, psi_nat, 3, 0));
  QXD_CUDA_OK(c, cudaEventRecord(c->ev1, c->stream));
  QXD_CUDA_OK(c, cudaEventSynchronize(c->ev1));
  float ms = 0.f;
  QXD_CUDA_OK(c, cudaEventElapsedTime(&ms, c->ev0, c->ev1));
  info->seconds = ms * 1e-3;
  if (status == QXD_ENOCONV) c->err = "solve: not converged (maxiter or breakdown); psi holds the best iterate";
  return status;
}


// ---------------------------------------------------------------------------------------------------------------
// Batched solve (rows a7 + a10, BASELINE config 4): nrhs independent CG iterations on the normal equations of D-hat
// run in lockstep, so that every sloppy operator application is one multi-RHS dslash launch (links and clover blocks
// read once for all right-hand sides, "solution of this system for many right-hand sides").  Every system
// keeps its own scalars (device arrays, SS doubles apart) and its own reliable-update schedule; a system that has met
// the fp64 residual target is frozen (alpha = beta = 0) until all are done.  Source preparation, reliable updates and
// reconstruction run per right-hand side through the single-RHS fp64 kernels.
// ---------------------------------------------------------------------------------------------------------------
int solve_eo_multi(qxd_ctx* c, int nrhs, const double* eta_nat, double* psi_nat, double tol, qxd_solve_info* info) {
  const int Vh = c->g.Vh;
  const int pop = info[0].sloppy;   // precision of the sloppy operator
  // binary16 operator: the Krylov vectors x, r, p stay in fp32 (reading R12) when the batch workspace is sized for fp32
  const bool h16 = (pop == 2 && c->mlo_size >= 4);
  const int plo = h16 ? 1 : pop;    // precision of the Krylov vectors
  if (nrhs < 1 || nrhs > c->nrhs) return fail(c, QXD_EINVAL, "solve_multi: nrhs exceeds the value the workspace was bound for");
  if (pop < 0 || pop >= NPREC || !((c->prec_mask >> pop) & 1)) return fail(c, QXD_EINVAL, "solve_multi: sloppy precision not bound");
  if (prec_size(plo) > c->mlo_size) return fail(c, QXD_EINVAL, "solve_multi: the batch workspace is sized for a narrower sloppy precision");
  if (info[0].algo != QXD_CGNE) return fail(c, QXD_EINVAL, "solve_multi: only QXD_CGNE is batched");
  if (!(tol > 0.0)) return fail(c, QXD_EINVAL, "solve_multi: tol must be > 0");
  const double delta = info[0].delta > 0.0 ? info[0].delta : 0.1;
  const int maxiter = info[0].maxiter > 0 ? info[0].maxiter : 10000;
  enum { SS = 8, M_GAM0 = 0, M_GAM1 = 1, M_TT = 2, M_RR = 3, M_RRT = 4 };
  const size_t rs_hi = half_bytes(0, Vh), rs_lo = (half_bytes(plo, Vh) + 255) & ~size_t(255);
  const size_t rs_op = (half_bytes(pop, Vh) + 255) & ~size_t(255);   // operator inputs / outputs
  const size_t vnat = size_t(c->V) * 24;
  // single-RHS scratch (fp64)
  SpinorPtr eta_e = half_view(0, c->full_a, Vh, 0), eta_o = half_view(0, c->full_a, Vh, 1);
  SpinorPtr out_e = half_view(0, c->full_b, Vh, 0), out_o = half_view(0, c->full_b, Vh, 1);
  SpinorPtr thi = hv(0, c->sp64[3], Vh), tmp_o_hi = hv(0, c->sp64[4], Vh), rhi = hv(0, c->sp64[2], Vh);
  // batch vectors
  SpinorPtr B = hv(0, c->mhi[0], Vh), X = hv(0, c->mhi[1], Vh);
  SpinorPtr xlo = hv(plo, c->mlo[0], Vh), rlo = hv(plo, c->mlo[1], Vh), p = hv(plo, c->mlo[2], Vh), t = hv(pop, c->mlo[3], Vh),
            tmp_o = hv(pop, c->mlo[4], Vh);
  SpinorPtr r16 = hv(pop, c->mlo[5], Vh), p16 = hv(pop, c->mlo[6], Vh);   // binary16 copies the operator reads (h16 only)
  const SpinorPtr& rin = h16 ? r16 : rlo;
  const SpinorPtr& pin = h16 ? p16 : p;
  double* ms = c->mscal;
  double* hs = c->h_mscal;
  Batch bl; bl.n = nrhs; bl.rs = rs_lo; bl.ss = SS; bl.act = c->mact;
  Batch bo = bl; bo.rs = rs_op;
  Batch bh; bh.n = nrhs; bh.rs = rs_hi; bh.ss = SS;

  QXD_CUDA_OK(c, cudaEventRecord(c->ev0, c->stream));
  double eta2[64], stop2[64], maxr[64], rr_true[64];
  int done[64], nrel[64], iters[64];
  // ---- per right-hand side: pack, |eta|^2, source preparation b_k = eta_e - D_eo A_oo^{-1} eta_o (row a8) ----
  for (int k = 0; k < nrhs; k++) {
    QXD_TRY(launch_spinor_pack(c, 0, eta_nat + vnat * k, c->full_a, 3, 0));
    QXD_TRY(blas_norm2(c, 0, eta_e, c->scal + SC_NE));
    QXD_TRY(blas_norm2(c, 0, eta_o, c->scal + SC_NO));
    double nn[2];
    QXD_TRY(read_scal(c, SC_NE, 2, nn));
    eta2[k] = nn[0] + nn[1];
    stop2[k] = tol * tol * eta2[k];
    QXD_TRY(launch_clover_apply(c, 0, 1, 1, eta_o, tmp_o_hi));
    DslashCall d{};
    d.prec = 0; d.mode = DS_X_MHOP; d.parity_out = 0; d.in[1] = tmp_o_hi; d.phi = eta_e; d.out[0] = rhs_view(B, rs_hi, k);
    QXD_TRY(launch_dslash(c, d));
  }
  QXD_TRY(blas_zero(c, 0, X, bh));
  QXD_TRY(blas_zero(c, plo, xlo, bl));
  QXD_TRY(blas_norm2(c, 0, B, ms + M_RRT, bh));
  QXD_TRY(launch_convert_spinor(c, 0, B, plo, rlo, nrhs, rs_hi, rs_lo));
  if (h16) QXD_TRY(launch_convert_spinor(c, 0, B, pop, r16, nrhs, rs_hi, rs_op));
  QXD_CUDA_OK(c, cudaMemcpyAsync(hs, ms, sizeof(double) * SS * nrhs, cudaMemcpyDeviceToHost, c->stream));
  QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
  int nactive = 0;
  for (int k = 0; k < nrhs; k++) {
    rr_true[k] = hs[k * SS + M_RRT];
    maxr[k] = std::sqrt(rr_true[k]);
    done[k] = (rr_true[k] <= stop2[k]) ? 1 : 0;   // includes eta_k = 0
    nrel[k] = 0; iters[k] = 0;
    c->h_mact[k] = done[k] ? 0.0 : 1.0;
    nactive += !done[k];
  }
  QXD_CUDA_OK(c, cudaMemcpyAsync(c->mact, c->h_mact, sizeof(double) * nrhs, cudaMemcpyHostToDevice, c->stream));
  // fp64 true residuals of the systems in `list`:  x_hi += x_lo; x_lo = 0; r = b - D-hat x_hi; r_lo = r.  All of them are
  // enqueued back to back (their |r|^2 go to the systems' own device slots) and read back with ONE host round trip.
  auto reliable = [&](const int* list, int n) -> int {
    if (n == 0) return QXD_OK;
    for (int i = 0; i < n; i++) {
      const int k = list[i];
      SpinorPtr xk = rhs_view(X, rs_hi, k);
      QXD_TRY(blas_acc_hi(c, plo, rhs_view(xlo, rs_lo, k), xk));
      QXD_TRY(apply_dhat(c, 0, xk, thi, tmp_o_hi, 0, nullptr));
      QXD_TRY(blas_sub_norm(c, 0, rhs_view(B, rs_hi, k), thi, rhi, ms + k * SS + M_RRT));
      QXD_TRY(launch_convert_spinor(c, 0, rhi, plo, rhs_view(rlo, rs_lo, k)));
      if (h16) QXD_TRY(launch_convert_spinor(c, 0, rhi, pop, rhs_view(r16, rs_op, k)));
      nrel[k]++;
    }
    QXD_CUDA_OK(c, cudaMemcpyAsync(hs, ms, sizeof(double) * SS * nrhs, cudaMemcpyDeviceToHost, c->stream));
    QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    for (int i = 0; i < n; i++) rr_true[list[i]] = hs[list[i] * SS + M_RRT];
    return QXD_OK;
  };
  int it = 0;
  if (nactive) {
    QXD_TRY(apply_dhat(c, pop, rin, t, tmp_o, 1, ms + M_GAM0, bo));   // s = A^dag r (s shares the buffer of t)
    QXD_TRY(launch_convert_spinor(c, pop, t, plo, p, nrhs, rs_op, rs_lo));
    if (h16) QXD_TRY(blas_copy(c, pop, t, p16, bo));
  }
  while (nactive && it < maxiter) {
    double* gam = ms + M_GAM0 + (it & 1);
    double* gam_next = ms + M_GAM0 + ((it + 1) & 1);
    QXD_TRY(apply_dhat(c, pop, pin, t, tmp_o, 0, ms + M_TT, bo));
    if (h16) QXD_TRY(blas_cg_xr_h(c, gam, ms + M_TT, p16, t, xlo, rlo, r16, ms + M_RR, bl, rs_op));
    else QXD_TRY(blas_cg_xr(c, plo, gam, ms + M_TT, p, t, xlo, rlo, ms + M_RR, bl));
    // the |r|^2 of all systems travel to the host while s = A^dag r of the whole batch is already running (as in the
    // single-RHS loop): the GPU does not idle on the round trip; systems that do a reliable update get their s redone below
    QXD_CUDA_OK(c, cudaMemcpyAsync(hs, ms, sizeof(double) * SS * nrhs, cudaMemcpyDeviceToHost, c->stream));
    QXD_CUDA_OK(c, cudaEventRecord(c->ev_scal, c->stream));
    QXD_TRY(apply_dhat(c, pop, rin, t, tmp_o, 1, gam_next, bo));
    QXD_CUDA_OK(c, cudaEventSynchronize(c->ev_scal));
    it++;
    bool changed = false;
    int upd[64], nupd = 0;
    for (int k = 0; k < nrhs; k++) {
      if (done[k]) continue;
      iters[k] = it;
      const double rr = hs[k * SS + M_RR];
      if (!(rr == rr)) {   // breakdown: freeze the system and drop its poisoned x_lo (x_hi of the last reliable update is returned)
        done[k] = 2; c->h_mact[k] = 0.0; changed = true; nactive--;
        QXD_TRY(blas_zero(c, plo, rhs_view(xlo, rs_lo, k)));
        continue;
      }
      const double rn = std::sqrt(rr);
      if (rn > maxr[k]) maxr[k] = rn;
      if (rn < delta * maxr[k] || rr <= stop2[k]) upd[nupd++] = k;
    }
    QXD_TRY(reliable(upd, nupd));
    for (int i = 0; i < nupd; i++) {
      const int k = upd[i];
      maxr[k] = std::sqrt(rr_true[k]);
      if (rr_true[k] <= stop2[k]) { done[k] = 1; c->h_mact[k] = 0.0; changed = true; nactive--; }
      else   // s_k = A^dag r_k from the corrected residual (single-RHS launch into the system's slots of the batch)
        QXD_TRY(apply_dhat(c, pop, rhs_view(rin, rs_op, k), rhs_view(t, rs_op, k), rhs_view(tmp_o, rs_op, k), 1, gam_next + k * SS));
    }
    if (changed) QXD_CUDA_OK(c, cudaMemcpyAsync(c->mact, c->h_mact, sizeof(double) * nrhs, cudaMemcpyHostToDevice, c->stream));
    if (!nactive) break;
    if (h16) QXD_TRY(blas_cg_p_h(c, gam_next, gam, t, p, p16, bl, rs_op));
    else QXD_TRY(blas_cg_p(c, plo, gam_next, gam, t, p, bl));
  }
  {   // systems that did not converge: leave the best iterate with its true residual
    int upd[64], nupd = 0;
    for (int k = 0; k < nrhs; k++) if (done[k] != 1) upd[nupd++] = k;
    QXD_TRY(reliable(upd, nupd));
    for (int i = 0; i < nupd; i++) if (rr_true[upd[i]] <= stop2[upd[i]]) done[upd[i]] = 1;
  }
  int status = QXD_OK;
  for (int k = 0; k < nrhs; k++) {
    if (done[k] != 1) status = QXD_ENOCONV;
    // reconstruction (row a8): psi_o = A_oo^{-1}(eta_o - D_oe psi_e)
    QXD_TRY(launch_spinor_pack(c, 0, eta_nat + vnat * k, c->full_a, 2, 0));
    DslashCall r{};
    r.prec = 0; r.mode = DS_AINV_X_MHOP; r.parity_out = 1; r.in[0] = rhs_view(X, rs_hi, k); r.phi = eta_o; r.out[1] = out_o;
    QXD_TRY(launch_dslash(c, r));
    QXD_TRY(blas_copy(c, 0, rhs_view(X, rs_hi, k), out_e));
    QXD_TRY(launch_spinor_unpack(c, 0, c->full_b, psi_nat + vnat * k, 3, 0));
  }
  QXD_CUDA_OK(c, cudaEventRecord(c->ev1, c->stream));
  QXD_CUDA_OK(c, cudaEventSynchronize(c->ev1));
  float ms_el = 0.f;
  QXD_CUDA_OK(c, cudaEventElapsedTime(&ms_el, c->ev0, c->ev1));
  for (int k = 0; k < nrhs; k++) {
    info[k].algo = info[0].algo; info[k].sloppy = pop; info[k].delta = delta; info[k].maxiter = maxiter;
    info[k].iters = iters[k]; info[k].n_reliable = nrel[k];
    info[k].true_res = eta2[k] > 0.0 ? std::sqrt(rr_true[k] / eta2[k]) : 0.0;
    info[k].seconds = ms_el * 1e-3;
  }
  if (status == QXD_ENOCONV) c->err = "solve_multi: at least one system not converged (maxiter or breakdown); psi holds the best iterates";
  return status;
}

}  // namespace qxd
