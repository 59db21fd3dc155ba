// gcr.cu -- SURVEY.md §8(f) row f3, the outer solver: flexible restarted GCR on the full-lattice D_w with the Schwarz
// alternating procedure (sap.cu) as preconditioner -- the solver family the paper measures ("heavily preconditioned GCR",
// PAPER.md:164; mixed half/single/double precision).
//
//   cycle:  for k < nkv:  z_k = M_sap r ;  w_k = D_w z_k (fp32) ;  w_k -= sum_{j<k} <w_j, w_k>/|w_j|^2 w_j ;
//                         r -= <w_k, r>/|w_k|^2 w_k
//   restart: solve the triangular system b y = c of the orthogonalisation coefficients (device, one thread),
//            psi += sum_k y_k z_k in fp64, r = eta - D_w psi in fp64 (the only residual convergence is declared on).
// All coefficients stay on the device; the host reads one scalar (|r|^2) per step to decide about restart and stop.
// A packed fp32 full-lattice spinor is a flat array of 12 Vh float4 (chunk-major per parity, qxd_common.cuh), so the
// vector kernels here are flat grid-stride loops; (re, im) pairs never straddle a float4.
#include "gcr_kernels.cuh"
#include <cmath>

namespace qxd {

namespace {

#define QXD_TRY(expr)        \
  do {                       \
    int rc__ = (expr);       \
    if (rc__) return rc__;   \
  } while (0)

// x (fp64 packed full lattice: 24 Vh double2) += sum_{k<K} y_k z_k (fp32).  fp32 chunk c of a parity holds the reals of the
// fp64 chunks 2c and 2c+1 of the same parity and site.
__global__ void __launch_bounds__(256) gcr_update_x_k(int Vh, VecList Z, int K, const double* __restrict__ y, double2* __restrict__ x) {
  __shared__ double yr[32], yi[32];
  if (threadIdx.x < K) { yr[threadIdx.x] = y[2 * threadIdx.x]; yi[threadIdx.x] = y[2 * threadIdx.x + 1]; }
  __syncthreads();
  const size_t n4 = size_t(12) * Vh;
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n4; i += size_t(gridDim.x) * blockDim.x) {
    const size_t pc = i / Vh, cb = i - pc * Vh;      // pc = parity * 6 + chunk
    const size_t i64 = (2 * pc) * Vh + cb;
    double2 a = x[i64], b = x[i64 + Vh];
    for (int k = 0; k < K; k++) {
      const float4 z = __ldg(Z.v[k] + i);
      a.x += yr[k] * z.x - yi[k] * z.y; a.y += yr[k] * z.y + yi[k] * z.x;
      b.x += yr[k] * z.z - yi[k] * z.w; b.y += yr[k] * z.w + yi[k] * z.z;
    }
    x[i64] = a; x[i64 + Vh] = b;
  }
}
// r64 = b - t (t may be null: r64 = b) ;  r32 = float(r64) ;  result = |r64|^2
__global__ void __launch_bounds__(256) gcr_resid_k(int Vh, const double2* __restrict__ b, const double2* __restrict__ t, double2* __restrict__ r64,
                                                   float4* __restrict__ r32, Reducer R) {
  const size_t n4 = size_t(12) * Vh;
  double acc[1] = {0.0};
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n4; i += size_t(gridDim.x) * blockDim.x) {
    const size_t pc = i / Vh, cb = i - pc * Vh;
    const size_t i64 = (2 * pc) * Vh + cb;
    double2 u = b[i64], v = b[i64 + Vh];
    if (t) { const double2 p = t[i64], q = t[i64 + Vh]; u.x -= p.x; u.y -= p.y; v.x -= q.x; v.y -= q.y; }
    r64[i64] = u; r64[i64 + Vh] = v;
    r32[i] = make_float4((float)u.x, (float)u.y, (float)v.x, (float)v.y);
    acc[0] += u.x * u.x + u.y * u.y + v.x * v.x + v.y * v.y;
  }
  grid_reduce<1>(acc, R, blockIdx.x, gridDim.x, 0);
}

struct Gcr {
  qxd_ctx* c;
  int nblk;
  size_t n4;
  Reducer red(double* result) const { Reducer R; R.partials = c->partials; R.result = result; R.rstride = 0; return R; }
  template <int N> int finalize(double* result) {
    reduce_finalize_k<N><<<dim3(1, 1), FINALIZE_THREADS, 0, c->stream>>>(red(result), nblk);
    QXD_LAUNCH_CHECK(c);
    return QXD_OK;
  }
  int read(int idx, int n, double* out) {
    QXD_CUDA_OK(c, cudaMemcpyAsync(c->h_scal, c->gscal + idx, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
    QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    for (int i = 0; i < n; i++) out[i] = c->h_scal[i];
    return QXD_OK;
  }
};

}  // namespace

// K steps of the flexible GCR in fp32 without any host round trip (the inverse iteration of the deflation setup, dfl.cu):
// on entry c->g_r holds the right-hand side b (it is overwritten with the residual), on exit x ~ D_w^{-1} b.  Uses the Krylov
// vectors gz / gw [0, K) and the scalars of the solver; no convergence test.
int gcr_cycle32(qxd_ctx* c, int pprec, bool use_dfl, int K, void* x) {
  const int Vh = c->g.Vh;
  if (K < 1 || K > c->gcr_nkv) return fail(c, QXD_EINVAL, "gcr_cycle32: 1 <= K <= nkv");
  Gcr G;
  G.c = c; G.n4 = size_t(12) * Vh;
  G.nblk = Vh / 128 < 1 ? 1 : (Vh / 128 > 148 * 8 ? 148 * 8 : Vh / 128);
  double* S = c->gscal;
  double* tmp = S + 3000;
  float4* r32 = static_cast<float4*>(c->g_r);
  VecList Z, W;
  for (int k = 0; k < 32; k++) { Z.v[k] = static_cast<const float4*>(c->gz[k]); W.v[k] = static_cast<const float4*>(c->gw[k]); }
  for (int k = 0; k < K; k++) {
    if (use_dfl) QXD_TRY(launch_dfl_precond(c, pprec, c->g_r, c->gz[k]));
    else QXD_TRY(launch_sap(c, pprec, c->g_r, c->gz[k]));
    DslashCall d{};
    d.prec = 1; d.mode = DS_DW_FULL; d.flags = 0;
    d.in[0] = half_view(1, c->gz[k], Vh, 0); d.in[1] = half_view(1, c->gz[k], Vh, 1);
    d.out[0] = half_view(1, c->gw[k], Vh, 0); d.out[1] = half_view(1, c->gw[k], Vh, 1);
    QXD_TRY(launch_dslash(c, d));
    float4* wk = static_cast<float4*>(c->gw[k]);
    for (int j0 = 0; j0 < k; j0 += 4) {
      const int nj = k - j0 < 4 ? k - j0 : 4;
      Reducer R = G.red(S + G_BR + (j0 * 32 + k) * 2);
      R.rstride = 64;
      if (nj == 4) gcr_dots_k<4><<<G.nblk, 256, 0, c->stream>>>(G.n4, W, j0, wk, R);
      else if (nj == 3) gcr_dots_k<3><<<G.nblk, 256, 0, c->stream>>>(G.n4, W, j0, wk, R);
      else if (nj == 2) gcr_dots_k<2><<<G.nblk, 256, 0, c->stream>>>(G.n4, W, j0, wk, R);
      else gcr_dots_k<1><<<G.nblk, 256, 0, c->stream>>>(G.n4, W, j0, wk, R);
      QXD_LAUNCH_CHECK(c);
      reduce_finalize_k<2><<<dim3(1, nj), FINALIZE_THREADS, 0, c->stream>>>(R, G.nblk);
      QXD_LAUNCH_CHECK(c);
    }
    gcr_orth_k<<<G.nblk, 256, 0, c->stream>>>(G.n4, W, k, S + G_BR + k * 2, S + G_N2, wk, r32, G.red(tmp));
    QXD_LAUNCH_CHECK(c);
    QXD_TRY(G.finalize<3>(tmp));
    gcr_store3_k<<<1, 1, 0, c->stream>>>(tmp, S + G_N2 + k, S + G_Q + 2 * k);
    QXD_LAUNCH_CHECK(c);
    gcr_update_r_k<<<G.nblk, 256, 0, c->stream>>>(G.n4, wk, S + G_Q + 2 * k, S + G_N2 + k, r32, G.red(S + G_RR));
    QXD_LAUNCH_CHECK(c);
    QXD_TRY(G.finalize<1>(S + G_RR));
  }
  gcr_backsub_k<<<1, 32, 0, c->stream>>>(K, S);
  QXD_LAUNCH_CHECK(c);
  gcr_update_x32_k<<<G.nblk, 256, 0, c->stream>>>(G.n4, Z, K, S + G_Y, static_cast<float4*>(x), 1);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

int solve_gcr(qxd_ctx* c, const double* eta_nat, double* psi_nat, double tol, qxd_solve_info* info) {
  const int Vh = c->g.Vh;
  const int pprec = info->sloppy;   // storage precision of the SAP block operator
  if (c->gcr_nkv < 1 || !c->gz[0]) return fail(c, QXD_EWORKSPACE, "solve: QXD_GCR needs qxd_set_gcr(nkv > 0) before qxd_workspace_bind");
  if (pprec != 1 && pprec != 2) return fail(c, QXD_EINVAL, "solve: QXD_GCR takes sloppy = QXD_F32 or QXD_F16 (storage of the SAP block operator)");
  if (!((c->prec_mask >> 1) & 1)) return fail(c, QXD_EINVAL, "solve: QXD_GCR needs fp32 bound (Krylov vectors and the fp32 D_w)");
  if (!(tol > 0.0)) return fail(c, QXD_EINVAL, "solve: tol must be > 0");
  QXD_TRY(sap_check_geometry(c));
  const bool use_dfl = info->algo == QXD_DFL_GCR;
  if (use_dfl && !c->dfl_ready) return fail(c, QXD_ESTATE, "solve: QXD_DFL_GCR needs qxd_deflation_setup (again after every change of the gauge field, quark or clover term)");
  const int maxiter = info->maxiter > 0 ? info->maxiter : 10000;
  const int nkv = c->gcr_nkv;
  Gcr G;
  G.c = c; G.n4 = size_t(12) * Vh;
  G.nblk = Vh / 128 < 1 ? 1 : (Vh / 128 > 148 * 8 ? 148 * 8 : Vh / 128);
  double* S = c->gscal;
  double* tmp = S + 3000;
  SpinorPtr b_e = half_view(0, c->full_a, Vh, 0), b_o = half_view(0, c->full_a, Vh, 1);
  SpinorPtr x_e = half_view(0, c->full_b, Vh, 0), x_o = half_view(0, c->full_b, Vh, 1);
  const double2* b64 = static_cast<const double2*>(c->full_a);
  double2* x64 = static_cast<double2*>(c->full_b);
  double2* r64 = static_cast<double2*>(c->g_r64);
  double2* t64 = static_cast<double2*>(c->g_t64);
  float4* r32 = static_cast<float4*>(c->g_r);
  VecList Z, W;
  for (int k = 0; k < 32; k++) { Z.v[k] = static_cast<const float4*>(c->gz[k]); W.v[k] = static_cast<const float4*>(c->gw[k]); }

  QXD_CUDA_OK(c, cudaEventRecord(c->ev0, c->stream));
  QXD_TRY(launch_spinor_pack(c, 0, eta_nat, c->full_a, 3, 0));
  QXD_TRY(blas_norm2(c, 0, b_e, S + G_NE));
  QXD_TRY(blas_norm2(c, 0, b_o, S + G_NO));
  double nn[2];
  QXD_TRY(G.read(G_NE, 2, nn));
  const double eta2 = nn[0] + nn[1];
  const double stop2 = tol * tol * eta2;
  QXD_TRY(blas_zero(c, 0, x_e));
  QXD_TRY(blas_zero(c, 0, x_o));
  int it = 0, nrel = 0, status = QXD_ENOCONV;
  double rr_true = eta2;
  if (eta2 == 0.0) status = QXD_OK;
  else {
    gcr_resid_k<<<G.nblk, 256, 0, c->stream>>>(Vh, b64, nullptr, r64, r32, G.red(S + G_RRT));
    QXD_LAUNCH_CHECK(c);
    QXD_TRY(G.finalize<1>(S + G_RRT));
  }
  int stalled = 0;
  while (status != QXD_OK && it < maxiter) {
    double rr = rr_true;
    const double rr0 = rr_true;
    int K = 0;
    for (int k = 0; k < nkv && it < maxiter; k++) {
      if (use_dfl) QXD_TRY(launch_dfl_precond(c, pprec, c->g_r, c->gz[k]));    // z_k = two-level preconditioner (dfl.cu)
      else QXD_TRY(launch_sap(c, pprec, c->g_r, c->gz[k]));                    // z_k = M_sap r
      DslashCall d{};                                                           // w_k = D_w z_k (fp32)
      d.prec = 1; d.mode = DS_DW_FULL; d.flags = 0;
      d.in[0] = half_view(1, c->gz[k], Vh, 0); d.in[1] = half_view(1, c->gz[k], Vh, 1);
      d.out[0] = half_view(1, c->gw[k], Vh, 0); d.out[1] = half_view(1, c->gw[k], Vh, 1);
      QXD_TRY(launch_dslash(c, d));
      float4* wk = static_cast<float4*>(c->gw[k]);
      for (int j0 = 0; j0 < k; j0 += 4) {                                       // raw <w_j, w_k>, four at a time
        const int nj = k - j0 < 4 ? k - j0 : 4;
        Reducer R = G.red(S + G_BR + (j0 * 32 + k) * 2);
        R.rstride = 64;
        if (nj == 4) gcr_dots_k<4><<<G.nblk, 256, 0, c->stream>>>(G.n4, W, j0, wk, R);
        else if (nj == 3) gcr_dots_k<3><<<G.nblk, 256, 0, c->stream>>>(G.n4, W, j0, wk, R);
        else if (nj == 2) gcr_dots_k<2><<<G.nblk, 256, 0, c->stream>>>(G.n4, W, j0, wk, R);
        else gcr_dots_k<1><<<G.nblk, 256, 0, c->stream>>>(G.n4, W, j0, wk, R);
        QXD_LAUNCH_CHECK(c);
        reduce_finalize_k<2><<<dim3(1, nj), FINALIZE_THREADS, 0, c->stream>>>(R, G.nblk);
        QXD_LAUNCH_CHECK(c);
      }
      gcr_orth_k<<<G.nblk, 256, 0, c->stream>>>(G.n4, W, k, S + G_BR + k * 2, S + G_N2, wk, r32, G.red(tmp));
      QXD_LAUNCH_CHECK(c);
      QXD_TRY(G.finalize<3>(tmp));
      gcr_store3_k<<<1, 1, 0, c->stream>>>(tmp, S + G_N2 + k, S + G_Q + 2 * k);
      QXD_LAUNCH_CHECK(c);
      gcr_update_r_k<<<G.nblk, 256, 0, c->stream>>>(G.n4, wk, S + G_Q + 2 * k, S + G_N2 + k, r32, G.red(S + G_RR));
      QXD_LAUNCH_CHECK(c);
      QXD_TRY(G.finalize<1>(S + G_RR));
      QXD_TRY(G.read(G_RR, 1, &rr));
      it++; K = k + 1;
      if (!(rr == rr)) break;                         // NaN: leave the cycle, the fp64 restart below decides
      // restart early when the fp32 recursion cannot be trusted further (residual down by 1e-4 within the cycle) or the
      // target looks reached (with a margin: the fp64 residual decides)
      if (rr <= 0.8 * stop2 || rr <= 1e-8 * rr0) break;
    }
    if (rr == rr && K > 0) {
      gcr_backsub_k<<<1, 32, 0, c->stream>>>(K, S);
      QXD_LAUNCH_CHECK(c);
      gcr_update_x_k<<<G.nblk, 256, 0, c->stream>>>(Vh, Z, K, S + G_Y, x64);
      QXD_LAUNCH_CHECK(c);
    }
    // true residual in fp64
    DslashCall d{};
    d.prec = 0; d.mode = DS_DW_FULL; d.flags = 0;
    d.in[0] = x_e; d.in[1] = x_o;
    d.out[0] = half_view(0, c->g_t64, Vh, 0); d.out[1] = half_view(0, c->g_t64, Vh, 1);
    QXD_TRY(launch_dslash(c, d));
    gcr_resid_k<<<G.nblk, 256, 0, c->stream>>>(Vh, b64, t64, r64, r32, G.red(S + G_RRT));
    QXD_LAUNCH_CHECK(c);
    QXD_TRY(G.finalize<1>(S + G_RRT));
    double rt;
    QXD_TRY(G.read(G_RRT, 1, &rt));
    nrel++;
    if (!(rt == rt)) break;                           // the iterate itself is poisoned: nothing left to return but the report
    const double prev = rr_true;
    rr_true = rt;
    if (rt <= stop2) { status = QXD_OK; break; }
    if (!(rr == rr)) break;                           // breakdown inside the cycle: psi holds the iterate of the last restart
    stalled = rt > 0.9801 * prev ? stalled + 1 : 0;   // less than 1 % gain in a whole cycle, three times in a row: stagnation
    if (stalled >= 3) break;
  }
  info->iters = it; info->n_reliable = nrel;
  info->true_res = eta2 > 0.0 ? std::sqrt(rr_true / eta2) : 0.0;
  QXD_TRY(launch_spinor_unpack(c, 0, c->full_b, psi_nat, 3, 0));
  QXD_CUDA_OK(c, cudaEventRecord(c->ev1, c->stream));
  QXD_CUDA_OK(c, cudaEventSynchronize(c->ev1));
  float ms = 0.f;
  QXD_CUDA_OK(c, cudaEventElapsedTime(&ms, c->ev0, c->ev1));
  info->seconds = ms * 1e-3;
  if (status == QXD_ENOCONV) c->err = "solve: GCR not converged (maxiter, stagnation or breakdown); psi holds the last iterate";
  return status;
}

}  // namespace qxd
