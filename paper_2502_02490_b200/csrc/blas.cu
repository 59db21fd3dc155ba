// blas.cu -- SURVEY.md §8 row a6: BLAS-1 on packed half-lattice spinors (axpy, xpay, complex dot, norm^2
// and the fused forms the solvers use).  The paper does not describe these kernels; any Krylov solver for
// D_w psi = eta needs them.  One thread per site (24 reals = 12/6/3 16-byte chunks,
// coalesced across the warp), fp64 accumulators for every storage precision, warp-shuffle -> block ->
// single-pass grid reduction (qxd_common.cuh).  Solver scalars (alpha, beta, ...) stay on the device: the
// kernels read numerator/denominator from device memory, so the inner loop needs no host round trip.
#include "qxd_ctx.h"

namespace qxd {

namespace {

template <typename S>
__global__ void __launch_bounds__(128) axpy_k(int Vh, double a, SpinorPtr x, SpinorPtr y) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  C vx[24], vy[24];
  load_spinor<S>(x, Vh, cb, vx);
  load_spinor<S>(y, Vh, cb, vy);
#pragma unroll
  for (int i = 0; i < 24; i++) vy[i] += (C)a * vx[i];
  store_spinor<S>(y, Vh, cb, vy);
}

// z = x + a*y + b*w, complex scalars by value (HASW = false: no w term)
template <typename S, bool HASW>
__global__ void __launch_bounds__(128) cxpaypbw_k(int Vh, SpinorPtr x, double ar_, double ai_, SpinorPtr y, double br_, double bi_, SpinorPtr w,
                                                  SpinorPtr z) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  const C ar = (C)ar_, ai = (C)ai_, br = (C)br_, bi = (C)bi_;
  C vx[24], vy[24];
  load_spinor<S>(x, Vh, cb, vx);
  load_spinor<S>(y, Vh, cb, vy);
#pragma unroll
  for (int k = 0; k < 12; k++) {
    C yr = vy[2 * k], yi = vy[2 * k + 1];
    vx[2 * k] += ar * yr - ai * yi;
    vx[2 * k + 1] += ar * yi + ai * yr;
  }
  if (HASW) {
    load_spinor<S>(w, Vh, cb, vy);
#pragma unroll
    for (int k = 0; k < 12; k++) {
      C yr = vy[2 * k], yi = vy[2 * k + 1];
      vx[2 * k] += br * yr - bi * yi;
      vx[2 * k + 1] += br * yi + bi * yr;
    }
  }
  store_spinor<S>(z, Vh, cb, vx);
}

// BiCGstab coefficients from the device-resident reduction results, so that the host need not read them back between the
// kernels of an iteration (one round trip per iteration instead of three):
//   alpha = rho / <r0,v>   (0 if <r0,v> vanishes: the step degenerates to the minimal-residual half, x and r stay consistent)
//   omega = <t,s> / |t|^2  (0 if t vanishes; dst = (Re <s,t>, Im <s,t>, |t|^2) as cdot_k leaves it)
constexpr double BICG_TINY = 1e-290;
__device__ __forceinline__ void bicg_alpha(double rho_re, double rho_im, const double* r0v, double& ar, double& ai) {
  const double br = r0v[0], bi = r0v[1], d = br * br + bi * bi;
  if (d < BICG_TINY) { ar = 0.0; ai = 0.0; return; }
  ar = (rho_re * br + rho_im * bi) / d; ai = (rho_im * br - rho_re * bi) / d;
}
__device__ __forceinline__ void bicg_omega(const double* dst, double& wr, double& wi) {
  const double tt = dst[2];
  if (!(tt > BICG_TINY)) { wr = 0.0; wi = 0.0; return; }
  wr = dst[0] / tt; wi = -dst[1] / tt;
}
//   s = r - alpha v
template <typename S>
__global__ void __launch_bounds__(128) bicg_s_k(int Vh, double rho_re, double rho_im, const double* r0v, SpinorPtr r, SpinorPtr v, SpinorPtr s) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  double ar_, ai_;
  bicg_alpha(rho_re, rho_im, r0v, ar_, ai_);
  const C ar = (C)(-ar_), ai = (C)(-ai_);
  C vx[24], vy[24];
  load_spinor<S>(r, Vh, cb, vx);
  load_spinor<S>(v, Vh, cb, vy);
#pragma unroll
  for (int k = 0; k < 12; k++) {
    C yr = vy[2 * k], yi = vy[2 * k + 1];
    vx[2 * k] += ar * yr - ai * yi;
    vx[2 * k + 1] += ar * yi + ai * yr;
  }
  store_spinor<S>(s, Vh, cb, vx);
}
// BiCGstab, end of an iteration in one pass:  x += alpha p + omega s ;  r = s - omega t ;  result = (<r0,r>, |r|^2)
template <typename S>
__global__ void __launch_bounds__(128) bicg_xr_k(int Vh, double rho_re, double rho_im, const double* r0v, const double* dst, SpinorPtr p, SpinorPtr s,
                                                 SpinorPtr t, SpinorPtr r0, SpinorPtr x, SpinorPtr r, Reducer R) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  double d[3] = {0.0, 0.0, 0.0};
  if (cb < Vh) {
    double ar_, ai_, wr_, wi_;
    bicg_alpha(rho_re, rho_im, r0v, ar_, ai_);
    bicg_omega(dst, wr_, wi_);
    const C ar = (C)ar_, ai = (C)ai_, wr = (C)wr_, wi = (C)wi_;
    C vx[24], va[24], vs[24];
    load_spinor<S>(x, Vh, cb, vx);
    load_spinor<S>(p, Vh, cb, va);
    load_spinor<S>(s, Vh, cb, vs);
#pragma unroll
    for (int k = 0; k < 12; k++) {
      vx[2 * k] += ar * va[2 * k] - ai * va[2 * k + 1] + wr * vs[2 * k] - wi * vs[2 * k + 1];
      vx[2 * k + 1] += ar * va[2 * k + 1] + ai * va[2 * k] + wr * vs[2 * k + 1] + wi * vs[2 * k];
    }
    store_spinor<S>(x, Vh, cb, vx);
    load_spinor<S>(t, Vh, cb, va);
#pragma unroll
    for (int k = 0; k < 12; k++) {
      vs[2 * k] -= wr * va[2 * k] - wi * va[2 * k + 1];
      vs[2 * k + 1] -= wr * va[2 * k + 1] + wi * va[2 * k];
    }
    load_spinor<S>(r0, Vh, cb, va);
    C p0 = 0, p1 = 0, p2 = 0;
#pragma unroll
    for (int k = 0; k < 12; k++) {
      const C xr = va[2 * k], xi = va[2 * k + 1], yr = vs[2 * k], yi = vs[2 * k + 1];
      p0 += xr * yr; p0 += xi * yi;
      p1 += xr * yi; p1 -= xi * yr;
      p2 += yr * yr; p2 += yi * yi;
    }
    d[0] = (double)p0; d[1] = (double)p1; d[2] = (double)p2;
    store_spinor<S>(r, Vh, cb, vs);
  }
  grid_reduce<3>(d, R);
}

// CG on the normal equations, step 1:  alpha = num/den ;  x += alpha p ;  r -= alpha t ;  result = |r|^2
// Batched form (row a10): blockIdx.y = right-hand side; vectors rs bytes apart, scalars ss doubles apart; act (may be null)
// holds 1.0 / 0.0 per right-hand side: a converged system is frozen (alpha = beta = 0).
template <typename S>
__global__ void __launch_bounds__(128) cg_xr_k(int Vh, const double* num, const double* den, SpinorPtr p, SpinorPtr t, SpinorPtr x,
                                               SpinorPtr r, Reducer R, size_t rs, int ss, const double* act) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  double nrm[1] = {0.0};
  const int k = blockIdx.y;
  p = rhs_view(p, rs, k); t = rhs_view(t, rs, k); x = rhs_view(x, rs, k); r = rhs_view(r, rs, k);
  if (cb < Vh) {
    const double dn = den[k * ss];
    const C al = (act && act[k] == 0.0) || dn == 0.0 ? (C)0 : (C)(num[k * ss] / dn);
    C vp[24], vx[24];
    load_spinor<S>(p, Vh, cb, vp);
    load_spinor<S>(x, Vh, cb, vx);
#pragma unroll
    for (int i = 0; i < 24; i++) vx[i] += al * vp[i];
    store_spinor<S>(x, Vh, cb, vx);
    load_spinor<S>(t, Vh, cb, vp);
    load_spinor<S>(r, Vh, cb, vx);
    C part = 0;   // per-site sum in the arithmetic type (fp32 for fp32/fp16 storage), fp64 across sites: the float->double
                  // conversions and DFMAs of a per-element fp64 sum cost more than the memory traffic of this kernel
#pragma unroll
    for (int i = 0; i < 24; i++) { vx[i] -= al * vp[i]; part += vx[i] * vx[i]; }
    nrm[0] = (double)part;
    store_spinor<S>(r, Vh, cb, vx);
  }
  grid_reduce<1>(nrm, R);
}
// step 2:  beta = num/den ;  p = s + beta p
template <typename S>
__global__ void __launch_bounds__(128) cg_p_k(int Vh, const double* num, const double* den, SpinorPtr s, SpinorPtr p, size_t rs, int ss,
                                              const double* act) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  const int k = blockIdx.y;
  s = rhs_view(s, rs, k); p = rhs_view(p, rs, k);
  const double dn = den[k * ss];
  const C be = (act && act[k] == 0.0) || dn == 0.0 ? (C)0 : (C)(num[k * ss] / dn);
  C vs[24], vp[24];
  load_spinor<S>(s, Vh, cb, vs);
  load_spinor<S>(p, Vh, cb, vp);
#pragma unroll
  for (int i = 0; i < 24; i++) vp[i] = vs[i] + be * vp[i];
  store_spinor<S>(p, Vh, cb, vp);
}

// fp16 sloppy operator with fp32 Krylov vectors (reading R12): the CG vectors x, r, p are kept in float,
// only the operator's inputs (p, r) and outputs (t, s) are binary16.  Rounding x, r and p themselves to 11-bit
// mantissas every iteration was measured to cost 2.8x the iterations of the fp32 solver at config c3.
//   x += alpha p16 ; r -= alpha t(half) ; r16 = half(r) ; result = |r|^2
// x takes the binary16 direction the operator was applied to (t = A p16), so that x and r stay consistent (r = b - A x up
// to fp32 rounding) and the fp32 p need not be read here.
__global__ void __launch_bounds__(128) cg_xr_h_k(int Vh, const double* num, const double* den, SpinorPtr p, SpinorPtr t, SpinorPtr x,
                                                 SpinorPtr r, SpinorPtr r16, Reducer R, size_t rs_v, size_t rs_o, int ss, const double* act) {
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  double nrm[1] = {0.0};
  const int k = blockIdx.y;   // right-hand side (batched form, row a10): fp32 vectors rs_v bytes apart, binary16 ones rs_o
  p = rhs_view(p, rs_o, k); x = rhs_view(x, rs_v, k); r = rhs_view(r, rs_v, k); t = rhs_view(t, rs_o, k); r16 = rhs_view(r16, rs_o, k);
  if (cb < Vh) {
    const double dn = den[k * ss];
    const float al = (act && act[k] == 0.0) || dn == 0.0 ? 0.f : (float)(num[k * ss] / dn);
    float vp[24], vx[24];
    load_spinor<__half>(p, Vh, cb, vp);
    load_spinor<float>(x, Vh, cb, vx);
#pragma unroll
    for (int i = 0; i < 24; i++) vx[i] += al * vp[i];
    store_spinor<float>(x, Vh, cb, vx);
    load_spinor<__half>(t, Vh, cb, vp);
    load_spinor<float>(r, Vh, cb, vx);
    float part = 0.f;
#pragma unroll
    for (int i = 0; i < 24; i++) { vx[i] -= al * vp[i]; part += vx[i] * vx[i]; }
    nrm[0] = (double)part;
    store_spinor<float>(r, Vh, cb, vx);
    store_spinor<__half>(r16, Vh, cb, vx);
  }
  grid_reduce<1>(nrm, R);
}
//   p = s(half) + beta p ; p16 = half(p)
__global__ void __launch_bounds__(128) cg_p_h_k(int Vh, const double* num, const double* den, SpinorPtr s, SpinorPtr p, SpinorPtr p16,
                                                size_t rs_v, size_t rs_o, int ss, const double* act) {
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  const int k = blockIdx.y;
  s = rhs_view(s, rs_o, k); p16 = rhs_view(p16, rs_o, k); p = rhs_view(p, rs_v, k);
  const double dn = den[k * ss];
  const float be = (act && act[k] == 0.0) || dn == 0.0 ? 0.f : (float)(num[k * ss] / dn);
  float vs[24], vp[24];
  load_spinor<__half>(s, Vh, cb, vs);
  load_spinor<float>(p, Vh, cb, vp);
#pragma unroll
  for (int i = 0; i < 24; i++) vp[i] = vs[i] + be * vp[i];
  store_spinor<float>(p, Vh, cb, vp);
  store_spinor<__half>(p16, Vh, cb, vp);
}

template <typename S, bool EXACT>
__global__ void __launch_bounds__(128) norm2_k(int Vh, SpinorPtr x, Reducer R, size_t rs) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  double nrm[1] = {0.0};
  x = rhs_view(x, rs, blockIdx.y);
  if (cb < Vh) {
    C v[24];
    load_spinor<S>(x, Vh, cb, v);
    if (EXACT) {
#pragma unroll
      for (int i = 0; i < 24; i++) nrm[0] += (double)v[i] * (double)v[i];
    } else {
      C part = 0;
#pragma unroll
      for (int i = 0; i < 24; i++) part += v[i] * v[i];
      nrm[0] = (double)part;
    }
  }
  grid_reduce<1>(nrm, R);
}
// <x,y> = sum conj(x) y  (re, im) and |y|^2 as a third component
template <typename S, bool EXACT>
__global__ void __launch_bounds__(128) cdot_k(int Vh, SpinorPtr x, SpinorPtr y, Reducer R) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  double d[3] = {0.0, 0.0, 0.0};
  if (cb < Vh) {
    C vx[24], vy[24];
    load_spinor<S>(x, Vh, cb, vx);
    load_spinor<S>(y, Vh, cb, vy);
    if (EXACT) {
#pragma unroll
      for (int k = 0; k < 12; k++) {
        double xr = vx[2 * k], xi = vx[2 * k + 1], yr = vy[2 * k], yi = vy[2 * k + 1];
        d[0] += xr * yr + xi * yi;
        d[1] += xr * yi - xi * yr;
        d[2] += yr * yr + yi * yi;
      }
    } else {
      C p0 = 0, p1 = 0, p2 = 0;
#pragma unroll
      for (int k = 0; k < 12; k++) {
        const C xr = vx[2 * k], xi = vx[2 * k + 1], yr = vy[2 * k], yi = vy[2 * k + 1];
        p0 += xr * yr; p0 += xi * yi;
        p1 += xr * yi; p1 -= xi * yr;
        p2 += yr * yr; p2 += yi * yi;
      }
      d[0] = (double)p0; d[1] = (double)p1; d[2] = (double)p2;
    }
  }
  grid_reduce<3>(d, R);
}

template <typename S>
__global__ void __launch_bounds__(128) zero_k(int Vh, SpinorPtr x, size_t rs) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  x = rhs_view(x, rs, blockIdx.y);
  C v[24];
#pragma unroll
  for (int i = 0; i < 24; i++) v[i] = 0;
  store_spinor<S>(x, Vh, cb, v);
}
// reliable update, solution part: x_hi (fp64) += x_lo (S) ; x_lo = 0
template <typename S>
__global__ void __launch_bounds__(128) acc_hi_k(int Vh, SpinorPtr xlo, SpinorPtr xhi) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  C v[24];
  double h[24];
  load_spinor<S>(xlo, Vh, cb, v);
  load_spinor<double>(xhi, Vh, cb, h);
#pragma unroll
  for (int i = 0; i < 24; i++) { h[i] += (double)v[i]; v[i] = 0; }
  store_spinor<double>(xhi, Vh, cb, h);
  store_spinor<S>(xlo, Vh, cb, v);
}
// r = b - t ; result = |r|^2
template <typename S>
__global__ void __launch_bounds__(128) sub_norm_k(int Vh, SpinorPtr b, SpinorPtr t, SpinorPtr r, Reducer R) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  double nrm[1] = {0.0};
  if (cb < Vh) {
    C vb[24], vt[24];
    load_spinor<S>(b, Vh, cb, vb);
    load_spinor<S>(t, Vh, cb, vt);
#pragma unroll
    for (int i = 0; i < 24; i++) { vb[i] -= vt[i]; nrm[0] += (double)vb[i] * (double)vb[i]; }
    store_spinor<S>(r, Vh, cb, vb);
  }
  grid_reduce<1>(nrm, R);
}

inline Reducer reducer(qxd_ctx* c, double* result, int rstride = 0) {
  Reducer R;
  R.partials = c->partials; R.result = result; R.rstride = rstride;
  return R;
}

}  // namespace

#define QXD_BY_PREC(prec, ...)                                 \
  do {                                                         \
    if ((prec) == 0) { typedef double S; __VA_ARGS__; }        \
    else if ((prec) == 1) { typedef float S; __VA_ARGS__; }    \
    else { typedef __half S; __VA_ARGS__; }                    \
  } while (0)

// second kernel of every reduction: adds the per-block partials of the launch before it (qxd_common.cuh)
#define QXD_FINALIZE(N, res, rstride, nslots)                                                                           \
  do {                                                                                                                  \
    QXD_LAUNCH_CHECK(c);                                                                                                \
    reduce_finalize_k<N><<<dim3(1, (nslots)), FINALIZE_THREADS, 0, c->stream>>>(reducer(c, (res), (rstride)), (c->g.Vh + 127) / 128); \
  } while (0)

#define QXD_GRID dim3((c->g.Vh + 127) / 128), 128, 0, c->stream
#define QXD_GRID_N(n) dim3((c->g.Vh + 127) / 128, (n)), 128, 0, c->stream

int blas_axpy(qxd_ctx* c, int prec, double a, const SpinorPtr& x, const SpinorPtr& y) {
  QXD_BY_PREC(prec, axpy_k<S><<<QXD_GRID>>>(c->g.Vh, a, x, y));
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_cxpaypbw(qxd_ctx* c, int prec, const SpinorPtr& x, double ar, double ai, const SpinorPtr& y, double br, double bi,
                  const SpinorPtr& w, const SpinorPtr& z) {
  if (br == 0.0 && bi == 0.0) QXD_BY_PREC(prec, cxpaypbw_k<S, false><<<QXD_GRID>>>(c->g.Vh, x, ar, ai, y, br, bi, w, z));
  else QXD_BY_PREC(prec, cxpaypbw_k<S, true><<<QXD_GRID>>>(c->g.Vh, x, ar, ai, y, br, bi, w, z));
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_bicg_s(qxd_ctx* c, int prec, double rho_re, double rho_im, const double* r0v, const SpinorPtr& r, const SpinorPtr& v, const SpinorPtr& s) {
  QXD_BY_PREC(prec, bicg_s_k<S><<<QXD_GRID>>>(c->g.Vh, rho_re, rho_im, r0v, r, v, s));
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_bicg_xr(qxd_ctx* c, int prec, double rho_re, double rho_im, const double* r0v, const double* dst, const SpinorPtr& p, const SpinorPtr& s,
                 const SpinorPtr& t, const SpinorPtr& r0, const SpinorPtr& x, const SpinorPtr& r, double* res3) {
  QXD_BY_PREC(prec, bicg_xr_k<S><<<QXD_GRID>>>(c->g.Vh, rho_re, rho_im, r0v, dst, p, s, t, r0, x, r, reducer(c, res3)));
  QXD_FINALIZE(3, res3, 0, 1);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_cg_xr(qxd_ctx* c, int prec, const double* num, const double* den, const SpinorPtr& p, const SpinorPtr& t, const SpinorPtr& x,
               const SpinorPtr& r, double* rr, const Batch& b) {
  QXD_BY_PREC(prec, cg_xr_k<S><<<QXD_GRID_N(b.n)>>>(c->g.Vh, num, den, p, t, x, r, reducer(c, rr, b.ss), b.rs, b.ss, b.act));
  QXD_FINALIZE(1, rr, b.ss, b.n);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_cg_p(qxd_ctx* c, int prec, const double* num, const double* den, const SpinorPtr& s, const SpinorPtr& p, const Batch& b) {
  QXD_BY_PREC(prec, cg_p_k<S><<<QXD_GRID_N(b.n)>>>(c->g.Vh, num, den, s, p, b.rs, b.ss, b.act));
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_cg_xr_h(qxd_ctx* c, const double* num, const double* den, const SpinorPtr& p, const SpinorPtr& t, const SpinorPtr& x,
                 const SpinorPtr& r, const SpinorPtr& r16, double* rr, const Batch& b, size_t rs_o) {
  cg_xr_h_k<<<QXD_GRID_N(b.n)>>>(c->g.Vh, num, den, p, t, x, r, r16, reducer(c, rr, b.ss), b.rs, rs_o, b.ss, b.act);
  QXD_FINALIZE(1, rr, b.ss, b.n);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_cg_p_h(qxd_ctx* c, const double* num, const double* den, const SpinorPtr& s, const SpinorPtr& p, const SpinorPtr& p16,
                const Batch& b, size_t rs_o) {
  cg_p_h_k<<<QXD_GRID_N(b.n)>>>(c->g.Vh, num, den, s, p, p16, b.rs, rs_o, b.ss, b.act);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_norm2(qxd_ctx* c, int prec, const SpinorPtr& x, double* res, const Batch& b, bool exact) {
  if (exact) QXD_BY_PREC(prec, norm2_k<S, true><<<QXD_GRID_N(b.n)>>>(c->g.Vh, x, reducer(c, res, b.ss), b.rs));
  else QXD_BY_PREC(prec, norm2_k<S, false><<<QXD_GRID_N(b.n)>>>(c->g.Vh, x, reducer(c, res, b.ss), b.rs));
  QXD_FINALIZE(1, res, b.ss, b.n);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_cdot(qxd_ctx* c, int prec, const SpinorPtr& x, const SpinorPtr& y, double* res3, bool exact) {
  if (exact) QXD_BY_PREC(prec, cdot_k<S, true><<<QXD_GRID>>>(c->g.Vh, x, y, reducer(c, res3)));
  else QXD_BY_PREC(prec, cdot_k<S, false><<<QXD_GRID>>>(c->g.Vh, x, y, reducer(c, res3)));
  QXD_FINALIZE(3, res3, 0, 1);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_zero(qxd_ctx* c, int prec, const SpinorPtr& x, const Batch& b) {
  QXD_BY_PREC(prec, zero_k<S><<<QXD_GRID_N(b.n)>>>(c->g.Vh, x, b.rs));
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_copy(qxd_ctx* c, int prec, const SpinorPtr& x, const SpinorPtr& y, const Batch& b) {
  return launch_convert_spinor(c, prec, x, prec, y, b.n, b.rs, b.rs);
}
int blas_acc_hi(qxd_ctx* c, int prec, const SpinorPtr& xlo, const SpinorPtr& xhi) {
  QXD_BY_PREC(prec, acc_hi_k<S><<<QXD_GRID>>>(c->g.Vh, xlo, xhi));
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int blas_sub_norm(qxd_ctx* c, int prec, const SpinorPtr& b, const SpinorPtr& t, const SpinorPtr& r, double* res) {
  QXD_BY_PREC(prec, sub_norm_k<S><<<QXD_GRID>>>(c->g.Vh, b, t, r, reducer(c, res)));
  QXD_FINALIZE(1, res, 0, 1);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // namespace qxd
