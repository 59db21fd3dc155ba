// dslash.cu -- launch front end of the dslash kernels (dslash_kernel.cuh) and the stand-alone clover multiply; SURVEY.md §8 rows a4 (D_w apply), a5 (D-hat even-odd passes) and the dslash-shaped parts
#include "dslash_args.h"
#include "block_algebra.cuh"
#include <cstdlib>

namespace qxd {

namespace {

// M v or M^{-1} v for one site; in the C*-paired layout the record is that of the physical site and the mirror image uses
// sigma2 M^* sigma2, applied as sigma2 conj(M conj(sigma2 v)) (see dslash_kernel.cuh)
template <typename S>
__device__ __forceinline__ void clover_mul(const void* CL, const Geom& g, int cb, const typename PT<S>::C* in, typename PT<S>::C* out) {
  typedef typename PT<S>::C C;
  const bool mir = g.pair && (cb & 1);
  const int rec = g.pair ? (cb >> 1) : cb;
  C b[36];
#pragma unroll
  for (int blk = 0; blk < 2; blk++) {
    if (blk == 0) load_reals<S, 0, 36>(CL, g.Vg, rec, b); else load_reals<S, 36, 36>(CL, g.Vg, rec, b);
    C a[12], w[12];
    mirror_in(in + 12 * blk, a, mir);
    block_mul(b, a, w);
    mirror_out(w, out + 12 * blk, mir);
  }
}

template <typename S, int INV_DUMMY>
__global__ void __launch_bounds__(128) clover_apply_k(Geom g, const void* CL, SpinorPtr in, SpinorPtr out) {
  typedef typename PT<S>::C C;
  const int Vh = g.Vh;
  const int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  C v[24], w[24];
  load_spinor<S>(in, Vh, cb, v);
  clover_mul<S>(CL, g, cb, v, w);
  store_spinor<S>(out, Vh, cb, w);
}

}  // namespace

int launch_dslash(qxd_ctx* c, const DslashCall& d) {
  if (d.prec < 0 || d.prec >= NPREC || !((c->prec_mask >> d.prec) & 1)) return fail(c, QXD_EINVAL, "dslash: precision not bound");
  DslashArgs a;
  a.g = c->g;
  a.in[0] = d.in[0]; a.in[1] = d.in[1];
  a.phi = d.phi;
  a.out[0] = d.out[0]; a.out[1] = d.out[1];
  a.W[0] = c->W[d.prec][0]; a.W[1] = c->W[d.prec][1];
  const bool inv = (d.mode == DS_HOP_AINV || d.mode == DS_AINV_X_MHOP);
  a.CL[0] = inv ? c->Mi[d.prec][0] : c->M[d.prec][0];
  a.CL[1] = inv ? c->Mi[d.prec][1] : c->M[d.prec][1];
  a.parity_out = d.parity_out;
  if (inv && !a.CL[d.parity_out & 1]) return fail(c, QXD_EINVAL, "dslash: the inverse clover blocks of the even sites exist in fp64 only");
  a.nrhs = d.nrhs > 1 ? d.nrhs : 1; a.ngroups = 1;
  a.rs_in = d.rs_in; a.rs_phi = d.rs_phi; a.rs_out = d.rs_out;
  a.tm = d.tm;
  a.t_lo = d.t_hi > 0 ? d.t_lo : 0; a.t_hi = d.t_hi > 0 ? d.t_hi : 0x7fffffff;
  if (a.nrhs > 64) return fail(c, QXD_EINVAL, "dslash: at most 64 right-hand sides per launch");
  a.R.partials = c->partials; a.R.result = d.norm_result; a.R.rstride = d.norm_stride;
  typedef int (*Dispatch)(qxd_ctx*, const DslashCall&, DslashArgs&);
  static const Dispatch table[3][2][2] = {   // [precision][14-real links][paired layout]
      {{dslash_dispatch_f64_l18_p0, dslash_dispatch_f64_l18_p1}, {dslash_dispatch_f64_l14_p0, dslash_dispatch_f64_l14_p1}},
      {{dslash_dispatch_f32_l18_p0, dslash_dispatch_f32_l18_p1}, {dslash_dispatch_f32_l14_p0, dslash_dispatch_f32_l14_p1}},
      {{dslash_dispatch_f16_l18_p0, dslash_dispatch_f16_l18_p1}, {dslash_dispatch_f16_l14_p0, dslash_dispatch_f16_l14_p1}}};
  int rc = table[d.prec][c->link_reals[d.prec] == 14 ? 1 : 0][c->g.pair ? 1 : 0](c, d, a);
  if (rc) return rc;
  QXD_LAUNCH_CHECK(c);
  if (d.flags & DSF_NORM) {   // second kernel of the fused norm: add the per-tile partials (qxd_common.cuh)
    reduce_finalize_k<1><<<dim3(1, a.nrhs), FINALIZE_THREADS, 0, c->stream>>>(a.R, (c->g.Vh + 127) / 128);
    QXD_LAUNCH_CHECK(c);
  } else if (d.flags & DSF_DOT) {
    reduce_finalize_k<3><<<dim3(1, a.nrhs), FINALIZE_THREADS, 0, c->stream>>>(a.R, (c->g.Vh + 127) / 128);
    QXD_LAUNCH_CHECK(c);
  }
  return QXD_OK;
}

int launch_clover_apply(qxd_ctx* c, int prec, int inverse, int parity, const SpinorPtr& in, const SpinorPtr& out) {
  const void* CL = inverse ? c->Mi[prec][parity] : c->M[prec][parity];
  dim3 gr((c->g.Vh + 127) / 128);
  if (prec == 0) clover_apply_k<double, 0><<<gr, 128, 0, c->stream>>>(c->g, CL, in, out);
  else if (prec == 1) clover_apply_k<float, 0><<<gr, 128, 0, c->stream>>>(c->g, CL, in, out);
  else clover_apply_k<__half, 0><<<gr, 128, 0, c->stream>>>(c->g, CL, in, out);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // namespace qxd
