// dslash_args.h -- kernel argument block of the dslash kernels (dslash_kernel.cuh) and the per-precision dispatchers.
#pragma once
#include "qxd_ctx.h"

namespace qxd {

struct DslashArgs {
  Geom g;
  SpinorPtr in[2];
  SpinorPtr phi;
  SpinorPtr out[2];
  const void* W[2];
  const void* CL[2];
  int parity_out;
  int nrhs;            // right-hand sides in this launch (row a10); 1 for the single-spinor entry points
  int ngroups;         // ceil(nrhs / R): consecutive CTAs work on the same tile for different groups of R right-hand sides
  size_t rs_in, rs_phi, rs_out;   // byte distance between consecutive right-hand sides
  Reducer R;
  TileMap tm;          // subset of tiles this launch works on (identity unless count > 0)
  int t_lo, t_hi;      // only sites with t_lo <= x0 < t_hi are computed (time-slab ranges of the domain decomposition; default: all)
};


// one translation unit per storage precision, link format and layout (dslash_f64_l18_p0.cu, ..., dslash_f16_l14_p1.cu)
int dslash_dispatch_f64_l18_p0(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f64_l18_p1(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f64_l14_p0(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f64_l14_p1(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f32_l18_p0(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f32_l18_p1(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f32_l14_p0(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f32_l14_p1(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f16_l18_p0(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f16_l18_p1(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f16_l14_p0(qxd_ctx* c, const DslashCall& d, DslashArgs& a);
int dslash_dispatch_f16_l14_p1(qxd_ctx* c, const DslashCall& d, DslashArgs& a);

}  // namespace qxd
