// dslash_f16_l14_p1.cu -- instantiates the dslash kernels (dslash_kernel.cuh) for __half storage,
// 14 stored reals per link (rows 0, 1 + det: 12-real reconstruct with the U(1) phase fused), C*-paired layout.
#include "dslash_kernel.cuh"

namespace qxd {
int dslash_dispatch_f16_l14_p1(qxd_ctx* c, const DslashCall& d, DslashArgs& a) { return dispatch<__half, 14, true>(c, d, a); }
}  // namespace qxd
