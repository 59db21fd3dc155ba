// dslash_f32_l14.cu -- instantiates the dslash kernels (dslash_kernel.cuh) for float storage
// with 14 stored reals per link (rows 0, 1 + det: 12-real reconstruct with the U(1) phase fused).
#include "dslash_kernel.cuh"

namespace qxd {
int dslash_dispatch_f32_l14(qxd_ctx* c, const DslashCall& d, DslashArgs& a) { return dispatch<float, 14>(c, d, a); }
}  // namespace qxd
