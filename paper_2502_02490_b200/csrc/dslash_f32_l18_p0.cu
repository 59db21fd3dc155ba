// dslash_f32_l18_p0.cu -- instantiates the dslash kernels (dslash_kernel.cuh) for float storage,
// 18 stored reals per link (full 3x3 links), extended-lattice layout.
#include "dslash_kernel.cuh"

namespace qxd {
int dslash_dispatch_f32_l18_p0(qxd_ctx* c, const DslashCall& d, DslashArgs& a) { return dispatch<float, 18, false>(c, d, a); }
}  // namespace qxd
