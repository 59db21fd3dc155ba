// dslash_f64_l18_p1.cu -- instantiates the dslash kernels (dslash_kernel.cuh) for double storage,
// 18 stored reals per link (full 3x3 links), C*-paired layout.
#include "dslash_kernel.cuh"

namespace qxd {
int dslash_dispatch_f64_l18_p1(qxd_ctx* c, const DslashCall& d, DslashArgs& a) { return dispatch<double, 18, true>(c, d, a); }
}  // namespace qxd
