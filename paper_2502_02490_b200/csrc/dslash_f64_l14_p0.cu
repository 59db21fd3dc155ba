// dslash_f64_l14_p0.cu -- instantiates the dslash kernels (dslash_kernel.cuh) for double storage,
// 14 stored reals per link (rows 0, 1 + det: 12-real reconstruct with the U(1) phase fused), extended-lattice layout.
#include "dslash_kernel.cuh"

namespace qxd {
int dslash_dispatch_f64_l14_p0(qxd_ctx* c, const DslashCall& d, DslashArgs& a) { return dispatch<double, 14, false>(c, d, a); }
}  // namespace qxd
