// dslash_f64.cu -- instantiates the dslash kernels (dslash_kernel.cuh) for double storage.
#include "dslash_kernel.cuh"

namespace qxd {
int dslash_dispatch_f64(qxd_ctx* c, const DslashCall& d, DslashArgs& a) { return dispatch<double>(c, d, a); }
}  // namespace qxd
