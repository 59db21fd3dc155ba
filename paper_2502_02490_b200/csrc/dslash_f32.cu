// dslash_f32.cu -- instantiates the dslash kernels (dslash_kernel.cuh) for float storage.
#include "dslash_kernel.cuh"

namespace qxd {
int dslash_dispatch_f32(qxd_ctx* c, const DslashCall& d, DslashArgs& a) { return dispatch<float>(c, d, a); }
}  // namespace qxd
