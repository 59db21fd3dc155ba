// dslash_f16.cu -- instantiates the dslash kernels (dslash_kernel.cuh) for __half storage.
#include "dslash_kernel.cuh"

namespace qxd {
int dslash_dispatch_f16(qxd_ctx* c, const DslashCall& d, DslashArgs& a) { return dispatch<__half>(c, d, a); }
}  // namespace qxd
