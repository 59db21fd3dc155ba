// block_algebra.cuh -- the site-local algebra of the clover term shared by the dslash kernels (dslash_kernel.cuh) and the
// stand-alone clover multiply (dslash.cu): Hermitian 6x6 block times 6-vector in the packing of PAPER.md:117, and the
// (re, im) permutations that turn the stored block of a physical site into that of its C* mirror image.
#pragma once
#include "qxd_common.cuh"

namespace qxd {

namespace {

// out(12 reals: one chirality) = Hermitian 6x6 block (36 packed reals) times in
template <typename C>
__device__ __forceinline__ void block_mul(const C* b, const C* in, C* out) {
#pragma unroll
  for (int i = 0; i < 6; i++) { out[2 * i] = b[i] * in[2 * i]; out[2 * i + 1] = b[i] * in[2 * i + 1]; }
  int k = 6;
#pragma unroll
  for (int i = 0; i < 6; i++)
#pragma unroll
    for (int j = i + 1; j < 6; j++) {
      const C ur = b[k], ui = b[k + 1];
      k += 2;
      // out_i += u in_j ; out_j += conj(u) in_i   (one FMA per product)
      out[2 * i] += ur * in[2 * j]; out[2 * i] -= ui * in[2 * j + 1];
      out[2 * i + 1] += ur * in[2 * j + 1]; out[2 * i + 1] += ui * in[2 * j];
      out[2 * j] += ur * in[2 * i]; out[2 * j] += ui * in[2 * i + 1];
      out[2 * j + 1] += ur * in[2 * i + 1]; out[2 * j + 1] -= ui * in[2 * i];
    }
}
// Paired layout: the clover block of the mirror site is sigma2 M^* sigma2, so (M' v) = sigma2 conj(M conj(sigma2 v)): the
// stored block is applied to a = conj(sigma2 v) = (i conj v1, -i conj v0) and the result w is mapped to (-i conj w1, i conj w0).
// In (re, im) pairs these are swaps and sign changes only; `mir` differs between neighbouring lanes, hence selects.
template <typename C>
__device__ __forceinline__ void mirror_in(const C* v, C* a, bool mir) {
#pragma unroll
  for (int c = 0; c < 3; c++) {
    a[2 * c] = mir ? v[6 + 2 * c + 1] : v[2 * c];            a[2 * c + 1] = mir ? v[6 + 2 * c] : v[2 * c + 1];
    a[6 + 2 * c] = mir ? -v[2 * c + 1] : v[6 + 2 * c];       a[6 + 2 * c + 1] = mir ? -v[2 * c] : v[6 + 2 * c + 1];
  }
}
template <typename C>
__device__ __forceinline__ void mirror_out(const C* w, C* y, bool mir) {
#pragma unroll
  for (int c = 0; c < 3; c++) {
    y[2 * c] = mir ? -w[6 + 2 * c + 1] : w[2 * c];           y[2 * c + 1] = mir ? -w[6 + 2 * c] : w[2 * c + 1];
    y[6 + 2 * c] = mir ? w[2 * c + 1] : w[6 + 2 * c];        y[6 + 2 * c + 1] = mir ? w[2 * c] : w[6 + 2 * c + 1];
  }
}
}  // namespace

}  // namespace qxd
