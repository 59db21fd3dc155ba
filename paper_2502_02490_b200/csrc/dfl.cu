// dfl.cu -- SURVEY.md §8(f) row f3, second level: the Schwarz-preconditioned GCR of sap.cu / gcr.cu with a coarse-grid
// (deflation) correction, the ingredient that makes the paper's solvers "heavily preconditioned" (deflated SAP-GCR
// on the CPU, multigrid GCR on the GPU).  Local-coherence deflation in the style of the host code's solver family:
//
//   setup   ns test vectors (random, passed in by the caller) are smoothed by ninv applications of M_sap, which damps the high
//           modes of D_w and leaves an approximate low-mode space; the vectors are restricted to the SAP blocks (256 sites) and
//           orthonormalised block by block: the deflation space is span{ P_b phi_i } (dimension ns per block);
//           with the chirality split (qxd_set_deflation_chirality) every phi_i gives two basis vectors per block, its upper and
//           lower spin components: dimension nc = 2 ns per block, coarse index 2 i + chi;
//           the coarse ("little") operator A_c = R D_w P is a nine-point stencil of nc x nc complex matrices (sap.cu).
//   apply   z = P A_c^{-1} R r  +  M_sap (r - D_w P A_c^{-1} R r):  coarse-grid correction, then Schwarz smoothing of what is left;
//           A_c^{-1} is nkc steps of GCR on the even-odd (Schur) form of the coarse system, matrices in binary16, all coefficients
//           on the device, no host round trip.
//
// R = P^dagger (block-wise inner products with the phi_i), P = block-wise linear combination.  Everything is fp32 (the block
// operator of M_sap and of the coarse-operator build in the storage precision of the solve).  The outer solver is the flexible
// GCR of gcr.cu: the preconditioner may be as inexact as it likes, convergence is declared on the fp64 residual only.
#include "gcr_kernels.cuh"
#include <cmath>
#include <vector>

namespace qxd {

namespace {

#define QXD_TRY(expr)        \
  do {                       \
    int rc__ = (expr);       \
    if (rc__) return rc__;   \
  } while (0)

struct PhiList {
  const float4* v[32];
};
// float4 index of chunk c of the thread's site (block b = blockIdx.x, 256 threads = 128 checkerboard indices x 2 parities)
__device__ __forceinline__ size_t own_index(int Vh) { return size_t(threadIdx.x >> 7) * 6 * Vh + size_t(blockIdx.x) * 128 + (threadIdx.x & 127); }

// out[b * ldo + j0 + j] = sum_{x in b} conj(u_{j0+j}(x)) . v(x),  j < NJ   (restriction, Gram-Schmidt coefficients, block norms).
// ch = 1 (chirality split): the sums over the upper (reals 0..11) and the lower (12..23) spin components are kept apart,
// out[b * ldo + 2 (j0 + j) + chi].
template <int NJ>
__global__ void __launch_bounds__(256) dfl_block_dots_k(int Vh, PhiList U, int j0, const float4* __restrict__ v, float2* __restrict__ out, int ldo, int ch) {
  __shared__ float red[8][4 * NJ];
  const size_t own = own_index(Vh);
  float y[24], part[4 * NJ];
#pragma unroll
  for (int c = 0; c < 6; c++) { const float4 t = __ldg(v + own + size_t(c) * Vh); y[4 * c] = t.x; y[4 * c + 1] = t.y; y[4 * c + 2] = t.z; y[4 * c + 3] = t.w; }
#pragma unroll
  for (int j = 0; j < NJ; j++) {
    float re[2] = {0.f, 0.f}, im[2] = {0.f, 0.f};
#pragma unroll
    for (int c = 0; c < 6; c++) {
      const float4 u = __ldg(U.v[j0 + j] + own + size_t(c) * Vh);
      const int h = c / 3;
      re[h] += u.x * y[4 * c]; re[h] += u.y * y[4 * c + 1]; re[h] += u.z * y[4 * c + 2]; re[h] += u.w * y[4 * c + 3];
      im[h] += u.x * y[4 * c + 1]; im[h] -= u.y * y[4 * c]; im[h] += u.z * y[4 * c + 3]; im[h] -= u.w * y[4 * c + 2];
    }
    part[4 * j] = re[0]; part[4 * j + 1] = im[0]; part[4 * j + 2] = re[1]; part[4 * j + 3] = im[1];
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
  for (int k = 0; k < 4 * NJ; k++) {
    float t = part[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    if (lane == 0) red[warp][k] = t;
  }
  __syncthreads();
  if (ch) {
    if (threadIdx.x < 4 * NJ) {
      float t = 0.f;
#pragma unroll
      for (int w = 0; w < 8; w++) t += red[w][threadIdx.x];
      reinterpret_cast<float*>(out + size_t(blockIdx.x) * ldo + 2 * j0)[threadIdx.x] = t;
    }
  } else if (threadIdx.x < 2 * NJ) {
    const int k = 4 * (threadIdx.x >> 1) + (threadIdx.x & 1);
    float t = 0.f;
#pragma unroll
    for (int w = 0; w < 8; w++) t += red[w][k] + red[w][k + 2];
    reinterpret_cast<float*>(out + size_t(blockIdx.x) * ldo + j0)[threadIdx.x] = t;
  }
}
// v(x) = beta v(x) + sign sum_{j<n} c[b * ldc + j] u_j(x)      (Gram-Schmidt update: beta 1, sign -1; prolongation: beta 0, sign +1)
// ch = 1: the upper spin components take c[b * ldc + 2 j], the lower ones c[b * ldc + 2 j + 1]  (n <= 16)
__global__ void __launch_bounds__(256) dfl_block_axpy_k(int Vh, PhiList U, int n, const float2* __restrict__ coef, int ldc, float beta, float sign,
                                                        float4* __restrict__ v, int ch) {
  __shared__ float2 cs[32];
  if (threadIdx.x < (ch ? 2 * n : n)) { const float2 t = coef[size_t(blockIdx.x) * ldc + threadIdx.x]; cs[threadIdx.x] = make_float2(sign * t.x, sign * t.y); }
  __syncthreads();
  const size_t own = own_index(Vh);
  float4 y[6];
#pragma unroll
  for (int c = 0; c < 6; c++) {
    y[c] = beta != 0.f ? v[own + size_t(c) * Vh] : make_float4(0.f, 0.f, 0.f, 0.f);
    if (beta != 0.f && beta != 1.f) { y[c].x *= beta; y[c].y *= beta; y[c].z *= beta; y[c].w *= beta; }
  }
  for (int j = 0; j < n; j++) {
    const float2 cu = ch ? cs[2 * j] : cs[j], cl = ch ? cs[2 * j + 1] : cs[j];
#pragma unroll
    for (int c = 0; c < 6; c++) {
      const float ar = c < 3 ? cu.x : cl.x, ai = c < 3 ? cu.y : cl.y;
      const float4 u = __ldg(U.v[j] + own + size_t(c) * Vh);
      y[c].x += ar * u.x - ai * u.y; y[c].y += ar * u.y + ai * u.x;
      y[c].z += ar * u.z - ai * u.w; y[c].w += ar * u.w + ai * u.z;
    }
  }
#pragma unroll
  for (int c = 0; c < 6; c++) v[own + size_t(c) * Vh] = y[c];
}
// v(x) /= sqrt(n2[b].x)  (block-wise normalisation; a vanishing block is left as it is); ch = 1: n2[b] and n2[b + 1] for the two chiralities
__global__ void __launch_bounds__(256) dfl_block_scale_k(int Vh, const float2* __restrict__ n2, int ld, float4* __restrict__ v, int ch) {
  const float du = n2[size_t(blockIdx.x) * ld].x, dl = ch ? n2[size_t(blockIdx.x) * ld + 1].x : du;
  const float su = du > 0.f ? rsqrtf(du) : 1.f, sl = dl > 0.f ? rsqrtf(dl) : 1.f;
  const size_t own = own_index(Vh);
#pragma unroll
  for (int c = 0; c < 6; c++) { const float sc = c < 3 ? su : sl; float4 t = v[own + size_t(c) * Vh]; t.x *= sc; t.y *= sc; t.z *= sc; t.w *= sc; v[own + size_t(c) * Vh] = t; }
}
// flat helpers on packed full-lattice fp32 vectors
__global__ void __launch_bounds__(256) dfl_scale_flat_k(size_t n4, const double* __restrict__ n2, float4* __restrict__ v) {
  const float s = *n2 > 0.0 ? (float)(1.0 / sqrt(*n2)) : 1.f;
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n4; i += size_t(gridDim.x) * blockDim.x) {
    float4 t = v[i]; t.x *= s; t.y *= s; t.z *= s; t.w *= s; v[i] = t;
  }
}
// z = a - b   /   z = a + b
__global__ void __launch_bounds__(256) dfl_addsub_flat_k(size_t n4, const float4* __restrict__ a, const float4* __restrict__ b, float sign, float4* __restrict__ z) {
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n4; i += size_t(gridDim.x) * blockDim.x) {
    const float4 x = a[i], y = b[i];
    z[i] = make_float4(x.x + sign * y.x, x.y + sign * y.y, x.z + sign * y.z, x.w + sign * y.w);
  }
}
// coarse operator: y[b][j] = sum_i A[b][0][j][i] x[b][i] + sum_{d<8} sum_i A[b][1+d][j][i] x[nbr[b][d]][i]; thread per (b, j)
__global__ void __launch_bounds__(256) dfl_coarse_apply_k(int nblocks, int ns, const float2* __restrict__ A, const int* __restrict__ nbr,
                                                          const float2* __restrict__ x, float2* __restrict__ y) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int b = t / ns, j = t - b * ns;
  if (b >= nblocks) return;
  float re = 0.f, im = 0.f;
  for (int d = 0; d < 9; d++) {
    const int nb = d == 0 ? b : nbr[b * 8 + d - 1];
    if (nb < 0) continue;
    const float2* row = A + ((size_t(b) * 9 + d) * ns + j) * ns;
    const float2* xv = x + size_t(nb) * ns;
    for (int i = 0; i < ns; i++) {
      const float2 a = __ldg(row + i), v = __ldg(xv + i);
      re += a.x * v.x - a.y * v.y; im += a.x * v.y + a.y * v.x;
    }
  }
  y[t] = make_float2(re, im);
}

// Dinv[b] = A[b][0]^{-1} (ns x ns complex, Gauss-Jordan with partial pivoting, one thread per block; setup only)
__global__ void __launch_bounds__(64) dfl_diag_inverse_k(int nblocks, int ns, const float2* __restrict__ A, float2* __restrict__ Dinv) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= nblocks) return;
  float2 m[32 * 32];
  float2* inv = Dinv + size_t(b) * ns * ns;
  const float2* src = A + size_t(b) * 9 * ns * ns;
  for (int i = 0; i < ns * ns; i++) { m[i] = src[i]; inv[i] = make_float2((i / ns) == (i % ns) ? 1.f : 0.f, 0.f); }
  for (int col = 0; col < ns; col++) {
    int piv = col; float best = m[col * ns + col].x * m[col * ns + col].x + m[col * ns + col].y * m[col * ns + col].y;
    for (int r = col + 1; r < ns; r++) { const float v = m[r * ns + col].x * m[r * ns + col].x + m[r * ns + col].y * m[r * ns + col].y; if (v > best) { best = v; piv = r; } }
    if (!(best > 0.f)) continue;
    if (piv != col) for (int j = 0; j < ns; j++) { float2 t = m[piv * ns + j]; m[piv * ns + j] = m[col * ns + j]; m[col * ns + j] = t; t = inv[piv * ns + j]; inv[piv * ns + j] = inv[col * ns + j]; inv[col * ns + j] = t; }
    const float2 p = m[col * ns + col];
    const float dr = p.x / best, di = -p.y / best;
    for (int j = 0; j < ns; j++) {
      float2 t = m[col * ns + j]; m[col * ns + j] = make_float2(t.x * dr - t.y * di, t.x * di + t.y * dr);
      t = inv[col * ns + j]; inv[col * ns + j] = make_float2(t.x * dr - t.y * di, t.x * di + t.y * dr);
    }
    for (int r = 0; r < ns; r++) {
      if (r == col) continue;
      const float2 f = m[r * ns + col];
      for (int j = 0; j < ns; j++) {
        const float2 a = m[col * ns + j], c2 = inv[col * ns + j];
        m[r * ns + j].x -= f.x * a.x - f.y * a.y; m[r * ns + j].y -= f.x * a.y + f.y * a.x;
        inv[r * ns + j].x -= f.x * c2.x - f.y * c2.y; inv[r * ns + j].y -= f.x * c2.y + f.y * c2.x;
      }
    }
  }
}
// y[b] = Dinv[b] x[b]  (block-Jacobi preconditioner of the coarse GCR); thread per (b, j)
__global__ void __launch_bounds__(256) dfl_diag_apply_k(int nblocks, int ns, const float2* __restrict__ Dinv, const float2* __restrict__ x, float2* __restrict__ y) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int b = t / ns, j = t - b * ns;
  if (b >= nblocks) return;
  const float2* row = Dinv + (size_t(b) * ns + j) * ns;
  const float2* xv = x + size_t(b) * ns;
  float re = 0.f, im = 0.f;
  for (int i = 0; i < ns; i++) { const float2 a = __ldg(row + i), v = __ldg(xv + i); re += a.x * v.x - a.y * v.y; im += a.x * v.y + a.y * v.x; }
  y[t] = make_float2(re, im);
}
// ---- even-odd (Schur) form of the coarse system ------------------------------------------------------------------------
// The blocks are two-coloured and every hop of the nine-point operator joins blocks of opposite colours, so with A_c = D + H
// (D the diagonal blocks) the coarse system splits as on the fine grid:
//     (1 - Dinv_e H_eo Dinv_o H_oe) x_e = Dinv_e (b_e - H_eo Dinv_o b_o),      x_o = Dinv_o (b_o - H_oe x_e).
// k GCR steps on the left-hand operator span the same space as 2k steps on the block-Jacobi preconditioned full operator, at
// half the matrix traffic each; the matrices are read from a transposed binary16 copy (thread j of a block reads column j:
// 4 ns contiguous bytes per row for the block's ns threads).
__global__ void __launch_bounds__(256) dfl_pack16_k(int nblocks, int ns, const float2* __restrict__ A, const float2* __restrict__ Dinv, __half2* __restrict__ Ah) {
  const size_t n = size_t(nblocks) * 9 * ns * ns;
  for (size_t t = size_t(blockIdx.x) * blockDim.x + threadIdx.x; t < n; t += size_t(gridDim.x) * blockDim.x) {
    const int j = int(t % ns), i = int((t / ns) % ns), slot = int((t / (size_t(ns) * ns)) % 9);
    const size_t b = t / (size_t(9) * ns * ns);
    const float2 v = slot < 8 ? A[((b * 9 + 1 + slot) * ns + j) * ns + i] : Dinv[(b * ns + j) * ns + i];
    Ah[t] = __floats2half2_rn(v.x, v.y);
  }
}
// y[b] = (u ? u[b] : 0) + sign * Dinv[b] sum_d A[b][1+d] x[nbr[b][d]] on the blocks of `colour`, 0 on the others.
// One CTA per pair of blocks (2k, 2k+1) -- they have opposite colours (sap_check_geometry) -- of 8 ns threads: thread (d, j)
// forms row j of hop d of the active block (ns loads of 4 bytes, contiguous over j), the eight partial sums meet in shared
// memory, the first ns threads multiply by Dinv and write both blocks (zeros for the other colour).
__global__ void __launch_bounds__(256) dfl_eo_hop_k(int ns, int colour, float sign, const __half2* __restrict__ Ah, const int* __restrict__ nbr,
                                                    const int* __restrict__ col, const float2* __restrict__ x, const float2* __restrict__ u, float2* __restrict__ y) {
  __shared__ float2 part[8 * 32];
  __shared__ float2 t[32];
  const int d = threadIdx.x / ns, j = threadIdx.x - d * ns;
  const int b = 2 * blockIdx.x + (col[2 * blockIdx.x] != colour ? 1 : 0);
  float re = 0.f, im = 0.f;
  const int nb = nbr[b * 8 + d];
  if (nb >= 0) {
    const __half2* At = Ah + ((size_t(b) * 9 + d) * ns) * ns + j;
    const float2* xv = x + size_t(nb) * ns;
#pragma unroll 8
    for (int i = 0; i < ns; i++) {
      const float2 a = __half22float2(At[size_t(i) * ns]), v = __ldg(xv + i);
      re += a.x * v.x - a.y * v.y; im += a.x * v.y + a.y * v.x;
    }
  }
  part[d * 32 + j] = make_float2(re, im);
  __syncthreads();
  if (threadIdx.x < ns) {
    float2 a = part[j];
#pragma unroll
    for (int k = 1; k < 8; k++) { a.x += part[k * 32 + j].x; a.y += part[k * 32 + j].y; }
    t[j] = a;
  }
  __syncthreads();
  if (threadIdx.x < ns) {
    const __half2* Dt = Ah + ((size_t(b) * 9 + 8) * ns) * ns + j;
    re = 0.f; im = 0.f;
#pragma unroll 8
    for (int i = 0; i < ns; i++) {
      const float2 a = __half22float2(Dt[size_t(i) * ns]), v = t[i];
      re += a.x * v.x - a.y * v.y; im += a.x * v.y + a.y * v.x;
    }
    float2 o = u ? u[size_t(b) * ns + j] : make_float2(0.f, 0.f);
    o.x += sign * re; o.y += sign * im;
    y[size_t(b) * ns + j] = o;
    y[size_t(b ^ 1) * ns + j] = make_float2(0.f, 0.f);
  }
}
struct Dfl {
  qxd_ctx* c;
  int Vh, nb, ns, nc, ch;   // ns null vectors; nc = coarse degrees of freedom per block (2 ns with the chirality split)
  size_t n4, nc4;     // float4 per fine / coarse vector
  int nblk, nblkc;
  PhiList phi() const { PhiList P; for (int i = 0; i < 32; i++) P.v[i] = static_cast<const float4*>(c->dphi[i]); return P; }
  Reducer red(double* result) const { Reducer R; R.partials = c->partials; R.result = result; R.rstride = 0; return R; }
};
Dfl make_dfl(qxd_ctx* c) {
  Dfl D;
  D.c = c; D.Vh = c->g.Vh; D.nb = c->g.Vh / 128; D.ns = c->dfl_ns; D.ch = c->dfl_chiral ? 1 : 0; D.nc = D.ns * (1 + D.ch);
  D.n4 = size_t(12) * D.Vh; D.nc4 = size_t(D.nb) * D.nc / 2;
  D.nblk = D.Vh / 128 < 1 ? 1 : (D.Vh / 128 > 148 * 8 ? 148 * 8 : D.Vh / 128);
  D.nblkc = int((D.nc4 + 255) / 256); if (D.nblkc > D.nblk) D.nblkc = D.nblk; if (D.nblkc < 1) D.nblkc = 1;
  return D;
}
// out[b][0..ns) = R v  (block inner products with all null vectors)
int restrict_to_coarse(const Dfl& D, const float4* v, float2* out) {
  for (int j0 = 0; j0 < D.ns; j0 += 4) {
    const int nj = D.ns - j0 < 4 ? D.ns - j0 : 4;
    if (nj == 4) dfl_block_dots_k<4><<<D.nb, 256, 0, D.c->stream>>>(D.Vh, D.phi(), j0, v, out, D.nc, D.ch);
    else if (nj == 3) dfl_block_dots_k<3><<<D.nb, 256, 0, D.c->stream>>>(D.Vh, D.phi(), j0, v, out, D.nc, D.ch);
    else if (nj == 2) dfl_block_dots_k<2><<<D.nb, 256, 0, D.c->stream>>>(D.Vh, D.phi(), j0, v, out, D.nc, D.ch);
    else dfl_block_dots_k<1><<<D.nb, 256, 0, D.c->stream>>>(D.Vh, D.phi(), j0, v, out, D.nc, D.ch);
    QXD_LAUNCH_CHECK(D.c);
  }
  return QXD_OK;
}

int eo_hop(const Dfl& D, int colour, float sign, const float2* x, const float2* u, float2* y) {
  dfl_eo_hop_k<<<D.nb / 2, 8 * D.nc, 0, D.c->stream>>>(D.nc, colour, sign, static_cast<const __half2*>(D.c->dAh), D.c->dnbr, D.c->dcol, x, u, y);
  QXD_LAUNCH_CHECK(D.c);
  return QXD_OK;
}
// x = (approximately) A_c^{-1} b: nkc GCR steps on the even-odd (Schur) form of the coarse system (z_k = current residual),
// every coefficient on the device, one back substitution at the end; no host synchronisation.
int coarse_solve(const Dfl& D, const float2* b, float2* x) {
  qxd_ctx* c = D.c;
  double* S = c->dscal;
  double* tmp = S + 3000;
  const int K = c->dfl_nkc;
  VecList Z, W;
  for (int k = 0; k < 32; k++) { Z.v[k] = static_cast<const float4*>(c->dcz[k]); W.v[k] = static_cast<const float4*>(c->dcw[k]); }
  float4* r = static_cast<float4*>(c->dcr);
  float2* s = static_cast<float2*>(c->dcs);
  float2* t = static_cast<float2*>(c->dct);
  dfl_diag_apply_k<<<(D.nb * D.nc + 255) / 256, 256, 0, c->stream>>>(D.nb, D.nc, static_cast<const float2*>(c->dDinv), b, s);   // s = Dinv b
  QXD_LAUNCH_CHECK(c);
  QXD_TRY(eo_hop(D, 0, -1.f, s, s, reinterpret_cast<float2*>(r)));                                   // r = s_e - Dinv_e H_eo s_o
  for (int k = 0; k < K; k++) {
    QXD_CUDA_OK(c, cudaMemcpyAsync(c->dcz[k], r, D.nc4 * sizeof(float4), cudaMemcpyDeviceToDevice, c->stream));   // z_k = r
    QXD_TRY(eo_hop(D, 1, +1.f, static_cast<const float2*>(c->dcz[k]), nullptr, t));                                 // t_o = Dinv_o H_oe z_k
    QXD_TRY(eo_hop(D, 0, -1.f, t, static_cast<const float2*>(c->dcz[k]), static_cast<float2*>(c->dcw[k])));         // w_k = z_k - Dinv_e H_eo t_o
    float4* wk = static_cast<float4*>(c->dcw[k]);
    for (int j0 = 0; j0 < k; j0 += 4) {
      const int nj = k - j0 < 4 ? k - j0 : 4;
      Reducer R = D.red(S + G_BR + (j0 * 32 + k) * 2);
      R.rstride = 64;
      if (nj == 4) gcr_dots_k<4><<<D.nblkc, 256, 0, c->stream>>>(D.nc4, W, j0, wk, R);
      else if (nj == 3) gcr_dots_k<3><<<D.nblkc, 256, 0, c->stream>>>(D.nc4, W, j0, wk, R);
      else if (nj == 2) gcr_dots_k<2><<<D.nblkc, 256, 0, c->stream>>>(D.nc4, W, j0, wk, R);
      else gcr_dots_k<1><<<D.nblkc, 256, 0, c->stream>>>(D.nc4, W, j0, wk, R);
      QXD_LAUNCH_CHECK(c);
      reduce_finalize_k<2><<<dim3(1, nj), FINALIZE_THREADS, 0, c->stream>>>(R, D.nblkc);
      QXD_LAUNCH_CHECK(c);
    }
    gcr_orth_k<<<D.nblkc, 256, 0, c->stream>>>(D.nc4, W, k, S + G_BR + k * 2, S + G_N2, wk, r, D.red(tmp));
    QXD_LAUNCH_CHECK(c);
    reduce_finalize_k<3><<<dim3(1, 1), FINALIZE_THREADS, 0, c->stream>>>(D.red(tmp), D.nblkc);
    QXD_LAUNCH_CHECK(c);
    gcr_store3_k<<<1, 1, 0, c->stream>>>(tmp, S + G_N2 + k, S + G_Q + 2 * k);
    QXD_LAUNCH_CHECK(c);
    gcr_update_r_k<<<D.nblkc, 256, 0, c->stream>>>(D.nc4, wk, S + G_Q + 2 * k, S + G_N2 + k, r, D.red(S + G_RR));
    QXD_LAUNCH_CHECK(c);
    reduce_finalize_k<1><<<dim3(1, 1), FINALIZE_THREADS, 0, c->stream>>>(D.red(S + G_RR), D.nblkc);
    QXD_LAUNCH_CHECK(c);
  }
  gcr_backsub_k<<<1, 32, 0, c->stream>>>(K, S);
  QXD_LAUNCH_CHECK(c);
  gcr_update_x32_k<<<D.nblkc, 256, 0, c->stream>>>(D.nc4, Z, K, S + G_Y, reinterpret_cast<float4*>(x), 1);          // x_e
  QXD_LAUNCH_CHECK(c);
  QXD_TRY(eo_hop(D, 1, -1.f, x, s, t));                                                                // t_o = s_o - Dinv_o H_oe x_e
  dfl_addsub_flat_k<<<D.nblkc, 256, 0, c->stream>>>(D.nc4, reinterpret_cast<const float4*>(x), reinterpret_cast<const float4*>(t), 1.f, reinterpret_cast<float4*>(x));
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

int apply_Dw32(qxd_ctx* c, void* in, void* out) {
  const int Vh = c->g.Vh;
  DslashCall d{};
  d.prec = 1; d.mode = DS_DW_FULL; d.flags = 0;
  d.in[0] = half_view(1, in, Vh, 0); d.in[1] = half_view(1, in, Vh, 1);
  d.out[0] = half_view(1, out, Vh, 0); d.out[1] = half_view(1, out, Vh, 1);
  return launch_dslash(c, d);
}

}  // namespace

// z = P A_c^{-1} R r + M_sap (r - D_w P A_c^{-1} R r);  r, z: fp32 packed full-lattice vectors; scratch: the context's d_t1, d_t2
int launch_dfl_precond(qxd_ctx* c, int prec, const void* r, void* z) {
  if (!c->dfl_ready) return fail(c, QXD_ESTATE, "deflated preconditioner: call qxd_deflation_setup first");
  const Dfl D = make_dfl(c);
  float2* cr = static_cast<float2*>(c->dcb);
  float2* cx = static_cast<float2*>(c->dcx);
  float4* z0 = static_cast<float4*>(z);
  float4* t1 = static_cast<float4*>(c->d_t1);
  float4* t2 = static_cast<float4*>(c->d_t2);
  QXD_TRY(restrict_to_coarse(D, static_cast<const float4*>(r), cr));
  QXD_TRY(coarse_solve(D, cr, cx));
  dfl_block_axpy_k<<<D.nb, 256, 0, c->stream>>>(D.Vh, D.phi(), D.ns, cx, D.nc, 0.f, 1.f, z0, D.ch);            // z0 = P cx
  QXD_LAUNCH_CHECK(c);
  QXD_TRY(apply_Dw32(c, z0, t1));                                                                            // t1 = D_w z0
  dfl_addsub_flat_k<<<D.nblk, 256, 0, c->stream>>>(D.n4, static_cast<const float4*>(r), t1, -1.f, t1);      // t1 = r - D_w z0
  QXD_LAUNCH_CHECK(c);
  QXD_TRY(launch_sap(c, prec, t1, t2));                                                                      // t2 = M_sap t1
  dfl_addsub_flat_k<<<D.nblk, 256, 0, c->stream>>>(D.n4, z0, t2, 1.f, z0);                                   // z = z0 + t2
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

namespace {
// v <- v / |v| (global norm) on a packed full-lattice fp32 vector
int normalise_flat(const Dfl& D, float4* v) {
  qxd_ctx* c = D.c;
  double* S = c->dscal;
  VecList L; for (int k = 0; k < 32; k++) L.v[k] = v;
  gcr_dots_k<1><<<D.nblk, 256, 0, c->stream>>>(D.n4, L, 0, v, D.red(S + 3900));
  QXD_LAUNCH_CHECK(c);
  reduce_finalize_k<2><<<dim3(1, 1), FINALIZE_THREADS, 0, c->stream>>>(D.red(S + 3900), D.nblk);
  QXD_LAUNCH_CHECK(c);
  dfl_scale_flat_k<<<D.nblk, 256, 0, c->stream>>>(D.n4, S + 3900, v);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
// block-wise Gram-Schmidt (twice) of the null vectors, then the coarse operator and the inverses of its diagonal blocks
int orthonormalise_and_build(const Dfl& D, int prec) {
  qxd_ctx* c = D.c;
  float2* coef = static_cast<float2*>(c->dcb);      // [nb][ns] scratch
  for (int i = 0; i < D.ns; i++) {
    float4* v = static_cast<float4*>(c->dphi[i]);
    for (int pass = 0; pass < 2 && i > 0; pass++) {
      for (int j0 = 0; j0 < i; j0 += 4) {
        const int nj = i - j0 < 4 ? i - j0 : 4;
        if (nj == 4) dfl_block_dots_k<4><<<D.nb, 256, 0, c->stream>>>(D.Vh, D.phi(), j0, v, coef, D.nc, D.ch);
        else if (nj == 3) dfl_block_dots_k<3><<<D.nb, 256, 0, c->stream>>>(D.Vh, D.phi(), j0, v, coef, D.nc, D.ch);
        else if (nj == 2) dfl_block_dots_k<2><<<D.nb, 256, 0, c->stream>>>(D.Vh, D.phi(), j0, v, coef, D.nc, D.ch);
        else dfl_block_dots_k<1><<<D.nb, 256, 0, c->stream>>>(D.Vh, D.phi(), j0, v, coef, D.nc, D.ch);
        QXD_LAUNCH_CHECK(c);
      }
      dfl_block_axpy_k<<<D.nb, 256, 0, c->stream>>>(D.Vh, D.phi(), i, coef, D.nc, 1.f, -1.f, v, D.ch);
      QXD_LAUNCH_CHECK(c);
    }
    PhiList self; for (int k = 0; k < 32; k++) self.v[k] = v;
    dfl_block_dots_k<1><<<D.nb, 256, 0, c->stream>>>(D.Vh, self, 0, v, coef, D.nc, D.ch);
    QXD_LAUNCH_CHECK(c);
    dfl_block_scale_k<<<D.nb, 256, 0, c->stream>>>(D.Vh, coef, D.nc, v, D.ch);     // coef[b * nc (+ 1)].x = |v|_b^2 (per chirality)
    QXD_LAUNCH_CHECK(c);
  }
  QXD_TRY(launch_coarse_build(c, prec, D.ns, c->dphi, c->dAc, c->dnbr));
  dfl_diag_inverse_k<<<(D.nb + 63) / 64, 64, 0, c->stream>>>(D.nb, D.nc, static_cast<const float2*>(c->dAc), static_cast<float2*>(c->dDinv));
  QXD_LAUNCH_CHECK(c);
  dfl_pack16_k<<<148 * 8, 256, 0, c->stream>>>(D.nb, D.nc, static_cast<const float2*>(c->dAc), static_cast<const float2*>(c->dDinv), static_cast<__half2*>(c->dAh));
  QXD_LAUNCH_CHECK(c);
  std::vector<int> col(D.nb);
  for (int b = 0; b < D.nb; b++) {
    int blk;
    QXD_TRY(qxd_sap_block_of(c, b * 128, 0, &blk, &col[b]));
  }
  QXD_CUDA_OK(c, cudaMemcpyAsync(c->dcol, col.data(), sizeof(int) * D.nb, cudaMemcpyHostToDevice, c->stream));
  QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));   // col leaves scope
  return QXD_OK;
}
}  // namespace

// Setup: smooth the caller's ns random vectors with ninv applications of M_sap (normalising in between), orthonormalise them
// block by block (Gram-Schmidt, twice), build the coarse operator.  Then nref rounds of adaptive refinement: every null vector
// is replaced by the two-level preconditioner applied to it (which amplifies exactly what the current method still converges
// slowly on), and the space and the coarse operator are rebuilt.
int dfl_setup(qxd_ctx* c, int prec, const void* random_vectors) {
  const Dfl D = make_dfl(c);
  const size_t vb = 2 * half_bytes(1, D.Vh);
  float4* t2 = static_cast<float4*>(c->d_t2);
  c->dfl_ready = false;
  for (int i = 0; i < D.ns; i++) {
    float4* v = static_cast<float4*>(c->dphi[i]);
    QXD_CUDA_OK(c, cudaMemcpyAsync(v, static_cast<const char*>(random_vectors) + vb * i, vb, cudaMemcpyDeviceToDevice, c->stream));
    for (int it = 0; it < c->dfl_ninv; it++) {
      QXD_TRY(launch_sap(c, prec, v, t2));
      QXD_TRY(normalise_flat(D, t2));
      QXD_CUDA_OK(c, cudaMemcpyAsync(v, t2, vb, cudaMemcpyDeviceToDevice, c->stream));
    }
  }
  QXD_TRY(orthonormalise_and_build(D, prec));
  c->dfl_ready = true; c->dfl_prec = prec;
  for (int round = 0; round < c->dfl_nref; round++) {
    // new vectors from the CURRENT two-level method, parked in the Krylov space of the fine-grid GCR until all are done
    // refk = 1: phi_i <- M_2level phi_i; refk > 1: inverse iteration, phi_i <- refk steps of the deflated GCR on D_w x = phi_i
    // (Krylov vectors [0, refk) of the fine-grid solver; the new vectors wait in the upper part of the Krylov space)
    const int refk = c->dfl_refk > 1 ? c->dfl_refk : 0, park = c->gcr_nkv - refk;
    if (D.ns > 2 * park) return fail(c, QXD_EWORKSPACE, "deflation refinement needs ns <= 2 (nkv - steps) scratch vectors (qxd_set_gcr)");
    for (int i = 0; i < D.ns; i++) {
      void* dst = i < park ? c->gz[refk + i] : c->gw[refk + i - park];
      if (refk) {
        QXD_CUDA_OK(c, cudaMemcpyAsync(c->g_r, c->dphi[i], vb, cudaMemcpyDeviceToDevice, c->stream));
        QXD_TRY(gcr_cycle32(c, prec, true, refk, dst));
      } else QXD_TRY(launch_dfl_precond(c, prec, c->dphi[i], dst));
      QXD_TRY(normalise_flat(D, static_cast<float4*>(dst)));
    }
    for (int i = 0; i < D.ns; i++) {
      void* src = i < park ? c->gz[refk + i] : c->gw[refk + i - park];
      QXD_CUDA_OK(c, cudaMemcpyAsync(c->dphi[i], src, vb, cudaMemcpyDeviceToDevice, c->stream));
    }
    c->dfl_ready = false;
    QXD_TRY(orthonormalise_and_build(D, prec));
    c->dfl_ready = true;
  }
  return QXD_OK;
}

// test / bench entry points on the coarse level: y = R x (x fine), x = P y, y = A_c x
int dfl_restrict(qxd_ctx* c, const void* fine, void* coarse) { const Dfl D = make_dfl(c); return restrict_to_coarse(D, static_cast<const float4*>(fine), static_cast<float2*>(coarse)); }
int dfl_prolong(qxd_ctx* c, const void* coarse, void* fine) {
  const Dfl D = make_dfl(c);
  dfl_block_axpy_k<<<D.nb, 256, 0, c->stream>>>(D.Vh, D.phi(), D.ns, static_cast<const float2*>(coarse), D.nc, 0.f, 1.f, static_cast<float4*>(fine), D.ch);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int dfl_coarse_solve(qxd_ctx* c, const void* b, void* x) { const Dfl D = make_dfl(c); return coarse_solve(D, static_cast<const float2*>(b), static_cast<float2*>(x)); }
int dfl_coarse_apply(qxd_ctx* c, const void* x, void* y) {
  const Dfl D = make_dfl(c);
  dfl_coarse_apply_k<<<(D.nb * D.nc + 255) / 256, 256, 0, c->stream>>>(D.nb, D.nc, static_cast<const float2*>(c->dAc), c->dnbr, static_cast<const float2*>(x),
                                                                      static_cast<float2*>(y));
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // namespace qxd
