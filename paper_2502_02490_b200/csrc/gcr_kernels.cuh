// gcr_kernels.cuh -- flat-vector kernels of the flexible GCR (row f3), shared by the fine-grid solver (gcr.cu) and the coarse-grid
// solver of the two-level preconditioner (dfl.cu).  A vector is a flat array of n4 float4 = 2 n4 complex numbers ((re, im) pairs
// never straddle a float4); reductions accumulate in fp64 across elements and finish in reduce_finalize_k (qxd_common.cuh).
#pragma once
#include "qxd_ctx.h"

namespace qxd {

namespace {

// layout of the device scalars of one GCR cycle (doubles)
enum { G_BR = 0 /* [32][32][2] raw <w_j, D z_k> */, G_N2 = 2048 /* [32] |w_k|^2 */, G_Q = 2080 /* [32][2] <w_k, r> */, G_Y = 2144 /* [32][2] */,
       G_RR = 2208, G_RRT = 2209, G_NE = 2210, G_NO = 2211 };


struct VecList {
  const float4* v[32];
};

// d_j = <w_j, v> for NJ vectors of the list starting at j0: result[(j0 + j) * rstride2 .. +1] = (re, im)
template <int NJ>
__global__ void __launch_bounds__(256) gcr_dots_k(size_t n4, VecList W, int j0, const float4* __restrict__ v, Reducer R) {
  double acc[2 * NJ];
#pragma unroll
  for (int i = 0; i < 2 * NJ; i++) acc[i] = 0.0;
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n4; i += size_t(gridDim.x) * blockDim.x) {
    const float4 y = __ldg(v + i);
#pragma unroll
    for (int j = 0; j < NJ; j++) {
      const float4 x = __ldg(W.v[j0 + j] + i);
      float re = x.x * y.x; re += x.y * y.y; re += x.z * y.z; re += x.w * y.w;
      float im = x.x * y.y; im -= x.y * y.x; im += x.z * y.w; im -= x.w * y.z;
      acc[2 * j] += (double)re; acc[2 * j + 1] += (double)im;
    }
  }
  grid_reduce<2 * NJ>(acc, R, blockIdx.x, gridDim.x, 0);
}

// v -= sum_{j<k} (braw_j / n2_j) w_j ;  result = (|v|^2, Re <v, r>, Im <v, r>)
__global__ void __launch_bounds__(256) gcr_orth_k(size_t n4, VecList W, int k, const double* __restrict__ braw /*[j][2], stride 64*/,
                                                  const double* __restrict__ n2, float4* __restrict__ v, const float4* __restrict__ r, Reducer R) {
  __shared__ float cr[32], ci[32];
  if (threadIdx.x < k) {
    const double d = n2[threadIdx.x];
    cr[threadIdx.x] = d > 0.0 ? (float)(braw[threadIdx.x * 64] / d) : 0.f;
    ci[threadIdx.x] = d > 0.0 ? (float)(braw[threadIdx.x * 64 + 1] / d) : 0.f;
  }
  __syncthreads();
  double acc[3] = {0.0, 0.0, 0.0};
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n4; i += size_t(gridDim.x) * blockDim.x) {
    float4 y = v[i];
    for (int j = 0; j < k; j++) {
      const float4 x = __ldg(W.v[j] + i);
      const float ar = cr[j], ai = ci[j];
      y.x -= ar * x.x - ai * x.y; y.y -= ar * x.y + ai * x.x;
      y.z -= ar * x.z - ai * x.w; y.w -= ar * x.w + ai * x.z;
    }
    v[i] = y;
    const float4 q = __ldg(r + i);
    float nn = y.x * y.x; nn += y.y * y.y; nn += y.z * y.z; nn += y.w * y.w;
    float re = y.x * q.x; re += y.y * q.y; re += y.z * q.z; re += y.w * q.w;
    float im = y.x * q.y; im -= y.y * q.x; im += y.z * q.w; im -= y.w * q.z;
    acc[0] += (double)nn; acc[1] += (double)re; acc[2] += (double)im;
  }
  grid_reduce<3>(acc, R, blockIdx.x, gridDim.x, 0);
}
// after the finalize of gcr_orth_k the three sums sit in tmp[0..2]: move them to their slots (n2[k], q[k])
__global__ void gcr_store3_k(const double* tmp, double* n2k, double* qk) { *n2k = tmp[0]; qk[0] = tmp[1]; qk[1] = tmp[2]; }

// r -= (q / n2) w ;  result = |r|^2
__global__ void __launch_bounds__(256) gcr_update_r_k(size_t n4, const float4* __restrict__ w, const double* __restrict__ q, const double* __restrict__ n2,
                                                      float4* __restrict__ r, Reducer R) {
  const double d = *n2;
  const float ar = d > 0.0 ? (float)(q[0] / d) : 0.f, ai = d > 0.0 ? (float)(q[1] / d) : 0.f;
  double acc[1] = {0.0};
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n4; i += size_t(gridDim.x) * blockDim.x) {
    const float4 x = __ldg(w + i);
    float4 y = r[i];
    y.x -= ar * x.x - ai * x.y; y.y -= ar * x.y + ai * x.x;
    y.z -= ar * x.z - ai * x.w; y.w -= ar * x.w + ai * x.z;
    r[i] = y;
    float nn = y.x * y.x; nn += y.y * y.y; nn += y.z * y.z; nn += y.w * y.w;
    acc[0] += (double)nn;
  }
  grid_reduce<1>(acc, R, blockIdx.x, gridDim.x, 0);
}

// Back substitution of  sum_k b_jk y_k = c_j  (j <= k < K) with b_jk = braw_jk / sqrt(n2_j) (j < k), b_kk = sqrt(n2_k),
// c_j = q_j / sqrt(n2_j): the coefficients of the solution update in terms of the z_k.  One thread.
__global__ void gcr_backsub_k(int K, double* s) {
  if (threadIdx.x || blockIdx.x) return;
  for (int k = K - 1; k >= 0; k--) {
    const double nk = sqrt(s[G_N2 + k]);
    if (!(nk > 0.0)) { s[G_Y + 2 * k] = 0.0; s[G_Y + 2 * k + 1] = 0.0; continue; }
    double yr = s[G_Q + 2 * k] / nk, yi = s[G_Q + 2 * k + 1] / nk;
    for (int l = k + 1; l < K; l++) {
      const double br = s[G_BR + (k * 32 + l) * 2] / nk, bi = s[G_BR + (k * 32 + l) * 2 + 1] / nk;
      const double zr = s[G_Y + 2 * l], zi = s[G_Y + 2 * l + 1];
      yr -= br * zr - bi * zi; yi -= br * zi + bi * zr;
    }
    s[G_Y + 2 * k] = yr / nk; s[G_Y + 2 * k + 1] = yi / nk;
  }
}

// x += sum_{k<K} y_k z_k on flat fp32 vectors (coarse-grid solution update)
__global__ void __launch_bounds__(256) gcr_update_x32_k(size_t n4, VecList Z, int K, const double* __restrict__ y, float4* __restrict__ x, int zero_first) {
  __shared__ float yr[32], yi[32];
  if (threadIdx.x < K) { yr[threadIdx.x] = (float)y[2 * threadIdx.x]; yi[threadIdx.x] = (float)y[2 * threadIdx.x + 1]; }
  __syncthreads();
  for (size_t i = size_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n4; i += size_t(gridDim.x) * blockDim.x) {
    float4 a = zero_first ? make_float4(0.f, 0.f, 0.f, 0.f) : x[i];
    for (int k = 0; k < K; k++) {
      const float4 z = __ldg(Z.v[k] + i);
      a.x += yr[k] * z.x - yi[k] * z.y; a.y += yr[k] * z.y + yi[k] * z.x;
      a.z += yr[k] * z.z - yi[k] * z.w; a.w += yr[k] * z.w + yi[k] * z.z;
    }
    x[i] = a;
  }
}

}  // namespace

}  // namespace qxd
