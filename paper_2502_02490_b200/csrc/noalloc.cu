// noalloc.cu -- the library's one entry point that needs NO memory from anybody: |x|^2 of a flat device array of reals.
//
// Every other reduction of the library (blas.cu: grid_reduce + reduce_finalize_k) parks its per-CTA partial sums in the
// caller's workspace, which the caller had to allocate.  Callers that cannot allocate (code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc) get this variant of the norm kernel: the partial sums live in a file-scope
// __device__ array of NA_MAX_PARTIALS = 65 536 doubles (512 KB, held by every GPU that loads the library until the process
// exits).  No cudaMalloc, cudaFree or allocating library routine is called here; no context, no workspace.
//
//   stage 1   CTA k sums the squares of reals [k CHUNK, (k+1) CHUNK) in fp64 and writes partial[k]      (n / CHUNK CTAs)
//   stage 2   one CTA adds partial[0 .. nchunks) in a fixed order and writes *out
//
// The result does not depend on the grid or on timing (fixed chunking, fixed order).  Every partial that stage 2 reads has been
// written by stage 1 of the same call, so nothing in the array has to start at zero and the contents left by the previous call
// are never read.  ALL calls on a device share the one array: two calls that overlap on the GPU (different streams without an
// ordering between them) race on it.  Calls on one stream are ordered and safe.
#include <cuda_runtime.h>
#include "../../include/qxd.h"
#include <cuda_fp16.h>
#include <mutex>
#include <string>

namespace qxd {
namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_CHUNK = 4096;                          // reals per stage-1 CTA
constexpr size_t NA_MAX_PARTIALS = 65536;               // 512 KB of doubles
constexpr size_t NA_MAX_REALS = NA_MAX_PARTIALS * NA_CHUNK;   // 268 435 456 reals (a c4 full-lattice spinor has 254 803 968)
constexpr int NA_MAX_DEVICES = 64;

// In host code this name is a host-side stand-in for the symbol, NOT a device address: the address that kernels are given
// comes from cudaGetSymbolAddress (na_setup below).  Device code of this file names the array directly.
static __device__ __align__(256) double na_partials[NA_MAX_PARTIALS];

thread_local std::string na_error;
std::mutex na_mutex;
double* na_ptr[NA_MAX_DEVICES] = {};                    // device address of na_partials on every device that was set up

int na_fail(int status, const std::string& msg) { na_error = msg; return status; }

__device__ __forceinline__ double na_block_sum(double v) {
  __shared__ double warp_sum[NA_THREADS / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = v;
  __syncthreads();
  double s = 0.0;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int w = 0; w < NA_THREADS / 32; w++) s += warp_sum[w];
  }
  __syncthreads();
  return s;    // valid in thread 0
}

template <typename T>
__global__ void __launch_bounds__(NA_THREADS) na_norm2_partial_k(const T* __restrict__ x, size_t n, double* __restrict__ partial) {
  const size_t base = size_t(blockIdx.x) * NA_CHUNK;
  double acc = 0.0;
#pragma unroll 4
  for (int i = threadIdx.x; i < NA_CHUNK; i += NA_THREADS) {
    const size_t k = base + i;
    if (k < n) { const double v = (double)x[k]; acc += v * v; }
  }
  const double s = na_block_sum(acc);
  if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

__global__ void __launch_bounds__(NA_THREADS) na_norm2_final_k(const double* __restrict__ partial, int nchunks, double* __restrict__ out) {
  double acc = 0.0;
  for (int i = threadIdx.x; i < nchunks; i += NA_THREADS) acc += partial[i];
  const double s = na_block_sum(acc);
  if (threadIdx.x == 0) *out = s;
}

// Set-up of the CURRENT device: the device address of the scratch array.  Once per device; later calls return the cached pointer.
int na_setup(double** ptr) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return na_fail(QXD_ECUDA, std::string("noalloc: cudaGetDevice: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= NA_MAX_DEVICES) return na_fail(QXD_EINVAL, "noalloc: device ordinal out of range (64 devices at most)");
  std::lock_guard<std::mutex> lock(na_mutex);
  if (!na_ptr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), na_partials);
    if (e != cudaSuccess || !p) return na_fail(QXD_ECUDA, std::string("noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
    na_ptr[dev] = p;
  }
  if (ptr) *ptr = na_ptr[dev];
  return QXD_OK;
}

}  // namespace
}  // namespace qxd

using namespace qxd;

extern "C" {

int qxd_noalloc_init(void) { return na_setup(nullptr); }

size_t qxd_noalloc_max_reals(void) { return NA_MAX_REALS; }

const char* qxd_noalloc_last_error(void) { return na_error.c_str(); }

int qxd_norm2_noalloc(int prec, const void* x, size_t nreals, double* out, void* stream) {
  if (!out || (!x && nreals > 0)) return na_fail(QXD_EINVAL, "norm2_noalloc: null pointer");
  if (prec != QXD_F64 && prec != QXD_F32) return na_fail(QXD_EINVAL, "norm2_noalloc: prec must be QXD_F64 or QXD_F32 (flat arrays of reals)");
  if (nreals > NA_MAX_REALS)
    return na_fail(QXD_EINVAL, "norm2_noalloc: " + std::to_string(nreals) + " reals exceed the static scratch (maximum " + std::to_string(NA_MAX_REALS) +
                                   " = " + std::to_string(NA_MAX_PARTIALS) + " partial sums of " + std::to_string(NA_CHUNK) + " reals)");
  double* partial = nullptr;
  const int rc = na_setup(&partial);
  if (rc) return rc;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int nchunks = int((nreals + NA_CHUNK - 1) / NA_CHUNK);
  if (nchunks > 0) {
    if (prec == QXD_F64) na_norm2_partial_k<double><<<nchunks, NA_THREADS, 0, s>>>(static_cast<const double*>(x), nreals, partial);
    else na_norm2_partial_k<float><<<nchunks, NA_THREADS, 0, s>>>(static_cast<const float*>(x), nreals, partial);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(QXD_ECUDA, std::string("norm2_noalloc: stage 1 launch: ") + cudaGetErrorString(e));
  }
  na_norm2_final_k<<<1, NA_THREADS, 0, s>>>(partial, nchunks, out);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return na_fail(QXD_ECUDA, std::string("norm2_noalloc: stage 2 launch: ") + cudaGetErrorString(e));
  return QXD_OK;
}

}  // extern "C"
