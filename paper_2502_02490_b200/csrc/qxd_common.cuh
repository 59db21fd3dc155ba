// qxd_common.cuh -- geometry, precision traits and 16-byte-chunk SoA record access.
//
// Site order on the device: the paper's host code orders sites in cache
// blocks, lexicographic inside a block, even sites first (Eq. (2)); we keep that idea
// with power-of-two tiles sized for the B200 L1/L2 and compute every index on the fly as a pure
// inlined function, as PAPER.md:105 advises (no lookup tables).
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>

namespace qxd {

struct Geom {
  // C*-paired layout (pair = 1): the index machinery below runs on the PHYSICAL lattice
  // (X[1] = L1) and an extended site is (physical site, mirror bit m): spinor index cb = 2 * cb_phys + m, so a site and
  // its mirror image x + L1 e1 are neighbours in memory and in the warp.  Links and clover blocks exist once per
  // physical site (record stride Vg = Vh / 2); the mirror site uses U^*, -A and sigma2 M^* sigma2 (reading R8).
  int pair;        // 0: extended-lattice layout, 1: C*-paired layout (cstar > 0 only)
  int Vg;          // stride of the link / clover records: Vh, or Vh / 2 in the paired layout
  int XE[4];       // extended extents T, X1 = 2 L1 (C*) or L1, L2, L3 -- the natural order of the ABI
  int X[4];        // extents of the indexed lattice: = XE, or the physical extents in the paired layout
  int L1;          // physical extent of direction 1 (the C* shift)
  int cstar;       // 0..3
  int antiper;     // fermions antiperiodic in time
  int Vh;          // V/2 = sites per parity = stride of every SoA record
  // Three-level site order (all extents powers of two except the number of blocks per direction):
  //   level 0  tile  b_mu  -- the sites one CTA works on (both parities), lexicographic, x3 fastest;
  //   level 1  block B_mu  -- B/b tiles, lexicographic; consecutive CTAs stay inside one block, so that
  //                           neighbour spinors and the second use of every link are L2 hits;
  //   level 2  blocks      -- lexicographic over X/B blocks, direction 0 slowest.
  int sh[4];       // log2 b_mu (sh[3] >= 1)
  int shB[4];      // log2 B_mu (>= sh)
  int s0[4];       // stride of the in-tile digit of direction mu (full-index units)
  int s1[4];       // stride of the tile-in-block digit
  int s2[4];       // stride of the block digit
  int nB[4];       // blocks per direction
};

// full index idx2(x) = sum_mu g_mu(x_mu); checkerboard index cb = idx2 >> 1; parity = sum x_mu & 1.
__host__ __device__ __forceinline__ int gmu(const Geom& g, int mu, int c) {
  return (c & ((1 << g.sh[mu]) - 1)) * g.s0[mu] + ((c & ((1 << g.shB[mu]) - 1)) >> g.sh[mu]) * g.s1[mu] + (c >> g.shB[mu]) * g.s2[mu];
}
__host__ __device__ __forceinline__ int idx2_of(const Geom& g, const int x[4]) {
  return gmu(g, 0, x[0]) + gmu(g, 1, x[1]) + gmu(g, 2, x[2]) + gmu(g, 3, x[3]);
}
// inverse on the indexed lattice: (cb, parity) -> coordinates
__host__ __device__ __forceinline__ void coords_int(const Geom& g, int cb, int parity, int x[4]) {
  const int tsh = g.sh[0] + g.sh[1] + g.sh[2] + g.sh[3] - 1;                            // log2(tile volume / 2)
  const int d3 = g.shB[3] - g.sh[3], d2 = g.shB[2] - g.sh[2], d1 = g.shB[1] - g.sh[1], d0 = g.shB[0] - g.sh[0];
  int r = cb & ((1 << tsh) - 1);
  int n = cb >> tsh;                                                                     // tile number
  int zh = r & ((1 << (g.sh[3] - 1)) - 1); r >>= (g.sh[3] - 1);
  int yl = r & ((1 << g.sh[2]) - 1); r >>= g.sh[2];
  int xl = r & ((1 << g.sh[1]) - 1); r >>= g.sh[1];
  int tl = r;
  int mz = n & ((1 << d3) - 1); n >>= d3;
  int my = n & ((1 << d2) - 1); n >>= d2;
  int mx = n & ((1 << d1) - 1); n >>= d1;
  int mt = n & ((1 << d0) - 1); n >>= d0;                                                // n = block number
  int bz = n % g.nB[3]; n /= g.nB[3];
  int by = n % g.nB[2]; n /= g.nB[2];
  int bx = n % g.nB[1];
  int bt = n / g.nB[1];
  x[0] = (bt << g.shB[0]) | (mt << g.sh[0]) | tl;
  x[1] = (bx << g.shB[1]) | (mx << g.sh[1]) | xl;
  x[2] = (by << g.shB[2]) | (my << g.sh[2]) | yl;
  int zb = (parity + x[0] + x[1] + x[2]) & 1;
  x[3] = (bz << g.shB[3]) | (mz << g.sh[3]) | (zh << 1) | zb;
}
// (spinor cb, parity) -> EXTENDED coordinates (x1 in [0, 2 L1) under C*)
__host__ __device__ __forceinline__ void coords_of(const Geom& g, int cb, int parity, int x[4]) {
  if (g.pair) {
    coords_int(g, cb >> 1, parity, x);
    x[1] += (cb & 1) * g.L1;
  } else coords_int(g, cb, parity, x);
}
// natural (application) order, Eq. (1) PAPER.md:93 with L1 -> X1, extended coordinates
__host__ __device__ __forceinline__ long lex_of(const Geom& g, const int x[4]) {
  return ((long(x[0]) * g.XE[1] + x[1]) * g.XE[2] + x[2]) * g.XE[3] + x[3];
}

// A subset of the tiles (128 checkerboard indices each) in launch order: tile(k) = base + (k >> lq) * mv + (k & qm), k < count.
// The identity map (count == 0) is the whole lattice.  A time slab of one tile thickness is such a subset for every site
// order (the t digit is the slowest one inside a block and over the blocks); qxd_apply_Dw_host pipelines over these slabs.
struct TileMap {
  int lq = 0, qm = 0, mv = 1, base = 0, count = 0;
};
__host__ __device__ __forceinline__ int tile_of(const TileMap& m, int k) { return m.base + (k >> m.lq) * m.mv + (k & m.qm); }

// Per-thread site context: coordinates and their index contributions (separable index).
struct Site {
  int x[4];     // coordinates on the indexed lattice (physical in the paired layout)
  int gx[4];
  int idx2;
  int m;        // mirror bit (paired layout), else 0
};
// PAIR: 0 / 1 = layout known at compile time (the dslash kernels), -1 = read g.pair
template <int PAIR = -1>
__host__ __device__ __forceinline__ void site_init(const Geom& g, int cb, int parity, Site& s) {
  const bool pair = PAIR < 0 ? (g.pair != 0) : (PAIR != 0);
  s.m = pair ? (cb & 1) : 0;
  coords_int(g, pair ? (cb >> 1) : cb, parity, s.x);
#pragma unroll
  for (int mu = 0; mu < 4; mu++) s.gx[mu] = gmu(g, mu, s.x[mu]);
  s.idx2 = s.gx[0] + s.gx[1] + s.gx[2] + s.gx[3];
}
// checkerboard index of x + dir*mu-hat with the boundary rules of reading R8: time and direction 1
// periodic (X1 = 2 L1 under C*), directions k in 2..cstar wrap with the shift x1 -> x1 + L1 mod 2 L1
// ("shifted boundaries").  The neighbour has the opposite parity.
template <int MU, int DIR, int PAIR = -1>
__host__ __device__ __forceinline__ int neighbour_cb(const Geom& g, const Site& s) {
  const bool pair = PAIR < 0 ? (g.pair != 0) : (PAIR != 0);
  int c = s.x[MU] + DIR;
  bool wrap = false;
  if (DIR > 0) { if (c >= g.X[MU]) { c = 0; wrap = true; } }
  else         { if (c < 0) { c = g.X[MU] - 1; wrap = true; } }
  int n = s.idx2 - s.gx[MU] + gmu(g, MU, c);
  if (pair) {
    // paired layout: every direction is periodic on the physical lattice; crossing a C* boundary (direction 1, and
    // directions 2..cstar) lands on the mirror image: the mirror bit flips
    const int flip = (wrap && MU >= 1 && MU <= (MU == 1 ? 1 : g.cstar)) ? 1 : 0;
    return ((n >> 1) << 1) | (s.m ^ flip);
  }
  if (MU >= 2) {
    if (wrap && MU <= g.cstar) {
      int y1 = s.x[1] + g.L1;
      if (y1 >= g.X[1]) y1 -= g.X[1];
      n += gmu(g, 1, y1) - s.gx[1];
    }
  }
  return n >> 1;
}
// run-time (mu,dir) version for the one-off kernels (clover build); also moves the Site.
__device__ __forceinline__ void site_step(const Geom& g, const Site& s, int mu, int dir, Site& o) {
  o = s;
  int c = s.x[mu] + dir;
  bool wrap = false;
  if (c >= g.X[mu]) { c = 0; wrap = true; }
  if (c < 0) { c = g.X[mu] - 1; wrap = true; }
  o.x[mu] = c; o.gx[mu] = gmu(g, mu, c);
  if (g.pair) {
    if (wrap && mu >= 1 && mu <= (mu == 1 ? 1 : g.cstar)) o.m = s.m ^ 1;
  } else if (wrap && mu >= 2 && mu <= g.cstar) {
    int y1 = s.x[1] + g.L1;
    if (y1 >= g.X[1]) y1 -= g.X[1];
    o.x[1] = y1; o.gx[1] = gmu(g, 1, y1);
  }
  o.idx2 = o.gx[0] + o.gx[1] + o.gx[2] + o.gx[3];
}
__device__ __forceinline__ int site_parity(const Site& s) { return (s.x[0] + s.x[1] + s.x[2] + s.x[3]) & 1; }

// ---------------------------------------------------------------------------------------------
// Storage precisions.  A "record" of NR reals per site is stored as ceil(NR/RPC) 16-byte chunks,
// chunk-major: element (chunk c, site cb) at vector index c*Vh + cb, so that consecutive threads
// (consecutive cb) issue one coalesced 128-bit access per chunk.
// ---------------------------------------------------------------------------------------------
template <typename S> struct PT;
template <> struct PT<double> { typedef double2 V; typedef double C; static constexpr int RPC = 2; static constexpr int ID = 0; };
template <> struct PT<float>  { typedef float4 V;  typedef float C;  static constexpr int RPC = 4; static constexpr int ID = 1; };
template <> struct PT<__half> { typedef uint4 V;   typedef float C;  static constexpr int RPC = 8; static constexpr int ID = 2; };

__device__ __forceinline__ void unpack_vec(const double2& v, double* o) { o[0] = v.x; o[1] = v.y; }
__device__ __forceinline__ void unpack_vec(const float4& v, float* o) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }
__device__ __forceinline__ void unpack_vec(const uint4& v, float* o) {
  const __half2* h = reinterpret_cast<const __half2*>(&v);
#pragma unroll
  for (int i = 0; i < 4; i++) { float2 f = __half22float2(h[i]); o[2 * i] = f.x; o[2 * i + 1] = f.y; }
}
__device__ __forceinline__ double2 pack_vec(const double* o, double2*) { return make_double2(o[0], o[1]); }
__device__ __forceinline__ float4 pack_vec(const float* o, float4*) { return make_float4(o[0], o[1], o[2], o[3]); }
__device__ __forceinline__ uint4 pack_vec(const float* o, uint4*) {
  uint4 v;
  __half2* h = reinterpret_cast<__half2*>(&v);
#pragma unroll
  for (int i = 0; i < 4; i++) h[i] = __floats2half2_rn(o[2 * i], o[2 * i + 1]);
  return v;
}

// Read-only 16-byte loads as volatile asm: the issue order written in the kernels (software-pipelined batches)
// is the order the compiler keeps; plain __ldg loads get sunk towards their use to save registers.
__device__ __forceinline__ double2 ldg_pinned(const double2* p) {
  double2 v;
  asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ float4 ldg_pinned(const float4* p) {
  float4 v;
  asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ uint4 ldg_pinned(const uint4* p) {
  uint4 v;
  asm volatile("ld.global.nc.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ float ldg_pinned(const float* p) {
  float v;
  asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}

// load reals [R0, R0+N) of the record of site cb (read-only path)
template <typename S, int R0, int N>
__device__ __forceinline__ void load_reals(const void* __restrict__ base, int Vh, int cb, typename PT<S>::C* out) {
  typedef typename PT<S>::V V;
  typedef typename PT<S>::C C;
  constexpr int RPC = PT<S>::RPC;
  constexpr int C0 = R0 / RPC, C1 = (R0 + N - 1) / RPC;
  const V* p = reinterpret_cast<const V*>(base);
#pragma unroll
  for (int c = C0; c <= C1; c++) {
    V v = __ldg(p + size_t(c) * Vh + cb);
    C tmp[RPC];
    unpack_vec(v, tmp);
#pragma unroll
    for (int k = 0; k < RPC; k++) {
      constexpr int dummy = 0; (void)dummy;
      int r = c * RPC + k;
      if (r >= R0 && r < R0 + N) out[r - R0] = tmp[k];
    }
  }
}
// store a whole record of NR reals (NR % RPC == 0)
template <typename S, int NR>
__device__ __forceinline__ void store_record(void* __restrict__ base, int Vh, int cb, const typename PT<S>::C* in) {
  typedef typename PT<S>::V V;
  constexpr int RPC = PT<S>::RPC;
  static_assert(NR % RPC == 0, "record must fill whole chunks");
  V* p = reinterpret_cast<V*>(base);
#pragma unroll
  for (int c = 0; c < NR / RPC; c++) p[size_t(c) * Vh + cb] = pack_vec(in + c * RPC, (V*)nullptr);
}

// A packed half-lattice spinor: 24 reals per site; fp16 adds one fp32 scale per site (block-float,
// reading R12): stored halves = value / scale, scale = max |component| of the site.
struct SpinorPtr {
  void* data;
  float* scale;  // fp16 only
};
template <typename S> __host__ __device__ inline size_t spinor_half_bytes(int Vh) {
  return size_t(Vh) * 24 * sizeof(S) + (PT<S>::ID == 2 ? size_t(Vh) * 4 : 0);
}
template <typename S> __host__ __device__ inline SpinorPtr spinor_view(void* base, int Vh, int parity) {
  char* b = static_cast<char*>(base) + size_t(parity) * spinor_half_bytes<S>(Vh);
  SpinorPtr p;
  p.data = b;
  p.scale = (PT<S>::ID == 2) ? reinterpret_cast<float*>(b + size_t(Vh) * 24 * sizeof(S)) : nullptr;
  return p;
}
template <typename S>
__device__ __forceinline__ void load_spinor(const SpinorPtr& p, int Vh, int cb, typename PT<S>::C* out) {
  load_reals<S, 0, 24>(p.data, Vh, cb, out);
  if (PT<S>::ID == 2) {
    float sc = __ldg(p.scale + cb);
#pragma unroll
    for (int i = 0; i < 24; i++) out[i] *= sc;
  }
}
template <typename S>
__device__ __forceinline__ void store_spinor(const SpinorPtr& p, int Vh, int cb, typename PT<S>::C* v) {
  if (PT<S>::ID == 2) {
    float m = 0.f;
#pragma unroll
    for (int i = 0; i < 24; i++) m = fmaxf(m, fabsf((float)v[i]));
    float inv = m > 0.f ? 1.0f / m : 0.f;
#pragma unroll
    for (int i = 0; i < 24; i++) v[i] *= inv;
    p.scale[cb] = m;
  }
  store_record<S, 24>(p.data, Vh, cb, v);
}

// ---------------------------------------------------------------------------------------------
// Reductions (row a6): warp shuffle -> block -> grid in two kernels.  Every block stores its partial sums and retires;
// reduce_finalize_k (one CTA per slot, launched right behind on the same stream) adds the partials in a fixed order, so the
// result is deterministic for a fixed launch configuration.  fp64 accumulators across sites for every storage type.
// (A single-pass version -- atomic ticket, last block adds -- kept every CTA of the dslash resident for a memory fence and
// an atomic round trip: the D-hat pass with the fused norm took 399 us instead of 333 at c3 fp32, 313 instead of 222 in fp16.)
// ---------------------------------------------------------------------------------------------
struct Reducer {
  double* partials;    // [slot][N][nparts]
  double* result;      // [slot * rstride + N]
  int rstride;         // distance (in doubles) between the results of consecutive slots (right-hand sides)
};
// part / nparts: this block's index among the blocks that contribute to `slot` and their number.
template <int N>
__device__ __forceinline__ void grid_reduce(double (&v)[N], const Reducer& R, int part, int nparts, int slot) {
  __shared__ double sm[N][32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  double* partials = R.partials + size_t(slot) * N * nparts;
  __syncthreads();  // sm may still be read by a previous call
#pragma unroll
  for (int k = 0; k < N; k++) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
    if (lane == 0) sm[k][w] = v[k];
  }
  __syncthreads();
  if (w == 0) {
#pragma unroll
    for (int k = 0; k < N; k++) {
      double t = lane < nw ? sm[k][lane] : 0.0;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
      if (lane == 0) partials[size_t(k) * nparts + part] = t;
    }
  }
}
// grid (1, nslots), FINALIZE_THREADS threads: result[slot * rstride + k] = sum_i partials[slot][k][i], fixed order
constexpr int FINALIZE_THREADS = 1024;
template <int N>
__global__ void __launch_bounds__(FINALIZE_THREADS) reduce_finalize_k(Reducer R, int nparts) {
  __shared__ double sm[N][32];
  const int slot = blockIdx.y, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const double* partials = R.partials + size_t(slot) * N * nparts;
  double t[N];
#pragma unroll
  for (int k = 0; k < N; k++) {
    double t0 = 0.0, t1 = 0.0, t2 = 0.0, t3 = 0.0;   // four independent loads in flight per thread
    int i = threadIdx.x;
    for (; i + 3 * FINALIZE_THREADS < nparts; i += 4 * FINALIZE_THREADS) {
      t0 += partials[size_t(k) * nparts + i]; t1 += partials[size_t(k) * nparts + i + FINALIZE_THREADS];
      t2 += partials[size_t(k) * nparts + i + 2 * FINALIZE_THREADS]; t3 += partials[size_t(k) * nparts + i + 3 * FINALIZE_THREADS];
    }
    for (; i < nparts; i += FINALIZE_THREADS) t0 += partials[size_t(k) * nparts + i];
    t[k] = (t0 + t1) + (t2 + t3);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t[k] += __shfl_xor_sync(0xffffffffu, t[k], o);
    if (lane == 0) sm[k][w] = t[k];
  }
  __syncthreads();
  if (w == 0) {
#pragma unroll
    for (int k = 0; k < N; k++) {
      double u = sm[k][lane];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) u += __shfl_xor_sync(0xffffffffu, u, o);
      if (lane == 0) R.result[size_t(slot) * R.rstride + k] = u;
    }
  }
}
// one slot per blockIdx.y (batched BLAS: blockIdx.y = right-hand side)
template <int N>
__device__ __forceinline__ void grid_reduce(double (&v)[N], const Reducer& R) {
  grid_reduce<N>(v, R, blockIdx.x, gridDim.x, blockIdx.y);
}

// Right-hand side r of a batch: consecutive right-hand sides are `stride` bytes apart (data and fp16 scales alike).
__host__ __device__ __forceinline__ SpinorPtr rhs_view(const SpinorPtr& p, size_t stride, int r) {
  SpinorPtr q;
  q.data = static_cast<char*>(p.data) + stride * r;
  q.scale = p.scale ? reinterpret_cast<float*>(reinterpret_cast<char*>(p.scale) + stride * r) : nullptr;
  return q;
}

}  // namespace qxd
