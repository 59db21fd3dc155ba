// pack.cu -- SURVEY.md §8 rows a2 (gauge load / pack) and a9 (spinor pack/unpack + precision convert).
// The paper's analogue is the reorder classes OpenQCDOrder / OpenQCDDiracOrder (PAPER.md:81-85,107-111,
// 133): per (checkerboard index, parity) compute the coordinates, map them to the application's index
// with a pure function and copy the site's numbers.  Here the application order is the
// natural order of include/qxd.h and the device order is the tiled even-odd SoA of qxd_common.cuh.
#include "qxd_ctx.h"

namespace qxd {

// ---- gauge: natural physical AoS -> extended even-odd SoA fp64; mirror half = conj(U), -A (reading R8)
__global__ void __launch_bounds__(128) gauge_pack_k(Geom g, const double* __restrict__ U, const double* __restrict__ A,
                                                    void* Ug0, void* Ug1, void* Ag0, void* Ag1) {
  int cb = blockIdx.x * blockDim.x + threadIdx.x;   // index of the link record: extended site, or physical site (paired layout)
  int parity = blockIdx.y;
  if (cb >= g.Vg) return;
  int x[4];
  coords_int(g, cb, parity, x);
  bool mirror = !g.pair && x[1] >= g.L1;
  int x1p = mirror ? x[1] - g.L1 : x[1];
  size_t sp = ((size_t(x[0]) * g.L1 + x1p) * g.X[2] + x[2]) * g.X[3] + x[3];
  double r[72];
  const double* u = U + sp * 72;
#pragma unroll
  for (int k = 0; k < 36; k++) {
    r[2 * k] = u[2 * k];
    r[2 * k + 1] = mirror ? -u[2 * k + 1] : u[2 * k + 1];
  }
  store_record<double, 72>(parity ? Ug1 : Ug0, g.Vg, cb, r);
  double a[4] = {0, 0, 0, 0};
  if (A) {
#pragma unroll
    for (int mu = 0; mu < 4; mu++) a[mu] = mirror ? -A[sp * 4 + mu] : A[sp * 4 + mu];
  }
  store_record<double, 4>(parity ? Ag1 : Ag0, g.Vg, cb, a);
}

// ---- hopping links W_mu(x) = e^{i q A_mu(x)} U_mu(x), fermion time-boundary sign folded
// into W_0 at x0 = T-1 (reading R9; the clover term is built from Ug and is unaffected).
// NL = 14: rows 0 and 1 of W and det W = e^{3 i q A} det U (-1 at the antiperiodic time boundary); the dslash rebuilds
// row 2 = det W * conj(row0 x row1).  det U is computed (not assumed 1), so U(3) input links are represented exactly.
template <typename S, int NL>
__global__ void __launch_bounds__(128) hoplinks_k(Geom g, double q, int use_a, const void* Ug0, const void* Ug1, const void* Ag0,
                                                  const void* Ag1, void* W0, void* W1) {
  typedef typename PT<S>::C C;
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  int parity = blockIdx.y;
  if (cb >= g.Vg) return;
  int x[4];
  coords_int(g, cb, parity, x);
  double u[72], a[4];
  load_reals<double, 0, 72>(parity ? Ug1 : Ug0, g.Vg, cb, u);
  load_reals<double, 0, 4>(parity ? Ag1 : Ag0, g.Vg, cb, a);
  C w[4 * NL];
#pragma unroll
  for (int mu = 0; mu < 4; mu++) {
    double c = 1.0, s = 0.0;
    if (use_a) sincos(q * a[mu], &s, &c);
    if (mu == 0 && g.antiper && x[0] == g.X[0] - 1) { c = -c; s = -s; }
    const double* m = u + 18 * mu;
#pragma unroll
    for (int k = 0; k < NL / 2 && k < 9; k++) {
      double re = m[2 * k], im = m[2 * k + 1];
      if (NL == 18 || k < 6) {
        w[NL * mu + 2 * k] = (C)(c * re - s * im);
        w[NL * mu + 2 * k + 1] = (C)(c * im + s * re);
      }
    }
    if (NL == 14) {
      // det U = sum_c row2[c] * (row0 x row1)[c]
      double dr = 0.0, di = 0.0;
#pragma unroll
      for (int cc = 0; cc < 3; cc++) {
        const int a0 = (cc + 1) % 3, b0 = (cc + 2) % 3;
        double zr = m[2 * a0] * m[6 + 2 * b0] - m[2 * a0 + 1] * m[6 + 2 * b0 + 1] - m[2 * b0] * m[6 + 2 * a0] + m[2 * b0 + 1] * m[6 + 2 * a0 + 1];
        double zi = m[2 * a0] * m[6 + 2 * b0 + 1] + m[2 * a0 + 1] * m[6 + 2 * b0] - m[2 * b0] * m[6 + 2 * a0 + 1] - m[2 * b0 + 1] * m[6 + 2 * a0];
        dr += m[12 + 2 * cc] * zr - m[12 + 2 * cc + 1] * zi;
        di += m[12 + 2 * cc] * zi + m[12 + 2 * cc + 1] * zr;
      }
      // (c + i s)^3 det U
      const double c3 = c * (c * c - 3.0 * s * s), s3 = s * (3.0 * c * c - s * s);
      w[NL * mu + 12] = (C)(c3 * dr - s3 * di);
      w[NL * mu + 13] = (C)(c3 * di + s3 * dr);
    }
  }
  store_record<S, 4 * NL>(parity ? W1 : W0, g.Vg, cb, w);
}

// ---- spinors: natural AoS fp64 <-> packed SoA in precision S
template <typename S>
__global__ void __launch_bounds__(128) spinor_pack_k(Geom g, const double* __restrict__ nat, SpinorPtr p0, SpinorPtr p1, int pmask,
                                                     int compact_even, TileMap tm) {
  typedef typename PT<S>::C C;
  int cb = tile_of(tm, blockIdx.x) * 128 + threadIdx.x;
  int parity = blockIdx.y;
  if (cb >= g.Vh || !((pmask >> parity) & 1)) return;
  int x[4];
  coords_of(g, cb, parity, x);
  size_t s = lex_of(g, x);
  if (compact_even) s >>= 1;
  const double2* src = reinterpret_cast<const double2*>(nat + s * 24);
  C v[24];
#pragma unroll
  for (int k = 0; k < 12; k++) { double2 z = src[k]; v[2 * k] = (C)z.x; v[2 * k + 1] = (C)z.y; }
  store_spinor<S>(parity ? p1 : p0, g.Vh, cb, v);
}
template <typename S>
__global__ void __launch_bounds__(128) spinor_unpack_k(Geom g, SpinorPtr p0, SpinorPtr p1, double* __restrict__ nat, int pmask,
                                                       int compact_even, TileMap tm) {
  typedef typename PT<S>::C C;
  int cb = tile_of(tm, blockIdx.x) * 128 + threadIdx.x;
  int parity = blockIdx.y;
  if (cb >= g.Vh || !((pmask >> parity) & 1)) return;
  int x[4];
  coords_of(g, cb, parity, x);
  size_t s = lex_of(g, x);
  if (compact_even) s >>= 1;
  C v[24];
  load_spinor<S>(parity ? p1 : p0, g.Vh, cb, v);
  double2* dst = reinterpret_cast<double2*>(nat + s * 24);
#pragma unroll
  for (int k = 0; k < 12; k++) dst[k] = make_double2((double)v[2 * k], (double)v[2 * k + 1]);
}

template <typename SF, typename ST>
__global__ void __launch_bounds__(128) convert_spinor_k(int Vh, SpinorPtr from, SpinorPtr to, size_t rs_from, size_t rs_to) {
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  from = rhs_view(from, rs_from, blockIdx.y); to = rhs_view(to, rs_to, blockIdx.y);
  typename PT<SF>::C v[24];
  typename PT<ST>::C w[24];
  load_spinor<SF>(from, Vh, cb, v);
#pragma unroll
  for (int i = 0; i < 24; i++) w[i] = (typename PT<ST>::C)v[i];
  store_spinor<ST>(to, Vh, cb, w);
}

template <typename ST>
__global__ void __launch_bounds__(128) convert72_k(int Vh, const void* from, void* to) {
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  double v[72];
  typename PT<ST>::C w[72];
  load_reals<double, 0, 72>(from, Vh, cb, v);
#pragma unroll
  for (int i = 0; i < 72; i++) w[i] = (typename PT<ST>::C)v[i];
  store_record<ST, 72>(to, Vh, cb, w);
}

// Packed 6x6 Hermitian block (PAPER.md:117 order, index i = 3 s + c) of the mirror site: M' = sigma2 M^* sigma2, i.e.
//   M'_(0c)(0c') = conj M_(1c)(1c'),  M'_(1c)(1c') = conj M_(0c)(0c'),  M'_(0c)(1c') = -conj M_(1c)(0c') = -M_(0c')(1c).
__host__ __device__ inline int packed_upper_index(int i, int j) { return i * 6 - (i * (i + 1)) / 2 + (j - i - 1); }
__device__ __forceinline__ void mirror_block(const double* b, double* o) {
#pragma unroll
  for (int c = 0; c < 3; c++) { o[c] = b[3 + c]; o[3 + c] = b[c]; }
#pragma unroll
  for (int c = 0; c < 3; c++)
#pragma unroll
    for (int d = 0; d < 3; d++) {
      if (d > c) {
        const int k00 = 6 + 2 * packed_upper_index(c, d), k11 = 6 + 2 * packed_upper_index(3 + c, 3 + d);
        o[k00] = b[k11]; o[k00 + 1] = -b[k11 + 1];
        o[k11] = b[k00]; o[k11 + 1] = -b[k00 + 1];
      }
      const int k01 = 6 + 2 * packed_upper_index(c, 3 + d), k10 = 6 + 2 * packed_upper_index(d, 3 + c);
      o[k01] = -b[k10]; o[k01 + 1] = -b[k10 + 1];
    }
}
__global__ void __launch_bounds__(128) clover_export_k(Geom g, const void* m0, const void* m1, double* __restrict__ out) {
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  int parity = blockIdx.y;
  if (cb >= g.Vh) return;
  int x[4];
  coords_of(g, cb, parity, x);
  size_t s = lex_of(g, x);
  double v[72];
  load_reals<double, 0, 72>(parity ? m1 : m0, g.Vg, g.pair ? (cb >> 1) : cb, v);
  if (g.pair && (cb & 1)) {   // mirror site: sigma2 M^* sigma2 of either block
    double t[72];
#pragma unroll
    for (int b = 0; b < 2; b++) mirror_block(v + 36 * b, t + 36 * b);
#pragma unroll
    for (int i = 0; i < 72; i++) v[i] = t[i];
  }
#pragma unroll
  for (int i = 0; i < 72; i++) out[s * 72 + i] = v[i];
}

static inline dim3 grid_for(int Vh, int ny) { return dim3((Vh + 127) / 128, ny); }

int launch_gauge_pack(qxd_ctx* c, const double* U, const double* A) {
  gauge_pack_k<<<grid_for(c->g.Vg, 2), 128, 0, c->stream>>>(c->g, U, A, c->Ug[0], c->Ug[1], c->Ag[0], c->Ag[1]);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

int launch_hoplinks(qxd_ctx* c, int prec) {
  dim3 gr = grid_for(c->g.Vg, 2);
  int ua = c->have_qed ? 1 : 0;
#define QXD_HOPLINKS(S, NL) hoplinks_k<S, NL><<<gr, 128, 0, c->stream>>>(c->g, c->q, ua, c->Ug[0], c->Ug[1], c->Ag[0], c->Ag[1], c->W[prec][0], c->W[prec][1])
  if (c->link_reals[prec] == 14) { if (prec == 0) QXD_HOPLINKS(double, 14); else if (prec == 1) QXD_HOPLINKS(float, 14); else QXD_HOPLINKS(__half, 14); }
  else { if (prec == 0) QXD_HOPLINKS(double, 18); else if (prec == 1) QXD_HOPLINKS(float, 18); else QXD_HOPLINKS(__half, 18); }
#undef QXD_HOPLINKS
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

int launch_spinor_pack(qxd_ctx* c, int prec, const double* nat, void* packed, int pmask, int compact_even, const TileMap& tm) {
  dim3 gr = tm.count > 0 ? dim3(tm.count, 2) : grid_for(c->g.Vh, 2);
  SpinorPtr p0 = half_view(prec, packed, c->g.Vh, 0), p1 = half_view(prec, packed, c->g.Vh, 1);
  if (prec == 0) spinor_pack_k<double><<<gr, 128, 0, c->stream>>>(c->g, nat, p0, p1, pmask, compact_even, tm);
  else if (prec == 1) spinor_pack_k<float><<<gr, 128, 0, c->stream>>>(c->g, nat, p0, p1, pmask, compact_even, tm);
  else spinor_pack_k<__half><<<gr, 128, 0, c->stream>>>(c->g, nat, p0, p1, pmask, compact_even, tm);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int launch_spinor_unpack(qxd_ctx* c, int prec, const void* packed, double* nat, int pmask, int compact_even, const TileMap& tm) {
  dim3 gr = tm.count > 0 ? dim3(tm.count, 2) : grid_for(c->g.Vh, 2);
  SpinorPtr p0 = half_view(prec, const_cast<void*>(packed), c->g.Vh, 0), p1 = half_view(prec, const_cast<void*>(packed), c->g.Vh, 1);
  if (prec == 0) spinor_unpack_k<double><<<gr, 128, 0, c->stream>>>(c->g, p0, p1, nat, pmask, compact_even, tm);
  else if (prec == 1) spinor_unpack_k<float><<<gr, 128, 0, c->stream>>>(c->g, p0, p1, nat, pmask, compact_even, tm);
  else spinor_unpack_k<__half><<<gr, 128, 0, c->stream>>>(c->g, p0, p1, nat, pmask, compact_even, tm);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

template <typename SF>
static void convert_from(qxd_ctx* c, const SpinorPtr& from, int pt, const SpinorPtr& to, int n, size_t rf, size_t rt) {
  dim3 gr = grid_for(c->g.Vh, n);
  if (pt == 0) convert_spinor_k<SF, double><<<gr, 128, 0, c->stream>>>(c->g.Vh, from, to, rf, rt);
  else if (pt == 1) convert_spinor_k<SF, float><<<gr, 128, 0, c->stream>>>(c->g.Vh, from, to, rf, rt);
  else convert_spinor_k<SF, __half><<<gr, 128, 0, c->stream>>>(c->g.Vh, from, to, rf, rt);
}
int launch_convert_spinor(qxd_ctx* c, int pf, const SpinorPtr& from, int pt, const SpinorPtr& to, int n, size_t rf, size_t rt) {
  if (pf == 0) convert_from<double>(c, from, pt, to, n, rf, rt);
  else if (pf == 1) convert_from<float>(c, from, pt, to, n, rf, rt);
  else convert_from<__half>(c, from, pt, to, n, rf, rt);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int launch_convert_record72(qxd_ctx* c, const void* from64, int pt, void* to) {
  dim3 gr = grid_for(c->g.Vg, 1);
  if (pt == 1) convert72_k<float><<<gr, 128, 0, c->stream>>>(c->g.Vg, from64, to);
  else if (pt == 2) convert72_k<__half><<<gr, 128, 0, c->stream>>>(c->g.Vg, from64, to);
  else return fail(c, QXD_EINVAL, "convert72: bad precision");
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int launch_clover_export(qxd_ctx* c, double* out, int inverse) {
  void* const* m = inverse ? c->Mi[0] : c->M[0];
  clover_export_k<<<grid_for(c->g.Vh, 2), 128, 0, c->stream>>>(c->g, m[0], m[1], out);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // namespace qxd
