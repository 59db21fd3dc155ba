// halo.cu -- SURVEY.md §8(f) row f2, the device side of the domain decomposition: the paper's codes run on rank-local
// lattices, exchange boundary data before the operator is applied and realise the C*
// boundary conditions through the neighbour map between ranks.  Here a rank's lattice carries ghost layers
// in the cut directions; what travels between ranks is the spin-PROJECTED boundary spinor -- 12 reals per face site and
// direction instead of 24 -- produced and consumed by the kernels of this file:
//
//   face_gather:   buf[f] = upper two spin components of (1 - sign gamma_mu) psi(x),  x_mu = coord     (project<MU,SIGN>)
//   face_scatter:  psi(x) = (h, 0) at the ghost sites x_mu = coord: a spinor whose projection (1 - sign gamma_mu) psi has the
//                  upper components h, which is all the hop from the first owned layer into the ghost layer reads
//                  (project = psi_upper + sign * (combination of psi_lower)); the source face site is shifted by `shift1`
//                  in direction 1 when the message crossed a C* boundary (the shifted boundaries of PAPER.md:137-139).
//   halo_zero:     psi(x) = 0 for lo <= x_mu < hi (ghost layers are cleared after use so that norms see owned sites only)
//
// Face sites are indexed lexicographically over the three other coordinates (extended local lattice, natural order, last
// coordinate fastest); a single-parity field uses the compact index f >> 1 (all extents are even).
#include "dslash_kernel.cuh"

namespace qxd {

namespace {

struct FaceGeom {
  int mu, coord;
  int d[3];      // the other three directions, increasing
  int n[3];      // their extended extents
  int nface;     // n[0] n[1] n[2]
};

__host__ __device__ __forceinline__ void face_coords(const FaceGeom& F, int f, int x[4]) {
  x[F.mu] = F.coord;
  x[F.d[2]] = f % F.n[2]; f /= F.n[2];
  x[F.d[1]] = f % F.n[1]; f /= F.n[1];
  x[F.d[0]] = f;
}
__host__ __device__ __forceinline__ int face_index(const FaceGeom& F, const int x[4]) {
  return (x[F.d[0]] * F.n[1] + x[F.d[1]]) * F.n[2] + x[F.d[2]];
}
// extended coordinates -> (checkerboard index, parity) in either layout (as qxd_site_index)
__device__ __forceinline__ int cb_of(const Geom& g, const int x[4], int& parity) {
  parity = (x[0] + x[1] + x[2] + x[3]) & 1;
  if (g.pair) {
    const int m = x[1] >= g.L1 ? 1 : 0;
    const int xp[4] = {x[0], x[1] - m * g.L1, x[2], x[3]};
    return ((idx2_of(g, xp) >> 1) << 1) | m;
  }
  return idx2_of(g, x) >> 1;
}
template <typename C>
__device__ __forceinline__ void project_rt(int mu, int sign, const C* psi, C* h) {
  if (sign > 0) {
    if (mu == 0) project<0, +1>(psi, h); else if (mu == 1) project<1, +1>(psi, h); else if (mu == 2) project<2, +1>(psi, h); else project<3, +1>(psi, h);
  } else {
    if (mu == 0) project<0, -1>(psi, h); else if (mu == 1) project<1, -1>(psi, h); else if (mu == 2) project<2, -1>(psi, h); else project<3, -1>(psi, h);
  }
}

template <typename S>
__global__ void __launch_bounds__(128) face_gather_k(Geom g, FaceGeom F, SpinorPtr p0, SpinorPtr p1, int pmask, int sign, typename PT<S>::C* buf) {
  typedef typename PT<S>::C C;
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= F.nface) return;
  int x[4], parity;
  face_coords(F, f, x);
  const int cb = cb_of(g, x, parity);
  if (!((pmask >> parity) & 1)) return;
  C psi[24], h[12];
  load_spinor<S>(parity ? p1 : p0, g.Vh, cb, psi);
  project_rt(F.mu, sign, psi, h);
  C* o = buf + size_t(pmask == 3 ? f : (f >> 1)) * 12;
#pragma unroll
  for (int i = 0; i < 12; i++) o[i] = h[i];
}
template <typename S>
__global__ void __launch_bounds__(128) face_scatter_k(Geom g, FaceGeom F, SpinorPtr p0, SpinorPtr p1, int pmask, int shift1, const typename PT<S>::C* buf) {
  typedef typename PT<S>::C C;
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= F.nface) return;
  int x[4], parity;
  face_coords(F, f, x);
  const int cb = cb_of(g, x, parity);
  if (!((pmask >> parity) & 1)) return;
  int y[4] = {x[0], x[1], x[2], x[3]};
  if (shift1) { y[1] += shift1; if (y[1] >= g.XE[1]) y[1] -= g.XE[1]; }
  const int fs = face_index(F, y);
  const C* in = buf + size_t(pmask == 3 ? fs : (fs >> 1)) * 12;
  C psi[24];
#pragma unroll
  for (int i = 0; i < 12; i++) { psi[i] = in[i]; psi[12 + i] = 0; }
  store_spinor<S>(parity ? p1 : p0, g.Vh, cb, psi);
}
template <typename S>
__global__ void __launch_bounds__(128) halo_zero_k(Geom g, FaceGeom F, SpinorPtr p0, SpinorPtr p1, int pmask, int lo, int hi) {
  typedef typename PT<S>::C C;
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= F.nface) return;
  C z[24];
  for (int c = lo; c < hi; c++) {
    F.coord = c;
    int x[4], parity;
    face_coords(F, f, x);
    const int cb = cb_of(g, x, parity);
    if (!((pmask >> parity) & 1)) continue;
#pragma unroll
    for (int i = 0; i < 24; i++) z[i] = 0;
    store_spinor<S>(parity ? p1 : p0, g.Vh, cb, z);
  }
}

int make_face(qxd_ctx* c, int mu, int coord, FaceGeom& F) {
  if (mu < 0 || mu > 3 || coord < 0 || coord >= c->g.XE[mu]) return fail(c, QXD_EINVAL, "face: direction or coordinate out of range");
  F.mu = mu; F.coord = coord;
  int k = 0;
  for (int nu = 0; nu < 4; nu++) if (nu != mu) { F.d[k] = nu; F.n[k] = c->g.XE[nu]; k++; }
  F.nface = F.n[0] * F.n[1] * F.n[2];
  return QXD_OK;
}

}  // namespace

size_t face_bytes(const qxd_ctx* c, int prec, int mu) {
  size_t n = 1;
  for (int nu = 0; nu < 4; nu++) if (nu != mu) n *= size_t(c->g.XE[nu]);
  return n * 12 * (prec == 0 ? 8 : 4);
}

int launch_face_gather(qxd_ctx* c, int prec, void* packed, int pmask, int mu, int coord, int sign, void* buf) {
  FaceGeom F;
  int rc = make_face(c, mu, coord, F);
  if (rc) return rc;
  const int Vh = c->g.Vh;
  dim3 gr((F.nface + 127) / 128);
  if (prec == 0) face_gather_k<double><<<gr, 128, 0, c->stream>>>(c->g, F, half_view(0, packed, Vh, 0), half_view(0, packed, Vh, 1), pmask, sign, (double*)buf);
  else if (prec == 1) face_gather_k<float><<<gr, 128, 0, c->stream>>>(c->g, F, half_view(1, packed, Vh, 0), half_view(1, packed, Vh, 1), pmask, sign, (float*)buf);
  else face_gather_k<__half><<<gr, 128, 0, c->stream>>>(c->g, F, half_view(2, packed, Vh, 0), half_view(2, packed, Vh, 1), pmask, sign, (float*)buf);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int launch_face_scatter(qxd_ctx* c, int prec, void* packed, int pmask, int mu, int coord, int shift1, const void* buf) {
  FaceGeom F;
  int rc = make_face(c, mu, coord, F);
  if (rc) return rc;
  if (shift1 < 0 || shift1 >= c->g.XE[1] || (shift1 & 1) || (mu == 1 && shift1)) return fail(c, QXD_EINVAL, "face_scatter: shift1 must be even, in [0, X1), and 0 for mu = 1");
  const int Vh = c->g.Vh;
  dim3 gr((F.nface + 127) / 128);
  if (prec == 0) face_scatter_k<double><<<gr, 128, 0, c->stream>>>(c->g, F, half_view(0, packed, Vh, 0), half_view(0, packed, Vh, 1), pmask, shift1, (const double*)buf);
  else if (prec == 1) face_scatter_k<float><<<gr, 128, 0, c->stream>>>(c->g, F, half_view(1, packed, Vh, 0), half_view(1, packed, Vh, 1), pmask, shift1, (const float*)buf);
  else face_scatter_k<__half><<<gr, 128, 0, c->stream>>>(c->g, F, half_view(2, packed, Vh, 0), half_view(2, packed, Vh, 1), pmask, shift1, (const float*)buf);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}
int launch_halo_zero(qxd_ctx* c, int prec, void* packed, int pmask, int mu, int lo, int hi) {
  FaceGeom F;
  if (mu < 0 || mu > 3 || lo < 0 || hi > c->g.XE[mu] || lo > hi) return fail(c, QXD_EINVAL, "halo_zero: bad range");
  if (lo == hi) return QXD_OK;
  int rc = make_face(c, mu, lo, F);
  if (rc) return rc;
  const int Vh = c->g.Vh;
  dim3 gr((F.nface + 127) / 128);
  if (prec == 0) halo_zero_k<double><<<gr, 128, 0, c->stream>>>(c->g, F, half_view(0, packed, Vh, 0), half_view(0, packed, Vh, 1), pmask, lo, hi);
  else if (prec == 1) halo_zero_k<float><<<gr, 128, 0, c->stream>>>(c->g, F, half_view(1, packed, Vh, 0), half_view(1, packed, Vh, 1), pmask, lo, hi);
  else halo_zero_k<__half><<<gr, 128, 0, c->stream>>>(c->g, F, half_view(2, packed, Vh, 0), half_view(2, packed, Vh, 1), pmask, lo, hi);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // namespace qxd
