// openqxd.cu -- SURVEY.md §8(f) row f1: the field orders of the paper's host code (§2, §4.1) as reorder kernels
// between openQxD order and this library's natural order, so that the host code's arrays can be handed over as they are.
//
//   site index   xhat = floor((V_B Lambda(n,N_B) + Lambda(b,B)) / 2) + P(x) V/2        Eq. (2)
//                (cache blocks B_mu, even points first), computed on the fly as a pure inlined function --
//                the paper's advice for GPUs instead of the host code's ipt[] table;
//   spinor       (xhat, alpha, a): 12 consecutive complex per site
//   clover       (xhat, +-, i): 2 x 36 reals per site, same packing as ours
//   gauge        (x_odd, +-mu, a, b): 8 links at every odd point, 3x3 row-major
//                entry 2 mu = U_mu(x), entry 2 mu + 1 = U_mu(x - mu)   (reading R20)
// The paper's load()/save() pair corresponds to the two directions of each kernel.  On one GPU the
// pre-call exchange of boundary links between ranks does not arise: every link is in the array.
#include "qxd_ctx.h"

namespace qxd {

namespace {

struct OqxdGeom {
  int X[4];    // extended extents
  int B[4];    // cache block
  int NB[4];   // blocks per direction
  int L1, cstar;
  long V;
  int VB;
};

__host__ __device__ __forceinline__ long oq_lam(const int x[4], const int L[4]) {
  return ((long(x[0]) * L[1] + x[1]) * L[2] + x[2]) * L[3] + x[3];   // Eq. (1)
}
__host__ __device__ __forceinline__ long oq_xhat(const OqxdGeom& o, const int x[4]) {
  int n[4], b[4];
#pragma unroll
  for (int m = 0; m < 4; m++) { n[m] = x[m] / o.B[m]; b[m] = x[m] - n[m] * o.B[m]; }
  const long par = (x[0] + x[1] + x[2] + x[3]) & 1;
  return (long(o.VB) * oq_lam(n, o.NB) + oq_lam(b, o.B)) / 2 + par * (o.V / 2);   // Eq. (2)
}
__host__ __device__ __forceinline__ void oq_coords(const int L[4], long s, int x[4]) {
  x[3] = int(s % L[3]); s /= L[3];
  x[2] = int(s % L[2]); s /= L[2];
  x[1] = int(s % L[1]);
  x[0] = int(s / L[1]);
}
// x + d mu-hat on the extended lattice with the shifted C* boundaries (reading R8)
__host__ __device__ __forceinline__ void oq_shift(const OqxdGeom& o, const int x[4], int mu, int d, int y[4]) {
#pragma unroll
  for (int m = 0; m < 4; m++) y[m] = x[m];
  y[mu] += d;
  bool wrap = false;
  if (y[mu] < 0) { y[mu] += o.X[mu]; wrap = true; }
  if (y[mu] >= o.X[mu]) { y[mu] -= o.X[mu]; wrap = true; }
  if (wrap && mu >= 2 && mu <= o.cstar) { y[1] += o.L1; if (y[1] >= o.X[1]) y[1] -= o.X[1]; }
}

// one thread per (natural-order site, complex pair of the record)
__global__ void __launch_bounds__(256) oq_reorder_k(OqxdGeom o, const double2* __restrict__ in, double2* __restrict__ out, int pairs, int to_oq) {
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i >= o.V * pairs) return;
  const long s = i / pairs;
  const int k = int(i - s * pairs);
  int x[4];
  oq_coords(o.X, s, x);
  const long h = oq_xhat(o, x);
  if (to_oq) out[h * pairs + k] = in[i];
  else out[i] = in[h * pairs + k];
}

__global__ void __launch_bounds__(256) oq_index_k(OqxdGeom o, const int* __restrict__ xs, long n, long* __restrict__ out) {
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i >= n) return;
  int x[4] = {xs[4 * i], xs[4 * i + 1], xs[4 * i + 2], xs[4 * i + 3]};
  out[i] = oq_xhat(o, x);
}

// value of real number r of link mu at the extended-lattice point z, from the physical natural-order field
// (NR = 18: SU(3) link, mirror = complex conjugate; NR = 1: U(1) field A, mirror = -A; reading R8)
template <int NR>
__device__ __forceinline__ double phys_link(const OqxdGeom& o, const double* __restrict__ nat, const int z[4], int mu, int r) {
  const bool mirror = o.cstar > 0 && z[1] >= o.L1;
  const int zp[4] = {z[0], mirror ? z[1] - o.L1 : z[1], z[2], z[3]};
  const int Lp[4] = {o.X[0], o.cstar > 0 ? o.L1 : o.X[1], o.X[2], o.X[3]};
  const double v = nat[(oq_lam(zp, Lp) * 4 + mu) * NR + r];
  if (!mirror) return v;
  return (NR == 1 || (r & 1)) ? -v : v;
}
// natural -> openQxD: one thread per (odd extended point, direction 0..7, real)
template <int NR>
__global__ void __launch_bounds__(256) oq_gauge_to_k(OqxdGeom o, const double* __restrict__ nat, double* __restrict__ ud) {
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i >= o.V * 8 * NR) return;   // loop over all extended points x 8 x NR; even points return below
  const int r = int(i % NR);
  const int d = int((i / NR) % 8);
  const long s = i / (8 * NR);
  int x[4];
  oq_coords(o.X, s, x);
  if (((x[0] + x[1] + x[2] + x[3]) & 1) == 0) return;
  const long od = oq_xhat(o, x) - o.V / 2;
  const int mu = d >> 1;
  int z[4];
  if (d & 1) oq_shift(o, x, mu, -1, z);
  else { z[0] = x[0]; z[1] = x[1]; z[2] = x[2]; z[3] = x[3]; }
  ud[(od * 8 + d) * NR + r] = phys_link<NR>(o, nat, z, mu, r);
}
// openQxD -> natural: one thread per (physical point y, mu, real)
template <int NR>
__global__ void __launch_bounds__(256) oq_gauge_from_k(OqxdGeom o, const double* __restrict__ ud, double* __restrict__ nat) {
  const int Lp[4] = {o.X[0], o.cstar > 0 ? o.L1 : o.X[1], o.X[2], o.X[3]};
  const long Vp = long(Lp[0]) * Lp[1] * Lp[2] * Lp[3];
  const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;
  if (i >= Vp * 4 * NR) return;
  const int r = int(i % NR);
  const int mu = int((i / NR) % 4);
  const long s = i / (4 * NR);
  int y[4];
  oq_coords(Lp, s, y);
  long od;
  int d;
  if ((y[0] + y[1] + y[2] + y[3]) & 1) { od = oq_xhat(o, y) - o.V / 2; d = 2 * mu; }
  else { int z[4]; oq_shift(o, y, mu, +1, z); od = oq_xhat(o, z) - o.V / 2; d = 2 * mu + 1; }
  nat[i] = ud[(od * 8 + d) * NR + r];
}

int make_geom(qxd_ctx* c, const int B[4], OqxdGeom& o) {
  if (!B) return fail(c, QXD_EINVAL, "openqxd: null block");
  o.V = c->V; o.L1 = c->g.L1; o.cstar = c->g.cstar; o.VB = 1;
  for (int m = 0; m < 4; m++) {
    o.X[m] = c->g.XE[m]; o.B[m] = B[m];
    if (B[m] < 1 || o.X[m] % B[m]) return fail(c, QXD_EINVAL, "openqxd: cache-block extents must divide the (extended) lattice extents");
    o.NB[m] = o.X[m] / B[m]; o.VB *= B[m];
  }
  // Eq. (2) pairs consecutive in-block points into one even and one odd index: needs an even innermost block extent
  if (B[3] % 2) return fail(c, QXD_EINVAL, "openqxd: cache-block extent B3 must be even (Eq. (2) halves the in-block index)");
  return QXD_OK;
}

}  // namespace

}  // namespace qxd

using namespace qxd;

extern "C" {

int qxd_openqxd_index(qxd_ctx* c, const int block[4], const int* xs, long n, long* out) {
  if (!c || !xs || !out || n < 0) return c ? fail(c, QXD_EINVAL, "openqxd_index: bad argument") : QXD_EINVAL;
  OqxdGeom o;
  int rc = make_geom(c, block, o);
  if (rc) return rc;
  if (n == 0) return QXD_OK;
  oq_index_k<<<unsigned((n + 255) / 256), 256, 0, c->stream>>>(o, xs, n, out);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

int qxd_openqxd_reorder(qxd_ctx* c, const int block[4], int reals_per_site, int to_openqxd, const double* in, double* out) {
  if (!c || !in || !out || in == out) return c ? fail(c, QXD_EINVAL, "openqxd_reorder: null or aliased pointers") : QXD_EINVAL;
  if (reals_per_site < 2 || reals_per_site % 2) return fail(c, QXD_EINVAL, "openqxd_reorder: reals_per_site must be even (24 spinor, 72 clover)");
  OqxdGeom o;
  int rc = make_geom(c, block, o);
  if (rc) return rc;
  const int pairs = reals_per_site / 2;
  const long n = o.V * pairs;
  oq_reorder_k<<<unsigned((n + 255) / 256), 256, 0, c->stream>>>(o, reinterpret_cast<const double2*>(in), reinterpret_cast<double2*>(out), pairs, to_openqxd ? 1 : 0);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

int qxd_openqxd_gauge(qxd_ctx* c, const int block[4], int reals_per_link, int to_openqxd, const double* in, double* out) {
  if (!c || !in || !out || in == out) return c ? fail(c, QXD_EINVAL, "openqxd_gauge: null or aliased pointers") : QXD_EINVAL;
  if (reals_per_link != 18 && reals_per_link != 1) return fail(c, QXD_EINVAL, "openqxd_gauge: reals_per_link is 18 (SU(3) links) or 1 (U(1) field)");
  OqxdGeom o;
  int rc = make_geom(c, block, o);
  if (rc) return rc;
  const long Vp = long(c->T) * c->L1 * c->L2 * c->L3;
  if (to_openqxd) {
    const long n = o.V * 8 * reals_per_link;
    if (reals_per_link == 18) oq_gauge_to_k<18><<<unsigned((n + 255) / 256), 256, 0, c->stream>>>(o, in, out);
    else oq_gauge_to_k<1><<<unsigned((n + 255) / 256), 256, 0, c->stream>>>(o, in, out);
  } else {
    const long n = Vp * 4 * reals_per_link;
    if (reals_per_link == 18) oq_gauge_from_k<18><<<unsigned((n + 255) / 256), 256, 0, c->stream>>>(o, in, out);
    else oq_gauge_from_k<1><<<unsigned((n + 255) / 256), 256, 0, c->stream>>>(o, in, out);
  }
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // extern "C"
