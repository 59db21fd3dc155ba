// dslash.cu -- SURVEY.md §8 rows a4 (D_w apply), a5 (D-hat even-odd passes) and the dslash-shaped parts
// of a8: the hand-written sm_100a stencil kernel.
//
//   (D_w psi)(x) = M(x) psi(x) - 1/2 sum_mu [ (1-gamma_mu) W_mu(x) psi(x+mu) + (1+gamma_mu) W_mu(x-mu)^dag psi(x-mu) ]
//
// (readings R1-R3; "connects nearest neighbor points ... indices for Dirac spin,
// color charge, and space-time"; W = e^{iqA} U; M = clover term.)
// One thread per output site: for each of the 8 neighbours the spinor is spin-projected to a half spinor
// (2 spin x 3 colour), multiplied by the link (or its adjoint), reconstructed and accumulated; the clover
// or inverse-clover multiplication is fused into the epilogue.  The path is bandwidth bound:
// all field accesses are 16-byte vector loads on chunk-major SoA records, coalesced across the warp.
//
// In the chiral basis of reading R3 (gamma_0 = [[0,-1],[-1,0]], gamma_k = [[0,-i s_k],[i s_k,0]]):
//   (1 -+ gamma_0) psi = (h, +-h),            h = psi_u +- psi_l
//   (1 -+ gamma_k) psi = (h, -+ i s_k h),     h = psi_u +- i s_k psi_l
// with the upper sign for the forward hop.
#include "qxd_ctx.h"
#include <cstdlib>

namespace qxd {

namespace {

struct DslashArgs {
  Geom g;
  SpinorPtr in[2];
  SpinorPtr phi;
  SpinorPtr out[2];
  const void* W[2];
  const void* CL[2];
  int parity_out;
  int prefetch;
  Reducer R;
};

// h = psi_u + SGN * (proj_lower), for direction MU; psi: 24 reals, h: 12 reals
template <int MU, int SGN, typename C>
__device__ __forceinline__ void project(const C* psi, C* h) {
  const C s = (C)SGN;
#pragma unroll
  for (int a = 0; a < 3; a++) {
    const C u0r = psi[2 * a], u0i = psi[2 * a + 1], u1r = psi[6 + 2 * a], u1i = psi[6 + 2 * a + 1];
    const C l0r = psi[12 + 2 * a], l0i = psi[12 + 2 * a + 1], l1r = psi[18 + 2 * a], l1i = psi[18 + 2 * a + 1];
    if (MU == 0) {        // + s * (l0, l1)
      h[2 * a] = u0r + s * l0r; h[2 * a + 1] = u0i + s * l0i;
      h[6 + 2 * a] = u1r + s * l1r; h[6 + 2 * a + 1] = u1i + s * l1i;
    } else if (MU == 1) { // + s * (i l1, i l0)
      h[2 * a] = u0r - s * l1i; h[2 * a + 1] = u0i + s * l1r;
      h[6 + 2 * a] = u1r - s * l0i; h[6 + 2 * a + 1] = u1i + s * l0r;
    } else if (MU == 2) { // + s * (l1, -l0)
      h[2 * a] = u0r + s * l1r; h[2 * a + 1] = u0i + s * l1i;
      h[6 + 2 * a] = u1r - s * l0r; h[6 + 2 * a + 1] = u1i - s * l0i;
    } else {              // + s * (i l0, -i l1)
      h[2 * a] = u0r - s * l0i; h[2 * a + 1] = u0i + s * l0r;
      h[6 + 2 * a] = u1r + s * l1i; h[6 + 2 * a + 1] = u1i - s * l1r;
    }
  }
}
// acc_u += r ; acc_l += lower part reconstructed from r
template <int MU, int SGN, typename C>
__device__ __forceinline__ void reconstruct(const C* r, C* acc) {
  const C s = (C)SGN;
#pragma unroll
  for (int a = 0; a < 3; a++) {
    const C r0r = r[2 * a], r0i = r[2 * a + 1], r1r = r[6 + 2 * a], r1i = r[6 + 2 * a + 1];
    acc[2 * a] += r0r; acc[2 * a + 1] += r0i;
    acc[6 + 2 * a] += r1r; acc[6 + 2 * a + 1] += r1i;
    if (MU == 0) {        // lower = s * (r0, r1)
      acc[12 + 2 * a] += s * r0r; acc[12 + 2 * a + 1] += s * r0i;
      acc[18 + 2 * a] += s * r1r; acc[18 + 2 * a + 1] += s * r1i;
    } else if (MU == 1) { // lower = -s * (i r1, i r0)
      acc[12 + 2 * a] += s * r1i; acc[12 + 2 * a + 1] -= s * r1r;
      acc[18 + 2 * a] += s * r0i; acc[18 + 2 * a + 1] -= s * r0r;
    } else if (MU == 2) { // lower = -s * (r1, -r0)
      acc[12 + 2 * a] -= s * r1r; acc[12 + 2 * a + 1] -= s * r1i;
      acc[18 + 2 * a] += s * r0r; acc[18 + 2 * a + 1] += s * r0i;
    } else {              // lower = -s * (i r0, -i r1)
      acc[12 + 2 * a] += s * r0i; acc[12 + 2 * a + 1] -= s * r0r;
      acc[18 + 2 * a] -= s * r1i; acc[18 + 2 * a + 1] += s * r1r;
    }
  }
}
// r[s][a] = sum_b W[a][b] h[s][b]   (ADJ: sum_b conj(W[b][a]) h[s][b])
template <bool ADJ, typename C>
__device__ __forceinline__ void link_mul(const C* w, const C* h, C* r) {
#pragma unroll
  for (int s = 0; s < 2; s++)
#pragma unroll
    for (int a = 0; a < 3; a++) {
      C re = 0, im = 0;
#pragma unroll
      for (int b = 0; b < 3; b++) {
        const C wr = ADJ ? w[2 * (3 * b + a)] : w[2 * (3 * a + b)];
        const C wi = ADJ ? -w[2 * (3 * b + a) + 1] : w[2 * (3 * a + b) + 1];
        const C hr = h[6 * s + 2 * b], hi = h[6 * s + 2 * b + 1];
        re += wr * hr - wi * hi;
        im += wr * hi + wi * hr;
      }
      r[6 * s + 2 * a] = re; r[6 * s + 2 * a + 1] = im;
    }
}

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
      // out_i += u in_j ; out_j += conj(u) in_i
      out[2 * i] += ur * in[2 * j] - ui * in[2 * j + 1];
      out[2 * i + 1] += ur * in[2 * j + 1] + ui * in[2 * j];
      out[2 * j] += ur * in[2 * i] + ui * in[2 * i + 1];
      out[2 * j + 1] += ur * in[2 * i + 1] - ui * in[2 * i];
    }
}
template <typename S>
__device__ __forceinline__ void clover_mul(const void* CL, int Vh, int cb, const typename PT<S>::C* in, typename PT<S>::C* out) {
  typename PT<S>::C b[36];
  load_reals<S, 0, 36>(CL, Vh, cb, b);
  block_mul(b, in, out);
  load_reals<S, 36, 36>(CL, Vh, cb, b);
  block_mul(b, in + 12, out + 12);
}

// One hop in flight: the raw 16-byte chunks of the neighbour spinor and of the link, exactly as loaded.  Keeping the
// packed vectors (not the unpacked reals) in registers between issue and use lets two hops be in flight per thread
// (software pipeline in hop_all below): the kernel is bound by memory latency x bytes in flight, not by arithmetic.
template <typename S>
struct HopRegs {
  typedef typename PT<S>::V V;
  static constexpr int RPC = PT<S>::RPC;
  static constexpr int NPSI = 24 / RPC;
  V psi[NPSI];
  static constexpr int NWC = RPC == 2 ? 9 : RPC == 4 ? 5 : 3;
  V w[NWC];      // chunks covering the 18 reals of one link
  float scale;   // fp16 block-float scale of the neighbour spinor
};
template <int MU, typename S> struct LinkChunks {
  static constexpr int RPC = PT<S>::RPC;
  static constexpr int C0 = (18 * MU) / RPC, C1 = (18 * MU + 17) / RPC, N = C1 - C0 + 1, OFF = 18 * MU - C0 * RPC;
};
template <typename S, int MU, int DIR>
__device__ __forceinline__ void hop_issue(const DslashArgs& a, const Site& s, int cb, int parity, HopRegs<S>& d) {
  typedef typename PT<S>::V V;
  typedef LinkChunks<MU, S> LC;
  const int Vh = a.g.Vh;
  const int nb = neighbour_cb<MU, DIR>(a.g, s);
  const V* p = reinterpret_cast<const V*>(a.in[1 - parity].data);
#pragma unroll
  for (int c = 0; c < HopRegs<S>::NPSI; c++) d.psi[c] = ldg_pinned(p + size_t(c) * Vh + nb);
  if (PT<S>::ID == 2) d.scale = ldg_pinned(a.in[1 - parity].scale + nb);
  // forward: W_mu(x) of the own parity; backward: W_mu(x-mu) of the other parity at the neighbour
  const V* w = reinterpret_cast<const V*>(DIR > 0 ? a.W[parity] : a.W[1 - parity]);
  const int wi = DIR > 0 ? cb : nb;
#pragma unroll
  for (int c = 0; c < LC::N; c++) d.w[c] = ldg_pinned(w + size_t(LC::C0 + c) * Vh + wi);
}
template <typename S, int MU, int DIR, bool G5IN>
__device__ __forceinline__ void hop_use(const HopRegs<S>& d, typename PT<S>::C* acc) {
  typedef typename PT<S>::C C;
  typedef LinkChunks<MU, S> LC;
  constexpr int RPC = PT<S>::RPC;
  C psi[24], h[12], wv[HopRegs<S>::NWC * RPC], r[12];
#pragma unroll
  for (int c = 0; c < HopRegs<S>::NPSI; c++) unpack_vec(d.psi[c], psi + c * RPC);
  if (PT<S>::ID == 2) {
#pragma unroll
    for (int i = 0; i < 24; i++) psi[i] *= d.scale;
  }
  if (G5IN) {
#pragma unroll
    for (int i = 12; i < 24; i++) psi[i] = -psi[i];
  }
  project<MU, DIR>(psi, h);
#pragma unroll
  for (int c = 0; c < LC::N; c++) unpack_vec(d.w[c], wv + c * RPC);
  link_mul<(DIR < 0)>(wv + LC::OFF, h, r);
  reconstruct<MU, DIR>(r, acc);
}
// all eight hops, two in flight
template <typename S, bool G5IN>
__device__ __forceinline__ void hop_all(const DslashArgs& a, const Site& s, int cb, int parity, typename PT<S>::C* acc) {
  HopRegs<S> d0, d1;
  hop_issue<S, 0, +1>(a, s, cb, parity, d0);
  hop_issue<S, 0, -1>(a, s, cb, parity, d1);
  hop_use<S, 0, +1, G5IN>(d0, acc);
  hop_issue<S, 1, +1>(a, s, cb, parity, d0);
  hop_use<S, 0, -1, G5IN>(d1, acc);
  hop_issue<S, 1, -1>(a, s, cb, parity, d1);
  hop_use<S, 1, +1, G5IN>(d0, acc);
  hop_issue<S, 2, +1>(a, s, cb, parity, d0);
  hop_use<S, 1, -1, G5IN>(d1, acc);
  hop_issue<S, 2, -1>(a, s, cb, parity, d1);
  hop_use<S, 2, +1, G5IN>(d0, acc);
  hop_issue<S, 3, +1>(a, s, cb, parity, d0);
  hop_use<S, 2, -1, G5IN>(d1, acc);
  hop_issue<S, 3, -1>(a, s, cb, parity, d1);
  hop_use<S, 3, +1, G5IN>(d0, acc);
  hop_use<S, 3, -1, G5IN>(d1, acc);
}

// Bulk L2 prefetch (cp.async.bulk.prefetch.L2, sm_90+): the compulsory DRAM streams of a CTA -- its own links, its
// clover blocks and its own spinors -- are contiguous 16 B x 128-site rows of the chunk-major SoA records.  One thread per
// row asks the L2 for the whole row when the CTA starts, so the per-thread 16-byte loads that follow (one hop after the
// other, bounded by registers) find their lines in L2 or already in flight instead of paying one DRAM latency per hop.
__device__ __forceinline__ void bulk_prefetch_l2(const void* p, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
template <typename S, int PHI, bool FULL>
__device__ __forceinline__ void cta_prefetch(const DslashArgs& a, int cb0) {
  constexpr int NW = 72 / PT<S>::RPC, NS = 24 / PT<S>::RPC;   // rows per parity: links, clover (NW each), spinor (NS)
  const int Vh = a.g.Vh;
  const int n = min(128, Vh - cb0);
  if (n <= 0) return;
  const unsigned bytes = unsigned(n) * 16u;
  const int t = threadIdx.x;
  if (FULL) {
    // rows: [parity][W NW | CL NW | psi NS]
    constexpr int PER = 2 * NW + NS;
    if (t < 2 * PER) {
      const int p = t / PER, r = t % PER;
      const char* base = r < NW ? (const char*)a.W[p] : r < 2 * NW ? (const char*)a.CL[p] : (const char*)a.in[p].data;
      const int c = r < NW ? r : r < 2 * NW ? r - NW : r - 2 * NW;
      bulk_prefetch_l2(base + (size_t(c) * Vh + cb0) * 16, bytes);
    }
  } else {
    // own forward links, clover (or inverse) block, phi
    constexpr int PER = 2 * NW + (PHI ? NS : 0);
    if (t < PER) {
      const int p = a.parity_out;
      const char* base = t < NW ? (const char*)a.W[p] : t < 2 * NW ? (const char*)a.CL[p] : (const char*)a.phi.data;
      const int c = t < NW ? t : t < 2 * NW ? t - NW : t - 2 * NW;
      bulk_prefetch_l2(base + (size_t(c) * Vh + cb0) * 16, bytes);
    }
  }
}

// PHI: 0 none, 1 phi, 2 M*phi (FULL: phi = in on the own parity).  POST: 1 = multiply the result by M^{-1}.
// Full-lattice launches (row a4) put both parities of 128 consecutive checkerboard indices -- one 4x4x4x4 tile with
// the default order -- into one CTA of 256 threads (warps 0-3 even, 4-7 odd): every link is then used twice by the same
// CTA (forward hop of x, backward hop of x+mu) and 3/4 of the neighbour spinors belong to the CTA's own tile.
template <typename S, int PHI, int POST, bool NEG, int FLAGS, bool FULL>
__global__ void __launch_bounds__(FULL ? 256 : 128, sizeof(S) == 8 ? 1 : (FULL ? 2 : 4)) dslash_k(const __grid_constant__ DslashArgs a) {
  typedef typename PT<S>::C C;
  const int Vh = a.g.Vh;
  const int cb = blockIdx.x * 128 + (threadIdx.x & 127);
  const int parity = FULL ? (threadIdx.x >> 7) : a.parity_out;
  if (a.prefetch) cta_prefetch<S, PHI, FULL>(a, blockIdx.x * 128);
  double nrm[1] = {0.0};
  if (cb < Vh) {
    Site s;
    site_init(a.g, cb, parity, s);
    C acc[24];
#pragma unroll
    for (int i = 0; i < 24; i++) acc[i] = 0;
    hop_all<S, (FLAGS & DSF_G5IN) != 0>(a, s, cb, parity, acc);
    const C hs = NEG ? (C)0.5 : (C)-0.5;  // +-hop = -+1/2 acc
#pragma unroll
    for (int i = 0; i < 24; i++) acc[i] *= ((FLAGS & DSF_G5HOP) && i >= 12) ? -hs : hs;
    if (PHI != 0) {
      C phi[24];
      load_spinor<S>(FULL ? a.in[parity] : a.phi, Vh, cb, phi);
      if (PHI == 2) {
        C mphi[24];
        clover_mul<S>(a.CL[parity], Vh, cb, phi, mphi);
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] += mphi[i];
      } else {
#pragma unroll
        for (int i = 0; i < 24; i++) acc[i] += phi[i];
      }
    }
    if (POST) {
      C t[24];
      clover_mul<S>(a.CL[parity], Vh, cb, acc, t);
#pragma unroll
      for (int i = 0; i < 24; i++) acc[i] = t[i];
    }
    if (FLAGS & DSF_NORM) {
#pragma unroll
      for (int i = 0; i < 24; i++) nrm[0] += (double)acc[i] * (double)acc[i];
    }
    store_spinor<S>(a.out[parity], Vh, cb, acc);
  }
  if (FLAGS & DSF_NORM) grid_reduce<1>(nrm, a.R);
}

template <typename S, int INV_DUMMY>
__global__ void __launch_bounds__(128) clover_apply_k(int Vh, const void* CL, SpinorPtr in, SpinorPtr out) {
  typedef typename PT<S>::C C;
  const int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  C v[24], w[24];
  load_spinor<S>(in, Vh, cb, v);
  clover_mul<S>(CL, Vh, cb, v, w);
  store_spinor<S>(out, Vh, cb, w);
}

template <typename S, int PHI, int POST, bool NEG, int FLAGS, bool FULL>
void launch_one(qxd_ctx* c, const DslashArgs& a) {
  dim3 gr((c->g.Vh + 127) / 128);
  dslash_k<S, PHI, POST, NEG, FLAGS, FULL><<<gr, FULL ? 256 : 128, 0, c->stream>>>(a);
}

template <typename S>
int dispatch(qxd_ctx* c, const DslashCall& d, const DslashArgs& a) {
  const int f = d.flags;
  switch (d.mode) {
    case DS_DW_FULL:
      if (f != 0) break;
      launch_one<S, 2, 0, false, 0, true>(c, a); return QXD_OK;
    case DS_HOP_AINV:
      if (f == 0) { launch_one<S, 0, 1, false, 0, false>(c, a); return QXD_OK; }
      if (f == DSF_G5IN) { launch_one<S, 0, 1, false, DSF_G5IN, false>(c, a); return QXD_OK; }
      break;
    case DS_A_XMHOP:
      if (f == 0) { launch_one<S, 2, 0, true, 0, false>(c, a); return QXD_OK; }
      if (f == DSF_NORM) { launch_one<S, 2, 0, true, DSF_NORM, false>(c, a); return QXD_OK; }
      if (f == DSF_G5HOP) { launch_one<S, 2, 0, true, DSF_G5HOP, false>(c, a); return QXD_OK; }
      if (f == (DSF_G5HOP | DSF_NORM)) { launch_one<S, 2, 0, true, DSF_G5HOP | DSF_NORM, false>(c, a); return QXD_OK; }
      break;
    case DS_X_MHOP:
      if (f == 0) { launch_one<S, 1, 0, true, 0, false>(c, a); return QXD_OK; }
      break;
    case DS_AINV_X_MHOP:
      if (f == 0) { launch_one<S, 1, 1, true, 0, false>(c, a); return QXD_OK; }
      break;
    default: break;
  }
  return fail(c, QXD_EINVAL, "dslash: unsupported mode/flags combination");
}

}  // namespace

int launch_dslash(qxd_ctx* c, const DslashCall& d) {
  if (d.prec < 0 || d.prec >= NPREC || !((c->prec_mask >> d.prec) & 1)) return fail(c, QXD_EINVAL, "dslash: precision not bound");
  DslashArgs a;
  a.g = c->g;
  a.in[0] = d.in[0]; a.in[1] = d.in[1];
  a.phi = d.phi;
  a.out[0] = d.out[0]; a.out[1] = d.out[1];
  a.W[0] = c->W[d.prec][0]; a.W[1] = c->W[d.prec][1];
  const bool inv = (d.mode == DS_HOP_AINV || d.mode == DS_AINV_X_MHOP);
  a.CL[0] = inv ? c->Mi[d.prec][0] : c->M[d.prec][0];
  a.CL[1] = inv ? c->Mi[d.prec][1] : c->M[d.prec][1];
  a.parity_out = d.parity_out;
  { static const int pf = getenv("QXD_PREFETCH") ? atoi(getenv("QXD_PREFETCH")) : 0; a.prefetch = pf; }
  a.R.partials = c->partials; a.R.ticket = c->ticket; a.R.result = d.norm_result;
  int rc = d.prec == 0 ? dispatch<double>(c, d, a) : d.prec == 1 ? dispatch<float>(c, d, a) : dispatch<__half>(c, d, a);
  if (rc) return rc;
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

int launch_clover_apply(qxd_ctx* c, int prec, int inverse, int parity, const SpinorPtr& in, const SpinorPtr& out) {
  const void* CL = inverse ? c->Mi[prec][parity] : c->M[prec][parity];
  dim3 gr((c->g.Vh + 127) / 128);
  if (prec == 0) clover_apply_k<double, 0><<<gr, 128, 0, c->stream>>>(c->g.Vh, CL, in, out);
  else if (prec == 1) clover_apply_k<float, 0><<<gr, 128, 0, c->stream>>>(c->g.Vh, CL, in, out);
  else clover_apply_k<__half, 0><<<gr, 128, 0, c->stream>>>(c->g.Vh, CL, in, out);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // namespace qxd
