// dslash_ilv.cu -- EXPERIMENT for SURVEY.md §8 row a10 (multi-RHS batched D_w): right-hand sides ACROSS LANES.
//
// The batched kernel of dslash_kernel.cuh gives every right-hand side of a tile its own CTA: each warp reads its links and clover
// blocks with 32 different 16-byte addresses (4 wavefronts of the 128 B/clk L1 path per instruction), and the out-of-tile
// neighbour spinors of the z faces use half of every 32-byte sector.  Here four right-hand sides are interleaved in memory,
//     chunk c of site cb of right-hand side j of a group  at vector index  (c Vh + cb) 4 + j
// (a group of four spinors IS a packed spinor of a lattice with 4 Vh sites per parity), and a warp works on 8 sites x 4
// right-hand sides: the four lanes of a site read the same link / clover words (one 128-byte wavefront per warp instruction
// instead of four), every spinor access of a warp is 8 runs of 64 contiguous bytes, and a neighbour site always contributes
// a full 64-byte run.  One thread still applies the operator of one site to one right-hand side (hop_use and
// clover_mul_multi are those of the tile kernel: identical arithmetic, identical results).  Full-lattice D_w only.
#include "dslash_kernel.cuh"

namespace qxd {

namespace {

constexpr int ILV = 4, ILV_SH = 2;

struct IlvArgs {
  Geom g;
  const char* in;        // groups of ILV interleaved right-hand sides, `rs` bytes apart; parity halves as in a packed spinor with ILV Vh sites
  char* out;
  const void* W[2];
  const void* CL[2];
  size_t rs;
  int ngroups;
};

template <typename S, int MU, int DIR, int NL, bool PAIR>
__device__ __forceinline__ void ilv_issue(const IlvArgs& a, const SpinorPtr (&in)[2], const Site& s, int cb, int parity, int j, HopRegs<S, 1, NL>& d) {
  typedef typename PT<S>::V V;
  typedef LinkChunks<MU, S, NL> LC;
  const int Vh = a.g.Vh, Vs = Vh << ILV_SH;
  const int nb = neighbour_cb<MU, DIR, PAIR ? 1 : 0>(a.g, s);
  const int nbs = (nb << ILV_SH) | j;
  const V* p = reinterpret_cast<const V*>(in[1 - parity].data);
#pragma unroll
  for (int c = 0; c < HopRegs<S, 1, NL>::NPSI; c++) d.psi[0][c] = ldg_pinned(p + size_t(c) * Vs + nbs);
  d.scale[0] = 1.f;
  if (PT<S>::ID == 2) d.scale[0] = ldg_pinned(in[1 - parity].scale + nbs);
  const V* w = reinterpret_cast<const V*>(DIR > 0 ? a.W[parity] : a.W[1 - parity]);
  int wi = DIR > 0 ? cb : nb;
  d.wsgn = 1.f;
  if (PAIR) { d.wsgn = (wi & 1) ? -1.f : 1.f; wi >>= 1; }
  const int Vw = PAIR ? a.g.Vg : Vh;
#pragma unroll
  for (int c = 0; c < LC::N; c++) d.w[c] = ldg_pinned(w + size_t(LC::C0 + c) * Vw + wi);
}

template <typename S, int NL, bool PAIR>
__global__ void __launch_bounds__(256, sizeof(S) == 8 ? 1 : 2) dw_ilv_k(const __grid_constant__ IlvArgs a) {
  typedef typename PT<S>::C C;
  const int Vh = a.g.Vh, Vs = Vh << ILV_SH;
  const int bt = blockIdx.x / a.ngroups, grp = blockIdx.x - bt * a.ngroups;     // groups fastest: a tile's links stay in L2 / L1
  const int parity = threadIdx.x >> 7;
  const int cb = bt * 32 + ((threadIdx.x >> ILV_SH) & 31);
  const int j = threadIdx.x & (ILV - 1);
  if (cb >= Vh) return;
  const int cbs = (cb << ILV_SH) | j;
  SpinorPtr in[2], out;
  {
    char* bi = const_cast<char*>(a.in) + a.rs * grp;
    in[0] = spinor_view<S>(bi, Vs, 0); in[1] = spinor_view<S>(bi, Vs, 1);
    out = spinor_view<S>(a.out + a.rs * grp, Vs, parity);
  }
  Site s;
  site_init<PAIR ? 1 : 0>(a.g, cb, parity, s);
  C acc[1][24];
#pragma unroll
  for (int i = 0; i < 24; i++) acc[0][i] = 0;
  {
    HopRegs<S, 1, NL> d0, d1;
    ilv_issue<S, 0, +1, NL, PAIR>(a, in, s, cb, parity, j, d0);
    ilv_issue<S, 0, -1, NL, PAIR>(a, in, s, cb, parity, j, d1);
    hop_use<S, 0, +1, false, 1, NL, PAIR>(d0, acc);
    ilv_issue<S, 1, +1, NL, PAIR>(a, in, s, cb, parity, j, d0);
    hop_use<S, 0, -1, false, 1, NL, PAIR>(d1, acc);
    ilv_issue<S, 1, -1, NL, PAIR>(a, in, s, cb, parity, j, d1);
    hop_use<S, 1, +1, false, 1, NL, PAIR>(d0, acc);
    ilv_issue<S, 2, +1, NL, PAIR>(a, in, s, cb, parity, j, d0);
    hop_use<S, 1, -1, false, 1, NL, PAIR>(d1, acc);
    ilv_issue<S, 2, -1, NL, PAIR>(a, in, s, cb, parity, j, d1);
    hop_use<S, 2, +1, false, 1, NL, PAIR>(d0, acc);
    ilv_issue<S, 3, +1, NL, PAIR>(a, in, s, cb, parity, j, d0);
    hop_use<S, 2, -1, false, 1, NL, PAIR>(d1, acc);
    ilv_issue<S, 3, -1, NL, PAIR>(a, in, s, cb, parity, j, d1);
    hop_use<S, 3, +1, false, 1, NL, PAIR>(d0, acc);
    hop_use<S, 3, -1, false, 1, NL, PAIR>(d1, acc);
  }
#pragma unroll
  for (int i = 0; i < 24; i++) acc[0][i] *= (C)-0.5;
  C phi[1][24], mphi[1][24];
  load_spinor<S>(in[parity], Vs, cbs, phi[0]);
  clover_mul_multi<S, 1, PAIR>(a.CL[parity], a.g, cb, phi, mphi);
#pragma unroll
  for (int i = 0; i < 24; i++) acc[0][i] += mphi[0][i];
  store_spinor<S>(out, Vs, cbs, acc[0]);
}

// raw copy between nrhs plain packed spinors (back to back) and nrhs / ILV interleaved groups, both parities
template <typename S>
__global__ void __launch_bounds__(128) ilv_convert_k(int Vh, int nrhs, char* plain, char* ilv, int to_ilv) {
  typedef typename PT<S>::V V;
  constexpr int NCH = 24 / PT<S>::RPC;
  const int cb = blockIdx.x * blockDim.x + threadIdx.x;
  const int k = blockIdx.y, parity = blockIdx.z;
  if (cb >= Vh) return;
  const int Vs = Vh << ILV_SH;
  const SpinorPtr p = spinor_view<S>(plain + size_t(k) * 2 * spinor_half_bytes<S>(Vh), Vh, parity);
  const SpinorPtr q = spinor_view<S>(ilv + size_t(k >> ILV_SH) * 2 * spinor_half_bytes<S>(Vs), Vs, parity);
  const int cbs = (cb << ILV_SH) | (k & (ILV - 1));
  V* pv = reinterpret_cast<V*>(p.data);
  V* qv = reinterpret_cast<V*>(q.data);
#pragma unroll
  for (int c = 0; c < NCH; c++) {
    if (to_ilv) qv[size_t(c) * Vs + cbs] = pv[size_t(c) * Vh + cb]; else pv[size_t(c) * Vh + cb] = qv[size_t(c) * Vs + cbs];
  }
  if (PT<S>::ID == 2) { if (to_ilv) q.scale[cbs] = p.scale[cb]; else p.scale[cb] = q.scale[cbs]; }
}

template <typename S, int NL, bool PAIR>
void ilv_launch(qxd_ctx* c, const IlvArgs& a) {
  const unsigned nt = unsigned((c->g.Vh + 31) / 32);
  dw_ilv_k<S, NL, PAIR><<<nt * unsigned(a.ngroups), 256, 0, c->stream>>>(a);
}

}  // namespace

int launch_dw_ilv(qxd_ctx* c, int prec, int nrhs, const void* in, void* out) {
  if (nrhs < ILV || nrhs % ILV) return fail(c, QXD_EINVAL, "apply_Dw_multi_interleaved: nrhs must be a multiple of 4");
  IlvArgs a;
  a.g = c->g; a.in = static_cast<const char*>(in); a.out = static_cast<char*>(out);
  for (int p = 0; p < 2; p++) { a.W[p] = c->W[prec][p]; a.CL[p] = c->M[prec][p]; }
  a.rs = 2 * half_bytes(prec, c->g.Vh << ILV_SH);
  a.ngroups = nrhs / ILV;
  const bool l14 = c->link_reals[prec] == 14, pr = c->g.pair != 0;
#define QXD_ILV(S) do { if (l14) { if (pr) ilv_launch<S, 14, true>(c, a); else ilv_launch<S, 14, false>(c, a); } \
                        else { if (pr) ilv_launch<S, 18, true>(c, a); else ilv_launch<S, 18, false>(c, a); } } while (0)
  if (prec == 0) QXD_ILV(double); else if (prec == 1) QXD_ILV(float); else QXD_ILV(__half);
#undef QXD_ILV
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

int launch_ilv_convert(qxd_ctx* c, int prec, int nrhs, void* plain, void* ilv, int to_ilv) {
  if (nrhs < ILV || nrhs % ILV) return fail(c, QXD_EINVAL, "multi_interleave: nrhs must be a multiple of 4");
  dim3 gr((c->g.Vh + 127) / 128, nrhs, 2);
  if (prec == 0) ilv_convert_k<double><<<gr, 128, 0, c->stream>>>(c->g.Vh, nrhs, (char*)plain, (char*)ilv, to_ilv);
  else if (prec == 1) ilv_convert_k<float><<<gr, 128, 0, c->stream>>>(c->g.Vh, nrhs, (char*)plain, (char*)ilv, to_ilv);
  else ilv_convert_k<__half><<<gr, 128, 0, c->stream>>>(c->g.Vh, nrhs, (char*)plain, (char*)ilv, to_ilv);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // namespace qxd
