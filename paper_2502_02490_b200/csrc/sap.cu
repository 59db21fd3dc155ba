// sap.cu -- SURVEY.md §8(f) row f3, the preconditioner: the Schwarz alternating procedure (SAP) named by the paper as the
// preconditioner of its CPU solver ("heavily preconditioned GCR ... Schwarz alternating procedure"), re-designed
// for the B200: a block is the 256 sites of one 128-index tile (both parities) and is solved by ONE thread block that keeps
// everything the block solve touches in shared memory -- the block residual (fp32, 24 KB) and the hopping links and clover
// blocks of the block (storage precision S: 36 + 36 KB in binary16, 72 + 72 KB in fp32) -- so that the nmr minimal-residual
// steps on the Dirichlet block operator D_Lambda = P_Lambda D_w P_Lambda run without touching L2 or HBM.
//
//   M_sap:  psi = 0, r = in;  for cy < ncy, for colour in (0, 1):  on every block Lambda of that colour
//              e = MR_nmr(D_Lambda, r|Lambda);   psi|Lambda += e;   r -= D_w e
// The update of r outside the block is done lazily: the kernel writes the in-block part (the MR residual) and the correction
// e; when a neighbouring block (of the other colour) is visited next, its prologue subtracts the hopping terms of the stored
// corrections across the block boundary.  With a proper two-colouring every correction is applied exactly once.
#include "dslash_kernel.cuh"

namespace qxd {

namespace {

struct SapArgs {
  Geom g;
  const void* W[2];       // hopping links W = e^{iqA} U of the sloppy precision S, NL stored reals per link
  const void* CL[2];      // clover blocks M (72 reals) of precision S
  const float4* src[2];   // residual the block solves start from: the preconditioner's input in cycle 0, `res` afterwards
  float4* res[2];         // block residuals (in-block part kept up to date)
  float4* corr[2];        // latest correction e of every site
  float4* psi[2];         // accumulated output
  int colour, prologue, init_psi, nmr;
  int boxsh[4];           // log2 of the block extents on the indexed lattice
  int colmask[4];         // 1 if the direction has more than one block (contributes to the colour)
};

__device__ __forceinline__ int colour_of(const SapArgs& a, const Site& s) {
  return ((a.colmask[0] ? (s.x[0] >> a.boxsh[0]) : 0) + (a.colmask[1] ? (s.x[1] >> a.boxsh[1]) : 0) +
          (a.colmask[2] ? (s.x[2] >> a.boxsh[2]) : 0) + (a.colmask[3] ? (s.x[3] >> a.boxsh[3]) : 0)) & 1;
}

// reals [R0, R0+N) of the record of local site l from a shared-memory array laid out [chunk][128]
template <typename S, int R0, int N>
__device__ __forceinline__ void lds_reals(const typename PT<S>::V* base, int l, float* out) {
  typedef typename PT<S>::V V;
  constexpr int RPC = PT<S>::RPC;
  constexpr int C0 = R0 / RPC, C1 = (R0 + N - 1) / RPC;
#pragma unroll
  for (int c = C0; c <= C1; c++) {
    const V v = base[c * 128 + l];
    float tmp[RPC];
    unpack_vec(v, tmp);
#pragma unroll
    for (int k = 0; k < RPC; k++) {
      const int r = c * RPC + k;
      if (r >= R0 && r < R0 + N) out[r - R0] = tmp[k];
    }
  }
}
__device__ __forceinline__ void unpack4(const float4& v, float* o) { o[0] = v.x; o[1] = v.y; o[2] = v.z; o[3] = v.w; }

template <typename S> struct SapShape {
  static constexpr int RPC = PT<S>::RPC;
  static constexpr int NCH = 72 / RPC;                       // chunks of a 72-real record (links of a site; clover blocks)
  static constexpr size_t RHO = size_t(2) * 6 * 128 * 16;    // fp32 block residual
  static constexpr size_t REC = size_t(2) * NCH * 128 * 16;  // one 72-real record per site of the block
  static constexpr size_t BYTES = RHO + 2 * REC;
  static constexpr int MINB = sizeof(S) == 2 ? 2 : 1;
};

// in-block hop from shared memory: acc += (1 -+ gamma_mu) W psi(x +- mu) for a neighbour inside the block, nothing otherwise
template <typename S, int MU, int DIR, bool PAIR>
__device__ __forceinline__ void hop_sm(const unsigned (&nbc)[2], int par, int l, const float4* rho,
                                       const typename PT<S>::V* Wsm, float* acc) {
  constexpr int D = 2 * MU + (DIR < 0 ? 1 : 0);
  const unsigned code = (nbc[D >> 2] >> (8 * (D & 3))) & 0xffu;   // bit 7: neighbour inside the block, bits 0-6: its local index
  if (!(code & 0x80u)) return;
  const int ln = code & 0x7f;
  float psi[24], w[18], h[12], t[12];
#pragma unroll
  for (int c = 0; c < 6; c++) unpack4(rho[((1 - par) * 6 + c) * 128 + ln], psi + 4 * c);
  if (DIR > 0) lds_reals<S, 18 * MU, 18>(Wsm + par * SapShape<S>::NCH * 128, l, w);
  else lds_reals<S, 18 * MU, 18>(Wsm + (1 - par) * SapShape<S>::NCH * 128, ln, w);
  project<MU, DIR>(psi, h);
  // packed fp32 FMAs (FFMA2) where the register budget allows (fp32 storage: one CTA per SM, 255 registers; measured at c3:
  // 9.8 -> 9.3 ms per M_sap); with binary16 storage (two CTAs per SM, 128 registers) the operand pairing spills: 6.4 -> 6.9 ms
  if constexpr (sizeof(S) == 4) { link_mul_x2<(DIR < 0)>(w, h, t); reconstruct_x2<MU, DIR, false>(t, acc, 1.0f); }
  else { link_mul<(DIR < 0)>(w, h, t); reconstruct<MU, DIR, false>(t, acc, 1.0f); }
}
// hop across the block boundary, from the stored corrections in global memory (prologue)
template <typename S, int MU, int DIR, int NL, bool PAIR>
__device__ __forceinline__ void hop_bnd(const SapArgs& a, const float4* __restrict__ nsrc, const Site& s, int tile, int par, int l,
                                        const typename PT<S>::V* Wsm, float* acc, int chmask = 0 /* 1 / 2: upper / lower chirality of the source only */) {
  const int nb = neighbour_cb<MU, DIR, PAIR ? 1 : 0>(a.g, s);
  if ((nb >> 7) == tile) return;
  const int Vh = a.g.Vh;
  float psi[24], w[18], h[12], t[12];
#pragma unroll
  for (int c = 0; c < 6; c++) unpack4(__ldg(nsrc + size_t(c) * Vh + nb), psi + 4 * c);
  if (chmask) {
#pragma unroll
    for (int k = 0; k < 12; k++) psi[(chmask == 1 ? 12 : 0) + k] = 0.f;
  }
  if (DIR > 0) lds_reals<S, 18 * MU, 18>(Wsm + par * SapShape<S>::NCH * 128, l, w);
  else {   // W_mu(x - mu): the forward link of the neighbour, from its global record
    int wi = nb;
    float sgn = 1.f;
    if (PAIR) { sgn = (wi & 1) ? -1.f : 1.f; wi >>= 1; }
    float wv[NL];
    load_reals<S, NL * MU, NL>(a.W[1 - par], PAIR ? a.g.Vg : Vh, wi, wv);
    if (PAIR) {
#pragma unroll
      for (int i = 1; i < NL; i += 2) wv[i] *= sgn;
    }
    if (NL == 14) reconstruct_row2(wv, w);
    else {
#pragma unroll
      for (int i = 0; i < 18; i++) w[i] = wv[i];
    }
  }
  project<MU, DIR>(psi, h);
  link_mul<(DIR < 0)>(w, h, t);
  reconstruct<MU, DIR, false>(t, acc, 1.0f);
}

template <typename S, int NL, bool PAIR, int MU>
__device__ __forceinline__ void stage_link(const SapArgs& a, int par, int Vs, int rec, bool mir, float* w72) {
  float wv[NL];
  load_reals<S, NL * MU, NL>(a.W[par], Vs, rec, wv);
  if (PAIR) {
#pragma unroll
    for (int i = 1; i < NL; i += 2) wv[i] = mir ? -wv[i] : wv[i];
  }
  if (NL == 14) reconstruct_row2(wv, w72 + 18 * MU);
  else {
#pragma unroll
    for (int i = 0; i < 18; i++) w72[18 * MU + i] = wv[i];
  }
}
// stage the four forward links of the thread's own site as 72 reals (18 per link; conjugated for a C* mirror site, row 2
// rebuilt from the 14-real format) and its clover record into shared memory
template <typename S, int NL, bool PAIR>
__device__ __forceinline__ void stage_site(const SapArgs& a, int cb, int par, int l, typename PT<S>::V* Wsm, typename PT<S>::V* Csm) {
  typedef typename PT<S>::V V;
  constexpr int RPC = PT<S>::RPC, NCH = SapShape<S>::NCH;
  const int rec = PAIR ? (cb >> 1) : cb;
  const int Vs = PAIR ? a.g.Vg : a.g.Vh;
  const bool mir = PAIR && (cb & 1);
  V* wdst = Wsm + par * NCH * 128 + l;
  if (NL == 18 && !PAIR) {
    const V* wsrc = reinterpret_cast<const V*>(a.W[par]);
#pragma unroll
    for (int c = 0; c < NCH; c++) wdst[c * 128] = __ldg(wsrc + size_t(c) * Vs + rec);
  } else {
    float w72[72];
    stage_link<S, NL, PAIR, 0>(a, par, Vs, rec, mir, w72); stage_link<S, NL, PAIR, 1>(a, par, Vs, rec, mir, w72);
    stage_link<S, NL, PAIR, 2>(a, par, Vs, rec, mir, w72); stage_link<S, NL, PAIR, 3>(a, par, Vs, rec, mir, w72);
#pragma unroll
    for (int c = 0; c < NCH; c++) wdst[c * 128] = pack_vec(w72 + c * RPC, (V*)nullptr);
  }
  const V* csrc = reinterpret_cast<const V*>(a.CL[par]);
  V* cdst = Csm + par * NCH * 128 + l;
#pragma unroll
  for (int c = 0; c < NCH; c++) cdst[c * 128] = __ldg(csrc + size_t(c) * Vs + rec);
}

// t = D_Lambda rho at the thread's site, all operands from shared memory
template <typename S, bool PAIR>
__device__ __forceinline__ void block_apply(const unsigned (&nbc)[2], int cb, int par, int l, const float4* rho,
                                            const typename PT<S>::V* Wsm, const typename PT<S>::V* Csm, const float* own, float* t) {
  float acc[24];
#pragma unroll
  for (int i = 0; i < 24; i++) acc[i] = 0.f;
  hop_sm<S, 0, +1, PAIR>(nbc, par, l, rho, Wsm, acc);
  hop_sm<S, 0, -1, PAIR>(nbc, par, l, rho, Wsm, acc);
  hop_sm<S, 1, +1, PAIR>(nbc, par, l, rho, Wsm, acc);
  hop_sm<S, 1, -1, PAIR>(nbc, par, l, rho, Wsm, acc);
  hop_sm<S, 2, +1, PAIR>(nbc, par, l, rho, Wsm, acc);
  hop_sm<S, 2, -1, PAIR>(nbc, par, l, rho, Wsm, acc);
  hop_sm<S, 3, +1, PAIR>(nbc, par, l, rho, Wsm, acc);
  hop_sm<S, 3, -1, PAIR>(nbc, par, l, rho, Wsm, acc);
  const bool mir = PAIR && (cb & 1);
  const typename PT<S>::V* cl = Csm + par * SapShape<S>::NCH * 128;
#pragma unroll
  for (int blk = 0; blk < 2; blk++) {
    float b[36], v[12], w[12];
    if (blk == 0) lds_reals<S, 0, 36>(cl, l, b); else lds_reals<S, 36, 36>(cl, l, b);
    if (PAIR) mirror_in(own + 12 * blk, v, mir);
    else {
#pragma unroll
      for (int i = 0; i < 12; i++) v[i] = own[12 * blk + i];
    }
    if constexpr (sizeof(S) == 4) block_mul_x2(b, v, w); else block_mul(b, v, w);
    if (PAIR) mirror_out(w, t + 12 * blk, mir);
    else {
#pragma unroll
      for (int i = 0; i < 12; i++) t[12 * blk + i] = w[i];
    }
  }
#pragma unroll
  for (int i = 0; i < 24; i++) t[i] -= 0.5f * acc[i];
}

template <typename S, int NL, bool PAIR>
__global__ void __launch_bounds__(256, SapShape<S>::MINB) sap_mr_k(const __grid_constant__ SapArgs a) {
  typedef typename PT<S>::V V;
  extern __shared__ __align__(16) unsigned char smem[];
  float4* rho = reinterpret_cast<float4*>(smem);                                   // [2 parities][6 chunks][128]
  V* Wsm = reinterpret_cast<V*>(smem + SapShape<S>::RHO);                          // [2][NCH][128]
  V* Csm = reinterpret_cast<V*>(smem + SapShape<S>::RHO + SapShape<S>::REC);       // [2][NCH][128]
  __shared__ float red[8][3];
  const int l = threadIdx.x & 127, par = threadIdx.x >> 7, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int Vh = a.g.Vh;
  // tiles 2j and 2j+1 have opposite colours (checked on the host): this block takes the one of the requested colour
  int tile;
  {
    Site s0;
    site_init<PAIR ? 1 : 0>(a.g, 2 * blockIdx.x * 128, 0, s0);
    tile = 2 * blockIdx.x + (colour_of(a, s0) != a.colour ? 1 : 0);
  }
  const int cb = tile * 128 + l;
  stage_site<S, NL, PAIR>(a, cb, par, l, Wsm, Csm);
  Site s;
  site_init<PAIR ? 1 : 0>(a.g, cb, par, s);
  // the eight neighbours, once: inside the block (bit 7) and local index (the index arithmetic is not repeated per MR step)
  unsigned nbc[2];
  {
    const int n[8] = {neighbour_cb<0, +1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<0, -1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<1, +1, PAIR ? 1 : 0>(a.g, s),
                      neighbour_cb<1, -1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<2, +1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<2, -1, PAIR ? 1 : 0>(a.g, s),
                      neighbour_cb<3, +1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<3, -1, PAIR ? 1 : 0>(a.g, s)};
    nbc[0] = 0; nbc[1] = 0;
#pragma unroll
    for (int d = 0; d < 8; d++) nbc[d >> 2] |= ((((n[d] >> 7) == tile) ? 0x80u : 0u) | unsigned(n[d] & 127)) << (8 * (d & 3));
  }
  float r[24], e[24];
#pragma unroll
  for (int c = 0; c < 6; c++) unpack4(__ldg(a.src[par] + size_t(c) * Vh + cb), r + 4 * c);
  __syncthreads();
  if (a.prologue) {   // r -= (hopping terms of the neighbouring blocks' latest corrections) = r + 1/2 acc
    float acc[24];
#pragma unroll
    for (int i = 0; i < 24; i++) acc[i] = 0.f;
    hop_bnd<S, 0, +1, NL, PAIR>(a, a.corr[1 - par], s, tile, par, l, Wsm, acc);
    hop_bnd<S, 0, -1, NL, PAIR>(a, a.corr[1 - par], s, tile, par, l, Wsm, acc);
    hop_bnd<S, 1, +1, NL, PAIR>(a, a.corr[1 - par], s, tile, par, l, Wsm, acc);
    hop_bnd<S, 1, -1, NL, PAIR>(a, a.corr[1 - par], s, tile, par, l, Wsm, acc);
    hop_bnd<S, 2, +1, NL, PAIR>(a, a.corr[1 - par], s, tile, par, l, Wsm, acc);
    hop_bnd<S, 2, -1, NL, PAIR>(a, a.corr[1 - par], s, tile, par, l, Wsm, acc);
    hop_bnd<S, 3, +1, NL, PAIR>(a, a.corr[1 - par], s, tile, par, l, Wsm, acc);
    hop_bnd<S, 3, -1, NL, PAIR>(a, a.corr[1 - par], s, tile, par, l, Wsm, acc);
#pragma unroll
    for (int i = 0; i < 24; i++) r[i] += 0.5f * acc[i];
  }
#pragma unroll
  for (int c = 0; c < 6; c++) rho[(par * 6 + c) * 128 + l] = make_float4(r[4 * c], r[4 * c + 1], r[4 * c + 2], r[4 * c + 3]);
#pragma unroll
  for (int i = 0; i < 24; i++) e[i] = 0.f;
  __syncthreads();
  for (int it = 0; it < a.nmr; it++) {
    float t[24];
    block_apply<S, PAIR>(nbc, cb, par, l, rho, Wsm, Csm, r, t);
    // alpha = <t, r> / <t, t> over the block (minimal residual step)
    float p0 = 0.f, p1 = 0.f, p2 = 0.f;
#pragma unroll
    for (int k = 0; k < 12; k++) {
      p0 += t[2 * k] * r[2 * k]; p0 += t[2 * k + 1] * r[2 * k + 1];
      p1 += t[2 * k] * r[2 * k + 1]; p1 -= t[2 * k + 1] * r[2 * k];
      p2 += t[2 * k] * t[2 * k]; p2 += t[2 * k + 1] * t[2 * k + 1];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      p0 += __shfl_xor_sync(0xffffffffu, p0, o); p1 += __shfl_xor_sync(0xffffffffu, p1, o); p2 += __shfl_xor_sync(0xffffffffu, p2, o);
    }
    if (lane == 0) { red[warp][0] = p0; red[warp][1] = p1; red[warp][2] = p2; }
    __syncthreads();   // also: every thread has finished reading its neighbours' rho
    p0 = 0.f; p1 = 0.f; p2 = 0.f;
#pragma unroll
    for (int w = 0; w < 8; w++) { p0 += red[w][0]; p1 += red[w][1]; p2 += red[w][2]; }
    const float ar = p2 > 0.f ? p0 / p2 : 0.f, ai = p2 > 0.f ? p1 / p2 : 0.f;
#pragma unroll
    for (int k = 0; k < 12; k++) {
      e[2 * k] += ar * r[2 * k] - ai * r[2 * k + 1]; e[2 * k + 1] += ar * r[2 * k + 1] + ai * r[2 * k];
      r[2 * k] -= ar * t[2 * k] - ai * t[2 * k + 1]; r[2 * k + 1] -= ar * t[2 * k + 1] + ai * t[2 * k];
    }
#pragma unroll
    for (int c = 0; c < 6; c++) rho[(par * 6 + c) * 128 + l] = make_float4(r[4 * c], r[4 * c + 1], r[4 * c + 2], r[4 * c + 3]);
    __syncthreads();
  }
#pragma unroll
  for (int c = 0; c < 6; c++) {
    const size_t i = size_t(c) * Vh + cb;
    a.res[par][i] = make_float4(r[4 * c], r[4 * c + 1], r[4 * c + 2], r[4 * c + 3]);
    float4 ev = make_float4(e[4 * c], e[4 * c + 1], e[4 * c + 2], e[4 * c + 3]);
    a.corr[par][i] = ev;
    if (!a.init_psi) { const float4 o = a.psi[par][i]; ev.x += o.x; ev.y += o.y; ev.z += o.z; ev.w += o.w; }
    a.psi[par][i] = ev;
  }
}

template <typename S, int NL, bool PAIR>
int sap_launch_t(qxd_ctx* c, const SapArgs& a, int nblocks) {
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(sap_mr_k<S, NL, PAIR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SapShape<S>::BYTES);
    if (e != cudaSuccess) return fail(c, QXD_ECUDA, std::string("sap: cudaFuncSetAttribute: ") + cudaGetErrorString(e));
    configured = true;
  }
  sap_mr_k<S, NL, PAIR><<<nblocks, 256, SapShape<S>::BYTES, c->stream>>>(a);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

// ---- coarse (little) Dirac operator of the two-level preconditioner (dfl.cu): for every block b and null vector phi_i the nine
// block rows  A[b][0][j][i] = <phi_j, D_b phi_i>_b  (Dirichlet block operator) and  A[b][1+d][j][i] = <phi_j, H_d phi_i>_b  (the
// hops that leave the block in direction d = 2 mu + (dir < 0), reading phi_i on the neighbouring block), built with the block
// machinery of the Schwarz kernel: links and clover blocks of the block staged in shared memory, phi_i of the block in the ring
// slot of the residual.  One CTA per block, all blocks.  Also records the neighbour block of every direction.
struct CoarseArgs {
  SapArgs a;
  const float4* phi[32];   // null vectors: fp32 packed full lattice (parity 1 at +6 Vh float4)
  int ns;                  // null vectors
  int ch;                  // 1: every null vector is split into its two chirality components (coarse dimension nc = 2 ns, index 2 i + chi)
  float2* A;               // [nblocks][9][nc][nc]
  int* nbr;                // [nblocks][8], -1 where the block is its own neighbour in that direction
};
// sums of the 64 per-thread partials over the CTA -> dst[0..32) (float2).  Within a warp a transposing butterfly: at the step
// with lane offset o every lane keeps one half of its values and hands the other half to its partner (32 + 16 + 8 + 4 + 2
// shuffles instead of 64 x 5); lane l ends up with the warp sums of values 2 l and 2 l + 1.
__device__ __forceinline__ void coarse_reduce_store(float (&part)[64], float* red /*[8][64]*/, float2* dst, int warp, int lane) {
#pragma unroll
  for (int h = 32, o = 16; h >= 2; h >>= 1, o >>= 1) {
    const bool up = (lane & o) != 0;
#pragma unroll
    for (int k = 0; k < h; k++) {
      const float send = up ? part[k] : part[k + h];
      const float keep = up ? part[k + h] : part[k];
      part[k] = keep + __shfl_xor_sync(0xffffffffu, send, o);
    }
  }
  reinterpret_cast<float2*>(red)[warp * 32 + lane] = make_float2(part[0], part[1]);
  __syncthreads();
  if (threadIdx.x < 64) {
    float v = 0.f;
#pragma unroll
    for (int w = 0; w < 8; w++) v += red[w * 64 + threadIdx.x];
    reinterpret_cast<float*>(dst)[threadIdx.x] = v;
  }
  __syncthreads();
}
template <typename S, int NL, bool PAIR>
__global__ void __launch_bounds__(256, 1) coarse_build_k(const __grid_constant__ CoarseArgs ca) {
  typedef typename PT<S>::V V;
  const SapArgs& a = ca.a;
  extern __shared__ __align__(16) unsigned char smem[];
  float4* rho = reinterpret_cast<float4*>(smem);
  V* Wsm = reinterpret_cast<V*>(smem + SapShape<S>::RHO);
  V* Csm = reinterpret_cast<V*>(smem + SapShape<S>::RHO + SapShape<S>::REC);
  __shared__ float red[8 * 64];
  const int l = threadIdx.x & 127, par = threadIdx.x >> 7, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int Vh = a.g.Vh, ns = ca.ns;
  const int tile = blockIdx.x;
  const int cb = tile * 128 + l;
  stage_site<S, NL, PAIR>(a, cb, par, l, Wsm, Csm);
  Site s;
  site_init<PAIR ? 1 : 0>(a.g, cb, par, s);
  unsigned nbc[2];
  int nbt[8];
  {
    const int n[8] = {neighbour_cb<0, +1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<0, -1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<1, +1, PAIR ? 1 : 0>(a.g, s),
                      neighbour_cb<1, -1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<2, +1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<2, -1, PAIR ? 1 : 0>(a.g, s),
                      neighbour_cb<3, +1, PAIR ? 1 : 0>(a.g, s), neighbour_cb<3, -1, PAIR ? 1 : 0>(a.g, s)};
    nbc[0] = 0; nbc[1] = 0;
#pragma unroll
    for (int d = 0; d < 8; d++) {
      nbt[d] = n[d] >> 7;
      nbc[d >> 2] |= (((nbt[d] == tile) ? 0x80u : 0u) | unsigned(n[d] & 127)) << (8 * (d & 3));
      if (nbt[d] != tile) ca.nbr[tile * 8 + d] = nbt[d];      // every face thread writes the same value
    }
  }
  const size_t own = size_t(par) * 6 * Vh + cb;     // float4 index of chunk 0 of the own site in a packed full-lattice vector
  const int ch = ca.ch, nc = ch ? 2 * ns : ns;
  for (int ic = 0; ic < nc; ic++) {                 // column of the coarse operator: null vector i, chirality chi (ch) or all of it
    const int i = ch ? (ic >> 1) : ic, chm = ch ? 1 + (ic & 1) : 0;
    float r[24], y[24], part[64];
#pragma unroll
    for (int c = 0; c < 6; c++) {
      float4 v = __ldg(ca.phi[i] + own + size_t(c) * Vh);
      if ((chm == 1 && c >= 3) || (chm == 2 && c < 3)) v = make_float4(0.f, 0.f, 0.f, 0.f);
      rho[(par * 6 + c) * 128 + l] = v;
      unpack4(v, r + 4 * c);
    }
    __syncthreads();
    const float4* nsrc = ca.phi[i] + size_t(1 - par) * 6 * Vh;
#pragma unroll 1
    for (int d = 0; d < 9; d++) {
      if (d == 0) block_apply<S, PAIR>(nbc, cb, par, l, rho, Wsm, Csm, r, y);
      else {
#pragma unroll
        for (int k = 0; k < 24; k++) y[k] = 0.f;
        switch (d) {
          case 1: hop_bnd<S, 0, +1, NL, PAIR>(a, nsrc, s, tile, par, l, Wsm, y, chm); break;
          case 2: hop_bnd<S, 0, -1, NL, PAIR>(a, nsrc, s, tile, par, l, Wsm, y, chm); break;
          case 3: hop_bnd<S, 1, +1, NL, PAIR>(a, nsrc, s, tile, par, l, Wsm, y, chm); break;
          case 4: hop_bnd<S, 1, -1, NL, PAIR>(a, nsrc, s, tile, par, l, Wsm, y, chm); break;
          case 5: hop_bnd<S, 2, +1, NL, PAIR>(a, nsrc, s, tile, par, l, Wsm, y, chm); break;
          case 6: hop_bnd<S, 2, -1, NL, PAIR>(a, nsrc, s, tile, par, l, Wsm, y, chm); break;
          case 7: hop_bnd<S, 3, +1, NL, PAIR>(a, nsrc, s, tile, par, l, Wsm, y, chm); break;
          default: hop_bnd<S, 3, -1, NL, PAIR>(a, nsrc, s, tile, par, l, Wsm, y, chm); break;
        }
#pragma unroll
        for (int k = 0; k < 24; k++) y[k] *= -0.5f;          // H = -1/2 sum (1 -+ gamma) W psi
      }
      // <phi_j, y> at this site, upper and lower chirality apart.  Out-of-block hops: y = 0 except on the face of direction d
      bool act = true;
      if (d > 0) act = ((nbc[(d - 1) >> 2] >> (8 * ((d - 1) & 3))) & 0x80u) == 0;
#pragma unroll
      for (int k = 0; k < 64; k++) part[k] = 0.f;
#pragma unroll
      for (int j = 0; j < 32; j++) {
        if (j < ns && act) {
          float re[2] = {0.f, 0.f}, im[2] = {0.f, 0.f};
#pragma unroll
          for (int c = 0; c < 6; c++) {
            const float4 u = __ldg(ca.phi[j] + own + size_t(c) * Vh);
            const int h = c / 3;
            re[h] += u.x * y[4 * c]; re[h] += u.y * y[4 * c + 1]; re[h] += u.z * y[4 * c + 2]; re[h] += u.w * y[4 * c + 3];
            im[h] += u.x * y[4 * c + 1]; im[h] -= u.y * y[4 * c]; im[h] += u.z * y[4 * c + 3]; im[h] -= u.w * y[4 * c + 2];
          }
          if (ch) { if (j < 16) { part[4 * j] = re[0]; part[4 * j + 1] = im[0]; part[4 * j + 2] = re[1]; part[4 * j + 3] = im[1]; } }
          else { part[2 * j] = re[0] + re[1]; part[2 * j + 1] = im[0] + im[1]; }
        }
      }
      // A[b][d][row][ic]: the reduction delivers a column; store transposed
      __shared__ float2 col[32];
      coarse_reduce_store(part, red, col, warp, lane);
      if (threadIdx.x < nc) ca.A[((size_t(tile) * 9 + d) * nc + threadIdx.x) * nc + ic] = col[threadIdx.x];
      __syncthreads();
    }
  }
}
template <typename S, int NL, bool PAIR>
int coarse_build_t(qxd_ctx* c, const CoarseArgs& ca, int nblocks) {
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(coarse_build_k<S, NL, PAIR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SapShape<S>::BYTES);
    if (e != cudaSuccess) return fail(c, QXD_ECUDA, std::string("coarse_build: cudaFuncSetAttribute: ") + cudaGetErrorString(e));
    configured = true;
  }
  coarse_build_k<S, NL, PAIR><<<nblocks, 256, SapShape<S>::BYTES, c->stream>>>(ca);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // namespace

// The SAP blocks are the 128-index tiles the kernels work on anyway: a run of 256 (128 in the paired layout) consecutive full
// indices idx2, which is a box of the indexed lattice as long as it is made of in-tile and tile-in-block digits (powers of
// two).  A two-colouring needs an even number of boxes in every direction that has more than one, and tiles 2j, 2j+1 must
// have opposite colours (the kernel picks its tile that way).  Host-only; the result is cached in the context.
int sap_check_geometry(qxd_ctx* c) {
  if (c->sap_ok == 1) return QXD_OK;
  const Geom& g = c->g;
  const char* why = nullptr;
  if (g.Vh % 128 || (g.Vh / 128) % 2) why = "the number of 128-index tiles must be even";
  int boxsh[4] = {0, 0, 0, 0};
  if (!why) {
    int bits = g.pair ? 7 : 8;
    const int order[8] = {3, 2, 1, 0, 3, 2, 1, 0};
    for (int k = 0; k < 8 && bits > 0; k++) {
      const int mu = order[k];
      const int avail = k < 4 ? g.sh[mu] : g.shB[mu] - g.sh[mu];
      const int take = bits < avail ? bits : avail;
      boxsh[mu] += take; bits -= take;
    }
    if (bits > 0) why = "a 128-index tile spans several blocks of the site order";
  }
  int colmask[4] = {0, 0, 0, 0};
  for (int mu = 0; mu < 4 && !why; mu++) {
    const int nb = g.X[mu] >> boxsh[mu];
    if (nb > 1) {
      colmask[mu] = 1;
      if (nb & 1) why = "odd number of SAP blocks in a direction";
    } else if (!g.pair && mu >= 2 && mu <= g.cstar && (g.X[1] >> boxsh[1]) > 1) {
      why = "a single SAP block in a C* direction whose shifted wrap leaves the block";
    }
    // extended-lattice layout: a hop across a C* boundary also shifts x1 by L1; the colour must flip exactly once
    if (!why && !g.pair && mu >= 2 && mu <= g.cstar && nb > 1 && ((g.L1 >> boxsh[1]) & 1))
      why = "the C* shift by L1 is an odd number of blocks in direction 1";
  }
  if (!why) {   // tiles 2j and 2j+1 must differ in colour
    const int ntiles = g.Vh / 128;
    for (int j = 0; j < ntiles / 2 && !why; j++) {
      int col[2];
      for (int k = 0; k < 2; k++) {
        int x[4];
        const int cb = (2 * j + k) * 128;
        coords_int(g, g.pair ? (cb >> 1) : cb, 0, x);
        col[k] = 0;
        for (int mu = 0; mu < 4; mu++) if (colmask[mu]) col[k] += x[mu] >> boxsh[mu];
        col[k] &= 1;
      }
      if (col[0] == col[1]) why = "consecutive tiles have the same colour in this site order";
    }
  }
  if (why) { c->sap_ok = 0; return fail(c, QXD_EINVAL, std::string("SAP: the geometry admits no two-colouring of the blocks (") + why + ")"); }
  for (int mu = 0; mu < 4; mu++) { c->sap_boxsh[mu] = boxsh[mu]; c->sap_colmask[mu] = colmask[mu]; }
  c->sap_ok = 1;
  return QXD_OK;
}

// out = M_sap in: 2 ncy half-steps of sap_mr_k; in, out: fp32 packed full-lattice spinors (parity 1 half_bytes after parity 0)
int launch_sap(qxd_ctx* c, int prec, const void* in, void* out) {
  if (prec != 1 && prec != 2) return fail(c, QXD_EINVAL, "SAP: the block operator is stored in fp32 or binary16");
  int rc = sap_check_geometry(c);
  if (rc) return rc;
  const int Vh = c->g.Vh;
  const size_t hb = half_bytes(1, Vh);
  SapArgs a;
  a.g = c->g;
  for (int p = 0; p < 2; p++) {
    a.W[p] = c->W[prec][p]; a.CL[p] = c->M[prec][p];
    a.res[p] = reinterpret_cast<float4*>(static_cast<char*>(c->g_res) + p * hb);
    a.corr[p] = reinterpret_cast<float4*>(static_cast<char*>(c->g_corr) + p * hb);
    a.psi[p] = reinterpret_cast<float4*>(static_cast<char*>(out) + p * hb);
  }
  for (int mu = 0; mu < 4; mu++) { a.boxsh[mu] = c->sap_boxsh[mu]; a.colmask[mu] = c->sap_colmask[mu]; }
  a.nmr = c->gcr_nmr;
  const int nblocks = Vh / 256;
  const int nl = c->link_reals[prec];
  for (int cy = 0; cy < c->gcr_ncy; cy++)
    for (int col = 0; col < 2; col++) {
      a.colour = col; a.prologue = (cy > 0 || col > 0) ? 1 : 0; a.init_psi = cy == 0 ? 1 : 0;
      for (int p = 0; p < 2; p++)
        a.src[p] = cy == 0 ? reinterpret_cast<const float4*>(static_cast<const char*>(in) + p * hb) : a.res[p];
      if (prec == 1) {
        if (nl == 14) rc = c->g.pair ? sap_launch_t<float, 14, true>(c, a, nblocks) : sap_launch_t<float, 14, false>(c, a, nblocks);
        else rc = c->g.pair ? sap_launch_t<float, 18, true>(c, a, nblocks) : sap_launch_t<float, 18, false>(c, a, nblocks);
      } else {
        if (nl == 14) rc = c->g.pair ? sap_launch_t<__half, 14, true>(c, a, nblocks) : sap_launch_t<__half, 14, false>(c, a, nblocks);
        else rc = c->g.pair ? sap_launch_t<__half, 18, true>(c, a, nblocks) : sap_launch_t<__half, 18, false>(c, a, nblocks);
      }
      if (rc) return rc;
    }
  return QXD_OK;
}


// Coarse operator of the two-level preconditioner (dfl.cu): A[b][9][ns][ns] and the neighbour-block table, from the ns null
// vectors phi (fp32 packed full-lattice), with the block operator in storage precision `prec` (fp32 or binary16).
int launch_coarse_build(qxd_ctx* c, int prec, int ns, void* const* phi, void* A, int* nbr) {
  if (prec != 1 && prec != 2) return fail(c, QXD_EINVAL, "coarse_build: block operator stored in fp32 or binary16");
  int rc = sap_check_geometry(c);
  if (rc) return rc;
  const int nblocks = c->g.Vh / 128;
  CoarseArgs ca;
  ca.a.g = c->g;
  for (int p = 0; p < 2; p++) {
    ca.a.W[p] = c->W[prec][p]; ca.a.CL[p] = c->M[prec][p];
    ca.a.src[p] = nullptr; ca.a.res[p] = nullptr; ca.a.corr[p] = nullptr; ca.a.psi[p] = nullptr;
  }
  for (int mu = 0; mu < 4; mu++) { ca.a.boxsh[mu] = c->sap_boxsh[mu]; ca.a.colmask[mu] = c->sap_colmask[mu]; }
  ca.a.colour = 0; ca.a.prologue = 0; ca.a.init_psi = 0; ca.a.nmr = 0;
  for (int i = 0; i < 32; i++) ca.phi[i] = i < ns ? static_cast<const float4*>(phi[i]) : nullptr;
  ca.ns = ns; ca.ch = c->dfl_chiral ? 1 : 0; ca.A = static_cast<float2*>(A); ca.nbr = nbr;
  QXD_CUDA_OK(c, cudaMemsetAsync(nbr, 0xff, size_t(nblocks) * 8 * sizeof(int), c->stream));
  const int nl = c->link_reals[prec];
  if (prec == 1) {
    if (nl == 14) rc = c->g.pair ? coarse_build_t<float, 14, true>(c, ca, nblocks) : coarse_build_t<float, 14, false>(c, ca, nblocks);
    else rc = c->g.pair ? coarse_build_t<float, 18, true>(c, ca, nblocks) : coarse_build_t<float, 18, false>(c, ca, nblocks);
  } else {
    if (nl == 14) rc = c->g.pair ? coarse_build_t<__half, 14, true>(c, ca, nblocks) : coarse_build_t<__half, 14, false>(c, ca, nblocks);
    else rc = c->g.pair ? coarse_build_t<__half, 18, true>(c, ca, nblocks) : coarse_build_t<__half, 18, false>(c, ca, nblocks);
  }
  return rc;
}

}  // namespace qxd
