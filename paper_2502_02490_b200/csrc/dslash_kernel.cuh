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
#pragma once
#include "dslash_args.h"
#include "block_algebra.cuh"

namespace qxd {

namespace {

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
// acc_u += sc * r ; acc_l += sc * (lower part reconstructed from r).  sc = 1 except for fp16 storage, where it is the
// block-float scale of the neighbour spinor: folding it into these FMAs costs nothing (the link multiply is linear).
template <int MU, int SGN, bool SCALED, typename C>
__device__ __forceinline__ void reconstruct(const C* r, C* acc, C sc) {
  const C p = SCALED ? sc : (C)1, sp = (C)SGN * p, sm = -sp;   // +-scale with the sign of the hop direction
#pragma unroll
  for (int a = 0; a < 3; a++) {
    const C r0r = r[2 * a], r0i = r[2 * a + 1], r1r = r[6 + 2 * a], r1i = r[6 + 2 * a + 1];
    acc[2 * a] += p * r0r; acc[2 * a + 1] += p * r0i;
    acc[6 + 2 * a] += p * r1r; acc[6 + 2 * a + 1] += p * r1i;
    if (MU == 0) {        // lower = s * (r0, r1)
      acc[12 + 2 * a] += sp * r0r; acc[12 + 2 * a + 1] += sp * r0i;
      acc[18 + 2 * a] += sp * r1r; acc[18 + 2 * a + 1] += sp * r1i;
    } else if (MU == 1) { // lower = -s * (i r1, i r0)
      acc[12 + 2 * a] += sp * r1i; acc[12 + 2 * a + 1] += sm * r1r;
      acc[18 + 2 * a] += sp * r0i; acc[18 + 2 * a + 1] += sm * r0r;
    } else if (MU == 2) { // lower = -s * (r1, -r0)
      acc[12 + 2 * a] += sm * r1r; acc[12 + 2 * a + 1] += sm * r1i;
      acc[18 + 2 * a] += sp * r0r; acc[18 + 2 * a + 1] += sp * r0i;
    } else {              // lower = -s * (i r0, -i r1)
      acc[12 + 2 * a] += sp * r0i; acc[12 + 2 * a + 1] += sm * r0r;
      acc[18 + 2 * a] += sm * r1i; acc[18 + 2 * a + 1] += sp * r1r;
    }
  }
}
// r[s][a] = sum_b W[a][b] h[s][b]   (ADJ: sum_b conj(W[b][a]) h[s][b])
// Written as chains of single multiply-adds so that every product is one FMA (re += a*b - c*d would cost three
// instructions: multiply, FMA, add).
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
        const C wi = ADJ ? w[2 * (3 * b + a) + 1] : w[2 * (3 * a + b) + 1];
        const C hr = h[6 * s + 2 * b], hi = h[6 * s + 2 * b + 1];
        if (b == 0) { re = wr * hr; im = wr * hi; } else { re += wr * hr; im += wr * hi; }
        if (ADJ) { re += wi * hi; im -= wi * hr; } else { re -= wi * hi; im += wi * hr; }
      }
      r[6 * s + 2 * a] = re; r[6 * s + 2 * a + 1] = im;
    }
}

// ---- packed fp32 arithmetic (sm_100a FFMA2 / FMUL2: two fp32 lanes per issue slot) ----------------------------------
// The fp32 FMA pipe is no faster with them, but the fp16-storage and C*-paired kernels are bound by instruction issue
// (profiles/r1c_dslash_family_c3.md), and a packed instruction takes one slot for two results.  ptxas folds lane
// broadcast (R.F32), lane swap (LO_HI) and negation into the operand, so the packing below costs no instruction where
// the register allocator can pair the operands.  Same products in the same order as the scalar code: bit-identical.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

// link multiply with the two spin components of the half spinor in the two lanes
template <bool ADJ>
__device__ __forceinline__ void link_mul_x2(const float* w, const float* h, float* r) {
  f32x2 Xr[3], Xi[3];
#pragma unroll
  for (int b = 0; b < 3; b++) { Xr[b] = pk2(h[2 * b], h[6 + 2 * b]); Xi[b] = pk2(h[2 * b + 1], h[6 + 2 * b + 1]); }
#pragma unroll
  for (int a = 0; a < 3; a++) {
    f32x2 re = 0, im = 0;
#pragma unroll
    for (int b = 0; b < 3; b++) {
      const float wr = ADJ ? w[2 * (3 * b + a)] : w[2 * (3 * a + b)];
      const float wi = ADJ ? w[2 * (3 * b + a) + 1] : w[2 * (3 * a + b) + 1];
      const f32x2 Wr = pk2(wr, wr), Wp = pk2(wi, wi), Wn = pk2(-wi, -wi);
      if (b == 0) { re = mul2(Wr, Xr[0]); im = mul2(Wr, Xi[0]); } else { re = fma2(Wr, Xr[b], re); im = fma2(Wr, Xi[b], im); }
      re = fma2(ADJ ? Wp : Wn, Xi[b], re);
      im = fma2(ADJ ? Wn : Wp, Xr[b], im);
    }
    upk2(re, r[2 * a], r[6 + 2 * a]);
    upk2(im, r[2 * a + 1], r[6 + 2 * a + 1]);
  }
}
// reconstruct with the same lanes: (upper spin 0, upper spin 1) and (lower spin 0, lower spin 1) per colour and re/im
template <int MU, int SGN, bool SCALED>
__device__ __forceinline__ void reconstruct_x2(const float* r, float* acc, float sc) {
  const float p = SCALED ? sc : 1.0f, sp = (float)SGN * p, sm = -sp;
  const f32x2 P = pk2(p, p), PP = pk2(sp, sp), MM = pk2(sm, sm), MP = pk2(sm, sp), PM = pk2(sp, sm);
#pragma unroll
  for (int a = 0; a < 3; a++) {
    const f32x2 Rr = pk2(r[2 * a], r[6 + 2 * a]), Ri = pk2(r[2 * a + 1], r[6 + 2 * a + 1]);
    const f32x2 Sr = pk2(r[6 + 2 * a], r[2 * a]), Si = pk2(r[6 + 2 * a + 1], r[2 * a + 1]);   // spins swapped
    f32x2 Ur = pk2(acc[2 * a], acc[6 + 2 * a]), Ui = pk2(acc[2 * a + 1], acc[6 + 2 * a + 1]);
    f32x2 Lr = pk2(acc[12 + 2 * a], acc[18 + 2 * a]), Li = pk2(acc[12 + 2 * a + 1], acc[18 + 2 * a + 1]);
    Ur = fma2(P, Rr, Ur); Ui = fma2(P, Ri, Ui);
    if (MU == 0) { Lr = fma2(PP, Rr, Lr); Li = fma2(PP, Ri, Li); }
    else if (MU == 1) { Lr = fma2(PP, Si, Lr); Li = fma2(MM, Sr, Li); }
    else if (MU == 2) { Lr = fma2(MP, Sr, Lr); Li = fma2(MP, Si, Li); }
    else { Lr = fma2(PM, Ri, Lr); Li = fma2(MP, Rr, Li); }
    upk2(Ur, acc[2 * a], acc[6 + 2 * a]); upk2(Ui, acc[2 * a + 1], acc[6 + 2 * a + 1]);
    upk2(Lr, acc[12 + 2 * a], acc[18 + 2 * a]); upk2(Li, acc[12 + 2 * a + 1], acc[18 + 2 * a + 1]);
  }
}
// Which kernels use the packed forms (measured at c3, same box, both layouts): fp16 storage gains 3-8 % (issue bound);
// fp32 storage loses 0-5 % (bound by DRAM and latency: the pairing constraints on the register allocation cost more
// than the issue slots bring), fp64 has no packed form.
#ifndef QXD_X2_F32
#define QXD_X2_F32 0
#endif
#ifndef QXD_X2_F16
#define QXD_X2_F16 7
#endif
// bit 0: link multiply, bit 1: reconstruct, bit 2: clover block multiply
template <typename S> struct UseX2 {
  static constexpr int MASK = PT<S>::ID == 2 ? QXD_X2_F16 : PT<S>::ID == 1 ? QXD_X2_F32 : 0;
  static constexpr bool LINK = (MASK & 1) != 0, RECON = (MASK & 2) != 0, BLOCK = (MASK & 4) != 0;
};

// (re, im) of one component in the two lanes; A = i * in supplies the products with the imaginary part of the block entry
__device__ __forceinline__ void block_mul_x2(const float* b, const float* in, float* out) {
  f32x2 I[6], A[6], O[6];
#pragma unroll
  for (int k = 0; k < 6; k++) { I[k] = pk2(in[2 * k], in[2 * k + 1]); A[k] = pk2(-in[2 * k + 1], in[2 * k]); }
#pragma unroll
  for (int i = 0; i < 6; i++) O[i] = mul2(pk2(b[i], b[i]), I[i]);
  int k = 6;
#pragma unroll
  for (int i = 0; i < 6; i++)
#pragma unroll
    for (int j = i + 1; j < 6; j++) {
      const float ur = b[k], ui = b[k + 1];
      k += 2;
      const f32x2 Ur = pk2(ur, ur);
      O[i] = fma2(Ur, I[j], O[i]); O[i] = fma2(pk2(ui, ui), A[j], O[i]);       // out_i += u in_j
      O[j] = fma2(Ur, I[i], O[j]); O[j] = fma2(pk2(-ui, -ui), A[i], O[j]);     // out_j += conj(u) in_i
    }
#pragma unroll
  for (int i = 0; i < 6; i++) upk2(O[i], out[2 * i], out[2 * i + 1]);
}
template <typename S, typename C>
__device__ __forceinline__ void block_mul_s(const C* b, const C* in, C* out) {
  if constexpr (UseX2<S>::BLOCK) block_mul_x2(b, in, out); else block_mul(b, in, out);
}
template <typename S>
__device__ __forceinline__ void clover_mul(const void* CL, int Vh, int cb, const typename PT<S>::C* in, typename PT<S>::C* out) {
  typename PT<S>::C b[36];
  load_reals<S, 0, 36>(CL, Vh, cb, b);
  block_mul_s<S>(b, in, out);
  load_reals<S, 36, 36>(CL, Vh, cb, b);
  block_mul_s<S>(b, in + 12, out + 12);
}
// the same blocks applied to R spinors (multi-RHS, row a10): each block is loaded once
template <typename S, int R, bool PAIR>
__device__ __forceinline__ void clover_mul_multi(const void* CL, const Geom& g, int cb, const typename PT<S>::C (*in)[24], typename PT<S>::C (*out)[24]) {
  typedef typename PT<S>::C C;
  C b[36];
  constexpr bool paired = PAIR;
  const bool mir = paired && (cb & 1);
  const int rec = paired ? (cb >> 1) : cb;
#pragma unroll
  for (int blk = 0; blk < 2; blk++) {
    if (blk == 0) load_reals<S, 0, 36>(CL, paired ? g.Vg : g.Vh, rec, b); else load_reals<S, 36, 36>(CL, paired ? g.Vg : g.Vh, rec, b);
#pragma unroll
    for (int r = 0; r < R; r++) {
      if (paired) {
        C a[12], w[12];
        mirror_in(in[r] + 12 * blk, a, mir);
        block_mul_s<S>(b, a, w);
        mirror_out(w, out[r] + 12 * blk, mir);
      } else block_mul_s<S>(b, in[r] + 12 * blk, out[r] + 12 * blk);
    }
  }
}

// One hop in flight: the raw 16-byte chunks of the neighbour spinor and of the link, exactly as loaded.  Keeping the
// packed vectors (not the unpacked reals) in registers between issue and use lets two hops be in flight per thread
// (software pipeline in hop_all below): the kernel is bound by memory latency x bytes in flight, not by arithmetic.
// NL = stored reals per link: 18 (full 3x3) or 14 (rows 0 and 1 + det W = e^{3iqA} (-1)^{bc}: "12-real reconstruct with
// the U(1) phase fused", row 2 = det W * conj(row0 x row1) for any U(3) matrix W; north_star).
template <typename S, int R, int NL>
struct HopRegs {
  typedef typename PT<S>::V V;
  static constexpr int RPC = PT<S>::RPC;
  static constexpr int NPSI = 24 / RPC;
  V psi[R][NPSI];
  static constexpr int NWC = NL == 18 ? (RPC == 2 ? 9 : RPC == 4 ? 5 : 3) : (RPC == 2 ? 7 : RPC == 4 ? 4 : 3);
  V w[NWC];        // chunks covering the NL reals of one link (loaded once for all R right-hand sides)
  float scale[R];  // fp16 block-float scale of the neighbour spinor
  float wsgn;      // paired layout: -1 if the link belongs to a mirror site (W^* = conj W), else +1
};
template <int MU, typename S, int NL> struct LinkChunks {
  static constexpr int RPC = PT<S>::RPC;
  static constexpr int C0 = (NL * MU) / RPC, C1 = (NL * MU + NL - 1) / RPC, N = C1 - C0 + 1, OFF = NL * MU - C0 * RPC;
};
// row 2 of a U(3) matrix from rows 0, 1 and its determinant: w[12..17] = det * conj(row0 x row1); in: w[0..11], det = (w[12], w[13])
template <typename C>
__device__ __forceinline__ void reconstruct_row2(const C* in, C* w) {
#pragma unroll
  for (int i = 0; i < 12; i++) w[i] = in[i];
  const C dr = in[12], di = in[13];
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const int a = (c + 1) % 3, b = (c + 2) % 3;
    const C ar = in[2 * a], ai = in[2 * a + 1], br = in[2 * b], bi = in[2 * b + 1];                    // row 0
    const C pr = in[6 + 2 * a], pi = in[6 + 2 * a + 1], qr = in[6 + 2 * b], qi = in[6 + 2 * b + 1];    // row 1
    C zr = ar * qr; zr -= ai * qi; zr -= br * pr; zr += bi * pi;                                       // z = r0[a] r1[b] - r0[b] r1[a]
    C zi = ar * qi; zi += ai * qr; zi -= br * pi; zi -= bi * pr;
    C rr = dr * zr; rr += di * zi;                                                                     // det * conj(z)
    C ri = di * zr; ri -= dr * zi;
    w[12 + 2 * c] = rr; w[12 + 2 * c + 1] = ri;
  }
}
template <typename S, int MU, int DIR, int R, int NL, bool PAIR>
__device__ __forceinline__ void hop_issue(const DslashArgs& a, const Site& s, int cb, int parity, int rhs0, HopRegs<S, R, NL>& d) {
  typedef typename PT<S>::V V;
  typedef LinkChunks<MU, S, NL> LC;
  const int Vh = a.g.Vh;
  const int nb = neighbour_cb<MU, DIR, PAIR ? 1 : 0>(a.g, s);
#pragma unroll
  for (int r = 0; r < R; r++) {
    if (R > 1 && rhs0 + r >= a.nrhs) break;
    const V* p = reinterpret_cast<const V*>(static_cast<const char*>(a.in[1 - parity].data) + a.rs_in * (rhs0 + r));
#pragma unroll
    for (int c = 0; c < HopRegs<S, R, NL>::NPSI; c++) d.psi[r][c] = ldg_pinned(p + size_t(c) * Vh + nb);
    d.scale[r] = 1.f;
    if (PT<S>::ID == 2) d.scale[r] = ldg_pinned(reinterpret_cast<const float*>(reinterpret_cast<const char*>(a.in[1 - parity].scale) + a.rs_in * (rhs0 + r)) + nb);
  }
  // forward: W_mu(x) of the own parity; backward: W_mu(x-mu) of the other parity at the neighbour
  const V* w = reinterpret_cast<const V*>(DIR > 0 ? a.W[parity] : a.W[1 - parity]);
  int wi = DIR > 0 ? cb : nb;
  d.wsgn = 1.f;
  if (PAIR) { d.wsgn = (wi & 1) ? -1.f : 1.f; wi >>= 1; }   // the record of the physical site; conjugate for the mirror image

  const int Vs = PAIR ? a.g.Vg : Vh;   // stride of the link records (the same register as the spinor stride unless paired)
#pragma unroll
  for (int c = 0; c < LC::N; c++) d.w[c] = ldg_pinned(w + size_t(LC::C0 + c) * Vs + wi);
}
template <typename S, int MU, int DIR, bool G5IN, int R, int NL, bool PAIR>
__device__ __forceinline__ void hop_use(const HopRegs<S, R, NL>& d, typename PT<S>::C (*acc)[24]) {
  typedef typename PT<S>::C C;
  typedef LinkChunks<MU, S, NL> LC;
  constexpr int RPC = PT<S>::RPC;
  C wv[HopRegs<S, R, NL>::NWC * RPC];
#pragma unroll
  for (int c = 0; c < LC::N; c++) unpack_vec(d.w[c], wv + c * RPC);
  if (PAIR) {   // links of mirror sites are the complex conjugates (rows, and det W with them)
#pragma unroll
    for (int i = 1; i < NL; i += 2) wv[LC::OFF + i] *= (C)d.wsgn;
  }
  C w18[18];
  if (NL == 14) reconstruct_row2(wv + LC::OFF, w18);
  const C* wl = NL == 14 ? w18 : wv + LC::OFF;
#pragma unroll
  for (int r = 0; r < R; r++) {
    C psi[24], h[12], t[12];
#pragma unroll
    for (int c = 0; c < HopRegs<S, R, NL>::NPSI; c++) unpack_vec(d.psi[r][c], psi + c * RPC);
    if (G5IN) {
#pragma unroll
      for (int i = 12; i < 24; i++) psi[i] = -psi[i];
    }
    project<MU, DIR>(psi, h);
    if constexpr (UseX2<S>::LINK) link_mul_x2<(DIR < 0)>(wl, h, t); else link_mul<(DIR < 0)>(wl, h, t);
    if constexpr (UseX2<S>::RECON) reconstruct_x2<MU, DIR, PT<S>::ID == 2>(t, acc[r], (C)d.scale[r]);
    else reconstruct<MU, DIR, PT<S>::ID == 2>(t, acc[r], (C)d.scale[r]);
  }
}
// EXPERIMENT (QXD_ASYNC_RING = depth >= 3, off by default): the hops in flight wait in a per-thread shared-memory ring filled by
// cp.async instead of in registers, so that `depth` hops (not two) are outstanding per thread.
#ifndef QXD_ASYNC_RING
#define QXD_ASYNC_RING 0
#endif
__device__ __forceinline__ void ring_cp16(void* smem, const void* gmem) {
  unsigned sa = static_cast<unsigned>(__cvta_generic_to_shared(smem));
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void ring_cp4(void* smem, const void* gmem) {
  unsigned sa = static_cast<unsigned>(__cvta_generic_to_shared(smem));
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(sa), "l"(gmem) : "memory");
}
template <int N> __device__ __forceinline__ void ring_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
template <typename S, int NL, int DEPTH> struct HopRing {
  typedef typename PT<S>::V V;
  static constexpr int NCH = HopRegs<S, 1, NL>::NPSI + HopRegs<S, 1, NL>::NWC;
  V v[DEPTH][NCH][128];
  float scale[DEPTH][128];
};
template <typename S, int H, int NL, bool PAIR, int DEPTH>
__device__ __forceinline__ void ring_issue(const DslashArgs& a, const Site& s, int cb, int parity, HopRing<S, NL, DEPTH>& ring, float (&wsgn)[DEPTH]) {
  typedef typename PT<S>::V V;
  constexpr int MU = H >> 1, DIR = (H & 1) ? -1 : +1, SLOT = H % DEPTH;
  typedef LinkChunks<MU, S, NL> LC;
  const int Vh = a.g.Vh, t = threadIdx.x & 127;
  const int nb = neighbour_cb<MU, DIR, PAIR ? 1 : 0>(a.g, s);
  const V* p = reinterpret_cast<const V*>(a.in[1 - parity].data);
#pragma unroll
  for (int c = 0; c < HopRegs<S, 1, NL>::NPSI; c++) ring_cp16(&ring.v[SLOT][c][t], p + size_t(c) * Vh + nb);
  if (PT<S>::ID == 2) ring_cp4(&ring.scale[SLOT][t], a.in[1 - parity].scale + nb);
  const V* w = reinterpret_cast<const V*>(DIR > 0 ? a.W[parity] : a.W[1 - parity]);
  int wi = DIR > 0 ? cb : nb;
  wsgn[SLOT] = 1.f;
  if (PAIR) { wsgn[SLOT] = (wi & 1) ? -1.f : 1.f; wi >>= 1; }
  const int Vs = PAIR ? a.g.Vg : Vh;
#pragma unroll
  for (int c = 0; c < LC::N; c++) ring_cp16(&ring.v[SLOT][HopRegs<S, 1, NL>::NPSI + c][t], w + size_t(LC::C0 + c) * Vs + wi);
  asm volatile("cp.async.commit_group;" ::: "memory");
}
template <typename S, int H, bool G5IN, int NL, bool PAIR, int DEPTH>
__device__ __forceinline__ void ring_step(const DslashArgs& a, const Site& s, int cb, int parity, HopRing<S, NL, DEPTH>& ring, float (&wsgn)[DEPTH],
                                          typename PT<S>::C (*acc)[24]) {
  constexpr int MU = H >> 1, DIR = (H & 1) ? -1 : +1, SLOT = H % DEPTH;
  typedef LinkChunks<MU, S, NL> LC;
  ring_wait<(7 - H < DEPTH - 1) ? 7 - H : DEPTH - 1>();
  const int t = threadIdx.x & 127;
  HopRegs<S, 1, NL> d;
#pragma unroll
  for (int c = 0; c < HopRegs<S, 1, NL>::NPSI; c++) d.psi[0][c] = ring.v[SLOT][c][t];
#pragma unroll
  for (int c = 0; c < LC::N; c++) d.w[c] = ring.v[SLOT][HopRegs<S, 1, NL>::NPSI + c][t];
  d.scale[0] = PT<S>::ID == 2 ? ring.scale[SLOT][t] : 1.f;
  d.wsgn = wsgn[SLOT];
  if constexpr (H + DEPTH < 8) ring_issue<S, H + DEPTH, NL, PAIR, DEPTH>(a, s, cb, parity, ring, wsgn);
  hop_use<S, MU, DIR, G5IN, 1, NL, PAIR>(d, acc);
}
// all eight hops; PIPE = 2: two hops in flight (software pipeline), PIPE = 1: one; PIPE >= 3: cp.async ring of that depth
template <typename S, bool G5IN, int R, int PIPE, int NL, bool PAIR>
__device__ __forceinline__ void hop_all(const DslashArgs& a, const Site& s, int cb, int parity, int rhs0, typename PT<S>::C (*acc)[24]) {
  if constexpr (PIPE >= 3) {
    __shared__ HopRing<S, NL, PIPE> ring;
    float wsgn[PIPE];
    ring_issue<S, 0, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn);
    ring_issue<S, 1, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn);
    ring_issue<S, 2, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn);
    if constexpr (PIPE >= 4) ring_issue<S, 3, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn);
    ring_step<S, 0, G5IN, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn, acc);
    ring_step<S, 1, G5IN, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn, acc);
    ring_step<S, 2, G5IN, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn, acc);
    ring_step<S, 3, G5IN, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn, acc);
    ring_step<S, 4, G5IN, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn, acc);
    ring_step<S, 5, G5IN, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn, acc);
    ring_step<S, 6, G5IN, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn, acc);
    ring_step<S, 7, G5IN, NL, PAIR, PIPE>(a, s, cb, parity, ring, wsgn, acc);
  } else if (PIPE == 2) {
    HopRegs<S, R, NL> d0, d1;
    hop_issue<S, 0, +1, R, NL, PAIR>(a, s, cb, parity, rhs0, d0);
    hop_issue<S, 0, -1, R, NL, PAIR>(a, s, cb, parity, rhs0, d1);
    hop_use<S, 0, +1, G5IN, R, NL, PAIR>(d0, acc);
    hop_issue<S, 1, +1, R, NL, PAIR>(a, s, cb, parity, rhs0, d0);
    hop_use<S, 0, -1, G5IN, R, NL, PAIR>(d1, acc);
    hop_issue<S, 1, -1, R, NL, PAIR>(a, s, cb, parity, rhs0, d1);
    hop_use<S, 1, +1, G5IN, R, NL, PAIR>(d0, acc);
    hop_issue<S, 2, +1, R, NL, PAIR>(a, s, cb, parity, rhs0, d0);
    hop_use<S, 1, -1, G5IN, R, NL, PAIR>(d1, acc);
    hop_issue<S, 2, -1, R, NL, PAIR>(a, s, cb, parity, rhs0, d1);
    hop_use<S, 2, +1, G5IN, R, NL, PAIR>(d0, acc);
    hop_issue<S, 3, +1, R, NL, PAIR>(a, s, cb, parity, rhs0, d0);
    hop_use<S, 2, -1, G5IN, R, NL, PAIR>(d1, acc);
    hop_issue<S, 3, -1, R, NL, PAIR>(a, s, cb, parity, rhs0, d1);
    hop_use<S, 3, +1, G5IN, R, NL, PAIR>(d0, acc);
    hop_use<S, 3, -1, G5IN, R, NL, PAIR>(d1, acc);
  } else {
    HopRegs<S, R, NL> d;
    hop_issue<S, 0, +1, R, NL, PAIR>(a, s, cb, parity, rhs0, d); hop_use<S, 0, +1, G5IN, R, NL, PAIR>(d, acc);
    hop_issue<S, 0, -1, R, NL, PAIR>(a, s, cb, parity, rhs0, d); hop_use<S, 0, -1, G5IN, R, NL, PAIR>(d, acc);
    hop_issue<S, 1, +1, R, NL, PAIR>(a, s, cb, parity, rhs0, d); hop_use<S, 1, +1, G5IN, R, NL, PAIR>(d, acc);
    hop_issue<S, 1, -1, R, NL, PAIR>(a, s, cb, parity, rhs0, d); hop_use<S, 1, -1, G5IN, R, NL, PAIR>(d, acc);
    hop_issue<S, 2, +1, R, NL, PAIR>(a, s, cb, parity, rhs0, d); hop_use<S, 2, +1, G5IN, R, NL, PAIR>(d, acc);
    hop_issue<S, 2, -1, R, NL, PAIR>(a, s, cb, parity, rhs0, d); hop_use<S, 2, -1, G5IN, R, NL, PAIR>(d, acc);
    hop_issue<S, 3, +1, R, NL, PAIR>(a, s, cb, parity, rhs0, d); hop_use<S, 3, +1, G5IN, R, NL, PAIR>(d, acc);
    hop_issue<S, 3, -1, R, NL, PAIR>(a, s, cb, parity, rhs0, d); hop_use<S, 3, -1, G5IN, R, NL, PAIR>(d, acc);
  }
}

// PHI: 0 none, 1 phi, 2 M*phi (FULL: phi = in on the own parity).  POST: 1 = multiply the result by M^{-1}.
// Full-lattice launches (row a4) work on both parities of 128 consecutive checkerboard indices -- one 4x4x4x4 tile with
// the default order -- at the same time (two consecutive 128-thread CTAs for one right-hand side, one 256-thread CTA
// for a batch): every link is then used twice within a few microseconds (forward hop of x, backward hop of x+mu) and
// 3/4 of the neighbour spinors belong to the tile itself.
// R > 1 (row a10, multi-RHS): every thread applies the operator of its site to R right-hand sides, loading each link
// and clover block once; ngroups consecutive CTAs cover all right-hand sides of one tile, so the links of a tile are
// read from DRAM once and from L2 by the other groups.
template <typename S, int R, bool FULL, int NL> struct KernelShape {
  // Full lattice, single right-hand side: either one 256-thread CTA per tile (both parities: the second use of every link
  // hits L1) or one 128-thread CTA per (tile, parity) in consecutive CTAs (links shared through L2).  Timed alone (ncu, 1.83
  // GHz) the split form is 4.5 % faster (534 vs 559 us, 18-real links); in a long run the GPU sits on its power cap and
  // the time follows the energy per apply: the extra 0.8 GB of L2 -> SM traffic of the split form costs 6 % (0.68 vs 0.64
  // ms sustained) with 18-real links, while with the 14-real format the split form stays ahead (0.61 vs 0.62 ms).
  static constexpr bool SPLIT = FULL && R == 1 && NL == 14;
  static constexpr int THREADS = (FULL && !SPLIT) ? 256 : 128;
  // CTAs per SM the register budget is sized for
  static constexpr int MINB = SPLIT ? (sizeof(S) == 8 ? 2 : 4) : sizeof(S) == 8 ? 1 : (R == 1 ? (FULL ? 2 : 4) : (R == 2 ? (FULL ? 1 : 3) : (FULL ? 1 : 2)));
  static constexpr int PIPE = (QXD_ASYNC_RING >= 3 && R == 1 && !FULL && sizeof(S) == 2) ? QXD_ASYNC_RING : (R == 1) ? 2 : 1;   // hops in flight per thread
};
template <typename S, int PHI, int POST, bool NEG, int FLAGS, bool FULL, int R, int NL, bool PAIR>
__global__ void __launch_bounds__(KernelShape<S, R, FULL, NL>::THREADS, KernelShape<S, R, FULL, NL>::MINB) dslash_k(const __grid_constant__ DslashArgs a) {
  typedef typename PT<S>::C C;
  const int Vh = a.g.Vh;
  constexpr bool SPLIT = KernelShape<S, R, FULL, NL>::SPLIT;
  // block index -> (tile, parity, group of R right-hand sides), groups fastest: the CTAs that need the links and clover
  // blocks of a tile run at the same time, so a batch reads them from DRAM once and from L2 afterwards
  const int bt = blockIdx.x / a.ngroups;
  const int rhs0 = (blockIdx.x - bt * a.ngroups) * R;
  const int tile = tile_of(a.tm, SPLIT ? (bt >> 1) : bt);
  const int cb = tile * 128 + (threadIdx.x & 127);
  const int parity = FULL ? (SPLIT ? (bt & 1) : (threadIdx.x >> 7)) : a.parity_out;
  constexpr int NRED = (FLAGS & DSF_DOT) ? 3 : 1;   // fused reductions: |out|^2, or <phi,out> and |out|^2
  double nrm[R][NRED];
#pragma unroll
  for (int r = 0; r < R; r++)
#pragma unroll
    for (int k = 0; k < NRED; k++) nrm[r][k] = 0.0;
  Site s;
  bool active = cb < Vh;
  if (active) {
    site_init<PAIR ? 1 : 0>(a.g, cb, parity, s);
    active = s.x[0] >= a.t_lo && s.x[0] < a.t_hi;   // time range of a slab-restricted launch (uniform over the CTA for whole slabs)
  }
  if (active) {
    C acc[R][24];
#pragma unroll
    for (int r = 0; r < R; r++)
#pragma unroll
      for (int i = 0; i < 24; i++) acc[r][i] = 0;
    const C hs = NEG ? (C)0.5 : (C)-0.5;  // +-hop = -+1/2 acc
    hop_all<S, (FLAGS & DSF_G5IN) != 0, R, KernelShape<S, R, FULL, NL>::PIPE, NL, PAIR>(a, s, cb, parity, rhs0, acc);
#pragma unroll
    for (int r = 0; r < R; r++)
#pragma unroll
      for (int i = 0; i < 24; i++) acc[r][i] *= ((FLAGS & DSF_G5HOP) && i >= 12) ? -hs : hs;
    if (PHI != 0) {
      C phi[R][24];
#pragma unroll
      for (int r = 0; r < R; r++) {
        if (R > 1 && rhs0 + r >= a.nrhs) break;
        load_spinor<S>(FULL ? rhs_view(a.in[parity], a.rs_in, rhs0 + r) : rhs_view(a.phi, a.rs_phi, rhs0 + r), Vh, cb, phi[r]);
      }
      if (PHI == 2) {
        C mphi[R][24];
        clover_mul_multi<S, R, PAIR>(a.CL[parity], a.g, cb, phi, mphi);
#pragma unroll
        for (int r = 0; r < R; r++)
#pragma unroll
          for (int i = 0; i < 24; i++) acc[r][i] += mphi[r][i];
      } else {
#pragma unroll
        for (int r = 0; r < R; r++)
#pragma unroll
          for (int i = 0; i < 24; i++) acc[r][i] += phi[r][i];
      }
    }
    if (POST) {
      C t[R][24];
      clover_mul_multi<S, R, PAIR>(a.CL[parity], a.g, cb, acc, t);
#pragma unroll
      for (int r = 0; r < R; r++)
#pragma unroll
        for (int i = 0; i < 24; i++) acc[r][i] = t[r][i];
    }
#pragma unroll
    for (int r = 0; r < R; r++) {
      if (R > 1 && rhs0 + r >= a.nrhs) break;
      if (FLAGS & DSF_DOT) {    // BiCGstab's <s,t> and |t|^2 for t = A s: phi = s is re-read (L1/L2) rather than kept in registers
        C ph[24];
        load_spinor<S>(rhs_view(a.phi, a.rs_phi, rhs0 + r), Vh, cb, ph);
        C p0 = 0, p1 = 0, p2 = 0;
#pragma unroll
        for (int k = 0; k < 12; k++) {
          const C xr = ph[2 * k], xi = ph[2 * k + 1], yr = acc[r][2 * k], yi = acc[r][2 * k + 1];
          p0 += xr * yr; p0 += xi * yi;
          p1 += xr * yi; p1 -= xi * yr;
          p2 += yr * yr; p2 += yi * yi;
        }
        nrm[r][0] = (double)p0; nrm[r][NRED > 1 ? 1 : 0] = (double)p1; nrm[r][NRED - 1] = (double)p2;
      } else if (FLAGS & DSF_NORM) {   // per-site sum in the arithmetic type, fp64 across sites (see blas.cu)
        C part = 0;
#pragma unroll
        for (int i = 0; i < 24; i++) part += acc[r][i] * acc[r][i];
        nrm[r][0] = (double)part;
      }
      store_spinor<S>(rhs_view(a.out[parity], a.rs_out, rhs0 + r), Vh, cb, acc[r]);
    }
  }
  if (FLAGS & (DSF_NORM | DSF_DOT)) {
    const int ntiles = gridDim.x / a.ngroups;
#pragma unroll
    for (int r = 0; r < R; r++) {
      if (R > 1 && rhs0 + r >= a.nrhs) break;   // uniform over the CTA
      grid_reduce<NRED>(nrm[r], a.R, tile, ntiles, rhs0 + r);
    }
  }
}

template <typename S, int PHI, int POST, bool NEG, int FLAGS, bool FULL, int R, int NL, bool PAIR>
void launch_r(qxd_ctx* c, DslashArgs& a) {
  a.ngroups = (a.nrhs + R - 1) / R;
  const unsigned ntiles = a.tm.count > 0 ? unsigned(a.tm.count) : unsigned((c->g.Vh + 127) / 128);
  dim3 gr(ntiles * unsigned(a.ngroups) * (KernelShape<S, R, FULL, NL>::SPLIT ? 2u : 1u));
  dslash_k<S, PHI, POST, NEG, FLAGS, FULL, R, NL, PAIR><<<gr, KernelShape<S, R, FULL, NL>::THREADS, 0, c->stream>>>(a);
}
// right-hand sides per thread: 1 for a single spinor; for a batch the value chosen by qxd_set_rhs_per_thread (default 1:
// measured at c3 with 12 right-hand sides, fp32: 0.43 ms per right-hand side against 0.59 (R = 2) and 0.50 (R = 3))
// MULTI: instantiate the R = 2, 3 kernels for this mode (only the modes the batched solver and bench use)
template <typename S, int NL, bool PAIR, int PHI, int POST, bool NEG, int FLAGS, bool FULL, bool MULTI>
int launch_one(qxd_ctx* c, DslashArgs& a) {
  int R = 1;
  if (a.nrhs > 1) {
    R = c->rhs_per_thread > 0 ? c->rhs_per_thread : 1;
    if (R > a.nrhs) R = a.nrhs;
  }
  if (MULTI && sizeof(S) < 8) {   // fp64: the accumulators of two spinors do not fit the register file
    if (R == 2) { launch_r<S, PHI, POST, NEG, FLAGS, FULL, (MULTI && sizeof(S) < 8) ? 2 : 1, NL, PAIR>(c, a); return QXD_OK; }
    if (R >= 3) { launch_r<S, PHI, POST, NEG, FLAGS, FULL, (MULTI && sizeof(S) < 8) ? 3 : 1, NL, PAIR>(c, a); return QXD_OK; }
  }
  // one right-hand side per thread, the right-hand sides of a tile in consecutive CTAs
  launch_r<S, PHI, POST, NEG, FLAGS, FULL, 1, NL, PAIR>(c, a);
  return QXD_OK;
}

template <typename S, int NL, bool PAIR>
int dispatch(qxd_ctx* c, const DslashCall& d, DslashArgs& a) {
  const int f = d.flags;
  switch (d.mode) {
    case DS_DW_FULL:
      if (f != 0) break;
      return launch_one<S, NL, PAIR, 2, 0, false, 0, true, true>(c, a);
    case DS_HOP_AINV:
      if (f == 0) { return launch_one<S, NL, PAIR, 0, 1, false, 0, false, true>(c, a); }
      if (f == DSF_G5IN) { return launch_one<S, NL, PAIR, 0, 1, false, DSF_G5IN, false, true>(c, a); }
      break;
    case DS_A_XMHOP:
      if (f == 0) { return launch_one<S, NL, PAIR, 2, 0, true, 0, false, true>(c, a); }
      if (f == DSF_NORM) { return launch_one<S, NL, PAIR, 2, 0, true, DSF_NORM, false, true>(c, a); }
      if (f == DSF_DOT) { return launch_one<S, NL, PAIR, 2, 0, true, DSF_DOT, false, false>(c, a); }
      if (f == DSF_G5HOP) { return launch_one<S, NL, PAIR, 2, 0, true, DSF_G5HOP, false, true>(c, a); }
      if (f == (DSF_G5HOP | DSF_NORM)) { return launch_one<S, NL, PAIR, 2, 0, true, DSF_G5HOP | DSF_NORM, false, true>(c, a); }
      break;
    case DS_X_MHOP:
      if (f == 0) { return launch_one<S, NL, PAIR, 1, 0, true, 0, false, false>(c, a); }
      break;
    case DS_AINV_X_MHOP:
      if (f == 0) { return launch_one<S, NL, PAIR, 1, 1, true, 0, false, false>(c, a); }
      break;
    default: break;
  }
  return fail(c, QXD_EINVAL, "dslash: unsupported mode/flags combination");
}

}  // namespace

}  // namespace qxd
