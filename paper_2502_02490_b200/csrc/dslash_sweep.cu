// dslash_sweep.cu -- an alternative full-lattice D_w kernel (SURVEY.md §8 row a4, fp32 storage, 18-real links, extended-lattice
// layout) built to cut the halo traffic of the tile kernel (dslash_kernel.cuh), whose DRAM traffic is 14.5 % above the
// algorithmic bytes, all of it out-of-tile neighbour spinors (profiles/r1d_dslash_fp32_c3.md).
//
// A CTA owns a spatial footprint of 8 x 8 x 4 sites (2 x 2 tiles in directions 1, 2) and SWEEPS a segment of time slices:
// thread <-> site of the slice (256 threads = 128 sites of each parity).  The spinors of the slices t-1, t, t+1 of the
// footprint live in a four-slot shared-memory ring (24 KB per slice) that is filled two slices ahead by per-thread
// cp.async copies (no registers held while the data are in flight, one __syncthreads per slice), so that
//   - the two time neighbours and every spatial neighbour inside the footprint are read from shared memory, and
//   - only the spatial faces of the footprint (1.0 out-of-footprint neighbours per site instead of 2.0 per site for a
//     4^4 tile) are read through L2, from CTAs that work on the same time segment at the same time.
// Links and clover blocks stream through registers exactly as in the tile kernel (hop_use / clover_mul_multi are shared).
// Reads and writes the same packed layout, so it is interchangeable with the tile kernel (qxd_set_dw_sweep).
#include "dslash_kernel.cuh"

namespace qxd {

namespace {

struct SweepArgs {
  Geom g;
  const float4* in[2];
  float4* out[2];
  const void* W[2];
  const void* CL[2];
  int ncx, ncy, ncz;   // footprints per direction 1, 2, 3
  int tseg;            // time slices per work unit
};

constexpr int SW_SLICE = 2 * 6 * 128;            // float4 per ring slot: [parity][chunk][128]
constexpr int SW_RING = 4;
constexpr size_t SW_SMEM = size_t(SW_RING) * SW_SLICE * sizeof(float4);   // 96 KB

__device__ __forceinline__ void cp_async16(float4* smem, const float4* gmem) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

struct SweepThread {
  int p, q, r;          // parity, tile of the footprint (qx = q >> 1, qy = q & 1), index inside the tile slice (xl, yl, zh)
  int lx, ly, zh;       // local coordinates in the footprint (lz = 2 zh + zb depends on t)
  int X0, Y0, Z0;
};

// one hop whose spinor comes from the ring (in-footprint) or from global memory (footprint face); the link always streams
struct SweepHop {
  HopRegs<float, 1, 18> d;
  int sidx;             // >= 0: float4 index of chunk 0 in the ring; -1: already loaded from global memory
};

template <int MU, int DIR>
__device__ __forceinline__ void sweep_issue(const SweepArgs& a, const Site& s, const SweepThread& th, int cb, int slot_t, int lz, SweepHop& h) {
  typedef LinkChunks<MU, float, 18> LC;
  const int Vh = a.g.Vh;
  const int nb = neighbour_cb<MU, DIR, 0>(a.g, s);
  int sidx = -1;
  if (MU == 0) {
    sidx = ((slot_t + DIR + SW_RING) & (SW_RING - 1)) * SW_SLICE + (1 - th.p) * 6 * 128 + th.q * 32 + th.r;
  } else if (MU == 1) {
    const int l = th.lx + DIR;
    if (l >= 0 && l < 8) sidx = slot_t * SW_SLICE + (1 - th.p) * 6 * 128 + ((((l >> 2) << 1) | (th.q & 1)) * 32) + (((l & 3) * 4 + (th.ly & 3)) * 2 + th.zh);
  } else if (MU == 2) {
    const int l = th.ly + DIR;
    if (l >= 0 && l < 8) sidx = slot_t * SW_SLICE + (1 - th.p) * 6 * 128 + (((th.q & 2) | (l >> 2)) * 32) + (((th.lx & 3) * 4 + (l & 3)) * 2 + th.zh);
  } else {
    const int l = lz + DIR;
    if (l >= 0 && l < 4) sidx = slot_t * SW_SLICE + (1 - th.p) * 6 * 128 + th.q * 32 + (((th.lx & 3) * 4 + (th.ly & 3)) * 2 + (l >> 1));
  }
  h.sidx = sidx;
  if (sidx < 0) {
    const float4* p = a.in[1 - th.p];
#pragma unroll
    for (int c = 0; c < 6; c++) h.d.psi[0][c] = ldg_pinned(p + size_t(c) * Vh + nb);
  }
  h.d.scale[0] = 1.f; h.d.wsgn = 1.f;
  const float4* w = reinterpret_cast<const float4*>(DIR > 0 ? a.W[th.p] : a.W[1 - th.p]);
  const int wi = DIR > 0 ? cb : nb;
#pragma unroll
  for (int c = 0; c < LC::N; c++) h.d.w[c] = ldg_pinned(w + size_t(LC::C0 + c) * Vh + wi);
}
template <int MU, int DIR>
__device__ __forceinline__ void sweep_use(SweepHop& h, const float4* ring, float (*acc)[24]) {
  if (h.sidx >= 0) {
#pragma unroll
    for (int c = 0; c < 6; c++) h.d.psi[0][c] = ring[h.sidx + c * 128];
  }
  hop_use<float, MU, DIR, false, 1, 18, false>(h.d, acc);
}

__global__ void __launch_bounds__(256, 2) dw_sweep_k(const __grid_constant__ SweepArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* ring = reinterpret_cast<float4*>(smem_raw);
  const Geom& g = a.g;
  const int Vh = g.Vh;
  const int ncol = a.ncx * a.ncy * a.ncz;
  const int seg = blockIdx.x / ncol, col = blockIdx.x - seg * ncol;
  SweepThread th;
  th.Z0 = (col % a.ncz) * 4; th.Y0 = ((col / a.ncz) % a.ncy) * 8; th.X0 = (col / (a.ncz * a.ncy)) * 8;
  const int tau = threadIdx.x;
  th.p = tau >> 7; th.q = (tau >> 5) & 3; th.r = tau & 31;
  const int xl = th.r >> 3, yl = (th.r >> 1) & 3;
  th.zh = th.r & 1;
  th.lx = 4 * (th.q >> 1) + xl; th.ly = 4 * (th.q & 1) + yl;
  const int T = g.X[0];
  const int t0 = seg * a.tseg;
  const int t1 = t0 + a.tseg < T ? t0 + a.tseg : T;       // slices [t0, t1)
  Site s;
  s.m = 0;
  s.x[1] = th.X0 + th.lx; s.x[2] = th.Y0 + th.ly;
  s.gx[1] = gmu(g, 1, s.x[1]); s.gx[2] = gmu(g, 2, s.x[2]);
  // checkerboard index of this thread's footprint site on slice tt (tt may be t0 - 1 or t1: wrapped) and parity th.p
  auto site_at = [&](int tt, Site& o) {
    const int tw = tt < 0 ? tt + T : (tt >= T ? tt - T : tt);
    o = s;
    o.x[0] = tw; o.gx[0] = gmu(g, 0, tw);
    const int zb = (th.p + tw + o.x[1] + o.x[2]) & 1;
    o.x[3] = th.Z0 + 2 * th.zh + zb; o.gx[3] = gmu(g, 3, o.x[3]);
    o.idx2 = o.gx[0] + o.gx[1] + o.gx[2] + o.gx[3];
  };
  auto prefetch = [&](int tt) {        // the thread's own site of slice tt -> ring slot tt & 3
    Site o;
    site_at(tt, o);
    const int cbp = o.idx2 >> 1;
    float4* dst = ring + ((tt + SW_RING) & (SW_RING - 1)) * SW_SLICE + th.p * 6 * 128 + th.q * 32 + th.r;
    const float4* src = a.in[th.p] + cbp;
#pragma unroll
    for (int c = 0; c < 6; c++) cp_async16(dst + c * 128, src + size_t(c) * Vh);
  };
  prefetch(t0 - 1); prefetch(t0); prefetch(t0 + 1);
  cp_async_commit();
  for (int t = t0; t < t1; t++) {
    cp_async_wait_all();
    __syncthreads();                   // slices <= t+1 are in the ring; everybody is done with slice t-2
    if (t + 2 <= t1) prefetch(t + 2);  // into the slot of slice t-2
    cp_async_commit();
    Site cur;
    site_at(t, cur);
    const int cb = cur.idx2 >> 1;
    const int lz = cur.x[3] - th.Z0;
    const int slot = t & (SW_RING - 1);
    float acc[1][24];
#pragma unroll
    for (int i = 0; i < 24; i++) acc[0][i] = 0.f;
    {
      SweepHop h0, h1;
      sweep_issue<0, +1>(a, cur, th, cb, slot, lz, h0);
      sweep_issue<0, -1>(a, cur, th, cb, slot, lz, h1);
      sweep_use<0, +1>(h0, ring, acc);
      sweep_issue<1, +1>(a, cur, th, cb, slot, lz, h0);
      sweep_use<0, -1>(h1, ring, acc);
      sweep_issue<1, -1>(a, cur, th, cb, slot, lz, h1);
      sweep_use<1, +1>(h0, ring, acc);
      sweep_issue<2, +1>(a, cur, th, cb, slot, lz, h0);
      sweep_use<1, -1>(h1, ring, acc);
      sweep_issue<2, -1>(a, cur, th, cb, slot, lz, h1);
      sweep_use<2, +1>(h0, ring, acc);
      sweep_issue<3, +1>(a, cur, th, cb, slot, lz, h0);
      sweep_use<2, -1>(h1, ring, acc);
      sweep_issue<3, -1>(a, cur, th, cb, slot, lz, h1);
      sweep_use<3, +1>(h0, ring, acc);
      sweep_use<3, -1>(h1, ring, acc);
    }
    float phi[1][24], mphi[1][24];
    {
      const float4* own = ring + slot * SW_SLICE + th.p * 6 * 128 + th.q * 32 + th.r;
#pragma unroll
      for (int c = 0; c < 6; c++) { const float4 v = own[c * 128]; phi[0][4 * c] = v.x; phi[0][4 * c + 1] = v.y; phi[0][4 * c + 2] = v.z; phi[0][4 * c + 3] = v.w; }
    }
    clover_mul_multi<float, 1, false>(a.CL[th.p], g, cb, phi, mphi);
    float4* o = a.out[th.p] + cb;
#pragma unroll
    for (int c = 0; c < 6; c++)
      o[size_t(c) * Vh] = make_float4(mphi[0][4 * c] - 0.5f * acc[0][4 * c], mphi[0][4 * c + 1] - 0.5f * acc[0][4 * c + 1],
                                      mphi[0][4 * c + 2] - 0.5f * acc[0][4 * c + 2], mphi[0][4 * c + 3] - 0.5f * acc[0][4 * c + 3]);
  }
  cp_async_wait_all();
}

}  // namespace

// out = D_w in with the sweep kernel; QXD_EINVAL if the geometry or the formats do not fit (the caller falls back)
int launch_dw_sweep(qxd_ctx* c, const SpinorPtr in[2], const SpinorPtr out[2]) {
  const Geom& g = c->g;
  if (g.pair || c->link_reals[1] != 18 || c->dw_sweep_tseg < 1) return QXD_EINVAL;
  if (c->tile[0] != 4 || c->tile[1] != 4 || c->tile[2] != 4 || c->tile[3] != 4 || g.X[1] % 8 || g.X[2] % 8 || g.X[3] % 4 || g.X[0] % 4) return QXD_EINVAL;
  static bool configured = false;
  if (!configured) {
    QXD_CUDA_OK(c, cudaFuncSetAttribute(dw_sweep_k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SW_SMEM));
    configured = true;
  }
  SweepArgs a;
  a.g = g;
  for (int p = 0; p < 2; p++) {
    a.in[p] = static_cast<const float4*>(in[p].data); a.out[p] = static_cast<float4*>(out[p].data);
    a.W[p] = c->W[1][p]; a.CL[p] = c->M[1][p];
  }
  a.ncx = g.X[1] / 8; a.ncy = g.X[2] / 8; a.ncz = g.X[3] / 4;
  a.tseg = c->dw_sweep_tseg;
  const int nseg = (g.X[0] + a.tseg - 1) / a.tseg;
  dw_sweep_k<<<a.ncx * a.ncy * a.ncz * nseg, 256, SW_SMEM, c->stream>>>(a);
  QXD_LAUNCH_CHECK(c);
  return QXD_OK;
}

}  // namespace qxd
