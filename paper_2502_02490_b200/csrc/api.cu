// api.cu -- the C-ABI entry points declared in include/qxd.h.  Argument checking,
// workspace carving and call sequencing only; every step of the path runs in the kernels of this library.
#include "qxd_ctx.h"
#include <new>
#include <cstring>
#include <vector>

using namespace qxd;

namespace qxd {
int apply_dhat(qxd_ctx* c, int prec, const SpinorPtr& in_e, const SpinorPtr& out_e, const SpinorPtr& tmp_o, int dagger, double* norm_slot);
}

namespace {

int pow2_le_dividing(int extent, int target) {
  int b = 1;
  while (b * 2 <= target && extent % (b * 2) == 0) b *= 2;
  return b;
}
int ilog2(int v) { int s = 0; while ((1 << s) < v) s++; return s; }

int set_order(qxd_ctx* c, const int b[4], const int B[4]) {
  Geom& g = c->g;
  for (int mu = 0; mu < 4; mu++) {
    if (b[mu] < 1 || (b[mu] & (b[mu] - 1)) || g.X[mu] % b[mu]) return fail(c, QXD_EINVAL, "tile extents must be powers of two dividing the extended extents");
    if (B[mu] < b[mu] || (B[mu] & (B[mu] - 1)) || g.X[mu] % B[mu]) return fail(c, QXD_EINVAL, "block extents must be powers of two, multiples of the tile extents, dividing the extended extents");
  }
  if (b[3] < 2) return fail(c, QXD_EINVAL, "tile extent b3 must be >= 2");
  int tv = 1, mv = 1;  // sites per tile, tiles per block
  for (int mu = 0; mu < 4; mu++) { g.sh[mu] = ilog2(b[mu]); g.shB[mu] = ilog2(B[mu]); g.nB[mu] = g.X[mu] / B[mu]; tv *= b[mu]; mv *= B[mu] / b[mu]; }
  g.s0[3] = 1; g.s0[2] = b[3]; g.s0[1] = b[3] * b[2]; g.s0[0] = b[3] * b[2] * b[1];
  g.s1[3] = tv; g.s1[2] = g.s1[3] * (B[3] / b[3]); g.s1[1] = g.s1[2] * (B[2] / b[2]); g.s1[0] = g.s1[1] * (B[1] / b[1]);
  const int bv = tv * mv;
  g.s2[3] = bv; g.s2[2] = bv * g.nB[3]; g.s2[1] = bv * g.nB[3] * g.nB[2]; g.s2[0] = bv * g.nB[3] * g.nB[2] * g.nB[1];
  for (int mu = 0; mu < 4; mu++) { c->tile[mu] = b[mu]; c->block[mu] = B[mu]; }
  return QXD_OK;
}

struct Carver {
  size_t off = 0;
  char* base;
  explicit Carver(char* b) : base(b) {}
  void* take(size_t bytes) {
    void* p = base ? base + off : nullptr;
    off += (bytes + 255) & ~size_t(255);
    return p;
  }
};

// One layout routine serves both the size query (base == nullptr) and the binding.
size_t carve(qxd_ctx* c, char* base, int prec_mask, int nrhs, bool assign) {
  const size_t Vh = c->g.Vh, Vg = c->g.Vg;
  Carver k(base);
  void* Ug[2]; void* Ag[2]; void* W[NPREC][2] = {}; void* M[NPREC][2] = {}; void* Mi[NPREC][2] = {};
  for (int p = 0; p < 2; p++) { Ug[p] = k.take(Vg * 72 * 8); Ag[p] = k.take(Vg * 4 * 8); }
  for (int pr = 0; pr < NPREC; pr++) {
    if (!((prec_mask >> pr) & 1)) continue;
    for (int p = 0; p < 2; p++) {
      W[pr][p] = k.take(Vg * 72 * prec_size(pr)); M[pr][p] = k.take(Vg * 72 * prec_size(pr));
      // block inverses: only A_oo^{-1} is ever applied (SURVEY.md §8 row a3 "odd sites only is enough"); the even-site inverses
      // exist in fp64 alone, for qxd_clover_export
      Mi[pr][p] = (pr == 0 || p == 1) ? k.take(Vg * 72 * prec_size(pr)) : nullptr;
    }
  }
  void* sp64[12]; void* splo[8];
  for (int i = 0; i < 12; i++) sp64[i] = k.take(half_bytes(0, Vh));
  for (int i = 0; i < 8; i++) splo[i] = k.take(half_bytes(0, Vh));  // sized for the widest sloppy type (fp64 when sloppy == hi)
  void* fa = k.take(2 * half_bytes(0, Vh));
  void* fb = k.take(2 * half_bytes(0, Vh));
  void* na = k.take(size_t(c->V) * 24 * 8);
  void* nb = k.take(size_t(c->V) * 24 * 8);
  const int max_blocks = int((Vh + 127) / 128) * 2 + 8;
  void* partials = k.take(size_t(max_blocks) * 4 * 8 * nrhs);
  void* scal = k.take(64 * 8);
  // batch vectors (row a10): fp64 b, x and five sloppy vectors per right-hand side; the sloppy ones are sized for the
  // widest bound precision below fp64 (fp64 itself if no other is bound)
  void* mhi[2] = {}; void* mlo[7] = {};
  const size_t mlo_size = (prec_mask & 2) ? 4 : (prec_mask & 4) ? 2 : 8;
  void* mscal = nullptr; void* mact = nullptr;
  if (nrhs > 1) {
    const int plo = mlo_size == 8 ? 0 : mlo_size == 4 ? 1 : 2;
    const size_t lo = (half_bytes(plo, Vh) + 255) & ~size_t(255);
    for (int i = 0; i < 2; i++) mhi[i] = k.take(half_bytes(0, Vh) * nrhs);
    // x, r, p, t, odd-site scratch; r16, p16 only for the binary16 operator with fp32 vectors
    for (int i = 0; i < 7; i++) mlo[i] = (i < 5 || (mlo_size == 4 && (prec_mask & 4))) ? k.take(lo * nrhs) : nullptr;
    mscal = k.take(64 * 8 * 8);
    mact = k.take(64 * 8);
  }
  // SAP-GCR (row f3): 2 nkv + 3 fp32 full-lattice vectors, 2 fp64 ones, scalars
  void* gz[32] = {}; void* gw[32] = {}; void* g_r = nullptr; void* g_res = nullptr; void* g_corr = nullptr; void* g_r64 = nullptr; void* g_t64 = nullptr;
  void* gscal = nullptr;
  if (c->gcr_nkv > 0) {
    const size_t f32 = 2 * half_bytes(1, Vh), f64 = 2 * half_bytes(0, Vh);
    for (int i = 0; i < c->gcr_nkv; i++) { gz[i] = k.take(f32); gw[i] = k.take(f32); }
    g_r = k.take(f32); g_res = k.take(f32); g_corr = k.take(f32); g_r64 = k.take(f64); g_t64 = k.take(f64);
    gscal = k.take(4096 * 8);
  }
  // two-level preconditioner (dfl.cu): ns + 2 fp32 full-lattice vectors, the coarse operator and the coarse-grid vectors
  void* dphi[32] = {}; void* dcz[32] = {}; void* dcw[32] = {};
  void* d_t1 = nullptr; void* d_t2 = nullptr; void* dAc = nullptr; void* dnbr = nullptr; void* dcb = nullptr; void* dcx = nullptr; void* dcr = nullptr;
  void* dscal = nullptr; void* dDinv = nullptr; void* dAh = nullptr; void* dcol = nullptr; void* dcs = nullptr; void* dct = nullptr;
  if (c->dfl_ns > 0) {
    const size_t ncd = size_t(c->dfl_ns) * (c->dfl_chiral ? 2 : 1);   // coarse dimension per block
    const size_t f32 = 2 * half_bytes(1, Vh), nb = Vh / 128 > 0 ? Vh / 128 : 1, cv = nb * ncd * 8;
    for (int i = 0; i < c->dfl_ns; i++) dphi[i] = k.take(f32);
    d_t1 = k.take(f32); d_t2 = k.take(f32);
    dAc = k.take(nb * 9 * ncd * ncd * 8); dnbr = k.take(nb * 8 * 4); dDinv = k.take(nb * ncd * ncd * 8);
    dcb = k.take(cv); dcx = k.take(cv); dcr = k.take(cv); dcs = k.take(cv); dct = k.take(cv);
    dAh = k.take(nb * 9 * ncd * ncd * 4); dcol = k.take(nb * 4);
    for (int i = 0; i < c->dfl_nkc; i++) { dcz[i] = k.take(cv); dcw[i] = k.take(cv); }
    dscal = k.take(4096 * 8);
  }
  if (assign) {
    for (int i = 0; i < 32; i++) { c->dphi[i] = dphi[i]; c->dcz[i] = dcz[i]; c->dcw[i] = dcw[i]; }
    c->d_t1 = d_t1; c->d_t2 = d_t2; c->dAc = dAc; c->dnbr = (int*)dnbr; c->dcb = dcb; c->dcx = dcx; c->dcr = dcr; c->dscal = (double*)dscal; c->dDinv = dDinv;
    c->dAh = dAh; c->dcol = (int*)dcol; c->dcs = dcs; c->dct = dct;
    c->dfl_ready = false;
    for (int i = 0; i < 32; i++) { c->gz[i] = gz[i]; c->gw[i] = gw[i]; }
    c->g_r = g_r; c->g_res = g_res; c->g_corr = g_corr; c->g_r64 = g_r64; c->g_t64 = g_t64; c->gscal = (double*)gscal;
    for (int i = 0; i < 2; i++) c->mhi[i] = mhi[i];
    for (int i = 0; i < 7; i++) c->mlo[i] = mlo[i];
    c->mlo_size = nrhs > 1 ? mlo_size : 0; c->mscal = (double*)mscal; c->mact = (double*)mact;
    for (int p = 0; p < 2; p++) { c->Ug[p] = Ug[p]; c->Ag[p] = Ag[p]; }
    for (int pr = 0; pr < NPREC; pr++) for (int p = 0; p < 2; p++) { c->W[pr][p] = W[pr][p]; c->M[pr][p] = M[pr][p]; c->Mi[pr][p] = Mi[pr][p]; }
    for (int i = 0; i < 12; i++) c->sp64[i] = sp64[i];
    for (int i = 0; i < 8; i++) c->splo[i] = splo[i];
    c->full_a = fa; c->full_b = fb; c->nat_a = (double*)na; c->nat_b = (double*)nb;
    c->partials = (double*)partials; c->scal = (double*)scal; c->max_blocks = max_blocks;
  }
  return k.off;
}

bool prec_ok(const qxd_ctx* c, int prec) { return prec >= 0 && prec < NPREC && ((c->prec_mask >> prec) & 1); }

}  // namespace

extern "C" {

const char* qxd_version(void) { return "qxd-b200 0.1 (sm_100a)"; }

int qxd_geometry_create(int T, int L1, int L2, int L3, int bc, qxd_ctx** out) {
  if (!out) return QXD_EINVAL;
  *out = nullptr;
  if (T < 2 || L1 < 2 || L2 < 2 || L3 < 2 || ((T | L1 | L2 | L3) & 1) || bc < 0 || bc > 7) return QXD_EINVAL;
  const int cstar = bc & 3;
  const long V = long(T) * (cstar ? 2 * L1 : L1) * L2 * L3;
  if (V / 2 * 72 > 0x7fffffffL) return QXD_EINVAL;  // chunk indices are 32-bit
  qxd_ctx* c = new (std::nothrow) qxd_ctx;
  if (!c) return QXD_EINVAL;
  c->T = T; c->L1 = L1; c->L2 = L2; c->L3 = L3; c->bc = bc; c->V = V;
  Geom& g = c->g;
  g.X[0] = T; g.X[1] = cstar ? 2 * L1 : L1; g.X[2] = L2; g.X[3] = L3;
  g.L1 = L1; g.cstar = cstar; g.antiper = (bc >> 2) & 1; g.Vh = int(V / 2);
  for (int mu = 0; mu < 4; mu++) g.XE[mu] = g.X[mu];
  g.pair = 0; g.Vg = g.Vh;
  // default order: 4x4x4x4 tiles (256 sites = one CTA of the full-lattice kernel), blocks of 4 tiles stacked in time and
  // time slabs 16 thick, so that only 1/8 of the sites have a neighbour in another slab
  int b[4] = {pow2_le_dividing(g.X[0], 4), pow2_le_dividing(g.X[1], 4), pow2_le_dividing(g.X[2], 4), pow2_le_dividing(g.X[3], 4)};
  int B[4] = {pow2_le_dividing(g.X[0], 16), b[1], b[2], b[3]};
  set_order(c, b, B);
  *out = c;
  // C* geometries use the paired layout by default; qxd_set_cstar_pairing(ctx, 0) selects the extended one
  if (cstar > 0) qxd_set_cstar_pairing(c, 1);
  return QXD_OK;
}

int qxd_geometry_destroy(qxd_ctx* c) {
  if (!c) return QXD_EINVAL;
  if (c->h_scal) cudaFreeHost(c->h_scal);
  if (c->ev0) cudaEventDestroy(c->ev0);
  if (c->ev1) cudaEventDestroy(c->ev1);
  if (c->ev_scal) cudaEventDestroy(c->ev_scal);
  for (int io = 0; io < 2; io++) for (int k = 0; k < 64; k++) if (c->ev_slab[io][k]) cudaEventDestroy(c->ev_slab[io][k]);
  if (c->s_in) cudaStreamDestroy(c->s_in);
  if (c->s_out) cudaStreamDestroy(c->s_out);
  delete c;
  return QXD_OK;
}

int qxd_set_tile(qxd_ctx* c, int b0, int b1, int b2, int b3) {
  if (!c) return QXD_EINVAL;
  if (c->ws) return fail(c, QXD_ESTATE, "qxd_set_tile must precede qxd_workspace_bind");
  int b[4] = {b0, b1, b2, b3};
  int B[4];
  for (int mu = 0; mu < 4; mu++) B[mu] = c->block[mu] > b[mu] && b[mu] > 0 && c->block[mu] % b[mu] == 0 ? c->block[mu] : b[mu];
  return set_order(c, b, B);
}

int qxd_set_block(qxd_ctx* c, int B0, int B1, int B2, int B3) {
  if (!c) return QXD_EINVAL;
  if (c->ws) return fail(c, QXD_ESTATE, "qxd_set_block must precede qxd_workspace_bind");
  int B[4] = {B0, B1, B2, B3};
  return set_order(c, c->tile, B);
}

int qxd_set_cstar_pairing(qxd_ctx* c, int on) {
  if (!c) return QXD_EINVAL;
  if (c->ws) return fail(c, QXD_ESTATE, "qxd_set_cstar_pairing must precede qxd_workspace_bind");
  Geom& g = c->g;
  if (on && g.cstar == 0) return fail(c, QXD_EINVAL, "set_cstar_pairing: the geometry has no C* direction");
  g.pair = on ? 1 : 0;
  g.X[1] = g.pair ? g.L1 : g.XE[1];
  g.Vg = g.pair ? g.Vh / 2 : g.Vh;
  // default site order on the indexed lattice (as in qxd_geometry_create)
  int b[4] = {pow2_le_dividing(g.X[0], 4), pow2_le_dividing(g.X[1], 4), pow2_le_dividing(g.X[2], 4), pow2_le_dividing(g.X[3], 4)};
  int B[4] = {pow2_le_dividing(g.X[0], 16), b[1], b[2], b[3]};
  return set_order(c, b, B);
}

long qxd_volume(const qxd_ctx* c) { return c ? c->V : 0; }

int qxd_site_index(const qxd_ctx* c, const int x[4], int* cb, int* parity) {
  if (!c || !x || !cb || !parity) return QXD_EINVAL;
  for (int mu = 0; mu < 4; mu++) if (x[mu] < 0 || x[mu] >= c->g.XE[mu]) return QXD_EINVAL;
  *parity = (x[0] + x[1] + x[2] + x[3]) & 1;
  if (c->g.pair) {   // (physical site, mirror bit)
    const int m = x[1] >= c->g.L1 ? 1 : 0;
    const int xp[4] = {x[0], x[1] - m * c->g.L1, x[2], x[3]};
    *cb = ((idx2_of(c->g, xp) >> 1) << 1) | m;
  } else *cb = idx2_of(c->g, x) >> 1;
  return QXD_OK;
}
int qxd_site_coords(const qxd_ctx* c, int cb, int parity, int x[4]) {
  if (!c || !x || cb < 0 || cb >= c->g.Vh || parity < 0 || parity > 1) return QXD_EINVAL;
  coords_of(c->g, cb, parity, x);
  return QXD_OK;
}
int qxd_site_neighbour(const qxd_ctx* c, int cb, int parity, int mu, int dir, int* cb_nb) {
  if (!c || !cb_nb || cb < 0 || cb >= c->g.Vh || parity < 0 || parity > 1 || mu < 0 || mu > 3 || (dir != 1 && dir != -1)) return QXD_EINVAL;
  Site s;
  site_init(c->g, cb, parity, s);
  switch (mu * 2 + (dir > 0 ? 0 : 1)) {
    case 0: *cb_nb = neighbour_cb<0, +1>(c->g, s); break;
    case 1: *cb_nb = neighbour_cb<0, -1>(c->g, s); break;
    case 2: *cb_nb = neighbour_cb<1, +1>(c->g, s); break;
    case 3: *cb_nb = neighbour_cb<1, -1>(c->g, s); break;
    case 4: *cb_nb = neighbour_cb<2, +1>(c->g, s); break;
    case 5: *cb_nb = neighbour_cb<2, -1>(c->g, s); break;
    case 6: *cb_nb = neighbour_cb<3, +1>(c->g, s); break;
    default: *cb_nb = neighbour_cb<3, -1>(c->g, s); break;
  }
  return QXD_OK;
}

size_t qxd_workspace_bytes(const qxd_ctx* c, int prec_mask, int nrhs) {
  if (!c || nrhs < 1 || nrhs > 64) return 0;
  return carve(const_cast<qxd_ctx*>(c), nullptr, (prec_mask | 1) & 7, nrhs, false);
}

int qxd_workspace_bind(qxd_ctx* c, void* dev, size_t bytes, int prec_mask, int nrhs) {
  if (!c || nrhs < 1 || nrhs > 64) return QXD_EINVAL;
  prec_mask = (prec_mask | 1) & 7;
  if (!dev || (reinterpret_cast<uintptr_t>(dev) & 255)) return fail(c, QXD_EWORKSPACE, "workspace must be a 256-byte aligned device pointer");
  const size_t need = carve(c, nullptr, prec_mask, nrhs, false);
  if (bytes < need) return fail(c, QXD_EWORKSPACE, "workspace too small");
  c->ws = static_cast<char*>(dev); c->ws_bytes = bytes; c->prec_mask = prec_mask; c->nrhs = nrhs;
  c->ws_used = carve(c, c->ws, prec_mask, nrhs, true);
  c->have_gauge = c->have_quark = c->have_clover = false;
  if (!c->h_scal) {
    QXD_CUDA_OK(c, cudaMallocHost((void**)&c->h_scal, (64 + 64 * 8 + 64) * sizeof(double)));
    c->h_mscal = c->h_scal + 64; c->h_mact = c->h_mscal + 64 * 8;
  }
  if (c->mscal) QXD_CUDA_OK(c, cudaMemsetAsync(c->mscal, 0, 64 * 8 * 8, c->stream));
  if (!c->ev0) QXD_CUDA_OK(c, cudaEventCreate(&c->ev0));
  if (!c->ev1) QXD_CUDA_OK(c, cudaEventCreate(&c->ev1));
  if (!c->ev_scal) QXD_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_scal, cudaEventDisableTiming));
  QXD_CUDA_OK(c, cudaMemsetAsync(c->scal, 0, 64 * 8, c->stream));
  return QXD_OK;
}

int qxd_set_stream(qxd_ctx* c, void* s) {
  if (!c) return QXD_EINVAL;
  c->stream = static_cast<cudaStream_t>(s);
  return QXD_OK;
}

// ---- field-status manager (row f4) ---------------------------------------------------------------
static int refresh_hoplinks(qxd_ctx* c) {
  for (int pr = 0; pr < NPREC; pr++)
    if ((c->prec_mask >> pr) & 1) { int rc = launch_hoplinks(c, pr); if (rc) return rc; }
  c->hop_stale = false; c->n_hop_refresh++;
  return QXD_OK;
}
static int refresh_clover(qxd_ctx* c) {
  int rc = launch_clover_build(c);
  if (rc) return rc;
  c->clover_stale = false; c->n_clover_refresh++;
  return QXD_OK;
}
// regenerate what a setter left stale; every entry point that reads derived fields calls it first
static int ensure_fresh(qxd_ctx* c) {
  if (c->hop_stale) { int rc = refresh_hoplinks(c); if (rc) return rc; }
  if (c->clover_stale) { int rc = refresh_clover(c); if (rc) return rc; }
  return QXD_OK;
}

int qxd_set_lazy_refresh(qxd_ctx* c, int on) {
  if (!c) return QXD_EINVAL;
  if (!on) { int rc = ensure_fresh(c); if (rc) return rc; }
  c->lazy = on != 0;
  return QXD_OK;
}
int qxd_refresh(qxd_ctx* c) { return c ? ensure_fresh(c) : QXD_EINVAL; }
int qxd_field_status(const qxd_ctx* c, int* status, long counts[2]) {
  if (!c || !status) return QXD_EINVAL;
  *status = (c->have_gauge ? QXD_FS_GAUGE : 0) | (c->have_quark && !c->hop_stale ? QXD_FS_HOPLINKS : 0) |
            (c->have_clover && !c->clover_stale ? QXD_FS_CLOVER : 0) | (c->hop_stale ? QXD_FS_HOPLINKS_STALE : 0) |
            (c->clover_stale ? QXD_FS_CLOVER_STALE : 0) | (c->lazy ? QXD_FS_LAZY : 0);
  if (counts) { counts[0] = c->n_hop_refresh; counts[1] = c->n_clover_refresh; }
  return QXD_OK;
}

int qxd_gauge_load(qxd_ctx* c, const double* U, const double* A, double qel) {
  if (!c || !U) return c ? fail(c, QXD_EINVAL, "gauge_load: U_su3 is null") : QXD_EINVAL;
  if (!c->ws) return fail(c, QXD_EWORKSPACE, "gauge_load: no workspace bound");
  if (A && !(qel != 0.0)) return fail(c, QXD_EINVAL, "gauge_load: qel must be non-zero");
  c->qel = A ? qel : 1.0;
  c->have_qed = (A != nullptr);
  int rc = launch_gauge_pack(c, U, A);
  if (rc) return rc;
  c->have_gauge = true; c->dfl_ready = false;
  if (c->lazy) {   // the quark and clover parameters stay; what they produced is stale until its next use
    c->hop_stale = c->have_quark; c->clover_stale = c->have_clover;
  } else { c->have_quark = false; c->have_clover = false; }
  return QXD_OK;
}

int qxd_set_quark(qxd_ctx* c, double kappa, double q) {
  if (!c) return QXD_EINVAL;
  if (!c->have_gauge) return fail(c, QXD_ESTATE, "set_quark: load a gauge field first");
  if (!(kappa > 0.0)) return fail(c, QXD_EINVAL, "set_quark: kappa must be > 0");
  c->kappa = kappa; c->q = q; c->m0 = 1.0 / (2.0 * kappa) - 4.0; c->dfl_ready = false;
  if (c->lazy) {   // the clover term depends on m0 and q: stale too if its coefficients are known
    c->have_quark = true; c->hop_stale = true; c->clover_stale = c->have_clover;
    return QXD_OK;
  }
  int rc = refresh_hoplinks(c);
  if (rc) return rc;
  c->have_quark = true; c->have_clover = false;
  return QXD_OK;
}

int qxd_set_gauge_reconstruct_prec(qxd_ctx* c, int prec, int recon) {
  if (!c) return QXD_EINVAL;
  if (prec < 0 || prec >= NPREC) return fail(c, QXD_EINVAL, "set_gauge_reconstruct: unknown precision");
  if (recon != QXD_RECON_NONE && recon != QXD_RECON_12) return fail(c, QXD_EINVAL, "set_gauge_reconstruct: QXD_RECON_NONE (18) or QXD_RECON_12 (12)");
  const int nl = recon == QXD_RECON_12 ? 14 : 18;
  if (nl == c->link_reals[prec]) return QXD_OK;
  c->link_reals[prec] = nl;
  // the hopping links are derived data: rewrite them in the new format (the clover term is unaffected)
  if (c->have_quark && !c->hop_stale && ((c->prec_mask >> prec) & 1)) return launch_hoplinks(c, prec);
  return QXD_OK;
}
int qxd_set_gauge_reconstruct(qxd_ctx* c, int recon) {
  if (!c) return QXD_EINVAL;
  for (int pr = 0; pr < NPREC; pr++) { int rc = qxd_set_gauge_reconstruct_prec(c, pr, recon); if (rc) return rc; }
  return QXD_OK;
}

int qxd_clover_build(qxd_ctx* c, double csw, double csw_qed) {
  if (!c) return QXD_EINVAL;
  if (!c->have_gauge || !c->have_quark) return fail(c, QXD_ESTATE, "clover_build: needs gauge_load and set_quark");
  c->csw = csw; c->csw_qed = csw_qed; c->dfl_ready = false;
  if (c->lazy) { c->have_clover = true; c->clover_stale = true; return QXD_OK; }
  int rc = refresh_clover(c);
  if (rc) return rc;
  c->have_clover = true;
  return QXD_OK;
}

int qxd_clover_stats(const qxd_ctx* c, long counts[2]) {
  if (!c || !counts) return QXD_EINVAL;
  counts[0] = c->n_inv_fast; counts[1] = c->n_inv_pivoted;
  return QXD_OK;
}

int qxd_clover_export(qxd_ctx* c, double* out, int inverse) {
  if (!c || !out) return QXD_EINVAL;
  if (!c->have_clover) return fail(c, QXD_ESTATE, "clover_export: build the clover term first");
  int rc = ensure_fresh(c);
  if (rc) return rc;
  return launch_clover_export(c, out, inverse);
}

static int check_apply(qxd_ctx* c, int prec, const void* a, const void* b, const char* who) {
  if (!c) return QXD_EINVAL;
  if (!a || !b) return fail(c, QXD_EINVAL, std::string(who) + ": null pointer");
  if (!c->have_clover) return fail(c, QXD_ESTATE, std::string(who) + ": needs gauge_load, set_quark and clover_build");
  if (!prec_ok(c, prec)) return fail(c, QXD_EINVAL, std::string(who) + ": precision not bound in the workspace");
  return ensure_fresh(c);
}

int qxd_apply_Dw_packed(qxd_ctx* c, int prec, const void* in, void* out) {
  int rc = check_apply(c, prec, in, out, "apply_Dw_packed");
  if (rc) return rc;
  const int Vh = c->g.Vh;
  DslashCall d{};
  d.prec = prec; d.mode = DS_DW_FULL; d.flags = 0;
  d.in[0] = half_view(prec, const_cast<void*>(in), Vh, 0); d.in[1] = half_view(prec, const_cast<void*>(in), Vh, 1);
  d.out[0] = half_view(prec, out, Vh, 0); d.out[1] = half_view(prec, out, Vh, 1);
  if (prec == 1 && c->dw_sweep_tseg > 0) {   // time-sweep kernel where it applies (fp32, 18-real links, extended layout, 4^4 tiles)
    rc = launch_dw_sweep(c, d.in, d.out);
    if (rc != QXD_EINVAL) return rc;
  }
  return launch_dslash(c, d);
}

int qxd_set_dw_sweep(qxd_ctx* c, int tseg) {
  if (!c || tseg < 0 || tseg == 1) return c ? fail(c, QXD_EINVAL, "set_dw_sweep: 0 (off) or a segment length >= 2") : QXD_EINVAL;
  c->dw_sweep_tseg = tseg;
  return QXD_OK;
}

int qxd_apply_Dw_multi_packed(qxd_ctx* c, int prec, int nrhs, const void* in, void* out) {
  int rc = check_apply(c, prec, in, out, "apply_Dw_multi_packed");
  if (rc) return rc;
  if (nrhs < 1 || nrhs > 64) return fail(c, QXD_EINVAL, "apply_Dw_multi_packed: nrhs must be in 1..64");
  if (size_t(c->max_blocks) * 4 * c->nrhs < size_t(nrhs)) return fail(c, QXD_EINVAL, "apply_Dw_multi_packed: nrhs exceeds the bound workspace");
  const int Vh = c->g.Vh;
  DslashCall d{};
  d.prec = prec; d.mode = DS_DW_FULL; d.flags = 0;
  d.in[0] = half_view(prec, const_cast<void*>(in), Vh, 0); d.in[1] = half_view(prec, const_cast<void*>(in), Vh, 1);
  d.out[0] = half_view(prec, out, Vh, 0); d.out[1] = half_view(prec, out, Vh, 1);
  d.nrhs = nrhs; d.rs_in = d.rs_phi = d.rs_out = 2 * half_bytes(prec, Vh);
  return launch_dslash(c, d);
}

int qxd_apply_Dw_multi_interleaved(qxd_ctx* c, int prec, int nrhs, const void* in, void* out) {
  int rc = check_apply(c, prec, in, out, "apply_Dw_multi_interleaved");
  if (rc) return rc;
  if (nrhs < 4 || nrhs > 64) return fail(c, QXD_EINVAL, "apply_Dw_multi_interleaved: nrhs must be a multiple of 4 in 4..64");
  return launch_dw_ilv(c, prec, nrhs, in, out);
}
int qxd_multi_interleave(qxd_ctx* c, int prec, int nrhs, void* plain, void* interleaved, int to_interleaved) {
  if (!c || !plain || !interleaved || prec < 0 || prec >= NPREC || !c->ws) return c ? fail(c, QXD_EINVAL, "multi_interleave: bad argument") : QXD_EINVAL;
  return launch_ilv_convert(c, prec, nrhs, plain, interleaved, to_interleaved);
}

int qxd_set_rhs_per_thread(qxd_ctx* c, int r) {
  if (!c || r < 0 || r > 3) return c ? fail(c, QXD_EINVAL, "set_rhs_per_thread: 0 (default), 1, 2 or 3") : QXD_EINVAL;
  c->rhs_per_thread = r;
  return QXD_OK;
}

int qxd_apply_Dhat_packed(qxd_ctx* c, int prec, const void* in_e, void* out_e, int dagger) {
  int rc = check_apply(c, prec, in_e, out_e, "apply_Dhat_packed");
  if (rc) return rc;
  const int Vh = c->g.Vh;
  return apply_dhat(c, prec, half_view(prec, const_cast<void*>(in_e), Vh, 0), half_view(prec, out_e, Vh, 0), half_view(prec, c->sp64[11], Vh, 0), dagger,
                    nullptr);
}

int qxd_apply_Dw(qxd_ctx* c, int prec, const double* psi, double* out) {
  int rc = check_apply(c, prec, psi, out, "apply_Dw");
  if (rc) return rc;
  if ((rc = launch_spinor_pack(c, prec, psi, c->full_a, 3, 0))) return rc;
  if ((rc = qxd_apply_Dw_packed(c, prec, c->full_a, c->full_b))) return rc;
  return launch_spinor_unpack(c, prec, c->full_b, out, 3, 0);
}

int qxd_apply_Dhat_eo(qxd_ctx* c, int prec, const double* psi_e, double* out_e, int dagger) {
  int rc = check_apply(c, prec, psi_e, out_e, "apply_Dhat_eo");
  if (rc) return rc;
  if ((rc = launch_spinor_pack(c, prec, psi_e, c->full_a, 1, 1))) return rc;
  if ((rc = qxd_apply_Dhat_packed(c, prec, c->full_a, c->full_b, dagger))) return rc;
  return launch_spinor_unpack(c, prec, c->full_b, out_e, 1, 1);
}

// Time slabs of one tile thickness as tile subsets (TileMap, qxd_common.cuh): inside a block the t digit of the tile index
// is the slowest one, and the blocks are lexicographic with direction 0 slowest, so slab (bt, mt) is
// { (bt NBsp + i) mv + mt q + j : i < NBsp, j < q } with mv tiles per block and q = mv / (tiles per block in t).
static bool time_slabs(const qxd_ctx* c, std::vector<TileMap>& maps, size_t& slab_sites) {
  const Geom& g = c->g;
  long tv = 1, mv = 1;
  for (int mu = 0; mu < 4; mu++) { tv *= c->tile[mu]; mv *= c->block[mu] / c->tile[mu]; }
  if (tv != 256 || g.Vh % 128) return false;   // the kernels' 128-index tiles must tile the geometric tiles
  // paired layout: a geometric tile (of the physical lattice) holds two 128-index kernel tiles per parity, (2 n, 2 n + 1)
  const int f = g.pair ? 2 : 1;
  const int ntt = c->block[0] / c->tile[0], q = int(mv / ntt), NBsp = g.nB[1] * g.nB[2] * g.nB[3];
  const int S = g.nB[0] * ntt;
  if (S < 3 || S > 64) return false;
  int lq = 0;
  while ((1 << lq) < q * f) lq++;
  maps.clear();
  for (int bt = 0; bt < g.nB[0]; bt++)
    for (int mt = 0; mt < ntt; mt++) {
      TileMap m;
      m.lq = lq; m.qm = q * f - 1; m.mv = int(mv) * f; m.base = (bt * NBsp * int(mv) + mt * q) * f; m.count = NBsp * q * f;
      maps.push_back(m);
    }
  slab_sites = size_t(c->tile[0]) * g.XE[1] * g.XE[2] * g.XE[3];
  return true;
}

// Host-pointer D_w (the shape of the paper's boundary: host arrays in, host arrays out).  The lattice is cut
// into time slabs of one tile thickness; slab k is copied in on its own stream, packed as soon as it has arrived, the operator
// is applied to a slab as soon as its two time neighbours are packed, and its result is unpacked and copied out on a third
// stream -- so the device->host copy of the first slabs overlaps the host->device copy of the last ones (PCIe is full duplex)
// and only the copies of about three slabs are exposed.  Orders without such slabs fall back to copy - apply - copy.
int qxd_apply_Dw_host(qxd_ctx* c, int prec, const double* psi_host, double* out_host) {
  int rc = check_apply(c, prec, psi_host, out_host, "apply_Dw_host");
  if (rc) return rc;
  const size_t bytes = size_t(c->V) * 24 * sizeof(double);
  std::vector<TileMap> maps;
  size_t slab_sites = 0;
  if (!time_slabs(c, maps, slab_sites)) {
    QXD_CUDA_OK(c, cudaMemcpyAsync(c->nat_a, psi_host, bytes, cudaMemcpyHostToDevice, c->stream));
    if ((rc = qxd_apply_Dw(c, prec, c->nat_a, c->nat_b))) return rc;
    QXD_CUDA_OK(c, cudaMemcpyAsync(out_host, c->nat_b, bytes, cudaMemcpyDeviceToHost, c->stream));
    QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
    return QXD_OK;
  }
  const int S = int(maps.size());
  if (!c->s_in) QXD_CUDA_OK(c, cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking));
  if (!c->s_out) QXD_CUDA_OK(c, cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking));
  for (int k = 0; k < S; k++)
    for (int io = 0; io < 2; io++)
      if (!c->ev_slab[io][k]) QXD_CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_slab[io][k], cudaEventDisableTiming));
  // the copy streams start after whatever is queued on the compute stream (it may still read the staging buffers)
  QXD_CUDA_OK(c, cudaEventRecord(c->ev_scal, c->stream));
  QXD_CUDA_OK(c, cudaStreamWaitEvent(c->s_in, c->ev_scal, 0));
  QXD_CUDA_OK(c, cudaStreamWaitEvent(c->s_out, c->ev_scal, 0));
  const size_t slab_reals = slab_sites * 24, slab_bytes = slab_reals * sizeof(double);
  for (int k = 0; k < S; k++) {
    QXD_CUDA_OK(c, cudaMemcpyAsync(c->nat_a + k * slab_reals, psi_host + k * slab_reals, slab_bytes, cudaMemcpyHostToDevice, c->s_in));
    QXD_CUDA_OK(c, cudaEventRecord(c->ev_slab[0][k], c->s_in));
  }
  const int Vh = c->g.Vh;
  bool packed[64] = {}, applied[64] = {};
  for (int k = 0; k < S; k++) {
    QXD_CUDA_OK(c, cudaStreamWaitEvent(c->stream, c->ev_slab[0][k], 0));
    if ((rc = launch_spinor_pack(c, prec, c->nat_a, c->full_a, 3, 0, maps[k]))) return rc;
    packed[k] = true;
    for (int j = 0; j < S; j++) {
      if (applied[j] || !(packed[(j + S - 1) % S] && packed[j] && packed[(j + 1) % S])) continue;
      DslashCall d{};
      d.prec = prec; d.mode = DS_DW_FULL; d.flags = 0;
      d.in[0] = half_view(prec, c->full_a, Vh, 0); d.in[1] = half_view(prec, c->full_a, Vh, 1);
      d.out[0] = half_view(prec, c->full_b, Vh, 0); d.out[1] = half_view(prec, c->full_b, Vh, 1);
      d.tm = maps[j];
      if ((rc = launch_dslash(c, d))) return rc;
      if ((rc = launch_spinor_unpack(c, prec, c->full_b, c->nat_b, 3, 0, maps[j]))) return rc;
      QXD_CUDA_OK(c, cudaEventRecord(c->ev_slab[1][j], c->stream));
      QXD_CUDA_OK(c, cudaStreamWaitEvent(c->s_out, c->ev_slab[1][j], 0));
      QXD_CUDA_OK(c, cudaMemcpyAsync(out_host + j * slab_reals, c->nat_b + j * slab_reals, slab_bytes, cudaMemcpyDeviceToHost, c->s_out));
      applied[j] = true;
    }
  }
  QXD_CUDA_OK(c, cudaStreamSynchronize(c->s_out));
  QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
  return QXD_OK;
}

// ---- domain decomposition building blocks (row f2) ------------------------------------------------------------------
int qxd_time_slabs(const qxd_ctx* c, int* nslabs, int* thickness) {
  if (!c || !nslabs || !thickness) return QXD_EINVAL;
  std::vector<TileMap> maps;
  size_t slab_sites = 0;
  if (!time_slabs(c, maps, slab_sites)) return QXD_EINVAL;
  *nslabs = int(maps.size()); *thickness = c->tile[0];
  return QXD_OK;
}

int qxd_dslash_packed(qxd_ctx* c, int prec, int mode, int flags, int parity_out, const void* in, const void* phi, void* out, int slab_lo, int slab_hi) {
  int rc = check_apply(c, prec, in, out, "dslash_packed");
  if (rc) return rc;
  if (mode < 0 || mode >= DS_NMODES || (flags & ~(DSF_G5IN | DSF_G5HOP)) || parity_out < 0 || parity_out > 1) return fail(c, QXD_EINVAL, "dslash_packed: bad mode, flags or parity");
  const bool needs_phi = mode == DS_A_XMHOP || mode == DS_X_MHOP || mode == DS_AINV_X_MHOP;
  if (needs_phi && !phi) return fail(c, QXD_EINVAL, "dslash_packed: this mode needs phi");
  std::vector<TileMap> maps;
  size_t slab_sites = 0;
  if (!time_slabs(c, maps, slab_sites)) return fail(c, QXD_EINVAL, "dslash_packed: the site order has no time slabs");
  if (slab_lo < 0 || slab_hi > int(maps.size()) || slab_lo > slab_hi) return fail(c, QXD_EINVAL, "dslash_packed: bad slab range");
  const int Vh = c->g.Vh;
  DslashCall d{};
  d.prec = prec; d.mode = mode; d.flags = flags; d.parity_out = parity_out;
  void* inp = const_cast<void*>(in);
  void* php = const_cast<void*>(phi);
  if (mode == DS_DW_FULL) {
    d.in[0] = half_view(prec, inp, Vh, 0); d.in[1] = half_view(prec, inp, Vh, 1);
    d.out[0] = half_view(prec, out, Vh, 0); d.out[1] = half_view(prec, out, Vh, 1);
  } else {
    d.in[1 - parity_out] = half_view(prec, inp, Vh, 1 - parity_out);
    if (needs_phi) d.phi = half_view(prec, php, Vh, parity_out);
    d.out[parity_out] = half_view(prec, out, Vh, parity_out);
  }
  if (slab_hi > slab_lo) {   // ONE launch over all tiles; the CTAs whose time slab lies outside the range retire at once
    d.t_lo = slab_lo * c->tile[0]; d.t_hi = slab_hi * c->tile[0];
    if ((rc = launch_dslash(c, d))) return rc;
  }
  return QXD_OK;
}

int qxd_clover_apply_packed(qxd_ctx* c, int prec, int inverse, int parity, const void* in, void* out) {
  int rc = check_apply(c, prec, in, out, "clover_apply_packed");
  if (rc) return rc;
  if (parity < 0 || parity > 1) return fail(c, QXD_EINVAL, "clover_apply_packed: parity 0 or 1");
  if (inverse && !c->Mi[prec][parity]) return fail(c, QXD_EINVAL, "clover_apply_packed: the even-site inverses exist in fp64 only");
  const int Vh = c->g.Vh;
  return launch_clover_apply(c, prec, inverse, parity, half_view(prec, const_cast<void*>(in), Vh, parity), half_view(prec, out, Vh, parity));
}

size_t qxd_face_bytes(const qxd_ctx* c, int prec, int mu) {
  if (!c || prec < 0 || prec >= NPREC || mu < 0 || mu > 3) return 0;
  return face_bytes(c, prec, mu);
}
static int check_halo(qxd_ctx* c, int prec, const void* a, const void* b, int pmask, int mu, const char* who) {
  if (!c) return QXD_EINVAL;
  if (!a || !b) return fail(c, QXD_EINVAL, std::string(who) + ": null pointer");
  if (!c->ws) return fail(c, QXD_EWORKSPACE, std::string(who) + ": no workspace bound");
  if (prec < 0 || prec >= NPREC || pmask < 1 || pmask > 3 || mu < 0 || mu > 3) return fail(c, QXD_EINVAL, std::string(who) + ": bad precision, parity mask or direction");
  return QXD_OK;
}
int qxd_face_gather(qxd_ctx* c, int prec, const void* packed, int pmask, int mu, int coord, int sign, void* buf) {
  int rc = check_halo(c, prec, packed, buf, pmask, mu, "face_gather");
  if (rc) return rc;
  if (sign != 1 && sign != -1) return fail(c, QXD_EINVAL, "face_gather: sign must be +1 or -1");
  return launch_face_gather(c, prec, const_cast<void*>(packed), pmask, mu, coord, sign, buf);
}
int qxd_face_scatter(qxd_ctx* c, int prec, void* packed, int pmask, int mu, int coord, int shift1, const void* buf) {
  int rc = check_halo(c, prec, packed, buf, pmask, mu, "face_scatter");
  if (rc) return rc;
  return launch_face_scatter(c, prec, packed, pmask, mu, coord, shift1, buf);
}
int qxd_halo_zero(qxd_ctx* c, int prec, void* packed, int pmask, int mu, int lo, int hi) {
  int rc = check_halo(c, prec, packed, packed, pmask, mu, "halo_zero");
  if (rc) return rc;
  return launch_halo_zero(c, prec, packed, pmask, mu, lo, hi);
}
static bool blas_args_ok(qxd_ctx* c, int prec) { return c && c->ws && prec >= 0 && prec < NPREC; }
static SpinorPtr hp(qxd_ctx* c, int prec, const void* p) { return half_view(prec, const_cast<void*>(p), c->g.Vh, 0); }
int qxd_blas_norm2_dev(qxd_ctx* c, int prec, const void* x, double* out) {
  if (!blas_args_ok(c, prec) || !x || !out) return QXD_EINVAL;
  return blas_norm2(c, prec, hp(c, prec, x), out, Batch(), true);
}
int qxd_blas_cg_xr(qxd_ctx* c, int prec, const double* num, const double* den, const void* p, const void* t, void* x, void* r, double* rr) {
  if (!blas_args_ok(c, prec) || !num || !den || !p || !t || !x || !r || !rr) return QXD_EINVAL;
  return blas_cg_xr(c, prec, num, den, hp(c, prec, p), hp(c, prec, t), hp(c, prec, x), hp(c, prec, r), rr);
}
int qxd_blas_cg_p(qxd_ctx* c, int prec, const double* num, const double* den, const void* s, void* p) {
  if (!blas_args_ok(c, prec) || !num || !den || !s || !p) return QXD_EINVAL;
  return blas_cg_p(c, prec, num, den, hp(c, prec, s), hp(c, prec, p));
}
int qxd_blas_cg_xr_h(qxd_ctx* c, const double* num, const double* den, const void* p16, const void* t16, void* x32, void* r32, void* r16, double* rr) {
  if (!blas_args_ok(c, 1) || !blas_args_ok(c, 2) || !num || !den || !p16 || !t16 || !x32 || !r32 || !r16 || !rr) return QXD_EINVAL;
  SpinorPtr x = hp(c, 1, x32), r = hp(c, 1, r32);
  x.scale = nullptr; r.scale = nullptr;
  return blas_cg_xr_h(c, num, den, hp(c, 2, p16), hp(c, 2, t16), x, r, hp(c, 2, r16), rr);
}
int qxd_blas_cg_p_h(qxd_ctx* c, const double* num, const double* den, const void* s16, void* p32, void* p16) {
  if (!blas_args_ok(c, 1) || !blas_args_ok(c, 2) || !num || !den || !s16 || !p32 || !p16) return QXD_EINVAL;
  SpinorPtr p = hp(c, 1, p32);
  p.scale = nullptr;
  return blas_cg_p_h(c, num, den, hp(c, 2, s16), p, hp(c, 2, p16));
}
int qxd_blas_copy(qxd_ctx* c, int prec, const void* x, void* y) {
  if (!blas_args_ok(c, prec) || !x || !y) return QXD_EINVAL;
  return blas_copy(c, prec, hp(c, prec, x), hp(c, prec, y));
}
int qxd_blas_zero(qxd_ctx* c, int prec, void* x) {
  if (!blas_args_ok(c, prec) || !x) return QXD_EINVAL;
  return blas_zero(c, prec, hp(c, prec, x));
}
int qxd_blas_convert(qxd_ctx* c, int prec_from, const void* x, int prec_to, void* y) {
  if (!blas_args_ok(c, prec_from) || !blas_args_ok(c, prec_to) || !x || !y) return QXD_EINVAL;
  return launch_convert_spinor(c, prec_from, hp(c, prec_from, x), prec_to, hp(c, prec_to, y));
}
int qxd_blas_acc_hi(qxd_ctx* c, int prec, void* x_lo, void* x_hi) {
  if (!blas_args_ok(c, prec) || !x_lo || !x_hi) return QXD_EINVAL;
  return blas_acc_hi(c, prec, hp(c, prec, x_lo), hp(c, 0, x_hi));
}
int qxd_blas_sub_norm_dev(qxd_ctx* c, int prec, const void* b, const void* t, void* r, double* rr) {
  if (!blas_args_ok(c, prec) || !b || !t || !r || !rr) return QXD_EINVAL;
  return blas_sub_norm(c, prec, hp(c, prec, b), hp(c, prec, t), hp(c, prec, r), rr);
}

int qxd_solve(qxd_ctx* c, const double* eta, double* psi, double tol, qxd_solve_info* info) {
  qxd_solve_info local;
  if (!info) { std::memset(&local, 0, sizeof(local)); info = &local; }
  int rc = check_apply(c, info->sloppy, eta, psi, "solve");
  if (rc) return rc;
  if (info->algo == QXD_GCR || info->algo == QXD_DFL_GCR) return solve_gcr(c, eta, psi, tol, info);
  if (info->algo != QXD_CGNE && info->algo != QXD_BICGSTAB) return fail(c, QXD_EINVAL, "solve: unknown algorithm");
  return solve_eo(c, eta, psi, tol, info);
}

int qxd_set_gcr(qxd_ctx* c, int nkv, int ncy, int nmr) {
  if (!c) return QXD_EINVAL;
  if (c->ws) return fail(c, QXD_ESTATE, "qxd_set_gcr must precede qxd_workspace_bind");
  if (nkv < 0 || nkv > 32 || ncy < 0 || nmr < 0) return fail(c, QXD_EINVAL, "set_gcr: 0 <= nkv <= 32, ncy >= 0, nmr >= 0");
  c->gcr_nkv = nkv; c->gcr_ncy = ncy > 0 ? ncy : 4; c->gcr_nmr = nmr > 0 ? nmr : 4;
  return QXD_OK;
}

int qxd_set_deflation(qxd_ctx* c, int ns, int ninv, int nkc, int nref) {
  if (!c) return QXD_EINVAL;
  if (c->ws) return fail(c, QXD_ESTATE, "qxd_set_deflation must precede qxd_workspace_bind");
  if (ns < 0 || ns > 32 || (ns & 1) || ninv < 0 || nkc < 0 || nkc > 32 || nref < 0) return fail(c, QXD_EINVAL, "set_deflation: ns even in 0..32, ninv >= 0, 0 <= nkc <= 32, nref >= 0");
  if (c->dfl_chiral && ns > 16) return fail(c, QXD_EINVAL, "set_deflation: at most 16 null vectors with the chirality split");
  c->dfl_ns = ns; c->dfl_ninv = ninv > 0 ? ninv : 4; c->dfl_nkc = nkc > 0 ? nkc : 16; c->dfl_nref = nref;
  return QXD_OK;
}
int qxd_set_deflation_refine(qxd_ctx* c, int nref, int steps) {
  if (!c) return QXD_EINVAL;
  if (nref < 0 || steps < 1 || steps > 16) return fail(c, QXD_EINVAL, "set_deflation_refine: nref >= 0, 1 <= steps <= 16");
  c->dfl_nref = nref; c->dfl_refk = steps;
  return QXD_OK;
}
int qxd_set_deflation_chirality(qxd_ctx* c, int on) {
  if (!c) return QXD_EINVAL;
  if (c->ws) return fail(c, QXD_ESTATE, "qxd_set_deflation_chirality must precede qxd_workspace_bind");
  if (on != 0 && on != 1) return fail(c, QXD_EINVAL, "set_deflation_chirality: 0 or 1");
  if (on && c->dfl_ns > 16) return fail(c, QXD_EINVAL, "set_deflation_chirality: at most 16 null vectors (32 coarse degrees of freedom per block)");
  c->dfl_chiral = on;
  return QXD_OK;
}
int qxd_deflation_setup(qxd_ctx* c, int prec, const void* random_vectors) {
  int rc = check_apply(c, prec, random_vectors, random_vectors, "deflation_setup");
  if (rc) return rc;
  if (c->dfl_ns < 2 || !c->dphi[0]) return fail(c, QXD_EWORKSPACE, "deflation_setup: call qxd_set_deflation before qxd_workspace_bind");
  if (c->gcr_nkv < 1) return fail(c, QXD_EWORKSPACE, "deflation_setup: needs the SAP workspace (qxd_set_gcr)");
  if (!prec_ok(c, 1) || (prec != 1 && prec != 2)) return fail(c, QXD_EINVAL, "deflation_setup: fp32 must be bound; block operator in fp32 or binary16");
  return dfl_setup(c, prec, random_vectors);
}
int qxd_deflation_info(const qxd_ctx* c, int* nblocks, int* ns, int* ready) {
  if (!c || !nblocks || !ns || !ready) return QXD_EINVAL;
  *nblocks = c->g.Vh / 128; *ns = c->dfl_ns * (c->dfl_chiral ? 2 : 1); *ready = c->dfl_ready ? 1 : 0;
  return QXD_OK;
}
int qxd_deflation_op(qxd_ctx* c, int op, const void* in, void* out) {
  if (!c || !in || !out) return QXD_EINVAL;
  if (!c->dfl_ready) return fail(c, QXD_ESTATE, "deflation_op: call qxd_deflation_setup first");
  switch (op) {
    case 0: return dfl_restrict(c, in, out);
    case 1: return dfl_prolong(c, in, out);
    case 2: return dfl_coarse_apply(c, in, out);
    case 3: return launch_dfl_precond(c, c->dfl_prec, in, out);
    case 4: return dfl_coarse_solve(c, in, out);
    default: return fail(c, QXD_EINVAL, "deflation_op: 0 restrict, 1 prolong, 2 coarse operator, 3 two-level preconditioner, 4 coarse solve");
  }
}

int qxd_sap_block_of(qxd_ctx* c, int cb, int parity, int* block, int* colour) {
  if (!c || !block || !colour || cb < 0 || cb >= c->g.Vh || parity < 0 || parity > 1) return QXD_EINVAL;
  int rc = sap_check_geometry(c);
  if (rc) return rc;
  int x[4];
  coords_int(c->g, c->g.pair ? (cb >> 1) : cb, parity, x);
  int col = 0;
  for (int mu = 0; mu < 4; mu++) if (c->sap_colmask[mu]) col += x[mu] >> c->sap_boxsh[mu];
  *block = cb >> 7; *colour = col & 1;
  return QXD_OK;
}

int qxd_apply_sap(qxd_ctx* c, int prec, const void* in, void* out) {
  int rc = check_apply(c, prec, in, out, "apply_sap");
  if (rc) return rc;
  if (c->gcr_nkv < 1) return fail(c, QXD_EWORKSPACE, "apply_sap: call qxd_set_gcr before qxd_workspace_bind");
  if (!prec_ok(c, 1)) return fail(c, QXD_EINVAL, "apply_sap: fp32 must be bound (the preconditioner works on fp32 vectors)");
  return launch_sap(c, prec, in, out);
}

int qxd_solve_multi(qxd_ctx* c, int nrhs, const double* eta, double* psi, double tol, qxd_solve_info* info) {
  if (!c || !info) return c ? fail(c, QXD_EINVAL, "solve_multi: info array is null") : QXD_EINVAL;
  int rc = check_apply(c, info[0].sloppy, eta, psi, "solve_multi");
  if (rc) return rc;
  if (c->nrhs < 2 || !c->mscal) return fail(c, QXD_EWORKSPACE, "solve_multi: bind the workspace with nrhs > 1");
  return solve_eo_multi(c, nrhs, eta, psi, tol, info);
}

int qxd_solve_host(qxd_ctx* c, const double* eta_host, double* psi_host, double tol, qxd_solve_info* info) {
  if (!c || !eta_host || !psi_host) return c ? fail(c, QXD_EINVAL, "solve_host: null pointer") : QXD_EINVAL;
  if (!c->ws) return fail(c, QXD_EWORKSPACE, "solve_host: no workspace bound");
  const size_t bytes = size_t(c->V) * 24 * sizeof(double);
  QXD_CUDA_OK(c, cudaMemcpyAsync(c->nat_a, eta_host, bytes, cudaMemcpyHostToDevice, c->stream));
  int rc = qxd_solve(c, c->nat_a, c->nat_b, tol, info);
  if (rc != QXD_OK && rc != QXD_ENOCONV) return rc;
  QXD_CUDA_OK(c, cudaMemcpyAsync(psi_host, c->nat_b, bytes, cudaMemcpyDeviceToHost, c->stream));
  QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
  return rc;
}

size_t qxd_packed_spinor_bytes(const qxd_ctx* c, int prec, int half_only) {
  if (!c || prec < 0 || prec >= NPREC) return 0;
  return half_bytes(prec, c->g.Vh) * (half_only ? 1 : 2);
}

int qxd_spinor_pack(qxd_ctx* c, int prec, const double* nat, void* packed) {
  if (!c || !nat || !packed || prec < 0 || prec >= NPREC) return QXD_EINVAL;
  return launch_spinor_pack(c, prec, nat, packed, 3, 0);
}
int qxd_spinor_unpack(qxd_ctx* c, int prec, const void* packed, double* nat) {
  if (!c || !nat || !packed || prec < 0 || prec >= NPREC) return QXD_EINVAL;
  return launch_spinor_unpack(c, prec, packed, nat, 3, 0);
}

static int read_result(qxd_ctx* c, int n, double* out) {
  QXD_CUDA_OK(c, cudaMemcpyAsync(c->h_scal + 32, c->scal + 32, sizeof(double) * n, cudaMemcpyDeviceToHost, c->stream));
  QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
  for (int i = 0; i < n; i++) out[i] = c->h_scal[32 + i];
  return QXD_OK;
}

int qxd_blas_axpy(qxd_ctx* c, int prec, double a, const void* x, void* y) {
  if (!c || !x || !y || prec < 0 || prec >= NPREC || !c->ws) return QXD_EINVAL;
  return blas_axpy(c, prec, a, half_view(prec, const_cast<void*>(x), c->g.Vh, 0), half_view(prec, y, c->g.Vh, 0));
}
int qxd_blas_cdot(qxd_ctx* c, int prec, const void* x, const void* y, double* re_im) {
  if (!c || !x || !y || !re_im || prec < 0 || prec >= NPREC || !c->ws) return QXD_EINVAL;
  int rc = blas_cdot(c, prec, half_view(prec, const_cast<void*>(x), c->g.Vh, 0), half_view(prec, const_cast<void*>(y), c->g.Vh, 0), c->scal + 32, true);
  if (rc) return rc;
  return read_result(c, 2, re_im);
}
int qxd_blas_norm2(qxd_ctx* c, int prec, const void* x, double* out) {
  if (!c || !x || !out || prec < 0 || prec >= NPREC || !c->ws) return QXD_EINVAL;
  int rc = blas_norm2(c, prec, half_view(prec, const_cast<void*>(x), c->g.Vh, 0), c->scal + 32, Batch(), true);
  if (rc) return rc;
  return read_result(c, 1, out);
}

long qxd_launch_count(const qxd_ctx* c) { return c ? c->launches : 0; }
const char* qxd_last_error(const qxd_ctx* c) { return c ? c->err.c_str() : "null context"; }

}  // extern "C"
