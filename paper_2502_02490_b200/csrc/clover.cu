// clover.cu -- SURVEY.md §8 row a3: on-device construction and inversion of the QCD+QED clover term.
// The paper computes this term on the CPU and uploads it and names its generation
// on the GPU as the next step; this file is that step.
//
//   M(x) = (4+m0) + c_sw (i/4) sum_{mu,nu} sigma_{mu nu} F-hat_{mu nu}(x)
//                 + q c_sw^{U(1)} (i/4) sum_{mu,nu} sigma_{mu nu} A-hat_{mu nu}(x)      (R1,R4,R5)
//
// In the chiral basis of reading R3 the term is block diagonal in chirality:
//   M_+- = (4+m0) + sum_k sigma_k (x) C^{+-}_k ,   C^{+-}_k = (i/2)(+-E_k - B_k),
//   E_k = X_{0k},  B_1 = X_{23}, B_2 = X_{31}, B_3 = X_{12},  X = c_sw F-hat + q c_sw^{U(1)} A-hat 1.
// Each block is stored as 36 reals in the order of PAPER.md:117.
#include "qxd_ctx.h"

namespace qxd {

namespace {

typedef double m3[18];  // 3x3 complex, row-major (re,im)

__device__ __forceinline__ void m3_mul(const double* a, const double* b, double* c) {  // c = a b
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      double re = 0, im = 0;
#pragma unroll
      for (int k = 0; k < 3; k++) {
        double ar = a[2 * (3 * i + k)], ai = a[2 * (3 * i + k) + 1], br = b[2 * (3 * k + j)], bi = b[2 * (3 * k + j) + 1];
        re += ar * br - ai * bi; im += ar * bi + ai * br;
      }
      c[2 * (3 * i + j)] = re; c[2 * (3 * i + j) + 1] = im;
    }
}
__device__ __forceinline__ void m3_mul_adj(const double* a, const double* b, double* c) {  // c = a b^dag
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      double re = 0, im = 0;
#pragma unroll
      for (int k = 0; k < 3; k++) {
        double ar = a[2 * (3 * i + k)], ai = a[2 * (3 * i + k) + 1], br = b[2 * (3 * j + k)], bi = -b[2 * (3 * j + k) + 1];
        re += ar * br - ai * bi; im += ar * bi + ai * br;
      }
      c[2 * (3 * i + j)] = re; c[2 * (3 * i + j) + 1] = im;
    }
}
__device__ __forceinline__ void m3_adj_mul(const double* a, const double* b, double* c) {  // c = a^dag b
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      double re = 0, im = 0;
#pragma unroll
      for (int k = 0; k < 3; k++) {
        double ar = a[2 * (3 * k + i)], ai = -a[2 * (3 * k + i) + 1], br = b[2 * (3 * k + j)], bi = b[2 * (3 * k + j) + 1];
        re += ar * br - ai * bi; im += ar * bi + ai * br;
      }
      c[2 * (3 * i + j)] = re; c[2 * (3 * i + j) + 1] = im;
    }
}

struct GaugePtrs { const void* U[2]; const void* A[2]; };

// links and A of a site; in the paired layout the records are those of the physical site and the mirror image
// (mirror bit = 1) takes U^* and -A (reading R8).  The plaquette arithmetic keeps only a handle of a neighbour site alive
// (record index, parity, mirror bit), and the plane (mu, nu) is a run-time argument: six unrolled template instances of
// the 12 matrix products were ~250 KB of code, and the kernel spent its time waiting for instructions
// (ncu: stall_no_instruction 11.5 per issue).
__device__ __forceinline__ int site_ref(const Site& s) { return ((s.idx2 >> 1) << 2) | (site_parity(s) << 1) | s.m; }
__device__ __forceinline__ void link_ref(const GaugePtrs& P, const Geom& g, int mu, int ref, double* m) {
  const double2* p = reinterpret_cast<const double2*>(P.U[(ref >> 1) & 1]) + size_t(9 * mu) * g.Vg + (ref >> 2);
  const double sg = (ref & 1) ? -1.0 : 1.0;
#pragma unroll
  for (int c = 0; c < 9; c++) {
    const double2 v = __ldg(p + size_t(c) * g.Vg);
    m[2 * c] = v.x; m[2 * c + 1] = sg * v.y;
  }
}
__device__ __forceinline__ double a_at(const GaugePtrs& P, const Geom& g, int mu, const Site& s) {
  const double a = __ldg(reinterpret_cast<const double*>(P.A[site_parity(s)]) + (size_t(mu >> 1) * g.Vg + (s.idx2 >> 1)) * 2 + (mu & 1));
  return s.m ? -a : a;
}
__device__ __forceinline__ double phi_at(const GaugePtrs& P, const Geom& g, int mu, int nu, const Site& y) {
  Site ypm, ypn;
  site_step(g, y, mu, +1, ypm);
  site_step(g, y, nu, +1, ypn);
  return a_at(P, g, mu, y) + a_at(P, g, nu, ypm) - a_at(P, g, mu, ypn) - a_at(P, g, nu, y);
}

// X_{mu nu}(x) = csw F-hat_{mu nu} + q csw_qed A-hat_{mu nu} 1   (anti-Hermitian 3x3)
__device__ __forceinline__ void plane_X(const GaugePtrs& P, const Geom& g, const Site& x, int mu, int nu, double csw, double qcq, double qel,
                                        int use_a, double* X) {
  int r_x, r_pm, r_pn, r_mm, r_mn, r_mmpn, r_mmmn, r_pmmn;
  {
    Site y, z;
    r_x = site_ref(x);
    site_step(g, x, mu, +1, y); r_pm = site_ref(y);
    site_step(g, y, nu, -1, z); r_pmmn = site_ref(z);
    site_step(g, x, nu, +1, y); r_pn = site_ref(y);
    site_step(g, x, nu, -1, y); r_mn = site_ref(y);
    site_step(g, x, mu, -1, y); r_mm = site_ref(y);
    site_step(g, y, nu, +1, z); r_mmpn = site_ref(z);
    site_step(g, y, nu, -1, z); r_mmmn = site_ref(z);
  }
  double Q[18];
#pragma unroll
  for (int i = 0; i < 18; i++) Q[i] = 0.0;
  if (csw != 0.0) {
    m3 a, b, t1, t2, t3;
    // leaf 1: U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
    link_ref(P, g, mu, r_x, a); link_ref(P, g, nu, r_pm, b); m3_mul(a, b, t1);
    link_ref(P, g, mu, r_pn, a); m3_mul_adj(t1, a, t2);
    link_ref(P, g, nu, r_x, a); m3_mul_adj(t2, a, t3);
#pragma unroll
    for (int i = 0; i < 18; i++) Q[i] += t3[i];
    // leaf 2: U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
    link_ref(P, g, nu, r_x, a); link_ref(P, g, mu, r_mmpn, b); m3_mul_adj(a, b, t1);
    link_ref(P, g, nu, r_mm, a); m3_mul_adj(t1, a, t2);
    link_ref(P, g, mu, r_mm, a); m3_mul(t2, a, t3);
#pragma unroll
    for (int i = 0; i < 18; i++) Q[i] += t3[i];
    // leaf 3: U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
    link_ref(P, g, nu, r_mmmn, a); link_ref(P, g, mu, r_mm, b); m3_mul(a, b, t1);   // (U_nu(x-mu-nu) U_mu(x-mu))
    link_ref(P, g, mu, r_mmmn, a); m3_adj_mul(t1, a, t2);                           // ^dag * U_mu(x-mu-nu)
    link_ref(P, g, nu, r_mn, a); m3_mul(t2, a, t3);
#pragma unroll
    for (int i = 0; i < 18; i++) Q[i] += t3[i];
    // leaf 4: U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
    link_ref(P, g, nu, r_mn, a); link_ref(P, g, mu, r_mn, b); m3_adj_mul(a, b, t1);
    link_ref(P, g, nu, r_pmmn, a); m3_mul(t1, a, t2);
    link_ref(P, g, mu, r_x, a); m3_mul_adj(t2, a, t3);
#pragma unroll
    for (int i = 0; i < 18; i++) Q[i] += t3[i];
  }
  // F-hat = (Q - Q^dag)/8
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      X[2 * (3 * i + j)] = csw * 0.125 * (Q[2 * (3 * i + j)] - Q[2 * (3 * j + i)]);
      X[2 * (3 * i + j) + 1] = csw * 0.125 * (Q[2 * (3 * i + j) + 1] + Q[2 * (3 * j + i) + 1]);
    }
  if (use_a && qcq != 0.0) {
    // A-hat = (i/(4 qel)) sum over the four leaves of sin(qel Phi)
    Site xmm, xmn, xmmmn;
    site_step(g, x, mu, -1, xmm); site_step(g, x, nu, -1, xmn); site_step(g, xmm, nu, -1, xmmmn);
    double s = sin(qel * phi_at(P, g, mu, nu, x)) + sin(qel * phi_at(P, g, mu, nu, xmm)) + sin(qel * phi_at(P, g, mu, nu, xmn)) +
               sin(qel * phi_at(P, g, mu, nu, xmmmn));
    double ah = qcq * s / (4.0 * qel);
    X[1] += ah; X[9] += ah; X[17] += ah;  // imaginary parts of the diagonal
  }
}

// C += sign * (i/2) X
__device__ __forceinline__ void acc_C(const double* X, double sign, double* C) {
#pragma unroll
  for (int k = 0; k < 9; k++) {
    C[2 * k] += sign * (-0.5 * X[2 * k + 1]);
    C[2 * k + 1] += sign * (0.5 * X[2 * k]);
  }
}

// write sigma_k (x) C contributions into a packed block (PAPER.md:117 order)
__device__ __forceinline__ int upper_index(int i, int j) {  // i<j, position among the 15 pairs, row-major
  return i * 6 - (i * (i + 1)) / 2 + (j - i - 1);
}
__device__ __forceinline__ void block_from_C(double diag, const double* C1, const double* C2, const double* C3, double* blk) {
  // block = diag + [[C3, C1 - i C2],[C1 + i C2, -C3]]
#pragma unroll
  for (int a = 0; a < 3; a++) {
    blk[a] = diag + C3[2 * (3 * a + a)];
    blk[3 + a] = diag - C3[2 * (3 * a + a)];
  }
#pragma unroll
  for (int a = 0; a < 3; a++)
#pragma unroll
    for (int b = 0; b < 3; b++) {
      if (b > a) {
        int k0 = 6 + 2 * upper_index(a, b);
        blk[k0] = C3[2 * (3 * a + b)]; blk[k0 + 1] = C3[2 * (3 * a + b) + 1];
        int k1 = 6 + 2 * upper_index(3 + a, 3 + b);
        blk[k1] = -C3[2 * (3 * a + b)]; blk[k1 + 1] = -C3[2 * (3 * a + b) + 1];
      }
      // (C1 - i C2)[a][b]
      int k2 = 6 + 2 * upper_index(a, 3 + b);
      blk[k2] = C1[2 * (3 * a + b)] + C2[2 * (3 * a + b) + 1];
      blk[k2 + 1] = C1[2 * (3 * a + b) + 1] - C2[2 * (3 * a + b)];
    }
}

// One thread per (site, plane): the six anti-Hermitian X_{mu nu} of a site are built by six warps of the CTA (a warp = one
// plane of 32 consecutive sites, so the template choice is warp-uniform and the link loads coalesce), parked in shared memory,
// and two threads per site then assemble the two chirality blocks.  (One thread per site held 2 x 54 accumulators next to
// the plane arithmetic: 255 registers and 428 B of spills.)
constexpr int CB_SITES = 32;
__global__ void __launch_bounds__(6 * CB_SITES, 2) clover_build_k(Geom g, GaugePtrs P, double diag, double csw, double qcq, double qel, int use_a,
                                                                void* M0, void* M1) {
  __shared__ double Xs[6][18][CB_SITES];
  const int lane = threadIdx.x & (CB_SITES - 1), pl = threadIdx.x / CB_SITES;
  const int cb = blockIdx.x * CB_SITES + lane;   // index of the clover record (physical site in the paired layout)
  const int parity = blockIdx.y;
  const bool act = cb < g.Vg;
  if (act) {
    Site x;
    site_init(g, g.pair ? 2 * cb : cb, parity, x);
    double X[18];
    // planes in the order E_1 = X_01, B_1 = X_23, E_2 = X_02, X_13 = -B_2, E_3 = X_03, B_3 = X_12
    const int mu = (0x101020 >> (4 * pl)) & 3, nu = (0x233231 >> (4 * pl)) & 3;
    plane_X(P, g, x, mu, nu, csw, qcq, qel, use_a, X);
#pragma unroll
    for (int i = 0; i < 18; i++) Xs[pl][i][lane] = X[i];
  }
  __syncthreads();
  if (!act || pl >= 2) return;
  // chirality block pl (0: C^+, 1: C^-).  E_k = X_{0k}: C^+ += (i/2) E, C^- -= (i/2) E;  B_k: C^+- -= (i/2) B  (B_2 = -X_13)
  double C[3][18], X[18];
#pragma unroll
  for (int k = 0; k < 3; k++) {
#pragma unroll
    for (int i = 0; i < 18; i++) C[k][i] = 0.0;
#pragma unroll
    for (int i = 0; i < 18; i++) X[i] = Xs[2 * k][i][lane];
    acc_C(X, pl == 0 ? +1.0 : -1.0, C[k]);
#pragma unroll
    for (int i = 0; i < 18; i++) X[i] = Xs[2 * k + 1][i][lane];
    acc_C(X, k == 1 ? +1.0 : -1.0, C[k]);
  }
  double out[36];
  block_from_C(diag, C[0], C[1], C[2], out);
  typedef PT<double>::V V;
  V* q = reinterpret_cast<V*>(parity ? M1 : M0);
#pragma unroll
  for (int k = 0; k < 18; k++) q[size_t(18 * pl + k) * g.Vg + cb] = make_double2(out[2 * k], out[2 * k + 1]);
}

// Fast path of the block inversion: in-place Gauss-Jordan WITHOUT pivoting, fully unrolled so that the 6x6 complex matrix
// lives in registers (the pivoted kernel below indexes its arrays at run time and works out of 2.3 KB of local memory:
// 9.7 ms per parity at c3 against ~1 ms here).  The blocks are (4 + m0) + O(c_sw F): diagonally dominant for every
// sensible field, so the unpivoted elimination is stable; a pivot below 1e-6 of the largest diagonal entry raises
// flag[1] and the caller redoes the parity with the pivoted kernel.  One thread per (site, chirality block).
__global__ void __launch_bounds__(128) clover_invert_fast_k(int Vh, const void* M, void* Mi, int* flag) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int cb = t >> 1, c = t & 1;
  if (cb >= Vh) return;
  double p[36];
  if (c == 0) load_reals<double, 0, 36>(M, Vh, cb, p); else load_reals<double, 36, 36>(M, Vh, cb, p);
  double ar[6][6], ai[6][6];
  double dmax = 0.0;
#pragma unroll
  for (int i = 0; i < 6; i++) {
    ar[i][i] = p[i]; ai[i][i] = 0.0;
    dmax = fmax(dmax, fabs(p[i]));
#pragma unroll
    for (int j = i + 1; j < 6; j++) {
      const int k = 6 + 2 * upper_index(i, j);
      ar[i][j] = p[k]; ai[i][j] = p[k + 1];
      ar[j][i] = p[k]; ai[j][i] = -p[k + 1];
    }
  }
  bool bad = false;
#pragma unroll
  for (int k = 0; k < 6; k++) {
    const double m2 = ar[k][k] * ar[k][k] + ai[k][k] * ai[k][k];
    if (!(m2 > 1e-12 * dmax * dmax)) bad = true;
    const double dr = ar[k][k] / m2, di = -ai[k][k] / m2;   // 1 / pivot
    ar[k][k] = 1.0; ai[k][k] = 0.0;
#pragma unroll
    for (int j = 0; j < 6; j++) {
      const double xr = ar[k][j], xi = ai[k][j];
      ar[k][j] = xr * dr - xi * di; ai[k][j] = xr * di + xi * dr;
    }
#pragma unroll
    for (int i = 0; i < 6; i++) {
      if (i == k) continue;
      const double fr = ar[i][k], fi = ai[i][k];
      ar[i][k] = 0.0; ai[i][k] = 0.0;
#pragma unroll
      for (int j = 0; j < 6; j++) {
        ar[i][j] -= fr * ar[k][j] - fi * ai[k][j];
        ai[i][j] -= fr * ai[k][j] + fi * ar[k][j];
      }
    }
  }
  if (bad) atomicExch(flag + 1, 1);
  double o[36];
#pragma unroll
  for (int i = 0; i < 6; i++) {
    o[i] = ar[i][i];
#pragma unroll
    for (int j = i + 1; j < 6; j++) {
      const int k = 6 + 2 * upper_index(i, j);
      o[k] = 0.5 * (ar[i][j] + ar[j][i]); o[k + 1] = 0.5 * (ai[i][j] - ai[j][i]);   // Hermitian average
    }
  }
  typedef PT<double>::V V;
  V* q = reinterpret_cast<V*>(Mi);
#pragma unroll
  for (int k = 0; k < 18; k++) q[size_t(18 * c + k) * Vh + cb] = make_double2(o[2 * k], o[2 * k + 1]);
}

// Inverse of both Hermitian 6x6 blocks of every site: Gauss-Jordan with partial pivoting in fp64,
// one thread per (site, chirality).  flag[0] is set if a block is numerically singular.
__global__ void __launch_bounds__(64) clover_invert_k(int Vh, const void* M, void* Mi, int* flag) {
  int cb = blockIdx.x * blockDim.x + threadIdx.x;
  if (cb >= Vh) return;
  double in[72], out[72];
  load_reals<double, 0, 72>(M, Vh, cb, in);
  for (int c = 0; c < 2; c++) {
    double ar[6][6], ai[6][6], br[6][6], bi[6][6];
    const double* p = in + 36 * c;
    for (int i = 0; i < 6; i++) {
      for (int j = 0; j < 6; j++) { br[i][j] = (i == j) ? 1.0 : 0.0; bi[i][j] = 0.0; }
      ar[i][i] = p[i]; ai[i][i] = 0.0;
      for (int j = i + 1; j < 6; j++) {
        int k = 6 + 2 * upper_index(i, j);
        ar[i][j] = p[k]; ai[i][j] = p[k + 1];
        ar[j][i] = p[k]; ai[j][i] = -p[k + 1];
      }
    }
    for (int col = 0; col < 6; col++) {
      int piv = col; double best = ar[col][col] * ar[col][col] + ai[col][col] * ai[col][col];
      for (int r = col + 1; r < 6; r++) { double m = ar[r][col] * ar[r][col] + ai[r][col] * ai[r][col]; if (m > best) { best = m; piv = r; } }
      if (!(best > 1e-300)) { atomicExch(flag, 1); best = 1.0; }
      if (piv != col)
        for (int j = 0; j < 6; j++) {
          double t;
          t = ar[piv][j]; ar[piv][j] = ar[col][j]; ar[col][j] = t; t = ai[piv][j]; ai[piv][j] = ai[col][j]; ai[col][j] = t;
          t = br[piv][j]; br[piv][j] = br[col][j]; br[col][j] = t; t = bi[piv][j]; bi[piv][j] = bi[col][j]; bi[col][j] = t;
        }
      double dr = ar[col][col] / best, di = -ai[col][col] / best;  // 1/pivot
      for (int j = 0; j < 6; j++) {
        double xr = ar[col][j], xi = ai[col][j];
        ar[col][j] = xr * dr - xi * di; ai[col][j] = xr * di + xi * dr;
        xr = br[col][j]; xi = bi[col][j];
        br[col][j] = xr * dr - xi * di; bi[col][j] = xr * di + xi * dr;
      }
      for (int r = 0; r < 6; r++) {
        if (r == col) continue;
        double fr = ar[r][col], fi = ai[r][col];
        for (int j = 0; j < 6; j++) {
          ar[r][j] -= fr * ar[col][j] - fi * ai[col][j]; ai[r][j] -= fr * ai[col][j] + fi * ar[col][j];
          br[r][j] -= fr * br[col][j] - fi * bi[col][j]; bi[r][j] -= fr * bi[col][j] + fi * br[col][j];
        }
      }
    }
    double* o = out + 36 * c;
    for (int i = 0; i < 6; i++) {
      o[i] = br[i][i];
      for (int j = i + 1; j < 6; j++) {
        int k = 6 + 2 * upper_index(i, j);
        // Hermitian average of the (i,j) and (j,i) entries
        o[k] = 0.5 * (br[i][j] + br[j][i]); o[k + 1] = 0.5 * (bi[i][j] - bi[j][i]);
      }
    }
  }
  store_record<double, 72>(Mi, Vh, cb, out);
}

}  // namespace

int launch_clover_build(qxd_ctx* c) {
  GaugePtrs P;
  P.U[0] = c->Ug[0]; P.U[1] = c->Ug[1]; P.A[0] = c->Ag[0]; P.A[1] = c->Ag[1];
  dim3 gr((c->g.Vg + CB_SITES - 1) / CB_SITES, 2);
  double diag = 4.0 + c->m0;
  clover_build_k<<<gr, 6 * CB_SITES, 0, c->stream>>>(c->g, P, diag, c->csw, c->q * c->csw_qed, c->qel, c->have_qed ? 1 : 0, c->M[0][0], c->M[0][1]);
  QXD_LAUNCH_CHECK(c);
  int* flag = reinterpret_cast<int*>(c->scal + 60);
  QXD_CUDA_OK(c, cudaMemsetAsync(flag, 0, 2 * sizeof(int), c->stream));
  for (int p = 0; p < 2; p++) {
    clover_invert_fast_k<<<(2 * c->g.Vg + 127) / 128, 128, 0, c->stream>>>(c->g.Vg, c->M[0][p], c->Mi[0][p], flag);
    QXD_LAUNCH_CHECK(c);
    c->n_inv_fast++;
  }
  int hflag[2] = {0, 0};
  QXD_CUDA_OK(c, cudaMemcpyAsync(hflag, flag, 2 * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
  QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
  if (hflag[1]) {   // a small pivot somewhere: redo with partial pivoting
    for (int p = 0; p < 2; p++) {
      clover_invert_k<<<(c->g.Vg + 63) / 64, 64, 0, c->stream>>>(c->g.Vg, c->M[0][p], c->Mi[0][p], flag);
      QXD_LAUNCH_CHECK(c);
      c->n_inv_pivoted++;
    }
    QXD_CUDA_OK(c, cudaMemcpyAsync(hflag, flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    QXD_CUDA_OK(c, cudaStreamSynchronize(c->stream));
  }
  if (hflag[0]) return fail(c, QXD_EINVAL, "clover_build: a clover block is singular");
  for (int pr = 1; pr < NPREC; pr++) {
    if (!((c->prec_mask >> pr) & 1)) continue;
    for (int p = 0; p < 2; p++) {
      int rc = launch_convert_record72(c, c->M[0][p], pr, c->M[pr][p]);
      if (rc) return rc;
      if (!c->Mi[pr][p]) continue;   // even-site inverses are kept in fp64 only (api.cu: carve)
      rc = launch_convert_record72(c, c->Mi[0][p], pr, c->Mi[pr][p]);
      if (rc) return rc;
    }
  }
  return QXD_OK;
}

}  // namespace qxd
