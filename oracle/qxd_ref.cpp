// =====================================================================================
// oracle/qxd_ref.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct fp64 CPU implementation of what the hot path computes:
// the O(a)-improved (clover) Wilson-Dirac operator D_w with SU(3)xU(1) links and C*
// spatial boundary conditions, its even-odd Schur complement D-hat, and the solution of
// D_w psi = eta.  It shares NO code with the CUDA path
// (paper_2502_02490_b200/csrc) and neither includes the other.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
//
// The paper never writes the operator down (it defers to refs [1][2]);
// the definition implemented here is the reading recorded in DESIGN.md "Readings"
// (= SURVEY.md §8(c)).  Every function cites the passage / reading it follows.
//
// Design rules of this file: natural-order array-of-structs fields on the explicitly
// stored EXTENDED lattice, generic 4x4 gamma / sigma matrices (x) 3x3 colour matrices,
// a dense 12x12 site matrix built from sigma_{mu nu} (x) X_{mu nu} (the chirality blocks
// are only EXTRACTED from it afterwards), no half-spinor projection, no 12-real
// reconstruct, no even-odd storage, no blocking, no fusion.  OpenMP over sites only.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): free-field momentum-space closed form
// (apply and solve), gamma5-hermiticity, SU(3)xU(1) gauge covariance, C* charge-conjugation
// symmetry, csw=0 -> Wilson, uniform abelian background clover closed form, SU(3)-formula
// on U(3) links -> q*A-hat, dense-matrix brute force with LU on 4^4 (independent numpy
// assembler); the SIGN of both SW terms by tree-level O(a) improvement: in a uniform abelian
// background the lowest Landau level of gamma5 D_w sits at (1 - c_sw) B/2 + O(B^2)
// (test_sw_term_sign_is_the_improving_one; "O(a)-improved").
// PARITY UNPINNED: only the choice of gamma-basis (ordering of the spin components at the
// ABI) relative to the paper's host code -- the paper prints no operator values; every
// chiral basis gives the same operator up to a fixed unitary change of spin components.
// =====================================================================================
#include <complex>
#include <vector>
#include <string>
#include <cmath>
#include <cstring>
#include <cstdio>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
static const cd I_(0.0, 1.0);

namespace {

// ---- gamma matrices: DESIGN.md reading R3; PAPER.md:53 requires a
// chiral basis (clover split in an upper "+" and lower "-" 6x6 block).
struct Gammas {
  cd g[4][4][4];        // gamma_mu
  cd g5[4][4];          // gamma_0 gamma_1 gamma_2 gamma_3
  cd sig[4][4][4][4];   // sigma_{mu nu} = (i/2)[gamma_mu, gamma_nu]
  Gammas() {
    std::memset((void*)g, 0, sizeof(g));
    cd s[4][2][2];  // Pauli matrices 1..3
    s[1][0][0] = 0; s[1][0][1] = 1;   s[1][1][0] = 1;  s[1][1][1] = 0;
    s[2][0][0] = 0; s[2][0][1] = -I_; s[2][1][0] = I_; s[2][1][1] = 0;
    s[3][0][0] = 1; s[3][0][1] = 0;   s[3][1][0] = 0;  s[3][1][1] = -1.0;
    // gamma_0 = [[0,-1],[-1,0]]
    for (int a = 0; a < 2; a++) { g[0][a][2 + a] = -1.0; g[0][2 + a][a] = -1.0; }
    // gamma_k = [[0,-i sigma_k],[i sigma_k,0]]
    for (int k = 1; k < 4; k++)
      for (int a = 0; a < 2; a++)
        for (int b = 0; b < 2; b++) { g[k][a][2 + b] = -I_ * s[k][a][b]; g[k][2 + a][b] = I_ * s[k][a][b]; }
    cd t[4][4], u[4][4];
    mul(g[0], g[1], t); mul(t, g[2], u); mul(u, g[3], g5);
    for (int m = 0; m < 4; m++)
      for (int n = 0; n < 4; n++) {
        cd ab[4][4], ba[4][4];
        mul(g[m], g[n], ab); mul(g[n], g[m], ba);
        for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) sig[m][n][i][j] = 0.5 * I_ * (ab[i][j] - ba[i][j]);
      }
  }
  static void mul(const cd a[4][4], const cd b[4][4], cd c[4][4]) {
    for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { cd z = 0; for (int k = 0; k < 4; k++) z += a[i][k] * b[k][j]; c[i][j] = z; }
  }
};
const Gammas GM;

// ---- 3x3 colour matrices, row-major
struct M3 { cd m[9]; };
inline M3 mul(const M3& a, const M3& b) { M3 c; for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) { cd z = 0; for (int k = 0; k < 3; k++) z += a.m[3 * i + k] * b.m[3 * k + j]; c.m[3 * i + j] = z; } return c; }
inline M3 dag(const M3& a) { M3 c; for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) c.m[3 * i + j] = std::conj(a.m[3 * j + i]); return c; }

struct Ref {
  int T, L1, L2, L3, cstar, antiper;
  int X[4];
  long V;
  double qel = 1.0, kappa = 0, q = 0, m0 = 0, csw = 0, csw_qed = 0;
  bool have_gauge = false, have_quark = false, have_csw = false, have_clover = false;
  std::vector<cd> U;      // [V][4][9]  extended SU(3) links (no phase, no BC sign)
  std::vector<double> A;  // [V][4]     extended U(1) field
  std::vector<cd> Mb;     // [V][2][36] chirality blocks of the site matrix, row-major 6x6
  std::vector<cd> Mi;     // [V][2][36] their inverses
  std::vector<cd> Mb_range;  // blocks of the site range [range_lo, range_hi) only (bounded-sample timing)
  long range_lo = 0, range_hi = 0;
  double max_offdiag = 0; // largest |entry| found outside the two chirality blocks (must be ~0)
  double max_antiherm = 0;// largest |M - M^dag| entry (must be ~0)

  long lex(const int x[4]) const { return ((long(x[0]) * X[1] + x[1]) * X[2] + x[2]) * X[3] + x[3]; }  // Eq. (1), PAPER.md:93, L1->X1
  void coords(long s, int x[4]) const { x[3] = s % X[3]; s /= X[3]; x[2] = s % X[2]; s /= X[2]; x[1] = s % X[1]; x[0] = s / X[1]; }
  int parity(const int x[4]) const { return (x[0] + x[1] + x[2] + x[3]) & 1; }

  // One lattice step x -> x + dir*mu-hat with the boundary conditions of reading R8
  // ("doubling of the lattice in x-direction and ... shifted
  // boundaries").  Returns 1 if the step crossed the time boundary (antiperiodic sign for spinors).
  int hop(const int x[4], int mu, int dir, int y[4]) const {
    y[0] = x[0]; y[1] = x[1]; y[2] = x[2]; y[3] = x[3];
    int c = x[mu] + dir, crossed_t = 0;
    if (c < 0 || c >= X[mu]) {
      c = (c + X[mu]) % X[mu];
      if (mu == 0) crossed_t = 1;
      if (mu >= 2 && mu <= cstar) y[1] = (x[1] + L1) % X[1];
    }
    y[mu] = c;
    return crossed_t;
  }
  M3 link(const int x[4], int mu) const { M3 r; std::memcpy((void*)r.m, (const void*)&U[(lex(x) * 4 + mu) * 9], sizeof(r.m)); return r; }
  double a_(const int x[4], int mu) const { return A.empty() ? 0.0 : A[lex(x) * 4 + mu]; }

  // W_mu(x) = exp(i q A_mu(x)) U_mu(x)
  M3 hoplink(const int x[4], int mu) const {
    M3 r = link(x, mu);
    double ph = q * a_(x, mu);
    cd e(std::cos(ph), std::sin(ph));
    for (int i = 0; i < 9; i++) r.m[i] *= e;
    return r;
  }

  // Q_{mu nu}(x): sum of the four plaquette leaves in the (mu,nu) plane that start and end at x,
  // all with the same orientation (reading R4); SU(3) links only.
  M3 Qleaves(const int x[4], int mu, int nu) const {
    int xpm[4], xpn[4], xmm[4], xmn[4], xmmpn[4], xmmmn[4], xpmmn[4];
    hop(x, mu, +1, xpm); hop(x, nu, +1, xpn); hop(x, mu, -1, xmm); hop(x, nu, -1, xmn);
    hop(xmm, nu, +1, xmmpn); hop(xmm, nu, -1, xmmmn); hop(xpm, nu, -1, xpmmn);
    M3 l1 = mul(mul(link(x, mu), link(xpm, nu)), mul(dag(link(xpn, mu)), dag(link(x, nu))));
    M3 l2 = mul(mul(link(x, nu), dag(link(xmmpn, mu))), mul(dag(link(xmm, nu)), link(xmm, mu)));
    M3 l3 = mul(mul(dag(link(xmm, mu)), dag(link(xmmmn, nu))), mul(link(xmmmn, mu), link(xmn, nu)));
    M3 l4 = mul(mul(dag(link(xmn, nu)), link(xmn, mu)), mul(link(xpmmn, nu), dag(link(x, mu))));
    M3 r;
    for (int i = 0; i < 9; i++) r.m[i] = l1.m[i] + l2.m[i] + l3.m[i] + l4.m[i];
    return r;
  }
  // F-hat_{mu nu}(x) = (1/8)(Q - Q^dag), anti-Hermitian, no trace subtraction (reading R4).
  M3 Fhat(const int x[4], int mu, int nu) const {
    M3 Q = Qleaves(x, mu, nu), Qd = dag(Q), r;
    for (int i = 0; i < 9; i++) r.m[i] = 0.125 * (Q.m[i] - Qd.m[i]);
    return r;
  }
  // Phi_{mu nu}(y) = A_mu(y) + A_nu(y+mu) - A_mu(y+nu) - A_nu(y)
  double Phi(const int y[4], int mu, int nu) const {
    int ypm[4], ypn[4];
    hop(y, mu, +1, ypm); hop(y, nu, +1, ypn);
    return a_(y, mu) + a_(ypm, nu) - a_(ypn, mu) - a_(y, nu);
  }
  // A-hat_{mu nu}(x) = (i/(4 qel)) sum over the leaves at y = x, x-mu, x-nu, x-mu-nu of sin(qel Phi(y))
  // (reading R5; "another SW-term proportional to c_SW^{U(1)}").
  cd Ahat(const int x[4], int mu, int nu) const {
    if (A.empty()) return 0.0;
    int xmm[4], xmn[4], xmmmn[4];
    hop(x, mu, -1, xmm); hop(x, nu, -1, xmn); hop(xmm, nu, -1, xmmmn);
    double s = std::sin(qel * Phi(x, mu, nu)) + std::sin(qel * Phi(xmm, mu, nu)) + std::sin(qel * Phi(xmn, mu, nu)) +
               std::sin(qel * Phi(xmmmn, mu, nu));
    return I_ * (s / (4.0 * qel));
  }

  // Site-diagonal part of D_w (reading R1/R2/R4/R5):
  // M(x) = (4+m0) 1 + csw (i/4) sum_{mu,nu} sigma_{mu nu} (x) F-hat_{mu nu}
  //                 + q csw_qed (i/4) sum_{mu,nu} sigma_{mu nu} A-hat_{mu nu} (x) 1_colour.
  // The sum runs over ALL ordered pairs mu != nu as written (no use of antisymmetry).
  void site_matrix(const int x[4], cd M[144]) const {
    for (int i = 0; i < 144; i++) M[i] = 0;
    for (int i = 0; i < 12; i++) M[13 * i] = 4.0 + m0;
    for (int mu = 0; mu < 4; mu++)
      for (int nu = 0; nu < 4; nu++) {
        if (mu == nu) continue;
        M3 X;
        for (int i = 0; i < 9; i++) X.m[i] = 0;
        if (csw != 0.0) { M3 F = Fhat(x, mu, nu); for (int i = 0; i < 9; i++) X.m[i] += csw * F.m[i]; }
        if (csw_qed != 0.0 && !A.empty()) { cd a = q * csw_qed * Ahat(x, mu, nu); X.m[0] += a; X.m[4] += a; X.m[8] += a; }
        for (int al = 0; al < 4; al++)
          for (int be = 0; be < 4; be++) {
            cd s = 0.25 * I_ * GM.sig[mu][nu][al][be];
            if (s == cd(0.0)) continue;
            for (int a = 0; a < 3; a++)
              for (int b = 0; b < 3; b++) M[(3 * al + a) * 12 + 3 * be + b] += s * X.m[3 * a + b];
          }
      }
  }
};

// dense n x n complex inverse, Gauss-Jordan with partial pivoting (textbook).
bool invert(int n, const cd* a_in, cd* inv) {
  std::vector<cd> a(a_in, a_in + n * n);
  for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) inv[i * n + j] = (i == j) ? 1.0 : 0.0;
  for (int c = 0; c < n; c++) {
    int p = c; double best = std::abs(a[c * n + c]);
    for (int r = c + 1; r < n; r++) if (std::abs(a[r * n + c]) > best) { best = std::abs(a[r * n + c]); p = r; }
    if (best == 0.0) return false;
    if (p != c) for (int j = 0; j < n; j++) { std::swap(a[p * n + j], a[c * n + j]); std::swap(inv[p * n + j], inv[c * n + j]); }
    cd d = 1.0 / a[c * n + c];
    for (int j = 0; j < n; j++) { a[c * n + j] *= d; inv[c * n + j] *= d; }
    for (int r = 0; r < n; r++) {
      if (r == c) continue;
      cd f = a[r * n + c];
      if (f == cd(0.0)) continue;
      for (int j = 0; j < n; j++) { a[r * n + j] -= f * a[c * n + j]; inv[r * n + j] -= f * inv[c * n + j]; }
    }
  }
  return true;
}

// Hopping part at one site (reading R1):
// (H psi)(x) = -1/2 sum_mu [ (1-gamma_mu) W_mu(x) psi(x+mu) + (1+gamma_mu) W_mu(x-mu)^dag psi(x-mu) ],
// spinors pick up -1 across the time boundary when antiperiodic (reading R9).
void hop_site(const Ref& g, const cd* psi, const int x[4], cd out[12]) {
  for (int i = 0; i < 12; i++) out[i] = 0;
  for (int mu = 0; mu < 4; mu++) {
    int y[4];
    // forward
    {
      int cr = g.hop(x, mu, +1, y);
      double sgn = (cr && g.antiper) ? -1.0 : 1.0;
      M3 W = g.hoplink(x, mu);
      const cd* p = psi + g.lex(y) * 12;
      for (int al = 0; al < 4; al++)
        for (int be = 0; be < 4; be++) {
          cd pr = ((al == be) ? 1.0 : 0.0) - GM.g[mu][al][be];
          if (pr == cd(0.0)) continue;
          for (int a = 0; a < 3; a++) {
            cd z = 0;
            for (int b = 0; b < 3; b++) z += W.m[3 * a + b] * p[3 * be + b];
            out[3 * al + a] += -0.5 * sgn * pr * z;
          }
        }
    }
    // backward
    {
      int cr = g.hop(x, mu, -1, y);
      double sgn = (cr && g.antiper) ? -1.0 : 1.0;
      M3 Wd = dag(g.hoplink(y, mu));
      const cd* p = psi + g.lex(y) * 12;
      for (int al = 0; al < 4; al++)
        for (int be = 0; be < 4; be++) {
          cd pr = ((al == be) ? 1.0 : 0.0) + GM.g[mu][al][be];
          if (pr == cd(0.0)) continue;
          for (int a = 0; a < 3; a++) {
            cd z = 0;
            for (int b = 0; b < 3; b++) z += Wd.m[3 * a + b] * p[3 * be + b];
            out[3 * al + a] += -0.5 * sgn * pr * z;
          }
        }
    }
  }
}

void diag_site(const cd* blk /*[2][36]*/, const cd* in, cd* out) {
  for (int c = 0; c < 2; c++)
    for (int i = 0; i < 6; i++) {
      cd z = 0;
      for (int j = 0; j < 6; j++) z += blk[c * 36 + i * 6 + j] * in[6 * c + j];
      out[6 * c + i] = z;
    }
}

// full-lattice helpers on natural-order fields [V][12]; parity_mask: 0 even, 1 odd, 2 all
void hop_field(const Ref& g, const cd* in, cd* out, int pm) {
#pragma omp parallel for schedule(static)
  for (long s = 0; s < g.V; s++) {
    int x[4]; g.coords(s, x);
    if (pm != 2 && g.parity(x) != pm) continue;
    hop_site(g, in, x, out + s * 12);
  }
}
void diag_field(const Ref& g, const std::vector<cd>& blk, const cd* in, cd* out, int pm) {
#pragma omp parallel for schedule(static)
  for (long s = 0; s < g.V; s++) {
    int x[4]; g.coords(s, x);
    if (pm != 2 && g.parity(x) != pm) continue;
    cd tmp[12];
    diag_site(&blk[s * 72], in + s * 12, tmp);
    for (int i = 0; i < 12; i++) out[s * 12 + i] = tmp[i];
  }
}

// D-hat = A_ee - D_eo A_oo^{-1} D_oe on even sites (reading R10); fields are
// natural-order full-lattice arrays whose odd entries are ignored on input and zero on output.
// dagger: D-hat^dag = gamma5 D-hat gamma5 (gamma5 = diag(1,1,-1,-1) in this basis).
void dhat_full(const Ref& g, const cd* in, cd* out, bool dagger, std::vector<cd>& w1, std::vector<cd>& w2) {
  const long n = g.V * 12;
  std::vector<cd>& v = w1; std::vector<cd>& t = w2;
  v.assign(n, 0.0); t.assign(n, 0.0);
#pragma omp parallel for schedule(static)
  for (long s = 0; s < g.V; s++) {
    int x[4]; g.coords(s, x);
    if (g.parity(x) != 0) continue;
    for (int i = 0; i < 12; i++) v[s * 12 + i] = (dagger && i >= 6) ? -in[s * 12 + i] : in[s * 12 + i];
  }
  hop_field(g, v.data(), t.data(), 1);          // t_o = D_oe v_e
  diag_field(g, g.Mi, t.data(), t.data(), 1);   // t_o = A_oo^{-1} t_o
  std::vector<cd> u(n, 0.0);
  hop_field(g, t.data(), u.data(), 0);          // u_e = D_eo t_o
  std::vector<cd> av(n, 0.0);
  diag_field(g, g.Mb, v.data(), av.data(), 0);  // A_ee v_e
#pragma omp parallel for schedule(static)
  for (long s = 0; s < g.V; s++) {
    int x[4]; g.coords(s, x);
    for (int i = 0; i < 12; i++) {
      cd z = 0.0;
      if (g.parity(x) == 0) { z = av[s * 12 + i] - u[s * 12 + i]; if (dagger && i >= 6) z = -z; }
      out[s * 12 + i] = z;
    }
  }
}

double norm2(const std::vector<cd>& a) {
  double s = 0;
#pragma omp parallel for reduction(+ : s) schedule(static)
  for (long i = 0; i < (long)a.size(); i++) s += std::norm(a[i]);
  return s;
}

}  // namespace

extern "C" {

int qxd_ref_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// bc = cstar (0..3) | antiperiodic_time << 2; extents are PHYSICAL (reading R18: all even, >= 2).
void* qxd_ref_create(int T, int L1, int L2, int L3, int bc) {
  int cstar = bc & 3, ap = (bc >> 2) & 1;
  if (T < 2 || L1 < 2 || L2 < 2 || L3 < 2 || (T | L1 | L2 | L3) & 1 || bc < 0 || bc > 7) return nullptr;
  Ref* g = new Ref;
  g->T = T; g->L1 = L1; g->L2 = L2; g->L3 = L3; g->cstar = cstar; g->antiper = ap;
  g->X[0] = T; g->X[1] = cstar > 0 ? 2 * L1 : L1; g->X[2] = L2; g->X[3] = L3;
  g->V = long(g->X[0]) * g->X[1] * g->X[2] * g->X[3];
  return g;
}
void qxd_ref_destroy(void* h) { delete (Ref*)h; }
long qxd_ref_volume(void* h) { return ((Ref*)h)->V; }

// U: [T][L1][L2][L3][4][3][3] complex (re,im) on the PHYSICAL lattice, A: [T][L1][L2][L3][4] or NULL.
// Mirror half (reading R8): U_mu(x + L1 1-hat) = U_mu(x)^*, A_mu(x + L1 1-hat) = -A_mu(x).
int qxd_ref_gauge_load(void* h, const double* U, const double* A, double qel) {
  Ref& g = *(Ref*)h;
  if (!U || qel == 0.0) return -1;
  g.qel = qel;
  g.U.assign(g.V * 36, 0.0);
  if (A) g.A.assign(g.V * 4, 0.0); else g.A.clear();
  for (long s = 0; s < g.V; s++) {
    int x[4]; g.coords(s, x);
    bool mirror = x[1] >= g.L1;
    long sp = ((long(x[0]) * g.L1 + (x[1] % g.L1)) * g.L2 + x[2]) * g.L3 + x[3];
    for (int k = 0; k < 36; k++) {
      cd z(U[(sp * 36 + k) * 2], U[(sp * 36 + k) * 2 + 1]);
      g.U[s * 36 + k] = mirror ? std::conj(z) : z;
    }
    if (A) for (int mu = 0; mu < 4; mu++) g.A[s * 4 + mu] = mirror ? -A[sp * 4 + mu] : A[sp * 4 + mu];
  }
  g.have_gauge = true; g.have_clover = false;
  return 0;
}

// m0 = 1/(2 kappa) - 4 (reading R2).
int qxd_ref_set_quark(void* h, double kappa, double q) {
  Ref& g = *(Ref*)h;
  if (!(kappa > 0.0)) return -1;
  g.kappa = kappa; g.q = q; g.m0 = 1.0 / (2.0 * kappa) - 4.0; g.have_quark = true; g.have_clover = false;
  return 0;
}

int qxd_ref_set_csw(void* h, double csw, double csw_qed) {
  Ref& g = *(Ref*)h;
  g.csw = csw; g.csw_qed = csw_qed; g.have_csw = true; g.have_clover = false;
  return 0;
}

// 12x12 site matrix from the definition, row-major complex (re,im): out[144][2].
int qxd_ref_site_matrix(void* h, long site, double* out) {
  Ref& g = *(Ref*)h;
  if (!g.have_gauge || !g.have_quark || !g.have_csw || site < 0 || site >= g.V) return -2;
  int x[4]; g.coords(site, x);
  cd M[144]; g.site_matrix(x, M);
  for (int i = 0; i < 144; i++) { out[2 * i] = M[i].real(); out[2 * i + 1] = M[i].imag(); }
  return 0;
}

// Builds the site matrix everywhere, extracts its two chirality blocks ("+" = spin 0,1; "-" = spin 2,3;
// PAPER.md:53) and inverts them (the term stays chirality-diagonal and Hermitian).
int qxd_ref_clover_build(void* h, double csw, double csw_qed) {
  Ref& g = *(Ref*)h;
  if (!g.have_gauge || !g.have_quark) return -2;
  qxd_ref_set_csw(h, csw, csw_qed);
  g.Mb.assign(g.V * 72, 0.0); g.Mi.assign(g.V * 72, 0.0);
  double moff = 0, mah = 0; int bad = 0;
#pragma omp parallel for schedule(static) reduction(max : moff, mah) reduction(+ : bad)
  for (long s = 0; s < g.V; s++) {
    int x[4]; g.coords(s, x);
    cd M[144]; g.site_matrix(x, M);
    for (int i = 0; i < 12; i++)
      for (int j = 0; j < 12; j++) {
        mah = std::max(mah, std::abs(M[i * 12 + j] - std::conj(M[j * 12 + i])));
        if ((i < 6) != (j < 6)) moff = std::max(moff, std::abs(M[i * 12 + j]));
      }
    for (int c = 0; c < 2; c++) {
      cd* b = &g.Mb[s * 72 + c * 36];
      for (int i = 0; i < 6; i++) for (int j = 0; j < 6; j++) b[i * 6 + j] = M[(6 * c + i) * 12 + 6 * c + j];
      if (!invert(6, b, &g.Mi[s * 72 + c * 36])) bad++;
    }
  }
  g.max_offdiag = moff; g.max_antiherm = mah;
  if (bad) return -3;
  g.have_clover = true;
  return 0;
}
double qxd_ref_clover_max_offdiag(void* h) { return ((Ref*)h)->max_offdiag; }
double qxd_ref_clover_max_antiherm(void* h) { return ((Ref*)h)->max_antiherm; }

// Packed blocks: per block 36 reals = 6 real diagonal entries, then (re,im) of the 15
// strictly-upper-triangular entries in row-major order.  out: [V][2][36].
int qxd_ref_clover_packed(void* h, double* out, int inverse) {
  Ref& g = *(Ref*)h;
  if (!g.have_clover) return -2;
  const std::vector<cd>& src = inverse ? g.Mi : g.Mb;
  for (long s = 0; s < g.V; s++)
    for (int c = 0; c < 2; c++) {
      const cd* b = &src[s * 72 + c * 36];
      double* o = out + s * 72 + c * 36;
      for (int i = 0; i < 6; i++) o[i] = b[i * 6 + i].real();
      int k = 6;
      for (int i = 0; i < 6; i++) for (int j = i + 1; j < 6; j++) { o[k++] = b[i * 6 + j].real(); o[k++] = b[i * 6 + j].imag(); }
    }
  return 0;
}

// psi, out: [T][X1][L2][L3][4][3] complex on the EXTENDED lattice (Eq. (1)).
int qxd_ref_apply_Dw(void* h, const double* psi, double* out) {
  Ref& g = *(Ref*)h;
  if (!g.have_clover) return -2;
  const cd* p = (const cd*)psi; cd* o = (cd*)out;
#pragma omp parallel for schedule(static)
  for (long s = 0; s < g.V; s++) {
    int x[4]; g.coords(s, x);
    cd hp[12], dg[12];
    hop_site(g, p, x, hp);
    diag_site(&g.Mb[s * 72], p + s * 12, dg);
    for (int i = 0; i < 12; i++) o[s * 12 + i] = dg[i] + hp[i];
  }
  return 0;
}

// (D_w psi)(x) at selected sites only, site matrix computed on the fly from the definition (full 12x12
// mat-vec, no block extraction): for sampled parity checks at sizes where a full apply is too slow.
int qxd_ref_apply_Dw_sites(void* h, const double* psi, long n, const long* sites, double* out) {
  Ref& g = *(Ref*)h;
  if (!g.have_gauge || !g.have_quark || !g.have_csw) return -2;
  const cd* p = (const cd*)psi; cd* o = (cd*)out;
  int bad = 0;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : bad)
  for (long k = 0; k < n; k++) {
    long s = sites[k];
    if (s < 0 || s >= g.V) { bad++; continue; }
    int x[4]; g.coords(s, x);
    cd hp[12], M[144];
    hop_site(g, p, x, hp);
    g.site_matrix(x, M);
    for (int i = 0; i < 12; i++) {
      cd z = hp[i];
      for (int j = 0; j < 12; j++) z += M[i * 12 + j] * p[s * 12 + j];
      o[k * 12 + i] = z;
    }
  }
  return bad ? -1 : 0;
}

// ---- bounded-sample variants (bench.py cpu_baseline / --impl reference): the same per-site arithmetic as
// qxd_ref_clover_build / qxd_ref_apply_Dw, restricted to the natural-order site range [lo, hi) so that a
// slab of a large lattice can be timed in seconds.  The blocks are kept in a range-sized array.
int qxd_ref_clover_build_range(void* h, double csw, double csw_qed, long lo, long hi) {
  Ref& g = *(Ref*)h;
  if (!g.have_gauge || !g.have_quark) return -2;
  if (lo < 0 || hi > g.V || lo >= hi) return -1;
  qxd_ref_set_csw(h, csw, csw_qed);
  g.range_lo = lo; g.range_hi = hi;
  g.Mb_range.assign((hi - lo) * 72, 0.0);
#pragma omp parallel for schedule(static)
  for (long s = lo; s < hi; s++) {
    int x[4]; g.coords(s, x);
    cd M[144]; g.site_matrix(x, M);
    for (int c = 0; c < 2; c++) {
      cd* b = &g.Mb_range[(s - lo) * 72 + c * 36];
      for (int i = 0; i < 6; i++) for (int j = 0; j < 6; j++) b[i * 6 + j] = M[(6 * c + i) * 12 + 6 * c + j];
    }
  }
  return 0;
}
// out: [(hi-lo)][4][3] complex = (D_w psi)(x) for the sites of the range built above; psi is the full field.
int qxd_ref_apply_Dw_range(void* h, const double* psi, double* out) {
  Ref& g = *(Ref*)h;
  if (g.Mb_range.empty()) return -2;
  const cd* p = (const cd*)psi; cd* o = (cd*)out;
  const long lo = g.range_lo, hi = g.range_hi;
#pragma omp parallel for schedule(static)
  for (long s = lo; s < hi; s++) {
    int x[4]; g.coords(s, x);
    cd hp[12], dg[12];
    hop_site(g, p, x, hp);
    diag_site(&g.Mb_range[(s - lo) * 72], p + s * 12, dg);
    for (int i = 0; i < 12; i++) o[(s - lo) * 12 + i] = dg[i] + hp[i];
  }
  return 0;
}

// Even-sublattice fields: [V/2][4][3] complex, the even sites in increasing Lambda order
// (all extents are even, so the k-th even site is the one with Lambda>>1 == k).
int qxd_ref_apply_Dhat(void* h, const double* psi_e, double* out_e, int dagger) {
  Ref& g = *(Ref*)h;
  if (!g.have_clover) return -2;
  std::vector<cd> in(g.V * 12, 0.0), out(g.V * 12), w1, w2;
  const cd* p = (const cd*)psi_e; cd* o = (cd*)out_e;
  for (long s = 0; s < g.V; s++) { int x[4]; g.coords(s, x); if (g.parity(x) == 0) for (int i = 0; i < 12; i++) in[s * 12 + i] = p[(s >> 1) * 12 + i]; }
  dhat_full(g, in.data(), out.data(), dagger != 0, w1, w2);
  for (long s = 0; s < g.V; s++) { int x[4]; g.coords(s, x); if (g.parity(x) == 0) for (int i = 0; i < 12; i++) o[(s >> 1) * 12 + i] = out[s * 12 + i]; }
  return 0;
}

// Solve D_w psi = eta by even-odd preconditioning and CG on the normal equations, keeping the SYSTEM
// residual explicitly (reading R10/R11, SURVEY.md §8(c4),(c5)):
//   eta-hat_e = eta_e - D_eo A_oo^{-1} eta_o ;  D-hat psi_e = eta-hat_e ;  psi_o = A_oo^{-1}(eta_o - D_oe psi_e)
//   x=0, r=b, s=A^dag r, p=s, gam=|s|^2; loop: t=Ap; al=gam/|t|^2; x+=al p; r-=al t;
//   stop if |r| <= tol |eta|; s=A^dag r; gam'=|s|^2; p=s+(gam'/gam)p; gam=gam'.
// Returns 0 on convergence, -5 if maxiter was hit (psi still holds the best iterate).
int qxd_ref_solve(void* h, const double* eta_, double* psi_, double tol, int maxiter, int* iters, double* relres) {
  Ref& g = *(Ref*)h;
  if (!g.have_clover) return -2;
  const long n = g.V * 12;
  const cd* eta = (const cd*)eta_; cd* psi = (cd*)psi_;
  std::vector<cd> b(n, 0.0), tmp(n, 0.0), tmp2(n, 0.0), w1, w2;
  std::vector<cd> etav(eta, eta + n);
  const double eta_norm = std::sqrt(norm2(etav));
  // source preparation
  diag_field(g, g.Mi, eta, tmp.data(), 1);       // tmp_o = A_oo^{-1} eta_o
  hop_field(g, tmp.data(), tmp2.data(), 0);      // tmp2_e = D_eo tmp_o
  for (long s = 0; s < g.V; s++) { int x[4]; g.coords(s, x); if (g.parity(x) == 0) for (int i = 0; i < 12; i++) b[s * 12 + i] = eta[s * 12 + i] - tmp2[s * 12 + i]; }
  std::vector<cd> x(n, 0.0), r(b), s(n), p(n), t(n);
  dhat_full(g, r.data(), s.data(), true, w1, w2);
  p = s;
  double gam = norm2(s);
  int it = 0, status = -5;
  double rn = std::sqrt(norm2(r));
  if (rn <= tol * eta_norm) status = 0;
  while (status != 0 && it < maxiter) {
    dhat_full(g, p.data(), t.data(), false, w1, w2);
    double al = gam / norm2(t);
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) { x[i] += al * p[i]; r[i] -= al * t[i]; }
    it++;
    rn = std::sqrt(norm2(r));
    if (rn <= tol * eta_norm) { status = 0; break; }
    dhat_full(g, r.data(), s.data(), true, w1, w2);
    double gam2 = norm2(s), be = gam2 / gam;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < n; i++) p[i] = s[i] + be * p[i];
    gam = gam2;
  }
  // reconstruction of the odd sites
  tmp.assign(n, 0.0);
  hop_field(g, x.data(), tmp.data(), 1);         // tmp_o = D_oe psi_e
  for (long k = 0; k < g.V; k++) { int c[4]; g.coords(k, c); if (g.parity(c) == 1) for (int i = 0; i < 12; i++) tmp[k * 12 + i] = eta[k * 12 + i] - tmp[k * 12 + i]; }
  diag_field(g, g.Mi, tmp.data(), tmp.data(), 1);
  for (long k = 0; k < g.V; k++) { int c[4]; g.coords(k, c); for (int i = 0; i < 12; i++) psi[k * 12 + i] = (g.parity(c) == 0) ? x[k * 12 + i] : tmp[k * 12 + i]; }
  if (iters) *iters = it;
  if (relres) *relres = rn / eta_norm;
  return status;
}

}  // extern "C"
