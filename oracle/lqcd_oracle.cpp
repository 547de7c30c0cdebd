// CPU ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, obviously-correct fp64 implementation of the Wilson-clover operator
//     M = A - kappa*D,   A = 1 - kappa*csw*sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}
// (Eq. 5; isotropic by default, the anisotropic weights nu/xi_0, c_SW^t, c_SW^r/xi_0
// through orc_set_anisotropy / orc_set_clover_aniso; kappa normalisation:
// the paper's a_t*M is this M/(2 kappa)), its even-odd Schur forms and CG / BiCGStab, written
// from the definitions in SURVEY.md §8(c) O1-O9 (the paper states conventions only:
// DeGrand-Rossi basis and cb2 layouts; BiCGStab/CG).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// use this file.  It shares no code with the CUDA path (paper_2411_08461_b200/csrc).
//
// Style: loops over the LEXICOGRAPHIC lattice; gamma and sigma matrices are built numerically
// from their definition (no hand-expanded projector tricks); every step is the textbook formula.
//
// Parity unpinned (conventions no invariant can see; fixed by DESIGN.md readings A4, A7):
//   * the trace of F_{mu nu} is not removed;
//   * the packed lower triangle of a clover block is row-major, (i,j), i>j at i(i-1)/2+j.
//
// Public layouts at this file's C entry points (complex = interleaved (re,im) doubles):
//   gauge   [4][2][Lt][Lz][Ly][Lx/2][3][3]   mu = 0..3 <-> x,y,z,t
//   spinor  [2][Lt][Lz][Ly][Lx/2][4][3]
//   clover  [2][Lt][Lz][Ly][Lx/2][2][36] reals: per chiral block 6 real diagonal
//           entries, then 15 complex strictly-lower entries
#include <algorithm>
#include <chrono>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const cplx I_(0.0, 1.0);

// ---------------------------------------------------------------------------------------------
// O1 geometry
// ---------------------------------------------------------------------------------------------
struct Geom {
  int L[4];
  long V, Vh;
  void coords(long lex, int x[4]) const {
    x[0] = lex % L[0]; lex /= L[0];
    x[1] = lex % L[1]; lex /= L[1];
    x[2] = lex % L[2];
    x[3] = lex / L[2];
  }
  long lex(const int x[4]) const { return x[0] + (long)L[0] * (x[1] + (long)L[1] * (x[2] + (long)L[2] * x[3])); }
  int parity(long l) const {
    int x[4];
    coords(l, x);
    return (x[0] + x[1] + x[2] + x[3]) & 1;
  }
  // position in the public [2][Vh] ordering
  long cb(long l) const { return (long)parity(l) * Vh + l / 2; }
  // neighbour of site l displaced by s (= +1/-1) in direction mu, periodic as an index
  long shift(long l, int mu, int s) const {
    int x[4];
    coords(l, x);
    x[mu] = (x[mu] + s + L[mu]) % L[mu];
    return lex(x);
  }
};

static bool make_geom(const int* dims, Geom& g) {
  g.V = 1;
  for (int i = 0; i < 4; i++) {
    if (dims[i] < 2 || (dims[i] & 1)) return false;
    g.L[i] = dims[i];
    g.V *= dims[i];
  }
  g.Vh = g.V / 2;
  return true;
}

// public cb2 <-> lexicographic copies of a field with n complex numbers per site
static void to_lex(const Geom& g, const cplx* pub, cplx* lexf, int n) {
#pragma omp parallel for schedule(static)
  for (long l = 0; l < g.V; l++) std::memcpy(lexf + l * n, pub + g.cb(l) * n, sizeof(cplx) * n);
}
static void from_lex(const Geom& g, const cplx* lexf, cplx* pub, int n) {
#pragma omp parallel for schedule(static)
  for (long l = 0; l < g.V; l++) std::memcpy(pub + g.cb(l) * n, lexf + l * n, sizeof(cplx) * n);
}
// gauge: public [4][2][Vh][9] -> lex [4][V][9]
static void gauge_to_lex(const Geom& g, const cplx* pub, cplx* lexf) {
  for (int mu = 0; mu < 4; mu++) to_lex(g, pub + (long)mu * g.V * 9, lexf + (long)mu * g.V * 9, 9);
}

// ---------------------------------------------------------------------------------------------
// O2 gamma matrices, DeGrand-Rossi basis: gamma_mu = [[0, B_mu], [B_mu^dag, 0]],
// B_x = i sigma^1, B_y = -i sigma^2, B_z = i sigma^3, B_t = 1.  gamma_5 = g_x g_y g_z g_t.
// sigma_{mu nu} = (i/2)[gamma_mu, gamma_nu].
// ---------------------------------------------------------------------------------------------
struct Gammas {
  cplx g[5][4][4];       // g[4] = gamma_5
  cplx sig[4][4][4][4];  // sig[mu][nu]
  Gammas() {
    const cplx s1[2][2] = {{0, 1}, {1, 0}};
    const cplx s2[2][2] = {{0, -I_}, {I_, 0}};
    const cplx s3[2][2] = {{1, 0}, {0, -1}};
    cplx B[4][2][2];
    for (int a = 0; a < 2; a++)
      for (int b = 0; b < 2; b++) {
        B[0][a][b] = I_ * s1[a][b];
        B[1][a][b] = -I_ * s2[a][b];
        B[2][a][b] = I_ * s3[a][b];
        B[3][a][b] = (a == b) ? 1.0 : 0.0;
      }
    for (int mu = 0; mu < 4; mu++) {
      for (int a = 0; a < 4; a++)
        for (int b = 0; b < 4; b++) g[mu][a][b] = 0;
      for (int a = 0; a < 2; a++)
        for (int b = 0; b < 2; b++) {
          g[mu][a][2 + b] = B[mu][a][b];
          g[mu][2 + a][b] = std::conj(B[mu][b][a]);
        }
    }
    cplx t1[4][4], t2[4][4];
    mul(g[0], g[1], t1);
    mul(t1, g[2], t2);
    mul(t2, g[3], g[4]);
    for (int mu = 0; mu < 4; mu++)
      for (int nu = 0; nu < 4; nu++) {
        mul(g[mu], g[nu], t1);
        mul(g[nu], g[mu], t2);
        for (int a = 0; a < 4; a++)
          for (int b = 0; b < 4; b++) sig[mu][nu][a][b] = 0.5 * I_ * (t1[a][b] - t2[a][b]);
      }
  }
  static void mul(const cplx a[4][4], const cplx b[4][4], cplx c[4][4]) {
    for (int i = 0; i < 4; i++)
      for (int j = 0; j < 4; j++) {
        cplx s = 0;
        for (int k = 0; k < 4; k++) s += a[i][k] * b[k][j];
        c[i][j] = s;
      }
  }
};
static const Gammas GM;

// ---------------------------------------------------------------------------------------------
// 3x3 colour-matrix helpers
// ---------------------------------------------------------------------------------------------
static inline void m3_mul(const cplx* a, const cplx* b, cplx* c) {  // c = a b
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      cplx s = 0;
      for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
      c[3 * i + j] = s;
    }
}
static inline void m3_dag(const cplx* a, cplx* c) {
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) c[3 * i + j] = std::conj(a[3 * j + i]);
}
// product of four matrices, each optionally daggered
static void m3_path(const cplx* a, bool da, const cplx* b, bool db, const cplx* c, bool dc, const cplx* d,
                    bool dd, cplx* out) {
  cplx A[9], B[9], C[9], D[9], t1[9], t2[9];
  if (da) m3_dag(a, A); else std::memcpy(A, a, sizeof(A));
  if (db) m3_dag(b, B); else std::memcpy(B, b, sizeof(B));
  if (dc) m3_dag(c, C); else std::memcpy(C, c, sizeof(C));
  if (dd) m3_dag(d, D); else std::memcpy(D, d, sizeof(D));
  m3_mul(A, B, t1);
  m3_mul(t1, C, t2);
  m3_mul(t2, D, out);
}

// ---------------------------------------------------------------------------------------------
// O3 hopping term on lexicographic fields.
//   (D psi)(x) = sum_mu [ (1 - g_mu) U_mu(x) psi(x+mu) + (1 + g_mu) U_mu^dag(x-mu) psi(x-mu) ]
// dagger swaps the two projector signs.  t_boundary = -1: hops across the t = Lt-1 -> 0 seam
// (both use U_t(., Lt-1)) get a factor -1.  only_parity = 0/1 restricts the OUTPUT sites to that
// parity (other output sites are set to zero); -1 = all sites.
// ---------------------------------------------------------------------------------------------
// w[mu]: weight of the hops in direction mu (Eq. 5: gamma_4 W_4 + (nu/xi_0) sum_i
// gamma_i W_i, i.e. w = (nu/xi_0, nu/xi_0, nu/xi_0, 1); isotropic: all 1).
static void hop(const Geom& g, int tb, const cplx* U, const cplx* in, cplx* out, int dagger, int only_parity,
                const double* w) {
  const double sgn = dagger ? -1.0 : 1.0;
#pragma omp parallel for schedule(static)
  for (long l = 0; l < g.V; l++) {
    cplx acc[4][3];
    for (int s = 0; s < 4; s++)
      for (int c = 0; c < 3; c++) acc[s][c] = 0;
    if (only_parity < 0 || g.parity(l) == only_parity) {
      int x[4];
      g.coords(l, x);
      for (int mu = 0; mu < 4; mu++) {
        // forward: (1 - sgn*g_mu) U_mu(x) psi(x+mu)
        {
          long lf = g.shift(l, mu, +1);
          const cplx* u = U + ((long)mu * g.V + l) * 9;
          const cplx* p = in + lf * 12;
          double bsign = (mu == 3 && tb < 0 && x[3] == g.L[3] - 1) ? -1.0 : 1.0;
          cplx up[4][3];
          for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++) {
              cplx v = 0;
              for (int b = 0; b < 3; b++) v += u[3 * a + b] * p[3 * s + b];
              up[s][a] = v;
            }
          for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++) {
              cplx v = up[s][a];
              for (int s2 = 0; s2 < 4; s2++)
                if (GM.g[mu][s][s2] != 0.0) v -= sgn * GM.g[mu][s][s2] * up[s2][a];
              acc[s][a] += w[mu] * bsign * v;
            }
        }
        // backward: (1 + sgn*g_mu) U_mu^dag(x-mu) psi(x-mu)
        {
          long lb = g.shift(l, mu, -1);
          const cplx* u = U + ((long)mu * g.V + lb) * 9;
          const cplx* p = in + lb * 12;
          double bsign = (mu == 3 && tb < 0 && x[3] == 0) ? -1.0 : 1.0;
          cplx up[4][3];
          for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++) {
              cplx v = 0;
              for (int b = 0; b < 3; b++) v += std::conj(u[3 * b + a]) * p[3 * s + b];
              up[s][a] = v;
            }
          for (int s = 0; s < 4; s++)
            for (int a = 0; a < 3; a++) {
              cplx v = up[s][a];
              for (int s2 = 0; s2 < 4; s2++)
                if (GM.g[mu][s][s2] != 0.0) v += sgn * GM.g[mu][s][s2] * up[s2][a];
              acc[s][a] += w[mu] * bsign * v;
            }
        }
      }
    }
    for (int s = 0; s < 4; s++)
      for (int c = 0; c < 3; c++) out[l * 12 + 3 * s + c] = acc[s][c];
  }
}

// ---------------------------------------------------------------------------------------------
// O4 field strength from the four clover leaves, all starting and ending at x, counter-clockwise
// in the mu-nu plane; raw periodic links (the boundary sign cancels inside every leaf).
//   F_{mu nu} = (Q - Q^dag) / (8 i),  Q = P1 + P2 + P3 + P4.   Trace NOT removed (reading A4).
// ---------------------------------------------------------------------------------------------
static void field_strength(const Geom& g, const cplx* U, long l, int mu, int nu, cplx* F) {
  auto link = [&](int d, long site) { return U + ((long)d * g.V + site) * 9; };
  const long xpm = g.shift(l, mu, +1), xpn = g.shift(l, nu, +1);
  const long xmm = g.shift(l, mu, -1), xmn = g.shift(l, nu, -1);
  const long xmm_pn = g.shift(xmm, nu, +1), xmm_mn = g.shift(xmm, nu, -1);
  const long xpm_mn = g.shift(xpm, nu, -1);
  cplx P[9], Q[9];
  for (int e = 0; e < 9; e++) Q[e] = 0;
  // P1 = U_mu(x) U_nu(x+mu) U_mu^dag(x+nu) U_nu^dag(x)
  m3_path(link(mu, l), false, link(nu, xpm), false, link(mu, xpn), true, link(nu, l), true, P);
  for (int e = 0; e < 9; e++) Q[e] += P[e];
  // P2 = U_nu(x) U_mu^dag(x-mu+nu) U_nu^dag(x-mu) U_mu(x-mu)
  m3_path(link(nu, l), false, link(mu, xmm_pn), true, link(nu, xmm), true, link(mu, xmm), false, P);
  for (int e = 0; e < 9; e++) Q[e] += P[e];
  // P3 = U_mu^dag(x-mu) U_nu^dag(x-mu-nu) U_mu(x-mu-nu) U_nu(x-nu)
  m3_path(link(mu, xmm), true, link(nu, xmm_mn), true, link(mu, xmm_mn), false, link(nu, xmn), false, P);
  for (int e = 0; e < 9; e++) Q[e] += P[e];
  // P4 = U_nu^dag(x-nu) U_mu(x-nu) U_nu(x+mu-nu) U_mu^dag(x)
  m3_path(link(nu, xmn), true, link(mu, xmn), false, link(nu, xpm_mn), false, link(mu, l), true, P);
  for (int e = 0; e < 9; e++) Q[e] += P[e];
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) F[3 * i + j] = (Q[3 * i + j] - std::conj(Q[3 * j + i])) / (8.0 * I_);
}

// O5: dense 12x12 clover matrix at one site, row/col index = 3*spin + colour
// csw = coefficient of the spatial planes (Eq. 5: c_SW^r/xi_0), csw_t = of the temporal planes
// (c_SW^t); isotropic: csw_t = csw.
static void clover_dense_site(const Geom& g, const cplx* U, long l, double kappa, double csw, double csw_t,
                              cplx* A /*144*/) {
  for (int e = 0; e < 144; e++) A[e] = 0;
  for (int i = 0; i < 12; i++) A[13 * i] = 1.0;
  for (int mu = 0; mu < 4; mu++)
    for (int nu = mu + 1; nu < 4; nu++) {
      cplx F[9];
      field_strength(g, U, l, mu, nu, F);
      for (int s = 0; s < 4; s++)
        for (int s2 = 0; s2 < 4; s2++) {
          cplx sg = GM.sig[mu][nu][s][s2];
          if (sg == 0.0) continue;
          for (int a = 0; a < 3; a++)
            for (int b = 0; b < 3; b++)
              A[(3 * s + a) * 12 + (3 * s2 + b)] -= kappa * (nu == 3 ? csw_t : csw) * sg * F[3 * a + b];
        }
    }
}

// pack / unpack one Hermitian 6x6 block <-> 36 reals (order: reading A7)
static void pack_block(const cplx* B /*36, row-major*/, double* p /*36*/) {
  for (int i = 0; i < 6; i++) p[i] = B[7 * i].real();
  for (int i = 1; i < 6; i++)
    for (int j = 0; j < i; j++) {
      int k = i * (i - 1) / 2 + j;
      p[6 + 2 * k] = B[6 * i + j].real();
      p[6 + 2 * k + 1] = B[6 * i + j].imag();
    }
}
static void unpack_block(const double* p, cplx* B) {
  for (int i = 0; i < 6; i++) B[7 * i] = p[i];
  for (int i = 1; i < 6; i++)
    for (int j = 0; j < i; j++) {
      int k = i * (i - 1) / 2 + j;
      cplx v(p[6 + 2 * k], p[6 + 2 * k + 1]);
      B[6 * i + j] = v;
      B[6 * j + i] = std::conj(v);
    }
}

// Build the packed clover field in lex order: [V][2][36].  Returns the largest magnitude found in
// the off-diagonal chiral 6x6 blocks and the largest anti-Hermitian part (both must be ~0).
static double clover_build_lex(const Geom& g, const cplx* U, double kappa, double csw, double csw_t, double* Apk) {
  double worst = 0;
#pragma omp parallel for schedule(static) reduction(max : worst)
  for (long l = 0; l < g.V; l++) {
    cplx A[144], B[36];
    clover_dense_site(g, U, l, kappa, csw, csw_t, A);
    for (int i = 0; i < 6; i++)
      for (int j = 0; j < 6; j++) {
        worst = std::max(worst, std::abs(A[i * 12 + 6 + j]));
        worst = std::max(worst, std::abs(A[(6 + i) * 12 + j]));
      }
    for (int i = 0; i < 12; i++)
      for (int j = 0; j < 12; j++) worst = std::max(worst, std::abs(A[i * 12 + j] - std::conj(A[j * 12 + i])));
    for (int k = 0; k < 2; k++) {
      for (int i = 0; i < 6; i++)
        for (int j = 0; j < 6; j++) B[6 * i + j] = A[(6 * k + i) * 12 + 6 * k + j];
      pack_block(B, Apk + (l * 2 + k) * 36);
    }
  }
  return worst;
}

// O6: inverse of a 6x6 complex matrix, Gauss-Jordan with partial pivoting. false if singular.
static bool invert6(const cplx* Bin, cplx* inv) {
  cplx a[6][12];
  double nrm = 0;
  for (int i = 0; i < 6; i++)
    for (int j = 0; j < 6; j++) {
      a[i][j] = Bin[6 * i + j];
      a[i][6 + j] = (i == j) ? 1.0 : 0.0;
      nrm = std::max(nrm, std::abs(Bin[6 * i + j]));
    }
  for (int c = 0; c < 6; c++) {
    int piv = c;
    for (int r = c + 1; r < 6; r++)
      if (std::abs(a[r][c]) > std::abs(a[piv][c])) piv = r;
    if (std::abs(a[piv][c]) <= 1e-12 * nrm) return false;
    if (piv != c)
      for (int j = 0; j < 12; j++) std::swap(a[piv][j], a[c][j]);
    cplx d = 1.0 / a[c][c];
    for (int j = 0; j < 12; j++) a[c][j] *= d;
    for (int r = 0; r < 6; r++) {
      if (r == c) continue;
      cplx f = a[r][c];
      if (f == 0.0) continue;
      for (int j = 0; j < 12; j++) a[r][j] -= f * a[c][j];
    }
  }
  for (int i = 0; i < 6; i++)
    for (int j = 0; j < 6; j++) inv[6 * i + j] = a[i][6 + j];
  return true;
}

static bool clover_invert_lex(const Geom& g, const double* Apk, double* Ainv) {
  int bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
  for (long q = 0; q < g.V * 2; q++) {
    cplx B[36], Bi[36], H[36];
    unpack_block(Apk + q * 36, B);
    if (!invert6(B, Bi)) {
      bad++;
      continue;
    }
    // the inverse of a Hermitian matrix is Hermitian; symmetrise the rounding before packing
    for (int i = 0; i < 6; i++)
      for (int j = 0; j < 6; j++) H[6 * i + j] = 0.5 * (Bi[6 * i + j] + std::conj(Bi[6 * j + i]));
    pack_block(H, Ainv + q * 36);
  }
  return bad == 0;
}

// out(x) = A(x) in(x) (or A^-1 if the packed inverse is passed); only_parity as in hop()
static void clover_apply_lex(const Geom& g, const double* Apk, const cplx* in, cplx* out, int only_parity) {
#pragma omp parallel for schedule(static)
  for (long l = 0; l < g.V; l++) {
    if (only_parity >= 0 && g.parity(l) != only_parity) {
      for (int e = 0; e < 12; e++) out[l * 12 + e] = 0;
      continue;
    }
    for (int k = 0; k < 2; k++) {
      cplx B[36];
      unpack_block(Apk + (l * 2 + k) * 36, B);
      for (int i = 0; i < 6; i++) {
        cplx s = 0;
        for (int j = 0; j < 6; j++) s += B[6 * i + j] * in[l * 12 + 6 * k + j];
        out[l * 12 + 6 * k + i] = s;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Problem = geometry + links + clover (all lexicographic), and the operators O7, O8.
// Even-odd fields are full-lattice arrays that are zero on the other parity.
// ---------------------------------------------------------------------------------------------
struct Problem {
  Geom g;
  int tb;
  double kappa, csw, defect;
  double w[4];                     // hop weights per direction (anisotropy); 1 = isotropic
  std::vector<cplx> U;             // [4][V][9]
  std::vector<double> A, Ainv;     // [V][2][36]
  long hops;                       // number of single-parity hop sweeps executed (full = 2)
  long n() const { return g.V * 12; }
};
typedef std::vector<cplx> Field;

static void op_hop(Problem& P, const Field& in, Field& out, int dagger, int only_parity) {
  hop(P.g, P.tb, P.U.data(), in.data(), out.data(), dagger, only_parity, P.w);
  P.hops += (only_parity < 0) ? 2 : 1;
}

// O7: M psi = A psi - kappa D psi ; M^dag psi = A psi - kappa D^dag psi
static void op_mat(Problem& P, const Field& in, Field& out, int dagger) {
  Field d(P.n()), a(P.n());
  op_hop(P, in, d, dagger, -1);
  clover_apply_lex(P.g, P.A.data(), in.data(), a.data(), -1);
  for (long i = 0; i < P.n(); i++) out[i] = a[i] - P.kappa * d[i];
}

// O8: even-even Schur complement on an even-supported field.
//   asymmetric (matpc 0): Mhat   = A_ee - k^2 D_eo A_oo^-1 D_oe         (dagger: every D daggered)
//   symmetric  (matpc 1): Mhat_s = 1 - k^2 A_ee^-1 D_eo A_oo^-1 D_oe
//                         Mhat_s^dag = 1 - k^2 D^dag_eo A_oo^-1 D^dag_oe A_ee^-1
static void op_mpc(Problem& P, const Field& in, Field& out, int matpc, int dagger) {
  const long n = P.n();
  const double k2 = P.kappa * P.kappa;
  Field t1(n), t2(n), t3(n);
  if (matpc == 0) {
    op_hop(P, in, t1, dagger, 1);                                         // D_oe x_e
    clover_apply_lex(P.g, P.Ainv.data(), t1.data(), t2.data(), 1);        // A_oo^-1 .
    op_hop(P, t2, t3, dagger, 0);                                         // D_eo .
    clover_apply_lex(P.g, P.A.data(), in.data(), t1.data(), 0);           // A_ee x_e
    for (long i = 0; i < n; i++) out[i] = t1[i] - k2 * t3[i];
  } else if (!dagger) {
    op_hop(P, in, t1, 0, 1);
    clover_apply_lex(P.g, P.Ainv.data(), t1.data(), t2.data(), 1);
    op_hop(P, t2, t3, 0, 0);
    clover_apply_lex(P.g, P.Ainv.data(), t3.data(), t1.data(), 0);        // A_ee^-1 .
    for (long i = 0; i < n; i++) out[i] = in[i] - k2 * t1[i];
  } else {
    clover_apply_lex(P.g, P.Ainv.data(), in.data(), t1.data(), 0);        // A_ee^-1 x_e
    op_hop(P, t1, t2, 1, 1);
    clover_apply_lex(P.g, P.Ainv.data(), t2.data(), t1.data(), 1);
    op_hop(P, t1, t3, 1, 0);
    for (long i = 0; i < n; i++) out[i] = in[i] - k2 * t3[i];
  }
  // keep the odd half exactly zero
  for (long l = 0; l < P.g.V; l++)
    if (P.g.parity(l) == 1)
      for (int e = 0; e < 12; e++) out[l * 12 + e] = 0;
}

// complex inner product <a,b> = sum conj(a_i) b_i
static cplx dot(const Field& a, const Field& b) {
  double re = 0, im = 0;
#pragma omp parallel for schedule(static) reduction(+ : re, im)
  for (long i = 0; i < (long)a.size(); i++) {
    cplx v = std::conj(a[i]) * b[i];
    re += v.real();
    im += v.imag();
  }
  return cplx(re, im);
}
static double norm2(const Field& a) { return dot(a, a).real(); }

struct orc_result {
  int status;       // 0 converged, 1 not converged, -7 breakdown
  int iterations;
  double iter_resid;   // |r_hat| / |b_full| from the recurrence
  double true_resid;   // |b - M x| / |b| with the full operator
  double seconds;
  long hops;           // single-parity hop sweeps
};

// ---------------------------------------------------------------------------------------------
// O9 solvers on  Mhat x = bhat  (x0 = 0).  stop = tol * |b_full|.
// ---------------------------------------------------------------------------------------------
static int solve_cgne(Problem& P, const Field& bh, Field& x, int matpc, double stop, int maxiter, int& it,
                      double& rnorm) {
  const long n = P.n();
  Field r = bh, p = bh, t(n), q(n);
  std::fill(x.begin(), x.end(), cplx(0));
  double rr = norm2(r);
  for (it = 0; it < maxiter && std::sqrt(rr) > stop; it++) {
    op_mpc(P, p, t, matpc, 1);             // t = Mhat^dag p
    double tt = norm2(t);                  // <p, Mhat Mhat^dag p>
    double alpha = rr / tt;
    for (long i = 0; i < n; i++) x[i] += alpha * t[i];   // x = Mhat^dag y
    op_mpc(P, t, q, matpc, 0);             // q = Mhat t
    for (long i = 0; i < n; i++) r[i] -= alpha * q[i];
    double rr_new = norm2(r);
    double beta = rr_new / rr;
    for (long i = 0; i < n; i++) p[i] = r[i] + beta * p[i];
    rr = rr_new;
  }
  rnorm = std::sqrt(rr);
  return rnorm <= stop ? 0 : 1;
}

static int solve_cgnr(Problem& P, const Field& bh, Field& x, int matpc, double stop, int maxiter, int& it,
                      double& rnorm) {
  const long n = P.n();
  Field res = bh, r(n), p(n), t(n), q(n);   // res = bhat - Mhat x ; r = Mhat^dag res
  std::fill(x.begin(), x.end(), cplx(0));
  op_mpc(P, res, r, matpc, 1);
  p = r;
  double rr = norm2(r), resn = norm2(res);
  for (it = 0; it < maxiter && std::sqrt(resn) > stop; it++) {
    op_mpc(P, p, t, matpc, 0);             // t = Mhat p
    double alpha = rr / norm2(t);
    for (long i = 0; i < n; i++) x[i] += alpha * p[i];
    for (long i = 0; i < n; i++) res[i] -= alpha * t[i];
    op_mpc(P, t, q, matpc, 1);             // q = Mhat^dag Mhat p
    for (long i = 0; i < n; i++) r[i] -= alpha * q[i];
    double rr_new = norm2(r);
    double beta = rr_new / rr;
    for (long i = 0; i < n; i++) p[i] = r[i] + beta * p[i];
    rr = rr_new;
    resn = norm2(res);
  }
  rnorm = std::sqrt(resn);
  return rnorm <= stop ? 0 : 1;
}

static int solve_bicgstab(Problem& P, const Field& bh, Field& x, int matpc, double stop, int maxiter, int& it,
                          double& rnorm) {
  const long n = P.n();
  Field r = bh, r0 = bh, p(n, 0), v(n, 0), s(n), t(n);
  std::fill(x.begin(), x.end(), cplx(0));
  cplx rho = 1, alpha = 1, omega = 1;
  double rr = norm2(r);
  bool restarted = false;
  for (it = 0; it < maxiter && std::sqrt(rr) > stop; it++) {
    cplx rho_new = dot(r0, r);
    if (std::abs(rho_new) < 1e-300 || std::abs(omega) < 1e-300) {
      if (restarted) { rnorm = std::sqrt(rr); return -7; }
      restarted = true;
      r0 = r; rho = alpha = omega = 1;
      std::fill(p.begin(), p.end(), cplx(0));
      std::fill(v.begin(), v.end(), cplx(0));
      rho_new = dot(r0, r);
    }
    cplx beta = (rho_new / rho) * (alpha / omega);
    for (long i = 0; i < n; i++) p[i] = r[i] + beta * (p[i] - omega * v[i]);
    op_mpc(P, p, v, matpc, 0);
    alpha = rho_new / dot(r0, v);
    for (long i = 0; i < n; i++) s[i] = r[i] - alpha * v[i];
    op_mpc(P, s, t, matpc, 0);
    omega = dot(t, s) / norm2(t);
    for (long i = 0; i < n; i++) x[i] += alpha * p[i] + omega * s[i];
    for (long i = 0; i < n; i++) r[i] = s[i] - omega * t[i];
    rho = rho_new;
    rr = norm2(r);
  }
  rnorm = std::sqrt(rr);
  return rnorm <= stop ? 0 : 1;
}

// full solve M x = b via the even-odd system (O8) and reconstruction; fills res
static int invert(Problem& P, const Field& b, Field& x, double tol, int maxiter, int solver, int matpc,
                  orc_result* res) {
  auto t0 = std::chrono::steady_clock::now();
  const long n = P.n();
  const Geom& g = P.g;
  P.hops = 0;
  Field t1(n), t2(n), bh(n), xe(n);
  double bnorm = std::sqrt(norm2(b));
  if (bnorm == 0) {
    std::fill(x.begin(), x.end(), cplx(0));
    *res = orc_result{0, 0, 0.0, 0.0, 0.0, 0};
    return 0;
  }
  // bhat = b_e + kappa D_eo A_oo^-1 b_o
  clover_apply_lex(g, P.Ainv.data(), b.data(), t1.data(), 1);
  op_hop(P, t1, t2, 0, 0);
  for (long l = 0; l < g.V; l++)
    for (int e = 0; e < 12; e++) bh[l * 12 + e] = (g.parity(l) == 0) ? b[l * 12 + e] + P.kappa * t2[l * 12 + e] : cplx(0);
  if (matpc == 1) {  // bhat_s = A_ee^-1 bhat
    clover_apply_lex(g, P.Ainv.data(), bh.data(), t1.data(), 0);
    bh = t1;
  }
  int it = 0, status;
  double rnorm = 0;
  const double stop = tol * bnorm;
  if (solver == 0) status = solve_cgne(P, bh, xe, matpc, stop, maxiter, it, rnorm);
  else if (solver == 1) status = solve_cgnr(P, bh, xe, matpc, stop, maxiter, it, rnorm);
  else status = solve_bicgstab(P, bh, xe, matpc, stop, maxiter, it, rnorm);
  // x_o = A_oo^-1 (b_o + kappa D_oe x_e)
  op_hop(P, xe, t1, 0, 1);
  for (long l = 0; l < g.V; l++)
    for (int e = 0; e < 12; e++) t2[l * 12 + e] = (g.parity(l) == 1) ? b[l * 12 + e] + P.kappa * t1[l * 12 + e] : cplx(0);
  clover_apply_lex(g, P.Ainv.data(), t2.data(), t1.data(), 1);
  for (long i = 0; i < n; i++) x[i] = xe[i] + t1[i];
  // true residual with the full operator
  long hops_solve = P.hops;
  op_mat(P, x, t1, 0);
  for (long i = 0; i < n; i++) t1[i] = b[i] - t1[i];
  res->status = status;
  res->iterations = it;
  res->iter_resid = rnorm / bnorm;
  res->true_resid = std::sqrt(norm2(t1)) / bnorm;
  res->hops = hops_solve;
  res->seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
  return status;
}

// ---------------------------------------------------------------------------------------------
// C entry points (public cb2 layouts in and out).
// ---------------------------------------------------------------------------------------------
static void spinor_in(const Problem& P, const double* pub, Field& f) {
  f.resize(P.n());
  to_lex(P.g, reinterpret_cast<const cplx*>(pub), f.data(), 12);
}
static void spinor_out(const Problem& P, const Field& f, double* pub) {
  from_lex(P.g, f.data(), reinterpret_cast<cplx*>(pub), 12);
}

extern "C" {

int orc_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// mu = 0..3 -> gamma_x..gamma_t, 4 -> gamma_5 ; out = 4x4 complex row-major
void orc_gamma(int mu, double* out) { std::memcpy(out, GM.g[mu], sizeof(cplx) * 16); }
void orc_sigma(int mu, int nu, double* out) { std::memcpy(out, GM.sig[mu][nu], sizeof(cplx) * 16); }

void* orc_create(const int* dims, int t_boundary, const double* U_public) {
  Problem* P = new Problem();
  if (!make_geom(dims, P->g) || (t_boundary != 1 && t_boundary != -1)) {
    delete P;
    return nullptr;
  }
  P->tb = t_boundary;
  P->kappa = 0; P->csw = 0; P->defect = 0; P->hops = 0;
  for (int mu = 0; mu < 4; mu++) P->w[mu] = 1.0;
  P->U.resize((size_t)4 * P->g.V * 9);
  gauge_to_lex(P->g, reinterpret_cast<const cplx*>(U_public), P->U.data());
  return P;
}
void orc_destroy(void* h) { delete static_cast<Problem*>(h); }

// Build A = 1 - kappa*csw*sigma.F and its inverse; also fixes kappa for orc_mat/orc_mpc/orc_invert.
// csw = 0 gives A = 1 (plain Wilson).  Returns 0, or -6 if some block is singular.
int orc_set_clover(void* h, double kappa, double csw) {
  Problem& P = *static_cast<Problem*>(h);
  P.kappa = kappa;
  P.csw = csw;
  P.A.assign((size_t)P.g.V * 72, 0.0);
  P.Ainv.assign((size_t)P.g.V * 72, 0.0);
  P.defect = clover_build_lex(P.g, P.U.data(), kappa, csw, csw, P.A.data());
  return clover_invert_lex(P.g, P.A.data(), P.Ainv.data()) ? 0 : -6;
}
// Anisotropic operator of Eq. 5 in kappa normalisation:
//   M = 1 - kappa [ D_t + (nu/xi_0) sum_i D_i ] - kappa [ c_SW^t sum_i sigma_i4 F_i4 + (c_SW^r/xi_0) sum_{i<j} sigma_ij F_ij ]
// orc_set_anisotropy fixes the spatial hop weight nu/xi_0 for every later operator call;
// orc_set_clover_aniso builds A with separate spatial (csw_s = c_SW^r/xi_0) and temporal (csw_t) coefficients.
void orc_set_anisotropy(void* h, double nu_over_xi0) {
  Problem& P = *static_cast<Problem*>(h);
  P.w[0] = P.w[1] = P.w[2] = nu_over_xi0;
  P.w[3] = 1.0;
}
int orc_set_clover_aniso(void* h, double kappa, double csw_s, double csw_t) {
  Problem& P = *static_cast<Problem*>(h);
  P.kappa = kappa;
  P.csw = csw_s;
  P.A.assign((size_t)P.g.V * 72, 0.0);
  P.Ainv.assign((size_t)P.g.V * 72, 0.0);
  P.defect = clover_build_lex(P.g, P.U.data(), kappa, csw_s, csw_t, P.A.data());
  return clover_invert_lex(P.g, P.A.data(), P.Ainv.data()) ? 0 : -6;
}
// largest |entry| of the off-diagonal chiral blocks / anti-Hermitian part seen by the last build
double orc_clover_defect(void* h) { return static_cast<Problem*>(h)->defect; }

// packed clover fields in the public layout [2][Vh][2][36]
void orc_get_clover(void* h, double* A_public, double* Ainv_public) {
  Problem& P = *static_cast<Problem*>(h);
  for (long l = 0; l < P.g.V; l++) {
    long c = P.g.cb(l);
    if (A_public) std::memcpy(A_public + c * 72, P.A.data() + l * 72, sizeof(double) * 72);
    if (Ainv_public) std::memcpy(Ainv_public + c * 72, P.Ainv.data() + l * 72, sizeof(double) * 72);
  }
}
// dense 12x12 clover matrices for every site, public site order: [2][Vh][12][12] complex
void orc_clover_dense(void* h, double kappa, double csw, double* out) {
  Problem& P = *static_cast<Problem*>(h);
  cplx* o = reinterpret_cast<cplx*>(out);
#pragma omp parallel for schedule(static)
  for (long l = 0; l < P.g.V; l++) clover_dense_site(P.g, P.U.data(), l, kappa, csw, csw, o + P.g.cb(l) * 144);
}
// F_{mu nu}(x) for all sites: [2][Vh][3][3] complex
void orc_fmunu(void* h, int mu, int nu, double* out) {
  Problem& P = *static_cast<Problem*>(h);
  cplx* o = reinterpret_cast<cplx*>(out);
#pragma omp parallel for schedule(static)
  for (long l = 0; l < P.g.V; l++) field_strength(P.g, P.U.data(), l, mu, nu, o + P.g.cb(l) * 9);
}

// out = D in (or D^dag in); only_parity = -1 all sites, 0/1 only that output parity (rest zero)
void orc_dslash(void* h, const double* in, double* out, int dagger, int only_parity) {
  Problem& P = *static_cast<Problem*>(h);
  Field fi, fo(P.n());
  spinor_in(P, in, fi);
  op_hop(P, fi, fo, dagger, only_parity);
  spinor_out(P, fo, out);
}
// (D in) at ONE output site given by its public index; out = 12 complex.  For sampled checks.
void orc_dslash_site(void* h, const double* in_public, long public_index, int dagger, double* out) {
  Problem& P = *static_cast<Problem*>(h);
  const Geom& g = P.g;
  long par = public_index / g.Vh, c = public_index % g.Vh, l = -1;
  for (long q = 2 * c; q < 2 * c + 2; q++)
    if (g.parity(q) == par) l = q;
  const cplx* in = reinterpret_cast<const cplx*>(in_public);
  const double sgn = dagger ? -1.0 : 1.0;
  cplx acc[12];
  for (int e = 0; e < 12; e++) acc[e] = 0;
  int x[4];
  g.coords(l, x);
  for (int mu = 0; mu < 4; mu++)
    for (int dir = 0; dir < 2; dir++) {
      long ln = g.shift(l, mu, dir == 0 ? +1 : -1);
      const cplx* u = P.U.data() + ((long)mu * g.V + (dir == 0 ? l : ln)) * 9;
      const cplx* p = in + g.cb(ln) * 12;
      double bs = 1.0;
      if (mu == 3 && P.tb < 0 && ((dir == 0 && x[3] == g.L[3] - 1) || (dir == 1 && x[3] == 0))) bs = -1.0;
      cplx up[4][3];
      for (int s = 0; s < 4; s++)
        for (int a = 0; a < 3; a++) {
          cplx v = 0;
          for (int b = 0; b < 3; b++) v += (dir == 0 ? u[3 * a + b] : std::conj(u[3 * b + a])) * p[3 * s + b];
          up[s][a] = v;
        }
      const double gs = (dir == 0 ? -1.0 : 1.0) * sgn;
      for (int s = 0; s < 4; s++)
        for (int a = 0; a < 3; a++) {
          cplx v = up[s][a];
          for (int s2 = 0; s2 < 4; s2++) v += gs * GM.g[mu][s][s2] * up[s2][a];
          acc[3 * s + a] += P.w[mu] * bs * v;
        }
    }
  std::memcpy(out, acc, sizeof(acc));
}

void orc_clover_apply(void* h, const double* in, double* out, int inverse, int only_parity) {
  Problem& P = *static_cast<Problem*>(h);
  Field fi, fo(P.n());
  spinor_in(P, in, fi);
  clover_apply_lex(P.g, inverse ? P.Ainv.data() : P.A.data(), fi.data(), fo.data(), only_parity);
  spinor_out(P, fo, out);
}

void orc_mat(void* h, const double* in, double* out, int dagger) {
  Problem& P = *static_cast<Problem*>(h);
  Field fi, fo(P.n());
  spinor_in(P, in, fi);
  op_mat(P, fi, fo, dagger);
  spinor_out(P, fo, out);
}

// in/out: full public spinors; the odd half of `in` is ignored, the odd half of `out` is zero
void orc_mpc(void* h, const double* in, double* out, int matpc, int dagger) {
  Problem& P = *static_cast<Problem*>(h);
  Field fi, fo(P.n());
  spinor_in(P, in, fi);
  for (long l = 0; l < P.g.V; l++)
    if (P.g.parity(l) == 1)
      for (int e = 0; e < 12; e++) fi[l * 12 + e] = 0;
  op_mpc(P, fi, fo, matpc, dagger);
  spinor_out(P, fo, out);
}

// solver: 0 CGNE, 1 CGNR, 2 BiCGStab ; matpc: 0 asymmetric, 1 symmetric
int orc_invert(void* h, const double* b, double* x, double tol, int maxiter, int solver, int matpc,
               orc_result* res) {
  Problem& P = *static_cast<Problem*>(h);
  Field fb, fx(P.n());
  spinor_in(P, b, fb);
  int st = invert(P, fb, fx, tol, maxiter, solver, matpc, res);
  spinor_out(P, fx, x);
  return st;
}

// |b - M x| / |b| with the full operator (used to verify solutions that come from elsewhere)
double orc_true_residual(void* h, const double* b, const double* x) {
  Problem& P = *static_cast<Problem*>(h);
  Field fb, fx, t(P.n());
  spinor_in(P, b, fb);
  spinor_in(P, x, fx);
  op_mat(P, fx, t, 0);
  for (long i = 0; i < P.n(); i++) t[i] = fb[i] - t[i];
  return std::sqrt(norm2(t) / norm2(fb));
}

}  // extern "C"
