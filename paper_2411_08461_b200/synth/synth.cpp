// Seeded synthetic-input generator.
//
// This module only MAKES inputs: SU(3) link fields U = exp(i*eps*H) and source vectors, in the
// paper's public cb2 layout (§II.A "Convention").  It holds none of the method's
// arithmetic (no gamma matrices, no hopping term, no clover, no solver) and is the only code
// that the CPU oracle's tests and the CUDA path's tests both use.
//
// Random numbers: counter-based.  Every value is a pure function of
// (seed, field id, lexicographic site, mu, component index), via a splitmix64 hash chain and
// Box-Muller, so a site's link does not depend on traversal order or thread count.
//
// Layouts written (all complex numbers as interleaved (re, im) doubles):
//   gauge  [4][2][Lt][Lz][Ly][Lx/2][3][3]   row-column colour order, mu = x,y,z,t
//   spinor [2][Lt][Lz][Ly][Lx/2][4][3]
//   colour matrix field [2][Lt][Lz][Ly][Lx/2][3][3]
// Site (x,y,z,t): parity = (x+y+z+t)&1, index inside a parity = (x + Lx*(y + Ly*(z + Lz*t)))/2.
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>

typedef std::complex<double> cplx;

static inline uint64_t mix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// key for one (seed, field, site, mu) cell; component counters are hashed on top of it
static inline uint64_t cell_key(uint64_t seed, uint64_t field, uint64_t site, uint64_t mu) {
  uint64_t k = mix64(seed);
  k = mix64(k ^ (field * 0xD1B54A32D192ED03ull));
  k = mix64(k ^ (site * 4 + mu));
  return k;
}
static inline uint64_t draw(uint64_t key, uint64_t counter) {
  return mix64(key + counter * 0x9E3779B97F4A7C15ull);
}
static inline double u01(uint64_t r) {  // (0,1]
  return ((double)(r >> 11) + 1.0) * (1.0 / 9007199254740992.0);
}
// two independent N(0,1) from counters (2c, 2c+1)
static inline void normal2(uint64_t key, uint64_t c, double& a, double& b) {
  double u1 = u01(draw(key, 2 * c)), u2 = u01(draw(key, 2 * c + 1));
  double r = std::sqrt(-2.0 * std::log(u1));
  a = r * std::cos(2.0 * M_PI * u2);
  b = r * std::sin(2.0 * M_PI * u2);
}

static void mat_mul(const cplx* a, const cplx* b, cplx* c) {
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      cplx s = 0;
      for (int k = 0; k < 3; k++) s += a[3 * i + k] * b[3 * k + j];
      c[3 * i + j] = s;
    }
}

// U = exp(i*eps*H), H = Hermitian traceless part of a complex Gaussian matrix; then reunitarise.
static void make_su3(uint64_t key, double eps, cplx* U) {
  cplx G[9], H[9];
  for (int e = 0; e < 9; e++) {
    double a, b;
    normal2(key, e, a, b);
    G[e] = cplx(a, b);
  }
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) H[3 * i + j] = 0.5 * (G[3 * i + j] + std::conj(G[3 * j + i]));
  cplx tr = (H[0] + H[4] + H[8]) / 3.0;
  H[0] -= tr; H[4] -= tr; H[8] -= tr;
  // X = i*eps*H / 2^s with small norm; Taylor series; square s times
  double nrm = 0;
  for (int e = 0; e < 9; e++) nrm += std::norm(H[e]);
  nrm = std::sqrt(nrm) * std::fabs(eps);
  int s = 0;
  while (nrm > 0.25) { nrm *= 0.5; s++; }
  double sc = eps / (double)(1ull << s);
  cplx X[9], T[9], E[9], W[9];
  for (int e = 0; e < 9; e++) X[e] = cplx(0, sc) * H[e];
  for (int e = 0; e < 9; e++) { E[e] = (e % 4 == 0) ? 1.0 : 0.0; T[e] = E[e]; }
  for (int n = 1; n <= 20; n++) {
    mat_mul(T, X, W);
    for (int e = 0; e < 9; e++) { T[e] = W[e] / (double)n; E[e] += T[e]; }
  }
  for (int q = 0; q < s; q++) {
    mat_mul(E, E, W);
    std::memcpy(E, W, sizeof(W));
  }
  // reunitarise: Gram-Schmidt rows 0,1; row 2 = conj(row0 x row1)
  double n0 = 0;
  for (int j = 0; j < 3; j++) n0 += std::norm(E[j]);
  n0 = 1.0 / std::sqrt(n0);
  for (int j = 0; j < 3; j++) E[j] *= n0;
  cplx d = 0;
  for (int j = 0; j < 3; j++) d += std::conj(E[j]) * E[3 + j];
  for (int j = 0; j < 3; j++) E[3 + j] -= d * E[j];
  double n1 = 0;
  for (int j = 0; j < 3; j++) n1 += std::norm(E[3 + j]);
  n1 = 1.0 / std::sqrt(n1);
  for (int j = 0; j < 3; j++) E[3 + j] *= n1;
  E[6] = std::conj(E[1] * E[5] - E[2] * E[4]);
  E[7] = std::conj(E[2] * E[3] - E[0] * E[5]);
  E[8] = std::conj(E[0] * E[4] - E[1] * E[3]);
  std::memcpy(U, E, sizeof(E));
}

struct Lat {
  int L[4];
  long V, Vh;
};
static bool make_lat(const int* dims, Lat& g) {
  g.V = 1;
  for (int i = 0; i < 4; i++) {
    if (dims[i] < 2 || (dims[i] & 1)) return false;
    g.L[i] = dims[i];
    g.V *= dims[i];
  }
  g.Vh = g.V / 2;
  return true;
}
static inline long cb_index(const Lat& g, long lex) {  // position in [2][Vh]
  int x = lex % g.L[0];
  long r = lex / g.L[0];
  int y = r % g.L[1]; r /= g.L[1];
  int z = r % g.L[2];
  int t = r / g.L[2];
  int par = (x + y + z + t) & 1;
  return par * g.Vh + lex / 2;
}

extern "C" {

// field ids: 1 = gauge, 2 = gauge transformation, 3 = source
int synth_gauge(const int* dims, double eps, uint64_t seed, double* U_public) {
  Lat g;
  if (!make_lat(dims, g)) return -1;
  cplx* out = reinterpret_cast<cplx*>(U_public);
#pragma omp parallel for schedule(static)
  for (long lex = 0; lex < g.V; lex++) {
    long cb = cb_index(g, lex);
    for (int mu = 0; mu < 4; mu++) {
      cplx U[9];
      make_su3(cell_key(seed, 1, (uint64_t)lex, mu), eps, U);
      std::memcpy(out + ((long)mu * g.V + cb) * 9, U, sizeof(U));
    }
  }
  return 0;
}

// one SU(3) matrix per site, for gauge-covariance tests
int synth_colour_rotation(const int* dims, double eps, uint64_t seed, double* g_public) {
  Lat g;
  if (!make_lat(dims, g)) return -1;
  cplx* out = reinterpret_cast<cplx*>(g_public);
#pragma omp parallel for schedule(static)
  for (long lex = 0; lex < g.V; lex++) {
    cplx U[9];
    make_su3(cell_key(seed, 2, (uint64_t)lex, 0), eps, U);
    std::memcpy(out + cb_index(g, lex) * 9, U, sizeof(U));
  }
  return 0;
}

// kind: 0 = point at the origin (spin, colour) ; 1 = Z2 (+-1 + 0i) ; 2 = Gaussian complex
int synth_source(const int* dims, int kind, uint64_t seed, int spin, int colour, double* b_public) {
  Lat g;
  if (!make_lat(dims, g)) return -1;
  if (kind < 0 || kind > 2) return -2;
  cplx* out = reinterpret_cast<cplx*>(b_public);
  if (kind == 0) {
    if (spin < 0 || spin > 3 || colour < 0 || colour > 2) return -2;
    std::memset(b_public, 0, sizeof(double) * 2 * 12 * g.V);
    out[0 * 12 + spin * 3 + colour] = 1.0;  // origin is even, cb index 0
    return 0;
  }
#pragma omp parallel for schedule(static)
  for (long lex = 0; lex < g.V; lex++) {
    uint64_t key = cell_key(seed, 3, (uint64_t)lex, 0);
    cplx* o = out + cb_index(g, lex) * 12;
    for (int e = 0; e < 12; e++) {
      if (kind == 1) {
        o[e] = (draw(key, e) >> 63) ? 1.0 : -1.0;
      } else {
        double a, b;
        normal2(key, e, a, b);
        o[e] = cplx(a, b);
      }
    }
  }
  return 0;
}

}  // extern "C"
