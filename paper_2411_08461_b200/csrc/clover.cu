// K4/K5: clover term from the clover-leaf field strength and its per-site inverse
// ("the clover field is then created"; PAPER.md:56 packed layout; SURVEY.md §8(c)
// O4-O6).  All arithmetic in fp64 whatever the storage precision; one thread per site.
//
//   F_{mu nu} = (Q - Q^dag)/(8i),  Q = sum of the four leaves around x (counter-clockwise)
//   A = 1 - kappa*csw*sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}.   In the DeGrand-Rossi basis
//   sigma_{mu nu} is block diagonal, so with  E3 = F_xy -/+ F_zt, E2 = F_xz +/- F_yt,
//   E1 = F_yz -/+ F_xt  (upper sign: spins 0,1; lower sign: spins 2,3)
//   A_block = 1 - kappa*csw * [[E3, E1 - i E2], [E1 + i E2, -E3]],  row index = 3*spin + colour.
//   Anisotropic form (Eq. 5): csw -> c_SW^r/xi_0 on the planes xy, xz, yz and c_SW^t on xt, yt, zt.
#include "lqcd_internal.cuh"

struct cd {
  double re, im;
};
__device__ __forceinline__ cd operator+(cd a, cd b) { return {a.re + b.re, a.im + b.im}; }
__device__ __forceinline__ cd operator-(cd a, cd b) { return {a.re - b.re, a.im - b.im}; }
__device__ __forceinline__ cd operator*(cd a, cd b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ cd conj(cd a) { return {a.re, -a.im}; }
__device__ __forceinline__ double abs2(cd a) { return a.re * a.re + a.im * a.im; }

struct M3 {
  cd m[9];
};
// c = a b, every term one DFMA (a*b + c*d + ... written with operators costs DMUL + DFMA + DADD per product)
__device__ __forceinline__ M3 mul(const M3& a, const M3& b) {
  M3 c;
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      double re = a.m[3 * i].re * b.m[j].re, im = a.m[3 * i].re * b.m[j].im;
      re = fma(-a.m[3 * i].im, b.m[j].im, re);
      im = fma(a.m[3 * i].im, b.m[j].re, im);
#pragma unroll
      for (int k = 1; k < 3; k++) {
        re = fma(a.m[3 * i + k].re, b.m[3 * k + j].re, re);
        re = fma(-a.m[3 * i + k].im, b.m[3 * k + j].im, re);
        im = fma(a.m[3 * i + k].re, b.m[3 * k + j].im, im);
        im = fma(a.m[3 * i + k].im, b.m[3 * k + j].re, im);
      }
      c.m[3 * i + j] = {re, im};
    }
  return c;
}
__device__ __forceinline__ M3 dag(const M3& a) {
  M3 c;
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) c.m[3 * i + j] = conj(a.m[3 * j + i]);
  return c;
}

// link U_mu at lattice coordinates (x,y,z,t) (already wrapped), promoted to fp64
template <typename T, int R>
__device__ __forceinline__ M3 link_at(const T* __restrict__ gauge, const Lat& L, int mu, const int* x) {
  const int par = (x[0] + x[1] + x[2] + x[3]) & 1;
  const int idx = (x[0] >> 1) + L.Lxh * (x[1] + L.Ly * (x[2] + L.Lz * x[3]));
  T U[18];
  load_link<T, R>(gauge + (size_t)(mu * 2 + par) * R * L.Vh, L.Vh, idx, U);
  M3 m;
#pragma unroll
  for (int e = 0; e < 9; e++) m.m[e] = {(double)U[2 * e], (double)U[2 * e + 1]};
  return m;
}

__device__ __forceinline__ void step(const Lat& L, int* x, int mu, int s) {
  const int ext = (mu == 0) ? 2 * L.Lxh : (mu == 1) ? L.Ly : (mu == 2) ? L.Lz : L.Lt;
  int v = x[mu] + s;
  x[mu] = v < 0 ? v + ext : (v >= ext ? v - ext : v);
}

// F_{mu nu}(x) as 9 complex numbers
template <typename T, int R>
__device__ void field_strength(const T* __restrict__ g, const Lat& L, const int* x0, int mu, int nu, cd* F) {
  int x[4], a[4], b[4], c[4];
  M3 Q;
  // P1 = U_mu(x) U_nu(x+mu) U_mu^dag(x+nu) U_nu^dag(x)
  for (int i = 0; i < 4; i++) x[i] = a[i] = b[i] = x0[i];
  step(L, a, mu, +1);
  step(L, b, nu, +1);
  Q = mul(mul(link_at<T, R>(g, L, mu, x), link_at<T, R>(g, L, nu, a)),
          mul(dag(link_at<T, R>(g, L, mu, b)), dag(link_at<T, R>(g, L, nu, x))));
  // P2 = U_nu(x) U_mu^dag(x-mu+nu) U_nu^dag(x-mu) U_mu(x-mu)
  for (int i = 0; i < 4; i++) a[i] = b[i] = x0[i];
  step(L, a, mu, -1);           // x-mu
  for (int i = 0; i < 4; i++) b[i] = a[i];
  step(L, b, nu, +1);           // x-mu+nu
  {
    M3 P = mul(mul(link_at<T, R>(g, L, nu, x), dag(link_at<T, R>(g, L, mu, b))),
               mul(dag(link_at<T, R>(g, L, nu, a)), link_at<T, R>(g, L, mu, a)));
    for (int e = 0; e < 9; e++) Q.m[e] = Q.m[e] + P.m[e];
  }
  // P3 = U_mu^dag(x-mu) U_nu^dag(x-mu-nu) U_mu(x-mu-nu) U_nu(x-nu)
  for (int i = 0; i < 4; i++) b[i] = a[i];
  step(L, b, nu, -1);           // x-mu-nu
  for (int i = 0; i < 4; i++) c[i] = x0[i];
  step(L, c, nu, -1);           // x-nu
  {
    M3 P = mul(mul(dag(link_at<T, R>(g, L, mu, a)), dag(link_at<T, R>(g, L, nu, b))),
               mul(link_at<T, R>(g, L, mu, b), link_at<T, R>(g, L, nu, c)));
    for (int e = 0; e < 9; e++) Q.m[e] = Q.m[e] + P.m[e];
  }
  // P4 = U_nu^dag(x-nu) U_mu(x-nu) U_nu(x+mu-nu) U_mu^dag(x)
  for (int i = 0; i < 4; i++) b[i] = c[i];
  step(L, b, mu, +1);           // x+mu-nu
  {
    M3 P = mul(mul(dag(link_at<T, R>(g, L, nu, c)), link_at<T, R>(g, L, mu, c)),
               mul(link_at<T, R>(g, L, nu, b), dag(link_at<T, R>(g, L, mu, x))));
    for (int e = 0; e < 9; e++) Q.m[e] = Q.m[e] + P.m[e];
  }
  // (Q - Q^dag)/(8i):  (z)/(i) = -i z
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      cd d = Q.m[3 * i + j] - conj(Q.m[3 * j + i]);
      F[3 * i + j] = {0.125 * d.im, -0.125 * d.re};
    }
}

// In-place Gauss-Jordan inverse with partial (row) pivoting of a 6x6 complex matrix (SURVEY.md §8(c)
// O6: no positive-definiteness assumed).  Every loop is unrolled with compile-time indices and the
// run-time pivot row only enters comparisons, so the 36 complex numbers stay in registers (the first
// version kept [A | 1] in local memory and spent 60 % of the build there).  Row swaps are recorded and
// undone as column swaps at the end.  Returns false when a pivot is below 1e-12 * max|A|.
__device__ __forceinline__ bool invert6(cd (&a)[6][6]) {
  double nrm = 0;
#pragma unroll
  for (int i = 0; i < 6; i++)
#pragma unroll
    for (int j = 0; j < 6; j++) nrm = fmax(nrm, abs2(a[i][j]));
  const double thresh = 1e-24 * nrm;
  int perm[6];
  bool ok = true;
#pragma unroll
  for (int c = 0; c < 6; c++) {
    int piv = c;
    double best = abs2(a[c][c]);
#pragma unroll
    for (int r = c + 1; r < 6; r++) {
      const double v = abs2(a[r][c]);
      if (v > best) { best = v; piv = r; }
    }
    ok = ok && (best > thresh);
    perm[c] = piv;
#pragma unroll
    for (int r = c + 1; r < 6; r++) {
      const bool sw = (piv == r);
#pragma unroll
      for (int j = 0; j < 6; j++) {
        const cd t = a[c][j], u = a[r][j];
        a[c][j] = sw ? u : t;
        a[r][j] = sw ? t : u;
      }
    }
    const cd p = a[c][c];
    const double ib = best > 0.0 ? 1.0 / best : 0.0;
    const cd inv = {p.re * ib, -p.im * ib};
    a[c][c] = {1.0, 0.0};
#pragma unroll
    for (int j = 0; j < 6; j++) a[c][j] = a[c][j] * inv;
#pragma unroll
    for (int r = 0; r < 6; r++) {
      if (r == c) continue;
      const cd f = a[r][c];
      a[r][c] = {0.0, 0.0};
#pragma unroll
      for (int j = 0; j < 6; j++) a[r][j] = a[r][j] - f * a[c][j];
    }
  }
  // (P A)^-1 = A^-1 P^T: undo the row swaps as column swaps, last first
#pragma unroll
  for (int c = 5; c >= 0; c--) {
#pragma unroll
    for (int r = c + 1; r < 6; r++) {
      const bool sw = (perm[c] == r);
#pragma unroll
      for (int i = 0; i < 6; i++) {
        const cd t = a[i][c], u = a[i][r];
        a[i][c] = sw ? u : t;
        a[i][r] = sw ? t : u;
      }
    }
  }
  return ok;
}

template <typename T>
__device__ __forceinline__ void store_block(T* __restrict__ field, int Vh, int idx, int k, const double* p36) {
  typedef typename V16<T>::vec vec;
  constexpr int N = V16<T>::N;
  vec* dst = reinterpret_cast<vec*>(field) + idx;
  for (int q = 0; q < 36 / N; q++) {
    T r[N];
    for (int e = 0; e < N; e++) r[e] = (T)p36[q * N + e];
    vec w;
    vec_set(w, r);
    dst[(size_t)(k * (36 / N) + q) * Vh] = w;
  }
}

// Thread layout: blockDim = (CB_SITES sites, 6 planes).  Phase 1: thread (s, pl) computes F of plane pl
// at site s (4 leaves, 12 matrix products, 16 link loads) and parks it in shared memory, so the six
// planes of a site run in parallel and no thread holds more than one F.  Phase 2: threads (s, k < 2)
// assemble chiral block k, pack it, invert it by Gauss-Jordan and store both.
constexpr int CB_SITES = 32;
#ifndef CB_ZC
#define CB_ZC 4  // z-planes per slab of the traversal order
#endif
#ifndef CB_MINB
#define CB_MINB 2  // 170 registers, 12 warps/SM: 5.84 -> 4.59 ms at 32^3x64 fp64 (3 blocks/SM spill: 9.1 ms)
#endif
// F of one plane for NS sites in shared memory.  F is Hermitian exactly (both triangles come from the same
// difference): 3 real diagonals, then (re, im) of F_01, F_02, F_12.
template <int NS>
__device__ __forceinline__ cd herm_entry(const double (&F)[9][NS], int i, int j, int ls) {
  if (i == j) return {F[i][ls], 0.0};
  const int lo = i < j ? i : j, hi = i < j ? j : i;
  const int e = 3 + 2 * (lo + hi - 1);  // (0,1) -> 3, (0,2) -> 5, (1,2) -> 7
  return {F[e][ls], i < j ? F[e + 1][ls] : -F[e + 1][ls]};
}
template <int NS>
__device__ __forceinline__ void herm_store(double (&F)[9][NS], int ls, const cd* f9) {
  F[0][ls] = f9[0].re;
  F[1][ls] = f9[4].re;
  F[2][ls] = f9[8].re;
  F[3][ls] = f9[1].re;
  F[4][ls] = f9[1].im;
  F[5][ls] = f9[2].re;
  F[6][ls] = f9[2].im;
  F[7][ls] = f9[5].re;
  F[8][ls] = f9[5].im;
}
// Inverse of a Hermitian positive definite 6x6 matrix held as its packed lower triangle (6 real diagonals dg, 15
// complex entries lo[i(i-1)/2+j], i > j) by the symmetric sweep operator: for k = 0..5
//   d = a_kk;  a_ij -= a_ik a_kj / d (i, j != k);  a_ik /= d;  a_kk = -1/d        and the result is -A^-1.
// The pivot of step k is the k-th pivot of the LDL^H factorisation, so "every pivot > thresh" proves positive
// definiteness, for which elimination without pivoting is stable.  Half the multiply-adds of Gauss-Jordan on the full
// matrix and no row exchanges (two thirds of invert6's instructions are the selects of its swap networks).  Returns
// false as soon as a pivot fails the test (the matrix is then left half swept).
__device__ __forceinline__ bool sweep6(double (&dg)[6], cd (&lo)[15], double thresh) {
  bool ok = true;
#pragma unroll
  for (int k = 0; k < 6; k++) {
    const double d = dg[k];
    ok = ok && (d > thresh);
    const double id = 1.0 / d;
    cd col[6];  // a_ik, i != k
#pragma unroll
    for (int i = 0; i < 6; i++) {
      if (i == k) continue;
      col[i] = i > k ? lo[i * (i - 1) / 2 + k] : conj(lo[k * (k - 1) / 2 + i]);
    }
#pragma unroll
    for (int i = 0; i < 6; i++) {
      if (i == k) continue;
      const cd bi = {col[i].re * id, col[i].im * id};
      dg[i] = fma(-bi.re, col[i].re, fma(-bi.im, col[i].im, dg[i]));
#pragma unroll
      for (int j = 0; j < i; j++) {
        if (j == k) continue;
        cd& a = lo[i * (i - 1) / 2 + j];  // a_ij -= (a_ik / d) conj(a_jk)
        a.re = fma(-bi.re, col[j].re, fma(-bi.im, col[j].im, a.re));
        a.im = fma(-bi.im, col[j].re, fma(bi.re, col[j].im, a.im));
      }
      if (i > k)
        lo[i * (i - 1) / 2 + k] = bi;
      else
        lo[k * (k - 1) / 2 + i] = conj(bi);
    }
    dg[k] = -id;
  }
  return ok;
}

// chiral block k of a site from the six F in shared memory: A_block = 1 - [[E3, E1 - i E2], [E1 + i E2, -E3]] with
// E3 = kc F_xy -/+ kt F_zt, E2 = kc F_xz +/- kt F_yt, E1 = kc F_yz -/+ kt F_xt (upper sign: k = 0);
// kc = kappa*csw on the spatial planes, kt = kappa*csw_t on the temporal ones (Eq. 5)
template <int NS>
__device__ __forceinline__ void assemble_block(const double (&Fs)[6][9][NS], int ls, int k, double kc, double kt, cd (&B)[6][6]) {
  const double st = (k == 0 ? 1.0 : -1.0) * kt;
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int j = 0; j < 3; j++) {
      const cd Fxy = herm_entry(Fs[0], i, j, ls), Fxz = herm_entry(Fs[1], i, j, ls), Fxt = herm_entry(Fs[2], i, j, ls),
               Fyz = herm_entry(Fs[3], i, j, ls), Fyt = herm_entry(Fs[4], i, j, ls), Fzt = herm_entry(Fs[5], i, j, ls);
      const cd E3 = {kc * Fxy.re - st * Fzt.re, kc * Fxy.im - st * Fzt.im};
      const cd E2 = {kc * Fxz.re + st * Fyt.re, kc * Fxz.im + st * Fyt.im};
      const cd E1 = {kc * Fyz.re - st * Fxt.re, kc * Fyz.im - st * Fxt.im};
      const double d = (i == j) ? 1.0 : 0.0;
      B[i][j] = {d - E3.re, -E3.im};
      B[3 + i][3 + j] = {d + E3.re, E3.im};
      B[i][3 + j] = {-(E1.re + E2.im), -(E1.im - E2.re)};  // E1 - i E2
      B[3 + i][j] = {-(E1.re - E2.im), -(E1.im + E2.re)};  // E1 + i E2
    }
}

// the rare path of clover_blocks, out of line so that its registers and spills are not the common path's
template <typename T, int NS>
__device__ __noinline__ void general_inverse_store(const double (&Fs)[6][9][NS], int ls, int k, double kc, double kt,
                                                   T* __restrict__ field, int Vh, int idx, int* flag) {
  double pk[36];
  cd a[6][6];
  assemble_block(Fs, ls, k, kc, kt, a);
  if (!invert6(a)) {
    atomicExch(flag, 1);
    for (int i = 0; i < 36; i++) pk[i] = 0;
  } else {
    for (int i = 0; i < 6; i++) pk[i] = a[i][i].re;
    for (int i = 1; i < 6; i++)
      for (int j = 0; j < i; j++) {
        // average the two triangles so rounding stays symmetric
        const int o = 6 + 2 * (i * (i - 1) / 2 + j);
        pk[o] = 0.5 * (a[i][j].re + a[j][i].re);
        pk[o + 1] = 0.5 * (a[i][j].im - a[j][i].im);
      }
  }
  store_block<T>(field, Vh, idx, k, pk);
}

// Phase 2 of either build: thread k < 2 of a site assembles chiral block k (exactly Hermitian: the shared-memory F
// are), packs and stores it, and inverts it: by the sweep above where every pivot exceeds 1e-6 of the largest
// diagonal entry (every block of a sensible field: at configs 3 and 4 the smallest pivot is 0.6), otherwise -- not
// positive definite or nearly singular -- by Gauss-Jordan with partial pivoting on the re-assembled block
// (no positive-definiteness assumed), which also decides LQCD_ERR_SINGULAR_CLOVER.
template <typename T, int NS>
__device__ __forceinline__ void clover_blocks(const double (&Fs)[6][9][NS], int ls, int k, T* __restrict__ clover,
                                              T* __restrict__ clover_inv, const Lat& L, int idx, int par, double kc, double kt,
                                              int* flag) {
  const size_t half = (size_t)72 * L.Vh;  // reals per parity of a clover field
  double pk[36];
  double dg[6];
  cd lo[15];
  {
    cd B[6][6];
    assemble_block(Fs, ls, k, kc, kt, B);
#pragma unroll
    for (int i = 0; i < 6; i++) pk[i] = dg[i] = B[i][i].re;
#pragma unroll
    for (int i = 1; i < 6; i++)
#pragma unroll
      for (int j = 0; j < i; j++) {
        const int o = i * (i - 1) / 2 + j;
        lo[o] = B[i][j];
        pk[6 + 2 * o] = B[i][j].re;
        pk[7 + 2 * o] = B[i][j].im;
      }
  }
  store_block<T>(clover + par * half, L.Vh, idx, k, pk);
  if (!clover_inv) return;
  double nrm = dg[0];
#pragma unroll
  for (int i = 1; i < 6; i++) nrm = fmax(nrm, dg[i]);
  if (sweep6(dg, lo, fmax(1e-6 * nrm, 0.0))) {
#pragma unroll
    for (int i = 0; i < 6; i++) pk[i] = -dg[i];
#pragma unroll
    for (int o = 0; o < 15; o++) {
      pk[6 + 2 * o] = -lo[o].re;
      pk[7 + 2 * o] = -lo[o].im;
    }
    store_block<T>(clover_inv + par * half, L.Vh, idx, k, pk);
  } else {
    general_inverse_store<T, NS>(Fs, ls, k, kc, kt, clover_inv + par * half, L.Vh, idx, flag);
  }
}

template <typename T, int R>
__global__ void __launch_bounds__(CB_SITES * 6, CB_MINB) clover_build_kernel(T* __restrict__ clover, T* __restrict__ clover_inv,
                                                                    const T* __restrict__ gauge, Lat L, double kc,
                                                                    double kt, int* flag) {
  __shared__ double Fs[6][9][CB_SITES];  // planes xy, xz, xt, yz, yt, zt
  const int ls = threadIdx.x, pl = threadIdx.y;
  // Traversal order.  Every link is needed by the 14 sites of its two-hop neighbourhood, of both parities; in plain
  // checkerboard order (all even sites, then all odd; t slowest) the reuse window is three whole time slices of all
  // links, twice over.  Here a block pair = the even and the odd sites of the same 32 checkerboard indices, and the
  // index runs (x, y, z within a slab of CB_ZC planes, t, slab): the window is three time slices of ONE z-slab
  // (7 MB at 32^3x64).  Measured (ncu, 32^3x64 fp64): DRAM reads 10.8 -> 7.1 GB, L2 hit rate 42 -> 55 %, time
  // unchanged (4.5 ms; any CB_ZC from 2 to 16): the kernel waits on its 12 warps per SM, not on DRAM.
  const int par = blockIdx.x & 1;
  const int k = (blockIdx.x >> 1) * CB_SITES + ls;
  const bool live = k < L.Vh;
  int idx = 0;
  if (live) {
    const int zc = (L.Lz % CB_ZC == 0) ? CB_ZC : 2;  // every extent is even
    const int plane = L.Lxh * L.Ly;
    const int xy = k % plane;
    int q = k / plane;
    const int zl = q % zc;
    q /= zc;
    const int t = q % L.Lt, slab = q / L.Lt;
    idx = xy + plane * ((slab * zc + zl) + L.Lz * t);
  }
  if (live) {
    const Site s = site_of(L, idx, par);
    const int x0[4] = {2 * s.xh + s.r, s.y, s.z, s.t};
    const int mu = pl < 3 ? 0 : (pl < 5 ? 1 : 2);
    const int nu = pl < 3 ? pl + 1 : (pl < 5 ? pl - 1 : 3);
    cd F[9];
    field_strength<T, R>(gauge, L, x0, mu, nu, F);
    herm_store(Fs[pl], ls, F);
  }
  __syncthreads();
  if (!live || pl >= 2) return;
  clover_blocks<T, CB_SITES>(Fs, ls, pl, clover, clover_inv, L, idx, par, kc, kt, flag);
}

// ---------------------------------------------------------------------------------------------------------------
// Three-pass build (the default).  The one-kernel build above gathers 72 links per site and multiplies 72 times; it
// waits on its loads (ncu: 52 % long-scoreboard stalls at 9 warps per SM, fp64 pipe 30 % busy).  The four leaves of a
// plane are the SAME plaquette seen from its four corners, and moving the starting corner is a transport by one link:
//   P(y)              = U_mu(y) U_nu(y+mu) [U_nu(y) U_mu(y+nu)]^dag                      (the leaf of y itself)
//   leaf of y at y+nu = U_nu(y)^dag P(y) U_nu(y),   at y+mu = U_mu(y)^dag P(y) U_mu(y),   at y+mu+nu: both in turn.
// Only Q - Q^dag enters F and the transport is linear, so each pass carries the anti-Hermitian part X = P - P^dag
// (9 reals: 3 imaginary diagonals, 3 complex entries above the diagonal):
//   pass 1: X1(x) = P(x) - P(x)^dag                                         3 products, 4 links
//   pass 2: X2(x) = X1(x) + U_nu(x-nu)^dag X1(x-nu) U_nu(x-nu)              2 products, 1 link
//   pass 3: X3(x) = X2(x) + U_mu(x-mu)^dag X2(x-mu) U_mu(x-mu) = Q - Q^dag  2 products, 1 link; F = X3/(8i); blocks, inverses
// 42 products and 36 link loads per site instead of 72 and 72, every pass a streaming kernel.  Scratch: two fields
// [6 planes][9][2 Vh] doubles (432 B per site each), owned by the context.
struct AH {
  double d[3];  // Im X_00, Im X_11, Im X_22
  cd o[3];      // X_01, X_02, X_12
};
__device__ __forceinline__ M3 expand(const AH& a) {
  M3 m;
  m.m[0] = {0.0, a.d[0]};
  m.m[4] = {0.0, a.d[1]};
  m.m[8] = {0.0, a.d[2]};
  m.m[1] = a.o[0];
  m.m[2] = a.o[1];
  m.m[5] = a.o[2];
  m.m[3] = {-a.o[0].re, a.o[0].im};  // X_ji = -conj(X_ij)
  m.m[6] = {-a.o[1].re, a.o[1].im};
  m.m[7] = {-a.o[2].re, a.o[2].im};
  return m;
}
__device__ __forceinline__ AH load_ah(const double* __restrict__ X, size_t V, int pl, size_t s) {
  const double* p = X + (size_t)pl * 9 * V + s;
  AH a;
  a.d[0] = p[0];
  a.d[1] = p[V];
  a.d[2] = p[2 * V];
#pragma unroll
  for (int e = 0; e < 3; e++) a.o[e] = {p[(3 + 2 * e) * V], p[(4 + 2 * e) * V]};
  return a;
}
__device__ __forceinline__ void store_ah(double* __restrict__ X, size_t V, int pl, size_t s, const AH& a) {
  double* p = X + (size_t)pl * 9 * V + s;
  p[0] = a.d[0];
  p[V] = a.d[1];
  p[2 * V] = a.d[2];
#pragma unroll
  for (int e = 0; e < 3; e++) {
    p[(3 + 2 * e) * V] = a.o[e].re;
    p[(4 + 2 * e) * V] = a.o[e].im;
  }
}
// entry (i, j) of a^dag b
__device__ __forceinline__ cd dag_mul_entry(const M3& a, const M3& b, int i, int j) {
  double re = a.m[i].re * b.m[j].re, im = a.m[i].re * b.m[j].im;
  re = fma(a.m[i].im, b.m[j].im, re);
  im = fma(-a.m[i].im, b.m[j].re, im);
#pragma unroll
  for (int k = 1; k < 3; k++) {
    re = fma(a.m[3 * k + i].re, b.m[3 * k + j].re, re);
    re = fma(a.m[3 * k + i].im, b.m[3 * k + j].im, re);
    im = fma(a.m[3 * k + i].re, b.m[3 * k + j].im, im);
    im = fma(-a.m[3 * k + i].im, b.m[3 * k + j].re, im);
  }
  return {re, im};
}
// the slab traversal of the one-kernel build: block pair = even and odd sites of the same 32 checkerboard indices
template <int NS = CB_SITES>
__device__ __forceinline__ bool cb_site(const Lat& L, int& idx, int& par) {
  par = blockIdx.x & 1;
  const int k = (blockIdx.x >> 1) * NS + threadIdx.x;
  if (k >= L.Vh) return false;
  const int zc = (L.Lz % CB_ZC == 0) ? CB_ZC : 2;
  const int plane = L.Lxh * L.Ly;
  const int xy = k % plane;
  int q = k / plane;
  const int zl = q % zc;
  q /= zc;
  const int t = q % L.Lt, slab = q / L.Lt;
  idx = xy + plane * ((slab * zc + zl) + L.Lz * t);
  return true;
}
__device__ __forceinline__ void plane_dirs(int pl, int& mu, int& nu) {
  mu = pl < 3 ? 0 : (pl < 5 ? 1 : 2);
  nu = pl < 3 ? pl + 1 : (pl < 5 ? pl - 1 : 3);
}
__device__ __forceinline__ size_t site_slot(const Lat& L, const int* x) {
  const int par = (x[0] + x[1] + x[2] + x[3]) & 1;
  return (size_t)par * L.Vh + (x[0] >> 1) + L.Lxh * (x[1] + L.Ly * (x[2] + L.Lz * x[3]));
}

#ifndef CB3_MINB
#define CB3_MINB 3
#endif
#ifndef CB1_MINB
#define CB1_MINB 2  // 168 registers: the four links of a leaf in flight at once (3 blocks: 96 registers, +9 %)
#endif
template <typename T, int R>
__global__ void __launch_bounds__(CB_SITES * 6, CB1_MINB) clover_plaquette_kernel(double* __restrict__ X1, const T* __restrict__ gauge, Lat L) {
  int idx, par;
  if (!cb_site(L, idx, par)) return;
  const int pl = threadIdx.y;
  int mu, nu;
  plane_dirs(pl, mu, nu);
  const Site s = site_of(L, idx, par);
  int x[4] = {2 * s.xh + s.r, s.y, s.z, s.t}, a[4], b[4];
  for (int i = 0; i < 4; i++) a[i] = b[i] = x[i];
  step(L, a, mu, +1);
  step(L, b, nu, +1);
  const M3 A = mul(link_at<T, R>(gauge, L, mu, x), link_at<T, R>(gauge, L, nu, a));
  const M3 B = mul(link_at<T, R>(gauge, L, nu, x), link_at<T, R>(gauge, L, mu, b));
  const M3 P = mul(A, dag(B));
  AH h;
#pragma unroll
  for (int i = 0; i < 3; i++) h.d[i] = 2.0 * P.m[4 * i].im;
  h.o[0] = P.m[1] - conj(P.m[3]);
  h.o[1] = P.m[2] - conj(P.m[6]);
  h.o[2] = P.m[5] - conj(P.m[7]);
  store_ah(X1, (size_t)2 * L.Vh, pl, (size_t)par * L.Vh + idx, h);
}

// X(x) + U_d(x-d)^dag X(x-d) U_d(x-d)
template <typename T, int R>
__device__ __forceinline__ AH transport_sum(const double* __restrict__ X, const T* __restrict__ gauge, const Lat& L, int pl,
                                            int d, const int* x0, size_t s0) {
  int xm[4];
  for (int i = 0; i < 4; i++) xm[i] = x0[i];
  step(L, xm, d, -1);
  const M3 U = link_at<T, R>(gauge, L, d, xm);
  const M3 Y = mul(expand(load_ah(X, (size_t)2 * L.Vh, pl, site_slot(L, xm))), U);
  AH r = load_ah(X, (size_t)2 * L.Vh, pl, s0);
#pragma unroll
  for (int i = 0; i < 3; i++) r.d[i] += dag_mul_entry(U, Y, i, i).im;
  r.o[0] = r.o[0] + dag_mul_entry(U, Y, 0, 1);
  r.o[1] = r.o[1] + dag_mul_entry(U, Y, 0, 2);
  r.o[2] = r.o[2] + dag_mul_entry(U, Y, 1, 2);
  return r;
}
template <typename T, int R>
__global__ void __launch_bounds__(CB_SITES * 6, CB3_MINB) clover_transport_kernel(double* __restrict__ X2, const double* __restrict__ X1,
                                                                           const T* __restrict__ gauge, Lat L) {
  int idx, par;
  if (!cb_site(L, idx, par)) return;
  const int pl = threadIdx.y;
  int mu, nu;
  plane_dirs(pl, mu, nu);
  const Site s = site_of(L, idx, par);
  const int x0[4] = {2 * s.xh + s.r, s.y, s.z, s.t};
  const size_t s0 = (size_t)par * L.Vh + idx;
  store_ah(X2, (size_t)2 * L.Vh, pl, s0, transport_sum<T, R>(X1, gauge, L, pl, nu, x0, s0));
}

// Pass 3.  Two threads per site in BOTH phases: thread (s, k) transports planes 3k..3k+2, then inverts chiral block k.
// (With one thread per plane, as in passes 1 and 2, four of a block's six warps idle through the inversions, whose
// dependent chains -- pivot search, reciprocal, elimination -- then run on 4 warps per SM: 1.4 of the pass's 1.9 ms.)
#ifndef CBF_SITES
#define CBF_SITES 64
#endif
#ifndef CBF_MINB
#define CBF_MINB 3
#endif
template <typename T, int R>
__global__ void __launch_bounds__(CBF_SITES * 2, CBF_MINB) clover_finish_kernel(T* __restrict__ clover, T* __restrict__ clover_inv,
                                                                          const double* __restrict__ X2, const T* __restrict__ gauge,
                                                                          Lat L, double kc, double kt, int* flag) {
  __shared__ double Fs[6][9][CBF_SITES];
  const int ls = threadIdx.x, k = threadIdx.y;
  int idx = 0, par = 0;
  const bool live = cb_site<CBF_SITES>(L, idx, par);
  if (live) {
    const Site s = site_of(L, idx, par);
    const int x0[4] = {2 * s.xh + s.r, s.y, s.z, s.t};
#pragma unroll
    for (int i = 0; i < 3; i++) {
      const int pl = 3 * k + i;
      int mu, nu;
      plane_dirs(pl, mu, nu);
      const AH q = transport_sum<T, R>(X2, gauge, L, pl, mu, x0, (size_t)par * L.Vh + idx);  // Q - Q^dag
      // F = (Q - Q^dag)/(8i): Hermitian
#pragma unroll
      for (int d = 0; d < 3; d++) Fs[pl][d][ls] = 0.125 * q.d[d];
#pragma unroll
      for (int e = 0; e < 3; e++) {
        Fs[pl][3 + 2 * e][ls] = 0.125 * q.o[e].im;
        Fs[pl][4 + 2 * e][ls] = -0.125 * q.o[e].re;
      }
    }
  }
  __syncthreads();
  if (!live) return;
  clover_blocks<T, CBF_SITES>(Fs, ls, k, clover, clover_inv, L, idx, par, kc, kt, flag);
}

template <typename T, int R>
static void clover_build_launch(lqcd_ctx* c, void* clover, void* clover_inv, const void* gauge, double kc, double kt, cudaStream_t st) {
  const int grid = 2 * ((c->lat.Vh + CB_SITES - 1) / CB_SITES);
  const dim3 block(CB_SITES, 6);
  if (!c->clover_onepass && !c->d_clover_scratch) {
    // two fields of 6 planes x 9 doubles per site; if they do not fit, the one-kernel build needs none
    if (cudaMalloc(&c->d_clover_scratch, sizeof(double) * 2 * 54 * (size_t)2 * c->lat.Vh) != cudaSuccess) {
      cudaGetLastError();
      c->d_clover_scratch = nullptr;
      c->clover_onepass = 1;
    }
  }
  if (c->clover_onepass) {
    clover_build_kernel<T, R><<<grid, block, 0, st>>>((T*)clover, (T*)clover_inv, (const T*)gauge, c->lat, kc, kt, c->d_flag);
    return;
  }
  double* X1 = c->d_clover_scratch;
  double* X2 = X1 + 54 * (size_t)2 * c->lat.Vh;
  clover_plaquette_kernel<T, R><<<grid, block, 0, st>>>(X1, (const T*)gauge, c->lat);
  clover_transport_kernel<T, R><<<grid, block, 0, st>>>(X2, X1, (const T*)gauge, c->lat);
  clover_finish_kernel<T, R><<<2 * ((c->lat.Vh + CBF_SITES - 1) / CBF_SITES), dim3(CBF_SITES, 2), 0, st>>>((T*)clover, (T*)clover_inv, X2, (const T*)gauge, c->lat, kc, kt, c->d_flag);
  c->launches += 2;  // LQCD_LAUNCH_CHECK counts the third
}

extern "C" int lqcd_clover_build_aniso(lqcd_ctx* c, void* clover, void* clover_inv, const void* gauge, double csw_s,
                                       double csw_t, double kappa, void* stream) {
  if (!c || !clover || !gauge) return LQCD_ERR_INVALID_ARG;
  if (c->half) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "clover_build: not available in a 16-bit context; build in an fp32 context and convert (lqcd_clover_to_half)");
  if (!lqcd_aligned16(clover) || !lqcd_aligned16(clover_inv) || !lqcd_aligned16(gauge))
    return lqcd_set_error(c, LQCD_ERR_ALIGN, "clover_build: alignment");
  cudaStream_t st = as_stream(stream);
  const double kc = kappa * csw_s, kt = kappa * csw_t;
  cudaMemsetAsync(c->d_flag, 0, sizeof(int), st);
  c->alg_bytes += (double)lqcd_gauge_bytes(c) + (clover_inv ? 2.0 : 1.0) * (double)lqcd_clover_bytes(c);
  if (c->prec == 4 && c->recon == 18)
    clover_build_launch<float, 18>(c, clover, clover_inv, gauge, kc, kt, st);
  else if (c->prec == 4)
    clover_build_launch<float, 12>(c, clover, clover_inv, gauge, kc, kt, st);
  else if (c->recon == 18)
    clover_build_launch<double, 18>(c, clover, clover_inv, gauge, kc, kt, st);
  else
    clover_build_launch<double, 12>(c, clover, clover_inv, gauge, kc, kt, st);
  LQCD_LAUNCH_CHECK(c, "clover_build");
  cudaMemcpyAsync(c->h_flag, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return lqcd_check_cuda(c, "clover_build sync");
  if (c->h_flag[0]) return lqcd_set_error(c, LQCD_ERR_SINGULAR_CLOVER, "clover_build: singular 6x6 block");
  return LQCD_OK;
}

extern "C" int lqcd_clover_build(lqcd_ctx* c, void* clover, void* clover_inv, const void* gauge, double csw,
                                 double kappa, void* stream) {
  return lqcd_clover_build_aniso(c, clover, clover_inv, gauge, csw, csw, kappa, stream);
}

// ---------------------------------------------------------------------------------------------------------------
// lqcd_clover_build_noalloc: the three-pass build for callers that cannot tolerate an allocation inside the call (code
// under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  lqcd_clover_build allocates its
// scratch (two fields of 6 planes x 9 doubles per site) with cudaMalloc on the first build of a context; here the
// scratch is a file-scope device array of fixed size, so the entry point calls no cudaMalloc, cudaFree or allocating
// library routine -- and serves lattices of at most LQCD_CLOVER_NOALLOC_MAX_SITES sites.
//   Size: 2 x 54 x 8 B x 32768 sites = 27 MiB, held by every GPU that loads the library until the process exits.
//   Sharing: ONE array per GPU for all contexts and calls.  It keeps the last call's contents; nothing in it has to
//   start at zero (pass 1 writes every entry of X1 that pass 2 reads, pass 2 every entry of X2 that pass 3 reads), so
//   nothing is cleared.  Two calls that overlap on the GPU (different streams, or different contexts on one device)
//   race on it: callers serialise them.
//   In host code the array's name is a host-side stand-in, not a device address; the device address is taken once per
//   device with cudaGetSymbolAddress while that device is current, and that pointer is what the kernels get.
// ---------------------------------------------------------------------------------------------------------------
constexpr long LQCD_CLOVER_NOALLOC_MAX_SITES = 32768;
static __device__ __align__(256) double clover_noalloc_scratch[2 * 54 * LQCD_CLOVER_NOALLOC_MAX_SITES];
static double* clover_noalloc_ptr[LQCD_MAX_DEVICES] = {};  // device address of the array, per device ordinal

extern "C" long lqcd_clover_noalloc_max_sites(void) { return LQCD_CLOVER_NOALLOC_MAX_SITES; }

template <typename T, int R>
static void clover_build_launch_static(lqcd_ctx* c, double* scratch, void* clover, void* clover_inv, const void* gauge,
                                       double kc, double kt, cudaStream_t st) {
  const int grid = 2 * ((c->lat.Vh + CB_SITES - 1) / CB_SITES);
  const dim3 block(CB_SITES, 6);
  double* X1 = scratch;
  double* X2 = X1 + 54 * (size_t)2 * c->lat.Vh;
  clover_plaquette_kernel<T, R><<<grid, block, 0, st>>>(X1, (const T*)gauge, c->lat);
  clover_transport_kernel<T, R><<<grid, block, 0, st>>>(X2, X1, (const T*)gauge, c->lat);
  clover_finish_kernel<T, R><<<2 * ((c->lat.Vh + CBF_SITES - 1) / CBF_SITES), dim3(CBF_SITES, 2), 0, st>>>(
      (T*)clover, (T*)clover_inv, X2, (const T*)gauge, c->lat, kc, kt, c->d_flag);
  c->launches += 2;  // LQCD_LAUNCH_CHECK counts the third
}

extern "C" int lqcd_clover_build_noalloc(lqcd_ctx* c, void* clover, void* clover_inv, const void* gauge, double csw,
                                         double kappa, void* stream) {
  if (!c || !clover || !gauge) return LQCD_ERR_INVALID_ARG;
  if (c->half) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "clover_build_noalloc: not available in a 16-bit context");
  if (!lqcd_aligned16(clover) || !lqcd_aligned16(clover_inv) || !lqcd_aligned16(gauge))
    return lqcd_set_error(c, LQCD_ERR_ALIGN, "clover_build_noalloc: alignment");
  const long sites = 2L * c->lat.Vh;
  if (sites > LQCD_CLOVER_NOALLOC_MAX_SITES)
    return lqcd_set_error(c, LQCD_ERR_WORKSPACE,
                          "clover_build_noalloc: lattice has %ld sites, the static scratch holds at most %ld (use lqcd_clover_build)",
                          sites, LQCD_CLOVER_NOALLOC_MAX_SITES);
  // set-up, once per device, with that device current
  if (!clover_noalloc_ptr[c->device]) {
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != c->device)
      return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "clover_build_noalloc: device %d of the context is not the current device (%d)",
                            c->device, cur);
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, clover_noalloc_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return lqcd_set_error(c, LQCD_ERR_CUDA, "clover_build_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    }
    clover_noalloc_ptr[c->device] = p;
  }
  double* scratch = clover_noalloc_ptr[c->device];
  cudaStream_t st = as_stream(stream);
  const double kc = kappa * csw;
  cudaMemsetAsync(c->d_flag, 0, sizeof(int), st);
  c->alg_bytes += (double)lqcd_gauge_bytes(c) + (clover_inv ? 2.0 : 1.0) * (double)lqcd_clover_bytes(c);
  if (c->prec == 4 && c->recon == 18)
    clover_build_launch_static<float, 18>(c, scratch, clover, clover_inv, gauge, kc, kc, st);
  else if (c->prec == 4)
    clover_build_launch_static<float, 12>(c, scratch, clover, clover_inv, gauge, kc, kc, st);
  else if (c->recon == 18)
    clover_build_launch_static<double, 18>(c, scratch, clover, clover_inv, gauge, kc, kc, st);
  else
    clover_build_launch_static<double, 12>(c, scratch, clover, clover_inv, gauge, kc, kc, st);
  LQCD_LAUNCH_CHECK(c, "clover_build_noalloc");
  cudaMemcpyAsync(c->h_flag, c->d_flag, sizeof(int), cudaMemcpyDeviceToHost, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return lqcd_check_cuda(c, "clover_build_noalloc sync");
  if (c->h_flag[0]) return lqcd_set_error(c, LQCD_ERR_SINGULAR_CLOVER, "clover_build_noalloc: singular 6x6 block");
  return LQCD_OK;
}
