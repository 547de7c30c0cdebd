// K2/K3 device code: Wilson hopping term (Eq. 5, the gamma_mu W_mu part; SURVEY.md
// §8(c) O3) and the chiral-block clover multiply, one thread per output site.
//
// DeGrand-Rossi basis: gamma_mu = [[0,B],[B^dag,0]] with B_x = i s1, B_y = -i s2,
// B_z = i s3, B_t = 1.  (1 + s*gamma_mu) psi has upper half h = psi_u + s*B psi_l and lower half
// s*B^dag h, so only the two-spin h is multiplied by the link: 8 x (12 + 132) + 168 = 1320 flop.
#pragma once
#include "lqcd_internal.cuh"

// spinor register layout: psi[2*(3*spin + colour) + (0 re | 1 im)]
#define RE(s, c) (2 * (3 * (s) + (c)))
#define IM(s, c) (2 * (3 * (s) + (c)) + 1)

// h = psi_u + S * B_mu psi_l          (S = -1: (1 - gamma_mu), S = +1: (1 + gamma_mu))
template <typename T, int MU, int S>
__device__ __forceinline__ void project(const T* psi, T* h) {
#pragma unroll
  for (int c = 0; c < 3; c++) {
    if (MU == 0) {  // B psi_l = (i psi_3, i psi_2)
      h[RE(0, c)] = psi[RE(0, c)] - S * psi[IM(3, c)];
      h[IM(0, c)] = psi[IM(0, c)] + S * psi[RE(3, c)];
      h[RE(1, c)] = psi[RE(1, c)] - S * psi[IM(2, c)];
      h[IM(1, c)] = psi[IM(1, c)] + S * psi[RE(2, c)];
    } else if (MU == 1) {  // B psi_l = (-psi_3, psi_2)
      h[RE(0, c)] = psi[RE(0, c)] - S * psi[RE(3, c)];
      h[IM(0, c)] = psi[IM(0, c)] - S * psi[IM(3, c)];
      h[RE(1, c)] = psi[RE(1, c)] + S * psi[RE(2, c)];
      h[IM(1, c)] = psi[IM(1, c)] + S * psi[IM(2, c)];
    } else if (MU == 2) {  // B psi_l = (i psi_2, -i psi_3)
      h[RE(0, c)] = psi[RE(0, c)] - S * psi[IM(2, c)];
      h[IM(0, c)] = psi[IM(0, c)] + S * psi[RE(2, c)];
      h[RE(1, c)] = psi[RE(1, c)] + S * psi[IM(3, c)];
      h[IM(1, c)] = psi[IM(1, c)] - S * psi[RE(3, c)];
    } else {  // B = 1
      h[RE(0, c)] = psi[RE(0, c)] + S * psi[RE(2, c)];
      h[IM(0, c)] = psi[IM(0, c)] + S * psi[IM(2, c)];
      h[RE(1, c)] = psi[RE(1, c)] + S * psi[RE(3, c)];
      h[IM(1, c)] = psi[IM(1, c)] + S * psi[IM(3, c)];
    }
  }
}

// acc_u += chi ; acc_l += S * B_mu^dag chi
template <typename T, int MU, int S>
__device__ __forceinline__ void reconstruct(T* acc, const T* chi) {
#pragma unroll
  for (int c = 0; c < 3; c++) {
    acc[RE(0, c)] += chi[RE(0, c)];
    acc[IM(0, c)] += chi[IM(0, c)];
    acc[RE(1, c)] += chi[RE(1, c)];
    acc[IM(1, c)] += chi[IM(1, c)];
    if (MU == 0) {  // B^dag chi = (-i chi_1, -i chi_0)
      acc[RE(2, c)] += S * chi[IM(1, c)];
      acc[IM(2, c)] -= S * chi[RE(1, c)];
      acc[RE(3, c)] += S * chi[IM(0, c)];
      acc[IM(3, c)] -= S * chi[RE(0, c)];
    } else if (MU == 1) {  // B^dag chi = (chi_1, -chi_0)
      acc[RE(2, c)] += S * chi[RE(1, c)];
      acc[IM(2, c)] += S * chi[IM(1, c)];
      acc[RE(3, c)] -= S * chi[RE(0, c)];
      acc[IM(3, c)] -= S * chi[IM(0, c)];
    } else if (MU == 2) {  // B^dag chi = (-i chi_0, i chi_1)
      acc[RE(2, c)] += S * chi[IM(0, c)];
      acc[IM(2, c)] -= S * chi[RE(0, c)];
      acc[RE(3, c)] -= S * chi[IM(1, c)];
      acc[IM(3, c)] += S * chi[RE(1, c)];
    } else {
      acc[RE(2, c)] += S * chi[RE(0, c)];
      acc[IM(2, c)] += S * chi[IM(0, c)];
      acc[RE(3, c)] += S * chi[RE(1, c)];
      acc[IM(3, c)] += S * chi[IM(1, c)];
    }
  }
}

// chi = U h (DAGGER_U = false) or U^dag h (true), for the two spin components of h
template <typename T, bool DAGGER_U>
__device__ __forceinline__ void su3_mul(const T* U, const T* h, T* chi) {
#pragma unroll
  for (int s = 0; s < 2; s++)
#pragma unroll
    for (int a = 0; a < 3; a++) {
      T re = 0, im = 0;
#pragma unroll
      for (int b = 0; b < 3; b++) {
        const T ur = DAGGER_U ? U[2 * (3 * b + a)] : U[2 * (3 * a + b)];
        const T ui = DAGGER_U ? -U[2 * (3 * b + a) + 1] : U[2 * (3 * a + b) + 1];
        re += ur * h[RE(s, b)] - ui * h[IM(s, b)];
        im += ur * h[IM(s, b)] + ui * h[RE(s, b)];
      }
      chi[RE(s, a)] = re;
      chi[IM(s, a)] = im;
    }
}

// one of the eight hops.  FWD: U_mu(x) psi(x+mu) with link block of the output parity at idx;
// backward: U_mu^dag(x-mu) psi(x-mu) with link block of the input parity at the neighbour index.
template <typename T, int R, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void hop(T* acc, const T* __restrict__ in, const T* __restrict__ links, int Vh,
                                    int nidx, int lidx, T bsign) {
  constexpr int S = (FWD != DAG) ? -1 : +1;
  T psi[24], U[18], h[12], chi[12];
  load_spinor<T>(in, Vh, nidx, psi);
  load_link<T, R>(links, Vh, lidx, U);
  project<T, MU, S>(psi, h);
  if (MU == 3) {
#pragma unroll
    for (int e = 0; e < 12; e++) h[e] *= bsign;
  }
  su3_mul<T, !FWD>(U, h, chi);
  reconstruct<T, MU, S>(acc, chi);
}

// all eight hops for output site idx of parity par.  gauge = native links [mu][parity][NGV][Vh].
template <typename T, int R, bool DAG>
__device__ __forceinline__ void dslash_site(T* acc, const T* __restrict__ in, const T* __restrict__ gauge,
                                            const Lat& L, int idx, int par) {
  const Site s = site_of(L, idx, par);
  const int Vh = L.Vh;
  const size_t blk = (size_t)R * Vh;  // reals per (mu, parity) link block
#pragma unroll
  for (int e = 0; e < 24; e++) acc[e] = 0;
  const T one = 1;
  const T sf = (L.tb < 0 && s.t == L.Lt - 1) ? -one : one;
  const T sb = (L.tb < 0 && s.t == 0) ? -one : one;
  int n;
  n = neighbour<0, +1>(L, idx, s);
  hop<T, R, 0, true, DAG>(acc, in, gauge + (0 * 2 + par) * blk, Vh, n, idx, one);
  n = neighbour<0, -1>(L, idx, s);
  hop<T, R, 0, false, DAG>(acc, in, gauge + (0 * 2 + 1 - par) * blk, Vh, n, n, one);
  n = neighbour<1, +1>(L, idx, s);
  hop<T, R, 1, true, DAG>(acc, in, gauge + (1 * 2 + par) * blk, Vh, n, idx, one);
  n = neighbour<1, -1>(L, idx, s);
  hop<T, R, 1, false, DAG>(acc, in, gauge + (1 * 2 + 1 - par) * blk, Vh, n, n, one);
  n = neighbour<2, +1>(L, idx, s);
  hop<T, R, 2, true, DAG>(acc, in, gauge + (2 * 2 + par) * blk, Vh, n, idx, one);
  n = neighbour<2, -1>(L, idx, s);
  hop<T, R, 2, false, DAG>(acc, in, gauge + (2 * 2 + 1 - par) * blk, Vh, n, n, one);
  n = neighbour<3, +1>(L, idx, s);
  hop<T, R, 3, true, DAG>(acc, in, gauge + (3 * 2 + par) * blk, Vh, n, idx, sf);
  n = neighbour<3, -1>(L, idx, s);
  hop<T, R, 3, false, DAG>(acc, in, gauge + (3 * 2 + 1 - par) * blk, Vh, n, n, sb);
}

// out = C v for the two Hermitian 6x6 chiral blocks of one site.  cl = one-parity clover field
// [NCV][Vh]; packed order per block: 6 real diagonal, then 15 complex lower entries row-major.
// v and out are 24-real spinors (block k acts on reals 12k..12k+11); they must not alias.
template <typename T>
__device__ __forceinline__ void clover_mul(const T* __restrict__ cl, int Vh, int idx, const T* v, T* out) {
  typedef typename V16<T>::vec vec;
  constexpr int N = V16<T>::N;
  const vec* p = reinterpret_cast<const vec*>(cl) + idx;
#pragma unroll
  for (int k = 0; k < 2; k++) {
    T a[36];
#pragma unroll
    for (int q = 0; q < 36 / N; q++) {
      vec w = ld_stream(p + (size_t)(k * (36 / N) + q) * Vh);
      vec_get(w, a + q * N);
    }
    const T* x = v + 12 * k;
    T* y = out + 12 * k;
#pragma unroll
    for (int i = 0; i < 6; i++) {
      T re = a[i] * x[2 * i], im = a[i] * x[2 * i + 1];
#pragma unroll
      for (int j = 0; j < 6; j++) {
        if (j < i) {  // L_ij x_j
          const int o = 6 + 2 * (i * (i - 1) / 2 + j);
          re += a[o] * x[2 * j] - a[o + 1] * x[2 * j + 1];
          im += a[o] * x[2 * j + 1] + a[o + 1] * x[2 * j];
        } else if (j > i) {  // conj(L_ji) x_j
          const int o = 6 + 2 * (j * (j - 1) / 2 + i);
          re += a[o] * x[2 * j] + a[o + 1] * x[2 * j + 1];
          im += a[o] * x[2 * j + 1] - a[o + 1] * x[2 * j];
        }
      }
      y[2 * i] = re;
      y[2 * i + 1] = im;
    }
  }
}
