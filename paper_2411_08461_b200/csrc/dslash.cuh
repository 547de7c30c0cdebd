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
#define CPK(a, s, c) pk2((a)[RE(s, c)], (a)[IM(s, c)])   // (re, im)
#define CSW(a, s, c) pk2((a)[IM(s, c)], (a)[RE(s, c)])   // (im, re): an operand swizzle, no instruction
#define CST(a, s, c, v) upk2((v), (a)[RE(s, c)], (a)[IM(s, c)])
template <int MU, int S>
__device__ __forceinline__ void project_packed(const float* psi, float* h) {
  const float p = (float)S, m = (float)-S;
#pragma unroll
  for (int c = 0; c < 3; c++) {
    if (MU == 0) {  // h0 = psi0 + S i psi3, h1 = psi1 + S i psi2;  S i (re, im) = (-S im, S re)
      CST(h, 0, c, fma2(pk2(m, p), CSW(psi, 3, c), CPK(psi, 0, c)));
      CST(h, 1, c, fma2(pk2(m, p), CSW(psi, 2, c), CPK(psi, 1, c)));
    } else if (MU == 1) {  // h0 = psi0 - S psi3, h1 = psi1 + S psi2
      CST(h, 0, c, fma2(pk2(m, m), CPK(psi, 3, c), CPK(psi, 0, c)));
      CST(h, 1, c, fma2(pk2(p, p), CPK(psi, 2, c), CPK(psi, 1, c)));
    } else if (MU == 2) {  // h0 = psi0 + S i psi2, h1 = psi1 - S i psi3
      CST(h, 0, c, fma2(pk2(m, p), CSW(psi, 2, c), CPK(psi, 0, c)));
      CST(h, 1, c, fma2(pk2(p, m), CSW(psi, 3, c), CPK(psi, 1, c)));
    } else {  // h0 = psi0 + S psi2, h1 = psi1 + S psi3
      CST(h, 0, c, fma2(pk2(p, p), CPK(psi, 2, c), CPK(psi, 0, c)));
      CST(h, 1, c, fma2(pk2(p, p), CPK(psi, 3, c), CPK(psi, 1, c)));
    }
  }
}

template <typename T, int MU, int S>
__device__ __forceinline__ void project(const T* psi, T* h) {
  if constexpr (UsePacked<T>::value) {
    project_packed<MU, S>(psi, h);
  } else {
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
}

// acc_u += w chi ; acc_l += w S B_mu^dag chi.  w = hop weight (boundary sign on t-hops, nu/xi_0 on
// spatial hops, Eq. 5): folded into the accumulation, every line is one FFMA/DFMA.
template <int MU, int S>
__device__ __forceinline__ void reconstruct_packed(float* acc, const float* chi, float w) {
  const float ws = S * w, wn = -ws;
#pragma unroll
  for (int c = 0; c < 3; c++) {
    CST(acc, 0, c, fma2(pk2(w, w), CPK(chi, 0, c), CPK(acc, 0, c)));
    CST(acc, 1, c, fma2(pk2(w, w), CPK(chi, 1, c), CPK(acc, 1, c)));
    if (MU == 0) {  // acc2 += ws (-i chi1) = (ws, -ws) o (im1, re1); acc3 likewise with chi0
      CST(acc, 2, c, fma2(pk2(ws, wn), CSW(chi, 1, c), CPK(acc, 2, c)));
      CST(acc, 3, c, fma2(pk2(ws, wn), CSW(chi, 0, c), CPK(acc, 3, c)));
    } else if (MU == 1) {  // acc2 += ws chi1; acc3 -= ws chi0
      CST(acc, 2, c, fma2(pk2(ws, ws), CPK(chi, 1, c), CPK(acc, 2, c)));
      CST(acc, 3, c, fma2(pk2(wn, wn), CPK(chi, 0, c), CPK(acc, 3, c)));
    } else if (MU == 2) {  // acc2 += ws (-i chi0); acc3 += ws (i chi1)
      CST(acc, 2, c, fma2(pk2(ws, wn), CSW(chi, 0, c), CPK(acc, 2, c)));
      CST(acc, 3, c, fma2(pk2(wn, ws), CSW(chi, 1, c), CPK(acc, 3, c)));
    } else {
      CST(acc, 2, c, fma2(pk2(ws, ws), CPK(chi, 0, c), CPK(acc, 2, c)));
      CST(acc, 3, c, fma2(pk2(ws, ws), CPK(chi, 1, c), CPK(acc, 3, c)));
    }
  }
}

template <typename T, int MU, int S>
__device__ __forceinline__ void reconstruct(T* acc, const T* chi, T w) {
  if constexpr (UsePacked<T>::value) {
    reconstruct_packed<MU, S>(acc, chi, w);
  } else {
  const T ws = S * w;
#pragma unroll
  for (int c = 0; c < 3; c++) {
    acc[RE(0, c)] += w * chi[RE(0, c)];
    acc[IM(0, c)] += w * chi[IM(0, c)];
    acc[RE(1, c)] += w * chi[RE(1, c)];
    acc[IM(1, c)] += w * chi[IM(1, c)];
    if (MU == 0) {  // B^dag chi = (-i chi_1, -i chi_0)
      acc[RE(2, c)] += ws * chi[IM(1, c)];
      acc[IM(2, c)] -= ws * chi[RE(1, c)];
      acc[RE(3, c)] += ws * chi[IM(0, c)];
      acc[IM(3, c)] -= ws * chi[RE(0, c)];
    } else if (MU == 1) {  // B^dag chi = (chi_1, -chi_0)
      acc[RE(2, c)] += ws * chi[RE(1, c)];
      acc[IM(2, c)] += ws * chi[IM(1, c)];
      acc[RE(3, c)] -= ws * chi[RE(0, c)];
      acc[IM(3, c)] -= ws * chi[IM(0, c)];
    } else if (MU == 2) {  // B^dag chi = (-i chi_0, i chi_1)
      acc[RE(2, c)] += ws * chi[IM(0, c)];
      acc[IM(2, c)] -= ws * chi[RE(0, c)];
      acc[RE(3, c)] -= ws * chi[IM(1, c)];
      acc[IM(3, c)] += ws * chi[RE(1, c)];
    } else {
      acc[RE(2, c)] += ws * chi[RE(0, c)];
      acc[IM(2, c)] += ws * chi[IM(0, c)];
      acc[RE(3, c)] += ws * chi[RE(1, c)];
      acc[IM(3, c)] += ws * chi[IM(1, c)];
    }
  }
  }
}

// chi = U h (DAGGER_U = false) or U^dag h (true), for the two spin components of h
template <bool DAGGER_U>
__device__ __forceinline__ void su3_mul_packed(const float* U, const float* h, float* chi) {
  // chi_a = sum_b ur_ab (hr, hi)_b  +  (-1, 1) o sum_b ui_ab (hi, hr)_b : the swizzled operand is free, the
  // sign of the imaginary-part products is applied once per output (7 FFMA2 per complex output)
#pragma unroll
  for (int s = 0; s < 2; s++)
#pragma unroll
    for (int a = 0; a < 3; a++) {
      u64 accr, acci;
#pragma unroll
      for (int b = 0; b < 3; b++) {
        const float ur = DAGGER_U ? U[2 * (3 * b + a)] : U[2 * (3 * a + b)];
        const float ui = DAGGER_U ? U[2 * (3 * b + a) + 1] : U[2 * (3 * a + b) + 1];
        accr = (b == 0) ? mul2(pk2(ur, ur), CPK(h, s, b)) : fma2(pk2(ur, ur), CPK(h, s, b), accr);
        acci = (b == 0) ? mul2(pk2(ui, ui), CSW(h, s, b)) : fma2(pk2(ui, ui), CSW(h, s, b), acci);
      }
      CST(chi, s, a, fma2(DAGGER_U ? pk2(1.f, -1.f) : pk2(-1.f, 1.f), acci, accr));
    }
}

template <typename T, bool DAGGER_U>
__device__ __forceinline__ void su3_mul(const T* U, const T* h, T* chi) {
  if constexpr (UsePacked<T>::value) {
    su3_mul_packed<DAGGER_U>(U, h, chi);
  } else {
#pragma unroll
  for (int s = 0; s < 2; s++)
#pragma unroll
    for (int a = 0; a < 3; a++) {
      T re = 0, im = 0;
#pragma unroll
      for (int b = 0; b < 3; b++) {
        const T ur = DAGGER_U ? U[2 * (3 * b + a)] : U[2 * (3 * a + b)];
        const T ui = DAGGER_U ? -U[2 * (3 * b + a) + 1] : U[2 * (3 * a + b) + 1];
        // one multiply-add per statement: each contracts to a single FFMA/DFMA (a*b - c*d + re would cost
        // FMUL + FFMA + FADD without reassociation)
        re += ur * h[RE(s, b)];
        re -= ui * h[IM(s, b)];
        im += ur * h[IM(s, b)];
        im += ui * h[RE(s, b)];
      }
      chi[RE(s, a)] = re;
      chi[IM(s, a)] = im;
    }
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
  su3_mul<T, !FWD>(U, h, chi);
  reconstruct<T, MU, S>(acc, chi, bsign);
}

// all eight hops for output site idx of parity par.  gauge = native links [mu][parity][NGV][Vh].
template <typename T, int R, bool DAG>
__device__ __forceinline__ void dslash_site(T* acc, const T* __restrict__ in, const T* __restrict__ gauge,
                                            const Lat& L, int idx, int par, T ws) {
  const Site s = site_of(L, idx, par);
  const int Vh = L.Vh;
  const size_t blk = (size_t)R * Vh;  // reals per (mu, parity) link block
#pragma unroll
  for (int e = 0; e < 24; e++) acc[e] = 0;
  const T one = ws;  // weight of the spatial hops (Eq. 5: nu/xi_0); the temporal hops carry the boundary sign
  const T sf = (L.tb < 0 && s.t == L.Lt - 1) ? (T)-1 : (T)1;
  const T sb = (L.tb < 0 && s.t == 0) ? (T)-1 : (T)1;
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

// ---------------------------------------------------------------------------------------------
// Link staging through shared memory with cp.async (LDGSTS).  Links are 67-75 % of the bytes, are
// streamed exactly once and need no sharing between threads, so each thread copies ITS OWN eight
// links global->shared asynchronously at kernel entry (one commit group per hop): all link bytes of
// a block are in flight at once without holding a single register, independently of how ptxas
// schedules the arithmetic.  Layout in shared memory: [slot = hop][vector][thread] (conflict free).
// A thread only reads what it copied itself, so cp.async.wait_group is the only synchronisation.
// ---------------------------------------------------------------------------------------------
template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem_dst, const void* gsrc) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  if (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <typename T, int R, int BLOCK>
__device__ __forceinline__ void stage_link(void* smem, int slot, const T* __restrict__ block, int Vh, int lidx) {
  typedef typename GV<T, R>::vec vec;
  constexpr int NGV = R / GV<T, R>::N;
  vec* sl = reinterpret_cast<vec*>(smem) + (size_t)slot * NGV * BLOCK + threadIdx.x;
  const vec* g = reinterpret_cast<const vec*>(block) + lidx;
#pragma unroll
  for (int v = 0; v < NGV; v++) cp_async<sizeof(vec)>(sl + v * BLOCK, g + (size_t)v * Vh);
  cp_async_commit();
}
template <typename T, int R, int BLOCK>
__device__ __forceinline__ void fetch_link(const void* smem, int slot, T* U) {
  typedef typename GV<T, R>::vec vec;
  constexpr int N = GV<T, R>::N, NGV = R / N;
  const vec* sl = reinterpret_cast<const vec*>(smem) + (size_t)slot * NGV * BLOCK + threadIdx.x;
#pragma unroll
  for (int v = 0; v < NGV; v++) {
    vec q = sl[v * BLOCK];
    vec_get(q, U + v * N);
  }
  if (R == 12) recon_row2<T>(U);
}

template <typename T, int R, int MU, bool FWD, bool DAG, int BLOCK, int SLOT>
__device__ __forceinline__ void hop_staged(T* acc, const T* __restrict__ in, const void* smem, int Vh, int nidx, T bsign) {
  constexpr int S = (FWD != DAG) ? -1 : +1;
  T psi[24], U[18], h[12], chi[12];
  load_spinor<T>(in, Vh, nidx, psi);
  project<T, MU, S>(psi, h);
  cp_async_wait<7 - SLOT>();
  fetch_link<T, R, BLOCK>(smem, SLOT, U);
  su3_mul<T, !FWD>(U, h, chi);
  reconstruct<T, MU, S>(acc, chi, bsign);
}

template <typename T, int R, bool DAG, int BLOCK>
__device__ __forceinline__ void dslash_site_staged(T* acc, const T* __restrict__ in, const T* __restrict__ gauge,
                                                   const Lat& L, int idx, int par, void* smem, T ws) {
  const Site s = site_of(L, idx, par);
  const int Vh = L.Vh;
  const size_t blk = (size_t)R * Vh;
  const int n0 = neighbour<0, +1>(L, idx, s), n1 = neighbour<0, -1>(L, idx, s);
  const int n2 = neighbour<1, +1>(L, idx, s), n3 = neighbour<1, -1>(L, idx, s);
  const int n4 = neighbour<2, +1>(L, idx, s), n5 = neighbour<2, -1>(L, idx, s);
  const int n6 = neighbour<3, +1>(L, idx, s), n7 = neighbour<3, -1>(L, idx, s);
  stage_link<T, R, BLOCK>(smem, 0, gauge + (0 * 2 + par) * blk, Vh, idx);
  stage_link<T, R, BLOCK>(smem, 1, gauge + (0 * 2 + 1 - par) * blk, Vh, n1);
  stage_link<T, R, BLOCK>(smem, 2, gauge + (1 * 2 + par) * blk, Vh, idx);
  stage_link<T, R, BLOCK>(smem, 3, gauge + (1 * 2 + 1 - par) * blk, Vh, n3);
  stage_link<T, R, BLOCK>(smem, 4, gauge + (2 * 2 + par) * blk, Vh, idx);
  stage_link<T, R, BLOCK>(smem, 5, gauge + (2 * 2 + 1 - par) * blk, Vh, n5);
  stage_link<T, R, BLOCK>(smem, 6, gauge + (3 * 2 + par) * blk, Vh, idx);
  stage_link<T, R, BLOCK>(smem, 7, gauge + (3 * 2 + 1 - par) * blk, Vh, n7);
#pragma unroll
  for (int e = 0; e < 24; e++) acc[e] = 0;
  const T one = ws;  // weight of the spatial hops (Eq. 5: nu/xi_0); the temporal hops carry the boundary sign
  const T sf = (L.tb < 0 && s.t == L.Lt - 1) ? (T)-1 : (T)1;
  const T sb = (L.tb < 0 && s.t == 0) ? (T)-1 : (T)1;
  hop_staged<T, R, 0, true, DAG, BLOCK, 0>(acc, in, smem, Vh, n0, one);
  hop_staged<T, R, 0, false, DAG, BLOCK, 1>(acc, in, smem, Vh, n1, one);
  hop_staged<T, R, 1, true, DAG, BLOCK, 2>(acc, in, smem, Vh, n2, one);
  hop_staged<T, R, 1, false, DAG, BLOCK, 3>(acc, in, smem, Vh, n3, one);
  hop_staged<T, R, 2, true, DAG, BLOCK, 4>(acc, in, smem, Vh, n4, one);
  hop_staged<T, R, 2, false, DAG, BLOCK, 5>(acc, in, smem, Vh, n5, one);
  hop_staged<T, R, 3, true, DAG, BLOCK, 6>(acc, in, smem, Vh, n6, sf);
  hop_staged<T, R, 3, false, DAG, BLOCK, 7>(acc, in, smem, Vh, n7, sb);
}

// y = B x for one packed Hermitian 6x6 block (6 real diagonals, 15 complex lower entries), packed fp32:
// y_i = sum_j ar_ij (xr, xi)_j + (-1, 1) o sum_j (+-ai_ij) (xi, xr)_j  (lower triangle +, conjugated upper -)
__device__ __forceinline__ void clover_block_packed(const float* a, const float* x, float* y) {
#pragma unroll
  for (int i = 0; i < 6; i++) {
    u64 accr = mul2(pk2(a[i], a[i]), pk2(x[2 * i], x[2 * i + 1]));
    u64 acci;
    bool first = true;
#pragma unroll
    for (int j = 0; j < 6; j++) {
      if (j == i) continue;
      const int o = j < i ? 6 + 2 * (i * (i - 1) / 2 + j) : 6 + 2 * (j * (j - 1) / 2 + i);
      const float ar = a[o], ai = j < i ? a[o + 1] : -a[o + 1];
      const u64 X = pk2(x[2 * j], x[2 * j + 1]), Xs = pk2(x[2 * j + 1], x[2 * j]);
      accr = fma2(pk2(ar, ar), X, accr);
      acci = first ? mul2(pk2(ai, ai), Xs) : fma2(pk2(ai, ai), Xs, acci);
      first = false;
    }
    upk2(fma2(pk2(-1.f, 1.f), acci, accr), y[2 * i], y[2 * i + 1]);
  }
}

// y = B x for one packed Hermitian 6x6 block a[36] (6 real diagonals, then the 15 complex lower entries row-major);
// the ONE block multiply of the library: clover apply, every fused epilogue, single and multi right-hand side
template <typename T>
__device__ __forceinline__ void clover_block(const T* a, const T* x, T* y) {
  if constexpr (UsePacked<T>::value) {
    clover_block_packed(a, x, y);
  } else {
#pragma unroll
    for (int i = 0; i < 6; i++) {
      T re = a[i] * x[2 * i], im = a[i] * x[2 * i + 1];
#pragma unroll
      for (int j = 0; j < 6; j++) {
        if (j < i) {  // L_ij x_j
          const int o = 6 + 2 * (i * (i - 1) / 2 + j);
          re += a[o] * x[2 * j];
          re -= a[o + 1] * x[2 * j + 1];
          im += a[o] * x[2 * j + 1];
          im += a[o + 1] * x[2 * j];
        } else if (j > i) {  // conj(L_ji) x_j
          const int o = 6 + 2 * (j * (j - 1) / 2 + i);
          re += a[o] * x[2 * j];
          re += a[o + 1] * x[2 * j + 1];
          im += a[o] * x[2 * j + 1];
          im -= a[o + 1] * x[2 * j];
        }
      }
      y[2 * i] = re;
      y[2 * i + 1] = im;
    }
  }
}

// one chiral block (k = 0 upper, 1 lower) of site idx from a one-parity clover field [NCV][Vh]
template <typename T>
__device__ __forceinline__ void load_clover_block(const T* __restrict__ cl, int Vh, int idx, int k, T* a) {
  typedef typename V16<T>::vec vec;
  constexpr int N = V16<T>::N;
  const vec* p = reinterpret_cast<const vec*>(cl) + idx;
#pragma unroll
  for (int q = 0; q < 36 / N; q++) {
    vec w = ld_stream(p + (size_t)(k * (36 / N) + q) * Vh);
    vec_get(w, a + q * N);
  }
}

// out = C v for the two Hermitian 6x6 chiral blocks of one site.  cl = one-parity clover field
// [NCV][Vh]; packed order per block: 6 real diagonal, then 15 complex lower entries row-major.
// v and out are 24-real spinors (block k acts on reals 12k..12k+11); they must not alias.
template <typename T>
__device__ __forceinline__ void clover_mul(const T* __restrict__ cl, int Vh, int idx, const T* v, T* out) {
#pragma unroll
  for (int k = 0; k < 2; k++) {
    T a[36];
    load_clover_block<T>(cl, Vh, idx, k, a);
    clover_block<T>(a, v + 12 * k, out + 12 * k);
  }
}

// res = x + scale * C v  and  res2 = C res  with ONE pass over the clover field: each 6x6 chiral block is loaded
// once and used for both products (dslash.cu epilogue 9).  v, x, res, res2 are 24-real spinors; no aliasing.
template <typename T>
__device__ __forceinline__ void clover_mul_twice(const T* __restrict__ cl, int Vh, int idx, const T* v, const T* x, T scale,
                                                 T* res, T* res2) {
#pragma unroll
  for (int k = 0; k < 2; k++) {
    T a[36], y[12];
    load_clover_block<T>(cl, Vh, idx, k, a);
    clover_block<T>(a, v + 12 * k, y);
#pragma unroll
    for (int e = 0; e < 12; e++) res[12 * k + e] = x[12 * k + e] + scale * y[e];
    clover_block<T>(a, res + 12 * k, res2 + 12 * k);
  }
}
