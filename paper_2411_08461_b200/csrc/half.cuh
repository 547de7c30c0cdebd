// 16-bit storage (second half, ref. [1] "mixed precision solvers on GPUs"):
// a context created with prec = 2 keeps its NATIVE fields as 16-bit fixed point and does all arithmetic in fp32
// registers.  It is meant as the inner context of lqcd_invert_mixed (fp64 defect correction outside), where it
// halves the bytes of every inner iteration against fp32 storage.
//
//   spinor, one parity : short4 v[6][Vh] ; float norm[Vh]        value = v * norm / 32767, norm = max |component| of
//                                                               the site (52 B per site instead of 96)
//   links              : [mu][parity] short2 u[9][Vh] (18 reals) or short4 u[3][Vh] (12 reals: third row rebuilt in
//                        fp32), value = u / 32767 (|U_ij| <= 1 for SU(3): no norm needed)
//   clover, one parity : short4 c[18][Vh] ; float norm[2][Vh]    one norm per chiral 6x6 block (152 B per site)
// Rounding: a component carries an absolute error of norm / 65534 (relative 1.5e-5 of the site's largest component),
// a link entry 1.5e-5 absolute.
#pragma once
#include "dslash.cuh"

constexpr float HALF_MAX = 32767.f;

__device__ __forceinline__ short quant(float x, float inv) { return (short)__float2int_rn(x * inv); }

// one-parity spinor at `base`: the norms follow the 6 Vh vectors
__device__ __forceinline__ const float* half_spinor_norms(const void* base, int Vh) {
  return reinterpret_cast<const float*>(reinterpret_cast<const short4*>(base) + (size_t)6 * Vh);
}
__device__ __forceinline__ void load_spinor_h(const void* base, int Vh, int idx, float* psi) {
  const short4* p = reinterpret_cast<const short4*>(base) + idx;
  const float s = __ldg(half_spinor_norms(base, Vh) + idx) * (1.f / HALF_MAX);
#pragma unroll
  for (int v = 0; v < 6; v++) {
    const short4 q = __ldg(p + (size_t)v * Vh);
    psi[4 * v] = q.x * s;
    psi[4 * v + 1] = q.y * s;
    psi[4 * v + 2] = q.z * s;
    psi[4 * v + 3] = q.w * s;
  }
}
// plain (coherent) loads: for kernels whose input may alias their output
__device__ __forceinline__ void load_spinor_h_plain(const void* base, int Vh, int idx, float* psi) {
  const short4* p = reinterpret_cast<const short4*>(base) + idx;
  const float s = half_spinor_norms(base, Vh)[idx] * (1.f / HALF_MAX);
#pragma unroll
  for (int v = 0; v < 6; v++) {
    const short4 q = p[(size_t)v * Vh];
    psi[4 * v] = q.x * s;
    psi[4 * v + 1] = q.y * s;
    psi[4 * v + 2] = q.z * s;
    psi[4 * v + 3] = q.w * s;
  }
}
__device__ __forceinline__ void store_spinor_h(void* base, int Vh, int idx, const float* psi) {
  float m = 0.f;
#pragma unroll
  for (int e = 0; e < 24; e++) m = fmaxf(m, fabsf(psi[e]));
  const float inv = m > 0.f ? HALF_MAX / m : 0.f;
  short4* p = reinterpret_cast<short4*>(base) + idx;
#pragma unroll
  for (int v = 0; v < 6; v++)
    p[(size_t)v * Vh] = make_short4(quant(psi[4 * v], inv), quant(psi[4 * v + 1], inv), quant(psi[4 * v + 2], inv), quant(psi[4 * v + 3], inv));
  const_cast<float*>(half_spinor_norms(base, Vh))[idx] = m;
}

// link block of one (mu, parity): R Vh shorts
template <int R>
__device__ __forceinline__ void load_link_h(const short* __restrict__ block, int Vh, int idx, float* U) {
  constexpr float s = 1.f / HALF_MAX;
  if (R == 18) {
    const short2* p = reinterpret_cast<const short2*>(block) + idx;
#pragma unroll
    for (int v = 0; v < 9; v++) {
      const short2 q = __ldcs(p + (size_t)v * Vh);
      U[2 * v] = q.x * s;
      U[2 * v + 1] = q.y * s;
    }
  } else {
    const short4* p = reinterpret_cast<const short4*>(block) + idx;
#pragma unroll
    for (int v = 0; v < 3; v++) {
      const short4 q = __ldcs(p + (size_t)v * Vh);
      U[4 * v] = q.x * s;
      U[4 * v + 1] = q.y * s;
      U[4 * v + 2] = q.z * s;
      U[4 * v + 3] = q.w * s;
    }
    recon_row2<float>(U);
  }
}

// chiral block k of site idx from a one-parity clover field: short4 c[18][Vh] ; float norm[2][Vh]
__device__ __forceinline__ void load_clover_block_h(const void* __restrict__ cl, int Vh, int idx, int k, float* a) {
  const short4* p = reinterpret_cast<const short4*>(cl) + idx;
  const float* n = reinterpret_cast<const float*>(reinterpret_cast<const short4*>(cl) + (size_t)18 * Vh);
  const float s = __ldcs(n + (size_t)k * Vh + idx) * (1.f / HALF_MAX);
#pragma unroll
  for (int q = 0; q < 9; q++) {
    const short4 w = __ldcs(p + (size_t)(9 * k + q) * Vh);
    a[4 * q] = w.x * s;
    a[4 * q + 1] = w.y * s;
    a[4 * q + 2] = w.z * s;
    a[4 * q + 3] = w.w * s;
  }
}
__device__ __forceinline__ void clover_mul_h(const void* __restrict__ cl, int Vh, int idx, const float* v, float* out) {
#pragma unroll
  for (int k = 0; k < 2; k++) {
    float a[36];
    load_clover_block_h(cl, Vh, idx, k, a);
    clover_block<float>(a, v + 12 * k, out + 12 * k);
  }
}
