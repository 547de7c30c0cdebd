// 16-bit storage (second half, ref. [1] "mixed precision solvers on GPUs"):
// a context created with prec = 2 keeps its NATIVE fields as 16-bit fixed point and does all arithmetic in fp32
// registers.  It is meant as the inner context of lqcd_invert_mixed (fp64 defect correction outside), where it
// halves the bytes of every inner iteration against fp32 storage.
//
//   spinor, one parity : 4 x 16 bit v[6][Vh] ; float norm[Vh]    value = v * norm / 32767, norm = max |component| of
//                                                               the site (52 B per site instead of 96)
//   links              : [mu][parity] 2 x 16 bit u[9][Vh] (18 reals) or 4 x 16 bit u[3][Vh] (12 reals: third row rebuilt in
//                        fp32), value = u / 32767 (|U_ij| <= 1 for SU(3): no norm needed)
//   clover, one parity : 4 x 16 bit c[18][Vh] ; float norm[2][Vh] one norm per chiral 6x6 block (152 B per site)
// Rounding: a component carries an absolute error of norm / 65534 (relative 1.5e-5 of the site's largest component),
// a link entry 1.5e-5 absolute.
#pragma once
#include "dslash.cuh"

constexpr float HALF_MAX = 32767.f;

// Stored integers are OFFSET BINARY, u = q + 32768 in an unsigned 16-bit field, so that both conversions run on the
// full-rate pipes instead of I2F / F2I (a quarter of the FP32 rate: 200 conversions per site made the first version of
// the 16-bit dslash slower than the fp32 one):
//   decode: PRMT puts u under the exponent of 2^23 -> the float 8388608 + u exactly; subtracting 8421376 = 2^23 + 2^15
//           (exact, both are integers below 2^24) leaves q; one multiply by the site's scale;
//   encode: fma(x, 32767 / norm, 12615680) with 12615680 = 1.5 * 2^23 + 2^15 rounds x * 32767 / norm to the nearest
//           integer (ties to even, a single rounding) and leaves u in the low 16 bits of the result.
// A zeroed buffer (u = 0, norm = 0) still reads as zero.
constexpr float HALF_DEC = 8421376.f, HALF_ENC = 12615680.f;
// two stored fields -> the two integers q as floats (exact): 2 PRMT + one packed add (fma.rn.f32x2 with multiplicand 1)
__device__ __forceinline__ void dec2_raw(unsigned w, float& lo, float& hi) {
  const u64 v = pk2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610)),   // bytes: w0 w1 00 4B
                    __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632)));  // bytes: w2 w3 00 4B
  upk2(fma2(v, pk2(1.f, 1.f), pk2(-HALF_DEC, -HALF_DEC)), lo, hi);
}
// ... and scaled: one packed multiply more
__device__ __forceinline__ void dec2(unsigned w, float s, float& lo, float& hi) {
  const u64 v = pk2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7610)), __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7632)));
  upk2(mul2(fma2(v, pk2(1.f, 1.f), pk2(-HALF_DEC, -HALF_DEC)), pk2(s, s)), lo, hi);
}
__device__ __forceinline__ unsigned enc2(float lo, float hi, float inv) {
  const unsigned a = __float_as_uint(fmaf(lo, inv, HALF_ENC)), b = __float_as_uint(fmaf(hi, inv, HALF_ENC));
  return __byte_perm(a, b, 0x5410);  // low halves of a and b
}

// one-parity spinor at `base`: the norms follow the 6 Vh vectors
__device__ __forceinline__ const float* half_spinor_norms(const void* base, int Vh) {
  return reinterpret_cast<const float*>(reinterpret_cast<const uint2*>(base) + (size_t)6 * Vh);
}
template <bool NC>
__device__ __forceinline__ void load_spinor_h_impl(const void* base, int Vh, int idx, float* psi) {
  const uint2* p = reinterpret_cast<const uint2*>(base) + idx;
  const float* np = half_spinor_norms(base, Vh) + idx;
  const float s = (NC ? __ldg(np) : *np) * (1.f / HALF_MAX);
#pragma unroll
  for (int v = 0; v < 6; v++) {
    const uint2 q = NC ? __ldg(p + (size_t)v * Vh) : p[(size_t)v * Vh];
    dec2(q.x, s, psi[4 * v], psi[4 * v + 1]);
    dec2(q.y, s, psi[4 * v + 2], psi[4 * v + 3]);
  }
}
__device__ __forceinline__ void load_spinor_h(const void* base, int Vh, int idx, float* psi) { load_spinor_h_impl<true>(base, Vh, idx, psi); }
// the 24 stored integers as floats and the site's scale norm / 32767 apart: projection, SU(3) multiply and
// reconstruction are linear, so a hop multiplies by the scale once, in its weight, instead of 24 times here
__device__ __forceinline__ float load_spinor_h_raw(const void* base, int Vh, int idx, float* q24) {
  const uint2* p = reinterpret_cast<const uint2*>(base) + idx;
#pragma unroll
  for (int v = 0; v < 6; v++) {
    const uint2 q = __ldg(p + (size_t)v * Vh);
    dec2_raw(q.x, q24[4 * v], q24[4 * v + 1]);
    dec2_raw(q.y, q24[4 * v + 2], q24[4 * v + 3]);
  }
  return __ldg(half_spinor_norms(base, Vh) + idx) * (1.f / HALF_MAX);
}
// plain (coherent) loads: for kernels whose input may alias their output
__device__ __forceinline__ void load_spinor_h_plain(const void* base, int Vh, int idx, float* psi) { load_spinor_h_impl<false>(base, Vh, idx, psi); }
__device__ __forceinline__ void store_spinor_h(void* base, int Vh, int idx, const float* psi) {
  float m = 0.f;
#pragma unroll
  for (int e = 0; e < 24; e++) m = fmaxf(m, fabsf(psi[e]));
  const float inv = m > 0.f ? HALF_MAX / m : 0.f;
  uint2* p = reinterpret_cast<uint2*>(base) + idx;
#pragma unroll
  for (int v = 0; v < 6; v++) p[(size_t)v * Vh] = make_uint2(enc2(psi[4 * v], psi[4 * v + 1], inv), enc2(psi[4 * v + 2], psi[4 * v + 3], inv));
  const_cast<float*>(half_spinor_norms(base, Vh))[idx] = m;
}

// link block of one (mu, parity): R Vh 16-bit fields
template <int R>
__device__ __forceinline__ void load_link_h(const short* __restrict__ block, int Vh, int idx, float* U) {
  constexpr float s = 1.f / HALF_MAX;
  if (R == 18) {
    const unsigned* p = reinterpret_cast<const unsigned*>(block) + idx;
#pragma unroll
    for (int v = 0; v < 9; v++) dec2(__ldcs(p + (size_t)v * Vh), s, U[2 * v], U[2 * v + 1]);
  } else {
    const uint2* p = reinterpret_cast<const uint2*>(block) + idx;
#pragma unroll
    for (int v = 0; v < 3; v++) {
      const uint2 q = __ldcs(p + (size_t)v * Vh);
      dec2(q.x, s, U[4 * v], U[4 * v + 1]);
      dec2(q.y, s, U[4 * v + 2], U[4 * v + 3]);
    }
    recon_row2<float>(U);
  }
}

// chiral block k of site idx from a one-parity clover field: 4 x 16 bit c[18][Vh] ; float norm[2][Vh]
__device__ __forceinline__ void load_clover_block_h(const void* __restrict__ cl, int Vh, int idx, int k, float* a) {
  const uint2* p = reinterpret_cast<const uint2*>(cl) + idx;
  const float* n = reinterpret_cast<const float*>(reinterpret_cast<const uint2*>(cl) + (size_t)18 * Vh);
  const float s = __ldcs(n + (size_t)k * Vh + idx) * (1.f / HALF_MAX);
#pragma unroll
  for (int q = 0; q < 9; q++) {
    const uint2 w = __ldcs(p + (size_t)(9 * k + q) * Vh);
    dec2(w.x, s, a[4 * q], a[4 * q + 1]);
    dec2(w.y, s, a[4 * q + 2], a[4 * q + 3]);
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
