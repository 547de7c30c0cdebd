// Kernels of the 16-bit-storage context (half.cuh): hopping term with the fused clover epilogues, clover apply,
// pack / unpack, conversions from fp32 natives, and the down / up conversions of the mixed-precision solver.
// Single right-hand side; fp32 arithmetic (the packed FFMA2 device functions of dslash.cuh).
#include "half.cuh"

namespace {

struct HalfArgs {
  void* out;
  const void* in;
  const short* gauge;
  const void* cl;  // one-parity clover field of the output parity (EPI 1, 2, 3)
  const void* x;   // one-parity spinor of the output parity (EPI 2, 3, 6)
  Lat lat;
  int parity;
  float scale, ws;
  // epilogues 9 and 10 (CG recurrences of the right-preconditioned form, as in dslash.cu)
  void* r;
  void* out2;
  double* partial;
  const double* scalars;
  int num, den;
};

template <int R, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void hop_h(float* acc, const void* in, const short* links, int Vh, int nidx, int lidx, float w) {
  constexpr int S = (FWD != DAG) ? -1 : +1;
  float psi[24], U[18], h[12], chi[12];
  const float s = load_spinor_h_raw(in, Vh, nidx, psi);  // integers; the site's scale goes into the hop weight
  load_link_h<R>(links, Vh, lidx, U);
  project<float, MU, S>(psi, h);
  su3_mul<float, !FWD>(U, h, chi);
  reconstruct<float, MU, S>(acc, chi, w * s);
}

// EPI as in dslash.cu: 0 scale*d ; 1 scale*C d ; 2 C x + scale*d ; 3 x + scale*C d ; 6 x + scale*d
// block sum -> partial[block] (summed in a fixed order by lqcd_partial_sum_launch: deterministic)
__device__ __forceinline__ void half_block_sum(double v, double* partial) {
  __shared__ double sm[4];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) partial[blockIdx.x] = (sm[0] + sm[1]) + (sm[2] + sm[3]);
}

#ifndef HALF_MINB
#define HALF_MINB 4
#endif
template <int R, bool DAG, int EPI>
__global__ void __launch_bounds__(128, HALF_MINB) dslash_half_kernel(const HalfArgs a) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const Lat& L = a.lat;
  const int Vh = L.Vh, par = a.parity;
  if (idx >= Vh) {
    if (EPI == 9 || EPI == 10) half_block_sum(0.0, a.partial);  // the reduction needs every thread of the block
    return;
  }
  const Site s = site_of(L, idx, par);
  const size_t blk = (size_t)R * Vh;  // shorts per (mu, parity) link block
  float acc[24];
#pragma unroll
  for (int e = 0; e < 24; e++) acc[e] = 0.f;
  const float sf = (L.tb < 0 && s.t == L.Lt - 1) ? -1.f : 1.f, sb = (L.tb < 0 && s.t == 0) ? -1.f : 1.f;
  int n;
  n = neighbour<0, +1>(L, idx, s);
  hop_h<R, 0, true, DAG>(acc, a.in, a.gauge + (0 * 2 + par) * blk, Vh, n, idx, a.ws);
  n = neighbour<0, -1>(L, idx, s);
  hop_h<R, 0, false, DAG>(acc, a.in, a.gauge + (0 * 2 + 1 - par) * blk, Vh, n, n, a.ws);
  n = neighbour<1, +1>(L, idx, s);
  hop_h<R, 1, true, DAG>(acc, a.in, a.gauge + (1 * 2 + par) * blk, Vh, n, idx, a.ws);
  n = neighbour<1, -1>(L, idx, s);
  hop_h<R, 1, false, DAG>(acc, a.in, a.gauge + (1 * 2 + 1 - par) * blk, Vh, n, n, a.ws);
  n = neighbour<2, +1>(L, idx, s);
  hop_h<R, 2, true, DAG>(acc, a.in, a.gauge + (2 * 2 + par) * blk, Vh, n, idx, a.ws);
  n = neighbour<2, -1>(L, idx, s);
  hop_h<R, 2, false, DAG>(acc, a.in, a.gauge + (2 * 2 + 1 - par) * blk, Vh, n, n, a.ws);
  n = neighbour<3, +1>(L, idx, s);
  hop_h<R, 3, true, DAG>(acc, a.in, a.gauge + (3 * 2 + par) * blk, Vh, n, idx, sf);
  n = neighbour<3, -1>(L, idx, s);
  hop_h<R, 3, false, DAG>(acc, a.in, a.gauge + (3 * 2 + 1 - par) * blk, Vh, n, n, sb);
  float res[24];
  if (EPI == 0) {
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] = a.scale * acc[e];
  } else if (EPI == 1) {
    clover_mul_h(a.cl, Vh, idx, acc, res);
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] *= a.scale;
  } else if (EPI == 2) {
    float xv[24];
    load_spinor_h(a.x, Vh, idx, xv);
    clover_mul_h(a.cl, Vh, idx, xv, res);
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] += a.scale * acc[e];
  } else if (EPI == 3) {
    float xv[24];
    load_spinor_h(a.x, Vh, idx, xv);
    clover_mul_h(a.cl, Vh, idx, acc, res);
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] = xv[e] + a.scale * res[e];
  } else if (EPI == 9) {  // t = x + scale * C d ; ta = C t ; |t|^2 (of the value kept, i.e. before it is rounded to 16 bits)
    float xv[24], res2[24];
    load_spinor_h(a.x, Vh, idx, xv);
    clover_mul_h(a.cl, Vh, idx, acc, res);
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] = xv[e] + a.scale * res[e];
    clover_mul_h(a.cl, Vh, idx, res, res2);
    store_spinor_h(a.out2, Vh, idx, res2);
  } else {  // 6, 10: x + scale * d
    load_spinor_h(a.x, Vh, idx, res);
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] += a.scale * acc[e];
  }
  if (EPI == 10) {  // q = res is not stored: r -= (s[num]/s[den]) q, |r|^2
    double local = 0;
    if (a.scalars[S_DONE] == 0.0) {
      const float alpha = (float)(a.scalars[a.num] / a.scalars[a.den]);
      float rv[24];
      load_spinor_h_plain(a.r, Vh, idx, rv);
#pragma unroll
      for (int e = 0; e < 24; e++) {
        rv[e] -= alpha * res[e];
        local += (double)rv[e] * rv[e];
      }
      store_spinor_h(a.r, Vh, idx, rv);
    }
    half_block_sum(local, a.partial);
    return;
  }
  store_spinor_h(a.out, Vh, idx, res);
  if (EPI == 9) {
    double local = 0;
#pragma unroll
    for (int e = 0; e < 24; e++) local += (double)res[e] * res[e];
    half_block_sum(local, a.partial);
  }
}

// in and out may alias: plain loads, a thread reads its whole site before it stores
__global__ void __launch_bounds__(128) clover_apply_half_kernel(void* out, const void* in, const void* __restrict__ cl, int Vh) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= Vh) return;
  float v[24], r[24];
  load_spinor_h_plain(in, Vh, idx, v);
  clover_mul_h(cl, Vh, idx, v, r);
  store_spinor_h(out, Vh, idx, r);
}

template <int R, bool DAG>
void launch_epi_h(const HalfArgs& a, int epi, cudaStream_t st) {
  const int grid = (a.lat.Vh + 127) / 128;
  switch (epi) {
    case 0: dslash_half_kernel<R, DAG, 0><<<grid, 128, 0, st>>>(a); break;
    case 1: dslash_half_kernel<R, DAG, 1><<<grid, 128, 0, st>>>(a); break;
    case 2: dslash_half_kernel<R, DAG, 2><<<grid, 128, 0, st>>>(a); break;
    case 3: dslash_half_kernel<R, DAG, 3><<<grid, 128, 0, st>>>(a); break;
    case 9: dslash_half_kernel<R, DAG, 9><<<grid, 128, 0, st>>>(a); break;
    case 10: dslash_half_kernel<R, DAG, 10><<<grid, 128, 0, st>>>(a); break;
    default: dslash_half_kernel<R, DAG, 6><<<grid, 128, 0, st>>>(a); break;
  }
}

}  // namespace

// bytes of a 16-bit dslash launch: 2 B per real of links, spinors, clover, + 4 B per spinor norm and 8 B of clover norms
double lqcd_half_dslash_bytes(const lqcd_ctx* c, int epi) {
  const double sp = 24 * 2 + 4, cl = 72 * 2 + 8;
  return (double)c->lat.Vh * (8.0 * c->recon * 2 + 2 * sp + (epi >= 1 && epi != 6 ? cl : 0.0) + (epi >= 2 ? sp : 0.0));
}

int lqcd_dslash_half_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                            int parity, double scale, int dagger, int epi, cudaStream_t st, const DslashFuse* f) {
  if (!(epi <= 3 || epi == 6 || ((epi == 9 || epi == 10) && f)))
    return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "16-bit context: epilogue %d not built", epi);
  HalfArgs a;
  a.r = f ? f->r : nullptr;
  a.out2 = f ? f->out2 : nullptr;
  a.partial = c->d_partial;
  a.scalars = c->d_scalars;
  a.num = f ? f->num : 0;
  a.den = f ? f->den : 0;
  a.out = out;
  a.in = in;
  a.gauge = (const short*)gauge;
  a.cl = cl;
  a.x = x;
  a.lat = c->lat;
  a.parity = parity;
  a.scale = (float)scale;
  a.ws = (float)c->ws;
  const double bytes = lqcd_half_dslash_bytes(c, epi == 9 ? 3 : (epi == 10 ? 6 : epi)) + (epi >= 9 ? 52.0 * c->lat.Vh : 0.0);
  c->alg_bytes += bytes;
  const bool rec = c->prof_on && c->prof_n < c->prof_cap;
  if (rec) cudaEventRecord(c->prof_ev[2 * c->prof_n], st);
  if (c->recon == 18) {
    if (dagger) launch_epi_h<18, true>(a, epi, st);
    else launch_epi_h<18, false>(a, epi, st);
  } else {
    if (dagger) launch_epi_h<12, true>(a, epi, st);
    else launch_epi_h<12, false>(a, epi, st);
  }
  if (rec) {
    cudaEventRecord(c->prof_ev[2 * c->prof_n + 1], st);
    c->prof_n++;
    c->prof_bytes += bytes;
  }
  LQCD_LAUNCH_CHECK(c, "dslash_half");
  if (epi >= 9) return lqcd_partial_sum_launch(c, (c->lat.Vh + 127) / 128, f->out_slot, st);
  return LQCD_OK;
}

int lqcd_clover_apply_half_launch(lqcd_ctx* c, void* out, const void* in, const void* cl_parity, cudaStream_t st) {
  const int Vh = c->lat.Vh;
  c->alg_bytes += (double)Vh * (152.0 + 2 * 52.0);
  clover_apply_half_kernel<<<(Vh + 127) / 128, 128, 0, st>>>(out, in, cl_parity, Vh);
  LQCD_LAUNCH_CHECK(c, "clover_apply_half");
  return LQCD_OK;
}

// ---------------------------------------------------------------------------------------------
// pack / unpack (public arrays of a 16-bit context are complex64, reading B1) and conversions
// ---------------------------------------------------------------------------------------------
namespace {

// public links [8 (mu, parity) blocks][Vh][18] floats -> native shorts, first R reals of every link
template <int R>
__global__ void __launch_bounds__(256) gauge_pack_half_kernel(short* __restrict__ nat, const float* __restrict__ pub, int Vh) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x, b = blockIdx.y;
  if (idx >= Vh) return;
  const float* src = pub + ((size_t)b * Vh + idx) * 18;
  short* dst = nat + (size_t)b * R * Vh;
  if (R == 18) {
    unsigned* p = reinterpret_cast<unsigned*>(dst) + idx;
#pragma unroll
    for (int v = 0; v < 9; v++) p[(size_t)v * Vh] = enc2(src[2 * v], src[2 * v + 1], HALF_MAX);
  } else {
    uint2* p = reinterpret_cast<uint2*>(dst) + idx;
#pragma unroll
    for (int v = 0; v < 3; v++)
      p[(size_t)v * Vh] = make_uint2(enc2(src[4 * v], src[4 * v + 1], HALF_MAX), enc2(src[4 * v + 2], src[4 * v + 3], HALF_MAX));
  }
}
// public spinor [nblocks parities][Vh][24] floats <-> native, one block per blockIdx.y
__global__ void __launch_bounds__(256) spinor_pack_half_kernel(char* __restrict__ nat, const float* __restrict__ pub, int Vh, size_t nat_stride) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= Vh) return;
  const float* src = pub + ((size_t)blockIdx.y * Vh + idx) * 24;
  float psi[24];
#pragma unroll
  for (int e = 0; e < 24; e++) psi[e] = src[e];
  store_spinor_h(nat + blockIdx.y * nat_stride, Vh, idx, psi);
}
__global__ void __launch_bounds__(256) spinor_unpack_half_kernel(float* __restrict__ pub, const char* __restrict__ nat, int Vh, size_t nat_stride) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= Vh) return;
  float psi[24];
  load_spinor_h(nat + blockIdx.y * nat_stride, Vh, idx, psi);
  float* dst = pub + ((size_t)blockIdx.y * Vh + idx) * 24;
#pragma unroll
  for (int e = 0; e < 24; e++) dst[e] = psi[e];
}
// fp32 native clover (float4 c[18][Vh] per parity) -> 16-bit native, one norm per chiral block
__global__ void __launch_bounds__(256) clover_to_half_kernel(char* __restrict__ dst, const float4* __restrict__ src, int Vh) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x, par = blockIdx.y;
  if (idx >= Vh) return;
  const float4* s = src + (size_t)par * 18 * Vh + idx;
  char* d = dst + (size_t)par * 152 * Vh;
  uint2* p = reinterpret_cast<uint2*>(d) + idx;
  float* n = reinterpret_cast<float*>(reinterpret_cast<uint2*>(d) + (size_t)18 * Vh);
#pragma unroll
  for (int k = 0; k < 2; k++) {
    float4 a[9];
    float m = 0.f;
#pragma unroll
    for (int q = 0; q < 9; q++) {
      a[q] = s[(size_t)(9 * k + q) * Vh];
      m = fmaxf(m, fmaxf(fmaxf(fabsf(a[q].x), fabsf(a[q].y)), fmaxf(fabsf(a[q].z), fabsf(a[q].w))));
    }
    const float inv = m > 0.f ? HALF_MAX / m : 0.f;
#pragma unroll
    for (int q = 0; q < 9; q++)
      p[(size_t)(9 * k + q) * Vh] = make_uint2(enc2(a[q].x, a[q].y, inv), enc2(a[q].z, a[q].w, inv));
    n[(size_t)k * Vh + idx] = m;
  }
}
// mixed-precision solver: fp64 native spinor -> 16-bit (scaled), and x(fp64) += a * e(16-bit)
__global__ void __launch_bounds__(256) spinor_down_half_kernel(void* __restrict__ out, const double2* __restrict__ in, int Vh, double scale) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= Vh) return;
  float psi[24];
#pragma unroll
  for (int u = 0; u < 12; u++) {
    const double2 a = in[(size_t)u * Vh + i];
    psi[2 * u] = (float)(scale * a.x);
    psi[2 * u + 1] = (float)(scale * a.y);
  }
  store_spinor_h(out, Vh, i, psi);
}
__global__ void __launch_bounds__(256) spinor_up_axpy_half_kernel(double2* __restrict__ x, const void* __restrict__ e, int Vh, double a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= Vh) return;
  float psi[24];
  load_spinor_h(e, Vh, i, psi);
#pragma unroll
  for (int u = 0; u < 12; u++) {
    double2 p = x[(size_t)u * Vh + i];
    p.x += a * psi[2 * u];
    p.y += a * psi[2 * u + 1];
    x[(size_t)u * Vh + i] = p;
  }
}

}  // namespace

int lqcd_gauge_pack_half(lqcd_ctx* c, void* native, const void* pub, cudaStream_t st) {
  const int Vh = c->lat.Vh;
  const dim3 grid((Vh + 255) / 256, 8);
  if (c->recon == 18) gauge_pack_half_kernel<18><<<grid, 256, 0, st>>>((short*)native, (const float*)pub, Vh);
  else gauge_pack_half_kernel<12><<<grid, 256, 0, st>>>((short*)native, (const float*)pub, Vh);
  c->alg_bytes += (double)4 * c->V * 18 * 4 + (double)lqcd_gauge_bytes(c);
  LQCD_LAUNCH_CHECK(c, "gauge_pack_half");
  return LQCD_OK;
}
int lqcd_spinor_pack_half(lqcd_ctx* c, void* native, const void* pub, int parities, cudaStream_t st) {
  const int Vh = c->lat.Vh;
  spinor_pack_half_kernel<<<dim3((Vh + 255) / 256, parities), 256, 0, st>>>((char*)native, (const float*)pub, Vh, lqcd_spinor_bytes(c));
  c->alg_bytes += (double)parities * Vh * (96.0 + 52.0);
  LQCD_LAUNCH_CHECK(c, "spinor_pack_half");
  return LQCD_OK;
}
int lqcd_spinor_unpack_half(lqcd_ctx* c, void* pub, const void* native, int parities, cudaStream_t st) {
  const int Vh = c->lat.Vh;
  spinor_unpack_half_kernel<<<dim3((Vh + 255) / 256, parities), 256, 0, st>>>((float*)pub, (const char*)native, Vh, lqcd_spinor_bytes(c));
  c->alg_bytes += (double)parities * Vh * (96.0 + 52.0);
  LQCD_LAUNCH_CHECK(c, "spinor_unpack_half");
  return LQCD_OK;
}
int lqcd_spinor_down_half(lqcd_ctx* c, void* out, const void* in_fp64, double scale, cudaStream_t st) {
  const int Vh = c->lat.Vh;
  spinor_down_half_kernel<<<(Vh + 255) / 256, 256, 0, st>>>(out, (const double2*)in_fp64, Vh, scale);
  c->alg_bytes += (double)Vh * (192.0 + 52.0);
  LQCD_LAUNCH_CHECK(c, "spinor_down_half");
  return LQCD_OK;
}
int lqcd_spinor_up_axpy_half(lqcd_ctx* c, void* x_fp64, const void* e, double a, cudaStream_t st) {
  const int Vh = c->lat.Vh;
  spinor_up_axpy_half_kernel<<<(Vh + 255) / 256, 256, 0, st>>>((double2*)x_fp64, e, Vh, a);
  c->alg_bytes += (double)Vh * (2 * 192.0 + 52.0);
  LQCD_LAUNCH_CHECK(c, "spinor_up_axpy_half");
  return LQCD_OK;
}

extern "C" int lqcd_clover_to_half(lqcd_ctx* c, void* clover_half, const void* clover_fp32_native, void* stream) {
  if (!c || !clover_half || !clover_fp32_native) return LQCD_ERR_INVALID_ARG;
  if (!c->half) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "clover_to_half: needs a 16-bit context (prec = 2)");
  if (!lqcd_aligned16(clover_half) || !lqcd_aligned16(clover_fp32_native)) return lqcd_set_error(c, LQCD_ERR_ALIGN, "clover_to_half: alignment");
  const int Vh = c->lat.Vh;
  clover_to_half_kernel<<<dim3((Vh + 255) / 256, 2), 256, 0, as_stream(stream)>>>((char*)clover_half, (const float4*)clover_fp32_native, Vh);
  c->alg_bytes += (double)c->V * (288.0 + 152.0);
  LQCD_LAUNCH_CHECK(c, "clover_to_half");
  return LQCD_OK;
}
