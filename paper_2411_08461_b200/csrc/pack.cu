// K1: public cb2 array-of-structures <-> native structure-of-arrays ("QUDA needs to
// convert the data format to its native one ... only at the beginning and end of a function").
// Pure index permutations; reconstruct-12 drops the third link row here.
#include "lqcd_internal.cuh"

// One thread per (site, vector): reads N consecutive reals of the site's AoS record and writes
// one SoA vector, so the SoA side is perfectly coalesced and the AoS side is sector-contiguous.
template <typename T, typename VEC, int N, int REALS_PUB, int NVEC>
__global__ void aos_to_soa_kernel(VEC* __restrict__ soa, const T* __restrict__ aos, int nsites, long nblocks) {
  // grid.y enumerates independent [NVEC][nsites] blocks (parity, or mu*2+parity)
  long blk = blockIdx.y;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nsites * NVEC || blk >= nblocks) return;
  int site = i / NVEC, v = i % NVEC;
  const T* src = aos + ((size_t)blk * nsites + site) * REALS_PUB + v * N;
  T r[N];
#pragma unroll
  for (int k = 0; k < N; k++) r[k] = src[k];
  VEC q;
  vec_set(q, r);
  soa[((size_t)blk * NVEC + v) * nsites + site] = q;
}

template <typename T, typename VEC, int N, int REALS_PUB, int NVEC>
__global__ void soa_to_aos_kernel(T* __restrict__ aos, const VEC* __restrict__ soa, int nsites, long nblocks) {
  long blk = blockIdx.y;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nsites * NVEC || blk >= nblocks) return;
  int site = i / NVEC, v = i % NVEC;
  VEC q = soa[((size_t)blk * NVEC + v) * nsites + site];
  T r[N];
  vec_get(q, r);
  T* dst = aos + ((size_t)blk * nsites + site) * REALS_PUB + v * N;
#pragma unroll
  for (int k = 0; k < N; k++) dst[k] = r[k];
}

template <typename T, typename VEC, int N, int REALS_PUB, int NVEC>
static void launch_to_soa(void* soa, const void* aos, int nsites, int nblocks, cudaStream_t st) {
  dim3 grid((unsigned)(((long)nsites * NVEC + 255) / 256), nblocks);
  aos_to_soa_kernel<T, VEC, N, REALS_PUB, NVEC><<<grid, 256, 0, st>>>((VEC*)soa, (const T*)aos, nsites, nblocks);
}
template <typename T, typename VEC, int N, int REALS_PUB, int NVEC>
static void launch_to_aos(void* aos, const void* soa, int nsites, int nblocks, cudaStream_t st) {
  dim3 grid((unsigned)(((long)nsites * NVEC + 255) / 256), nblocks);
  soa_to_aos_kernel<T, VEC, N, REALS_PUB, NVEC><<<grid, 256, 0, st>>>((T*)aos, (const VEC*)soa, nsites, nblocks);
}

extern "C" {

int lqcd_gauge_pack(lqcd_ctx* c, void* native, const void* pub, void* stream) {
  if (!c || !native || !pub) return LQCD_ERR_INVALID_ARG;
  if (!lqcd_aligned16(native) || !lqcd_aligned16(pub)) return lqcd_set_error(c, LQCD_ERR_ALIGN, "gauge_pack: alignment");
  cudaStream_t st = as_stream(stream);
  const int Vh = c->lat.Vh;
  if (c->half) return lqcd_gauge_pack_half(c, native, pub, st);
  if (c->prec == 4 && c->recon == 18) launch_to_soa<float, float2, 2, 18, 9>(native, pub, Vh, 8, st);
  else if (c->prec == 4) launch_to_soa<float, float4, 4, 18, 3>(native, pub, Vh, 8, st);
  else if (c->recon == 18) launch_to_soa<double, double2, 2, 18, 9>(native, pub, Vh, 8, st);
  else launch_to_soa<double, double2, 2, 18, 6>(native, pub, Vh, 8, st);
  c->alg_bytes += (double)4 * c->V * 18 * c->prec + (double)lqcd_gauge_bytes(c);
  LQCD_LAUNCH_CHECK(c, "gauge_pack");
  return LQCD_OK;
}

int lqcd_spinor_pack(lqcd_ctx* c, void* native, const void* pub, void* stream) {
  if (!c || !native || !pub) return LQCD_ERR_INVALID_ARG;
  if (!lqcd_aligned16(native) || !lqcd_aligned16(pub)) return lqcd_set_error(c, LQCD_ERR_ALIGN, "spinor_pack: alignment");
  cudaStream_t st = as_stream(stream);
  if (c->half) return lqcd_spinor_pack_half(c, native, pub, 2, st);
  if (c->prec == 4) launch_to_soa<float, float4, 4, 24, 6>(native, pub, c->lat.Vh, 2, st);
  else launch_to_soa<double, double2, 2, 24, 12>(native, pub, c->lat.Vh, 2, st);
  c->alg_bytes += 4.0 * (double)lqcd_spinor_bytes(c);
  LQCD_LAUNCH_CHECK(c, "spinor_pack");
  return LQCD_OK;
}

int lqcd_spinor_unpack(lqcd_ctx* c, void* pub, const void* native, void* stream) {
  if (!c || !native || !pub) return LQCD_ERR_INVALID_ARG;
  if (!lqcd_aligned16(native) || !lqcd_aligned16(pub)) return lqcd_set_error(c, LQCD_ERR_ALIGN, "spinor_unpack: alignment");
  cudaStream_t st = as_stream(stream);
  if (c->half) return lqcd_spinor_unpack_half(c, pub, native, 2, st);
  if (c->prec == 4) launch_to_aos<float, float4, 4, 24, 6>(pub, native, c->lat.Vh, 2, st);
  else launch_to_aos<double, double2, 2, 24, 12>(pub, native, c->lat.Vh, 2, st);
  c->alg_bytes += 4.0 * (double)lqcd_spinor_bytes(c);
  LQCD_LAUNCH_CHECK(c, "spinor_unpack");
  return LQCD_OK;
}

int lqcd_clover_unpack(lqcd_ctx* c, void* pub, const void* native, void* stream) {
  if (!c || !native || !pub) return LQCD_ERR_INVALID_ARG;
  if (!lqcd_aligned16(native) || !lqcd_aligned16(pub)) return lqcd_set_error(c, LQCD_ERR_ALIGN, "clover_unpack: alignment");
  cudaStream_t st = as_stream(stream);
  if (c->half) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "clover_unpack: not available in a 16-bit context (convert from an fp32 one: lqcd_clover_to_half)");
  if (c->prec == 4) launch_to_aos<float, float4, 4, 72, 18>(pub, native, c->lat.Vh, 2, st);
  else launch_to_aos<double, double2, 2, 72, 36>(pub, native, c->lat.Vh, 2, st);
  c->alg_bytes += 2.0 * (double)lqcd_clover_bytes(c);
  LQCD_LAUNCH_CHECK(c, "clover_unpack");
  return LQCD_OK;
}

// public packed clover [2][Vh][2][36] reals -> native (the inverse of lqcd_clover_unpack): a field built elsewhere, e.g.
// the sub-lattice's part of a clover field built on the whole lattice (domain decomposition, dd.py)
int lqcd_clover_pack(lqcd_ctx* c, void* native, const void* pub, void* stream) {
  if (!c || !native || !pub) return LQCD_ERR_INVALID_ARG;
  if (!lqcd_aligned16(native) || !lqcd_aligned16(pub)) return lqcd_set_error(c, LQCD_ERR_ALIGN, "clover_pack: alignment");
  if (c->half) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "clover_pack: not available in a 16-bit context (lqcd_clover_to_half)");
  cudaStream_t st = as_stream(stream);
  if (c->prec == 4) launch_to_soa<float, float4, 4, 72, 18>(native, pub, c->lat.Vh, 2, st);
  else launch_to_soa<double, double2, 2, 72, 36>(native, pub, c->lat.Vh, 2, st);
  c->alg_bytes += 2.0 * (double)lqcd_clover_bytes(c);
  LQCD_LAUNCH_CHECK(c, "clover_pack");
  return LQCD_OK;
}

}  // extern "C"

// one-parity spinor pack/unpack (used by the *_host entry points)
int lqcd_spinor_pack_parity(lqcd_ctx* c, void* native, const void* pub, cudaStream_t st) {
  if (c->half) return lqcd_spinor_pack_half(c, native, pub, 1, st);
  if (c->prec == 4) launch_to_soa<float, float4, 4, 24, 6>(native, pub, c->lat.Vh, 1, st);
  else launch_to_soa<double, double2, 2, 24, 12>(native, pub, c->lat.Vh, 1, st);
  c->alg_bytes += 2.0 * (double)lqcd_spinor_bytes(c);
  LQCD_LAUNCH_CHECK(c, "spinor_pack_parity");
  return LQCD_OK;
}
int lqcd_spinor_unpack_parity(lqcd_ctx* c, void* pub, const void* native, cudaStream_t st) {
  if (c->half) return lqcd_spinor_unpack_half(c, pub, native, 1, st);
  if (c->prec == 4) launch_to_aos<float, float4, 4, 24, 6>(pub, native, c->lat.Vh, 1, st);
  else launch_to_aos<double, double2, 2, 24, 12>(pub, native, c->lat.Vh, 1, st);
  c->alg_bytes += 2.0 * (double)lqcd_spinor_bytes(c);
  LQCD_LAUNCH_CHECK(c, "spinor_unpack_parity");
  return LQCD_OK;
}
