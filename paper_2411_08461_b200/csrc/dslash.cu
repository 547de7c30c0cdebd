// K2 dslash kernel with fused epilogues and K3 clover apply.
#include "dslash.cuh"
#include "dslash_tiled.cuh"

// Epilogues (EPI), with d = D_{p,1-p} in  and C = the clover-like field passed in `cl`:
//   0: out = scale * d
//   1: out = scale * C d                 (e.g. A_oo^-1 D_oe x)
//   2: out = C x + scale * d             (asymmetric Mhat:  A_ee x - k^2 D_eo t)
//   3: out = x + scale * C d             (symmetric  Mhat:  x - k^2 A_ee^-1 D_eo t)
// Epilogues fused with the CG recurrences (single right-hand side; fp64 reduction, deterministic:
// per-block partials summed in block order by the last block to finish):
//   4: out = C x + scale * d ; s[out_slot] = |out|^2                          (t = Mhat^dag p, <p, A p>)
//   5: q   = C x + scale * d ; r -= (s[num]/s[den]) q ; s[out_slot] = |r|^2   (q never stored)
// Symmetric form (Mhat_s = 1 - k^2 A_ee^-1 D_eo A_oo^-1 D_oe; its adjoint ends in a hop with no clover factor):
//   6: out = x + scale * d               (Mhat_s^dag y = y - k^2 D^dag_eo A_oo^-1 D^dag_oe A_ee^-1 y)
//   7: as 6 ; s[out_slot] = |out|^2
//   8: q   = x + scale * C d ; r -= (s[num]/s[den]) q ; s[out_slot] = |r|^2   (3 fused with the recurrence)
// Right-preconditioned symmetric form (Mhat_r = 1 - k^2 D_eo A_oo^-1 D_oe A_ee^-1, unknown y = A_ee x_e):
//   9: out = x + scale * C d ; out2 = C out ; s[out_slot] = |out|^2           (t = Mhat_r^dag p and A_ee^-1 t)
//  10: q   = x + scale * d   ; r -= (s[num]/s[den]) q ; s[out_slot] = |r|^2   (q = Mhat_r t never stored)
// BiCGStab on the left-symmetric form (as in dslash_mrhs.cu): epilogue 3 with the inner products of the next step,
//  11: out = x + scale * C d ; s[out_slot..+2] = Re<out,x>, Im<out,x>, |out|^2        (t = Mhat s: <t,s>, |t|^2)
//  12: out = x + scale * C d ; s[out_slot..+2] = Re<y,out>, Im<y,out>, |y|^2, y = r   (v = Mhat p: <r0,v>)
// Closing steps of a solve (as in dslash_mrhs.cu):
//  13: s[out_slot] = |y - (C x + scale * d)|^2, y = r, nothing stored   (one parity of the true residual b - M x)
//  14: out = C (x + scale * d)                                           (b-hat of the left-symmetric form; x_o)
template <typename T> struct DslashArgs {
  T* out;
  const T* in;
  const T* gauge;
  const T* cl;  // one-parity clover field of the OUTPUT parity (every EPI but 0, 6, 7)
  const T* x;   // one-parity spinor of the OUTPUT parity (EPI >= 2)
  Lat lat;
  int parity;
  T scale;
  T ws;  // weight of the spatial hops (anisotropy nu/xi_0; 1 = isotropic)
  // EPI 4, 5, 7, 8, 9, 10 only
  T* r;
  T* out2;  // EPI 9: second output, C * out
  double* partial;
  double* scalars;
  int num, den;
};

// Launch shape per precision (threads per block, minimum resident blocks per SM = register budget).
// The kernel is latency bound: what matters is how many independent loads ptxas can hoist per
// thread, which the register budget controls; values chosen by the round-1 sweep (profiles/r01d_tuning.md; the first sweep is in the git history).
#ifndef DSLASH_BLOCK_F32
#define DSLASH_BLOCK_F32 128
#endif
#ifndef DSLASH_MINB_F32
#define DSLASH_MINB_F32 4
#endif
#ifndef DSLASH_BLOCK_F64
#define DSLASH_BLOCK_F64 64
#endif
#ifndef DSLASH_MINB_F64
#define DSLASH_MINB_F64 5
#endif
#ifndef DSLASH_STAGE_F64_R12
#define DSLASH_STAGE_F64_R12 1  // cp.async link staging pays for fp64 12-real links only (round-1 sweep, profiles/r01d_tuning.md)
#endif
#ifndef DSLASH_MINB_F64_R12
#define DSLASH_MINB_F64_R12 4
#endif
template <typename T, int R> struct Tune;
template <> struct Tune<float, 18> { static constexpr int BLOCK = DSLASH_BLOCK_F32, MINB = DSLASH_MINB_F32; static constexpr bool STAGE = false; };
template <> struct Tune<float, 12> { static constexpr int BLOCK = DSLASH_BLOCK_F32, MINB = DSLASH_MINB_F32; static constexpr bool STAGE = false; };
template <> struct Tune<double, 18> { static constexpr int BLOCK = DSLASH_BLOCK_F64, MINB = DSLASH_MINB_F64; static constexpr bool STAGE = false; };
template <> struct Tune<double, 12> { static constexpr int BLOCK = DSLASH_BLOCK_F64, MINB = DSLASH_MINB_F64_R12; static constexpr bool STAGE = DSLASH_STAGE_F64_R12; };

// Deterministic fp64 grid reduction of the fused epilogues: block sum -> partial[block] (no fence, no
// atomic: a ticket scheme inside the stencil kernel cost 25 us per launch in block-retirement latency),
// then one small kernel sums the partials in a fixed order -> scalars[out_slot].
template <int BLOCK>
__device__ __forceinline__ void dslash_reduce(double v, double* partial) {
  __shared__ double sm[BLOCK / 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if (lane == 0) sm[warp] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0;
#pragma unroll
    for (int w = 0; w < BLOCK / 32; w++) t += sm[w];
    partial[blockIdx.x] = t;
  }
}
// three sums per block (epilogues 11, 12): partial[k * gridDim.x + block]
template <int BLOCK>
__device__ __forceinline__ void dslash_reduce3(const double (&v)[3], double* partial) {
  __shared__ double sm3[3][BLOCK / 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < 3; k++) {
    double t = v[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    if (lane == 0) sm3[k][warp] = t;
  }
  __syncthreads();
  if (threadIdx.x < 3) {
    double t = 0;
#pragma unroll
    for (int w = 0; w < BLOCK / 32; w++) t += sm3[threadIdx.x][w];
    partial[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = t;
  }
}
constexpr int PSUM_BLOCK = 1024;
__global__ void __launch_bounds__(PSUM_BLOCK) partial_sum_kernel(const double* __restrict__ partial, int n, double* out) {
  __shared__ double sm[PSUM_BLOCK / 32];
  partial += (size_t)blockIdx.x * n;  // block k: the k-th sum of the launch (epilogues 11, 12: three), consecutive slots
  out += blockIdx.x;
  double t0 = 0, t1 = 0, t2 = 0, t3 = 0;  // four independent chains, fixed assignment: deterministic
  int b = threadIdx.x;
  for (; b + 3 * PSUM_BLOCK < n; b += 4 * PSUM_BLOCK) {
    t0 += partial[b];
    t1 += partial[b + PSUM_BLOCK];
    t2 += partial[b + 2 * PSUM_BLOCK];
    t3 += partial[b + 3 * PSUM_BLOCK];
  }
  for (; b < n; b += PSUM_BLOCK) t0 += partial[b];
  double v = (t0 + t1) + (t2 + t3);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if (lane == 0) sm[warp] = v;
  __syncthreads();
  if (warp == 0) {
    v = sm[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) *out = v;
  }
}

__host__ __device__ constexpr bool epi_reduces(int epi) { return epi == 4 || epi == 5 || (epi >= 7 && epi != 14); }

// epilogue of one output site (EPI as listed at the top); `local` collects the fp64 reduction term
template <typename T, int EPI>
__device__ __forceinline__ void dslash_epilogue(const DslashArgs<T>& a, int idx, const T* acc, double (&loc)[3]) {
  double& local = loc[0];
  const int Vh = a.lat.Vh;
  T res[24];
  if (EPI == 0) {
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] = a.scale * acc[e];
  } else if (EPI == 1) {
    clover_mul<T>(a.cl, Vh, idx, acc, res);
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] *= a.scale;
  } else if (EPI == 2 || EPI == 4 || EPI == 5 || EPI == 13) {
    T xv[24];
    load_spinor<T>(a.x, Vh, idx, xv);
    clover_mul<T>(a.cl, Vh, idx, xv, res);
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] += a.scale * acc[e];
  } else if (EPI == 6 || EPI == 7 || EPI == 10) {
    load_spinor<T>(a.x, Vh, idx, res);
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] += a.scale * acc[e];
  } else if (EPI == 14) {
    T xv[24];
    load_spinor<T>(a.x, Vh, idx, xv);
#pragma unroll
    for (int e = 0; e < 24; e++) xv[e] += a.scale * acc[e];
    clover_mul<T>(a.cl, Vh, idx, xv, res);
  } else if (EPI == 9) {
    T xv[24], res2[24];
    load_spinor<T>(a.x, Vh, idx, xv);
    clover_mul_twice<T>(a.cl, Vh, idx, acc, xv, a.scale, res, res2);
    store_spinor<T>(a.out2, Vh, idx, res2);
  } else {
    T xv[24];
    load_spinor<T>(a.x, Vh, idx, xv);
    clover_mul<T>(a.cl, Vh, idx, acc, res);
#pragma unroll
    for (int e = 0; e < 24; e++) res[e] = xv[e] + a.scale * res[e];
  }
  if (EPI == 5 || EPI == 8 || EPI == 10) {
    if (a.scalars[S_DONE] != 0.0) return;  // converged (device-side stopping test, solver.cu): r keeps its value
    const T alpha = (T)(a.scalars[a.num] / a.scalars[a.den]);
    T rv[24];
    load_spinor<T>(a.r, Vh, idx, rv);
#pragma unroll
    for (int e = 0; e < 24; e++) {
      rv[e] -= alpha * res[e];
      local += (double)rv[e] * rv[e];
    }
    store_spinor<T>(a.r, Vh, idx, rv);
  } else if (EPI == 13) {
    T yv[24];
    load_spinor<T>(a.r, Vh, idx, yv);
#pragma unroll
    for (int e = 0; e < 24; e++) {
      const double dlt = (double)yv[e] - (double)res[e];
      local += dlt * dlt;
    }
  } else {
    if (EPI == 4 || EPI == 7 || EPI == 9) {
#pragma unroll
      for (int e = 0; e < 24; e++) local += (double)res[e] * res[e];
    }
    if (EPI == 11 || EPI == 12) {
      // <u,w> = sum conj(u) w with (u, w) = (out, x) for 11, (y, out) for 12
      T wv[24];
      load_spinor<T>(EPI == 11 ? a.x : a.r, Vh, idx, wv);
#pragma unroll
      for (int e = 0; e < 24; e += 2) {
        const double ur = EPI == 11 ? res[e] : wv[e], ui = EPI == 11 ? res[e + 1] : wv[e + 1];
        const double wr = EPI == 11 ? wv[e] : res[e], wi = EPI == 11 ? wv[e + 1] : res[e + 1];
        loc[0] += ur * wr + ui * wi;
        loc[1] += ur * wi - ui * wr;
        loc[2] += ur * ur + ui * ui;
      }
    }
    store_spinor<T>(a.out, Vh, idx, res);
  }
}

template <typename T, int R, bool DAG, int EPI>
__global__ void __launch_bounds__(Tune<T, R>::BLOCK, Tune<T, R>::MINB) dslash_kernel(const DslashArgs<T> a) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = idx < a.lat.Vh;
  if (!epi_reduces(EPI) && !live) return;
  double local[3] = {0, 0, 0};
  if (live) {
    T acc[24];
    if (Tune<T, R>::STAGE) {
      extern __shared__ __align__(16) unsigned char dslash_smem[];
      dslash_site_staged<T, R, DAG, Tune<T, R>::BLOCK>(acc, a.in, a.gauge, a.lat, idx, a.parity, dslash_smem, a.ws);
    } else {
      dslash_site<T, R, DAG>(acc, a.in, a.gauge, a.lat, idx, a.parity, a.ws);
    }
    dslash_epilogue<T, EPI>(a, idx, acc, local);
  }
  if (EPI == 11 || EPI == 12) dslash_reduce3<Tune<T, R>::BLOCK>(local, a.partial);
  else if (epi_reduces(EPI)) dslash_reduce<Tune<T, R>::BLOCK>(local[0], a.partial);
}

// in and out may alias (lqcd.h: lqcd_clover_apply; the solvers apply A_ee^-1 in place): no __restrict__ and plain
// (coherent) loads on `in`; a thread reads its whole site before it stores
template <typename T>
__global__ void __launch_bounds__(128) clover_apply_kernel(T* out, const T* in, const T* __restrict__ cl, int Vh) {
  typedef typename V16<T>::vec vec;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= Vh) return;
  out += (size_t)blockIdx.y * 24 * Vh;  // right-hand side
  in += (size_t)blockIdx.y * 24 * Vh;
  T v[24], r[24];
  const vec* p = reinterpret_cast<const vec*>(in) + idx;
#pragma unroll
  for (int q = 0; q < Lay<T>::NSV; q++) {
    const vec w = p[(size_t)q * Vh];
    vec_get(w, v + q * V16<T>::N);
  }
  clover_mul<T>(cl, Vh, idx, v, r);
  store_spinor<T>(out, Vh, idx, r);
}

// ---------------------------------------------------------------------------------------------
// Tiled kernel (dslash_tiled.cuh): block = one 4-D tile of output sites, neighbour spinors staged through
// shared memory.  Tile shape and resident blocks per precision (sweep in profiles/r01d_tuning.md).
// ---------------------------------------------------------------------------------------------
// output sites per tile: XH (checkerboard sites in x), Y, Z, T
#ifndef TILE_F32_XH
#define TILE_F32_XH 4
#define TILE_F32_Y 4
#define TILE_F32_Z 4
#define TILE_F32_T 4
#endif
#ifndef TILE_F64_XH
#define TILE_F64_XH 4
#define TILE_F64_Y 4
#define TILE_F64_Z 4
#define TILE_F64_T 2
#endif
#define TILE_F32 TILE_F32_XH, TILE_F32_Y, TILE_F32_Z, TILE_F32_T
#define TILE_F64 TILE_F64_XH, TILE_F64_Y, TILE_F64_Z, TILE_F64_T
#ifndef TILE_MINB_F32
#define TILE_MINB_F32 2
#endif
#ifndef TILE_MINB_F64
#define TILE_MINB_F64 2
#endif
template <typename T> struct TileOf;
template <> struct TileOf<float> { typedef TileShape<TILE_F32> TS; static constexpr int MINB = TILE_MINB_F32, NOUT = TS::NOUT; };
template <> struct TileOf<double> { typedef TileShape<TILE_F64> TS; static constexpr int MINB = TILE_MINB_F64, NOUT = TS::NOUT; };

template <typename T, int R, bool DAG, int EPI>
__global__ void __launch_bounds__(TileOf<T>::NOUT, TileOf<T>::MINB) dslash_tiled_kernel(const DslashArgs<T> a) {
  typedef typename TileOf<T>::TS TS;
  extern __shared__ __align__(16) unsigned char dslash_smem[];
  const Lat& L = a.lat;
  const int ntx = L.Lxh / TS::TXH, nty = L.Ly / TS::TY, ntz = L.Lz / TS::TZ;
  int b = blockIdx.x;
  const int x0 = 2 * TS::TXH * (b % ntx);
  b /= ntx;
  const int y0 = TS::TY * (b % nty);
  b /= nty;
  const int z0 = TS::TZ * (b % ntz);
  const int t0 = TS::TT * (b / ntz);
  tile_stage<T, TS>(dslash_smem, a.in, L, x0, y0, z0, t0, 1 - a.parity);
  int q = threadIdx.x;
  const int lxh = q % TS::TXH;
  q /= TS::TXH;
  const int ly = q % TS::TY;
  q /= TS::TY;
  const int lz = q % TS::TZ, lt = q / TS::TZ;
  Site s;
  s.xh = (x0 >> 1) + lxh;
  s.y = y0 + ly;
  s.z = z0 + lz;
  s.t = t0 + lt;
  s.r = (a.parity + s.y + s.z + s.t) & 1;
  const int idx = s.xh + L.Lxh * (s.y + L.Ly * (s.z + L.Lz * s.t));
  cp_async_wait<0>();
  __syncthreads();
  T acc[24];
  dslash_site_tiled<T, TS, R, DAG>(acc, dslash_smem, a.gauge, L, idx, a.parity, lxh, ly, lz, lt, s, a.ws);
  double local[3] = {0, 0, 0};
  dslash_epilogue<T, EPI>(a, idx, acc, local);
  if (epi_reduces(EPI)) dslash_reduce<TS::NOUT>(local[0], a.partial);
}

template <typename T> static bool tile_fits(const Lat& L) {
  typedef typename TileOf<T>::TS TS;
  return L.Lxh % TS::TXH == 0 && L.Ly % TS::TY == 0 && L.Lz % TS::TZ == 0 && L.Lt % TS::TT == 0;
}
bool lqcd_dslash_tiled(const lqcd_ctx* c) {
  return c->tiled && (c->prec == 4 ? tile_fits<float>(c->lat) : tile_fits<double>(c->lat));
}
// blocks of a launch of dslash_kernel (= per-block partials of the epilogues that reduce; those never run tiled)
int lqcd_dslash_grid(const lqcd_ctx* c) {
  const int block = c->prec == 4 ? DSLASH_BLOCK_F32 : DSLASH_BLOCK_F64;
  return (c->lat.Vh + block - 1) / block;
}

template <typename T, int R, bool DAG>
static void launch_tiled(const DslashArgs<T>& a, int epi, int device, cudaStream_t st) {
  typedef typename TileOf<T>::TS TS;
  const int grid = a.lat.Vh / TS::NOUT;
  const size_t smem = (size_t)TS::NSLOT * 24 * sizeof(T);
  static bool configured[LQCD_MAX_DEVICES] = {};  // per (T, R, DAG) instantiation and device
  if (!configured[device]) {
    cudaFuncSetAttribute(dslash_tiled_kernel<T, R, DAG, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_tiled_kernel<T, R, DAG, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_tiled_kernel<T, R, DAG, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_tiled_kernel<T, R, DAG, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_tiled_kernel<T, R, DAG, 6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    configured[device] = true;
  }
  switch (epi) {
    case 0: dslash_tiled_kernel<T, R, DAG, 0><<<grid, TS::NOUT, smem, st>>>(a); break;
    case 1: dslash_tiled_kernel<T, R, DAG, 1><<<grid, TS::NOUT, smem, st>>>(a); break;
    case 2: dslash_tiled_kernel<T, R, DAG, 2><<<grid, TS::NOUT, smem, st>>>(a); break;
    case 3: dslash_tiled_kernel<T, R, DAG, 3><<<grid, TS::NOUT, smem, st>>>(a); break;
    default: dslash_tiled_kernel<T, R, DAG, 6><<<grid, TS::NOUT, smem, st>>>(a); break;
  }
}

template <typename T, int R, bool DAG>
static void launch_epi(const DslashArgs<T>& a, int epi, int device, cudaStream_t st) {
  const int block = Tune<T, R>::BLOCK;
  const int grid = (a.lat.Vh + block - 1) / block;
  const size_t smem = Tune<T, R>::STAGE ? (size_t)8 * R * sizeof(T) * block : 0;  // eight links per thread
  static bool configured[LQCD_MAX_DEVICES] = {};  // per (T, R, DAG) instantiation and device: the attribute is per device
  if (!configured[device] && smem > 40 * 1024) {  // the epilogues that reduce add static shared memory on top of `smem`
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 5>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 7>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 9>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 10>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 11>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 12>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 13>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_kernel<T, R, DAG, 14>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  configured[device] = true;
  switch (epi) {
    case 0: dslash_kernel<T, R, DAG, 0><<<grid, block, smem, st>>>(a); break;
    case 1: dslash_kernel<T, R, DAG, 1><<<grid, block, smem, st>>>(a); break;
    case 2: dslash_kernel<T, R, DAG, 2><<<grid, block, smem, st>>>(a); break;
    case 3: dslash_kernel<T, R, DAG, 3><<<grid, block, smem, st>>>(a); break;
    case 4: dslash_kernel<T, R, DAG, 4><<<grid, block, smem, st>>>(a); break;
    case 5: dslash_kernel<T, R, DAG, 5><<<grid, block, smem, st>>>(a); break;
    case 6: dslash_kernel<T, R, DAG, 6><<<grid, block, smem, st>>>(a); break;
    case 7: dslash_kernel<T, R, DAG, 7><<<grid, block, smem, st>>>(a); break;
    case 8: dslash_kernel<T, R, DAG, 8><<<grid, block, smem, st>>>(a); break;
    case 9: dslash_kernel<T, R, DAG, 9><<<grid, block, smem, st>>>(a); break;
    case 11: dslash_kernel<T, R, DAG, 11><<<grid, block, smem, st>>>(a); break;
    case 12: dslash_kernel<T, R, DAG, 12><<<grid, block, smem, st>>>(a); break;
    case 13: dslash_kernel<T, R, DAG, 13><<<grid, block, smem, st>>>(a); break;
    case 14: dslash_kernel<T, R, DAG, 14><<<grid, block, smem, st>>>(a); break;
    default: dslash_kernel<T, R, DAG, 10><<<grid, block, smem, st>>>(a); break;
  }
}

template <typename T>
static void launch_typed(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                         int parity, double scale, int dagger, int epi, const DslashFuse* f, cudaStream_t st) {
  DslashArgs<T> a;
  a.r = f ? (T*)f->r : nullptr;
  a.out2 = f ? (T*)f->out2 : nullptr;
  a.partial = c->d_partial;
  a.scalars = c->d_scalars;
  a.num = f ? f->num : 0;
  a.den = f ? f->den : 0;
  a.out = (T*)out;
  a.in = (const T*)in;
  a.gauge = (const T*)gauge;
  a.cl = (const T*)cl;
  a.x = (const T*)x;
  a.lat = c->lat;
  a.parity = parity;
  a.scale = (T)scale;
  a.ws = (T)c->ws;
  if (lqcd_dslash_tiled(c) && (epi <= 3 || epi == 6)) {  // the tiled form exists for the epilogues without a reduction
    if (c->recon == 18) {
      if (dagger) launch_tiled<T, 18, true>(a, epi, c->device, st);
      else launch_tiled<T, 18, false>(a, epi, c->device, st);
    } else {
      if (dagger) launch_tiled<T, 12, true>(a, epi, c->device, st);
      else launch_tiled<T, 12, false>(a, epi, c->device, st);
    }
    return;
  }
  if (c->recon == 18) {
    if (dagger) launch_epi<T, 18, true>(a, epi, c->device, st);
    else launch_epi<T, 18, false>(a, epi, c->device, st);
  } else {
    if (dagger) launch_epi<T, 12, true>(a, epi, c->device, st);
    else launch_epi<T, 12, false>(a, epi, c->device, st);
  }
}

// internal entry used by the C ABI and by the solvers.  cl: one-parity clover block of the output
// parity (or NULL for epi 0); x: one-parity spinor (epi 2,3).  nrhs > 1: `in`, `out`, `x` are nrhs
// consecutive one-parity spinors and the multi-right-hand-side kernel (dslash_mrhs.cu) runs.
int lqcd_dslash_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                       int parity, double scale, int dagger, int epi, int nrhs, cudaStream_t st) {
  if (c->half) {
    if (nrhs > 1) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "16-bit context: one right-hand side only");
    return lqcd_dslash_half_launch(c, out, in, gauge, cl, x, parity, scale, dagger, epi, st);
  }
  if (nrhs > 1) return lqcd_dslash_mrhs_launch(c, out, in, gauge, cl, x, parity, scale, dagger, epi, nrhs, st);
  // algorithmic bytes: every link once, input spinor once, output once (+ clover, + x)
  const double bytes = (double)c->lat.Vh * c->prec *
                       (8.0 * c->recon + 48.0 + (epi >= 1 && epi != 6 ? 72.0 : 0.0) + (epi >= 2 ? 24.0 : 0.0));
  c->alg_bytes += bytes;
  const bool rec = c->prof_on && c->prof_n < c->prof_cap;
  if (rec) cudaEventRecord(c->prof_ev[2 * c->prof_n], st);
  if (c->prec == 4) launch_typed<float>(c, out, in, gauge, cl, x, parity, scale, dagger, epi, nullptr, st);
  else launch_typed<double>(c, out, in, gauge, cl, x, parity, scale, dagger, epi, nullptr, st);
  if (rec) {
    cudaEventRecord(c->prof_ev[2 * c->prof_n + 1], st);
    c->prof_n++;
    c->prof_bytes += bytes;
  }
  LQCD_LAUNCH_CHECK(c, "dslash");
  return LQCD_OK;
}

// CG-fused epilogues (4, 5) are available when the per-block partials fit the context's scratch
bool lqcd_dslash_fuse_ok(const lqcd_ctx* c) {
  return !c->half && (long)lqcd_dslash_grid(c) <= 4L * c->max_red_blocks * LQCD_MAX_RHS;
}
// ... and the epilogues with three sums (11, 12) when three times as many do
bool lqcd_dslash_fuse3_ok(const lqcd_ctx* c) {
  return !c->half && 3L * lqcd_dslash_grid(c) <= 4L * c->max_red_blocks * LQCD_MAX_RHS;
}

int lqcd_partial_sum_launch(lqcd_ctx* c, int n, int slot, cudaStream_t st) {
  partial_sum_kernel<<<1, PSUM_BLOCK, 0, st>>>(c->d_partial, n, c->d_scalars + slot);
  LQCD_LAUNCH_CHECK(c, "partial_sum");
  return LQCD_OK;
}

int lqcd_dslash_fused_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                             int parity, double scale, int dagger, int epi, const DslashFuse* f, cudaStream_t st) {
  if (c->half) return lqcd_dslash_half_launch(c, out, in, gauge, cl, x, parity, scale, dagger, epi, st, f);
  // epi 4: as epi 2; epi 7: as epi 6 (no clover); epi 9: as epi 3 + a second output.  epi 5, 8, 10: no output
  // store, r read and written instead
  // epi 11: as epi 3 ; epi 12: as epi 3 + y read
  const double bytes = (double)c->lat.Vh * c->prec *
                       (8.0 * c->recon + 48.0 + (epi == 7 || epi == 10 ? 0.0 : 72.0) + 24.0 +
                        (epi == 5 || epi == 8 || epi == 9 || epi == 10 || epi == 12 ? 24.0 : 0.0));
  c->alg_bytes += bytes;
  const bool rec = c->prof_on && c->prof_n < c->prof_cap;
  if (rec) cudaEventRecord(c->prof_ev[2 * c->prof_n], st);
  if (c->prec == 4) launch_typed<float>(c, out, in, gauge, cl, x, parity, scale, dagger, epi, f, st);
  else launch_typed<double>(c, out, in, gauge, cl, x, parity, scale, dagger, epi, f, st);
  partial_sum_kernel<<<epi == 11 || epi == 12 ? 3 : 1, PSUM_BLOCK, 0, st>>>(c->d_partial, lqcd_dslash_grid(c), c->d_scalars + f->out_slot);
  c->launches++;
  if (rec) {
    cudaEventRecord(c->prof_ev[2 * c->prof_n + 1], st);
    c->prof_n++;
    c->prof_bytes += bytes;
  }
  LQCD_LAUNCH_CHECK(c, "dslash_fused");
  return LQCD_OK;
}

int lqcd_clover_apply_launch(lqcd_ctx* c, void* out, const void* in, const void* cl_parity, int nrhs, cudaStream_t st) {
  if (c->half) {
    if (nrhs > 1) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "16-bit context: one right-hand side only");
    return lqcd_clover_apply_half_launch(c, out, in, cl_parity, st);
  }
  const int Vh = c->lat.Vh, block = 128;
  const dim3 grid((Vh + block - 1) / block, nrhs);
  c->alg_bytes += (double)Vh * c->prec * (72.0 + 48.0 * nrhs);
  if (c->prec == 4) clover_apply_kernel<float><<<grid, block, 0, st>>>((float*)out, (const float*)in, (const float*)cl_parity, Vh);
  else clover_apply_kernel<double><<<grid, block, 0, st>>>((double*)out, (const double*)in, (const double*)cl_parity, Vh);
  LQCD_LAUNCH_CHECK(c, "clover_apply");
  return LQCD_OK;
}

extern "C" {

int lqcd_dslash(lqcd_ctx* c, void* out, const void* in, const void* gauge, int parity, double scale, int dagger,
                void* stream) {
  if (!c || !out || !in || !gauge || (parity != 0 && parity != 1)) return LQCD_ERR_INVALID_ARG;
  if (out == in) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "dslash: out aliases in");
  if (!lqcd_aligned16(out) || !lqcd_aligned16(in) || !lqcd_aligned16(gauge))
    return lqcd_set_error(c, LQCD_ERR_ALIGN, "dslash: alignment");
  return lqcd_dslash_launch(c, out, in, gauge, nullptr, nullptr, parity, scale, dagger ? 1 : 0, 0, 1, as_stream(stream));
}

int lqcd_clover_apply(lqcd_ctx* c, void* out, const void* in, const void* clover, int parity, void* stream) {
  if (!c || !out || !in || !clover || (parity != 0 && parity != 1)) return LQCD_ERR_INVALID_ARG;
  if (!lqcd_aligned16(out) || !lqcd_aligned16(in) || !lqcd_aligned16(clover))
    return lqcd_set_error(c, LQCD_ERR_ALIGN, "clover_apply: alignment");
  const char* cl = (const char*)clover + (size_t)parity * (lqcd_clover_bytes(c) / 2);
  return lqcd_clover_apply_launch(c, out, in, cl, 1, as_stream(stream));
}

}  // extern "C"
