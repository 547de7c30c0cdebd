// Multi-right-hand-side dslash, tiled form: the kernel that lifts the
// bound of dslash_mrhs.cu.  There every neighbour spinor of every column crosses the L2->SM crossbar once per
// hop (768 B per site and column; ncu: 10-11 TB/s of crossbar traffic at 4-5 TB/s of DRAM traffic).  Here a block
// owns a 4-D tile of NOUT output sites (dslash_tiled.cuh) and CS column slots; slot k walks the columns
// k, k+CS, ...: the input spinors of the tile + halo of its NEXT column are copied to shared memory with
// cp.async while the eight hops of the CURRENT column read theirs from shared memory (two buffers per slot,
// one named barrier per slot: the slots never wait for one another).  Crossbar traffic per site and column
// falls to (NSLOT/NOUT) x 96 B = 312 B; the tile's links are re-read per column through L1.
//
// Unlike the single-RHS tiled kernel (slower than one thread per site: copy -> barrier -> compute leaves the
// memory pipe idle), the column loop keeps a copy in flight during every compute phase.
#define DSLASH_FFMA2 1
#include "dslash_tiled.cuh"

template <typename T> struct MrhsTArgs {
  T* out;
  const T* in;
  const T* gauge;
  const T* cl;
  const T* x;
  Lat lat;
  int parity;
  T scale;
  T ws;
  size_t stride;  // reals between consecutive right-hand sides (24 * Vh)
  int nrhs;
};

#ifndef MRHS_TILE_XH
#define MRHS_TILE_XH 4
#define MRHS_TILE_Y 4
#define MRHS_TILE_Z 4
#define MRHS_TILE_T 2
#endif
#ifndef MRHS_TILE_CS
#define MRHS_TILE_CS 2
#endif
typedef TileShape<MRHS_TILE_XH, MRHS_TILE_Y, MRHS_TILE_Z, MRHS_TILE_T> MTS;
constexpr int MCS = MRHS_TILE_CS;
constexpr int MSPT = (MTS::NSLOT + MTS::NOUT - 1) / MTS::NOUT;  // slots staged per thread

__device__ __forceinline__ void slot_barrier(int id, int count) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}

template <typename T, int R, bool DAG, int EPI>
__global__ void __launch_bounds__(MTS::NOUT * MCS, 1) dslash_mrhs_tiled_kernel(const MrhsTArgs<T> a) {
  typedef MTS TS;
  typedef typename V16<T>::vec vec;
  constexpr int NSV = Lay<T>::NSV;
  extern __shared__ __align__(16) unsigned char mt_smem[];
  const Lat& L = a.lat;
  const int Vh = L.Vh, par = a.parity, cs = threadIdx.y;
  const int ntx = L.Lxh / TS::TXH, nty = L.Ly / TS::TY, ntz = L.Lz / TS::TZ;
  int b = blockIdx.x;
  const int x0 = 2 * TS::TXH * (b % ntx);
  b /= ntx;
  const int y0 = TS::TY * (b % nty);
  b /= nty;
  const int z0 = TS::TZ * (b % ntz);
  const int t0 = TS::TT * (b / ntz);
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
  s.r = (par + s.y + s.z + s.t) & 1;
  const int idx = s.xh + L.Lxh * (s.y + L.Ly * (s.z + L.Lz * s.t));
  // the shared-memory slots this thread fills are the same for every column
  int gsite[MSPT];
#pragma unroll
  for (int k = 0; k < MSPT; k++) {
    const int sl = threadIdx.x + k * TS::NOUT;
    gsite[k] = sl < TS::NSLOT ? tile_slot_site<TS>(L, sl, x0, y0, z0, t0, 1 - par) : -1;
  }
  vec* buf = reinterpret_cast<vec*>(mt_smem) + (size_t)cs * 2 * NSV * TS::NSLOT;  // this slot's two buffers
  auto stage = [&](int col, int bi) {
    const vec* g = reinterpret_cast<const vec*>(a.in + (size_t)col * a.stride);
    vec* d = buf + (size_t)bi * NSV * TS::NSLOT;
#pragma unroll
    for (int k = 0; k < MSPT; k++) {
      if (gsite[k] < 0) continue;
#pragma unroll
      for (int v = 0; v < NSV; v++) cp_async<16>(d + v * TS::NSLOT + threadIdx.x + k * TS::NOUT, g + (size_t)v * Vh + gsite[k]);
    }
  };
  int bi = 0;
  if (cs < a.nrhs) stage(cs, 0);
  cp_async_commit();
  for (int col = cs; col < a.nrhs; col += MCS) {
    if (col + MCS < a.nrhs) stage(col + MCS, bi ^ 1);
    cp_async_commit();
    cp_async_wait<1>();              // this thread's copies of column `col` have landed
    slot_barrier(1 + cs, TS::NOUT);  // ... and everybody else's in this slot
    T acc[24];
    dslash_site_tiled<T, TS, R, DAG, true>(acc, buf + (size_t)bi * NSV * TS::NSLOT, a.gauge, L, idx, par, lxh, ly, lz, lt, s, a.ws);
    const size_t first = (size_t)col * a.stride;
    T res[24];
    if (EPI == 0) {
#pragma unroll
      for (int e = 0; e < 24; e++) res[e] = a.scale * acc[e];
    } else if (EPI == 1) {
      clover_mul<T>(a.cl, Vh, idx, acc, res);
#pragma unroll
      for (int e = 0; e < 24; e++) res[e] *= a.scale;
    } else if (EPI == 2) {
      T xv[24];
      load_spinor<T>(a.x + first, Vh, idx, xv);
      clover_mul<T>(a.cl, Vh, idx, xv, res);
#pragma unroll
      for (int e = 0; e < 24; e++) res[e] += a.scale * acc[e];
    } else {
      T xv[24];
      load_spinor<T>(a.x + first, Vh, idx, xv);
      clover_mul<T>(a.cl, Vh, idx, acc, res);
#pragma unroll
      for (int e = 0; e < 24; e++) res[e] = xv[e] + a.scale * res[e];
    }
    store_spinor<T>(a.out + first, Vh, idx, res);
    slot_barrier(1 + cs, TS::NOUT);  // buffer bi is free again: the next iteration copies into it
    bi ^= 1;
  }
}

template <typename T, int R, bool DAG>
static void launch_mt(const MrhsTArgs<T>& a, int epi, cudaStream_t st) {
  const dim3 block(MTS::NOUT, MCS);
  const int grid = a.lat.Vh / MTS::NOUT;
  const size_t smem = (size_t)MCS * 2 * MTS::NSLOT * 24 * sizeof(T);
  static bool configured = false;  // one flag per (T, R, DAG) instantiation
  if (!configured) {
    cudaFuncSetAttribute(dslash_mrhs_tiled_kernel<T, R, DAG, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_tiled_kernel<T, R, DAG, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_tiled_kernel<T, R, DAG, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_tiled_kernel<T, R, DAG, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    configured = true;
  }
  switch (epi) {
    case 0: dslash_mrhs_tiled_kernel<T, R, DAG, 0><<<grid, block, smem, st>>>(a); break;
    case 1: dslash_mrhs_tiled_kernel<T, R, DAG, 1><<<grid, block, smem, st>>>(a); break;
    case 2: dslash_mrhs_tiled_kernel<T, R, DAG, 2><<<grid, block, smem, st>>>(a); break;
    default: dslash_mrhs_tiled_kernel<T, R, DAG, 3><<<grid, block, smem, st>>>(a); break;
  }
}

// fp32 only (two buffers per slot of an fp64 tile do not fit beside a useful number of warps); the tile must
// divide the lattice
bool lqcd_mrhs_tiled_ok(const lqcd_ctx* c) {
  const Lat& L = c->lat;
  return c->mrhs_tiled && c->prec == 4 && L.Lxh % MTS::TXH == 0 && L.Ly % MTS::TY == 0 && L.Lz % MTS::TZ == 0 &&
         L.Lt % MTS::TT == 0;
}

void lqcd_dslash_mrhs_tiled_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                                   int parity, double scale, int dagger, int epi, int nrhs, cudaStream_t st) {
  MrhsTArgs<float> a;
  a.out = (float*)out;
  a.in = (const float*)in;
  a.gauge = (const float*)gauge;
  a.cl = (const float*)cl;
  a.x = (const float*)x;
  a.lat = c->lat;
  a.parity = parity;
  a.scale = (float)scale;
  a.ws = (float)c->ws;
  a.stride = (size_t)24 * c->lat.Vh;
  a.nrhs = nrhs;
  if (c->recon == 18) {
    if (dagger) launch_mt<float, 18, true>(a, epi, st);
    else launch_mt<float, 18, false>(a, epi, st);
  } else {
    if (dagger) launch_mt<float, 12, true>(a, epi, st);
    else launch_mt<float, 12, false>(a, epi, st);
  }
}
