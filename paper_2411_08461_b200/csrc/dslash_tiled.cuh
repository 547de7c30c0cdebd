// K2, tiled form: the eight-fold neighbour reuse of the hopping term (Eq. 5; SURVEY.md §8(a)
// a6) staged through shared memory.
//
// Why: in the one-thread-per-site kernel (dslash.cu) every neighbour spinor comes from L2 (ncu: each input
// spinor is fetched 6.1 times over the L2->SM crossbar).  All four precision/reconstruction variants and the
// multi-RHS kernel then run at the same 8.5-9.7 TB/s of L2->L1 traffic whatever their DRAM traffic is: the
// crossbar, not HBM, bounds them.  Here a block owns a 4-D tile of output sites, copies the input spinors
// of the tile plus its one-site halo (no corners: the stencil has none) into shared memory ONCE with
// asynchronous 16-byte copies (cp.async.cg, no registers, L1 bypassed), and all eight hops read them from
// shared memory: 2.75-3.25 fetches per spinor instead of 6.1.  Links are read exactly once, straight to
// registers, as before.
//
// Tile = TXH x TY x TZ x TT output sites of parity p (TXH counts checkerboard sites: 2*TXH lattice sites
// in x).  Input slots in shared memory, structure-of-arrays [vector][slot] of 16-byte vectors:
//   interior rows  [TT][TZ][TY][TXH+1] : row (y,z,t) holds the TXH+1 sites of the input parity at
//                                        x = x0 - q + 2j, q = (1-p+y+z+t)&1 (one x-halo site per row)
//   y halo         [2][TT][TZ][TXH], z halo [2][TT][TY][TXH], t halo [2][TZ][TY][TXH]
// An output site (lxh,ly,lz,lt) with x = x0 + 2 lxh + qo finds its -x/+x neighbours at interior entries
// j = lxh, lxh+1 of its own row and its y/z/t neighbours at entry lxh + qo of the neighbouring interior
// row, or at entry lxh of the halo row when the neighbour lies outside the tile.
#pragma once
#include "dslash.cuh"

template <int TXH_, int TY_, int TZ_, int TT_> struct TileShape {
  static constexpr int TXH = TXH_, TY = TY_, TZ = TZ_, TT = TT_;
  static constexpr int NOUT = TXH * TY * TZ * TT;  // threads per block
  static constexpr int NINT = (TXH + 1) * TY * TZ * TT;
  static constexpr int NY = 2 * TXH * TZ * TT, NZ = 2 * TXH * TY * TT, NT = 2 * TXH * TY * TZ;
  static constexpr int OFF_Y = NINT, OFF_Z = OFF_Y + NY, OFF_T = OFF_Z + NZ;
  static constexpr int NSLOT = OFF_T + NT;
};

// global checkerboard index (input parity) of shared-memory slot s of the tile at (x0,y0,z0,t0)
template <typename TS>
__device__ __forceinline__ int tile_slot_site(const Lat& L, int s, int x0, int y0, int z0, int t0, int pin) {
  int x, y, z, t;
  if (s < TS::NINT) {
    const int j = s % (TS::TXH + 1);
    int q = s / (TS::TXH + 1);
    y = y0 + q % TS::TY;
    q /= TS::TY;
    z = z0 + q % TS::TZ;
    t = t0 + q / TS::TZ;
    const int qin = (pin + y + z + t) & 1;
    x = x0 - qin + 2 * j;
    const int Lx = 2 * L.Lxh;
    x = x < 0 ? x + Lx : (x >= Lx ? x - Lx : x);
  } else {
    int lxh, side;
    if (s < TS::OFF_Z) {
      int q = s - TS::OFF_Y;
      lxh = q % TS::TXH;
      q /= TS::TXH;
      z = z0 + q % TS::TZ;
      q /= TS::TZ;
      t = t0 + q % TS::TT;
      side = q / TS::TT;
      y = side ? y0 + TS::TY : y0 - 1;
    } else if (s < TS::OFF_T) {
      int q = s - TS::OFF_Z;
      lxh = q % TS::TXH;
      q /= TS::TXH;
      y = y0 + q % TS::TY;
      q /= TS::TY;
      t = t0 + q % TS::TT;
      side = q / TS::TT;
      z = side ? z0 + TS::TZ : z0 - 1;
    } else {
      int q = s - TS::OFF_T;
      lxh = q % TS::TXH;
      q /= TS::TXH;
      y = y0 + q % TS::TY;
      q /= TS::TY;
      z = z0 + q % TS::TZ;
      side = q / TS::TZ;
      t = side ? t0 + TS::TT : t0 - 1;
    }
    // parity of the row before wrapping (every extent is even, so wrapping keeps it)
    const int qin = (pin + y + z + t) & 1;
    x = x0 + 2 * lxh + qin;
    y = y < 0 ? y + L.Ly : (y >= L.Ly ? y - L.Ly : y);
    z = z < 0 ? z + L.Lz : (z >= L.Lz ? z - L.Lz : z);
    t = t < 0 ? t + L.Lt : (t >= L.Lt ? t - L.Lt : t);
  }
  return (x >> 1) + L.Lxh * (y + L.Ly * (z + L.Lz * t));
}

// asynchronous copy of the tile's input spinors into shared memory [NSV][NSLOT]
template <typename T, typename TS>
__device__ __forceinline__ void tile_stage(void* smem, const T* __restrict__ in, const Lat& L, int x0, int y0, int z0,
                                           int t0, int pin) {
  typedef typename V16<T>::vec vec;
  vec* sm = reinterpret_cast<vec*>(smem);
  const vec* g = reinterpret_cast<const vec*>(in);
  for (int s = threadIdx.x; s < TS::NSLOT; s += TS::NOUT) {
    const int idx = tile_slot_site<TS>(L, s, x0, y0, z0, t0, pin);
#pragma unroll
    for (int v = 0; v < Lay<T>::NSV; v++) cp_async<16>(sm + v * TS::NSLOT + s, g + (size_t)v * L.Vh + idx);
  }
  cp_async_commit();
}

// link through the streaming path (single RHS: read once) or the L1-allocating path (multi-RHS: re-read per column)
template <typename T, int R, bool L1>
__device__ __forceinline__ void load_link_sel(const T* __restrict__ block, int Vh, int idx, T* U) {
  if (!L1) {
    load_link<T, R>(block, Vh, idx, U);
  } else {
    typedef typename GV<T, R>::vec vec;
    constexpr int N = GV<T, R>::N;
    const vec* p = reinterpret_cast<const vec*>(block) + idx;
#pragma unroll
    for (int v = 0; v < R / N; v++) {
      vec q = ld_cached(p + (size_t)v * Vh);
      vec_get(q, U + v * N);
    }
    if (R == 12) recon_row2<T>(U);
  }
}

template <typename T, typename TS, int R, int MU, bool FWD, bool DAG, bool L1LINKS>
__device__ __forceinline__ void hop_tiled(T* acc, const void* smem, int slot, const T* __restrict__ links, int Vh,
                                          int lidx, T w) {
  typedef typename V16<T>::vec vec;
  constexpr int S = (FWD != DAG) ? -1 : +1;
  T psi[24], U[18], h[12], chi[12];
  load_link_sel<T, R, L1LINKS>(links, Vh, lidx, U);
  const vec* sm = reinterpret_cast<const vec*>(smem) + slot;
#pragma unroll
  for (int v = 0; v < Lay<T>::NSV; v++) {
    vec q = sm[v * TS::NSLOT];
    vec_get(q, psi + v * V16<T>::N);
  }
  project<T, MU, S>(psi, h);
  su3_mul<T, !FWD>(U, h, chi);
  reconstruct<T, MU, S>(acc, chi, w);
}

// all eight hops of the output site (lxh,ly,lz,lt) of the tile; idx = its global checkerboard index
template <typename T, typename TS, int R, bool DAG, bool L1LINKS = false>
__device__ __forceinline__ void dslash_site_tiled(T* acc, const void* smem, const T* __restrict__ gauge, const Lat& L,
                                                  int idx, int par, int lxh, int ly, int lz, int lt, const Site& s, T ws) {
  const int Vh = L.Vh;
  const size_t blk = (size_t)R * Vh;
  constexpr int W = TS::TXH + 1;
  const int row = (lt * TS::TZ + lz) * TS::TY + ly;  // interior row of this site
  const int jq = lxh + s.r;                          // entry of the same x in a neighbouring interior row
#pragma unroll
  for (int e = 0; e < 24; e++) acc[e] = 0;
  const T sf = (L.tb < 0 && s.t == L.Lt - 1) ? (T)-1 : (T)1;
  const T sb = (L.tb < 0 && s.t == 0) ? (T)-1 : (T)1;
  int n, slot;
  // x
  slot = row * W + lxh + 1;
  hop_tiled<T, TS, R, 0, true, DAG, L1LINKS>(acc, smem, slot, gauge + (0 * 2 + par) * blk, Vh, idx, ws);
  n = neighbour<0, -1>(L, idx, s);
  slot = row * W + lxh;
  hop_tiled<T, TS, R, 0, false, DAG, L1LINKS>(acc, smem, slot, gauge + (0 * 2 + 1 - par) * blk, Vh, n, ws);
  // y
  slot = ly + 1 < TS::TY ? (row + 1) * W + jq : TS::OFF_Y + ((1 * TS::TT + lt) * TS::TZ + lz) * TS::TXH + lxh;
  hop_tiled<T, TS, R, 1, true, DAG, L1LINKS>(acc, smem, slot, gauge + (1 * 2 + par) * blk, Vh, idx, ws);
  n = neighbour<1, -1>(L, idx, s);
  slot = ly > 0 ? (row - 1) * W + jq : TS::OFF_Y + ((0 * TS::TT + lt) * TS::TZ + lz) * TS::TXH + lxh;
  hop_tiled<T, TS, R, 1, false, DAG, L1LINKS>(acc, smem, slot, gauge + (1 * 2 + 1 - par) * blk, Vh, n, ws);
  // z
  slot = lz + 1 < TS::TZ ? (row + TS::TY) * W + jq : TS::OFF_Z + ((1 * TS::TT + lt) * TS::TY + ly) * TS::TXH + lxh;
  hop_tiled<T, TS, R, 2, true, DAG, L1LINKS>(acc, smem, slot, gauge + (2 * 2 + par) * blk, Vh, idx, ws);
  n = neighbour<2, -1>(L, idx, s);
  slot = lz > 0 ? (row - TS::TY) * W + jq : TS::OFF_Z + ((0 * TS::TT + lt) * TS::TY + ly) * TS::TXH + lxh;
  hop_tiled<T, TS, R, 2, false, DAG, L1LINKS>(acc, smem, slot, gauge + (2 * 2 + 1 - par) * blk, Vh, n, ws);
  // t
  slot = lt + 1 < TS::TT ? (row + TS::TY * TS::TZ) * W + jq : TS::OFF_T + ((1 * TS::TZ + lz) * TS::TY + ly) * TS::TXH + lxh;
  hop_tiled<T, TS, R, 3, true, DAG, L1LINKS>(acc, smem, slot, gauge + (3 * 2 + par) * blk, Vh, idx, sf);
  n = neighbour<3, -1>(L, idx, s);
  slot = lt > 0 ? (row - TS::TY * TS::TZ) * W + jq : TS::OFF_T + ((0 * TS::TZ + lz) * TS::TY + ly) * TS::TXH + lxh;
  hop_tiled<T, TS, R, 3, false, DAG, L1LINKS>(acc, smem, slot, gauge + (3 * 2 + 1 - par) * blk, Vh, n, sb);
}
