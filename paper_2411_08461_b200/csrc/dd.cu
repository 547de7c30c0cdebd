// 4-D domain decomposition of the hopping term ("the lattice are
// divided equally ... 4D Cartesian grid ... rank varies fastest in the t direction").  Every rank holds one
// sub-lattice (its own context, links and spinors).  In a partitioned direction mu the hops that leave the
// sub-lattice are taken out of the kernel and served by faces of projected HALF spinors (12 reals per site instead of
// 24, DeGrand-Rossi projectors of dslash.cuh):
//   forward ghost (dir = +1):  the receiver needs (1 -+ g_mu) U_mu(x) psi(x + mu) at its upper edge; the +mu neighbour
//       packs h = P psi of its FIRST slice; the receiver multiplies by its own link U_mu(x) and reconstructs;
//   backward ghost (dir = -1): the receiver needs (1 +- g_mu) U_mu^dag(x - mu) psi(x - mu) at its lower edge; the link
//       lives on the -mu neighbour, which packs chi = U_mu^dag(y) P psi(y) of its LAST slice; the receiver reconstructs.
// lqcd_dslash_dd_interior computes every hop that stays inside (the others get weight 0), lqcd_face_pack /
// lqcd_face_unpack are the two halves of the exchange; moving the buffers is the caller's business (device copies on
// one GPU, send / recv between ranks: paper_2411_08461_b200/dd.py).  Plain scale * D only (no fused epilogue): the
// clover factors of M-hat are applied by lqcd_clover_apply in the decomposed path.
//
// Face order (the same on both sides of a cut, which is all that matters): for mu = y, z, t the face sites of a parity
// in checkerboard order with the mu coordinate removed, f = xh + Lxh * (rest); for mu = x one site per (y, z, t) row
// whose x = 0 (or Lx - 1) site has that parity, f = index of the row among those rows in (y, z, t) order.
// Buffer layout: [12 reals][nface] (structure of arrays, the context's real type).
#include "dslash.cuh"

namespace {

template <typename T> struct DdArgs {
  T* out;
  const T* in;
  const T* gauge;
  Lat lat;
  int parity, mask;  // mask bit mu: direction mu is partitioned
  T scale, ws;
};

template <typename T, int R, bool DAG>
__global__ void __launch_bounds__(128) dslash_dd_interior_kernel(const DdArgs<T> a) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const Lat& L = a.lat;
  const int Vh = L.Vh, par = a.parity;
  if (idx >= Vh) return;
  const Site s = site_of(L, idx, par);
  const size_t blk = (size_t)R * Vh;
  const int x = 2 * s.xh + s.r, Lx = 2 * L.Lxh;
  // weight of each hop: 0 if it leaves a partitioned direction; else nu/xi_0 (space) or the boundary sign (time)
  const T z = (T)0;
  const T wxf = ((a.mask & 1) && x == Lx - 1) ? z : a.ws, wxb = ((a.mask & 1) && x == 0) ? z : a.ws;
  const T wyf = ((a.mask & 2) && s.y == L.Ly - 1) ? z : a.ws, wyb = ((a.mask & 2) && s.y == 0) ? z : a.ws;
  const T wzf = ((a.mask & 4) && s.z == L.Lz - 1) ? z : a.ws, wzb = ((a.mask & 4) && s.z == 0) ? z : a.ws;
  const T sf = (L.tb < 0 && s.t == L.Lt - 1) ? (T)-1 : (T)1, sb = (L.tb < 0 && s.t == 0) ? (T)-1 : (T)1;
  const T wtf = ((a.mask & 8) && s.t == L.Lt - 1) ? z : sf, wtb = ((a.mask & 8) && s.t == 0) ? z : sb;
  T acc[24];
#pragma unroll
  for (int e = 0; e < 24; e++) acc[e] = 0;
  int n;
  n = neighbour<0, +1>(L, idx, s);
  hop<T, R, 0, true, DAG>(acc, a.in, a.gauge + (0 * 2 + par) * blk, Vh, n, idx, wxf);
  n = neighbour<0, -1>(L, idx, s);
  hop<T, R, 0, false, DAG>(acc, a.in, a.gauge + (0 * 2 + 1 - par) * blk, Vh, n, n, wxb);
  n = neighbour<1, +1>(L, idx, s);
  hop<T, R, 1, true, DAG>(acc, a.in, a.gauge + (1 * 2 + par) * blk, Vh, n, idx, wyf);
  n = neighbour<1, -1>(L, idx, s);
  hop<T, R, 1, false, DAG>(acc, a.in, a.gauge + (1 * 2 + 1 - par) * blk, Vh, n, n, wyb);
  n = neighbour<2, +1>(L, idx, s);
  hop<T, R, 2, true, DAG>(acc, a.in, a.gauge + (2 * 2 + par) * blk, Vh, n, idx, wzf);
  n = neighbour<2, -1>(L, idx, s);
  hop<T, R, 2, false, DAG>(acc, a.in, a.gauge + (2 * 2 + 1 - par) * blk, Vh, n, n, wzb);
  n = neighbour<3, +1>(L, idx, s);
  hop<T, R, 3, true, DAG>(acc, a.in, a.gauge + (3 * 2 + par) * blk, Vh, n, idx, wtf);
  n = neighbour<3, -1>(L, idx, s);
  hop<T, R, 3, false, DAG>(acc, a.in, a.gauge + (3 * 2 + 1 - par) * blk, Vh, n, n, wtb);
#pragma unroll
  for (int e = 0; e < 24; e++) acc[e] *= a.scale;
  store_spinor<T>(a.out, Vh, idx, acc);
}

// checkerboard index (parity `par`) of face site f of the slice coord_mu = c
template <int MU>
__device__ __forceinline__ int face_site(const Lat& L, int f, int c, int par) {
  if (MU == 0) {
    // rows (y, z, t) in order; the row's site at x = c has parity par iff (c + y + z + t) & 1 == par: every second y
    const int hy = L.Ly >> 1;
    const int yh = f % hy;
    int q = f / hy;
    const int z = q % L.Lz, t = q / L.Lz;
    const int y = 2 * yh + ((par + c + z + t) & 1);
    return (c >> 1) + L.Lxh * (y + L.Ly * (z + L.Lz * t));
  } else if (MU == 1) {
    const int xh = f % L.Lxh;
    int q = f / L.Lxh;
    const int z = q % L.Lz, t = q / L.Lz;
    return xh + L.Lxh * (c + L.Ly * (z + L.Lz * t));
  } else if (MU == 2) {
    const int xh = f % L.Lxh;
    int q = f / L.Lxh;
    const int y = q % L.Ly, t = q / L.Ly;
    return xh + L.Lxh * (y + L.Ly * (c + L.Lz * t));
  } else {
    const int xh = f % L.Lxh;
    int q = f / L.Lxh;
    const int y = q % L.Ly, z = q / L.Ly;
    return xh + L.Lxh * (y + L.Ly * (z + L.Lz * c));
  }
}
__host__ __device__ inline int face_extent(const Lat& L, int mu) { return mu == 0 ? 2 * L.Lxh : (mu == 1 ? L.Ly : (mu == 2 ? L.Lz : L.Lt)); }
__host__ __device__ inline int face_count(const Lat& L, int mu) { return L.Vh / face_extent(L, mu); }

// sender side.  FWD = true: forward ghost of the receiver = my slice coord 0, h = P psi.  FWD = false: backward ghost =
// my slice coord L-1, chi = U_mu^dag P psi with my link.  `par` = parity of the sites packed (the INPUT parity).
template <typename T, int R, int MU, bool FWD, bool DAG>
__global__ void __launch_bounds__(128) face_pack_kernel(T* __restrict__ buf, const T* __restrict__ in, const T* __restrict__ gauge,
                                                        const Lat L, int par, int nface) {
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= nface) return;
  constexpr int S = (FWD != DAG) ? -1 : +1;
  const int c = FWD ? 0 : face_extent(L, MU) - 1;
  const int idx = face_site<MU>(L, f, c, par);
  T psi[24], h[12];
  load_spinor<T>(in, L.Vh, idx, psi);
  project<T, MU, S>(psi, h);
  if (!FWD) {
    T U[18], chi[12];
    load_link<T, R>(gauge + (size_t)(MU * 2 + par) * R * L.Vh, L.Vh, idx, U);
    su3_mul<T, true>(U, h, chi);
#pragma unroll
    for (int e = 0; e < 12; e++) h[e] = chi[e];
  }
#pragma unroll
  for (int e = 0; e < 12; e++) buf[(size_t)e * nface + f] = h[e];
}

// receiver side: out(x) += scale * w * (reconstruction of the ghost), x on my upper (FWD) or lower edge, parity `par`
template <typename T, int R, int MU, bool FWD, bool DAG>
__global__ void __launch_bounds__(128) face_unpack_kernel(T* __restrict__ out, const T* __restrict__ buf, const T* __restrict__ gauge,
                                                          const Lat L, int par, int nface, T scale, T w) {
  const int f = blockIdx.x * blockDim.x + threadIdx.x;
  if (f >= nface) return;
  constexpr int S = (FWD != DAG) ? -1 : +1;
  const int c = FWD ? face_extent(L, MU) - 1 : 0;
  const int idx = face_site<MU>(L, f, c, par);
  T h[12], chi[12], acc[24], o[24];
#pragma unroll
  for (int e = 0; e < 12; e++) h[e] = buf[(size_t)e * nface + f];
  if (FWD) {
    T U[18];
    load_link<T, R>(gauge + (size_t)(MU * 2 + par) * R * L.Vh, L.Vh, idx, U);
    su3_mul<T, false>(U, h, chi);
  } else {
#pragma unroll
    for (int e = 0; e < 12; e++) chi[e] = h[e];
  }
#pragma unroll
  for (int e = 0; e < 24; e++) acc[e] = 0;
  reconstruct<T, MU, S>(acc, chi, w);
  typedef typename V16<T>::vec vec;
  vec* p = reinterpret_cast<vec*>(out) + idx;
#pragma unroll
  for (int v = 0; v < Lay<T>::NSV; v++) {
    vec q = p[(size_t)v * L.Vh];
    vec_get(q, o + v * V16<T>::N);
  }
#pragma unroll
  for (int e = 0; e < 24; e++) o[e] += scale * acc[e];
  store_spinor<T>(out, L.Vh, idx, o);
}

template <typename T, int R, int MU, bool DAG>
void pack_dir(lqcd_ctx* c, void* buf, const void* in, const void* gauge, int dir, int par, int nface, cudaStream_t st) {
  const int grid = (nface + 127) / 128;
  if (dir > 0) face_pack_kernel<T, R, MU, true, DAG><<<grid, 128, 0, st>>>((T*)buf, (const T*)in, (const T*)gauge, c->lat, par, nface);
  else face_pack_kernel<T, R, MU, false, DAG><<<grid, 128, 0, st>>>((T*)buf, (const T*)in, (const T*)gauge, c->lat, par, nface);
}
template <typename T, int R, int MU, bool DAG>
void unpack_dir(lqcd_ctx* c, void* out, const void* buf, const void* gauge, int dir, int par, int nface, double scale, double w,
                cudaStream_t st) {
  const int grid = (nface + 127) / 128;
  if (dir > 0) face_unpack_kernel<T, R, MU, true, DAG><<<grid, 128, 0, st>>>((T*)out, (const T*)buf, (const T*)gauge, c->lat, par, nface, (T)scale, (T)w);
  else face_unpack_kernel<T, R, MU, false, DAG><<<grid, 128, 0, st>>>((T*)out, (const T*)buf, (const T*)gauge, c->lat, par, nface, (T)scale, (T)w);
}
template <typename T, int R, bool DAG>
void pack_mu(lqcd_ctx* c, void* buf, const void* in, const void* gauge, int mu, int dir, int par, int nface, cudaStream_t st) {
  switch (mu) {
    case 0: pack_dir<T, R, 0, DAG>(c, buf, in, gauge, dir, par, nface, st); break;
    case 1: pack_dir<T, R, 1, DAG>(c, buf, in, gauge, dir, par, nface, st); break;
    case 2: pack_dir<T, R, 2, DAG>(c, buf, in, gauge, dir, par, nface, st); break;
    default: pack_dir<T, R, 3, DAG>(c, buf, in, gauge, dir, par, nface, st); break;
  }
}
template <typename T, int R, bool DAG>
void unpack_mu(lqcd_ctx* c, void* out, const void* buf, const void* gauge, int mu, int dir, int par, int nface, double scale,
               double w, cudaStream_t st) {
  switch (mu) {
    case 0: unpack_dir<T, R, 0, DAG>(c, out, buf, gauge, dir, par, nface, scale, w, st); break;
    case 1: unpack_dir<T, R, 1, DAG>(c, out, buf, gauge, dir, par, nface, scale, w, st); break;
    case 2: unpack_dir<T, R, 2, DAG>(c, out, buf, gauge, dir, par, nface, scale, w, st); break;
    default: unpack_dir<T, R, 3, DAG>(c, out, buf, gauge, dir, par, nface, scale, w, st); break;
  }
}

bool dd_ok(lqcd_ctx* c, int mu, int dir) { return c && !c->half && mu >= 0 && mu < 4 && (dir == 1 || dir == -1); }

}  // namespace

#define DD_DISPATCH(CALL)                                   \
  do {                                                      \
    if (c->prec == 4) {                                     \
      if (c->recon == 18) {                                 \
        if (dagger) CALL(float, 18, true);                  \
        else CALL(float, 18, false);                        \
      } else {                                              \
        if (dagger) CALL(float, 12, true);                  \
        else CALL(float, 12, false);                        \
      }                                                     \
    } else {                                                \
      if (c->recon == 18) {                                 \
        if (dagger) CALL(double, 18, true);                 \
        else CALL(double, 18, false);                       \
      } else {                                              \
        if (dagger) CALL(double, 12, true);                 \
        else CALL(double, 12, false);                       \
      }                                                     \
    }                                                       \
  } while (0)

extern "C" {

int lqcd_set_partition(lqcd_ctx* c, const int partitioned[4]) {
  if (!c || !partitioned) return LQCD_ERR_INVALID_ARG;
  c->part_mask = 0;
  for (int mu = 0; mu < 4; mu++)
    if (partitioned[mu]) c->part_mask |= 1 << mu;
  return LQCD_OK;
}

size_t lqcd_face_bytes(const lqcd_ctx* c, int mu) {
  if (!c || mu < 0 || mu > 3) return 0;
  return (size_t)face_count(c->lat, mu) * 12 * c->prec;
}

int lqcd_dslash_dd_interior(lqcd_ctx* c, void* out, const void* in, const void* gauge, int parity, double scale, int dagger,
                            void* stream) {
  if (!c || !out || !in || !gauge || (parity != 0 && parity != 1) || c->half) return LQCD_ERR_INVALID_ARG;
  if (out == in) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "dslash_dd_interior: out aliases in");
  if (!lqcd_aligned16(out) || !lqcd_aligned16(in) || !lqcd_aligned16(gauge)) return lqcd_set_error(c, LQCD_ERR_ALIGN, "dslash_dd_interior: alignment");
  cudaStream_t st = as_stream(stream);
  const int grid = (c->lat.Vh + 127) / 128;
#define CALL(T, R, DAG)                                                                     \
  do {                                                                                      \
    DdArgs<T> a;                                                                            \
    a.out = (T*)out; a.in = (const T*)in; a.gauge = (const T*)gauge; a.lat = c->lat;        \
    a.parity = parity; a.mask = c->part_mask; a.scale = (T)scale; a.ws = (T)c->ws;          \
    dslash_dd_interior_kernel<T, R, DAG><<<grid, 128, 0, st>>>(a);                          \
  } while (0)
  DD_DISPATCH(CALL);
#undef CALL
  c->alg_bytes += (double)c->lat.Vh * c->prec * (8.0 * c->recon + 48.0);
  LQCD_LAUNCH_CHECK(c, "dslash_dd_interior");
  return LQCD_OK;
}

int lqcd_face_pack(lqcd_ctx* c, void* buf, const void* in, const void* gauge, int mu, int dir, int parity_in, int dagger,
                   void* stream) {
  if (!dd_ok(c, mu, dir) || !buf || !in || !gauge || (parity_in != 0 && parity_in != 1)) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  const int nface = face_count(c->lat, mu);
#define CALL(T, R, DAG) pack_mu<T, R, DAG>(c, buf, in, gauge, mu, dir, parity_in, nface, st)
  DD_DISPATCH(CALL);
#undef CALL
  c->alg_bytes += (double)nface * c->prec * (24.0 + 12.0 + (dir < 0 ? c->recon : 0));
  LQCD_LAUNCH_CHECK(c, "face_pack");
  return LQCD_OK;
}

int lqcd_face_unpack(lqcd_ctx* c, void* out, const void* buf, const void* gauge, int mu, int dir, int parity_out, double scale,
                     double weight, int dagger, void* stream) {
  if (!dd_ok(c, mu, dir) || !buf || !out || !gauge || (parity_out != 0 && parity_out != 1)) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  const int nface = face_count(c->lat, mu);
#define CALL(T, R, DAG) unpack_mu<T, R, DAG>(c, out, buf, gauge, mu, dir, parity_out, nface, scale, weight, st)
  DD_DISPATCH(CALL);
#undef CALL
  c->alg_bytes += (double)nface * c->prec * (48.0 + 12.0 + (dir > 0 ? c->recon : 0));
  LQCD_LAUNCH_CHECK(c, "face_unpack");
  return LQCD_OK;
}

}  // extern "C"
