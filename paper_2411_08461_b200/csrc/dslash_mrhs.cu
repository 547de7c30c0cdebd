// Multi-right-hand-side dslash (the 12 spin-colour columns of
// a propagator are 12 solves with the same links and clover).  Links are 67-75 % of the compulsory
// bytes of a single-RHS dslash and are identical for every column, so this kernel loads each link
// ONCE per site for NRHS spinors: bytes per site and column fall from (8R+48)w to (8R/NRHS+48)w.
//
// Field layout: NRHS consecutive one-parity native spinors, [rhs][NSV][Vh] vec16.
// Thread layout: blockDim = (SITES, G).  threadIdx.x = site of the block (a warp = 32 consecutive
// sites: coalesced 512 B rows), threadIdx.y = group of NB columns kept in registers (NB x 24
// accumulators), NRHS = G * NB.  The eight links and the clover rows of the block's sites are copied to
// shared memory ONCE per block (streaming loads, the column groups share the copying) and every column
// of every group reads them from there: re-reading them per column through L1 put up to (8R+72)w bytes
// per site and column on the L2->SM crossbar, which is what bounds this kernel (12 columns at 32^3x64, fp32
// 18-real links: 1037 -> 850 us, M-hat 2884 -> 2130 us).  Epilogues are those of dslash.cu.
// Packed FFMA2 arithmetic (lqcd_internal.cuh) is off in this file: measured at 32^3x64, 12 columns, it changes nothing
// for 12-real links (1015 vs 1008 us) and the paired registers push the 18-real kernel into spills (round 1).
#define DSLASH_FFMA2 0
#include "dslash.cuh"

#ifndef MRHS_NB_F32
#define MRHS_NB_F32 1
#endif
#ifndef MRHS_NB_F64
#define MRHS_NB_F64 1
#endif
#ifndef MRHS_SITES
#define MRHS_SITES 32
#endif
#ifndef MRHS_MINB_F32
#define MRHS_MINB_F32 5
#endif
#ifndef MRHS_MINB_F64
#define MRHS_MINB_F64 3
#endif
#ifndef MRHS_GMAX
#define MRHS_GMAX 4                                  // column groups resident in one block
#endif
constexpr int MRHS_MAXT = MRHS_SITES * MRHS_GMAX;    // threads per block (register allocation bound)

template <typename T> struct MrhsArgs {
  T* out;
  const T* in;
  const T* gauge;
  const T* cl;
  const T* x;
  Lat lat;
  int parity;
  T scale;
  T ws;           // weight of the spatial hops (anisotropy nu/xi_0)
  size_t stride;  // reals between consecutive right-hand sides (24 * Vh)
  int ngroups;    // nrhs / NB column groups; group g is handled by threadIdx.y = g mod blockDim.y
  // epilogues 9 and 10 (CG recurrences fused per column, as in dslash.cu)
  T* r;             // epi 10: residual block, r -= (s[num]/s[den]) q, per column
  T* out2;          // epi 9: second output, C * out
  double* partial;  // [sum k][column][block]: one partial per warp (= 32 sites of one column), k < 3
  const double* scalars;
  int num, den, nblocks;
  int zslab;  // z-planes per slab of the sweep (0: plain order)
};
__host__ __device__ constexpr bool mrhs_clover(int epi) { return epi == 1 || epi == 2 || epi == 3 || epi == 9 || epi == 11 || epi == 12 || epi == 13 || epi == 14; }
// Block order of the sweep: 32-site blocks run x, y, then z inside a slab of `zslab` planes, then t, then the slab, so
// that the +-t reuse window of all columns (2 x slab x nrhs columns) stays in L2 (round 1: 1.5 x the algorithmic DRAM
// bytes with 12 columns in plain checkerboard order).  zslab = 0, or a plane that is not a whole number of blocks: identity.
__device__ __forceinline__ int sweep_block(const Lat& L, int b, int zslab) {
  const int plane = L.Lxh * L.Ly;
  if (zslab <= 0 || zslab >= L.Lz || plane % MRHS_SITES || L.Lz % zslab) return b;
  const int pb = plane / MRHS_SITES;
  const int xy = b % pb;
  int q = b / pb;
  const int zl = q % zslab;
  q /= zslab;
  const int t = q % L.Lt, slab = q / L.Lt;
  return xy + pb * ((slab * zslab + zl) + L.Lz * t);
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}

template <typename T, int R, int MU, bool FWD, bool DAG, int NB>
__device__ __forceinline__ void hop_mrhs(T (*acc)[24], const T* __restrict__ in, size_t stride,
                                         const typename GV<T, R>::vec* lk, int Vh, int nidx, T bsign, bool seam) {
  constexpr int S = (FWD != DAG) ? -1 : +1;
  constexpr int GN = GV<T, R>::N;
  T U[18];
  // this site's link of this hop, from the block's shared-memory copy [vector][site] (stage_links_block)
#pragma unroll
  for (int v = 0; v < R / GN; v++) {
    typename GV<T, R>::vec q = lk[v * MRHS_SITES];
    vec_get(q, U + v * GN);
  }
  if (R == 12) recon_row2<T>(U);
  // t: antiperiodic seam; x,y,z: hop weight; folded into the accumulation (reconstruct)
  const T sg = (MU == 3) ? (seam ? (T)-1 : (T)1) : bsign;
#pragma unroll
  for (int r = 0; r < NB; r++) {
    T psi[24], h[12], chi[12];
    load_spinor<T>(in + r * stride, Vh, nidx, psi);
    project<T, MU, S>(psi, h);
    su3_mul<T, !FWD>(U, h, chi);
    reconstruct<T, MU, S>(acc[r], chi, sg);
  }
}

// The clover rows of a block's MRHS_SITES sites, copied to shared memory once per block ([vector][site]): every
// column of every column group multiplies by the same 72 reals per site, and reloading them per column from
// L1/L2 put 288 B x nrhs per site on the L2->SM crossbar (ncu: +3.6 GB per 12-column launch, +250-300 us).
template <typename T>
__device__ __forceinline__ void stage_clover_block(typename V16<T>::vec* sm, const T* __restrict__ cl, int Vh, int site0) {
  typedef typename V16<T>::vec vec;
  const vec* g = reinterpret_cast<const vec*>(cl);
  const int nthr = blockDim.x * blockDim.y, tid = threadIdx.y * blockDim.x + threadIdx.x;
  for (int e = tid; e < Lay<T>::NCV * MRHS_SITES; e += nthr) {
    const int q = e / MRHS_SITES, sl = e % MRHS_SITES;
    if (site0 + sl < Vh) sm[e] = ld_stream(g + (size_t)q * Vh + site0 + sl);
  }
}

// out[r] = C v[r] for NB vectors; C from the block's shared-memory copy (stage_clover_block), site = threadIdx.x
template <typename T, int NB>
__device__ __forceinline__ void clover_mul_mrhs(const typename V16<T>::vec* sm, const T (*v)[24], T (*out)[24]) {
  typedef typename V16<T>::vec vec;
  constexpr int N = V16<T>::N;
  const vec* p = sm + threadIdx.x;
#pragma unroll
  for (int k = 0; k < 2; k++) {
    T a[36];
#pragma unroll
    for (int q = 0; q < 36 / N; q++) {
      vec w = p[(k * (36 / N) + q) * MRHS_SITES];
      vec_get(w, a + q * N);
    }
#pragma unroll
    for (int r = 0; r < NB; r++) {
      const T* x = v[r] + 12 * k;
      T* y = out[r] + 12 * k;
      clover_block<T>(a, x, y);
    }
  }
}

template <typename T> struct MrhsTune;
template <> struct MrhsTune<float> { static constexpr int MINB = MRHS_MINB_F32, NB = MRHS_NB_F32; };
template <> struct MrhsTune<double> { static constexpr int MINB = MRHS_MINB_F64, NB = MRHS_NB_F64; };

template <typename T, int R, bool DAG, int EPI, int NB>
__global__ void __launch_bounds__(MRHS_MAXT, MrhsTune<T>::MINB) dslash_mrhs_kernel(const MrhsArgs<T> a) {
  typedef typename GV<T, R>::vec gvec;
  constexpr int NGV = R / GV<T, R>::N;
  const int blk0 = sweep_block(a.lat, blockIdx.x, a.zslab);  // block of 32 consecutive sites this thread block computes
  const int idx = blk0 * blockDim.x + threadIdx.x;
  __shared__ typename V16<T>::vec cl_sm[mrhs_clover(EPI) ? Lay<T>::NCV * MRHS_SITES : 1];
  extern __shared__ __align__(16) unsigned char mrhs_lk_smem[];  // the eight links of the block's sites: [hop][vector][site]
  gvec* lk_sm = reinterpret_cast<gvec*>(mrhs_lk_smem);
  const Lat& L = a.lat;
  const int Vh = L.Vh, par = a.parity;
  const bool live = idx < Vh;
  const size_t stride = a.stride;
  const Site s = site_of(L, live ? idx : 0, par);
  const size_t blk = (size_t)R * Vh;
  int nb[8];
  {
    const int i0 = live ? idx : 0;
    nb[0] = neighbour<0, +1>(L, i0, s);
    nb[1] = neighbour<0, -1>(L, i0, s);
    nb[2] = neighbour<1, +1>(L, i0, s);
    nb[3] = neighbour<1, -1>(L, i0, s);
    nb[4] = neighbour<2, +1>(L, i0, s);
    nb[5] = neighbour<2, -1>(L, i0, s);
    nb[6] = neighbour<3, +1>(L, i0, s);
    nb[7] = neighbour<3, -1>(L, i0, s);
  }
  // links and clover rows are the same for every column: copied once per block (column group y copies hops y, y+G, ...)
  if (live) {
    for (int h = threadIdx.y; h < 8; h += blockDim.y) {
      const gvec* gp = reinterpret_cast<const gvec*>(a.gauge + ((h >> 1) * 2 + ((h & 1) ? 1 - par : par)) * blk) + ((h & 1) ? nb[h] : idx);
#pragma unroll
      for (int v = 0; v < NGV; v++) lk_sm[(h * NGV + v) * MRHS_SITES + threadIdx.x] = ld_stream(gp + (size_t)v * Vh);
    }
  }
  if (mrhs_clover(EPI)) stage_clover_block<T>(cl_sm, a.cl, Vh, blk0 * blockDim.x);
  __syncthreads();
  if (!live) return;
  for (int g = threadIdx.y; g < a.ngroups; g += blockDim.y) {
  const size_t first = (size_t)g * NB * stride;  // first column of this thread's group
  const T* in = a.in + first;
  T acc[NB][24];
#pragma unroll
  for (int r = 0; r < NB; r++)
#pragma unroll
    for (int e = 0; e < 24; e++) acc[r][e] = 0;
  const T one = a.ws;
  const bool anti = L.tb < 0;
  const bool seam_f = anti && s.t == L.Lt - 1, seam_b = anti && s.t == 0;
  hop_mrhs<T, R, 0, true, DAG, NB>(acc, in, stride, lk_sm + 0 * NGV * MRHS_SITES + threadIdx.x, Vh, nb[0], one, false);
  hop_mrhs<T, R, 0, false, DAG, NB>(acc, in, stride, lk_sm + 1 * NGV * MRHS_SITES + threadIdx.x, Vh, nb[1], one, false);
  hop_mrhs<T, R, 1, true, DAG, NB>(acc, in, stride, lk_sm + 2 * NGV * MRHS_SITES + threadIdx.x, Vh, nb[2], one, false);
  hop_mrhs<T, R, 1, false, DAG, NB>(acc, in, stride, lk_sm + 3 * NGV * MRHS_SITES + threadIdx.x, Vh, nb[3], one, false);
  hop_mrhs<T, R, 2, true, DAG, NB>(acc, in, stride, lk_sm + 4 * NGV * MRHS_SITES + threadIdx.x, Vh, nb[4], one, false);
  hop_mrhs<T, R, 2, false, DAG, NB>(acc, in, stride, lk_sm + 5 * NGV * MRHS_SITES + threadIdx.x, Vh, nb[5], one, false);
  hop_mrhs<T, R, 3, true, DAG, NB>(acc, in, stride, lk_sm + 6 * NGV * MRHS_SITES + threadIdx.x, Vh, nb[6], -one, seam_f);
  hop_mrhs<T, R, 3, false, DAG, NB>(acc, in, stride, lk_sm + 7 * NGV * MRHS_SITES + threadIdx.x, Vh, nb[7], -one, seam_b);

  T* out = a.out + first;
  if (EPI == 0) {
#pragma unroll
    for (int r = 0; r < NB; r++) {
#pragma unroll
      for (int e = 0; e < 24; e++) acc[r][e] *= a.scale;
      store_spinor<T>(out + r * stride, Vh, idx, acc[r]);
    }
  } else if (EPI == 6) {  // out = x + scale * d (dslash.cu epilogue 6: the hop without a clover factor of the symmetric forms)
#pragma unroll
    for (int r = 0; r < NB; r++) {
      T xv[24];
      load_spinor<T>(a.x + first + r * stride, Vh, idx, xv);
#pragma unroll
      for (int e = 0; e < 24; e++) xv[e] += a.scale * acc[r][e];
      store_spinor<T>(out + r * stride, Vh, idx, xv);
    }
  } else if (EPI == 14) {  // out = C (x + scale * d): b-hat of the left-symmetric form, x_o = A_oo^-1 (b_o + kappa D_oe x_e)
    T res[NB][24];
#pragma unroll
    for (int r = 0; r < NB; r++) {
      T xv[24];
      load_spinor<T>(a.x + first + r * stride, Vh, idx, xv);
#pragma unroll
      for (int e = 0; e < 24; e++) acc[r][e] = xv[e] + a.scale * acc[r][e];
    }
    clover_mul_mrhs<T, NB>(cl_sm, acc, res);
#pragma unroll
    for (int r = 0; r < NB; r++) store_spinor<T>(out + r * stride, Vh, idx, res[r]);
  } else if (EPI == 1) {
    T res[NB][24];
    clover_mul_mrhs<T, NB>(cl_sm, acc, res);
#pragma unroll
    for (int r = 0; r < NB; r++) {
#pragma unroll
      for (int e = 0; e < 24; e++) res[r][e] *= a.scale;
      store_spinor<T>(out + r * stride, Vh, idx, res[r]);
    }
  } else if (EPI == 2) {
    T xv[NB][24], res[NB][24];
#pragma unroll
    for (int r = 0; r < NB; r++) load_spinor<T>(a.x + first + r * stride, Vh, idx, xv[r]);
    clover_mul_mrhs<T, NB>(cl_sm, xv, res);
#pragma unroll
    for (int r = 0; r < NB; r++) {
#pragma unroll
      for (int e = 0; e < 24; e++) res[r][e] += a.scale * acc[r][e];
      store_spinor<T>(out + r * stride, Vh, idx, res[r]);
    }
  } else if (EPI == 9) {  // t = x + scale * C d ; ta = C t ; |t|^2 per column (Vh a multiple of 32: full warps)
    T res[NB][24], res2[NB][24];
    clover_mul_mrhs<T, NB>(cl_sm, acc, res);
#pragma unroll
    for (int r = 0; r < NB; r++) {
      T xv[24];
      load_spinor<T>(a.x + first + r * stride, Vh, idx, xv);
#pragma unroll
      for (int e = 0; e < 24; e++) res[r][e] = xv[e] + a.scale * res[r][e];
    }
    clover_mul_mrhs<T, NB>(cl_sm, res, res2);
#pragma unroll
    for (int r = 0; r < NB; r++) {
      double local = 0;
#pragma unroll
      for (int e = 0; e < 24; e++) local += (double)res[r][e] * res[r][e];
      store_spinor<T>(out + r * stride, Vh, idx, res[r]);
      store_spinor<T>(a.out2 + first + r * stride, Vh, idx, res2[r]);
      local = warp_sum(local);
      if (threadIdx.x == 0) a.partial[(size_t)(g * NB + r) * a.nblocks + blockIdx.x] = local;
    }
  } else if (EPI == 11 || EPI == 12) {
    // BiCGStab: out = x + scale * C d (epilogue 3) with the inner products the next step needs, per column:
    //   11: Re<out,x>, Im<out,x>, |out|^2   (t = Mhat s: <t,s>, |t|^2)      12: Re<y,out>, Im<y,out>, |y|^2, y = a.r   (<r0,v>)
    T res[NB][24];
    clover_mul_mrhs<T, NB>(cl_sm, acc, res);
#pragma unroll
    for (int r = 0; r < NB; r++) {
      T xv[24], yv[24];
      load_spinor<T>(a.x + first + r * stride, Vh, idx, xv);
#pragma unroll
      for (int e = 0; e < 24; e++) res[r][e] = xv[e] + a.scale * res[r][e];
      store_spinor<T>(out + r * stride, Vh, idx, res[r]);
      if (EPI == 12) load_spinor<T>(a.r + first + r * stride, Vh, idx, yv);
      double s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
      for (int e = 0; e < 24; e += 2) {
        // <u,w> = sum conj(u) w with (u, w) = (out, x) for 11, (y, out) for 12
        const double ur = EPI == 11 ? res[r][e] : yv[e], ui = EPI == 11 ? res[r][e + 1] : yv[e + 1];
        const double wr = EPI == 11 ? xv[e] : res[r][e], wi = EPI == 11 ? xv[e + 1] : res[r][e + 1];
        s0 += ur * wr + ui * wi;
        s1 += ur * wi - ui * wr;
        s2 += ur * ur + ui * ui;
      }
      s0 = warp_sum(s0);
      s1 = warp_sum(s1);
      s2 = warp_sum(s2);
      if (threadIdx.x == 0) {
        const size_t col = g * NB + r;
        a.partial[(0 * LQCD_MAX_RHS + col) * a.nblocks + blockIdx.x] = s0;
        a.partial[(1 * LQCD_MAX_RHS + col) * a.nblocks + blockIdx.x] = s1;
        a.partial[(2 * LQCD_MAX_RHS + col) * a.nblocks + blockIdx.x] = s2;
      }
    }
  } else if (EPI == 13) {
    // closing step of a solve: |y - (C x + scale * d)|^2 per column with y = a.r, nothing stored (one parity of the true
    // residual b - M x: epilogue 2 whose result goes straight into the norm)
    T xv[NB][24], res[NB][24];
#pragma unroll
    for (int r = 0; r < NB; r++) load_spinor<T>(a.x + first + r * stride, Vh, idx, xv[r]);
    clover_mul_mrhs<T, NB>(cl_sm, xv, res);
#pragma unroll
    for (int r = 0; r < NB; r++) {
      T yv[24];
      load_spinor<T>(a.r + first + r * stride, Vh, idx, yv);
      double local = 0;
#pragma unroll
      for (int e = 0; e < 24; e++) {
        const double dlt = (double)yv[e] - ((double)res[r][e] + (double)a.scale * (double)acc[r][e]);
        local += dlt * dlt;
      }
      local = warp_sum(local);
      if (threadIdx.x == 0) a.partial[(size_t)(g * NB + r) * a.nblocks + blockIdx.x] = local;
    }
  } else if (EPI == 10) {  // q = x + scale * d not stored ; r -= (s[num]/s[den]) q ; |r|^2 per column
#pragma unroll
    for (int r = 0; r < NB; r++) {
      const double* sc = a.scalars + (size_t)(g * NB + r) * SC_STRIDE;
      double local = 0;
      if (sc[S_DONE] == 0.0) {  // a converged column keeps its r
        const T alpha = (T)(sc[a.num] / sc[a.den]);
        T xv[24], rv[24];
        load_spinor<T>(a.x + first + r * stride, Vh, idx, xv);
        load_spinor<T>(a.r + first + r * stride, Vh, idx, rv);
#pragma unroll
        for (int e = 0; e < 24; e++) {
          rv[e] -= alpha * (xv[e] + a.scale * acc[r][e]);
          local += (double)rv[e] * rv[e];
        }
        store_spinor<T>(a.r + first + r * stride, Vh, idx, rv);
      }
      local = warp_sum(local);
      if (threadIdx.x == 0) a.partial[(size_t)(g * NB + r) * a.nblocks + blockIdx.x] = local;
    }
  } else {
    T res[NB][24];
    clover_mul_mrhs<T, NB>(cl_sm, acc, res);
#pragma unroll
    for (int r = 0; r < NB; r++) {
      T xv[24];
      load_spinor<T>(a.x + first + r * stride, Vh, idx, xv);
#pragma unroll
      for (int e = 0; e < 24; e++) res[r][e] = xv[e] + a.scale * res[r][e];
      store_spinor<T>(out + r * stride, Vh, idx, res[r]);
    }
  }
  }  // column groups
}

// sums the per-warp partials of one column in a fixed order -> scalars[column][slot] (deterministic)
__global__ void __launch_bounds__(256) partial_sum_mrhs_kernel(const double* __restrict__ partial, int nblocks, double* scalars, int slot) {
  __shared__ double sm[8];
  const double* p = partial + ((size_t)blockIdx.y * LQCD_MAX_RHS + blockIdx.x) * nblocks;  // blockIdx.y: which of up to 3 sums
  slot += blockIdx.y;
  double v = 0;
  for (int b = threadIdx.x; b < nblocks; b += 256) v += p[b];
  v = warp_sum(v);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0;
    for (int w = 0; w < 8; w++) t += sm[w];
    scalars[(size_t)blockIdx.x * SC_STRIDE + slot] = t;
  }
}

// ---------------------------------------------------------------------------------------------
// Staged form (one column per thread): the neighbour spinors of a thread's (site, column) are copied
// global -> shared memory with per-thread asynchronous 16-byte copies (cp.async.cg), HPR hops per round,
// two rounds of buffers: while round k is multiplied, round k+1 (the next hops, or the first hops of the
// thread's NEXT column) is in flight without holding a register.  The one-thread-per-site kernel above
// is latency bound (ncu: issue slots 43 % busy, DRAM 45 %, 6.5 warps per issue waiting on the long
// scoreboard, and removing 24 % of its instructions changed nothing): here every thread keeps
// HPR * 24 reals in flight at all times.  A thread reads only what it copied itself: cp.async.wait_group
// is the only synchronisation.  Shared memory per thread: 2 * HPR * 24 reals.
// ---------------------------------------------------------------------------------------------
// Measured at 32^3x64, 12 columns (profiles/r01d_tuning.md): fp32 12-real links 1003 -> 886 us with one hop per
// round and 5 blocks/SM; 18-real links and fp64 lose 4-25 % (more shared memory per thread, fewer warps), so the
// staged kernel runs for <float, 12> only.  HPR = hops per round; 0 = off.
#ifndef MRHS_HPR_F32_R12
#define MRHS_HPR_F32_R12 1
#endif
#ifndef MRHS_HPR_F32_R18
#define MRHS_HPR_F32_R18 0
#endif
#ifndef MRHS_HPR_F64
#define MRHS_HPR_F64 0
#endif
#ifndef MRHS_SMINB_F32
#define MRHS_SMINB_F32 5
#endif
#ifndef MRHS_SMINB_F64
#define MRHS_SMINB_F64 3
#endif
template <typename T, int R> struct MrhsStage;
template <> struct MrhsStage<float, 12> { static constexpr int HPR = MRHS_HPR_F32_R12, MINB = MRHS_SMINB_F32; };
template <> struct MrhsStage<float, 18> { static constexpr int HPR = MRHS_HPR_F32_R18, MINB = MRHS_SMINB_F32; };
template <> struct MrhsStage<double, 12> { static constexpr int HPR = MRHS_HPR_F64, MINB = MRHS_SMINB_F64; };
template <> struct MrhsStage<double, 18> { static constexpr int HPR = MRHS_HPR_F64, MINB = MRHS_SMINB_F64; };

template <typename T, int R, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void hop_mrhs_staged(T* acc, const typename V16<T>::vec* sm, const typename GV<T, R>::vec* lk, T w) {
  typedef typename V16<T>::vec vec;
  constexpr int S = (FWD != DAG) ? -1 : +1;
  constexpr int GN = GV<T, R>::N;
  T U[18], psi[24], h[12], chi[12];
  // this site's link of this hop, from the block's shared-memory copy [vector][site]
#pragma unroll
  for (int v = 0; v < R / GN; v++) {
    typename GV<T, R>::vec q = lk[v * MRHS_SITES];
    vec_get(q, U + v * GN);
  }
  if (R == 12) recon_row2<T>(U);
#pragma unroll
  for (int v = 0; v < Lay<T>::NSV; v++) {
    vec q = sm[v * MRHS_MAXT];
    vec_get(q, psi + v * V16<T>::N);
  }
  project<T, MU, S>(psi, h);
  su3_mul<T, !FWD>(U, h, chi);
  reconstruct<T, MU, S>(acc, chi, w);
}

template <typename T, int R, bool DAG, int EPI>
__global__ void __launch_bounds__(MRHS_MAXT, MrhsStage<T, R>::MINB) dslash_mrhs_staged_kernel(const MrhsArgs<T> a) {
  typedef typename V16<T>::vec vec;
  constexpr int HPR = MrhsStage<T, R>::HPR > 0 ? MrhsStage<T, R>::HPR : 1, NR = 8 / HPR, NSV = Lay<T>::NSV;
  extern __shared__ __align__(16) unsigned char mrhs_smem[];
  const int blk0 = sweep_block(a.lat, blockIdx.x, a.zslab);
  const int idx = blk0 * blockDim.x + threadIdx.x;
  typedef typename GV<T, R>::vec gvec;
  constexpr int NGV = R / GV<T, R>::N;
  __shared__ vec cl_sm[mrhs_clover(EPI) ? Lay<T>::NCV * MRHS_SITES : 1];
  __shared__ gvec lk_sm[8 * NGV * MRHS_SITES];  // the eight links of the block's sites: [hop][vector][site]
  const Lat& L = a.lat;
  const int Vh = L.Vh, par = a.parity;
  const bool live = idx < Vh;
  const size_t stride = a.stride;
  const Site s = site_of(L, live ? idx : 0, par);
  const size_t blk = (size_t)R * Vh;
  int n[8];
  {
    const int i0 = live ? idx : 0;
    n[0] = neighbour<0, +1>(L, i0, s);
    n[1] = neighbour<0, -1>(L, i0, s);
    n[2] = neighbour<1, +1>(L, i0, s);
    n[3] = neighbour<1, -1>(L, i0, s);
    n[4] = neighbour<2, +1>(L, i0, s);
    n[5] = neighbour<2, -1>(L, i0, s);
    n[6] = neighbour<3, +1>(L, i0, s);
    n[7] = neighbour<3, -1>(L, i0, s);
  }
  // every column of every column group multiplies by the same eight links per site: copied once per block (the column
  // groups share the work: group y copies hops y, y + G, ...), instead of one L1/L2 read per column
  if (live) {
    for (int h = threadIdx.y; h < 8; h += blockDim.y) {
      const gvec* gp = reinterpret_cast<const gvec*>(a.gauge + ((h >> 1) * 2 + ((h & 1) ? 1 - par : par)) * blk) + ((h & 1) ? n[h] : idx);
#pragma unroll
      for (int v = 0; v < NGV; v++) lk_sm[(h * NGV + v) * MRHS_SITES + threadIdx.x] = ld_stream(gp + (size_t)v * Vh);
    }
  }
  if (mrhs_clover(EPI)) stage_clover_block<T>(cl_sm, a.cl, Vh, blk0 * blockDim.x);
  __syncthreads();
  if (!live) return;
  // shared memory [buffer][hop of the round][vector][thread]
  vec* sm = reinterpret_cast<vec*>(mrhs_smem) + threadIdx.y * MRHS_SITES + threadIdx.x;
  const bool anti = L.tb < 0;
  const T wf = (anti && s.t == L.Lt - 1) ? (T)-1 : (T)1, wb = (anti && s.t == 0) ? (T)-1 : (T)1;
  // copies of round rnd (hops rnd*HPR ...) of column `col` into buffer rnd & 1
  auto issue = [&](const T* __restrict__ col, int rnd) {
#pragma unroll
    for (int k = 0; k < HPR; k++) {
      const vec* g = reinterpret_cast<const vec*>(col) + n[rnd * HPR + k];
      vec* d = sm + (size_t)((rnd & 1) * HPR + k) * NSV * MRHS_MAXT;
#pragma unroll
      for (int v = 0; v < NSV; v++) cp_async<16>(d + v * MRHS_MAXT, g + (size_t)v * Vh);
    }
  };
  int g = threadIdx.y;
  if (g < a.ngroups) issue(a.in + (size_t)g * stride, 0);
  cp_async_commit();
  for (; g < a.ngroups; g += blockDim.y) {
    const size_t first = (size_t)g * stride;
    const T* in = a.in + first;
    const bool more = g + (int)blockDim.y < a.ngroups;
    T acc[1][24];
#pragma unroll
    for (int e = 0; e < 24; e++) acc[0][e] = 0;
#pragma unroll
    for (int rnd = 0; rnd < NR; rnd++) {
      if (rnd + 1 < NR) issue(in, rnd + 1);
      else if (more) issue(in + (size_t)blockDim.y * stride, 0);
      cp_async_commit();
      cp_async_wait<1>();
#pragma unroll
      for (int k = 0; k < HPR; k++) {
        const int H = rnd * HPR + k;
        const vec* b = sm + (size_t)((rnd & 1) * HPR + k) * NSV * MRHS_MAXT;
        switch (H) {
          case 0: hop_mrhs_staged<T, R, 0, true, DAG>(acc[0], b, lk_sm + 0 * NGV * MRHS_SITES + threadIdx.x, a.ws); break;
          case 1: hop_mrhs_staged<T, R, 0, false, DAG>(acc[0], b, lk_sm + 1 * NGV * MRHS_SITES + threadIdx.x, a.ws); break;
          case 2: hop_mrhs_staged<T, R, 1, true, DAG>(acc[0], b, lk_sm + 2 * NGV * MRHS_SITES + threadIdx.x, a.ws); break;
          case 3: hop_mrhs_staged<T, R, 1, false, DAG>(acc[0], b, lk_sm + 3 * NGV * MRHS_SITES + threadIdx.x, a.ws); break;
          case 4: hop_mrhs_staged<T, R, 2, true, DAG>(acc[0], b, lk_sm + 4 * NGV * MRHS_SITES + threadIdx.x, a.ws); break;
          case 5: hop_mrhs_staged<T, R, 2, false, DAG>(acc[0], b, lk_sm + 5 * NGV * MRHS_SITES + threadIdx.x, a.ws); break;
          case 6: hop_mrhs_staged<T, R, 3, true, DAG>(acc[0], b, lk_sm + 6 * NGV * MRHS_SITES + threadIdx.x, wf); break;
          default: hop_mrhs_staged<T, R, 3, false, DAG>(acc[0], b, lk_sm + 7 * NGV * MRHS_SITES + threadIdx.x, wb); break;
        }
      }
    }
    T* out = a.out + first;
    if (EPI == 0) {
#pragma unroll
      for (int e = 0; e < 24; e++) acc[0][e] *= a.scale;
      store_spinor<T>(out, Vh, idx, acc[0]);
    } else if (EPI == 6) {
      T xv[24];
      load_spinor<T>(a.x + first, Vh, idx, xv);
#pragma unroll
      for (int e = 0; e < 24; e++) xv[e] += a.scale * acc[0][e];
      store_spinor<T>(out, Vh, idx, xv);
    } else if (EPI == 1) {
      T res[1][24];
      clover_mul_mrhs<T, 1>(cl_sm, acc, res);
#pragma unroll
      for (int e = 0; e < 24; e++) res[0][e] *= a.scale;
      store_spinor<T>(out, Vh, idx, res[0]);
    } else if (EPI == 2) {
      T xv[1][24], res[1][24];
      load_spinor<T>(a.x + first, Vh, idx, xv[0]);
      clover_mul_mrhs<T, 1>(cl_sm, xv, res);
#pragma unroll
      for (int e = 0; e < 24; e++) res[0][e] += a.scale * acc[0][e];
      store_spinor<T>(out, Vh, idx, res[0]);
    } else {
      T res[1][24], xv[24];
      clover_mul_mrhs<T, 1>(cl_sm, acc, res);
      load_spinor<T>(a.x + first, Vh, idx, xv);
#pragma unroll
      for (int e = 0; e < 24; e++) res[0][e] = xv[e] + a.scale * res[0][e];
      store_spinor<T>(out, Vh, idx, res[0]);
    }
  }
}

template <typename T, int R, bool DAG>
static void launch_mrhs_staged(MrhsArgs<T> a, int epi, int nrhs, cudaStream_t st) {
  a.ngroups = nrhs;
  const dim3 block(MRHS_SITES, a.ngroups < MRHS_GMAX ? a.ngroups : MRHS_GMAX);
  const int grid = (a.lat.Vh + MRHS_SITES - 1) / MRHS_SITES;
  const size_t smem = (size_t)2 * MrhsStage<T, R>::HPR * 24 * sizeof(T) * MRHS_MAXT;
  static bool configured = false;  // one flag per (T, R, DAG) instantiation
  if (!configured && smem > 40 * 1024) {
    cudaFuncSetAttribute(dslash_mrhs_staged_kernel<T, R, DAG, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_staged_kernel<T, R, DAG, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_staged_kernel<T, R, DAG, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_staged_kernel<T, R, DAG, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_staged_kernel<T, R, DAG, 6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  configured = true;
  switch (epi) {
    case 0: dslash_mrhs_staged_kernel<T, R, DAG, 0><<<grid, block, smem, st>>>(a); break;
    case 1: dslash_mrhs_staged_kernel<T, R, DAG, 1><<<grid, block, smem, st>>>(a); break;
    case 2: dslash_mrhs_staged_kernel<T, R, DAG, 2><<<grid, block, smem, st>>>(a); break;
    case 3: dslash_mrhs_staged_kernel<T, R, DAG, 3><<<grid, block, smem, st>>>(a); break;
    default: dslash_mrhs_staged_kernel<T, R, DAG, 6><<<grid, block, smem, st>>>(a); break;
  }
}

template <typename T, int R, bool DAG, int NB>
static void launch_mrhs_epi(MrhsArgs<T> a, int epi, int nrhs, cudaStream_t st) {
  a.ngroups = nrhs / NB;
  const dim3 block(MRHS_SITES, a.ngroups < MRHS_GMAX ? a.ngroups : MRHS_GMAX);
  const int grid = (a.lat.Vh + MRHS_SITES - 1) / MRHS_SITES;
  const size_t smem = (size_t)8 * R * sizeof(T) * MRHS_SITES;  // the block's links
  static bool configured = false;  // one flag per (T, R, DAG, NB) instantiation; the clover rows are static shared memory on top
  if (!configured && smem + 72 * sizeof(T) * MRHS_SITES > 40 * 1024) {
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 0, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 1, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 2, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 3, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 6, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 9, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 10, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 11, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 12, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 13, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaFuncSetAttribute(dslash_mrhs_kernel<T, R, DAG, 14, NB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  configured = true;
  switch (epi) {
    case 0: dslash_mrhs_kernel<T, R, DAG, 0, NB><<<grid, block, smem, st>>>(a); break;
    case 1: dslash_mrhs_kernel<T, R, DAG, 1, NB><<<grid, block, smem, st>>>(a); break;
    case 2: dslash_mrhs_kernel<T, R, DAG, 2, NB><<<grid, block, smem, st>>>(a); break;
    case 3: dslash_mrhs_kernel<T, R, DAG, 3, NB><<<grid, block, smem, st>>>(a); break;
    case 9: dslash_mrhs_kernel<T, R, DAG, 9, NB><<<grid, block, smem, st>>>(a); break;
    case 10: dslash_mrhs_kernel<T, R, DAG, 10, NB><<<grid, block, smem, st>>>(a); break;
    case 11: dslash_mrhs_kernel<T, R, DAG, 11, NB><<<grid, block, smem, st>>>(a); break;
    case 12: dslash_mrhs_kernel<T, R, DAG, 12, NB><<<grid, block, smem, st>>>(a); break;
    case 13: dslash_mrhs_kernel<T, R, DAG, 13, NB><<<grid, block, smem, st>>>(a); break;
    case 14: dslash_mrhs_kernel<T, R, DAG, 14, NB><<<grid, block, smem, st>>>(a); break;
    default: dslash_mrhs_kernel<T, R, DAG, 6, NB><<<grid, block, smem, st>>>(a); break;
  }
}

template <typename T, int R, bool DAG>
static void launch_mrhs_nb(const MrhsArgs<T>& a, int epi, int nrhs, cudaStream_t st) {
  if constexpr (MrhsStage<T, R>::HPR > 0) {
    if (epi <= 6) {  // the epilogues with a reduction (9, 10) exist in the register kernel only
      launch_mrhs_staged<T, R, DAG>(a, epi, nrhs, st);
      return;
    }
  }
  // columns per thread: the tuned NB when it divides nrhs, else one per thread
  if (nrhs % MrhsTune<T>::NB == 0) launch_mrhs_epi<T, R, DAG, MrhsTune<T>::NB>(a, epi, nrhs, st);
  else launch_mrhs_epi<T, R, DAG, 1>(a, epi, nrhs, st);
}

template <typename T>
static void launch_mrhs_typed(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                              int parity, double scale, int dagger, int epi, int nrhs, cudaStream_t st,
                              const DslashFuse* f = nullptr) {
  MrhsArgs<T> a;
  a.r = f ? (T*)f->r : nullptr;
  a.out2 = f ? (T*)f->out2 : nullptr;
  a.partial = c->d_partial_mrhs;
  a.scalars = c->d_scalars;
  a.num = f ? f->num : 0;
  a.den = f ? f->den : 0;
  a.nblocks = (c->lat.Vh + MRHS_SITES - 1) / MRHS_SITES;
  a.zslab = 2 * (c->mrhs_zslab < 0 ? 2 : c->mrhs_zslab);  // LQCD_MRHS_ZSLAB counts pairs of z-planes; default 2 (sweep: 1890 / 1709 / 1736 / 1654 us for 0 / 4 / 8 / 2, fp64)
  a.out = (T*)out;
  a.in = (const T*)in;
  a.gauge = (const T*)gauge;
  a.cl = (const T*)cl;
  a.x = (const T*)x;
  a.lat = c->lat;
  a.parity = parity;
  a.scale = (T)scale;
  a.ws = (T)c->ws;
  a.stride = (size_t)24 * c->lat.Vh;
  if (c->recon == 18) {
    if (dagger) launch_mrhs_nb<T, 18, true>(a, epi, nrhs, st);
    else launch_mrhs_nb<T, 18, false>(a, epi, nrhs, st);
  } else {
    if (dagger) launch_mrhs_nb<T, 12, true>(a, epi, nrhs, st);
    else launch_mrhs_nb<T, 12, false>(a, epi, nrhs, st);
  }
}

// internal entry (solvers and the C ABI): nrhs >= 2 consecutive one-parity native spinors in `in`,
// `out` and (epilogues 2, 3) `x`.
int lqcd_dslash_mrhs_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                            int parity, double scale, int dagger, int epi, int nrhs, cudaStream_t st) {
  const double bytes = (double)c->lat.Vh * c->prec *
                       (8.0 * c->recon + nrhs * 48.0 + (epi >= 1 && epi != 6 ? 72.0 : 0.0) + (epi >= 2 ? nrhs * 24.0 : 0.0));
  c->alg_bytes += bytes;
  const bool rec = c->prof_on && c->prof_n < c->prof_cap;
  if (rec) cudaEventRecord(c->prof_ev[2 * c->prof_n], st);
  if (lqcd_mrhs_tma_ok(c, epi)) {
    const int rc = lqcd_dslash_mrhs_tma_launch(c, out, in, gauge, cl, x, parity, scale, dagger, epi, nrhs, st);
    if (rc) return rc;
  } else if (c->prec == 4) launch_mrhs_typed<float>(c, out, in, gauge, cl, x, parity, scale, dagger, epi, nrhs, st);
  else launch_mrhs_typed<double>(c, out, in, gauge, cl, x, parity, scale, dagger, epi, nrhs, st);
  if (rec) {
    cudaEventRecord(c->prof_ev[2 * c->prof_n + 1], st);
    c->prof_n++;
    c->prof_bytes += bytes;
  }
  LQCD_LAUNCH_CHECK(c, "dslash_mrhs");
  return LQCD_OK;
}

// Krylov recurrences fused per column into the epilogue (9: t, ta = C t, |t|^2 ; 10: r -= alpha q, |r|^2, as in dslash.cu;
// 11, 12: epilogue 3 with BiCGStab's inner products);
// the register kernel of this file, whatever the plain epilogues run on.  Needs whole warps: Vh a multiple of 32.
bool lqcd_mrhs_fuse_ok(const lqcd_ctx* c) { return !c->half && c->lat.Vh % MRHS_SITES == 0; }

int lqcd_dslash_mrhs_fused_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                                  int parity, double scale, int dagger, int epi, int nrhs, const DslashFuse* f, cudaStream_t st) {
  const int nblocks = (c->lat.Vh + MRHS_SITES - 1) / MRHS_SITES;
  if (!c->d_partial_mrhs) {
    if (cudaMalloc(&c->d_partial_mrhs, sizeof(double) * 3 * LQCD_MAX_RHS * nblocks) != cudaSuccess) return lqcd_check_cuda(c, "mrhs partials");
  }
  // epi 9: links, clover, in, x, out, out2 per column ; epi 10: links, in, x, r read and written
  // epi 11: as epi 3 (links, clover, in, x, out) ; epi 12: + y ; epi 13: links, clover, in, x, y (nothing written)
  const double bytes = (double)c->lat.Vh * c->prec *
                       (8.0 * c->recon + (epi == 10 ? 0.0 : 72.0) + nrhs * (epi == 11 || epi == 13 ? 72.0 : 96.0));
  c->alg_bytes += bytes;
  const bool rec = c->prof_on && c->prof_n < c->prof_cap;
  if (rec) cudaEventRecord(c->prof_ev[2 * c->prof_n], st);
  int nsum = nblocks;  // partials per sum and column
  if ((epi == 11 || epi == 12) && lqcd_mrhs_tma_fused_ok(c)) {
    // where the TMA-tiled kernel serves epilogue 3 it serves 11 and 12 too (one partial per 128-site tile)
    nsum = lqcd_mrhs_tma_fused_blocks(c);
    const int rc = lqcd_dslash_mrhs_tma_fused_launch(c, out, in, gauge, cl, x, parity, scale, dagger, epi, nrhs, f->r,
                                                     c->d_partial_mrhs, st);
    if (rc) return rc;
  } else if (c->prec == 4) launch_mrhs_typed<float>(c, out, in, gauge, cl, x, parity, scale, dagger, epi, nrhs, st, f);
  else launch_mrhs_typed<double>(c, out, in, gauge, cl, x, parity, scale, dagger, epi, nrhs, st, f);
  partial_sum_mrhs_kernel<<<dim3(nrhs, epi == 11 || epi == 12 ? 3 : 1), 256, 0, st>>>(c->d_partial_mrhs, nsum, c->d_scalars, f->out_slot);
  c->launches++;
  if (rec) {
    cudaEventRecord(c->prof_ev[2 * c->prof_n + 1], st);
    c->prof_n++;
    c->prof_bytes += bytes;
  }
  LQCD_LAUNCH_CHECK(c, "dslash_mrhs_fused");
  return LQCD_OK;
}

extern "C" {

int lqcd_dslash_mrhs(lqcd_ctx* c, void* out, const void* in, const void* gauge, int parity, double scale, int dagger,
                     int nrhs, void* stream) {
  if (!c || !out || !in || !gauge || (parity != 0 && parity != 1) || nrhs < 1 || nrhs > LQCD_MAX_RHS)
    return LQCD_ERR_INVALID_ARG;
  if (out == in) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "dslash_mrhs: out aliases in");
  if (!lqcd_aligned16(out) || !lqcd_aligned16(in) || !lqcd_aligned16(gauge))
    return lqcd_set_error(c, LQCD_ERR_ALIGN, "dslash_mrhs: alignment");
  return lqcd_dslash_launch(c, out, in, gauge, nullptr, nullptr, parity, scale, dagger ? 1 : 0, 0, nrhs, as_stream(stream));
}

}  // extern "C"
