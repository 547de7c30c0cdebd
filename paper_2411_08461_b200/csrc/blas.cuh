// K6: fused BLAS-1 kernels of the solvers.
// One generic streaming kernel parameterised by an "op": up to 6 one-parity spinors are read as
// flat arrays of 16-byte vectors, updated complex element by complex element, written back, and
// up to 4 fp64 reductions are produced.  Coefficients (alpha, beta, omega) are computed on the
// device from reduction slots in ctx->d_scalars, so a whole Krylov iteration is enqueued without
// a host round-trip.  Reductions: warp shuffle -> block (shared memory) -> per-block partials;
// the last block to finish (ticket counter) sums the partials in block order, so results are
// deterministic for a fixed grid.  Accumulation is fp64 in both precisions.
#pragma once
#include "lqcd_internal.cuh"
#include "half.cuh"

constexpr int BLAS_BLOCK = 256;
constexpr int BLAS_MAXV = 6;
// Batched (multi-right-hand-side) form: blockIdx.y selects the right-hand side; every vector is a
// block of nrhs consecutive one-parity spinors, every right-hand side owns SC_STRIDE scalar slots,
// its own partials and its own ticket.  Slot S_DONE != 0 freezes a right-hand side (its blocks exit
// at once: a converged column is no longer updated); slot S_FIRST marks BiCGStab's first iteration.
constexpr int BLAS_MAXR = 4;  // reductions per launch

template <typename T> struct BlasVecs {
  T* v[BLAS_MAXV];
};

struct cplxd {
  double re, im;
};
__device__ __forceinline__ cplxd cmul(cplxd a, cplxd b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
__device__ __forceinline__ cplxd cdiv(cplxd a, cplxd b) {
  const double d = b.re * b.re + b.im * b.im;
  return {(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d};
}

// omega = <t,s>/<t,t> of BiCGStab from slots ts..ts+2; t = 0 happens when the half step s = r - alpha v already
// solved the system (s = 0, "lucky breakdown"): omega = 0 then, so x += alpha p and r = s = 0, not 0/0
__device__ __forceinline__ cplxd bicg_omega(const double* s, int ts) {
  const double tt = s[ts + 2];
  if (!(tt > 0.0)) return {0.0, 0.0};
  return {s[ts] / tt, s[ts + 1] / tt};
}

template <int NR>
__device__ __forceinline__ void block_reduce_finish(double* acc, double* partial, int max_blocks, unsigned int* ticket,
                                                    double* scalars, const int* out_slots) {
  __shared__ double sm[NR][BLAS_BLOCK / 32];
  __shared__ bool last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int k = 0; k < NR; k++) {
    double v = acc[k];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (lane == 0) sm[k][warp] = v;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < NR; k++) {
      double v = 0;
      for (int w = 0; w < BLAS_BLOCK / 32; w++) v += sm[k][w];
      partial[k * max_blocks + blockIdx.x] = v;
    }
    __threadfence();
    const unsigned int t = atomicAdd(ticket, 1u);
    last = (t == gridDim.x - 1);
  }
  __syncthreads();
  if (last) {
    // fixed-order sum over blocks: each of the first NR warps handles one output
    if (warp < NR) {
      __threadfence();
      double v = 0;
      for (int b = lane; b < (int)gridDim.x; b += 32) v += __ldcg(&partial[warp * max_blocks + b]);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
      if (lane == 0) scalars[out_slots[warp]] = v;
    }
    if (threadIdx.x == 0) *ticket = 0;
  }
}

struct RedArgs {
  double* partial;
  double* scalars;
  unsigned int* ticket;
  int max_blocks;
  int rhs0;       // first right-hand side of this launch
  size_t stride;  // reals between consecutive right-hand sides of a vector block
  int out[4];
};

// Op interface:
//   static constexpr int NV, NR; static constexpr unsigned LOAD, STORE (bit masks over vectors)
//   __device__ void init(const double* scalars);
//   __device__ void elem(T* re_im[NV] ... ) -> implemented as elem(T (*z)[2], double* acc)
template <typename T, typename Op>
__global__ void __launch_bounds__(BLAS_BLOCK) blas_kernel(Op op, BlasVecs<T> vecs, long nvec, RedArgs red) {
  typedef typename V16<T>::vec vec;
  constexpr int N = V16<T>::N;
  const int rhs = red.rhs0 + blockIdx.y;
  red.scalars += (size_t)rhs * SC_STRIDE;
  if (red.scalars[S_DONE] != 0.0) return;  // frozen right-hand side (uniform over its blocks)
  red.partial += (size_t)rhs * BLAS_MAXR * red.max_blocks;
  red.ticket += rhs;
#pragma unroll
  for (int a = 0; a < Op::NV; a++) vecs.v[a] += (size_t)rhs * red.stride;
  op.init(red.scalars);
  double acc[Op::NR > 0 ? Op::NR : 1];
#pragma unroll
  for (int k = 0; k < (Op::NR > 0 ? Op::NR : 1); k++) acc[k] = 0;
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (long)gridDim.x * blockDim.x) {
    T z[Op::NV][N];
#pragma unroll
    for (int a = 0; a < Op::NV; a++) {
      if (Op::LOAD & (1u << a)) {
        vec q = reinterpret_cast<const vec*>(vecs.v[a])[i];
        vec_get(q, z[a]);
      }
    }
#pragma unroll
    for (int e = 0; e < N; e += 2) {
      T w[Op::NV][2];
#pragma unroll
      for (int a = 0; a < Op::NV; a++) { w[a][0] = z[a][e]; w[a][1] = z[a][e + 1]; }
      op.elem(w, acc);
#pragma unroll
      for (int a = 0; a < Op::NV; a++) { z[a][e] = w[a][0]; z[a][e + 1] = w[a][1]; }
    }
#pragma unroll
    for (int a = 0; a < Op::NV; a++) {
      if (Op::STORE & (1u << a)) {
        vec q;
        vec_set(q, z[a]);
        reinterpret_cast<vec*>(vecs.v[a])[i] = q;
      }
    }
  }
  if (Op::NR > 0) block_reduce_finish<(Op::NR > 0 ? Op::NR : 1)>(acc, red.partial, red.max_blocks, red.ticket, red.scalars, red.out);
}

// --------------------------------------------------------------------------------------------
// ops.  Vector order is given in each comment; "s[k]" are reduction slots in ctx->d_scalars.
// --------------------------------------------------------------------------------------------
template <typename T> struct OpNorm2 {  // v0 = x ; out0 = |x|^2
  static constexpr int NV = 1, NR = 1;
  static constexpr unsigned LOAD = 1, STORE = 0;
  __device__ void init(const double*) {}
  __device__ void elem(T (*w)[2], double* acc) { acc[0] += (double)w[0][0] * w[0][0] + (double)w[0][1] * w[0][1]; }
};
template <typename T> struct OpCdot {  // v0 = x, v1 = y ; out = Re<x,y>, Im<x,y>, |x|^2
  static constexpr int NV = 2, NR = 3;
  static constexpr unsigned LOAD = 3, STORE = 0;
  __device__ void init(const double*) {}
  __device__ void elem(T (*w)[2], double* acc) {
    const double xr = w[0][0], xi = w[0][1], yr = w[1][0], yi = w[1][1];
    acc[0] += xr * yr + xi * yi;
    acc[1] += xr * yi - xi * yr;
    acc[2] += xr * xr + xi * xi;
  }
};
template <typename T> struct OpAxpyNorm {  // v0 = x, v1 = y ; y += a x (a real, host) ; out0 = |y|^2
  static constexpr int NV = 2, NR = 1;
  static constexpr unsigned LOAD = 3, STORE = 2;
  double a;
  __device__ void init(const double*) {}
  __device__ void elem(T (*w)[2], double* acc) {
    w[1][0] += (T)a * w[0][0];
    w[1][1] += (T)a * w[0][1];
    acc[0] += (double)w[1][0] * w[1][0] + (double)w[1][1] * w[1][1];
  }
};
template <typename T> struct OpXpay {  // v0 = x, v1 = y ; y = x + a y (a real, host)
  static constexpr int NV = 2, NR = 0;
  static constexpr unsigned LOAD = 3, STORE = 2;
  double a;
  __device__ void init(const double*) {}
  __device__ void elem(T (*w)[2], double*) {
    w[1][0] = w[0][0] + (T)a * w[1][0];
    w[1][1] = w[0][1] + (T)a * w[1][1];
  }
};
template <typename T> struct OpXpayNorm {  // v0 = x, v1 = y ; y = x + a y (a real, host) ; out0 = |y|^2
  static constexpr int NV = 2, NR = 1;
  static constexpr unsigned LOAD = 3, STORE = 2;
  double a;
  __device__ void init(const double*) {}
  __device__ void elem(T (*w)[2], double* acc) {
    w[1][0] = w[0][0] + (T)a * w[1][0];
    w[1][1] = w[0][1] + (T)a * w[1][1];
    acc[0] += (double)w[1][0] * w[1][0] + (double)w[1][1] * w[1][1];
  }
};
template <typename T> struct OpCaxpbypz {  // v0 = x, v1 = y, v2 = z ; z += a x + b y (complex, host)
  static constexpr int NV = 3, NR = 0;
  static constexpr unsigned LOAD = 7, STORE = 4;
  cplxd a, b;
  __device__ void init(const double*) {}
  __device__ void elem(T (*w)[2], double*) {
    const T ar = (T)a.re, ai = (T)a.im, br = (T)b.re, bi = (T)b.im;
    w[2][0] += ar * w[0][0] - ai * w[0][1] + br * w[1][0] - bi * w[1][1];
    w[2][1] += ar * w[0][1] + ai * w[0][0] + br * w[1][1] + bi * w[1][0];
  }
};
// CG update (O9): alpha = s[num]/s[den] ; v0 = x += alpha v1(t) ; v2 = r -= alpha v3(q) ; out0 = |r|^2
template <typename T> struct OpCgUpdate {
  static constexpr int NV = 4, NR = 1;
  static constexpr unsigned LOAD = 15, STORE = 5;
  int num, den;
  T alpha;
  __device__ void init(const double* s) { alpha = (T)(s[num] / s[den]); }
  __device__ void elem(T (*w)[2], double* acc) {
    w[0][0] += alpha * w[1][0];
    w[0][1] += alpha * w[1][1];
    w[2][0] -= alpha * w[3][0];
    w[2][1] -= alpha * w[3][1];
    acc[0] += (double)w[2][0] * w[2][0] + (double)w[2][1] * w[2][1];
  }
};
// x += (s[num]/s[den]) t                            v0 = x, v1 = t
template <typename T> struct OpAxpyRatio {
  static constexpr int NV = 2, NR = 0;
  static constexpr unsigned LOAD = 3, STORE = 1;
  int num, den;
  T alpha;
  __device__ void init(const double* s) { alpha = (T)(s[num] / s[den]); }
  __device__ void elem(T (*w)[2], double*) {
    w[0][0] += alpha * w[1][0];
    w[0][1] += alpha * w[1][1];
  }
};
// r -= (s[num]/s[den]) q ; out0 = |r|^2            v0 = r, v1 = q
template <typename T> struct OpAxmyNormRatio {
  static constexpr int NV = 2, NR = 1;
  static constexpr unsigned LOAD = 3, STORE = 1;
  int num, den;
  T alpha;
  __device__ void init(const double* s) { alpha = (T)(s[num] / s[den]); }
  __device__ void elem(T (*w)[2], double* acc) {
    w[0][0] -= alpha * w[1][0];
    w[0][1] -= alpha * w[1][1];
    acc[0] += (double)w[0][0] * w[0][0] + (double)w[0][1] * w[0][1];
  }
};
// p = r + (s[num]/s[den]) p                        v0 = p, v1 = r
template <typename T> struct OpXpayRatio {
  static constexpr int NV = 2, NR = 0;
  static constexpr unsigned LOAD = 3, STORE = 1;
  int num, den;
  T beta;
  __device__ void init(const double* s) { beta = (T)(s[num] / s[den]); }
  __device__ void elem(T (*w)[2], double*) {
    w[0][0] = w[1][0] + beta * w[0][0];
    w[0][1] = w[1][1] + beta * w[0][1];
  }
};
// BiCGStab (O9).  Slots: rho (2: <r0,r> of this iteration), r0v (3: <r0,v>, |r0|^2 unused),
// ts (3: Re<t,s>, Im<t,s>, |t|^2).
//   p = r + beta (p - omega v), beta = (rho/r0v_prev)/omega_prev ; first iteration: p = r.   v0=p v1=r v2=v
template <typename T> struct OpBicgP {
  static constexpr int NV = 3, NR = 0;
  static constexpr unsigned LOAD = 7, STORE = 1;
  int rho, r0v, ts;
  bool first;
  cplxd beta, omega;
  __device__ void init(const double* s) {
    first = s[S_FIRST] != 0.0;
    if (first) { beta = {0, 0}; omega = {0, 0}; return; }
    omega = bicg_omega(s, ts);
    beta = cdiv(cdiv({s[rho], s[rho + 1]}, {s[r0v], s[r0v + 1]}), omega);
  }
  __device__ void elem(T (*w)[2], double*) {
    if (first) {  // p, v hold garbage on the first iteration: do not touch them
      w[0][0] = w[1][0];
      w[0][1] = w[1][1];
      return;
    }
    const T br = (T)beta.re, bi = (T)beta.im, orr = (T)omega.re, oi = (T)omega.im;
    const T ur = w[0][0] - (orr * w[2][0] - oi * w[2][1]);
    const T ui = w[0][1] - (orr * w[2][1] + oi * w[2][0]);
    w[0][0] = w[1][0] + br * ur - bi * ui;
    w[0][1] = w[1][1] + br * ui + bi * ur;
  }
};
//   s = r - alpha v, alpha = rho / r0v                                                   v0=s v1=r v2=v
template <typename T> struct OpBicgS {
  static constexpr int NV = 3, NR = 0;
  static constexpr unsigned LOAD = 6, STORE = 1;
  int rho, r0v;
  cplxd alpha;
  __device__ void init(const double* s) { alpha = cdiv({s[rho], s[rho + 1]}, {s[r0v], s[r0v + 1]}); }
  __device__ void elem(T (*w)[2], double*) {
    const T ar = (T)alpha.re, ai = (T)alpha.im;
    w[0][0] = w[1][0] - (ar * w[2][0] - ai * w[2][1]);
    w[0][1] = w[1][1] - (ar * w[2][1] + ai * w[2][0]);
  }
};
//   x += alpha p + omega s ; r = s - omega t ; out = |r|^2, Re<r0,r>, Im<r0,r>   v0=x v1=r v2=p v3=s v4=t v5=r0
template <typename T> struct OpBicgXR {
  static constexpr int NV = 6, NR = 3;
  static constexpr unsigned LOAD = 1 | 4 | 8 | 16 | 32, STORE = 3;
  int rho, r0v, ts;
  cplxd alpha, omega;
  __device__ void init(const double* s) {
    alpha = cdiv({s[rho], s[rho + 1]}, {s[r0v], s[r0v + 1]});
    omega = bicg_omega(s, ts);
  }
  __device__ void elem(T (*w)[2], double* acc) {
    const T ar = (T)alpha.re, ai = (T)alpha.im, orr = (T)omega.re, oi = (T)omega.im;
    w[0][0] += ar * w[2][0] - ai * w[2][1] + orr * w[3][0] - oi * w[3][1];
    w[0][1] += ar * w[2][1] + ai * w[2][0] + orr * w[3][1] + oi * w[3][0];
    w[1][0] = w[3][0] - (orr * w[4][0] - oi * w[4][1]);
    w[1][1] = w[3][1] - (orr * w[4][1] + oi * w[4][0]);
    const double rr = w[1][0], ri = w[1][1], zr = w[5][0], zi = w[5][1];
    acc[0] += rr * rr + ri * ri;
    acc[1] += zr * rr + zi * ri;
    acc[2] += zr * ri - zi * rr;
  }
};

// v[a]: base of vector block a (right-hand side 0); right-hand sides rhs0 .. rhs0+nrhs-1 are processed
template <typename T, typename Op>
static inline int blas_launch(lqcd_ctx* c, const Op& op, void* const* v, const int* out_slots, int nrhs, int rhs0,
                              cudaStream_t st) {
  BlasVecs<T> vecs;
  for (int a = 0; a < BLAS_MAXV; a++) vecs.v[a] = a < Op::NV ? (T*)v[a] : nullptr;
  const long nvec = (long)Lay<T>::NSV * c->lat.Vh;
  long want = (nvec + BLAS_BLOCK - 1) / BLAS_BLOCK;
  int grid = (int)(want < c->max_red_blocks ? want : c->max_red_blocks);
  RedArgs red;
  red.partial = c->d_partial;
  red.scalars = c->d_scalars;
  red.ticket = c->d_ticket;
  red.max_blocks = c->max_red_blocks;
  red.rhs0 = rhs0;
  red.stride = (size_t)24 * c->lat.Vh;
  for (int k = 0; k < 4; k++) red.out[k] = out_slots ? out_slots[k] : 0;
  const int acct = (c->acct_rhs > 0 && c->acct_rhs < nrhs) ? c->acct_rhs : nrhs;  // frozen columns move no bytes
  c->alg_bytes += (double)(__builtin_popcount(Op::LOAD) + __builtin_popcount(Op::STORE)) * 24.0 * sizeof(T) * c->lat.Vh * acct;
  blas_kernel<T, Op><<<dim3(grid, nrhs), BLAS_BLOCK, 0, st>>>(op, vecs, nvec, red);
  LQCD_LAUNCH_CHECK(c, "blas");
  return LQCD_OK;
}

// --------------------------------------------------------------------------------------------
// 16-bit storage (half.cuh): the same ops, one thread per SITE, because a stored vector needs the site's norm
// (the largest of its 24 components) before its first component can be written.  Single right-hand side.
// --------------------------------------------------------------------------------------------
template <typename Op>
__global__ void __launch_bounds__(BLAS_BLOCK) blas_half_kernel(Op op, BlasVecs<void> vecs, int Vh, RedArgs red) {
  if (red.scalars[S_DONE] != 0.0) return;
  op.init(red.scalars);
  double acc[Op::NR > 0 ? Op::NR : 1];
#pragma unroll
  for (int k = 0; k < (Op::NR > 0 ? Op::NR : 1); k++) acc[k] = 0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < Vh; i += gridDim.x * blockDim.x) {
    float z[Op::NV][24];
#pragma unroll
    for (int a = 0; a < Op::NV; a++)
      if (Op::LOAD & (1u << a)) load_spinor_h_plain(vecs.v[a], Vh, i, z[a]);
#pragma unroll
    for (int e = 0; e < 24; e += 2) {
      float w[Op::NV][2];
#pragma unroll
      for (int a = 0; a < Op::NV; a++) { w[a][0] = z[a][e]; w[a][1] = z[a][e + 1]; }
      op.elem(w, acc);
#pragma unroll
      for (int a = 0; a < Op::NV; a++) { z[a][e] = w[a][0]; z[a][e + 1] = w[a][1]; }
    }
#pragma unroll
    for (int a = 0; a < Op::NV; a++)
      if (Op::STORE & (1u << a)) store_spinor_h(vecs.v[a], Vh, i, z[a]);
  }
  if (Op::NR > 0) block_reduce_finish<(Op::NR > 0 ? Op::NR : 1)>(acc, red.partial, red.max_blocks, red.ticket, red.scalars, red.out);
}

template <typename Op>
static inline int blas_half_launch(lqcd_ctx* c, const Op& op, void* const* v, const int* out_slots, int nrhs, int rhs0,
                                   cudaStream_t st) {
  if (nrhs != 1 || rhs0 != 0) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "16-bit context: one right-hand side only");
  BlasVecs<void> vecs;
  for (int a = 0; a < BLAS_MAXV; a++) vecs.v[a] = a < Op::NV ? v[a] : nullptr;
  const int Vh = c->lat.Vh;
  const long want = (Vh + BLAS_BLOCK - 1) / BLAS_BLOCK;
  const int grid = (int)(want < c->max_red_blocks ? want : c->max_red_blocks);
  RedArgs red;
  red.partial = c->d_partial;
  red.scalars = c->d_scalars;
  red.ticket = c->d_ticket;
  red.max_blocks = c->max_red_blocks;
  red.rhs0 = 0;
  red.stride = 0;
  for (int k = 0; k < 4; k++) red.out[k] = out_slots ? out_slots[k] : 0;
  c->alg_bytes += (double)(__builtin_popcount(Op::LOAD) + __builtin_popcount(Op::STORE)) * 52.0 * Vh;
  blas_half_kernel<Op><<<grid, BLAS_BLOCK, 0, st>>>(op, vecs, Vh, red);
  LQCD_LAUNCH_CHECK(c, "blas_half");
  return LQCD_OK;
}
