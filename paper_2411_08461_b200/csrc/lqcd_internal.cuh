// Internal declarations of liblqcd (CUDA, sm_100a).  Not part of the C ABI (include/lqcd.h).
// Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include "lqcd.h"

// ---------------------------------------------------------------------------------------------
// Lattice geometry handed to kernels by value.  Checkerboard index of a site of parity p
// (cb2 layout [2][Lt][Lz][Ly][Lx/2]):  c = xh + Lxh*(y + Ly*(z + Lz*t)),
// x = 2*xh + ((p + y + z + t) & 1).
// ---------------------------------------------------------------------------------------------
struct Lat {
  int Lxh, Ly, Lz, Lt;
  int Vh;
  int tb;  // +1 periodic, -1 antiperiodic in t
};

constexpr int LQCD_MAX_DEVICES = 64;
// Scalar slots of one right-hand side in ctx->d_scalars (SC_STRIDE doubles each).  The solvers' own reduction slots
// are in solver.cu; these are shared with the kernels: S_DONE != 0 freezes a right-hand side (its BLAS blocks exit at
// once, the fused epilogues leave r alone), S_FIRST marks BiCGStab's first iteration, and the device-side stopping
// test (solver.cu, conv_check_kernel) keeps its threshold, its iteration counter, a flag (1 NaN, 2 rho/omega
// underflow) and the last live residual in S_STOP, S_ITERS, S_FLAG, S_RRFIN.
constexpr int SC_STRIDE = 64;
constexpr int S_STOP = 56, S_ITERS = 57, S_FLAG = 58, S_RRFIN = 59, S_DONE = 60, S_FIRST = 61;  // lqcd_create refuses a larger ordinal (per-device launch configuration flags)

// an instantiated CUDA graph of `stride` Krylov iterations (solver.cu), reused while the solve's buffers stay the same
struct GraphSlot {
  unsigned long long key;
  cudaGraphExec_t exec;
  long launches, dslashes;  // what one replay adds to the counters
  double bytes;
};

struct lqcd_ctx {
  int L[4];
  Lat lat;
  long V;
  int prec, recon, device, sm_count;  // prec: bytes of a real of the PUBLIC arrays and of the arithmetic (4 | 8)
  int half;  // 1: native fields in 16-bit fixed point (half.cuh; created with prec = 2: fp32 arithmetic and public arrays)
  cudaStream_t graph_stream;  // the legacy default stream cannot be captured: small-lattice solves called on it run here
  cudaEvent_t ev_graph;
  GraphSlot graphs[4];
  long graph_launches;  // blocks replayed so far (lqcd_graph_launch_count)
  int graph_next, graphs_on;  // LQCD_GRAPHS=0 (at creation) keeps every iteration a sequence of plain launches
  int part_mask;  // bit mu: direction mu is cut between ranks (lqcd_set_partition; dd.cu)
  double ws;  // weight of the spatial hops: nu/xi_0 of Eq. 5; 1 = isotropic
  int mrhs_tma;    // 1 (default): TMA-tiled multi-RHS kernel (dslash_mrhs_tma.cu) where it applies; LQCD_MRHS_TMA=0 turns it off
  int mrhs_fuse_dots;  // batched BiCGStab: inner products in the multi-RHS epilogues (LQCD_MRHS_FUSE_DOTS: 1 on, 0 off; unset = -1: where measured faster)
  int mrhs_zslab;  // z-tiles per slab of its sweep (LQCD_MRHS_ZSLAB; 0 = the whole z extent)
  int tiled;  // 1: shared-memory tiled dslash where the tile divides the lattice (opt-in: LQCD_DSLASH_TILED=1)
  long launches;
  char err[256];
  // reduction scratch (device): per-block partials, ticket counter, result slots; pinned host mirror
  double* d_partial;
  double* d_partial_mrhs;  // [column][32-site warp]: partials of the multi-RHS fused epilogues (allocated on first use)
  double* d_clover_scratch;  // clover build in three passes: two fields of 6 planes x 9 doubles per site (allocated on first use)
  double mixed_last_margin;   // mixed solves: an outer step is taken for the last when the inner residual estimate is below this x the bar
  int clover_onepass;         // LQCD_CLOVER_ONEPASS=1: the one-kernel build (also the fallback when the scratch cannot be allocated)
  double* d_scalars;
  unsigned int* d_ticket;
  int* d_flag;
  double* h_scalars;
  double* h_consts;  // pinned {0.0, 1.0}: sources of small asynchronous flag writes
  double* h_stop;    // pinned, one per right-hand side: source of the asynchronous writes of the stopping thresholds
  int* h_flag;
  int max_red_blocks;
  cudaEvent_t ev0, ev1;
  cudaStream_t copy_stream;      // lqcd_solve_host: uploads run here, beside the kernels of the caller's stream
  cudaEvent_t ev_copy[3];        // entry fence, links uploaded, source uploaded
  // accounting: algorithmic bytes of every launch; optional per-launch event timing of dslash
  double alg_bytes;
  int acct_rhs;  // active right-hand sides of a batched solve (byte accounting of frozen columns)
  int prof_on, prof_n, prof_cap;
  cudaEvent_t* prof_ev;  // 2 events per recorded launch
  double prof_bytes;
};

int lqcd_set_error(lqcd_ctx* ctx, int code, const char* fmt, ...);
int lqcd_check_cuda(lqcd_ctx* ctx, const char* what);
static inline bool lqcd_aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

// ---------------------------------------------------------------------------------------------
// Native structure-of-arrays layouts: arrays of 16-byte vectors, vector index slowest.
//   spinor (one parity): [NSV][Vh] vec16,  24 reals per site in (spin, colour, re/im) order
//   clover (one parity): [NCV][Vh] vec16,  72 reals per site in the public packed order
//   links               : [mu][parity][NGV][Vh] gauge-vec; first R reals of the row-major 3x3
// fp32: vec16 = float4 (4 reals), fp64: vec16 = double2 (2 reals).  fp32 recon-18 links use
// float2 (9 per link); every other link variant uses 16-byte vectors.
// ---------------------------------------------------------------------------------------------
template <typename T> struct V16;
template <> struct V16<float> { typedef float4 vec; static constexpr int N = 4; };
template <> struct V16<double> { typedef double2 vec; static constexpr int N = 2; };

template <typename T, int R> struct GV { typedef typename V16<T>::vec vec; static constexpr int N = V16<T>::N; };
template <> struct GV<float, 18> { typedef float2 vec; static constexpr int N = 2; };

template <typename T> struct Lay {
  static constexpr int N = V16<T>::N;
  static constexpr int NSV = 24 / N;  // vectors per spinor site
  static constexpr int NCV = 72 / N;  // vectors per clover site
};

__device__ __forceinline__ void vec_get(const float4& v, float* r) { r[0] = v.x; r[1] = v.y; r[2] = v.z; r[3] = v.w; }
__device__ __forceinline__ void vec_get(const double2& v, double* r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ void vec_get(const float2& v, float* r) { r[0] = v.x; r[1] = v.y; }
__device__ __forceinline__ void vec_set(float4& v, const float* r) { v = make_float4(r[0], r[1], r[2], r[3]); }
__device__ __forceinline__ void vec_set(double2& v, const double* r) { v = make_double2(r[0], r[1]); }
__device__ __forceinline__ void vec_set(float2& v, const float* r) { v = make_float2(r[0], r[1]); }

// read-only streaming load (links, clover: touched once per sweep) and default cached load
template <typename V> __device__ __forceinline__ V ld_stream(const V* p) { return __ldcs(p); }
template <typename V> __device__ __forceinline__ V ld_cached(const V* p) { return __ldg(p); }

template <typename T>
__device__ __forceinline__ void load_spinor(const T* __restrict__ base, int Vh, int idx, T* psi) {
  typedef typename V16<T>::vec vec;
  const vec* p = reinterpret_cast<const vec*>(base) + idx;
#pragma unroll
  for (int v = 0; v < Lay<T>::NSV; v++) {
    vec q = ld_cached(p + (size_t)v * Vh);
    vec_get(q, psi + v * V16<T>::N);
  }
}
template <typename T>
__device__ __forceinline__ void store_spinor(T* __restrict__ base, int Vh, int idx, const T* psi) {
  typedef typename V16<T>::vec vec;
  vec* p = reinterpret_cast<vec*>(base) + idx;
#pragma unroll
  for (int v = 0; v < Lay<T>::NSV; v++) {
    vec q;
    vec_set(q, psi + v * V16<T>::N);
    p[(size_t)v * Vh] = q;
  }
}

// bytes of one link-field block [NGV][Vh] for (mu, parity)
template <typename T, int R> __host__ __device__ constexpr int gauge_nvec() { return R / GV<T, R>::N; }

// ---------------------------------------------------------------------------------------------
// Packed fp32 arithmetic (Blackwell FFMA2: fma.rn.f32x2, two IEEE fp32 FMAs per issue slot; measured on
// B200: same 73 TFLOP/s as FFMA, i.e. half the issue slots for the same flops).  A complex number
// (re, im) sits in one 64-bit register pair; ptxas folds pk2(a, a) into a scalar-broadcast operand and
// pk2(hi, lo) into an operand swizzle, so a complex multiply-accumulate acc += u * h is two FFMA2:
//   acc = fma2((ur, ur), (hr, hi), acc);  acc = fma2((ui, ui), (-hi, hr), acc)
// with the rotated copy (-hi, hr) = i*h made once per half-spinor component and used for three rows.
// Every lane is the same fused multiply-add, in the same order, as the scalar code below.
// ---------------------------------------------------------------------------------------------
#ifndef DSLASH_FFMA2
#define DSLASH_FFMA2 1
#endif
typedef unsigned long long u64;
__device__ __forceinline__ u64 pk2(float lo, float hi) {
  u64 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void upk2(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
  u64 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
  u64 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
template <typename T> struct UsePacked { static constexpr bool value = false; };
template <> struct UsePacked<float> { static constexpr bool value = DSLASH_FFMA2 != 0; };

// recon-12: row2[c] = conj(row0[a]*row1[b] - row0[b]*row1[a]),  (a,b) = (1,2),(2,0),(0,1)
template <typename T>
__device__ __forceinline__ void recon_row2(T* U) {
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const int a = (c + 1) % 3, b = (c + 2) % 3;
    if constexpr (UsePacked<T>::value) {
      const u64 Vb = pk2(U[6 + 2 * b], U[6 + 2 * b + 1]), Vbs = pk2(U[6 + 2 * b + 1], U[6 + 2 * b]);
      const u64 Va = pk2(U[6 + 2 * a], U[6 + 2 * a + 1]), Vas = pk2(U[6 + 2 * a + 1], U[6 + 2 * a]);
      u64 zr = mul2(pk2(U[2 * a], U[2 * a]), Vb);
      zr = fma2(pk2(-U[2 * b], -U[2 * b]), Va, zr);
      u64 zi = mul2(pk2(U[2 * a + 1], U[2 * a + 1]), Vbs);
      zi = fma2(pk2(-U[2 * b + 1], -U[2 * b + 1]), Vas, zi);
      float re, im;
      upk2(fma2(pk2(-1.f, 1.f), zi, zr), re, im);
      U[12 + 2 * c] = re;
      U[12 + 2 * c + 1] = -im;
    } else {
      T re = U[2 * a] * U[6 + 2 * b] - U[2 * a + 1] * U[6 + 2 * b + 1] - U[2 * b] * U[6 + 2 * a] +
             U[2 * b + 1] * U[6 + 2 * a + 1];
      T im = U[2 * a] * U[6 + 2 * b + 1] + U[2 * a + 1] * U[6 + 2 * b] - U[2 * b] * U[6 + 2 * a + 1] -
             U[2 * b + 1] * U[6 + 2 * a];
      U[12 + 2 * c] = re;
      U[12 + 2 * c + 1] = -im;
    }
  }
}

// load one link into U[18] (row-major, (re,im)); recon-12 rebuilds row 2 = conj(row0 x row1)
template <typename T, int R>
__device__ __forceinline__ void load_link(const T* __restrict__ block, int Vh, int idx, T* U) {
  typedef typename GV<T, R>::vec vec;
  constexpr int N = GV<T, R>::N;
  const vec* p = reinterpret_cast<const vec*>(block) + idx;
#pragma unroll
  for (int v = 0; v < R / N; v++) {
    vec q = ld_stream(p + (size_t)v * Vh);
    vec_get(q, U + v * N);
  }
  if (R == 12) recon_row2<T>(U);
}

// site coordinates of checkerboard index idx of parity par
struct Site {
  int xh, y, z, t, r;  // r = (par + y + z + t) & 1 : x = 2*xh + r
};
__device__ __forceinline__ Site site_of(const Lat& L, int idx, int par) {
  Site s;
  s.xh = idx % L.Lxh;
  int q = idx / L.Lxh;
  s.y = q % L.Ly;
  q /= L.Ly;
  s.z = q % L.Lz;
  s.t = q / L.Lz;
  s.r = (par + s.y + s.z + s.t) & 1;
  return s;
}
// checkerboard index (in the opposite parity) of the neighbour at +1/-1 in direction mu
template <int MU, int DIR>
__device__ __forceinline__ int neighbour(const Lat& L, int idx, const Site& s) {
  if (MU == 0) {
    if (DIR > 0) return s.r ? (s.xh == L.Lxh - 1 ? idx - (L.Lxh - 1) : idx + 1) : idx;
    return s.r ? idx : (s.xh == 0 ? idx + (L.Lxh - 1) : idx - 1);
  } else if (MU == 1) {
    const int st = L.Lxh;
    if (DIR > 0) return s.y == L.Ly - 1 ? idx - (L.Ly - 1) * st : idx + st;
    return s.y == 0 ? idx + (L.Ly - 1) * st : idx - st;
  } else if (MU == 2) {
    const int st = L.Lxh * L.Ly;
    if (DIR > 0) return s.z == L.Lz - 1 ? idx - (L.Lz - 1) * st : idx + st;
    return s.z == 0 ? idx + (L.Lz - 1) * st : idx - st;
  } else {
    const int st = L.Lxh * L.Ly * L.Lz;
    if (DIR > 0) return s.t == L.Lt - 1 ? idx - (L.Lt - 1) * st : idx + st;
    return s.t == 0 ? idx + (L.Lt - 1) * st : idx - st;
  }
}

// launchers implemented per translation unit
#define LQCD_LAUNCH_CHECK(ctx, what)                 \
  do {                                               \
    (ctx)->launches++;                               \
    cudaError_t e__ = cudaPeekAtLastError();         \
    if (e__ != cudaSuccess) return lqcd_check_cuda((ctx), what); \
  } while (0)

static inline cudaStream_t as_stream(void* s) { return reinterpret_cast<cudaStream_t>(s); }

// internal launchers shared between translation units
int lqcd_dslash_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                       int parity, double scale, int dagger, int epi, int nrhs, cudaStream_t st);
// CG recurrences fused into the dslash epilogue (dslash.cu, epilogues 4 and 5; single right-hand side)
struct DslashFuse {
  void* r;       // epi 5: residual updated in place, r -= (s[num]/s[den]) q
  int out_slot;  // reduction result: |out|^2 (epi 4, 7, 9) or |r|^2 (epi 5, 8, 10) -> d_scalars[out_slot]
  int num, den;
  void* out2;    // epi 9: second output, C * out
};
bool lqcd_dslash_fuse_ok(const lqcd_ctx* c);
bool lqcd_dslash_fuse3_ok(const lqcd_ctx* c);
int lqcd_dslash_fused_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                             int parity, double scale, int dagger, int epi, const DslashFuse* f, cudaStream_t st);
int lqcd_dslash_mrhs_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                            int parity, double scale, int dagger, int epi, int nrhs, cudaStream_t st);
bool lqcd_mrhs_fuse_ok(const lqcd_ctx* c);
int lqcd_dslash_mrhs_fused_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                                  int parity, double scale, int dagger, int epi, int nrhs, const DslashFuse* f, cudaStream_t st);
bool lqcd_mrhs_tma_ok(const lqcd_ctx* c, int epi);
bool lqcd_mrhs_tma_fused_ok(const lqcd_ctx* c);
int lqcd_mrhs_tma_fused_blocks(const lqcd_ctx* c);
int lqcd_dslash_mrhs_tma_fused_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                                      int parity, double scale, int dagger, int epi, int nrhs, const void* r, double* partial,
                                      cudaStream_t st);
int lqcd_dslash_mrhs_tma_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                                int parity, double scale, int dagger, int epi, int nrhs, cudaStream_t st);
// 16-bit-storage context (half.cu)
struct DslashFuse;
int lqcd_dslash_half_launch(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* cl, const void* x,
                            int parity, double scale, int dagger, int epi, cudaStream_t st, const DslashFuse* f = nullptr);
int lqcd_partial_sum_launch(lqcd_ctx* c, int n, int slot, cudaStream_t st);  // d_partial[0..n) -> d_scalars[slot], fixed order
int lqcd_clover_apply_half_launch(lqcd_ctx* c, void* out, const void* in, const void* cl_parity, cudaStream_t st);
int lqcd_gauge_pack_half(lqcd_ctx* c, void* native, const void* pub, cudaStream_t st);
int lqcd_spinor_pack_half(lqcd_ctx* c, void* native, const void* pub, int parities, cudaStream_t st);
int lqcd_spinor_unpack_half(lqcd_ctx* c, void* pub, const void* native, int parities, cudaStream_t st);
int lqcd_spinor_down_half(lqcd_ctx* c, void* out, const void* in_fp64, double scale, cudaStream_t st);
int lqcd_spinor_up_axpy_half(lqcd_ctx* c, void* x_fp64, const void* e, double a, cudaStream_t st);
int lqcd_clover_apply_launch(lqcd_ctx* c, void* out, const void* in, const void* cl_parity, int nrhs, cudaStream_t st);
int lqcd_spinor_pack_parity(lqcd_ctx* c, void* native, const void* pub, cudaStream_t st);
int lqcd_spinor_unpack_parity(lqcd_ctx* c, void* pub, const void* native, cudaStream_t st);
