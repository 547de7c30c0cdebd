// Sources, propagator assembly and per-time-slice contractions of the paper's Listing 1
// (Eqs. 6-8).
// Everything here works on PUBLIC layouts: site axes [2][Lt][Lz][Ly][Lx/2] ("wtzyx"),
// spinor [...][4][3], propagator [...][j sink spin][i source spin][b sink colour][a source colour].
// For fixed (w, t) the (z, y, xh, component) range is contiguous, so all kernels are flat, coalesced
// sweeps over one (parity, time-slice) chunk; reductions are fp64 and deterministic (fixed grid,
// per-block partials summed in block order by a second kernel).
#include "lqcd_internal.cuh"

template <typename T> struct Cx { T re, im; };
constexpr int CT_BLOCK = 256;

__device__ __forceinline__ void site_xyz(const Lat& L, int w, int t, int s, int& x, int& y, int& z) {
  const int xh = s % L.Lxh;
  int q = s / L.Lxh;
  y = q % L.Ly;
  z = q / L.Ly;
  x = 2 * xh + ((w + y + z + t) & 1);
}

// phase[w][t][z][y][xh] = exp(2 pi i (nx x/Lx + ny y/Ly + nz z/Lz)); the argument is reduced mod 1
// in integer arithmetic before sincospi, so the result is correctly rounded fp64 whatever the size
template <typename T>
__global__ void __launch_bounds__(CT_BLOCK) phase_kernel(Cx<T>* __restrict__ out, Lat L, int nx, int ny, int nz) {
  const long n = 2L * L.Vh;
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int slice = L.Lxh * L.Ly * L.Lz;
  const int w = (int)(i / L.Vh), r = (int)(i % L.Vh), t = r / slice, s = r % slice;
  int x, y, z;
  site_xyz(L, w, t, s, x, y, z);
  const int Lx = 2 * L.Lxh;
  const long long den = (long long)Lx * L.Ly * L.Lz;
  long long num = (long long)nx * x * L.Ly * L.Lz + (long long)ny * y * Lx * L.Lz + (long long)nz * z * Lx * L.Ly;
  num %= den;
  if (num < 0) num += den;
  double sn, cs;
  sincospi(2.0 * (double)num / (double)den, &sn, &cs);
  out[i].re = (T)cs;
  out[i].im = (T)sn;
}

// wall (t0 >= 0, site < 0) or point (site = cb index within parity w0 at t0) source, one column
template <typename T>
__global__ void __launch_bounds__(CT_BLOCK) source_kernel(Cx<T>* __restrict__ b, const Cx<T>* __restrict__ phase, Lat L,
                                                          int t0, int comp, int w0, int site) {
  const long n = 2L * L.Vh;
  const long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int slice = L.Lxh * L.Ly * L.Lz;
  const int w = (int)(i / L.Vh), r = (int)(i % L.Vh), t = r / slice;
  Cx<T> v = {0, 0};
  if (t == t0 && (site < 0 || (w == w0 && r == site))) v = phase ? phase[i] : Cx<T>{1, 0};
#pragma unroll
  for (int e = 0; e < 12; e++) b[i * 12 + e] = (e == comp) ? v : Cx<T>{0, 0};
}

// a12: prop[site][j][i][b][a] = column[3i+a][site][j][b]   (split = the inverse copy)
template <typename T, bool SPLIT>
__global__ void __launch_bounds__(CT_BLOCK) assemble_kernel(Cx<T>* __restrict__ prop, Cx<T>* __restrict__ cols, long nsite) {
  const long k = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nsite * 144) return;
  const long site = k / 144;
  const int e = (int)(k % 144), j = e / 36, i = (e / 9) % 4, bb = (e / 3) % 3, a = e % 3;
  Cx<T>* c = cols + ((long)(3 * i + a) * nsite + site) * 12 + 3 * j + bb;
  if (SPLIT) *c = prop[k];
  else prop[k] = *c;
}

struct Gamma4 { double re[16], im[16]; };  // row-major 4x4

__device__ __forceinline__ void block_sum2(double& re, double& im, double* partial_re_im) {
  __shared__ double sm[2][CT_BLOCK / 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    re += __shfl_down_sync(0xffffffffu, re, o);
    im += __shfl_down_sync(0xffffffffu, im, o);
  }
  if (lane == 0) { sm[0][warp] = re; sm[1][warp] = im; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0, b = 0;
    for (int w = 0; w < CT_BLOCK / 32; w++) { a += sm[0][w]; b += sm[1][w]; }
    partial_re_im[0] = a;
    partial_re_im[1] = b;
  }
}

// Eq. 6: partial[(w*Lt+t)*nblk + blk] = sum over the block's share of conj(ph) conj(S0) Sp
template <typename T>
__global__ void __launch_bounds__(CT_BLOCK) twopt_kernel(double* __restrict__ partial, const Cx<T>* __restrict__ phase,
                                                         const Cx<T>* __restrict__ S0, const Cx<T>* __restrict__ Sp, long slice) {
  const long chunk = (long)blockIdx.y * slice;  // first site of this (w, t)
  const long n = slice * 144;
  double re = 0, im = 0;
  for (long k = (long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long)gridDim.x * blockDim.x) {
    const long site = chunk + k / 144;
    const Cx<T> a = S0[chunk * 144 + k], b = Sp[chunk * 144 + k];
    // conj(a) * b
    const double pr = (double)a.re * b.re + (double)a.im * b.im, pi = (double)a.re * b.im - (double)a.im * b.re;
    double cr = 1.0, ci = 0.0;
    if (phase) { cr = phase[site].re; ci = -(double)phase[site].im; }
    re += cr * pr - ci * pi;
    im += cr * pi + ci * pr;
  }
  block_sum2(re, im, partial + 2 * ((long)blockIdx.y * gridDim.x + blockIdx.x));
}

// Eq. 7: sum_{j,k} conj(S_p0[j,i,b,a]) Gamma[j][k] S_p[k,i,b,a]
template <typename T>
__global__ void __launch_bounds__(CT_BLOCK) threept_kernel(double* __restrict__ partial, const Cx<T>* __restrict__ Sp0,
                                                           const Cx<T>* __restrict__ Sp, Gamma4 g, long slice) {
  const long chunk = (long)blockIdx.y * slice;
  const long n = slice * 36;
  double re = 0, im = 0;
  for (long q = (long)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (long)gridDim.x * blockDim.x) {
    const long base = (chunk + q / 36) * 144 + q % 36;
    double br[4], bi[4];
#pragma unroll
    for (int k = 0; k < 4; k++) { br[k] = Sp[base + 36 * k].re; bi[k] = Sp[base + 36 * k].im; }
#pragma unroll
    for (int j = 0; j < 4; j++) {
      double vr = 0, vi = 0;  // (Gamma S_p)_j
#pragma unroll
      for (int k = 0; k < 4; k++) {
        vr += g.re[4 * j + k] * br[k] - g.im[4 * j + k] * bi[k];
        vi += g.re[4 * j + k] * bi[k] + g.im[4 * j + k] * br[k];
      }
      const double ar = Sp0[base + 36 * j].re, ai = Sp0[base + 36 * j].im;
      re += ar * vr + ai * vi;
      im += ar * vi - ai * vr;
    }
  }
  block_sum2(re, im, partial + 2 * ((long)blockIdx.y * gridDim.x + blockIdx.x));
}

// out[t] = sum_w sum_blk partial, fixed order
__global__ void slice_sum_kernel(double* __restrict__ out, const double* __restrict__ partial, int Lt, int nblk) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= Lt) return;
  double re = 0, im = 0;
  for (int w = 0; w < 2; w++)
    for (int b = 0; b < nblk; b++) {
      re += partial[2 * ((long)(w * Lt + t) * nblk + b)];
      im += partial[2 * ((long)(w * Lt + t) * nblk + b) + 1];
    }
  out[2 * t] = re;
  out[2 * t + 1] = im;
}

// Eq. 8: X[site][i][k][a][b] = conj(ph) sum_j Gamma[i][j] S0[site][j][k][a][b] on time-slice t, 0 elsewhere
template <typename T>
__global__ void __launch_bounds__(CT_BLOCK) seqsrc_kernel(Cx<T>* __restrict__ X, const Cx<T>* __restrict__ phase,
                                                          const Cx<T>* __restrict__ S0, Gamma4 g, Lat L, int t0) {
  const long n = 2L * L.Vh * 36;
  const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= n) return;
  const long site = q / 36, base = site * 144 + q % 36;
  const int slice = L.Lxh * L.Ly * L.Lz;
  const int t = (int)((site % L.Vh) / slice);
  if (t != t0) {
#pragma unroll
    for (int i = 0; i < 4; i++) X[base + 36 * i] = Cx<T>{0, 0};
    return;
  }
  double sr[4], si[4];
#pragma unroll
  for (int j = 0; j < 4; j++) { sr[j] = S0[base + 36 * j].re; si[j] = S0[base + 36 * j].im; }
  double cr = 1.0, ci = 0.0;
  if (phase) { cr = phase[site].re; ci = -(double)phase[site].im; }
#pragma unroll
  for (int i = 0; i < 4; i++) {
    double vr = 0, vi = 0;
#pragma unroll
    for (int j = 0; j < 4; j++) {
      vr += g.re[4 * i + j] * sr[j] - g.im[4 * i + j] * si[j];
      vi += g.re[4 * i + j] * si[j] + g.im[4 * i + j] * sr[j];
    }
    X[base + 36 * i] = Cx<T>{(T)(cr * vr - ci * vi), (T)(cr * vi + ci * vr)};
  }
}

// ---------------------------------------------------------------------------------------------
// C ABI
// ---------------------------------------------------------------------------------------------
static Gamma4 make_gamma(const double* g) {
  Gamma4 G;
  for (int e = 0; e < 16; e++) { G.re[e] = g[2 * e]; G.im[e] = g[2 * e + 1]; }
  return G;
}
static inline int grid_for(long n) { return (int)((n + CT_BLOCK - 1) / CT_BLOCK); }

// per-slice reduction scratch inside ctx->d_partial: [2*Lt*nblk complex partials][Lt complex results]
static int slice_scratch(lqcd_ctx* c, int* nblk, double** partial, double** out) {
  const long cap = 4L * c->max_red_blocks * LQCD_MAX_RHS;  // doubles
  const int Lt = c->lat.Lt;
  int nb = 32;
  while (nb > 1 && 4L * Lt * nb + 2L * Lt > cap) nb >>= 1;
  if (4L * Lt * nb + 2L * Lt > cap) return lqcd_set_error(c, LQCD_ERR_DIMS, "contract: Lt too large for the reduction scratch");
  *nblk = nb;
  *partial = c->d_partial;
  *out = c->d_partial + 4L * Lt * nb;
  return LQCD_OK;
}
static int slice_finish(lqcd_ctx* c, double* out_host, double* partial, double* out, int nblk, cudaStream_t st) {
  const int Lt = c->lat.Lt;
  slice_sum_kernel<<<(Lt + 63) / 64, 64, 0, st>>>(out, partial, Lt, nblk);
  LQCD_LAUNCH_CHECK(c, "slice_sum");
  cudaMemcpyAsync(out_host, out, sizeof(double) * 2 * Lt, cudaMemcpyDeviceToHost, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return lqcd_check_cuda(c, "contract sync");
  return LQCD_OK;
}

extern "C" {

int lqcd_momentum_phase(lqcd_ctx* c, void* phase, const int mom[3], void* stream) {
  if (!c || !phase || !mom) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  const long n = 2L * c->lat.Vh;
  if (c->prec == 4) phase_kernel<float><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<float>*)phase, c->lat, mom[0], mom[1], mom[2]);
  else phase_kernel<double><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<double>*)phase, c->lat, mom[0], mom[1], mom[2]);
  c->alg_bytes += (double)n * 2 * c->prec;
  LQCD_LAUNCH_CHECK(c, "momentum_phase");
  return LQCD_OK;
}

static int source_launch(lqcd_ctx* c, void* b, const void* phase, int t0, int spin, int colour, int w0, int site, cudaStream_t st) {
  const long n = 2L * c->lat.Vh;
  const int comp = 3 * spin + colour;
  if (c->prec == 4) source_kernel<float><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<float>*)b, (const Cx<float>*)phase, c->lat, t0, comp, w0, site);
  else source_kernel<double><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<double>*)b, (const Cx<double>*)phase, c->lat, t0, comp, w0, site);
  c->alg_bytes += (double)n * 24 * c->prec;
  LQCD_LAUNCH_CHECK(c, "source");
  return LQCD_OK;
}

int lqcd_source_wall(lqcd_ctx* c, void* b_public, int t0, int spin, int colour, const void* phase, void* stream) {
  if (!c || !b_public || t0 < 0 || t0 >= c->lat.Lt || spin < 0 || spin > 3 || colour < 0 || colour > 2)
    return LQCD_ERR_INVALID_ARG;
  return source_launch(c, b_public, phase, t0, spin, colour, 0, -1, as_stream(stream));
}

int lqcd_source_point(lqcd_ctx* c, void* b_public, const int x[4], int spin, int colour, void* stream) {
  if (!c || !b_public || !x || spin < 0 || spin > 3 || colour < 0 || colour > 2) return LQCD_ERR_INVALID_ARG;
  for (int d = 0; d < 4; d++)
    if (x[d] < 0 || x[d] >= c->L[d]) return LQCD_ERR_INVALID_ARG;
  const int w0 = (x[0] + x[1] + x[2] + x[3]) & 1;
  const int site = (x[0] >> 1) + c->lat.Lxh * (x[1] + c->lat.Ly * (x[2] + c->lat.Lz * x[3]));
  return source_launch(c, b_public, nullptr, x[3], spin, colour, w0, site, as_stream(stream));
}

static int assemble_launch(lqcd_ctx* c, void* prop, void* cols, bool split, cudaStream_t st) {
  const long nsite = 2L * c->lat.Vh, n = nsite * 144;
  if (c->prec == 4) {
    if (split) assemble_kernel<float, true><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<float>*)prop, (Cx<float>*)cols, nsite);
    else assemble_kernel<float, false><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<float>*)prop, (Cx<float>*)cols, nsite);
  } else {
    if (split) assemble_kernel<double, true><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<double>*)prop, (Cx<double>*)cols, nsite);
    else assemble_kernel<double, false><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<double>*)prop, (Cx<double>*)cols, nsite);
  }
  c->alg_bytes += (double)n * 4 * c->prec;
  LQCD_LAUNCH_CHECK(c, "propagator_assemble");
  return LQCD_OK;
}
int lqcd_propagator_assemble(lqcd_ctx* c, void* prop_public, const void* columns_public, void* stream) {
  if (!c || !prop_public || !columns_public) return LQCD_ERR_INVALID_ARG;
  return assemble_launch(c, prop_public, (void*)columns_public, false, as_stream(stream));
}
int lqcd_propagator_split(lqcd_ctx* c, void* columns_public, const void* prop_public, void* stream) {
  if (!c || !prop_public || !columns_public) return LQCD_ERR_INVALID_ARG;
  return assemble_launch(c, (void*)prop_public, columns_public, true, as_stream(stream));
}

int lqcd_contract_twopt(lqcd_ctx* c, double* out_host, const void* phase, const void* S_0, const void* S_p, void* stream) {
  if (!c || !out_host || !S_0 || !S_p) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  int nblk, rc;
  double *partial, *out;
  if ((rc = slice_scratch(c, &nblk, &partial, &out))) return rc;
  const long slice = (long)c->lat.Lxh * c->lat.Ly * c->lat.Lz;
  const dim3 grid(nblk, 2 * c->lat.Lt);
  if (c->prec == 4) twopt_kernel<float><<<grid, CT_BLOCK, 0, st>>>(partial, (const Cx<float>*)phase, (const Cx<float>*)S_0, (const Cx<float>*)S_p, slice);
  else twopt_kernel<double><<<grid, CT_BLOCK, 0, st>>>(partial, (const Cx<double>*)phase, (const Cx<double>*)S_0, (const Cx<double>*)S_p, slice);
  c->alg_bytes += 2.0 * c->lat.Vh * (2 * 288 + (phase ? 2 : 0)) * c->prec;
  LQCD_LAUNCH_CHECK(c, "contract_twopt");
  return slice_finish(c, out_host, partial, out, nblk, st);
}

int lqcd_contract_threept(lqcd_ctx* c, double* out_host, const void* S_p0, const double gamma[32], const void* S_p, void* stream) {
  if (!c || !out_host || !S_p0 || !S_p || !gamma) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  int nblk, rc;
  double *partial, *out;
  if ((rc = slice_scratch(c, &nblk, &partial, &out))) return rc;
  const long slice = (long)c->lat.Lxh * c->lat.Ly * c->lat.Lz;
  const dim3 grid(nblk, 2 * c->lat.Lt);
  const Gamma4 G = make_gamma(gamma);
  if (c->prec == 4) threept_kernel<float><<<grid, CT_BLOCK, 0, st>>>(partial, (const Cx<float>*)S_p0, (const Cx<float>*)S_p, G, slice);
  else threept_kernel<double><<<grid, CT_BLOCK, 0, st>>>(partial, (const Cx<double>*)S_p0, (const Cx<double>*)S_p, G, slice);
  c->alg_bytes += 2.0 * c->lat.Vh * 2 * 288 * c->prec;
  LQCD_LAUNCH_CHECK(c, "contract_threept");
  return slice_finish(c, out_host, partial, out, nblk, st);
}

int lqcd_sequential_source(lqcd_ctx* c, void* X_prop, const void* phase, const double gamma[32], const void* S_0, int t, void* stream) {
  if (!c || !X_prop || !S_0 || !gamma || t < 0 || t >= c->lat.Lt || X_prop == S_0) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  const long n = 2L * c->lat.Vh * 36;
  const Gamma4 G = make_gamma(gamma);
  if (c->prec == 4) seqsrc_kernel<float><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<float>*)X_prop, (const Cx<float>*)phase, (const Cx<float>*)S_0, G, c->lat, t);
  else seqsrc_kernel<double><<<grid_for(n), CT_BLOCK, 0, st>>>((Cx<double>*)X_prop, (const Cx<double>*)phase, (const Cx<double>*)S_0, G, c->lat, t);
  c->alg_bytes += 2.0 * c->lat.Vh * 288 * c->prec * (1.0 + 1.0 / c->lat.Lt);
  LQCD_LAUNCH_CHECK(c, "sequential_source");
  return LQCD_OK;
}

}  // extern "C"
