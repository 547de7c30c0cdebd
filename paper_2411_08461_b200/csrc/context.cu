// Context, error reporting and size queries of liblqcd (include/lqcd.h).
#include <stdarg.h>
#include <string.h>
#include <stdlib.h>
#include "lqcd_internal.cuh"

int lqcd_set_error(lqcd_ctx* ctx, int code, const char* fmt, ...) {
  if (ctx) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
    va_end(ap);
  }
  return code;
}

int lqcd_check_cuda(lqcd_ctx* ctx, const char* what) {
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) return LQCD_OK;
  return lqcd_set_error(ctx, LQCD_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

extern "C" {

const char* lqcd_strerror(int code) {
  switch (code) {
    case LQCD_OK: return "ok";
    case LQCD_NOT_CONVERGED: return "not converged within maxiter";
    case LQCD_ERR_INVALID_ARG: return "invalid argument";
    case LQCD_ERR_DIMS: return "unsupported lattice dimensions";
    case LQCD_ERR_ALIGN: return "device pointer not 16-byte aligned";
    case LQCD_ERR_WORKSPACE: return "workspace too small";
    case LQCD_ERR_CUDA: return "CUDA error";
    case LQCD_ERR_SINGULAR_CLOVER: return "singular clover block";
    case LQCD_ERR_BREAKDOWN: return "solver breakdown";
    default: return "unknown error code";
  }
}

const char* lqcd_last_error(const lqcd_ctx* ctx) { return ctx ? ctx->err : "null context"; }
long lqcd_launch_count(const lqcd_ctx* ctx) { return ctx ? ctx->launches : 0; }
long lqcd_graph_launch_count(const lqcd_ctx* ctx) { return ctx ? ctx->graph_launches : 0; }

int lqcd_create(lqcd_ctx** out, const int dims[4], int prec, int recon, int t_boundary, int device) {
  if (!out || !dims) return LQCD_ERR_INVALID_ARG;
  *out = nullptr;
  if ((prec != 4 && prec != 8 && prec != 2) || (recon != 18 && recon != 12) || (t_boundary != 1 && t_boundary != -1))
    return LQCD_ERR_INVALID_ARG;
  long V = 1;
  for (int i = 0; i < 4; i++) {
    if (dims[i] < 4 || (dims[i] & 1)) return LQCD_ERR_DIMS;
    V *= dims[i];
  }
  if (V / 2 > 0x3fffffffL) return LQCD_ERR_DIMS;  // 32-bit site indices inside kernels
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev || device >= LQCD_MAX_DEVICES) {
    cudaGetLastError();
    return LQCD_ERR_CUDA;  // no CPU fallback: without a device the library does nothing
  }
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return LQCD_ERR_CUDA;
  if (prop.major != 10) return LQCD_ERR_CUDA;  // kernels are built for sm_100a only
  if (cudaSetDevice(device) != cudaSuccess) return LQCD_ERR_CUDA;

  lqcd_ctx* c = new lqcd_ctx();
  memset(c, 0, sizeof(*c));
  for (int i = 0; i < 4; i++) c->L[i] = dims[i];
  c->V = V;
  c->lat.Lxh = dims[0] / 2;
  c->lat.Ly = dims[1];
  c->lat.Lz = dims[2];
  c->lat.Lt = dims[3];
  c->lat.Vh = (int)(V / 2);
  c->lat.tb = t_boundary;
  c->prec = prec == 2 ? 4 : prec;  // 16-bit storage: fp32 arithmetic and public arrays
  c->half = prec == 2 ? 1 : 0;
  c->ws = 1.0;
  {
    // shared-memory tiled dslash (dslash_tiled.cuh): parity-tested, measured slower than the one-thread-per-site
    // kernel at every tile shape tried (profiles/r01d_tuning.md), so it is opt-in: LQCD_DSLASH_TILED=1
    const char* e = getenv("LQCD_DSLASH_TILED");
    c->tiled = (e && e[0] == '1') ? 1 : 0;
    const char* m = getenv("LQCD_MRHS_TMA");  // TMA-tiled multi-RHS kernel: on unless LQCD_MRHS_TMA=0 (A/B measurements, parity tests of both)
    c->mrhs_tma = (m && m[0] == '0') ? 0 : ((m && m[0] == '2') ? 2 : 1);
    const char* fd = getenv("LQCD_MRHS_FUSE_DOTS");
    c->mrhs_fuse_dots = fd ? (fd[0] == '1') : -1;  // -1: where the register kernel runs the plain epilogues anyway
    const char* gr = getenv("LQCD_GRAPHS");
    c->graphs_on = (gr && gr[0] == '0') ? 0 : 1;
    const char* ml = getenv("LQCD_MIXED_LAST_MARGIN");
    c->mixed_last_margin = ml ? atof(ml) : 0.9;
    const char* co = getenv("LQCD_CLOVER_ONEPASS");
    c->clover_onepass = (co && co[0] == '1') ? 1 : 0;
    const char* z = getenv("LQCD_MRHS_ZSLAB");
    c->mrhs_zslab = z ? atoi(z) : -1;  // pairs of z-planes per slab; -1: each kernel's own default (4 TMA-tiled, 2 register kernels)
  }
  c->recon = recon;
  c->device = device;
  c->sm_count = prop.multiProcessorCount;
  c->max_red_blocks = 8 * c->sm_count;
  strcpy(c->err, "ok");
  bool ok = cudaMalloc(&c->d_partial, sizeof(double) * 4 * c->max_red_blocks * LQCD_MAX_RHS) == cudaSuccess &&
            cudaMalloc(&c->d_scalars, sizeof(double) * 64 * LQCD_MAX_RHS) == cudaSuccess &&
            cudaMalloc(&c->d_ticket, sizeof(unsigned int) * LQCD_MAX_RHS) == cudaSuccess &&
            cudaMalloc(&c->d_flag, sizeof(int) * 4) == cudaSuccess &&
            cudaMallocHost(&c->h_scalars, sizeof(double) * 64 * LQCD_MAX_RHS) == cudaSuccess &&
            cudaMallocHost(&c->h_consts, sizeof(double) * 2) == cudaSuccess &&
            cudaMallocHost(&c->h_stop, sizeof(double) * LQCD_MAX_RHS) == cudaSuccess &&
            cudaMallocHost(&c->h_flag, sizeof(int) * 4) == cudaSuccess &&
            cudaEventCreate(&c->ev0) == cudaSuccess && cudaEventCreate(&c->ev1) == cudaSuccess &&
            cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&c->graph_stream, cudaStreamNonBlocking) == cudaSuccess &&
            cudaEventCreateWithFlags(&c->ev_graph, cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&c->ev_copy[0], cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&c->ev_copy[1], cudaEventDisableTiming) == cudaSuccess &&
            cudaEventCreateWithFlags(&c->ev_copy[2], cudaEventDisableTiming) == cudaSuccess;
  if (ok) {
    c->h_consts[0] = 0.0;
    c->h_consts[1] = 1.0;
    ok = cudaMemset(c->d_ticket, 0, sizeof(unsigned int) * LQCD_MAX_RHS) == cudaSuccess &&
         cudaMemset(c->d_flag, 0, sizeof(int) * 4) == cudaSuccess &&
         cudaMemset(c->d_scalars, 0, sizeof(double) * 64 * LQCD_MAX_RHS) == cudaSuccess;
  }
  if (!ok) {
    cudaGetLastError();
    lqcd_destroy(c);
    return LQCD_ERR_CUDA;
  }
  *out = c;
  return LQCD_OK;
}

int lqcd_destroy(lqcd_ctx* c) {
  if (!c) return LQCD_ERR_INVALID_ARG;
  cudaSetDevice(c->device);
  if (c->d_partial) cudaFree(c->d_partial);
  if (c->d_partial_mrhs) cudaFree(c->d_partial_mrhs);
  if (c->d_clover_scratch) cudaFree(c->d_clover_scratch);
  if (c->d_scalars) cudaFree(c->d_scalars);
  if (c->d_ticket) cudaFree(c->d_ticket);
  if (c->d_flag) cudaFree(c->d_flag);
  if (c->h_scalars) cudaFreeHost(c->h_scalars);
  for (int i = 0; i < 4; i++)
    if (c->graphs[i].exec) cudaGraphExecDestroy(c->graphs[i].exec);
  if (c->h_consts) cudaFreeHost(c->h_consts);
  if (c->h_stop) cudaFreeHost(c->h_stop);
  if (c->h_flag) cudaFreeHost(c->h_flag);
  if (c->ev0) cudaEventDestroy(c->ev0);
  if (c->ev1) cudaEventDestroy(c->ev1);
  for (int i = 0; i < 3; i++)
    if (c->ev_copy[i]) cudaEventDestroy(c->ev_copy[i]);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  if (c->graph_stream) cudaStreamDestroy(c->graph_stream);
  if (c->ev_graph) cudaEventDestroy(c->ev_graph);
  if (c->prof_ev) {
    for (int i = 0; i < 2 * c->prof_cap; i++) cudaEventDestroy(c->prof_ev[i]);
    delete[] c->prof_ev;
  }
  delete c;
  return LQCD_OK;
}

int lqcd_set_anisotropy(lqcd_ctx* c, double nu_over_xi0) {
  if (!c || !(nu_over_xi0 > 0)) return LQCD_ERR_INVALID_ARG;
  c->ws = nu_over_xi0;
  return LQCD_OK;
}

double lqcd_algorithmic_bytes(const lqcd_ctx* c) { return c ? c->alg_bytes : 0.0; }

int lqcd_profile_enable(lqcd_ctx* c, int enable) {
  if (!c) return LQCD_ERR_INVALID_ARG;
  if (enable && !c->prof_ev) {
    c->prof_cap = 8192;
    c->prof_ev = new cudaEvent_t[2 * c->prof_cap];
    for (int i = 0; i < 2 * c->prof_cap; i++)
      if (cudaEventCreate(&c->prof_ev[i]) != cudaSuccess) return lqcd_check_cuda(c, "profile events");
  }
  c->prof_on = enable ? 1 : 0;
  return LQCD_OK;
}

int lqcd_profile_read(lqcd_ctx* c, long* launches, double* total_ms, double* total_bytes) {
  if (!c || !launches || !total_ms || !total_bytes) return LQCD_ERR_INVALID_ARG;
  double ms = 0;
  for (int i = 0; i < c->prof_n; i++) {
    if (cudaEventSynchronize(c->prof_ev[2 * i + 1]) != cudaSuccess) return lqcd_check_cuda(c, "profile sync");
    float t = 0;
    cudaEventElapsedTime(&t, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]);
    ms += t;
  }
  *launches = c->prof_n;
  *total_ms = ms;
  *total_bytes = c->prof_bytes;
  c->prof_n = 0;
  c->prof_bytes = 0;
  return LQCD_OK;
}

// 16-bit storage (half.cuh): 2 B per real, + one fp32 norm per spinor site, + two per clover site
size_t lqcd_gauge_bytes(const lqcd_ctx* c) { return c ? (size_t)4 * c->V * c->recon * (c->half ? 2 : c->prec) : 0; }
size_t lqcd_spinor_bytes(const lqcd_ctx* c) { return c ? (c->half ? (size_t)c->lat.Vh * 52 : (size_t)c->lat.Vh * 24 * c->prec) : 0; }
size_t lqcd_clover_bytes(const lqcd_ctx* c) { return c ? (c->half ? (size_t)c->V * 152 : (size_t)c->V * 72 * c->prec) : 0; }

}  // extern "C"
