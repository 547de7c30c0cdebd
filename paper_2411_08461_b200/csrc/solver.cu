// Operators M, Mhat and the Krylov solvers (§8(c) O7-O9;
// PAPER.md:94 "BiCGStab for Wilson/clover and CG", PAPER.md:227-230 invert), for nrhs >= 1
// right-hand sides advanced in lock step.  Every "vector" below is a block
// of nrhs consecutive one-parity native spinors; every right-hand side has its own scalar slots,
// coefficients and stopping test.  nrhs = 1 is the single solve and runs the single-RHS kernels.
#include <math.h>
#include <string.h>
#include "blas.cuh"

static inline char* off(const void* p, size_t bytes) { return (char*)p + bytes; }

// reduction slots of one right-hand side (SC_STRIDE doubles each) in ctx->d_scalars
enum { S_BB = 0, S_RR0 = 2, S_RR1 = 3, S_TT = 4, S_RES = 5, S_RHO0 = 8, S_RHO1 = 10, S_R0V = 12, S_TS = 16, S_RR = 20, S_TRUE = 24 };

#define BLAS_CALL(c, OPNAME, SETUP, vecs, outs, nrhs, rhs0, st)                       \
  ((c)->half ? [&]() { OPNAME<float> op; SETUP; return blas_half_launch<OPNAME<float>>((c), op, (vecs), (outs), (nrhs), (rhs0), (st)); }() \
   : (c)->prec == 4 ? [&]() { OPNAME<float> op; SETUP; return blas_launch<float, OPNAME<float>>((c), op, (vecs), (outs), (nrhs), (rhs0), (st)); }() \
                  : [&]() { OPNAME<double> op; SETUP; return blas_launch<double, OPNAME<double>>((c), op, (vecs), (outs), (nrhs), (rhs0), (st)); }())

// all slots of the first nrhs right-hand sides -> pinned host mirror; synchronises the stream
static int read_scalars(lqcd_ctx* c, int nrhs, cudaStream_t st) {
  cudaMemcpyAsync(c->h_scalars, c->d_scalars, sizeof(double) * SC_STRIDE * nrhs, cudaMemcpyDeviceToHost, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return lqcd_check_cuda(c, "scalar read-back");
  return LQCD_OK;
}
static inline double hs(const lqcd_ctx* c, int rhs, int slot) { return c->h_scalars[(size_t)rhs * SC_STRIDE + slot]; }
// write 0.0 / 1.0 into one slot of one right-hand side, or of all of them (stream ordered)
static void set_slot(lqcd_ctx* c, int rhs, int slot, bool one, cudaStream_t st) {
  cudaMemcpyAsync(c->d_scalars + (size_t)rhs * SC_STRIDE + slot, c->h_consts + (one ? 1 : 0), sizeof(double),
                  cudaMemcpyHostToDevice, st);
}
static void set_slot_all(lqcd_ctx* c, int nrhs, int slot, bool one, cudaStream_t st) {
  for (int j = 0; j < nrhs; j++) set_slot(c, j, slot, one, st);
}

// Mhat (O8) on blocks of nrhs one-parity native spinors.  Two fused dslash launches:
//   asym:       tmp = A_oo^-1 D_oe in ; out = A_ee in - k^2 D_eo tmp
//   sym:        tmp = A_oo^-1 D_oe in ; out = in - k^2 A_ee^-1 D_eo tmp
//   sym dagger: out(scratch) = A_ee^-1 in ; tmp = A_oo^-1 D^dag_oe out ; out = in - k^2 D^dag_eo tmp
static int mpc_apply(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* clover,
                     const void* clover_inv, double kappa, int matpc, int dagger, void* tmp, int nrhs, cudaStream_t st) {
  const size_t half = lqcd_clover_bytes(c) / 2;
  const void* A_e = clover;
  const void* Ai_e = clover_inv;
  const void* Ai_o = off(clover_inv, half);
  const double k2 = -kappa * kappa;
  int rc;
  if (matpc == LQCD_MATPC_ASYMMETRIC) {
    if ((rc = lqcd_dslash_launch(c, tmp, in, gauge, Ai_o, nullptr, 1, 1.0, dagger, 1, nrhs, st))) return rc;
    return lqcd_dslash_launch(c, out, tmp, gauge, A_e, in, 0, k2, dagger, 2, nrhs, st);
  }
  if (matpc == LQCD_MATPC_SYMMETRIC_RIGHT) {
    //   right:        out(scratch) = A_ee^-1 in ; tmp = A_oo^-1 D_oe out ; out = in - k^2 D_eo tmp
    //   right dagger: tmp = A_oo^-1 D^dag_oe in ; out = in - k^2 A_ee^-1 D^dag_eo tmp
    if (dagger) {
      if ((rc = lqcd_dslash_launch(c, tmp, in, gauge, Ai_o, nullptr, 1, 1.0, 1, 1, nrhs, st))) return rc;
      return lqcd_dslash_launch(c, out, tmp, gauge, Ai_e, in, 0, k2, 1, 3, nrhs, st);
    }
    if ((rc = lqcd_clover_apply_launch(c, out, in, Ai_e, nrhs, st))) return rc;
    if ((rc = lqcd_dslash_launch(c, tmp, out, gauge, Ai_o, nullptr, 1, 1.0, 0, 1, nrhs, st))) return rc;
    return lqcd_dslash_launch(c, out, tmp, gauge, nullptr, in, 0, k2, 0, 6, nrhs, st);
  }
  if (!dagger) {
    if ((rc = lqcd_dslash_launch(c, tmp, in, gauge, Ai_o, nullptr, 1, 1.0, 0, 1, nrhs, st))) return rc;
    return lqcd_dslash_launch(c, out, tmp, gauge, Ai_e, in, 0, k2, 0, 3, nrhs, st);
  }
  if ((rc = lqcd_clover_apply_launch(c, out, in, Ai_e, nrhs, st))) return rc;
  if ((rc = lqcd_dslash_launch(c, tmp, out, gauge, Ai_o, nullptr, 1, 1.0, 1, 1, nrhs, st))) return rc;
  return lqcd_dslash_launch(c, out, tmp, gauge, nullptr, in, 0, k2, 1, 6, nrhs, st);  // out = in + k2 D^dag_eo tmp
}

// full M (O7): out_p = A_pp in_p - kappa D_{p,1-p} in_{1-p}; fields are [parity][nrhs][one-parity]
static int mat_apply(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* clover, double kappa,
                     int dagger, int nrhs, cudaStream_t st) {
  const size_t blk = lqcd_spinor_bytes(c) * nrhs, half = lqcd_clover_bytes(c) / 2;
  int rc;
  if ((rc = lqcd_dslash_launch(c, out, off(in, blk), gauge, clover, in, 0, -kappa, dagger, 2, nrhs, st))) return rc;
  return lqcd_dslash_launch(c, off(out, blk), in, gauge, off(clover, half), off(in, blk), 1, -kappa, dagger, 2, nrhs, st);
}

static bool check_ptrs(lqcd_ctx* c, const void* const* p, int n, const char* what) {
  for (int i = 0; i < n; i++)
    if (!lqcd_aligned16(p[i])) {
      lqcd_set_error(c, LQCD_ERR_ALIGN, "%s: pointer %d not 16-byte aligned", what, i);
      return false;
    }
  return true;
}

extern "C" {

int lqcd_mpc_apply_mrhs(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* clover,
                        const void* clover_inv, double kappa, int matpc, int dagger, void* tmp, int nrhs, void* stream) {
  if (!c || !out || !in || !gauge || !clover || !clover_inv || !tmp || matpc < 0 || matpc > 2 || nrhs < 1 ||
      nrhs > LQCD_MAX_RHS)
    return LQCD_ERR_INVALID_ARG;
  if (out == in || tmp == in || tmp == out) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "mpc_apply: aliasing");
  const void* p[6] = {out, in, gauge, clover, clover_inv, tmp};
  if (!check_ptrs(c, p, 6, "mpc_apply")) return LQCD_ERR_ALIGN;
  return mpc_apply(c, out, in, gauge, clover, clover_inv, kappa, matpc, dagger ? 1 : 0, tmp, nrhs, as_stream(stream));
}

int lqcd_mpc_apply(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* clover,
                   const void* clover_inv, double kappa, int matpc, int dagger, void* tmp, void* stream) {
  return lqcd_mpc_apply_mrhs(c, out, in, gauge, clover, clover_inv, kappa, matpc, dagger, tmp, 1, stream);
}

int lqcd_mat_apply(lqcd_ctx* c, void* out, const void* in, const void* gauge, const void* clover, double kappa,
                   int dagger, void* stream) {
  if (!c || !out || !in || !gauge || !clover) return LQCD_ERR_INVALID_ARG;
  if (out == in) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "mat_apply: out aliases in");
  const void* p[4] = {out, in, gauge, clover};
  if (!check_ptrs(c, p, 4, "mat_apply")) return LQCD_ERR_ALIGN;
  return mat_apply(c, out, in, gauge, clover, kappa, dagger ? 1 : 0, 1, as_stream(stream));
}

// workspace: nrhs x (2 two-parity + 9 one-parity spinors) (+ clover pair when built inside)
size_t lqcd_invert_multi_workspace_bytes(const lqcd_ctx* c, int solver, int nrhs) {
  (void)solver;
  if (!c || nrhs < 1) return 0;
  return (size_t)nrhs * 13 * lqcd_spinor_bytes(c) + 2 * lqcd_clover_bytes(c);
}
size_t lqcd_invert_workspace_bytes(const lqcd_ctx* c, int solver) { return lqcd_invert_multi_workspace_bytes(c, solver, 1); }

}  // extern "C"

struct Work {
  int nrhs;
  char* b;      // source, [parity][nrhs][one-parity native]
  char* x;      // solution, same layout
  char* v[9];   // scratch blocks of nrhs one-parity spinors
  char* clover; // optional
  char* clover_inv;
};

// per-right-hand-side bookkeeping of a batched solve (host)
struct Cols {
  int n;
  bool active[LQCD_MAX_RHS];
  double stop2[LQCD_MAX_RHS], bb[LQCD_MAX_RHS], rr[LQCD_MAX_RHS];
  int base_it[LQCD_MAX_RHS];  // iterations of earlier passes (residual-replacement restarts, invert_native)
  bool warm;                  // start from the x already in w.x (r = bhat - Mhat x by the operator), not from x = 0
  int nactive() const { int k = 0; for (int j = 0; j < n; j++) k += active[j]; return k; }
};
// freeze column j: its BLAS blocks exit from now on, so x_j, r_j keep the values of this iteration
static void freeze(lqcd_ctx* c, Cols& cols, int j, cudaStream_t st) {
  cols.active[j] = false;
  set_slot(c, j, S_DONE, true, st);
  c->acct_rhs = cols.nactive();
}

// Device-side stopping test, one thread per right-hand side, launched at the end of every Krylov iteration: a column
// whose recurrence residual passed its threshold (or went NaN, or whose BiCGStab rho / omega underflowed) is frozen
// on the device at once, so the host need not look at every iteration: it reads the slots back every `stride`
// iterations only (small lattices, where a blocking read-back per iteration was most of the iteration: 67 us per
// iteration at 4^3x8 against 8 launches of 2-4 us).  The iterations a frozen column sits out change nothing of it.
__global__ void conv_check_kernel(double* scalars, int n, int slot_rr, int slot_rho, int slot_ts) {
  const int j = threadIdx.x;
  if (j >= n) return;
  double* s = scalars + (size_t)j * SC_STRIDE;
  if (s[S_DONE] != 0.0) return;
  s[S_ITERS] += 1.0;
  const double rr = s[slot_rr];
  s[S_RRFIN] = rr;
  if (!(rr == rr)) {
    s[S_FLAG] = 1.0;
    s[S_DONE] = 1.0;
  } else if (!(rr > s[S_STOP])) {
    s[S_DONE] = 1.0;
  } else if (slot_rho >= 0) {
    const double rho = s[slot_rho] * s[slot_rho] + s[slot_rho + 1] * s[slot_rho + 1];
    const double om = s[slot_ts] * s[slot_ts] + s[slot_ts + 1] * s[slot_ts + 1];
    if (rho < 1e-300 || om < 1e-300) {
      s[S_FLAG] = 2.0;
      s[S_DONE] = 1.0;
    }
  }
}
static int conv_check(lqcd_ctx* c, int n, int slot_rr, int slot_rho, int slot_ts, cudaStream_t st) {
  conv_check_kernel<<<1, LQCD_MAX_RHS, 0, st>>>(c->d_scalars, n, slot_rr, slot_rho, slot_ts);
  LQCD_LAUNCH_CHECK(c, "conv_check");
  return LQCD_OK;
}
// thresholds and counters of the device-side test for the columns still active
static void arm_check(lqcd_ctx* c, const Cols& cols, cudaStream_t st) {
  for (int j = 0; j < cols.n; j++) {
    c->h_stop[j] = cols.stop2[j];
    cudaMemcpyAsync(c->d_scalars + (size_t)j * SC_STRIDE + S_STOP, c->h_stop + j, sizeof(double), cudaMemcpyHostToDevice, st);
    set_slot(c, j, S_ITERS, false, st);
    set_slot(c, j, S_FLAG, false, st);
  }
}
// host reads every `stride` iterations: 1 where an iteration is long against a read-back, 4 on the small lattices
static int check_stride(const lqcd_ctx* c, int n) { return (long)c->lat.Vh * n <= 131072 ? 4 : 1; }

// ---- CUDA graphs for the iteration body (SURVEY.md §7 "small-lattice solve time is launch bound: CUDA graphs for the
// iteration body; check convergence every k iterations").  A block of `stride` iterations (an even number, starting at
// an even iteration: the reduction slots alternate with the parity of the iteration) is captured once from the very
// launches the plain path makes, instantiated, and replayed; the instantiated graph is kept in the context and reused
// by later solves as long as every buffer, coefficient and shape it baked in is the same (key).
static unsigned long long mix(unsigned long long h, unsigned long long v) {
  h ^= v + 0x9e3779b97f4a7c15ull + (h << 6) + (h >> 2);
  return h;
}
static unsigned long long graph_key(const lqcd_ctx* c, int tag, const Work& w, const void* gauge, const void* A, const void* Ai,
                                    double kappa, int matpc, int variant, int stride) {
  unsigned long long h = 0x12345 + tag;
  const void* ptrs[] = {w.x, w.v[0], w.v[1], w.v[2], w.v[3], w.v[4], w.v[5], w.v[6], w.v[7], gauge, A, Ai};
  for (const void* p : ptrs) h = mix(h, (unsigned long long)(uintptr_t)p);
  unsigned long long kb, wb;
  memcpy(&kb, &kappa, 8);
  memcpy(&wb, &c->ws, 8);
  h = mix(h, kb);
  h = mix(h, wb);
  h = mix(h, (unsigned long long)w.nrhs << 32 | (unsigned)matpc << 16 | (unsigned)variant << 8 | (unsigned)stride);
  h = mix(h, (unsigned long long)c->part_mask << 8 | (unsigned)c->lat.tb + 2);
  return h | 1;  // never 0: 0 marks an empty slot
}
// runs iterations it0 .. it0+stride-1 as one graph launch; `iterate(it)` enqueues one iteration on `st`
template <typename F>
static int run_block(lqcd_ctx* c, unsigned long long key, int stride, int it0, F& iterate, long& dslashes, cudaStream_t st) {
  for (int i = 0; i < 4; i++)
    if (c->graphs[i].key == key && c->graphs[i].exec) {
      GraphSlot& g = c->graphs[i];
      if (cudaGraphLaunch(g.exec, st) != cudaSuccess) return lqcd_check_cuda(c, "graph launch");
      c->graph_launches++;
      c->launches += g.launches;
      c->alg_bytes += g.bytes;
      dslashes += g.dslashes;
      return LQCD_OK;
    }
  const long l0 = c->launches, d0 = dslashes;
  const double b0 = c->alg_bytes;
  if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
    cudaGetLastError();
    c->graphs_on = 0;
    return -1000;  // not capturable here: the caller falls back to plain launches
  }
  int rc = LQCD_OK;
  for (int i = 0; i < stride && !rc; i++) rc = iterate(it0 + i);
  cudaGraph_t graph = nullptr;
  const cudaError_t e = cudaStreamEndCapture(st, &graph);
  cudaGraphExec_t exec = nullptr;
  if (rc || e != cudaSuccess || cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) {
    if (graph) cudaGraphDestroy(graph);
    cudaGetLastError();
    c->graphs_on = 0;
    c->launches = l0;
    c->alg_bytes = b0;
    dslashes = d0;
    return rc ? rc : -1000;
  }
  cudaGraphDestroy(graph);
  GraphSlot& g = c->graphs[c->graph_next];
  c->graph_next = (c->graph_next + 1) & 3;
  if (g.exec) cudaGraphExecDestroy(g.exec);
  g.key = key;
  g.exec = exec;
  g.launches = c->launches - l0;
  g.bytes = c->alg_bytes - b0;
  g.dslashes = dslashes - d0;
  if (cudaGraphLaunch(exec, st) != cudaSuccess) return lqcd_check_cuda(c, "graph launch");
  c->graph_launches++;
  return LQCD_OK;
}

static int solve_cg(lqcd_ctx* c, const Work& w, const void* gauge, const void* A, const void* Ai, double kappa,
                    int matpc, int normal_residual, Cols& cols, int maxiter, lqcd_result* res, cudaStream_t st) {
  // CGNE (normal_residual = 0): Mhat Mhat^dag y = bhat, x = Mhat^dag y.   bhat in v[0], x_e in w.x
  // CGNR (normal_residual = 1): Mhat^dag Mhat x = Mhat^dag bhat; `resv` tracks bhat - Mhat x
  char *r = w.v[1], *p = w.v[2], *t = w.v[3], *q = w.v[4], *tmp = w.v[5], *resv = w.v[6];
  const int n = w.nrhs;
  const size_t blk = lqcd_spinor_bytes(c) * n;
  char* x = w.x;
  int rc;
  long dslashes = 0;
  // residual of the start vector: x = 0 -> bhat; warm start (residual replacement) -> bhat - Mhat x by the operator
  char* res0 = normal_residual ? resv : r;
  if (!cols.warm) {
    cudaMemsetAsync(x, 0, blk, st);
    cudaMemcpyAsync(res0, w.v[0], blk, cudaMemcpyDeviceToDevice, st);
  } else {
    if ((rc = mpc_apply(c, res0, x, gauge, A, Ai, kappa, matpc, 0, tmp, n, st))) return rc;
    dslashes += 2;
    void* u[2] = {w.v[0], res0};
    if ((rc = BLAS_CALL(c, OpXpay, op.a = -1.0, u, nullptr, n, 0, st))) return rc;  // res0 = bhat - Mhat x
  }
  if (normal_residual) {
    if ((rc = mpc_apply(c, r, resv, gauge, A, Ai, kappa, matpc, 1, tmp, n, st))) return rc;
    dslashes += 2;
  }
  cudaMemcpyAsync(p, r, blk, cudaMemcpyDeviceToDevice, st);
  {
    void* v[1] = {r};
    int outs[4] = {S_RR0, 0, 0, 0};
    if ((rc = BLAS_CALL(c, OpNorm2, (void)op, v, outs, n, 0, st))) return rc;
    void* v2[1] = {normal_residual ? resv : r};
    int outs2[4] = {S_RES, 0, 0, 0};
    if ((rc = BLAS_CALL(c, OpNorm2, (void)op, v2, outs2, n, 0, st))) return rc;
  }
  if ((rc = read_scalars(c, n, st))) return rc;
  for (int j = 0; j < n; j++) {
    if (!cols.active[j]) continue;
    cols.rr[j] = hs(c, j, S_RES);
    if (!(cols.rr[j] > cols.stop2[j])) freeze(c, cols, j, st);
  }
  const bool fused = n == 1 && lqcd_dslash_fuse_ok(c);
  const bool fused_half = n == 1 && c->half && matpc == LQCD_MATPC_SYMMETRIC_RIGHT;  // 16-bit context: epilogues 9, 10 only
  const int stride = check_stride(c, n);
  arm_check(c, cols, st);
  // one iteration, enqueued on `st` (plain launches, or recorded into a graph by run_block)
  auto iterate = [&](int it) -> int {
    const int cur = (it & 1) ? S_RR1 : S_RR0, nxt = (it & 1) ? S_RR0 : S_RR1;
    int outs[4] = {S_TT, 0, 0, 0};
    if (!normal_residual && (fused || fused_half) && matpc == LQCD_MATPC_SYMMETRIC_RIGHT) {
      // right-preconditioned symmetric form, recurrences fused into the epilogues (dslash.cu EPI 9, 10):
      //   tmp = A_oo^-1 D^dag_oe p ; t = p - k^2 A_ee^-1 D^dag_eo tmp, ta = A_ee^-1 t and |t|^2 in one launch ;
      //   tmp = A_oo^-1 D_oe ta ; q = t - k^2 D_eo tmp is never stored: r -= alpha q, |r|^2 in its launch
      const size_t half = lqcd_clover_bytes(c) / 2;
      const double k2 = -kappa * kappa;
      char* ta = q;  // q is not stored in this path
      DslashFuse f9 = {nullptr, S_TT, 0, 0, ta}, f10 = {r, nxt, cur, S_TT, nullptr};
      if ((rc = lqcd_dslash_launch(c, tmp, p, gauge, off(Ai, half), nullptr, 1, 1.0, 1, 1, 1, st))) return rc;
      if ((rc = lqcd_dslash_fused_launch(c, t, tmp, gauge, Ai, p, 0, k2, 1, 9, &f9, st))) return rc;
      if ((rc = lqcd_dslash_launch(c, tmp, ta, gauge, off(Ai, half), nullptr, 1, 1.0, 0, 1, 1, st))) return rc;
      if ((rc = lqcd_dslash_fused_launch(c, nullptr, tmp, gauge, nullptr, t, 0, k2, 0, 10, &f10, st))) return rc;
      void* u[2] = {x, t};
      if ((rc = BLAS_CALL(c, OpAxpyRatio, (op.num = cur, op.den = S_TT), u, nullptr, n, 0, st))) return rc;  // y += a t
    } else if (!normal_residual && n > 1 && matpc == LQCD_MATPC_SYMMETRIC_RIGHT && lqcd_mrhs_fuse_ok(c)) {
      // the same for a batch of columns: per-column |t|^2 and r -= alpha q, |r|^2 in the multi-RHS epilogues 9, 10
      const size_t half = lqcd_clover_bytes(c) / 2;
      const double k2 = -kappa * kappa;
      char* ta = q;
      DslashFuse f9 = {nullptr, S_TT, 0, 0, ta}, f10 = {r, nxt, cur, S_TT, nullptr};
      if ((rc = lqcd_dslash_launch(c, tmp, p, gauge, off(Ai, half), nullptr, 1, 1.0, 1, 1, n, st))) return rc;
      if ((rc = lqcd_dslash_mrhs_fused_launch(c, t, tmp, gauge, Ai, p, 0, k2, 1, 9, n, &f9, st))) return rc;
      if ((rc = lqcd_dslash_launch(c, tmp, ta, gauge, off(Ai, half), nullptr, 1, 1.0, 0, 1, n, st))) return rc;
      if ((rc = lqcd_dslash_mrhs_fused_launch(c, nullptr, tmp, gauge, nullptr, t, 0, k2, 0, 10, n, &f10, st))) return rc;
      void* u[2] = {x, t};
      if ((rc = BLAS_CALL(c, OpAxpyRatio, (op.num = cur, op.den = S_TT), u, nullptr, n, 0, st))) return rc;  // y += a t
    } else if (!normal_residual && fused && matpc == LQCD_MATPC_SYMMETRIC) {
      // symmetric form, recurrences fused into the epilogues (dslash.cu EPI 7, 8):
      //   pa = A_ee^-1 p ; tmp = A_oo^-1 D^dag_oe pa ; t = p - k^2 D^dag_eo tmp and |t|^2 in one launch ;
      //   tmp = A_oo^-1 D_oe t ; q = t - k^2 A_ee^-1 D_eo tmp is never stored: r -= alpha q, |r|^2 in its launch
      const size_t half = lqcd_clover_bytes(c) / 2;
      const double k2 = -kappa * kappa;
      char* pa = q;  // q is not stored in this path
      DslashFuse f7 = {nullptr, S_TT, 0, 0, nullptr}, f8 = {r, nxt, cur, S_TT, nullptr};
      if ((rc = lqcd_clover_apply_launch(c, pa, p, Ai, 1, st))) return rc;
      if ((rc = lqcd_dslash_launch(c, tmp, pa, gauge, off(Ai, half), nullptr, 1, 1.0, 1, 1, 1, st))) return rc;
      if ((rc = lqcd_dslash_fused_launch(c, t, tmp, gauge, nullptr, p, 0, k2, 1, 7, &f7, st))) return rc;
      if ((rc = lqcd_dslash_launch(c, tmp, t, gauge, off(Ai, half), nullptr, 1, 1.0, 0, 1, 1, st))) return rc;
      if ((rc = lqcd_dslash_fused_launch(c, nullptr, tmp, gauge, Ai, t, 0, k2, 0, 8, &f8, st))) return rc;
      void* u[2] = {x, t};
      if ((rc = BLAS_CALL(c, OpAxpyRatio, (op.num = cur, op.den = S_TT), u, nullptr, n, 0, st))) return rc;  // x += a t
    } else if (!normal_residual && fused) {
      // CGNE with the recurrences fused into the dslash epilogues (dslash.cu EPI 4, 5):
      //   t = Mhat^dag p and |t|^2 in one launch; q = Mhat t is never stored: r -= alpha q, |r|^2 in its launch
      const size_t half = lqcd_clover_bytes(c) / 2;
      const double k2 = -kappa * kappa;
      DslashFuse f4 = {nullptr, S_TT, 0, 0, nullptr}, f5 = {r, nxt, cur, S_TT, nullptr};
      if ((rc = lqcd_dslash_launch(c, tmp, p, gauge, off(Ai, half), nullptr, 1, 1.0, 1, 1, 1, st))) return rc;
      if ((rc = lqcd_dslash_fused_launch(c, t, tmp, gauge, A, p, 0, k2, 1, 4, &f4, st))) return rc;
      if ((rc = lqcd_dslash_launch(c, tmp, t, gauge, off(Ai, half), nullptr, 1, 1.0, 0, 1, 1, st))) return rc;
      if ((rc = lqcd_dslash_fused_launch(c, nullptr, tmp, gauge, A, t, 0, k2, 0, 5, &f5, st))) return rc;
      void* u[2] = {x, t};
      if ((rc = BLAS_CALL(c, OpAxpyRatio, (op.num = cur, op.den = S_TT), u, nullptr, n, 0, st))) return rc;  // x += a t
    } else if (!normal_residual) {
      if ((rc = mpc_apply(c, t, p, gauge, A, Ai, kappa, matpc, 1, tmp, n, st))) return rc;   // t = Mhat^dag p
      void* v[1] = {t};
      if ((rc = BLAS_CALL(c, OpNorm2, (void)op, v, outs, n, 0, st))) return rc;              // <p, Mhat Mhat^dag p>
      if ((rc = mpc_apply(c, q, t, gauge, A, Ai, kappa, matpc, 0, tmp, n, st))) return rc;   // q = Mhat t
      void* u[4] = {x, t, r, q};
      int o2[4] = {nxt, 0, 0, 0};
      if ((rc = BLAS_CALL(c, OpCgUpdate, (op.num = cur, op.den = S_TT), u, o2, n, 0, st))) return rc;  // x += a t ; r -= a q
    } else {
      if ((rc = mpc_apply(c, t, p, gauge, A, Ai, kappa, matpc, 0, tmp, n, st))) return rc;   // t = Mhat p
      void* v[1] = {t};
      if ((rc = BLAS_CALL(c, OpNorm2, (void)op, v, outs, n, 0, st))) return rc;
      void* u[4] = {x, p, resv, t};
      int o2[4] = {S_RES, 0, 0, 0};
      if ((rc = BLAS_CALL(c, OpCgUpdate, (op.num = cur, op.den = S_TT), u, o2, n, 0, st))) return rc;  // x += a p ; res -= a t
      if ((rc = mpc_apply(c, q, t, gauge, A, Ai, kappa, matpc, 1, tmp, n, st))) return rc;   // q = Mhat^dag t
      void* u2[2] = {r, q};
      int o3[4] = {nxt, 0, 0, 0};
      if ((rc = BLAS_CALL(c, OpAxmyNormRatio, (op.num = cur, op.den = S_TT), u2, o3, n, 0, st))) return rc;
    }
    dslashes += 4;
    void* u3[2] = {p, r};
    if ((rc = BLAS_CALL(c, OpXpayRatio, (op.num = nxt, op.den = cur), u3, nullptr, n, 0, st))) return rc;  // p = r + beta p
    return conv_check(c, n, normal_residual ? S_RES : nxt, -1, -1, st);
  };
  const bool graphs = c->graphs_on && stride > 1 && !c->prof_on;
  const unsigned long long key = graph_key(c, 1 + normal_residual, w, gauge, A, Ai, kappa, matpc, fused, stride);
  int it = 0, since_read = 0;
  while (it < maxiter && cols.nactive() > 0) {
    bool block = graphs && c->graphs_on && it >= 2 && !(it & 1) && it + stride <= maxiter;
    if (block) {
      rc = run_block(c, key, stride, it, iterate, dslashes, st);
      if (rc == -1000) block = false;
      else if (rc) return rc;
      else {
        it += stride;
        since_read = stride;
      }
    }
    if (!block) {
      if ((rc = iterate(it))) return rc;
      it++;
      since_read++;
    }
    if (since_read < stride && it < maxiter) continue;
    since_read = 0;
    if ((rc = read_scalars(c, n, st))) return rc;
    for (int j = 0; j < n; j++) {
      if (!cols.active[j]) continue;
      cols.rr[j] = hs(c, j, S_RRFIN);
      res[j].iterations = cols.base_it[j] + (int)hs(c, j, S_ITERS);
      if (hs(c, j, S_DONE) == 0.0) continue;
      if (hs(c, j, S_FLAG) != 0.0) res[j].status = LQCD_ERR_BREAKDOWN;
      cols.active[j] = false;  // frozen on the device already
      c->acct_rhs = cols.nactive();
    }
  }
  for (int j = 0; j < n; j++) res[j].dslash_count += dslashes;
  return LQCD_OK;
}

static int solve_bicgstab(lqcd_ctx* c, const Work& w, const void* gauge, const void* A, const void* Ai, double kappa,
                          int matpc, Cols& cols, int maxiter, lqcd_result* res, cudaStream_t st) {
  char *r = w.v[1], *r0 = w.v[2], *p = w.v[3], *v = w.v[4], *s = w.v[6], *t = w.v[7], *tmp = w.v[5];
  const int n = w.nrhs;
  const size_t sp = lqcd_spinor_bytes(c), blk = sp * n;
  char* x = w.x;
  int rc;
  long dslashes = 0;
  bool restarted[LQCD_MAX_RHS] = {false};
  if (!cols.warm) {
    cudaMemsetAsync(x, 0, blk, st);
    cudaMemcpyAsync(r, w.v[0], blk, cudaMemcpyDeviceToDevice, st);
  } else {  // residual replacement: r = bhat - Mhat x by the operator
    if ((rc = mpc_apply(c, r, x, gauge, A, Ai, kappa, matpc, 0, tmp, n, st))) return rc;
    dslashes += 2;
    void* u[2] = {w.v[0], r};
    if ((rc = BLAS_CALL(c, OpXpay, op.a = -1.0, u, nullptr, n, 0, st))) return rc;
  }
  cudaMemcpyAsync(r0, r, blk, cudaMemcpyDeviceToDevice, st);
  {
    // rho_0 = <r0,r> = |r|^2
    void* u[2] = {r0, r};
    int outs[4] = {S_RHO0, S_RHO0 + 1, S_RR, 0};
    if ((rc = BLAS_CALL(c, OpCdot, (void)op, u, outs, n, 0, st))) return rc;
  }
  set_slot_all(c, n, S_FIRST, true, st);  // first iteration: p = r (p, v hold garbage)
  bool first_pending = true;
  if ((rc = read_scalars(c, n, st))) return rc;
  for (int j = 0; j < n; j++) {
    if (!cols.active[j]) continue;
    cols.rr[j] = hs(c, j, S_RR);
    if (!(cols.rr[j] > cols.stop2[j])) freeze(c, cols, j, st);
  }
  const int stride = check_stride(c, n);
  arm_check(c, cols, st);
  // one iteration, enqueued on `st` (plain launches, or recorded into a graph by run_block)
  auto iterate = [&](int it) -> int {
    const int rho = (it & 1) ? S_RHO1 : S_RHO0, rho_next = (it & 1) ? S_RHO0 : S_RHO1;
    {
      void* u[3] = {p, r, v};
      if ((rc = BLAS_CALL(c, OpBicgP, (op.rho = rho, op.r0v = S_R0V, op.ts = S_TS), u, nullptr, n, 0, st))) return rc;
    }
    if (first_pending) {
      set_slot_all(c, n, S_FIRST, false, st);
      first_pending = false;
    }
    // batch of columns, left-symmetric form: <r0,v> and <t,s>, |t|^2 come out of the epilogue that produces v and t
    // (multi-RHS epilogues 12 and 11), two vector passes fewer each
    // (measured: 16^3x32 fp32 6.09 -> 5.60 ms, 32^3x64 fp64 195.8 -> 186.0 ms per 12-column solve); the fused launch runs on
    // the TMA-tiled kernel where that serves epilogue 3, on the register kernel elsewhere.  LQCD_MRHS_FUSE_DOTS=0: off.
    const bool fuse_dots = n > 1 && matpc == LQCD_MATPC_SYMMETRIC && lqcd_mrhs_fuse_ok(c) && c->mrhs_fuse_dots != 0;
    // one column: the same two epilogues in the single-RHS kernel (dslash.cu)
    const bool fuse1 = n == 1 && matpc == LQCD_MATPC_SYMMETRIC && lqcd_dslash_fuse3_ok(c) && c->mrhs_fuse_dots != 0;
    const size_t half = lqcd_clover_bytes(c) / 2;
    const double k2 = -kappa * kappa;
    if (fuse1) {
      DslashFuse f12 = {r0, S_R0V, 0, 0, nullptr};
      if ((rc = lqcd_dslash_launch(c, tmp, p, gauge, off(Ai, half), nullptr, 1, 1.0, 0, 1, 1, st))) return rc;
      if ((rc = lqcd_dslash_fused_launch(c, v, tmp, gauge, Ai, p, 0, k2, 0, 12, &f12, st))) return rc;
    } else if (fuse_dots) {
      DslashFuse f12 = {r0, S_R0V, 0, 0, nullptr};
      if ((rc = lqcd_dslash_launch(c, tmp, p, gauge, off(Ai, half), nullptr, 1, 1.0, 0, 1, n, st))) return rc;
      if ((rc = lqcd_dslash_mrhs_fused_launch(c, v, tmp, gauge, Ai, p, 0, k2, 0, 12, n, &f12, st))) return rc;
    } else {
      if ((rc = mpc_apply(c, v, p, gauge, A, Ai, kappa, matpc, 0, tmp, n, st))) return rc;   // v = Mhat p
      void* u[2] = {r0, v};
      int outs[4] = {S_R0V, S_R0V + 1, S_R0V + 2, 0};
      if ((rc = BLAS_CALL(c, OpCdot, (void)op, u, outs, n, 0, st))) return rc;
    }
    {
      void* u2[3] = {s, r, v};
      if ((rc = BLAS_CALL(c, OpBicgS, (op.rho = rho, op.r0v = S_R0V), u2, nullptr, n, 0, st))) return rc;
    }
    if (fuse1) {
      DslashFuse f11 = {nullptr, S_TS, 0, 0, nullptr};
      if ((rc = lqcd_dslash_launch(c, tmp, s, gauge, off(Ai, half), nullptr, 1, 1.0, 0, 1, 1, st))) return rc;
      if ((rc = lqcd_dslash_fused_launch(c, t, tmp, gauge, Ai, s, 0, k2, 0, 11, &f11, st))) return rc;
    } else if (fuse_dots) {
      DslashFuse f11 = {nullptr, S_TS, 0, 0, nullptr};
      if ((rc = lqcd_dslash_launch(c, tmp, s, gauge, off(Ai, half), nullptr, 1, 1.0, 0, 1, n, st))) return rc;
      if ((rc = lqcd_dslash_mrhs_fused_launch(c, t, tmp, gauge, Ai, s, 0, k2, 0, 11, n, &f11, st))) return rc;
    } else {
      if ((rc = mpc_apply(c, t, s, gauge, A, Ai, kappa, matpc, 0, tmp, n, st))) return rc;   // t = Mhat s
      void* u[2] = {t, s};
      int outs[4] = {S_TS, S_TS + 1, S_TS + 2, 0};
      if ((rc = BLAS_CALL(c, OpCdot, (void)op, u, outs, n, 0, st))) return rc;             // <t,s>, |t|^2
    }
    {
      void* u2[6] = {x, r, p, s, t, r0};
      int o2[4] = {S_RR, rho_next, rho_next + 1, 0};
      if ((rc = BLAS_CALL(c, OpBicgXR, (op.rho = rho, op.r0v = S_R0V, op.ts = S_TS), u2, o2, n, 0, st))) return rc;
    }
    dslashes += 4;
    return conv_check(c, n, S_RR, rho_next, S_TS, st);
  };
  const bool graphs = c->graphs_on && stride > 1 && !c->prof_on;
  const unsigned long long key = graph_key(c, 3, w, gauge, A, Ai, kappa, matpc, 0, stride);
  int it = 0, since_read = 0;
  while (it < maxiter && cols.nactive() > 0) {
    // a block never contains a first iteration (start, or a restarted column): those clear S_FIRST from the host
    bool block = graphs && c->graphs_on && !first_pending && it >= 2 && !(it & 1) && it + stride <= maxiter;
    if (block) {
      rc = run_block(c, key, stride, it, iterate, dslashes, st);
      if (rc == -1000) block = false;
      else if (rc) return rc;
      else {
        it += stride;
        since_read = stride;
      }
    }
    if (!block) {
      if ((rc = iterate(it))) return rc;
      it++;
      since_read++;
    }
    if (since_read < stride && it < maxiter) continue;
    since_read = 0;
    if ((rc = read_scalars(c, n, st))) return rc;
    for (int j = 0; j < n; j++) {
      if (!cols.active[j]) continue;
      cols.rr[j] = hs(c, j, S_RRFIN);
      res[j].iterations = cols.base_it[j] + (int)hs(c, j, S_ITERS);
      if (hs(c, j, S_DONE) == 0.0) continue;
      const double flag = hs(c, j, S_FLAG);
      if (flag == 2.0 && !restarted[j]) {
        // rho or omega underflowed: one restart with r0 = r (O9), for this column only.  The column was frozen at the
        // end of the iteration that broke down; the slots the NEXT iteration reads as rho get <r0, r>.
        restarted[j] = true;
        const int rho_in = (it & 1) ? S_RHO1 : S_RHO0;
        set_slot(c, j, S_FLAG, false, st);
        set_slot(c, j, S_DONE, false, st);
        set_slot(c, j, S_FIRST, true, st);
        first_pending = true;
        cudaMemcpyAsync(r0 + (size_t)j * sp, r + (size_t)j * sp, sp, cudaMemcpyDeviceToDevice, st);
        void* u[2] = {r0, r};
        int outs[4] = {rho_in, rho_in + 1, S_RR, 0};
        if ((rc = BLAS_CALL(c, OpCdot, (void)op, u, outs, 1, j, st))) return rc;
        continue;
      }
      if (flag != 0.0) res[j].status = LQCD_ERR_BREAKDOWN;
      cols.active[j] = false;  // frozen on the device already
      c->acct_rhs = cols.nactive();
    }
  }
  for (int j = 0; j < n; j++) res[j].dslash_count += dslashes;
  return LQCD_OK;
}

static void carve(lqcd_ctx* c, void* workspace, Work& w, int nrhs, bool with_clover) {
  const size_t blk = lqcd_spinor_bytes(c) * nrhs;
  char* p = (char*)workspace;
  w.nrhs = nrhs;
  w.b = p; p += 2 * blk;
  w.x = p; p += 2 * blk;
  for (int i = 0; i < 9; i++) { w.v[i] = p; p += blk; }
  w.clover = with_clover ? p : nullptr;
  w.clover_inv = with_clover ? p + lqcd_clover_bytes(c) : nullptr;
}

// ---------------------------------------------------------------------------------------------
// Mixed precision: fp64 defect correction around fp32 Krylov solves.
//   x = 0, r = bhat;  repeat { e = Mhat^-1 (r/|r|) in fp32 to tol_k ; x += |r| e ; r = bhat - Mhat x in fp64 }
// The fp64 residual is recomputed from x every outer step, so the result meets the same stopping
// test |r_hat| <= tol |b| as the pure fp64 solve; the fp32 inner solves carry ~all the bytes at half
// the width.  tol_k = max(inner_tol, 0.25 * tol|b| / |r|): the last inner solve is not over-solved.
// ---------------------------------------------------------------------------------------------
struct Mixed {
  lqcd_ctx* ci;  // fp32 context (same lattice, boundary, device)
  Work wi;
  const void *gauge, *A, *Ai;  // fp32 natives
  double inner_tol;
};

__global__ void __launch_bounds__(256) spinor_down_kernel(float4* __restrict__ out, const double2* __restrict__ in, int Vh,
                                                          double scale) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= Vh) return;
#pragma unroll
  for (int u = 0; u < 6; u++) {
    const double2 a = in[(size_t)(2 * u) * Vh + i], b = in[(size_t)(2 * u + 1) * Vh + i];
    out[(size_t)u * Vh + i] = make_float4((float)(scale * a.x), (float)(scale * a.y), (float)(scale * b.x), (float)(scale * b.y));
  }
}
__global__ void __launch_bounds__(256) spinor_up_axpy_kernel(double2* __restrict__ x, const float4* __restrict__ e, int Vh,
                                                             double a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= Vh) return;
#pragma unroll
  for (int u = 0; u < 6; u++) {
    const float4 v = e[(size_t)u * Vh + i];
    double2 p = x[(size_t)(2 * u) * Vh + i], q = x[(size_t)(2 * u + 1) * Vh + i];
    p.x += a * v.x; p.y += a * v.y; q.x += a * v.z; q.y += a * v.w;
    x[(size_t)(2 * u) * Vh + i] = p;
    x[(size_t)(2 * u + 1) * Vh + i] = q;
  }
}

static int solve_cg(lqcd_ctx* c, const Work& w, const void* gauge, const void* A, const void* Ai, double kappa,
                    int matpc, int normal_residual, Cols& cols, int maxiter, lqcd_result* res, cudaStream_t st);
static int solve_bicgstab(lqcd_ctx* c, const Work& w, const void* gauge, const void* A, const void* Ai, double kappa,
                          int matpc, Cols& cols, int maxiter, lqcd_result* res, cudaStream_t st);

// bhat in w.v[0], x_e (zeroed) in w.x, w.nrhs columns in lock step: every outer step runs ONE batched fp32 solve
// over the columns still above their fp64 stopping test (the others are frozen in the inner solve and skipped
// in the fp64 update); fills cols.rr[j], res[j].iterations (inner iterations that column took part in).
// The last outer step needs no fp64 Schur residual of its own: when the inner recurrences say that every live column
// will be below its bar (|r|^2 * (inner relative residual)^2 <= 0.9 stop^2), the closing steps of the solve
// (`closing`: x_o and the TRUE residual of the full operator into true_rr, which the caller owes anyway) decide.  If
// they pass, *closed = true and cols.rr is the recurrence's estimate |r|^2 * (inner relative residual)^2; if not,
// `reopen` undoes what the closing steps did to x and the loop goes on as usual.
// A wrong guess costs one closing pass (x_o and the true residual, about 1.5 fp64 M-hat) and nothing else;
// LQCD_MIXED_LAST_MARGIN (read at context creation; default 0.9, 0 = never guess) is the factor, and the tests set it
// huge to force wrong guesses through `reopen`.
template <class Closing, class Reopen>
static int solve_mixed(lqcd_ctx* c, const Work& w, const void* gauge, const void* A, const void* Ai, double kappa,
                       int matpc, int solver, Cols& cols, int maxiter, lqcd_result* res, Mixed& m, cudaStream_t st,
                       Closing&& closing, Reopen&& reopen, const double* true_rr, bool* closed) {
  lqcd_ctx* ci = m.ci;
  char *bh = w.v[0], *r = w.v[1], *mx = w.v[2], *tmp = w.v[5], *x = w.x;
  const int n = w.nrhs;
  const size_t sp = lqcd_spinor_bytes(c), spi = lqcd_spinor_bytes(ci);
  const int Vh = c->lat.Vh, grid = (Vh + 255) / 256;
  int rc;
  cudaMemcpyAsync(r, bh, sp * n, cudaMemcpyDeviceToDevice, st);
  double rr[LQCD_MAX_RHS];
  bool live[LQCD_MAX_RHS];
  int iters[LQCD_MAX_RHS];
  {
    void* v[1] = {r};
    int o[4] = {S_RES, 0, 0, 0};
    if ((rc = BLAS_CALL(c, OpNorm2, (void)op, v, o, n, 0, st))) return rc;
    if ((rc = read_scalars(c, n, st))) return rc;
  }
  int nlive = 0;
  for (int j = 0; j < n; j++) {
    rr[j] = cols.active[j] ? hs(c, j, S_RES) : 0.0;
    live[j] = cols.active[j] && rr[j] > cols.stop2[j];
    iters[j] = 0;
    nlive += live[j];
  }
  int total = 0, outer = 0;
  while (nlive > 0 && total < maxiter && outer < 64) {
    Cols ic;
    ic.n = n;
    ic.warm = false;
    cudaMemsetAsync(ci->d_scalars, 0, sizeof(double) * SC_STRIDE * n, st);
    double rn[LQCD_MAX_RHS];
    for (int j = 0; j < n; j++) {
      ic.active[j] = live[j];
      ic.base_it[j] = 0;
      ic.bb[j] = 1.0;
      ic.rr[j] = 1.0;
      ic.stop2[j] = 1.0;
      if (!live[j]) {
        set_slot(ci, j, S_DONE, true, st);
        continue;
      }
      rn[j] = sqrt(rr[j]);
      if (ci->half) {
        if ((rc = lqcd_spinor_down_half(c, m.wi.v[0] + j * spi, r + j * sp, 1.0 / rn[j], st))) return rc;
      } else {
        spinor_down_kernel<<<grid, 256, 0, st>>>((float4*)(m.wi.v[0] + j * spi), (const double2*)(r + j * sp), Vh, 1.0 / rn[j]);
        c->alg_bytes += (double)Vh * 24 * 12;
        LQCD_LAUNCH_CHECK(c, "spinor_down");
      }
      // inner fp32 solve of Mhat e = r/|r|, relative tolerance tol_k
      const double need = 0.25 * sqrt(cols.stop2[j] / rr[j]);
      const double tol_k = need > m.inner_tol ? need : m.inner_tol;
      ic.stop2[j] = tol_k * tol_k;
    }
    lqcd_result ri[LQCD_MAX_RHS];
    memset(ri, 0, sizeof(ri));
    ci->acct_rhs = nlive;
    if (solver == LQCD_SOLVER_BICGSTAB) rc = solve_bicgstab(ci, m.wi, m.gauge, m.A, m.Ai, kappa, matpc, ic, maxiter - total, ri, st);
    else rc = solve_cg(ci, m.wi, m.gauge, m.A, m.Ai, kappa, matpc, solver == LQCD_SOLVER_CGNR, ic, maxiter - total, ri, st);
    ci->acct_rhs = 0;
    if (rc) return lqcd_set_error(c, rc, "invert_mixed: inner solve: %s", ci->err);
    int step = 0;
    bool broke = false;
    for (int j = 0; j < n; j++) {
      if (!live[j]) continue;
      iters[j] += ri[j].iterations;
      step = ri[j].iterations > step ? ri[j].iterations : step;
      res[j].dslash_count += ri[j].dslash_count;
      if (ri[j].status < 0) { res[j].status = ri[j].status; live[j] = false; nlive--; broke = true; continue; }
      // x += |r| e
      if (ci->half) {
        if ((rc = lqcd_spinor_up_axpy_half(c, x + j * sp, m.wi.x + j * spi, rn[j], st))) return rc;
      } else {
        spinor_up_axpy_kernel<<<grid, 256, 0, st>>>((double2*)(x + j * sp), (const float4*)(m.wi.x + j * spi), Vh, rn[j]);
        c->alg_bytes += (double)Vh * 24 * 20;
        LQCD_LAUNCH_CHECK(c, "spinor_up_axpy");
      }
    }
    total += step;
    if (broke && n == 1) break;
    // |r|^2 times the inner recurrence's (|r_inner| / |rhs|)^2 at exit estimates the next fp64 residual
    bool expect_last = !broke;
    for (int j = 0; j < n; j++) expect_last = expect_last && (!live[j] || rr[j] * ic.rr[j] <= c->mixed_last_margin * cols.stop2[j]);
    if (expect_last) {
      if ((rc = closing())) return rc;
      bool pass = true;
      for (int j = 0; j < n; j++) pass = pass && (!live[j] || !(true_rr[j] > cols.stop2[j]));
      if (pass) {
        for (int j = 0; j < n; j++)
          if (live[j]) {
            rr[j] *= ic.rr[j];  // the inner recurrence's |r|^2 / |rhs|^2 at exit
            if (true_rr[j] < rr[j]) rr[j] = true_rr[j];  // the estimate never reports worse than what was measured
            live[j] = false;
          }
        nlive = 0;
        *closed = true;
        break;
      }
      if ((rc = reopen())) return rc;
    }
    // r = bhat - Mhat x in fp64, all columns (a frozen column reproduces its residual)
    if ((rc = mpc_apply(c, mx, x, gauge, A, Ai, kappa, matpc, 0, tmp, n, st))) return rc;
    for (int j = 0; j < n; j++) res[j].dslash_count += 2;
    {
      void* v[2] = {bh, mx};
      int o[4] = {S_RES, 0, 0, 0};
      if ((rc = BLAS_CALL(c, OpXpayNorm, op.a = -1.0, v, o, n, 0, st))) return rc;  // mx = bhat - Mhat x and its norm, one pass
      if ((rc = read_scalars(c, n, st))) return rc;
    }
    char* sw = r; r = mx; mx = sw;
    outer++;
    for (int j = 0; j < n; j++) {
      if (!live[j]) continue;
      const double rr_new = hs(c, j, S_RES);
      const bool nan = !(rr_new == rr_new), stalled = rr_new > 0.81 * rr[j];  // fp32 solves no longer reduce the fp64 residual
      rr[j] = rr_new;
      if (nan) res[j].status = LQCD_ERR_BREAKDOWN;
      if (nan || stalled || !(rr_new > cols.stop2[j])) { live[j] = false; nlive--; }
    }
  }
  for (int j = 0; j < n; j++) {
    if (!cols.active[j]) continue;
    cols.rr[j] = rr[j];
    res[j].iterations = iters[j];
  }
  return LQCD_OK;
}

// the whole solve on native fields already in w.b; result in w.x (both parities).
// Residual replacement (SURVEY.md §7 "add a reliable-update restart if the true residual misses"): the Krylov loops
// stop on the recurrence residual; the solve then closes with x_o (a10) and the true residual |b - M x| of the full
// operator (a11), which costs nothing extra.  A column whose recurrence converged but whose TRUE residual is still
// above tol |b| (an fp32 recurrence drifts from the true residual near 2e-7; the left-symmetric form stops on
// |A_ee^-1 r_hat|) is restarted from its x: r = bhat - Mhat x recomputed with the operator replaces the recurrence
// residual and the iteration goes on to a target tightened by 1/2 per pass, the other columns frozen.  At most
// MAX_PASSES passes; a column that no longer improves stops.  status = NOT_CONVERGED if the true residual stays
// above tol |b| (the precision floor of the storage type).
static int invert_native_body(lqcd_ctx* c, Work& w, const void* gauge, const void* A, const void* Ai, double kappa,
                              double tol, int maxiter, int solver, int matpc, lqcd_result* res, cudaStream_t st,
                              Mixed* mixed) {
  constexpr int MAX_PASSES = 4;
  const int n = w.nrhs;
  const size_t sp = lqcd_spinor_bytes(c), blk = sp * n, half = lqcd_clover_bytes(c) / 2;
  const void* Ai_e = Ai;
  const void* Ai_o = off(Ai, half);
  char *b_e = w.b, *b_o = w.b + blk, *x_e = w.x, *x_o = w.x + blk;
  int rc;
  cudaMemsetAsync(c->d_scalars, 0, sizeof(double) * SC_STRIDE * n, st);  // clears S_DONE / S_FIRST too
  c->acct_rhs = 0;
  // |b|^2 over both parities
  {
    void* v[1] = {b_e};
    int o[4] = {S_BB, 0, 0, 0};
    if ((rc = BLAS_CALL(c, OpNorm2, (void)op, v, o, n, 0, st))) return rc;
    void* v2[1] = {b_o};
    int o2[4] = {S_BB + 1, 0, 0, 0};
    if ((rc = BLAS_CALL(c, OpNorm2, (void)op, v2, o2, n, 0, st))) return rc;
  }
  if ((rc = read_scalars(c, n, st))) return rc;
  Cols cols;
  cols.n = n;
  cols.warm = false;
  double stop2[LQCD_MAX_RHS], true_rr[LQCD_MAX_RHS];
  bool solvable[LQCD_MAX_RHS];
  for (int j = 0; j < n; j++) {
    cols.bb[j] = hs(c, j, S_BB) + hs(c, j, S_BB + 1);
    const bool finite = cols.bb[j] == cols.bb[j] && cols.bb[j] <= 1.7e308;
    stop2[j] = cols.stop2[j] = tol * tol * cols.bb[j];
    cols.rr[j] = 0;
    cols.base_it[j] = 0;
    true_rr[j] = 0;
    // a zero source has the zero solution: nothing to iterate; a non-finite source cannot be solved
    solvable[j] = cols.active[j] = finite && cols.bb[j] > 0.0;
    res[j].status = finite ? LQCD_OK : LQCD_ERR_BREAKDOWN;
  }
  cudaMemsetAsync(w.x, 0, 2 * blk, st);
  if (cols.nactive() == 0) return LQCD_OK;
  // a5: bhat = b_e + kappa D_eo A_oo^-1 b_o   (sym: bhat_s = A_ee^-1 bhat)
  char* bh = w.v[0];
  if ((rc = lqcd_clover_apply_launch(c, w.v[5], b_o, Ai_o, n, st))) return rc;
  // the sum rides on the hop (epilogue 6: x + scale * d), one vector pass less; in a batch the clover factor of the
  // left-symmetric form rides too (multi-RHS epilogue 14: C (x + scale * d))
  const bool ride = n > 1 ? lqcd_mrhs_fuse_ok(c) : (!c->half && lqcd_dslash_fuse_ok(c));
  if (matpc == LQCD_MATPC_SYMMETRIC && ride) {
    if ((rc = lqcd_dslash_launch(c, bh, w.v[5], gauge, Ai_e, b_e, 0, kappa, 0, 14, n, st))) return rc;
  } else {
    if ((rc = lqcd_dslash_launch(c, bh, w.v[5], gauge, nullptr, b_e, 0, kappa, 0, 6, n, st))) return rc;
    if (matpc == LQCD_MATPC_SYMMETRIC)
      if ((rc = lqcd_clover_apply_launch(c, bh, bh, Ai_e, n, st))) return rc;
  }
  // closing steps for n columns given by their own pointers (all columns of the batch, or one column of it):
  // unknown back to x_e (right-preconditioned form), a10: x_o = A_oo^-1 (b_o + kappa D_oe x_e), a11: the true residual
  // b - M x with the full operator into (r1, r2), its norms into S_TRUE, S_TRUE + 1
  auto finish = [&](char* be, char* bo, char* xe, char* xo, char* r1, char* r2, char* t5, int m) -> int {
    int e;
    if (matpc == LQCD_MATPC_SYMMETRIC_RIGHT)     // the Krylov unknown was y = A_ee x_e
      if ((e = lqcd_clover_apply_launch(c, xe, xe, Ai_e, m, st))) return e;
    const bool ride1 = m == 1 && !c->half && lqcd_dslash_fuse_ok(c);  // one column: the same epilogues in dslash.cu
    if ((m > 1 && lqcd_mrhs_fuse_ok(c)) || ride1) {  // x_o = A_oo^-1 (b_o + kappa D_oe x_e) in one launch
      if ((e = lqcd_dslash_launch(c, xo, xe, gauge, Ai_o, bo, 1, kappa, 0, 14, m, st))) return e;
    } else {
      if ((e = lqcd_dslash_launch(c, t5, xe, gauge, nullptr, bo, 1, kappa, 0, 6, m, st))) return e;  // b_o + kappa D_oe x_e
      if ((e = lqcd_clover_apply_launch(c, xo, t5, Ai_o, m, st))) return e;
    }
    if (m > 1 && lqcd_mrhs_fuse_ok(c)) {
      // batch: each parity of A x - kappa D x goes straight into |b - (...)|^2 (multi-RHS epilogue 13), nothing is stored
      DslashFuse fe = {be, S_TRUE, 0, 0, nullptr}, fo = {bo, S_TRUE + 1, 0, 0, nullptr};
      if ((e = lqcd_dslash_mrhs_fused_launch(c, nullptr, xo, gauge, A, xe, 0, -kappa, 0, 13, m, &fe, st))) return e;
      if ((e = lqcd_dslash_mrhs_fused_launch(c, nullptr, xe, gauge, off(A, half), xo, 1, -kappa, 0, 13, m, &fo, st))) return e;
      return read_scalars(c, m, st);
    }
    if (ride1) {
      DslashFuse fe = {be, S_TRUE, 0, 0, nullptr}, fo = {bo, S_TRUE + 1, 0, 0, nullptr};
      if ((e = lqcd_dslash_fused_launch(c, nullptr, xo, gauge, A, xe, 0, -kappa, 0, 13, &fe, st))) return e;
      if ((e = lqcd_dslash_fused_launch(c, nullptr, xe, gauge, off(A, half), xo, 1, -kappa, 0, 13, &fo, st))) return e;
      return read_scalars(c, 1, st);
    }
    if ((e = lqcd_dslash_launch(c, r1, xo, gauge, A, xe, 0, -kappa, 0, 2, m, st))) return e;
    if ((e = lqcd_dslash_launch(c, r2, xe, gauge, off(A, half), xo, 1, -kappa, 0, 2, m, st))) return e;
    {
      void* v[2] = {be, r1};
      int o[4] = {S_TRUE, 0, 0, 0};
      if ((e = BLAS_CALL(c, OpAxpyNorm, op.a = -1.0, v, o, m, 0, st))) return e;
      void* v2[2] = {bo, r2};
      int o2[4] = {S_TRUE + 1, 0, 0, 0};
      if ((e = BLAS_CALL(c, OpAxpyNorm, op.a = -1.0, v2, o2, m, 0, st))) return e;
    }
    return read_scalars(c, m, st);
  };
  // pass 0: all columns in lock step
  for (int j = 0; j < n; j++)
    if (!cols.active[j]) set_slot(c, j, S_DONE, true, st);
  c->acct_rhs = cols.nactive();
  bool closed = false;  // the closing steps already ran on the final x (mixed solve, last outer step)
  auto closing = [&]() -> int {
    set_slot_all(c, n, S_DONE, false, st);  // the closing steps update every column
    const int e = finish(b_e, b_o, x_e, x_o, w.v[1], w.v[2], w.v[5], n);
    for (int j = 0; j < n && !e; j++) true_rr[j] = solvable[j] ? hs(c, j, S_TRUE) + hs(c, j, S_TRUE + 1) : 0.0;
    return e;
  };
  auto reopen = [&]() -> int {
    if (matpc == LQCD_MATPC_SYMMETRIC_RIGHT)  // back to the Krylov unknown y = A_ee x_e
      if (int e = lqcd_clover_apply_launch(c, x_e, x_e, A, n, st)) return e;
    for (int j = 0; j < n; j++)
      if (!solvable[j]) set_slot(c, j, S_DONE, true, st);
    return LQCD_OK;
  };
  if (mixed) rc = solve_mixed(c, w, gauge, A, Ai, kappa, matpc, solver, cols, maxiter, res, *mixed, st, closing, reopen, true_rr, &closed);
  else if (solver == LQCD_SOLVER_BICGSTAB) rc = solve_bicgstab(c, w, gauge, A, Ai, kappa, matpc, cols, maxiter, res, st);
  else rc = solve_cg(c, w, gauge, A, Ai, kappa, matpc, solver == LQCD_SOLVER_CGNR, cols, maxiter, res, st);
  c->acct_rhs = 0;
  if (rc) return rc;
  if (!closed && (rc = closing())) return rc;
  for (int j = 0; j < n; j++) res[j].dslash_count += 4;  // prepare, reconstruct, two for the true residual
  // residual replacement, column by column (a one-column view of the batch: the single-RHS kernels run, the other
  // columns are not touched): only where the recurrence converged and the true residual is still above the bar
  for (int j = 0; j < n && !mixed; j++) {
    if (!solvable[j] || res[j].status != LQCD_OK) continue;
    Work w1 = w;
    w1.nrhs = 1;
    w1.x = x_e + j * sp;
    for (int i = 0; i < 9; i++) w1.v[i] = w.v[i] + j * sp;
    double target = stop2[j];
    for (int pass = 1; pass < MAX_PASSES; pass++) {
      if (cols.rr[j] > target || !(true_rr[j] > stop2[j]) || res[j].iterations >= maxiter) break;
      target *= 0.25;
      if (matpc == LQCD_MATPC_SYMMETRIC_RIGHT)  // back to the Krylov unknown y = A_ee x_e
        if ((rc = lqcd_clover_apply_launch(c, w1.x, w1.x, A, 1, st))) return rc;
      Cols c1;
      c1.n = 1;
      c1.warm = true;
      c1.active[0] = true;
      c1.stop2[0] = target;
      c1.bb[0] = cols.bb[j];
      c1.rr[0] = cols.rr[j];
      c1.base_it[0] = res[j].iterations;
      c->acct_rhs = 1;
      const int left = maxiter - res[j].iterations;
      if (solver == LQCD_SOLVER_BICGSTAB) rc = solve_bicgstab(c, w1, gauge, A, Ai, kappa, matpc, c1, left, res + j, st);
      else rc = solve_cg(c, w1, gauge, A, Ai, kappa, matpc, solver == LQCD_SOLVER_CGNR, c1, left, res + j, st);
      c->acct_rhs = 0;
      if (rc) return rc;
      set_slot(c, 0, S_DONE, false, st);
      if ((rc = finish(b_e + j * sp, b_o + j * sp, w1.x, x_o + j * sp, w1.v[1], w1.v[2], w1.v[5], 1))) return rc;
      res[j].dslash_count += 3;
      cols.rr[j] = c1.rr[0];
      const double t2 = hs(c, 0, S_TRUE) + hs(c, 0, S_TRUE + 1), before = true_rr[j];
      true_rr[j] = t2;
      if (res[j].status != LQCD_OK || !(t2 < 0.5 * before)) break;  // no longer improving: the floor of the storage type
    }
    cols.stop2[j] = target;
  }
  for (int j = 0; j < n; j++) {
    if (!solvable[j]) continue;
    res[j].iter_resid = sqrt(cols.rr[j] / cols.bb[j]);
    res[j].true_resid = sqrt(true_rr[j] / cols.bb[j]);
    if (res[j].status == LQCD_OK && (cols.rr[j] > stop2[j] || true_rr[j] > stop2[j])) res[j].status = LQCD_NOT_CONVERGED;
  }
  return LQCD_OK;
}

// freeze flags and the first-iteration flag never outlive a solve, whatever path it returned by: the public
// lqcd_blas_* calls and the next solve on this context (or on the inner context of a mixed solve) start clean
static int invert_native(lqcd_ctx* c, Work& w, const void* gauge, const void* A, const void* Ai, double kappa,
                         double tol, int maxiter, int solver, int matpc, lqcd_result* res, cudaStream_t st,
                         Mixed* mixed = nullptr) {
  const int rc = invert_native_body(c, w, gauge, A, Ai, kappa, tol, maxiter, solver, matpc, res, st, mixed);
  c->acct_rhs = 0;
  set_slot_all(c, w.nrhs, S_DONE, false, st);
  set_slot_all(c, w.nrhs, S_FIRST, false, st);
  if (mixed) {
    mixed->ci->acct_rhs = 0;
    set_slot_all(mixed->ci, w.nrhs, S_DONE, false, st);
    set_slot_all(mixed->ci, w.nrhs, S_FIRST, false, st);
  }
  return rc;
}

static int worst_status(const lqcd_result* res, int n) {
  int worst = LQCD_OK;
  for (int j = 0; j < n; j++) {
    if (res[j].status < 0) worst = (worst < 0 && worst < res[j].status) ? worst : res[j].status;
    else if (res[j].status > 0 && worst == LQCD_OK) worst = res[j].status;
  }
  return worst;
}

static int invert_common(lqcd_ctx* c, void* x_public, const void* b_public, const void* gauge, const void* clover,
                         const void* clover_inv, double kappa, double csw, double tol, int maxiter, int solver,
                         int matpc, int nrhs, void* workspace, size_t workspace_bytes, lqcd_result* res, cudaStream_t st,
                         Mixed* mixed = nullptr) {
  if (!c || !x_public || !b_public || !gauge || !workspace || !res) return LQCD_ERR_INVALID_ARG;
  if (solver < 0 || solver > 2 || matpc < 0 || matpc > 2 || maxiter < 0 || !(tol >= 0) || (clover && !clover_inv) ||
      nrhs < 1 || nrhs > LQCD_MAX_RHS || (c->half && (nrhs > 1 || !clover)))
    return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "invert: bad solver/matpc/maxiter/tol/nrhs (16-bit context: one column, clover fields required)");
  if (workspace_bytes < lqcd_invert_multi_workspace_bytes(c, solver, nrhs))
    return lqcd_set_error(c, LQCD_ERR_WORKSPACE, "invert: workspace %zu < %zu", workspace_bytes,
                          lqcd_invert_multi_workspace_bytes(c, solver, nrhs));
  const void* p[6] = {x_public, b_public, gauge, clover, clover_inv, workspace};
  if (!check_ptrs(c, p, 6, "invert")) return LQCD_ERR_ALIGN;
  memset(res, 0, sizeof(*res) * nrhs);
  // A small-lattice solve replays its iterations as CUDA graphs, and the legacy default stream (what PyTorch hands out
  // unless told otherwise) cannot be captured: such a solve runs on a stream of the context, ordered after the work
  // already queued on the caller's stream; the call synchronises before it returns, as lqcd_invert always does.
  if (c->graphs_on && (st == nullptr || st == cudaStreamLegacy) && check_stride(c, nrhs) > 1) {
    cudaEventRecord(c->ev_graph, st);
    cudaStreamWaitEvent(c->graph_stream, c->ev_graph, 0);
    st = c->graph_stream;
  }
  const long launches0 = c->launches, mixed_launches0 = mixed ? mixed->ci->launches : 0;
  const size_t sp = lqcd_spinor_bytes(c);
  const size_t psp = (size_t)c->lat.Vh * 24 * c->prec;  // one parity of a PUBLIC spinor (16-bit context: complex64)
  Work w;
  carve(c, workspace, w, nrhs, clover == nullptr);
  int rc;
  cudaEventRecord(c->ev0, st);
  if (!clover) {
    void* s = (void*)st;
    if ((rc = lqcd_clover_build(c, w.clover, w.clover_inv, gauge, csw, kappa, s))) return rc;
    clover = w.clover;
    clover_inv = w.clover_inv;
  }
  for (int j = 0; j < nrhs; j++)
    for (int par = 0; par < 2; par++)
      if ((rc = lqcd_spinor_pack_parity(c, w.b + ((size_t)par * nrhs + j) * sp,
                                        (const char*)b_public + ((size_t)2 * j + par) * psp, st))) return rc;
  if ((rc = invert_native(c, w, gauge, clover, clover_inv, kappa, tol, maxiter, solver, matpc, res, st, mixed))) return rc;
  for (int j = 0; j < nrhs; j++)
    for (int par = 0; par < 2; par++)
      if ((rc = lqcd_spinor_unpack_parity(c, (char*)x_public + ((size_t)2 * j + par) * psp,
                                          w.x + ((size_t)par * nrhs + j) * sp, st))) return rc;
  cudaEventRecord(c->ev1, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return lqcd_check_cuda(c, "invert sync");
  float ms = 0;
  cudaEventElapsedTime(&ms, c->ev0, c->ev1);
  for (int j = 0; j < nrhs; j++) {
    res[j].seconds = ms * 1e-3;  // of the whole (batched) call
    res[j].kernel_launches = c->launches - launches0 + (mixed ? mixed->ci->launches - mixed_launches0 : 0);
  }
  return worst_status(res, nrhs);
}

extern "C" {

int lqcd_invert(lqcd_ctx* c, void* x_public, const void* b_public, const void* gauge, const void* clover,
                const void* clover_inv, double kappa, double csw, double tol, int maxiter, int solver, int matpc,
                void* workspace, size_t workspace_bytes, lqcd_result* res, void* stream) {
  return invert_common(c, x_public, b_public, gauge, clover, clover_inv, kappa, csw, tol, maxiter, solver, matpc, 1,
                       workspace, workspace_bytes, res, as_stream(stream));
}

int lqcd_invert_multi(lqcd_ctx* c, void* x_public, const void* b_public, const void* gauge, const void* clover,
                      const void* clover_inv, double kappa, double tol, int maxiter, int solver, int matpc, int nrhs,
                      void* workspace, size_t workspace_bytes, lqcd_result* res, void* stream) {
  if (!clover || !clover_inv) return LQCD_ERR_INVALID_ARG;
  return invert_common(c, x_public, b_public, gauge, clover, clover_inv, kappa, 0.0, tol, maxiter, solver, matpc, nrhs,
                       workspace, workspace_bytes, res, as_stream(stream));
}

int lqcd_invert_multi_mixed(lqcd_ctx* c, lqcd_ctx* ci, void* x_public, const void* b_public, const void* gauge,
                            const void* clover, const void* clover_inv, const void* gauge_lo, const void* clover_lo,
                            const void* clover_inv_lo, double kappa, double tol, double inner_tol, int maxiter, int solver,
                            int matpc, int nrhs, void* workspace, size_t workspace_bytes, void* workspace_lo,
                            size_t workspace_lo_bytes, lqcd_result* res, void* stream) {
  if (!c || !ci || !clover || !clover_inv || !gauge_lo || !clover_lo || !clover_inv_lo || !workspace_lo)
    return LQCD_ERR_INVALID_ARG;
  if (c->prec != 8 || ci->prec != 4 || c->device != ci->device || c->lat.tb != ci->lat.tb || c->L[0] != ci->L[0] ||
      c->L[1] != ci->L[1] || c->L[2] != ci->L[2] || c->L[3] != ci->L[3] || !(inner_tol > 0) || !(inner_tol < 1) ||
      nrhs < 1 || nrhs > LQCD_MAX_RHS || c->half || (ci->half && nrhs > 1))
    return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "invert_mixed: needs an fp64 and an fp32 (or, one column, 16-bit) context of the same lattice");
  if (workspace_lo_bytes < lqcd_invert_multi_workspace_bytes(ci, solver, nrhs))
    return lqcd_set_error(c, LQCD_ERR_WORKSPACE, "invert_mixed: low-precision workspace too small");
  const void* p[4] = {gauge_lo, clover_lo, clover_inv_lo, workspace_lo};
  if (!check_ptrs(c, p, 4, "invert_mixed")) return LQCD_ERR_ALIGN;
  Mixed m;
  m.ci = ci;
  carve(ci, workspace_lo, m.wi, nrhs, false);
  m.gauge = gauge_lo;
  m.A = clover_lo;
  m.Ai = clover_inv_lo;
  m.inner_tol = inner_tol;
  return invert_common(c, x_public, b_public, gauge, clover, clover_inv, kappa, 0.0, tol, maxiter, solver, matpc, nrhs,
                       workspace, workspace_bytes, res, as_stream(stream), &m);
}

int lqcd_invert_mixed(lqcd_ctx* c, lqcd_ctx* ci, void* x_public, const void* b_public, const void* gauge,
                      const void* clover, const void* clover_inv, const void* gauge_lo, const void* clover_lo,
                      const void* clover_inv_lo, double kappa, double tol, double inner_tol, int maxiter, int solver,
                      int matpc, void* workspace, size_t workspace_bytes, void* workspace_lo, size_t workspace_lo_bytes,
                      lqcd_result* res, void* stream) {
  return lqcd_invert_multi_mixed(c, ci, x_public, b_public, gauge, clover, clover_inv, gauge_lo, clover_lo, clover_inv_lo,
                                 kappa, tol, inner_tol, maxiter, solver, matpc, 1, workspace, workspace_bytes, workspace_lo,
                                 workspace_lo_bytes, res, stream);
}

size_t lqcd_host_scratch_bytes(const lqcd_ctx* c, int solver) {
  return c ? 4 * lqcd_spinor_bytes(c) + lqcd_invert_workspace_bytes(c, solver) : 0;
}

int lqcd_gauge_pack_host(lqcd_ctx* c, void* native, const void* pub_host, void* scratch, void* stream) {
  if (!c || !native || !pub_host || !scratch) return LQCD_ERR_INVALID_ARG;
  if (c->half) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "gauge_pack_host: not available in a 16-bit context");
  cudaStream_t st = as_stream(stream);
  cudaMemcpyAsync(scratch, pub_host, (size_t)4 * c->V * 18 * c->prec, cudaMemcpyHostToDevice, st);
  return lqcd_gauge_pack(c, native, scratch, stream);
}

// scratch: [public in (1 parity)] [public out (1 parity)] [native in] [native out]
int lqcd_dslash_host(lqcd_ctx* c, void* out_host, const void* in_host, const void* gauge, int parity, double scale,
                     int dagger, void* scratch, void* stream) {
  if (!c || !out_host || !in_host || !gauge || !scratch || (parity != 0 && parity != 1)) return LQCD_ERR_INVALID_ARG;
  if (c->half) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "dslash_host: not available in a 16-bit context");
  if (!lqcd_aligned16(scratch) || !lqcd_aligned16(gauge)) return lqcd_set_error(c, LQCD_ERR_ALIGN, "dslash_host: alignment");
  cudaStream_t st = as_stream(stream);
  const size_t sp = lqcd_spinor_bytes(c);
  char* s = (char*)scratch;
  int rc;
  cudaMemcpyAsync(s, (const char*)in_host + (size_t)(1 - parity) * sp, sp, cudaMemcpyHostToDevice, st);
  if ((rc = lqcd_spinor_pack_parity(c, s + 2 * sp, s, st))) return rc;
  if ((rc = lqcd_dslash_launch(c, s + 3 * sp, s + 2 * sp, gauge, nullptr, nullptr, parity, scale, dagger ? 1 : 0, 0, 1, st))) return rc;
  if ((rc = lqcd_spinor_unpack_parity(c, s + sp, s + 3 * sp, st))) return rc;
  cudaMemcpyAsync((char*)out_host + (size_t)parity * sp, s + sp, sp, cudaMemcpyDeviceToHost, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return lqcd_check_cuda(c, "dslash_host sync");
  return LQCD_OK;
}

int lqcd_invert_host(lqcd_ctx* c, void* x_host, const void* b_host, const void* gauge, const void* clover,
                     const void* clover_inv, double kappa, double tol, int maxiter, int solver, int matpc,
                     void* scratch, size_t scratch_bytes, lqcd_result* res, void* stream) {
  if (!c || !x_host || !b_host || !scratch || !clover || !clover_inv) return LQCD_ERR_INVALID_ARG;
  if (c->half) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "invert_host: not available in a 16-bit context");
  if (scratch_bytes < lqcd_host_scratch_bytes(c, solver)) return lqcd_set_error(c, LQCD_ERR_WORKSPACE, "invert_host: scratch too small");
  cudaStream_t st = as_stream(stream);
  const size_t sp = lqcd_spinor_bytes(c);
  char* s = (char*)scratch;
  cudaMemcpyAsync(s, b_host, 2 * sp, cudaMemcpyHostToDevice, st);
  int rc = invert_common(c, s + 2 * sp, s, gauge, clover, clover_inv, kappa, 0.0, tol, maxiter, solver, matpc, 1,
                         s + 4 * sp, scratch_bytes - 4 * sp, res, st);
  if (rc < 0) return rc;
  cudaMemcpyAsync(x_host, s + 2 * sp, 2 * sp, cudaMemcpyDeviceToHost, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return lqcd_check_cuda(c, "invert_host sync");
  return rc;
}

// The whole path from host buffers in one call: links and source go up on the context's copy stream while the
// caller's stream packs the links and builds the clover field (the source upload hides behind pack + build), then
// the solve, then the solution goes down.  g_scratch: >= 4*V*18*prec bytes; scratch: as lqcd_invert_host.
int lqcd_solve_host(lqcd_ctx* c, void* x_host, const void* b_host, const void* gauge_public_host, void* gauge,
                    void* clover, void* clover_inv, double csw, double kappa, double tol, int maxiter, int solver,
                    int matpc, void* g_scratch, void* scratch, size_t scratch_bytes, lqcd_result* res, void* stream) {
  if (!c || !x_host || !b_host || !gauge_public_host || !gauge || !clover || !clover_inv || !g_scratch || !scratch || !res)
    return LQCD_ERR_INVALID_ARG;
  if (c->half) return lqcd_set_error(c, LQCD_ERR_INVALID_ARG, "solve_host: not available in a 16-bit context");
  if (scratch_bytes < lqcd_host_scratch_bytes(c, solver)) return lqcd_set_error(c, LQCD_ERR_WORKSPACE, "solve_host: scratch too small");
  cudaStream_t st = as_stream(stream), cp = c->copy_stream;
  const size_t sp = lqcd_spinor_bytes(c);
  char* s = (char*)scratch;
  int rc;
  cudaEventRecord(c->ev_copy[0], st);        // the scratch buffers may still be in use by earlier work on `stream`
  cudaStreamWaitEvent(cp, c->ev_copy[0], 0);
  cudaMemcpyAsync(g_scratch, gauge_public_host, (size_t)4 * c->V * 18 * c->prec, cudaMemcpyHostToDevice, cp);
  cudaEventRecord(c->ev_copy[1], cp);
  cudaMemcpyAsync(s, b_host, 2 * sp, cudaMemcpyHostToDevice, cp);
  cudaEventRecord(c->ev_copy[2], cp);
  cudaStreamWaitEvent(st, c->ev_copy[1], 0);
  if ((rc = lqcd_gauge_pack(c, gauge, g_scratch, stream))) return rc;
  if ((rc = lqcd_clover_build(c, clover, clover_inv, gauge, csw, kappa, stream))) return rc;
  cudaStreamWaitEvent(st, c->ev_copy[2], 0);
  rc = invert_common(c, s + 2 * sp, s, gauge, clover, clover_inv, kappa, 0.0, tol, maxiter, solver, matpc, 1, s + 4 * sp,
                     scratch_bytes - 4 * sp, res, st);
  if (rc < 0) return rc;
  cudaMemcpyAsync(x_host, s + 2 * sp, 2 * sp, cudaMemcpyDeviceToHost, st);
  if (cudaStreamSynchronize(st) != cudaSuccess) return lqcd_check_cuda(c, "solve_host sync");
  return rc;
}

// BLAS-1 entry points: single right-hand side, slot S_DONE of column 0 cleared by every solve's end
int lqcd_blas_axpy_norm(lqcd_ctx* c, double a, const void* x, void* y, double* norm2_host, void* stream) {
  if (!c || !x || !y || !norm2_host) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  void* v[2] = {(void*)x, y};
  int o[4] = {S_TRUE, 0, 0, 0};
  int rc;
  if ((rc = BLAS_CALL(c, OpAxpyNorm, op.a = a, v, o, 1, 0, st))) return rc;
  if ((rc = read_scalars(c, 1, st))) return rc;
  *norm2_host = c->h_scalars[S_TRUE];
  return LQCD_OK;
}

int lqcd_blas_xpay(lqcd_ctx* c, const void* x, double a, void* y, void* stream) {
  if (!c || !x || !y) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  void* v[2] = {(void*)x, y};
  int rc;
  if ((rc = BLAS_CALL(c, OpXpay, op.a = a, v, nullptr, 1, 0, st))) return rc;
  return LQCD_OK;
}

int lqcd_blas_cdot(lqcd_ctx* c, const void* x, const void* y, double out_host[3], void* stream) {
  if (!c || !x || !y || !out_host) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  void* v[2] = {(void*)x, (void*)y};
  int o[4] = {S_TRUE, S_TRUE + 1, S_TRUE + 2, 0};
  int rc;
  if ((rc = BLAS_CALL(c, OpCdot, (void)op, v, o, 1, 0, st))) return rc;
  if ((rc = read_scalars(c, 1, st))) return rc;
  for (int i = 0; i < 3; i++) out_host[i] = c->h_scalars[S_TRUE + i];
  return LQCD_OK;
}

int lqcd_blas_caxpbypz(lqcd_ctx* c, const double a[2], const void* x, const double b[2], const void* y, void* z,
                       void* stream) {
  if (!c || !a || !b || !x || !y || !z) return LQCD_ERR_INVALID_ARG;
  cudaStream_t st = as_stream(stream);
  void* v[3] = {(void*)x, (void*)y, z};
  int rc;
  if ((rc = BLAS_CALL(c, OpCaxpbypz, (op.a = {a[0], a[1]}, op.b = {b[0], b[1]}), v, nullptr, 1, 0, st))) return rc;
  return LQCD_OK;
}

}  // extern "C"
