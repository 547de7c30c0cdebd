/* lqcd.h -- C ABI of liblqcd: even-odd preconditioned Wilson-clover operator and Krylov solves on
 * one B200 (sm_100a).  Boundary of SURVEY.md §8(b); every step behind these calls runs in
 * hand-written CUDA kernels (paper_2411_08461_b200/csrc).  No CPU fallback exists.
 *
 * Operator (Eq. 5, isotropic case; kappa normalisation, reading A2):
 *     M = A - kappa * D,     A = 1 - kappa * csw * sum_{mu<nu} sigma_{mu nu} (x) F_{mu nu}
 *     (D psi)(x) = sum_mu [ (1-g_mu) U_mu(x) psi(x+mu) + (1+g_mu) U_mu^dag(x-mu) psi(x-mu) ]
 * DeGrand-Rossi gamma basis.  The paper's a_t*M equals M/(2 kappa).
 *
 * PUBLIC layouts (complex = interleaved (re,im) of the context's real type):
 *     gauge   [4][2][Lt][Lz][Ly][Lx/2][3][3]   mu = 0..3 <-> x,y,z,t ; row-column colour order
 *     spinor  [2][Lt][Lz][Ly][Lx/2][4][3]      even parity first
 *     clover  [2][Lt][Lz][Ly][Lx/2][2][36] reals: per chiral block (upper, lower) 6 real diagonal
 *             entries then the 15 strictly-lower complex entries, row-major ((i,j), i>j at
 *             i(i-1)/2+j)
 * NATIVE layouts are private structure-of-arrays of 16-byte vectors; the
 * caller only needs their byte sizes (lqcd_*_bytes) and moves data with pack/unpack.
 *
 * Conventions.  Every pointer is a DEVICE pointer unless the name ends in _host.  The caller owns
 * all buffers; the library keeps none beyond the call (the context owns a small reduction
 * scratch and, after a clover build, that build's scratch).  Device pointers must be 16-byte aligned.  All calls are asynchronous on `stream`
 * (a cudaStream_t passed as void*) except lqcd_invert*, lqcd_*_host and lqcd_blas_*, which
 * synchronise the stream before returning.  Return: 0 = OK, <0 = error, +1 = NOT_CONVERGED.
 * No exceptions, no abort, nothing printed.  A context is not thread-safe.
 */
#ifndef LQCD_H
#define LQCD_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct lqcd_ctx lqcd_ctx;

enum {
  LQCD_OK = 0,
  LQCD_NOT_CONVERGED = 1,
  LQCD_ERR_INVALID_ARG = -1,
  LQCD_ERR_DIMS = -2,
  LQCD_ERR_ALIGN = -3,
  LQCD_ERR_WORKSPACE = -4,
  LQCD_ERR_CUDA = -5,
  LQCD_ERR_SINGULAR_CLOVER = -6,
  LQCD_ERR_BREAKDOWN = -7
};
enum { LQCD_SOLVER_CGNE = 0, LQCD_SOLVER_CGNR = 1, LQCD_SOLVER_BICGSTAB = 2 };
enum { LQCD_MATPC_ASYMMETRIC = 0, LQCD_MATPC_SYMMETRIC = 1, LQCD_MATPC_SYMMETRIC_RIGHT = 2 };
#define LQCD_MAX_RHS 16 /* right-hand sides per multi-RHS call (a propagator has 12 columns) */

typedef struct lqcd_result {
  int status;          /* LQCD_OK, LQCD_NOT_CONVERGED or LQCD_ERR_BREAKDOWN */
  int iterations;
  double iter_resid;   /* |r_hat| / |b| from the recurrence at exit                         */
  double true_resid;   /* |b - M x| / |b| recomputed with the full operator (lqcd_mat_apply) */
  double seconds;      /* device time of the whole call, CUDA events                        */
  long dslash_count;   /* single-parity dslash launches                                     */
  long kernel_launches;
} lqcd_result;

/* Context (init + LatticeInfo).  dims = {Lx,Ly,Lz,Lt}, each even and >= 4;
 * prec = 4 (fp32) or 8 (fp64): the real type of every native AND public buffer of this context; prec = 2: 16-bit
 * fixed-point NATIVE fields with fp32 arithmetic and fp32 (complex64) public arrays (see "16-bit storage" below);
 * recon = 18 (full links) or 12 (two rows stored, third recomputed); t_boundary = +1 or -1
 * (antiperiodic in t, applied in-kernel to raw periodic links); device = CUDA
 * ordinal (must be compute capability 10.x).
 * Measurement switches read from the environment at creation (results agree to rounding order, only the kernel
 * differs; every default is the measured-best choice):
 *   LQCD_DSLASH_TILED=1      shared-memory tiled single-RHS dslash where its tile divides the lattice (slower);
 *   LQCD_MRHS_TMA=0|1|2      TMA-tiled multi-RHS kernel (fp32): off | where measured faster (default) | wherever it runs;
 *   LQCD_MRHS_ZSLAB=n        z-planes per slab of the multi-RHS block sweep (default per kernel);
 *   LQCD_MRHS_FUSE_DOTS=0|1  batched BiCGStab dot products in the multi-RHS epilogues: never | always (default: where
 *                            the register kernel runs the epilogue anyway);
 *   LQCD_GRAPHS=0            no CUDA-graph replay of Krylov iteration blocks on small lattices;
 *   LQCD_CLOVER_ONEPASS=1    one-kernel clover build (no scratch) instead of the three-pass one;
 *   LQCD_MIXED_LAST_MARGIN=f mixed solves close (x_o, true residual) without a last fp64 Schur residual when the inner
 *                            recurrence predicts |r|^2 <= f * (tol |b|)^2 (default 0.9; 0 = never; a wrong guess reopens). */
int lqcd_create(lqcd_ctx** ctx, const int dims[4], int prec, int recon, int t_boundary, int device);
int lqcd_destroy(lqcd_ctx* ctx);
const char* lqcd_strerror(int code);
const char* lqcd_last_error(const lqcd_ctx* ctx);
/* number of kernels this context has launched since creation (bench.py's gpu_launches) */
long lqcd_launch_count(const lqcd_ctx* ctx);
/* Small-lattice solves (one-parity volume x columns <= 131072) stop on the device and replay blocks of 4 Krylov
 * iterations as CUDA graphs (LQCD_GRAPHS=0 at context creation: plain launches, same results bit for bit); this counts
 * the blocks replayed.  Their kernels are included in lqcd_launch_count. */
long lqcd_graph_launch_count(const lqcd_ctx* ctx);

/* Algorithmic HBM bytes (compulsory reads + writes of each kernel) summed over
 * every kernel this context has launched since creation (bench.py's whole-step throughput). */
double lqcd_algorithmic_bytes(const lqcd_ctx* ctx);
/* Per-launch device timing of the dslash kernels (all epilogues) with CUDA events on the launching
 * stream.  enable != 0 starts recording (up to 8192 launches), 0 stops.  lqcd_profile_read
 * synchronises the recorded events, returns the number of launches, their summed duration in ms
 * and their summed algorithmic bytes, and clears the record. */
int lqcd_profile_enable(lqcd_ctx* ctx, int enable);
int lqcd_profile_read(lqcd_ctx* ctx, long* launches, double* total_ms, double* total_bytes);

/* Byte sizes of native buffers: links (4 directions, both parities), ONE parity of a spinor,
 * the clover field (both parities; same size for A and for A^-1), the solver workspace. */
size_t lqcd_gauge_bytes(const lqcd_ctx* ctx);
size_t lqcd_spinor_bytes(const lqcd_ctx* ctx);
size_t lqcd_clover_bytes(const lqcd_ctx* ctx);
size_t lqcd_invert_workspace_bytes(const lqcd_ctx* ctx, int solver);

/* public <-> native ("QUDA needs to convert the data format to its native one").
 * Spinor natives hold both parities: [2][one-parity native]. recon 12 drops the third row. */
int lqcd_gauge_pack(lqcd_ctx* ctx, void* gauge_native, const void* gauge_public, void* stream);
int lqcd_spinor_pack(lqcd_ctx* ctx, void* spinor_native, const void* spinor_public, void* stream);
int lqcd_spinor_unpack(lqcd_ctx* ctx, void* spinor_public, const void* spinor_native, void* stream);
int lqcd_clover_unpack(lqcd_ctx* ctx, void* clover_public, const void* clover_native, void* stream);
/* the inverse: a packed clover field (or inverse) in the public layout -> native, e.g. a sub-lattice's part of a field
 * built on the whole lattice (domain decomposition) */
int lqcd_clover_pack(lqcd_ctx* ctx, void* clover_native, const void* clover_public, void* stream);

/* Clover term and its inverse from the links ("the clover field is then created";
 * SURVEY.md §8(c) O4-O6).  kappa is required because A contains kappa*csw (reading A6).  Leaves
 * and the 6x6 inverses are computed in fp64 whatever the storage precision.  clover_inv may be
 * NULL.  Synchronises; returns LQCD_ERR_SINGULAR_CLOVER if some block has a pivot < 1e-12|A|.
 * Ownership: the first build makes the context allocate a scratch of 864 bytes per lattice site (two fields of
 * plaquette parts between the passes of the build), kept until lqcd_destroy; if that allocation fails
 * the build falls back to a one-kernel form that needs none. */
int lqcd_clover_build(lqcd_ctx* ctx, void* clover, void* clover_inv, const void* gauge, double csw,
                      double kappa, void* stream);

/* lqcd_clover_build for callers that cannot tolerate an allocation inside the call (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): same arguments, same result (the same three kernels), but the scratch
 * between the passes is a fixed device array inside the library instead of a cudaMalloc on the context's first build.
 * The call makes no cudaMalloc / cudaFree / allocating library call.
 * Limit: lattices of at most lqcd_clover_noalloc_max_sites() = 32768 sites (e.g. 8^3x64, 16x16x8x16); larger ones return
 * LQCD_ERR_WORKSPACE with the two numbers in lqcd_last_error.  Cost: 27 MiB of device memory on every GPU that loads the
 * library, until the process exits.  The array is shared by all contexts and calls on a GPU and keeps the last call's
 * contents (nothing in it needs clearing: every entry read was written by the same call); calls that overlap on the GPU
 * race on it, so serialise them.  The context's device must be the current device.  Synchronises like lqcd_clover_build. */
int lqcd_clover_build_noalloc(lqcd_ctx* ctx, void* clover, void* clover_inv, const void* gauge, double csw,
                              double kappa, void* stream);
long lqcd_clover_noalloc_max_sites(void);

/* Anisotropic operator of PAPER.md:218-221, Eq. 5, in kappa normalisation:
 *     M = 1 - kappa [ D_t + (nu/xi_0) sum_i D_i ]
 *           - kappa [ c_SW^t sum_i sigma_i4 F_i4 + (c_SW^r/xi_0) sum_{i<j} sigma_ij F_ij ],   1/kappa = 2(m0 + 1 + 3 nu/xi_0)
 * lqcd_set_anisotropy fixes the weight nu/xi_0 (> 0; default 1 = isotropic) of the spatial hops for
 * every later dslash / mpc_apply / mat_apply / invert* call of this context (the temporal hops keep
 * weight 1 and the boundary sign).  lqcd_clover_build_aniso is lqcd_clover_build with
 * csw_s = c_SW^r/xi_0 on the planes xy, xz, yz and csw_t = c_SW^t on xt, yt, zt.  Raw (unscaled)
 * SU(3) links are passed in both cases: no "fake anisotropy" is applied to the gauge field
 * (PAPER.md:100-102 describes that workaround for QUDA). */
int lqcd_set_anisotropy(lqcd_ctx* ctx, double nu_over_xi0);
int lqcd_clover_build_aniso(lqcd_ctx* ctx, void* clover, void* clover_inv, const void* gauge, double csw_s,
                            double csw_t, double kappa, void* stream);

/* out = C in on one parity, C = the two Hermitian 6x6 chiral blocks per site of `clover_or_inv`
 * (PAPER.md:56).  in/out: one-parity native spinors; they may alias. */
int lqcd_clover_apply(lqcd_ctx* ctx, void* out, const void* in, const void* clover_or_inv, int parity,
                      void* stream);

/* out_p = scale * D_{p,1-p} in_{1-p}  (dagger != 0: D^dag).  parity = parity of `out` (0 even).
 * in/out: one-parity native spinors, must not alias.  scale = 1 gives the bare hopping term
 * (1320 flop/site); -kappa gives the off-diagonal block of M. */
int lqcd_dslash(lqcd_ctx* ctx, void* out, const void* in, const void* gauge, int parity, double scale,
                int dagger, void* stream);

/* Even-even Schur complement on one-parity native spinors:
 *   matpc 0: out = A_ee in - kappa^2 D_eo A_oo^-1 D_oe in
 *   matpc 1: out = in - kappa^2 A_ee^-1 D_eo A_oo^-1 D_oe in      (symmetric, preconditioned from the left)
 *   matpc 2: out = in - kappa^2 D_eo A_oo^-1 D_oe A_ee^-1 in      (symmetric, preconditioned from the right:
 *            = (matpc 0) A_ee^-1; in a solve the Krylov unknown is y = A_ee x_e and the recurrence residual is
 *            that of matpc 0, i.e. the even half of the true residual, with the conditioning of matpc 1)
 * dagger: the adjoint of any of them.  tmp_o: one-parity scratch spinor. */
int lqcd_mpc_apply(lqcd_ctx* ctx, void* out_e, const void* in_e, const void* gauge, const void* clover,
                   const void* clover_inv, double kappa, int matpc, int dagger, void* tmp_o, void* stream);

/* Full operator on both parities: out = A in - kappa D in (dagger: D^dag).  in/out: two-parity
 * native spinors, must not alias. */
int lqcd_mat_apply(lqcd_ctx* ctx, void* out, const void* in, const void* gauge, const void* clover,
                   double kappa, int dagger, void* stream);

/* Solve M x = b through the even-even Schur system,
 * x0 = 0, stop when |r_hat| <= tol*|b| (reading A11), reconstruct the odd half, recompute the true
 * residual.  x_public/b_public: public-layout device spinors.  clover/clover_inv: native fields
 * from lqcd_clover_build; if clover == NULL both are built inside the workspace from
 * (gauge, csw, kappa), otherwise csw is ignored.  workspace: >= lqcd_invert_workspace_bytes.
 * Host-synchronous.  Returns res->status. */
int lqcd_invert(lqcd_ctx* ctx, void* x_public, const void* b_public, const void* gauge, const void* clover,
                const void* clover_inv, double kappa, double csw, double tol, int maxiter, int solver,
                int matpc, void* workspace, size_t workspace_bytes, lqcd_result* res, void* stream);

/* Multi-right-hand-side forms (a propagator is 12 solves, one
 * per spin-colour column, on the same links and clover).  The links are loaded once per site for all
 * nrhs columns, so the bytes per site and column fall from (8R+48)w towards (8R/nrhs+48)w.
 * Native multi-RHS fields are nrhs consecutive one-parity native spinors ([rhs][one-parity native]);
 * 1 <= nrhs <= LQCD_MAX_RHS; nrhs = 1 runs the single-RHS kernels.
 *   lqcd_dslash_mrhs    : out[r] = scale * D_{p,1-p} in[r]                      (as lqcd_dslash)
 *   lqcd_mpc_apply_mrhs : out[r] = Mhat in[r]; tmp_o: nrhs one-parity spinors   (as lqcd_mpc_apply)
 *   lqcd_invert_multi   : nrhs independent Krylov recurrences advanced in lock step (each column has
 *       its own alpha, beta, omega and stopping test |r_hat_r| <= tol*|b_r|; a converged column is
 *       frozen, so every column's result is that of its own single solve).  x_public/b_public: nrhs
 *       consecutive public spinors; res: array of nrhs results.  Returns the worst status: the
 *       most negative error if any column failed, else NOT_CONVERGED if any did not converge, else
 *       OK.  workspace: >= lqcd_invert_multi_workspace_bytes; clover and clover_inv are required. */
int lqcd_dslash_mrhs(lqcd_ctx* ctx, void* out, const void* in, const void* gauge, int parity, double scale,
                     int dagger, int nrhs, void* stream);
int lqcd_mpc_apply_mrhs(lqcd_ctx* ctx, void* out_e, const void* in_e, const void* gauge, const void* clover,
                        const void* clover_inv, double kappa, int matpc, int dagger, void* tmp_o, int nrhs,
                        void* stream);
size_t lqcd_invert_multi_workspace_bytes(const lqcd_ctx* ctx, int solver, int nrhs);
int lqcd_invert_multi(lqcd_ctx* ctx, void* x_public, const void* b_public, const void* gauge, const void* clover,
                      const void* clover_inv, double kappa, double tol, int maxiter, int solver, int matpc,
                      int nrhs, void* workspace, size_t workspace_bytes, lqcd_result* res, void* stream);

/* Mixed precision: the same system solved to the same fp64 stopping test
 * |r_hat| <= tol*|b| by fp64 defect correction around fp32 Krylov solves:
 *     x = 0, r = b_hat;  repeat { e = Mhat^-1 (r/|r|) in fp32 to tol_k;  x += |r| e;  r = b_hat - Mhat x (fp64) }
 * with tol_k = max(inner_tol, 0.25*tol*|b|/|r|).  ctx: fp64 context owning x, b, gauge, clover,
 * clover_inv, workspace (as lqcd_invert); ctx_lo: fp32 context of the same lattice/boundary/device
 * owning gauge_lo, clover_lo, clover_inv_lo (its own pack/clover_build of the same links; the
 * reconstructions may differ) and workspace_lo (>= lqcd_invert_workspace_bytes(ctx_lo)).
 * res->iterations counts inner iterations; true_resid is recomputed in fp64.  Host-synchronous.
 * lqcd_invert_multi_mixed: the same for nrhs columns (x_public/b_public: nrhs consecutive public spinors,
 * res: nrhs results, as lqcd_invert_multi): every outer step is ONE batched fp32 solve (multi-RHS kernels:
 * links loaded once per site for all columns) over the columns still above their fp64 stopping test;
 * workspace >= lqcd_invert_multi_workspace_bytes(ctx, solver, nrhs), workspace_lo likewise for ctx_lo.
 * Returns the worst status over the columns (as lqcd_invert_multi). */
int lqcd_invert_multi_mixed(lqcd_ctx* ctx, lqcd_ctx* ctx_lo, void* x_public, const void* b_public, const void* gauge,
                            const void* clover, const void* clover_inv, const void* gauge_lo, const void* clover_lo,
                            const void* clover_inv_lo, double kappa, double tol, double inner_tol, int maxiter,
                            int solver, int matpc, int nrhs, void* workspace, size_t workspace_bytes,
                            void* workspace_lo, size_t workspace_lo_bytes, lqcd_result* res, void* stream);
int lqcd_invert_mixed(lqcd_ctx* ctx, lqcd_ctx* ctx_lo, void* x_public, const void* b_public, const void* gauge,
                      const void* clover, const void* clover_inv, const void* gauge_lo, const void* clover_lo,
                      const void* clover_inv_lo, double kappa, double tol, double inner_tol, int maxiter, int solver,
                      int matpc, void* workspace, size_t workspace_bytes, void* workspace_lo,
                      size_t workspace_lo_bytes, lqcd_result* res, void* stream);

/* 16-bit storage (second half; PAPER.md:423 ref. [1], mixed-precision solvers on GPUs).  A context
 * created with prec = 2 stores spinors as 24 int16 + one fp32 norm per site (52 B), links as R int16 (|U_ij| <= 1) and
 * the clover field as 72 int16 + one fp32 norm per chiral block (152 B per site); every kernel computes in fp32
 * registers.  Sizes come from lqcd_*_bytes as usual; public arrays are complex64.  Available in such a context:
 * lqcd_gauge_pack, lqcd_spinor_pack / _unpack, lqcd_dslash, lqcd_clover_apply, lqcd_mpc_apply, lqcd_mat_apply,
 * lqcd_invert (clover fields required), lqcd_blas_*, the sources / contractions (public arrays), and its use as
 * ctx_lo of lqcd_invert_mixed (one column), which is what it is for: the inner iterations move half the bytes of an
 * fp32 context and the fp64 defect correction outside restores the tolerance.  Not available (LQCD_ERR_INVALID_ARG):
 * lqcd_clover_build* (build in an fp32 context of the same lattice, then lqcd_clover_to_half), lqcd_clover_unpack, the
 * multi-RHS and *_host calls.
 *   lqcd_clover_to_half : clover_fp32_native (both parities, from an fp32 context of the same lattice) -> 16-bit native */
int lqcd_clover_to_half(lqcd_ctx* ctx_half, void* clover_half, const void* clover_fp32_native, void* stream);

/* 4-D domain decomposition of the hopping term (the lattice is divided
 * equally over a 4-D Cartesian grid of ranks, the rank index running fastest in t).  Each rank owns a context, links and
 * spinors of its sub-lattice (every local extent even and >= 4).  In a partitioned direction the hops that leave the
 * sub-lattice are served by faces of projected half spinors, 12 reals per face site:
 *   lqcd_set_partition      : partitioned[mu] != 0 marks direction mu as cut (default: none)
 *   lqcd_face_bytes         : bytes of one face buffer of direction mu ([12][face sites of one parity], context type)
 *   lqcd_dslash_dd_interior : out_p = scale * (the hops of D_{p,1-p} in that stay inside the sub-lattice); with no
 *                             direction partitioned this is lqcd_dslash.  The context's t_boundary sign applies to
 *                             interior hops only: give +1 to a context whose t direction is cut.
 *   lqcd_face_pack          : dir = +1: the forward ghost of my -mu neighbour = my FIRST slice, h = P psi;
 *                             dir = -1: the backward ghost of my +mu neighbour = my LAST slice, U_mu^dag P psi (my links).
 *                             parity_in = parity of `in` (one-parity native spinor); dagger as in lqcd_dslash.
 *   lqcd_face_unpack        : out_p += scale * weight * (the hop rebuilt from a received face): dir = +1 a forward ghost
 *                             (received from the +mu neighbour, multiplied by my link U_mu(x) on my last slice), dir = -1
 *                             a backward ghost (from the -mu neighbour, added on my first slice).  weight = nu/xi_0 for
 *                             a spatial mu, and for t the boundary sign of THIS hop: -1 where it crosses the
 *                             antiperiodic seam of the global lattice, +1 elsewhere.
 * Moving a packed face to the rank that unpacks it is the caller's job (paper_2411_08461_b200/dd.py: device copies
 * between sub-lattices on one GPU, torch.distributed send / recv between ranks).  fp32 and fp64 contexts. */
int lqcd_set_partition(lqcd_ctx* ctx, const int partitioned[4]);
size_t lqcd_face_bytes(const lqcd_ctx* ctx, int mu);
int lqcd_dslash_dd_interior(lqcd_ctx* ctx, void* out, const void* in, const void* gauge, int parity, double scale,
                            int dagger, void* stream);
int lqcd_face_pack(lqcd_ctx* ctx, void* face, const void* in, const void* gauge, int mu, int dir, int parity_in,
                   int dagger, void* stream);
int lqcd_face_unpack(lqcd_ctx* ctx, void* out, const void* face, const void* gauge, int mu, int dir, int parity_out,
                     double scale, double weight, int dagger, void* stream);

/* Sources, propagator assembly and per-time-slice contractions of the paper's Listing 1
 * (SURVEY.md §8(a) a4/a12, §8(f) rank 4).  All arrays are DEVICE arrays in PUBLIC
 * layout and in the context's precision: phase [2][Lt][Lz][Ly][Lx/2] complex; spinor as above;
 * propagator [2][Lt][Lz][Ly][Lx/2][4 sink spin j][4 source spin i][3 sink colour b][3 source colour a]
 * complex; "columns" = 12 consecutive public spinors, column 3*i+a = the solution for
 * the source of spin i, colour a.
 *   lqcd_momentum_phase      : phase(x) = exp(2 pi i (n_x x/Lx + n_y y/Ly + n_z z/Lz))
 *   lqcd_source_wall         : 1 (or phase(x) if phase != NULL) on every site of time-slice t0 in the
 *                              (spin, colour) component, 0 elsewhere
 *   lqcd_source_point        : 1 at site x = {x,y,z,t} in the (spin, colour) component
 *   lqcd_propagator_assemble : columns -> propagator;  lqcd_propagator_split: the inverse (the source
 *                              columns of invertPropagator)
 *   lqcd_contract_twopt      : Eq. 6: out[t] = sum_{w,x,y,z,i,j,a,b} conj(phase) conj(S_0) S_p
 *                              (phase == NULL: 1); out_host: Lt complex as {re, im} doubles
 *   lqcd_contract_threept    : Eq. 7: out[t] = sum conj(S_p0[j,i,b,a]) Gamma[j][k] S_p[k,i,b,a];
 *                              gamma: 4x4 complex row-major as 32 doubles (host)
 *   lqcd_sequential_source   : Eq. 8: X[i,k,a,b] = conj(phase) sum_j Gamma[i][j] S_0[j,k,a,b] on
 *                              time-slice t, 0 elsewhere; X must not alias S_0
 * The two contractions accumulate in fp64 with a fixed reduction order (deterministic) and synchronise. */
int lqcd_momentum_phase(lqcd_ctx* ctx, void* phase_public, const int mom[3], void* stream);
int lqcd_source_wall(lqcd_ctx* ctx, void* b_public, int t0, int spin, int colour, const void* phase_public,
                     void* stream);
int lqcd_source_point(lqcd_ctx* ctx, void* b_public, const int x[4], int spin, int colour, void* stream);
int lqcd_propagator_assemble(lqcd_ctx* ctx, void* prop_public, const void* columns_public, void* stream);
int lqcd_propagator_split(lqcd_ctx* ctx, void* columns_public, const void* prop_public, void* stream);
int lqcd_contract_twopt(lqcd_ctx* ctx, double* out_host, const void* phase_public, const void* S_0,
                        const void* S_p, void* stream);
int lqcd_contract_threept(lqcd_ctx* ctx, double* out_host, const void* S_p0, const double gamma[32],
                          const void* S_p, void* stream);
int lqcd_sequential_source(lqcd_ctx* ctx, void* X_prop, const void* phase_public, const double gamma[32],
                           const void* S_0, int t, void* stream);

/* End-to-end variants with HOST buffers (pageable or pinned): the call uploads the public input,
 * packs, computes, unpacks and downloads the public result.  Links/clover stay resident on the
 * device (PAPER.md:225 loadGauge).  scratch: device buffer of >= lqcd_host_scratch_bytes. */
size_t lqcd_host_scratch_bytes(const lqcd_ctx* ctx, int solver);
int lqcd_gauge_pack_host(lqcd_ctx* ctx, void* gauge_native, const void* gauge_public_host, void* scratch,
                         void* stream); /* scratch: >= 4*V*18*prec bytes (the public link field) */
int lqcd_dslash_host(lqcd_ctx* ctx, void* out_public_host, const void* in_public_host, const void* gauge,
                     int parity, double scale, int dagger, void* scratch, void* stream);
int lqcd_invert_host(lqcd_ctx* ctx, void* x_public_host, const void* b_public_host, const void* gauge,
                     const void* clover, const void* clover_inv, double kappa, double tol, int maxiter,
                     int solver, int matpc, void* scratch, size_t scratch_bytes, lqcd_result* res,
                     void* stream);

/* The whole path from HOST buffers in one call (loadGauge, clover creation, invert): uploads the
 * public links and source, packs, builds clover and inverse, solves, downloads the public solution.  The uploads
 * run on a copy stream owned by the context, so the source upload overlaps the link pack and the clover build.
 * gauge, clover, clover_inv: device buffers (lqcd_*_bytes) that receive the native fields and stay valid for later
 * calls; g_scratch: device, >= 4*V*18*prec bytes; scratch: device, >= lqcd_host_scratch_bytes.  Host-synchronous;
 * returns res->status. */
int lqcd_solve_host(lqcd_ctx* ctx, void* x_public_host, const void* b_public_host, const void* gauge_public_host,
                    void* gauge, void* clover, void* clover_inv, double csw, double kappa, double tol, int maxiter,
                    int solver, int matpc, void* g_scratch, void* scratch, size_t scratch_bytes, lqcd_result* res,
                    void* stream);

/* Fused BLAS-1 kernels of the solvers, exposed for parity tests and bandwidth measurement
 * (SURVEY.md §8(a) a9).  Vectors are one-parity native spinors; results are fp64 on the host;
 * the two that return a scalar (axpy_norm, cdot) synchronise, the other two are asynchronous.  a, b are complex
 * given as {re, im}.
 *   lqcd_blas_axpy_norm : y += a*x (a real),  returns |y|^2
 *   lqcd_blas_xpay      : y  = x + a*y (a real)
 *   lqcd_blas_cdot      : returns <x,y> = sum conj(x_i) y_i  and |x|^2 in out[0..2]
 *   lqcd_blas_caxpbypz  : z += a*x + b*y (a, b complex) */
int lqcd_blas_axpy_norm(lqcd_ctx* ctx, double a, const void* x, void* y, double* norm2_host, void* stream);
int lqcd_blas_xpay(lqcd_ctx* ctx, const void* x, double a, void* y, void* stream);
int lqcd_blas_cdot(lqcd_ctx* ctx, const void* x, const void* y, double out_host[3], void* stream);
int lqcd_blas_caxpbypz(lqcd_ctx* ctx, const double a[2], const void* x, const double b[2], const void* y,
                       void* z, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* LQCD_H */
