"""Thin Python binding of liblqcd (include/lqcd.h): argument marshalling only.

PyTorch supplies device memory and the CUDA stream; every step of the path runs in the CUDA
kernels behind the C ABI.  There is no CPU fallback: if the shared library is missing or no
sm_100 device is present, creating a context raises.
"""
import ctypes
import os

import numpy as np
import torch

from . import build as _build

_lib = None


class Result(ctypes.Structure):
    _fields_ = [("status", ctypes.c_int), ("iterations", ctypes.c_int),
                ("iter_resid", ctypes.c_double), ("true_resid", ctypes.c_double),
                ("seconds", ctypes.c_double), ("dslash_count", ctypes.c_long),
                ("kernel_launches", ctypes.c_long)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


SOLVERS = {"cgne": 0, "cgnr": 1, "bicgstab": 2}
SYMBOLS = [
    "lqcd_create", "lqcd_destroy", "lqcd_strerror", "lqcd_last_error", "lqcd_launch_count",
    "lqcd_algorithmic_bytes", "lqcd_profile_enable", "lqcd_profile_read", "lqcd_gauge_pack_host",
    "lqcd_gauge_bytes", "lqcd_spinor_bytes", "lqcd_clover_bytes", "lqcd_invert_workspace_bytes",
    "lqcd_gauge_pack", "lqcd_spinor_pack", "lqcd_spinor_unpack", "lqcd_clover_unpack",
    "lqcd_clover_build_noalloc", "lqcd_clover_noalloc_max_sites",
    "lqcd_clover_build", "lqcd_clover_apply", "lqcd_dslash", "lqcd_mpc_apply", "lqcd_mat_apply",
    "lqcd_invert", "lqcd_host_scratch_bytes", "lqcd_dslash_host", "lqcd_invert_host",
    "lqcd_blas_axpy_norm", "lqcd_blas_xpay", "lqcd_blas_cdot", "lqcd_blas_caxpbypz",
    "lqcd_dslash_mrhs", "lqcd_mpc_apply_mrhs", "lqcd_invert_multi_workspace_bytes", "lqcd_invert_multi",
    "lqcd_invert_mixed", "lqcd_invert_multi_mixed", "lqcd_solve_host", "lqcd_set_anisotropy", "lqcd_clover_build_aniso",
    "lqcd_momentum_phase", "lqcd_source_wall", "lqcd_source_point", "lqcd_propagator_assemble",
    "lqcd_propagator_split", "lqcd_contract_twopt", "lqcd_contract_threept", "lqcd_sequential_source",
    "lqcd_clover_to_half", "lqcd_set_partition", "lqcd_face_bytes", "lqcd_dslash_dd_interior", "lqcd_face_pack",
    "lqcd_face_unpack", "lqcd_clover_pack", "lqcd_graph_launch_count",
]
MAX_RHS = 16


def library_path():
    return _build.SO


def load():
    """dlopen liblqcd.so (built in-tree by build.py) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_build.SO):
        raise RuntimeError("liblqcd.so is missing: run `python -m paper_2411_08461_b200.build` "
                           "(there is no CPU fallback)")
    L = ctypes.CDLL(_build.SO)
    vp, ci, cd, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    L.lqcd_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(ci), ci, ci, ci, ci]
    L.lqcd_destroy.argtypes = [vp]
    L.lqcd_strerror.restype = ctypes.c_char_p
    L.lqcd_strerror.argtypes = [ci]
    L.lqcd_last_error.restype = ctypes.c_char_p
    L.lqcd_last_error.argtypes = [vp]
    L.lqcd_launch_count.restype = ctypes.c_long
    L.lqcd_launch_count.argtypes = [vp]
    L.lqcd_graph_launch_count.restype = ctypes.c_long
    L.lqcd_graph_launch_count.argtypes = [vp]
    L.lqcd_algorithmic_bytes.restype = cd
    L.lqcd_algorithmic_bytes.argtypes = [vp]
    L.lqcd_profile_enable.argtypes = [vp, ci]
    L.lqcd_profile_read.argtypes = [vp, ctypes.POINTER(ctypes.c_long), ctypes.POINTER(cd), ctypes.POINTER(cd)]
    L.lqcd_gauge_pack_host.argtypes = [vp, vp, vp, vp, vp]
    for f in ("lqcd_gauge_bytes", "lqcd_spinor_bytes", "lqcd_clover_bytes"):
        getattr(L, f).restype = sz
        getattr(L, f).argtypes = [vp]
    for f in ("lqcd_invert_workspace_bytes", "lqcd_host_scratch_bytes"):
        getattr(L, f).restype = sz
        getattr(L, f).argtypes = [vp, ci]
    for f in ("lqcd_gauge_pack", "lqcd_spinor_pack", "lqcd_spinor_unpack", "lqcd_clover_unpack", "lqcd_clover_pack"):
        getattr(L, f).argtypes = [vp, vp, vp, vp]
    L.lqcd_clover_build.argtypes = [vp, vp, vp, vp, cd, cd, vp]
    L.lqcd_clover_build_noalloc.argtypes = [vp, vp, vp, vp, cd, cd, vp]
    L.lqcd_clover_noalloc_max_sites.argtypes = []
    L.lqcd_clover_noalloc_max_sites.restype = ctypes.c_long
    ip = ctypes.POINTER(ci)
    dp = ctypes.POINTER(cd)
    L.lqcd_momentum_phase.argtypes = [vp, vp, ip, vp]
    L.lqcd_source_wall.argtypes = [vp, vp, ci, ci, ci, vp, vp]
    L.lqcd_source_point.argtypes = [vp, vp, ip, ci, ci, vp]
    L.lqcd_propagator_assemble.argtypes = [vp, vp, vp, vp]
    L.lqcd_propagator_split.argtypes = [vp, vp, vp, vp]
    L.lqcd_contract_twopt.argtypes = [vp, dp, vp, vp, vp, vp]
    L.lqcd_contract_threept.argtypes = [vp, dp, vp, dp, vp, vp]
    L.lqcd_sequential_source.argtypes = [vp, vp, vp, dp, vp, ci, vp]
    L.lqcd_clover_to_half.argtypes = [vp, vp, vp, vp]
    L.lqcd_set_partition.argtypes = [vp, ctypes.POINTER(ci)]
    L.lqcd_face_bytes.restype = sz
    L.lqcd_face_bytes.argtypes = [vp, ci]
    L.lqcd_dslash_dd_interior.argtypes = [vp, vp, vp, vp, ci, cd, ci, vp]
    L.lqcd_face_pack.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, vp]
    L.lqcd_face_unpack.argtypes = [vp, vp, vp, vp, ci, ci, ci, cd, cd, ci, vp]
    L.lqcd_set_anisotropy.argtypes = [vp, cd]
    L.lqcd_clover_build_aniso.argtypes = [vp, vp, vp, vp, cd, cd, cd, vp]
    L.lqcd_clover_apply.argtypes = [vp, vp, vp, vp, ci, vp]
    L.lqcd_dslash.argtypes = [vp, vp, vp, vp, ci, cd, ci, vp]
    L.lqcd_mpc_apply.argtypes = [vp, vp, vp, vp, vp, vp, cd, ci, ci, vp, vp]
    L.lqcd_mat_apply.argtypes = [vp, vp, vp, vp, vp, cd, ci, vp]
    L.lqcd_invert.argtypes = [vp, vp, vp, vp, vp, vp, cd, cd, cd, ci, ci, ci, vp, sz,
                              ctypes.POINTER(Result), vp]
    L.lqcd_dslash_mrhs.argtypes = [vp, vp, vp, vp, ci, cd, ci, ci, vp]
    L.lqcd_mpc_apply_mrhs.argtypes = [vp, vp, vp, vp, vp, vp, cd, ci, ci, vp, ci, vp]
    L.lqcd_invert_multi_workspace_bytes.restype = sz
    L.lqcd_invert_multi_workspace_bytes.argtypes = [vp, ci, ci]
    L.lqcd_invert_multi.argtypes = [vp, vp, vp, vp, vp, vp, cd, cd, ci, ci, ci, ci, vp, sz,
                                    ctypes.POINTER(Result), vp]
    L.lqcd_invert_mixed.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, cd, cd, cd, ci, ci, ci, vp, sz, vp, sz,
                                    ctypes.POINTER(Result), vp]
    L.lqcd_invert_multi_mixed.argtypes = [vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, cd, cd, cd, ci, ci, ci, ci, vp, sz,
                                          vp, sz, ctypes.POINTER(Result), vp]
    L.lqcd_dslash_host.argtypes = [vp, vp, vp, vp, ci, cd, ci, vp, vp]
    L.lqcd_invert_host.argtypes = [vp, vp, vp, vp, vp, vp, cd, cd, ci, ci, ci, vp, sz,
                                   ctypes.POINTER(Result), vp]
    L.lqcd_solve_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, cd, cd, cd, ci, ci, ci, vp, vp, sz,
                                  ctypes.POINTER(Result), vp]
    L.lqcd_blas_axpy_norm.argtypes = [vp, cd, vp, vp, ctypes.POINTER(cd), vp]
    L.lqcd_blas_xpay.argtypes = [vp, vp, cd, vp, vp]
    L.lqcd_blas_cdot.argtypes = [vp, vp, vp, ctypes.POINTER(cd), vp]
    L.lqcd_blas_caxpbypz.argtypes = [vp, ctypes.POINTER(cd), vp, ctypes.POINTER(cd), vp, vp, vp]
    _lib = L
    return L


class LqcdError(RuntimeError):
    pass


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _p(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else ctypes.c_void_p(0)


def shard_columns(n, rank, world):
    """Contiguous block [lo, hi) of n independent right-hand sides owned by `rank` of `world` (sizes differ by at
    most one; the first n % world ranks take the extra column)."""
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def sharded_solve(sources, solve, group=None):
    """The n independent columns of `sources` ([n, ...]) sharded over the ranks of a torch.distributed group
    (the 12 spin-colour columns of a propagator): links and clover are
    replicated, rank r solves the contiguous block shard_columns(n, r, world) with ONE batched call
    `solve(block) -> (x, results, status)`, and one all-gather of the ranks' blocks (padded to the largest block, so
    every rank sends ceil(n / world) columns, not n) brings the solutions to every rank.  No collective on the data
    path of the solves.  Returns (x [n, ...], iterations per column, worst status over the ranks)."""
    import torch.distributed as dist
    on = dist.is_available() and dist.is_initialized()
    world = dist.get_world_size(group) if on else 1
    rank = dist.get_rank(group) if on else 0
    n = sources.shape[0]
    lo, hi = shard_columns(n, rank, world)
    width = -(-n // world)  # columns of the largest block
    mine = torch.zeros((width,) + tuple(sources.shape[1:]), dtype=sources.dtype, device=sources.device)
    my_it = torch.zeros(width, dtype=torch.int64, device=sources.device)
    rc = 0
    if hi > lo:
        x, res, rc = solve(sources[lo:hi])
        mine[:hi - lo] = x
        my_it[:hi - lo] = torch.tensor([r.iterations for r in res], dtype=torch.int64, device=sources.device)
    if world == 1:
        return mine[:n], my_it[:n].tolist(), rc
    flat = torch.view_as_real(mine) if mine.is_complex() else mine
    blocks = [torch.empty_like(flat) for _ in range(world)]
    its = [torch.empty_like(my_it) for _ in range(world)]
    dist.all_gather(blocks, flat.contiguous(), group=group)
    dist.all_gather(its, my_it, group=group)
    worst = torch.tensor([min(rc, 0), max(rc, 0)], dtype=torch.int64, device=sources.device)
    neg, pos = worst[:1].clone(), worst[1:].clone()
    dist.all_reduce(neg, op=dist.ReduceOp.MIN, group=group)
    dist.all_reduce(pos, op=dist.ReduceOp.MAX, group=group)
    x_full = torch.empty_like(sources)
    iters = []
    for r in range(world):
        l, h = shard_columns(n, r, world)
        if h > l:
            blk = torch.view_as_complex(blocks[r]) if sources.is_complex() else blocks[r]
            x_full[l:h] = blk[:h - l]
            iters += its[r][:h - l].tolist()
    neg, pos = int(neg), int(pos)
    return x_full, iters, (neg if neg < 0 else pos)


class Context:
    """One lattice, precision and link reconstruction (init + LatticeInfo)."""

    def __init__(self, dims, prec=8, recon=18, t_boundary=-1, device=0):
        self.lib = load()
        self.dims = tuple(int(d) for d in dims)
        self.prec, self.recon, self.device = prec, recon, device
        h = ctypes.c_void_p()
        rc = self.lib.lqcd_create(ctypes.byref(h), (ctypes.c_int * 4)(*self.dims), prec, recon,
                                  t_boundary, device)
        if rc != 0:
            raise LqcdError("lqcd_create failed: %s (no CUDA sm_100 device => no fallback)"
                            % self.lib.lqcd_strerror(rc).decode())
        self.h = h
        self.dev = torch.device("cuda", device)
        # prec = 2: 16-bit native storage (int16 buffers), fp32 arithmetic, complex64 public arrays
        self.rdtype = {2: torch.int16, 4: torch.float32, 8: torch.float64}[prec]
        self.pub_rdtype = torch.float64 if prec == 8 else torch.float32
        self.cdtype = torch.complex128 if prec == 8 else torch.complex64
        self.np_cdtype = np.complex128 if prec == 8 else np.complex64
        Lx, Ly, Lz, Lt = self.dims
        self.site_shape = (2, Lt, Lz, Ly, Lx // 2)
        self.Vh = Lx * Ly * Lz * Lt // 2
        self.gauge_bytes = self.lib.lqcd_gauge_bytes(h)
        self.spinor_bytes = self.lib.lqcd_spinor_bytes(h)
        self.clover_bytes = self.lib.lqcd_clover_bytes(h)

    def close(self):
        if getattr(self, "h", None):
            self.lib.lqcd_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- helpers ---------------------------------------------------------------------------
    def _check(self, rc, allow_not_converged=False):
        if rc == 0 or (allow_not_converged and rc == 1):
            return rc
        raise LqcdError("%s: %s" % (self.lib.lqcd_strerror(rc).decode(),
                                    self.lib.lqcd_last_error(self.h).decode()))

    def launch_count(self):
        return self.lib.lqcd_launch_count(self.h)

    def graph_launch_count(self):
        return self.lib.lqcd_graph_launch_count(self.h)

    def algorithmic_bytes(self):
        return self.lib.lqcd_algorithmic_bytes(self.h)

    def profile_enable(self, on=True):
        self._check(self.lib.lqcd_profile_enable(self.h, int(on)))

    def profile_read(self):
        """(launches, total ms, total algorithmic bytes) of the dslash kernels recorded so far."""
        n, ms, by = ctypes.c_long(), ctypes.c_double(), ctypes.c_double()
        self._check(self.lib.lqcd_profile_read(self.h, ctypes.byref(n), ctypes.byref(ms), ctypes.byref(by)))
        return n.value, ms.value, by.value

    def gauge_pack_host(self, gauge_native, U_host, scratch):
        self._check(self.lib.lqcd_gauge_pack_host(self.h, _p(gauge_native), _p(U_host), _p(scratch), _stream()))
        return gauge_native

    def empty(self, nbytes):
        return torch.empty(nbytes // self.prec, dtype=self.rdtype, device=self.dev)

    def new_spinor(self, parities=1):
        return self.empty(self.spinor_bytes * parities)

    def to_device(self, a):
        """numpy public-layout array -> device tensor in this context's precision."""
        t = torch.from_numpy(np.ascontiguousarray(a))
        if t.is_complex():
            t = t.to(self.cdtype)
        else:
            t = t.to(self.pub_rdtype)
        return t.to(self.dev).contiguous()

    # ---- pack / unpack ---------------------------------------------------------------------
    def gauge_pack(self, U_public):
        g = self.empty(self.gauge_bytes)
        self._check(self.lib.lqcd_gauge_pack(self.h, _p(g), _p(U_public), _stream()))
        return g

    def spinor_pack(self, psi_public):
        s = self.new_spinor(2)
        self._check(self.lib.lqcd_spinor_pack(self.h, _p(s), _p(psi_public), _stream()))
        return s

    def spinor_unpack(self, s_native):
        out = torch.empty(self.site_shape + (4, 3), dtype=self.cdtype, device=self.dev)
        self._check(self.lib.lqcd_spinor_unpack(self.h, _p(out), _p(s_native), _stream()))
        return out

    def clover_unpack(self, cl_native):
        out = torch.empty(self.site_shape + (2, 36), dtype=self.pub_rdtype, device=self.dev)
        self._check(self.lib.lqcd_clover_unpack(self.h, _p(out), _p(cl_native), _stream()))
        return out

    def clover_pack(self, cl_public):
        out = self.empty(self.clover_bytes)
        self._check(self.lib.lqcd_clover_pack(self.h, _p(out), _p(cl_public), _stream()))
        return out

    def parity(self, s_native, p):
        n = self.spinor_bytes // self.prec
        return s_native[p * n:(p + 1) * n]

    # ---- operators -------------------------------------------------------------------------
    def clover_build(self, gauge, csw, kappa, want_inverse=True):
        A = self.empty(self.clover_bytes)
        Ai = self.empty(self.clover_bytes) if want_inverse else None
        self._check(self.lib.lqcd_clover_build(self.h, _p(A), _p(Ai), _p(gauge), csw, kappa, _stream()))
        return A, Ai

    def clover_build_noalloc(self, gauge, csw, kappa, out=None, out_inv=None):
        """lqcd_clover_build_noalloc: the build with the library's static scratch (at most clover_noalloc_max_sites()
        sites).  `out`, `out_inv`: native clover buffers of the caller (allocated here if None -- by torch, not by the
        library call)."""
        A = self.empty(self.clover_bytes) if out is None else out
        Ai = self.empty(self.clover_bytes) if out_inv is None else out_inv
        self._check(self.lib.lqcd_clover_build_noalloc(self.h, _p(A), _p(Ai), _p(gauge), csw, kappa, _stream()))
        return A, Ai

    def clover_noalloc_max_sites(self):
        return int(self.lib.lqcd_clover_noalloc_max_sites())

    def clover_to_half(self, clover_fp32_native):
        """self: 16-bit context; clover_fp32_native: A or A^-1 of an fp32 context of the same lattice."""
        out = self.empty(self.clover_bytes)
        self._check(self.lib.lqcd_clover_to_half(self.h, _p(out), _p(clover_fp32_native), _stream()))
        return out

    # ---- domain decomposition (include/lqcd.h; the exchange itself is in dd.py) ---------------------
    def set_partition(self, partitioned):
        self._check(self.lib.lqcd_set_partition(self.h, (ctypes.c_int * 4)(*[int(bool(v)) for v in partitioned])))
        return self

    def face_buffer(self, mu):
        return self.empty(self.lib.lqcd_face_bytes(self.h, mu))

    def dslash_dd_interior(self, out, inp, gauge, parity, scale=1.0, dagger=False):
        self._check(self.lib.lqcd_dslash_dd_interior(self.h, _p(out), _p(inp), _p(gauge), parity, scale, int(dagger), _stream()))
        return out

    def face_pack(self, face, inp, gauge, mu, direction, parity_in, dagger=False):
        self._check(self.lib.lqcd_face_pack(self.h, _p(face), _p(inp), _p(gauge), mu, direction, parity_in, int(dagger), _stream()))
        return face

    def face_unpack(self, out, face, gauge, mu, direction, parity_out, scale=1.0, weight=1.0, dagger=False):
        self._check(self.lib.lqcd_face_unpack(self.h, _p(out), _p(face), _p(gauge), mu, direction, parity_out, scale, weight,
                                              int(dagger), _stream()))
        return out

    def set_anisotropy(self, nu_over_xi0):
        self._check(self.lib.lqcd_set_anisotropy(self.h, nu_over_xi0))
        return self

    def clover_build_aniso(self, gauge, csw_s, csw_t, kappa, want_inverse=True):
        A = self.empty(self.clover_bytes)
        Ai = self.empty(self.clover_bytes) if want_inverse else None
        self._check(self.lib.lqcd_clover_build_aniso(self.h, _p(A), _p(Ai), _p(gauge), csw_s, csw_t, kappa, _stream()))
        return A, Ai

    def clover_apply(self, out, inp, clover, parity):
        self._check(self.lib.lqcd_clover_apply(self.h, _p(out), _p(inp), _p(clover), parity, _stream()))
        return out

    def dslash(self, out, inp, gauge, parity, scale=1.0, dagger=False):
        self._check(self.lib.lqcd_dslash(self.h, _p(out), _p(inp), _p(gauge), parity, scale,
                                         int(dagger), _stream()))
        return out

    def mpc_apply(self, out, inp, gauge, clover, clover_inv, kappa, matpc=0, dagger=False, tmp=None):
        tmp = tmp if tmp is not None else self.new_spinor()
        self._check(self.lib.lqcd_mpc_apply(self.h, _p(out), _p(inp), _p(gauge), _p(clover),
                                            _p(clover_inv), kappa, matpc, int(dagger), _p(tmp), _stream()))
        return out

    def mat_apply(self, out, inp, gauge, clover, kappa, dagger=False):
        self._check(self.lib.lqcd_mat_apply(self.h, _p(out), _p(inp), _p(gauge), _p(clover), kappa,
                                            int(dagger), _stream()))
        return out

    def workspace(self, solver="cgne"):
        n = self.lib.lqcd_invert_workspace_bytes(self.h, SOLVERS[solver])
        return self.empty(n), n

    def invert(self, b_public, gauge, clover, clover_inv, kappa, csw=0.0, tol=1e-10, maxiter=1000,
               solver="cgne", matpc=0, workspace=None):
        if workspace is None:
            workspace, _ = self.workspace(solver)
        x = torch.empty_like(b_public)
        res = Result()
        rc = self.lib.lqcd_invert(self.h, _p(x), _p(b_public), _p(gauge), _p(clover), _p(clover_inv),
                                  kappa, csw, tol, maxiter, SOLVERS[solver], matpc, _p(workspace),
                                  workspace.numel() * self.prec, ctypes.byref(res), _stream())
        self._check(rc, allow_not_converged=True)
        return x, res

    # ---- multi-right-hand-side forms (nrhs consecutive one-parity native spinors) -----------------
    def dslash_mrhs(self, out, inp, gauge, parity, nrhs, scale=1.0, dagger=False):
        self._check(self.lib.lqcd_dslash_mrhs(self.h, _p(out), _p(inp), _p(gauge), parity, scale,
                                              int(dagger), nrhs, _stream()))
        return out

    def mpc_apply_mrhs(self, out, inp, gauge, clover, clover_inv, kappa, nrhs, matpc=0, dagger=False, tmp=None):
        tmp = tmp if tmp is not None else self.new_spinor(nrhs)
        self._check(self.lib.lqcd_mpc_apply_mrhs(self.h, _p(out), _p(inp), _p(gauge), _p(clover),
                                                 _p(clover_inv), kappa, matpc, int(dagger), _p(tmp), nrhs,
                                                 _stream()))
        return out

    def workspace_multi(self, nrhs, solver="cgne"):
        n = self.lib.lqcd_invert_multi_workspace_bytes(self.h, SOLVERS[solver], nrhs)
        return self.empty(n), n

    def invert_multi(self, b_public, gauge, clover, clover_inv, kappa, tol=1e-10, maxiter=1000,
                     solver="cgne", matpc=0, workspace=None):
        """b_public: [nrhs, 2, Lt, Lz, Ly, Lx/2, 4, 3] device tensor; returns (x, [Result]*nrhs, status)."""
        nrhs = b_public.shape[0]
        if workspace is None:
            workspace, _ = self.workspace_multi(nrhs, solver)
        x = torch.empty_like(b_public)
        res = (Result * nrhs)()
        rc = self.lib.lqcd_invert_multi(self.h, _p(x), _p(b_public), _p(gauge), _p(clover), _p(clover_inv),
                                        kappa, tol, maxiter, SOLVERS[solver], matpc, nrhs, _p(workspace),
                                        workspace.numel() * self.prec, res, _stream())
        if rc < 0 and rc != -7:  # a breakdown of some column is reported per column
            self._check(rc)
        return x, list(res), rc

    def invert_mixed(self, lo, b_public, gauge, clover, clover_inv, gauge_lo, clover_lo, clover_inv_lo, kappa,
                     tol=1e-10, inner_tol=1e-4, maxiter=1000, solver="cgne", matpc=0, workspace=None,
                     workspace_lo=None):
        """self: fp64 context, lo: fp32 context of the same lattice (its own natives *_lo)."""
        if workspace is None:
            workspace, _ = self.workspace(solver)
        if workspace_lo is None:
            workspace_lo, _ = lo.workspace(solver)
        x = torch.empty_like(b_public)
        res = Result()
        rc = self.lib.lqcd_invert_mixed(self.h, lo.h, _p(x), _p(b_public), _p(gauge), _p(clover), _p(clover_inv),
                                        _p(gauge_lo), _p(clover_lo), _p(clover_inv_lo), kappa, tol, inner_tol,
                                        maxiter, SOLVERS[solver], matpc, _p(workspace),
                                        workspace.numel() * self.prec, _p(workspace_lo),
                                        workspace_lo.numel() * lo.prec, ctypes.byref(res), _stream())
        self._check(rc, allow_not_converged=True)
        return x, res

    def invert_multi_mixed(self, lo, b_public, gauge, clover, clover_inv, gauge_lo, clover_lo, clover_inv_lo, kappa,
                           tol=1e-10, inner_tol=1e-4, maxiter=1000, solver="cgne", matpc=0, workspace=None,
                           workspace_lo=None):
        """Batched mixed-precision solve.  b_public: [nrhs, 2, Lt, Lz, Ly, Lx/2, 4, 3] fp64 device tensor;
        returns (x, [Result]*nrhs, status)."""
        nrhs = b_public.shape[0]
        if workspace is None:
            workspace, _ = self.workspace_multi(nrhs, solver)
        if workspace_lo is None:
            workspace_lo, _ = lo.workspace_multi(nrhs, solver)
        x = torch.empty_like(b_public)
        res = (Result * nrhs)()
        rc = self.lib.lqcd_invert_multi_mixed(self.h, lo.h, _p(x), _p(b_public), _p(gauge), _p(clover), _p(clover_inv),
                                              _p(gauge_lo), _p(clover_lo), _p(clover_inv_lo), kappa, tol, inner_tol,
                                              maxiter, SOLVERS[solver], matpc, nrhs, _p(workspace),
                                              workspace.numel() * self.prec, _p(workspace_lo),
                                              workspace_lo.numel() * lo.prec, res, _stream())
        if rc < 0 and rc != -7:
            self._check(rc)
        return x, list(res), rc

    # ---- sources, propagators, contractions ----------------------------------
    def _gamma(self, g):
        g = np.ascontiguousarray(g, dtype=np.complex128).reshape(16)
        return (ctypes.c_double * 32)(*np.stack([g.real, g.imag], axis=1).ravel())

    def momentum_phase(self, mom):
        ph = torch.empty(self.site_shape, dtype=self.cdtype, device=self.dev)
        self._check(self.lib.lqcd_momentum_phase(self.h, _p(ph), (ctypes.c_int * 3)(*mom), _stream()))
        return ph

    def source_wall(self, t0, spin, colour, phase=None):
        b = torch.empty(self.site_shape + (4, 3), dtype=self.cdtype, device=self.dev)
        self._check(self.lib.lqcd_source_wall(self.h, _p(b), t0, spin, colour, _p(phase), _stream()))
        return b

    def source_point(self, x, spin, colour):
        b = torch.empty(self.site_shape + (4, 3), dtype=self.cdtype, device=self.dev)
        self._check(self.lib.lqcd_source_point(self.h, _p(b), (ctypes.c_int * 4)(*x), spin, colour, _stream()))
        return b

    def propagator_assemble(self, columns):
        prop = torch.empty(self.site_shape + (4, 4, 3, 3), dtype=self.cdtype, device=self.dev)
        self._check(self.lib.lqcd_propagator_assemble(self.h, _p(prop), _p(columns), _stream()))
        return prop

    def propagator_split(self, prop):
        cols = torch.empty((12,) + self.site_shape + (4, 3), dtype=self.cdtype, device=self.dev)
        self._check(self.lib.lqcd_propagator_split(self.h, _p(cols), _p(prop), _stream()))
        return cols

    def contract_twopt(self, phase, S_0, S_p):
        out = (ctypes.c_double * (2 * self.dims[3]))()
        self._check(self.lib.lqcd_contract_twopt(self.h, out, _p(phase), _p(S_0), _p(S_p), _stream()))
        return np.array(out).reshape(-1, 2) @ np.array([1, 1j])

    def contract_threept(self, S_p0, gamma, S_p):
        out = (ctypes.c_double * (2 * self.dims[3]))()
        self._check(self.lib.lqcd_contract_threept(self.h, out, _p(S_p0), self._gamma(gamma), _p(S_p), _stream()))
        return np.array(out).reshape(-1, 2) @ np.array([1, 1j])

    def sequential_source(self, phase, gamma, S_0, t):
        X = torch.empty_like(S_0)
        self._check(self.lib.lqcd_sequential_source(self.h, _p(X), _p(phase), self._gamma(gamma), _p(S_0), t, _stream()))
        return X

    def propagator(self, sources, gauge, clover, clover_inv, kappa, tol=1e-10, maxiter=1000, solver="cgne",
                   matpc=0, workspace=None):
        """The paper's `invert`: 12 source columns [12, site..., 4, 3] -> propagator, by
        one lqcd_invert_multi call and lqcd_propagator_assemble.  Returns (prop, results, status)."""
        x, res, rc = self.invert_multi(sources, gauge, clover, clover_inv, kappa, tol, maxiter, solver, matpc,
                                       workspace)
        return self.propagator_assemble(x), res, rc

    def propagator_sharded(self, sources, gauge, clover, clover_inv, kappa, tol=1e-10, maxiter=1000, solver="cgne",
                           matpc=0, group=None):
        """The paper's `invert` over several GPUs: see sharded_solve.
        Returns (prop, iterations per column, status)."""
        solve = lambda blk: self.invert_multi(blk, gauge, clover, clover_inv, kappa, tol, maxiter, solver, matpc)
        x, iters, rc = sharded_solve(sources, solve, group)
        return self.propagator_assemble(x), iters, rc

    # ---- host-buffer (end-to-end) entry points -----------------------------------------------
    def host_scratch(self, solver="cgne"):
        n = self.lib.lqcd_host_scratch_bytes(self.h, SOLVERS[solver])
        return self.empty(n), n

    def dslash_host(self, out_host, in_host, gauge, parity, scratch, scale=1.0, dagger=False):
        """out_host/in_host: pinned or pageable CPU tensors in the public two-parity layout."""
        self._check(self.lib.lqcd_dslash_host(self.h, _p(out_host), _p(in_host), _p(gauge), parity,
                                              scale, int(dagger), _p(scratch), _stream()))
        return out_host

    def invert_host(self, x_host, b_host, gauge, clover, clover_inv, kappa, scratch, tol=1e-10,
                    maxiter=1000, solver="cgne", matpc=0):
        res = Result()
        rc = self.lib.lqcd_invert_host(self.h, _p(x_host), _p(b_host), _p(gauge), _p(clover),
                                       _p(clover_inv), kappa, tol, maxiter, SOLVERS[solver], matpc,
                                       _p(scratch), scratch.numel() * self.prec, ctypes.byref(res),
                                       _stream())
        self._check(rc, allow_not_converged=True)
        return x_host, res

    def solve_host(self, x_host, b_host, U_host, gauge, clover, clover_inv, csw, kappa, g_scratch, scratch,
                   tol=1e-10, maxiter=1000, solver="cgne", matpc=0):
        """Host links + host source -> host solution in one call (uploads overlap the pack and the clover build)."""
        res = Result()
        rc = self.lib.lqcd_solve_host(self.h, _p(x_host), _p(b_host), _p(U_host), _p(gauge), _p(clover),
                                      _p(clover_inv), csw, kappa, tol, maxiter, SOLVERS[solver], matpc,
                                      _p(g_scratch), _p(scratch), scratch.numel() * self.prec, ctypes.byref(res),
                                      _stream())
        self._check(rc, allow_not_converged=True)
        return x_host, res

    # ---- BLAS-1 ----------------------------------------------------------------------------
    def blas_axpy_norm(self, a, x, y):
        out = ctypes.c_double()
        self._check(self.lib.lqcd_blas_axpy_norm(self.h, a, _p(x), _p(y), ctypes.byref(out), _stream()))
        return out.value

    def blas_xpay(self, x, a, y):
        self._check(self.lib.lqcd_blas_xpay(self.h, _p(x), a, _p(y), _stream()))

    def blas_cdot(self, x, y):
        out = (ctypes.c_double * 3)()
        self._check(self.lib.lqcd_blas_cdot(self.h, _p(x), _p(y), out, _stream()))
        return complex(out[0], out[1]), out[2]

    def blas_caxpbypz(self, a, x, b, y, z):
        A = (ctypes.c_double * 2)(a.real, a.imag)
        B = (ctypes.c_double * 2)(b.real, b.imag)
        self._check(self.lib.lqcd_blas_caxpbypz(self.h, A, _p(x), B, _p(y), _p(z), _stream()))
