"""4-D domain decomposition of the hopping term: host logic.

The lattice is divided equally over a Cartesian grid of ranks [Gx, Gy, Gz, Gt]; the rank index runs fastest in t
(PAPER.md:82).  Every rank owns one sub-lattice: its own lqcd.Context, links and spinors.  One application of D is
    interior hops (lqcd_dslash_dd_interior)  |  pack the faces (lqcd_face_pack)  ->  move them  ->  lqcd_face_unpack
with faces of projected half spinors (12 reals per face site).  This module holds the rank grid, the exchange
schedule, the two ways of moving faces (between sub-lattices held by one process on one GPU; between ranks with
torch.distributed send / recv), and the index permutations that cut a global field into sub-lattices.  No arithmetic
of the operator happens here: every multiply is in csrc/dd.cu.
"""
import numpy as np
import torch


class Partition:
    """dims = global (Lx, Ly, Lz, Lt), grid = (Gx, Gy, Gz, Gt).  Local extents must be even and >= 4, so that a local
    site has the parity of its global site and the kernels' own wrap-around never meets a cut."""

    def __init__(self, dims, grid, t_boundary=-1):
        self.dims, self.grid, self.t_boundary = tuple(dims), tuple(grid), t_boundary
        for L, G in zip(self.dims, self.grid):
            if G < 1 or L % G or (L // G) % 2 or L // G < 4:
                raise ValueError("every local extent L/G must be an even integer >= 4: %r / %r" % (dims, grid))
        self.local = tuple(L // G for L, G in zip(self.dims, self.grid))
        self.size = int(np.prod(self.grid))
        self.partitioned = [G > 1 for G in self.grid]

    def coords(self, rank):
        """(gx, gy, gz, gt) of a rank; t runs fastest."""
        Gx, Gy, Gz, Gt = self.grid
        gt = rank % Gt
        rank //= Gt
        gz = rank % Gz
        rank //= Gz
        return (rank // Gy, rank % Gy, gz, gt)

    def rank(self, c):
        Gx, Gy, Gz, Gt = self.grid
        return ((c[0] % Gx * Gy + c[1] % Gy) * Gz + c[2] % Gz) * Gt + c[3] % Gt

    def neighbour(self, rank, mu, direction):
        c = list(self.coords(rank))
        c[mu] += direction
        return self.rank(c)

    def origin(self, rank):
        return tuple(g * l for g, l in zip(self.coords(rank), self.local))

    def local_t_boundary(self):
        """t_boundary of the sub-lattice contexts: with t cut no interior hop crosses the global seam."""
        return 1 if self.grid[3] > 1 else self.t_boundary

    def ghost_weight(self, rank, mu, kind, ws=1.0):
        """Weight of the hop served by a ghost face on `rank`: kind = +1 forward ghost (hop from my upper edge), -1
        backward ghost (hop from my lower edge).  Spatial: nu/xi_0.  t: -1 where the hop crosses the antiperiodic seam
        between global t = Lt-1 and 0."""
        if mu < 3:
            return ws
        gt = self.coords(rank)[3]
        at_seam = gt == self.grid[3] - 1 if kind > 0 else gt == 0
        return float(self.t_boundary) if at_seam else 1.0

    def messages(self, rank):
        """The faces `rank` sends and receives in one application, as (mu, kind, peer, tag): kind = +1 a forward ghost
        (packed from the sender's FIRST slice, sent to its -mu neighbour, unpacked on the receiver's upper edge),
        kind = -1 a backward ghost (sender's LAST slice, to its +mu neighbour).  tag = 2 mu + (kind > 0): with two ranks
        in a direction both neighbours are the same rank and only the tag tells the two faces apart."""
        sends, recvs = [], []
        for mu in range(4):
            if not self.partitioned[mu]:
                continue
            for kind in (+1, -1):
                tag = 2 * mu + (1 if kind > 0 else 0)
                sends.append((mu, kind, self.neighbour(rank, mu, -kind), tag))   # my first slice goes down, my last slice up
                recvs.append((mu, kind, self.neighbour(rank, mu, +kind), tag))   # a forward ghost comes from above
        return sends, recvs


# ---- cutting global cb2 fields [2, Lt, Lz, Ly, Lx/2, ...] into sub-lattices (index permutations only) -------------
def _cb_to_lex(f, dims):
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return f[(x + y + z + t) & 1, t, z, y, x // 2]


def _lex_to_cb(f, dims):
    Lx, Ly, Lz, Lt = dims
    par, t, z, y, xh = np.meshgrid(np.arange(2), np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx // 2), indexing="ij")
    return f[t, z, y, 2 * xh + ((par + y + z + t) & 1)]


def split_field(part, field):
    """Global public field [2, Lt, Lz, Ly, Lx/2, ...] -> list over ranks of local public fields."""
    lex = _cb_to_lex(field, part.dims)
    lx, ly, lz, lt = part.local
    out = []
    for r in range(part.size):
        ox, oy, oz, ot = part.origin(r)
        out.append(np.ascontiguousarray(_lex_to_cb(lex[ot:ot + lt, oz:oz + lz, oy:oy + ly, ox:ox + lx], part.local)))
    return out


def join_field(part, pieces):
    lx, ly, lz, lt = part.local
    Lx, Ly, Lz, Lt = part.dims
    lex = np.empty((Lt, Lz, Ly, Lx) + pieces[0].shape[5:], dtype=pieces[0].dtype)
    for r, p in enumerate(pieces):
        ox, oy, oz, ot = part.origin(r)
        lex[ot:ot + lt, oz:oz + lz, oy:oy + ly, ox:ox + lx] = _cb_to_lex(p, part.local)
    return _lex_to_cb(lex, part.dims)


def split_gauge(part, U):
    """Global public links [4, 2, Lt, Lz, Ly, Lx/2, 3, 3] -> list over ranks of local public links."""
    per_mu = [split_field(part, U[mu]) for mu in range(4)]
    return [np.stack([per_mu[mu][r] for mu in range(4)]) for r in range(part.size)]


# ---- one application of D on a decomposed lattice ------------------------------------------------------------------
def _pack_all(part, rank, ctx, inp, gauge, parity_out, dagger):
    """Interior hops are launched by the caller; here: every face this rank sends, keyed by tag."""
    faces = {}
    for mu, kind, peer, tag in part.messages(rank)[0]:
        buf = ctx.face_buffer(mu)
        ctx.face_pack(buf, inp, gauge, mu, kind, 1 - parity_out, dagger)
        faces[tag] = (buf, peer)
    return faces


def _unpack_all(part, rank, ctx, out, gauge, received, parity_out, scale, dagger, ws):
    for mu, kind, peer, tag in part.messages(rank)[1]:
        ctx.face_unpack(out, received[tag], gauge, mu, kind, parity_out, scale, part.ghost_weight(rank, mu, kind, ws), dagger)


def dslash_dd_emulated(part, ctxs, outs, ins, gauges, parity, scale=1.0, dagger=False, ws=1.0):
    """All ranks of `part` held by this process on one device (tests; a single-GPU stand-in for the multi-GPU path):
    outs[r] = scale * D_{p,1-p} ins[r] on every sub-lattice, faces moved by device copies."""
    sent = []
    for r in range(part.size):
        ctxs[r].dslash_dd_interior(outs[r], ins[r], gauges[r], parity, scale, dagger)
        sent.append(_pack_all(part, r, ctxs[r], ins[r], gauges[r], parity, dagger))
    for r in range(part.size):
        received = {}
        for mu, kind, peer, tag in part.messages(r)[1]:
            buf, dest = sent[peer][tag]
            assert dest == r, "exchange schedule: the face with tag %d of rank %d is not addressed to rank %d" % (tag, peer, r)
            received[tag] = buf.clone()
        _unpack_all(part, r, ctxs[r], outs[r], gauges[r], received, parity, scale, dagger, ws)
    return outs


def exchange(part, rank, faces, group=None):
    """Move the packed faces between ranks with torch.distributed point-to-point calls.  faces: {tag: (tensor, peer)}
    as _pack_all returns them; returns {tag: received tensor}.  Receives are posted first; a face and its reply to
    the same peer differ by their tag."""
    import torch.distributed as dist
    received, reqs = {}, []
    for mu, kind, peer, tag in part.messages(rank)[1]:
        buf = torch.empty_like(faces[tag][0])
        received[tag] = buf
        reqs.append(dist.irecv(buf, src=peer, group=group, tag=tag))
    for tag, (buf, peer) in faces.items():
        reqs.append(dist.isend(buf, dst=peer, group=group, tag=tag))
    for q in reqs:
        q.wait()
    return received


def dslash_dd(part, rank, ctx, out, inp, gauge, parity, scale=1.0, dagger=False, ws=1.0, group=None):
    """This rank's share of out = scale * D_{p,1-p} in on a lattice decomposed over a torch.distributed group
    (one process per GPU): the faces are packed first, the interior hops run while they travel."""
    faces = _pack_all(part, rank, ctx, inp, gauge, parity, dagger)
    torch.cuda.current_stream().synchronize()  # the faces are complete before they are handed to the transport
    ctx.dslash_dd_interior(out, inp, gauge, parity, scale, dagger)
    received = exchange(part, rank, faces, group)
    _unpack_all(part, rank, ctx, out, gauge, received, parity, scale, dagger, ws)
    return out


# ---- M-hat and an even-odd CGNE solve on a decomposed lattice ------------------------------------------------------
class Decomposed:
    """The sub-lattices this process holds (all of them on one device: emulation and tests; exactly one, with a
    torch.distributed group: one process per GPU) with their contexts and native fields, and the three things a Krylov
    solve needs across them: D with its face exchange, sums over all ranks, and the BLAS-1 calls of the C ABI with
    host coefficients.  The solve is host-driven (one scalar round trip per reduction): it is the correctness
    reference of the decomposed path, not a tuned solver.  The clover fields are given (cut from a field built on the
    whole lattice: a sub-lattice cannot build its edge sites' clover leaves from its own links alone)."""

    def __init__(self, part, ranks, ctxs, gauges, A, Ai, group=None, ws=1.0):
        self.part, self.ranks, self.ctxs, self.gauges, self.A, self.Ai = part, list(ranks), ctxs, gauges, A, Ai
        self.group, self.ws = group, ws
        self.emulated = group is None
        if self.emulated and len(self.ranks) != part.size:
            raise ValueError("without a process group this process must hold every sub-lattice")
        if not self.emulated and len(self.ranks) != 1:
            raise ValueError("with a process group a process holds one sub-lattice")

    def new(self):
        return [c.new_spinor(1) for c in self.ctxs]

    def dslash(self, outs, ins, parity, scale=1.0, dagger=False):
        if self.emulated:
            return dslash_dd_emulated(self.part, self.ctxs, outs, ins, self.gauges, parity, scale, dagger, self.ws)
        dslash_dd(self.part, self.ranks[0], self.ctxs[0], outs[0], ins[0], self.gauges[0], parity, scale, dagger, self.ws, self.group)
        return outs

    def allsum(self, values):
        """values: one float or complex per held sub-lattice -> the sum over ALL ranks."""
        s = complex(sum(values))
        if not self.emulated:
            import torch.distributed as dist
            t = torch.tensor([s.real, s.imag], dtype=torch.float64)
            if dist.get_backend(self.group) == "nccl":
                t = t.cuda()
            dist.all_reduce(t, group=self.group)
            s = complex(float(t[0]), float(t[1]))
        return s

    def clover(self, outs, ins, field, parity):
        for c, o, i, f in zip(self.ctxs, outs, ins, field):
            c.clover_apply(o, i, f, parity)
        return outs

    def mpc(self, outs, ins, kappa, dagger, tmp, tmp2):
        """Asymmetric even-even Schur complement: out = A_ee in - kappa^2 D_eo A_oo^-1 D_oe in."""
        self.dslash(tmp2, ins, 1, 1.0, dagger)
        self.clover(tmp, tmp2, self.Ai, 1)
        self.dslash(outs, tmp, 0, -kappa * kappa, dagger)
        self.clover(tmp2, ins, self.A, 0)
        for c, o, t2 in zip(self.ctxs, outs, tmp2):
            c.blas_caxpbypz(1.0, t2, 0.0, t2, o)        # out += A_ee in
        return outs

    def norm2(self, xs):
        return self.allsum([c.blas_cdot(x, x)[1] for c, x in zip(self.ctxs, xs)]).real

    def cgne(self, x, bhat, kappa, tol2_abs, maxiter):
        """CGNE (O9) on Mhat Mhat^dag y = bhat, x = Mhat^dag y; x is zeroed here.  Returns (iterations, |r|^2)."""
        r, p, t, q, tmp, tmp2 = (self.new() for _ in range(6))
        for xx, rr, pp, b in zip(x, r, p, bhat):
            xx.zero_()
            rr.copy_(b)
            pp.copy_(b)
        rr2 = self.norm2(r)
        it = 0
        while it < maxiter and rr2 > tol2_abs:
            self.mpc(t, p, kappa, True, tmp, tmp2)          # t = Mhat^dag p
            alpha = rr2 / self.norm2(t)
            self.mpc(q, t, kappa, False, tmp, tmp2)         # q = Mhat t
            for c, xx, tt, rr, qq in zip(self.ctxs, x, t, r, q):
                c.blas_caxpbypz(alpha, tt, 0.0, tt, xx)     # x += alpha t
                c.blas_caxpbypz(-alpha, qq, 0.0, qq, rr)    # r -= alpha q
            new = self.norm2(r)
            for c, pp, rr in zip(self.ctxs, p, r):
                c.blas_xpay(rr, new / rr2, pp)              # p = r + beta p
            rr2 = new
            it += 1
        return it, rr2

    def invert(self, b_natives, kappa, tol=1e-10, maxiter=2000):
        """M x = b through the even-even system (O8): b_natives / result: two-parity native spinors per held sub-lattice."""
        cs = self.ctxs
        b_e = [c.parity(b, 0) for c, b in zip(cs, b_natives)]
        b_o = [c.parity(b, 1) for c, b in zip(cs, b_natives)]
        bb = self.norm2(b_e) + self.norm2(b_o)
        xs = [c.new_spinor(2) for c in cs]
        x_e = [c.parity(x, 0) for c, x in zip(cs, xs)]
        x_o = [c.parity(x, 1) for c, x in zip(cs, xs)]
        bhat, tmp = self.new(), self.new()
        self.clover(tmp, b_o, self.Ai, 1)
        self.dslash(bhat, tmp, 0, kappa)                    # kappa D_eo A_oo^-1 b_o
        for c, bh, be in zip(cs, bhat, b_e):
            c.blas_caxpbypz(1.0, be, 0.0, be, bh)           # + b_e
        it, rr2 = self.cgne(x_e, bhat, kappa, tol * tol * bb, maxiter)
        self.dslash(tmp, x_e, 1, kappa)                     # x_o = A_oo^-1 (b_o + kappa D_oe x_e)
        for c, t, bo in zip(cs, tmp, b_o):
            c.blas_caxpbypz(1.0, bo, 0.0, bo, t)
        self.clover(x_o, tmp, self.Ai, 1)
        return xs, it, (rr2 / bb) ** 0.5
