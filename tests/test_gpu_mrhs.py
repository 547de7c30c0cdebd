"""GPU parity of the multi-right-hand-side path against the
oracle: every column of lqcd_dslash_mrhs / lqcd_mpc_apply_mrhs equals the oracle's operator on that
column (north_star tolerances), and every column of lqcd_invert_multi meets reading A17 (oracle's
solution within 10*tol, oracle-evaluated true residual below tol)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2411_08461_b200 import synth
from latt import rel_err
from test_gpu_parity import Setup, TOL, from_cfg, lq

pytestmark = pytest.mark.gpu


def pack_block(s, psis, parity):
    """list of public spinors -> device block [nrhs][one-parity native] of the given parity."""
    return torch.cat([s.ctx.parity(s.up(p), parity) for p in psis])


def unpack_block(s, block, nrhs, parity):
    n = s.ctx.spinor_bytes // s.ctx.prec
    out = []
    for r in range(nrhs):
        full = s.ctx.new_spinor(2)
        full.zero_()
        s.ctx.parity(full, parity).copy_(block[r * n:(r + 1) * n])
        out.append(s.down(full)[parity])
    return out


@pytest.mark.parametrize("prec,recon", [(8, 18), (8, 12), (4, 18), (4, 12)])
@pytest.mark.parametrize("dims,tb,nrhs", [((4, 6, 8, 10), -1, 12), ((8, 8, 8, 16), -1, 12), ((12, 4, 6, 4), 1, 5),
                                          ((4, 4, 4, 8), -1, 16), ((4, 4, 4, 8), -1, 2)])
def test_dslash_mrhs_matches_oracle(prec, recon, dims, tb, nrhs):
    s = Setup(dims, 0.5, 2, 0.124, 1.2, prec, recon, tb, with_clover=False)
    psis = [s.spinor("gaussian", 200 + r) for r in range(nrhs)]
    n = s.ctx.spinor_bytes // s.ctx.prec
    for dagger in (False, True):
        wants = [s.orc.dslash(p, dagger=dagger) for p in psis]
        for par in (0, 1):
            inp = pack_block(s, psis, 1 - par)
            out = s.ctx.new_spinor(nrhs)
            s.ctx.dslash_mrhs(out, inp, s.gauge, par, nrhs, 1.0, dagger)
            gots = unpack_block(s, out, nrhs, par)
            for r in range(nrhs):
                assert rel_err(gots[r], wants[r][par]) < TOL[prec], (dagger, par, r)
            # every column equals the single-RHS kernel's result up to rounding order
            single = s.ctx.new_spinor(1)
            s.ctx.dslash(single, inp[:n], s.gauge, par, 1.0, dagger)
            assert rel_err(out[:n].cpu().numpy().astype(np.float64), single.cpu().numpy().astype(np.float64)) < TOL[prec]


@pytest.mark.parametrize("prec,recon", [(8, 18), (4, 12)])
@pytest.mark.parametrize("nrhs", [12, 7])
def test_mpc_apply_mrhs(prec, recon, nrhs):
    s, c = from_cfg(2, prec, recon)
    psis = [s.spinor("gaussian", 300 + r) for r in range(nrhs)]
    for p in psis:
        p[1] = 0
    inp = pack_block(s, psis, 0)
    for matpc in (0, 1):
        for dagger in (False, True):
            out = s.ctx.new_spinor(nrhs)
            s.ctx.mpc_apply_mrhs(out, inp, s.gauge, s.A, s.Ai, s.kappa, nrhs, matpc, dagger)
            gots = unpack_block(s, out, nrhs, 0)
            for r in range(nrhs):
                assert rel_err(gots[r], s.orc.mpc(psis[r], matpc, dagger)[0]) < TOL[prec], (matpc, dagger, r)


@pytest.mark.parametrize("solver", ["cgne", "cgnr", "bicgstab"])
def test_invert_multi_fp64_config2(solver):
    """Columns of different difficulty (point, Z2, Gaussian, zero) in one batch: each column must be
    the solution of its own system, frozen at its own convergence."""
    s, c = from_cfg(2, 8, 18)
    dims = c["dims"]
    bs = [synth.source(dims, "point", spin=1, colour=2), synth.source(dims, "z2", 102),
          synth.source(dims, "gaussian", 5), np.zeros_like(synth.source(dims, "point")),
          synth.source(dims, "point", spin=3, colour=0)]
    B = s.ctx.to_device(np.stack(bs))
    x, res, rc = s.ctx.invert_multi(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, maxiter=2000, solver=solver)
    assert rc == 0
    xs = x.cpu().numpy()
    its = []  # per-column iteration counts (columns freeze independently; the zero column never starts)
    for r, b in enumerate(bs):
        assert res[r].status == 0
        if not b.any():
            assert res[r].iterations == 0 and not xs[r].any()
            continue
        true = s.orc.true_residual(b, xs[r])
        assert true < 1e-10 and abs(true - res[r].true_resid) < 5e-11, (r, true, res[r].as_dict())
        xo, ro = s.orc.invert(b, 1e-10, 2000, "bicgstab", 0)
        assert rel_err(xs[r], xo) < 1e-9, r
        # same answer and iteration count as the column's own single solve
        x1, r1 = s.ctx.invert(s.ctx.to_device(b), s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, maxiter=2000, solver=solver)
        assert r1.iterations == res[r].iterations
        assert rel_err(xs[r], x1.cpu().numpy()) < 1e-12
        its.append(res[r].iterations)


def test_invert_multi_maxiter_and_errors():
    s, c = from_cfg(1, 8, 18)
    bs = np.stack([synth.source(c["dims"], "gaussian", 9), synth.source(c["dims"], "point")])
    B = s.ctx.to_device(bs)
    x, res, rc = s.ctx.invert_multi(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, maxiter=3, solver="cgne")
    assert rc == 1 and all(r.status == 1 and r.iterations == 3 for r in res)
    with pytest.raises(lq().LqcdError):
        s.ctx.invert_multi(B, s.gauge, s.A, s.Ai, s.kappa, workspace=s.ctx.empty(1024))
    big = s.ctx.to_device(np.stack([bs[0]] * 17))
    with pytest.raises(lq().LqcdError):
        s.ctx.invert_multi(big, s.gauge, s.A, s.Ai, s.kappa)


def test_config3_propagator_12_columns_batched_fp32_recon12():
    """BASELINE config 3 through the batched path: the 12 spin-colour columns of a point-source
    propagator in ONE lqcd_invert_multi call (fp32, reconstruct-12, CGNE to 1e-6)."""
    s, c = from_cfg(3, 4, 12)
    dims = c["dims"]
    bs = [synth.source(dims, "point", spin=sp, colour=col) for sp in range(4) for col in range(3)]
    B = s.ctx.to_device(np.stack(bs))
    x, res, rc = s.ctx.invert_multi(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-6, solver="cgne")
    assert rc == 0
    xs = x.cpu().numpy().astype(np.complex128)
    for r in range(12):  # every column, oracle-evaluated, below the tolerance asked for (reading A17)
        assert s.orc.true_residual(bs[r], xs[r]) < 1e-6, (r, res[r].as_dict())
    for r in (0, 5, 10):
        xo, ro = s.orc.invert(bs[r], 1e-9, 2000, "cgne", 0)
        assert rel_err(xs[r], xo) < 1e-5, r
    # sink-source assembly [.., s_sink, s_src, c_sink, c_src] and gamma5-hermiticity at the source
    prop = np.zeros(s.orc.site_shape + (4, 4, 3, 3), dtype=np.complex128)
    for r in range(12):
        prop[..., :, r // 3, :, r % 3] = xs[r]
    S00 = prop[0, 0, 0, 0, 0].transpose(0, 2, 1, 3).reshape(12, 12)
    g5 = np.repeat([1, 1, -1, -1.0], 3)
    assert np.abs(g5[:, None] * S00 * g5[None, :] - S00.conj().T).max() < 1e-5 * np.abs(S00).max()


@pytest.mark.parametrize("solver", ["cgne", "bicgstab"])
def test_invert_multi_mixed_fp64_tolerance_config2(solver):
    """Batched mixed precision (SURVEY.md §8(f) ranks 1+2): fp64 defect correction around ONE batched fp32
    reconstruct-12 solve per outer step.  Every column (point, Z2, Gaussian, zero, point) must meet the bar of
    its own pure fp64 solve (reading A17): oracle solution within 10*tol, oracle-evaluated true residual < tol."""
    s, c = from_cfg(2, 8, 18)
    dims = c["dims"]
    lo = lq().Context(dims, 4, 12, -1)
    g_lo = lo.gauge_pack(lo.to_device(s.U))
    A_lo, Ai_lo = lo.clover_build(g_lo, c["csw"], c["kappa"])
    bs = [synth.source(dims, "point", spin=1, colour=2), synth.source(dims, "z2", 102),
          synth.source(dims, "gaussian", 5), np.zeros_like(synth.source(dims, "point")),
          synth.source(dims, "point", spin=3, colour=0)]
    B = s.ctx.to_device(np.stack(bs))
    x, res, rc = s.ctx.invert_multi_mixed(lo, B, s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo, s.kappa, tol=1e-10,
                                          inner_tol=1e-4, maxiter=2000, solver=solver)
    assert rc == 0, [r.as_dict() for r in res]
    xs = x.cpu().numpy()
    for r, b in enumerate(bs):
        assert res[r].status == 0
        if not b.any():
            assert res[r].iterations == 0 and not xs[r].any()
            continue
        true = s.orc.true_residual(b, xs[r])
        assert true < 1e-10 and abs(true - res[r].true_resid) < 5e-11, (r, true, res[r].as_dict())
        xo, ro = s.orc.invert(b, 1e-12, 2000, "bicgstab", 0)
        assert rel_err(xs[r], xo) < 1e-9, r
    # one column through the batched entry point = lqcd_invert_mixed
    x1, res1, rc1 = s.ctx.invert_multi_mixed(lo, B[1:2], s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo, s.kappa, tol=1e-10,
                                             inner_tol=1e-4, maxiter=2000, solver=solver)
    x2, res2 = s.ctx.invert_mixed(lo, B[1], s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo, s.kappa, tol=1e-10,
                                  inner_tol=1e-4, maxiter=2000, solver=solver)
    assert rc1 == 0 and res1[0].iterations == res2.iterations
    assert np.array_equal(x1[0].cpu().numpy(), x2.cpu().numpy())


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("dims,zslab", [((16, 4, 4, 4), "1"), ((32, 4, 6, 8), "3"), ((16, 8, 4, 6), "0"), ((32, 8, 8, 4), "2")])
def test_tma_mrhs_kernel_matches_oracle(dims, zslab, recon, monkeypatch):
    """The TMA-tiled multi-RHS kernel (csrc/dslash_mrhs_tma.cu; fp32, x-rows of 8 or 16 checkerboard sites): tiles
    whose halo wraps onto the tile itself (extent = tile), several z-slabs, odd column counts (the two ring stages
    change roles), dagger, both parities, every epilogue through the three Schur forms -- against the oracle, and
    against the kernels of dslash_mrhs.cu (LQCD_MRHS_TMA=0) which must give the same field to rounding."""
    monkeypatch.setenv("LQCD_MRHS_ZSLAB", zslab)
    monkeypatch.setenv("LQCD_MRHS_TMA", "2")  # also where it is not the default (x-rows of 8)
    s = Setup(dims, 0.5, 2, 0.124, 1.2, 4, recon, -1)
    monkeypatch.setenv("LQCD_MRHS_TMA", "0")
    ref = lq().Context(dims, 4, recon, -1)
    for nrhs in (12, 5, 2):
        psis = [s.spinor("gaussian", 200 + r) for r in range(nrhs)]
        for dagger in (False, True):
            wants = [s.orc.dslash(p, dagger=dagger) for p in psis]
            for par in (0, 1):
                out, out_ref = s.ctx.new_spinor(nrhs), s.ctx.new_spinor(nrhs)
                blk = pack_block(s, psis, 1 - par)
                s.ctx.dslash_mrhs(out, blk, s.gauge, par, nrhs, 0.7, dagger)
                ref.dslash_mrhs(out_ref, blk, s.gauge, par, nrhs, 0.7, dagger)
                assert float((out - out_ref).abs().max()) < 2e-5 * float(out_ref.abs().max())
                gots = unpack_block(s, out, nrhs, par)
                for r in range(nrhs):
                    assert rel_err(gots[r], 0.7 * wants[r][par]) < TOL[4], (nrhs, dagger, par, r)
        for matpc in (0, 1, 2):
            for dagger in (False, True):
                out = s.ctx.new_spinor(nrhs)
                s.ctx.mpc_apply_mrhs(out, pack_block(s, psis, 0), s.gauge, s.A, s.Ai, s.kappa, nrhs, matpc, dagger)
                gots = unpack_block(s, out, nrhs, 0)
                for r in range(nrhs):
                    pe = psis[r].copy()
                    pe[1] = 0
                    if matpc < 2:
                        want = s.orc.mpc(pe, matpc, dagger)
                    elif not dagger:  # Mhat_r = Mhat A_ee^-1, composed from the oracle's pieces (test_gpu_parity.py)
                        want = s.orc.mpc(s.orc.clover_apply(pe, inverse=True, only_parity=0), 0, False)
                    else:
                        want = s.orc.clover_apply(s.orc.mpc(pe, 0, True), inverse=True, only_parity=0)
                    assert rel_err(gots[r], want[0]) < TOL[4], (nrhs, matpc, dagger, r)


@pytest.mark.parametrize("nrhs", [12, 5])
def test_batched_bicgstab_inner_products_in_the_epilogues(nrhs, monkeypatch):
    """Batched BiCGStab on the left-symmetric form takes <r0,v> and <t,s>, |t|^2 from multi-RHS epilogues 12 and 11: in
    the TMA-tiled kernel where that serves epilogue 3 (fp32, 12-real links, x-rows of 16), in the register kernel
    (LQCD_MRHS_TMA=0), or from separate BLAS-1 passes (LQCD_MRHS_FUSE_DOTS=0).  All three must meet reading A17 on every
    column and agree on the iteration counts to +-1 (the sums differ in rounding order only)."""
    dims, kappa, csw = (32, 4, 6, 8), 0.124, 1.2
    bs = [synth.round_fp32(synth.source(dims, "gaussian", 300 + r)) for r in range(nrhs)]
    iters = {}
    for name, env in (("tma", {}), ("register", {"LQCD_MRHS_TMA": "0"}), ("blas", {"LQCD_MRHS_FUSE_DOTS": "0"})):
        for k in ("LQCD_MRHS_TMA", "LQCD_MRHS_FUSE_DOTS"):
            monkeypatch.delenv(k, raising=False)
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        s = Setup(dims, 0.5, 2, kappa, csw, 4, 12, -1)
        x, res, rc = s.ctx.invert_multi(s.ctx.to_device(np.stack(bs)), s.gauge, s.A, s.Ai, kappa, tol=1e-6, maxiter=500,
                                        solver="bicgstab", matpc=1)
        assert rc == 0, name
        xs = x.cpu().numpy().astype(np.complex128)
        for r, b in enumerate(bs):
            assert res[r].status == 0 and s.orc.true_residual(b, xs[r]) < 1e-6, (name, r, res[r].as_dict())
        iters[name] = [r.iterations for r in res]
        s.ctx.close()
    for name in ("register", "blas"):
        assert max(abs(a - b) for a, b in zip(iters["tma"], iters[name])) <= 1, iters


@pytest.mark.parametrize("solver,matpc", [("bicgstab", 1), ("cgne", 2)])
@pytest.mark.parametrize("recon", [12, 18])
def test_batched_solves_are_bitwise_reproducible(solver, matpc, recon):
    """Every reduction of the batched path is summed in a fixed order (per-warp shuffles, per-block partials, one block
    per column adding them in block order), so two runs of the same solve give the same bits and the same iteration
    counts -- in the TMA-tiled kernels (x-rows of 16) as in the register kernels.  A race in the shared-memory stages, the
    half-sum exchange or the partial buffers would show up here as a difference."""
    dims = (32, 8, 4, 6)
    s = Setup(dims, 0.5, 11, 0.124, 1.2, 4, recon, -1)
    bs = np.stack([synth.round_fp32(synth.source(dims, "gaussian", 400 + r)) for r in range(12)])
    B = s.ctx.to_device(bs)
    runs = []
    for _ in range(3):
        x, res, rc = s.ctx.invert_multi(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-6, maxiter=500, solver=solver, matpc=matpc)
        assert rc == 0
        runs.append((x.clone(), [r.iterations for r in res], [r.true_resid for r in res]))
    for x, its, tr in runs[1:]:
        assert its == runs[0][1] and tr == runs[0][2]
        assert torch.equal(x, runs[0][0])
    s.ctx.close()


def test_propagator_sharded_single_rank_equals_propagator():
    """Without a process group the column-sharded propagator is the batched one."""
    s, c = from_cfg(2, 8, 18)
    dims = c["dims"]
    cols = np.stack([synth.source(dims, "point", spin=sp, colour=co) for sp in range(4) for co in range(3)])
    B = s.ctx.to_device(cols)
    p1, res, rc1 = s.ctx.propagator(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, solver="bicgstab")
    p2, iters, rc2 = s.ctx.propagator_sharded(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, solver="bicgstab")
    assert rc1 == 0 and rc2 == 0 and iters == [r.iterations for r in res]
    assert torch.equal(p1, p2)


@pytest.mark.parametrize("solver", ["cgne", "bicgstab"])
@pytest.mark.parametrize("matpc", [1, 2])
def test_invert_multi_symmetric_forms_config2(solver, matpc):
    """Batched solves on the symmetric Schur complements (left and right; multi-RHS epilogue 6 and the batched clover
    apply for the clover-first products): every column meets reading A17 and equals the column's own single solve."""
    s, c = from_cfg(2, 8, 18)
    dims = c["dims"]
    bs = [synth.source(dims, "point", spin=1, colour=2), synth.source(dims, "z2", 102), synth.source(dims, "gaussian", 5)]
    B = s.ctx.to_device(np.stack(bs))
    x, res, rc = s.ctx.invert_multi(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, maxiter=2000, solver=solver, matpc=matpc)
    assert rc == 0
    xs = x.cpu().numpy()
    for r, b in enumerate(bs):
        true = s.orc.true_residual(b, xs[r])
        assert res[r].status == 0 and true < 1e-10 and abs(true - res[r].true_resid) < 5e-11, (r, true, res[r].as_dict())
        xo, ro = s.orc.invert(b, 1e-12, 2000, "bicgstab", 0)
        assert rel_err(xs[r], xo) < 1e-9, r
        x1, r1 = s.ctx.invert(s.ctx.to_device(b), s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, maxiter=2000, solver=solver,
                              matpc=matpc)
        assert r1.iterations == res[r].iterations and rel_err(xs[r], x1.cpu().numpy()) < 1e-11


@pytest.mark.parametrize("solver,matpc", [("cgne", 2), ("bicgstab", 1)])
def test_invert_multi_mixed_symmetric_forms_config2(solver, matpc):
    """The forms bench.py times for the mixed-precision rows (CGNE: right, BiCGStab: left), batched, against the oracle."""
    s, c = from_cfg(2, 8, 18)
    dims = c["dims"]
    lo = lq().Context(dims, 4, 12, -1)
    g_lo = lo.gauge_pack(lo.to_device(s.U))
    A_lo, Ai_lo = lo.clover_build(g_lo, c["csw"], c["kappa"])
    bs = [synth.source(dims, "point", spin=0, colour=1), synth.source(dims, "gaussian", 6), synth.source(dims, "z2", 103)]
    B = s.ctx.to_device(np.stack(bs))
    x, res, rc = s.ctx.invert_multi_mixed(lo, B, s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo, s.kappa, tol=1e-10,
                                          inner_tol=1e-4, maxiter=2000, solver=solver, matpc=matpc)
    assert rc == 0, [r.as_dict() for r in res]
    xs = x.cpu().numpy()
    for r, b in enumerate(bs):
        true = s.orc.true_residual(b, xs[r])
        assert true < 1e-10 and abs(true - res[r].true_resid) < 5e-11, (r, true, res[r].as_dict())
        xo, ro = s.orc.invert(b, 1e-12, 2000, "bicgstab", 0)
        assert rel_err(xs[r], xo) < 1e-9, r
    x1, r1 = s.ctx.invert_mixed(lo, B[1], s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo, s.kappa, tol=1e-10, inner_tol=1e-4,
                                maxiter=2000, solver=solver, matpc=matpc)
    assert r1.status == 0 and s.orc.true_residual(bs[1], x1.cpu().numpy()) < 1e-10
