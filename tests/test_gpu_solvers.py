"""GPU parity of lqcd_invert against the oracle's solvers and operator (reading A17): the solution
is unique, so the GPU's x must agree with the oracle's x within 10*tol, and the TRUE residual of
the GPU's x, evaluated by the oracle's own M, must be below tol."""
import numpy as np
import pytest
import torch

import oracle
from paper_2411_08461_b200 import synth
from latt import rel_err
from test_gpu_parity import Setup, from_cfg, lq

pytestmark = pytest.mark.gpu


def solve_and_check(s, b, solver, matpc, tol, oracle_solution=None, resid_bound=None):
    bd = s.ctx.to_device(b)
    x, res = s.ctx.invert(bd, s.gauge, s.A, s.Ai, s.kappa, tol=tol, maxiter=2000, solver=solver, matpc=matpc)
    xg = x.cpu().numpy().astype(np.complex128)
    assert res.status == 0, (solver, matpc, res.as_dict())
    true = s.orc.true_residual(b, xg)
    bound = resid_bound if resid_bound is not None else tol
    assert true < bound, (solver, matpc, true, res.as_dict())
    assert abs(res.true_resid - true) < 0.5 * bound
    if oracle_solution is not None:
        assert rel_err(xg, oracle_solution) < 10 * tol, (solver, matpc)
    return xg, res


def test_config1_point_source_cgne_fp64():
    s, c = from_cfg(1, 8, 18)
    b = synth.source(c["dims"], "point")
    xo, ro = s.orc.invert(b, 1e-10, 2000, "cgne", 0)
    assert ro.status == 0
    xg, res = solve_and_check(s, b, "cgne", 0, 1e-10, xo)
    assert abs(res.iterations - ro.iterations) <= 1
    # paper's normalisation: a_t M = M/(2 kappa), so its propagator is 2 kappa x (reading A2)
    assert res.dslash_count > 0 and res.kernel_launches > 0 and res.seconds > 0


@pytest.mark.parametrize("solver", ["cgne", "cgnr", "bicgstab"])
@pytest.mark.parametrize("matpc", [0, 1, 2])
def test_config2_z2_source_fp64(solver, matpc):
    s, c = from_cfg(2, 8, 18)
    b = synth.source(c["dims"], "z2", c["src_seed"])
    xo, ro = s.orc.invert(b, 1e-10, 2000, "bicgstab", 0)
    xg, res = solve_and_check(s, b, solver, matpc, 1e-10, xo)


@pytest.mark.parametrize("recon", [18, 12])
def test_config2_bicgstab_fp32(recon):
    s, c = from_cfg(2, 4, recon)
    b = synth.source(c["dims"], "z2", c["src_seed"])
    xo, ro = s.orc.invert(b, 1e-10, 2000, "bicgstab", 0)
    # north_star: fp32 solve to 1e-6; the oracle-evaluated true residual must be < 1e-6 as well (reading A17):
    # a column whose true residual misses is restarted from its x with the recomputed residual (solver.cu)
    solve_and_check(s, b, "bicgstab", 0, 1e-6, xo)
    solve_and_check(s, b, "cgne", 0, 1e-6, xo)
    # the symmetric forms in fp32 (packed FFMA2 epilogues 6-10, clover_mul_twice)
    for matpc in (1, 2):
        solve_and_check(s, b, "cgne", matpc, 1e-6, xo)
        solve_and_check(s, b, "bicgstab", matpc, 1e-6, xo)


def test_invert_builds_clover_when_absent_and_edge_cases():
    s, c = from_cfg(1, 8, 18)
    b = synth.source(c["dims"], "gaussian", 9)
    bd = s.ctx.to_device(b)
    x1, r1 = s.ctx.invert(bd, s.gauge, None, None, s.kappa, csw=s.csw, tol=1e-10, solver="bicgstab")
    x2, r2 = s.ctx.invert(bd, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, solver="bicgstab")
    assert r1.status == 0 and torch.equal(x1, x2)
    # zero source -> zero solution, no iterations
    x0, r0 = s.ctx.invert(torch.zeros_like(bd), s.gauge, s.A, s.Ai, s.kappa)
    assert r0.status == 0 and r0.iterations == 0 and float(x0.abs().max()) == 0.0
    # maxiter exhausted -> NOT_CONVERGED (+1), x is still the best iterate
    x3, r3 = s.ctx.invert(bd, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, maxiter=3, solver="cgne")
    assert r3.status == 1 and r3.iterations == 3 and r3.true_resid > 1e-10
    xo, ro = s.orc.invert(b, 1e-10, 3, "cgne", 0)
    assert rel_err(x3.cpu().numpy(), xo) < 1e-12
    # workspace too small / bad solver id
    ws = s.ctx.empty(1024)
    with pytest.raises(lq().LqcdError):
        s.ctx.invert(bd, s.gauge, s.A, s.Ai, s.kappa, workspace=ws)


def test_host_entry_points():
    s, c = from_cfg(1, 8, 18)
    b = synth.source(c["dims"], "gaussian", 9)
    bh = torch.from_numpy(b).pin_memory()
    xh = torch.empty_like(bh).pin_memory()
    scratch, _ = s.ctx.host_scratch("bicgstab")
    _, res = s.ctx.invert_host(xh, bh, s.gauge, s.A, s.Ai, s.kappa, scratch, tol=1e-10, solver="bicgstab")
    assert res.status == 0 and s.orc.true_residual(b, xh.numpy()) < 1e-10
    oh = torch.zeros_like(bh)
    for p in (0, 1):
        s.ctx.dslash_host(oh, bh, s.gauge, p, scratch)
    assert rel_err(oh.numpy(), s.orc.dslash(b)) < 1e-13
    # the whole path from host buffers in one call: host links + host source -> host solution, native fields left
    # behind for later calls
    Uh = torch.from_numpy(s.U).pin_memory()
    gauge, g_scr = s.ctx.empty(s.ctx.gauge_bytes), s.ctx.empty(Uh.numel() * 16)
    A, Ai = s.ctx.empty(s.ctx.clover_bytes), s.ctx.empty(s.ctx.clover_bytes)
    for matpc in (0, 2):
        x2 = torch.zeros_like(bh).pin_memory()
        _, r2 = s.ctx.solve_host(x2, bh, Uh, gauge, A, Ai, s.csw, s.kappa, g_scr, scratch, tol=1e-10, solver="cgne",
                                 matpc=matpc)
        assert r2.status == 0 and s.orc.true_residual(b, x2.numpy()) < 1e-10
        assert rel_err(x2.numpy(), xh.numpy()) < 1e-9
    assert torch.equal(gauge, s.gauge) and torch.equal(A, s.A) and torch.equal(Ai, s.Ai)


def test_config3_propagator_12_columns_fp32_recon12():
    """BASELINE config 3: 16^3x32, fp32, reconstruct-12, point source, all 12 spin-colour columns by
    CGNE, assembled sink-source.  Every column's true residual is checked with the
    oracle's operator (< tol, reading A17); three columns are compared with the oracle's own solve."""
    s, c = from_cfg(3, 4, 12)
    dims = c["dims"]
    prop = np.zeros(s.orc.site_shape + (4, 4, 3, 3), dtype=np.complex128)
    ws, _ = s.ctx.workspace("cgne")
    for spin in range(4):
        for col in range(3):
            b = synth.source(dims, "point", spin=spin, colour=col)
            x, res = s.ctx.invert(s.ctx.to_device(b), s.gauge, s.A, s.Ai, s.kappa, tol=1e-6, solver="cgne",
                                  workspace=ws)
            assert res.status == 0
            xg = x.cpu().numpy().astype(np.complex128)
            prop[..., :, spin, :, col] = xg
            assert s.orc.true_residual(b, xg) < 1e-6, (spin, col, res.as_dict())
            if (spin, col) in ((0, 0), (1, 2), (3, 1)):
                xo, ro = s.orc.invert(b, 1e-9, 2000, "cgne", 0)
                assert rel_err(xg, xo) < 1e-5
    # gamma5-hermiticity of the point-to-point propagator at the source: g5 S(0,0) g5 = S(0,0)^dag
    S00 = prop[0, 0, 0, 0, 0].transpose(0, 2, 1, 3).reshape(12, 12)   # (s_sink,c_sink),(s_src,c_src)
    g5 = np.repeat([1, 1, -1, -1.0], 3)
    assert np.abs(g5[:, None] * S00 * g5[None, :] - S00.conj().T).max() < 1e-5 * np.abs(S00).max()


@pytest.mark.parametrize("solver", ["cgne", "bicgstab"])
@pytest.mark.parametrize("recon_lo", [18, 12])
def test_config2_mixed_precision_reaches_fp64_tolerance(solver, recon_lo):
    """fp64 defect correction around fp32 solves must meet the SAME bar as the
    pure fp64 solve (reading A17): oracle solution within 10*tol, oracle-evaluated true residual < tol."""
    s, c = from_cfg(2, 8, 18)
    lo = lq().Context(c["dims"], 4, recon_lo, -1)
    g_lo = lo.gauge_pack(lo.to_device(s.U))
    A_lo, Ai_lo = lo.clover_build(g_lo, c["csw"], c["kappa"])
    b = synth.source(c["dims"], "z2", c["src_seed"])
    xo, ro = s.orc.invert(b, 1e-12, 2000, "bicgstab", 0)
    x, res = s.ctx.invert_mixed(lo, s.ctx.to_device(b), s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo, s.kappa,
                                tol=1e-10, inner_tol=1e-4, maxiter=2000, solver=solver)
    assert res.status == 0, res.as_dict()
    xg = x.cpu().numpy()
    true = s.orc.true_residual(b, xg)
    assert true < 1e-10 and abs(true - res.true_resid) < 5e-11, (true, res.as_dict())
    assert rel_err(xg, xo) < 1e-9
    # a tolerance below the fp32 floor of the inner solver is still reached (more outer steps)
    x2, res2 = s.ctx.invert_mixed(lo, s.ctx.to_device(b), s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo, s.kappa,
                                  tol=1e-13, inner_tol=1e-3, maxiter=4000, solver=solver)
    assert res2.status == 0 and s.orc.true_residual(b, x2.cpu().numpy()) < 1e-13
    # argument checks: contexts swapped / same precision
    with pytest.raises(lq().LqcdError):
        s.ctx.invert_mixed(s.ctx, s.ctx.to_device(b), s.gauge, s.A, s.Ai, s.gauge, s.A, s.Ai, s.kappa)


@pytest.mark.parametrize("prec,recon,tol", [(8, 18, 1e-10), (8, 12, 1e-10), (4, 12, 1e-6)])
def test_single_bicgstab_inner_products_in_the_epilogues(prec, recon, tol, monkeypatch):
    """BiCGStab on the left-symmetric form, one column: <r0,v> and <t,s>, |t|^2 come out of epilogues 12 and 11 of the
    single-RHS dslash kernel (three per-block partials, fixed-order sums); LQCD_MRHS_FUSE_DOTS=0 takes them from BLAS-1
    passes instead.  Both meet reading A17, agree on the iteration count to +-1, and the fused solve is reproducible
    bit for bit."""
    dims = (8, 6, 8, 12)
    b = synth.source(dims, "gaussian", 77)
    out = {}
    for name, env in (("fused", None), ("blas", "0")):
        if env is None:
            monkeypatch.delenv("LQCD_MRHS_FUSE_DOTS", raising=False)
        else:
            monkeypatch.setenv("LQCD_MRHS_FUSE_DOTS", env)
        s = Setup(dims, 0.5, 4, 0.124, 1.2, prec, recon)
        bb = synth.round_fp32(b) if prec == 4 else b
        runs = []
        for _ in range(2):
            x, res = s.ctx.invert(s.ctx.to_device(bb), s.gauge, s.A, s.Ai, s.kappa, tol=tol, maxiter=500, solver="bicgstab", matpc=1)
            runs.append(x.clone())
        assert torch.equal(runs[0], runs[1])
        true = s.orc.true_residual(bb, x.cpu().numpy().astype(np.complex128))
        assert res.status == 0 and true < tol, (name, true, res.as_dict())
        out[name] = res.iterations
        s.ctx.close()
    assert abs(out["fused"] - out["blas"]) <= 1, out


@pytest.mark.parametrize("margin", ["1e30", "0", None])
@pytest.mark.parametrize("solver,matpc", [("cgne", 2), ("bicgstab", 1), ("cgne", 0)])
def test_mixed_last_outer_step_guess(solver, matpc, margin, monkeypatch):
    """A mixed solve closes (x_o, true residual) as soon as the inner recurrences say the bar is met, without an fp64
    Schur residual of its own; a wrong guess must reopen the iteration.  LQCD_MIXED_LAST_MARGIN=1e30 makes every outer
    step a guess (so the early ones are wrong), 0 never guesses, unset is the default: the same bar is met each time,
    single and batched (the batch freezes columns as they finish)."""
    if margin is None:
        monkeypatch.delenv("LQCD_MIXED_LAST_MARGIN", raising=False)
    else:
        monkeypatch.setenv("LQCD_MIXED_LAST_MARGIN", margin)
    s, c = from_cfg(2, 8, 18)
    lo = lq().Context(c["dims"], 4, 12, -1)
    g_lo = lo.gauge_pack(lo.to_device(s.U))
    A_lo, Ai_lo = lo.clover_build(g_lo, c["csw"], c["kappa"])
    bs = [synth.source(c["dims"], "z2", c["src_seed"]), synth.source(c["dims"], "point", spin=2, colour=1),
          synth.source(c["dims"], "gaussian", 7)]
    x, res = s.ctx.invert_mixed(lo, s.ctx.to_device(bs[0]), s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo, s.kappa,
                                tol=1e-10, inner_tol=1e-3, maxiter=2000, solver=solver, matpc=matpc)
    true = s.orc.true_residual(bs[0], x.cpu().numpy())
    assert res.status == 0 and true < 1e-10 and abs(true - res.true_resid) < 5e-11, (true, res.as_dict())
    xm, resm, rc = s.ctx.invert_multi_mixed(lo, s.ctx.to_device(np.stack(bs)), s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo,
                                            s.kappa, tol=1e-10, inner_tol=1e-3, maxiter=2000, solver=solver, matpc=matpc)
    assert rc == 0
    xs = xm.cpu().numpy()
    for r, b in enumerate(bs):
        true = s.orc.true_residual(b, xs[r])
        assert resm[r].status == 0 and true < 1e-10 and abs(true - resm[r].true_resid) < 5e-11, (r, true, resm[r].as_dict())


@pytest.mark.parametrize("matpc", [0, 1, 2])
def test_config2_cgne_fp64_recon12(matpc):
    """fp64 with reconstruct-12 links: the kernel variant that stages its links through shared memory with cp.async
    (exactly 48 KB of dynamic shared memory) under the CG-fused epilogues, which add static shared memory of their own."""
    s, c = from_cfg(2, 8, 12)
    b = synth.source(c["dims"], "z2", c["src_seed"])
    xo, ro = s.orc.invert(b, 1e-10, 2000, "bicgstab", 0)
    solve_and_check(s, b, "cgne", matpc, 1e-10, xo)


@pytest.mark.parametrize("solver", ["cgne", "bicgstab"])
def test_fp32_status_is_honest_about_the_true_residual(solver):
    """PAPER.md:158, 221 (tol is the solver's tolerance): status OK means the TRUE residual, evaluated by the oracle,
    is below tol -- the recurrence residual of an fp32 solve drifts from it near 2e-7, so a column that misses is
    restarted with the recomputed residual (solver.cu, invert_native).  Below the fp32 floor the call must say
    NOT_CONVERGED, not OK."""
    s, c = from_cfg(2, 4, 18)
    b = synth.source(c["dims"], "z2", c["src_seed"])
    ok = 0
    for tol in (1e-6, 5e-7, 3e-7, 1e-7, 1e-8):
        for matpc in (0, 1, 2):
            x, res = s.ctx.invert(s.ctx.to_device(b), s.gauge, s.A, s.Ai, s.kappa, tol=tol, maxiter=500, solver=solver,
                                  matpc=matpc)
            true = s.orc.true_residual(b, x.cpu().numpy().astype(np.complex128))
            assert res.status in (0, 1), res.as_dict()
            if res.status == 0:
                assert true < tol, (tol, matpc, true, res.as_dict())
                ok += 1
            else:
                assert res.true_resid > tol or res.iter_resid > tol
            if tol >= 5e-7:
                assert res.status == 0, (tol, matpc, res.as_dict())
    assert ok >= 6


def test_freeze_flags_do_not_outlive_a_solve():
    """a mixed solve freezes the converged columns of its fp32 context; the flags must be cleared at exit
    (also on the stalled / not-converged paths), or the public BLAS-1 calls on that context silently do nothing."""
    s, c = from_cfg(1, 8, 18)
    lo = lq().Context(c["dims"], 4, 18, -1)
    g_lo = lo.gauge_pack(lo.to_device(s.U))
    A_lo, Ai_lo = lo.clover_build(g_lo, c["csw"], c["kappa"])
    b = synth.source(c["dims"], "gaussian", 3)
    for tol, want in ((1e-10, 0), (1e-18, 1)):  # 1e-18 is below the fp64 floor: the outer loop stalls -> NOT_CONVERGED
        x, res = s.ctx.invert_mixed(lo, s.ctx.to_device(b), s.gauge, s.A, s.Ai, g_lo, A_lo, Ai_lo, s.kappa, tol=tol,
                                    inner_tol=1e-4, maxiter=3000, solver="bicgstab")
        assert res.status == want, res.as_dict()
        assert s.orc.true_residual(b, x.cpu().numpy()) < 1e-10
        for ctx in (lo, s.ctx):
            u = torch.randn(ctx.spinor_bytes // ctx.prec, dtype=ctx.rdtype, device=ctx.dev)
            v = torch.randn_like(u)
            dot, nrm = ctx.blas_cdot(u, v)
            assert abs(nrm - float((u.double() ** 2).sum())) < 1e-5 * nrm
            w = v.clone()
            ctx.blas_xpay(u, 2.0, w)
            assert torch.allclose(w, u + 2.0 * v)


def test_degenerate_sources_and_lucky_breakdown():
    s, c = from_cfg(1, 8, 18)
    b = synth.source(c["dims"], "gaussian", 5)
    # a non-finite source is an error of that column, not a successful solve
    bad = b.copy()
    bad[0, 0, 0, 0, 0, 0, 0] = np.nan
    B = s.ctx.to_device(np.stack([b, bad]))
    x, res, rc = s.ctx.invert_multi(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, solver="cgne")
    assert res[0].status == 0 and res[1].status == -7 and rc == -7
    assert s.orc.true_residual(b, x[0].cpu().numpy()) < 1e-10
    # kappa = 0: M = 1, the first BiCGStab half step already solves the system (s = 0, t = 0, omega = 0/0 guarded)
    A1, Ai1 = s.ctx.clover_build(s.gauge, c["csw"], 0.0)
    for solver in ("bicgstab", "cgne"):
        x1, r1 = s.ctx.invert(s.ctx.to_device(b), s.gauge, A1, Ai1, 0.0, tol=1e-12, solver=solver)
        assert r1.status == 0 and r1.iterations <= 1, r1.as_dict()
        assert rel_err(x1.cpu().numpy(), b) < 1e-14


@pytest.mark.parametrize("solver,matpc", [("cgne", 0), ("cgne", 2), ("cgnr", 1), ("bicgstab", 1)])
def test_graph_replayed_iterations_equal_plain_launches(solver, matpc, monkeypatch):
    """Small lattices run blocks of 4 iterations as one CUDA graph and stop on the device (solver.cu): the result must
    be bit for bit that of the plain launch sequence (LQCD_GRAPHS=0), also when the instantiated graph is reused by a
    second solve with the same workspace and a different source, and for a batch of columns that stop at different
    iterations."""
    s, c = from_cfg(2, 8, 18)
    monkeypatch.setenv("LQCD_GRAPHS", "0")
    plain = lq().Context(c["dims"], 8, 18, -1)
    ws, _ = s.ctx.workspace(solver)
    wp, _ = plain.workspace(solver)
    for seed in (1, 2):
        b = s.ctx.to_device(synth.source(c["dims"], "gaussian", seed))
        x1, r1 = s.ctx.invert(b, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, solver=solver, matpc=matpc, workspace=ws)
        x2, r2 = plain.invert(b, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, solver=solver, matpc=matpc, workspace=wp)
        assert r1.status == 0 and r1.iterations == r2.iterations and r1.iterations > 6
        assert torch.equal(x1, x2) and r1.true_resid == r2.true_resid
    assert s.ctx.graph_launch_count() >= 2 and plain.graph_launch_count() == 0
    cols = np.stack([synth.source(c["dims"], "gaussian", 3), synth.source(c["dims"], "point"), 1e-3 * synth.source(c["dims"], "z2", 4)])
    B = s.ctx.to_device(cols)
    xa, ra, _ = s.ctx.invert_multi(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, solver=solver, matpc=matpc)
    xb, rb, _ = plain.invert_multi(B, s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, solver=solver, matpc=matpc)
    assert [r.iterations for r in ra] == [r.iterations for r in rb] and torch.equal(xa, xb)
