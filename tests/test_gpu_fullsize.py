"""GPU parity at BASELINE.json's full sizes (configs 4 and 5), in the launch configuration bench.py
times.  The oracle still finishes a full-lattice operator application in seconds at these sizes, so
dslash, clover, clover-inverse and M-hat are compared on EVERY site (relative L2, north_star
tolerances), plus element-wise on sampled sites through the oracle's one-site entry points
(`dslash_site`), and every solve is checked through the oracle-evaluated true residual
(at 48^3x96 the solve is verified through the true residual only)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2411_08461_b200 import synth
from latt import rel_err
from test_gpu_parity import TOL, lq

pytestmark = pytest.mark.gpu

_cache = {}


def host_inputs(n, prec):
    """(U, oracle with clover, source) of config n, rounded to fp32 first when prec == 4 (A16)."""
    key = (n, prec)
    if key not in _cache:
        _cache.clear()  # one full-size lattice resident at a time (host memory)
        c = synth.CONFIGS[n]
        U = synth.gauge(c["dims"], c["eps"], c["seed"])
        b = synth.source(c["dims"], c["source"], c["src_seed"])
        if prec == 4:
            U, b = synth.round_fp32(U), synth.round_fp32(b)
        orc = oracle.Oracle(c["dims"], U, -1).set_clover(c["kappa"], c["csw"])
        _cache[key] = (U, orc, b)
    return _cache[key]


class Dev:
    def __init__(self, n, prec, recon):
        c = synth.CONFIGS[n]
        self.c, self.prec = c, prec
        self.U, self.orc, self.b = host_inputs(n, prec)
        self.ctx = lq().Context(c["dims"], prec, recon, -1)
        self.gauge = self.ctx.gauge_pack(self.ctx.to_device(self.U))
        self.A, self.Ai = self.ctx.clover_build(self.gauge, c["csw"], c["kappa"])
        torch.cuda.synchronize()

    def up(self, psi):
        return self.ctx.spinor_pack(self.ctx.to_device(psi))

    def down(self, nat):
        return self.ctx.spinor_unpack(nat).cpu().numpy().astype(np.complex128)


def sampled_sites(shape, k, seed):
    rng = np.random.default_rng(seed)
    n = int(np.prod(shape))
    # always include the corners of the index range (origin, last site of each parity)
    return np.unique(np.concatenate([[0, n // 2 - 1, n // 2, n - 1], rng.integers(0, n, k)]))


def check_operators(d, check_A=True):
    ctx, orc, psi, tol = d.ctx, d.orc, d.b, TOL[d.prec]
    nat = d.up(psi)
    out = ctx.new_spinor(2)
    # a6: bare hopping term, both parities, every site; then sampled sites element by element
    for dagger in (False, True):
        for p in (0, 1):
            ctx.dslash(ctx.parity(out, p), ctx.parity(nat, 1 - p), d.gauge, p, 1.0, dagger)
        got = d.down(out)
        want = orc.dslash(psi, dagger=dagger)
        assert rel_err(got, want) < tol, dagger
        flat = got.reshape(-1, 4, 3)
        for s in sampled_sites(orc.site_shape, 60, 7 + dagger):
            ws = orc.dslash_site(psi, int(s), dagger)
            assert np.abs(flat[s] - ws).max() <= 4 * tol * max(np.abs(ws).max(), 1.0), (dagger, s)
    # a2/a3: clover and inverse, every site
    A_o, Ai_o = orc.clover()
    if check_A:
        assert rel_err(ctx.clover_unpack(d.A).cpu().numpy().astype(np.float64), A_o) < tol
    assert rel_err(ctx.clover_unpack(d.Ai).cpu().numpy().astype(np.float64), Ai_o) < tol
    del A_o, Ai_o
    # a7: clover-inverse apply
    for p in (0, 1):
        ctx.clover_apply(ctx.parity(out, p), ctx.parity(nat, p), d.Ai, p)
    assert rel_err(d.down(out), orc.clover_apply(psi, inverse=True)) < tol
    # a8: M-hat (two fused launches) and full M
    pe = psi.copy()
    pe[1] = 0
    out.zero_()
    ctx.mpc_apply(ctx.parity(out, 0), ctx.parity(nat, 0), d.gauge, d.A, d.Ai, d.c["kappa"], 0, False)
    assert rel_err(d.down(out), orc.mpc(pe, 0, False)) < tol
    ctx.mat_apply(out, nat, d.gauge, d.A, d.c["kappa"], False)
    assert rel_err(d.down(out), orc.mat(psi, False)) < tol


@pytest.mark.parametrize("recon", [18, 12])
def test_config4_operators_every_site_fp64(recon):
    check_operators(Dev(4, 8, recon))


@pytest.mark.parametrize("matpc", [0, 1, 2])
def test_config4_cgne_fp64_true_residual(matpc):
    """BASELINE config 4: mixed-precision-free fp64 CG (CGNE) to 1e-10, with the asymmetric and the symmetric
    Schur complements (left: fused epilogues 7 and 8; right: 9 and 10, the one bench.py times); the oracle's own operator
    evaluates the true residual of the GPU's solution, and the two solutions are the same x."""
    d = Dev(4, 8, 18)
    x, res = d.ctx.invert(d.ctx.to_device(d.b), d.gauge, d.A, d.Ai, d.c["kappa"], tol=1e-10, solver="cgne", matpc=matpc)
    assert res.status == 0 and res.iterations < 200
    xg = x.cpu().numpy()
    true = d.orc.true_residual(d.b, xg)
    assert true < 1e-10 and abs(true - res.true_resid) < 1e-11, (true, res.as_dict())
    if matpc >= 1:
        x0, res0 = d.ctx.invert(d.ctx.to_device(d.b), d.gauge, d.A, d.Ai, d.c["kappa"], tol=1e-10, solver="cgne", matpc=0)
        assert res.iterations < res0.iterations
        assert rel_err(xg, x0.cpu().numpy()) < 1e-9


def test_config4_mixed_precision_cgne():
    """fp64-accurate solve at 32^3x64 by fp64 defect correction around fp32 reconstruct-12 CGNE
    (SURVEY.md §8(f) rank 2); same bar as the pure fp64 solve."""
    d = Dev(4, 8, 18)
    lo = lq().Context(d.c["dims"], 4, 12, -1)
    g_lo = lo.gauge_pack(lo.to_device(d.U))
    A_lo, Ai_lo = lo.clover_build(g_lo, d.c["csw"], d.c["kappa"])
    x, res = d.ctx.invert_mixed(lo, d.ctx.to_device(d.b), d.gauge, d.A, d.Ai, g_lo, A_lo, Ai_lo, d.c["kappa"],
                                tol=1e-10, inner_tol=1e-4, solver="cgne")
    assert res.status == 0, res.as_dict()
    true = d.orc.true_residual(d.b, x.cpu().numpy())
    assert true < 1e-10 and abs(true - res.true_resid) < 1e-11, (true, res.as_dict())


@pytest.mark.parametrize("recon", [18, 12])
def test_config4_operators_every_site_fp32(recon):
    check_operators(Dev(4, 4, recon))


def test_config4_bicgstab_fp32_true_residual():
    d = Dev(4, 4, 18)
    x, res = d.ctx.invert(d.ctx.to_device(d.b), d.gauge, d.A, d.Ai, d.c["kappa"], tol=1e-6, solver="bicgstab")
    assert res.status == 0
    assert d.orc.true_residual(d.b, x.cpu().numpy().astype(np.complex128)) < 1e-6, res.as_dict()


def test_config5_capacity_fp32_recon12():
    """BASELINE config 5: 48^3x96 (10.6M sites), fp32 reconstruct-12: dslash, clover-inverse apply
    and a BiCGStab solve to 1e-6 (true residual by the oracle below the tolerance, reading A17)."""
    d = Dev(5, 4, 12)
    check_operators(d)
    x, res = d.ctx.invert(d.ctx.to_device(d.b), d.gauge, d.A, d.Ai, d.c["kappa"], tol=1e-6, solver="bicgstab")
    assert res.status == 0, res.as_dict()
    assert d.orc.true_residual(d.b, x.cpu().numpy().astype(np.complex128)) < 1e-6, res.as_dict()
    _cache.clear()
