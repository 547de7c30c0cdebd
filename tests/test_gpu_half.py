"""GPU parity of the 16-bit-storage context (include/lqcd.h "16-bit storage", second half;
PAPER.md:423): pack / unpack bit-exact against the format's numpy restatement (halfmodel.py), the operators against the
oracle applied to the values the context actually holds, and the mixed-precision solve with a 16-bit inner context
against the same bar as the fp64 solve (reading A17)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2411_08461_b200 import synth
from halfmodel import quantise_spinor, round_spinor, round_links
from latt import rel_err
from test_gpu_parity import Setup, from_cfg, lq

pytestmark = pytest.mark.gpu


class HalfSetup:
    """fp32 context (pack, clover build) + 16-bit context of the same lattice; the oracle runs on the ROUNDED links."""

    def __init__(self, dims, eps, seed, kappa, csw, recon):
        self.dims, self.kappa, self.csw = dims, kappa, csw
        U = synth.round_fp32(synth.gauge(dims, eps, seed))
        self.U = U
        self.f32 = lq().Context(dims, 4, recon, -1)
        g32 = self.f32.gauge_pack(self.f32.to_device(U))
        self.A32, self.Ai32 = self.f32.clover_build(g32, csw, kappa)
        self.ctx = lq().Context(dims, 2, recon, -1)
        self.gauge = self.ctx.gauge_pack(self.ctx.to_device(U))
        self.A, self.Ai = self.ctx.clover_to_half(self.A32), self.ctx.clover_to_half(self.Ai32)
        self.orc = oracle.Oracle(dims, round_links(U, recon), -1)   # hopping term of the links the kernels see
        self.orc_full = oracle.Oracle(dims, U, -1).set_clover(kappa, csw)

    def up(self, psi):
        return self.ctx.spinor_pack(self.ctx.to_device(psi))

    def down(self, nat):
        return self.ctx.spinor_unpack(nat).cpu().numpy().astype(np.complex128)


def test_pack_unpack_is_the_format_bit_for_bit():
    s = HalfSetup((4, 6, 4, 8), 0.4, 3, 0.12, 1.0, 18)
    psi = synth.source(s.dims, "gaussian", 11)
    psi[0, 0, 0, 0, 0] = 0
    nat = s.up(psi)
    Vh = s.ctx.Vh
    raw = nat.cpu().numpy().view(np.uint16)
    q, n = quantise_spinor(psi)                       # [2, T, Z, Y, Xh, 24], [2, T, Z, Y, Xh]
    for par in range(2):
        blk = raw[par * 26 * Vh:(par + 1) * 26 * Vh]  # 52 B per site = 26 int16
        got_q = (blk[:24 * Vh].reshape(6, Vh, 4).transpose(1, 0, 2).reshape(Vh, 24).astype(np.int32) - 32768).astype(np.int16)  # offset binary
        got_n = np.ascontiguousarray(blk[24 * Vh:]).view(np.float32)
        assert np.array_equal(got_q, q[par].reshape(Vh, 24))
        assert np.array_equal(got_n, n[par].reshape(Vh))
    assert np.array_equal(s.down(nat), round_spinor(psi))


@pytest.mark.parametrize("recon", [18, 12])
def test_dslash_and_clover_apply_match_oracle_on_rounded_inputs(recon):
    s = HalfSetup((8, 8, 8, 16), 0.5, 2, 0.124, 1.2, recon)
    psi = synth.source(s.dims, "gaussian", 21)
    held = round_spinor(psi)
    nat = s.up(psi)
    for dagger in (False, True):
        want = s.orc.dslash(held, dagger=dagger)
        out = s.ctx.new_spinor(2)
        for par in (0, 1):
            s.ctx.dslash(s.ctx.parity(out, par), s.ctx.parity(nat, 1 - par), s.gauge, par, 1.0, dagger)
        # what is left: fp32 arithmetic and the rounding of the OUTPUT (1.5e-5 of a site's largest component)
        assert rel_err(s.down(out), want) < 3e-5, dagger
    # clover apply against the oracle's exact clover term: + the rounding of the stored clover blocks
    for inverse, cl in ((False, s.A), (True, s.Ai)):
        out = s.ctx.new_spinor(2)
        for par in (0, 1):
            s.ctx.clover_apply(s.ctx.parity(out, par), s.ctx.parity(nat, par), cl, par)
        assert rel_err(s.down(out), s.orc_full.clover_apply(held, inverse=inverse)) < 6e-5, inverse
    # Mhat through the fused epilogues, all three Schur forms, against the full-precision oracle
    pe = held.copy()
    pe[1] = 0
    for matpc in (0, 1):
        for dagger in (False, True):
            out = s.ctx.new_spinor(2)
            out.zero_()
            s.ctx.mpc_apply(s.ctx.parity(out, 0), s.ctx.parity(nat, 0), s.gauge, s.A, s.Ai, s.kappa, matpc, dagger)
            got = s.down(out)
            got[1] = 0
            assert rel_err(got, s.orc_full.mpc(pe, matpc, dagger)) < 1e-4, (matpc, dagger)


def test_blas_in_16_bit_storage():
    s = HalfSetup((4, 6, 4, 8), 0.4, 3, 0.12, 1.0, 18)
    xs, ys = synth.source(s.dims, "gaussian", 1), synth.source(s.dims, "gaussian", 2)
    x, y = s.ctx.parity(s.up(xs), 0), s.ctx.parity(s.up(ys), 0)
    xe, ye = round_spinor(xs)[0], round_spinor(ys)[0]
    dot, nrm = s.ctx.blas_cdot(x, y)
    assert abs(dot - np.vdot(xe, ye)) < 1e-6 * abs(np.vdot(xe, ye)) + 1e-9 and abs(nrm - np.vdot(xe, xe).real) < 1e-6 * nrm
    s.ctx.blas_xpay(x, 0.5, y)                       # y = x + 0.5 y, stored in 16 bits again
    full = s.ctx.new_spinor(2)
    full.zero_()
    s.ctx.parity(full, 0).copy_(y)
    assert rel_err(s.down(full)[0], xe + 0.5 * ye) < 3e-5
    n2 = s.ctx.blas_axpy_norm(-1.0, x, y)            # y -= x -> 0.5 ye (rounded)
    assert abs(n2 - np.vdot(0.5 * ye, 0.5 * ye).real) < 1e-3 * n2


@pytest.mark.parametrize("solver,matpc", [("cgne", 0), ("cgne", 2), ("bicgstab", 1), ("bicgstab", 0)])
@pytest.mark.parametrize("recon", [18, 12])
def test_config2_mixed_precision_with_16_bit_inner_context(solver, matpc, recon):
    """The bar of test_config2_mixed_precision_reaches_fp64_tolerance, with the 16-bit context inside: oracle solution
    within 10 tol, oracle-evaluated true residual < tol = 1e-10."""
    s, c = from_cfg(2, 8, 18)
    h = HalfSetup(c["dims"], c["eps"], c["seed"], c["kappa"], c["csw"], recon)
    b = synth.source(c["dims"], "z2", c["src_seed"])
    xo, ro = s.orc.invert(b, 1e-12, 2000, "bicgstab", 0)
    x, res = s.ctx.invert_mixed(h.ctx, s.ctx.to_device(b), s.gauge, s.A, s.Ai, h.gauge, h.A, h.Ai, s.kappa,
                                tol=1e-10, inner_tol=2e-3, maxiter=4000, solver=solver, matpc=matpc)
    assert res.status == 0, res.as_dict()
    xg = x.cpu().numpy()
    true = s.orc.true_residual(b, xg)
    assert true < 1e-10 and abs(true - res.true_resid) < 5e-11, (true, res.as_dict())
    assert rel_err(xg, xo) < 1e-9
    assert res.iterations < 400


def test_config4_mixed_precision_cgne_16_bit():
    """32^3x64 (BASELINE config 4): fp64 defect correction around 16-bit CGNE; true residual by the oracle."""
    s, c = from_cfg(4, 8, 18)
    h = HalfSetup(c["dims"], c["eps"], c["seed"], c["kappa"], c["csw"], 12)
    b = synth.source(c["dims"], c["source"], c["src_seed"])
    x, res = s.ctx.invert_mixed(h.ctx, s.ctx.to_device(b), s.gauge, s.A, s.Ai, h.gauge, h.A, h.Ai, s.kappa,
                                tol=1e-10, inner_tol=2e-3, maxiter=4000, solver="cgne", matpc=2)
    assert res.status == 0, res.as_dict()
    assert s.orc.true_residual(b, x.cpu().numpy()) < 1e-10


def test_unsupported_calls_say_so():
    s = HalfSetup((4, 4, 4, 8), 0.3, 1, 0.12, 1.0, 18)
    with pytest.raises(lq().LqcdError):
        s.ctx.clover_build(s.gauge, 1.0, 0.12)
    with pytest.raises(lq().LqcdError):
        s.ctx.dslash_mrhs(s.ctx.new_spinor(2), s.ctx.new_spinor(2), s.gauge, 0, 2)
    # a pure 16-bit solve works to the accuracy the storage allows
    b = synth.source(s.dims, "gaussian", 5)
    x, res = s.ctx.invert(s.ctx.to_device(b), s.gauge, s.A, s.Ai, s.kappa, tol=1e-3, maxiter=200, solver="cgne")
    assert res.status == 0 and s.orc_full.true_residual(b, x.cpu().numpy().astype(np.complex128)) < 2e-3
