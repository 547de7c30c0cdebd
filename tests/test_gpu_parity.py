"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Tolerances (north_star): relative L2 error 1e-13 in fp64, 2e-6 in fp32
for dslash / clover; solutions within 10*tol of the oracle's and true residual < tol as evaluated
by the oracle's operator (reading A17).  fp32 protocol (A16): inputs are rounded to
fp32 and the oracle runs in fp64 on the rounded values."""
import numpy as np
import pytest
import torch

import oracle
from paper_2411_08461_b200 import synth
from latt import rel_err

pytestmark = pytest.mark.gpu

TOL = {8: 1e-13, 4: 2e-6}


def lq():
    from paper_2411_08461_b200 import lqcd
    return lqcd


class Setup:
    def __init__(self, dims, eps, seed, kappa, csw, prec, recon, tb=-1, with_clover=True):
        self.dims, self.kappa, self.csw, self.prec = dims, kappa, csw, prec
        U = synth.gauge(dims, eps, seed)
        if prec == 4:
            U = synth.round_fp32(U)
        self.U = U
        self.orc = oracle.Oracle(dims, U, tb)
        self.ctx = lq().Context(dims, prec, recon, tb)
        self.gauge = self.ctx.gauge_pack(self.ctx.to_device(U))
        if with_clover:
            self.orc.set_clover(kappa, csw)
            self.A, self.Ai = self.ctx.clover_build(self.gauge, csw, kappa)

    def spinor(self, kind, seed):
        b = synth.source(self.dims, kind, seed)
        return synth.round_fp32(b) if self.prec == 4 else b

    def up(self, psi):  # public numpy -> native two-parity device spinor
        return self.ctx.spinor_pack(self.ctx.to_device(psi))

    def down(self, native):
        return self.ctx.spinor_unpack(native).cpu().numpy().astype(np.complex128)


def from_cfg(n, prec, recon, **kw):
    c = synth.CONFIGS[n]
    return Setup(c["dims"], c["eps"], c["seed"], c["kappa"], c["csw"], prec, recon, **kw), c


# --------------------------------------------------------------------------------------------
def test_pack_unpack_roundtrip():
    for prec in (8, 4):
        s = Setup((4, 6, 4, 8), 0.4, 3, 0.12, 1.0, prec, 18, with_clover=False)
        psi = s.spinor("gaussian", 5)
        back = s.down(s.up(psi))
        assert np.array_equal(back, psi)


@pytest.mark.parametrize("prec,recon", [(8, 18), (8, 12), (4, 18), (4, 12)])
@pytest.mark.parametrize("dims,tb", [((4, 4, 4, 8), -1), ((4, 6, 8, 10), -1), ((8, 8, 8, 16), 1), ((12, 4, 6, 4), -1),
                                     # shared-memory tiled kernel (csrc/dslash_tiled.cuh): several tiles in every
                                     # direction, and tiles that span a whole extent (halo wraps onto the tile itself)
                                     ((16, 8, 4, 8), -1), ((8, 4, 8, 4), -1), ((24, 12, 8, 6), 1)])
def test_dslash_matches_oracle(prec, recon, dims, tb):
    s = Setup(dims, 0.5, 2, 0.124, 1.2, prec, recon, tb, with_clover=False)
    psi = s.spinor("gaussian", 102)
    nat = s.up(psi)
    out = s.ctx.new_spinor(2)
    for dagger in (False, True):
        want = s.orc.dslash(psi, dagger=dagger)
        for p in (0, 1):
            s.ctx.dslash(s.ctx.parity(out, p), s.ctx.parity(nat, 1 - p), s.gauge, p, 1.0, dagger)
        got = s.down(out)
        for p in (0, 1):
            assert rel_err(got[p], want[p]) < TOL[prec], (dagger, p)
    # scale argument
    s.ctx.dslash(s.ctx.parity(out, 0), s.ctx.parity(nat, 1), s.gauge, 0, -0.37, False)
    assert rel_err(s.down(out)[0], -0.37 * s.orc.dslash(psi)[0]) < TOL[prec]


def test_config1_twenty_chained_dslash():
    """BASELINE config 1 / reading A13: 20 chained applications alternating parity; each output is
    compared with the oracle applied to the GPU's own input of that step, then renormalised."""
    s, c = from_cfg(1, 8, 18, with_clover=False)
    psi = s.spinor("gaussian", 7)
    psi[1] = 0
    for step in range(20):
        p_out = (step + 1) & 1
        nat = s.up(psi)
        out = s.ctx.new_spinor(2)
        out.zero_()
        s.ctx.dslash(s.ctx.parity(out, p_out), s.ctx.parity(nat, 1 - p_out), s.gauge, p_out, 1.0, step % 3 == 0)
        got = s.down(out)
        want = s.orc.dslash(psi, dagger=(step % 3 == 0), only_parity=p_out)
        assert rel_err(got, want) < 1e-13, step
        psi = got / np.linalg.norm(got.ravel())


@pytest.mark.parametrize("prec,recon", [(8, 18), (4, 18), (4, 12)])
def test_clover_build_and_apply(prec, recon):
    s, c = from_cfg(2, prec, recon)
    A_o, Ai_o = s.orc.clover()
    A_g = s.ctx.clover_unpack(s.A).cpu().numpy().astype(np.float64)
    Ai_g = s.ctx.clover_unpack(s.Ai).cpu().numpy().astype(np.float64)
    assert rel_err(A_g, A_o) < TOL[prec]
    assert rel_err(Ai_g, Ai_o) < TOL[prec]
    psi = s.spinor("gaussian", 11)
    nat = s.up(psi)
    out = s.ctx.new_spinor(2)
    for inverse, field in ((False, s.A), (True, s.Ai)):
        for p in (0, 1):
            s.ctx.clover_apply(s.ctx.parity(out, p), s.ctx.parity(nat, p), field, p)
        assert rel_err(s.down(out), s.orc.clover_apply(psi, inverse=inverse)) < TOL[prec]


@pytest.mark.parametrize("onepass", ["0", "1"])
def test_clover_inverse_of_indefinite_blocks_and_both_build_forms(onepass, monkeypatch):
    """kappa*csw = 1.2 on a rough field makes most 6x6 blocks indefinite: the Hermitian sweep must hand every such block
    to the pivoted elimination.  Run for the three-pass build and for the one-kernel build (LQCD_CLOVER_ONEPASS=1);
    both against the oracle, whose inverse is a general pivoted one."""
    monkeypatch.setenv("LQCD_CLOVER_ONEPASS", onepass)
    for dims, kappa, csw in (((4, 6, 8, 10), 0.12, 10.0), ((8, 8, 8, 16), 0.124, 1.2)):
        s = Setup(dims, 0.7, 9, kappa, csw, 8, 18)
        A_o, Ai_o = s.orc.clover()
        A_g = s.ctx.clover_unpack(s.A).cpu().numpy()
        Ai_g = s.ctx.clover_unpack(s.Ai).cpu().numpy()
        if csw > 5:
            assert (A_o[..., :6] < 0).any()  # negative diagonal entries: certainly not positive definite
        assert rel_err(A_g, A_o) < 1e-13
        # an indefinite block may be badly conditioned; bound the error blockwise by its condition
        scale = np.abs(Ai_o).max(axis=-1, keepdims=True)
        assert (np.abs(Ai_g - Ai_o) / scale).max() < 1e-10
        assert rel_err(Ai_g, Ai_o) < 1e-11
        s.ctx.close()


def test_clover_build_csw_zero_and_singular():
    s = Setup((4, 4, 4, 8), 0.3, 1, 0.12, 0.0, 8, 18)
    A = s.ctx.clover_unpack(s.A).cpu().numpy()
    ref = np.zeros(36)
    ref[:6] = 1
    assert np.array_equal(A, np.broadcast_to(ref, A.shape))
    # kappa*csw*sigma.F = 1 on a constant abelian field makes a block exactly singular
    dims = (4, 4, 4, 4)
    B = 2 * np.pi / 16
    U = synth.unit_gauge(dims)
    from latt import coords
    xs = coords(dims)
    T = np.array([1.0, -1.0, 0.0])
    U[0] = 0
    for cc in range(3):
        U[0][..., cc, cc] = np.exp(-1j * B * xs[1] * T[cc])
        U[1][..., cc, cc] = np.where(xs[1] == 3, np.exp(1j * B * 4 * xs[0] * T[cc]), 1.0)
    ctx = lq().Context(dims, 8, 18, -1)
    g = ctx.gauge_pack(ctx.to_device(U))
    with pytest.raises(lq().LqcdError, match="singular"):
        ctx.clover_build(g, 1.0 / np.sin(B), 1.0)


@pytest.mark.parametrize("prec,recon", [(8, 18), (4, 12)])
def test_mat_and_mpc_apply(prec, recon):
    s, c = from_cfg(2, prec, recon)
    psi = s.spinor("z2", 102)
    nat = s.up(psi)
    out = s.ctx.new_spinor(2)
    for dagger in (False, True):
        s.ctx.mat_apply(out, nat, s.gauge, s.A, s.kappa, dagger)
        assert rel_err(s.down(out), s.orc.mat(psi, dagger)) < TOL[prec]
    pe = psi.copy()
    pe[1] = 0
    for matpc in (0, 1):
        for dagger in (False, True):
            out.zero_()
            s.ctx.mpc_apply(s.ctx.parity(out, 0), s.ctx.parity(nat, 0), s.gauge, s.A, s.Ai, s.kappa, matpc, dagger)
            assert rel_err(s.down(out), s.orc.mpc(pe, matpc, dagger)) < TOL[prec], (matpc, dagger)


@pytest.mark.parametrize("prec,recon", [(8, 18), (4, 12)])
def test_mpc_apply_right_preconditioned(prec, recon):
    """matpc 2 (include/lqcd.h): Mhat_r = 1 - k^2 D_eo A_oo^-1 D_oe A_ee^-1 = (asymmetric Mhat) A_ee^-1 by definition;
    expected values compose the oracle's clover-inverse apply and its asymmetric Schur complement."""
    s, c = from_cfg(2, prec, recon)
    psi = s.spinor("gaussian", 31)
    psi[1] = 0
    nat = s.up(psi)
    out = s.ctx.new_spinor(2)
    want = s.orc.mpc(s.orc.clover_apply(psi, inverse=True, only_parity=0), 0, False)
    want_dag = s.orc.clover_apply(s.orc.mpc(psi, 0, True), inverse=True, only_parity=0)
    for dagger, w in ((False, want), (True, want_dag)):
        out.zero_()
        s.ctx.mpc_apply(s.ctx.parity(out, 0), s.ctx.parity(nat, 0), s.gauge, s.A, s.Ai, s.kappa, 2, dagger)
        assert rel_err(s.down(out)[0], w[0]) < TOL[prec], dagger


def test_blas_kernels():
    for prec in (8, 4):
        s = Setup((4, 6, 4, 8), 0.4, 3, 0.12, 1.0, prec, 18, with_clover=False)
        ctx = s.ctx
        xs, ys, zs = (s.spinor("gaussian", k) for k in (1, 2, 3))
        x, y, z = (ctx.parity(s.up(v), 0) for v in (xs, ys, zs))
        xe, ye, ze = xs[0], ys[0], zs[0]
        tol = 1e-14 if prec == 8 else 1e-6
        d, n2 = ctx.blas_cdot(x, y)
        assert abs(d - np.vdot(xe, ye)) < tol * abs(np.vdot(xe, xe)) and abs(n2 - np.vdot(xe, xe).real) < tol * n2
        n = ctx.blas_axpy_norm(0.37, x, y)
        ye = ye + 0.37 * xe
        assert abs(n - np.vdot(ye, ye).real) < tol * n
        ctx.blas_xpay(x, -1.25, y)
        ye = xe - 1.25 * ye
        ctx.blas_caxpbypz(0.3 - 0.7j, x, -1.1 + 0.2j, y, z)
        ze = ze + (0.3 - 0.7j) * xe + (-1.1 + 0.2j) * ye
        full = ctx.new_spinor(2)
        full.zero_()
        ctx.parity(full, 0).copy_(z)
        assert rel_err(s.down(full)[0], ze) < 10 * tol
        # deterministic: the same reduction twice gives the same bits
        assert ctx.blas_cdot(x, y) == ctx.blas_cdot(x, y)


@pytest.mark.parametrize("prec,recon", [(8, 18), (8, 12), (4, 18), (4, 12)])
@pytest.mark.parametrize("dims,tb", [((16, 8, 4, 8), -1), ((8, 8, 8, 16), -1), ((8, 4, 8, 4), 1)])
def test_tiled_dslash_matches_oracle(prec, recon, dims, tb, monkeypatch):
    """The opt-in shared-memory tiled kernel (csrc/dslash_tiled.cuh, LQCD_DSLASH_TILED=1 at context creation):
    several tiles per direction, tiles spanning a whole extent (the halo wraps onto the tile itself), the seam in t,
    every epilogue without a reduction through M and M-hat (both forms, adjoints: 0-3 and 6), and a CGNE solve in which
    the tiled kernel does the A^-1 D hops and the default kernel the epilogues that reduce."""
    monkeypatch.setenv("LQCD_DSLASH_TILED", "1")
    s = Setup(dims, 0.5, 2, 0.124, 1.2, prec, recon, tb)
    psi = s.spinor("gaussian", 102)
    nat = s.up(psi)
    out = s.ctx.new_spinor(2)
    for dagger in (False, True):
        want = s.orc.dslash(psi, dagger=dagger)
        for p in (0, 1):
            s.ctx.dslash(s.ctx.parity(out, p), s.ctx.parity(nat, 1 - p), s.gauge, p, 1.0, dagger)
        got = s.down(out)
        for p in (0, 1):
            assert rel_err(got[p], want[p]) < TOL[prec], (dagger, p)
        s.ctx.mat_apply(out, nat, s.gauge, s.A, s.kappa, dagger)
        assert rel_err(s.down(out), s.orc.mat(psi, dagger)) < TOL[prec]
    pe = psi.copy()
    pe[1] = 0
    for matpc in (0, 1):
        for dagger in (False, True):
            out.zero_()
            s.ctx.mpc_apply(s.ctx.parity(out, 0), s.ctx.parity(nat, 0), s.gauge, s.A, s.Ai, s.kappa, matpc, dagger)
            assert rel_err(s.down(out), s.orc.mpc(pe, matpc, dagger)) < TOL[prec], (matpc, dagger)
    tol = 1e-10 if prec == 8 else 1e-6
    x, res = s.ctx.invert(s.ctx.to_device(psi), s.gauge, s.A, s.Ai, s.kappa, tol=tol, maxiter=2000, solver="cgne", matpc=0)
    assert res.status == 0
    assert s.orc.true_residual(psi, x.cpu().numpy().astype(np.complex128)) < tol, res.as_dict()
