"""GPU parity of the anisotropic operator (Eq. 5) against
the oracle: hopping term with spatial weight nu/xi_0, clover term with separate c_SW^r/xi_0 and
c_SW^t, M, M-hat and the solves, at the paper's Listing-1 parameters (xi_0, nu = 2.464, 0.95;
m_0 = 0.3; c_SW^t, c_SW^r = 0.91, 1.07, reading A18) on synthetic links."""
import numpy as np
import pytest
import torch

import oracle
from paper_2411_08461_b200 import synth
from latt import rel_err
from test_gpu_parity import Setup, TOL, lq

pytestmark = pytest.mark.gpu

XI0, NU, M0, CSW_T, CSW_R = 2.464, 0.95, 0.3, 0.91, 1.07
WS = NU / XI0
KAPPA = 1.0 / (2 * (M0 + 1 + 3 * WS))


class Aniso(Setup):
    def __init__(self, dims, prec, recon, tb=-1):
        super().__init__(dims, 0.4, 11, KAPPA, 0.0, prec, recon, tb, with_clover=False)
        self.orc.set_anisotropy(WS).set_clover_aniso(KAPPA, CSW_R / XI0, CSW_T)
        self.ctx.set_anisotropy(WS)
        self.A, self.Ai = self.ctx.clover_build_aniso(self.gauge, CSW_R / XI0, CSW_T, KAPPA)


@pytest.mark.parametrize("prec,recon", [(8, 18), (8, 12), (4, 18), (4, 12)])
@pytest.mark.parametrize("dims", [(4, 4, 4, 8), (4, 6, 8, 10), (8, 8, 8, 16)])
def test_aniso_operators_match_oracle(prec, recon, dims):
    s = Aniso(dims, prec, recon)
    tol = TOL[prec]
    psi = s.spinor("gaussian", 31)
    nat = s.up(psi)
    out = s.ctx.new_spinor(2)
    for dagger in (False, True):
        for p in (0, 1):
            s.ctx.dslash(s.ctx.parity(out, p), s.ctx.parity(nat, 1 - p), s.gauge, p, 1.0, dagger)
        assert rel_err(s.down(out), s.orc.dslash(psi, dagger=dagger)) < tol
    A_o, Ai_o = s.orc.clover()
    assert rel_err(s.ctx.clover_unpack(s.A).cpu().numpy().astype(np.float64), A_o) < tol
    assert rel_err(s.ctx.clover_unpack(s.Ai).cpu().numpy().astype(np.float64), Ai_o) < tol
    for dagger in (False, True):
        s.ctx.mat_apply(out, nat, s.gauge, s.A, s.kappa, dagger)
        assert rel_err(s.down(out), s.orc.mat(psi, dagger)) < tol
    pe = psi.copy()
    pe[1] = 0
    for matpc in (0, 1):
        out.zero_()
        s.ctx.mpc_apply(s.ctx.parity(out, 0), s.ctx.parity(nat, 0), s.gauge, s.A, s.Ai, s.kappa, matpc, False)
        assert rel_err(s.down(out), s.orc.mpc(pe, matpc, False)) < tol
    # multi-RHS kernel carries the same weight
    n = s.ctx.spinor_bytes // s.ctx.prec
    inp = torch.cat([s.ctx.parity(nat, 1)] * 3)
    o3 = s.ctx.new_spinor(3)
    s.ctx.dslash_mrhs(o3, inp, s.gauge, 0, 3)
    full = s.ctx.new_spinor(2)
    full.zero_()
    s.ctx.parity(full, 0).copy_(o3[2 * n:3 * n])
    assert rel_err(s.down(full)[0], s.orc.dslash(psi)[0]) < tol


@pytest.mark.parametrize("solver", ["cgne", "bicgstab"])
def test_aniso_solve_fp64(solver):
    s = Aniso((8, 8, 8, 16), 8, 18)
    b = synth.source(s.dims, "point", spin=2, colour=1)
    xo, ro = s.orc.invert(b, 1e-12, 4000, "bicgstab", 0)
    x, res = s.ctx.invert(s.ctx.to_device(b), s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, maxiter=4000, solver=solver)
    assert res.status == 0, res.as_dict()
    xg = x.cpu().numpy()
    assert s.orc.true_residual(b, xg) < 1e-10
    assert rel_err(xg, xo) < 1e-9
    # the isotropic operator gives a different answer: the weights are really in the solve
    s.ctx.set_anisotropy(1.0)
    x1, r1 = s.ctx.invert(s.ctx.to_device(b), s.gauge, s.A, s.Ai, s.kappa, tol=1e-10, maxiter=4000, solver=solver)
    assert rel_err(x1.cpu().numpy(), xo) > 1e-2
    with pytest.raises(lq().LqcdError):
        s.ctx.set_anisotropy(0.0)
