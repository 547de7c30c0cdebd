"""GPU parity of the Listing-1 steps against oracle/contract.py:
momentum phase, wall/point sources, propagator assembly/split, Eq. 6 two-point, Eq. 7 three-point, Eq. 8
sequential source - first on random propagators (every entry exercised), then the listing end to end:
wall-source propagators S_0, S_p by the batched solver, sequential source, S_p0, both correlators."""
import numpy as np
import pytest
import torch

import oracle
from oracle import contract as oc
from paper_2411_08461_b200 import synth
from latt import rel_err
from test_gpu_parity import Setup, TOL, from_cfg, lq
from test_oracle_pins import G, G5

pytestmark = pytest.mark.gpu


def dev(ctx, a):
    return ctx.to_device(a)


def host(t):
    return t.cpu().numpy().astype(np.complex128)


@pytest.mark.parametrize("prec", [8, 4])
@pytest.mark.parametrize("dims", [(4, 6, 4, 8), (8, 4, 6, 4)])
def test_sources_phase_assemble_contract_on_random_fields(prec, dims):
    ctx = lq().Context(dims, prec, 18, -1)
    tol = 1e-13 if prec == 8 else 2e-6
    mom = [1, -2, 3]
    ph_o = oc.momentum_phase(dims, mom)
    ph = ctx.momentum_phase(mom)
    # numpy evaluates exp(i theta) at |theta| <= 2 pi sum|n_i| ~ 38 without reducing the argument, so the
    # ORACLE carries |theta| * eps ~ 4e-15; the kernel reduces n.x/L mod 1 in integers before sincospi
    assert np.abs(host(ph) - ph_o).max() < (1e-14 if prec == 8 else 1e-7)
    assert np.array_equal(host(ctx.source_wall(3, 2, 1)), oc.wall_source(dims, 3, 2, 1))
    assert np.abs(host(ctx.source_wall(0, 3, 0, ph)) - oc.wall_source(dims, 0, 3, 0, host(ph))).max() == 0
    assert np.array_equal(host(ctx.source_point((0, 0, 0, 0), 0, 0)), synth.source(dims, "point"))
    pt = host(ctx.source_point((3, 1, 2, 3), 1, 2))
    assert np.count_nonzero(pt) == 1 and pt[(3 + 1 + 2 + 3) & 1, 3, 2, 1, 1, 1, 2] == 1
    rng = np.random.default_rng(3)
    shp = (2, dims[3], dims[2], dims[1], dims[0] // 2)
    cols = rng.normal(size=(12,) + shp + (4, 3)) + 1j * rng.normal(size=(12,) + shp + (4, 3))
    if prec == 4:
        cols = synth.round_fp32(cols)
    P = ctx.propagator_assemble(dev(ctx, cols))
    assert np.array_equal(host(P), oc.assemble(cols))
    assert np.array_equal(host(ctx.propagator_split(P)), cols)
    S0 = rng.normal(size=shp + (4, 4, 3, 3)) + 1j * rng.normal(size=shp + (4, 4, 3, 3))
    Sp = rng.normal(size=shp + (4, 4, 3, 3)) + 1j * rng.normal(size=shp + (4, 4, 3, 3))
    if prec == 4:
        S0, Sp = synth.round_fp32(S0), synth.round_fp32(Sp)
    pho = host(ph)
    d0, dp = dev(ctx, S0), dev(ctx, Sp)
    assert rel_err(ctx.contract_twopt(ph, d0, dp), oc.twopt(pho, S0, Sp)) < tol
    assert rel_err(ctx.contract_twopt(None, d0, d0), oc.twopt(np.ones_like(pho), S0, S0)) < tol
    gam = G5 @ G[2]  # gamma_5 gamma_3 of Eq. 7 (paper's gamma(15) @ gamma(4), reading A8)
    assert rel_err(ctx.contract_threept(d0, gam, dp), oc.threept(S0, gam, Sp)) < tol
    assert ctx.contract_twopt(ph, d0, dp).tolist() == ctx.contract_twopt(ph, d0, dp).tolist()  # deterministic
    X = ctx.sequential_source(ph, G5, d0, 2)
    assert rel_err(host(X), oc.sequential_source(pho, G5, S0, 2)) < (1e-14 if prec == 8 else 2e-7)


def test_listing1_end_to_end_config1():
    """PAPER.md:151-211 on the 4^3x8 lattice of BASELINE configs[0] (isotropic clover, synthetic links):
    S_0 and S_p from wall sources at t0 = 0 (momentum mode [0,0,1]), two-point function Eq. 6, sequential
    source Eq. 8 at t = 4 through gamma_5, S_p0 = M^-1 X, three-point function Eq. 7.  Every propagator
    column is checked through the oracle's true residual, the correlators against the oracle's einsum on
    the GPU's propagators AND against an all-oracle run of the listing."""
    s, c = from_cfg(1, 8, 18)
    ctx, dims, kappa = s.ctx, c["dims"], c["kappa"]
    t0, tsnk, mom = 0, 4, [0, 0, 1]
    ph = ctx.momentum_phase(mom)
    pho = oc.momentum_phase(dims, mom)

    def gpu_prop(sources):
        prop, res, rc = ctx.propagator(sources, s.gauge, s.A, s.Ai, kappa, tol=1e-11, solver="bicgstab")
        assert rc == 0
        return prop

    def orc_prop(sources):
        return oc.assemble([s.orc.invert(b, 1e-12, 2000, "bicgstab", 0)[0] for b in sources])

    src0 = torch.stack([ctx.source_wall(t0, i, a) for i in range(4) for a in range(3)])
    srcp = torch.stack([ctx.source_wall(t0, i, a, ph) for i in range(4) for a in range(3)])
    S0, Sp = gpu_prop(src0), gpu_prop(srcp)
    cols0 = host(ctx.propagator_split(S0))
    for k in (0, 7, 11):
        assert s.orc.true_residual(host(src0[k]), cols0[k]) < 1e-10
    X = ctx.sequential_source(ph, G5, S0, tsnk)
    Sp0 = gpu_prop(ctx.propagator_split(X))
    two = ctx.contract_twopt(ph, S0, Sp)
    three = ctx.contract_threept(Sp0, G5 @ G[2], Sp)
    # the GPU contractions against the oracle's einsum on the same (GPU-made) propagators
    assert rel_err(two, oc.twopt(pho, host(S0), host(Sp))) < 1e-13
    assert rel_err(three, oc.threept(host(Sp0), G5 @ G[2], host(Sp))) < 1e-13
    # the whole listing by the oracle alone
    o_src0 = [oc.wall_source(dims, t0, i, a) for i in range(4) for a in range(3)]
    o_srcp = [oc.wall_source(dims, t0, i, a, pho) for i in range(4) for a in range(3)]
    oS0, oSp = orc_prop(o_src0), orc_prop(o_srcp)
    oX = oc.sequential_source(pho, G5, oS0, tsnk)
    oSp0 = orc_prop([oX[..., :, i, :, a] for i in range(4) for a in range(3)])
    assert rel_err(host(S0), oS0) < 1e-9 and rel_err(host(Sp0), oSp0) < 1e-9
    assert rel_err(two, oc.twopt(pho, oS0, oSp)) < 1e-9
    assert rel_err(three, oc.threept(oSp0, G5 @ G[2], oSp)) < 1e-9
