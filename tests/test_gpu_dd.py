"""GPU parity of the domain-decomposed hopping term (csrc/dd.cu, paper_2411_08461_b200/dd.py; SURVEY.md §8(f) rank 4b;
PAPER.md:82): sub-lattices held on ONE device exchange their faces through device memory and must reproduce the
oracle's full-lattice D (which knows nothing of the decomposition), for cuts in every direction, both parities, dagger,
antiperiodic t, anisotropic weight, fp64 and fp32, 18 and 12 reals per link."""
import numpy as np
import pytest
import torch

import oracle
from paper_2411_08461_b200 import dd, synth
from latt import rel_err
from test_gpu_parity import TOL, lq

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("grid", [(1, 1, 1, 2), (1, 1, 2, 2), (2, 2, 1, 1), (2, 1, 1, 4), (2, 2, 2, 2), (1, 1, 1, 1)])
@pytest.mark.parametrize("prec,recon", [(8, 18), (4, 12)])
def test_decomposed_dslash_matches_full_lattice_oracle(grid, prec, recon):
    dims, ws = (8, 8, 8, 16), 0.8
    part = dd.Partition(dims, grid, t_boundary=-1)
    U = synth.gauge(dims, 0.5, 2)
    psi = synth.source(dims, "gaussian", 77)
    if prec == 4:
        U, psi = synth.round_fp32(U), synth.round_fp32(psi)
    orc = oracle.Oracle(dims, U, -1).set_anisotropy(ws)
    Us, psis = dd.split_gauge(part, U), dd.split_field(part, psi)
    ctxs, gauges, ins = [], [], []
    for r in range(part.size):
        c = lq().Context(part.local, prec, recon, part.local_t_boundary()).set_anisotropy(ws).set_partition(part.partitioned)
        ctxs.append(c)
        gauges.append(c.gauge_pack(c.to_device(Us[r])))
        ins.append(c.spinor_pack(c.to_device(psis[r])))
    for dagger in (False, True):
        want = orc.dslash(psi, dagger=dagger)
        outs = [c.new_spinor(2) for c in ctxs]
        for par in (0, 1):
            dd.dslash_dd_emulated(part, ctxs, [c.parity(o, par) for c, o in zip(ctxs, outs)],
                                  [c.parity(i, 1 - par) for c, i in zip(ctxs, ins)], gauges, par, 0.7, dagger, ws)
        got = dd.join_field(part, [c.spinor_unpack(o).cpu().numpy().astype(np.complex128) for c, o in zip(ctxs, outs)])
        assert rel_err(got, 0.7 * want) < TOL[prec], (grid, dagger)


def test_interior_alone_misses_exactly_the_cut_hops():
    """With t cut in two, the interior kernel of the lower half equals D with the links across the two cuts set to
    zero (the oracle takes any 3x3 matrices as links)."""
    dims = (4, 4, 4, 16)
    part = dd.Partition(dims, (1, 1, 1, 2), t_boundary=-1)
    U = synth.gauge(dims, 0.4, 9)
    psi = synth.source(dims, "gaussian", 5)
    Ucut = U.copy()
    Ucut[3, :, 7] = 0     # t-links leaving t = 7 (into the upper half) and t = 15 (the seam)
    Ucut[3, :, 15] = 0
    want = dd.split_field(part, oracle.Oracle(dims, Ucut, -1).dslash(psi))[0]
    c = lq().Context(part.local, 8, 18, 1).set_partition(part.partitioned)
    g = c.gauge_pack(c.to_device(dd.split_gauge(part, U)[0]))
    nat = c.spinor_pack(c.to_device(dd.split_field(part, psi)[0]))
    out = c.new_spinor(2)
    for par in (0, 1):
        c.dslash_dd_interior(c.parity(out, par), c.parity(nat, 1 - par), g, par)
    assert rel_err(c.spinor_unpack(out).cpu().numpy(), want) < 1e-13


@pytest.mark.parametrize("grid", [(1, 1, 2, 2), (2, 1, 1, 2)])
def test_decomposed_mhat_and_cgne_solve_match_oracle(grid):
    """M-hat and the even-odd CGNE solve over sub-lattices (dd.Decomposed: D by interior + faces, sums over ranks, the
    C ABI's BLAS-1 with host coefficients) against the oracle on the whole lattice: M-hat to 1e-13, solution within
    10 tol, oracle-evaluated true residual < tol (reading A17).  The clover fields are cut from a whole-lattice build."""
    c2 = synth.CONFIGS[2]
    dims, kappa, csw = c2["dims"], c2["kappa"], c2["csw"]
    part = dd.Partition(dims, grid, t_boundary=-1)
    U = synth.gauge(dims, c2["eps"], c2["seed"])
    b = synth.source(dims, "z2", c2["src_seed"])
    orc = oracle.Oracle(dims, U, -1).set_clover(kappa, csw)
    whole = lq().Context(dims, 8, 18, -1)
    gw = whole.gauge_pack(whole.to_device(U))
    Aw, Aiw = whole.clover_build(gw, csw, kappa)
    A_pub, Ai_pub = (dd.split_field(part, whole.clover_unpack(f).cpu().numpy()) for f in (Aw, Aiw))
    Us, bs = dd.split_gauge(part, U), dd.split_field(part, b)
    ctxs = [lq().Context(part.local, 8, 18, part.local_t_boundary()).set_partition(part.partitioned) for _ in range(part.size)]
    gauges = [c.gauge_pack(c.to_device(u)) for c, u in zip(ctxs, Us)]
    A = [c.clover_pack(c.to_device(a)) for c, a in zip(ctxs, A_pub)]
    Ai = [c.clover_pack(c.to_device(a)) for c, a in zip(ctxs, Ai_pub)]
    D = dd.Decomposed(part, range(part.size), ctxs, gauges, A, Ai)
    nat = [c.spinor_pack(c.to_device(p)) for c, p in zip(ctxs, bs)]
    # M-hat and its adjoint
    be = b.copy()
    be[1] = 0
    for dagger in (False, True):
        outs = [c.new_spinor(2) for c in ctxs]
        for o in outs:
            o.zero_()
        D.mpc([c.parity(o, 0) for c, o in zip(ctxs, outs)], [c.parity(n, 0) for c, n in zip(ctxs, nat)], kappa, dagger, D.new(), D.new())
        got = dd.join_field(part, [c.spinor_unpack(o).cpu().numpy() for c, o in zip(ctxs, outs)])
        assert rel_err(got, orc.mpc(be, 0, dagger)) < 1e-13, dagger
    xs, it, resid = D.invert(nat, kappa, tol=1e-10)
    x = dd.join_field(part, [c.spinor_unpack(v).cpu().numpy() for c, v in zip(ctxs, xs)])
    xo, ro = orc.invert(b, 1e-10, 2000, "cgne", 0)
    assert abs(it - ro.iterations) <= 1 and resid < 1e-10
    assert orc.true_residual(b, x) < 1e-10 and rel_err(x, xo) < 1e-9
