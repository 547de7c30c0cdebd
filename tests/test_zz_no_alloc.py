"""lqcd_clover_build_noalloc (include/lqcd.h): the clover build whose scratch is a fixed device array inside the library
instead of a cudaMalloc made by the call.  Checked against the existing path (lqcd_clover_build) within the tolerances
of tests/test_gpu_parity.py, on calls in a row that share the static array (different lattices and links, so a call
that relied on what the previous one left there would show), plus the size limit.  Collected last on purpose (the
suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

from paper_2411_08461_b200 import synth
from latt import rel_err

pytestmark = pytest.mark.gpu

TOL = {8: 1e-13, 4: 2e-6}  # as tests/test_gpu_parity.py


def lq():
    from paper_2411_08461_b200 import lqcd
    return lqcd


def build_both(dims, eps, seed, kappa, csw, prec, recon, check_no_alloc=False):
    U = synth.gauge(dims, eps, seed)
    if prec == 4:
        U = synth.round_fp32(U)
    ctx = lq().Context(dims, prec, recon, -1)
    g = ctx.gauge_pack(ctx.to_device(U))
    A0, Ai0 = ctx.clover_build(g, csw, kappa)  # existing path (allocates its scratch on the context's first build)
    A1, Ai1 = ctx.empty(ctx.clover_bytes), ctx.empty(ctx.clover_bytes)
    A1.fill_(0)
    Ai1.fill_(0)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ctx.clover_build_noalloc(g, csw, kappa, out=A1, out_inv=Ai1)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    if check_no_alloc:  # kernels and the array are resident after the first call: device memory must not move
        assert free1 >= free0, (free0, free1)
    pub = [ctx.clover_unpack(t).cpu().numpy().astype(np.float64) for t in (A0, Ai0, A1, Ai1)]
    ctx.close()
    return pub


def test_noalloc_clover_build_matches_existing_path_on_calls_in_a_row():
    cases = [
        # dims, eps, seed, kappa, csw, prec, recon
        ((8, 8, 8, 16), 0.5, 2, 0.124, 1.2, 8, 18),    # BASELINE config 2
        ((4, 6, 8, 10), 0.7, 9, 0.120, 1.0, 8, 12),    # smaller, ragged, other links: the array holds the last call's data
        ((8, 8, 8, 16), 0.5, 2, 0.124, 1.2, 8, 18),    # the first one again
        ((16, 8, 8, 16), 0.6, 5, 0.124, 1.5, 4, 12),   # fp32 storage, 16384 sites
        ((16, 16, 8, 16), 0.6, 6, 0.124, 1.5, 4, 18),  # exactly the limit: 32768 sites
    ]
    first = None
    for i, (dims, eps, seed, kappa, csw, prec, recon) in enumerate(cases):
        A0, Ai0, A1, Ai1 = build_both(dims, eps, seed, kappa, csw, prec, recon, check_no_alloc=i > 0)
        assert np.abs(A0).max() > 0.5 and np.abs(Ai1).max() > 0.5
        assert rel_err(A1, A0) < TOL[prec], (i, rel_err(A1, A0))
        assert rel_err(Ai1, Ai0) < TOL[prec], (i, rel_err(Ai1, Ai0))
        if i == 0:
            first = (A1, Ai1)
        if i == 2:  # same inputs, same kernels: the same bits, whatever ran in between
            assert np.array_equal(A1, first[0]) and np.array_equal(Ai1, first[1])


def test_noalloc_clover_build_rejects_lattices_beyond_the_static_scratch():
    L = lq()
    dims = (16, 16, 16, 16)  # 65536 sites
    ctx = L.Context(dims, 4, 12, -1)
    assert ctx.clover_noalloc_max_sites() == 32768
    g = ctx.empty(ctx.gauge_bytes)
    with pytest.raises(L.LqcdError, match="65536 sites.*at most 32768"):
        ctx.clover_build_noalloc(g, 1.0, 0.12)
    ctx.close()
