"""Pins of oracle/contract.py (Listing 1 sources and contractions) against brute-force
loops over explicit lattice coordinates, closed forms and invariants.  CPU only."""
import numpy as np
import pytest

from oracle import contract as oc
from latt import coords
from test_oracle_pins import G, G5

DIMS = (4, 6, 4, 8)


def rand_prop(seed):
    rng = np.random.default_rng(seed)
    shp = (2, DIMS[3], DIMS[2], DIMS[1], DIMS[0] // 2, 4, 4, 3, 3)
    return rng.normal(size=shp) + 1j * rng.normal(size=shp)


def test_momentum_phase_and_wall_source_by_coordinates():
    mom = [1, -2, 3]
    ph = oc.momentum_phase(DIMS, mom)
    x, y, z, t = coords(DIMS)  # independent index helper of the test suite
    for idx in [(0, 0, 0, 0, 0), (1, 3, 2, 5, 1), (0, 7, 3, 4, 0), (1, 7, 3, 5, 1)]:
        X, Y, Z = x[idx], y[idx], z[idx]
        want = np.exp(2j * np.pi * (mom[0] * X / DIMS[0] + mom[1] * Y / DIMS[1] + mom[2] * Z / DIMS[2]))
        assert abs(ph[idx] - want) < 1e-14
    assert np.allclose(np.abs(ph), 1) and np.allclose(oc.momentum_phase(DIMS, [0, 0, 0]), 1)
    # lattice periodicity: shifting n_x by Lx changes nothing
    assert np.allclose(oc.momentum_phase(DIMS, [1 + DIMS[0], 0, 0]), oc.momentum_phase(DIMS, [1, 0, 0]))
    b = oc.wall_source(DIMS, 3, 2, 1, ph)
    assert np.count_nonzero(b) == DIMS[0] * DIMS[1] * DIMS[2]
    assert np.array_equal(b[:, 3, ..., 2, 1], ph[:, 3]) and not b[:, 2].any() and not b[..., 0, 0].any()
    assert oc.wall_source(DIMS, 0, 0, 0).sum() == DIMS[0] * DIMS[1] * DIMS[2]


def test_twopt_and_threept_brute_force():
    S0, Sp, ph = rand_prop(1), rand_prop(2), oc.momentum_phase(DIMS, [0, 1, 2])
    gam = G5 @ G[2]
    two, three = oc.twopt(ph, S0, Sp), oc.threept(S0, gam, Sp)
    for t in (0, 5):
        acc2 = acc3 = 0
        for w in range(2):
            for z in range(DIMS[2]):
                for y in range(DIMS[1]):
                    for xh in range(DIMS[0] // 2):
                        a, b = S0[w, t, z, y, xh], Sp[w, t, z, y, xh]
                        acc2 += np.conj(ph[w, t, z, y, xh]) * np.sum(np.conj(a) * b)
                        for i in range(4):
                            for c1 in range(3):
                                for c2 in range(3):
                                    acc3 += np.conj(a[:, i, c1, c2]) @ gam @ b[:, i, c1, c2]
        assert abs(two[t] - acc2) < 1e-10 * abs(acc2) and abs(three[t] - acc3) < 1e-10 * abs(acc3)
    # p = 0, S_p = S_0: the pion correlator is the squared norm per time-slice (real, positive)
    one = np.ones_like(ph)
    c = oc.twopt(one, S0, S0)
    assert np.allclose(c.imag, 0) and np.allclose(c.real, (np.abs(S0) ** 2).sum(axis=(0, 2, 3, 4, 5, 6, 7, 8)))
    # Gamma = 1 reduces Eq. 7 to Eq. 6 at zero momentum
    assert np.allclose(oc.threept(S0, np.eye(4), Sp), oc.twopt(one, S0, Sp))


def test_sequential_source_and_assemble():
    S0, ph = rand_prop(3), oc.momentum_phase(DIMS, [0, 0, 1])
    X = oc.sequential_source(ph, G5, S0, 4)
    assert not X[:, 3].any() and not X[:, 5].any()
    w, z, y, xh = 1, 2, 3, 1
    want = np.conj(ph[w, 4, z, y, xh]) * np.einsum("ij,jkab->ikab", G5, S0[w, 4, z, y, xh])
    assert np.allclose(X[w, 4, z, y, xh], want)
    # gamma5 is diagonal (1,1,-1,-1): rows 2,3 of the sink spin change sign
    assert np.allclose(X[:, 4, ..., 2:, :, :, :], -np.conj(ph[:, 4])[..., None, None, None, None] * S0[:, 4, ..., 2:, :, :, :])
    rng = np.random.default_rng(5)
    cols = rng.normal(size=(12, 2, 2, 2, 2, 2, 4, 3)) + 0j
    P = oc.assemble(cols)
    assert P.shape == (2, 2, 2, 2, 2, 4, 4, 3, 3)
    assert np.array_equal(P[1, 0, 1, 0, 1, 2, 3, 1, 2], cols[3 * 3 + 2][1, 0, 1, 0, 1, 2, 1])
