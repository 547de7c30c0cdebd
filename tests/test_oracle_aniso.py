"""Pins for the oracle's anisotropic operator (Eq. 5):
    M = 1 - kappa [ D_t + (nu/xi_0) sum_i D_i ] - kappa [ c_SW^t sum_i sigma_i4 F_i4 + (c_SW^r/xi_0) sum_{i<j} sigma_ij F_ij ]
checked against closed forms typed out here (free field with direction-dependent weights, constant
abelian field plane by plane), the isotropic limit, gamma5-hermiticity and the solved system.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_2411_08461_b200 import synth
from latt import coords, rel_err
from test_oracle_pins import G, G5, SIG, rand_spinor, vdot


@pytest.mark.parametrize("dims,n", [((4, 4, 4, 8), (1, 0, 3, 2)), ((4, 6, 2, 4), (3, 5, 1, 0))])
def test_p15_free_field_plane_wave_with_weights(dims, n):
    kappa, ws = 0.115, 0.37
    orc = oracle.Oracle(dims, synth.unit_gauge(dims), -1).set_anisotropy(ws).set_clover_aniso(kappa, 0.9, 1.7)
    x, y, z, t = coords(dims)
    p = [2 * np.pi * n[0] / dims[0], 2 * np.pi * n[1] / dims[1], 2 * np.pi * n[2] / dims[2],
         2 * np.pi * (n[3] + 0.5) / dims[3]]
    w = [ws, ws, ws, 1.0]
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    rng = np.random.default_rng(11)
    u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
    psi = phase[..., None, None] * u
    Mp = (1 - 2 * kappa * sum(w[mu] * np.cos(p[mu]) for mu in range(4))) * np.eye(4) \
        + 2j * kappa * sum(w[mu] * np.sin(p[mu]) * G[mu] for mu in range(4))
    assert rel_err(orc.mat(psi), phase[..., None, None] * (Mp @ u)) < 1e-14
    assert rel_err(orc.mat(psi, dagger=True), phase[..., None, None] * (Mp.conj().T @ u)) < 1e-14
    Dp = sum(w[mu] * (2 * np.cos(p[mu]) * np.eye(4) - 2j * np.sin(p[mu]) * G[mu]) for mu in range(4))
    assert rel_err(orc.dslash(psi), phase[..., None, None] * (Dp @ u)) < 1e-14
    # one-site entry point carries the same weights
    flat = orc.dslash(psi).reshape(-1, 4, 3)
    for s in (0, 5, flat.shape[0] - 1):
        assert np.abs(orc.dslash_site(psi, s) - flat[s]).max() < 1e-13


@pytest.mark.parametrize("mu,nu", [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)])
def test_p16_constant_abelian_field_picks_the_plane_coefficient(mu, nu):
    """F_mu_nu = sin(B) T on one plane only: A = 1 - kappa * c(plane) * sin(B) sigma_mu_nu (x) T with
    c = csw_t on the temporal planes (nu = t) and csw_s on the spatial ones."""
    dims = (4, 6, 4, 8)
    B = 2 * np.pi / (dims[mu] * dims[nu])
    T = np.array([1.0, -1.0, 0.0])
    xs = coords(dims)
    U = synth.unit_gauge(dims)
    U[mu] = np.zeros_like(U[mu])
    for c in range(3):
        U[mu][..., c, c] = np.exp(-1j * B * xs[nu] * T[c])
        U[nu][..., c, c] = np.where(xs[nu] == dims[nu] - 1, np.exp(1j * B * dims[nu] * xs[mu] * T[c]), 1.0)
    kappa, cs, ct = 0.13, 0.8, 2.1
    o = oracle.Oracle(dims, U, -1).set_anisotropy(0.5).set_clover_aniso(kappa, cs, ct)
    coef = ct if nu == 3 else cs
    want = np.eye(12) - kappa * coef * np.sin(B) * np.kron(SIG(mu, nu), np.diag(T))
    psi = rand_spinor(dims, 3)
    got = o.clover_apply(psi)
    ref = np.einsum("ij,...j->...i", want, psi.reshape(psi.shape[:-2] + (12,))).reshape(psi.shape)
    assert rel_err(got, ref) < 1e-14
    inv = o.clover_apply(got, inverse=True)
    assert rel_err(inv, psi) < 1e-13


def test_p17_isotropic_limit_hermiticity_and_solve():
    dims = (4, 4, 4, 8)
    U = synth.gauge(dims, 0.4, 21)
    kappa = 0.118
    iso = oracle.Oracle(dims, U, -1).set_clover(kappa, 1.3)
    same = oracle.Oracle(dims, U, -1).set_anisotropy(1.0).set_clover_aniso(kappa, 1.3, 1.3)
    psi, chi = rand_spinor(dims, 1), rand_spinor(dims, 2)
    assert np.array_equal(iso.mat(psi), same.mat(psi))
    A1, _ = iso.clover()
    A2, _ = same.clover()
    assert np.array_equal(A1, A2)
    # anisotropic: gamma5-hermiticity and adjoint, Schur-preconditioned solves give M x = b
    an = oracle.Oracle(dims, U, -1).set_anisotropy(0.45).set_clover_aniso(kappa, 0.7, 1.9)
    g5 = np.array([1, 1, -1, -1.0])[:, None]
    lhs = vdot(psi, g5 * an.mat(chi))
    rhs = vdot(g5 * an.mat(psi), chi)
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    assert abs(vdot(psi, an.mat(chi, dagger=True)) - vdot(an.mat(psi), chi)) < 1e-12 * abs(lhs)
    assert rel_err(an.mat(psi), iso.mat(psi)) > 1e-2  # the weights really changed the operator
    b = synth.source(dims, "gaussian", 4)
    for solver, matpc in (("cgne", 0), ("bicgstab", 1), ("cgnr", 0)):
        x, res = an.invert(b, 1e-12, 2000, solver, matpc)
        assert res.status == 0 and rel_err(an.mat(x), b) < 1e-11
        assert an.true_residual(b, x) < 1e-11
    # temporal planes only / spatial planes only differ from each other (c_t and c_s both act)
    a_t = oracle.Oracle(dims, U, -1).set_clover_aniso(kappa, 0.0, 1.5).clover_apply(psi)
    a_s = oracle.Oracle(dims, U, -1).set_clover_aniso(kappa, 1.5, 0.0).clover_apply(psi)
    full = oracle.Oracle(dims, U, -1).set_clover_aniso(kappa, 1.5, 1.5).clover_apply(psi)
    assert rel_err(a_t + a_s - psi, full) < 1e-14 and rel_err(a_t, a_s) > 1e-2
