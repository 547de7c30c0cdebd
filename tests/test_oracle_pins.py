"""Pins for the CPU oracle: the oracle is checked against what the
paper's conventions and the mathematics fix -- closed forms, invariants, brute force -- none of
which re-use the oracle's own formulas.  CPU only."""
import numpy as np
import pytest

import oracle
from paper_2411_08461_b200 import synth
from latt import (coords, cb_to_lex, lex_to_cb, gauge_cb_to_lex, gauge_lex_to_cb, shift, dagger,
                  rel_err)

# DeGrand-Rossi gamma matrices typed out as literals (Chroma's convention), NOT taken
# from the oracle, so that a slip in the oracle's block construction shows up.
i = 1j
G = [
    np.array([[0, 0, 0, i], [0, 0, i, 0], [0, -i, 0, 0], [-i, 0, 0, 0]]),
    np.array([[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]], dtype=complex),
    np.array([[0, 0, i, 0], [0, 0, 0, -i], [-i, 0, 0, 0], [0, i, 0, 0]]),
    np.array([[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]], dtype=complex),
]
G5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(complex)


def SIG(mu, nu):
    return 0.5j * (G[mu] @ G[nu] - G[nu] @ G[mu])


def rand_spinor(dims, seed):
    return synth.source(dims, "gaussian", seed)


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


# ------------------------------------------------------------------------------------------ P1
def test_p1_gamma_algebra():
    for mu in range(4):
        g = oracle.gamma(mu)
        assert np.array_equal(g, G[mu])
        assert np.allclose(g, g.conj().T)
        for nu in range(4):
            anti = g @ oracle.gamma(nu) + oracle.gamma(nu) @ g
            assert np.allclose(anti, 2.0 * (mu == nu) * np.eye(4), atol=0)
    g5 = oracle.gamma(4)
    assert np.array_equal(g5, G5)  # gamma(15) = g1 g2 g3 g4 = diag(1,1,-1,-1)
    for mu in range(4):
        for nu in range(4):
            s = oracle.sigma(mu, nu)
            assert np.allclose(s, SIG(mu, nu), atol=0)
            assert np.all(s[:2, 2:] == 0) and np.all(s[2:, :2] == 0)  # chiral basis: block diagonal


# ------------------------------------------------------------------------------------------ P2
@pytest.mark.parametrize("dims,n", [((4, 4, 4, 8), (1, 0, 3, 2)), ((4, 6, 2, 4), (3, 5, 1, 0)),
                                    ((2, 2, 2, 2), (1, 1, 0, 1))])
@pytest.mark.parametrize("tb", [-1, 1])
def test_p2_free_field_plane_wave(dims, n, tb):
    kappa = 0.119
    orc = oracle.Oracle(dims, synth.unit_gauge(dims), tb).set_clover(kappa, 1.3)
    x, y, z, t = coords(dims)
    p = [2 * np.pi * n[0] / dims[0], 2 * np.pi * n[1] / dims[1], 2 * np.pi * n[2] / dims[2],
         2 * np.pi * (n[3] + (0.5 if tb < 0 else 0.0)) / dims[3]]
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    rng = np.random.default_rng(7)
    u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
    psi = phase[..., None, None] * u
    Mp = (1 - 2 * kappa * sum(np.cos(pm) for pm in p)) * np.eye(4) \
        + 2j * kappa * sum(np.sin(p[mu]) * G[mu] for mu in range(4))
    Mdp = Mp.conj().T
    assert rel_err(orc.mat(psi), phase[..., None, None] * (Mp @ u)) < 1e-14
    assert rel_err(orc.mat(psi, dagger=True), phase[..., None, None] * (Mdp @ u)) < 1e-14
    # bare hopping term: D(p) = sum_mu [2 cos p - 2 i gamma sin p]
    Dp = sum(2 * np.cos(p[mu]) * np.eye(4) - 2j * np.sin(p[mu]) * G[mu] for mu in range(4))
    assert rel_err(orc.dslash(psi), phase[..., None, None] * (Dp @ u)) < 1e-14


# ------------------------------------------------------------------------------------------ P3
def test_p3_free_propagator_closed_form():
    dims = (4, 4, 4, 8)
    kappa = 0.12
    V = np.prod(dims)
    orc = oracle.Oracle(dims, synth.unit_gauge(dims), -1).set_clover(kappa, 1.0)
    x, y, z, t = coords(dims)
    s0, c0 = 2, 1
    b = synth.source(dims, "point", spin=s0, colour=c0)
    expect = np.zeros(b.shape, dtype=complex)
    for nx in range(dims[0]):
        for ny in range(dims[1]):
            for nz in range(dims[2]):
                for nt in range(dims[3]):
                    p = [2 * np.pi * nx / dims[0], 2 * np.pi * ny / dims[1], 2 * np.pi * nz / dims[2],
                         2 * np.pi * (nt + 0.5) / dims[3]]
                    a = 1 - 2 * kappa * sum(np.cos(q) for q in p)
                    bm = [2 * kappa * np.sin(q) for q in p]
                    Minv = (a * np.eye(4) - 1j * sum(bm[mu] * G[mu] for mu in range(4))) / \
                        (a * a + sum(q * q for q in bm))
                    ph = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t)) / V
                    expect[..., :, c0] += ph[..., None] * Minv[:, s0]
    for solver in ("cgne", "cgnr", "bicgstab"):
        sol, res = orc.invert(b, tol=1e-13, maxiter=500, solver=solver)
        assert res.status == 0
        assert rel_err(sol, expect) < 1e-11, solver


# ------------------------------------------------------------------------------------------ P4
@pytest.mark.parametrize("tb", [-1, 1])
def test_p4_gamma5_hermiticity_and_dagger(tb):
    dims = (4, 4, 4, 8)
    orc = oracle.Oracle(dims, synth.gauge(dims, 0.5, 11), tb).set_clover(0.124, 1.2)
    xv, yv = rand_spinor(dims, 1), rand_spinor(dims, 2)
    g5 = np.array([1, 1, -1, -1.0])[:, None]
    lhs = vdot(xv, g5 * orc.mat(yv))
    rhs = vdot(g5 * orc.mat(xv), yv)
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)
    assert abs(vdot(xv, orc.mat(yv, dagger=True)) - vdot(orc.mat(xv), yv)) < 1e-11 * abs(lhs)
    assert abs(vdot(xv, orc.dslash(yv, dagger=True)) - vdot(orc.dslash(xv), yv)) < 1e-11 * abs(lhs)
    # asymmetric Mhat is gamma5-hermitian; both forms obey <x, Mhat^dag y> = <Mhat x, y>
    xe, ye = xv.copy(), yv.copy()
    xe[1] = 0
    ye[1] = 0
    for matpc in (0, 1):
        a = vdot(xe, orc.mpc(ye, matpc, dagger=True))
        c = vdot(orc.mpc(xe, matpc), ye)
        assert abs(a - c) < 1e-11 * abs(a)
    assert rel_err(g5 * orc.mpc(g5 * ye, 0), orc.mpc(ye, 0, dagger=True)) < 1e-13


# ------------------------------------------------------------------------------------------ P5
def transform_gauge(U, g, dims):
    Ul, gl = gauge_cb_to_lex(U, dims), cb_to_lex(g, dims)
    out = np.stack([gl @ Ul[mu] @ dagger(shift(gl, mu, +1)) for mu in range(4)])
    return gauge_lex_to_cb(out, dims)


def rotate(g, psi):  # (g psi)_a = sum_b g_ab psi_b on the colour index
    return np.einsum("...ab,...sb->...sa", g, psi)


def test_p5_gauge_covariance():
    dims = (4, 4, 4, 8)
    kappa, csw = 0.124, 1.2
    U = synth.gauge(dims, 0.5, 21)
    g = synth.colour_rotation(dims, 22)
    U2 = transform_gauge(U, g, dims)
    o1 = oracle.Oracle(dims, U, -1).set_clover(kappa, csw)
    o2 = oracle.Oracle(dims, U2, -1).set_clover(kappa, csw)
    psi = rand_spinor(dims, 3)
    assert rel_err(o2.mat(rotate(g, psi)), rotate(g, o1.mat(psi))) < 1e-14
    assert rel_err(o2.dslash(rotate(g, psi), dagger=True), rotate(g, o1.dslash(psi, dagger=True))) < 1e-14
    assert rel_err(o2.clover_apply(rotate(g, psi)), rotate(g, o1.clover_apply(psi))) < 1e-14
    x1, r1 = o1.invert(psi, 1e-12, 500, "bicgstab")
    x2, r2 = o2.invert(rotate(g, psi), 1e-12, 500, "bicgstab")
    assert r1.status == 0 and r2.status == 0
    assert rel_err(x2, rotate(g, x1)) < 1e-10


# ------------------------------------------------------------------------------------------ P6
def test_p6_pure_gauge_is_free():
    dims = (4, 4, 4, 8)
    kappa = 0.12
    g = synth.colour_rotation(dims, 31)
    U = transform_gauge(synth.unit_gauge(dims), g, dims)
    o = oracle.Oracle(dims, U, -1).set_clover(kappa, 1.7)
    for mu in range(4):
        for nu in range(mu + 1, 4):
            assert np.abs(o.fmunu(mu, nu)).max() < 1e-14
    A, Ai = o.clover()
    ref = np.zeros(36)
    ref[:6] = 1
    assert np.abs(A - ref).max() < 1e-14 and np.abs(Ai - ref).max() < 1e-14
    # propagator = g(x) S_free(x,0) g^dag(0)
    free = oracle.Oracle(dims, synth.unit_gauge(dims), -1).set_clover(kappa, 1.7)
    b = synth.source(dims, "point", spin=1, colour=2)
    xs, _ = o.invert(b, 1e-12, 500, "bicgstab")
    g0d = g[0, 0, 0, 0, 0].conj().T
    acc = np.zeros_like(xs)
    for c in range(3):
        xf, _ = free.invert(synth.source(dims, "point", spin=1, colour=c), 1e-12, 500, "bicgstab")
        acc += rotate(g, xf) * g0d[c, 2]
    assert rel_err(xs, acc) < 1e-10


# ------------------------------------------------------------------------------------------ P7
@pytest.mark.parametrize("mu,nu", [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)])
def test_p7_constant_abelian_field(mu, nu):
    dims = (4, 6, 4, 8)
    k = 1
    B = 2 * np.pi * k / (dims[mu] * dims[nu])
    T = np.array([1.0, -1.0, 0.0])
    xs = coords(dims)
    U = synth.unit_gauge(dims)
    U[mu] = np.zeros_like(U[mu])
    for c in range(3):
        U[mu][..., c, c] = np.exp(-1j * B * xs[nu] * T[c])
        U[nu][..., c, c] = np.where(xs[nu] == dims[nu] - 1, np.exp(1j * B * dims[nu] * xs[mu] * T[c]), 1.0)
    kappa, csw = 0.13, 1.4
    o = oracle.Oracle(dims, U, -1).set_clover(kappa, csw)
    for a in range(4):
        for b in range(a + 1, 4):
            F = o.fmunu(a, b)
            want = np.diag(np.sin(B) * T) if (a, b) == (mu, nu) else np.zeros((3, 3))
            assert np.abs(F - want).max() < 1e-15
    assert np.abs(o.fmunu(nu, mu) + np.diag(np.sin(B) * T)).max() < 1e-15  # antisymmetry
    dense = o.clover_dense(kappa, csw)
    want = np.eye(12) - kappa * csw * np.sin(B) * np.kron(SIG(mu, nu), np.diag(T))
    assert np.abs(dense - want).max() < 1e-15


# ------------------------------------------------------------------------------------------ P8
def unpack_blocks(Apk):
    """packed [...,2,36] -> dense Hermitian [...,2,6,6]; order per PAPER.md:56 + reading A7."""
    out = np.zeros(Apk.shape[:-1] + (6, 6), dtype=complex)
    for d in range(6):
        out[..., d, d] = Apk[..., d]
    for r in range(1, 6):
        for c in range(r):
            kk = r * (r - 1) // 2 + c
            v = Apk[..., 6 + 2 * kk] + 1j * Apk[..., 6 + 2 * kk + 1]
            out[..., r, c] = v
            out[..., c, r] = np.conj(v)
    return out


def test_p8_clover_structure_and_inverse():
    dims = (4, 4, 4, 8)
    kappa, csw = 0.124, 1.2
    o = oracle.Oracle(dims, synth.gauge(dims, 0.5, 41), -1).set_clover(kappa, csw)
    assert o.clover_defect() < 1e-15
    dense = o.clover_dense(kappa, csw)
    assert np.abs(dense - dagger(dense)).max() < 1e-15
    assert np.abs(dense[..., :6, 6:]).max() == 0 and np.abs(dense[..., 6:, :6]).max() == 0
    A, Ai = o.clover()
    blocks = unpack_blocks(A)
    assert np.abs(blocks[..., 0, :, :] - dense[..., :6, :6]).max() < 1e-15
    assert np.abs(blocks[..., 1, :, :] - dense[..., 6:, 6:]).max() < 1e-15
    prod = unpack_blocks(A) @ unpack_blocks(Ai)
    assert np.abs(prod - np.eye(6)).max() < 1e-14
    psi = rand_spinor(dims, 4)
    assert rel_err(o.clover_apply(o.clover_apply(psi), inverse=True), psi) < 1e-14
    # clover apply == dense 12x12 times the (spin,colour) vector
    want = np.einsum("...ij,...j->...i", dense, psi.reshape(psi.shape[:-2] + (12,))).reshape(psi.shape)
    assert rel_err(o.clover_apply(psi), want) < 1e-15
    # F is Hermitian, antisymmetric in (mu,nu), and the clover term does not see t_boundary
    F = o.fmunu(1, 3)
    assert np.abs(F - dagger(F)).max() < 1e-15
    o2 = oracle.Oracle(dims, synth.gauge(dims, 0.5, 41), +1).set_clover(kappa, csw)
    assert np.array_equal(o2.clover()[0], A)


# ------------------------------------------------------------------------------------------ P9
def smooth_field(dims, amp, seed):
    rng = np.random.default_rng(seed)
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    X = [x.astype(float), y.astype(float), z.astype(float), t.astype(float)]
    modes = []
    for mu in range(4):
        ms = []
        for _ in range(3):
            Gm = rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3))
            H = (Gm + Gm.conj().T) / 2
            H -= np.trace(H) / 3 * np.eye(3)
            ms.append((H, rng.integers(-1, 2, size=4), rng.uniform(0, 2 * np.pi)))
        modes.append(ms)
    U = []
    for mu in range(4):
        A = np.zeros(x.shape + (3, 3), dtype=complex)
        for H, n, ph in modes[mu]:
            arg = sum(2 * np.pi * n[d] * (X[d] + (0.5 if d == mu else 0.0)) / dims[d] for d in range(4)) + ph
            A += amp * np.cos(arg)[..., None, None] * H
        w, v = np.linalg.eigh(A)
        U.append(np.einsum("...ij,...j,...kj->...ik", v, np.exp(1j * w), v.conj()))
    psi = np.zeros(x.shape + (4, 3), dtype=complex)
    for _ in range(3):
        n = rng.integers(-1, 2, size=4)
        u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
        arg = sum(2 * np.pi * n[d] * X[d] / dims[d] for d in range(4))
        psi += np.exp(1j * arg)[..., None, None] * u
    return np.stack(U), psi


def test_p9_csw_sign_and_scale():
    """sum_{mu<nu} sigma F psi -> sum_{mu<nu} gamma_mu gamma_nu [nabla_mu, nabla_nu] psi on smooth fields."""
    ratios = []
    for L in (8, 16):
        dims = (L, L, L, L)
        Ul, psil = smooth_field(dims, 2.0 / L, 5)  # fixed physical field: a*A ~ 1/L
        kappa, csw = 0.125, 1.0
        o = oracle.Oracle(dims, gauge_lex_to_cb(Ul, dims), +1).set_clover(kappa, csw)
        psi = lex_to_cb(psil, dims)
        sigF = cb_to_lex((psi - o.clover_apply(psi)) / (kappa * csw), dims)

        def nabla(mu, f):
            fwd = np.einsum("...ab,...sb->...sa", Ul[mu], shift(f, mu, +1))
            bwd = shift(np.einsum("...ba,...sb->...sa", Ul[mu].conj(), f), mu, -1)
            return 0.5 * (fwd - bwd)

        comm = np.zeros_like(psil)
        for mu in range(4):
            for nu in range(mu + 1, 4):
                c = nabla(mu, nabla(nu, psil)) - nabla(nu, nabla(mu, psil))
                comm += np.einsum("st,...tc->...sc", G[mu] @ G[nu], c)
        ratios.append((rel_err(comm, sigF), rel_err(-comm, sigF)))
    (r8, w8), (r16, w16) = ratios
    assert r8 < 0.7 and r16 < 0.2 and r16 < r8 / 3.0, ratios   # O(a^2) convergence, right sign
    assert w8 > 1.4 and w16 > 1.8, ratios                      # wrong sign is ~2


# ----------------------------------------------------------------------------------------- P10
@pytest.mark.parametrize("matpc", [0, 1])
def test_p10_schur_identities(matpc):
    dims = (4, 4, 4, 8)
    kappa = 0.124
    o = oracle.Oracle(dims, synth.gauge(dims, 0.5, 51), -1).set_clover(kappa, 1.2)
    b, xe = rand_spinor(dims, 5), rand_spinor(dims, 6)
    xe[1] = 0
    be, bo = b.copy(), b.copy()
    be[1] = 0
    bo[0] = 0
    # x_o = A_oo^-1 (b_o + kappa D_oe x_e)
    xo = o.clover_apply(bo + kappa * o.dslash(xe, only_parity=1), inverse=True, only_parity=1)
    Mx = o.mat(xe + xo)
    assert rel_err(Mx[1], b[1]) < 1e-14                                      # (M x)_o = b_o
    corr = kappa * o.dslash(o.clover_apply(bo, inverse=True, only_parity=1), only_parity=0)
    Mx_e = Mx.copy()
    Mx_e[1] = 0
    if matpc == 0:   # (M x)_e = Mhat x_e - kappa D_eo A_oo^-1 b_o
        assert rel_err(Mx_e, o.mpc(xe, 0) - corr) < 1e-14
    else:            # A_ee^-1 (M x)_e = Mhat_s x_e - kappa A_ee^-1 D_eo A_oo^-1 b_o
        lhs = o.clover_apply(Mx_e, inverse=True, only_parity=0)
        assert rel_err(lhs, o.mpc(xe, 1) - o.clover_apply(corr, inverse=True, only_parity=0)) < 1e-14
    # only_parity really restricts the output, and D only connects opposite parities
    full = o.dslash(xe)
    assert np.abs(full[0]).max() == 0 and np.array_equal(o.dslash(xe, only_parity=1)[1], full[1])


# ----------------------------------------------------------------------------------------- P11
def test_p11_dense_brute_force_2x2x2x2():
    dims = (2, 2, 2, 2)
    kappa, csw = 0.11, 1.1
    o = oracle.Oracle(dims, synth.gauge(dims, 0.4, 61), -1).set_clover(kappa, csw)
    n = 16 * 12
    shape = (2, 2, 2, 2, 1, 4, 3)
    M = np.zeros((n, n), dtype=complex)
    Md = np.zeros((n, n), dtype=complex)
    for j in range(n):
        e = np.zeros(n, dtype=complex)
        e[j] = 1
        M[:, j] = o.mat(e.reshape(shape)).ravel()
        Md[:, j] = o.mat(e.reshape(shape), dagger=True).ravel()
    assert np.abs(Md - M.conj().T).max() < 1e-15
    g5 = np.tile(np.repeat([1, 1, -1, -1.0], 3), 16)
    assert np.abs(g5[:, None] * M * g5[None, :] - M.conj().T).max() < 1e-15
    b = rand_spinor(dims, 7)
    want = np.linalg.solve(M, b.ravel()).reshape(shape)
    for solver in ("cgne", "cgnr", "bicgstab"):
        for matpc in (0, 1):
            x, res = o.invert(b, 1e-13, 400, solver, matpc)
            assert res.status == 0, (solver, matpc)
            assert rel_err(x, want) < 1e-11, (solver, matpc)
            assert res.true_resid < 1e-12
    # dense Schur complement of the even-even block equals Mhat
    ne = n // 2
    Mee, Meo, Moe, Moo = M[:ne, :ne], M[:ne, ne:], M[ne:, :ne], M[ne:, ne:]
    S = Mee - Meo @ np.linalg.solve(Moo, Moe)
    xe = rand_spinor(dims, 8)
    xe[1] = 0
    assert rel_err(o.mpc(xe, 0).ravel()[:ne], S @ xe.ravel()[:ne]) < 1e-14
    Ss = np.linalg.solve(Mee + Meo @ np.zeros_like(Moe), S)   # A_ee^-1 S  (M_ee is exactly A_ee)
    assert rel_err(o.mpc(xe, 1).ravel()[:ne], Ss @ xe.ravel()[:ne]) < 1e-13
    assert rel_err(o.mpc(xe, 1, dagger=True).ravel()[:ne], Ss.conj().T @ xe.ravel()[:ne]) < 1e-13


# ----------------------------------------------------------------------------------------- P12
def test_p12_solvers_agree_and_true_residual():
    cfg = synth.CONFIGS[1]
    dims = cfg["dims"]
    o = oracle.Oracle(dims, synth.gauge(dims, cfg["eps"], cfg["seed"]), -1).set_clover(cfg["kappa"], cfg["csw"])
    b = synth.source(dims, "point")
    sols = {}
    for solver in ("cgne", "cgnr", "bicgstab"):
        x, res = o.invert(b, 1e-10, 1000, solver, 0)
        assert res.status == 0 and res.true_resid < 1e-10 and res.iter_resid <= 1e-10
        assert abs(o.true_residual(b, x) - res.true_resid) < 1e-14
        sols[solver] = x
    assert rel_err(sols["cgnr"], sols["cgne"]) < 1e-9
    assert rel_err(sols["bicgstab"], sols["cgne"]) < 1e-9
    xs, res = o.invert(b, 1e-10, 1000, "bicgstab", 1)
    assert res.status == 0 and rel_err(xs, sols["cgne"]) < 1e-9
    # maxiter reached -> status 1, x still the best iterate
    _, res = o.invert(b, 1e-10, 3, "cgne", 0)
    assert res.status == 1 and res.iterations == 3 and res.true_resid > 1e-10


# ----------------------------------------------------------------------------------------- P13
def test_p13_generator_su3_and_plaquette():
    dims = (4, 4, 4, 8)
    plaq = {}
    for eps in (0.0, 0.3, 0.8):
        U = synth.gauge(dims, eps, 1)
        assert np.abs(U @ dagger(U) - np.eye(3)).max() < 1e-14
        assert np.abs(np.linalg.det(U) - 1).max() < 1e-14
        Ul = gauge_cb_to_lex(U, dims)
        s, cnt = 0.0, 0
        for mu in range(4):
            for nu in range(mu + 1, 4):
                P = Ul[mu] @ shift(Ul[nu], mu, 1) @ dagger(shift(Ul[mu], nu, 1)) @ dagger(Ul[nu])
                s += np.trace(P, axis1=-2, axis2=-1).real.mean() / 3
                cnt += 1
        plaq[eps] = s / cnt
    assert abs(plaq[0.0] - 1) < 1e-15
    assert 0.5 < plaq[0.3] < 0.75        # ~0.62 at eps 0.3
    assert abs(plaq[0.8]) < 0.08         # ~0.0125 at eps 0.8
    # counter-based: same (seed, site) -> same link, independent of thread count or call order
    assert np.array_equal(synth.gauge(dims, 0.3, 1), synth.gauge(dims, 0.3, 1))
    assert not np.array_equal(synth.gauge(dims, 0.3, 1), synth.gauge(dims, 0.3, 2))
    z2 = synth.source(dims, "z2", 3)
    assert set(np.unique(z2.real)) == {-1.0, 1.0} and np.all(z2.imag == 0)
    ga = synth.source((8, 8, 8, 16), "gaussian", 3)
    assert abs(ga.real.std() - 1) < 0.01 and abs(ga.imag.std() - 1) < 0.01 and abs(ga.mean()) < 0.02
    pt = synth.source(dims, "point")
    assert pt[0, 0, 0, 0, 0, 0, 0] == 1 and np.abs(pt).sum() == 1


def test_dslash_site_matches_sweep():
    dims = (4, 6, 4, 8)
    o = oracle.Oracle(dims, synth.gauge(dims, 0.5, 71), -1)
    psi = rand_spinor(dims, 9)
    for dag in (False, True):
        full = o.dslash(psi, dagger=dag).reshape(-1, 4, 3)
        for idx in (0, 1, 17, 383, 384, 500, 767):
            assert np.abs(o.dslash_site(psi, idx, dag) - full[idx]).max() < 1e-14
