"""Pins P1-P6, P15 of SURVEY.md 8(c): the oracle's gamma algebra, operator, even-odd
algebra and covariance, checked against closed forms, invariants and brute force."""
import itertools

import numpy as np
import pytest

import oracle
from paper_1211_0126_b200 import workloads as W
from dense_helpers import coords, dense_from_apply, parity, volume

G5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)


def g5(psi):
    return np.einsum("ab,xbc->xac", G5, psi)


def inner(a, b):
    return np.vdot(a.reshape(-1), b.reshape(-1))


# ---------------------------------------------------------------- P1 gamma algebra
def test_p1_gamma_algebra():
    g = [oracle.gamma(2 + m) for m in range(4)]
    one = np.eye(4)
    for m, n in itertools.product(range(4), repeat=2):
        assert np.allclose(g[m] @ g[n] + g[n] @ g[m], 2 * one * (m == n), atol=0)
    for m in range(4):
        assert np.array_equal(g[m], g[m].conj().T)
    assert np.array_equal(oracle.gamma(0), one)
    assert np.array_equal(oracle.gamma(1), G5)
    assert np.array_equal(g[0] @ g[1] @ g[2] @ g[3], G5)
    # C3 as printed: gamma_3 = [[0,1],[1,0]], gamma_k upper-right block = -i sigma_k
    assert np.array_equal(g[3], np.block([[np.zeros((2, 2)), np.eye(2)], [np.eye(2), np.zeros((2, 2))]]))
    sig = [np.array([[0, 1], [1, 0]]), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]])]
    for k in range(3):
        assert np.array_equal(g[k][:2, 2:], -1j * sig[k])
        assert np.array_equal(g[k][2:, :2], 1j * sig[k])
        assert not g[k][:2, :2].any() and not g[k][2:, 2:].any()
    for m in range(4):
        assert np.array_equal(oracle.gamma(6 + m), G5 @ g[m])
        assert np.array_equal(oracle.gamma(6 + m).conj().T, -oracle.gamma(6 + m))  # anti-hermitian
    pairs = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    for i, (m, n) in enumerate(pairs):
        s = oracle.gamma(10 + i)
        assert np.array_equal(s, 0.5j * (g[m] @ g[n] - g[n] @ g[m]))
        assert np.array_equal(s, s.conj().T)
    allg = np.stack([oracle.gamma(i).reshape(-1) for i in range(16)])
    assert np.linalg.matrix_rank(allg) == 16
    for i in range(16):  # one non-zero per row, in {+-1, +-i}
        G = oracle.gamma(i)
        assert ((G != 0).sum(axis=1) == 1).all()
        assert set(np.round(G[G != 0], 12).tolist()) <= {1, -1, 1j, -1j}


def test_p1_projection_identity():
    """(1 +- gamma_mu) psi = [h; +- a_mu^dag h], h = psi_up +- a_mu psi_low (C3)."""
    rng = np.random.default_rng(1)
    psi = rng.standard_normal(4) + 1j * rng.standard_normal(4)
    for m in range(4):
        gm = oracle.gamma(2 + m)
        a = gm[:2, 2:]
        for sgn in (+1, -1):
            full = psi + sgn * gm @ psi
            h = psi[:2] + sgn * a @ psi[2:]
            assert np.allclose(full, np.concatenate([h, sgn * a.conj().T @ h]), atol=1e-15)


# ---------------------------------------------------------------- P2 free field
@pytest.mark.parametrize("theta", [+1, -1])
def test_p2_free_field_spectrum(theta):
    dims = (2, 2, 2, 4)
    kappa, mu = 0.12, 0.3
    a = 2 * kappa * mu
    U = W.unit_links(dims)
    V = volume(dims)
    M = dense_from_apply(lambda v: oracle.apply_M(dims, theta, kappa, mu, U, v), V)
    ev = np.linalg.eigvals(M)
    expect = []
    for n in itertools.product(*[range(L) for L in dims]):
        p = [2 * np.pi * n[i] / dims[i] for i in range(3)]
        p.append(2 * np.pi * n[3] / dims[3] if theta == 1 else (2 * n[3] + 1) * np.pi / dims[3])
        A = 1 - 2 * kappa * sum(np.cos(p))
        B2 = sum((2 * kappa * np.sin(q)) ** 2 for q in p)
        expect += [A + 1j * np.sqrt(B2 + a * a)] * 6 + [A - 1j * np.sqrt(B2 + a * a)] * 6
    expect = np.array(expect)
    # match the two multisets: sort by (real, imag) rounded
    key = lambda z: np.lexsort((np.round(z.imag, 9), np.round(z.real, 9)))
    assert np.allclose(ev[key(ev)], expect[key(expect)], atol=1e-12)


@pytest.mark.parametrize("theta", [+1, -1])
def test_p2_plane_waves_mdagm_scalar(theta):
    """|M psi|^2 = (A^2 + B^2 + a^2)|psi|^2 for every plane wave, any constant spinor."""
    dims = (4, 6, 4, 8)
    kappa, mu = 0.13, 0.21
    a = 2 * kappa * mu
    U = W.unit_links(dims)
    xs = coords(dims)
    rng = np.random.default_rng(5)
    for n in [(0, 0, 0, 0), (1, 2, 3, 5), (3, 5, 1, 7), (2, 0, 1, 4)]:
        p = [2 * np.pi * n[i] / dims[i] for i in range(3)]
        p.append(2 * np.pi * n[3] / dims[3] if theta == 1 else (2 * n[3] + 1) * np.pi / dims[3])
        u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
        psi = np.exp(1j * (xs @ np.array(p)))[:, None, None] * u[None]
        out = oracle.apply_M(dims, theta, kappa, mu, U, psi)
        A = 1 - 2 * kappa * sum(np.cos(p))
        B2 = sum((2 * kappa * np.sin(q)) ** 2 for q in p)
        assert np.isclose(np.vdot(out, out).real, (A * A + B2 + a * a) * np.vdot(psi, psi).real, rtol=1e-12)
        # the plane wave stays a plane wave: M psi = e^{ipx} (M(p) u)
        ratio = out / np.exp(1j * (xs @ np.array(p)))[:, None, None]
        assert np.allclose(ratio, ratio[0][None], atol=1e-12)


# ---------------------------------------------------------------- P3 / P4 hermiticity, twisted mass
def _setup(dims=(4, 4, 2, 6), eps=0.6, seed=3):
    U = W.random_su3_links(dims, eps, seed)
    phi = W.random_spinor(dims, 11)
    psi = W.random_spinor(dims, 12)
    return dims, U, phi, psi


@pytest.mark.parametrize("theta", [+1, -1])
def test_p3_gamma5_hermiticity(theta):
    dims, U, phi, psi = _setup()
    kappa, mu = 0.16, 0.05
    lhs = inner(phi, oracle.apply_M(dims, theta, kappa, mu, U, psi))
    rhs = inner(g5(oracle.apply_M(dims, theta, kappa, -mu, U, g5(phi))), psi)
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)


@pytest.mark.parametrize("theta", [+1, -1])
def test_p3_mhat_dag_is_the_adjoint(theta):
    dims, U, phi, psi = _setup()
    kappa, mu = 0.16, 0.05
    even = parity(dims) == 0
    phi = phi * even[:, None, None]
    psi = psi * even[:, None, None]
    lhs = inner(phi, oracle.apply_Mhat(dims, theta, kappa, mu, U, psi))
    rhs = inner(oracle.apply_Mhat_dag(dims, theta, kappa, mu, U, phi), psi)
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)
    # D_eo^dag = gamma5 D_oe gamma5
    odd = ~even
    chi = W.random_spinor(dims, 13) * odd[:, None, None]
    lhs = inner(psi, oracle.hop(dims, theta, U, chi, 0))
    rhs = inner(g5(oracle.hop(dims, theta, U, g5(psi), 1)), chi)
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)
    # Mhat keeps odd sites empty
    assert not oracle.apply_Mhat(dims, theta, kappa, mu, U, psi)[odd].any()


def test_p4_twisted_mass_identities():
    """M(mu) - M(-mu) = 2 i a gamma5 and lambda_min(M^dag M) >= a^2."""
    dims, U, phi, psi = _setup()
    kappa, mu = 0.16, 0.05
    a = 2 * kappa * mu
    d = oracle.apply_M(dims, -1, kappa, mu, U, psi) - oracle.apply_M(dims, -1, kappa, -mu, U, psi)
    assert np.allclose(d, 2j * a * g5(psi), atol=1e-13)
    # M(mu) + M(-mu) = 2 (1 - kappa D_hop): independent of mu
    s1 = oracle.apply_M(dims, -1, kappa, mu, U, psi) + oracle.apply_M(dims, -1, kappa, -mu, U, psi)
    s2 = 2 * oracle.apply_M(dims, -1, kappa, 0.0, U, psi)
    assert np.allclose(s1, s2, atol=1e-13)
    Mpsi = oracle.apply_M(dims, -1, kappa, mu, U, psi)
    assert np.vdot(Mpsi, Mpsi).real >= a * a * np.vdot(psi, psi).real
    # dense: near-critical kappa so that the bound is what keeps the spectrum away from 0
    dims2 = (2, 2, 2, 4)
    U2 = W.random_su3_links(dims2, 0.7, 9)
    for kap, m in [(0.18, 0.4), (0.20, 1.0)]:
        M = dense_from_apply(lambda v: oracle.apply_M(dims2, -1, kap, m, U2, v), volume(dims2))
        lam = np.linalg.eigvalsh(M.conj().T @ M)
        assert lam.min() >= (2 * kap * m) ** 2 * (1 - 1e-12)
        # M^dag M = Q^2 + a^2 with Q = gamma5 (1 - kappa D_hop) hermitian
        M0 = dense_from_apply(lambda v: oracle.apply_M(dims2, -1, kap, 0.0, U2, v), volume(dims2))
        Q = np.kron(np.eye(volume(dims2)), np.kron(G5, np.eye(3))) @ M0
        assert np.allclose(Q, Q.conj().T, atol=1e-13)
        assert np.allclose(M.conj().T @ M, Q @ Q + (2 * kap * m) ** 2 * np.eye(len(Q)), atol=1e-12)


# ---------------------------------------------------------------- P5 even-odd algebra
def test_p5_even_odd_blocks_and_schur():
    dims = (2, 2, 2, 4)
    kappa, mu, theta = 0.17, 0.3, -1
    a = 2 * kappa * mu
    U = W.random_su3_links(dims, 0.7, 21)
    V = volume(dims)
    par = parity(dims)
    e, o = par == 0, par == 1
    M = dense_from_apply(lambda v: oracle.apply_M(dims, theta, kappa, mu, U, v), V)
    sel_e = np.arange(12 * V).reshape(V, 12)[e].reshape(-1)
    sel_o = np.arange(12 * V).reshape(V, 12)[o].reshape(-1)
    Mee, Meo = M[np.ix_(sel_e, sel_e)], M[np.ix_(sel_e, sel_o)]
    Moe, Moo = M[np.ix_(sel_o, sel_e)], M[np.ix_(sel_o, sel_o)]
    R = np.kron(np.eye(V // 2), np.kron(np.eye(4) + 1j * a * G5, np.eye(3)))
    assert np.allclose(Mee, R, atol=1e-14) and np.allclose(Moo, R, atol=1e-14)  # no same-parity hops
    Mhat = dense_from_apply(lambda v: oracle.apply_Mhat(dims, theta, kappa, mu, U, v), V, site_mask=e)
    assert np.allclose(Mhat, Mee - Meo @ np.linalg.inv(Moo) @ Moe, atol=1e-13)
    Mhd = dense_from_apply(lambda v: oracle.apply_Mhat_dag(dims, theta, kappa, mu, U, v), V, site_mask=e)
    assert np.allclose(Mhd, Mhat.conj().T, atol=1e-13)


def test_p5_solve_satisfies_full_system():
    wl = W.WORKLOADS[1]
    U = wl.links()
    eta = oracle.noise(wl.dims, wl.noise_seed, 0)
    for tol in (1e-10, 1e-4):
        s, info = oracle.solve(wl.dims, -1, wl.kappa, wl.mu, U, eta, tol, 500)
        res = eta - oracle.apply_M(wl.dims, -1, wl.kappa, wl.mu, U, s)
        rel = np.linalg.norm(res) / np.linalg.norm(eta)
        assert rel < 2 * tol
        assert np.isclose(rel, info["rel_resid_true"], rtol=1e-6)
        assert np.isclose(rel, oracle.true_residual(wl.dims, -1, wl.kappa, wl.mu, U, eta, s), rtol=1e-6)
    assert info["status"] == 0


# ---------------------------------------------------------------- P6 gauge covariance
def test_p6_gauge_covariance():
    dims = (4, 4, 4, 4)
    kappa, mu, theta = 0.15, 0.02, -1
    U = W.random_su3_links(dims, 0.5, 31)
    Om = W.random_su3_sites(dims, 32)
    assert np.allclose(np.einsum("nij,nkj->nik", Om, Om.conj()), np.eye(3)[None], atol=1e-13)
    assert np.allclose(np.linalg.det(Om), 1, atol=1e-13)
    Ug = W.gauge_transform(dims, U, Om)
    psi = W.random_spinor(dims, 33)
    rot = lambda f: np.einsum("nij,naj->nai", Om, f)
    assert np.allclose(oracle.apply_M(dims, theta, kappa, mu, Ug, rot(psi)),
                       rot(oracle.apply_M(dims, theta, kappa, mu, U, psi)), atol=1e-12)
    eta = oracle.noise(dims, 77, 3)
    s, _ = oracle.solve(dims, theta, kappa, mu, U, eta, 1e-12, 500)
    sg, _ = oracle.solve(dims, theta, kappa, mu, Ug, rot(eta), 1e-12, 500)
    assert np.allclose(sg, rot(s), atol=1e-9)
    L0 = oracle.all_loops(dims, theta, U, eta, s, True)
    L1 = oracle.all_loops(dims, theta, Ug, rot(eta), sg, True)
    assert np.abs(L0 - L1).max() < 1e-8 * np.abs(L0).max()
    # exact covariance of the contraction itself (same s on both sides)
    L2 = oracle.all_loops(dims, theta, Ug, rot(eta), rot(s), True)
    assert np.abs(L0 - L2).max() < 1e-12 * np.abs(L0).max()


# ---------------------------------------------------------------- P15 delta-source stencil
@pytest.mark.parametrize("theta", [+1, -1])
def test_p15_delta_source_blocks(theta):
    dims = (4, 6, 4, 4)
    V = volume(dims)
    U = W.random_su3_links(dims, 0.8, 41)
    xs = coords(dims)
    lex = lambda x: x[0] + dims[0] * (x[1] + dims[1] * (x[2] + dims[2] * x[3]))
    for y in [(1, 2, 3, 0), (0, 0, 0, 3), (3, 5, 3, 3)]:
        ly = lex(y)
        for beta, cc in [(0, 0), (2, 1), (3, 2)]:
            src = np.zeros((V, 4, 3), dtype=np.complex128)
            src[ly, beta, cc] = 1.0
            out = oracle.hop(dims, theta, U, src)
            expect = np.zeros_like(out)
            for m in range(4):
                gm = oracle.gamma(2 + m)
                xm = list(y); xm[m] = (y[m] - 1) % dims[m]      # x = y - mu sees y as x + mu
                xp = list(y); xp[m] = (y[m] + 1) % dims[m]      # x = y + mu sees y as x - mu
                php = theta if (m == 3 and xm[3] == dims[3] - 1) else 1
                phm = theta if (m == 3 and xp[3] == 0) else 1
                expect[lex(xm)] += php * np.outer((np.eye(4) - gm)[:, beta], U[m, lex(xm)][:, cc])
                expect[lex(xp)] += phm * np.outer((np.eye(4) + gm)[:, beta], U[m, ly].conj().T[:, cc])
            assert np.allclose(out, expect, atol=1e-14)
            nz = np.unique(np.nonzero(np.abs(out).sum(axis=(1, 2)))[0])
            assert len(nz) == 8 and ((xs[nz].sum(axis=1) & 1) != (sum(y) & 1)).all()
    # parity-restricted hop = full hop masked
    psi = W.random_spinor(dims, 42)
    full = oracle.hop(dims, theta, U, psi)
    par = parity(dims)
    for p in (0, 1):
        assert np.array_equal(oracle.hop(dims, theta, U, psi, p), full * (par == p)[:, None, None])
