"""Pins for the clover-term oracle (oracle/clover.py, Eq 47-49), CPU only.

The expected values come from hand algebra (abelian backgrounds, sigma matrices typed from Eq 1-3), from a
brute-force loop over plaquette angles written with explicit site arithmetic, and from symmetries (gauge
covariance, Hermiticity, [sigma, gamma_5] = 0); none re-types the oracle's leaf products.
"""
import numpy as np
import pytest

from oracle import clover
from harness import synth

FUND, ADJ, SYM, ASY = 0, 1, 2, 3
BC = (-1, 1, 1, 1)
S1 = np.array([[0, 1], [1, 0]], dtype=complex)
S2 = np.array([[0, -1j], [1j, 0]], dtype=complex)
S3 = np.array([[1, 0], [0, -1]], dtype=complex)
Z2 = np.zeros((2, 2), dtype=complex)


def blockdiag(a, b):
    return np.block([[a, Z2], [Z2, b]])


# sigma_{mu nu} = (i/2)[gamma_mu, gamma_nu] with gamma from Eq 3, e_0 = -1, e_k = -i sigma_k, worked out by hand:
# upper block (i/2)(e_mu e_nu^+ - e_nu e_mu^+), lower block (i/2)(e_mu^+ e_nu - e_nu^+ e_mu)
SIGMA = {(0, 1): blockdiag(S1, -S1), (0, 2): blockdiag(S2, -S2), (0, 3): blockdiag(S3, -S3),
         (1, 2): blockdiag(-S3, -S3), (1, 3): blockdiag(S2, S2), (2, 3): blockdiag(-S1, -S1)}


def test_sigma_matches_hand_algebra():
    for (mu, nu), s in SIGMA.items():
        np.testing.assert_allclose(clover.sigma(mu, nu), s, atol=1e-15)
        np.testing.assert_allclose(clover.sigma(nu, mu), -s, atol=1e-15)


def abelian_links(theta):
    """U_mu(x) = exp(i theta_mu(x)) as 1x1 'represented' links [V,4,1,1]."""
    return np.exp(1j * theta).reshape(-1, 4, 1, 1)


@pytest.mark.parametrize("mu,nu", list(SIGMA))
def test_constant_abelian_field(mu, nu):
    """theta_nu(x) = phi x_mu gives P_{mu nu} = e^{i phi} everywhere (phi * extent = 2 pi k), so C = 4 e^{i phi},
    F_{mu nu} = i sin(phi) and (i/4)(sigma_{mu nu}F_{mu nu} + sigma_{nu mu}F_{nu mu}) = -(1/2) sin(phi) sigma_{mu nu}."""
    T, L = 6, 4
    ext = (T, L, L, L)
    phi = 2 * np.pi / ext[mu]
    c = synth.site_coords(T, L)
    theta = np.zeros((T * L ** 3, 4))
    theta[:, nu] = phi * c[:, mu]
    A = clover.clover_term(T, L, abelian_links(theta)).reshape(-1, 4, 4)
    want = -0.5 * np.sin(phi) * SIGMA[(mu, nu)]
    np.testing.assert_allclose(A, np.broadcast_to(want, A.shape), atol=1e-14)


def test_random_abelian_field_brute_force():
    """F_{mu nu}(x) = (i/4) sum of sin(plaquette angle) over the four plaquettes based at x, x-mu, x-mu-nu, x-nu
    (the base points Eq 48 prints), angles from explicit site arithmetic."""
    T, L = 4, 4
    ext = np.array([T, L, L, L])
    rng = np.random.default_rng(5)
    theta = rng.uniform(-np.pi, np.pi, size=(T, L, L, L, 4))

    def th(x, mu):
        return theta[tuple(np.mod(x, ext))][mu]

    def angle(y, mu, nu):
        e = np.eye(4, dtype=int)
        return th(y, mu) + th(y + e[mu], nu) - th(y + e[nu], mu) - th(y, nu)

    R = abelian_links(theta.reshape(-1, 4))
    e = np.eye(4, dtype=int)
    for mu, nu in [(0, 1), (1, 3), (3, 2)]:
        F = clover.field_strength(T, L, R, mu, nu).reshape(T, L, L, L)
        for x in [np.array(v) for v in [(0, 0, 0, 0), (3, 1, 2, 0), (1, 3, 3, 3), (2, 0, 1, 2)]]:
            s = sum(np.sin(angle(y, mu, nu)) for y in (x, x - e[mu], x - e[mu] - e[nu], x - e[nu]))
            assert abs(F[tuple(x)] - 0.25j * s) < 1e-14


def random_problem(oracle, T, L, n, rep, seed):
    cfg = synth.Config("t", T, L, n, rep, -0.3, "haar", seed, ())
    U, (psi, phi) = synth.make_inputs(cfg, n_spinors=2)
    return cfg, U, oracle.represent_field(n, rep, U), psi, phi


@pytest.mark.parametrize("n,rep", [(2, FUND), (3, FUND), (2, ADJ), (3, SYM), (4, ASY)])
def test_hermitian_traceless_chiral(oracle, n, rep):
    T, L = 4, 2
    _, _, R, _, _ = random_problem(oracle, T, L, n, rep, 3)
    A = clover.clover_term(T, L, R)
    V, _, d = A.shape[:3]
    M = A.reshape(V, 4 * d, 4 * d)
    assert np.abs(M).max() > 0.1
    np.testing.assert_allclose(M, np.conj(np.swapaxes(M, 1, 2)), atol=1e-13)
    assert np.abs(np.trace(M, axis1=1, axis2=2)).max() < 1e-12
    assert np.abs(A[:, :2, :, 2:, :]).max() == 0 and np.abs(A[:, 2:, :, :2, :]).max() == 0
    B = clover.chiral_blocks(T, L, R)
    # each chirality block is [[H, B], [B^+, -H]]: sigma_k (x) H_k
    np.testing.assert_allclose(B[:, :, :d, :d], -B[:, :, d:, d:], atol=1e-13)


@pytest.mark.parametrize("n,rep", [(2, FUND), (3, FUND), (2, ADJ)])
def test_pure_gauge_vanishes_and_gauge_covariance(oracle, n, rep):
    T, L = 4, 2
    V = T * L ** 3
    rng = np.random.default_rng(9)
    g = synth.haar_sun(rng, V, n)
    c = synth.site_coords(T, L)
    ext = np.array([T, L, L, L])

    def transform(U):
        out = np.empty_like(U)
        for mu in range(4):
            cn = c.copy()
            cn[:, mu] = (cn[:, mu] + 1) % ext[mu]
            nb = ((cn[:, 0] * L + cn[:, 1]) * L + cn[:, 2]) * L + cn[:, 3]
            out[:, mu] = g @ U[:, mu] @ np.conj(np.swapaxes(g[nb], 1, 2))
        return out

    one = np.broadcast_to(np.eye(n, dtype=complex), (V, 4, n, n)).copy()
    A0 = clover.clover_term(T, L, oracle.represent_field(n, rep, transform(one)))
    assert np.abs(A0).max() < 1e-13
    _, U, R, _, _ = random_problem(oracle, T, L, n, rep, 4)
    A = clover.clover_term(T, L, R)
    Ag = clover.clover_term(T, L, oracle.represent_field(n, rep, transform(U)))
    Rg = oracle.represent_field(n, rep, g)
    want = np.einsum("xab,xsbtc,xdc->xsatd", Rg, A, np.conj(Rg))
    np.testing.assert_allclose(Ag, want, atol=1e-12)


def test_g5_hermiticity_of_clover_operator(oracle):
    T, L, n, rep = 4, 2, 3, FUND
    _, _, R, psi, phi = random_problem(oracle, T, L, n, rep, 6)
    g5 = np.array([1, 1, -1, -1])[None, :, None]
    D = lambda v: clover.Dphi_clover(T, L, -0.2, 1.3, R, v, BC)
    lhs = np.vdot(phi, g5 * D(psi))
    rhs = np.vdot(g5 * D(phi), psi)
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)
    # c_sw = 0 reduces to the unimproved operator
    np.testing.assert_allclose(clover.Dphi_clover(T, L, -0.2, 0.0, R, psi, BC),
                               oracle.Dphi(T, L, 3, -0.2, R, psi, BC), atol=1e-13)


def test_clover_schur_form_against_dense_matrix(oracle):
    """Eq 43 for the clover operator: build the dense matrix of Dphi_clover column by column on 4x2^3, take the Schur
    complement D_ee - D_eo D_oo^{-1} D_oe with numpy's dense solver on the full odd block, compare with the oracle's
    site-by-site version; and det D = det D_oo det D_hat (Eq 42)."""
    from oracle import dense
    T, L, n, rep = 4, 2, 2, FUND
    _, _, R, psi, _ = random_problem(oracle, T, L, n, rep, 8)
    m0, csw = 0.3, 1.1
    V, d = T * L ** 3, 2
    N = V * 4 * d
    D = np.zeros((N, N), dtype=complex)
    for k in range(N):
        e = np.zeros(N, dtype=complex)
        e[k] = 1
        D[:, k] = clover.Dphi_clover(T, L, m0, csw, R, e.reshape(V, 4, d), BC).reshape(-1)
    ie, io = dense.parity_index(T, L, d, 0), dense.parity_index(T, L, d, 1)
    Dee, Deo, Doe, Doo = D[np.ix_(ie, ie)], D[np.ix_(ie, io)], D[np.ix_(io, ie)], D[np.ix_(io, io)]
    S = Dee - Deo @ np.linalg.solve(Doo, Doe)
    ev = synth.parity_sites(T, L, 0)
    got = clover.Dphi_clover_hat(T, L, m0, csw, R, psi[ev], BC).reshape(-1)
    want = S @ psi[ev].reshape(-1)
    assert np.linalg.norm(got - want) < 1e-12 * np.linalg.norm(want)
    s1, l1 = np.linalg.slogdet(D)
    s2, l2 = np.linalg.slogdet(Doo)
    s3, l3 = np.linalg.slogdet(S)
    assert abs(l1 - l2 - l3) < 1e-9 and abs(s1 - s2 * s3) < 1e-9
    # the inverse of the diagonal blocks undoes Cphi
    back = clover.Cphi_inv(T, L, m0, csw, R, clover.Cphi(T, L, m0, csw, R, psi))
    np.testing.assert_allclose(back, psi, atol=1e-12)


def test_exponential_clover_blocks(oracle):
    """Eq 50: closed forms and expansions.  det = (4+m)^(2d) (A traceless), E(c_sw) E^{-1}(c_sw) = 1, c_sw = 0 gives (4+m),
    the expansion to second order in c_sw agrees with (4+m) + c_sw A + c_sw^2 A^2 / (2(4+m)) up to O(c_sw^3), an
    independent Taylor series of the exponential (40 terms, plain matrix products), and the constant abelian background
    where exp(-x sigma_01) = cosh x - sigma_01 sinh x."""
    T, L, n, rep = 4, 2, 3, FUND
    _, _, R, psi, _ = random_problem(oracle, T, L, n, rep, 12)
    m0, csw = -0.2, 1.3
    A = clover.chiral_blocks(T, L, R)
    E = clover.exp_blocks(T, L, m0, csw, R)
    Ei = clover.exp_blocks(T, L, m0, csw, R, inverse=True)
    nn = A.shape[-1]
    eye = np.eye(nn)
    np.testing.assert_allclose(np.linalg.det(E), (4 + m0) ** nn * np.ones(E.shape[:2]), rtol=1e-12)
    np.testing.assert_allclose(E @ Ei, np.broadcast_to(eye, E.shape), atol=1e-13)
    np.testing.assert_allclose(clover.exp_blocks(T, L, m0, 0.0, R), np.broadcast_to((4 + m0) * eye, E.shape), atol=1e-14)
    eps = 1e-3
    E2 = (4 + m0) * eye + eps * A + eps ** 2 * (A @ A) / (2 * (4 + m0))
    assert np.abs(clover.exp_blocks(T, L, m0, eps, R) - E2).max() < 10 * eps ** 3
    X = csw / (4 + m0) * A
    term, ser = np.broadcast_to(eye, A.shape).astype(complex), np.broadcast_to(eye, A.shape).astype(complex)
    for k in range(1, 40):
        term = term @ X / k
        ser = ser + term
    np.testing.assert_allclose(E, (4 + m0) * ser, atol=1e-12)
    # constant abelian background in the (0,1) plane: A = -(1/2) sin(phi) sigma_01, sigma_01^2 = 1
    Ta, La = 6, 4
    phi = 2 * np.pi / Ta
    c = synth.site_coords(Ta, La)
    theta = np.zeros((Ta * La ** 3, 4))
    theta[:, 1] = phi * c[:, 0]
    Eab = clover.exp_blocks(Ta, La, m0, csw, abelian_links(theta))
    x = csw / (4 + m0) * 0.5 * np.sin(phi)
    for cblk, s in ((0, S1), (1, -S1)):
        want = (4 + m0) * (np.cosh(x) * np.eye(2) - np.sinh(x) * s)
        np.testing.assert_allclose(Eab[:, cblk], np.broadcast_to(want, Eab[:, cblk].shape), atol=1e-13)
    # operator level: gamma_5-Hermiticity of the full operator and the Schur form against its definition
    g5 = np.array([1, 1, -1, -1])[None, :, None]
    _, _, _, psi, phi_s = random_problem(oracle, T, L, n, rep, 12)
    D = lambda v: clover.Dphi_expclover(T, L, m0, csw, R, v, BC)
    lhs, rhs = np.vdot(phi_s, g5 * D(psi)), np.vdot(g5 * D(phi_s), psi)
    assert abs(lhs - rhs) < 1e-11 * abs(lhs)
    ev, od = synth.parity_sites(T, L, 0), synth.parity_sites(T, L, 1)
    # solve D (x_e, x_o) = (b, 0) blockwise: D_hat x_e = b with x_o = -D_oo^{-1} D_oe x_e
    xe = psi[ev]
    xo = -clover.apply_blocks(Ei[od], oracle.Dphi_oe(T, L, 3, R, xe, BC))
    full = np.zeros_like(psi)
    full[ev], full[od] = xe, xo
    out = D(full)
    assert np.abs(out[od]).max() < 1e-12
    np.testing.assert_allclose(out[ev], clover.Dphi_expclover_hat(T, L, m0, csw, R, xe, BC), atol=1e-12)
