"""Pins for the oracle's Dirac operator (CPU only): closed forms, invariants, brute force.

None of these re-types the oracle's formula: the free-field symbol is derived by hand from Eq 8, gamma_5
hermiticity / gauge covariance / translation covariance are symmetries of the continuum-motivated operator,
and the dense matrix is assembled by an independent numpy program (oracle/dense.py).
"""
import numpy as np
import pytest

from oracle import dense
from harness import synth

FUND, ADJ, SYM, ASY = 0, 1, 2, 3
BC = (-1, 1, 1, 1)


def small_problem(oracle, T, L, n, rep, seed, links="haar"):
    cfg = synth.Config("t", T, L, n, rep, -0.3, links, seed, ())
    U, (psi, phi) = synth.make_inputs(cfg, n_spinors=2)
    R = oracle.represent_field(n, rep, U)
    return cfg, U, R, psi, phi


# ------------------------------------------------------------------------ free field, closed form
@pytest.mark.parametrize("T,L,n,rep", [(4, 2, 2, FUND), (6, 4, 3, FUND), (4, 2, 2, ADJ), (4, 2, 3, SYM), (4, 4, 4, ASY)])
def test_free_field_plane_wave(oracle, T, L, n, rep):
    """U = 1: D psi = [(4+m - sum cos p) + i sum gamma_mu sin p_mu] psi for psi = exp(ipx) chi,
    p_0 = (2 n_0+1) pi/T (antiperiodic), p_k = 2 pi n_k/L.  From Eq 8:
    -1/2[(1-g)e^{ip} + (1+g)e^{-ip}] = -cos p + i g sin p."""
    d = oracle.rep_dim(n, rep)
    m0 = 0.37
    V = T * L ** 3
    U = np.broadcast_to(np.eye(n, dtype=complex), (V, 4, n, n)).copy()
    R = oracle.represent_field(n, rep, U)
    g, g5 = oracle.gamma(), oracle.gamma5()
    rng = np.random.default_rng(11)
    c = synth.site_coords(T, L)
    for n_mom in [(0, 0, 0, 0), (1, 1, 0, L - 1), (T - 1, 0, 1, 1)]:
        p = np.array([(2 * n_mom[0] + 1) * np.pi / T] + [2 * np.pi * k / L for k in n_mom[1:]])
        chi = rng.standard_normal((4, d)) + 1j * rng.standard_normal((4, d))
        psi = np.exp(1j * (c @ p))[:, None, None] * chi[None]
        M = 4 + m0 - np.cos(p).sum()
        slash = sum(g[mu] * np.sin(p[mu]) for mu in range(4))
        symbol = M * np.eye(4) + 1j * slash
        ref = np.einsum("ab,xbi->xai", symbol, psi)
        out = oracle.Dphi(T, L, d, m0, R, psi, BC)
        assert oracle.rel_l2(out, ref) < 1e-13
        # Q^2 = M^2 + sum sin^2 (a scalar)
        out2 = oracle.g5Dphi_sq(T, L, d, m0, R, psi, BC)
        assert oracle.rel_l2(out2, (M * M + (np.sin(p) ** 2).sum()) * psi) < 1e-13
        # D_hat on the even-restricted wave: (4+m)^2 - (sum cos - i sum g sin)^2
        ev = synth.parity_sites(T, L, 0)
        H = np.cos(p).sum() * np.eye(4) - 1j * slash
        ref_hat = np.einsum("ab,xbi->xai", (4 + m0) ** 2 * np.eye(4) - H @ H, psi[ev])
        out_hat = oracle.Dphi_hat(T, L, d, m0, R, psi[ev], BC)
        assert oracle.rel_l2(out_hat, ref_hat) < 1e-13
    # spectrum multiplicity: eigenvalues M +- i sqrt(sum sin^2), each 2 d-fold (checked on the 4x4 symbol)
    ev4 = np.linalg.eigvals(symbol)
    s = np.sqrt((np.sin(p) ** 2).sum())
    assert np.allclose(sorted(ev4.imag), [-s, -s, s, s], atol=1e-12) and np.allclose(ev4.real, M)


def test_free_field_periodic_time(oracle):
    """bc = +1 in time: momenta p_0 = 2 pi n/T instead (checks that bc is really applied per direction)."""
    T, L, n = 4, 2, 2
    d, m0 = 2, -0.1
    U = np.broadcast_to(np.eye(n, dtype=complex), (T * L ** 3, 4, n, n)).copy()
    g = oracle.gamma()
    c = synth.site_coords(T, L)
    p = np.array([2 * np.pi * 1 / T, 0, np.pi, 0])
    chi = np.arange(8).reshape(4, 2) + 1j
    psi = np.exp(1j * (c @ p))[:, None, None] * chi[None]
    symbol = (4 + m0 - np.cos(p).sum()) * np.eye(4) + 1j * sum(g[mu] * np.sin(p[mu]) for mu in range(4))
    out = oracle.Dphi(T, L, d, m0, U, psi, (1, 1, 1, 1))
    assert oracle.rel_l2(out, np.einsum("ab,xbi->xai", symbol, psi)) < 1e-13
    # antiperiodic in x: p_1 = pi (2n+1)/L
    p = np.array([0, np.pi * 3 / L, 0, 0])
    psi = np.exp(1j * (c @ p))[:, None, None] * chi[None]
    symbol = (4 + m0 - np.cos(p).sum()) * np.eye(4) + 1j * sum(g[mu] * np.sin(p[mu]) for mu in range(4))
    out = oracle.Dphi(T, L, d, m0, U, psi, (1, -1, 1, 1))
    assert oracle.rel_l2(out, np.einsum("ab,xbi->xai", symbol, psi)) < 1e-13


# ------------------------------------------------------------------------------------- invariants
CASES = [(4, 2, 2, FUND), (4, 4, 3, FUND), (2, 4, 2, ADJ), (4, 2, 3, SYM), (4, 2, 4, ASY), (2, 2, 3, ADJ)]


@pytest.mark.parametrize("T,L,n,rep", CASES)
def test_gamma5_hermiticity(oracle, T, L, n, rep):
    cfg, U, R, psi, phi = small_problem(oracle, T, L, n, rep, seed=21)
    d, m0 = cfg.d_R, cfg.m0
    lhs = np.vdot(phi, oracle.g5(oracle.Dphi(T, L, d, m0, R, psi, BC)))
    rhs = np.conj(np.vdot(psi, oracle.g5(oracle.Dphi(T, L, d, m0, R, phi, BC))))
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    q2 = np.vdot(psi, oracle.g5Dphi_sq(T, L, d, m0, R, psi, BC))
    nrm = np.linalg.norm(oracle.Dphi(T, L, d, m0, R, psi, BC)) ** 2
    assert abs(q2.imag) < 1e-12 * nrm and abs(q2.real - nrm) < 1e-12 * nrm    # <psi,Q^2 psi> = |Q psi|^2 > 0
    # gamma5 D_hat is Hermitian as well (Eq 45)
    ev = synth.parity_sites(T, L, 0)
    a = np.vdot(phi[ev], oracle.g5(oracle.Dphi_hat(T, L, d, m0, R, psi[ev], BC)))
    b = np.conj(np.vdot(psi[ev], oracle.g5(oracle.Dphi_hat(T, L, d, m0, R, phi[ev], BC))))
    assert abs(a - b) < 1e-12 * abs(a)


@pytest.mark.parametrize("T,L,n,rep", CASES)
def test_gauge_covariance(oracle, T, L, n, rep):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger, psi' = R(g) psi  =>  D[U'] psi' = R(g) D[U] psi."""
    cfg, U, R, psi, _ = small_problem(oracle, T, L, n, rep, seed=22)
    d, m0 = cfg.d_R, cfg.m0
    V = cfg.volume
    gs = synth.haar_sun(np.random.default_rng(5), V, n)
    c = synth.site_coords(T, L)
    ext = np.array([T, L, L, L])
    Up = np.empty_like(U)
    for mu in range(4):
        cn = c.copy(); cn[:, mu] = (cn[:, mu] + 1) % ext[mu]
        nb = ((cn[:, 0] * L + cn[:, 1]) * L + cn[:, 2]) * L + cn[:, 3]
        Up[:, mu] = gs @ U[:, mu] @ np.conj(np.swapaxes(gs[nb], 1, 2))
    Rg = oracle.represent_field(n, rep, gs)
    Rp = oracle.represent_field(n, rep, Up)
    psip = np.einsum("xij,xaj->xai", Rg, psi)
    lhs = oracle.Dphi(T, L, d, m0, Rp, psip, BC)
    rhs = np.einsum("xij,xaj->xai", Rg, oracle.Dphi(T, L, d, m0, R, psi, BC))
    assert oracle.rel_l2(lhs, rhs) < 1e-13


def test_structural_identities(oracle):
    T, L, n, rep = 4, 4, 3, FUND
    cfg, U, R, psi, phi = small_problem(oracle, T, L, n, rep, seed=23)
    d = cfg.d_R
    D = lambda m, f: oracle.Dphi(T, L, d, m, R, f, BC)
    # linearity and mass shift
    a, b = 0.3 - 0.2j, -1.1 + 0.5j
    assert oracle.rel_l2(D(0.1, a * psi + b * phi), a * D(0.1, psi) + b * D(0.1, phi)) < 1e-14
    assert oracle.rel_l2(D(0.7, psi) - D(-0.2, psi), 0.9 * psi) < 1e-13
    # even/odd decomposition (Eq 41): (D psi)_e = (4+m) psi_e + D_eo psi_o, and likewise for odd
    ev, od = synth.parity_sites(T, L, 0), synth.parity_sites(T, L, 1)
    full = D(0.1, psi)
    assert oracle.rel_l2(full[ev], 4.1 * psi[ev] + oracle.Dphi_eo(T, L, d, R, psi[od], BC)) < 1e-14
    assert oracle.rel_l2(full[od], 4.1 * psi[od] + oracle.Dphi_oe(T, L, d, R, psi[ev], BC)) < 1e-14
    # hop_field is D at m = -4
    assert oracle.rel_l2(oracle.hop_field(T, L, d, R, psi, BC), D(-4.0, psi)) < 1e-14
    # translation covariance in a periodic direction (y): shift links and spinor by one site
    sh = lambda f: np.roll(f.reshape((T, L, L, L) + f.shape[1:]), 1, axis=2).reshape(f.shape)
    assert oracle.rel_l2(oracle.Dphi(T, L, d, 0.1, sh(R), sh(psi), BC), sh(full)) < 1e-14


def test_hop_local_matches_field(oracle):
    """The per-site entry point used for sampled full-size parity is the same function the field loop calls;
    check the neighbour bookkeeping done on the Python side of the sampled tests against the field result."""
    T, L, n, rep = 4, 4, 2, ADJ
    cfg, U, R, psi, _ = small_problem(oracle, T, L, n, rep, seed=24)
    d = cfg.d_R
    full = oracle.hop_field(T, L, d, R, psi, BC)
    c = synth.site_coords(T, L)
    ext = [T, L, L, L]
    for ix in (0, 5, T * L ** 3 - 1, 77):
        Rf, Rb, pf, pb, sf, sb = [], [], [], [], [], []
        for mu in range(4):
            cf = c[ix].copy(); cf[mu] += 1; s = 1
            if cf[mu] == ext[mu]: cf[mu] = 0; s = BC[mu]
            kf = ((cf[0] * L + cf[1]) * L + cf[2]) * L + cf[3]
            sf.append(s); pf.append(psi[kf]); Rf.append(R[ix, mu])
            cb = c[ix].copy(); cb[mu] -= 1; s = 1
            if cb[mu] < 0: cb[mu] = ext[mu] - 1; s = BC[mu]
            kb = ((cb[0] * L + cb[1]) * L + cb[2]) * L + cb[3]
            sb.append(s); pb.append(psi[kb]); Rb.append(R[kb, mu])
        assert np.array_equal(oracle.hop_local(d, Rf, Rb, pf, pb, sf, sb), full[ix])


# ------------------------------------------------------------------------- dense brute force
def test_dense_matrix_config1_4x4x4x4(oracle):
    """BASELINE configs[0]: SU(2) fundamental, 4^4, m0 = 0.1 -- independent dense assembly vs the C oracle."""
    cfg = synth.CONFIGS["C1"]
    U, (psi,) = synth.make_inputs(cfg)
    D = dense.dense_D(cfg.T, cfg.L, cfg.n_g, cfg.rep, U, cfg.m0, BC)
    assert D.shape == (2048, 2048)
    ref = (D @ psi.ravel()).reshape(psi.shape)
    out = oracle.Dphi(cfg.T, cfg.L, cfg.d_R, cfg.m0, oracle.represent_field(2, FUND, U), psi, BC)
    assert oracle.rel_l2(out, ref) < 1e-14
    # gamma5-hermiticity of the matrix itself
    G5 = np.kron(np.eye(cfg.volume), np.kron(dense.gamma5(), np.eye(cfg.d_R)))
    Q = G5 @ D
    assert np.abs(Q - Q.conj().T).max() < 1e-14
    # blocks of Eq 41
    e, o = dense.parity_index(cfg.T, cfg.L, cfg.d_R, 0), dense.parity_index(cfg.T, cfg.L, cfg.d_R, 1)
    Dee, Deo, Doe, Doo = D[np.ix_(e, e)], D[np.ix_(e, o)], D[np.ix_(o, e)], D[np.ix_(o, o)]
    assert np.allclose(Dee, (4 + cfg.m0) * np.eye(len(e))) and np.allclose(Doo, (4 + cfg.m0) * np.eye(len(o)))
    R = oracle.represent_field(2, FUND, U)
    ev, od = synth.parity_sites(cfg.T, cfg.L, 0), synth.parity_sites(cfg.T, cfg.L, 1)
    assert oracle.rel_l2(oracle.Dphi_eo(4, 4, 2, R, psi[od], BC).ravel(), Deo @ psi[od].ravel()) < 1e-14
    assert oracle.rel_l2(oracle.Dphi_oe(4, 4, 2, R, psi[ev], BC).ravel(), Doe @ psi[ev].ravel()) < 1e-14
    # Eq 44 and its relation to the Schur complement Eq 43
    Dhat44 = (4 + cfg.m0) ** 2 * np.eye(len(e)) - Deo @ Doe
    assert oracle.rel_l2(oracle.Dphi_hat(4, 4, 2, cfg.m0, R, psi[ev], BC).ravel(), Dhat44 @ psi[ev].ravel()) < 1e-14
    schur = Dee - Deo @ np.linalg.inv(Doo) @ Doe
    assert np.allclose(Dhat44, (4 + cfg.m0) * schur, atol=1e-12)
    # Q^2 from the matrix
    assert oracle.rel_l2(oracle.g5Dphi_sq(4, 4, 2, cfg.m0, R, psi, BC).ravel(), Q @ (Q @ psi.ravel())) < 1e-14


@pytest.mark.parametrize("n,rep", [(2, ADJ), (3, SYM), (4, ASY), (3, ADJ), (2, SYM)])
def test_dense_matrix_higher_reps_2x2x2x2(oracle, n, rep):
    """Extent-2 lattice (both hops reach the same neighbour, reading A8), higher representations.  The dense
    program builds R(U) with its own numpy formulas, so this also cross-checks the C representation code."""
    T = L = 2
    cfg = synth.Config("t", T, L, n, rep, -0.4, "haar", 31, ())
    U, (psi,) = synth.make_inputs(cfg)
    D = dense.dense_D(T, L, n, rep, U, cfg.m0, BC)
    R = oracle.represent_field(n, rep, U)
    assert oracle.rel_l2(oracle.Dphi(T, L, cfg.d_R, cfg.m0, R, psi, BC).ravel(), D @ psi.ravel()) < 1e-13
    # determinant factorisation Eq 42: det D = det D_oo * det(Schur)
    e, o = dense.parity_index(T, L, cfg.d_R, 0), dense.parity_index(T, L, cfg.d_R, 1)
    Dee, Deo, Doe, Doo = D[np.ix_(e, e)], D[np.ix_(e, o)], D[np.ix_(o, e)], D[np.ix_(o, o)]
    s1, l1 = np.linalg.slogdet(D)
    s2, l2 = np.linalg.slogdet(Doo)
    s3, l3 = np.linalg.slogdet(Dee - Deo @ np.linalg.inv(Doo) @ Doe)
    assert abs(l1 - l2 - l3) < 1e-9 and abs(s1 - s2 * s3) < 1e-9


def test_antiperiodic_bc_equals_link_sign_on_last_time_slice(oracle):
    """L945: antiperiodic BCs = negative sign on the represented links of one time slice.  The oracle applies
    the literal Eq 61 sign on the wrapped hop; flipping U^R_0(t=T-1) with periodic BCs must give the same D."""
    T, L, n, rep = 4, 2, 3, ASY
    cfg, U, R, psi, _ = small_problem(oracle, T, L, n, rep, seed=41)
    d = cfg.d_R
    R2 = R.reshape(T, L ** 3, 4, d, d).copy()
    R2[T - 1, :, 0] *= -1
    out_sign = oracle.Dphi(T, L, d, 0.2, R2.reshape(R.shape), psi, (1, 1, 1, 1))
    out_bc = oracle.Dphi(T, L, d, 0.2, R, psi, BC)
    assert oracle.rel_l2(out_sign, out_bc) < 1e-15
    # a different slice is a different matrix
    R3 = R.reshape(T, L ** 3, 4, d, d).copy()
    R3[0, :, 0] *= -1
    assert oracle.rel_l2(oracle.Dphi(T, L, d, 0.2, R3.reshape(R.shape), psi, (1, 1, 1, 1)), out_bc) > 1e-3


# ------------------------------------------------------------------ twisted mass (Eq 51) and Eq 43
def test_twisted_mass_pins(oracle):
    """Eq 51 / Eq 43 for the twisted-mass diagonal term: free-field symbol, the identity
    (D^tm)^dagger D^tm = D^dagger D + mu^2, and the dense 4^4 matrix with its Schur complement."""
    # (i) free field: D^tm psi = [M(p) + i sum gamma sin p + i mu gamma_5] psi
    T, L, n, rep, m0, mu = 4, 2, 3, FUND, 0.37, 0.21
    d, V = 3, 4 * 8
    U = np.broadcast_to(np.eye(n, dtype=complex), (V, 4, n, n)).copy()
    R = oracle.represent_field(n, rep, U)
    g, g5 = oracle.gamma(), oracle.gamma5()
    c = synth.site_coords(T, L)
    p = np.array([3 * np.pi / T, 2 * np.pi / L, 0.0, 2 * np.pi / L])
    rng = np.random.default_rng(4)
    chi = rng.standard_normal((4, d)) + 1j * rng.standard_normal((4, d))
    psi = np.exp(1j * (c @ p))[:, None, None] * chi[None]
    symbol = (4 + m0 - np.cos(p).sum()) * np.eye(4) + 1j * sum(g[k] * np.sin(p[k]) for k in range(4)) + 1j * mu * g5
    assert oracle.rel_l2(oracle.Dphi_tm(T, L, d, m0, mu, R, psi, BC), np.einsum("ab,xbi->xai", symbol, psi)) < 1e-13
    # (ii) random links: (D^tm)^dag D^tm = Q^2 + mu^2 (the cross terms cancel by gamma_5-hermiticity), any sign of mu
    cfg = synth.CONFIGS["C1"]
    Uc, (b, phi) = synth.make_inputs(cfg, 2)
    Rc = oracle.represent_field(cfg.n_g, cfg.rep, Uc)
    T, L, d = cfg.T, cfg.L, cfg.d_R
    for sgn in (+1, -1):
        lhs = oracle.Dphi_tm_sq(T, L, d, m0, sgn * mu, Rc, b, BC)
        rhs = oracle.g5Dphi_sq(T, L, d, m0, Rc, b, BC) + mu * mu * b
        assert oracle.rel_l2(lhs, rhs) < 1e-13
    # (iii) dense: D^tm = D + i mu G5; its dagger; the Schur complement of Eq 43
    D = dense.dense_D(T, L, cfg.n_g, cfg.rep, Uc, m0, BC)
    G5 = np.kron(np.eye(cfg.volume), np.kron(dense.gamma5(), np.eye(d)))
    Dtm = D + 1j * mu * G5
    out = oracle.Dphi_tm(T, L, d, m0, mu, Rc, b, BC)
    assert np.linalg.norm(out.ravel() - Dtm @ b.ravel()) < 1e-13 * np.linalg.norm(out)
    sq = oracle.Dphi_tm_sq(T, L, d, m0, mu, Rc, b, BC)
    assert np.linalg.norm(sq.ravel() - Dtm.conj().T @ (Dtm @ b.ravel())) < 1e-13 * np.linalg.norm(sq)
    e, o = dense.parity_index(T, L, d, 0), dense.parity_index(T, L, d, 1)
    schur = Dtm[np.ix_(e, e)] - Dtm[np.ix_(e, o)] @ np.linalg.solve(Dtm[np.ix_(o, o)], Dtm[np.ix_(o, e)])
    ev = synth.parity_sites(T, L, 0)
    hat = oracle.Dphi_tm_hat(T, L, d, m0, mu, Rc, phi[ev], BC)
    assert np.linalg.norm(hat.ravel() - schur @ phi[ev].ravel()) < 1e-13 * np.linalg.norm(hat)
    # mu = 0 reduces to Eq 43 = Eq 44 / (4+m)
    hat0 = oracle.Dphi_tm_hat(T, L, d, m0, 0.0, Rc, phi[ev], BC)
    assert oracle.rel_l2((4 + m0) * hat0, oracle.Dphi_hat(T, L, d, m0, Rc, phi[ev], BC)) < 1e-13
    # gamma_5 linear combination: hand values on one site
    one = np.zeros((1, 4, 1), complex); one[0, :, 0] = [1, 2j, 3, -1]
    assert np.array_equal(oracle.g5_lc(2.0, 1j, one)[0, :, 0], np.array([2 + 1j, 4j - 2, 6 - 3j, -2 + 1j]))
