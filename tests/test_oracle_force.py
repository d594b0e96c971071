"""Pins of the force oracle (oracle/force.py; Eq 20-21) against what the paper and the mathematics fix.

The paper prints no numbers for the force, and Eq 21 is garbled (reading A32), so the pin is the DEFINITION of a force in
Hamilton's equations (Eq 14-18): F^a_mu(x) = -(1/T_FUND) dS_f / d omega^a for U_mu(x) -> exp(i omega^a T^a) U_mu(x), with
S_f = psi^dagger (Q_m^2)^-1 psi evaluated by an independent dense solve (oracle/dense.py, numpy) -- a dropped term, a wrong
sign, a transposed outer product, a missing boundary factor or a wrong generator normalisation all fail it.  Plus: gauge
covariance (the force rotates in the adjoint), the representation generators against Tbl 1, and the symmetry of Eq 20.
"""
import numpy as np
import pytest

from harness import synth
from oracle import dense
from oracle import force as of

FUND, ADJ, SYM, ASY = 0, 1, 2, 3
BC = (-1, 1, 1, 1)


def expm_herm(H, eps):
    w, v = np.linalg.eigh(H)
    return (v * np.exp(1j * eps * w)) @ v.conj().T


def action(T, L, n, rep, U, m0, phi, bc):
    D = dense.dense_D(T, L, n, rep, U, m0, bc)
    d = D.shape[0] // (T * L ** 3 * 4)
    g5 = np.kron(np.eye(T * L ** 3), np.kron(dense.gamma5(), np.eye(d)))
    Q = g5 @ D
    eta = np.linalg.solve(Q @ Q, phi.ravel())
    return float(np.real(np.vdot(phi.ravel(), eta))), eta, Q


@pytest.mark.parametrize("n,rep,T,L,bc", [(3, FUND, 2, 2, BC), (2, ADJ, 2, 2, BC), (4, ASY, 2, 2, (1, 1, 1, 1)), (2, SYM, 4, 2, (-1, 1, -1, 1)),
                                          (3, SYM, 2, 2, BC), (2, FUND, 4, 2, BC)])
def test_force_is_minus_derivative_of_the_action(oracle, n, rep, T, L, bc):
    cfg = synth.Config("t", T, L, n, rep, 0.35, "haar", 4000 + 10 * n + rep, ())
    U, (phi,) = synth.make_inputs(cfg)
    V, d, m0 = cfg.volume, cfg.d_R, cfg.m0
    S0, eta, Q = action(T, L, n, rep, U, m0, phi, bc)
    xi = Q @ eta
    R = oracle.represent_field(n, rep, U)
    F = of.force_hopping(T, L, n, rep, R, eta.reshape(V, 4, d), xi.reshape(V, 4, d), bc)
    assert F.shape == (V, 4, n * n - 1) and F.dtype == np.float64
    Tf = oracle.generators(n)
    rng = np.random.default_rng(1)
    eps = 1e-4
    # boundary links (t = T-1, mu = 0 and an edge in a spatial direction) and interior ones, several generators
    picks = [(V - 1, 0), (0, 0), (V - 1, 2), (int(rng.integers(V)), 1), (int(rng.integers(V)), 3)]
    for ix, mu in picks:
        for a in sorted(set([0, len(Tf) - 1, int(rng.integers(len(Tf)))])):
            Up, Um = U.copy(), U.copy()
            Up[ix, mu] = expm_herm(Tf[a], +eps) @ U[ix, mu]
            Um[ix, mu] = expm_herm(Tf[a], -eps) @ U[ix, mu]
            dS = (action(T, L, n, rep, Up, m0, phi, bc)[0] - action(T, L, n, rep, Um, m0, phi, bc)[0]) / (2 * eps)
            assert abs(F[ix, mu, a] + dS / of.T_FUND) < 2e-6 * max(1.0, abs(dS)), (ix, mu, a, F[ix, mu, a], -dS / of.T_FUND)


@pytest.mark.parametrize("n,rep", [(3, FUND), (2, ADJ), (3, ASY), (2, SYM)])
def test_force_gauge_covariance(oracle, n, rep):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dagger, eta' = R(g) eta, xi' = R(g) xi  =>  F'^a_mu(x) T^a = g(x) F^b_mu(x) T^b g(x)^dagger,
    i.e. F' = Ad(g(x)) F with the adjoint representation matrix (real, orthogonal)."""
    T, L = 2, 4
    cfg = synth.Config("t", T, L, n, rep, 0.0, "haar", 4100 + 10 * n + rep, ())
    U, (eta, xi) = synth.make_inputs(cfg, 2)
    V = cfg.volume
    rng = np.random.Generator(np.random.PCG64(9))
    g = synth.haar_sun(rng, V, n)
    c = synth.site_coords(T, L)
    ext = np.array([T, L, L, L])
    Ug = np.empty_like(U)
    for mu in range(4):
        cf = c.copy(); cf[:, mu] = (cf[:, mu] + 1) % ext[mu]
        nb = ((cf[:, 0] * L + cf[:, 1]) * L + cf[:, 2]) * L + cf[:, 3]
        Ug[:, mu] = g @ U[:, mu] @ np.conj(np.swapaxes(g[nb], 1, 2))
    Rg = np.array([oracle.rep_matrix(n, rep, m) for m in g])
    F = of.force_hopping(T, L, n, rep, oracle.represent_field(n, rep, U), eta, xi, BC)
    Fg = of.force_hopping(T, L, n, rep, oracle.represent_field(n, rep, Ug), np.einsum("xij,xsj->xsi", Rg, eta),
                          np.einsum("xij,xsj->xsi", Rg, xi), BC)
    Ad = np.array([oracle.rep_matrix(n, ADJ, m).real for m in g])
    assert np.allclose(Fg, np.einsum("xab,xmb->xma", Ad, F), atol=1e-12 * np.abs(F).max())


@pytest.mark.parametrize("n,rep,t_r", [(2, FUND, 0.5), (3, FUND, 0.5), (2, ADJ, 2.0), (3, ADJ, 3.0), (3, SYM, 2.5), (4, ASY, 1.0), (3, ASY, 0.5)])
def test_rep_generators_exact(oracle, n, rep, t_r):
    """T_R^a (A33): Hermitian, traceless, tr(T_R^a T_R^b) = T_R delta^ab (Tbl 1, L213-220, A12), a representation of the algebra
    ([T_R^a, T_R^b] = i f^abc T_R^c with the f of the fundamental), and equal to the small-angle derivative of R."""
    TR = of.rep_generators(n, rep)
    Tf = oracle.generators(n)
    na = n * n - 1
    assert TR.shape == (na, oracle.rep_dim(n, rep), oracle.rep_dim(n, rep))
    gram = np.einsum("aij,bji->ab", TR, TR)
    assert np.allclose(gram, t_r * np.eye(na), atol=1e-13)
    assert np.allclose(TR, np.conj(np.swapaxes(TR, 1, 2)), atol=1e-14) and np.allclose(np.einsum("aii->a", TR), 0, atol=1e-14)
    for a, b in [(0, 1), (1, na - 1), (0, na - 1)]:
        comm_f = Tf[a] @ Tf[b] - Tf[b] @ Tf[a]
        coef = np.array([2 * np.trace(comm_f @ Tf[c]) for c in range(na)])          # [T^a,T^b] = sum_c coef_c T^c
        assert np.allclose(TR[a] @ TR[b] - TR[b] @ TR[a], np.einsum("c,cij->ij", coef, TR), atol=1e-13)
    eps = 1e-5
    fd = (oracle.rep_matrix(n, rep, expm_herm(Tf[1], eps)) - oracle.rep_matrix(n, rep, expm_herm(Tf[1], -eps))) / (2j * eps)
    assert np.allclose(fd, TR[1], atol=1e-9)


def test_traced_operator_symmetry_and_fund_projection(oracle):
    """Eq 20 is symmetric under eta <-> xi, and Hermitian-conjugating the colour matrix U T maps the two terms into each other
    only through the trace, so F is real by construction; for FUND the projection onto S_ij, A_ij is an entry of U T."""
    T, L, n = 2, 2, 3
    cfg = synth.Config("t", T, L, n, FUND, 0.0, "haar", 4200, ())
    U, (eta, xi) = synth.make_inputs(cfg, 2)
    R = oracle.represent_field(n, FUND, U)
    F1 = of.force_hopping(T, L, n, FUND, R, eta, xi, BC)
    F2 = of.force_hopping(T, L, n, FUND, R, xi, eta, BC)
    assert np.array_equal(F1, F2) or np.allclose(F1, F2, rtol=0, atol=1e-13)
    M = np.einsum("xjk,xki->xji", R[:, 1], of.traced_operator(T, L, 1, eta, xi, BC))
    # generator 0 is S_01 = (E_01 + E_10)/2: -(1/T_F) Re tr[i S M] = 2 * Im(M_01 + M_10)/2
    assert np.allclose(F1[:, 1, 0], np.imag(M[:, 0, 1] + M[:, 1, 0]), atol=1e-13)
    # generator 1 is A_01 = -i(E_01 - E_10)/2: tr[A M] = -i(M_10 - M_01)/2  ->  F = 2 Im(tr[A M]) = -(Re M_10 - Re M_01)
    assert np.allclose(F1[:, 1, 1], -(np.real(M[:, 1, 0]) - np.real(M[:, 0, 1])), atol=1e-13)
