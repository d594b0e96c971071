"""Pins of oracle/linalg.py against what the paper and the mathematics fix (no GPU, no CUDA code).

Compensated sums: Alg 1-4 against exact rational arithmetic and the textbook cancellation
example; products/norms (Eq 27, 32, 33) against exact rationals and their algebraic properties; linear combinations
(Eq 22-26) against hand-computed values and mutual identities; CG (L730, L772) against a dense direct solve of the
independently assembled 4^4 matrix (oracle/dense.py) and the finite-termination property.
"""
from fractions import Fraction

import numpy as np
import pytest

from oracle import dense
from oracle import linalg as la
from harness import synth

BC = (-1, 1, 1, 1)


def exact(a):
    return sum((Fraction(float(x)) for x in a), Fraction(0))


# ------------------------------------------------------------------------------------------ Alg 1-4
def test_fast_two_sum_is_exact():
    rng = np.random.default_rng(1)
    for _ in range(2000):
        a, b = float(rng.normal() * 10.0 ** rng.integers(-20, 20)), float(rng.normal() * 10.0 ** rng.integers(-20, 20))
        s, c = la.fast_two_sum(a, b)
        assert s == a + b                                         # s = fl(a + b)
        assert Fraction(s) + Fraction(c) == Fraction(a) + Fraction(b)   # s + c = a + b exactly (L640)


def test_textbook_cancellation_example():
    # the standard example separating Kahan from Neumaier: naive (and Kahan) give 0, Neumaier gives the exact 2
    a = [1.0, 1e100, 1.0, -1e100]
    assert la.naive_sum(a) == 0.0
    assert la.neumaier(a) == 2.0
    assert la.second_order_neumaier(a) == 2.0
    assert la.double_double_sum(a) == 2.0


def test_compensated_sums_error_does_not_grow():
    """L698: the error of the compensated sums stays O(eps) while the naive error grows with the number of terms."""
    rng = np.random.default_rng(7)
    a = (rng.normal(size=200000) * 10.0 ** rng.uniform(-6, 6, size=200000)).tolist()
    ex = exact(a)
    scale = float(sum(abs(Fraction(x)) for x in a))
    err = lambda v: abs(float(Fraction(v) - ex)) / scale
    assert err(la.neumaier(a)) < 2.0 ** -52
    assert err(la.second_order_neumaier(a)) < 2.0 ** -52
    assert err(la.double_double_sum(a)) < 2.0 ** -52
    # positive terms: the naive sum drifts by many ulps of the result, the compensated ones are within one ulp
    b = rng.uniform(0.0, 1.0, size=300000).tolist()
    exb = exact(b)
    ulp = float(exb) * 2.0 ** -52
    assert abs(float(Fraction(la.naive_sum(b)) - exb)) > 4 * ulp
    for f in (la.neumaier, la.second_order_neumaier, la.double_double_sum):
        assert abs(float(Fraction(f(b)) - exb)) <= ulp


def test_compensated_sums_on_ill_conditioned_sum():
    # condition number ~1e20 (sum = 500, sum of |terms| ~ 1e23): naive summation loses everything, the three
    # compensated algorithms (error eps^2 * n * sum|a| << 1) return the exact sum
    a = []
    rng = np.random.default_rng(3)
    for _ in range(500):
        big = float(rng.normal() * 1e20)
        mid = float(rng.normal() * 1e8)
        a += [big, mid, 1.0, -big, -mid]
    assert float(exact(a)) == 500.0
    assert la.neumaier(a) == 500.0
    assert la.double_double_sum(a) == 500.0
    assert la.second_order_neumaier(a) == 500.0
    assert abs(la.naive_sum(a) - 500.0) > 1.0


# --------------------------------------------------------------------------------------- Eq 27, 32, 33
def test_products_and_norms():
    rng = np.random.default_rng(11)
    xi = rng.normal(size=(50, 4, 3)) + 1j * rng.normal(size=(50, 4, 3))
    eta = rng.normal(size=(50, 4, 3)) + 1j * rng.normal(size=(50, 4, 3))
    # Eq 27 against exact rational arithmetic
    ex_re = sum(Fraction(float(a.real)) * Fraction(float(b.real)) + Fraction(float(a.imag)) * Fraction(float(b.imag))
                for a, b in zip(xi.ravel(), eta.ravel()))
    ex_im = sum(Fraction(float(a.real)) * Fraction(float(b.imag)) - Fraction(float(a.imag)) * Fraction(float(b.real))
                for a, b in zip(xi.ravel(), eta.ravel()))
    p = la.prod(xi, eta)
    mag = float(np.sum(np.abs(xi) * np.abs(eta)))
    assert abs(p.real - float(ex_re)) <= 2.0 ** -52 * mag and abs(p.imag - float(ex_im)) <= 2.0 ** -52 * mag
    # conj(xi) on the LEFT (a wrong side would flip the sign of the imaginary part)
    assert p.imag != 0 and la.prod(eta, xi) == p.conjugate()
    assert abs(la.prod(1j * xi, eta) - (-1j) * p) < 1e-12 * mag      # antilinear in the first argument
    assert abs(la.prod(xi, 1j * eta) - 1j * p) < 1e-12 * mag         # linear in the second
    assert la.sqnorm(xi) == la.prod(xi, xi).real and la.prod(xi, xi).imag == 0.0
    assert la.norm2(xi) == pytest.approx(np.linalg.norm(xi.ravel()), rel=1e-14)
    assert abs(p) <= la.norm2(xi) * la.norm2(eta)                    # Cauchy-Schwarz
    # Eq 33 on a hand-made field
    z = np.array([[0.5 - 3.0j, 2.0 + 1.0j], [-2.5 + 0.1j, 0.0]])
    assert la.max_norm(z) == 3.0
    assert la.max_norm(np.array([1.0 - 7.0j])) == 7.0 and la.max_norm(np.array([-9.0 + 7.0j])) == 9.0


# ------------------------------------------------------------------------------------------ Eq 22-26
def test_linear_combinations_hand_values_and_identities():
    eta = np.array([1.0 + 2.0j, -1.0j])
    zeta = np.array([0.5, 2.0 - 1.0j])
    xi = np.array([3.0, 1.0 + 1.0j])
    assert np.array_equal(la.lc(2.0, eta, -1.0, zeta), np.array([1.5 + 4.0j, -2.0 - 1.0j]))            # Eq 22
    c1, c2 = 1.0j, 2.0
    assert np.array_equal(la.clc(c1, eta, c2, zeta), np.array([-2.0 + 1.0j + 1.0, 1.0 + 4.0 - 2.0j]))    # Eq 23
    assert np.array_equal(la.lc1(xi, c1, eta), np.array([3.0 - 2.0 + 1.0j, 1.0 + 1.0j + 1.0]))           # Eq 24
    assert np.array_equal(la.lc2(xi, c1, c2, eta), np.array([3.0j + 2.0 + 4.0j, 1.0j - 1.0 - 2.0j]))     # Eq 25
    assert np.array_equal(la.lc3(xi, c1, eta, c2, zeta), la.clc(c1, eta, c2, zeta) - xi)                 # Eq 26
    assert np.array_equal(la.lc2(xi, 1.0, c2, eta), la.lc1(xi, c2, eta))
    assert np.array_equal(la.lc_add_assign(xi, 2.0, eta, -1.0, zeta), xi + la.lc(2.0, eta, -1.0, zeta))
    assert np.array_equal(la.clc_add_assign(xi, c1, eta, c2, zeta), xi + la.clc(c1, eta, c2, zeta))


# ---------------------------------------------------------------------------------------------- CG
def test_cg_finite_termination_and_direct_solve():
    """CG on an n x n Hermitian positive-definite matrix with k distinct eigenvalues converges in k steps (textbook
    property); the solution matches numpy's direct solve."""
    rng = np.random.default_rng(5)
    n = 24
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n)))
    lam = np.repeat([0.5, 1.0, 3.0, 7.0], n // 4)
    A = (Q * lam) @ Q.conj().T
    b = rng.normal(size=n) + 1j * rng.normal(size=n)
    x, it, res, hist = la.cg(lambda v: A @ v, b, 1e-13, 100)
    assert it == 4
    assert np.linalg.norm(x - np.linalg.solve(A, b)) < 1e-12 * np.linalg.norm(x)
    assert res <= 1e-13 and len(hist) == it + 1


def test_cg_on_dense_Qsq_4x4x4x4(oracle):
    """BASELINE configs[0] lattice: CG with the C oracle's g5Dphi_sq equals the direct solve with the independently
    assembled dense (gamma5 D)^2 (oracle/dense.py); the recurrence residual equals the true residual."""
    cfg = synth.CONFIGS["C1"]
    U, (b,) = synth.make_inputs(cfg)
    R = oracle.represent_field(cfg.n_g, cfg.rep, U)
    m0 = 0.6                                     # heavier than the BASELINE mass: ~60 iterations instead of hundreds
    D = dense.dense_D(cfg.T, cfg.L, cfg.n_g, cfg.rep, U, m0, BC)
    G5 = np.kron(np.eye(cfg.volume), np.kron(dense.gamma5(), np.eye(cfg.d_R)))
    A = G5 @ D @ G5 @ D
    shape = b.shape
    apply_A = lambda v: oracle.g5Dphi_sq(cfg.T, cfg.L, cfg.d_R, m0, R, v.reshape(shape), BC)
    x, it, res, hist = la.cg(apply_A, b, 1e-12, 2000)
    assert 5 < it < 2000 and res <= 1e-12
    x_direct = np.linalg.solve(A, b.ravel())
    assert np.linalg.norm(x.ravel() - x_direct) < 1e-9 * np.linalg.norm(x_direct)
    true_res = np.linalg.norm(b.ravel() - A @ x.ravel()) / np.linalg.norm(b.ravel())
    assert true_res < 1e-10
    # the A-norm of the error decreases monotonically (defining property of CG); checked via the energy functional
    assert all(h >= 0 for h in hist)


def test_eo_preconditioned_solve_equals_dense_full_solve(oracle):
    """Eq 41-45 end to end on the 4^4 lattice: Q_hat = gamma_5 D_hat is Hermitian and equals the dense block
    expression; solving D_m x = b through the Schur complement -- D_hat x_e = (4+m) b_e - D_eo b_o by CG on Q_hat^2,
    x_o = (b_o - D_oe x_e)/(4+m) -- reproduces numpy's direct solve of the independently assembled dense D_m."""
    cfg = synth.CONFIGS["C1"]
    T, L, d = cfg.T, cfg.L, cfg.d_R
    U, (b, phi) = synth.make_inputs(cfg, 2)
    R = oracle.represent_field(cfg.n_g, cfg.rep, U)
    m0, a = 0.6, 4.6
    ev, od = synth.parity_sites(T, L, 0), synth.parity_sites(T, L, 1)
    D = dense.dense_D(T, L, cfg.n_g, cfg.rep, U, m0, BC)
    e, o = dense.parity_index(T, L, d, 0), dense.parity_index(T, L, d, 1)
    G5e = np.kron(np.eye(cfg.volume // 2), np.kron(dense.gamma5(), np.eye(d)))
    Qhat = G5e @ (a * a * np.eye(len(e)) - D[np.ix_(e, o)] @ D[np.ix_(o, e)])
    assert np.linalg.norm(Qhat - Qhat.conj().T) < 1e-12 * np.linalg.norm(Qhat)               # Hermitian (Eq 45)
    got = oracle.g5Dphi_hat(T, L, d, m0, R, phi[ev], BC)
    assert np.linalg.norm(got.ravel() - Qhat @ phi[ev].ravel()) < 1e-13 * np.linalg.norm(got)
    got2 = oracle.g5Dphi_hat_sq(T, L, d, m0, R, phi[ev], BC)
    assert np.linalg.norm(got2.ravel() - Qhat @ (Qhat @ phi[ev].ravel())) < 1e-13 * np.linalg.norm(got2)
    # the solve
    c = a * b[ev] - oracle.Dphi_eo(T, L, d, R, b[od], BC)
    rhs = oracle.g5Dphi_hat(T, L, d, m0, R, oracle.g5(c), BC)
    x_e, it, res, _ = la.cg(lambda v: oracle.g5Dphi_hat_sq(T, L, d, m0, R, v, BC), rhs, 1e-13, 2000)
    x_o = (b[od] - oracle.Dphi_oe(T, L, d, R, x_e, BC)) / a
    x = np.zeros_like(b)
    x[ev], x[od] = x_e, x_o
    x_direct = np.linalg.solve(D, b.ravel())
    assert np.linalg.norm(x.ravel() - x_direct) < 1e-9 * np.linalg.norm(x_direct)
    # even-odd preconditioning pays: fewer iterations than CG on the full Q^2 for the same residual
    _, it_full, _, _ = la.cg(lambda v: oracle.g5Dphi_sq(T, L, d, m0, R, v, BC), b, 1e-13, 2000)
    assert it < it_full


def test_cg_zero_rhs_and_initial_guess():
    A = np.diag([1.0, 2.0, 3.0]).astype(complex)
    x, it, res, _ = la.cg(lambda v: A @ v, np.zeros(3, complex), 1e-10, 10)
    assert it == 0 and np.all(x == 0)
    b = np.array([1.0, 1.0j, -2.0])
    x, it, res, _ = la.cg(lambda v: A @ v, b, 1e-14, 10, x0=np.linalg.solve(A, b))
    assert it == 0


def test_multishift_cg_against_direct_solves(oracle):
    """Every shifted solution of the multi-shift CG equals the direct solve of (A + sigma_k) x = b -- on a random
    Hermitian positive-definite matrix and on the dense (gamma_5 D)^2 of the 4^4 lattice -- and the zero shift
    reproduces plain CG iterate for iterate."""
    rng = np.random.default_rng(8)
    n = 40
    Q, _ = np.linalg.qr(rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n)))
    A = (Q * rng.uniform(0.2, 5.0, size=n)) @ Q.conj().T
    b = rng.normal(size=n) + 1j * rng.normal(size=n)
    shifts = [0.0, 0.05, 0.7, 3.0]
    xs, it, res = la.cg_mshift(lambda v: A @ v, b, shifts, 1e-13, 500)
    assert res <= 1e-13
    for sg, x in zip(shifts, xs):
        ref = np.linalg.solve(A + sg * np.eye(n), b)
        assert np.linalg.norm(x - ref) < 1e-11 * np.linalg.norm(ref), sg
    x0, it0, _, _ = la.cg(lambda v: A @ v, b, 1e-13, 500)
    assert it0 == it and np.linalg.norm(xs[0] - x0) < 1e-12 * np.linalg.norm(x0)
    # the lattice operator
    cfg = synth.CONFIGS["C1"]
    U, (bl,) = synth.make_inputs(cfg)
    R = oracle.represent_field(cfg.n_g, cfg.rep, U)
    m0 = 0.6
    D = dense.dense_D(cfg.T, cfg.L, cfg.n_g, cfg.rep, U, m0, BC)
    G5 = np.kron(np.eye(cfg.volume), np.kron(dense.gamma5(), np.eye(cfg.d_R)))
    Qsq = G5 @ D @ G5 @ D
    shape = bl.shape
    shifts = [0.01, 0.3, 2.0]
    xs, it, res = la.cg_mshift(lambda v: oracle.g5Dphi_sq(cfg.T, cfg.L, cfg.d_R, m0, R, v.reshape(shape), BC), bl, shifts, 1e-12, 3000)
    assert res <= 1e-12
    for sg, x in zip(shifts, xs):
        ref = np.linalg.solve(Qsq + sg * np.eye(Qsq.shape[0]), bl.ravel())
        assert np.linalg.norm(x.ravel() - ref) < 1e-9 * np.linalg.norm(ref), sg


def test_bicgstab_against_direct_solves(oracle):
    """BiCGstab on a random non-Hermitian matrix and on the dense D_m / D_hat of the 4^4 lattice equals numpy's direct
    solve; it needs fewer operator applications than CG on the normal equations (the paper's remark, L730)."""
    rng = np.random.default_rng(12)
    n = 50
    A = 3.0 * np.eye(n) + 0.3 * (rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n)))
    b = rng.normal(size=n) + 1j * rng.normal(size=n)
    x, it, res = la.bicgstab(lambda v: A @ v, b, 1e-13, 500)
    assert res <= 1e-13 and np.linalg.norm(x - np.linalg.solve(A, b)) < 1e-11 * np.linalg.norm(x)
    cfg = synth.CONFIGS["C1"]
    U, (bl,) = synth.make_inputs(cfg)
    R = oracle.represent_field(cfg.n_g, cfg.rep, U)
    T, L, d, m0 = cfg.T, cfg.L, cfg.d_R, 0.3
    D = dense.dense_D(T, L, cfg.n_g, cfg.rep, U, m0, BC)
    shape = bl.shape
    x, it, res = la.bicgstab(lambda v: oracle.Dphi(T, L, d, m0, R, v.reshape(shape), BC), bl, 1e-12, 2000)
    ref = np.linalg.solve(D, bl.ravel())
    assert res <= 1e-12 and np.linalg.norm(x.ravel() - ref) < 1e-9 * np.linalg.norm(ref)
    _, it_cg, _, _ = la.cg(lambda v: oracle.g5Dphi_sq(T, L, d, m0, R, v.reshape(shape), BC), bl, 1e-12, 2000)
    assert 2 * it < 2 * it_cg                      # operator applications: 2 per BiCGstab iteration, 2 per CG iteration on Q^2
    # even-odd preconditioned operator
    ev = synth.parity_sites(T, L, 0)
    e, o = dense.parity_index(T, L, d, 0), dense.parity_index(T, L, d, 1)
    a = 4.0 + m0
    Dhat = a * a * np.eye(len(e)) - D[np.ix_(e, o)] @ D[np.ix_(o, e)]
    xe, it, res = la.bicgstab(lambda v: oracle.Dphi_hat(T, L, d, m0, R, v, BC), bl[ev], 1e-12, 2000)
    ref = np.linalg.solve(Dhat, bl[ev].ravel())
    assert np.linalg.norm(xe.ravel() - ref) < 1e-9 * np.linalg.norm(ref)
