"""Pins for the oracle's gamma matrices and representation maps (CPU only).

Every check is against something the paper or the mathematics fixes, not against the oracle's own formula:
Clifford algebra from Eq 1-3; Table 1 values (tests/golden/table1_reps.txt); group homomorphism, unitarity,
the textbook SO(3) rotation for the SU(2) adjoint, Cauchy-Binet 2x2 minors for 2AS, permanents for SYM.
"""
import os

import numpy as np
import pytest

from harness import synth

FUND, ADJ, SYM, ASY = 0, 1, 2, 3
REP_ID = {"FUND": FUND, "ADJ": ADJ, "SYM": SYM, "2AS": ASY}
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "table1_reps.txt")


def golden_rows():
    rows = []
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        n, rep, d, tr, c2 = line.split()
        rows.append((int(n), REP_ID[rep], int(d), float(tr), float(c2)))
    return rows


def rand_su(n, k, seed):
    return synth.haar_sun(np.random.default_rng(seed), k, n)


# ------------------------------------------------------------------------------------------ gamma
def test_gamma_clifford_algebra(oracle):
    g = oracle.gamma()
    for mu in range(4):
        assert np.allclose(g[mu], g[mu].conj().T)                      # Hermitian
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * (mu == nu) * np.eye(4), atol=1e-15)


def test_gamma_explicit_entries_from_eq_2_3(oracle):
    # Eq 2-3 typed out by hand: gamma_0 = [[0,-1],[-1,0]], gamma_k = [[0,-i sigma_k],[i sigma_k,0]]
    g = oracle.gamma()
    z, one = np.zeros((2, 2)), np.eye(2)
    s1 = np.array([[0, 1], [1, 0]]); s2 = np.array([[0, -1j], [1j, 0]]); s3 = np.array([[1, 0], [0, -1]])
    assert np.array_equal(g[0], np.block([[z, -one], [-one, z]]))
    for k, s in enumerate((s1, s2, s3), start=1):
        assert np.array_equal(g[k], np.block([[z, -1j * s], [1j * s, z]]))


def test_gamma5_is_diag_and_anticommutes(oracle):
    g, g5 = oracle.gamma(), oracle.gamma5()
    assert np.allclose(g5, np.diag([1, 1, -1, -1]), atol=1e-15)         # reading A1
    assert np.allclose(g5 @ g5, np.eye(4))
    for mu in range(4):
        assert np.allclose(g5 @ g[mu] + g[mu] @ g5, 0, atol=1e-15)


def test_half_spinor_rank(oracle):
    # (1 -+ gamma_mu) are rank-2 projectors times 2: the fact the GPU path's spin projection rests on
    g = oracle.gamma()
    for mu in range(4):
        for sgn in (-1, 1):
            P = np.eye(4) + sgn * g[mu]
            assert np.linalg.matrix_rank(P) == 2
            assert np.allclose(P @ P, 2 * P)


# ---------------------------------------------------------------------------------- generators
@pytest.mark.parametrize("n", [2, 3, 4, 6])
def test_generators_normalisation_and_textbook(oracle, n):
    T = oracle.generators(n)
    assert T.shape == (n * n - 1, n, n)
    for a in range(len(T)):
        assert np.allclose(T[a], T[a].conj().T) and abs(np.trace(T[a])) < 1e-15
        for b in range(len(T)):
            assert abs(np.trace(T[a] @ T[b]) - 0.5 * (a == b)) < 1e-14   # T_FUND = 1/2 (Tbl 1)
    if n == 2:
        s = [np.array([[0, 1], [1, 0]]), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]])]
        for a in range(3):
            assert np.allclose(T[a], s[a] / 2)
    if n == 3:   # Gell-Mann lambda_3 and lambda_8
        assert np.allclose(T[2], np.diag([1, -1, 0]) / 2)
        assert np.allclose(T[7], np.diag([1, 1, -2]) / (2 * np.sqrt(3)))


# ------------------------------------------------------------------------------ representations
@pytest.mark.parametrize("n,rep,d,t_r,c2", golden_rows())
def test_table1_dimension_trace_norm_casimir(oracle, n, rep, d, t_r, c2):
    """d_R, T_R, C_2(R) of Table 1 from T_R^a = -i dR/d omega^a at the identity (Eq 7)."""
    assert oracle.rep_dim(n, rep) == d
    Tf = oracle.generators(n)
    eps = 1e-4
    TR = []
    for a in range(len(Tf)):
        w, v = np.linalg.eigh(Tf[a])
        up = (v * np.exp(1j * eps * w)) @ v.conj().T
        um = (v * np.exp(-1j * eps * w)) @ v.conj().T
        TR.append((oracle.rep_matrix(n, rep, up) - oracle.rep_matrix(n, rep, um)) / (2j * eps))
    TR = np.array(TR)
    assert TR.shape[1:] == (d, d)
    # only a subset of (a,b) pairs for the big ones
    idx = range(len(TR)) if len(TR) <= 15 else [0, 1, 7, 20, 34]
    for a in idx:
        assert np.allclose(TR[a], TR[a].conj().T, atol=1e-7)
        for b in idx:
            assert abs(np.trace(TR[a] @ TR[b]) - t_r * (a == b)) < 1e-6
    cas = sum(t @ t for t in TR)
    assert np.allclose(cas, c2 * np.eye(d), atol=1e-6)


@pytest.mark.parametrize("n,rep", [(2, FUND), (2, ADJ), (2, SYM), (3, FUND), (3, ADJ), (3, SYM), (3, ASY),
                                   (4, ASY), (4, SYM), (4, ADJ), (6, ADJ), (6, ASY)])
def test_homomorphism_unitarity_identity(oracle, n, rep):
    U, V = rand_su(n, 2, seed=10 * n + rep)
    RU, RV, RUV = (oracle.rep_matrix(n, rep, m) for m in (U, V, U @ V))
    d = oracle.rep_dim(n, rep)
    assert np.allclose(RUV, RU @ RV, atol=1e-12)                         # R(UV) = R(U) R(V)
    assert np.allclose(RU @ RU.conj().T, np.eye(d), atol=1e-12)          # unitary
    assert np.allclose(oracle.rep_matrix(n, rep, np.eye(n)), np.eye(d), atol=1e-14)
    assert np.allclose(oracle.rep_matrix(n, rep, U.conj().T), RU.conj().T, atol=1e-12)
    assert abs(np.linalg.det(RU) - 1) < 1e-10
    if rep == ADJ:
        assert np.all(RU.imag == 0)                                      # real representation (Tbl 2, A9)
        assert np.allclose(RU @ RU.T, np.eye(d), atol=1e-12)


def test_su2_adjoint_is_textbook_rotation(oracle):
    # U = a0 + i a.sigma  ->  R_ab = (a0^2-|a|^2) d_ab + 2 a_a a_b + 2 a0 eps_abc a_c
    rng = np.random.default_rng(5)
    eps = np.zeros((3, 3, 3))
    eps[0, 1, 2] = eps[1, 2, 0] = eps[2, 0, 1] = 1
    eps[0, 2, 1] = eps[2, 1, 0] = eps[1, 0, 2] = -1
    for _ in range(4):
        q = rng.standard_normal(4); q /= np.linalg.norm(q)
        a0, a = q[0], q[1:]
        U = np.array([[a0 + 1j * a[2], a[1] + 1j * a[0]], [-a[1] + 1j * a[0], a0 - 1j * a[2]]])
        R = oracle.rep_matrix(2, ADJ, U).real
        ref = (a0 * a0 - a @ a) * np.eye(3) + 2 * np.outer(a, a) + 2 * a0 * np.einsum("abc,c->ab", eps, a)
        assert np.allclose(R, ref, atol=1e-14)


@pytest.mark.parametrize("n", [2, 3, 4, 6])
def test_2as_is_2x2_minors(oracle, n):
    U = rand_su(n, 1, seed=77 + n)[0]
    R = oracle.rep_matrix(n, ASY, U)
    pairs = [(i, j) for i in range(n) for j in range(i + 1, n)]
    for A, (i, j) in enumerate(pairs):
        for B, (k, l) in enumerate(pairs):
            assert abs(R[A, B] - (U[i, k] * U[j, l] - U[i, l] * U[j, k])) < 1e-14


def test_su2_2as_is_the_trivial_representation(oracle):
    """SU(2) 2AS: d_R = N(N-1)/2 = 1 (Tbl 1, L213-220) and R(U) = det U = 1 -- the singlet.  With unit represented links the
    operator is the free one, whatever the gauge field."""
    for U in rand_su(2, 4, seed=5):
        R = oracle.rep_matrix(2, ASY, U)
        assert R.shape == (1, 1) and abs(R[0, 0] - 1.0) < 1e-14


@pytest.mark.parametrize("n", [2, 3, 4])
def test_sym_is_symmetrised_products(oracle, n):
    """R_(ij),(kl) = c_A c_B * sum over the distinct orderings (p,q) of (i,j) and (r,s) of (k,l) of U_pr U_qs,
    c = 1 for a diagonal pair, 1/sqrt2 otherwise (permanent-like closed form of Psi -> U Psi U^T)."""
    U = rand_su(n, 1, seed=99 + n)[0]
    R = oracle.rep_matrix(n, SYM, U)
    pairs = [(i, j) for i in range(n) for j in range(i, n)]

    def orderings(i, j):
        return [(i, i)] if i == j else [(i, j), (j, i)]

    for A, (i, j) in enumerate(pairs):
        for B, (k, l) in enumerate(pairs):
            ca = 1.0 if i == j else np.sqrt(0.5)
            cb = 1.0 if k == l else np.sqrt(0.5)
            ref = ca * cb * sum(U[p, r] * U[q, s] for (p, q) in orderings(i, j) for (r, s) in orderings(k, l))
            assert abs(R[A, B] - ref) < 1e-14


@pytest.mark.parametrize("n,rep", [(3, SYM), (4, ASY), (3, ASY)])
def test_two_index_rep_is_tensor_action(oracle, n, rep):
    """R is the matrix of Psi -> U Psi U^T on (anti)symmetric N x N tensors (reading A11), checked by acting
    on a random tensor rather than entry by entry."""
    U = rand_su(n, 1, seed=3 * n + rep)[0]
    R = oracle.rep_matrix(n, rep, U)
    B = oracle.tensor_basis(n, rep)
    for a in range(len(B)):                      # orthonormal basis of the right symmetry
        assert np.allclose(B[a].T, B[a] if rep == SYM else -B[a])
        for b in range(len(B)):
            assert abs(np.sum(B[a] * B[b]) - (a == b)) < 1e-15
    rng = np.random.default_rng(1)
    c = rng.standard_normal(len(B)) + 1j * rng.standard_normal(len(B))
    Psi = np.einsum("a,aij->ij", c, B)
    Psi2 = U @ Psi @ U.T
    c2 = np.einsum("aij,ij->a", B, Psi2)
    assert np.allclose(R @ c, c2, atol=1e-13)


def test_represent_field_matches_single(oracle):
    U = rand_su(3, 6, seed=4).reshape(3, 2, 3, 3)
    Rf = oracle.represent_field(3, SYM, U)
    assert Rf.shape == (3, 2, 6, 6)
    assert np.array_equal(Rf[1, 1], oracle.rep_matrix(3, SYM, U[1, 1]))
