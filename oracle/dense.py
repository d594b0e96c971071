"""Second, even more naive oracle for tiny lattices: the dense matrix of D_m.  TEST INFRASTRUCTURE ONLY.

Independent of hirep_oracle.c (different language, assembled entry-block by entry-block with numpy Kronecker
products), written from the same passages of PAPER.md:

  gamma matrices   Eq 1-3 (L171-182)                      D_m        Eq 8 (L207), a = 1
  even/odd blocks  Eq 41 (L795), parity (t+x+y+z)%2 L793  D_hat      Eq 43/44 (L803-808)
  boundary factor  Eq 58/61 (L930-938)                    reps       Eq 7 + readings A10/A11 of DESIGN.md

Row/column index of the matrix: (ix*4 + spin)*d_R + colour with ix the canonical site index.
"""
from __future__ import annotations

import itertools

import numpy as np

FUND, ADJ, SYM, ASY = 0, 1, 2, 3


def pauli():
    return [np.array([[0, 1], [1, 0]], dtype=complex),
            np.array([[0, -1j], [1j, 0]], dtype=complex),
            np.array([[1, 0], [0, -1]], dtype=complex)]


def gammas():
    """gamma_mu = [[0, e_mu], [e_mu^dagger, 0]], e_0 = -1, e_k = -i sigma_k (Eq 2-3)."""
    e = [-np.eye(2, dtype=complex)] + [-1j * s for s in pauli()]
    z = np.zeros((2, 2), dtype=complex)
    return [np.block([[z, em], [em.conj().T, z]]) for em in e]


def gamma5():
    g = gammas()
    return g[0] @ g[1] @ g[2] @ g[3]


def su_generators(n):
    """Generalised Gell-Mann matrices / 2 in the order of reading A10."""
    gens = []
    for j in range(1, n):
        for i in range(j):
            s = np.zeros((n, n), dtype=complex); s[i, j] = s[j, i] = 0.5
            a = np.zeros((n, n), dtype=complex); a[i, j] = -0.5j; a[j, i] = 0.5j
            gens += [s, a]
        d = np.zeros((n, n), dtype=complex)
        d[np.arange(j), np.arange(j)] = 1.0
        d[j, j] = -j
        gens.append(d / np.sqrt(2.0 * j * (j + 1)))
    return gens


def tensor_basis(n, rep):
    out = []
    for i, j in itertools.combinations_with_replacement(range(n), 2):
        e = np.zeros((n, n))
        if rep == ASY:
            if i == j:
                continue
            e[i, j], e[j, i] = 1 / np.sqrt(2), -1 / np.sqrt(2)
        else:
            if i == j:
                e[i, i] = 1.0
            else:
                e[i, j] = e[j, i] = 1 / np.sqrt(2)
        out.append(e)
    return out


def rep_matrix(n, rep, U):
    U = np.asarray(U, dtype=complex)
    if rep == FUND:
        return U.copy()
    if rep == ADJ:
        T = su_generators(n)
        return np.array([[2 * np.trace(ta @ U @ tb @ U.conj().T).real for tb in T] for ta in T], dtype=complex)
    B = tensor_basis(n, rep)
    return np.array([[np.trace(ea.T @ U @ eb @ U.T) for eb in B] for ea in B], dtype=complex)


def coords(T, L):
    return [(t, x, y, z) for t in range(T) for x in range(L) for y in range(L) for z in range(L)]


def dense_D(T, L, n_g, rep, links, m0, bc=(-1, 1, 1, 1)):
    """Dense D_m (Eq 8).  links: canonical fundamental [V,4,N,N]."""
    ext = (T, L, L, L)
    g = gammas()
    one = np.eye(4, dtype=complex)
    cs = coords(T, L)
    index = {c: k for k, c in enumerate(cs)}
    R = [[rep_matrix(n_g, rep, links[k, mu]) for mu in range(4)] for k in range(len(cs))]
    d = R[0][0].shape[0]
    n = 4 * d
    D = np.zeros((len(cs) * n, len(cs) * n), dtype=complex)
    for k, c in enumerate(cs):
        D[k * n:(k + 1) * n, k * n:(k + 1) * n] += (4.0 + m0) * np.eye(n)
        for mu in range(4):
            cf = list(c); cf[mu] += 1; sf = 1.0
            if cf[mu] == ext[mu]:
                cf[mu] = 0; sf = bc[mu]
            cb = list(c); cb[mu] -= 1; sb = 1.0
            if cb[mu] < 0:
                cb[mu] = ext[mu] - 1; sb = bc[mu]
            kf, kb = index[tuple(cf)], index[tuple(cb)]
            D[k * n:(k + 1) * n, kf * n:(kf + 1) * n] += -0.5 * sf * np.kron(one - g[mu], R[k][mu])
            D[k * n:(k + 1) * n, kb * n:(kb + 1) * n] += -0.5 * sb * np.kron(one + g[mu], R[kb][mu].conj().T)
    return D


def parity_index(T, L, d, parity):
    """Matrix row indices belonging to the sites of the given parity, in increasing site order."""
    n = 4 * d
    rows = []
    for k, c in enumerate(coords(T, L)):
        if sum(c) % 2 == parity:
            rows.extend(range(k * n, (k + 1) * n))
    return np.array(rows)
