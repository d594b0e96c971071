"""Oracle of the fermion force of the hopping term.  TEST INFRASTRUCTURE ONLY: imported by tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline leg, never by the product path; shares no code with the CUDA library.

Follows PAPER.md L273-278 (Sect. 2.5) step by step, in the paper's notation, plain numpy in fp64:

  eta = (Q_m^2)^-1 psi,  xi = Q_m eta                                                          (L273)
  T_mu(x) = tr_spin[ gamma_5 (1 - gamma_mu) { eta(x+mu) (x) xi^dagger(x) + xi(x+mu) (x) eta^dagger(x) } ]     (Eq 20)
  F^a_mu(x) = -(1/T_FUND) Re tr[ i T_R^a U^R_mu(x) T_mu(x) ]                                   (Eq 21, reading A32)

Readings:
  A32  Eq 21 is printed as "F^a_F(x) = -(1/T_FUND) Re tr[U^R_mu(x) T_mu(x)]": the index a does not appear on the right-hand side
       and mu not on the left.  By analogy with Eq 19 (Re tr[i T_R^a U V^dagger]) the generator i T_R^a of the REPRESENTED algebra is
       what the extraction garbled; with it the formula is exactly -(1/T_FUND) dS_f/d omega^a for S_f = psi^dagger (Q_m^2)^-1 psi and
       U_mu(x) -> exp(i omega^a T^a) U_mu(x) (Eq 17), which is what Hamilton's equations with H_pi of Eq 15 require (Eq 18).  That
       identity is the pin (tests/test_oracle_force.py: finite differences of the action on a dense 2^4 / 4x2^3 operator).
  A33  T_R^a = -i dR(exp(i omega T^a))/d omega at omega = 0 (Eq 7: U^R = exp(i omega^a T_R^a)).  R is a polynomial of degree <= 2 in
       (U, U^dagger) (A17), so the derivative is taken EXACTLY as the odd part [R(1 + iT^a) - R(1 - iT^a)] / (2i).
  A34  boundary conditions: psi(x + L_mu) = bc_mu psi(x) (Eq 58-61) applies to eta and xi alike: the neighbour reached across
       the edge carries bc_mu.
The outer product a (x) b^dagger is the matrix (a b^dagger)_{(beta i),(alpha j)} = a_{beta i} conj(b_{alpha j}) in spin (x) colour; the spin
trace with Gamma leaves the colour matrix T_ij = sum_{alpha beta} Gamma_{alpha beta} a_{beta i} conj(b_{alpha j}).
"""
from __future__ import annotations

import numpy as np

from . import oracle as orc

T_FUND = 0.5   # Tbl 1 (L213-220)


def rep_generators(n_g: int, rep: int) -> np.ndarray:
    """T_R^a, a = 0..N^2-2, as [N^2-1, d_R, d_R] complex (reading A33)."""
    Tf = orc.generators(n_g)
    one = np.eye(n_g, dtype=np.complex128)
    return np.array([(orc.rep_matrix(n_g, rep, one + 1j * t) - orc.rep_matrix(n_g, rep, one - 1j * t)) / 2j for t in Tf])


def shift_forward(field: np.ndarray, mu: int, T: int, L: int, bc) -> np.ndarray:
    """field(x + mu) with the boundary factor of Eq 61 on the sites whose neighbour lies across the edge.  field: [V, ...]."""
    ext = (T, L, L, L)
    f = field.reshape(ext + field.shape[1:])
    out = np.roll(f, -1, axis=mu).copy()
    edge = [slice(None)] * 4
    edge[mu] = ext[mu] - 1
    out[tuple(edge)] *= bc[mu]
    return out.reshape(field.shape)


def traced_operator(T: int, L: int, mu: int, eta: np.ndarray, xi: np.ndarray, bc) -> np.ndarray:
    """T_mu(x) of Eq 20 as [V, d_R, d_R]."""
    G = orc.gamma()
    Gam = orc.gamma5() @ (np.eye(4) - G[mu])
    eta_f, xi_f = shift_forward(eta, mu, T, L, bc), shift_forward(xi, mu, T, L, bc)
    return (np.einsum("ab,xbi,xaj->xij", Gam, eta_f, np.conj(xi)) + np.einsum("ab,xbi,xaj->xij", Gam, xi_f, np.conj(eta)))


def force_hopping(T: int, L: int, n_g: int, rep: int, Rlinks: np.ndarray, eta: np.ndarray, xi: np.ndarray,
                  bc=orc.DEFAULT_BC) -> np.ndarray:
    """F^a_mu(x) of Eq 21 as [V, 4, N^2-1] real.  Rlinks: represented links [V,4,d_R,d_R] (oracle.represent_field)."""
    TR = rep_generators(n_g, rep)
    V = T * L ** 3
    F = np.empty((V, 4, TR.shape[0]))
    for mu in range(4):
        Tm = traced_operator(T, L, mu, eta, xi, bc)
        UT = np.einsum("xjk,xki->xji", Rlinks[:, mu], Tm)                 # U^R_mu(x) T_mu(x)
        F[:, mu, :] = -(1.0 / T_FUND) * np.real(1j * np.einsum("aij,xji->xa", TR, UT))
    return F
