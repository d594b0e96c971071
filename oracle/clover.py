"""Clover term of the Wilson-Dirac operator -- TEST ORACLE (plain numpy, fp64), not part of the product path.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs may import this module.

What it follows:
  * Eq 47 (L859):  D_ee,m + D_oo,m = (4+m) + c_sw (i/4) sum_{mu,nu} sigma_{mu nu} F_{mu nu}
  * Eq 48 (L864):  C_{mu nu}(x) = sum of the four plaquettes that touch x in the (mu,nu) plane
  * Eq 49 (L869):  F_{mu nu} = (1/8) (C_{mu nu} - C_{mu nu}^dagger)
  * Eq 13 (L243):  P_{mu nu}(x) = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dagger U_nu(x)^dagger
  * Eq 3  (L182):  gamma_mu = [[0, e_mu], [e_mu^dagger, 0]]

Readings (A26-A28):
  A26  Eq 48 as printed adds plaquettes based at four different sites (not gauge covariant, and two of the four run
       clockwise); it is read as the standard clover: the four plaquette loops in the (mu,nu) plane that pass
       through x, each written as a closed path that starts and ends at x, all with the orientation of P_{mu nu}(x).
  A27  Eq 49's second equality repeats Eq 48 and contradicts the first; the first is taken:
       F = (C - C^dagger)/8, anti-Hermitian.
  A28  sigma_{mu nu} is not defined in the paper; sigma_{mu nu} = (i/2) [gamma_mu, gamma_nu] (Hermitian) is taken, the
       sum in Eq 47 runs over all ordered pairs (mu,nu), so the term is Hermitian and commutes with gamma_5.
  The links are the represented links R(U_mu(x)); boundary signs +-1 cancel in every closed plaquette loop.

Pins (tests/test_oracle_clover.py): sigma matrices typed from hand algebra, constant abelian background (closed form),
random abelian background against a brute-force sum over the four base points Eq 48 prints, gauge covariance, pure
gauge = 0, Hermiticity / tracelessness / chirality blocks, gamma_5-Hermiticity of the full operator, c_sw = 0.
Parity unpinned in one respect: the overall sign convention of the c_sw term (A28) -- the paper prints nothing that
fixes sigma_{mu nu} beyond the name.

Layout: Rlinks [V, 4, d, d] complex, V = T L^3 canonical sites ((t*L + x)*L + y)*L + z; spinors [V, 4, d].
"""
from __future__ import annotations

import numpy as np

from . import dense


def _field(T, L, Rlinks):
    d = Rlinks.shape[-1]
    return np.asarray(Rlinks, dtype=np.complex128).reshape(T, L, L, L, 4, d, d)


def _shift(A, mu, s):
    """A'(x) = A(x + s mu), periodic."""
    return np.roll(A, -s, axis=mu)


def _dag(A):
    return np.conj(np.swapaxes(A, -1, -2))


def clover_leaves(T, L, Rlinks, mu, nu):
    """C_{mu nu}(x) (Eq 48, reading A26) as an array [T,L,L,L,d,d]."""
    U = _field(T, L, Rlinks)
    Um, Un = U[..., mu, :, :], U[..., nu, :, :]
    mm = np.matmul
    # leaf 1: x -> x+mu -> x+mu+nu -> x+nu -> x
    l1 = mm(mm(Um, _shift(Un, mu, 1)), mm(_dag(_shift(Um, nu, 1)), _dag(Un)))
    # leaf 2: x -> x+nu -> x-mu+nu -> x-mu -> x
    Um_m = _shift(Um, mu, -1)                      # U_mu(x-mu)
    l2 = mm(mm(Un, _dag(_shift(Um_m, nu, 1))), mm(_dag(_shift(Un, mu, -1)), Um_m))
    # leaf 3: x -> x-mu -> x-mu-nu -> x-nu -> x
    Un_n = _shift(Un, nu, -1)                      # U_nu(x-nu)
    l3 = mm(mm(_dag(Um_m), _dag(_shift(Un_n, mu, -1))), mm(_shift(Um_m, nu, -1), Un_n))
    # leaf 4: x -> x-nu -> x+mu-nu -> x+mu -> x
    l4 = mm(mm(_dag(Un_n), _shift(Um, nu, -1)), mm(_shift(Un_n, mu, 1), _dag(Um)))
    return l1 + l2 + l3 + l4


def field_strength(T, L, Rlinks, mu, nu):
    """F_{mu nu}(x) = (C - C^dagger)/8 (Eq 49, reading A27), [T,L,L,L,d,d]."""
    C = clover_leaves(T, L, Rlinks, mu, nu)
    return (C - _dag(C)) / 8.0


def sigma(mu, nu):
    """sigma_{mu nu} = (i/2)[gamma_mu, gamma_nu] (reading A28), 4x4."""
    g = dense.gammas()
    return 0.5j * (g[mu] @ g[nu] - g[nu] @ g[mu])


def clover_term(T, L, Rlinks):
    """(i/4) sum_{mu,nu} sigma_{mu nu} F_{mu nu}(x) as [V, 4, d, 4, d] (spin, colour, spin', colour')."""
    d = Rlinks.shape[-1]
    V = T * L ** 3
    A = np.zeros((V, 4, d, 4, d), dtype=np.complex128)
    for mu in range(4):
        for nu in range(4):
            if mu == nu:
                continue
            F = field_strength(T, L, Rlinks, mu, nu).reshape(V, d, d)
            A += 0.25j * np.einsum("st,xab->xsatb", sigma(mu, nu), F)
    return A


def Cphi(T, L, m0, csw, Rlinks, psi):
    """((4+m) + c_sw (i/4) sum sigma F) psi (Eq 47): the diagonal blocks D_ee,m + D_oo,m."""
    A = clover_term(T, L, Rlinks)
    psi = np.asarray(psi, dtype=np.complex128)
    return (4.0 + m0) * psi + csw * np.einsum("xsatb,xtb->xsa", A, psi)


def chiral_blocks(T, L, Rlinks):
    """The two (2d x 2d) Hermitian blocks of the clover term (spin 0,1 and spin 2,3), [V, 2, 2d, 2d]; the
    off-diagonal chirality blocks vanish because sigma_{mu nu} commutes with gamma_5 (checked in the tests)."""
    A = clover_term(T, L, Rlinks)
    V, _, d = A.shape[:3]
    out = np.zeros((V, 2, 2 * d, 2 * d), dtype=np.complex128)
    for c in range(2):
        out[:, c] = A[:, 2 * c:2 * c + 2, :, 2 * c:2 * c + 2, :].reshape(V, 2 * d, 2 * d)
    return out


def Dphi_clover(T, L, m0, csw, Rlinks, psi, bc):
    """Eq 8 with the diagonal term of Eq 47: hopping term (the C oracle's field loop) + Cphi."""
    from . import oracle as _o
    d = Rlinks.shape[-1]
    return _o.hop_field(T, L, d, Rlinks, psi, bc) + Cphi(T, L, m0, csw, Rlinks, psi)


def _parity_sites(T, L, parity):
    t, x, y, z = np.meshgrid(np.arange(T), np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    return np.nonzero(((t + x + y + z) % 2).reshape(-1) == parity)[0]


def diag_blocks(T, L, m0, csw, Rlinks):
    """The site-diagonal blocks of D_ee,m / D_oo,m (Eq 47) per chirality: (4+m) 1 + c_sw A_c, [V, 2, 2d, 2d]."""
    B = csw * chiral_blocks(T, L, Rlinks)
    n = B.shape[-1]
    return B + (4.0 + m0) * np.eye(n)


def Cphi_inv(T, L, m0, csw, Rlinks, psi, sites=None):
    """((4+m) + c_sw (i/4) sum sigma F)^{-1} psi, site by site (numpy's dense inverse of each 2d x 2d block);
    psi [n, 4, d] on the canonical sites `sites` (all sites if None)."""
    M = diag_blocks(T, L, m0, csw, Rlinks)
    if sites is not None:
        M = M[sites]
    psi = np.asarray(psi, dtype=np.complex128)
    n, _, d = psi.shape
    v = psi.reshape(n, 2, 2 * d)
    return np.einsum("xcij,xcj->xci", np.linalg.inv(M), v).reshape(n, 4, d)


def Dphi_clover_hat(T, L, m0, csw, Rlinks, psi_even, bc):
    """Eq 43 with the clover diagonal blocks of Eq 47: D_ee psi_e - D_eo D_oo^{-1} D_oe psi_e (even sites)."""
    from . import oracle as _o
    d = Rlinks.shape[-1]
    ev, od = _parity_sites(T, L, 0), _parity_sites(T, L, 1)
    psi_even = np.asarray(psi_even, dtype=np.complex128)
    M = diag_blocks(T, L, m0, csw, Rlinks)
    dee = np.einsum("xcij,xcj->xci", M[ev], psi_even.reshape(len(ev), 2, 2 * d)).reshape(len(ev), 4, d)
    t = _o.Dphi_oe(T, L, d, Rlinks, psi_even, bc)
    u = Cphi_inv(T, L, m0, csw, Rlinks, t, sites=od)
    return dee - _o.Dphi_eo(T, L, d, Rlinks, u, bc)


def exp_blocks(T, L, m0, csw, Rlinks, inverse=False):
    """Exponential clover (Eq 50): the site-diagonal blocks (4+m0) exp(c_sw/(4+m0) A_c), [V, 2, 2d, 2d], through the
    Hermitian eigendecomposition A_c = V diag(lambda) V^+ (exp of a Hermitian matrix by its definition on the spectrum);
    inverse=True gives their inverses exp(-c_sw/(4+m0) A_c)/(4+m0)."""
    A = chiral_blocks(T, L, Rlinks)
    lam, vec = np.linalg.eigh(A)
    x = csw / (4.0 + m0) * lam
    f = np.exp(-x) / (4.0 + m0) if inverse else (4.0 + m0) * np.exp(x)
    return np.einsum("xcik,xck,xcjk->xcij", vec, f, np.conj(vec))


def apply_blocks(blocks, psi):
    """Site-diagonal chirality blocks [n, 2, 2d, 2d] applied to spinors [n, 4, d]."""
    psi = np.asarray(psi, dtype=np.complex128)
    n, _, d = psi.shape
    return np.einsum("xcij,xcj->xci", blocks, psi.reshape(n, 2, 2 * d)).reshape(n, 4, d)


def Dphi_expclover(T, L, m0, csw, Rlinks, psi, bc):
    """Eq 8 with the diagonal term of Eq 50."""
    from . import oracle as _o
    d = Rlinks.shape[-1]
    return _o.hop_field(T, L, d, Rlinks, psi, bc) + apply_blocks(exp_blocks(T, L, m0, csw, Rlinks), psi)


def Dphi_expclover_hat(T, L, m0, csw, Rlinks, psi_even, bc):
    """Eq 43 with the blocks of Eq 50: D_ee psi_e - D_eo D_oo^{-1} D_oe psi_e."""
    from . import oracle as _o
    d = Rlinks.shape[-1]
    ev, od = _parity_sites(T, L, 0), _parity_sites(T, L, 1)
    E = exp_blocks(T, L, m0, csw, Rlinks)
    Einv = exp_blocks(T, L, m0, csw, Rlinks, inverse=True)
    t = _o.Dphi_oe(T, L, d, Rlinks, psi_even, bc)
    return apply_blocks(E[ev], psi_even) - _o.Dphi_eo(T, L, d, Rlinks, apply_blocks(Einv[od], t), bc)
