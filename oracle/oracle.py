"""ctypes wrapper of the CPU oracle (oracle/hirep_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports the CUDA package.  All arrays are numpy complex128 in the canonical layout described in
hirep_oracle.c.  `build()` compiles the C file with gcc (building the checker is not using it).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hirep_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

FUND, ADJ, SYM, ASY = 0, 1, 2, 3

_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-o", _LIB, _SRC, "-lm"])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.oracle_rep_dim.restype = ctypes.c_int
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a, a.ctypes.data_as(ctypes.c_void_p)


def _bc(bc):
    return (ctypes.c_int * 4)(*[int(b) for b in bc])


DEFAULT_BC = (-1, 1, 1, 1)   # antiperiodic in time, periodic in space (BASELINE.json configs[0]; reading A7)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def rep_dim(n_g: int, rep: int) -> int:
    return int(lib().oracle_rep_dim(n_g, rep))


def gamma() -> np.ndarray:
    g = np.zeros((4, 4, 4), dtype=np.complex128)
    lib().oracle_gamma(g.ctypes.data_as(ctypes.c_void_p))
    return g


def gamma5() -> np.ndarray:
    g = np.zeros((4, 4), dtype=np.complex128)
    lib().oracle_gamma5(g.ctypes.data_as(ctypes.c_void_p))
    return g


def generators(n_g: int) -> np.ndarray:
    t = np.zeros((n_g * n_g - 1, n_g, n_g), dtype=np.complex128)
    lib().oracle_generators(n_g, t.ctypes.data_as(ctypes.c_void_p))
    return t


def tensor_basis(n_g: int, rep: int) -> np.ndarray:
    b = np.zeros((rep_dim(n_g, rep), n_g, n_g), dtype=np.float64)
    lib().oracle_tensor_basis(n_g, rep, b.ctypes.data_as(ctypes.c_void_p))
    return b


def rep_matrix(n_g: int, rep: int, U: np.ndarray) -> np.ndarray:
    d = rep_dim(n_g, rep)
    U, pU = _c(U)
    R = np.zeros((d, d), dtype=np.complex128)
    lib().oracle_rep_matrix(n_g, rep, pU, R.ctypes.data_as(ctypes.c_void_p))
    return R


def represent_field(n_g: int, rep: int, links: np.ndarray) -> np.ndarray:
    """links [..., N, N] -> [..., d_R, d_R] (complex128; ADJ has zero imaginary part)."""
    d = rep_dim(n_g, rep)
    links, pl = _c(links)
    n = links.size // (n_g * n_g)
    R = np.zeros(links.shape[:-2] + (d, d), dtype=np.complex128)
    lib().oracle_represent_field(n_g, rep, ctypes.c_long(n), pl, R.ctypes.data_as(ctypes.c_void_p))
    return R


def hop_local(d_R, Rf, Rb, psi_f, psi_b, sf, sb) -> np.ndarray:
    """One site of the hopping term from its 8 represented links and 8 neighbour spinors (Eq 8)."""
    keep = []

    def ptrs(arrs):
        out = (ctypes.c_void_p * 4)()
        for k, a in enumerate(arrs):
            a, p = _c(a)
            keep.append(a)
            out[k] = p
        return out

    out = np.zeros((4, d_R), dtype=np.complex128)
    sf = (ctypes.c_double * 4)(*[float(s) for s in sf])
    sb = (ctypes.c_double * 4)(*[float(s) for s in sb])
    lib().oracle_hop_local(d_R, ptrs(Rf), ptrs(Rb), ptrs(psi_f), ptrs(psi_b), sf, sb,
                           out.ctypes.data_as(ctypes.c_void_p))
    return out


def hop_field(T, L, d_R, Rlinks, psi, bc=DEFAULT_BC) -> np.ndarray:
    Rlinks, pR = _c(Rlinks)
    psi, pp = _c(psi)
    out = np.zeros_like(psi)
    lib().oracle_hop_field(T, L, d_R, _bc(bc), pR, pp, out.ctypes.data_as(ctypes.c_void_p))
    return out


def Dphi(T, L, d_R, m0, Rlinks, psi, bc=DEFAULT_BC) -> np.ndarray:
    Rlinks, pR = _c(Rlinks)
    psi, pp = _c(psi)
    out = np.zeros_like(psi)
    lib().oracle_Dphi(T, L, d_R, _bc(bc), ctypes.c_double(m0), pR, pp, out.ctypes.data_as(ctypes.c_void_p))
    return out


def _offdiag(T, L, d_R, pin, Rlinks, psi_half, bc):
    Rlinks, pR = _c(Rlinks)
    psi_half, pp = _c(psi_half)
    out = np.zeros_like(psi_half)
    lib().oracle_Dphi_offdiag(T, L, d_R, _bc(bc), pin, pR, pp, out.ctypes.data_as(ctypes.c_void_p))
    return out


def Dphi_eo(T, L, d_R, Rlinks, psi_odd, bc=DEFAULT_BC) -> np.ndarray:
    """odd in -> even out (row e, column o of Eq 41)."""
    return _offdiag(T, L, d_R, 1, Rlinks, psi_odd, bc)


def Dphi_oe(T, L, d_R, Rlinks, psi_even, bc=DEFAULT_BC) -> np.ndarray:
    return _offdiag(T, L, d_R, 0, Rlinks, psi_even, bc)


def Dphi_hat(T, L, d_R, m0, Rlinks, psi_even, bc=DEFAULT_BC) -> np.ndarray:
    Rlinks, pR = _c(Rlinks)
    psi_even, pp = _c(psi_even)
    out = np.zeros_like(psi_even)
    lib().oracle_Dphi_hat(T, L, d_R, _bc(bc), ctypes.c_double(m0), pR, pp, out.ctypes.data_as(ctypes.c_void_p))
    return out


def g5(psi) -> np.ndarray:
    psi, pp = _c(psi)
    out = np.zeros_like(psi)
    d_R = psi.shape[-1]
    lib().oracle_g5(ctypes.c_long(psi.size // (4 * d_R)), d_R, pp, out.ctypes.data_as(ctypes.c_void_p))
    return out


def g5Dphi_sq(T, L, d_R, m0, Rlinks, psi, bc=DEFAULT_BC) -> np.ndarray:
    Rlinks, pR = _c(Rlinks)
    psi, pp = _c(psi)
    out = np.zeros_like(psi)
    lib().oracle_g5Dphi_sq(T, L, d_R, _bc(bc), ctypes.c_double(m0), pR, pp, out.ctypes.data_as(ctypes.c_void_p))
    return out


def g5Dphi_hat(T, L, d_R, m0, Rlinks, psi_even, bc=DEFAULT_BC) -> np.ndarray:
    """Q_hat psi_e = gamma_5 D_hat psi_e (Eq 45) with D_hat in the normalisation of Eq 44 (L808): the literal
    composition of the two oracle functions above (reading A22 of DESIGN.md)."""
    return g5(Dphi_hat(T, L, d_R, m0, Rlinks, psi_even, bc))


def g5Dphi_hat_sq(T, L, d_R, m0, Rlinks, psi_even, bc=DEFAULT_BC) -> np.ndarray:
    """Q_hat^2 psi_e: the operator the even-odd preconditioned CG inverts (L772, L806)."""
    return g5Dphi_hat(T, L, d_R, m0, Rlinks, g5Dphi_hat(T, L, d_R, m0, Rlinks, psi_even, bc), bc)


# ---- twisted mass (Eq 51) and the general Schur form it needs (Eq 43); SURVEY 8(f) NEXT-2 ---------------
def g5_lc(c1, c2, eta) -> np.ndarray:
    """xi = c1 eta + c2 gamma_5 eta (the gamma_5-fused linear combination, L447)."""
    return complex(c1) * np.asarray(eta, dtype=np.complex128) + complex(c2) * g5(eta)


def Dphi_tm(T, L, d_R, m0, mu, Rlinks, psi, bc=DEFAULT_BC) -> np.ndarray:
    """Eq 51 for the tau^3 = +1 flavour: D^tm psi = D_m psi + i mu gamma_5 psi (the other flavour is mu -> -mu)."""
    return Dphi(T, L, d_R, m0, Rlinks, psi, bc) + 1j * float(mu) * g5(psi)


def Dphi_tm_hat(T, L, d_R, m0, mu, Rlinks, psi_even, bc=DEFAULT_BC) -> np.ndarray:
    """Eq 43 literally, with D_ee = D_oo = (4+m) + i mu gamma_5 (site-diagonal, so its inverse is
    ((4+m) - i mu gamma_5) / ((4+m)^2 + mu^2)):  D_hat psi_e = D_ee psi_e - D_eo D_oo^{-1} D_oe psi_e."""
    a, mu = 4.0 + float(m0), float(mu)
    t = Dphi_oe(T, L, d_R, Rlinks, psi_even, bc)
    t = g5_lc(a / (a * a + mu * mu), -1j * mu / (a * a + mu * mu), t)
    return g5_lc(a, 1j * mu, psi_even) - Dphi_eo(T, L, d_R, Rlinks, t, bc)


def Dphi_tm_sq(T, L, d_R, m0, mu, Rlinks, psi, bc=DEFAULT_BC) -> np.ndarray:
    """(D^tm)^dagger D^tm psi, with (D^tm(mu))^dagger = gamma_5 D^tm(-mu) gamma_5 (gamma_5-hermiticity of D_m, and
    (i mu gamma_5)^dagger = -i mu gamma_5): the Hermitian positive-definite operator of the twisted-mass monomial."""
    return g5(Dphi_tm(T, L, d_R, m0, -mu, Rlinks, g5(Dphi_tm(T, L, d_R, m0, mu, Rlinks, psi, bc)), bc))


def rel_l2(a: np.ndarray, b: np.ndarray) -> float:
    """||a - b||_2 / ||b||_2 in fp64 with compensated (math.fsum) accumulation."""
    import math
    a = np.asarray(a, dtype=np.complex128).ravel()
    b = np.asarray(b, dtype=np.complex128).ravel()
    d = a - b
    num = math.fsum((d.real ** 2 + d.imag ** 2).tolist()) if d.size < (1 << 22) else float(np.sum(np.abs(d) ** 2))
    den = math.fsum((b.real ** 2 + b.imag ** 2).tolist()) if b.size < (1 << 22) else float(np.sum(np.abs(b) ** 2))
    return math.sqrt(num / den) if den > 0 else math.sqrt(num)
