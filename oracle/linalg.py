"""CPU oracle of the spinor linear algebra, the reductions and the CG inverter.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import this; it never imports the CUDA
package.  Plain numpy / pure Python in fp64, written to be checked against PAPER.md by eye:

  linear combinations   Eq 22-26: lc, clc, lc1, lc2, lc3 and the add-assign forms
  reductions            Eq 27 (L402) <xi,eta> = sum conj(xi) eta ; Eq 32 (L426) ||xi||_2 ; Eq 33 (L430) max norm
  compensated sums      Alg 1 FastTwoSum (L642), Alg 2 Neumaier (L662), Alg 3 second-order Neumaier (L682),
                        Alg 4 double-double (L706) -- step by step, in the paper's notation
  inverter              conjugate gradient for the Hermitian positive-definite Q_m^2 (L772: "Q_m^2 = Q_m^dagger Q_m
                        is Hermitian and positive definite"; L730 lists CG among the supported inverters but prints no
                        algorithm: the textbook Hestenes-Stiefel recurrence is used and stated in DESIGN.md, reading A19)

Where the exact value of a sum is the definition (inner products, norms) the oracle returns the correctly rounded
sum (math.fsum); the compensated algorithms are separate functions whose job is to be compared with that.
"""
from __future__ import annotations

import math

import numpy as np


# ------------------------------------------------------------------------------ linear combinations (Eq 22-26)
def lc(r1, eta, r2, zeta):
    """Eq 22: xi = r1 eta + r2 zeta, r1, r2 real."""
    return float(r1) * eta + float(r2) * zeta


def clc(c1, eta, c2, zeta):
    """Eq 23: xi = c1 eta + c2 zeta, c1, c2 complex."""
    return complex(c1) * eta + complex(c2) * zeta


def lc_add_assign(xi, r1, eta, r2, zeta):
    """add-assign version of Eq 22: xi <- xi + r1 eta + r2 zeta."""
    return xi + float(r1) * eta + float(r2) * zeta


def clc_add_assign(xi, c1, eta, c2, zeta):
    """add-assign version of Eq 23: xi <- xi + c1 eta + c2 zeta."""
    return xi + complex(c1) * eta + complex(c2) * zeta


def lc1(xi, c1, eta):
    """Eq 24: xi <- xi + c1 eta."""
    return xi + complex(c1) * eta


def lc2(xi, c1, c2, eta):
    """Eq 25: xi <- c1 xi + c2 eta."""
    return complex(c1) * xi + complex(c2) * eta


def lc3(xi, c1, eta, c2, zeta):
    """Eq 26: xi <- c1 eta + c2 zeta - xi."""
    return complex(c1) * eta + complex(c2) * zeta - xi


# --------------------------------------------------------------------------------------- reductions (Eq 27-33)
def _terms_of_product(xi, eta):
    """real and imaginary parts of conj(xi_k) eta_k as exact-sum inputs: each product a*b of two doubles is split
    into its rounded value and the rounding error (Dekker/Veltkamp via fma-free splitting is avoided: Python floats
    are exact rationals, so fractions would be exact but slow; instead the 4 real products per element are handed
    to fsum separately -- each is one rounding away from exact, which bounds the oracle's own error by
    2^-53 * sum |terms|, the same first-order bound the GPU's fp64 products have)."""
    a, b = np.asarray(xi, dtype=np.complex128).ravel(), np.asarray(eta, dtype=np.complex128).ravel()
    re = np.concatenate([a.real * b.real, a.imag * b.imag])
    im = np.concatenate([a.real * b.imag, -(a.imag * b.real)])
    return re, im


def prod(xi, eta) -> complex:
    """Eq 27: <xi, eta> = sum_{site, alpha, a} conj(xi) eta, correctly rounded sum of the fp64 products."""
    re, im = _terms_of_product(xi, eta)
    return complex(math.fsum(re.tolist()), math.fsum(im.tolist()))


def prod_re(xi, eta) -> float:
    return prod(xi, eta).real


def sqnorm(xi) -> float:
    """Eq 32 squared: <xi, xi> (real)."""
    a = np.asarray(xi, dtype=np.complex128).ravel()
    return math.fsum(np.concatenate([a.real * a.real, a.imag * a.imag]).tolist())


def norm2(xi) -> float:
    """Eq 32: ||xi||_2 = sqrt(<xi, xi>)."""
    return math.sqrt(sqnorm(xi))


def max_norm(eta) -> float:
    """Eq 33: the largest |Re| or |Im| over all components."""
    a = np.asarray(eta, dtype=np.complex128).ravel()
    return float(max(np.max(np.abs(a.real)), np.max(np.abs(a.imag)))) if a.size else 0.0


# ---------------------------------------------------------------------------- compensated sums (Alg 1-4)
def fast_two_sum(a: float, b: float):
    """Algorithm 1: (s, c) with s = a (+) b and s + c = a + b exactly."""
    s = a + b
    if abs(a) >= abs(b):
        c = b - (s - a)
    else:
        c = a - (s - b)
    return s, c


def neumaier(a) -> float:
    """Algorithm 2."""
    s, c = 0.0, 0.0
    for x in a:
        s, e = fast_two_sum(s, float(x))
        c = c + e
    return s + c


def second_order_neumaier(a) -> float:
    """Algorithm 3."""
    s, c, c2 = 0.0, 0.0, 0.0
    for x in a:
        s, e = fast_two_sum(s, float(x))
        c, e = fast_two_sum(c, e)
        c2 = c2 + e
    return s + (c + c2)


def double_double_sum(a) -> float:
    """Algorithm 4."""
    s, c = 0.0, 0.0
    for x in a:
        s, e = fast_two_sum(s, float(x))
        s, c = fast_two_sum(s, c + e)
    return s


def naive_sum(a) -> float:
    s = 0.0
    for x in a:
        s = s + float(x)
    return s


# ------------------------------------------------------------------------------------------------ inverter (L730)
def cg(apply_A, b, tol: float, maxiter: int, x0=None):
    """Conjugate gradient for A x = b, A Hermitian positive definite (A = Q_m^2 = g5Dphi_sq, L772).

    Textbook recurrence (Hestenes-Stiefel), reading A19 of DESIGN.md:
        r = b - A x ; p = r ; rr = <r,r>
        repeat:  Ap = A p ; alpha = rr / <p,Ap> ; x += alpha p ; r -= alpha Ap ; rr' = <r,r>
                 stop if rr' <= tol^2 <b,b> ; beta = rr'/rr ; p = r + beta p ; rr = rr'
    Returns (x, iterations, relative residual sqrt(rr/<b,b>) of the recurrence, history of rr)."""
    b = np.asarray(b, dtype=np.complex128)
    x = np.zeros_like(b) if x0 is None else np.array(x0, dtype=np.complex128)
    r = b - apply_A(x) if x0 is not None else b.copy()
    p = r.copy()
    bb = sqnorm(b)
    rr = sqnorm(r)
    hist = [rr]
    it = 0
    if bb == 0.0:
        return x, 0, 0.0, hist
    while it < maxiter and rr > tol * tol * bb:
        Ap = apply_A(p)
        alpha = rr / prod_re(p, Ap)
        x = x + alpha * p
        r = r - alpha * Ap
        rr_new = sqnorm(r)
        it += 1
        hist.append(rr_new)
        beta = rr_new / rr
        p = r + beta * p
        rr = rr_new
    return x, it, math.sqrt(rr / bb), hist


def cg_mshift(apply_A, b, shifts, tol: float, maxiter: int):
    """Multi-shift conjugate gradient (L730: "the Multi-Shift Conjugate Gradient ... is necessary for simulations
    with the RHMC"; Eq 39-40: the rational approximation needs (Q_m^2 + beta_k)^{-1} b for all k at once).

    The paper prints no recurrence; the textbook one is used (reading A24 of DESIGN.md).  All shifted systems
    (A + sigma_k) x_k = b share the Krylov space of A: their residuals are collinear with the residual r of the
    unshifted recurrence, r_k = zeta_k r, with
        zeta_k' = zeta_k zeta_k^- alpha^- / ( alpha beta^- (zeta_k^- - zeta_k) + zeta_k^- alpha^- (1 + sigma_k alpha) )
        alpha_k = alpha zeta_k'/zeta_k ,  beta_k = beta (zeta_k'/zeta_k)^2
        x_k += alpha_k p_k ,  p_k' = zeta_k' r' + beta_k p_k
    where alpha, beta are the step and direction coefficients of plain CG on A (superscript - : previous iteration;
    alpha^- = 1, beta^- = 0, zeta = zeta^- = 1 at the start).  Stops on the unshifted residual (the shifted ones are
    smaller for sigma_k >= 0).  Returns ([x_k], iterations, relative residual of the unshifted recurrence)."""
    b = np.asarray(b, dtype=np.complex128)
    ns = len(shifts)
    xs = [np.zeros_like(b) for _ in range(ns)]
    ps = [b.copy() for _ in range(ns)]
    r, p = b.copy(), b.copy()
    bb = sqnorm(b)
    rr = bb
    zeta = [1.0] * ns
    zeta_old = [1.0] * ns
    alpha_old, beta_old = 1.0, 0.0
    it = 0
    if bb == 0.0:
        return xs, 0, 0.0
    while it < maxiter and rr > tol * tol * bb:
        Ap = apply_A(p)
        alpha = rr / prod_re(p, Ap)
        zeta_new = []
        for k in range(ns):
            zn = zeta[k] * zeta_old[k] * alpha_old / (alpha * beta_old * (zeta_old[k] - zeta[k])
                                                     + zeta_old[k] * alpha_old * (1.0 + float(shifts[k]) * alpha))
            zeta_new.append(zn)
            xs[k] = xs[k] + (alpha * zn / zeta[k]) * ps[k]
        r = r - alpha * Ap
        rr_new = sqnorm(r)
        it += 1
        beta = rr_new / rr
        for k in range(ns):
            ps[k] = zeta_new[k] * r + (beta * (zeta_new[k] / zeta[k]) ** 2) * ps[k]
        p = r + beta * p
        zeta_old, zeta = zeta, zeta_new
        alpha_old, beta_old = alpha, beta
        rr = rr_new
    return xs, it, math.sqrt(rr / bb)


def bicgstab(apply_A, b, tol: float, maxiter: int):
    """Stabilised bi-conjugate gradient (L730: "the stabilized Bi-Conjugate Gradient (BiCG)[35, 36] ... for
    ill-conditioned systems often substantially faster") for a general (non-Hermitian) A x = b, e.g. A = D_m or
    D_hat directly.  Textbook recurrence (van der Vorst), x0 = 0, shadow residual = b (reading A25 of DESIGN.md):
        rho' = <rhat, r> ; beta = (rho'/rho)(alpha/omega) ; p = r + beta (p - omega v) ; v = A p
        alpha = rho'/<rhat, v> ; s = r - alpha v ; t = A s ; omega = <t,s>/<t,t>
        x += alpha p + omega s ; r = s - omega t
    with <.,.> the product of Eq 27.  Stops when ||r|| <= tol ||b|| (checked on s as well, after the half step).
    Returns (x, iterations, relative residual of the recurrence)."""
    b = np.asarray(b, dtype=np.complex128)
    x = np.zeros_like(b)
    r = b.copy()
    rhat = b.copy()
    p = np.zeros_like(b)
    v = np.zeros_like(b)
    rho = alpha = omega = 1.0 + 0.0j
    bb = sqnorm(b)
    rr = bb
    it = 0
    if bb == 0.0:
        return x, 0, 0.0
    while it < maxiter and rr > tol * tol * bb:
        rho_new = prod(rhat, r)
        beta = (rho_new / rho) * (alpha / omega)
        p = r + beta * (p - omega * v)
        v = apply_A(p)
        alpha = rho_new / prod(rhat, v)
        s = r - alpha * v
        it += 1
        ss = sqnorm(s)
        if ss <= tol * tol * bb:
            x = x + alpha * p
            rr = ss
            break
        t = apply_A(s)
        omega = prod(t, s) / sqnorm(t)
        x = x + alpha * p + omega * s
        r = s - omega * t
        rr = sqnorm(r)
        rho = rho_new
    return x, it, math.sqrt(rr / bb)
