"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path.  It holds
none of the method's arithmetic (no gamma matrices, no representation maps, no stencil): it
only draws random SU(N) matrices and Gaussian spinors in the *canonical* interchange layout

    site index   ix = ((t*L + x)*L + y)*L + z            (z fastest, mu = 0 is time)
    spinor       [ix][spin 0..3][colour 0..d_R-1]         complex   (Tbl 2)
    links        [ix][mu 0..3][row i][col j]              complex, (U psi)_i = sum_j U_ij psi_j

The inputs stand in for the paper's thermalised gauge ensembles, which are
not available; the kernel's cost is data independent, so random links of the same shape have the
same byte footprint and access pattern.  Recipes are stated in DESIGN.md ("Input recipe").

numpy is used for host generation (tests, oracle); `*_torch` variants generate the same
distributions directly on a torch device for the full-size lattices, where host generation of
10^7..10^8 matrices would take minutes.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np

FUND, ADJ, SYM, ASY = 0, 1, 2, 3
REP_NAMES = {FUND: "FUND", ADJ: "ADJ", SYM: "SYM", ASY: "2AS"}


def rep_dim(n_g: int, rep: int) -> int:
    """d_R of Tbl 1."""
    return {FUND: n_g, ADJ: n_g * n_g - 1, SYM: n_g * (n_g + 1) // 2, ASY: n_g * (n_g - 1) // 2}[rep]


@dataclass(frozen=True)
class Config:
    name: str
    T: int
    L: int
    n_g: int
    rep: int
    m0: float
    links: str          # "haar" | "near_identity"
    seed: int
    ops: tuple
    eps: float = 0.3

    @property
    def d_R(self) -> int:
        return rep_dim(self.n_g, self.rep)

    @property
    def volume(self) -> int:
        return self.T * self.L ** 3

    def resized(self, T: int, L: int) -> "Config":
        return replace(self, T=T, L=L)


# BASELINE.json configs[0..4]
CONFIGS = {
    "C1": Config("C1", 4, 4, 2, FUND, +0.1, "haar", 1001, ("Dphi",)),
    "C2": Config("C2", 32, 32, 3, FUND, -0.2, "haar", 1002, ("Dphi_eo", "Dphi_hat")),
    "C3": Config("C3", 48, 48, 2, ADJ, -0.5, "haar", 1003, ("Dphi_eo",)),
    "C4": Config("C4", 96, 48, 4, ASY, -0.3, "near_identity", 1004, ("Dphi_hat", "g5Dphi_sq")),
    "C5": Config("C5", 32, 16, 6, ADJ, -0.4, "haar", 1005, ("Dphi_eo",)),
}


# ----------------------------------------------------------------------------- numpy (host)
def haar_su2(rng: np.random.Generator, n: int) -> np.ndarray:
    """Normalised Gaussian quaternion a -> [[a0+i a3, a2+i a1], [-a2+i a1, a0-i a3]]."""
    a = rng.standard_normal((n, 4))
    a /= np.linalg.norm(a, axis=1, keepdims=True)
    u = np.empty((n, 2, 2), dtype=np.complex128)
    u[:, 0, 0] = a[:, 0] + 1j * a[:, 3]
    u[:, 0, 1] = a[:, 2] + 1j * a[:, 1]
    u[:, 1, 0] = -a[:, 2] + 1j * a[:, 1]
    u[:, 1, 1] = a[:, 0] - 1j * a[:, 3]
    return u


def haar_sun(rng: np.random.Generator, n: int, n_g: int) -> np.ndarray:
    """QR of a complex Gaussian matrix, column phases fixed by diag(R), then det -> 1."""
    if n_g == 2:
        return haar_su2(rng, n)
    z = rng.standard_normal((n, n_g, n_g)) + 1j * rng.standard_normal((n, n_g, n_g))
    q, r = np.linalg.qr(z)
    d = np.diagonal(r, axis1=1, axis2=2)
    q = q * (d / np.abs(d))[:, None, :]
    det = np.linalg.det(q)
    q = q * np.exp(-1j * np.angle(det) / n_g)[:, None, None]
    return q


def gaussian_su_algebra(rng: np.random.Generator, n: int, n_g: int) -> np.ndarray:
    """Hermitian traceless H distributed as sum_a w_a T^a, w_a iid N(0,1), tr(T^a T^b) = delta/2.

    Drawn without any generator table: H = (A + A^dag)/2 - tr/N with A_ij = N(0,1/2) + i N(0,1/2)
    has the same law (off-diagonal E|H_ij|^2 = 1/2, diagonal covariance (delta_ij - 1/N)/2).
    """
    s = np.sqrt(0.5)
    a = s * rng.standard_normal((n, n_g, n_g)) + 1j * s * rng.standard_normal((n, n_g, n_g))
    h = 0.5 * (a + np.conj(np.swapaxes(a, 1, 2)))
    tr = np.trace(h, axis1=1, axis2=2).real / n_g
    h -= tr[:, None, None] * np.eye(n_g)
    return h


def near_identity_sun(rng: np.random.Generator, n: int, n_g: int, eps: float) -> np.ndarray:
    """U = exp(i eps H) by Hermitian eigendecomposition."""
    h = gaussian_su_algebra(rng, n, n_g)
    w, v = np.linalg.eigh(h)
    return (v * np.exp(1j * eps * w)[:, None, :]) @ np.conj(np.swapaxes(v, 1, 2))


def gaussian_spinor(rng: np.random.Generator, nsites: int, d_R: int) -> np.ndarray:
    return rng.standard_normal((nsites, 4, d_R)) + 1j * rng.standard_normal((nsites, 4, d_R))


def make_links(cfg: Config, rng: np.random.Generator) -> np.ndarray:
    n = cfg.volume * 4
    if cfg.links == "haar":
        u = haar_sun(rng, n, cfg.n_g)
    elif cfg.links == "near_identity":
        u = near_identity_sun(rng, n, cfg.n_g, cfg.eps)
    else:
        raise ValueError(cfg.links)
    return np.ascontiguousarray(u.reshape(cfg.volume, 4, cfg.n_g, cfg.n_g))


def make_inputs(cfg: Config, n_spinors: int = 1):
    """(links [V,4,N,N] c128, [spinor [V,4,d_R] c128, ...]) drawn in this order from PCG64(seed)."""
    rng = np.random.Generator(np.random.PCG64(cfg.seed))
    links = make_links(cfg, rng)
    spinors = [gaussian_spinor(rng, cfg.volume, cfg.d_R) for _ in range(n_spinors)]
    return links, spinors


def round_to_precision(a: np.ndarray, prec: str) -> np.ndarray:
    """fp32 runs use the fp64 arrays rounded to fp32 (widened back so the oracle sees the same values)."""
    if prec == "f64":
        return a
    return a.astype(np.complex64).astype(np.complex128)


# ------------------------------------------------------------------------ site bookkeeping
def site_coords(T: int, L: int) -> np.ndarray:
    """[V,4] integer coordinates (t,x,y,z) of canonical site index ix."""
    ix = np.arange(T * L ** 3)
    z = ix % L
    y = (ix // L) % L
    x = (ix // (L * L)) % L
    t = ix // (L * L * L)
    return np.stack([t, x, y, z], axis=1)


def parity_sites(T: int, L: int, parity: int) -> np.ndarray:
    """Canonical indices of the sites with (t+x+y+z) mod 2 == parity, increasing."""
    c = site_coords(T, L)
    return np.nonzero(c.sum(axis=1) % 2 == parity)[0]


# ------------------------------------------------------------------------------ torch (device)
def make_inputs_torch(cfg: Config, device, dtype_complex, n_spinors: int = 1, chunk_sites: int = 1 << 20):
    """Same distributions generated with torch on `device` (different random stream than numpy).

    Returns canonical tensors (links [V,4,N,N], [spinor [V,4,d_R], ...]) of `dtype_complex`.
    Generation is done in fp64 and rounded at the end, chunked to bound temporary memory.
    """
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(cfg.seed)
    V, N = cfg.volume, cfg.n_g
    links = torch.empty((V, 4, N, N), dtype=dtype_complex, device=device)
    for s0 in range(0, V, chunk_sites):
        n = (min(V, s0 + chunk_sites) - s0) * 4
        if cfg.links == "haar" and N == 2:
            a = torch.randn((n, 4), generator=g, device=device, dtype=torch.float64)
            a = a / a.norm(dim=1, keepdim=True)
            u = torch.empty((n, 2, 2), dtype=torch.complex128, device=device)
            u[:, 0, 0] = torch.complex(a[:, 0], a[:, 3])
            u[:, 0, 1] = torch.complex(a[:, 2], a[:, 1])
            u[:, 1, 0] = torch.complex(-a[:, 2], a[:, 1])
            u[:, 1, 1] = torch.complex(a[:, 0], -a[:, 3])
        elif cfg.links == "haar":
            # Gram-Schmidt on the columns of a complex Gaussian matrix = the Q of its QR factorisation with
            # diag(R) > 0, i.e. the numpy recipe above, but vectorised over the batch (two passes per column)
            z = torch.randn((n, N, N), generator=g, device=device, dtype=torch.complex128)
            cols = []
            for j in range(N):
                v = z[:, :, j]
                for _ in range(2):
                    for qk in cols:
                        v = v - (qk.conj() * v).sum(dim=1, keepdim=True) * qk
                cols.append(v / v.norm(dim=1, keepdim=True))
            q = torch.stack(cols, dim=2)
            det = torch.linalg.det(q)
            u = q * torch.exp(-1j * torch.angle(det) / N)[:, None, None]
        else:
            a = torch.randn((n, N, N), generator=g, device=device, dtype=torch.complex128)  # var 1/2 per part
            h = 0.5 * (a + a.mH)
            tr = torch.diagonal(h, dim1=1, dim2=2).sum(dim=1).real / N
            h = h - tr[:, None, None] * torch.eye(N, device=device, dtype=torch.complex128)
            u = torch.linalg.matrix_exp(1j * cfg.eps * h)
        links[s0:s0 + n // 4] = u.reshape(-1, 4, N, N).to(dtype_complex)
        del u
    spinors = []
    for _ in range(n_spinors):
        sp = torch.empty((V, 4, cfg.d_R), dtype=dtype_complex, device=device)
        for s0 in range(0, V, chunk_sites):
            n = min(V, s0 + chunk_sites) - s0
            re = torch.randn((n, 4, cfg.d_R), generator=g, device=device, dtype=torch.float64)
            im = torch.randn((n, 4, cfg.d_R), generator=g, device=device, dtype=torch.float64)
            sp[s0:s0 + n] = torch.complex(re, im).to(dtype_complex)
        spinors.append(sp)
    return links, spinors
