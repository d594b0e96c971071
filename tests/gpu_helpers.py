"""Helpers of the GPU parity tests: problem set-up and sampled oracle evaluation at full lattice sizes.

The neighbour bookkeeping here is test code, written against the canonical layout only (it knows nothing about
the library's native layout) and checked against the oracle's own field loop in tests/test_oracle_dirac.py
(test_hop_local_matches_field).
"""
from __future__ import annotations

import numpy as np

from harness import synth

BC = (-1, 1, 1, 1)
TOL = {"f64": 1e-13, "f32": 1e-5}          # BASELINE.json north_star: relative L2


def coords_of(ix, T, L):
    return np.array([ix // (L ** 3), (ix // (L * L)) % L, (ix // L) % L, ix % L])


def index_of(c, L):
    return int(((c[0] * L + c[1]) * L + c[2]) * L + c[3])


class SampledOracle:
    """Evaluates the oracle's operators at single sites from GPU-resident canonical tensors.

    links_canon: torch [V,4,N,N] (device), fetch_spinor(ix) -> np [4,d_R] complex128.
    Represented links are built per link by the oracle (oracle.rep_matrix) and memoised.
    """

    def __init__(self, oracle, cfg, links_canon, bc=BC):
        self.o, self.cfg, self.links, self.bc = oracle, cfg, links_canon, bc
        self.T, self.L, self.d = cfg.T, cfg.L, cfg.d_R
        self.ext = (cfg.T, cfg.L, cfg.L, cfg.L)
        self._R = {}

    def R(self, ix, mu):
        key = (ix, mu)
        if key not in self._R:
            U = self.links[ix, mu].cpu().numpy().astype(np.complex128)
            self._R[key] = self.o.rep_matrix(self.cfg.n_g, self.cfg.rep, U)
        return self._R[key]

    def neighbours(self, ix):
        c = coords_of(ix, self.T, self.L)
        fwd, bwd = [], []
        for mu in range(4):
            cf = c.copy(); cf[mu] += 1; s = 1
            if cf[mu] == self.ext[mu]:
                cf[mu] = 0; s = self.bc[mu]
            fwd.append((index_of(cf, self.L), s))
            cb = c.copy(); cb[mu] -= 1; s = 1
            if cb[mu] < 0:
                cb[mu] = self.ext[mu] - 1; s = self.bc[mu]
            bwd.append((index_of(cb, self.L), s))
        return fwd, bwd

    def hop(self, field, ix):
        """hop(field)(ix); `field(ix)` returns the [4,d] spinor at canonical site ix."""
        fwd, bwd = self.neighbours(ix)
        Rf = [self.R(ix, mu) for mu in range(4)]
        Rb = [self.R(bwd[mu][0], mu) for mu in range(4)]
        pf = [field(fwd[mu][0]) for mu in range(4)]
        pb = [field(bwd[mu][0]) for mu in range(4)]
        return self.o.hop_local(self.d, Rf, Rb, pf, pb, [f[1] for f in fwd], [b[1] for b in bwd])

    def Dphi(self, field, ix, m0):
        return (4.0 + m0) * field(ix) + self.hop(field, ix)

    def Dphi_hat(self, field_even, ix, m0):
        """(4+m)^2 psi(ix) - D_eo D_oe psi at an even site; field_even is only evaluated on even sites."""
        inner = lambda iy: self.hop(field_even, iy)          # (D_oe psi)(iy), iy odd
        return (4.0 + m0) ** 2 * field_even(ix) - self.hop(inner, ix)

    def g5Dphi_sq(self, field, ix, m0):
        G5 = self.o.gamma5()                                  # the oracle's own gamma_5 (4 x 4), pinned in test_oracle_dirac.py
        inner = lambda iy: G5 @ self.Dphi(field, iy, m0)
        return G5 @ self.Dphi(inner, ix, m0)


def torch_field_fetch(canon):
    """canon: torch [V,4,d] on any device -> fetch(ix) as complex128 numpy."""
    cache = {}

    def fetch(ix):
        if ix not in cache:
            cache[ix] = canon[ix].cpu().numpy().astype(np.complex128)
        return cache[ix]
    return fetch


def sample_sites(cfg, n, parity=None, seed=0):
    """Canonical indices: the lattice corners/edges (boundary wraps), sites of the last tile of the kernels' grid rounds,
    plus random interior sites."""
    T, L = cfg.T, cfg.L
    rng = np.random.default_rng(seed)
    picks = [0, cfg.volume - 1, index_of((T - 1, 0, L - 1, 0), L), index_of((0, L - 1, 0, L - 1), L),
             index_of((T // 2, L // 2, 1, L - 1), L), index_of((T - 1, L - 1, L - 1, L - 2), L)]
    if n >= 16:
        picks += round_end_sites(cfg, parity, n // 2, seed)
    picks += list(rng.integers(0, cfg.volume, size=4 * n))
    out = []
    for ix in picks:
        ix = int(ix)
        if parity is not None and int(coords_of(ix, T, L).sum()) % 2 != parity:
            ix = ix ^ 1              # flip z parity (L even): neighbouring site of the other parity
        if ix not in out:
            out.append(ix)
        if len(out) == n:
            break
    return out


def native_to_canonical(cfg, parity, h):
    """Canonical index of the site with half index h of `parity` in the library's documented site order (DESIGN.md 4:
    h = ((t L + x) L + y) L/2 + zh, z = 2 zh + ((t+x+y+parity) & 1)).  Used only to AIM samples at particular tiles."""
    L, Lh = cfg.L, cfg.L // 2
    zh = h % Lh; r = h // Lh
    y = r % L; r //= L
    x = r % L; t = r // L
    z = 2 * zh + ((t + x + y + parity) & 1)
    return index_of((t, x, y, z), L)


def round_end_sites(cfg, parity, n, seed=0):
    """Sites in the LAST tile of a grid round of the persistent kernels (a round = all warps / pairs / groups of the grid
    take one tile each), for every plausible round size, spread over the lattice, plus the ragged last tile."""
    rng = np.random.default_rng(seed)
    nh = cfg.volume // 2
    n_tiles = (nh + 31) // 32
    tiles = {n_tiles - 1}
    for per_sm in (1, 2, 3, 4, 6, 8, 12, 16):          # tiles in flight per SM: groups, pairs or warps per CTA
        R = 148 * per_sm
        for k in (1, 2, 3, max(1, n_tiles // (2 * R)), max(1, n_tiles // R)):
            for full_lattice in (1, 2):                # full-lattice launches interleave the parities: half the tiles per round
                tl = k * R // full_lattice - 1
                if 0 <= tl < n_tiles:
                    tiles.add(tl)
    tiles = sorted(tiles)
    picks = []
    for tl in tiles:
        h = min(tl * 32 + int(rng.integers(0, 32)), nh - 1)
        picks.append(native_to_canonical(cfg, parity if parity is not None else int(rng.integers(0, 2)), h))
    rng.shuffle(picks)
    return [int(v) for v in picks[:n]]


def half_rank(ix):
    """Row of canonical site ix inside the half-lattice canonical spinor of its parity."""
    return ix >> 1
