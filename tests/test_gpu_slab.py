"""Sharded operator on ONE GPU: the lattice is block-partitioned in t into 2 or 4 slabs, every "rank" is a
slab geometry with two ghost slices, the projected half-spinor faces are packed / copied device-to-device / unpacked by the
library's kernels, and the stitched result is compared with the oracle on the UNDIVIDED lattice.  The ranks' kernels run one
after the other (no kernel waits for another).  Real multi-GPU transport (NCCL isend/irecv) is covered on CPU by
tests/test_slab_host.py; scaling is unmeasured on hardware this round."""
import numpy as np
import pytest

from harness import synth
from paper_2503_06721_b200 import slab
from tests.gpu_helpers import TOL
from tests.test_gpu_parity import env, np_c  # noqa: F401  (env is a fixture)

pytestmark = pytest.mark.gpu


class Rank:
    def __init__(self, env, cfg, prec, bc, t_start, T_loc, U, psi):
        torch, hirep = env["torch"], env["hirep"]
        T, L, d = cfg.T, cfg.L, cfg.d_R
        self.ts = [(t_start - 1 + k) % T for k in range(T_loc + 2)]        # global slices of the local lattice (ghosts at both ends)
        S = L ** 3
        self.geom = hirep.Geometry(T_loc, L, cfg.n_g, cfg.rep, prec, device=env["dev"], bc=bc, slab=(T, t_start))
        U_loc = U.reshape(T, S, 4, cfg.n_g, cfg.n_g)[self.ts].reshape(-1, 4, cfg.n_g, cfg.n_g)
        self.links = self.geom.links_to_rep(self.geom.links_import(torch.from_numpy(U_loc.astype(np_c(prec)))))
        loc = psi.reshape(T, S, 4, d)[self.ts].copy()
        loc[0] = 0; loc[-1] = 0                                              # ghost slices start EMPTY: only the halo can fill them
        self.x = self.geom.spinor_import(torch.from_numpy(loc.reshape(-1, 4, d).astype(np_c(prec))), hirep.FULL)
        self.T_loc, self.S, self.d = T_loc, S, d

    def owned(self, native_full, hirep):
        out = self.geom.spinor_export(native_full, hirep.FULL).cpu().numpy().astype(np.complex128)
        return out.reshape(self.T_loc + 2, self.S, 4, self.d)[1:-1]


def halo_exchange(ranks, halves_of):
    """every rank's faces -> its neighbours' ghost slices (device-to-device; the buffers stand in for the transport)"""
    R = len(ranks)
    for r, rk in enumerate(ranks):
        for hsel in halves_of:
            src = hsel(rk)
            f0, f1 = rk.geom.halo_pack(0, src), rk.geom.halo_pack(1, src)
            prv, nxt = slab.neighbours(r, R)
            ranks[prv].geom.halo_unpack(0, hsel(ranks[prv]), f0.clone())   # first owned slice -> previous rank's last ghost slice
            ranks[nxt].geom.halo_unpack(1, hsel(ranks[nxt]), f1.clone())   # last owned slice  -> next rank's ghost slice 0


@pytest.mark.parametrize("name,T,L,world", [("C2", 8, 4, 2), ("C2", 8, 4, 4), ("C3", 8, 6, 2), ("C4", 12, 4, 3), ("C5", 4, 4, 2)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_sharded_operators_match_the_undivided_lattice(env, name, T, L, world, prec):
    torch, hirep, oracle = env["torch"], env["hirep"], env["oracle"]
    cfg = synth.CONFIGS[name].resized(T, L)
    bc = (-1, 1, 1, -1)
    U, (psi,) = synth.make_inputs(cfg)
    U, psi = synth.round_to_precision(U, prec), synth.round_to_precision(psi, prec)
    R = oracle.represent_field(cfg.n_g, cfg.rep, U)
    ranks = [Rank(env, cfg, prec, bc, t0, n, U, psi) for t0, n in slab.partition(T, world)]
    hb = ranks[0].geom.sizes["spinor_half"]
    halo_exchange(ranks, [lambda rk: rk.x[:hb], lambda rk: rk.x[hb:]])
    # full-lattice Dphi: region OWNED in one go, and INTERIOR + BOUNDARY (the split of Fig 1) must agree with it bit for bit
    ref = oracle.Dphi(T, L, cfg.d_R, cfg.m0, R, psi, bc)
    parts, parts_split = [], []
    for rk in ranks:
        y = rk.geom.Dphi(cfg.m0, rk.x, rk.links)
        parts.append(rk.owned(y, hirep))
        y2 = torch.zeros_like(y)
        rk.geom.set_region(hirep.REGION_INTERIOR); rk.geom.Dphi(cfg.m0, rk.x, rk.links, out=y2)
        rk.geom.set_region(hirep.REGION_BOUNDARY); rk.geom.Dphi(cfg.m0, rk.x, rk.links, out=y2)
        rk.geom.set_region(hirep.REGION_OWNED)
        parts_split.append(rk.owned(y2, hirep))
    got = np.concatenate(parts).reshape(-1, 4, cfg.d_R)
    assert oracle.rel_l2(got, ref) < TOL[prec], (name, world, prec)
    assert np.array_equal(np.concatenate(parts_split).reshape(-1, 4, cfg.d_R), got)
    # even-odd piece: GLOBAL even output <- GLOBAL odd input; on a slab (t_start even, one ghost slice in front) local parity =
    # global parity XOR 1, so that is the LOCAL Dphi_oe: local-even input half -> local-odd output half
    ev, od = synth.parity_sites(T, L, 0), synth.parity_sites(T, L, 1)
    ref_eo = oracle.Dphi_eo(T, L, cfg.d_R, R, psi[od], bc)
    outs = []
    for rk in ranks:
        y = torch.zeros_like(rk.x)
        rk.geom.Dphi_oe(rk.x[:hb], rk.links, out=y[hb:])
        outs.append(rk.owned(y, hirep))
    got_full = np.concatenate(outs).reshape(-1, 4, cfg.d_R)
    assert oracle.rel_l2(got_full[ev], ref_eo) < TOL[prec], (name, world, prec)


def test_slab_errors_and_two_pass_guard(env):
    hirep = env["hirep"]
    with pytest.raises(hirep.HirepError):
        hirep.hirep_geom_create_slab(8, 4, 3, 0, 0, 1, 4)          # odd t_start
    with pytest.raises(hirep.HirepError):
        hirep.hirep_geom_create_slab(8, 4, 3, 0, 0, 6, 4)          # runs past the lattice
    g = hirep.Geometry(4, 4, 3, 0, "f64", device=env["dev"], slab=(8, 0))
    x, lr = g.new_spinor(hirep.FULL), g.new_links_rep()
    with pytest.raises(hirep.HirepError, match="slab"):
        g.g5Dphi_sq(0.1, x, lr)
    plain = hirep.Geometry(4, 4, 3, 0, "f64", device=env["dev"])
    with pytest.raises(hirep.HirepError, match="slab"):
        plain.set_region(hirep.REGION_INTERIOR)
    with pytest.raises(hirep.HirepError, match="slab"):
        plain.halo_pack(0, plain.new_spinor(hirep.EVEN))
