"""GPU parity tests: the CUDA library (through the C-ABI binding) against the CPU oracle, element by element.

Tolerance (BASELINE.json north_star): relative L2 <= 1e-13 (fp64), <= 1e-5 (fp32).  fp32 runs feed the oracle the
fp32-rounded inputs widened to fp64, so the error measures arithmetic only.  Index/byte work (layout round trips)
is bit exact.  Reduced lattices span several 32-site tiles and a ragged tail; the full BASELINE sizes are checked
on sampled output sites (tests/gpu_helpers.py) in the launch configuration bench.py times.
"""
import numpy as np
import pytest

from harness import synth
from tests.gpu_helpers import BC, TOL, SampledOracle, half_rank, sample_sites, torch_field_fetch

pytestmark = pytest.mark.gpu

FUND, ADJ, SYM, ASY = 0, 1, 2, 3


@pytest.fixture(scope="module")
def env(oracle):
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import __graft_entry__ as ge
    import os
    if not os.path.exists(ge.LIB):
        ge.build_cuda()
    from paper_2503_06721_b200 import hirep
    hirep.load()
    return dict(torch=torch, hirep=hirep, oracle=oracle, dev=torch.device("cuda:0"))


def np_c(prec):
    return np.complex128 if prec == "f64" else np.complex64


class Problem:
    def __init__(self, env, cfg, prec, bc=BC, n_spinors=1):
        torch, hirep = env["torch"], env["hirep"]
        self.env, self.cfg, self.prec, self.bc = env, cfg, prec, bc
        U, spinors = synth.make_inputs(cfg, n_spinors)
        self.U = synth.round_to_precision(U, prec)
        self.spinors = [synth.round_to_precision(s, prec) for s in spinors]
        self.geom = hirep.Geometry(cfg.T, cfg.L, cfg.n_g, cfg.rep, prec, device=env["dev"], bc=bc)
        self.links_fund = self.geom.links_import(torch.from_numpy(self.U.astype(np_c(prec))))
        self.links_rep = self.geom.links_to_rep(self.links_fund)
        self._R = None
        self.ev = synth.parity_sites(cfg.T, cfg.L, 0)
        self.od = synth.parity_sites(cfg.T, cfg.L, 1)

    @property
    def R(self):
        if self._R is None:
            self._R = self.env["oracle"].represent_field(self.cfg.n_g, self.cfg.rep, self.U)
        return self._R

    def to_native(self, canon, which):
        return self.geom.spinor_import(self.env["torch"].from_numpy(canon.astype(np_c(self.prec))), which)

    def to_numpy(self, native, which):
        return self.geom.spinor_export(native, which).cpu().numpy().astype(np.complex128)


# ------------------------------------------------------------------------------ layout, bit exact
@pytest.mark.parametrize("T,L,n,rep", [(2, 2, 2, FUND), (4, 4, 3, FUND), (2, 6, 2, ADJ), (6, 6, 4, ASY), (4, 2, 6, ADJ)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_spinor_roundtrip_bit_exact(env, T, L, n, rep, prec):
    torch, hirep = env["torch"], env["hirep"]
    cfg = synth.Config("t", T, L, n, rep, 0.0, "haar", 7, ())
    geom = hirep.Geometry(T, L, n, rep, prec, device=env["dev"])
    psi = synth.gaussian_spinor(np.random.default_rng(3), cfg.volume, cfg.d_R).astype(np_c(prec))
    full = geom.spinor_export(geom.spinor_import(torch.from_numpy(psi), hirep.FULL), hirep.FULL).cpu().numpy()
    assert np.array_equal(full, psi)
    for which, sites in ((hirep.EVEN, synth.parity_sites(T, L, 0)), (hirep.ODD, synth.parity_sites(T, L, 1))):
        half = geom.spinor_export(geom.spinor_import(torch.from_numpy(psi[sites]), which), which).cpu().numpy()
        assert np.array_equal(half, psi[sites])
    # the full-lattice native buffer is the even half followed by the odd half
    nat = geom.spinor_import(torch.from_numpy(psi), hirep.FULL)
    hb = geom.sizes["spinor_half"]
    ev = geom.spinor_export(nat[:hb], hirep.EVEN).cpu().numpy()
    od = geom.spinor_export(nat[hb:], hirep.ODD).cpu().numpy()
    assert np.array_equal(ev, psi[synth.parity_sites(T, L, 0)]) and np.array_equal(od, psi[synth.parity_sites(T, L, 1)])


# ------------------------------------------------------------------------ links_to_rep vs oracle
REPS = [(2, FUND), (3, FUND), (4, FUND), (2, ADJ), (3, ADJ), (4, ADJ), (6, ADJ), (2, SYM), (3, SYM), (4, SYM),
        (2, ASY), (3, ASY), (4, ASY), (5, ASY), (6, ASY)]


@pytest.mark.parametrize("n,rep", REPS)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_links_to_rep(env, n, rep, prec):
    oracle = env["oracle"]
    T, L = 4, 2
    cfg = synth.Config("t", T, L, n, rep, 0.0, "haar", 100 + 10 * n + rep, ())
    p = Problem(env, cfg, prec)
    fwd = p.geom.links_rep_export(p.links_rep).cpu().numpy().astype(np.complex128)
    bwd = p.geom.links_rep_export(p.links_rep, bwd=True).cpu().numpy().astype(np.complex128)
    c = synth.site_coords(T, L)
    ext = np.array([T, L, L, L])
    tol = 1e-13 if prec == "f64" else 2e-6
    ref_f = p.R.copy()
    ref_b = np.empty_like(ref_f)
    for mu in range(4):
        ref_f[c[:, mu] == ext[mu] - 1, mu] *= BC[mu]                   # forward hop crosses the edge (L945)
        cb = c.copy(); cb[:, mu] = (cb[:, mu] - 1) % ext[mu]
        ib = ((cb[:, 0] * L + cb[:, 1]) * L + cb[:, 2]) * L + cb[:, 3]
        ref_b[:, mu] = np.conj(np.swapaxes(p.R[ib, mu], -1, -2))
        ref_b[c[:, mu] == 0, mu] *= BC[mu]
    assert oracle.rel_l2(fwd, ref_f) < tol
    assert oracle.rel_l2(bwd, ref_b) < tol
    if rep == ADJ:
        assert p.geom.sizes["rep_is_real"]


# ------------------------------------------------------------------ operators on reduced lattices
SMALL = [  # (config, T, L) : several tiles + ragged tail (Nh % 32 != 0) except C1 which is the BASELINE size
    ("C1", 4, 4), ("C2", 6, 6), ("C3", 6, 6), ("C4", 6, 6), ("C5", 4, 6),
]


def check_all_ops(env, p, variant=0, rebuild=False):
    oracle, hirep = env["oracle"], env["hirep"]
    cfg, g = p.cfg, p.geom
    g.set_link_mode(hirep.LINKS_REBUILD if rebuild else hirep.LINKS_STORED)
    links = p.links_fund if rebuild else p.links_rep
    T, L, d, m0 = cfg.T, cfg.L, cfg.d_R, cfg.m0
    tol = TOL[p.prec]
    g.set_kernel_variant(variant)
    psi = p.spinors[0]
    errs = {}
    out = p.to_numpy(g.Dphi(m0, p.to_native(psi, hirep.FULL), links), hirep.FULL)
    errs["Dphi"] = oracle.rel_l2(out, oracle.Dphi(T, L, d, m0, p.R, psi, p.bc))
    out = p.to_numpy(g.Dphi_eo(p.to_native(psi[p.od], hirep.ODD), links), hirep.EVEN)
    errs["Dphi_eo"] = oracle.rel_l2(out, oracle.Dphi_eo(T, L, d, p.R, psi[p.od], p.bc))
    out = p.to_numpy(g.Dphi_oe(p.to_native(psi[p.ev], hirep.EVEN), links), hirep.ODD)
    errs["Dphi_oe"] = oracle.rel_l2(out, oracle.Dphi_oe(T, L, d, p.R, psi[p.ev], p.bc))
    out = p.to_numpy(g.Dphi_hat(m0, p.to_native(psi[p.ev], hirep.EVEN), links), hirep.EVEN)
    errs["Dphi_hat"] = oracle.rel_l2(out, oracle.Dphi_hat(T, L, d, m0, p.R, psi[p.ev], p.bc))
    out = p.to_numpy(g.g5Dphi_sq(m0, p.to_native(psi, hirep.FULL), links), hirep.FULL)
    errs["g5Dphi_sq"] = oracle.rel_l2(out, oracle.g5Dphi_sq(T, L, d, m0, p.R, psi, p.bc))
    g.sync()
    for k, v in errs.items():
        assert v < tol, (k, v, errs)
    return errs


@pytest.mark.parametrize("name,T,L", SMALL)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_operators_vs_oracle_reduced(env, name, T, L, prec):
    cfg = synth.CONFIGS[name].resized(T, L)
    p = Problem(env, cfg, prec)
    errs = check_all_ops(env, p)
    print(name, prec, {k: "%.2e" % v for k, v in errs.items()})


@pytest.mark.parametrize("name,T,L", [("C1", 4, 4), ("C2", 6, 6), ("C3", 2, 6), ("C4", 4, 6)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("variant", [1, 2, 3, 4, 5])
def test_kernel_variants(env, name, T, L, prec, variant):
    p = Problem(env, synth.CONFIGS[name].resized(T, L), prec)
    check_all_ops(env, p, variant)


@pytest.mark.parametrize("name,prec,variant", [("C2", "f64", 3), ("C2", "f32", 3), ("C3", "f64", 3), ("C4", "f32", 3),
                                               ("C4", "f64", 4), ("C2", "f64", 4), ("C3", "f32", 4),
                                               ("C1", "f64", 5), ("C2", "f64", 5), ("C2", "f32", 5), ("C3", "f64", 5), ("C3", "f32", 5),
                                               ("C4", "f64", 5), ("C4", "f32", 5)])
@pytest.mark.parametrize("max_ctas", [1, 3])
def test_persistent_loop(env, name, prec, variant, max_ctas):
    """Persistent kernels with MANY tiles per warp (grid capped at 1-3 CTAs: the bulk-copy ring wraps across tile
    boundaries many times, mbarrier phases flip) on a 4x8^3 lattice (32 tiles per parity)."""
    hirep = env["hirep"]
    p = Problem(env, synth.CONFIGS[name].resized(4, 8), prec)
    p.geom.set_tuning(hirep.TUNE_MAX_CTAS, max_ctas)
    check_all_ops(env, p, variant)


@pytest.mark.parametrize("n,rep", [(3, SYM), (3, ASY), (2, SYM), (4, FUND), (5, FUND), (3, ADJ), (4, SYM), (6, ASY), (4, ADJ),
                                   (5, ASY), (5, SYM), (6, SYM), (5, ADJ), (2, ASY)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_other_representations(env, n, rep, prec):
    """Every (N_g <= 6, rep) the library instantiates beyond the BASELINE configs (d_R up to 24)."""
    cfg = synth.Config("t", 4, 4, n, rep, -0.25, "haar", 500 + 10 * n + rep, ())
    check_all_ops(env, Problem(env, cfg, prec))


@pytest.mark.parametrize("n,rep", [(3, ADJ), (4, SYM), (6, ASY), (6, ADJ)])
@pytest.mark.parametrize("max_ctas,variant", [(1, 0), (3, 0), (0, 1)])
def test_large_dR_kernels(env, n, rep, max_ctas, variant):
    """d_R >= 8: the row-group ring kernel with many tiles per group (capped grid), and the direct-load kernel."""
    hirep = env["hirep"]
    cfg = synth.Config("t", 4, 6, n, rep, -0.4, "haar", 900 + 10 * n + rep, ())
    p = Problem(env, cfg, "f64")
    p.geom.set_tuning(hirep.TUNE_MAX_CTAS, max_ctas)
    check_all_ops(env, p, variant)


REBUILD = [(2, FUND), (3, FUND), (4, FUND), (5, FUND), (6, FUND), (2, ADJ), (2, SYM), (3, SYM), (2, ASY), (3, ASY), (4, ASY),
           (3, ADJ), (4, ADJ), (5, ADJ), (6, ADJ)]        # the last four: matrix-free adjoint (hop_adjmf.cuh)


@pytest.mark.parametrize("n,rep", REBUILD)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_rebuild_mode(env, n, rep, prec):
    """Link mode REBUILD (`links` = the fundamental field, R rebuilt in registers, boundary sign applied to the
    half spinor) against the oracle, every (N_g, rep) with d_R <= 6 and the matrix-free adjoint of SU(3..6); non-trivial
    signs in two directions and a ragged tail."""
    cfg = synth.Config("t", 6, 6, n, rep, -0.3, "haar", 700 + 10 * n + rep, ())
    check_all_ops(env, Problem(env, cfg, prec, bc=(-1, 1, -1, 1)), rebuild=True)


def test_rebuild_mode_persistent_and_unsupported(env):
    hirep = env["hirep"]
    p = Problem(env, synth.CONFIGS["C4"].resized(4, 8), "f64")
    p.geom.set_tuning(hirep.TUNE_MAX_CTAS, 2)
    check_all_ops(env, p, rebuild=True)
    # stored and rebuilt agree with each other to rounding
    x = p.to_native(p.spinors[0][p.ev], hirep.EVEN)
    a = p.to_numpy(p.geom.Dphi_hat(-0.3, x, p.links_fund), hirep.EVEN)
    p.geom.set_link_mode(hirep.LINKS_STORED)
    b = p.to_numpy(p.geom.Dphi_hat(-0.3, x, p.links_rep), hirep.EVEN)
    assert env["oracle"].rel_l2(a, b) < 1e-14
    # 2-index representations with d_R > 6 have no rebuild kernel: loud error, no fallback
    q = Problem(env, synth.Config("t", 2, 2, 4, SYM, -0.4, "haar", 5, ()), "f64")
    q.geom.set_link_mode(hirep.LINKS_REBUILD)
    with pytest.raises(hirep.HirepError, match="no kernel instantiated"):
        q.geom.Dphi_eo(q.to_native(q.spinors[0][q.od], hirep.ODD), q.links_fund)


@pytest.mark.parametrize("bc", [(1, 1, 1, 1), (1, -1, 1, 1), (-1, -1, -1, -1), (-1, 1, 1, -1)])
def test_boundary_conditions(env, bc):
    cfg = synth.CONFIGS["C2"].resized(4, 4)
    check_all_ops(env, Problem(env, cfg, "f64", bc=bc))


def test_degenerate_extents(env):
    """Extent 2: the +mu and -mu neighbours are the same site (A8); smallest lattice pads one tile."""
    for T, L in [(2, 2), (4, 2), (2, 4)]:
        check_all_ops(env, Problem(env, synth.CONFIGS["C2"].resized(T, L), "f64"))
        check_all_ops(env, Problem(env, synth.CONFIGS["C3"].resized(T, L), "f32"))


def test_fp32_close_to_fp64(env):
    hirep = env["hirep"]
    cfg = synth.CONFIGS["C2"].resized(4, 4)
    p64, p32 = Problem(env, cfg, "f64"), Problem(env, cfg, "f32")
    a = p64.to_numpy(p64.geom.Dphi(cfg.m0, p64.to_native(p64.spinors[0], hirep.FULL), p64.links_rep), hirep.FULL)
    b = p32.to_numpy(p32.geom.Dphi(cfg.m0, p32.to_native(p32.spinors[0], hirep.FULL), p32.links_rep), hirep.FULL)
    assert env["oracle"].rel_l2(b, a) < 1e-6


def test_runtime_errors(env):
    hirep, torch = env["hirep"], env["torch"]
    p = Problem(env, synth.CONFIGS["C2"].resized(4, 4), "f64")
    x = p.to_native(p.spinors[0][p.od], hirep.ODD)
    p.geom.set_kernel_variant(99)
    with pytest.raises(hirep.HirepError, match="no kernel instantiated"):
        p.geom.Dphi_eo(x, p.links_rep)
    p.geom.set_kernel_variant(0)
    with pytest.raises(hirep.HirepError, match="alias"):
        p.geom.Dphi_eo(x, p.links_rep, out=x)
    p.geom.set_link_mode(hirep.LINKS_REBUILD)
    p.geom.set_link_mode(hirep.LINKS_STORED)
    before = p.geom.launch_count()
    p.geom.Dphi_hat(0.1, p.to_native(p.spinors[0][p.ev], hirep.EVEN), p.links_rep)
    assert p.geom.launch_count() - before == 3        # import + two stencil passes
    p.geom.sync()


def test_apply_host_end_to_end(env):
    """hirep_apply_host with pinned host buffers equals the oracle (and the device-resident path)."""
    torch, hirep, oracle = env["torch"], env["hirep"], env["oracle"]
    cfg = synth.CONFIGS["C2"].resized(4, 4)
    p = Problem(env, cfg, "f64")
    U_h = torch.from_numpy(p.U).pin_memory()
    psi = p.spinors[0]
    for op, inp, ref in [
        (hirep.OP_DPHI, psi, oracle.Dphi(4, 4, 3, cfg.m0, p.R, psi, BC)),
        (hirep.OP_DPHI_EO, psi[p.od], oracle.Dphi_eo(4, 4, 3, p.R, psi[p.od], BC)),
        (hirep.OP_DPHI_OE, psi[p.ev], oracle.Dphi_oe(4, 4, 3, p.R, psi[p.ev], BC)),
        (hirep.OP_DPHI_HAT, psi[p.ev], oracle.Dphi_hat(4, 4, 3, cfg.m0, p.R, psi[p.ev], BC)),
        (hirep.OP_G5DPHI_SQ, psi, oracle.g5Dphi_sq(4, 4, 3, cfg.m0, p.R, psi, BC)),
    ]:
        x_h = torch.from_numpy(np.ascontiguousarray(inp)).pin_memory()
        out = p.geom.apply_host(op, cfg.m0, x_h, U_h)
        assert oracle.rel_l2(out.numpy(), ref) < 1e-13
    # links stay resident when none are passed
    out = p.geom.apply_host(hirep.OP_DPHI, cfg.m0, torch.from_numpy(psi).pin_memory(), None)
    assert oracle.rel_l2(out.numpy(), oracle.Dphi(4, 4, 3, cfg.m0, p.R, psi, BC)) < 1e-13


def test_apply_host_async_pipeline(env):
    """hirep_apply_host_async: several calls in flight (results leave on a second stream from two staging buffers)
    give, after hirep_sync, bit for bit what the synchronous entry gives."""
    torch, hirep = env["torch"], env["hirep"]
    cfg = synth.CONFIGS["C2"].resized(6, 6)
    p = Problem(env, cfg, "f64")
    U_h = torch.from_numpy(p.U).pin_memory()
    psi = p.spinors[0]
    ins = {"f": torch.from_numpy(psi).pin_memory(), "e": torch.from_numpy(np.ascontiguousarray(psi[p.ev])).pin_memory(),
           "o": torch.from_numpy(np.ascontiguousarray(psi[p.od])).pin_memory()}
    seq = [(hirep.OP_DPHI_EO, "o", "e"), (hirep.OP_DPHI_OE, "e", "o"), (hirep.OP_DPHI, "f", "f"), (hirep.OP_DPHI_HAT, "e", "e"),
           (hirep.OP_G5DPHI_SQ, "f", "f"), (hirep.OP_DPHI_EO, "o", "e"), (hirep.OP_DPHI, "f", "f")]
    ref = [p.geom.apply_host(op, cfg.m0, ins[i], U_h if k == 0 else None) for k, (op, i, o) in enumerate(seq)]
    outs = [torch.empty_like(ins[o]).pin_memory() for (_, _, o) in seq]
    for rep in range(2):
        for k, (op, i, o) in enumerate(seq):
            hirep.hirep_apply_host_async(p.geom.handle, op, cfg.m0, outs[k].data_ptr(), ins[i].data_ptr(), U_h.data_ptr() if k == 0 else None)
        p.geom.sync()
        for k in range(len(seq)):
            assert torch.equal(outs[k], ref[k]), (rep, k)


# --------------------------------------------------------- full BASELINE sizes, sampled outputs
def full_size_problem(env, name, prec, rebuild=False):
    torch, hirep = env["torch"], env["hirep"]
    cfg = synth.CONFIGS[name]
    cdt = torch.complex128 if prec == "f64" else torch.complex64
    links, (psi,) = synth.make_inputs_torch(cfg, env["dev"], cdt, n_spinors=1)
    geom = hirep.Geometry(cfg.T, cfg.L, cfg.n_g, cfg.rep, prec, device=env["dev"])
    lf = geom.links_import(links)
    if rebuild:
        geom.set_link_mode(hirep.LINKS_REBUILD)   # the operators read the fundamental field
        return cfg, geom, links, psi, lf
    lr = geom.links_to_rep(lf)
    del lf
    torch.cuda.empty_cache()
    return cfg, geom, links, psi, lr


def half_canon(env, cfg, psi, parity):
    """canonical half-lattice spinor = rows of that parity in increasing ix; row of ix is ix >> 1"""
    torch = env["torch"]
    idx = torch.arange(cfg.volume, device=env["dev"])
    c = (idx // cfg.L ** 3) + (idx // cfg.L ** 2) % cfg.L + (idx // cfg.L) % cfg.L + idx % cfg.L
    return psi[(c % 2) == parity].contiguous()


def compare_sampled(out_canon, sites, ref_fn, row_of, tol, tag):
    num = den = 0.0
    for ix in sites:
        ref = ref_fn(ix)
        got = out_canon[row_of(ix)].cpu().numpy().astype(np.complex128)
        num += float(np.sum(np.abs(got - ref) ** 2)); den += float(np.sum(np.abs(ref) ** 2))
        assert np.linalg.norm(got - ref) <= 10 * tol * np.linalg.norm(ref), (tag, ix)
    assert np.sqrt(num / den) < tol, tag


NSAMP = 64      # sampled sites per operator: corners, the last tile of the kernels' grid rounds, random interior sites

FULL = [("C2", "f64"), ("C2", "f32"), ("C3", "f64"), ("C3", "f32"), ("C4", "f64"), ("C4", "f32"), ("C5", "f64"), ("C5", "f32")]


def run_sampled(env, name, prec, rebuild):
    torch, hirep, oracle = env["torch"], env["hirep"], env["oracle"]
    cfg, geom, links, psi, lk = full_size_problem(env, name, prec, rebuild)
    so = SampledOracle(oracle, cfg, links)
    fetch = torch_field_fetch(psi)
    tol = TOL[prec]
    tag = (name, prec, "rebuild" if rebuild else "stored")
    if "Dphi_eo" in cfg.ops:
        x = geom.spinor_import(half_canon(env, cfg, psi, 1), hirep.ODD)
        out = geom.spinor_export(geom.Dphi_eo(x, lk), hirep.EVEN)
        compare_sampled(out, sample_sites(cfg, NSAMP, parity=0, seed=1), lambda ix: so.hop(fetch, ix), half_rank, tol, tag + ("Dphi_eo",))
        del x, out
    if "Dphi_hat" in cfg.ops:
        x = geom.spinor_import(half_canon(env, cfg, psi, 0), hirep.EVEN)
        out = geom.spinor_export(geom.Dphi_hat(cfg.m0, x, lk), hirep.EVEN)
        compare_sampled(out, sample_sites(cfg, NSAMP, parity=0, seed=2), lambda ix: so.Dphi_hat(fetch, ix, cfg.m0), half_rank, tol, tag + ("Dphi_hat",))
        del x, out
    if "g5Dphi_sq" in cfg.ops:
        x = geom.spinor_import(psi, hirep.FULL)
        out = geom.spinor_export(geom.g5Dphi_sq(cfg.m0, x, lk), hirep.FULL)
        compare_sampled(out, sample_sites(cfg, NSAMP, seed=3), lambda ix: so.g5Dphi_sq(fetch, ix, cfg.m0), lambda ix: ix, tol, tag + ("g5Dphi_sq",))
        del x, out
    geom.sync()
    del lk, links, psi
    torch.cuda.empty_cache()


@pytest.mark.parametrize("name,prec", FULL)
def test_full_size_sampled(env, name, prec):
    """BASELINE lattice sizes, default launch configuration (the one bench.py times); outputs compared with the oracle on
    64 sampled sites per operator: the lattice corners (all boundary wraps), a site from the last tile of every grid
    round of the persistent kernels, random interior sites."""
    run_sampled(env, name, prec, rebuild=False)


@pytest.mark.parametrize("name", ["C4", "C5"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_full_size_sampled_rebuild(env, name, prec):
    """Link mode REBUILD (R rebuilt in the kernel from the fundamental links; C5: the matrix-free adjoint) at the full sizes
    bench.py times it on."""
    run_sampled(env, name, prec, rebuild=True)


def test_adjoint_matrix_free_capped_grid(env):
    """hop_adjmf.cuh with many site groups per warp (grid capped), SU(3) and SU(6), all operators."""
    hirep = env["hirep"]
    for n in (3, 6):
        p = Problem(env, synth.Config("t", 4, 6, n, ADJ, -0.4, "haar", 910 + n, ()), "f64")
        p.geom.set_tuning(hirep.TUNE_MAX_CTAS, 2)
        check_all_ops(env, p, rebuild=True)


# ------------------------------------------------ full BASELINE sizes, the WHOLE output field (C2: all ops; C3: Dphi_eo)
@pytest.mark.parametrize("name,prec", [("C2", "f64"), ("C2", "f32"), ("C3", "f64"), ("C3", "f32")])
def test_full_size_whole_field(env, name, prec):
    """Every output element of the bench launch configuration against the oracle at the BASELINE size: the oracle runs a
    32^4 step in ~2 s, so C2 (all five operators) and C3 (Dphi_eo) are compared over the whole field, not on samples."""
    torch, hirep, oracle = env["torch"], env["hirep"], env["oracle"]
    cfg, geom, links, psi, lr = full_size_problem(env, name, prec, rebuild=False)
    T, L, d, m0 = cfg.T, cfg.L, cfg.d_R, cfg.m0
    tol = TOL[prec]
    U = links.cpu().numpy().astype(np.complex128)
    psi_h = psi.cpu().numpy().astype(np.complex128)
    R = oracle.represent_field(cfg.n_g, cfg.rep, U)
    del U
    ev, od = synth.parity_sites(T, L, 0), synth.parity_sites(T, L, 1)
    imp = lambda a, w: geom.spinor_import(torch.from_numpy(np.ascontiguousarray(a)).to(env["dev"]), w)
    exp = lambda n, w: geom.spinor_export(n, w).cpu().numpy().astype(np.complex128)
    errs = {}
    errs["Dphi_eo"] = oracle.rel_l2(exp(geom.Dphi_eo(imp(psi_h[od], hirep.ODD), lr), hirep.EVEN), oracle.Dphi_eo(T, L, d, R, psi_h[od], BC))
    if name == "C2":
        errs["Dphi_oe"] = oracle.rel_l2(exp(geom.Dphi_oe(imp(psi_h[ev], hirep.EVEN), lr), hirep.ODD), oracle.Dphi_oe(T, L, d, R, psi_h[ev], BC))
        errs["Dphi_hat"] = oracle.rel_l2(exp(geom.Dphi_hat(m0, imp(psi_h[ev], hirep.EVEN), lr), hirep.EVEN), oracle.Dphi_hat(T, L, d, m0, R, psi_h[ev], BC))
        xf = imp(psi_h, hirep.FULL)
        errs["Dphi"] = oracle.rel_l2(exp(geom.Dphi(m0, xf, lr), hirep.FULL), oracle.Dphi(T, L, d, m0, R, psi_h, BC))
        errs["g5Dphi_sq"] = oracle.rel_l2(exp(geom.g5Dphi_sq(m0, xf, lr), hirep.FULL), oracle.g5Dphi_sq(T, L, d, m0, R, psi_h, BC))
    geom.sync()
    print(name, prec, {k: "%.2e" % v for k, v in errs.items()})
    for k, v in errs.items():
        assert v < tol, (name, prec, k, v)
    del lr, links, psi, R
    torch.cuda.empty_cache()


@pytest.mark.parametrize("name,prec,variant", [("C2", "f64", 0), ("C4", "f32", 0), ("C4", "f64", 5), ("C3", "f64", 0)])
def test_round_pacing_is_result_neutral(env, name, prec, variant):
    """HIREP_TUNE_PACE_WINDOW throttles leading warp groups of the tile-pair kernel; results are bit-identical with and without it
    (many rounds: 8x8^3 lattice on a capped grid, window 1 and 3)."""
    hirep = env["hirep"]
    p = Problem(env, synth.CONFIGS[name].resized(8, 8), prec)
    g = p.geom
    g.set_kernel_variant(variant)
    x = p.to_native(p.spinors[0], hirep.FULL)
    ref = g.Dphi(p.cfg.m0, x, p.links_rep).clone()
    for cap in (0, 5):
        g.set_tuning(hirep.TUNE_MAX_CTAS, cap)
        for w in (1, 3):
            g.set_tuning(hirep.TUNE_PACE_WINDOW, w)
            assert env["torch"].equal(g.Dphi(p.cfg.m0, x, p.links_rep), ref), (cap, w)
    g.set_tuning(hirep.TUNE_PACE_WINDOW, 0)
    check_all_ops(env, p, variant)
