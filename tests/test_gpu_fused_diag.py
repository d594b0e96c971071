"""GPU parity of the operators with site-diagonal matrices in BOTH of their forms ("fused into the
second pass"; Eq 43, Eq 47-50): fused = the matrices are applied inside the stencil epilogues (one launch per
stencil pass: Dphi_clover / Dphi_blocks 1 launch, the Schur forms 2), composed = separate block-apply launches (2 resp. 4;
hirep_set_tuning(HIREP_TUNE_FUSE_DIAG, 0)).  Each form is compared with oracle/clover.py element by element at the usual
tolerances, and the launch counts prove which form ran."""
import numpy as np
import pytest

from harness import synth
from tests.gpu_helpers import BC, TOL
from tests.test_gpu_parity import Problem, env  # noqa: F401  (env is a fixture)

pytestmark = pytest.mark.gpu

# (config, T, L, fused form instantiated in fp64, in fp32): ring kernel d_R <= 4 in fp64, <= 6 in fp32, pair kernel d_R = 5, 6;
# C3 has real links; C5 (d_R = 35, row-group kernel) keeps the composed form
CASES = [("C1", 4, 4, True, True), ("C2", 6, 6, True, True), ("C3", 4, 8, True, True), ("C4", 4, 6, True, True), ("C5", 2, 4, False, False)]


def launches(g, fn):
    n0 = g.launch_count()
    out = fn()
    return out, g.launch_count() - n0


@pytest.mark.parametrize("name,T,L,f64_fused,f32_fused", CASES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("max_ctas", [0, 2])
def test_fused_and_composed_forms(env, name, T, L, f64_fused, f32_fused, prec, max_ctas):
    """Dphi_clover, Dphi_clover_hat, Dphi_blocks, Dphi_blocks_hat (exponential clover): both forms against the oracle.
    max_ctas = 2: a capped persistent grid, every warp walks several tiles (the ring runs across tile boundaries with the
    matrix pieces between the link chunks of consecutive tiles)."""
    from oracle import clover as oc
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS[name].resized(T, L)
    p = Problem(env, cfg, prec)
    g, m0, tol = p.geom, cfg.m0, TOL[prec]
    fused_here = f64_fused if prec == "f64" else f32_fused
    g.set_tuning(hirep.TUNE_MAX_CTAS, max_ctas)
    cl = g.clover_field(p.links_rep)
    psi = p.spinors[0]
    x = p.to_native(psi, hirep.FULL)
    xe = p.to_native(psi[p.ev], hirep.EVEN)
    csw_c, csw_s, csw_e = 1.7, 0.5, 1.2
    inv_odd = g.clover_inv_field(m0, csw_s, hirep.ODD, cl)
    E = g.clover_exp_field(m0, csw_e, cl)
    Ei = g.clover_exp_field(m0, csw_e, cl, inverse=True)
    nb = E.numel() // 2
    want = {
        "Dphi_clover": oc.Dphi_clover(T, L, m0, csw_c, p.R, psi, BC),
        "Dphi_clover_hat": oc.Dphi_clover_hat(T, L, m0, csw_s, p.R, psi[p.ev], BC),
        "Dphi_blocks": oc.Dphi_expclover(T, L, m0, csw_e, p.R, psi, BC),
        "Dphi_blocks_hat": oc.Dphi_expclover_hat(T, L, m0, csw_e, p.R, psi[p.ev], BC),
    }
    results = {}
    for fuse in (1, 0):
        g.set_tuning(hirep.TUNE_FUSE_DIAG, fuse)
        full = 1 if (fuse and fused_here) else 2
        hat = 2 if (fuse and fused_here) else 4
        out, n = launches(g, lambda: g.Dphi_clover(m0, csw_c, x, p.links_rep, cl))
        assert n == full
        results[("Dphi_clover", fuse)] = p.to_numpy(out, hirep.FULL)
        out, n = launches(g, lambda: g.Dphi_clover_hat(m0, csw_s, xe, p.links_rep, cl, inv_odd))
        assert n == hat
        results[("Dphi_clover_hat", fuse)] = p.to_numpy(out, hirep.EVEN)
        out, n = launches(g, lambda: g.Dphi_blocks(x, p.links_rep, E))
        assert n == full
        results[("Dphi_blocks", fuse)] = p.to_numpy(out, hirep.FULL)
        out, n = launches(g, lambda: g.Dphi_blocks_hat(xe, p.links_rep, E, Ei[nb:]))
        assert n == hat
        results[("Dphi_blocks_hat", fuse)] = p.to_numpy(out, hirep.EVEN)
    for (op, fuse), got in results.items():
        assert np.isfinite(got).all(), (op, fuse)
        assert oracle.rel_l2(got, want[op]) < tol, (op, fuse)
        assert np.abs(got - want[op]).max() < 100 * tol * np.abs(want[op]).max(), (op, fuse)


@pytest.mark.parametrize("n,rep,T,L,prec,variant", [(2, 3, 4, 4, "f64", 0), (2, 0, 2, 6, "f64", 0), (4, 0, 4, 4, "f64", 0), (5, 0, 4, 2, "f64", 0),
                                                    (3, 2, 4, 4, "f64", 0), (2, 2, 4, 4, "f32", 0), (3, 3, 2, 6, "f32", 0), (5, 0, 4, 2, "f32", 0),
                                                    (3, 2, 4, 4, "f32", 0), (4, 0, 6, 4, "f32", 0), (5, 0, 4, 2, "f32", 4), (3, 2, 2, 6, "f32", 4),
                                                    (3, 0, 4, 4, "f64", 3)])
def test_fused_form_every_instantiation(env, n, rep, T, L, prec, variant):
    """d_R = 1 (SU(2) 2AS: one-entry ring slots), 2, 4 (ring kernel), 5, 6 (pair kernel) in fp64; d_R = 3, 3, 5, 6, 4 in fp32 (ring
    kernel) and d_R = 5, 6 on the pair kernel (variant 4) -- every d_R the fused epilogue is instantiated for beyond the BASELINE
    configs; ragged tails (4^4: 4 tiles; 2x6^3: 6.75 tiles)."""
    from oracle import clover as oc
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.Config("t", T, L, n, rep, -0.15, "haar", 29, ())
    p = Problem(env, cfg, prec)
    g, m0, tol = p.geom, cfg.m0, TOL[prec]
    g.set_kernel_variant(variant)
    cl = g.clover_field(p.links_rep)
    psi = p.spinors[0]
    x = p.to_native(psi, hirep.FULL)
    xe = p.to_native(psi[p.ev], hirep.EVEN)
    out, nl = launches(g, lambda: g.Dphi_clover(m0, 0.9, x, p.links_rep, cl))
    assert nl == 1
    assert oracle.rel_l2(p.to_numpy(out, hirep.FULL), oc.Dphi_clover(T, L, m0, 0.9, p.R, psi, BC)) < tol
    inv_odd = g.clover_inv_field(m0, 0.4, hirep.ODD, cl)
    out, nl = launches(g, lambda: g.Dphi_clover_hat(m0, 0.4, xe, p.links_rep, cl, inv_odd))
    assert nl == 2
    assert oracle.rel_l2(p.to_numpy(out, hirep.EVEN), oc.Dphi_clover_hat(T, L, m0, 0.4, p.R, psi[p.ev], BC)) < tol
    E = g.clover_exp_field(m0, 0.8, cl)
    Ei = g.clover_exp_field(m0, 0.8, cl, inverse=True)
    out, nl = launches(g, lambda: g.Dphi_blocks(x, p.links_rep, E))
    assert nl == 1
    assert oracle.rel_l2(p.to_numpy(out, hirep.FULL), oc.Dphi_expclover(T, L, m0, 0.8, p.R, psi, BC)) < tol
    out, nl = launches(g, lambda: g.Dphi_blocks_hat(xe, p.links_rep, E, Ei[E.numel() // 2:]))
    assert nl == 2
    assert oracle.rel_l2(p.to_numpy(out, hirep.EVEN), oc.Dphi_expclover_hat(T, L, m0, 0.8, p.R, psi[p.ev], BC)) < tol


@pytest.mark.parametrize("name,T,L,prec", [("C2", 4, 6, "f64"), ("C4", 4, 4, "f64"), ("C3", 4, 4, "f64"), ("C4", 4, 4, "f32"), ("C2", 4, 4, "f32")])
def test_fused_form_g5_squares_and_cg(env, name, T, L, prec):
    """(gamma_5 D_clover)^2 and the even-odd (gamma_5 D_hat)^2 run on the fused passes (2 resp. 4 launches) and agree with the
    composed forms to rounding; the clover CGs -- whose two reductions then ride in the epilogues of those passes (ring kernel: C2,
    C3 with real links, C4 in fp32; pair kernel: C4 in fp64) -- converge to the same solution in both forms."""
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS[name].resized(T, L)
    p = Problem(env, cfg, prec)
    g, m0 = p.geom, 0.3
    tol, cg_tol, sol_tol = (1e-13, 1e-10, 1e-7) if prec == "f64" else (1e-5, 1e-5, 2e-3)
    cl = g.clover_field(p.links_rep)
    inv_odd = g.clover_inv_field(m0, 0.6, hirep.ODD, cl)
    psi = p.spinors[0]
    x = p.to_native(psi, hirep.FULL)
    xe = p.to_native(psi[p.ev], hirep.EVEN)
    res = {}
    for fuse in (1, 0):
        g.set_tuning(hirep.TUNE_FUSE_DIAG, fuse)
        out, n = launches(g, lambda: g.g5Dphi_clover_sq(m0, 0.6, x, p.links_rep, cl))
        assert n == (2 if fuse else 4)
        res[("sq", fuse)] = p.to_numpy(out, hirep.FULL)
        out, n = launches(g, lambda: g.g5Dphi_clover_hat_sq(m0, 0.6, xe, p.links_rep, cl, inv_odd))
        assert n == (4 if fuse else 8)
        res[("hat_sq", fuse)] = p.to_numpy(out, hirep.EVEN)
        sol, it, rel = g.cg_g5Dphi_clover_sq(m0, 0.6, x, p.links_rep, cl, cg_tol, 500)
        assert rel <= cg_tol
        res[("cg", fuse)] = p.to_numpy(sol, hirep.FULL)
        res[("cg_it", fuse)] = it
        sol, it, rel = g.cg_g5Dphi_clover_hat_sq(m0, 0.6, xe, p.links_rep, cl, inv_odd, cg_tol, 500)
        assert rel <= cg_tol
        res[("cg_hat", fuse)] = p.to_numpy(sol, hirep.EVEN)
        res[("cg_hat_it", fuse)] = it
    assert oracle.rel_l2(res[("sq", 1)], res[("sq", 0)]) < tol
    assert oracle.rel_l2(res[("hat_sq", 1)], res[("hat_sq", 0)]) < tol
    assert oracle.rel_l2(res[("cg", 1)], res[("cg", 0)]) < sol_tol
    assert oracle.rel_l2(res[("cg_hat", 1)], res[("cg_hat", 0)]) < sol_tol
    assert abs(res[("cg_it", 1)] - res[("cg_it", 0)]) <= 2 and abs(res[("cg_hat_it", 1)] - res[("cg_hat_it", 0)]) <= 2
    # true residual of the fused solution through the composed operator
    g.set_tuning(hirep.TUNE_FUSE_DIAG, 0)
    Ax = p.to_numpy(g.g5Dphi_clover_hat_sq(m0, 0.6, p.to_native(res[("cg_hat", 1)], hirep.EVEN), p.links_rep, cl, inv_odd), hirep.EVEN)
    b = psi[p.ev]
    assert np.linalg.norm((Ax - b).ravel()) < 20 * cg_tol * np.linalg.norm(b.ravel())


def test_full_size_fused_clover_C4_f64(env):
    """The 2-index BASELINE config at full size (SU(4) 2AS, 96 x 48^3, fp64), bench launch configuration: Dphi_clover through the pair
    kernel's fused epilogue (one launch) at sampled sites incl. the lattice corners.  The clover term at x only involves links in
    the 3^4 neighbourhood of x: the oracle runs, as it stands, on that neighbourhood cut out as a 3 x 3^3 lattice and is read at the
    centre; the hopping term comes from the sampled oracle of the Wilson tests (tests/gpu_helpers.py).  (The block export of
    tests/test_gpu_clover.py::test_full_size_clover_sampled would not fit beside the 49 GB of links here.)"""
    import itertools
    from oracle import clover as oc
    from tests.gpu_helpers import SampledOracle, coords_of, index_of, sample_sites, torch_field_fetch
    from tests.test_gpu_parity import full_size_problem
    torch, hirep, oracle = env["torch"], env["hirep"], env["oracle"]
    cfg, geom, links, psi, lr = full_size_problem(env, "C4", "f64")
    so = SampledOracle(oracle, cfg, links)
    fetch = torch_field_fetch(psi)
    tol, m0, csw, d = TOL["f64"], cfg.m0, 1.3, cfg.d_R
    ext = np.array([cfg.T, cfg.L, cfg.L, cfg.L])
    cl = geom.clover_field(lr)
    x = geom.spinor_import(psi, hirep.FULL)
    y, n = launches(geom, lambda: geom.Dphi_clover(m0, csw, x, lr, cl))
    assert n == 1
    out_d = geom.spinor_export(y, hirep.FULL)
    del y, x
    centre = index_of((1, 1, 1, 1), 3)
    num = den = 0.0
    for ix in sample_sites(cfg, 8, seed=11):
        c = coords_of(ix, cfg.T, cfg.L)
        idx = [index_of((c + np.array(off) - 1) % ext, cfg.L) for off in itertools.product(range(3), repeat=4)]
        Up = links[torch.tensor(idx, device=links.device)].cpu().numpy().astype(np.complex128)          # [81,4,N,N]
        Rp = np.array([[oracle.rep_matrix(cfg.n_g, cfg.rep, Up[s, mu]) for mu in range(4)] for s in range(81)])
        pp = np.zeros((81, 4, d), dtype=np.complex128)
        pp[centre] = fetch(ix)
        want = oc.Cphi(3, 3, m0, csw, Rp, pp)[centre] + so.hop(fetch, ix)
        got = out_d[ix].cpu().numpy().astype(np.complex128)
        assert np.linalg.norm(got - want) <= 10 * tol * np.linalg.norm(want), ix
        num += float(np.sum(np.abs(got - want) ** 2)); den += float(np.sum(np.abs(want) ** 2))
    assert np.sqrt(num / den) < tol
    geom.sync()
    del cl, out_d, lr, links, psi
    torch.cuda.empty_cache()
