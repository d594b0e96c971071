"""GPU parity of the twisted-mass operators (Eq 51) and their even-odd Schur form (Eq 43) -- the first part
of SURVEY.md 8(f) NEXT-2 -- against oracle.Dphi_tm / Dphi_tm_hat / Dphi_tm_sq / g5_lc, through the C-ABI binding.
Same tolerances as the Wilson operators: relative L2 <= 1e-13 (fp64) / 1e-5 (fp32)."""
import numpy as np
import pytest

from harness import synth
from tests.gpu_helpers import BC, TOL
from tests.test_gpu_parity import Problem, env  # noqa: F401  (env is a fixture)

pytestmark = pytest.mark.gpu

# every kernel family: ring (C1, C2, C3), pair (C4), rows (C5); ragged tails and whole tiles
CASES = [("C1", 4, 4), ("C2", 6, 6), ("C3", 4, 8), ("C4", 4, 6), ("C5", 2, 4)]


@pytest.mark.parametrize("name,T,L", CASES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("mu", [0.35, -1.2])
def test_twisted_mass_operators(env, name, T, L, prec, mu):
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS[name].resized(T, L)
    p = Problem(env, cfg, prec)
    g, d, m0, tol = p.geom, cfg.d_R, cfg.m0, TOL[prec]
    psi = p.spinors[0]
    x = p.to_native(psi, hirep.FULL)
    got = p.to_numpy(g.Dphi_tm(m0, mu, x, p.links_rep), hirep.FULL)
    assert oracle.rel_l2(got, oracle.Dphi_tm(T, L, d, m0, mu, p.R, psi, BC)) < tol
    got = p.to_numpy(g.Dphi_tm_sq(m0, mu, x, p.links_rep), hirep.FULL)
    assert oracle.rel_l2(got, oracle.Dphi_tm_sq(T, L, d, m0, mu, p.R, psi, BC)) < tol
    xe = p.to_native(psi[p.ev], hirep.EVEN)
    got = p.to_numpy(g.Dphi_tm_hat(m0, mu, xe, p.links_rep), hirep.EVEN)
    assert oracle.rel_l2(got, oracle.Dphi_tm_hat(T, L, d, m0, mu, p.R, psi[p.ev], BC)) < tol
    # mu -> 0 leaves the Wilson results bit-for-bit (the twisted term is skipped, not multiplied by zero)
    a = p.to_numpy(g.Dphi_tm(m0, 0.0, x, p.links_rep), hirep.FULL)
    b = p.to_numpy(g.Dphi(m0, x, p.links_rep), hirep.FULL)
    assert np.array_equal(a, b)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("which", ["full", "even", "odd"])
def test_g5_linear_combination(env, prec, which):
    hirep, oracle = env["hirep"], env["oracle"]
    p = Problem(env, synth.CONFIGS["C4"].resized(2, 6), prec)
    w = {"full": hirep.FULL, "even": hirep.EVEN, "odd": hirep.ODD}[which]
    sel = {"full": slice(None), "even": p.ev, "odd": p.od}[which]
    eta = p.spinors[0][sel]
    c1, c2 = 0.75 - 0.5j, -1.25 + 2.0j
    e = p.to_native(eta, w)
    xi = p.geom.new_spinor(w)
    p.geom.g5_lc(w, xi, c1, c2, e)
    assert oracle.rel_l2(p.to_numpy(xi, w), oracle.g5_lc(c1, c2, eta)) < TOL[prec]
    # in place, pure gamma_5: bit exact sign flips of the lower components
    p.geom.g5_lc(w, e, 0.0, 1.0, e)
    assert np.array_equal(p.to_numpy(e, w), oracle.g5(eta))


def test_twisted_mass_rebuild_mode_and_persistent_grid(env):
    """The twisted diagonal term through link mode REBUILD and a capped grid (many tiles per warp)."""
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS["C4"].resized(4, 8)
    p = Problem(env, cfg, "f64")
    p.geom.set_tuning(hirep.TUNE_MAX_CTAS, 2)
    psi, mu = p.spinors[0], 0.4
    ref = oracle.Dphi_tm_hat(cfg.T, cfg.L, cfg.d_R, cfg.m0, mu, p.R, psi[p.ev], BC)
    xe = p.to_native(psi[p.ev], hirep.EVEN)
    assert oracle.rel_l2(p.to_numpy(p.geom.Dphi_tm_hat(cfg.m0, mu, xe, p.links_rep), hirep.EVEN), ref) < 1e-13
    p.geom.set_link_mode(hirep.LINKS_REBUILD)
    assert oracle.rel_l2(p.to_numpy(p.geom.Dphi_tm_hat(cfg.m0, mu, xe, p.links_fund), hirep.EVEN), ref) < 1e-13


def test_twisted_mass_schur_form_fused_and_fallback(env):
    """Dphi_tm_hat applies D_oo^-1 = (a - i mu gamma_5)/(a^2 + mu^2) in the epilogue of its D_oe pass (2 launches) on the persistent
    kernels -- here also the matrix-free adjoint (C5 in link mode REBUILD) and the explicit variants 3, 4 -- and falls back to the separate
    gamma_5 combination (3 launches) on the direct-load kernels (variants 1, 2)."""
    hirep, oracle = env["hirep"], env["oracle"]
    mu = -0.7
    cfg = synth.CONFIGS["C5"].resized(2, 4)
    p = Problem(env, cfg, "f64")
    psi = p.spinors[0]
    ref = oracle.Dphi_tm_hat(cfg.T, cfg.L, cfg.d_R, cfg.m0, mu, p.R, psi[p.ev], BC)
    xe = p.to_native(psi[p.ev], hirep.EVEN)
    p.geom.set_link_mode(hirep.LINKS_REBUILD)
    n0 = p.geom.launch_count()
    y = p.geom.Dphi_tm_hat(cfg.m0, mu, xe, p.links_fund)
    assert p.geom.launch_count() - n0 == 2
    assert oracle.rel_l2(p.to_numpy(y, hirep.EVEN), ref) < 1e-13
    for prec in ("f64", "f32"):
        cfg = synth.CONFIGS["C2"].resized(4, 6)
        p = Problem(env, cfg, prec)
        psi = p.spinors[0]
        ref = oracle.Dphi_tm_hat(cfg.T, cfg.L, cfg.d_R, cfg.m0, mu, p.R, psi[p.ev], BC)
        xe = p.to_native(psi[p.ev], hirep.EVEN)
        for variant, nl in ((0, 2), (3, 2), (4, 2), (1, 3), (2, 3)):
            p.geom.set_kernel_variant(variant)
            n0 = p.geom.launch_count()
            y = p.geom.Dphi_tm_hat(cfg.m0, mu, xe, p.links_rep)
            assert p.geom.launch_count() - n0 == nl, (prec, variant)
            assert oracle.rel_l2(p.to_numpy(y, hirep.EVEN), ref) < TOL[prec], (prec, variant)


def test_twisted_mass_cg(env):
    """CG on (D^tm)^dag D^tm: the twist lifts the spectrum by mu^2, so the solve needs fewer iterations than mu = 0;
    solution against the oracle's CG and the true residual through the oracle operator."""
    from oracle import linalg as la
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS["C2"].resized(4, 4)
    p = Problem(env, cfg, "f64")
    T, L, d, m0, mu = 4, 4, cfg.d_R, 0.2, 0.5
    b = p.spinors[0]
    A = lambda v: oracle.Dphi_tm_sq(T, L, d, m0, mu, p.R, v, BC)
    x_ref, it_ref, _, _ = la.cg(A, b, 1e-10, 3000)
    xs, it, res = p.geom.cg_Dphi_tm_sq(m0, mu, p.to_native(b, hirep.FULL), p.links_rep, 1e-10, 3000)
    x = p.to_numpy(xs, hirep.FULL)
    assert res <= 1e-10 and abs(it - it_ref) <= 2
    assert oracle.rel_l2(x, x_ref) < 1e-7
    assert np.linalg.norm((b - A(x)).ravel()) < 1e-9 * np.linalg.norm(b.ravel())
    _, it0, _ = p.geom.cg_g5Dphi_sq(m0, p.to_native(b, hirep.FULL), p.links_rep, 1e-10, 3000)
    assert it < it0
    # the solve above ran with the reductions in the stencil epilogues (tile-pair kernel, 5 launches per iteration); the explicit
    # ring variant runs the separate reduction kernels (7): same solution
    n0 = p.geom.launch_count()
    p.geom.cg_Dphi_tm_sq(m0, mu, p.to_native(b, hirep.FULL), p.links_rep, 1e-30, 4)
    fused_launches = p.geom.launch_count() - n0
    p.geom.set_kernel_variant(3)
    n0 = p.geom.launch_count()
    p.geom.cg_Dphi_tm_sq(m0, mu, p.to_native(b, hirep.FULL), p.links_rep, 1e-30, 4)
    assert p.geom.launch_count() - n0 > fused_launches
    xs3, it3, res3 = p.geom.cg_Dphi_tm_sq(m0, mu, p.to_native(b, hirep.FULL), p.links_rep, 1e-10, 3000)
    assert res3 <= 1e-10 and abs(it3 - it) <= 2
    assert oracle.rel_l2(p.to_numpy(xs3, hirep.FULL), x) < 1e-7


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_g5_fused_forms(env, prec):
    """The gamma_5 add-mul-assign form and the fused reduction <xi, gamma_5 eta> against the oracle
    composition g5() + lc / prod."""
    from oracle import linalg as la
    hirep, oracle = env["hirep"], env["oracle"]
    p = Problem(env, synth.CONFIGS["C3"].resized(4, 6), prec, n_spinors=2)
    xi0, eta0 = p.spinors
    for w, sel in ((hirep.FULL, slice(None)), (hirep.ODD, p.od)):
        a, b = xi0[sel], eta0[sel]
        c0, c1, c2 = 0.5 + 0.25j, -1.5j, 2.0 - 1.0j
        xi, e = p.to_native(a, w), p.to_native(b, w)
        p.geom.g5_lc_add_assign(w, xi, c0, c1, c2, e)
        assert oracle.rel_l2(p.to_numpy(xi, w), c0 * a + oracle.g5_lc(c1, c2, b)) < TOL[prec]
        got = p.geom.g5_prod(w, p.to_native(a, w), e)
        ref = la.prod(a, oracle.g5(b))
        mag = float(np.sum(np.abs(a) * np.abs(b))) * 2
        assert abs(got - ref) <= 8 * 2.0 ** -52 * mag
        assert abs(got - ref) <= 1e-12 * mag


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_gamma_matrix_application(env, prec):
    """Eq 34: xi = gamma_mu eta against the oracle's 4x4 gamma matrices (Eq 1-3); sign flips and factors of i only,
    so the result is bit exact.  Ragged lattice, every extent selector."""
    hirep, oracle = env["hirep"], env["oracle"]
    p = Problem(env, synth.CONFIGS["C4"].resized(2, 6), prec)
    gam = {mu: oracle.gamma()[mu] for mu in range(4)}
    gam[5] = oracle.gamma5()
    for w, sel in ((hirep.FULL, slice(None)), (hirep.EVEN, p.ev), (hirep.ODD, p.od)):
        eta = p.spinors[0][sel]
        e = p.to_native(eta, w)
        for mu in (0, 1, 2, 3, 5):
            xi = p.geom.new_spinor(w)
            p.geom.gamma(w, mu, xi, e)
            assert np.array_equal(p.to_numpy(xi, w), np.einsum("ab,xbi->xai", gam[mu], eta)), mu
    with pytest.raises(hirep.HirepError):
        p.geom.gamma(hirep.FULL, 4, p.geom.new_spinor(hirep.FULL), p.to_native(p.spinors[0], hirep.FULL))
