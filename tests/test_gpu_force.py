"""GPU parity of the fermion force of the hopping term (Eq 20-21) against oracle/force.py,
element by element through the C-ABI.  Tolerance: relative L2 <= 1e-13 (fp64) / 1e-5 (fp32) over the force field, like the
operators (the force is a sum of ~16 d_R products per generator entry; fp32 runs feed the oracle the fp32-rounded inputs)."""
import numpy as np
import pytest

from harness import synth
from oracle import force as of
from tests.gpu_helpers import BC
from tests.test_gpu_parity import Problem, env, np_c  # noqa: F401  (env is a fixture)

pytestmark = pytest.mark.gpu

FUND, ADJ, SYM, ASY = 0, 1, 2, 3
TOL = {"f64": 1e-13, "f32": 1e-5}


def check_force(env, p, seed=0):
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = p.cfg
    eta, xi = p.spinors[0], p.spinors[1]
    F = p.geom.force_hopping(p.to_native(eta, hirep.FULL), p.to_native(xi, hirep.FULL), p.links_rep).cpu().numpy().astype(np.float64)
    ref = of.force_hopping(cfg.T, cfg.L, cfg.n_g, cfg.rep, p.R, eta, xi, p.bc)
    assert F.shape == ref.shape
    err = oracle.rel_l2(F, ref) if np.abs(ref).max() > 0 else float(np.abs(F).max())
    assert err < TOL[p.prec], (cfg.n_g, cfg.rep, p.prec, err)
    return err


@pytest.mark.parametrize("n,rep", [(2, FUND), (3, FUND), (4, FUND), (6, FUND), (2, ADJ), (3, ADJ), (4, ADJ), (6, ADJ), (2, SYM), (3, SYM), (4, SYM),
                                   (2, ASY), (3, ASY), (4, ASY), (6, ASY)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_force_all_representations(env, n, rep, prec):
    """6x4^3 (ragged last tile), antiperiodic in t and y: every representation the library instantiates."""
    cfg = synth.Config("t", 6, 4, n, rep, 0.0, "haar", 6000 + 10 * n + rep, ())
    check_force(env, Problem(env, cfg, prec, bc=(-1, 1, -1, 1), n_spinors=2))


@pytest.mark.parametrize("name,T,L", [("C1", 4, 4), ("C2", 6, 6), ("C3", 6, 6), ("C4", 6, 6), ("C5", 2, 4)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_force_baseline_configs_reduced(env, name, T, L, prec):
    check_force(env, Problem(env, synth.CONFIGS[name].resized(T, L), prec, n_spinors=2))


@pytest.mark.parametrize("n", [2, 3, 4, 5, 6])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_force_adjoint_matrix_free(env, n, prec):
    """Link mode REBUILD, adjoint representation: the commutator form on the FUNDAMENTAL links against the same oracle (and so against
    the sparse-generator kernel on the stored adjoint links); 6x4^3 with a ragged site-group tail, antiperiodic t and y."""
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.Config("t", 6, 4, n, ADJ, 0.0, "haar", 6100 + n, ())
    p = Problem(env, cfg, prec, bc=(-1, 1, -1, 1), n_spinors=2)
    eta, xi = p.spinors
    p.geom.set_link_mode(hirep.LINKS_REBUILD)
    F = p.geom.force_hopping(p.to_native(eta, hirep.FULL), p.to_native(xi, hirep.FULL), p.links_fund).cpu().numpy().astype(np.float64)
    ref = of.force_hopping(cfg.T, cfg.L, n, ADJ, p.R, eta, xi, p.bc)
    assert oracle.rel_l2(F, ref) < TOL[prec], (n, prec, oracle.rel_l2(F, ref))
    p.geom.set_link_mode(hirep.LINKS_STORED)
    G = p.geom.force_hopping(p.to_native(eta, hirep.FULL), p.to_native(xi, hirep.FULL), p.links_rep).cpu().numpy().astype(np.float64)
    assert oracle.rel_l2(F, G) < 10 * TOL[prec]


def test_force_degenerate_and_errors(env):
    hirep = env["hirep"]
    for T, L in [(2, 2), (4, 2)]:
        check_force(env, Problem(env, synth.CONFIGS["C2"].resized(T, L), "f64", n_spinors=2))
    p = Problem(env, synth.CONFIGS["C4"].resized(2, 4), "f64", n_spinors=2)
    e, x = p.to_native(p.spinors[0], hirep.FULL), p.to_native(p.spinors[1], hirep.FULL)
    p.geom.set_link_mode(hirep.LINKS_REBUILD)
    with pytest.raises(hirep.HirepError, match="stored represented links"):
        p.geom.force_hopping(e, x, p.links_fund)
    p.geom.set_link_mode(hirep.LINKS_STORED)
    a = p.geom.force_hopping(e, x, p.links_rep)
    b = p.geom.force_hopping(x, e, p.links_rep)          # Eq 20 is symmetric under eta <-> xi
    assert float((a - b).abs().max()) <= 1e-13 * float(a.abs().max())


def test_force_is_the_derivative_of_the_action_on_the_gpu(env):
    """End to end on the device: eta by hirep_cg_g5Dphi_sq, xi = gamma_5 D eta, F by hirep_force_hopping; then the action
    S = <psi, eta> is re-evaluated by the GPU CG with one link rotated by exp(+-i eps T^a): F = -(1/T_FUND) dS/d omega."""
    torch, hirep, oracle = env["torch"], env["hirep"], env["oracle"]
    cfg = synth.Config("t", 4, 4, 3, FUND, 0.4, "haar", 6400, ())
    p = Problem(env, cfg, "f64")
    g, m0 = p.geom, cfg.m0
    psi = p.to_native(p.spinors[0], hirep.FULL)

    def solve(U):
        lr = g.links_to_rep(g.links_import(torch.from_numpy(U)))
        eta, it, res = g.cg_g5Dphi_sq(m0, psi, lr, 1e-13, 2000)
        return lr, eta, float(g.prod(hirep.FULL, psi, eta).real)

    lr, eta, S0 = solve(p.U)
    xi = g.new_spinor(hirep.FULL)
    g.gamma(hirep.FULL, 5, xi, g.Dphi(m0, eta, lr))          # xi = Q_m eta = gamma_5 D_m eta
    F = g.force_hopping(eta, xi, lr).cpu().numpy()
    Tf = oracle.generators(3)
    eps = 1e-4
    for ix, mu, a in [(cfg.volume - 1, 0, 3), (17, 2, 7), (100, 1, 0)]:
        w, v = np.linalg.eigh(Tf[a])
        Ss = []
        for sgn in (+1, -1):
            U = p.U.copy()
            U[ix, mu] = ((v * np.exp(1j * sgn * eps * w)) @ v.conj().T) @ U[ix, mu]
            Ss.append(solve(U)[2])
        dS = (Ss[0] - Ss[1]) / (2 * eps)
        assert abs(F[ix, mu, a] + 2.0 * dS) < 1e-5 * max(1.0, abs(dS)), (ix, mu, a, F[ix, mu, a], -2 * dS)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_force_full_size_C2_whole_field(env, prec):
    """BASELINE configs[1] size (32^4): the whole force field against the oracle."""
    torch, hirep, oracle = env["torch"], env["hirep"], env["oracle"]
    cfg = synth.CONFIGS["C2"]
    cdt = torch.complex128 if prec == "f64" else torch.complex64
    links, (eta, xi) = synth.make_inputs_torch(cfg, env["dev"], cdt, n_spinors=2)
    geom = hirep.Geometry(cfg.T, cfg.L, cfg.n_g, cfg.rep, prec, device=env["dev"])
    lr = geom.links_to_rep(geom.links_import(links))
    F = geom.force_hopping(geom.spinor_import(eta, hirep.FULL), geom.spinor_import(xi, hirep.FULL), lr).cpu().numpy().astype(np.float64)
    R = oracle.represent_field(cfg.n_g, cfg.rep, links.cpu().numpy().astype(np.complex128))
    ref = of.force_hopping(cfg.T, cfg.L, cfg.n_g, cfg.rep, R, eta.cpu().numpy().astype(np.complex128), xi.cpu().numpy().astype(np.complex128), BC)
    assert oracle.rel_l2(F, ref) < TOL[prec]
