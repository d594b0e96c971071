"""GPU parity of the spinor linear algebra, the reductions and the CG inverter against
oracle/linalg.py, through the C-ABI binding.

Tolerances: linear combinations -- relative L2 <= 1e-13 (fp64) / 1e-5 (fp32) like the operators (one or two
roundings per element); reductions -- the GPU's Neumaier sum against the correctly rounded sum of the same fp64
products: |diff| <= 4 ulp of sum|terms| (compensated summation leaves O(eps) relative to the result plus the
products' own rounding, which both sides share); max norm -- bit exact; CG -- both sides run the same recurrence to
tol = 1e-10, so the two solutions differ by at most ~2 tol cond(Q^2): checked at 1e-7, and the true residual of the
GPU solution (oracle operator) at 1e-9.
"""
import numpy as np
import pytest

from oracle import linalg as la
from harness import synth
from tests.gpu_helpers import BC
from tests.test_gpu_parity import Problem, env, np_c  # noqa: F401  (env is a fixture)

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-13, "f32": 1e-5}
CASES = [("C2", 6, 6), ("C3", 4, 8), ("C4", 2, 6)]     # ragged tail (Nh % 32 != 0) and whole tiles


def fields(p, n, seed):
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(n):
        f = synth.gaussian_spinor(rng, p.cfg.volume, p.cfg.d_R)
        out.append(synth.round_to_precision(f, p.prec))
    return out


@pytest.mark.parametrize("name,T,L", CASES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("which", ["full", "even", "odd"])
def test_linear_combinations(env, name, T, L, prec, which):
    hirep, oracle = env["hirep"], env["oracle"]
    p = Problem(env, synth.CONFIGS[name].resized(T, L), prec)
    w = {"full": hirep.FULL, "even": hirep.EVEN, "odd": hirep.ODD}[which]
    sel = {"full": slice(None), "even": p.ev, "odd": p.od}[which]
    xi0, eta0, zeta0 = [f[sel] for f in fields(p, 3, 42)]
    g = p.geom
    nat = lambda f: p.to_native(f, w)
    c1, c2, r1, r2 = 0.75 - 1.25j, -0.5 + 2.0j, 1.5, -0.625
    cases = [
        ("lc", lambda xi, e, z: g.lc(w, xi, r1, e, r2, z), la.lc(r1, eta0, r2, zeta0)),
        ("clc", lambda xi, e, z: g.clc(w, xi, c1, e, c2, z), la.clc(c1, eta0, c2, zeta0)),
        ("lc_add_assign", lambda xi, e, z: g.lc_add_assign(w, xi, r1, e, r2, z), la.lc_add_assign(xi0, r1, eta0, r2, zeta0)),
        ("clc_add_assign", lambda xi, e, z: g.clc_add_assign(w, xi, c1, e, c2, z), la.clc_add_assign(xi0, c1, eta0, c2, zeta0)),
        ("lc1", lambda xi, e, z: g.lc1(w, xi, c1, e), la.lc1(xi0, c1, eta0)),
        ("lc2", lambda xi, e, z: g.lc2(w, xi, c1, c2, e), la.lc2(xi0, c1, c2, eta0)),
        ("lc3", lambda xi, e, z: g.lc3(w, xi, c1, e, c2, z), la.lc3(xi0, c1, eta0, c2, zeta0)),
    ]
    for nm, run, ref in cases:
        xi, e, z = nat(xi0), nat(eta0), nat(zeta0)
        run(xi, e, z)
        got = p.to_numpy(xi, w)
        assert oracle.rel_l2(got, ref) < TOL[prec], nm
        # inputs untouched
        assert np.array_equal(p.to_numpy(e, w), eta0) and np.array_equal(p.to_numpy(z, w), zeta0), nm


@pytest.mark.parametrize("name,T,L", CASES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_reductions(env, name, T, L, prec):
    hirep = env["hirep"]
    p = Problem(env, synth.CONFIGS[name].resized(T, L), prec)
    xi0, eta0 = fields(p, 2, 7)
    # plant the maximum on an imaginary part with negative sign, and make the sum ill conditioned
    xi0[5, 1, 0] = complex(0.25, -7.5)
    eps = 2.0 ** -52
    for w, sel in ((hirep.FULL, slice(None)), (hirep.EVEN, p.ev), (hirep.ODD, p.od)):
        a, b = xi0[sel], eta0[sel]
        xa, xb = p.to_native(a, w), p.to_native(b, w)
        mag = float(np.sum(np.abs(a.real * b.real)) + np.sum(np.abs(a.imag * b.imag)) + np.sum(np.abs(a.real * b.imag)) + np.sum(np.abs(a.imag * b.real)))
        got, ref = p.geom.prod(w, xa, xb), la.prod(a, b)
        assert abs(got - ref) <= 4 * eps * mag
        assert abs(got - ref) <= 1e-13 * abs(ref) + 4 * eps * mag
        n_got, n_ref = p.geom.sqnorm(w, xa), la.sqnorm(a)
        assert abs(n_got - n_ref) <= 4 * eps * n_ref
        assert p.geom.max_norm(w, xa) == la.max_norm(a)              # bit exact
    # conj on the left: <xi,eta> = conj <eta,xi>
    xa, xb = p.to_native(xi0, hirep.FULL), p.to_native(eta0, hirep.FULL)
    assert p.geom.prod(hirep.FULL, xb, xa) == p.geom.prod(hirep.FULL, xa, xb).conjugate()


def test_reduction_is_compensated(env):
    """A sum that naive fp64 accumulation gets wrong by many ulps: 2^20 terms of size ~1 plus a few of size 2^40.
    The GPU result must be within 2 ulp of the exact sum (Algorithm 2), far below the naive error."""
    hirep = env["hirep"]
    cfg = synth.CONFIGS["C2"].resized(8, 8)
    p = Problem(env, cfg, "f64")
    rng = np.random.default_rng(99)
    f = (rng.uniform(0.5, 1.5, size=(cfg.volume, 4, cfg.d_R)) + 1j * rng.uniform(0.5, 1.5, size=(cfg.volume, 4, cfg.d_R)))
    f[::997, 0, 0] = 2.0 ** 20
    ref = la.sqnorm(f)
    got = p.geom.sqnorm(hirep.FULL, p.to_native(f, hirep.FULL))
    assert abs(got - ref) <= 2 * 2.0 ** -52 * ref
    naive = la.naive_sum(np.concatenate([f.real.ravel() ** 2, f.imag.ravel() ** 2]).tolist())
    assert abs(naive - ref) > 8 * 2.0 ** -52 * ref


@pytest.mark.parametrize("alg", [2, 3, 4])
def test_summation_algorithms(env, alg):
    """Algorithms 2, 3, 4 (Neumaier, second-order Neumaier, double-double), selected through
    hirep_set_tuning.  (i) A well-conditioned field: within 2 ulp of the exact sum.  (ii) A product whose real part
    cancels to ~1e-17 of the sum of |terms| (+-2^30 pairs plus small terms): every compensated algorithm recovers it
    to 1e-9 relative, where the naive fp64 sum has no correct digit."""
    hirep = env["hirep"]
    cfg = synth.CONFIGS["C2"].resized(8, 8)
    p = Problem(env, cfg, "f64")
    p.geom.set_tuning(hirep.TUNE_SUM_ALGORITHM, alg)
    rng = np.random.default_rng(5)
    f = rng.uniform(0.5, 1.5, size=(cfg.volume, 4, cfg.d_R)) + 1j * rng.uniform(0.5, 1.5, size=(cfg.volume, 4, cfg.d_R))
    ref = la.sqnorm(f)
    assert abs(p.geom.sqnorm(hirep.FULL, p.to_native(f, hirep.FULL)) - ref) <= 2 * 2.0 ** -52 * ref
    # cancellation: xi = (big, -big, small...), eta = (big, big, small...) -> the big products cancel exactly
    xi = (rng.uniform(-1, 1, size=f.shape) + 0j)
    eta = (rng.uniform(-1, 1, size=f.shape) + 0j)
    big = 2.0 ** 30
    xi[0::2, 0, 0], eta[0::2, 0, 0] = big, big
    xi[1::2, 0, 0], eta[1::2, 0, 0] = -big, big
    ref = la.prod(xi, eta).real
    got = p.geom.prod(hirep.FULL, p.to_native(xi, hirep.FULL), p.to_native(eta, hirep.FULL)).real
    assert abs(got - ref) <= 1e-9 * abs(ref), (alg, got, ref)
    naive = la.naive_sum((xi.real * eta.real).ravel().tolist())
    assert abs(naive - ref) > 1e-3 * abs(ref)
    with pytest.raises(hirep.HirepError):
        p.geom.set_tuning(hirep.TUNE_SUM_ALGORITHM, 7)


@pytest.mark.parametrize("name,T,L,prec,m0", [("C1", 4, 4, "f64", 0.6), ("C2", 4, 4, "f64", 0.4), ("C3", 4, 4, "f64", 0.5), ("C2", 4, 4, "f32", 0.6)])
def test_cg_vs_oracle(env, name, T, L, prec, m0):
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS[name].resized(T, L)
    p = Problem(env, cfg, prec)
    b = p.spinors[0]
    d = cfg.d_R
    apply_A = lambda v: oracle.g5Dphi_sq(T, L, d, m0, p.R, v, BC)
    tol = 1e-10 if prec == "f64" else 1e-5
    x_ref, it_ref, res_ref, _ = la.cg(apply_A, b, tol, 3000)
    x_nat, it, res = p.geom.cg_g5Dphi_sq(m0, p.to_native(b, hirep.FULL), p.links_rep, tol, 3000)
    x = p.to_numpy(x_nat, hirep.FULL)
    assert res <= tol and abs(it - it_ref) <= max(2, it_ref // 20), (it, it_ref)
    bn = np.linalg.norm(b.ravel())
    true_res = np.linalg.norm((b - apply_A(x)).ravel()) / bn
    if prec == "f64":
        assert oracle.rel_l2(x, x_ref) < 1e-7
        assert true_res < 1e-9
    else:
        assert oracle.rel_l2(x, x_ref) < 1e-3
        assert true_res < 1e-4
    # maxiter is honoured and reported, not an error
    _, it2, res2 = p.geom.cg_g5Dphi_sq(m0, p.to_native(b, hirep.FULL), p.links_rep, tol, 3)
    assert it2 == 3 and res2 > tol


@pytest.mark.parametrize("name,T,L,prec", [("C1", 4, 4, "f64"), ("C2", 6, 6, "f64"), ("C3", 4, 6, "f32"), ("C4", 4, 6, "f64"), ("C5", 2, 4, "f64")])
def test_g5Dphi_hat_and_square(env, name, T, L, prec):
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS[name].resized(T, L)
    p = Problem(env, cfg, prec)
    psi_e = p.spinors[0][p.ev]
    x = p.to_native(psi_e, hirep.EVEN)
    tol = TOL[prec]
    got = p.to_numpy(p.geom.g5Dphi_hat(cfg.m0, x, p.links_rep), hirep.EVEN)
    assert oracle.rel_l2(got, oracle.g5Dphi_hat(T, L, cfg.d_R, cfg.m0, p.R, psi_e, BC)) < tol
    got = p.to_numpy(p.geom.g5Dphi_hat_sq(cfg.m0, x, p.links_rep), hirep.EVEN)
    assert oracle.rel_l2(got, oracle.g5Dphi_hat_sq(T, L, cfg.d_R, cfg.m0, p.R, psi_e, BC)) < tol
    # Hermitian positive definite: <phi, Q^2 psi> = conj <psi, Q^2 phi>, <psi, Q^2 psi> = ||Q psi||^2 > 0 (GPU reductions)
    q = p.geom.g5Dphi_hat(cfg.m0, x, p.links_rep)
    q2 = p.geom.g5Dphi_hat_sq(cfg.m0, x, p.links_rep)
    lhs, rhs = p.geom.prod(hirep.EVEN, x, q2).real, p.geom.sqnorm(hirep.EVEN, q)
    assert abs(lhs - rhs) <= (1e-12 if prec == "f64" else 1e-5) * rhs and rhs > 0


def test_eo_preconditioned_solve_on_gpu(env):
    """The production solve: D_m x = b through the Schur complement with every step on the GPU (Dphi_eo, lc, Q_hat,
    CG on Q_hat^2, Dphi_oe), against the oracle's CG and a direct check of the residual of the FULL system."""
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS["C2"].resized(4, 4)
    T, L, d, m0 = 4, 4, cfg.d_R, 0.3
    a = 4.0 + m0
    p = Problem(env, cfg, "f64")
    g, b = p.geom, p.spinors[0]
    b_e, b_o = p.to_native(b[p.ev], hirep.EVEN), p.to_native(b[p.od], hirep.ODD)
    c = g.Dphi_eo(b_o, p.links_rep)                                   # D_eo b_o
    g.lc(hirep.EVEN, c, a, b_e, -1.0, c)                              # c = a b_e - D_eo b_o     (xi aliases zeta)
    c_np = oracle.g5(p.to_numpy(c, hirep.EVEN))                       # gamma_5 c (host: no standalone gamma_5 entry)
    rhs = g.g5Dphi_hat(m0, p.to_native(c_np, hirep.EVEN), p.links_rep)
    x_e, it, res = g.cg_g5Dphi_hat_sq(m0, rhs, p.links_rep, 1e-12, 2000)
    assert res <= 1e-12 and it > 3
    x_o = g.Dphi_oe(x_e, p.links_rep)
    g.lc(hirep.ODD, x_o, 1.0 / a, b_o, -1.0 / a, x_o)                 # x_o = (b_o - D_oe x_e) / a
    x = np.zeros_like(b)
    x[p.ev], x[p.od] = p.to_numpy(x_e, hirep.EVEN), p.to_numpy(x_o, hirep.ODD)
    resid = np.linalg.norm((b - oracle.Dphi(T, L, d, m0, p.R, x, BC)).ravel()) / np.linalg.norm(b.ravel())
    assert resid < 1e-10
    # the oracle's CG on the same preconditioned system needs the same number of iterations (+-2) and agrees
    rhs_np = p.to_numpy(rhs, hirep.EVEN)
    x_ref, it_ref, _, _ = la.cg(lambda v: oracle.g5Dphi_hat_sq(T, L, d, m0, p.R, v, BC), rhs_np, 1e-12, 2000)
    assert abs(it - it_ref) <= 2
    assert oracle.rel_l2(p.to_numpy(x_e, hirep.EVEN), x_ref) < 1e-8


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_full_size_linalg_and_cg(env, prec):
    """BASELINE configs[1] at full size (SU(3) fundamental, 32^4), the launch configuration bench.py times:
    reductions against the correctly rounded sum of the downloaded field, a linear combination on sampled sites, and
    the CG solution checked on sampled sites with the per-site oracle: (Q^2 x)(ix) = b(ix)."""
    from tests.gpu_helpers import SampledOracle, sample_sites, torch_field_fetch
    from tests.test_gpu_parity import full_size_problem
    torch, hirep, oracle = env["torch"], env["hirep"], env["oracle"]
    cfg, geom, links, psi, lr = full_size_problem(env, "C2", prec)
    x = geom.spinor_import(psi, hirep.FULL)
    host = psi.cpu().numpy().astype(np.complex128)
    eps = 2.0 ** -52
    ref = la.sqnorm(host)
    assert abs(geom.sqnorm(hirep.FULL, x) - ref) <= 4 * eps * ref
    assert geom.max_norm(hirep.FULL, x) == la.max_norm(host)
    # y = 0.5 x - 1.5 i x on sampled rows (lc2 with xi = a copy of x)
    y = geom.new_spinor(hirep.FULL)
    y.copy_(x)
    geom.lc2(hirep.FULL, y, 0.5, -1.5j, x)
    yc = geom.spinor_export(y, hirep.FULL)
    sites = sample_sites(cfg, 8, seed=5)
    for ix in sites:
        got = yc[ix].cpu().numpy().astype(np.complex128)
        assert np.linalg.norm(got - (0.5 - 1.5j) * host[ix]) <= TOL[prec] * np.linalg.norm(host[ix])
    prod = geom.prod(hirep.FULL, x, y)                       # <x, (0.5-1.5i) x> = (0.5-1.5i) ||x||^2
    assert abs(prod - (0.5 - 1.5j) * ref) <= (1e-12 if prec == "f64" else 1e-6) * abs(ref)
    # CG on Q^2 at a heavy mass (converges in a few tens of iterations)
    m0 = 1.0
    tol = 1e-9 if prec == "f64" else 2e-5
    sol, it, res = geom.cg_g5Dphi_sq(m0, x, lr, tol, 500)
    assert res <= tol and 5 < it < 500
    so = SampledOracle(oracle, cfg, links)
    fetch = torch_field_fetch(geom.spinor_export(sol, hirep.FULL))
    bnorm = np.sqrt(ref / cfg.volume)                        # typical |b(ix)| per site
    for ix in sites[:5]:
        r = host[ix] - so.g5Dphi_sq(fetch, ix, m0)
        assert np.linalg.norm(r) <= (1e-6 if prec == "f64" else 2e-3) * bnorm * np.sqrt(4 * cfg.d_R), (ix, np.linalg.norm(r))
    geom.sync()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_multishift_cg(env, prec):
    """Multi-shift CG on Q^2 (L730, Eq 39-40): every shifted solution against the oracle's multi-shift CG and, through
    the oracle operator, the true residual of its own system; same iteration count as the oracle (+-2)."""
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS["C2"].resized(4, 4)
    p = Problem(env, cfg, prec)
    T, L, d, m0 = 4, 4, cfg.d_R, 0.3
    b = p.spinors[0]
    shifts = [0.0, 0.02, 0.5, 4.0]
    tol = 1e-10 if prec == "f64" else 1e-5
    A = lambda v: oracle.g5Dphi_sq(T, L, d, m0, p.R, v, BC)
    xs_ref, it_ref, _ = la.cg_mshift(A, b, shifts, tol, 3000)
    xs, it, res = p.geom.cg_mshift_g5Dphi_sq(m0, shifts, p.to_native(b, hirep.FULL), p.links_rep, tol, 3000)
    assert res <= tol and abs(it - it_ref) <= max(2, it_ref // 20)
    bn = np.linalg.norm(b.ravel())
    for sg, xn, xr in zip(shifts, xs, xs_ref):
        x = p.to_numpy(xn, hirep.FULL)
        assert oracle.rel_l2(x, xr) < (1e-7 if prec == "f64" else 1e-3), sg
        assert np.linalg.norm((b - A(x) - sg * x).ravel()) < (1e-9 if prec == "f64" else 1e-4) * bn, sg
    # the zero shift is plain CG
    x0, it0, _ = p.geom.cg_g5Dphi_sq(m0, p.to_native(b, hirep.FULL), p.links_rep, tol, 3000)
    assert it0 == it and oracle.rel_l2(p.to_numpy(xs[0], hirep.FULL), p.to_numpy(x0, hirep.FULL)) < (1e-12 if prec == "f64" else 1e-5)
    with pytest.raises(hirep.HirepError):
        p.geom.cg_mshift_g5Dphi_sq(m0, [-1.0], p.to_native(b, hirep.FULL), p.links_rep, tol, 10)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("op", ["Dphi", "Dphi_hat"])
def test_bicgstab(env, prec, op):
    """BiCGstab (L730) on D_m (full lattice) and D_hat (even sites): solution against the oracle's BiCGstab and the true
    residual through the oracle operator.  BiCGstab iterates are more sensitive to rounding than CG's (the products
    rho, omega are not norms), so iteration counts may differ by a few."""
    hirep, oracle = env["hirep"], env["oracle"]
    cfg = synth.CONFIGS["C2"].resized(4, 4)
    p = Problem(env, cfg, prec)
    T, L, d, m0 = 4, 4, cfg.d_R, 0.3
    tol = 1e-10 if prec == "f64" else 1e-5
    if op == "Dphi":
        b, w, code = p.spinors[0], hirep.FULL, hirep.OP_DPHI
        A = lambda v: oracle.Dphi(T, L, d, m0, p.R, v, BC)
    else:
        b, w, code = p.spinors[0][p.ev], hirep.EVEN, hirep.OP_DPHI_HAT
        A = lambda v: oracle.Dphi_hat(T, L, d, m0, p.R, v, BC)
    x_ref, it_ref, _ = la.bicgstab(A, b, tol, 3000)
    xn, it, res = p.geom.bicgstab(code, m0, p.to_native(b, w), p.links_rep, tol, 3000)
    x = p.to_numpy(xn, w)
    assert res <= tol and abs(it - it_ref) <= max(3, it_ref // 5), (it, it_ref)
    assert oracle.rel_l2(x, x_ref) < (1e-7 if prec == "f64" else 1e-3)
    assert np.linalg.norm((b - A(x)).ravel()) < (1e-9 if prec == "f64" else 1e-4) * np.linalg.norm(b.ravel())
    with pytest.raises(hirep.HirepError):
        p.geom.bicgstab(hirep.OP_G5DPHI_SQ, m0, p.to_native(b, w), p.links_rep, tol, 10)


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_elementary_operations(env, prec):
    """zero / copy / multiplication by a scalar / minus on a ragged lattice, also in place."""
    hirep, oracle = env["hirep"], env["oracle"]
    p = Problem(env, synth.CONFIGS["C2"].resized(6, 6), prec)
    h = p.geom.handle
    for w, sel in ((hirep.FULL, slice(None)), (hirep.EVEN, p.ev)):
        eta = p.spinors[0][sel]
        e = p.to_native(eta, w)
        xi = p.geom.new_spinor(w)
        xi.fill_(0xFF)                                                  # NaN bit patterns
        hirep.hirep_spinor_zero(h, w, xi.data_ptr())
        assert not p.to_numpy(xi, w).any()
        hirep.hirep_spinor_copy(h, w, xi.data_ptr(), e.data_ptr())
        assert np.array_equal(p.to_numpy(xi, w), eta)
        hirep.hirep_spinor_minus(h, w, xi.data_ptr(), xi.data_ptr())    # in place
        assert np.array_equal(p.to_numpy(xi, w), -eta)
        hirep.hirep_spinor_mul(h, w, xi.data_ptr(), 0.5 - 2.0j, e.data_ptr())
        assert oracle.rel_l2(p.to_numpy(xi, w), (0.5 - 2.0j) * eta) < TOL[prec]


def test_solver_breakdown_is_reported(env):
    """a NaN right-hand side, a NaN residual or an indefinite operator must return HIREP_EBREAKDOWN (stream
    drained, x undefined) and never HIREP_OK with relres = 0."""
    hirep, torch = env["hirep"], env["torch"]
    cfg = synth.CONFIGS["C2"].resized(4, 4)
    p = Problem(env, cfg, "f64")
    b = p.spinors[0].copy()
    b[5, 1, 2] = np.nan
    bn = p.to_native(b, hirep.FULL)
    for call in (lambda: p.geom.cg_g5Dphi_sq(0.3, bn, p.links_rep, 1e-10, 50),
                 lambda: p.geom.cg_mshift_g5Dphi_sq(0.3, [0.0, 0.5], bn, p.links_rep, 1e-10, 50),
                 lambda: p.geom.bicgstab(hirep.OP_DPHI, 0.3, bn, p.links_rep, 1e-10, 50)):
        with pytest.raises(hirep.HirepError) as ei:
            call()
        assert ei.value.rc == hirep.EBREAKDOWN, ei.value
    be = p.to_native(b[p.ev], hirep.EVEN)
    with pytest.raises(hirep.HirepError) as ei:
        p.geom.cg_g5Dphi_hat_sq(0.3, be, p.links_rep, 1e-10, 50)
    assert ei.value.rc == hirep.EBREAKDOWN
    # site-diagonal blocks that contain NaN: <p,Ap> = ||B p||^2 is NaN in the first iteration
    good = p.to_native(p.spinors[0], hirep.FULL)
    nb = hirep.hirep_clover_inv_bytes(p.geom.handle)
    blocks = torch.zeros(2 * nb, dtype=torch.uint8, device=env["dev"])
    blocks.view(torch.float64)[::7] = float("nan")
    with pytest.raises(hirep.HirepError) as ei:
        p.geom.cg_g5Dphi_blocks_sq(good, p.links_rep, blocks, 1e-10, 20)
    assert ei.value.rc == hirep.EBREAKDOWN
    # the geometry is still usable afterwards (stream drained, no sticky error)
    x, it, res = p.geom.cg_g5Dphi_sq(0.3, good, p.links_rep, 1e-10, 500)
    assert res <= 1e-10 and it > 0
    # zero right-hand side: x = 0 after zero iterations, not an error
    z = torch.zeros_like(good)
    x, it, res = p.geom.cg_g5Dphi_sq(0.3, z, p.links_rep, 1e-10, 50)
    assert it == 0 and res == 0.0 and not bool(x.any())
