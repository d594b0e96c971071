"""Robustness checks of the CUDA kernels that need no oracle (compute-sanitizer is not available on the GPU pool):
  * determinism -- every operator gives bit-identical output when repeated (a shared-memory or mbarrier race in the
    bulk-copy rings, the pair exchange or the row-group half-spinor buffers would show up as run-to-run differences);
  * guard bands -- outputs are written into a slice of a larger buffer whose bytes before and after the slice keep
    their fill pattern (no out-of-bounds store), and the padding lanes of the last tile keep theirs (stores of
    inactive lanes are predicated)."""
import numpy as np
import pytest

from harness import synth
from tests.test_gpu_parity import Problem, env  # noqa: F401  (env is a fixture)

pytestmark = pytest.mark.gpu

GUARD = 4096
CASES = [("C1", 4, 4, "f64"), ("C2", 6, 6, "f64"), ("C2", 6, 6, "f32"), ("C3", 4, 8, "f32"), ("C4", 6, 6, "f64"),
         ("C4", 6, 6, "f32"), ("C5", 2, 6, "f64"), ("C5", 2, 6, "f32")]


def guarded(torch, dev, nbytes):
    big = torch.full((nbytes + 2 * GUARD,), 0xA5, dtype=torch.uint8, device=dev)
    return big, big[GUARD:GUARD + nbytes]


@pytest.mark.parametrize("name,T,L,prec", CASES)
@pytest.mark.parametrize("max_ctas", [0, 2])
def test_determinism_and_guard_bands(env, name, T, L, prec, max_ctas):
    torch, hirep = env["torch"], env["hirep"]
    cfg = synth.CONFIGS[name].resized(T, L)
    p = Problem(env, cfg, prec)
    g = p.geom
    g.set_tuning(hirep.TUNE_MAX_CTAS, max_ctas)
    x = p.to_native(p.spinors[0], hirep.FULL)
    hb, fb = g.sizes["spinor_half"], g.sizes["spinor_full"]
    ops = [
        ("Dphi", fb, lambda out: g.Dphi(cfg.m0, x, p.links_rep, out=out)),
        ("Dphi_eo", hb, lambda out: g.Dphi_eo(x[hb:], p.links_rep, out=out)),
        ("Dphi_oe", hb, lambda out: g.Dphi_oe(x[:hb], p.links_rep, out=out)),
        ("Dphi_hat", hb, lambda out: g.Dphi_hat(cfg.m0, x[:hb], p.links_rep, out=out)),
        ("g5Dphi_sq", fb, lambda out: g.g5Dphi_sq(cfg.m0, x, p.links_rep, out=out)),
        ("Dphi_tm_hat", hb, lambda out: g.Dphi_tm_hat(cfg.m0, 0.3, x[:hb], p.links_rep, out=out)),
    ]
    # lanes of the last tile beyond Nh are padding: [tile][comp][lane] -> mask of padding bytes of one half-lattice buffer
    nh = cfg.volume // 2
    valid = nh % 32 or 32
    w = 16 if prec == "f64" else 8
    ncomp = 4 * cfg.d_R
    pad_mask = np.zeros(hb, dtype=bool)
    if valid != 32:
        last = (hb // (ncomp * 32 * w) - 1) * ncomp * 32 * w
        m = pad_mask[last:].reshape(ncomp, 32, w)
        m[:, valid:, :] = True
    for nm, nbytes, run in ops:
        results = []
        for rep in range(3):
            big, out = guarded(torch, env["dev"], nbytes)
            run(out)
            g.sync()
            host = big.cpu().numpy()
            assert (host[:GUARD] == 0xA5).all() and (host[GUARD + nbytes:] == 0xA5).all(), (nm, "guard band overwritten")
            body = host[GUARD:GUARD + nbytes]
            for h0 in range(0, nbytes, hb):
                assert (body[h0:h0 + hb][pad_mask] == 0xA5).all(), (nm, "padding lanes written")
            results.append(body.copy())
        assert np.array_equal(results[0], results[1]) and np.array_equal(results[0], results[2]), (nm, "not deterministic")


NEW_KERNELS = [  # (N, rep, T, L, prec, variant, rebuild): hop_full in all its shapes (variant 5) and the matrix-free adjoint (REBUILD)
    (3, 0, 8, 8, "f64", 5, False), (3, 0, 8, 8, "f32", 5, False), (2, 1, 4, 12, "f64", 5, False), (2, 1, 4, 12, "f32", 5, False),
    (4, 3, 4, 12, "f64", 5, False), (4, 3, 4, 12, "f32", 5, False), (5, 0, 4, 6, "f64", 5, False), (4, 0, 6, 6, "f32", 5, False),
    (3, 1, 4, 8, "f64", 0, True), (6, 1, 4, 6, "f64", 0, True), (6, 1, 4, 6, "f32", 0, True), (4, 1, 6, 6, "f32", 0, True)]


@pytest.mark.parametrize("n,rep,T,L,prec,variant,rebuild", NEW_KERNELS)
@pytest.mark.parametrize("max_ctas", [0, 3])
def test_determinism_of_the_round2_kernels(env, n, rep, T, L, prec, variant, rebuild, max_ctas):
    """compute-sanitizer is closed on the GPU pool, so races in the tile-pair staging (mbarrier slots shared by bulk copies and
    per-lane cp.async gathers, register neighbours, staged input tiles refilled during the last direction) and in the per-warp
    areas of the matrix-free adjoint are hunted the other way: six repetitions must agree bit for bit, with guard bands around the
    output and L^3/2 not a multiple of the tile (ragged rows, in-pair and out-of-pair neighbours mixed within a warp)."""
    torch, hirep = env["torch"], env["hirep"]
    cfg = synth.Config("t", T, L, n, rep, -0.3, "haar", 321, ())
    p = Problem(env, cfg, prec)
    g = p.geom
    g.set_kernel_variant(variant)
    g.set_tuning(hirep.TUNE_MAX_CTAS, max_ctas)
    links = p.links_rep
    if rebuild:
        g.set_link_mode(hirep.LINKS_REBUILD)
        links = p.links_fund
    x = p.to_native(p.spinors[0], hirep.FULL)
    fb = g.sizes["spinor_full"]
    for nm, run in [("Dphi", lambda out: g.Dphi(cfg.m0, x, links, out=out)), ("g5Dphi_sq", lambda out: g.g5Dphi_sq(cfg.m0, x, links, out=out)),
                    ("Dphi_tm", lambda out: g.Dphi_tm(cfg.m0, 0.25, x, links, out=out))]:
        first = None
        for rep_ in range(6):
            big, out = guarded(torch, env["dev"], fb)
            run(out)
            g.sync()
            host = big.cpu().numpy()
            assert (host[:GUARD] == 0xA5).all() and (host[GUARD + fb:] == 0xA5).all(), (nm, "guard band overwritten")
            body = host[GUARD:GUARD + fb].copy()
            if first is None:
                first = body
            assert np.array_equal(first, body), (nm, rep_, "not deterministic")


def test_reductions_and_cg_are_deterministic(env):
    hirep = env["hirep"]
    p = Problem(env, synth.CONFIGS["C2"].resized(6, 6), "f64")
    x = p.to_native(p.spinors[0], hirep.FULL)
    vals = {(p.geom.sqnorm(hirep.FULL, x), p.geom.prod(hirep.FULL, x, x)) for _ in range(5)}
    assert len(vals) == 1
    sols = []
    for _ in range(2):
        s, it, res = p.geom.cg_g5Dphi_sq(0.5, x, p.links_rep, 1e-10, 500)
        sols.append((p.to_numpy(s, hirep.FULL), it, res))
    assert sols[0][1:] == sols[1][1:] and np.array_equal(sols[0][0], sols[1][0])


def test_cuda_graph_capture_and_replay(env):
    """The operator calls only enqueue kernels on the geometry's stream (no allocation or synchronisation once the
    workspaces exist), so a whole step can be captured in a CUDA graph and replayed -- the launch-bound small-lattice
    case of BASELINE configs[0] (4^4).  Replay must reproduce the eager result bit for bit."""
    torch, hirep = env["torch"], env["hirep"]
    cfg = synth.CONFIGS["C1"]
    U, (psi,) = synth.make_inputs(cfg)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        g = hirep.Geometry(cfg.T, cfg.L, cfg.n_g, cfg.rep, "f64", device=env["dev"])
        lf = g.links_import(torch.from_numpy(U).to(env["dev"]))
        lr = g.links_to_rep(lf)
        x = g.spinor_import(torch.from_numpy(psi).to(env["dev"]))
        hb = g.sizes["spinor_half"]
        ye, yf = g.new_spinor(hirep.EVEN), g.new_spinor(hirep.FULL)

        def step():
            g.links_to_rep(lf, out=lr)
            g.Dphi_hat(cfg.m0, x[:hb], lr, out=ye)
            g.g5Dphi_sq(cfg.m0, x, lr, out=yf)
            g.Dphi_tm_hat(cfg.m0, 0.2, x[:hb], lr, out=ye)

        for _ in range(2):
            step()                       # warm-up: workspaces and kernel attributes are set up outside the capture
        s.synchronize()
        ref_e, ref_f = ye.clone(), yf.clone()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            step()
        ye.zero_(); yf.zero_()
        for _ in range(3):
            graph.replay()
        s.synchronize()
        assert torch.equal(ye, ref_e) and torch.equal(yf, ref_f)


def test_reserve_then_first_call_inside_capture(env):
    """hirep_geom_reserve allocates the workspaces up front: the FIRST Dphi_hat / g5Dphi_sq / Dphi_clover_hat of a geometry may then
    be issued inside a CUDA-graph capture (no cudaMalloc in the call); the replayed results equal those of a second, eagerly used
    geometry bit for bit."""
    torch, hirep = env["torch"], env["hirep"]
    cfg = synth.CONFIGS["C2"].resized(4, 6)
    U, (psi,) = synth.make_inputs(cfg)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        outs = []
        for captured in (False, True):
            g = hirep.Geometry(cfg.T, cfg.L, cfg.n_g, cfg.rep, "f64", device=env["dev"])
            lf = g.links_import(torch.from_numpy(U).to(env["dev"]))
            lr = g.links_to_rep(lf)
            x = g.spinor_import(torch.from_numpy(psi).to(env["dev"]))
            cl = g.clover_field(lr)
            inv = g.clover_inv_field(cfg.m0, 0.5, hirep.ODD, cl)
            hb = g.sizes["spinor_half"]
            ye, yf, yc = g.new_spinor(hirep.EVEN), g.new_spinor(hirep.FULL), g.new_spinor(hirep.EVEN)

            def step():
                g.Dphi_hat(cfg.m0, x[:hb], lr, out=ye)
                g.g5Dphi_sq(cfg.m0, x, lr, out=yf)
                g.Dphi_clover_hat(cfg.m0, 0.5, x[:hb], lr, cl, inv, out=yc)

            if captured:
                g.reserve(hirep.RESERVE_OPERATORS)
                g.reserve(hirep.RESERVE_OPERATORS | hirep.RESERVE_SOLVERS)      # idempotent
                s.synchronize()
                graph = torch.cuda.CUDAGraph()
                with torch.cuda.graph(graph, stream=s):
                    step()
                graph.replay()
            else:
                step()
            s.synchronize()
            # canonical export: the padding lanes of the ragged last tile (13.5 tiles per parity) are never written and hold whatever
            # torch.empty returned
            outs.append((g.spinor_export(ye, hirep.EVEN), g.spinor_export(yf, hirep.FULL), g.spinor_export(yc, hirep.EVEN)))
        for a, b in zip(*outs):
            assert torch.equal(a, b) and bool(torch.isfinite(a.real).all()) and float(a.abs().max()) > 0
    with pytest.raises(hirep.HirepError):
        g.reserve(0)
