"""hirep_Dphi_hat_static (include/hirep_b200.h): Dphi_hat (Eq 44) with the odd intermediate field in a static device array,
for callers that cannot call cudaMalloc.  Checked against the existing hirep_Dphi_hat on two calls in a row (the second on other
inputs, with the shared array dirtied by another geometry in between), against the oracle, and for the size limit.

Collected last on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`.
"""
import numpy as np
import pytest

from harness import synth
from tests.gpu_helpers import BC, TOL
from tests.test_gpu_parity import Problem, env, np_c  # noqa: F401  (env is a fixture)

pytestmark = pytest.mark.gpu

M0 = -0.3


def rel(a, b):
    a, b = a.astype(np.complex128).ravel(), b.astype(np.complex128).ravel()
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def even_native(p, k):
    torch, hirep = p.env["torch"], p.env["hirep"]
    return p.geom.spinor_import(torch.from_numpy(p.spinors[k][p.ev].astype(np_c(p.prec))), hirep.EVEN)


# 6^4: 648 sites per parity = 20 tiles + a ragged one of 8 lanes (the padding the call has to clear); 8^4: whole tiles
@pytest.mark.parametrize("name,T,L", [("C2", 8, 8), ("C2", 6, 6), ("C3", 6, 6), ("C4", 4, 6), ("C5", 4, 4)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_static_scratch_matches_Dphi_hat_on_two_calls_in_a_row(env, name, T, L, prec):
    torch, hirep, oracle = env["torch"], env["hirep"], env["oracle"]
    p = Problem(env, synth.CONFIGS[name].resized(T, L), prec, n_spinors=2)
    assert p.geom.sizes["spinor_half"] <= hirep.STATIC_SCRATCH_BYTES
    x0, x1 = even_native(p, 0), even_native(p, 1)
    # expected values first: the existing path, its intermediate field in the handle's own workspace
    ref0 = p.geom.spinor_export(p.geom.Dphi_hat(M0, x0, p.links_rep), hirep.EVEN).cpu().numpy()
    ref1 = p.geom.spinor_export(p.geom.Dphi_hat(M0, x1, p.links_rep), hirep.EVEN).cpu().numpy()
    # dirty the shared array with another geometry's intermediate field (more tiles, another component count, NaN-free but large)
    q = Problem(env, synth.CONFIGS["C4"].resized(6, 6), "f64")
    xq = q.geom.spinor_import(torch.from_numpy(q.spinors[0][q.ev] * 1e30), hirep.EVEN)
    q.geom.Dphi_hat_static(M0, xq, q.links_rep, q.geom.new_spinor(hirep.EVEN))
    # two calls in a row on the same stream, different inputs, the caller's output buffers
    o0 = p.geom.Dphi_hat_static(M0, x0, p.links_rep, p.geom.new_spinor(hirep.EVEN))
    o1 = p.geom.Dphi_hat_static(M0, x1, p.links_rep, p.geom.new_spinor(hirep.EVEN))
    got0 = p.geom.spinor_export(o0, hirep.EVEN).cpu().numpy()
    got1 = p.geom.spinor_export(o1, hirep.EVEN).cpu().numpy()
    assert np.isfinite(got0.view(np.float64 if prec == "f64" else np.float32)).all()
    assert rel(got0, ref0) <= TOL[prec], (rel(got0, ref0), "first call")
    assert rel(got1, ref1) <= TOL[prec], (rel(got1, ref1), "second call")
    # same kernels, same launch order, same inputs: in fact bit for bit
    assert np.array_equal(got0, ref0) and np.array_equal(got1, ref1)
    # and against the oracle (full field at this size)
    want = oracle.Dphi_hat(p.cfg.T, p.cfg.L, p.cfg.d_R, M0, p.R, p.spinors[1][p.ev], p.bc)
    assert rel(got1, want) <= TOL[prec], rel(got1, want)


def test_static_scratch_rebuild_mode(env):
    """link mode REBUILD (represented links rebuilt in registers from the fundamental field) goes through the same entry point"""
    torch, hirep = env["torch"], env["hirep"]
    p = Problem(env, synth.CONFIGS["C4"].resized(4, 6), "f64", n_spinors=2)
    p.geom.set_link_mode(hirep.LINKS_REBUILD)
    for k in (0, 1):
        x = even_native(p, k)
        ref = p.geom.spinor_export(p.geom.Dphi_hat(M0, x, p.links_fund), hirep.EVEN).cpu().numpy()
        got = p.geom.spinor_export(p.geom.Dphi_hat_static(M0, x, p.links_fund, p.geom.new_spinor(hirep.EVEN)), hirep.EVEN).cpu().numpy()
        assert rel(got, ref) <= TOL["f64"] and np.array_equal(got, ref)


def test_static_scratch_allocates_nothing(env):
    """free device memory does not move across the call on a FRESH handle (where hirep_Dphi_hat would allocate its workspace)"""
    torch, hirep = env["torch"], env["hirep"]
    cfg = synth.CONFIGS["C2"].resized(16, 16)             # 6.3 MB per half spinor: above the driver's allocation granularity
    warm = Problem(env, cfg, "f64")                        # loads the kernels of this instantiation, resolves the symbol
    warm.geom.Dphi_hat_static(M0, even_native(warm, 0), warm.links_rep, warm.geom.new_spinor(hirep.EVEN))
    p = Problem(env, cfg, "f64")
    x, out = even_native(p, 0), p.geom.new_spinor(hirep.EVEN)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    p.geom.Dphi_hat_static(M0, x, p.links_rep, out)
    p.geom.Dphi_hat_static(M0, x, p.links_rep, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before
    ref = p.geom.Dphi_hat(M0, x, p.links_rep)
    assert torch.equal(ref, out)


def test_static_scratch_rejects_sizes_beyond_the_maximum(env):
    torch, hirep = env["torch"], env["hirep"]
    geom = hirep.Geometry(48, 16, 3, 0, "f64", device=env["dev"], bc=BC)       # 98304 sites per parity * 192 B = 18 MiB > 16 MiB
    assert geom.sizes["spinor_half"] > hirep.STATIC_SCRATCH_BYTES
    x, out = geom.new_spinor(hirep.EVEN), geom.new_spinor(hirep.EVEN)
    links = torch.zeros(geom.sizes["links_rep"], dtype=torch.uint8, device=env["dev"])
    n0 = geom.launch_count()
    with pytest.raises(hirep.HirepError) as ei:
        geom.Dphi_hat_static(M0, x, links, out)
    assert ei.value.rc == hirep.EINVAL and "HIREP_STATIC_SCRATCH_BYTES" in str(ei.value)
    assert geom.launch_count() == n0                                          # nothing was launched
    with pytest.raises(hirep.HirepError):
        geom.Dphi_hat_static(M0, x, links, x)                                 # aliasing is rejected as in hirep_Dphi_hat
