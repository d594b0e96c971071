"""Thin ctypes binding of libhirep_b200.so (C-ABI: include/hirep_b200.h).

Argument marshalling only: every step of the path runs in the library's CUDA kernels.  torch supplies device
memory (`tensor.data_ptr()`) and the stream.  Module-level functions carry the C names and take raw pointers;
`Geometry` is a convenience wrapper that allocates native buffers as torch tensors.

There is NO CPU fallback: `load()` raises if the shared library is missing, and every compute call raises
`HirepError` with the library's message if CUDA is unavailable.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("HIREP_B200_LIB", os.path.join(_HERE, "libhirep_b200.so"))   # override: A/B builds

FUND, ADJ, SYM, ASY = 0, 1, 2, 3
F64, F32 = 0, 1
EVEN, ODD, FULL = 0, 1, 2
LINKS_STORED, LINKS_REBUILD = 0, 1
OP_DPHI, OP_DPHI_EO, OP_DPHI_OE, OP_DPHI_HAT, OP_G5DPHI_SQ = 0, 1, 2, 3, 4
TUNE_MAX_CTAS, TUNE_SUM_ALGORITHM, TUNE_PACE_WINDOW, TUNE_FUSE_DIAG = 1, 2, 3, 4
REGION_ALL, REGION_OWNED, REGION_INTERIOR, REGION_BOUNDARY = 0, 1, 2, 3
STATIC_SCRATCH_BYTES = 16 << 20   # HIREP_STATIC_SCRATCH_BYTES
RESERVE_OPERATORS, RESERVE_SOLVERS = 1, 2
OK, EINVAL, EUNSUPPORTED, ECUDA, ENOMEM, EBREAKDOWN = 0, -1, -2, -3, -4, -5

# every symbol include/hirep_b200.h declares
SYMBOLS = [
    "hirep_geom_create", "hirep_geom_destroy", "hirep_geom_set_bc", "hirep_geom_set_stream", "hirep_geom_sizes", "hirep_geom_reserve",
    "hirep_spinor_import", "hirep_spinor_export", "hirep_links_import", "hirep_links_rep_export",
    "hirep_links_rep_export_bwd", "hirep_links_to_rep", "hirep_Dphi", "hirep_Dphi_eo", "hirep_Dphi_oe",
    "hirep_Dphi_hat", "hirep_Dphi_hat_static", "hirep_g5Dphi_sq", "hirep_g5Dphi_hat", "hirep_g5Dphi_hat_sq", "hirep_cg_g5Dphi_hat_sq", "hirep_set_link_mode", "hirep_set_kernel_variant", "hirep_set_tuning", "hirep_launch_count",
    "hirep_apply_host", "hirep_apply_host_async", "hirep_spinor_zero", "hirep_spinor_copy", "hirep_spinor_mul", "hirep_spinor_minus",
    "hirep_spinor_lc", "hirep_spinor_clc", "hirep_spinor_lc_add_assign", "hirep_spinor_clc_add_assign",
    "hirep_spinor_lc1", "hirep_spinor_lc2", "hirep_spinor_lc3", "hirep_spinor_prod", "hirep_spinor_sqnorm",
    "hirep_spinor_max_norm", "hirep_cg_g5Dphi_sq", "hirep_spinor_g5_lc", "hirep_spinor_gamma", "hirep_spinor_g5_lc_add_assign", "hirep_spinor_g5_prod", "hirep_Dphi_tm", "hirep_Dphi_tm_sq",
    "hirep_Dphi_tm_hat", "hirep_cg_Dphi_tm_sq", "hirep_cg_mshift_g5Dphi_sq", "hirep_bicgstab", "hirep_fma_peak", "hirep_sync", "hirep_last_error",
    "hirep_clover_bytes", "hirep_clover_field", "hirep_clover_export", "hirep_Cphi", "hirep_Dphi_clover",
    "hirep_clover_inv_bytes", "hirep_clover_inv_field", "hirep_Cphi_inv", "hirep_Dphi_clover_hat",
    "hirep_clover_exp_field", "hirep_Dphi_blocks", "hirep_Dphi_blocks_hat", "hirep_g5Dphi_clover_sq", "hirep_cg_g5Dphi_clover_sq",
    "hirep_g5Dphi_clover_hat_sq", "hirep_g5Dphi_blocks_hat_sq", "hirep_cg_g5Dphi_clover_hat_sq", "hirep_cg_g5Dphi_blocks_hat_sq",
    "hirep_g5Dphi_blocks_sq", "hirep_cg_g5Dphi_blocks_sq", "hirep_force_bytes", "hirep_force_hopping",
    "hirep_geom_create_slab", "hirep_set_region", "hirep_halo_bytes", "hirep_halo_pack", "hirep_halo_unpack",
]


class HirepError(RuntimeError):
    def __init__(self, msg, rc=None):
        super().__init__(msg)
        self.rc = rc


_lib = None


def load():
    """dlopen the CUDA library and check that it exports every declared symbol.  Needs no GPU."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise HirepError(
            "CUDA library %s not found: run `python __graft_entry__.py` (nvcc, sm_100a) first. "
            "There is no CPU fallback." % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    for name in SYMBOLS:
        if not hasattr(lib, name):
            raise HirepError("libhirep_b200.so does not export %s" % name)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    lib.hirep_geom_create.argtypes = [ci, ci, ci, ci, ci, ctypes.POINTER(vp)]
    lib.hirep_geom_destroy.argtypes = [vp]
    lib.hirep_geom_set_bc.argtypes = [vp, ctypes.POINTER(ci)]
    lib.hirep_geom_set_stream.argtypes = [vp, vp]
    lib.hirep_geom_reserve.argtypes = [vp, ci]
    lib.hirep_geom_sizes.argtypes = [vp] + [ctypes.POINTER(ctypes.c_size_t)] * 4 + [ctypes.POINTER(ci)] * 2
    for n in ("hirep_spinor_import", "hirep_spinor_export"):
        getattr(lib, n).argtypes = [vp, vp, vp, ci]
    for n in ("hirep_links_import", "hirep_links_rep_export", "hirep_links_rep_export_bwd", "hirep_links_to_rep"):
        getattr(lib, n).argtypes = [vp, vp, vp]
    for n in ("hirep_Dphi", "hirep_Dphi_hat", "hirep_Dphi_hat_static", "hirep_g5Dphi_sq", "hirep_g5Dphi_hat", "hirep_g5Dphi_hat_sq"):
        getattr(lib, n).argtypes = [vp, cd, vp, vp, vp]
    for n in ("hirep_Dphi_eo", "hirep_Dphi_oe"):
        getattr(lib, n).argtypes = [vp, vp, vp, vp]
    lib.hirep_set_link_mode.argtypes = [vp, ci]
    lib.hirep_set_kernel_variant.argtypes = [vp, ci]
    lib.hirep_set_tuning.argtypes = [vp, ci, ci]
    lib.hirep_launch_count.argtypes = [vp]
    lib.hirep_launch_count.restype = ctypes.c_long
    lib.hirep_apply_host.argtypes = [vp, ci, cd, vp, vp, vp]
    lib.hirep_apply_host_async.argtypes = [vp, ci, cd, vp, vp, vp]
    c2p = ctypes.POINTER(cd)
    for n in ("hirep_spinor_lc", "hirep_spinor_lc_add_assign"):
        getattr(lib, n).argtypes = [vp, ci, vp, cd, vp, cd, vp]
    for n in ("hirep_spinor_clc", "hirep_spinor_clc_add_assign", "hirep_spinor_lc3"):
        getattr(lib, n).argtypes = [vp, ci, vp, c2p, vp, c2p, vp]
    lib.hirep_spinor_zero.argtypes = [vp, ci, vp]
    lib.hirep_spinor_copy.argtypes = [vp, ci, vp, vp]
    lib.hirep_spinor_minus.argtypes = [vp, ci, vp, vp]
    lib.hirep_spinor_mul.argtypes = [vp, ci, vp, c2p, vp]
    lib.hirep_spinor_lc1.argtypes = [vp, ci, vp, c2p, vp]
    lib.hirep_spinor_lc2.argtypes = [vp, ci, vp, c2p, c2p, vp]
    lib.hirep_spinor_prod.argtypes = [vp, ci, vp, vp, c2p]
    lib.hirep_spinor_sqnorm.argtypes = [vp, ci, vp, c2p]
    lib.hirep_spinor_max_norm.argtypes = [vp, ci, vp, c2p]
    lib.hirep_cg_g5Dphi_sq.argtypes = [vp, cd, vp, vp, vp, cd, ci, ctypes.POINTER(ci), c2p]
    lib.hirep_cg_g5Dphi_hat_sq.argtypes = [vp, cd, vp, vp, vp, cd, ci, ctypes.POINTER(ci), c2p]
    lib.hirep_spinor_g5_lc.argtypes = [vp, ci, vp, c2p, c2p, vp]
    lib.hirep_spinor_gamma.argtypes = [vp, ci, ci, vp, vp]
    lib.hirep_spinor_g5_lc_add_assign.argtypes = [vp, ci, vp, c2p, c2p, c2p, vp]
    lib.hirep_spinor_g5_prod.argtypes = [vp, ci, vp, vp, c2p]
    for n in ("hirep_Dphi_tm", "hirep_Dphi_tm_sq", "hirep_Dphi_tm_hat"):
        getattr(lib, n).argtypes = [vp, cd, cd, vp, vp, vp]
    lib.hirep_cg_mshift_g5Dphi_sq.argtypes = [vp, cd, ci, c2p, ctypes.POINTER(vp), vp, vp, cd, ci, ctypes.POINTER(ci), c2p]
    lib.hirep_bicgstab.argtypes = [vp, ci, cd, vp, vp, vp, cd, ci, ctypes.POINTER(ci), c2p]
    lib.hirep_cg_Dphi_tm_sq.argtypes = [vp, cd, cd, vp, vp, vp, cd, ci, ctypes.POINTER(ci), c2p]
    lib.hirep_fma_peak.argtypes = [ci, ctypes.POINTER(cd)]
    lib.hirep_clover_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_size_t)]
    lib.hirep_clover_field.argtypes = [vp, vp, vp]
    lib.hirep_clover_export.argtypes = [vp, vp, vp]
    lib.hirep_Cphi.argtypes = [vp, cd, cd, vp, vp, vp]
    lib.hirep_Dphi_clover.argtypes = [vp, cd, cd, vp, vp, vp, vp]
    lib.hirep_clover_inv_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_size_t)]
    lib.hirep_clover_inv_field.argtypes = [vp, cd, cd, ci, vp, vp]
    lib.hirep_Cphi_inv.argtypes = [vp, vp, vp, vp]
    lib.hirep_Dphi_clover_hat.argtypes = [vp, cd, cd, vp, vp, vp, vp, vp]
    lib.hirep_clover_exp_field.argtypes = [vp, cd, cd, ci, ci, vp, vp]
    lib.hirep_g5Dphi_clover_sq.argtypes = [vp, cd, cd, vp, vp, vp, vp]
    lib.hirep_cg_g5Dphi_clover_sq.argtypes = [vp, cd, cd, vp, vp, vp, vp, cd, ci, ctypes.POINTER(ci), c2p]
    lib.hirep_Dphi_blocks.argtypes = [vp, vp, vp, vp, vp]
    lib.hirep_Dphi_blocks_hat.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.hirep_geom_create_slab.argtypes = [ci, ci, ci, ci, ci, ci, ci, ctypes.POINTER(vp)]
    lib.hirep_set_region.argtypes = [vp, ci]
    lib.hirep_halo_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_size_t)]
    lib.hirep_halo_pack.argtypes = [vp, ci, vp, vp]
    lib.hirep_halo_unpack.argtypes = [vp, ci, vp, vp]
    lib.hirep_force_bytes.argtypes = [vp, ctypes.POINTER(ctypes.c_size_t), ctypes.POINTER(ci)]
    lib.hirep_force_hopping.argtypes = [vp, vp, vp, vp, vp]
    lib.hirep_g5Dphi_blocks_sq.argtypes = [vp, vp, vp, vp, vp]
    lib.hirep_cg_g5Dphi_blocks_sq.argtypes = [vp, vp, vp, vp, vp, cd, ci, ctypes.POINTER(ci), c2p]
    lib.hirep_g5Dphi_clover_hat_sq.argtypes = [vp, cd, cd, vp, vp, vp, vp, vp]
    lib.hirep_g5Dphi_blocks_hat_sq.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.hirep_cg_g5Dphi_clover_hat_sq.argtypes = [vp, cd, cd, vp, vp, vp, vp, vp, cd, ci, ctypes.POINTER(ci), c2p]
    lib.hirep_cg_g5Dphi_blocks_hat_sq.argtypes = [vp, vp, vp, vp, vp, vp, cd, ci, ctypes.POINTER(ci), c2p]
    lib.hirep_sync.argtypes = [vp]
    lib.hirep_last_error.restype = ctypes.c_char_p
    for n in SYMBOLS:
        if n not in ("hirep_launch_count", "hirep_last_error"):
            getattr(lib, n).restype = ci
    _lib = lib
    return lib


def hirep_last_error() -> str:
    return load().hirep_last_error().decode()


def _check(rc: int):
    if rc != 0:
        raise HirepError("hirep error %d: %s" % (rc, hirep_last_error()), rc)


# ---- same-name module-level functions (raw handles / pointers) -----------------------------------------
def hirep_geom_create(T, L, N_g, rep, prec):
    h = ctypes.c_void_p()
    _check(load().hirep_geom_create(T, L, N_g, rep, prec, ctypes.byref(h)))
    return h


def hirep_geom_destroy(g):
    _check(load().hirep_geom_destroy(g))


def hirep_geom_set_bc(g, sign):
    _check(load().hirep_geom_set_bc(g, (ctypes.c_int * 4)(*[int(s) for s in sign])))


def hirep_geom_reserve(g, what):
    _check(load().hirep_geom_reserve(g, int(what)))


def hirep_geom_set_stream(g, cuda_stream):
    _check(load().hirep_geom_set_stream(g, ctypes.c_void_p(cuda_stream)))


def hirep_geom_sizes(g):
    sz = [ctypes.c_size_t() for _ in range(4)]
    d, r = ctypes.c_int(), ctypes.c_int()
    _check(load().hirep_geom_sizes(g, *[ctypes.byref(s) for s in sz], ctypes.byref(d), ctypes.byref(r)))
    return dict(spinor_full=sz[0].value, spinor_half=sz[1].value, links_fund=sz[2].value, links_rep=sz[3].value,
                d_R=d.value, rep_is_real=bool(r.value))


def hirep_spinor_import(g, native, canonical, which): _check(load().hirep_spinor_import(g, native, canonical, which))
def hirep_spinor_export(g, canonical, native, which): _check(load().hirep_spinor_export(g, canonical, native, which))
def hirep_links_import(g, native_fund, canonical_fund): _check(load().hirep_links_import(g, native_fund, canonical_fund))
def hirep_links_rep_export(g, canonical_rep, native_rep): _check(load().hirep_links_rep_export(g, canonical_rep, native_rep))
def hirep_links_rep_export_bwd(g, canonical_rep, native_rep): _check(load().hirep_links_rep_export_bwd(g, canonical_rep, native_rep))
def hirep_links_to_rep(g, native_rep, native_fund): _check(load().hirep_links_to_rep(g, native_rep, native_fund))
def hirep_Dphi(g, m0, out, inp, links): _check(load().hirep_Dphi(g, m0, out, inp, links))
def hirep_Dphi_eo(g, out, inp, links): _check(load().hirep_Dphi_eo(g, out, inp, links))
def hirep_Dphi_oe(g, out, inp, links): _check(load().hirep_Dphi_oe(g, out, inp, links))
def hirep_Dphi_hat(g, m0, out, inp, links): _check(load().hirep_Dphi_hat(g, m0, out, inp, links))
def hirep_Dphi_hat_static(g, m0, out, inp, links): _check(load().hirep_Dphi_hat_static(g, m0, out, inp, links))
def hirep_g5Dphi_sq(g, m0, out, inp, links): _check(load().hirep_g5Dphi_sq(g, m0, out, inp, links))
def hirep_g5Dphi_hat(g, m0, out, inp, links): _check(load().hirep_g5Dphi_hat(g, m0, out, inp, links))
def hirep_g5Dphi_hat_sq(g, m0, out, inp, links): _check(load().hirep_g5Dphi_hat_sq(g, m0, out, inp, links))
def hirep_set_link_mode(g, mode): _check(load().hirep_set_link_mode(g, mode))
def hirep_set_kernel_variant(g, variant): _check(load().hirep_set_kernel_variant(g, variant))
def hirep_set_tuning(g, key, value): _check(load().hirep_set_tuning(g, key, value))
def hirep_launch_count(g): return int(load().hirep_launch_count(g))
def _c2(z):
    z = complex(z)
    return (ctypes.c_double * 2)(z.real, z.imag)


def hirep_spinor_zero(g, which, xi): _check(load().hirep_spinor_zero(g, which, xi))
def hirep_spinor_copy(g, which, xi, eta): _check(load().hirep_spinor_copy(g, which, xi, eta))
def hirep_spinor_minus(g, which, xi, eta): _check(load().hirep_spinor_minus(g, which, xi, eta))
def hirep_spinor_mul(g, which, xi, c, eta): _check(load().hirep_spinor_mul(g, which, xi, _c2(c), eta))
def hirep_spinor_lc(g, which, xi, r1, eta, r2, zeta): _check(load().hirep_spinor_lc(g, which, xi, r1, eta, r2, zeta))
def hirep_spinor_clc(g, which, xi, c1, eta, c2, zeta): _check(load().hirep_spinor_clc(g, which, xi, _c2(c1), eta, _c2(c2), zeta))
def hirep_spinor_lc_add_assign(g, which, xi, r1, eta, r2, zeta): _check(load().hirep_spinor_lc_add_assign(g, which, xi, r1, eta, r2, zeta))
def hirep_spinor_clc_add_assign(g, which, xi, c1, eta, c2, zeta): _check(load().hirep_spinor_clc_add_assign(g, which, xi, _c2(c1), eta, _c2(c2), zeta))
def hirep_spinor_lc1(g, which, xi, c1, eta): _check(load().hirep_spinor_lc1(g, which, xi, _c2(c1), eta))
def hirep_spinor_lc2(g, which, xi, c1, c2, eta): _check(load().hirep_spinor_lc2(g, which, xi, _c2(c1), _c2(c2), eta))
def hirep_spinor_lc3(g, which, xi, c1, eta, c2, zeta): _check(load().hirep_spinor_lc3(g, which, xi, _c2(c1), eta, _c2(c2), zeta))


def hirep_spinor_prod(g, which, xi, eta):
    out = (ctypes.c_double * 2)()
    _check(load().hirep_spinor_prod(g, which, xi, eta, out))
    return complex(out[0], out[1])


def hirep_spinor_sqnorm(g, which, xi):
    out = (ctypes.c_double * 2)()
    _check(load().hirep_spinor_sqnorm(g, which, xi, out))
    return out[0]


def hirep_spinor_max_norm(g, which, eta):
    out = (ctypes.c_double * 2)()
    _check(load().hirep_spinor_max_norm(g, which, eta, out))
    return out[0]


def hirep_cg_g5Dphi_sq(g, m0, x, b, links, tol, maxiter):
    it, res = ctypes.c_int(), (ctypes.c_double * 2)()
    _check(load().hirep_cg_g5Dphi_sq(g, m0, x, b, links, tol, maxiter, ctypes.byref(it), res))
    return it.value, res[0]


def hirep_spinor_g5_lc(g, which, xi, c1, c2, eta): _check(load().hirep_spinor_g5_lc(g, which, xi, _c2(c1), _c2(c2), eta))
def hirep_spinor_gamma(g, which, mu, xi, eta): _check(load().hirep_spinor_gamma(g, which, mu, xi, eta))


def hirep_spinor_g5_lc_add_assign(g, which, xi, c0, c1, c2, eta):
    _check(load().hirep_spinor_g5_lc_add_assign(g, which, xi, _c2(c0), _c2(c1), _c2(c2), eta))


def hirep_spinor_g5_prod(g, which, xi, eta):
    out = (ctypes.c_double * 2)()
    _check(load().hirep_spinor_g5_prod(g, which, xi, eta, out))
    return complex(out[0], out[1])


def hirep_Dphi_tm(g, m0, mu, out, inp, links): _check(load().hirep_Dphi_tm(g, m0, mu, out, inp, links))
def hirep_Dphi_tm_sq(g, m0, mu, out, inp, links): _check(load().hirep_Dphi_tm_sq(g, m0, mu, out, inp, links))
def hirep_clover_bytes(g) -> int:
    n = ctypes.c_size_t(0)
    _check(load().hirep_clover_bytes(g, ctypes.byref(n)))
    return n.value


def hirep_clover_field(g, clover, links_rep): _check(load().hirep_clover_field(g, clover, links_rep))
def hirep_clover_export(g, canonical, clover): _check(load().hirep_clover_export(g, canonical, clover))
def hirep_Cphi(g, m0, csw, out, inp, clover): _check(load().hirep_Cphi(g, m0, csw, out, inp, clover))
def hirep_Dphi_clover(g, m0, csw, out, inp, links, clover): _check(load().hirep_Dphi_clover(g, m0, csw, out, inp, links, clover))
def hirep_clover_inv_bytes(g) -> int:
    n = ctypes.c_size_t(0)
    _check(load().hirep_clover_inv_bytes(g, ctypes.byref(n)))
    return n.value


def hirep_clover_inv_field(g, m0, csw, parity, inv, clover): _check(load().hirep_clover_inv_field(g, m0, csw, parity, inv, clover))
def hirep_Cphi_inv(g, out, inp, inv): _check(load().hirep_Cphi_inv(g, out, inp, inv))
def hirep_Dphi_clover_hat(g, m0, csw, out, inp, links, clover, inv_odd): _check(load().hirep_Dphi_clover_hat(g, m0, csw, out, inp, links, clover, inv_odd))
def hirep_clover_exp_field(g, m0, csw, parity, inverse, blocks, clover): _check(load().hirep_clover_exp_field(g, m0, csw, parity, inverse, blocks, clover))
def hirep_Dphi_blocks(g, out, inp, links, blocks): _check(load().hirep_Dphi_blocks(g, out, inp, links, blocks))
def hirep_Dphi_blocks_hat(g, out, inp, links, blocks_even, inv_blocks_odd): _check(load().hirep_Dphi_blocks_hat(g, out, inp, links, blocks_even, inv_blocks_odd))
def hirep_Dphi_tm_hat(g, m0, mu, out, inp, links): _check(load().hirep_Dphi_tm_hat(g, m0, mu, out, inp, links))


def hirep_cg_mshift_g5Dphi_sq(g, m0, shifts, xs, b, links, tol, maxiter):
    n = len(shifts)
    sh = (ctypes.c_double * n)(*[float(s) for s in shifts])
    xp = (ctypes.c_void_p * n)(*xs)
    it, res = ctypes.c_int(), (ctypes.c_double * 2)()
    _check(load().hirep_cg_mshift_g5Dphi_sq(g, m0, n, sh, xp, b, links, tol, maxiter, ctypes.byref(it), res))
    return it.value, res[0]


def hirep_bicgstab(g, op, m0, x, b, links, tol, maxiter):
    it, res = ctypes.c_int(), (ctypes.c_double * 2)()
    _check(load().hirep_bicgstab(g, op, m0, x, b, links, tol, maxiter, ctypes.byref(it), res))
    return it.value, res[0]


def hirep_cg_Dphi_tm_sq(g, m0, mu, x, b, links, tol, maxiter):
    it, res = ctypes.c_int(), (ctypes.c_double * 2)()
    _check(load().hirep_cg_Dphi_tm_sq(g, m0, mu, x, b, links, tol, maxiter, ctypes.byref(it), res))
    return it.value, res[0]


def hirep_g5Dphi_clover_sq(g, m0, csw, out, inp, links, clover): _check(load().hirep_g5Dphi_clover_sq(g, m0, csw, out, inp, links, clover))


def hirep_cg_g5Dphi_clover_sq(g, m0, csw, x, b, links, clover, tol, maxiter):
    it, res = ctypes.c_int(), (ctypes.c_double * 2)()
    _check(load().hirep_cg_g5Dphi_clover_sq(g, m0, csw, x, b, links, clover, tol, maxiter, ctypes.byref(it), res))
    return it.value, res[0]


def hirep_geom_create_slab(T_glob, L, N_g, rep, prec, t_start, T_loc):
    h = ctypes.c_void_p()
    _check(load().hirep_geom_create_slab(T_glob, L, N_g, rep, prec, t_start, T_loc, ctypes.byref(h)))
    return h


def hirep_set_region(g, region): _check(load().hirep_set_region(g, region))


def hirep_halo_bytes(g):
    nb = ctypes.c_size_t()
    _check(load().hirep_halo_bytes(g, ctypes.byref(nb)))
    return nb.value


def hirep_halo_pack(g, face, buf, spinor_half): _check(load().hirep_halo_pack(g, face, buf, spinor_half))
def hirep_halo_unpack(g, face, spinor_half, buf): _check(load().hirep_halo_unpack(g, face, spinor_half, buf))


def hirep_force_bytes(g):
    nb, na = ctypes.c_size_t(), ctypes.c_int()
    _check(load().hirep_force_bytes(g, ctypes.byref(nb), ctypes.byref(na)))
    return nb.value, na.value


def hirep_force_hopping(g, force, eta, xi, links): _check(load().hirep_force_hopping(g, force, eta, xi, links))


def hirep_g5Dphi_blocks_sq(g, out, inp, links, blocks_full): _check(load().hirep_g5Dphi_blocks_sq(g, out, inp, links, blocks_full))


def hirep_cg_g5Dphi_blocks_sq(g, x, b, links, blocks_full, tol, maxiter):
    it, res = ctypes.c_int(), (ctypes.c_double * 2)()
    _check(load().hirep_cg_g5Dphi_blocks_sq(g, x, b, links, blocks_full, tol, maxiter, ctypes.byref(it), res))
    return it.value, res[0]


def hirep_g5Dphi_clover_hat_sq(g, m0, csw, out, inp, links, clover, inv_odd):
    _check(load().hirep_g5Dphi_clover_hat_sq(g, m0, csw, out, inp, links, clover, inv_odd))


def hirep_g5Dphi_blocks_hat_sq(g, out, inp, links, blocks_even, inv_blocks_odd):
    _check(load().hirep_g5Dphi_blocks_hat_sq(g, out, inp, links, blocks_even, inv_blocks_odd))


def hirep_cg_g5Dphi_clover_hat_sq(g, m0, csw, x, b, links, clover, inv_odd, tol, maxiter):
    it, res = ctypes.c_int(), (ctypes.c_double * 2)()
    _check(load().hirep_cg_g5Dphi_clover_hat_sq(g, m0, csw, x, b, links, clover, inv_odd, tol, maxiter, ctypes.byref(it), res))
    return it.value, res[0]


def hirep_cg_g5Dphi_blocks_hat_sq(g, x, b, links, blocks_even, inv_blocks_odd, tol, maxiter):
    it, res = ctypes.c_int(), (ctypes.c_double * 2)()
    _check(load().hirep_cg_g5Dphi_blocks_hat_sq(g, x, b, links, blocks_even, inv_blocks_odd, tol, maxiter, ctypes.byref(it), res))
    return it.value, res[0]


def hirep_cg_g5Dphi_hat_sq(g, m0, x, b, links, tol, maxiter):
    it, res = ctypes.c_int(), (ctypes.c_double * 2)()
    _check(load().hirep_cg_g5Dphi_hat_sq(g, m0, x, b, links, tol, maxiter, ctypes.byref(it), res))
    return it.value, res[0]


def hirep_fma_peak(prec):
    out = ctypes.c_double()
    _check(load().hirep_fma_peak(prec, ctypes.byref(out)))
    return out.value


def hirep_sync(g): _check(load().hirep_sync(g))


def hirep_apply_host(g, op, m0, out_host_ptr, in_host_ptr, links_host_ptr):
    _check(load().hirep_apply_host(g, op, m0, out_host_ptr, in_host_ptr, links_host_ptr))


def hirep_apply_host_async(g, op, m0, out_host_ptr, in_host_ptr, links_host_ptr):
    _check(load().hirep_apply_host_async(g, op, m0, out_host_ptr, in_host_ptr, links_host_ptr))


# ---- convenience wrapper ---------------------------------------------------------------------------------
class Geometry:
    """Owns a hirep_geom handle; allocates native buffers as uint8 torch tensors on `device`."""

    def __init__(self, T, L, N_g, rep, prec="f64", device=None, bc=None, slab=None):
        """slab = (T_glob, t_start): T is then the number of OWNED slices and the local lattice has T + 2 (two ghost slices)."""
        import torch
        self.torch = torch
        self.prec = {"f64": F64, "f32": F32}[prec] if isinstance(prec, str) else prec
        self.device = torch.device(device if device is not None else "cuda:0")
        if slab is not None:
            self.handle = hirep_geom_create_slab(slab[0], L, N_g, rep, self.prec, slab[1], T)
            T = T + 2
        else:
            self.handle = hirep_geom_create(T, L, N_g, rep, self.prec)
        self.T, self.L, self.N_g, self.rep = T, L, N_g, rep
        self.sizes = hirep_geom_sizes(self.handle)
        self.d_R = self.sizes["d_R"]
        self.cdtype = torch.complex128 if self.prec == F64 else torch.complex64
        self.rdtype = torch.float64 if self.prec == F64 else torch.float32
        self.V = T * L ** 3
        if bc is not None:
            hirep_geom_set_bc(self.handle, bc)
        self.use_current_stream()

    def __del__(self):
        try:
            if getattr(self, "handle", None):
                hirep_geom_destroy(self.handle)
                self.handle = None
        except Exception:
            pass

    def use_current_stream(self):
        if self.device.type == "cuda" and self.torch.cuda.is_available():
            with self.torch.cuda.device(self.device):
                hirep_geom_set_stream(self.handle, self.torch.cuda.current_stream().cuda_stream)

    def _buf(self, nbytes):
        return self.torch.empty(nbytes, dtype=self.torch.uint8, device=self.device)

    def new_spinor(self, which=FULL):
        return self._buf(self.sizes["spinor_full" if which == FULL else "spinor_half"])

    def new_links_fund(self):
        return self._buf(self.sizes["links_fund"])

    def new_links_rep(self):
        return self._buf(self.sizes["links_rep"])

    # canonical <-> native
    def spinor_import(self, canonical, which=FULL):
        canonical = canonical.to(self.device, self.cdtype).contiguous()
        n = self.V if which == FULL else self.V // 2
        assert canonical.shape == (n, 4, self.d_R), canonical.shape
        native = self.new_spinor(which)
        hirep_spinor_import(self.handle, native.data_ptr(), canonical.data_ptr(), which)
        return native

    def spinor_export(self, native, which=FULL):
        n = self.V if which == FULL else self.V // 2
        canonical = self.torch.empty((n, 4, self.d_R), dtype=self.cdtype, device=self.device)
        hirep_spinor_export(self.handle, canonical.data_ptr(), native.data_ptr(), which)
        return canonical

    def links_import(self, canonical_fund):
        canonical_fund = canonical_fund.to(self.device, self.cdtype).contiguous()
        assert canonical_fund.shape == (self.V, 4, self.N_g, self.N_g), canonical_fund.shape
        native = self.new_links_fund()
        hirep_links_import(self.handle, native.data_ptr(), canonical_fund.data_ptr())
        return native

    def links_to_rep(self, native_fund, out=None):
        out = self.new_links_rep() if out is None else out
        hirep_links_to_rep(self.handle, out.data_ptr(), native_fund.data_ptr())
        return out

    def links_rep_export(self, native_rep, bwd=False):
        dt = self.rdtype if self.sizes["rep_is_real"] else self.cdtype
        canonical = self.torch.empty((self.V, 4, self.d_R, self.d_R), dtype=dt, device=self.device)
        (hirep_links_rep_export_bwd if bwd else hirep_links_rep_export)(self.handle, canonical.data_ptr(), native_rep.data_ptr())
        return canonical

    # operators (allocate `out` unless given)
    def Dphi(self, m0, inp, links, out=None):
        out = self.new_spinor(FULL) if out is None else out
        hirep_Dphi(self.handle, m0, out.data_ptr(), inp.data_ptr(), links.data_ptr())
        return out

    def Dphi_eo(self, inp_odd, links, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        hirep_Dphi_eo(self.handle, out.data_ptr(), inp_odd.data_ptr(), links.data_ptr())
        return out

    def Dphi_oe(self, inp_even, links, out=None):
        out = self.new_spinor(ODD) if out is None else out
        hirep_Dphi_oe(self.handle, out.data_ptr(), inp_even.data_ptr(), links.data_ptr())
        return out

    def Dphi_hat(self, m0, inp_even, links, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        hirep_Dphi_hat(self.handle, m0, out.data_ptr(), inp_even.data_ptr(), links.data_ptr())
        return out

    def Dphi_hat_static(self, m0, inp_even, links, out):
        """hirep_Dphi_hat_static: no allocation inside the call, so the caller passes `out` (include/hirep_b200.h)."""
        hirep_Dphi_hat_static(self.handle, m0, out.data_ptr(), inp_even.data_ptr(), links.data_ptr())
        return out

    def g5Dphi_sq(self, m0, inp, links, out=None):
        out = self.new_spinor(FULL) if out is None else out
        hirep_g5Dphi_sq(self.handle, m0, out.data_ptr(), inp.data_ptr(), links.data_ptr())
        return out

    def g5Dphi_hat(self, m0, inp_even, links, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        hirep_g5Dphi_hat(self.handle, m0, out.data_ptr(), inp_even.data_ptr(), links.data_ptr())
        return out

    def g5Dphi_hat_sq(self, m0, inp_even, links, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        hirep_g5Dphi_hat_sq(self.handle, m0, out.data_ptr(), inp_even.data_ptr(), links.data_ptr())
        return out

    def apply_host(self, op, m0, inp_host, links_host=None):
        """End-to-end through hirep_apply_host: host (ideally pinned) canonical tensors in, host tensor out."""
        out = self.torch.empty_like(inp_host)
        if inp_host.is_pinned():
            out = out.pin_memory()
        hirep_apply_host(self.handle, op, m0, out.data_ptr(), inp_host.data_ptr(),
                         links_host.data_ptr() if links_host is not None else None)
        return out

    # linear algebra / reductions / CG on native buffers (tensors); `which` gives the extent
    def lc(self, which, xi, r1, eta, r2, zeta): hirep_spinor_lc(self.handle, which, xi.data_ptr(), r1, eta.data_ptr(), r2, zeta.data_ptr())
    def clc(self, which, xi, c1, eta, c2, zeta): hirep_spinor_clc(self.handle, which, xi.data_ptr(), c1, eta.data_ptr(), c2, zeta.data_ptr())
    def lc_add_assign(self, which, xi, r1, eta, r2, zeta): hirep_spinor_lc_add_assign(self.handle, which, xi.data_ptr(), r1, eta.data_ptr(), r2, zeta.data_ptr())
    def clc_add_assign(self, which, xi, c1, eta, c2, zeta): hirep_spinor_clc_add_assign(self.handle, which, xi.data_ptr(), c1, eta.data_ptr(), c2, zeta.data_ptr())
    def lc1(self, which, xi, c1, eta): hirep_spinor_lc1(self.handle, which, xi.data_ptr(), c1, eta.data_ptr())
    def lc2(self, which, xi, c1, c2, eta): hirep_spinor_lc2(self.handle, which, xi.data_ptr(), c1, c2, eta.data_ptr())
    def lc3(self, which, xi, c1, eta, c2, zeta): hirep_spinor_lc3(self.handle, which, xi.data_ptr(), c1, eta.data_ptr(), c2, zeta.data_ptr())
    def prod(self, which, xi, eta): return hirep_spinor_prod(self.handle, which, xi.data_ptr(), eta.data_ptr())
    def sqnorm(self, which, xi): return hirep_spinor_sqnorm(self.handle, which, xi.data_ptr())
    def max_norm(self, which, eta): return hirep_spinor_max_norm(self.handle, which, eta.data_ptr())

    def cg_g5Dphi_sq(self, m0, b, links, tol, maxiter, out=None):
        out = self.new_spinor(FULL) if out is None else out
        it, res = hirep_cg_g5Dphi_sq(self.handle, m0, out.data_ptr(), b.data_ptr(), links.data_ptr(), tol, maxiter)
        return out, it, res

    def g5_lc(self, which, xi, c1, c2, eta): hirep_spinor_g5_lc(self.handle, which, xi.data_ptr(), c1, c2, eta.data_ptr())

    def g5_lc_add_assign(self, which, xi, c0, c1, c2, eta): hirep_spinor_g5_lc_add_assign(self.handle, which, xi.data_ptr(), c0, c1, c2, eta.data_ptr())
    def gamma(self, which, mu, xi, eta): hirep_spinor_gamma(self.handle, which, mu, xi.data_ptr(), eta.data_ptr())
    def g5_prod(self, which, xi, eta): return hirep_spinor_g5_prod(self.handle, which, xi.data_ptr(), eta.data_ptr())

    def Dphi_tm(self, m0, mu, inp, links, out=None):
        out = self.new_spinor(FULL) if out is None else out
        hirep_Dphi_tm(self.handle, m0, mu, out.data_ptr(), inp.data_ptr(), links.data_ptr())
        return out

    def Dphi_tm_sq(self, m0, mu, inp, links, out=None):
        out = self.new_spinor(FULL) if out is None else out
        hirep_Dphi_tm_sq(self.handle, m0, mu, out.data_ptr(), inp.data_ptr(), links.data_ptr())
        return out

    def Dphi_tm_hat(self, m0, mu, inp_even, links, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        hirep_Dphi_tm_hat(self.handle, m0, mu, out.data_ptr(), inp_even.data_ptr(), links.data_ptr())
        return out

    # clover term (Eq 47-49)
    def clover_field(self, links_rep, out=None):
        if out is None:
            out = self.torch.empty(hirep_clover_bytes(self.handle), dtype=self.torch.uint8, device=self.device)
        hirep_clover_field(self.handle, out.data_ptr(), links_rep.data_ptr())
        return out

    def clover_export(self, clover):
        canonical = self.torch.empty((self.V, 2, 2 * self.d_R, 2 * self.d_R), dtype=self.cdtype, device=self.device)
        hirep_clover_export(self.handle, canonical.data_ptr(), clover.data_ptr())
        return canonical

    def Cphi(self, m0, csw, inp, clover, out=None):
        out = self.new_spinor(FULL) if out is None else out
        hirep_Cphi(self.handle, m0, csw, out.data_ptr(), inp.data_ptr(), clover.data_ptr())
        return out

    def Dphi_clover(self, m0, csw, inp, links, clover, out=None):
        out = self.new_spinor(FULL) if out is None else out
        hirep_Dphi_clover(self.handle, m0, csw, out.data_ptr(), inp.data_ptr(), links.data_ptr(), clover.data_ptr())
        return out

    def clover_inv_field(self, m0, csw, parity, clover, out=None):
        if out is None:
            out = self.torch.empty(hirep_clover_inv_bytes(self.handle), dtype=self.torch.uint8, device=self.device)
        hirep_clover_inv_field(self.handle, m0, csw, parity, out.data_ptr(), clover.data_ptr())
        return out

    def Cphi_inv(self, parity, inp_half, inv, out=None):
        out = self.new_spinor(parity) if out is None else out
        hirep_Cphi_inv(self.handle, out.data_ptr(), inp_half.data_ptr(), inv.data_ptr())
        return out

    def Dphi_clover_hat(self, m0, csw, inp_even, links, clover, inv_odd, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        hirep_Dphi_clover_hat(self.handle, m0, csw, out.data_ptr(), inp_even.data_ptr(), links.data_ptr(), clover.data_ptr(), inv_odd.data_ptr())
        return out

    def clover_exp_field(self, m0, csw, clover, inverse=False):
        """Full-lattice block field of Eq 50: even blocks followed by odd blocks (or their inverses)."""
        nb = hirep_clover_inv_bytes(self.handle)
        out = self.torch.empty(2 * nb, dtype=self.torch.uint8, device=self.device)
        for parity in (EVEN, ODD):
            hirep_clover_exp_field(self.handle, m0, csw, parity, int(inverse), out[parity * nb:].data_ptr(), clover.data_ptr())
        return out

    def Dphi_blocks(self, inp, links, blocks_full, out=None):
        out = self.new_spinor(FULL) if out is None else out
        hirep_Dphi_blocks(self.handle, out.data_ptr(), inp.data_ptr(), links.data_ptr(), blocks_full.data_ptr())
        return out

    def Dphi_blocks_hat(self, inp_even, links, blocks_even, inv_blocks_odd, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        hirep_Dphi_blocks_hat(self.handle, out.data_ptr(), inp_even.data_ptr(), links.data_ptr(), blocks_even.data_ptr(), inv_blocks_odd.data_ptr())
        return out

    def cg_mshift_g5Dphi_sq(self, m0, shifts, b, links, tol, maxiter):
        outs = [self.new_spinor(FULL) for _ in shifts]
        it, res = hirep_cg_mshift_g5Dphi_sq(self.handle, m0, shifts, [o.data_ptr() for o in outs], b.data_ptr(), links.data_ptr(), tol, maxiter)
        return outs, it, res

    def bicgstab(self, op, m0, b, links, tol, maxiter, out=None):
        out = self.new_spinor(FULL if op == OP_DPHI else EVEN) if out is None else out
        it, res = hirep_bicgstab(self.handle, op, m0, out.data_ptr(), b.data_ptr(), links.data_ptr(), tol, maxiter)
        return out, it, res

    def cg_Dphi_tm_sq(self, m0, mu, b, links, tol, maxiter, out=None):
        out = self.new_spinor(FULL) if out is None else out
        it, res = hirep_cg_Dphi_tm_sq(self.handle, m0, mu, out.data_ptr(), b.data_ptr(), links.data_ptr(), tol, maxiter)
        return out, it, res

    def g5Dphi_clover_sq(self, m0, csw, inp, links, clover, out=None):
        out = self.new_spinor(FULL) if out is None else out
        hirep_g5Dphi_clover_sq(self.handle, m0, csw, out.data_ptr(), inp.data_ptr(), links.data_ptr(), clover.data_ptr())
        return out

    def cg_g5Dphi_clover_sq(self, m0, csw, b, links, clover, tol, maxiter, out=None):
        out = self.new_spinor(FULL) if out is None else out
        it, res = hirep_cg_g5Dphi_clover_sq(self.handle, m0, csw, out.data_ptr(), b.data_ptr(), links.data_ptr(), clover.data_ptr(), tol, maxiter)
        return out, it, res

    def set_region(self, region): hirep_set_region(self.handle, region)

    def halo_pack(self, face, spinor_half):
        buf = self._buf(hirep_halo_bytes(self.handle))
        hirep_halo_pack(self.handle, face, buf.data_ptr(), spinor_half.data_ptr())
        return buf

    def halo_unpack(self, face, spinor_half, buf): hirep_halo_unpack(self.handle, face, spinor_half.data_ptr(), buf.data_ptr())

    def force_hopping(self, eta, xi, links, out=None):
        """F^a_mu(x) of Eq 20-21 as a real tensor [V, 4, N_g^2 - 1] in canonical site order."""
        nb, na = hirep_force_bytes(self.handle)
        out = out if out is not None else self.torch.empty((self.V, 4, na), dtype=self.rdtype, device=self.device)
        hirep_force_hopping(self.handle, out.data_ptr(), eta.data_ptr(), xi.data_ptr(), links.data_ptr())
        return out

    def g5Dphi_blocks_sq(self, inp, links, blocks_full, out=None):
        out = self.new_spinor(FULL) if out is None else out
        hirep_g5Dphi_blocks_sq(self.handle, out.data_ptr(), inp.data_ptr(), links.data_ptr(), blocks_full.data_ptr())
        return out

    def cg_g5Dphi_blocks_sq(self, b, links, blocks_full, tol, maxiter, out=None):
        out = self.new_spinor(FULL) if out is None else out
        it, res = hirep_cg_g5Dphi_blocks_sq(self.handle, out.data_ptr(), b.data_ptr(), links.data_ptr(), blocks_full.data_ptr(), tol, maxiter)
        return out, it, res

    def g5Dphi_clover_hat_sq(self, m0, csw, inp_even, links, clover, inv_odd, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        hirep_g5Dphi_clover_hat_sq(self.handle, m0, csw, out.data_ptr(), inp_even.data_ptr(), links.data_ptr(), clover.data_ptr(), inv_odd.data_ptr())
        return out

    def g5Dphi_blocks_hat_sq(self, inp_even, links, blocks_even, inv_blocks_odd, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        hirep_g5Dphi_blocks_hat_sq(self.handle, out.data_ptr(), inp_even.data_ptr(), links.data_ptr(), blocks_even.data_ptr(), inv_blocks_odd.data_ptr())
        return out

    def cg_g5Dphi_clover_hat_sq(self, m0, csw, b_even, links, clover, inv_odd, tol, maxiter, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        it, res = hirep_cg_g5Dphi_clover_hat_sq(self.handle, m0, csw, out.data_ptr(), b_even.data_ptr(), links.data_ptr(), clover.data_ptr(),
                                                inv_odd.data_ptr(), tol, maxiter)
        return out, it, res

    def cg_g5Dphi_blocks_hat_sq(self, b_even, links, blocks_even, inv_blocks_odd, tol, maxiter, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        it, res = hirep_cg_g5Dphi_blocks_hat_sq(self.handle, out.data_ptr(), b_even.data_ptr(), links.data_ptr(), blocks_even.data_ptr(),
                                                inv_blocks_odd.data_ptr(), tol, maxiter)
        return out, it, res

    def cg_g5Dphi_hat_sq(self, m0, b_even, links, tol, maxiter, out=None):
        out = self.new_spinor(EVEN) if out is None else out
        it, res = hirep_cg_g5Dphi_hat_sq(self.handle, m0, out.data_ptr(), b_even.data_ptr(), links.data_ptr(), tol, maxiter)
        return out, it, res

    def set_link_mode(self, mode): hirep_set_link_mode(self.handle, mode)
    def set_kernel_variant(self, v): hirep_set_kernel_variant(self.handle, v)
    def set_tuning(self, key, value): hirep_set_tuning(self.handle, key, value)
    def reserve(self, what=RESERVE_OPERATORS | RESERVE_SOLVERS): hirep_geom_reserve(self.handle, what)
    def set_bc(self, sign): hirep_geom_set_bc(self.handle, sign)
    def sync(self): hirep_sync(self.handle)
    def launch_count(self): return hirep_launch_count(self.handle)
