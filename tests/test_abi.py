"""CPU-only checks of the boundary: the library loads, exports every symbol include/hirep_b200.h declares, and
its host-side logic (argument validation, sizes, error reporting) behaves as documented.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def hirep():
    import __graft_entry__ as ge
    ge.build_cuda()
    from paper_2503_06721_b200 import hirep as h
    h.load()
    return h


def header_symbols():
    text = open(os.path.join(ROOT, "include", "hirep_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hirep_[A-Za-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(hirep):
    syms = header_symbols()
    assert len(syms) >= 20
    lib = ctypes.CDLL(hirep.LIB_PATH)
    for s in syms:
        assert hasattr(lib, s), s
    assert sorted(hirep.SYMBOLS) == syms          # the Python binding lists exactly the header's functions


def test_geom_create_validation_and_sizes(hirep):
    for bad in [(3, 4, 3, 0, 0), (4, 5, 3, 0, 0), (0, 4, 3, 0, 0), (4, 4, 1, 0, 0), (4, 4, 7, 0, 0), (4, 4, 3, 9, 0), (4, 4, 3, 0, 5)]:
        with pytest.raises(hirep.HirepError):
            hirep.hirep_geom_create(*bad)
    assert "N_g" in hirep.hirep_last_error() or "precision" in hirep.hirep_last_error()
    g = hirep.hirep_geom_create(4, 4, 2, hirep.ASY, 0)       # SU(2) 2AS, d_R = 1 (R = det U = 1): allowed
    assert hirep.hirep_geom_sizes(g)["d_R"] == 1
    hirep.hirep_geom_destroy(g)
    # sizes: SU(3) FUND 32^4 fp64 (BASELINE configs[1]) -- SURVEY.md 8(a) table: 201 MB spinor, 604 MB links (x2 gather copies)
    g = hirep.hirep_geom_create(32, 32, 3, hirep.FUND, hirep.F64)
    sz = hirep.hirep_geom_sizes(g)
    V = 32 ** 4
    assert sz["d_R"] == 3 and not sz["rep_is_real"]
    assert sz["spinor_full"] == V * 12 * 16 and sz["spinor_half"] * 2 == sz["spinor_full"]
    assert sz["links_fund"] == 2 * (V // 2) * 8 * 9 * 16 == sz["links_rep"]
    hirep.hirep_geom_destroy(g)
    # SU(2) ADJ fp32: real links, d_R = 3; ragged lattice pads the last tile
    g = hirep.hirep_geom_create(2, 6, 2, hirep.ADJ, hirep.F32)
    sz = hirep.hirep_geom_sizes(g)
    nh = 2 * 6 ** 3 // 2
    ntiles = (nh + 31) // 32
    assert sz["rep_is_real"] and sz["d_R"] == 3
    assert sz["links_rep"] == 2 * ntiles * 8 * 9 * 32 * 4
    assert sz["spinor_half"] == ntiles * 12 * 32 * 8
    hirep.hirep_geom_destroy(g)


def test_maximum_sizes(hirep):
    """Largest lattices: byte counts are computed in size_t without overflow, and a lattice whose half-volume does not
    fit 32-bit site indices is rejected (no partial handle)."""
    g = hirep.hirep_geom_create(256, 128, 6, hirep.ADJ, hirep.F64)          # V = 2^29 sites, d_R = 35
    sz = hirep.hirep_geom_sizes(g)
    V = 256 * 128 ** 3
    assert sz["spinor_full"] == V * 4 * 35 * 16                              # 1.2 TB: far beyond one GPU, still exact
    assert sz["links_rep"] == 2 * (V // 2) * 8 * 35 * 35 * 8 and sz["links_fund"] == 2 * (V // 2) * 8 * 36 * 16
    hirep.hirep_geom_destroy(g)
    with pytest.raises(hirep.HirepError, match="too large"):
        hirep.hirep_geom_create(4096, 128, 3, hirep.FUND, hirep.F64)         # V/2 = 2^32 sites
    g = hirep.hirep_geom_create(2, 2, 2, hirep.FUND, hirep.F32)              # smallest lattice: 8 sites per parity, one padded tile
    sz = hirep.hirep_geom_sizes(g)
    assert sz["spinor_half"] == 1 * 8 * 32 * 8 and sz["links_fund"] == 2 * 1 * 8 * 4 * 32 * 8
    hirep.hirep_geom_destroy(g)


@pytest.mark.parametrize("n,rep,d", [(2, 0, 2), (3, 0, 3), (2, 1, 3), (4, 3, 6), (6, 1, 35), (3, 2, 6), (4, 2, 10), (6, 3, 15)])
def test_rep_dimensions_table1(hirep, n, rep, d):
    g = hirep.hirep_geom_create(4, 4, n, rep, hirep.F64)
    assert hirep.hirep_geom_sizes(g)["d_R"] == d            # Tbl 1
    hirep.hirep_geom_destroy(g)


def test_argument_errors_without_gpu(hirep):
    g = hirep.hirep_geom_create(4, 4, 3, hirep.FUND, hirep.F64)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_geom_set_bc(g, (1, 1, 0, 1))
    hirep.hirep_geom_set_bc(g, (1, -1, 1, 1))
    with pytest.raises(hirep.HirepError):
        hirep.hirep_set_link_mode(g, 7)
    # null / misaligned / aliased pointers are rejected before any CUDA call
    with pytest.raises(hirep.HirepError):
        hirep.hirep_Dphi_eo(g, None, 4096, 8192)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_Dphi_eo(g, 4096 + 8, 8192, 16384)
    assert "aligned" in hirep.hirep_last_error()
    with pytest.raises(hirep.HirepError):
        hirep.hirep_Dphi(g, 0.1, 4096, 4096, 8192)
    assert "alias" in hirep.hirep_last_error()
    assert hirep.hirep_launch_count(g) == 0
    hirep.hirep_geom_destroy(g)
    hirep.hirep_geom_destroy(None)


def test_new_entry_points_argument_errors_without_gpu(hirep):
    g = hirep.hirep_geom_create(4, 4, 3, hirep.FUND, hirep.F64)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_spinor_lc(g, hirep.FULL, None, 1.0, 4096, 1.0, 8192)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_spinor_lc(g, 5, 4096, 1.0, 8192, 1.0, 12288)          # bad extent selector
    with pytest.raises(hirep.HirepError):
        hirep.hirep_spinor_prod(g, hirep.EVEN, 4096 + 4, 8192)            # misaligned
    with pytest.raises(hirep.HirepError):
        hirep.hirep_cg_g5Dphi_sq(g, 0.1, 4096, 4096, 8192, 1e-8, 10)      # x aliases b
    with pytest.raises(hirep.HirepError):
        hirep.hirep_cg_g5Dphi_sq(g, 0.1, 4096, 8192, 12288, 0.0, 10)      # tol must be positive
    with pytest.raises(hirep.HirepError):
        hirep.hirep_set_tuning(g, 99, 1)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_set_tuning(g, hirep.TUNE_FUSE_DIAG, 2)
    hirep.hirep_set_tuning(g, hirep.TUNE_FUSE_DIAG, 0)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_geom_reserve(g, 0)                                     # no flag
    with pytest.raises(hirep.HirepError):
        hirep.hirep_geom_reserve(g, 8)                                     # unknown flag
    with pytest.raises(hirep.HirepError) as ei:
        hirep.hirep_geom_reserve(g, hirep.RESERVE_OPERATORS)               # no device here: an error, not a silent success
    assert ei.value.rc in (hirep.ECUDA, hirep.ENOMEM)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_set_tuning(g, hirep.TUNE_MAX_CTAS, -2)
    hirep.hirep_set_tuning(g, hirep.TUNE_MAX_CTAS, 4)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_fma_peak(7)
    assert hirep.hirep_launch_count(g) == 0
    hirep.hirep_geom_destroy(g)


def test_clover_entry_points_argument_errors_without_gpu(hirep):
    g = hirep.hirep_geom_create(4, 4, 3, hirep.FUND, hirep.F64)
    # 4 d_R^2 complex per site, 256 sites (= 8 tiles of 32 lanes), 16 bytes per complex: both fields are the same size
    assert hirep.hirep_clover_bytes(g) == 256 * 4 * 9 * 16
    assert hirep.hirep_clover_inv_bytes(g) == 128 * 2 * 36 * 16
    with pytest.raises(hirep.HirepError):
        hirep.hirep_clover_field(g, None, 4096)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_Cphi(g, 0.1, 1.0, 4096, 4096, 8192)                    # out aliases in
    with pytest.raises(hirep.HirepError):
        hirep.hirep_Dphi_clover(g, 0.1, 1.0, 4096, 8192, 12288 + 8, 16384)  # misaligned links
    with pytest.raises(hirep.HirepError):
        hirep.hirep_clover_inv_field(g, 0.1, 1.0, hirep.FULL, 4096, 8192)  # parity must be EVEN or ODD
    with pytest.raises(hirep.HirepError):
        hirep.hirep_clover_exp_field(g, -4.0, 1.0, hirep.ODD, 0, 4096, 8192)   # 4 + m0 = 0
    with pytest.raises(hirep.HirepError):
        hirep.hirep_Dphi_blocks_hat(g, 4096, 4096, 8192, 12288, 16384)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_cg_g5Dphi_clover_sq(g, 0.1, 1.0, 4096, 4096, 8192, 12288, 1e-8, 10)   # x aliases b
    with pytest.raises(hirep.HirepError):
        hirep.hirep_g5Dphi_clover_hat_sq(g, 0.1, 1.0, 4096, 4096, 8192, 12288, 16384)      # out aliases in
    with pytest.raises(hirep.HirepError):
        hirep.hirep_g5Dphi_blocks_sq(g, 4096, 4096, 8192, 12288)                           # out aliases in
    with pytest.raises(hirep.HirepError):
        hirep.hirep_cg_g5Dphi_blocks_sq(g, 4096, 8192, 12288, 16384, 1e-8, -1)             # maxiter < 0
    with pytest.raises(hirep.HirepError):
        hirep.hirep_g5Dphi_blocks_hat_sq(g, 4096, 8192, 12288, None, 16384)                # NULL blocks
    with pytest.raises(hirep.HirepError):
        hirep.hirep_cg_g5Dphi_clover_hat_sq(g, 0.1, 1.0, 4096, 4096, 8192, 12288, 16384, 1e-8, 10)   # x aliases b
    with pytest.raises(hirep.HirepError):
        hirep.hirep_cg_g5Dphi_blocks_hat_sq(g, 4096, 8192, 12288, 16384, 20480, -1.0, 10)  # tol <= 0
    hirep.hirep_set_link_mode(g, hirep.LINKS_REBUILD)
    with pytest.raises(hirep.HirepError):
        hirep.hirep_clover_field(g, 4096, 8192)                            # needs the stored represented links
    assert hirep.hirep_launch_count(g) == 0
    hirep.hirep_geom_destroy(g)


def test_compute_without_device_is_an_error_not_a_fallback(hirep):
    """On a box without a GPU every compute entry point reports HIREP_ECUDA (-3); nothing is computed on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("needs a box without a CUDA device")
    g = hirep.hirep_geom_create(4, 4, 3, hirep.FUND, hirep.F64)
    buf = (ctypes.c_char * (1 << 20))()
    base = (ctypes.addressof(buf) + 255) & ~255
    with pytest.raises(hirep.HirepError, match="hirep error -3"):
        hirep.hirep_Dphi_eo(g, base, base + 65536, base + 131072)
    with pytest.raises(hirep.HirepError, match="hirep error -3"):
        hirep.hirep_links_to_rep(g, base, base + 262144)
    with pytest.raises(hirep.HirepError, match="hirep error -3"):
        hirep.hirep_spinor_lc(g, hirep.EVEN, base, 1.0, base + 65536, 1.0, base + 131072)
    hirep.hirep_geom_destroy(g)


def test_missing_library_fails_loudly(hirep, monkeypatch):
    """The product path must not fall back to anything when the CUDA library is absent."""
    monkeypatch.setattr(hirep, "_lib", None)
    monkeypatch.setattr(hirep, "LIB_PATH", os.path.join(ROOT, "no_such_dir", "libhirep_b200.so"))
    with pytest.raises(hirep.HirepError, match="no CPU fallback"):
        hirep.load()


def test_product_does_not_import_oracle():
    """Neither the package nor bench's product arm may route through oracle/ (checked textually on the package)."""
    pkg = os.path.join(ROOT, "paper_2503_06721_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                for needle in ("import oracle", "from oracle", "liboracle", "hirep_oracle", "oracle/"):
                    assert needle not in src, (needle, os.path.join(dirpath, f))
