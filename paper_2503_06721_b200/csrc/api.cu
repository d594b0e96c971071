// api.cu -- the C-ABI of include/hirep_b200.h: argument checking, workspace, operator composition.
//
// Operator composition out of stencil passes (hop_small.cuh / hop_large.cuh), out = a*self + b*hop(in):
//   Dphi_eo / Dphi_oe : a = 0,        b = -1/2                                  (Eq 41)
//   Dphi              : a = 4 + m,    b = -1/2, both parities in one launch     (Eq 8,  L207)
//   Dphi_hat          : tmp_o = D_oe in_e ; out_e = (4+m)^2 in_e + 1/2 hop(tmp_o)   (Eq 44)
//   g5Dphi_sq         : tmp = g5 D in ; out = g5 D tmp                          (Eq 11; L772)
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/hirep_b200.h"
#include "hop_dispatch.cuh"

using namespace hirep;

struct hirep_geom {
    Geo geo;
    int N, rep, prec, dR, real;
    int mode, variant;
    int tune_max_ctas, sum_alg, tune_pace, tune_fuse_diag;   // hirep_set_tuning
    int slab, region;             // hirep_geom_create_slab / hirep_set_region
    cudaStream_t stream;
    void *ws_half, *ws_half2, *ws_half3, *ws_full;   // workspace spinors (lazy)
    void *ws_red;                   // reduction partials + 4 result doubles (lazy)
    void *ws_red2;                  // partials written by stencil launches with a fused reduction (lazy)
    void *cg_r, *cg_p, *cg_Ap;      // CG work fields (lazy)
    void *ms_p[HIREP_MAX_SHIFTS];    // multi-shift CG direction fields (lazy)
    void *bi_s, *bi_t;              // BiCGstab work fields (lazy)
    void *ws_exp;                   // hirep_clover_exp_field work matrices (lazy)
    // hirep_apply_host staging (lazy)
    void *h_links_canon, *h_links_fund, *h_links_rep, *h_in_canon, *h_in_native, *h_out_native, *h_out_canon, *h_out_canon2;
    cudaStream_t copy_stream;       // device -> host copies of hirep_apply_host[_async] (lazy)
    cudaEvent_t ev_done[2], ev_copied[2];
    int host_slot, host_events;
    int host_links_ready;
    double *h_scal;                 // pinned: the CG's scalars read back without blocking the launches behind them (lazy)
    cudaEvent_t ev_scal;
    int *force_rowptr, *force_jk;   // sparse represented generators T_R^a for hirep_force_hopping (lazy)
    void *force_val, *force_dense;  // ... and the dense table [a][j][k] (double2)
    int *dev_flags;                 // device word set by kernels that met a numerical breakdown (clover block inverse / exponential); read by hirep_sync
    long launches;
    int device;                     // CUDA device current at hirep_geom_create (-1: none); compute calls check it
    size_t bytes_spinor_half, bytes_links_fund, bytes_links_rep;
};

static thread_local char g_err[512] = "";

static int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}
static int cuda_fail(cudaError_t e, const char *what) {
    return fail(HIREP_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}
static int kern_result(hirep_geom *g, int rc, const char *what, int nlaunch = 1) {
    if (rc == 0) { g->launches += nlaunch; return HIREP_OK; }
    if (rc == KERR_UNSUPPORTED)
        return fail(HIREP_EUNSUPPORTED, "%s: no kernel instantiated for N_g=%d rep=%d prec=%d mode=%d variant=%d", what, g->N,
                    g->rep, g->prec, g->mode, g->variant);
    return cuda_fail((cudaError_t)rc, what);
}
static bool misaligned(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) != 0; }
// a solver stopped on a non-finite or degenerate scalar: drain the stream (kernels may be queued ahead), then report.
// The solution field is undefined after a breakdown (include/hirep_b200.h).
static int breakdown(hirep_geom *g, const char *fmt, ...) {
    cudaStreamSynchronize(g->stream);
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return HIREP_EBREAKDOWN;
}

extern "C" const char *hirep_last_error(void) { return g_err; }

static int rep_dim(int N, int rep) {
    switch (rep) {
    case HIREP_FUND: return N;
    case HIREP_ADJ: return N * N - 1;
    case HIREP_SYM: return N * (N + 1) / 2;
    case HIREP_ASY: return N * (N - 1) / 2;
    }
    return -1;
}

extern "C" int hirep_geom_create(int T, int L, int N_g, int rep, int prec, hirep_geom **out) {
    if (!out) return fail(HIREP_EINVAL, "hirep_geom_create: out is NULL");
    *out = nullptr;
    if (T < 2 || L < 2 || (T & 1) || (L & 1)) return fail(HIREP_EINVAL, "hirep_geom_create: extents must be even and >= 2 (T=%d L=%d)", T, L);
    if (N_g < 2 || N_g > 6) return fail(HIREP_EINVAL, "hirep_geom_create: N_g=%d outside 2..6", N_g);
    if (rep < 0 || rep > 3) return fail(HIREP_EINVAL, "hirep_geom_create: unknown representation %d", rep);
    if (prec != HIREP_F64 && prec != HIREP_F32) return fail(HIREP_EINVAL, "hirep_geom_create: unknown precision %d", prec);
    const long long V = (long long)T * L * L * L;
    if (V / 2 + 32 >= (1LL << 31)) return fail(HIREP_EINVAL, "hirep_geom_create: lattice too large for 32-bit site indices");
    const int dR = rep_dim(N_g, rep);
    hirep_geom *g = new (std::nothrow) hirep_geom;
    if (!g) return fail(HIREP_ENOMEM, "hirep_geom_create: out of host memory");
    memset(g, 0, sizeof(*g));
    g->geo.T = T; g->geo.L = L; g->geo.Lh = L / 2;
    g->geo.Nh = (int)(V / 2);
    g->geo.n_tiles = (g->geo.Nh + TILE - 1) / TILE;
    g->geo.bc[0] = -1; g->geo.bc[1] = g->geo.bc[2] = g->geo.bc[3] = 1;
    g->geo.t0 = 0; g->geo.Tg = T;
    g->tune_max_ctas = 0; g->sum_alg = 2; g->tune_fuse_diag = 1;
    g->N = N_g; g->rep = rep; g->prec = prec; g->dR = dR; g->real = (rep == HIREP_ADJ);
    const size_t w = prec == HIREP_F64 ? 8 : 4;
    g->bytes_spinor_half = (size_t)g->geo.n_tiles * 4 * dR * TILE * 2 * w;
    g->bytes_links_fund = (size_t)2 * g->geo.n_tiles * 8 * N_g * N_g * TILE * 2 * w;
    g->bytes_links_rep = (size_t)2 * g->geo.n_tiles * 8 * dR * dR * TILE * (g->real ? 1 : 2) * w;
    if (cudaGetDevice(&g->device) != cudaSuccess) { g->device = -1; cudaGetLastError(); }
    *out = g;
    return HIREP_OK;
}

// ---- slab of a lattice block-partitioned in t (Fig 1) ---------------------------------
extern "C" int hirep_geom_create_slab(int T_glob, int L, int N_g, int rep, int prec, int t_start, int T_loc, hirep_geom **out) {
    if (!out) return fail(HIREP_EINVAL, "hirep_geom_create_slab: out is NULL");
    *out = nullptr;
    if (T_glob < 2 || (T_glob & 1) || T_loc < 2 || (T_loc & 1) || t_start < 0 || (t_start & 1) || t_start + T_loc > T_glob)
        return fail(HIREP_EINVAL, "hirep_geom_create_slab: T_glob=%d t_start=%d T_loc=%d (all even, T_loc >= 2, t_start + T_loc <= T_glob)", T_glob, t_start, T_loc);
    const int rc = hirep_geom_create(T_loc + 2, L, N_g, rep, prec, out);
    if (rc) return rc;
    (*out)->geo.t0 = (t_start - 1 + T_glob) % T_glob;   // local slice 0 is the ghost slice before the first owned one
    (*out)->geo.Tg = T_glob;
    (*out)->slab = 1;
    (*out)->region = HIREP_REGION_OWNED;
    return HIREP_OK;
}
extern "C" int hirep_set_region(hirep_geom *g, int region) {
    if (!g) return fail(HIREP_EINVAL, "hirep_set_region: NULL geometry");
    if (region < HIREP_REGION_ALL || region > HIREP_REGION_BOUNDARY) return fail(HIREP_EINVAL, "hirep_set_region: unknown region %d", region);
    if (!g->slab && region != HIREP_REGION_ALL) return fail(HIREP_EINVAL, "hirep_set_region: only a slab geometry has owned / interior / boundary regions");
    g->region = region;
    return HIREP_OK;
}
static size_t halo_bytes(const hirep_geom *g) {
    return (size_t)g->geo.L * g->geo.L * g->geo.Lh * 2 * g->dR * 2 * (g->prec == HIREP_F64 ? 8 : 4);
}
extern "C" int hirep_halo_bytes(const hirep_geom *g, size_t *bytes) {
    if (!g || !bytes) return fail(HIREP_EINVAL, "hirep_halo_bytes: NULL argument");
    *bytes = halo_bytes(g);
    return HIREP_OK;
}

extern "C" int hirep_geom_destroy(hirep_geom *g) {
    if (!g) return HIREP_OK;
    for (void *b : g->ms_p)
        if (b) cudaFree(b);
    void *bufs[] = {g->ws_red2, g->dev_flags, g->force_rowptr, g->force_jk, g->force_val, g->force_dense, g->ws_exp, g->ws_half, g->ws_half2, g->ws_half3, g->ws_full, g->ws_red, g->cg_r, g->cg_p, g->cg_Ap, g->bi_s, g->bi_t, g->h_links_canon, g->h_links_fund, g->h_links_rep, g->h_in_canon,
                    g->h_in_native, g->h_out_native, g->h_out_canon, g->h_out_canon2};
    if (g->host_events) {
        for (int i = 0; i < 2; ++i) { cudaEventDestroy(g->ev_done[i]); cudaEventDestroy(g->ev_copied[i]); }
        cudaStreamDestroy(g->copy_stream);
    }
    for (void *b : bufs)
        if (b) cudaFree(b);
    if (g->h_scal) { cudaFreeHost(g->h_scal); cudaEventDestroy(g->ev_scal); }
    delete g;
    return HIREP_OK;
}

extern "C" int hirep_geom_set_bc(hirep_geom *g, const int sign[4]) {
    if (!g || !sign) return fail(HIREP_EINVAL, "hirep_geom_set_bc: NULL argument");
    for (int mu = 0; mu < 4; ++mu)
        if (sign[mu] != 1 && sign[mu] != -1) return fail(HIREP_EINVAL, "hirep_geom_set_bc: sign[%d]=%d is not +-1", mu, sign[mu]);
    for (int mu = 0; mu < 4; ++mu) g->geo.bc[mu] = sign[mu];
    g->host_links_ready = 0;
    return HIREP_OK;
}

extern "C" int hirep_geom_set_stream(hirep_geom *g, void *cuda_stream) {
    if (!g) return fail(HIREP_EINVAL, "hirep_geom_set_stream: NULL geometry");
    g->stream = (cudaStream_t)cuda_stream;
    return HIREP_OK;
}

extern "C" int hirep_geom_sizes(const hirep_geom *g, size_t *spinor_full, size_t *spinor_half, size_t *links_fund,
                                size_t *links_rep, int *d_R, int *rep_is_real) {
    if (!g) return fail(HIREP_EINVAL, "hirep_geom_sizes: NULL geometry");
    if (spinor_full) *spinor_full = 2 * g->bytes_spinor_half;
    if (spinor_half) *spinor_half = g->bytes_spinor_half;
    if (links_fund) *links_fund = g->bytes_links_fund;
    if (links_rep) *links_rep = g->bytes_links_rep;
    if (d_R) *d_R = g->dR;
    if (rep_is_real) *rep_is_real = g->real;
    return HIREP_OK;
}

extern "C" int hirep_set_link_mode(hirep_geom *g, int mode) {
    if (!g) return fail(HIREP_EINVAL, "hirep_set_link_mode: NULL geometry");
    if (mode != HIREP_LINKS_STORED && mode != HIREP_LINKS_REBUILD) return fail(HIREP_EINVAL, "hirep_set_link_mode: unknown mode %d", mode);
    g->mode = mode;
    return HIREP_OK;
}
extern "C" int hirep_set_kernel_variant(hirep_geom *g, int variant) {
    if (!g) return fail(HIREP_EINVAL, "hirep_set_kernel_variant: NULL geometry");
    if (variant < 0) return fail(HIREP_EINVAL, "hirep_set_kernel_variant: negative variant");
    g->variant = variant;
    return HIREP_OK;
}
extern "C" int hirep_set_tuning(hirep_geom *g, int key, int value) {
    if (!g) return fail(HIREP_EINVAL, "hirep_set_tuning: NULL geometry");
    switch (key) {
    case HIREP_TUNE_SUM_ALGORITHM:
        if (value < 2 || value > 4) return fail(HIREP_EINVAL, "hirep_set_tuning: summation algorithm %d (2, 3 or 4)", value);
        g->sum_alg = value;
        return HIREP_OK;
    case HIREP_TUNE_MAX_CTAS:
        if (value < 0) return fail(HIREP_EINVAL, "hirep_set_tuning: max CTAs %d", value);
        g->tune_max_ctas = value;
        return HIREP_OK;
    case HIREP_TUNE_PACE_WINDOW:
        if (value < 0 || value > 64) return fail(HIREP_EINVAL, "hirep_set_tuning: pace window %d (0 = off, 1..64 rounds)", value);
        g->tune_pace = value;
        return HIREP_OK;
    case HIREP_TUNE_FUSE_DIAG:
        if (value != 0 && value != 1) return fail(HIREP_EINVAL, "hirep_set_tuning: fuse-diagonal switch %d (0 or 1)", value);
        g->tune_fuse_diag = value;
        return HIREP_OK;
    }
    return fail(HIREP_EINVAL, "hirep_set_tuning: unknown key %d", key);
}
extern "C" long hirep_launch_count(const hirep_geom *g) { return g ? g->launches : 0; }

// a geometry belongs to the device that was current when it was created (its workspaces live there)
static bool wrong_device(const hirep_geom *g) {
    int dev = -1;
    if (g->device < 0 || cudaGetDevice(&dev) != cudaSuccess) return false;   // no device: the launch itself reports HIREP_ECUDA
    return dev != g->device;
}
#define CHECK_PTRS(name, ...)                                                                                      \
    do {                                                                                                           \
        if (!g) return fail(HIREP_EINVAL, name ": NULL geometry");                                                 \
        if (wrong_device(g)) return fail(HIREP_EINVAL, name ": the geometry was created on CUDA device %d, which is not the current device", g->device); \
        const void *ptrs_[] = {__VA_ARGS__};                                                                       \
        for (const void *p_ : ptrs_) {                                                                             \
            if (!p_) return fail(HIREP_EINVAL, name ": NULL pointer argument");                                    \
            if (misaligned(p_)) return fail(HIREP_EINVAL, name ": pointer %p is not 16-byte aligned", p_);         \
        }                                                                                                          \
    } while (0)

extern "C" int hirep_spinor_import(hirep_geom *g, void *native, const void *canonical, int which) {
    CHECK_PTRS("hirep_spinor_import", native, canonical);
    if (which < 0 || which > 2) return fail(HIREP_EINVAL, "hirep_spinor_import: parity_or_full=%d", which);
    return kern_result(g, k_spinor_import(g->geo, g->prec, g->dR, native, canonical, which, g->stream), "hirep_spinor_import",
                       1 + (g->geo.Nh % TILE ? 1 : 0));
}
extern "C" int hirep_spinor_export(hirep_geom *g, void *canonical, const void *native, int which) {
    CHECK_PTRS("hirep_spinor_export", native, canonical);
    if (which < 0 || which > 2) return fail(HIREP_EINVAL, "hirep_spinor_export: parity_or_full=%d", which);
    return kern_result(g, k_spinor_export(g->geo, g->prec, g->dR, canonical, native, which, g->stream), "hirep_spinor_export");
}
extern "C" int hirep_links_import(hirep_geom *g, void *native_fund, const void *canonical_fund) {
    CHECK_PTRS("hirep_links_import", native_fund, canonical_fund);
    return kern_result(g, k_links_import(g->geo, g->prec, g->N, native_fund, canonical_fund, g->stream), "hirep_links_import");
}
extern "C" int hirep_links_rep_export(hirep_geom *g, void *canonical_rep, const void *native_rep) {
    CHECK_PTRS("hirep_links_rep_export", native_rep, canonical_rep);
    return kern_result(g, k_links_rep_export(g->geo, g->prec, g->dR, g->real, canonical_rep, native_rep, 0, g->stream), "hirep_links_rep_export");
}
extern "C" int hirep_links_rep_export_bwd(hirep_geom *g, void *canonical_rep, const void *native_rep) {
    CHECK_PTRS("hirep_links_rep_export_bwd", native_rep, canonical_rep);
    return kern_result(g, k_links_rep_export(g->geo, g->prec, g->dR, g->real, canonical_rep, native_rep, 1, g->stream), "hirep_links_rep_export_bwd");
}
extern "C" int hirep_links_to_rep(hirep_geom *g, void *native_rep, const void *native_fund) {
    CHECK_PTRS("hirep_links_to_rep", native_rep, native_fund);
    if (native_rep == native_fund) return fail(HIREP_EINVAL, "hirep_links_to_rep: output aliases input");
    return kern_result(g, k_links_to_rep(g->geo, g->prec, g->N, g->rep, native_rep, native_fund, g->stream), "hirep_links_to_rep");
}

// ---- operators ------------------------------------------------------------------------------------
static int workspace(void **slot, size_t bytes);
static int hop_range(hirep_geom *g, HopLaunch L, int tb, int te, const char *what) {
    L.tile_begin = tb; L.tile_end = te;
    const int rc = g->prec == HIREP_F64 ? k_hop_f64(g->geo, g->N, g->rep, g->mode, g->variant, L, g->stream)
                                        : k_hop_f32(g->geo, g->N, g->rep, g->mode, g->variant, L, g->stream);
    return kern_result(g, rc, what);
}
// Regions of a slab in tiles of each parity (slice t = half indices [t S, (t+1) S), S = L^3/2; local slices 0 and T-1 are ghosts):
//   OWNED    = slices 1 .. T-2;  INTERIOR = the tiles that lie entirely in slices 2 .. T-3 (no hop reaches a ghost slice);
//   BOUNDARY = the rest of OWNED, i.e. the tiles touching slice 1 and those touching slice T-2 (two launches, one if they meet).
// Tiles that straddle a slice boundary also compute a few sites of the neighbouring slice (ghost outputs are scratch).
static int hop(hirep_geom *g, HopLaunch L, const char *what) {
    L.max_ctas = g->tune_max_ctas;
    static const int dbg = getenv("HIREP_DBG") ? atoi(getenv("HIREP_DBG")) : 0;
    L.dbg = dbg;
    if (g->tune_pace > 0 && L.nsets == 2) {   // hirep_set_tuning(HIREP_TUNE_PACE_WINDOW): round pacing of the tile-pair kernel
        int rc0 = workspace((void **)&g->dev_flags, 64);
        if (rc0) return rc0;
        L.pace = (unsigned *)g->dev_flags + 4;
        L.pace_every = g->tune_pace;
        const cudaError_t pe = cudaMemsetAsync(L.pace, 0, sizeof(unsigned), g->stream);
        if (pe != cudaSuccess) return cuda_fail(pe, what);
    }
    if (!g->slab || g->region == HIREP_REGION_ALL) return hop_range(g, L, 0, 0, what);
    const long S = (long)g->geo.L * g->geo.L * g->geo.Lh;
    const int T = g->geo.T;
    const int own_b = (int)(S / TILE), own_e = (int)(((T - 1) * S + TILE - 1) / TILE);
    int int_b = (int)((2 * S + TILE - 1) / TILE), int_e = (int)(((T - 2) * S) / TILE);
    if (int_e < int_b) int_e = int_b = (own_b + own_e) / 2 > own_b ? (own_b + own_e) / 2 : own_b;   // no interior: split point only
    if (int_b < own_b) int_b = own_b;
    if (int_e > own_e) int_e = own_e;
    if (g->region == HIREP_REGION_OWNED) return hop_range(g, L, own_b, own_e, what);
    if (g->region == HIREP_REGION_INTERIOR) return int_e > int_b ? hop_range(g, L, int_b, int_e, what) : HIREP_OK;
    int rc = int_b > own_b ? hop_range(g, L, own_b, int_b, what) : HIREP_OK;
    if (rc) return rc;
    return own_e > int_e ? hop_range(g, L, int_e, own_e, what) : HIREP_OK;
}
extern "C" int hirep_halo_pack(hirep_geom *g, int face, void *buf, const void *spinor_half) {
    CHECK_PTRS("hirep_halo_pack", buf, spinor_half);
    if (!g->slab) return fail(HIREP_EINVAL, "hirep_halo_pack: not a slab geometry");
    if (face != 0 && face != 1) return fail(HIREP_EINVAL, "hirep_halo_pack: face=%d (0 first owned slice, 1 last owned slice)", face);
    return kern_result(g, k_halo_pack(g->geo, g->prec, g->dR, 0, face, buf, spinor_half, g->stream), "hirep_halo_pack");
}
extern "C" int hirep_halo_unpack(hirep_geom *g, int face, void *spinor_half, const void *buf) {
    CHECK_PTRS("hirep_halo_unpack", spinor_half, buf);
    if (!g->slab) return fail(HIREP_EINVAL, "hirep_halo_unpack: not a slab geometry");
    if (face != 0 && face != 1) return fail(HIREP_EINVAL, "hirep_halo_unpack: face=%d", face);
    return kern_result(g, k_halo_unpack(g->geo, g->prec, g->dR, 0, face, spinor_half, buf, g->stream), "hirep_halo_unpack");
}
static const char *links_parity(const hirep_geom *g, const void *links, int p) {
    const size_t total = g->mode == HIREP_LINKS_STORED ? g->bytes_links_rep : g->bytes_links_fund;
    return (const char *)links + (size_t)p * (total / 2);
}
static int workspace(void **slot, size_t bytes) {
    if (*slot) return HIREP_OK;
    cudaError_t e = cudaMalloc(slot, bytes);
    if (e != cudaSuccess) { *slot = nullptr; cudaGetLastError(); return fail(HIREP_ENOMEM, "workspace allocation of %zu bytes failed: %s", bytes, cudaGetErrorString(e)); }
    // once, at allocation: padding lanes of the library's own work fields hold zeros, never stale memory (they are excluded from every
    // reduction, but kernels that copy whole tiles would otherwise carry garbage into the caller's padding)
    e = cudaMemset(*slot, 0, bytes);
    if (e != cudaSuccess) return cuda_fail(e, "workspace initialisation");
    return HIREP_OK;
}

// Allocate (and zero) now what the operator / solver entry points would otherwise allocate on their first call, so that a first call
// may already sit inside a CUDA-graph capture or any region where cudaMalloc is not allowed (lazy allocation).
extern "C" int hirep_geom_reserve(hirep_geom *g, int what) {
    if (!g) return fail(HIREP_EINVAL, "hirep_geom_reserve: NULL geometry");
    if (wrong_device(g)) return fail(HIREP_EINVAL, "hirep_geom_reserve: the geometry was created on CUDA device %d, which is not the current device", g->device);
    if (what <= 0 || (what & ~(HIREP_RESERVE_OPERATORS | HIREP_RESERVE_SOLVERS))) return fail(HIREP_EINVAL, "hirep_geom_reserve: flags %d", what);
    int rc = HIREP_OK;
    const size_t hb = g->bytes_spinor_half;
    if (what & HIREP_RESERVE_OPERATORS) {
        if ((rc = workspace(&g->ws_half, hb)) || (rc = workspace(&g->ws_half2, hb)) || (rc = workspace(&g->ws_half3, hb)) ||
            (rc = workspace(&g->ws_full, 2 * hb)) || (rc = workspace((void **)&g->dev_flags, 64)))
            return rc;
    }
    if (what & HIREP_RESERVE_SOLVERS) {
        if ((rc = workspace(&g->ws_red, (size_t)k_reduce_workspace_bytes() + 64)) || (rc = workspace(&g->ws_red2, (size_t)k_reduce_workspace_bytes())) ||
            (rc = workspace(&g->cg_r, 2 * hb)) || (rc = workspace(&g->cg_p, 2 * hb)) || (rc = workspace(&g->cg_Ap, 2 * hb)) ||
            (rc = workspace(&g->bi_s, 2 * hb)) || (rc = workspace(&g->bi_t, 2 * hb)))
            return rc;
        if (!g->h_scal) {
            cudaError_t e = cudaHostAlloc((void **)&g->h_scal, 8 * sizeof(double), cudaHostAllocDefault);
            if (e != cudaSuccess) { g->h_scal = nullptr; return cuda_fail(e, "hirep_geom_reserve"); }
            if ((e = cudaEventCreateWithFlags(&g->ev_scal, cudaEventDisableTiming)) != cudaSuccess) {
                cudaFreeHost(g->h_scal); g->h_scal = nullptr;
                return cuda_fail(e, "hirep_geom_reserve");
            }
        }
    }
    return HIREP_OK;
}

static int offdiag(hirep_geom *g, void *out, const void *in, const void *links, int p_out, const char *what) {
    HopLaunch L{};
    L.nsets = 1;
    L.set[0] = HopSet{in, out, nullptr, links_parity(g, links, p_out), p_out};
    L.a = 0.0; L.b = -0.5; L.g5 = 0;
    return hop(g, L, what);
}

extern "C" int hirep_Dphi_eo(hirep_geom *g, void *out_even, const void *in_odd, const void *links) {
    CHECK_PTRS("hirep_Dphi_eo", out_even, in_odd, links);
    if (out_even == in_odd) return fail(HIREP_EINVAL, "hirep_Dphi_eo: out aliases in");
    return offdiag(g, out_even, in_odd, links, 0, "hirep_Dphi_eo");
}
extern "C" int hirep_Dphi_oe(hirep_geom *g, void *out_odd, const void *in_even, const void *links) {
    CHECK_PTRS("hirep_Dphi_oe", out_odd, in_even, links);
    if (out_odd == in_even) return fail(HIREP_EINVAL, "hirep_Dphi_oe: out aliases in");
    return offdiag(g, out_odd, in_even, links, 1, "hirep_Dphi_oe");
}

struct FusedRed { int mode; void *r; const double *num, *den; };
static int dphi_full(hirep_geom *g, double m0, void *out, const void *in, const void *links, int g5, const char *what, double am = 0.0,
                     const FusedRed *red = nullptr) {
    const size_t hb = g->bytes_spinor_half;
    const char *in_e = (const char *)in, *in_o = in_e + hb;
    char *out_e = (char *)out, *out_o = out_e + hb;
    HopLaunch L{};
    L.nsets = 2;
    L.set[0] = HopSet{in_o, out_e, in_e, links_parity(g, links, 0), 0};
    L.set[1] = HopSet{in_e, out_o, in_o, links_parity(g, links, 1), 1};
    L.a = 4.0 + m0; L.b = -0.5; L.g5 = g5; L.am = am;
    if (red) {
        L.red_mode = red->mode; L.red_alg = g->sum_alg; L.red_partial = g->ws_red2;
        L.red_r = red->r; L.red_num = red->num; L.red_den = red->den;
    }
    return hop(g, L, what);
}
// does a default full-lattice launch of this geometry run the tile-pair kernel, whose epilogue can carry the CG's reductions?
static bool fused_cg_ok(const hirep_geom *g) {
    if (g->mode != HIREP_LINKS_STORED || g->variant != 0 || g->slab || g->tune_max_ctas < 0) return false;
    const bool f64 = g->prec == HIREP_F64;
    return (g->dR <= 3 && (f64 || !g->real)) || (!f64 && !g->real && g->dR != 5 && g->dR <= 6);
}

extern "C" int hirep_Dphi(hirep_geom *g, double m0, void *out_full, const void *in_full, const void *links) {
    CHECK_PTRS("hirep_Dphi", out_full, in_full, links);
    if (out_full == in_full) return fail(HIREP_EINVAL, "hirep_Dphi: out aliases in");
    return dphi_full(g, m0, out_full, in_full, links, 0, "hirep_Dphi");
}

// out_even = [gamma_5] ((4+m)^2 in_even - D_eo D_oe in_even): two half-lattice passes through the odd workspace
// `red` (CG only): the reduction fused into the epilogue of the SECOND pass, which writes the result (FusedRed, above)
static int dphi_hat(hirep_geom *g, double m0, void *out_even, const void *in_even, const void *links, int g5, const char *what,
                    const FusedRed *red = nullptr) {
    if (g->slab) return fail(HIREP_EUNSUPPORTED, "%s: on a slab compose the two passes yourself (Dphi_oe, halo exchange, Dphi_eo)", what);
    int rc = workspace(&g->ws_half, g->bytes_spinor_half);
    if (rc) return rc;
    rc = offdiag(g, g->ws_half, in_even, links, 1, what);
    if (rc) return rc;
    HopLaunch L{};
    L.nsets = 1;
    L.set[0] = HopSet{g->ws_half, out_even, in_even, links_parity(g, links, 0), 0};
    L.a = (4.0 + m0) * (4.0 + m0);
    L.b = +0.5;   // - D_eo = -(-1/2) hop
    L.g5 = g5;
    if (red) {
        L.red_mode = red->mode; L.red_alg = g->sum_alg; L.red_partial = g->ws_red2;
        L.red_r = red->r; L.red_num = red->num; L.red_den = red->den;
    }
    return hop(g, L, what);
}
// does a default half-lattice launch of this geometry run the ring / pair kernels, whose epilogues can carry the CG's reductions?
static bool fused_cg_eo_ok(const hirep_geom *g) {
    return g->mode == HIREP_LINKS_STORED && g->variant == 0 && !g->slab && g->tune_max_ctas >= 0 && g->dR <= 6;
}

extern "C" int hirep_Dphi_hat(hirep_geom *g, double m0, void *out_even, const void *in_even, const void *links) {
    CHECK_PTRS("hirep_Dphi_hat", out_even, in_even, links);
    if (out_even == in_even) return fail(HIREP_EINVAL, "hirep_Dphi_hat: out aliases in");
    return dphi_hat(g, m0, out_even, in_even, links, 0, "hirep_Dphi_hat");
}

// ---- hirep_Dphi_hat_static: Dphi_hat for callers that cannot call cudaMalloc (CUDA graph capture, serving loops) ----------
// The odd intermediate field D_oe in_e of Eq 44 (L808) lives in a file-scope device array instead of the handle's lazily
// allocated workspace.  Every GPU that loads the library holds HIREP_STATIC_SCRATCH_BYTES until exit.  In host code the array's
// name is only a stand-in for the symbol: the device address is resolved once per device with cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_static_scratch[HIREP_STATIC_SCRATCH_BYTES];
static void *g_static_scratch_addr[64];   // per CUDA device ordinal
static std::mutex g_static_scratch_mu;
static int static_scratch(const hirep_geom *g, void **ptr, const char *what) {
    int dev = g->device;
    cudaError_t e = dev >= 0 ? cudaSuccess : cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, what);
    if (dev < 0 || dev >= 64) return fail(HIREP_EUNSUPPORTED, "%s: CUDA device ordinal %d outside the table of 64", what, dev);
    std::lock_guard<std::mutex> lk(g_static_scratch_mu);
    if (!g_static_scratch_addr[dev]) {   // the geometry's device is the current one (CHECK_PTRS): the address is that device's copy
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) return cuda_fail(e, "hirep_Dphi_hat_static: cudaGetSymbolAddress");
        g_static_scratch_addr[dev] = p;
    }
    *ptr = g_static_scratch_addr[dev];
    return HIREP_OK;
}
extern "C" int hirep_Dphi_hat_static(hirep_geom *g, double m0, void *out_even, const void *in_even, const void *links) {
    const char *what = "hirep_Dphi_hat_static";
    CHECK_PTRS("hirep_Dphi_hat_static", out_even, in_even, links);
    if (out_even == in_even) return fail(HIREP_EINVAL, "%s: out aliases in", what);
    if (g->slab) return fail(HIREP_EUNSUPPORTED, "%s: on a slab compose the two passes yourself (Dphi_oe, halo exchange, Dphi_eo)", what);
    if (g->bytes_spinor_half > (size_t)HIREP_STATIC_SCRATCH_BYTES)
        return fail(HIREP_EINVAL, "%s: one half-lattice spinor of this geometry is %zu bytes, the static scratch holds %zu (HIREP_STATIC_SCRATCH_BYTES); use hirep_Dphi_hat",
                    what, g->bytes_spinor_half, (size_t)HIREP_STATIC_SCRATCH_BYTES);
    void *tmp = nullptr;
    int rc = static_scratch(g, &tmp, what);
    if (rc) return rc;
    // The array keeps the previous call's contents, possibly of another geometry.  Every site lane is overwritten by the first pass; the
    // padding lanes of a ragged last tile are not, and the handle's own workspace holds zeros there: clear that tile.
    if (g->geo.Nh % TILE) {
        const size_t tile_bytes = g->bytes_spinor_half / (size_t)g->geo.n_tiles;
        const cudaError_t e = cudaMemsetAsync((char *)tmp + (size_t)(g->geo.n_tiles - 1) * tile_bytes, 0, tile_bytes, g->stream);
        if (e != cudaSuccess) return cuda_fail(e, what);
    }
    rc = offdiag(g, tmp, in_even, links, 1, what);
    if (rc) return rc;
    HopLaunch L{};
    L.nsets = 1;
    L.set[0] = HopSet{tmp, out_even, in_even, links_parity(g, links, 0), 0};
    L.a = (4.0 + m0) * (4.0 + m0);
    L.b = +0.5;
    L.g5 = 0;
    return hop(g, L, what);
}

extern "C" int hirep_g5Dphi_hat(hirep_geom *g, double m0, void *out_even, const void *in_even, const void *links) {
    CHECK_PTRS("hirep_g5Dphi_hat", out_even, in_even, links);
    if (out_even == in_even) return fail(HIREP_EINVAL, "hirep_g5Dphi_hat: out aliases in");
    return dphi_hat(g, m0, out_even, in_even, links, 1, "hirep_g5Dphi_hat");
}

extern "C" int hirep_g5Dphi_hat_sq(hirep_geom *g, double m0, void *out_even, const void *in_even, const void *links) {
    CHECK_PTRS("hirep_g5Dphi_hat_sq", out_even, in_even, links);
    if (out_even == in_even) return fail(HIREP_EINVAL, "hirep_g5Dphi_hat_sq: out aliases in");
    int rc = workspace(&g->ws_half2, g->bytes_spinor_half);
    if (rc) return rc;
    rc = dphi_hat(g, m0, g->ws_half2, in_even, links, 1, "hirep_g5Dphi_hat_sq (first Q_hat)");
    if (rc) return rc;
    return dphi_hat(g, m0, out_even, g->ws_half2, links, 1, "hirep_g5Dphi_hat_sq (second Q_hat)");
}

extern "C" int hirep_g5Dphi_sq(hirep_geom *g, double m0, void *out_full, const void *in_full, const void *links) {
    CHECK_PTRS("hirep_g5Dphi_sq", out_full, in_full, links);
    if (out_full == in_full) return fail(HIREP_EINVAL, "hirep_g5Dphi_sq: out aliases in");
    if (g->slab) return fail(HIREP_EUNSUPPORTED, "hirep_g5Dphi_sq: on a slab compose the two applications yourself with a halo exchange in between");
    int rc = workspace(&g->ws_full, 2 * g->bytes_spinor_half);
    if (rc) return rc;
    rc = dphi_full(g, m0, g->ws_full, in_full, links, 1, "hirep_g5Dphi_sq (first g5 D)");
    if (rc) return rc;
    return dphi_full(g, m0, out_full, g->ws_full, links, 1, "hirep_g5Dphi_sq (second g5 D)");
}

// ---- twisted mass (Eq 51) and its Schur form (Eq 43): SURVEY.md 8(f) NEXT-2, first part --------
extern "C" int hirep_spinor_g5_lc(hirep_geom *g, int which, void *xi, const double c1[2], const double c2[2], const void *eta) {
    CHECK_PTRS("hirep_spinor_g5_lc", xi, eta);
    if (!c1 || !c2) return fail(HIREP_EINVAL, "hirep_spinor_g5_lc: NULL coefficient");
    if (which < 0 || which > 2) return fail(HIREP_EINVAL, "hirep_spinor_g5_lc: parity_or_full=%d", which);
    const long n = (long)g->geo.n_tiles * 4 * g->dR * TILE * (which == HIREP_FULL ? 2 : 1);
    static const double zero2[2] = {0.0, 0.0};
    return kern_result(g, k_g5_lincomb(g->prec, n, g->dR, xi, zero2, 0, c1, c2, eta, g->stream), "hirep_spinor_g5_lc");
}
extern "C" int hirep_spinor_gamma(hirep_geom *g, int which, int mu, void *xi, const void *eta) {
    CHECK_PTRS("hirep_spinor_gamma", xi, eta);
    if (which < 0 || which > 2) return fail(HIREP_EINVAL, "hirep_spinor_gamma: parity_or_full=%d", which);
    if (!((mu >= 0 && mu <= 3) || mu == 5)) return fail(HIREP_EINVAL, "hirep_spinor_gamma: mu=%d (0..3 or 5)", mu);
    if (xi == eta) return fail(HIREP_EINVAL, "hirep_spinor_gamma: xi aliases eta");
    return kern_result(g, k_gamma(g->geo, g->prec, g->dR, which == HIREP_FULL ? 2 : 1, mu, xi, eta, g->stream), "hirep_spinor_gamma");
}
extern "C" int hirep_spinor_g5_lc_add_assign(hirep_geom *g, int which, void *xi, const double c0[2], const double c1[2], const double c2[2],
                                             const void *eta) {
    CHECK_PTRS("hirep_spinor_g5_lc_add_assign", xi, eta);
    if (!c0 || !c1 || !c2) return fail(HIREP_EINVAL, "hirep_spinor_g5_lc_add_assign: NULL coefficient");
    if (which < 0 || which > 2) return fail(HIREP_EINVAL, "hirep_spinor_g5_lc_add_assign: parity_or_full=%d", which);
    const long n = (long)g->geo.n_tiles * 4 * g->dR * TILE * (which == HIREP_FULL ? 2 : 1);
    return kern_result(g, k_g5_lincomb(g->prec, n, g->dR, xi, c0, 1, c1, c2, eta, g->stream), "hirep_spinor_g5_lc_add_assign");
}

extern "C" int hirep_Dphi_tm(hirep_geom *g, double m0, double mu, void *out_full, const void *in_full, const void *links) {
    CHECK_PTRS("hirep_Dphi_tm", out_full, in_full, links);
    if (out_full == in_full) return fail(HIREP_EINVAL, "hirep_Dphi_tm: out aliases in");
    return dphi_full(g, m0, out_full, in_full, links, 0, "hirep_Dphi_tm", mu);
}

// (D^tm)^dagger D^tm = gamma_5 D^tm(-mu) gamma_5 D^tm(mu): two full-lattice launches with the gamma_5 fused in the store
extern "C" int hirep_Dphi_tm_sq(hirep_geom *g, double m0, double mu, void *out_full, const void *in_full, const void *links) {
    CHECK_PTRS("hirep_Dphi_tm_sq", out_full, in_full, links);
    if (out_full == in_full) return fail(HIREP_EINVAL, "hirep_Dphi_tm_sq: out aliases in");
    int rc = workspace(&g->ws_full, 2 * g->bytes_spinor_half);
    if (rc) return rc;
    rc = dphi_full(g, m0, g->ws_full, in_full, links, 1, "hirep_Dphi_tm_sq (gamma_5 D^tm(mu))", mu);
    if (rc) return rc;
    return dphi_full(g, m0, out_full, g->ws_full, links, 1, "hirep_Dphi_tm_sq (gamma_5 D^tm(-mu))", -mu);
}

// Eq 43 with D_ee = D_oo = (4+m) + i mu gamma_5:  out_e = D_ee in_e - D_eo D_oo^{-1} D_oe in_e.
// Three launches: D_oe pass; D_oo^{-1} = ((4+m) - i mu gamma_5)/((4+m)^2 + mu^2) as a gamma_5 linear combination in
// place; D_eo pass with the diagonal term (a + i mu gamma_5) in_e fused in the epilogue.
extern "C" int hirep_Dphi_tm_hat(hirep_geom *g, double m0, double mu, void *out_even, const void *in_even, const void *links) {
    CHECK_PTRS("hirep_Dphi_tm_hat", out_even, in_even, links);
    if (out_even == in_even) return fail(HIREP_EINVAL, "hirep_Dphi_tm_hat: out aliases in");
    int rc = workspace(&g->ws_half, g->bytes_spinor_half);
    if (rc) return rc;
    const double a = 4.0 + m0, den = a * a + mu * mu;
    // D_oo^-1 = (a - i mu gamma_5)/(a^2 + mu^2) multiplies the hop sum of the D_oe pass: in the epilogue of that pass (kernel variants 0, 3, 4:
    // the persistent kernels), else as a separate gamma_5 linear combination
    if (g->variant == 0 || g->variant == 3 || g->variant == 4) {
        HopLaunch L1{};
        L1.nsets = 1;
        L1.set[0] = HopSet{in_even, g->ws_half, nullptr, links_parity(g, links, 1), 1};
        L1.a = 0.0; L1.b = -0.5 * a / den; L1.bi = 0.5 * mu / den;
        if ((rc = hop(g, L1, "hirep_Dphi_tm_hat (D_oo^-1 D_oe pass)"))) return rc;
    } else {
        if ((rc = offdiag(g, g->ws_half, in_even, links, 1, "hirep_Dphi_tm_hat (D_oe pass)"))) return rc;
        const double c1[2] = {a / den, 0.0}, c2[2] = {0.0, -mu / den};
        if ((rc = hirep_spinor_g5_lc(g, HIREP_ODD, g->ws_half, c1, c2, g->ws_half))) return rc;
    }
    HopLaunch L{};
    L.nsets = 1;
    L.set[0] = HopSet{g->ws_half, out_even, in_even, links_parity(g, links, 0), 0};
    L.a = a;
    L.am = mu;
    L.b = +0.5;   // - D_eo = -(-1/2) hop
    L.g5 = 0;
    return hop(g, L, "hirep_Dphi_tm_hat (D_eo pass)");
}

// ---- clover term (Eq 47-49): SURVEY.md 8(f) NEXT-2, second part ----------------------------------------
static size_t clover_bytes(const hirep_geom *g) {
    return (size_t)2 * g->geo.n_tiles * 4 * g->dR * g->dR * TILE * 2 * (g->prec == HIREP_F64 ? 8 : 4);
}
extern "C" int hirep_clover_bytes(const hirep_geom *g, size_t *bytes) {
    if (!g || !bytes) return fail(HIREP_EINVAL, "hirep_clover_bytes: NULL argument");
    *bytes = clover_bytes(g);
    return HIREP_OK;
}
extern "C" int hirep_clover_field(hirep_geom *g, void *clover, const void *links_rep) {
    CHECK_PTRS("hirep_clover_field", clover, links_rep);
    if (g->mode != HIREP_LINKS_STORED) return fail(HIREP_EINVAL, "hirep_clover_field: needs the stored represented links (HIREP_LINKS_STORED)");
    return kern_result(g, k_clover_field(g->geo, g->prec, g->dR, g->real, clover, links_rep, g->stream), "hirep_clover_field");
}
extern "C" int hirep_clover_export(hirep_geom *g, void *canonical_out, const void *clover) {
    CHECK_PTRS("hirep_clover_export", canonical_out, clover);
    return kern_result(g, k_clover_export(g->geo, g->prec, g->dR, canonical_out, clover, g->stream), "hirep_clover_export");
}
extern "C" int hirep_Cphi(hirep_geom *g, double m0, double csw, void *out_full, const void *in_full, const void *clover) {
    CHECK_PTRS("hirep_Cphi", out_full, in_full, clover);
    if (out_full == in_full) return fail(HIREP_EINVAL, "hirep_Cphi: out aliases in");
    return kern_result(g, k_cphi(g->prec, g->dR, 2 * g->geo.n_tiles, 4.0 + m0, csw, clover, in_full, out_full, g->stream), "hirep_Cphi");
}
// Are the site-diagonal matrices applied inside the stencil epilogue (one launch per stencil pass, "fused into the second pass",
// SURVEY 8(f) row 2) or by separate block-apply launches?  Fused where the thread-per-site ring kernel is instantiated
// (k_hop_diag_supported) unless hirep_set_tuning(HIREP_TUNE_FUSE_DIAG, 0); slab geometries keep the composed form.
static bool fuse_diag(const hirep_geom *g) {
    return g->tune_fuse_diag && !g->slab && k_hop_diag_supported(g->prec == HIREP_F64 ? 0 : 1, g->dR, g->real, g->mode, g->variant);
}
// one stencil pass over parity p_out with the diagonal matrices `diag` of that parity in its epilogue (kernels.h DIAG_*)
static void set_red(hirep_geom *g, HopLaunch &L, const FusedRed *red) {   // the CG's reduction in this launch's epilogue (FusedRed)
    if (!red) return;
    L.red_mode = red->mode; L.red_alg = g->sum_alg; L.red_partial = g->ws_red2;
    L.red_r = red->r; L.red_num = red->num; L.red_den = red->den;
}
static int hop_diag_half(hirep_geom *g, int diag_mode, double a, double csw, double b, int g5, void *out, const void *in, const void *self,
                         const void *links, const void *diag, int p_out, const char *what, const FusedRed *red = nullptr) {
    HopLaunch L{};
    L.nsets = 1;
    L.set[0] = HopSet{in, out, self, links_parity(g, links, p_out), p_out, diag};
    L.a = a; L.b = b; L.g5 = g5; L.diag_mode = diag_mode; L.diag_csw = csw;
    set_red(g, L, red);
    return hop(g, L, what);
}
// the same over both parities in one launch: out = [gamma_5] (Diag in + b hop(in)); diag_full = both parities, even first
static int hop_diag_full(hirep_geom *g, int diag_mode, double a, double csw, int g5, void *out_full, const void *in_full, const void *links,
                         const void *diag_full, size_t diag_parity_bytes, const char *what, const FusedRed *red = nullptr) {
    const size_t hb = g->bytes_spinor_half;
    const char *in_e = (const char *)in_full, *in_o = in_e + hb;
    char *out_e = (char *)out_full, *out_o = out_e + hb;
    HopLaunch L{};
    L.nsets = 2;
    L.set[0] = HopSet{in_o, out_e, in_e, links_parity(g, links, 0), 0, diag_full};
    L.set[1] = HopSet{in_e, out_o, in_o, links_parity(g, links, 1), 1, (const char *)diag_full + diag_parity_bytes};
    L.a = a; L.b = -0.5; L.g5 = g5; L.diag_mode = diag_mode; L.diag_csw = csw;
    set_red(g, L, red);
    return hop(g, L, what);
}
// out = [gamma_5] (Cphi in - 1/2 hop(in)).  Fused: one stencil launch whose epilogue applies (4+m) + c_sw A to the site's own
// input.  Composed: Cphi writes out, the hopping pass accumulates onto it in place (every site's own
// value is read before it is written, by the same tile); gamma_5 commutes with the diagonal blocks
static int dphi_clover(hirep_geom *g, double m0, double csw, void *out_full, const void *in_full, const void *links, const void *clover, int g5,
                       const char *what, const FusedRed *red = nullptr) {
    if (fuse_diag(g)) return hop_diag_full(g, DIAG_HB, 4.0 + m0, csw, g5, out_full, in_full, links, clover, clover_bytes(g) / 2, what, red);
    if (red) return fail(HIREP_EINVAL, "%s: fused reductions need the fused epilogue", what);
    int rc = kern_result(g, k_cphi(g->prec, g->dR, 2 * g->geo.n_tiles, 4.0 + m0, csw, clover, in_full, out_full, g->stream), what);
    if (rc) return rc;
    const size_t hb = g->bytes_spinor_half;
    const char *in_e = (const char *)in_full, *in_o = in_e + hb;
    char *out_e = (char *)out_full, *out_o = out_e + hb;
    HopLaunch L{};
    L.nsets = 2;
    L.set[0] = HopSet{in_o, out_e, out_e, links_parity(g, links, 0), 0};
    L.set[1] = HopSet{in_e, out_o, out_o, links_parity(g, links, 1), 1};
    L.a = 1.0; L.b = -0.5; L.g5 = g5; L.am = 0.0;
    return hop(g, L, what);
}
extern "C" int hirep_Dphi_clover(hirep_geom *g, double m0, double csw, void *out_full, const void *in_full, const void *links, const void *clover) {
    CHECK_PTRS("hirep_Dphi_clover", out_full, in_full, links, clover);
    if (out_full == in_full) return fail(HIREP_EINVAL, "hirep_Dphi_clover: out aliases in");
    return dphi_clover(g, m0, csw, out_full, in_full, links, clover, 0, "hirep_Dphi_clover");
}
// (gamma_5 D_clover)^2, Hermitian positive definite: the operator of the CG with the clover term (L772)
extern "C" int hirep_g5Dphi_clover_sq(hirep_geom *g, double m0, double csw, void *out_full, const void *in_full, const void *links,
                                      const void *clover) {
    CHECK_PTRS("hirep_g5Dphi_clover_sq", out_full, in_full, links, clover);
    if (out_full == in_full) return fail(HIREP_EINVAL, "hirep_g5Dphi_clover_sq: out aliases in");
    int rc = workspace(&g->ws_full, 2 * g->bytes_spinor_half);
    if (rc) return rc;
    rc = dphi_clover(g, m0, csw, g->ws_full, in_full, links, clover, 1, "hirep_g5Dphi_clover_sq (first g5 D)");
    if (rc) return rc;
    return dphi_clover(g, m0, csw, out_full, g->ws_full, links, clover, 1, "hirep_g5Dphi_clover_sq (second g5 D)");
}
// the Schur form Eq 43 with the clover blocks: out_e = D_ee in_e - D_eo D_oo^{-1} D_oe in_e
extern "C" int hirep_clover_inv_bytes(const hirep_geom *g, size_t *bytes) {
    if (!g || !bytes) return fail(HIREP_EINVAL, "hirep_clover_inv_bytes: NULL argument");
    *bytes = clover_bytes(g);   // one parity, (2 d_R)^2 = 4 d_R^2 per chirality: the same count as the H,B field of both parities
    return HIREP_OK;
}
extern "C" int hirep_clover_inv_field(hirep_geom *g, double m0, double csw, int parity, void *inv, const void *clover) {
    CHECK_PTRS("hirep_clover_inv_field", inv, clover);
    if (parity != HIREP_EVEN && parity != HIREP_ODD) return fail(HIREP_EINVAL, "hirep_clover_inv_field: parity=%d", parity);
    if (inv == clover) return fail(HIREP_EINVAL, "hirep_clover_inv_field: inv aliases clover");
    int rc = workspace((void **)&g->dev_flags, 64);
    if (rc) return rc;
    return kern_result(g, k_clover_inv(g->geo, g->prec, g->dR, parity, 4.0 + m0, csw, clover, inv, g->dev_flags, g->stream), "hirep_clover_inv_field");
}
extern "C" int hirep_Cphi_inv(hirep_geom *g, void *out_half, const void *in_half, const void *inv) {
    CHECK_PTRS("hirep_Cphi_inv", out_half, in_half, inv);
    if (out_half == in_half) return fail(HIREP_EINVAL, "hirep_Cphi_inv: out aliases in");
    return kern_result(g, k_cblock(g->prec, g->dR, g->geo.n_tiles, inv, in_half, out_half, g->stream), "hirep_Cphi_inv");
}
extern "C" int hirep_Dphi_clover_hat(hirep_geom *g, double m0, double csw, void *out_even, const void *in_even, const void *links,
                                     const void *clover, const void *inv_odd) {
    CHECK_PTRS("hirep_Dphi_clover_hat", out_even, in_even, links, clover, inv_odd);
    if (out_even == in_even) return fail(HIREP_EINVAL, "hirep_Dphi_clover_hat: out aliases in");
    int rc = workspace(&g->ws_half, g->bytes_spinor_half);
    if (rc) return rc;
    if (fuse_diag(g)) {   // two launches: D_oo^-1 in the epilogue of the D_oe pass, D_ee in the epilogue of the D_eo pass
        rc = hop_diag_half(g, DIAG_POST, 0.0, 0.0, -0.5, 0, g->ws_half, in_even, nullptr, links, inv_odd, 1, "hirep_Dphi_clover_hat (D_oo^-1 D_oe pass)");
        if (rc) return rc;
        return hop_diag_half(g, DIAG_HB, 4.0 + m0, csw, +0.5, 0, out_even, g->ws_half, in_even, links, clover, 0, "hirep_Dphi_clover_hat (D_ee - D_eo pass)");
    }
    rc = workspace(&g->ws_half2, g->bytes_spinor_half);
    if (rc) return rc;
    rc = offdiag(g, g->ws_half, in_even, links, 1, "hirep_Dphi_clover_hat (D_oe pass)");
    if (rc) return rc;
    rc = kern_result(g, k_cblock(g->prec, g->dR, g->geo.n_tiles, inv_odd, g->ws_half, g->ws_half2, g->stream), "hirep_Dphi_clover_hat (D_oo^-1)");
    if (rc) return rc;
    rc = kern_result(g, k_cphi(g->prec, g->dR, g->geo.n_tiles, 4.0 + m0, csw, clover, in_even, out_even, g->stream), "hirep_Dphi_clover_hat (D_ee)");
    if (rc) return rc;
    HopLaunch L{};
    L.nsets = 1;
    L.set[0] = HopSet{g->ws_half2, out_even, out_even, links_parity(g, links, 0), 0};
    L.a = 1.0;
    L.b = +0.5;   // - D_eo = -(-1/2) hop
    L.g5 = 0;
    return hop(g, L, "hirep_Dphi_clover_hat (D_eo pass)");
}

// ---- exponential clover (Eq 50) and operators with general site-diagonal chirality blocks -----------------------
extern "C" int hirep_clover_exp_field(hirep_geom *g, double m0, double csw, int parity, int inverse, void *blocks, const void *clover) {
    CHECK_PTRS("hirep_clover_exp_field", blocks, clover);
    if (parity != HIREP_EVEN && parity != HIREP_ODD) return fail(HIREP_EINVAL, "hirep_clover_exp_field: parity=%d", parity);
    if (4.0 + m0 == 0.0) return fail(HIREP_EINVAL, "hirep_clover_exp_field: 4 + m0 = 0");
    if (blocks == clover) return fail(HIREP_EINVAL, "hirep_clover_exp_field: blocks aliases clover");
    int rc = workspace(&g->ws_exp, 2 * clover_bytes(g));
    if (rc) return rc;
    if ((rc = workspace((void **)&g->dev_flags, 64))) return rc;
    const double x = (inverse ? -1.0 : 1.0) * csw / (4.0 + m0), pref = inverse ? 1.0 / (4.0 + m0) : 4.0 + m0;
    return kern_result(g, k_clover_exp(g->geo, g->prec, g->dR, parity, x, pref, clover, blocks, g->ws_exp, g->dev_flags, g->stream), "hirep_clover_exp_field");
}
// out = [gamma_5] (blocks in - 1/2 hop(in)); gamma_5 commutes with the chirality blocks
static int dphi_blocks(hirep_geom *g, void *out_full, const void *in_full, const void *links, const void *blocks_full, int g5, const char *what,
                       const FusedRed *red = nullptr) {
    if (fuse_diag(g)) return hop_diag_full(g, DIAG_PRE, 0.0, 0.0, g5, out_full, in_full, links, blocks_full, clover_bytes(g), what, red);
    if (red) return fail(HIREP_EINVAL, "%s: fused reductions need the fused epilogue", what);
    int rc = kern_result(g, k_cblock(g->prec, g->dR, 2 * g->geo.n_tiles, blocks_full, in_full, out_full, g->stream), what);
    if (rc) return rc;
    const size_t hb = g->bytes_spinor_half;
    const char *in_e = (const char *)in_full, *in_o = in_e + hb;
    char *out_e = (char *)out_full, *out_o = out_e + hb;
    HopLaunch L{};
    L.nsets = 2;
    L.set[0] = HopSet{in_o, out_e, out_e, links_parity(g, links, 0), 0};
    L.set[1] = HopSet{in_e, out_o, out_o, links_parity(g, links, 1), 1};
    L.a = 1.0; L.b = -0.5; L.g5 = g5; L.am = 0.0;
    return hop(g, L, what);
}
extern "C" int hirep_Dphi_blocks(hirep_geom *g, void *out_full, const void *in_full, const void *links, const void *blocks_full) {
    CHECK_PTRS("hirep_Dphi_blocks", out_full, in_full, links, blocks_full);
    if (out_full == in_full) return fail(HIREP_EINVAL, "hirep_Dphi_blocks: out aliases in");
    return dphi_blocks(g, out_full, in_full, links, blocks_full, 0, "hirep_Dphi_blocks");
}
// (gamma_5 D)^2 with Hermitian site-diagonal blocks (the exponential clover's): Hermitian positive definite; gamma_5 D in is
// left in ws_full for the CG
extern "C" int hirep_g5Dphi_blocks_sq(hirep_geom *g, void *out_full, const void *in_full, const void *links, const void *blocks_full) {
    CHECK_PTRS("hirep_g5Dphi_blocks_sq", out_full, in_full, links, blocks_full);
    if (out_full == in_full) return fail(HIREP_EINVAL, "hirep_g5Dphi_blocks_sq: out aliases in");
    int rc = workspace(&g->ws_full, 2 * g->bytes_spinor_half);
    if (rc) return rc;
    rc = dphi_blocks(g, g->ws_full, in_full, links, blocks_full, 1, "hirep_g5Dphi_blocks_sq (first g5 D)");
    if (rc) return rc;
    return dphi_blocks(g, out_full, g->ws_full, links, blocks_full, 1, "hirep_g5Dphi_blocks_sq (second g5 D)");
}
extern "C" int hirep_Dphi_blocks_hat(hirep_geom *g, void *out_even, const void *in_even, const void *links, const void *blocks_even,
                                     const void *inv_blocks_odd) {
    CHECK_PTRS("hirep_Dphi_blocks_hat", out_even, in_even, links, blocks_even, inv_blocks_odd);
    if (out_even == in_even) return fail(HIREP_EINVAL, "hirep_Dphi_blocks_hat: out aliases in");
    int rc = workspace(&g->ws_half, g->bytes_spinor_half);
    if (rc) return rc;
    if (fuse_diag(g)) {
        rc = hop_diag_half(g, DIAG_POST, 0.0, 0.0, -0.5, 0, g->ws_half, in_even, nullptr, links, inv_blocks_odd, 1, "hirep_Dphi_blocks_hat (D_oo^-1 D_oe pass)");
        if (rc) return rc;
        return hop_diag_half(g, DIAG_PRE, 0.0, 0.0, +0.5, 0, out_even, g->ws_half, in_even, links, blocks_even, 0, "hirep_Dphi_blocks_hat (D_ee - D_eo pass)");
    }
    rc = workspace(&g->ws_half2, g->bytes_spinor_half);
    if (rc) return rc;
    rc = offdiag(g, g->ws_half, in_even, links, 1, "hirep_Dphi_blocks_hat (D_oe pass)");
    if (rc) return rc;
    rc = kern_result(g, k_cblock(g->prec, g->dR, g->geo.n_tiles, inv_blocks_odd, g->ws_half, g->ws_half2, g->stream), "hirep_Dphi_blocks_hat (D_oo^-1)");
    if (rc) return rc;
    rc = kern_result(g, k_cblock(g->prec, g->dR, g->geo.n_tiles, blocks_even, in_even, out_even, g->stream), "hirep_Dphi_blocks_hat (D_ee)");
    if (rc) return rc;
    HopLaunch L{};
    L.nsets = 1;
    L.set[0] = HopSet{g->ws_half2, out_even, out_even, links_parity(g, links, 0), 0};
    L.a = 1.0; L.b = +0.5; L.g5 = 0;
    return hop(g, L, "hirep_Dphi_blocks_hat (D_eo pass)");
}

// [gamma_5] D_hat for site-diagonal blocks (Eq 43): D_ee is either Cphi from the clover field (clover != NULL) or the
// given even blocks; gamma_5 commutes with the blocks, so it is applied once in the last stencil epilogue
static int blocks_hat(hirep_geom *g, double m0, double csw, void *out_even, const void *in_even, const void *links, const void *clover,
                      const void *blocks_even, const void *inv_odd, int g5, const char *what, const FusedRed *red = nullptr) {
    int rc = workspace(&g->ws_half, g->bytes_spinor_half);
    if (rc) return rc;
    if (fuse_diag(g)) {
        rc = hop_diag_half(g, DIAG_POST, 0.0, 0.0, -0.5, 0, g->ws_half, in_even, nullptr, links, inv_odd, 1, what);
        if (rc) return rc;
        return clover ? hop_diag_half(g, DIAG_HB, 4.0 + m0, csw, +0.5, g5, out_even, g->ws_half, in_even, links, clover, 0, what, red)
                      : hop_diag_half(g, DIAG_PRE, 0.0, 0.0, +0.5, g5, out_even, g->ws_half, in_even, links, blocks_even, 0, what, red);
    }
    if (red) return fail(HIREP_EINVAL, "%s: fused reductions need the fused epilogue", what);
    rc = workspace(&g->ws_half2, g->bytes_spinor_half);
    if (rc) return rc;
    rc = offdiag(g, g->ws_half, in_even, links, 1, what);
    if (rc) return rc;
    rc = kern_result(g, k_cblock(g->prec, g->dR, g->geo.n_tiles, inv_odd, g->ws_half, g->ws_half2, g->stream), what);
    if (rc) return rc;
    rc = clover ? kern_result(g, k_cphi(g->prec, g->dR, g->geo.n_tiles, 4.0 + m0, csw, clover, in_even, out_even, g->stream), what)
                : kern_result(g, k_cblock(g->prec, g->dR, g->geo.n_tiles, blocks_even, in_even, out_even, g->stream), what);
    if (rc) return rc;
    HopLaunch L{};
    L.nsets = 1;
    L.set[0] = HopSet{g->ws_half2, out_even, out_even, links_parity(g, links, 0), 0};
    L.a = 1.0; L.b = +0.5; L.g5 = g5;
    return hop(g, L, what);
}
// Q_hat^2 = (gamma_5 D_hat)^2 with D_hat of Eq 43: gamma_5 D_hat is Hermitian when the blocks are (gamma_5 D_ee gamma_5 =
// D_ee^dagger, gamma_5 D_eo gamma_5 = D_oe^dagger), so this is Hermitian positive definite: the even-odd preconditioned
// CG operator with a clover or exponential clover term (L803, L815).  Q_hat in is left in ws_half3 for the CG.
static int blocks_hat_sq(hirep_geom *g, double m0, double csw, void *out_even, const void *in_even, const void *links, const void *clover,
                         const void *blocks_even, const void *inv_odd, const char *what) {
    int rc = workspace(&g->ws_half3, g->bytes_spinor_half);
    if (rc) return rc;
    rc = blocks_hat(g, m0, csw, g->ws_half3, in_even, links, clover, blocks_even, inv_odd, 1, what);
    if (rc) return rc;
    return blocks_hat(g, m0, csw, out_even, g->ws_half3, links, clover, blocks_even, inv_odd, 1, what);
}
extern "C" int hirep_g5Dphi_clover_hat_sq(hirep_geom *g, double m0, double csw, void *out_even, const void *in_even, const void *links,
                                          const void *clover, const void *inv_odd) {
    CHECK_PTRS("hirep_g5Dphi_clover_hat_sq", out_even, in_even, links, clover, inv_odd);
    if (out_even == in_even) return fail(HIREP_EINVAL, "hirep_g5Dphi_clover_hat_sq: out aliases in");
    return blocks_hat_sq(g, m0, csw, out_even, in_even, links, clover, nullptr, inv_odd, "hirep_g5Dphi_clover_hat_sq");
}
extern "C" int hirep_g5Dphi_blocks_hat_sq(hirep_geom *g, void *out_even, const void *in_even, const void *links, const void *blocks_even,
                                          const void *inv_blocks_odd) {
    CHECK_PTRS("hirep_g5Dphi_blocks_hat_sq", out_even, in_even, links, blocks_even, inv_blocks_odd);
    if (out_even == in_even) return fail(HIREP_EINVAL, "hirep_g5Dphi_blocks_hat_sq: out aliases in");
    return blocks_hat_sq(g, 0.0, 0.0, out_even, in_even, links, nullptr, blocks_even, inv_blocks_odd, "hirep_g5Dphi_blocks_hat_sq");
}

static long spinor_elems(const hirep_geom *g, int which) {   // complex elements of a native buffer, padding included
    return (long)g->geo.n_tiles * 4 * g->dR * TILE * (which == HIREP_FULL ? 2 : 1);
}
static int lincomb(hirep_geom *g, int which, void *xi, const double c0[2], int use_xi, const void *eta, const double c1[2],
                   const void *zeta, const double c2[2], int use_zeta, const char *what) {
    if (which < 0 || which > 2) return fail(HIREP_EINVAL, "%s: parity_or_full=%d", what, which);
    return kern_result(g, k_lincomb(g->prec, spinor_elems(g, which), xi, c0, use_xi, eta, c1, zeta, c2, use_zeta, g->stream), what);
}
static const double ZERO2[2] = {0.0, 0.0}, ONE2[2] = {1.0, 0.0}, MINUS2[2] = {-1.0, 0.0};

extern "C" int hirep_spinor_lc(hirep_geom *g, int which, void *xi, double r1, const void *eta, double r2, const void *zeta) {
    CHECK_PTRS("hirep_spinor_lc", xi, eta, zeta);
    const double c1[2] = {r1, 0.0}, c2[2] = {r2, 0.0};
    return lincomb(g, which, xi, ZERO2, 0, eta, c1, zeta, c2, 1, "hirep_spinor_lc");
}
extern "C" int hirep_spinor_clc(hirep_geom *g, int which, void *xi, const double c1[2], const void *eta, const double c2[2], const void *zeta) {
    CHECK_PTRS("hirep_spinor_clc", xi, eta, zeta);
    if (!c1 || !c2) return fail(HIREP_EINVAL, "hirep_spinor_clc: NULL coefficient");
    return lincomb(g, which, xi, ZERO2, 0, eta, c1, zeta, c2, 1, "hirep_spinor_clc");
}
extern "C" int hirep_spinor_lc_add_assign(hirep_geom *g, int which, void *xi, double r1, const void *eta, double r2, const void *zeta) {
    CHECK_PTRS("hirep_spinor_lc_add_assign", xi, eta, zeta);
    const double c1[2] = {r1, 0.0}, c2[2] = {r2, 0.0};
    return lincomb(g, which, xi, ONE2, 1, eta, c1, zeta, c2, 1, "hirep_spinor_lc_add_assign");
}
extern "C" int hirep_spinor_clc_add_assign(hirep_geom *g, int which, void *xi, const double c1[2], const void *eta, const double c2[2], const void *zeta) {
    CHECK_PTRS("hirep_spinor_clc_add_assign", xi, eta, zeta);
    if (!c1 || !c2) return fail(HIREP_EINVAL, "hirep_spinor_clc_add_assign: NULL coefficient");
    return lincomb(g, which, xi, ONE2, 1, eta, c1, zeta, c2, 1, "hirep_spinor_clc_add_assign");
}
extern "C" int hirep_spinor_lc1(hirep_geom *g, int which, void *xi, const double c1[2], const void *eta) {
    CHECK_PTRS("hirep_spinor_lc1", xi, eta);
    if (!c1) return fail(HIREP_EINVAL, "hirep_spinor_lc1: NULL coefficient");
    return lincomb(g, which, xi, ONE2, 1, eta, c1, eta, ZERO2, 0, "hirep_spinor_lc1");
}
extern "C" int hirep_spinor_lc2(hirep_geom *g, int which, void *xi, const double c1[2], const double c2[2], const void *eta) {
    CHECK_PTRS("hirep_spinor_lc2", xi, eta);
    if (!c1 || !c2) return fail(HIREP_EINVAL, "hirep_spinor_lc2: NULL coefficient");
    return lincomb(g, which, xi, c1, 1, eta, c2, eta, ZERO2, 0, "hirep_spinor_lc2");
}
extern "C" int hirep_spinor_lc3(hirep_geom *g, int which, void *xi, const double c1[2], const void *eta, const double c2[2], const void *zeta) {
    CHECK_PTRS("hirep_spinor_lc3", xi, eta, zeta);
    if (!c1 || !c2) return fail(HIREP_EINVAL, "hirep_spinor_lc3: NULL coefficient");
    return lincomb(g, which, xi, MINUS2, 1, eta, c1, zeta, c2, 1, "hirep_spinor_lc3");
}

// the elementary operations of L365-371: zero, copy, multiplication by a scalar, global minus sign (one streaming
// kernel each, as the paper prefers over memset/memcpy)
extern "C" int hirep_spinor_zero(hirep_geom *g, int which, void *xi) {
    CHECK_PTRS("hirep_spinor_zero", xi);
    if (which < 0 || which > 2) return fail(HIREP_EINVAL, "hirep_spinor_zero: parity_or_full=%d", which);
    const cudaError_t e = cudaMemsetAsync(xi, 0, (which == HIREP_FULL ? 2 : 1) * g->bytes_spinor_half, g->stream);   // exact zeros, also over NaNs
    return e == cudaSuccess ? HIREP_OK : cuda_fail(e, "hirep_spinor_zero");
}
extern "C" int hirep_spinor_copy(hirep_geom *g, int which, void *xi, const void *eta) {
    CHECK_PTRS("hirep_spinor_copy", xi, eta);
    if (xi == eta) return HIREP_OK;
    return lincomb(g, which, xi, ZERO2, 0, eta, ONE2, eta, ZERO2, 0, "hirep_spinor_copy");
}
extern "C" int hirep_spinor_mul(hirep_geom *g, int which, void *xi, const double c[2], const void *eta) {
    CHECK_PTRS("hirep_spinor_mul", xi, eta);
    if (!c) return fail(HIREP_EINVAL, "hirep_spinor_mul: NULL coefficient");
    return lincomb(g, which, xi, ZERO2, 0, eta, c, eta, ZERO2, 0, "hirep_spinor_mul");
}
extern "C" int hirep_spinor_minus(hirep_geom *g, int which, void *xi, const void *eta) {
    CHECK_PTRS("hirep_spinor_minus", xi, eta);
    return lincomb(g, which, xi, ZERO2, 0, eta, MINUS2, eta, ZERO2, 0, "hirep_spinor_minus");
}

static int red_workspace(hirep_geom *g) { return workspace(&g->ws_red, (size_t)k_reduce_workspace_bytes() + 64); }
static double *red_out(hirep_geom *g) { return (double *)((char *)g->ws_red + k_reduce_workspace_bytes()); }
static int fetch_result(hirep_geom *g, double *host, int n, const char *what) {
    cudaError_t e = cudaMemcpyAsync(host, red_out(g), n * sizeof(double), cudaMemcpyDeviceToHost, g->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(g->stream);
    if (e != cudaSuccess) return cuda_fail(e, what);
    return HIREP_OK;
}
static int reduce_prod(hirep_geom *g, int which, int mode, const void *xi, const void *eta, double *host, const char *what) {
    if (which < 0 || which > 2) return fail(HIREP_EINVAL, "%s: parity_or_full=%d", what, which);
    int rc = red_workspace(g);
    if (rc) return rc;
    rc = kern_result(g, k_prod(g->geo, g->prec, g->dR, which == HIREP_FULL ? 2 : 1, mode, g->sum_alg, xi, eta, g->ws_red, red_out(g), g->stream), what, 2);
    if (rc) return rc;
    return fetch_result(g, host, 2, what);
}
extern "C" int hirep_spinor_prod(hirep_geom *g, int which, const void *xi, const void *eta, double out[2]) {
    CHECK_PTRS("hirep_spinor_prod", xi, eta);
    if (!out) return fail(HIREP_EINVAL, "hirep_spinor_prod: NULL result pointer");
    return reduce_prod(g, which, 0, xi, eta, out, "hirep_spinor_prod");
}
extern "C" int hirep_spinor_g5_prod(hirep_geom *g, int which, const void *xi, const void *eta, double out[2]) {
    CHECK_PTRS("hirep_spinor_g5_prod", xi, eta);
    if (!out) return fail(HIREP_EINVAL, "hirep_spinor_g5_prod: NULL result pointer");
    return reduce_prod(g, which, 2, xi, eta, out, "hirep_spinor_g5_prod");
}
extern "C" int hirep_spinor_sqnorm(hirep_geom *g, int which, const void *xi, double *out) {
    CHECK_PTRS("hirep_spinor_sqnorm", xi);
    if (!out) return fail(HIREP_EINVAL, "hirep_spinor_sqnorm: NULL result pointer");
    double r[2];
    const int rc = reduce_prod(g, which, 1, xi, xi, r, "hirep_spinor_sqnorm");
    if (rc == HIREP_OK) *out = r[0];
    return rc;
}
extern "C" int hirep_spinor_max_norm(hirep_geom *g, int which, const void *eta, double *out) {
    CHECK_PTRS("hirep_spinor_max_norm", eta);
    if (!out) return fail(HIREP_EINVAL, "hirep_spinor_max_norm: NULL result pointer");
    if (which < 0 || which > 2) return fail(HIREP_EINVAL, "hirep_spinor_max_norm: parity_or_full=%d", which);
    int rc = red_workspace(g);
    if (rc) return rc;
    rc = kern_result(g, k_maxnorm(g->geo, g->prec, g->dR, which == HIREP_FULL ? 2 : 1, eta, g->ws_red, red_out(g), g->stream), "hirep_spinor_max_norm", 2);
    if (rc) return rc;
    return fetch_result(g, out, 1, "hirep_spinor_max_norm");
}

// Conjugate gradient for A x = b with A = Q_m^2 = g5Dphi_sq (full lattice) or A = Q_hat^2 = g5Dphi_hat_sq (even
// sites), both Hermitian positive definite (L772, L815).  Textbook recurrence (reading A19): x0 = 0; r = b;
// p = r; repeat { Ap; alpha = rr/<p,Ap>; x += alpha p; r -= alpha Ap; rr' = <r,r>; stop if rr' <= tol^2 <b,b>;
// beta = rr'/rr; p = r + beta p }.  Per iteration: the operator (2 or 4 stencil launches), <p,Ap> = ||B p||^2 (2 launches),
// r -= alpha Ap fused with ||r||^2 (2), x += alpha p fused with the p update (1): 8 spinor passes of linear algebra.
// alpha, beta never leave the device and the next operator application is queued before the host reads ||r||^2 (see below).
static int cg_solve(hirep_geom *g, int full, double m0, void *x, const void *b, const void *links, double tol, int maxiter, int *iters,
                    double *relres, const char *what, int twisted = 0, double mu = 0.0, const void *clover = nullptr, double csw = 0.0,
                    const void *blocks_even = nullptr, const void *inv_odd = nullptr) {
    if (x == b) return fail(HIREP_EINVAL, "%s: x aliases b", what);
    if (!(tol > 0.0) || maxiter < 0) return fail(HIREP_EINVAL, "%s: tol=%g maxiter=%d", what, tol, maxiter);
    const int which = full ? HIREP_FULL : HIREP_EVEN, halves = full ? 2 : 1;
    const size_t fb = halves * g->bytes_spinor_half;
    int rc;
    // work fields are allocated at full-lattice size once and serve both operators
    const size_t wb = 2 * g->bytes_spinor_half;
    if ((rc = workspace(&g->cg_r, wb)) || (rc = workspace(&g->cg_p, wb)) || (rc = workspace(&g->cg_Ap, wb)) || (rc = red_workspace(g))) return rc;
    cudaError_t e = cudaMemsetAsync(x, 0, fb, g->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(g->cg_r, b, fb, cudaMemcpyDeviceToDevice, g->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(g->cg_p, b, fb, cudaMemcpyDeviceToDevice, g->stream);
    if (e != cudaSuccess) return cuda_fail(e, what);
    if (!g->h_scal) {
        if ((e = cudaHostAlloc((void **)&g->h_scal, 8 * sizeof(double), cudaHostAllocDefault)) != cudaSuccess) return cuda_fail(e, what);
        if ((e = cudaEventCreateWithFlags(&g->ev_scal, cudaEventDisableTiming)) != cudaSuccess) {
            cudaFreeHost(g->h_scal); g->h_scal = nullptr;
            return cuda_fail(e, what);
        }
    }
    double bb, rr;
    if ((rc = hirep_spinor_sqnorm(g, which, b, &bb))) return rc;
    rr = bb;
    if (!std::isfinite(bb)) return breakdown(g, "%s: <b,b> = %g is not finite", what, bb);
    // The scalars stay on the device: d[0..1] = <p,Ap>, d[2..3] / d[4..5] = ||r||^2 of the even / odd iterations; alpha and beta
    // are formed in the update kernels by the same IEEE divisions the host would do.  The host only reads ||r||^2 (and <p,Ap>,
    // to report a non-positive value) for the stopping rule, and it does so AFTER it has queued the next operator application, so
    // the GPU never idles on the round trip; a solve that stops on the tolerance has queued one operator application too many
    // (it writes only Ap and the operator's workspaces).
    double *d = red_out(g);
    if ((e = cudaMemcpyAsync(d + 2, d, sizeof(double), cudaMemcpyDeviceToDevice, g->stream)) != cudaSuccess) return cuda_fail(e, what);
    auto apply_op = [&]() -> int {
        int rc2 = inv_odd ? blocks_hat_sq(g, m0, csw, g->cg_Ap, g->cg_p, links, clover, blocks_even, inv_odd, what)
                : blocks_even ? hirep_g5Dphi_blocks_sq(g, g->cg_Ap, g->cg_p, links, blocks_even)
                : clover ? hirep_g5Dphi_clover_sq(g, m0, csw, g->cg_Ap, g->cg_p, links, clover)
                : twisted ? hirep_Dphi_tm_sq(g, m0, mu, g->cg_Ap, g->cg_p, links)
                          : full ? hirep_g5Dphi_sq(g, m0, g->cg_Ap, g->cg_p, links) : hirep_g5Dphi_hat_sq(g, m0, g->cg_Ap, g->cg_p, links);
        if (rc2) return rc2;
        // A = B^dagger B with B p left in the operator's workspace (gamma_5 D p, Q_hat p, gamma_5 D^tm p; gamma_5 is
        // unitary), so <p, A p> = ||B p||^2: one field read instead of two
        const void *Bp = inv_odd ? g->ws_half3 : (full || twisted) ? g->ws_full : g->ws_half2;
        return kern_result(g, k_prod(g->geo, g->prec, g->dR, halves, 1, g->sum_alg, Bp, Bp, g->ws_red, d, g->stream), what, 2);
    };
    // Fused form (plain Wilson Q^2 on the full lattice, when the tile-pair kernel runs it): pass 1 = gamma_5 D p with ||B p||^2 = <p,Ap>
    // accumulated in its epilogue; pass 2 = gamma_5 D (B p) whose epilogue does r -= alpha A p and accumulates ||r||^2 without ever
    // storing A p: 3 spinor passes and 2 launches fewer per iteration (the separate ||Bp||^2 and residual-update kernels are gone).
    // Even-odd form (Q_hat^2, ring / pair kernels): the same two reductions ride on the second pass of each Q_hat application.
    // Operators with site-diagonal matrices (clover, exponential clover; full lattice and Schur form): when their matrices ride in the
    // stencil epilogues (fuse_diag) the last launch of each B = gamma_5 D [hat] application is a ring / pair kernel launch whose
    // epilogue carries the same two reductions.
    const bool plain = !twisted && !clover && !blocks_even && !inv_odd;
    const bool diag = !twisted && !plain;
    // Twisted mass ((D^tm)^dagger D^tm = [gamma_5 D^tm(-mu)] [gamma_5 D^tm(mu)], full lattice): the same two passes with +-mu in the epilogues.
    const bool fused = plain ? (full ? fused_cg_ok(g) : fused_cg_eo_ok(g)) : twisted ? (full && fused_cg_ok(g)) : (diag && fuse_diag(g) && fused_cg_eo_ok(g));
    const int nred = k_reduce_workspace_bytes() / (int)(2 * 3 * sizeof(double));   // Acc pairs the partial buffer holds
    void *Bp_f = nullptr;   // B p of the fused form
    if (fused) {
        void **slot = inv_odd ? &g->ws_half3 : full ? &g->ws_full : &g->ws_half2;
        if ((rc = workspace(&g->ws_red2, (size_t)k_reduce_workspace_bytes())) || (rc = workspace(slot, (full ? 2 : 1) * g->bytes_spinor_half))) return rc;
        if ((e = cudaMemsetAsync(g->ws_red2, 0, (size_t)k_reduce_workspace_bytes(), g->stream)) != cudaSuccess) return cuda_fail(e, what);
        Bp_f = *slot;
    }
    // one application of B with the reduction `fr` in the epilogue of its last launch
    auto apply_B = [&](void *out, const void *in, const FusedRed *fr) -> int {
        if (twisted) return dphi_full(g, m0, out, in, links, 1, what, fr->mode == 1 ? mu : -mu, fr);   // pass 1: gamma_5 D^tm(mu), pass 2: gamma_5 D^tm(-mu)
        if (inv_odd) return blocks_hat(g, m0, csw, out, in, links, clover, blocks_even, inv_odd, 1, what, fr);
        if (blocks_even) return dphi_blocks(g, out, in, links, blocks_even, 1, what, fr);
        if (clover) return dphi_clover(g, m0, csw, out, in, links, clover, 1, what, fr);
        return full ? dphi_full(g, m0, out, in, links, 1, what, 0.0, fr) : dphi_hat(g, m0, out, in, links, 1, what, fr);
    };
    auto fused_pass1 = [&]() -> int {
        const FusedRed fr{1, nullptr, nullptr, nullptr};
        int rc2 = apply_B(Bp_f, g->cg_p, &fr);
        if (rc2) return rc2;
        return kern_result(g, k_reduce_final(nred, g->sum_alg, g->ws_red2, d, g->stream), what);
    };
    int it = 0;
    bool more = bb > 0.0 && it < maxiter && !(rr <= tol * tol * bb);
    if (more && (rc = fused ? fused_pass1() : apply_op())) return rc;
    while (more) {
        double *rr_old = d + 2 + 2 * (it & 1), *rr_new_d = d + 2 + 2 * ((it + 1) & 1);
        if (fused) {
            const FusedRed fr{2, g->cg_r, rr_old, d};
            if ((rc = apply_B(g->cg_Ap, Bp_f, &fr))) return rc;
            if ((rc = kern_result(g, k_reduce_final(nred, g->sum_alg, g->ws_red2, rr_new_d, g->stream), what))) return rc;
        } else {
            rc = kern_result(g, k_cg_update(g->geo, g->prec, g->dR, halves, g->sum_alg, 0.0, rr_old, d, nullptr, g->cg_r, g->cg_p, g->cg_Ap, g->ws_red, rr_new_d, g->stream), what, 2);
            if (rc) return rc;
        }
        if ((rc = kern_result(g, k_cg_xp(g->geo, g->prec, g->dR, halves, 0.0, 0.0, rr_old, d, rr_new_d, x, g->cg_p, g->cg_r, g->stream), what))) return rc;
        if ((e = cudaMemcpyAsync(g->h_scal, d, sizeof(double), cudaMemcpyDeviceToHost, g->stream)) != cudaSuccess) return cuda_fail(e, what);
        if ((e = cudaMemcpyAsync(g->h_scal + 1, rr_new_d, sizeof(double), cudaMemcpyDeviceToHost, g->stream)) != cudaSuccess) return cuda_fail(e, what);
        if ((e = cudaEventRecord(g->ev_scal, g->stream)) != cudaSuccess) return cuda_fail(e, what);
        ++it;
        if (it < maxiter && (rc = fused ? fused_pass1() : apply_op())) return rc;   // queued before the host looks at ||r||^2
        if ((e = cudaEventSynchronize(g->ev_scal)) != cudaSuccess) return cuda_fail(e, what);
        const double pAp = g->h_scal[0];
        if (!(pAp > 0.0) || !std::isfinite(pAp))
            return breakdown(g, "%s: <p,Ap> = %g is not positive and finite (operator not positive definite?); x is undefined", what, pAp);
        rr = g->h_scal[1];
        if (!std::isfinite(rr)) return breakdown(g, "%s: ||r||^2 = %g is not finite; x is undefined", what, rr);
        more = it < maxiter && !(rr <= tol * tol * bb);
    }
    if (iters) *iters = it;
    if (relres) *relres = bb > 0.0 ? sqrt(rr / bb) : 0.0;
    return hirep_sync(g);
}

// Multi-shift CG for (Q_m^2 + sigma_k) x_k = b, k < nshift (L730; Eq 39-40: what the RHMC's rational approximation
// needs).  One Krylov space: the unshifted recurrence (r, p, alpha, beta) plus, per shift, zeta_k, x_k and p_k
// (recurrence: DESIGN.md A24).  Per iteration: the operator, <p,Ap>, the residual update +
// ||r||^2, the p update, and two fused linear combinations per shift.
extern "C" int hirep_cg_mshift_g5Dphi_sq(hirep_geom *g, double m0, int nshift, const double *shifts, void *const *x_full, const void *b_full,
                                         const void *links, double tol, int maxiter, int *iters, double *relres) {
    CHECK_PTRS("hirep_cg_mshift_g5Dphi_sq", b_full, links);
    const char *what = "hirep_cg_mshift_g5Dphi_sq";
    if (!shifts || !x_full || nshift < 1 || nshift > HIREP_MAX_SHIFTS) return fail(HIREP_EINVAL, "%s: nshift=%d (1..%d), shifts/x must be given", what, nshift, HIREP_MAX_SHIFTS);
    if (!(tol > 0.0) || maxiter < 0) return fail(HIREP_EINVAL, "%s: tol=%g maxiter=%d", what, tol, maxiter);
    for (int k = 0; k < nshift; ++k) {
        if (!x_full[k] || misaligned(x_full[k]) || x_full[k] == b_full) return fail(HIREP_EINVAL, "%s: bad solution pointer %d", what, k);
        if (!(shifts[k] >= 0.0)) return fail(HIREP_EINVAL, "%s: shift %d = %g must be >= 0", what, k, shifts[k]);
    }
    const size_t fb = 2 * g->bytes_spinor_half;
    int rc;
    if ((rc = workspace(&g->cg_r, fb)) || (rc = workspace(&g->cg_p, fb)) || (rc = workspace(&g->cg_Ap, fb)) || (rc = red_workspace(g))) return rc;
    cudaError_t e = cudaMemcpyAsync(g->cg_r, b_full, fb, cudaMemcpyDeviceToDevice, g->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(g->cg_p, b_full, fb, cudaMemcpyDeviceToDevice, g->stream);
    for (int k = 0; k < nshift && e == cudaSuccess; ++k) {
        if ((rc = workspace(&g->ms_p[k], fb))) return rc;
        e = cudaMemsetAsync(x_full[k], 0, fb, g->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(g->ms_p[k], b_full, fb, cudaMemcpyDeviceToDevice, g->stream);
    }
    if (e != cudaSuccess) return cuda_fail(e, what);
    double bb, rr, res[2];
    if ((rc = hirep_spinor_sqnorm(g, HIREP_FULL, b_full, &bb))) return rc;
    rr = bb;
    if (!std::isfinite(bb)) return breakdown(g, "%s: <b,b> = %g is not finite", what, bb);
    double zeta[HIREP_MAX_SHIFTS], zeta_old[HIREP_MAX_SHIFTS], zeta_new[HIREP_MAX_SHIFTS];
    for (int k = 0; k < nshift; ++k) zeta[k] = zeta_old[k] = 1.0;
    double alpha_old = 1.0, beta_old = 0.0;
    int it = 0;
    while (bb > 0.0 && it < maxiter && !(rr <= tol * tol * bb)) {
        if ((rc = hirep_g5Dphi_sq(g, m0, g->cg_Ap, g->cg_p, links))) return rc;
        if ((rc = reduce_prod(g, HIREP_FULL, 0, g->cg_p, g->cg_Ap, res, what))) return rc;
        if (!(res[0] > 0.0) || !std::isfinite(res[0])) return breakdown(g, "%s: <p,Ap> = %g is not positive and finite; x is undefined", what, res[0]);
        const double alpha = rr / res[0];
        for (int k = 0; k < nshift; ++k) {
            zeta_new[k] = zeta[k] * zeta_old[k] * alpha_old /
                          (alpha * beta_old * (zeta_old[k] - zeta[k]) + zeta_old[k] * alpha_old * (1.0 + shifts[k] * alpha));
            const double ak[2] = {alpha * zeta_new[k] / zeta[k], 0.0};
            if ((rc = lincomb(g, HIREP_FULL, x_full[k], ONE2, 1, g->ms_p[k], ak, g->ms_p[k], ZERO2, 0, what))) return rc;   // x_k += alpha_k p_k
        }
        rc = kern_result(g, k_cg_update(g->geo, g->prec, g->dR, 2, g->sum_alg, alpha, nullptr, nullptr, nullptr, g->cg_r, g->cg_p, g->cg_Ap, g->ws_red, red_out(g), g->stream), what, 2);
        if (rc) return rc;
        if ((rc = fetch_result(g, res, 2, what))) return rc;
        const double rr_new = res[0], beta = rr_new / rr;
        if (!std::isfinite(rr_new)) return breakdown(g, "%s: ||r||^2 = %g is not finite; x is undefined", what, rr_new);
        ++it;
        for (int k = 0; k < nshift; ++k) {
            const double q = zeta_new[k] / zeta[k];
            const double bk[2] = {beta * q * q, 0.0}, zk[2] = {zeta_new[k], 0.0};
            if ((rc = lincomb(g, HIREP_FULL, g->ms_p[k], bk, 1, g->cg_r, zk, g->cg_r, ZERO2, 0, what))) return rc;   // p_k = zeta_k' r + beta_k p_k
            zeta_old[k] = zeta[k];
            zeta[k] = zeta_new[k];
        }
        const double b2[2] = {beta, 0.0};
        if ((rc = lincomb(g, HIREP_FULL, g->cg_p, b2, 1, g->cg_r, ONE2, g->cg_r, ZERO2, 0, what))) return rc;
        alpha_old = alpha;
        beta_old = beta;
        rr = rr_new;
    }
    if (iters) *iters = it;
    if (relres) *relres = bb > 0.0 ? sqrt(rr / bb) : 0.0;
    return hirep_sync(g);
}

// BiCGstab (L730) for D_m x = b (op = HIREP_OP_DPHI, full lattice) or D_hat x = b (op = HIREP_OP_DPHI_HAT, even sites).
// Textbook recurrence (A25), x0 = 0, shadow residual = b.  Work fields: r (cg_r), p (cg_p), v (cg_Ap), s and t
// (bi_s, bi_t), rhat = b itself.  Per iteration: 2 operator applications, 4 products / norms, 4 fused linear combinations.
extern "C" int hirep_bicgstab(hirep_geom *g, int op, double m0, void *x, const void *b, const void *links, double tol, int maxiter,
                              int *iters, double *relres) {
    CHECK_PTRS("hirep_bicgstab", x, b, links);
    const char *what = "hirep_bicgstab";
    if (op != HIREP_OP_DPHI && op != HIREP_OP_DPHI_HAT) return fail(HIREP_EINVAL, "%s: op %d (HIREP_OP_DPHI or HIREP_OP_DPHI_HAT)", what, op);
    if (x == b) return fail(HIREP_EINVAL, "%s: x aliases b", what);
    if (!(tol > 0.0) || maxiter < 0) return fail(HIREP_EINVAL, "%s: tol=%g maxiter=%d", what, tol, maxiter);
    const int full = op == HIREP_OP_DPHI, which = full ? HIREP_FULL : HIREP_EVEN;
    const size_t fb = (full ? 2 : 1) * g->bytes_spinor_half, wb = 2 * g->bytes_spinor_half;
    int rc;
    if ((rc = workspace(&g->cg_r, wb)) || (rc = workspace(&g->cg_p, wb)) || (rc = workspace(&g->cg_Ap, wb)) || (rc = workspace(&g->bi_s, wb)) ||
        (rc = workspace(&g->bi_t, wb)) || (rc = red_workspace(g)))
        return rc;
    void *r = g->cg_r, *p = g->cg_p, *v = g->cg_Ap, *sv = g->bi_s, *t = g->bi_t;
    cudaError_t e = cudaMemsetAsync(x, 0, fb, g->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(r, b, fb, cudaMemcpyDeviceToDevice, g->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(p, 0, fb, g->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(v, 0, fb, g->stream);
    if (e != cudaSuccess) return cuda_fail(e, what);
    auto apply = [&](void *out, const void *in) { return full ? hirep_Dphi(g, m0, out, in, links) : hirep_Dphi_hat(g, m0, out, in, links); };
    auto cdiv = [](const double a[2], const double c[2], double out[2]) {
        const double d = c[0] * c[0] + c[1] * c[1];
        out[0] = (a[0] * c[0] + a[1] * c[1]) / d;
        out[1] = (a[1] * c[0] - a[0] * c[1]) / d;
    };
    auto cmul2 = [](const double a[2], const double c[2], double out[2]) {
        const double re = a[0] * c[0] - a[1] * c[1], im = a[0] * c[1] + a[1] * c[0];
        out[0] = re; out[1] = im;
    };
    double bb, rr, rho[2] = {1, 0}, alpha[2] = {1, 0}, omega[2] = {1, 0};
    if ((rc = hirep_spinor_sqnorm(g, which, b, &bb))) return rc;
    rr = bb;
    if (!std::isfinite(bb)) return breakdown(g, "%s: <b,b> = %g is not finite", what, bb);
    auto zero_or_nan = [](const double c[2]) { return !std::isfinite(c[0]) || !std::isfinite(c[1]) || (c[0] == 0.0 && c[1] == 0.0); };
    int it = 0;
    while (bb > 0.0 && it < maxiter && !(rr <= tol * tol * bb)) {
        double rho_new[2], q1[2], q2[2], beta[2], mbw[2], rv[2], ss, tt, ts[2];
        if ((rc = reduce_prod(g, which, 0, b, r, rho_new, what))) return rc;                     // rho' = <rhat, r>
        if (zero_or_nan(rho_new)) return breakdown(g, "%s: breakdown (rho = <rhat,r> = %g%+gi); x is undefined", what, rho_new[0], rho_new[1]);
        cdiv(rho_new, rho, q1); cdiv(alpha, omega, q2); cmul2(q1, q2, beta);                      // beta = (rho'/rho)(alpha/omega)
        cmul2(beta, omega, mbw); mbw[0] = -mbw[0]; mbw[1] = -mbw[1];
        if ((rc = lincomb(g, which, p, beta, 1, r, ONE2, v, mbw, 1, what))) return rc;            // p = r + beta p - beta omega v
        if ((rc = apply(v, p))) return rc;                                                        // v = A p
        if ((rc = reduce_prod(g, which, 0, b, v, rv, what))) return rc;
        if (zero_or_nan(rv)) return breakdown(g, "%s: breakdown (<rhat,v> = %g%+gi); x is undefined", what, rv[0], rv[1]);
        cdiv(rho_new, rv, alpha);                                                                 // alpha = rho'/<rhat, v>
        const double malpha[2] = {-alpha[0], -alpha[1]};
        if ((rc = lincomb(g, which, sv, ZERO2, 0, r, ONE2, v, malpha, 1, what))) return rc;       // s = r - alpha v
        ++it;
        if ((rc = hirep_spinor_sqnorm(g, which, sv, &ss))) return rc;
        if (!std::isfinite(ss)) return breakdown(g, "%s: ||s||^2 = %g is not finite; x is undefined", what, ss);
        if (ss <= tol * tol * bb) {
            if ((rc = lincomb(g, which, x, ONE2, 1, p, alpha, p, ZERO2, 0, what))) return rc;     // x += alpha p
            rr = ss;
            break;
        }
        if ((rc = apply(t, sv))) return rc;                                                       // t = A s
        if ((rc = reduce_prod(g, which, 0, t, sv, ts, what))) return rc;
        if ((rc = hirep_spinor_sqnorm(g, which, t, &tt))) return rc;
        if (!(tt > 0.0) || !std::isfinite(tt)) return breakdown(g, "%s: breakdown (<t,t> = %g); x is undefined", what, tt);
        if (zero_or_nan(ts)) return breakdown(g, "%s: breakdown (omega = <t,s>/<t,t> = 0 or not finite); x is undefined", what);
        omega[0] = ts[0] / tt; omega[1] = ts[1] / tt;                                             // omega = <t,s>/<t,t>
        if ((rc = lincomb(g, which, x, ONE2, 1, p, alpha, sv, omega, 1, what))) return rc;        // x += alpha p + omega s
        const double momega[2] = {-omega[0], -omega[1]};
        if ((rc = lincomb(g, which, r, ZERO2, 0, sv, ONE2, t, momega, 1, what))) return rc;       // r = s - omega t
        if ((rc = hirep_spinor_sqnorm(g, which, r, &rr))) return rc;
        if (!std::isfinite(rr)) return breakdown(g, "%s: ||r||^2 = %g is not finite; x is undefined", what, rr);
        rho[0] = rho_new[0]; rho[1] = rho_new[1];
    }
    if (iters) *iters = it;
    if (relres) *relres = bb > 0.0 ? sqrt(rr / bb) : 0.0;
    return hirep_sync(g);
}

extern "C" int hirep_cg_g5Dphi_sq(hirep_geom *g, double m0, void *x_full, const void *b_full, const void *links, double tol,
                                  int maxiter, int *iters, double *relres) {
    CHECK_PTRS("hirep_cg_g5Dphi_sq", x_full, b_full, links);
    return cg_solve(g, 1, m0, x_full, b_full, links, tol, maxiter, iters, relres, "hirep_cg_g5Dphi_sq");
}
extern "C" int hirep_cg_g5Dphi_clover_sq(hirep_geom *g, double m0, double csw, void *x_full, const void *b_full, const void *links,
                                         const void *clover, double tol, int maxiter, int *iters, double *relres) {
    CHECK_PTRS("hirep_cg_g5Dphi_clover_sq", x_full, b_full, links, clover);
    return cg_solve(g, 1, m0, x_full, b_full, links, tol, maxiter, iters, relres, "hirep_cg_g5Dphi_clover_sq", 0, 0.0, clover, csw);
}
extern "C" int hirep_cg_Dphi_tm_sq(hirep_geom *g, double m0, double mu, void *x_full, const void *b_full, const void *links, double tol,
                                   int maxiter, int *iters, double *relres) {
    CHECK_PTRS("hirep_cg_Dphi_tm_sq", x_full, b_full, links);
    return cg_solve(g, 1, m0, x_full, b_full, links, tol, maxiter, iters, relres, "hirep_cg_Dphi_tm_sq", 1, mu);
}
extern "C" int hirep_cg_g5Dphi_hat_sq(hirep_geom *g, double m0, void *x_even, const void *b_even, const void *links, double tol,
                                      int maxiter, int *iters, double *relres) {
    CHECK_PTRS("hirep_cg_g5Dphi_hat_sq", x_even, b_even, links);
    return cg_solve(g, 0, m0, x_even, b_even, links, tol, maxiter, iters, relres, "hirep_cg_g5Dphi_hat_sq");
}

// CG on the even-odd preconditioned operator with site-diagonal blocks, A = (gamma_5 D_hat)^2 with D_hat of Eq 43 (L803, L815):
// the clover term (D_ee from the clover field, D_oo^{-1} from hirep_clover_inv_field) or any Hermitian blocks (exponential
// clover: hirep_clover_exp_field and its inverse)
extern "C" int hirep_cg_g5Dphi_clover_hat_sq(hirep_geom *g, double m0, double csw, void *x_even, const void *b_even, const void *links,
                                             const void *clover, const void *inv_odd, double tol, int maxiter, int *iters, double *relres) {
    CHECK_PTRS("hirep_cg_g5Dphi_clover_hat_sq", x_even, b_even, links, clover, inv_odd);
    return cg_solve(g, 0, m0, x_even, b_even, links, tol, maxiter, iters, relres, "hirep_cg_g5Dphi_clover_hat_sq", 0, 0.0, clover, csw, nullptr, inv_odd);
}
extern "C" int hirep_cg_g5Dphi_blocks_sq(hirep_geom *g, void *x_full, const void *b_full, const void *links, const void *blocks_full, double tol,
                                         int maxiter, int *iters, double *relres) {
    CHECK_PTRS("hirep_cg_g5Dphi_blocks_sq", x_full, b_full, links, blocks_full);
    return cg_solve(g, 1, 0.0, x_full, b_full, links, tol, maxiter, iters, relres, "hirep_cg_g5Dphi_blocks_sq", 0, 0.0, nullptr, 0.0, blocks_full, nullptr);
}
extern "C" int hirep_cg_g5Dphi_blocks_hat_sq(hirep_geom *g, void *x_even, const void *b_even, const void *links, const void *blocks_even,
                                             const void *inv_blocks_odd, double tol, int maxiter, int *iters, double *relres) {
    CHECK_PTRS("hirep_cg_g5Dphi_blocks_hat_sq", x_even, b_even, links, blocks_even, inv_blocks_odd);
    return cg_solve(g, 0, 0.0, x_even, b_even, links, tol, maxiter, iters, relres, "hirep_cg_g5Dphi_blocks_hat_sq", 0, 0.0, nullptr, 0.0, blocks_even,
                    inv_blocks_odd);
}

// ---- fermion force of the hopping term (Eq 20-21): SURVEY.md 8(f) NEXT-4 --------------------------------------------
static int force_table(hirep_geom *g) {
    if (g->force_rowptr) return HIREP_OK;
    const int NA = g->N * g->N - 1, d = g->dR;
    const size_t n = (size_t)NA * d * d;
    double2 *dense = nullptr;
    cudaError_t e = cudaMalloc((void **)&dense, n * sizeof(double2));
    if (e != cudaSuccess) { cudaGetLastError(); return fail(HIREP_ENOMEM, "hirep_force_hopping: generator table: %s", cudaGetErrorString(e)); }
    int rc = k_rep_generators(g->N, g->rep, dense, g->stream);
    if (rc) { cudaFree(dense); return kern_result(g, rc, "hirep_force_hopping (generator table)"); }
    std::vector<double2> h(n);
    e = cudaMemcpyAsync(h.data(), dense, n * sizeof(double2), cudaMemcpyDeviceToHost, g->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(g->stream);
    if (e != cudaSuccess) { cudaFree(dense); return cuda_fail(e, "hirep_force_hopping (generator table)"); }
    g->launches += 1;
    std::vector<int> rowptr(NA + 1, 0), jk;
    std::vector<double2> val;
    for (int a = 0; a < NA; ++a) {
        for (int j = 0; j < d; ++j)
            for (int k = 0; k < d; ++k) {
                const double2 v = h[((size_t)a * d + j) * d + k];
                if (fabs(v.x) > 1e-14 || fabs(v.y) > 1e-14) { jk.push_back(j * d + k); val.push_back(v); }
            }
        rowptr[a + 1] = (int)jk.size();
    }
    if (jk.empty()) { jk.push_back(0); val.push_back(make_double2(0, 0)); }   // SU(2) 2AS: the trivial representation has T_R = 0
    void *p0 = nullptr, *p1 = nullptr, *p2 = nullptr;
    e = cudaMalloc(&p0, rowptr.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&p1, jk.size() * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&p2, val.size() * sizeof(double2));
    if (e == cudaSuccess) e = cudaMemcpy(p0, rowptr.data(), rowptr.size() * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(p1, jk.data(), jk.size() * sizeof(int), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(p2, val.data(), val.size() * sizeof(double2), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(p0); cudaFree(p1); cudaFree(p2); cudaFree(dense); cudaGetLastError();
        return fail(HIREP_ENOMEM, "hirep_force_hopping: generator table upload: %s", cudaGetErrorString(e));
    }
    g->force_rowptr = (int *)p0; g->force_jk = (int *)p1; g->force_val = p2; g->force_dense = dense;
    return HIREP_OK;
}
extern "C" int hirep_force_bytes(const hirep_geom *g, size_t *bytes, int *n_generators) {
    if (!g) return fail(HIREP_EINVAL, "hirep_force_bytes: NULL geometry");
    const int NA = g->N * g->N - 1;
    if (bytes) *bytes = (size_t)2 * g->geo.Nh * 4 * NA * (g->prec == HIREP_F64 ? 8 : 4);
    if (n_generators) *n_generators = NA;
    return HIREP_OK;
}
extern "C" int hirep_force_hopping(hirep_geom *g, void *force_canonical, const void *eta_full, const void *xi_full, const void *links_rep) {
    CHECK_PTRS("hirep_force_hopping", force_canonical, eta_full, xi_full, links_rep);
    if (g->mode == HIREP_LINKS_REBUILD && g->rep == HIREP_ADJ)   // `links` is the fundamental field: matrix-free commutator form
        return kern_result(g, k_force_hopping_adj(g->geo, g->prec, g->N, eta_full, xi_full, links_rep, force_canonical, g->stream), "hirep_force_hopping (adjoint, matrix-free)");
    if (g->mode != HIREP_LINKS_STORED) return fail(HIREP_EINVAL, "hirep_force_hopping: needs the stored represented links (HIREP_LINKS_STORED), or the adjoint representation in HIREP_LINKS_REBUILD mode");
    int rc = force_table(g);
    if (rc) return rc;
    return kern_result(g, k_force_hopping(g->geo, g->prec, g->dR, g->real, g->rep == HIREP_FUND, eta_full, xi_full, links_rep, g->force_rowptr, g->force_jk, g->force_val,
                                          g->force_dense, g->N * g->N - 1, force_canonical, g->stream), "hirep_force_hopping");
}

extern "C" int hirep_fma_peak(int prec, double *tflops) {
    if (!tflops) return fail(HIREP_EINVAL, "hirep_fma_peak: NULL result pointer");
    if (prec != HIREP_F64 && prec != HIREP_F32) return fail(HIREP_EINVAL, "hirep_fma_peak: unknown precision %d", prec);
    const int rc = k_fma_peak(prec, tflops, 0);
    if (rc != 0) return cuda_fail((cudaError_t)rc, "hirep_fma_peak");
    return HIREP_OK;
}

extern "C" int hirep_sync(hirep_geom *g) {
    if (!g) return fail(HIREP_EINVAL, "hirep_sync: NULL geometry");
    cudaError_t e = cudaStreamSynchronize(g->stream);
    if (e == cudaSuccess && g->host_events) e = cudaStreamSynchronize(g->copy_stream);
    if (e != cudaSuccess) return cuda_fail(e, "hirep_sync");
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "hirep_sync (deferred)");
    if (g->dev_flags) {   // numerical breakdowns reported by kernels since the last sync
        int fl = 0;
        e = cudaMemcpy(&fl, g->dev_flags, sizeof(int), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return cuda_fail(e, "hirep_sync (flags)");
        if (fl) {
            cudaMemset(g->dev_flags, 0, sizeof(int));
            return fail(HIREP_EBREAKDOWN, "hirep_sync: %s%s%s", (fl & 1) ? "hirep_clover_inv_field met a vanishing or non-finite pivot (block not positive definite: c_sw |A| against 4+m0)" : "",
                        (fl & 3) == 3 ? "; " : "", (fl & 2) ? "hirep_clover_exp_field: |c_sw/(4+m0) A| > 8 at some site, outside the range of the exponential series" : "");
        }
    }
    return HIREP_OK;
}

// ---- end-to-end host entry -------------------------------------------------------------------------
static int apply_host_impl(hirep_geom *g, int op, double m0, void *out_host, const void *in_host, const void *links_fund_host, bool async) {
    if (!g || !out_host || !in_host) return fail(HIREP_EINVAL, "hirep_apply_host: NULL argument");
    if (op < HIREP_OP_DPHI || op > HIREP_OP_G5DPHI_SQ) return fail(HIREP_EINVAL, "hirep_apply_host: unknown op %d", op);
    const bool full = (op == HIREP_OP_DPHI || op == HIREP_OP_G5DPHI_SQ);
    const size_t w = g->prec == HIREP_F64 ? 8 : 4;
    const size_t V = (size_t)2 * g->geo.Nh;
    const size_t canon_links = V * 4 * g->N * g->N * 2 * w;
    const size_t canon_sp = (full ? V : V / 2) * 4 * g->dR * 2 * w;
    const size_t native_sp = (full ? 2 : 1) * g->bytes_spinor_half;
    if (!links_fund_host && !g->host_links_ready) return fail(HIREP_EINVAL, "hirep_apply_host: no links given and none resident");
    int rc;
    if ((rc = workspace(&g->h_links_rep, g->bytes_links_rep))) return rc;
    if ((rc = workspace(&g->h_in_canon, V * 4 * g->dR * 2 * w))) return rc;
    if ((rc = workspace(&g->h_out_canon, V * 4 * g->dR * 2 * w))) return rc;
    if ((rc = workspace(&g->h_out_canon2, V * 4 * g->dR * 2 * w))) return rc;
    if (!g->host_events) {
        cudaError_t ce = cudaStreamCreateWithFlags(&g->copy_stream, cudaStreamNonBlocking);
        for (int i = 0; i < 2 && ce == cudaSuccess; ++i) {
            ce = cudaEventCreateWithFlags(&g->ev_done[i], cudaEventDisableTiming);
            if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&g->ev_copied[i], cudaEventDisableTiming);
            if (ce == cudaSuccess) ce = cudaEventRecord(g->ev_copied[i], g->copy_stream);   // "slot free"
        }
        if (ce != cudaSuccess) return cuda_fail(ce, "hirep_apply_host: stream/event setup");
        g->host_events = 1;
    }
    if ((rc = workspace(&g->h_in_native, 2 * g->bytes_spinor_half))) return rc;
    if ((rc = workspace(&g->h_out_native, 2 * g->bytes_spinor_half))) return rc;
    cudaError_t e;
    if (links_fund_host) {
        if ((rc = workspace(&g->h_links_canon, canon_links))) return rc;
        if ((rc = workspace(&g->h_links_fund, g->bytes_links_fund))) return rc;
        e = cudaMemcpyAsync(g->h_links_canon, links_fund_host, canon_links, cudaMemcpyHostToDevice, g->stream);
        if (e != cudaSuccess) return cuda_fail(e, "hirep_apply_host: links H2D");
        if ((rc = hirep_links_import(g, g->h_links_fund, g->h_links_canon))) return rc;
        if ((rc = hirep_links_to_rep(g, g->h_links_rep, g->h_links_fund))) return rc;
        g->host_links_ready = 1;
    }
    e = cudaMemcpyAsync(g->h_in_canon, in_host, canon_sp, cudaMemcpyHostToDevice, g->stream);
    if (e != cudaSuccess) return cuda_fail(e, "hirep_apply_host: spinor H2D");
    const int in_which = full ? HIREP_FULL : (op == HIREP_OP_DPHI_EO ? HIREP_ODD : HIREP_EVEN);
    const int out_which = full ? HIREP_FULL : (op == HIREP_OP_DPHI_OE ? HIREP_ODD : HIREP_EVEN);
    if ((rc = hirep_spinor_import(g, g->h_in_native, g->h_in_canon, in_which))) return rc;
    const void *links = g->mode == HIREP_LINKS_STORED ? g->h_links_rep : g->h_links_fund;
    switch (op) {
    case HIREP_OP_DPHI: rc = hirep_Dphi(g, m0, g->h_out_native, g->h_in_native, links); break;
    case HIREP_OP_DPHI_EO: rc = hirep_Dphi_eo(g, g->h_out_native, g->h_in_native, links); break;
    case HIREP_OP_DPHI_OE: rc = hirep_Dphi_oe(g, g->h_out_native, g->h_in_native, links); break;
    case HIREP_OP_DPHI_HAT: rc = hirep_Dphi_hat(g, m0, g->h_out_native, g->h_in_native, links); break;
    default: rc = hirep_g5Dphi_sq(g, m0, g->h_out_native, g->h_in_native, links); break;
    }
    if (rc) return rc;
    // the result goes home on a second stream from one of two staging buffers, so that the device -> host copy of this
    // call overlaps the host -> device copy and the kernels of the next one (PCIe is full duplex)
    const int slot = g->host_slot;
    g->host_slot ^= 1;
    void *stage = slot ? g->h_out_canon2 : g->h_out_canon;
    e = cudaStreamWaitEvent(g->stream, g->ev_copied[slot], 0);          // the buffer's previous copy has left
    if (e != cudaSuccess) return cuda_fail(e, "hirep_apply_host: wait for staging buffer");
    if ((rc = hirep_spinor_export(g, stage, g->h_out_native, out_which))) return rc;
    e = cudaEventRecord(g->ev_done[slot], g->stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(g->copy_stream, g->ev_done[slot], 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out_host, stage, canon_sp, cudaMemcpyDeviceToHost, g->copy_stream);
    if (e == cudaSuccess) e = cudaEventRecord(g->ev_copied[slot], g->copy_stream);
    if (e != cudaSuccess) return cuda_fail(e, "hirep_apply_host: result D2H");
    (void)native_sp;
    if (async) return HIREP_OK;
    return hirep_sync(g);
}

extern "C" int hirep_apply_host(hirep_geom *g, int op, double m0, void *out_host, const void *in_host, const void *links_fund_host) {
    return apply_host_impl(g, op, m0, out_host, in_host, links_fund_host, false);
}
extern "C" int hirep_apply_host_async(hirep_geom *g, int op, double m0, void *out_host, const void *in_host, const void *links_fund_host) {
    return apply_host_impl(g, op, m0, out_host, in_host, links_fund_host, true);
}
