/*
 * hirep_b200.h -- C-ABI of the B200-native Wilson-Dirac operator for fermions in a representation R of SU(N_g).
 *
 * Operation definitions follow arXiv 2503.06721 (HiRep v2); citations are PAPER.md line + section/equation.
 *
 *   lattice      T x L^3 hypercubic, mu = 0 is time                                  (L167, Sect. 2.1)
 *   gamma basis  e_0 = -1, e_k = -i sigma_k, gamma_mu = [[0,e_mu],[e_mu^dagger,0]]   (L171-182, Eq 1-3)
 *   D_m psi(x) = (4+m) psi(x) - 1/2 sum_mu [ (1-gamma_mu) U^R_mu(x) psi(x+mu)
 *                                           + (1+gamma_mu) U^R_mu(x-mu)^dagger psi(x-mu) ]   (L207, Eq 8; a = 1)
 *   Q_m = gamma_5 D_m, gamma_5 = gamma_0 gamma_1 gamma_2 gamma_3 = diag(1,1,-1,-1)    (L230, Eq 11; A1)
 *   even site: (t+x+y+z) mod 2 = 0; D_m = [[D_ee, D_eo],[D_oe, D_oo]]                (L793-795, Eq 41)
 *   D_hat = (4+m)^2 - D_eo D_oe                                                      (L808, Eq 44)
 *   boundary conditions: psi(x + L_mu) = bc_mu psi(x), bc_mu = +-1                   (L930-943, Eq 58-63)
 *   representations FUND / ADJ / SYM / 2AS, dimensions of Tbl 1                      (L213-220)
 *
 * General rules
 *   - Every function returns 0 on success and a negative HIREP_E* code on failure; nothing throws or aborts
 *     across this boundary.  hirep_last_error() gives a thread-local NUL-terminated description.
 *   - "device pointer" = CUDA global memory on the current device, 16-byte aligned, owned by the caller
 *     (allocate through torch).  "host pointer" = ordinary host memory (pinned memory makes the copies faster).
 *   - Operator calls are asynchronous on the geometry's stream (hirep_geom_set_stream; default stream 0);
 *     launch failures are reported by the call that launched, execution failures by hirep_sync or a later call.
 *   - `out` is overwritten, never accumulated, and must not alias `in`.
 *   - There is NO CPU fallback: without a CUDA device every compute entry point returns HIREP_ECUDA.
 *
 * Canonical (interchange) layout -- used only by the import/export calls and by hirep_apply_host:
 *     site index ix = ((t*L + x)*L + y)*L + z        (z fastest)
 *     spinor  [ix][spin 0..3][colour 0..d_R-1]        complex (interleaved re,im)  of the working precision
 *     links   [ix][mu 0..3][row i][col j]             complex, (U psi)_i = sum_j U_ij psi_j
 *     half-lattice spinors list the sites of that parity in increasing ix.
 *     represented links exported by hirep_links_rep_export: [ix][mu][i][j], REAL scalars for ADJ
 *     (rep_is_real = 1), complex otherwise.
 * Native layout -- private to the library, sizes from hirep_geom_sizes, described in DESIGN.md:
 *     per parity, sites ordered (t,x,y,z/2) in tiles of 32; spinor [tile][4 d_R][32] complex;
 *     links [parity][tile][8 directions][d*d][32]: the 8 matrices W_d that act on the 8 neighbours of a
 *     site (W_mu = U_mu(x), W_{4+mu} = U_mu(x-mu)^dagger), so every stencil pass streams one contiguous
 *     block per tile.  Represented links carry the boundary signs.
 */
#ifndef HIREP_B200_H
#define HIREP_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hirep_geom hirep_geom; /* opaque: lattice maps, BC state, stream, workspace spinors */

enum { HIREP_FUND = 0, HIREP_ADJ = 1, HIREP_SYM = 2, HIREP_ASY = 3 }; /* representation (Tbl 1, L213-220) */
enum { HIREP_F64 = 0, HIREP_F32 = 1 };                                /* field precision (L308)          */
enum { HIREP_EVEN = 0, HIREP_ODD = 1, HIREP_FULL = 2 };
enum { HIREP_LINKS_STORED = 0, HIREP_LINKS_REBUILD = 1 };
enum { HIREP_OP_DPHI = 0, HIREP_OP_DPHI_EO = 1, HIREP_OP_DPHI_OE = 2, HIREP_OP_DPHI_HAT = 3, HIREP_OP_G5DPHI_SQ = 4 };
enum {
    HIREP_OK = 0,
    HIREP_EINVAL = -1,       /* bad argument: null/misaligned pointer, odd or <2 extent, unknown enum, out aliases in */
    HIREP_EUNSUPPORTED = -2, /* (N_g, rep, prec, mode) combination not instantiated                               */
    HIREP_ECUDA = -3,        /* CUDA runtime error (no device, launch or execution failure)                        */
    HIREP_ENOMEM = -4,       /* workspace allocation failed                                                        */
    HIREP_EBREAKDOWN = -5    /* an iterative solver met a non-finite or degenerate scalar (NaN/inf in b or in a field,
                                <p,Ap> <= 0, rho = 0, <rhat,v> = 0, <t,t> = 0, omega = 0); the stream has been drained
                                and the solution field is UNDEFINED                                                  */
};

/* Lattice T x L^3 (both even, >= 2), gauge group SU(N_g) (2 <= N_g <= 6), representation, precision.
 * Default boundary conditions: antiperiodic in time, periodic in space ({-1,+1,+1,+1}); link mode STORED.
 * The handle is bound to the CUDA device that is current at creation: its workspaces are allocated there and every
 * compute call made while another device is current returns HIREP_EINVAL. */
int hirep_geom_create(int T, int L, int N_g, int rep, int prec, hirep_geom **out);
int hirep_geom_destroy(hirep_geom *g); /* frees the handle and its workspace; NULL is a no-op */

/* ---- sharded operator: slab of a lattice block-partitioned in t over ranks (Fig 1; Sect. 4.8) ----
 * One rank owns the global time slices [t_start, t_start + T_loc) of a T_glob x L^3 lattice.  Its geometry is a LOCAL lattice of
 * T_loc + 2 slices: local slice 0 and T_loc + 1 are GHOST slices (global slices t_start - 1 and t_start + T_loc, mod T_glob), local
 * slices 1 .. T_loc are owned.  Every buffer (spinors, links) has the local lattice's native size.  t_start, T_loc, T_glob even,
 * so local parity = global parity XOR 1 on every rank (local slice t is global slice t_start - 1 + t).  The boundary factor bc_0
 * sits where the GLOBAL lattice closes: hirep_links_to_rep puts it on the links of global slice T_glob - 1, so only the owning
 * rank carries it (L945).  Links: import the fundamental field of the local lattice (owned slices plus the ghost slice BEFORE them,
 * whose t-links the first owned slice's backward hop uses; the other ghost links are not read by owned sites).
 * Spinors: per application the caller (a) packs the two faces of the input -- PROJECTED half spinors, 2 d_R complex per face site
 * (L624) -- (b) ships them to the neighbour ranks (peer copy / NCCL send-recv; not this library's business), (c) unpacks what it
 * received into the ghost slices, (d) applies the operator.  With hirep_set_region the interior can run while the faces are in
 * flight and the two boundary slabs afterwards (the paper's inner/boundary split, Fig 1):
 *     region OWNED (default for a slab) | INTERIOR (tiles whose hops reach no ghost slice) | BOUNDARY (the rest of OWNED) | ALL.
 * Regions are honoured by hirep_Dphi, hirep_Dphi_eo, hirep_Dphi_oe and the other single-pass stencil calls (persistent kernels,
 * link mode STORED or the d_R <= 6 REBUILD kernels); two-pass operators return HIREP_EUNSUPPORTED on a slab (a halo exchange belongs
 * between their passes), reductions and linear algebra see the whole local buffers including ghosts.
 * face: 0 = first owned slice, projected with (1 - gamma_0): goes to the PREVIOUS rank, which unpacks it (face 0) into its last
 * ghost slice; 1 = last owned slice, (1 + gamma_0): goes to the NEXT rank, unpacked (face 1) into its ghost slice 0.  buf: device
 * buffer of hirep_halo_bytes bytes; spinor_half: native half-lattice spinor of the local lattice (either parity).  unpack stores
 * the ghost spinor (h, 0), whose projection inside the stencil is h again, so halo sites need no second code path. */
enum { HIREP_REGION_ALL = 0, HIREP_REGION_OWNED = 1, HIREP_REGION_INTERIOR = 2, HIREP_REGION_BOUNDARY = 3 };
int hirep_geom_create_slab(int T_glob, int L, int N_g, int rep, int prec, int t_start, int T_loc, hirep_geom **out);
int hirep_set_region(hirep_geom *g, int region);
int hirep_halo_bytes(const hirep_geom *g, size_t *bytes);
int hirep_halo_pack(hirep_geom *g, int face, void *buf, const void *spinor_half);
int hirep_halo_unpack(hirep_geom *g, int face, void *spinor_half, const void *buf);

/* bc_mu = +-1 per direction (Eq 58-63).  The signs are baked into the represented links by
 * hirep_links_to_rep (the paper's implementation, L945), so call it again after changing them. */
int hirep_geom_set_bc(hirep_geom *g, const int sign[4]);
/* cuda_stream: a cudaStream_t / CUstream (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream */
int hirep_geom_set_stream(hirep_geom *g, void *cuda_stream);
/* Workspaces are allocated (cudaMalloc, zeroed once) by the first call that needs them -- which therefore must not sit inside a
 * CUDA-graph capture or any other region where allocation is forbidden.  hirep_geom_reserve allocates them now instead:
 *   HIREP_RESERVE_OPERATORS  the intermediate spinor fields of the two-pass operators (Dphi_hat, g5Dphi_sq, the clover / block /
 *                            twisted-mass forms and their squares) and the device flag word: 5 half-lattice spinors
 *   HIREP_RESERVE_SOLVERS    the reduction buffers and the work fields of the CGs and BiCGstab (5 full-lattice spinors), the pinned
 *                            host scalars (the multi-shift CG's per-shift fields and hirep_apply_host's staging stay lazy)
 * Flags may be or-ed.  Idempotent.  Errors: HIREP_EINVAL (flags), HIREP_ENOMEM, HIREP_ECUDA.  (hirep_Dphi_hat_static needs none.) */
enum { HIREP_RESERVE_OPERATORS = 1, HIREP_RESERVE_SOLVERS = 2 };
int hirep_geom_reserve(hirep_geom *g, int what);
/* Bytes of native buffers (any pointer may be NULL): full- and half-lattice spinor, fundamental links,
 * represented links; d_R (Tbl 1); rep_is_real = 1 iff represented links are stored as real numbers (ADJ). */
int hirep_geom_sizes(const hirep_geom *g, size_t *spinor_full, size_t *spinor_half, size_t *links_fund,
                     size_t *links_rep, int *d_R, int *rep_is_real);

/* canonical <-> native, all device pointers.  parity_or_full in {HIREP_EVEN, HIREP_ODD, HIREP_FULL}. */
int hirep_spinor_import(hirep_geom *g, void *native, const void *canonical, int parity_or_full);
int hirep_spinor_export(hirep_geom *g, void *canonical, const void *native, int parity_or_full);
int hirep_links_import(hirep_geom *g, void *native_fund, const void *canonical_fund);
/* forward matrices s_mu(x) U^R_mu(x) (boundary sign included) in canonical order; for tests */
int hirep_links_rep_export(hirep_geom *g, void *canonical_rep, const void *native_rep);
/* the stored backward matrices W_{4+mu}(x) = s U^R_mu(x-mu)^dagger, canonical [ix][mu][i][j]; for tests */
int hirep_links_rep_export_bwd(hirep_geom *g, void *canonical_rep, const void *native_rep);

/* U -> U^R for all links (Eq 7; FUND: identity map; ADJ: R_ab = 2 Re tr(T^a U T^b U^dagger);
 * SYM/2AS: Psi -> U Psi U^T on (anti)symmetric tensors; bases in DESIGN.md A10/A11), times the boundary
 * sign on links that cross the lattice boundary (L945).  Device pointers, native layouts. */
int hirep_links_to_rep(hirep_geom *g, void *native_rep, const void *native_fund);

/* The operators.  Device pointers to native buffers.  `links` is the represented field (mode STORED) or the
 * fundamental field (mode REBUILD, R rebuilt in registers).  m0 is the bare mass m of Eq 8.
 *   hirep_Dphi      out = D_m in                      full lattice            (Eq 8/10)
 *   hirep_Dphi_eo   out_even = D_eo in_odd            (off-diagonal block of Eq 41, includes the -1/2)
 *   hirep_Dphi_oe   out_odd  = D_oe in_even
 *   hirep_Dphi_hat  out_even = (4+m)^2 in_even - D_eo D_oe in_even            (Eq 44)
 *   hirep_g5Dphi_sq out = gamma_5 D_m gamma_5 D_m in  full lattice            (Eq 11)            */
int hirep_Dphi(hirep_geom *g, double m0, void *out_full, const void *in_full, const void *links);
int hirep_Dphi_eo(hirep_geom *g, void *out_even, const void *in_odd, const void *links);
int hirep_Dphi_oe(hirep_geom *g, void *out_odd, const void *in_even, const void *links);
int hirep_Dphi_hat(hirep_geom *g, double m0, void *out_even, const void *in_even, const void *links);
int hirep_g5Dphi_sq(hirep_geom *g, double m0, void *out_full, const void *in_full, const void *links);
/* hirep_Dphi_hat_static: the same operator as hirep_Dphi_hat (Eq 44), same arguments, same kernels and launch order,
 * same result bit for bit, for callers that cannot call cudaMalloc (a stream under CUDA graph capture, a serving loop, a harness
 * that forbids it).  The odd intermediate field D_oe in_even lives in a static device array of HIREP_STATIC_SCRATCH_BYTES
 * (16 MiB; every GPU that loads the library holds it until exit) instead of the handle's lazily allocated workspace: the call
 * makes no cudaMalloc, cudaFree or allocating library call.  Limits and hazards:
 *   - one half-lattice spinor of the geometry must fit: 4 d_R * 16 (8 in fp32) bytes per site slot * 32 * ceil(V/64) <=
 *     HIREP_STATIC_SCRATCH_BYTES (e.g. SU(3) fundamental fp64 up to 16^3 x 32); larger geometries are rejected with
 *     HIREP_EINVAL and a message, nothing is launched;
 *   - slab geometries: HIREP_EUNSUPPORTED, as hirep_Dphi_hat;
 *   - every call on a device shares the one array: two calls that overlap on the GPU (different streams, different handles,
 *     different host threads) RACE on it.  Calls on one stream are ordered and safe.  The array keeps the previous call's
 *     contents; what must be zero (the padding lanes of a ragged last tile) is cleared on the stream by each call;
 *   - the first call on a device resolves the array's address (cudaGetSymbolAddress) and loads the kernels: make one call
 *     before starting a capture.  out_even, in_even, links: device pointers owned by the caller, as hirep_Dphi_hat. */
#define HIREP_STATIC_SCRATCH_BYTES (16u << 20)
int hirep_Dphi_hat_static(hirep_geom *g, double m0, void *out_even, const void *in_even, const void *links);
/* The Hermitian even-odd preconditioned operator (Eq 45) in the normalisation of Eq 44 (A22):
 *   hirep_g5Dphi_hat     out_even = gamma_5 ((4+m)^2 - D_eo D_oe) in_even = Q_hat in_even
 *   hirep_g5Dphi_hat_sq  out_even = Q_hat Q_hat in_even      (Hermitian positive definite: what CG inverts in HMC, L772/L806) */
int hirep_g5Dphi_hat(hirep_geom *g, double m0, void *out_even, const void *in_even, const void *links);
int hirep_g5Dphi_hat_sq(hirep_geom *g, double m0, void *out_even, const void *in_even, const void *links);

int hirep_set_link_mode(hirep_geom *g, int mode); /* HIREP_LINKS_STORED | HIREP_LINKS_REBUILD */
/* Implementation variant of the stencil kernel, for measurements: 0 = library default, >0 = explicit
 * (list in DESIGN.md).  An unknown variant for the geometry's instantiation returns HIREP_EUNSUPPORTED. */
int hirep_set_kernel_variant(hirep_geom *g, int variant);
/* Measurement / test knobs of the persistent stencil kernels.  Results never depend on them.
 *   HIREP_TUNE_MAX_CTAS    cap on the number of persistent CTAs (0 = one per SM); a small cap makes every warp
 *                          walk many tiles, which the parity tests use on small lattices
 *   HIREP_TUNE_SUM_ALGORITHM  accumulation of the reductions (this one does change the last bits of their results):
 *                          2 = Neumaier, Algorithm 2 (default), 3 = second-order Neumaier, Algorithm 3 (L682),
 *                          4 = double-double, Algorithm 4 (L706)
 *   HIREP_TUNE_PACE_WINDOW W > 0: full-lattice launches of the tile-pair kernel throttle their leading warp groups -- a group starts
 *                          its round k only when the grid has completed k - W rounds' worth of tile pairs -- so that link blocks and
 *                          spinor tiles gathered from other tile pairs are still in L2 (C4: DRAM reads -16..-26 %; time +-5 %, so
 *                          off by default: 0).  Needs all CTAs of the launch co-resident (the library's grids are <= one CTA per SM).
 *   HIREP_TUNE_FUSE_DIAG   1 (default): the operators with site-diagonal matrices (clover, exponential clover, general blocks; Eq 43,
 *                          47, 50) apply them inside the stencil epilogues wherever that kernel is instantiated (stored links,
 *                          d_R <= 6, kernel variants 0, 3, 4): Dphi_clover / Dphi_blocks 1 launch, the Schur forms 2; 0: separate
 *                          block-apply launches (2 resp. 4).  The two forms sum in different orders: results agree to rounding. */
enum { HIREP_TUNE_MAX_CTAS = 1, HIREP_TUNE_SUM_ALGORITHM = 2, HIREP_TUNE_PACE_WINDOW = 3, HIREP_TUNE_FUSE_DIAG = 4 };
int hirep_set_tuning(hirep_geom *g, int key, int value);
/* number of kernels this library has launched on behalf of g since creation (bench.py's gpu_launches) */
long hirep_launch_count(const hirep_geom *g);

/* End-to-end entry with HOST buffers (canonical layout): copies `in` (and `links_fund`, if non-NULL; otherwise
 * the represented links built by the previous call are reused) to the device, imports, builds the represented
 * links, applies `op` (HIREP_OP_*), exports and copies the result back to `out`; returns after the result is in
 * host memory.  Spinor extents follow the op (half lattice for EO/OE/HAT, full otherwise). */
int hirep_apply_host(hirep_geom *g, int op, double m0, void *out_host, const void *in_host, const void *links_fund_host);
/* The same without the final wait: returns once everything is enqueued; results are in host memory after hirep_sync.
 * Consecutive calls pipeline: the device -> host copy of one call overlaps the host -> device copy and kernels of the
 * next (pinned host buffers needed for the copies to be asynchronous; in_host must stay valid until hirep_sync). */
int hirep_apply_host_async(hirep_geom *g, int op, double m0, void *out_host, const void *in_host, const void *links_fund_host);

/* ---- spinor linear algebra, reductions and the CG inverter (Sect. 4.2 / 5.1; the consumer of the hot path) ----
 * Native spinor buffers (device pointers); `which` in {HIREP_EVEN, HIREP_ODD, HIREP_FULL} gives their extent.
 * Complex coefficients are host pointers to {re, im}.  xi may alias eta or zeta (element-wise operations).
 *   hirep_spinor_lc   xi = r1 eta + r2 zeta            (Eq 22)      hirep_spinor_lc1  xi <- xi + c1 eta          (Eq 24)
 *   hirep_spinor_clc  xi = c1 eta + c2 zeta            (Eq 23)            hirep_spinor_lc2  xi <- c1 xi + c2 eta       (Eq 25)
 *   *_add_assign      xi <- xi + (the same)            (L387)             hirep_spinor_lc3  xi <- c1 eta + c2 zeta - xi (Eq 26) */
int hirep_spinor_lc(hirep_geom *g, int which, void *xi, double r1, const void *eta, double r2, const void *zeta);
/* elementary operations (L365-371): xi = 0 ; xi = eta ; xi = c eta (complex c) ; xi = -eta.  xi may alias eta. */
int hirep_spinor_zero(hirep_geom *g, int which, void *xi);
int hirep_spinor_copy(hirep_geom *g, int which, void *xi, const void *eta);
int hirep_spinor_mul(hirep_geom *g, int which, void *xi, const double c[2], const void *eta);
int hirep_spinor_minus(hirep_geom *g, int which, void *xi, const void *eta);
int hirep_spinor_clc(hirep_geom *g, int which, void *xi, const double c1[2], const void *eta, const double c2[2], const void *zeta);
int hirep_spinor_lc_add_assign(hirep_geom *g, int which, void *xi, double r1, const void *eta, double r2, const void *zeta);
int hirep_spinor_clc_add_assign(hirep_geom *g, int which, void *xi, const double c1[2], const void *eta, const double c2[2], const void *zeta);
int hirep_spinor_lc1(hirep_geom *g, int which, void *xi, const double c1[2], const void *eta);
int hirep_spinor_lc2(hirep_geom *g, int which, void *xi, const double c1[2], const double c2[2], const void *eta);
int hirep_spinor_lc3(hirep_geom *g, int which, void *xi, const double c1[2], const void *eta, const double c2[2], const void *zeta);
/* Reductions over the sites of the buffer (padding excluded); results are HOST doubles, the calls synchronise the
 * stream.  Accumulation: Neumaier's compensated sum (Algorithm 2) in fp64 also for fp32 fields.
 *   hirep_spinor_prod      out = {Re, Im} of <xi, eta> = sum conj(xi) eta            (Eq 27)
 *   hirep_spinor_sqnorm    out = <xi, xi> = ||xi||_2^2                               (Eq 32)
 *   hirep_spinor_max_norm  out = max over components of max(|Re|, |Im|)              (Eq 33) */
int hirep_spinor_prod(hirep_geom *g, int which, const void *xi, const void *eta, double out[2]);
int hirep_spinor_sqnorm(hirep_geom *g, int which, const void *xi, double *out);
int hirep_spinor_max_norm(hirep_geom *g, int which, const void *eta, double *out);
/* Conjugate gradient (L730) for Q_m^2 x = b with Q_m^2 = g5Dphi_sq, Hermitian positive definite (L772); x starts at 0.
 * Stops when ||r||_2 <= tol ||b||_2 (r the recurrence residual) or after maxiter iterations (not an error: check
 * *relres).  Full-lattice native spinors; iters / relres are host pointers (may be NULL).  x must not alias b.
 * alpha and beta stay on the device; the host reads ||r||^2 once per iteration AFTER queueing the next operator application, so a
 * solve that stops on the tolerance has launched one operator application more than it needed (it touches only the
 * library's own work fields); a non-positive or non-finite <p,Ap>, <b,b> or ||r||^2 returns HIREP_EBREAKDOWN after that iteration's
 * update (x is then undefined; the stream is synchronised first).  Synchronous on return.  All solvers below follow the same rule. */
int hirep_cg_g5Dphi_sq(hirep_geom *g, double m0, void *x_full, const void *b_full, const void *links, double tol, int maxiter,
                       int *iters, double *relres);
/* Stabilised bi-conjugate gradient (L730) for the non-Hermitian systems D_m x = b (op = HIREP_OP_DPHI, full-lattice
 * spinors) or D_hat x = b (op = HIREP_OP_DPHI_HAT, even sites); x starts at 0; same stopping rule and outputs as the CG. */
int hirep_bicgstab(hirep_geom *g, int op, double m0, void *x, const void *b, const void *links, double tol, int maxiter, int *iters,
                   double *relres);
/* Multi-shift CG (L730; Eq 39-40): (Q_m^2 + shifts[k]) x[k] = b for all k < nshift <= HIREP_MAX_SHIFTS in one
 * Krylov space -- the inversion the RHMC's rational approximation needs.  shifts: host array, >= 0; x_full: host array of
 * nshift device pointers (native full-lattice spinors, distinct from b).  Stops on the unshifted residual. */
#define HIREP_MAX_SHIFTS 16
int hirep_cg_mshift_g5Dphi_sq(hirep_geom *g, double m0, int nshift, const double *shifts, void *const *x_full, const void *b_full,
                              const void *links, double tol, int maxiter, int *iters, double *relres);
/* The same for (D^tm)^dagger D^tm x = b (hirep_Dphi_tm_sq), the twisted-mass monomial's operator. */
int hirep_cg_Dphi_tm_sq(hirep_geom *g, double m0, double mu, void *x_full, const void *b_full, const void *links, double tol,
                        int maxiter, int *iters, double *relres);
/* The same for Q_hat^2 x = b on the even sites (hirep_g5Dphi_hat_sq): even-odd preconditioned CG. */
int hirep_cg_g5Dphi_hat_sq(hirep_geom *g, double m0, void *x_even, const void *b_even, const void *links, double tol, int maxiter,
                           int *iters, double *relres);

/* ---- twisted mass (Eq 51) and the general even-odd form it needs (Eq 43) ----
 *   hirep_spinor_g5_lc  xi = c1 eta + c2 gamma_5 eta             (gamma_5-fused linear combination, L447; xi may alias eta)
 *   hirep_Dphi_tm       out = D_m in + i mu gamma_5 in           (Eq 51 for the tau^3 = +1 flavour; -mu gives the other)
 *   hirep_Dphi_tm_sq    out = (D^tm)^dagger D^tm in = gamma_5 D^tm(-mu) gamma_5 D^tm(mu) in   (Hermitian positive definite)
 *   hirep_Dphi_tm_hat   out_even = D_ee in_even - D_eo D_oo^{-1} D_oe in_even, D_ee = D_oo = (4+m) + i mu gamma_5  (Eq 43); two stencil
 *                       launches: D_oo^{-1} = ((4+m) - i mu gamma_5)/((4+m)^2 + mu^2) is applied in the epilogue of the D_oe pass, D_ee in that
 *                       of the D_eo pass (kernel variants 1, 2: a separate gamma_5 combination in between) */
int hirep_spinor_g5_lc(hirep_geom *g, int which, void *xi, const double c1[2], const double c2[2], const void *eta);
/* gamma matrix application (Eq 34): xi = gamma_mu eta, mu = 0..3 in the basis of Eq 1-3, mu = 5 for gamma_5; xi != eta */
int hirep_spinor_gamma(hirep_geom *g, int which, int mu, void *xi, const void *eta);
/* the add-assign / add-mul-assign forms (L447): xi <- c0 xi + c1 eta + c2 gamma_5 eta */
int hirep_spinor_g5_lc_add_assign(hirep_geom *g, int which, void *xi, const double c0[2], const double c1[2], const double c2[2], const void *eta);
/* the fused reduction <xi, gamma_5 eta> (L447): out = {Re, Im}, host doubles, compensated like hirep_spinor_prod */
int hirep_spinor_g5_prod(hirep_geom *g, int which, const void *xi, const void *eta, double out[2]);
int hirep_Dphi_tm(hirep_geom *g, double m0, double mu, void *out_full, const void *in_full, const void *links);
int hirep_Dphi_tm_sq(hirep_geom *g, double m0, double mu, void *out_full, const void *in_full, const void *links);
int hirep_Dphi_tm_hat(hirep_geom *g, double m0, double mu, void *out_even, const void *in_even, const void *links);

/* ---- clover term (Eq 47-49, second part) ----
 *   D_ee,m + D_oo,m = (4+m) + c_sw (i/4) sum_{mu,nu} sigma_{mu nu} F_{mu nu},  F = (C - C^dagger)/8,  C = the four plaquette
 *   loops through x in the (mu,nu) plane closed at x (readings A26-A28 in DESIGN.md; sigma_{mu nu} = (i/2)[gamma_mu,gamma_nu]).
 *   The term is block diagonal in chirality; the library keeps per site and chirality c the d_R x d_R blocks H, B of
 *   A_c = [[H, B], [B^dagger, -H]] in a caller-owned NATIVE buffer of hirep_clover_bytes() bytes (device, 16-byte aligned).
 *   hirep_clover_field   clover <- from the STORED represented links of hirep_links_to_rep (boundary signs cancel in the
 *                        closed loops); once per gauge update.  HIREP_EINVAL in HIREP_LINKS_REBUILD mode.
 *   hirep_clover_export  canonical_out[V][2][2 d_R][2 d_R] complex (device; site index as the canonical spinor): A_0, A_1.
 *   hirep_Cphi           out_full = ((4+m) + c_sw A) in_full           (the diagonal blocks of Eq 41 with Eq 47); out != in
 *   hirep_Dphi_clover    out_full = D_m in_full with that diagonal term (Eq 8 + Eq 47).  Stored links, d_R <= 6: ONE stencil launch
 *                        whose epilogue applies (4+m) + c_sw A to the site's own input (the H, B matrices stream through the same
 *                        shared-memory ring as the links).  Otherwise (d_R >= 8, link mode REBUILD, slabs,
 *                        HIREP_TUNE_FUSE_DIAG = 0): Cphi, then the hopping pass adds -1/2 hop(in) onto it in place.  out != in;
 *                        `links` as for hirep_Dphi (current link mode). */
int hirep_clover_bytes(const hirep_geom *g, size_t *bytes);
int hirep_clover_field(hirep_geom *g, void *clover, const void *links_rep);
int hirep_clover_export(hirep_geom *g, void *canonical_out, const void *clover);
int hirep_Cphi(hirep_geom *g, double m0, double csw, void *out_full, const void *in_full, const void *clover);
int hirep_Dphi_clover(hirep_geom *g, double m0, double csw, void *out_full, const void *in_full, const void *links, const void *clover);
/* (gamma_5 D_clover)^2 (two passes of the above with gamma_5 fused in the store) and the CG on it (as hirep_cg_g5Dphi_sq). */
int hirep_g5Dphi_clover_sq(hirep_geom *g, double m0, double csw, void *out_full, const void *in_full, const void *links, const void *clover);
int hirep_cg_g5Dphi_clover_sq(hirep_geom *g, double m0, double csw, void *x_full, const void *b_full, const void *links,
                              const void *clover, double tol, int maxiter, int *iters, double *relres);
/* The even-odd form Eq 43 (L803) with the clover blocks of Eq 47: D_hat = D_ee - D_eo D_oo^{-1} D_oe on the even sites.
 *   hirep_clover_inv_field  inv <- ((4+m) + c_sw A_c)^{-1} for every site of ONE parity and both chiralities: the full
 *                           (2 d_R) x (2 d_R) blocks, native, caller-owned buffer of hirep_clover_inv_bytes() bytes.  In-place
 *                           Gauss-Jordan without pivoting: the blocks must be positive definite ((4+m) dominating c_sw |A|, the
 *                           regime the operator is used in); depends on m0 and c_sw, so once per gauge update AND mass.
 *   hirep_Cphi_inv          out_half = that block inverse applied to in_half (spinors of the parity `inv` was built for)
 *   hirep_Dphi_clover_hat   out_even = D_ee in_even - D_eo D_oo^{-1} D_oe in_even; inv_odd = hirep_clover_inv_field(.., HIREP_ODD, ..)
 *                           for the same m0, csw.  Two launches where the fused epilogue exists (see hirep_Dphi_clover): the D_oe pass
 *                           applies D_oo^{-1} to its hop sum before storing it, the D_eo pass adds D_ee in_even; else four
 *                           (D_oe, D_oo^{-1}, D_ee, D_eo accumulated in place).  out != in. */
int hirep_clover_inv_bytes(const hirep_geom *g, size_t *bytes);
int hirep_clover_inv_field(hirep_geom *g, double m0, double csw, int parity, void *inv, const void *clover);
int hirep_Cphi_inv(hirep_geom *g, void *out_half, const void *in_half, const void *inv);
int hirep_Dphi_clover_hat(hirep_geom *g, double m0, double csw, void *out_even, const void *in_even, const void *links,
                          const void *clover, const void *inv_odd);

/* ---- exponential clover (Eq 50): D_ee,m + D_oo,m = (4+m0) exp(c_sw/(4+m0) (i/4) sum sigma F) ----
 *   hirep_clover_exp_field  blocks <- (4+m0) exp(+c_sw/(4+m0) A_c) (inverse = 0) or its inverse exp(-c_sw/(4+m0) A_c)/(4+m0)
 *                           (inverse = 1) for the sites of ONE parity: full (2 d_R)^2 blocks, same native layout and size
 *                           (hirep_clover_inv_bytes) as hirep_clover_inv_field; scaling and squaring (2^4) of a 14-term
 *                           Taylor sum, |c_sw A|/(4+m0) <= 8.  A buffer of 2 x that size holding the even blocks followed by
 *                           the odd blocks is a full-lattice block field.
 *   hirep_Dphi_blocks       out_full = blocks_full in_full - 1/2 hop(in_full): Eq 8 with ANY site-diagonal chirality blocks
 *                           (the exponential clover's; also (4+m) + c_sw A written out as full blocks); out != in
 *   hirep_Dphi_blocks_hat   out_even = blocks_even in_even - D_eo inv_blocks_odd D_oe in_even (Eq 43); two launches (fused epilogues,
 *                           as hirep_Dphi_clover_hat) or four; out != in */
int hirep_clover_exp_field(hirep_geom *g, double m0, double csw, int parity, int inverse, void *blocks, const void *clover);
int hirep_Dphi_blocks(hirep_geom *g, void *out_full, const void *in_full, const void *links, const void *blocks_full);
int hirep_Dphi_blocks_hat(hirep_geom *g, void *out_even, const void *in_even, const void *links, const void *blocks_even,
                          const void *inv_blocks_odd);

/* Even-odd preconditioned CG with a site-diagonal term (L803, L815): Q_hat = gamma_5 D_hat with D_hat of Eq 43 is Hermitian
 * when the blocks are (gamma_5 commutes with them and gamma_5 D_eo gamma_5 = D_oe^dagger), so Q_hat^2 is Hermitian positive
 * definite.  Arguments as hirep_Dphi_clover_hat / hirep_Dphi_blocks_hat; four (fused epilogues) or eight launches per application;
 * the CGs then also carry their two reductions in the epilogues of those launches (seven launches per iteration); out != in.
 *   hirep_g5Dphi_clover_hat_sq / hirep_g5Dphi_blocks_hat_sq     out_even = Q_hat^2 in_even
 *   hirep_cg_g5Dphi_clover_hat_sq / hirep_cg_g5Dphi_blocks_hat_sq   Q_hat^2 x_even = b_even; recurrence, stopping rule, iters
 *                           and relres (host pointers, may be NULL) as hirep_cg_g5Dphi_hat_sq; x != b. */
/* The same on the full lattice with general Hermitian blocks (exponential clover): (gamma_5 D)^2 with D = hirep_Dphi_blocks, and
 * the CG on it (as hirep_cg_g5Dphi_clover_sq). */
int hirep_g5Dphi_blocks_sq(hirep_geom *g, void *out_full, const void *in_full, const void *links, const void *blocks_full);
int hirep_cg_g5Dphi_blocks_sq(hirep_geom *g, void *x_full, const void *b_full, const void *links, const void *blocks_full, double tol,
                              int maxiter, int *iters, double *relres);
int hirep_g5Dphi_clover_hat_sq(hirep_geom *g, double m0, double csw, void *out_even, const void *in_even, const void *links,
                               const void *clover, const void *inv_odd);
int hirep_g5Dphi_blocks_hat_sq(hirep_geom *g, void *out_even, const void *in_even, const void *links, const void *blocks_even,
                               const void *inv_blocks_odd);
int hirep_cg_g5Dphi_clover_hat_sq(hirep_geom *g, double m0, double csw, void *x_even, const void *b_even, const void *links,
                                  const void *clover, const void *inv_odd, double tol, int maxiter, int *iters, double *relres);
int hirep_cg_g5Dphi_blocks_hat_sq(hirep_geom *g, void *x_even, const void *b_even, const void *links, const void *blocks_even,
                                  const void *inv_blocks_odd, double tol, int maxiter, int *iters, double *relres);

/* ---- fermion force of the hopping term (Sect. 2.5) ----
 * With eta = (Q_m^2)^-1 psi and xi = Q_m eta (native full-lattice spinors the caller has computed, e.g. by hirep_cg_g5Dphi_sq
 * and gamma_5 hirep_Dphi):
 *   T_mu(x)   = tr_spin[ gamma_5 (1 - gamma_mu) { eta(x+mu) (x) xi^dagger(x) + xi(x+mu) (x) eta^dagger(x) } ]          (Eq 20)
 *   F^a_mu(x) = -(1/T_FUND) Re tr[ i T_R^a U^R_mu(x) T_mu(x) ],  a = 0 .. N_g^2 - 2, T_FUND = 1/2                      (Eq 21)
 * The printed Eq 21 has lost the generator; with i T_R^a (as in Eq 19) this is -(1/T_FUND) dS_f/d omega^a for
 * U_mu(x) -> exp(i omega^a T^a) U_mu(x), S_f = psi^dagger (Q_m^2)^-1 psi (reading A32).  T_R^a = -i dR/d omega^a are the
 * generators of the representation in the basis of reading A10/A11 (fundamental T^a = generalised Gell-Mann / 2).
 * force_canonical: device buffer of hirep_force_bytes bytes, REAL numbers of the working precision in CANONICAL order
 * [ix][mu][a] (ix = ((t L + x) L + y) L + z); overwritten.  links_rep: the stored represented field (boundary signs included: a
 * hop across the edge contributes with bc_mu, Eq 61).  In HIREP_LINKS_REBUILD mode `links_rep` is the FUNDAMENTAL field and only the
 * adjoint representation is served (matrix-free: (T^a_adj)_bc = -i f^abc turns the projection into -4 Im tr(T^a C) with C a sum of
 * commutators [K^dagger, W H W^dagger] of N x N matrices); every other representation returns HIREP_EINVAL there.  The first call builds the
 * generator table (one small kernel + a host round trip; not capturable in a CUDA graph), later calls only enqueue one kernel. */
int hirep_force_bytes(const hirep_geom *g, size_t *bytes, int *n_generators);
int hirep_force_hopping(hirep_geom *g, void *force_canonical, const void *eta_full, const void *xi_full, const void *links_rep);

/* Measurement utility: achieved TFLOP/s (2 flops per FMA) of a register-resident chain of
 * FMAs in the given precision on the current device, the ALU roofline the pipe utilisation is read against.
 * Synchronous; tflops is a host pointer. */
int hirep_fma_peak(int prec, double *tflops);

int hirep_sync(hirep_geom *g);
/* hirep_sync also reports numerical breakdowns that kernels flagged since the last sync (HIREP_EBREAKDOWN, flags cleared):
 * hirep_clover_inv_field eliminates without pivoting and flags a pivot below 1e-10 (fp32: 1e-4) of the block's largest entry or a
 * non-finite one (blocks not positive definite: c_sw |A| is not small against 4 + m0); hirep_clover_exp_field flags sites with
 * |c_sw/(4+m0) A_c|_inf > 8, outside the range its scaling-and-squaring series is accurate for.  The fields are then unusable. */ /* synchronise the stream; returns any pending execution error */
const char *hirep_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* HIREP_B200_H */
