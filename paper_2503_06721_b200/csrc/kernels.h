// kernels.h -- host-side launchers (type-erased on precision / representation) used by api.cu.
// Each returns 0, a positive cudaError_t, or KERR_UNSUPPORTED when the combination is not instantiated.
#pragma once
#include "common.cuh"

namespace hirep {

constexpr int KERR_UNSUPPORTED = -2;

// one stencil pass over the sites of parity p_out:  out = a*self + b*hop(in)   (optionally times gamma_5)
//   hop(in)(x) = sum_d P_d W_d(x) in(nbr_d(x)),  P_d = (1 -+ gamma_mu)        (the bracket of Eq 8)
struct HopSet {
    const void *in;     // spinor on parity 1-p_out
    void *out;          // spinor on parity p_out
    const void *self;   // spinor on parity p_out (may be null when a == 0)
    const void *links;  // gather block of parity p_out: represented (stored) or fundamental (rebuild)
    int p_out;
    const void *diag;   // site-diagonal matrices of parity p_out when HopLaunch::diag_mode != 0 (tile-major, [tile][entry][lane] complex)
};
// Site-diagonal term applied inside the stencil epilogue (Eq 43 / 47 / 50: "fused into the second pass").
// The matrices ride through the same bulk-copy ring as the links, after the eight directions of a tile.
//   DIAG_HB   : out = (a + csw A) self + b hop(in),  A_c = [[H, B], [B^+, -H]] from the clover field (4 d_R^2 complex per site)
//   DIAG_PRE  : out = M self + b hop(in),            M = full (2 d_R)^2 chirality blocks (8 d_R^2 complex per site)
//   DIAG_POST : out = M (b hop(in))                  (D_oo^-1 D_oe of the Schur form; no self)
enum { DIAG_NONE = 0, DIAG_HB = 1, DIAG_PRE = 2, DIAG_POST = 3 };
struct HopLaunch {
    HopSet set[2];
    int nsets;          // 1 = half lattice, 2 = both parities in one launch
    double a, b;
    double bi;          // the hop sum is scaled by (b + i bi gamma_5): D_oo^-1 = (a - i mu gamma_5)/(a^2 + mu^2) of the twisted-mass Schur form (Eq 43, 51)
                        // fused into the D_oe pass; ring / pair / row-group / matrix-free adjoint kernels, 0 elsewhere
    double am;          // twisted mass mu: the diagonal term is (a + i am gamma_5) self (Eq 51); 0 = plain Wilson
    int g5;             // multiply the result by gamma_5 = diag(1,1,-1,-1)
    int diag_mode;      // DIAG_*: site-diagonal matrices HopSet::diag applied in the epilogue (ring / pair kernels, stored links)
    double diag_csw;    // DIAG_HB: c_sw (a is the (4+m) of Eq 47)
    int max_ctas;       // cap on the persistent grid (0 = one CTA per SM); tests use it to force many tiles per warp
    int tile_begin, tile_end;   // tiles [begin, end) of each parity to compute (slab regions: interior / boundary); end = 0: all
    // reductions fused into the epilogue of the tile-pair kernel (hop_full.cuh; the CG on Q^2):
    //   red_mode 1: the result is stored as usual and sum |out|^2 over the real sites is accumulated
    //   red_mode 2: the result is NOT stored; red_r -= (red_num / red_den) * result, sum |red_r|^2 is accumulated
    // per-CTA partial sums (compensated, algorithm red_alg) go to red_partial[2 * blockIdx.x] (an Acc of reduce.cuh, second one zero)
    int red_mode, red_alg;
    void *red_partial;
    void *red_r;                        // native full-lattice spinor (even half, then odd half)
    const double *red_num, *red_den;    // device scalars
    unsigned *pace;     // hop_full.cuh: device counter of the round pacing (NULL / pace_every = 0: off)
    int pace_every;     // grid-wide rendezvous every pace_every tile rounds
    int dbg;            // HIREP_DBG (development only, results become wrong): bit mu skips the backward-link gather of direction mu,
                        // bit 4+mu the neighbour-spinor gathers of +-mu in hop_full.cuh -- traffic attribution under ncu
};

inline __host__ __device__ int launch_tiles(const Geo &g, const HopLaunch &L) { return L.tile_end > 0 ? L.tile_end - L.tile_begin : g.n_tiles; }

// slab halo (half-spinor faces, L624): face = 0 first owned slice (projected with 1-gamma_0, for the previous rank's forward hop),
// face = 1 last owned slice (1+gamma_0, for the next rank's backward hop); unpack writes ghost slice T-1 (face 0 data) or 0 (face 1 data)
int k_halo_pack(const Geo &g, int prec, int dR, int parity, int face, void *buf, const void *spinor_half, cudaStream_t s);
int k_halo_unpack(const Geo &g, int prec, int dR, int parity, int face, void *spinor_half, const void *buf, cudaStream_t s);
int k_spinor_import(const Geo &g, int prec, int dR, void *native, const void *canon, int which, cudaStream_t s);
int k_spinor_export(const Geo &g, int prec, int dR, void *canon, const void *native, int which, cudaStream_t s);
int k_links_import(const Geo &g, int prec, int N, void *native_fund, const void *canon, cudaStream_t s);
int k_links_rep_export(const Geo &g, int prec, int dR, int real, void *canon, const void *native, int bwd, cudaStream_t s);
int k_links_to_rep(const Geo &g, int prec, int N, int rep, void *native_rep, const void *native_fund, cudaStream_t s);
// variant: 0 default; see hop_dispatch.cu.  mode: 0 stored represented links, 1 rebuild from fundamental (N, rep).
int k_hop(const Geo &g, int prec, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s);
// whether a launch with HopLaunch::diag_mode != 0 is instantiated for this configuration (else the caller composes the
// operator from separate block-apply launches)
bool k_hop_diag_supported(int prec, int dR, int real, int mode, int variant);
// linalg.cu: spinor linear algebra / reductions on native buffers (n = complex elements incl. padding; halves = 1 | 2)
int k_reduce_workspace_bytes();
// second stage of a reduction whose per-CTA partials a stencil launch has written (HopLaunch::red_partial): out_dev[0..1]
int k_reduce_final(int nblocks, int alg, const void *partial, double *out_dev, cudaStream_t s);
int k_lincomb(int prec, long n, void *xi, const double c0[2], int use_xi, const void *eta, const double c1[2], const void *zeta,
              const double c2[2], int use_zeta, cudaStream_t s);
int k_gamma(const Geo &g, int prec, int dR, int halves, int mu, void *xi, const void *eta, cudaStream_t s);
int k_g5_lincomb(int prec, long n, int dR, void *xi, const double c0[2], int use_xi, const double c1[2], const double c2[2], const void *eta,
                 cudaStream_t s);
int k_prod(const Geo &g, int prec, int dR, int halves, int mode, int alg, const void *xi, const void *eta, void *ws, double *out_dev, cudaStream_t s);
int k_maxnorm(const Geo &g, int prec, int dR, int halves, const void *xi, void *ws, double *out_dev, cudaStream_t s);
// num/den, rr_old/pAp/rr_new: device-resident scalars (alpha = num/den; alpha = rr_old/pAp, beta = rr_new/rr_old) used instead of
// the by-value alpha, beta when non-null: the pipelined CG never waits for the host between the operator and the updates
int k_cg_update(const Geo &g, int prec, int dR, int halves, int alg, double alpha, const double *num, const double *den, void *x, void *r,
                const void *p, const void *Ap, void *ws, double *out_dev, cudaStream_t s);
int k_cg_xp(const Geo &g, int prec, int dR, int halves, double alpha, double beta, const double *rr_old, const double *pAp, const double *rr_new,
            void *x, void *p, const void *r, cudaStream_t s);
int k_fma_peak(int prec, double *tflops, cudaStream_t s);   // fma_peak.cu: measured FP64/FP32 FMA throughput
// clover.cu: clover term (Eq 47-49); native clover field = 4 dR^2 complex per site
int k_clover_field(const Geo &g, int prec, int dR, int real, void *clover, const void *links_rep, cudaStream_t s);
int k_clover_export(const Geo &g, int prec, int dR, void *canon, const void *clover, cudaStream_t s);
int k_cphi(int prec, int dR, int ntile, double a, double csw, const void *clover, const void *in, void *out, cudaStream_t s);
// inverse diagonal blocks of one parity ((2 dR)^2 complex per site and chirality) and their application
int k_clover_inv(const Geo &g, int prec, int dR, int parity, double a, double csw, const void *clover, void *inv, int *flags, cudaStream_t s);
// blocks of one parity <- pref * exp(x A_c) (Eq 50); work = 2 x the bytes of `blocks`
int k_clover_exp(const Geo &g, int prec, int dR, int parity, double x, double pref, const void *clover, void *blocks, void *work, int *flags, cudaStream_t s);
int k_cblock(int prec, int dR, int ntile, const void *blk, const void *in, void *out, cudaStream_t s);
// force.cu: fermion force of the hopping term (Eq 20-21).  k_rep_generators fills a dense double2 table [N^2-1][dR][dR] of the
// represented generators; k_force_hopping takes them as a sparse list (entries of generator a: rowptr[a]..rowptr[a+1], jk = j*dR+k)
// and, for the register kernel at small d_R, the dense table itself
int k_rep_generators(int N, int rep, void *table_dev, cudaStream_t s);
// fund: the representation is the fundamental one (its generators are known in closed form, reading A10)
int k_force_hopping(const Geo &g, int prec, int dR, int real, int fund, const void *eta, const void *xi, const void *links, const int *rowptr,
                    const int *jk, const void *val, const void *dense, int NA, void *force, cudaStream_t s);
int k_force_hopping_adj(const Geo &g, int prec, int N, const void *eta, const void *xi, const void *links_fund, void *force, cudaStream_t s);
// number of distinct kernel launches k_hop issues for this configuration (for launch accounting): always 1.

}  // namespace hirep
