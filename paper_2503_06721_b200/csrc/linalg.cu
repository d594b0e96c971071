// linalg.cu -- spinor linear algebra and reductions on native-layout spinors.
//
//   linear combinations   Eq 22-26: every form is xi = c0*xi + c1*eta + c2*zeta with complex
//                         coefficients (a real coefficient is a complex one with zero imaginary part), one fused
//                         kernel -- "fusing together one or more linear algebra kernels" (L379)
//   reductions            Eq 27 (L402) <xi,eta>, Eq 32 (L426) ||xi||^2, Eq 33 (L430) max norm, accumulated with
//                         Neumaier's compensated sum, Algorithm 2 (L662) -- the paper's default; Algorithms 3 and 4
//                         (second-order Neumaier, double-double) selectable -- per thread, and
//                         merged across lanes / warps / blocks with the branch-free two-sum (L654: "either variant
//                         can be used"); fp32 fields are accumulated in fp64 (their products are exact in fp64)
//   cg_update / cg_xp     the CG step in two fused passes:  r -= alpha Ap ; ||r||^2   and, once beta is known,
//                         x += alpha p ; p = r + beta p   (8 spinor passes per iteration instead of 9)
//
// All kernels are HBM-bound streaming passes: 128-bit accesses, grid = 4 CTAs per SM, grid-stride loops.  The
// padding lanes of the last tile (sites h >= Nh) are excluded from every reduction.
#include "kernels.h"
#include "reduce.cuh"

namespace hirep {

namespace {

constexpr int RED_THREADS = 256;

// block-wide merge of NV accumulators per thread; result valid in thread 0
template <int NV> __device__ void block_merge(Acc (&a)[NV], int alg) {
    __shared__ Acc sh[NV][RED_THREADS / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const Acc b = acc_shfl_down(a[v], off);
            acc_merge(a[v], b, alg);
        }
        if (lane == 0) sh[v][warp] = a[v];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int v = 0; v < NV; ++v) {
            Acc x = lane < RED_THREADS / 32 ? sh[v][lane] : Acc{0.0, 0.0, 0.0};
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) {
                const Acc b = acc_shfl_down(x, off);
                acc_merge(x, b, alg);
            }
            a[v] = x;
        }
    }
}

// Which elements of a native spinor buffer are real sites: element i = (row r = i >> 5, lane = i & 31), row =
// (half, tile, component); only the LAST tile of each half lattice has padding lanes (lane >= Nh % 32).  No division.
struct Pad {
    long rows_per_half;   // n_tiles * ncomp
    int ncomp, valid;     // valid lanes of the last tile (32 = no padding)
};
__device__ __forceinline__ bool is_site(const Pad &P, long i) {
    if (P.valid == TILE) return true;
    long r = i >> 5;
    if (r >= P.rows_per_half) r -= P.rows_per_half;
    return r < P.rows_per_half - P.ncomp || (int)(i & (TILE - 1)) < P.valid;
}

// ---- xi = c0*xi + c1*eta + c2*zeta --------------------------------------------------------------------------
template <typename T, bool USE_XI, bool USE_ZETA>
__global__ void __launch_bounds__(256) lincomb_kernel(long n, cplx<T> *xi, double2 c0, const cplx<T> *eta,
                                                      double2 c1, const cplx<T> *zeta, double2 c2) {
    const T c0x = (T)c0.x, c0y = (T)c0.y, c1x = (T)c1.x, c1y = (T)c1.y, c2x = (T)c2.x, c2y = (T)c2.y;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
        const cplx<T> e = eta[i];
        T re = c1x * e.x - c1y * e.y, im = c1x * e.y + c1y * e.x;
        if (USE_ZETA) {
            const cplx<T> z = zeta[i];
            re += c2x * z.x - c2y * z.y;
            im += c2x * z.y + c2y * z.x;
        }
        if (USE_XI) {
            const cplx<T> x = xi[i];
            re += c0x * x.x - c0y * x.y;
            im += c0x * x.y + c0y * x.x;
        }
        xi[i] = mk<T>(re, im);
    }
}

// ---- xi = c1*eta + c2*gamma_5*eta: the factor is c1 + c2 on the upper two spin components, c1 - c2 on the lower two
template <typename T>
__global__ void __launch_bounds__(256) g5_lincomb_kernel(long n, int ncomp, cplx<T> *xi, const cplx<T> *eta,
                                                         double2 cu, double2 cl, double2 c0, int use_xi) {
    const T ux = (T)cu.x, uy = (T)cu.y, lx = (T)cl.x, ly = (T)cl.y, c0x = (T)c0.x, c0y = (T)c0.y;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
        const int comp = (int)((i >> 5) % ncomp);          // row = (half, tile, component)
        const bool lower = 2 * comp >= ncomp;
        const T cx = lower ? lx : ux, cy = lower ? ly : uy;
        const cplx<T> e = eta[i];
        T re = cx * e.x - cy * e.y, im = cx * e.y + cy * e.x;
        if (use_xi) {   // add-(mul-)assign forms (L447): xi <- c0 xi + c1 eta + c2 gamma_5 eta
            const cplx<T> x = xi[i];
            re += c0x * x.x - c0y * x.y;
            im += c0x * x.y + c0y * x.x;
        }
        xi[i] = mk<T>(re, im);
    }
}

// ---- xi = gamma_mu eta (Eq 34), gamma_mu = [[0, e_mu], [e_mu^dagger, 0]] in the basis of Eq 1-3 (L171-182):
// e_0 = -1, e_k = -i sigma_k.  One thread per (site, colour): the four spin components of that colour.  mu = 5: gamma_5.
template <typename T>
__global__ void __launch_bounds__(256) gamma_kernel(long nrows32, int dR, int mu, cplx<T> *__restrict__ xi, const cplx<T> *__restrict__ eta) {
    // element (tile-row block, colour c, lane): components at ((tile*4*dR) + s*dR + c)*32 + lane, s = 0..3
    const long total = nrows32 * dR * TILE;   // nrows32 = number of tiles (halves included)
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long)gridDim.x * blockDim.x) {
        const int lane = (int)(i & (TILE - 1));
        const long tc = i >> 5;
        const int c = (int)(tc % dR);
        const long tile = tc / dR;
        const size_t base = ((size_t)tile * 4 * dR + c) * TILE + lane, st = (size_t)dR * TILE;
        const cplx<T> a0 = eta[base], a1 = eta[base + st], a2 = eta[base + 2 * st], a3 = eta[base + 3 * st];
        cplx<T> o0, o1, o2, o3;
        auto neg = [](cplx<T> z) { return mk<T>(-z.x, -z.y); };
        auto muli = [](cplx<T> z) { return mk<T>(-z.y, z.x); };      // i z
        auto mulmi = [](cplx<T> z) { return mk<T>(z.y, -z.x); };     // -i z
        switch (mu) {
        case 0: o0 = neg(a2); o1 = neg(a3); o2 = neg(a0); o3 = neg(a1); break;                  // e_0 = -1
        case 1: o0 = mulmi(a3); o1 = mulmi(a2); o2 = muli(a1); o3 = muli(a0); break;             // e_1 = -i sigma_1
        case 2: o0 = neg(a3); o1 = a2; o2 = a1; o3 = neg(a0); break;                             // e_2 = -i sigma_2 = [[0,-1],[1,0]]
        case 3: o0 = mulmi(a2); o1 = muli(a3); o2 = muli(a0); o3 = mulmi(a1); break;             // e_3 = -i sigma_3
        default: o0 = a0; o1 = a1; o2 = neg(a2); o3 = neg(a3); break;                            // gamma_5
        }
        xi[base] = o0; xi[base + st] = o1; xi[base + 2 * st] = o2; xi[base + 3 * st] = o3;
    }
}

// ---- partial reductions: one Acc pair (or quadruple) per block -------------------------------------------------
// mode 0: <xi,eta> (re, im)   mode 1: ||xi||^2 (re only)   mode 2: <xi, gamma_5 eta> (the fused reduction of L447)
template <typename T, int MODE>
__global__ void __launch_bounds__(RED_THREADS) prod_partial_kernel(Pad P, long n, int alg, const cplx<T> *__restrict__ xi,
                                                                   const cplx<T> *__restrict__ eta, Acc *__restrict__ partial) {
    Acc a[2] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
        if (!is_site(P, i)) continue;
        const cplx<T> x = xi[i];
        const double xr = (double)x.x, xm = (double)x.y;
        if (MODE == 1) {
            acc_add(a[0], __dmul_rn(xr, xr), alg);
            acc_add(a[0], __dmul_rn(xm, xm), alg);
        } else {
            const cplx<T> e = eta[i];
            double er = (double)e.x, em = (double)e.y;
            if (MODE == 2 && 2 * (int)((i >> 5) % P.ncomp) >= P.ncomp) { er = -er; em = -em; }   // lower spin components
            acc_add(a[0], __dmul_rn(xr, er), alg);
            acc_add(a[0], __dmul_rn(xm, em), alg);
            acc_add(a[1], __dmul_rn(xr, em), alg);
            acc_add(a[1], -__dmul_rn(xm, er), alg);
        }
    }
    block_merge<2>(a, alg);
    if (threadIdx.x == 0) { partial[2 * blockIdx.x] = a[0]; partial[2 * blockIdx.x + 1] = a[1]; }
}

// fused CG step: x += alpha p ; r -= alpha Ap ; partial ||r||^2          (alpha real: A is Hermitian positive definite)
template <typename T>
__global__ void __launch_bounds__(RED_THREADS) cg_update_kernel(Pad P, long n, int alg, double alpha, const double *__restrict__ num,
                                                                const double *__restrict__ den, cplx<T> *__restrict__ x,
                                                                cplx<T> *__restrict__ r, const cplx<T> *__restrict__ p,
                                                                const cplx<T> *__restrict__ Ap, Acc *__restrict__ partial) {
    Acc a[2] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
    if (num != nullptr) alpha = __ddiv_rn(num[0], den[0]);   // device-resident scalars: the same IEEE division the host would do
    const T al = (T)alpha;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
        const cplx<T> av = Ap[i];
        cplx<T> rv = r[i];
        if (x != nullptr) {   // null: only the residual is updated (multi-shift CG keeps its own x_k, p_k)
            const cplx<T> pv = p[i];
            cplx<T> xv = x[i];
            xv.x += al * pv.x; xv.y += al * pv.y;
            x[i] = xv;
        }
        rv.x -= al * av.x; rv.y -= al * av.y;
        r[i] = rv;
        if (is_site(P, i)) {
            acc_add(a[0], __dmul_rn((double)rv.x, (double)rv.x), alg);
            acc_add(a[0], __dmul_rn((double)rv.y, (double)rv.y), alg);
        }
    }
    block_merge<2>(a, alg);
    if (threadIdx.x == 0) { partial[2 * blockIdx.x] = a[0]; partial[2 * blockIdx.x + 1] = a[1]; }
}

// second half of the CG step, after beta is known:  x += alpha p ; p = r + beta p   (one pass: reads x, p, r; writes x, p)
template <typename T>
__global__ void __launch_bounds__(256) cg_xp_kernel(long n, double alpha, double beta, const double *__restrict__ rr_old,
                                                    const double *__restrict__ pAp, const double *__restrict__ rr_new, cplx<T> *__restrict__ x,
                                                    cplx<T> *__restrict__ p, const cplx<T> *__restrict__ r) {
    if (rr_old != nullptr) { alpha = __ddiv_rn(rr_old[0], pAp[0]); beta = __ddiv_rn(rr_new[0], rr_old[0]); }
    const T al = (T)alpha, be = (T)beta;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
        const cplx<T> pv = p[i], rv = r[i];
        cplx<T> xv = x[i];
        xv.x += al * pv.x; xv.y += al * pv.y;
        x[i] = xv;
        p[i] = mk<T>(rv.x + be * pv.x, rv.y + be * pv.y);
    }
}

// second stage: merge the per-block accumulators (fixed order: deterministic), out[v] = the algorithm's final value
__global__ void __launch_bounds__(RED_THREADS) reduce_final_kernel(int nblocks, int alg, const Acc *__restrict__ partial, double *__restrict__ out) {
    Acc a[2] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
    for (int b = threadIdx.x; b < nblocks; b += RED_THREADS) {
        acc_merge(a[0], partial[2 * b], alg);
        acc_merge(a[1], partial[2 * b + 1], alg);
    }
    block_merge<2>(a, alg);
    if (threadIdx.x == 0) { out[0] = acc_value(a[0], alg); out[1] = acc_value(a[1], alg); }
}

template <typename T>
__global__ void __launch_bounds__(RED_THREADS) maxnorm_partial_kernel(Pad P, long n, const cplx<T> *__restrict__ xi, double *__restrict__ partial) {
    double m = 0.0;
    for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
        if (!is_site(P, i)) continue;
        const cplx<T> x = xi[i];
        m = fmax(m, fmax(fabs((double)x.x), fabs((double)x.y)));
    }
    __shared__ double sh[RED_THREADS / 32];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) m = fmax(m, __shfl_down_sync(0xffffffffu, m, off));
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < RED_THREADS / 32; ++w) m = fmax(m, sh[w]);
        partial[blockIdx.x] = m;
    }
}
__global__ void maxnorm_final_kernel(int nblocks, const double *__restrict__ partial, double *__restrict__ out) {
    double m = 0.0;
    for (int b = 0; b < nblocks; ++b) m = fmax(m, partial[b]);
    out[0] = m;
}

// partial-sum blocks of the reductions: a constant (4 CTAs per SM of the 148-SM B200 this library is written for), so that the
// workspace size and the summation order do not depend on which device of a process asks first
int red_blocks() { return 4 * 148; }
int blocks_for(long n) {
    const long need = (n + RED_THREADS - 1) / RED_THREADS;
    const int cap = red_blocks();
    return (int)(need < cap ? (need > 0 ? need : 1) : cap);
}

template <typename T>
int lincomb_t(long n, void *xi, double2 c0, bool use_xi, const void *eta, double2 c1, const void *zeta, double2 c2, bool use_zeta, cudaStream_t s) {
    const int nb = blocks_for(n);
    auto X = (cplx<T> *)xi;
    auto E = (const cplx<T> *)eta;
    auto Z = (const cplx<T> *)zeta;
    if (use_xi && use_zeta) lincomb_kernel<T, true, true><<<nb, 256, 0, s>>>(n, X, c0, E, c1, Z, c2);
    else if (use_xi) lincomb_kernel<T, true, false><<<nb, 256, 0, s>>>(n, X, c0, E, c1, Z, c2);
    else if (use_zeta) lincomb_kernel<T, false, true><<<nb, 256, 0, s>>>(n, X, c0, E, c1, Z, c2);
    else lincomb_kernel<T, false, false><<<nb, 256, 0, s>>>(n, X, c0, E, c1, Z, c2);
    return (int)cudaGetLastError();
}

}  // namespace

int k_reduce_workspace_bytes() { return red_blocks() * 2 * (int)sizeof(Acc) + 64; }

// n = number of complex elements of the buffer (padding included); halves = 1 or 2
int k_lincomb(int prec, long n, void *xi, const double c0[2], int use_xi, const void *eta, const double c1[2], const void *zeta,
              const double c2[2], int use_zeta, cudaStream_t s) {
    const double2 a = make_double2(c0[0], c0[1]), b = make_double2(c1[0], c1[1]), c = make_double2(c2[0], c2[1]);
    return prec == 0 ? lincomb_t<double>(n, xi, a, use_xi, eta, b, zeta, c, use_zeta, s)
                     : lincomb_t<float>(n, xi, a, use_xi, eta, b, zeta, c, use_zeta, s);
}

int k_gamma(const Geo &g, int prec, int dR, int halves, int mu, void *xi, const void *eta, cudaStream_t s) {
    const long tiles = (long)g.n_tiles * halves;
    const int nb = blocks_for(tiles * dR * TILE);
    if (prec == 0) gamma_kernel<double><<<nb, 256, 0, s>>>(tiles, dR, mu, (double2 *)xi, (const double2 *)eta);
    else gamma_kernel<float><<<nb, 256, 0, s>>>(tiles, dR, mu, (float2 *)xi, (const float2 *)eta);
    return (int)cudaGetLastError();
}

int k_g5_lincomb(int prec, long n, int dR, void *xi, const double c0[2], int use_xi, const double c1[2], const double c2[2], const void *eta,
                 cudaStream_t s) {
    const double2 cu = make_double2(c1[0] + c2[0], c1[1] + c2[1]), cl = make_double2(c1[0] - c2[0], c1[1] - c2[1]);
    const double2 cx = make_double2(c0[0], c0[1]);
    const int nb = blocks_for(n);
    if (prec == 0) g5_lincomb_kernel<double><<<nb, 256, 0, s>>>(n, 4 * dR, (double2 *)xi, (const double2 *)eta, cu, cl, cx, use_xi);
    else g5_lincomb_kernel<float><<<nb, 256, 0, s>>>(n, 4 * dR, (float2 *)xi, (const float2 *)eta, cu, cl, cx, use_xi);
    return (int)cudaGetLastError();
}

// mode 0: <xi,eta> -> out_dev[0..1] ; mode 1: ||xi||^2 -> out_dev[0] ; ws = k_reduce_workspace_bytes() device bytes
int k_prod(const Geo &g, int prec, int dR, int halves, int mode, int alg, const void *xi, const void *eta, void *ws, double *out_dev, cudaStream_t s) {
    const int ncomp = 4 * dR;
    const long half_elems = (long)g.n_tiles * ncomp * TILE, n = half_elems * halves;
    const Pad P{(long)g.n_tiles * ncomp, ncomp, g.Nh % TILE == 0 ? TILE : g.Nh % TILE};
    const int nb = blocks_for(n);
    Acc *partial = (Acc *)ws;
    if (prec == 0) {
        if (mode == 0) prod_partial_kernel<double, 0><<<nb, RED_THREADS, 0, s>>>(P, n, alg, (const double2 *)xi, (const double2 *)eta, partial);
        else if (mode == 2) prod_partial_kernel<double, 2><<<nb, RED_THREADS, 0, s>>>(P, n, alg, (const double2 *)xi, (const double2 *)eta, partial);
        else prod_partial_kernel<double, 1><<<nb, RED_THREADS, 0, s>>>(P, n, alg, (const double2 *)xi, (const double2 *)eta, partial);
    } else {
        if (mode == 0) prod_partial_kernel<float, 0><<<nb, RED_THREADS, 0, s>>>(P, n, alg, (const float2 *)xi, (const float2 *)eta, partial);
        else if (mode == 2) prod_partial_kernel<float, 2><<<nb, RED_THREADS, 0, s>>>(P, n, alg, (const float2 *)xi, (const float2 *)eta, partial);
        else prod_partial_kernel<float, 1><<<nb, RED_THREADS, 0, s>>>(P, n, alg, (const float2 *)xi, (const float2 *)eta, partial);
    }
    reduce_final_kernel<<<1, RED_THREADS, 0, s>>>(nb, alg, partial, out_dev);
    return (int)cudaGetLastError();
}

int k_reduce_final(int nblocks, int alg, const void *partial, double *out_dev, cudaStream_t s) {
    reduce_final_kernel<<<1, RED_THREADS, 0, s>>>(nblocks, alg, (const Acc *)partial, out_dev);
    return (int)cudaGetLastError();
}

int k_maxnorm(const Geo &g, int prec, int dR, int halves, const void *xi, void *ws, double *out_dev, cudaStream_t s) {
    const int ncomp = 4 * dR;
    const long half_elems = (long)g.n_tiles * ncomp * TILE, n = half_elems * halves;
    const Pad P{(long)g.n_tiles * ncomp, ncomp, g.Nh % TILE == 0 ? TILE : g.Nh % TILE};
    const int nb = blocks_for(n);
    if (prec == 0) maxnorm_partial_kernel<double><<<nb, RED_THREADS, 0, s>>>(P, n, (const double2 *)xi, (double *)ws);
    else maxnorm_partial_kernel<float><<<nb, RED_THREADS, 0, s>>>(P, n, (const float2 *)xi, (double *)ws);
    maxnorm_final_kernel<<<1, 1, 0, s>>>(nb, (const double *)ws, out_dev);
    return (int)cudaGetLastError();
}

int k_cg_xp(const Geo &g, int prec, int dR, int halves, double alpha, double beta, const double *rr_old, const double *pAp, const double *rr_new,
            void *x, void *p, const void *r, cudaStream_t s) {
    const long n = (long)g.n_tiles * 4 * dR * TILE * halves;
    const int nb = blocks_for(n);
    if (prec == 0) cg_xp_kernel<double><<<nb, 256, 0, s>>>(n, alpha, beta, rr_old, pAp, rr_new, (double2 *)x, (double2 *)p, (const double2 *)r);
    else cg_xp_kernel<float><<<nb, 256, 0, s>>>(n, alpha, beta, rr_old, pAp, rr_new, (float2 *)x, (float2 *)p, (const float2 *)r);
    return (int)cudaGetLastError();
}

int k_cg_update(const Geo &g, int prec, int dR, int halves, int alg, double alpha, const double *num, const double *den, void *x, void *r,
                const void *p, const void *Ap, void *ws, double *out_dev, cudaStream_t s) {
    const int ncomp = 4 * dR;
    const long half_elems = (long)g.n_tiles * ncomp * TILE, n = half_elems * halves;
    const Pad P{(long)g.n_tiles * ncomp, ncomp, g.Nh % TILE == 0 ? TILE : g.Nh % TILE};
    const int nb = blocks_for(n);
    Acc *partial = (Acc *)ws;
    if (prec == 0) cg_update_kernel<double><<<nb, RED_THREADS, 0, s>>>(P, n, alg, alpha, num, den, (double2 *)x, (double2 *)r, (const double2 *)p, (const double2 *)Ap, partial);
    else cg_update_kernel<float><<<nb, RED_THREADS, 0, s>>>(P, n, alg, alpha, num, den, (float2 *)x, (float2 *)r, (const float2 *)p, (const float2 *)Ap, partial);
    reduce_final_kernel<<<1, RED_THREADS, 0, s>>>(nb, alg, partial, out_dev);
    return (int)cudaGetLastError();
}

}  // namespace hirep
