// clover.cu -- clover term of the Wilson-Dirac operator (Eq 47-49).
//
//   D_ee,m + D_oo,m = (4+m) + c_sw (i/4) sum_{mu,nu} sigma_{mu nu} F_{mu nu}                       (Eq 47)
//   C_{mu nu}(x) = the four plaquette loops through x in the (mu,nu) plane, each closed at x         (Eq 48; DESIGN A26)
//   F_{mu nu} = (C_{mu nu} - C_{mu nu}^dagger)/8                                                    (Eq 49; DESIGN A27)
//
// With gamma_mu = [[0,e_mu],[e_mu^+,0]], e_0 = -1, e_k = -i sigma_k (Eq 2-3) and sigma_{mu nu} = (i/2)[gamma_mu,gamma_nu]
// (DESIGN A28) the term is block diagonal in chirality, A = diag(A_0, A_1), A_c acting on spins (2c, 2c+1):
//   sigma_01 = (s1,-s1)  sigma_02 = (s2,-s2)  sigma_03 = (s3,-s3)  sigma_12 = (-s3,-s3)  sigma_13 = (s2,s2)  sigma_23 = (-s1,-s1)
//   A_c = s1 (x) K1 + s2 (x) K2 + s3 (x) K3 = [[H, B], [B^+, -H]],   H = K3,  B = K1 - i K2,   with (+ for c = 0, - for c = 1)
//   K1 = (i/2)(+-F01 - F23),  K2 = (i/2)(+-F02 + F13),  K3 = (i/2)(+-F03 - F12)       (Hermitian, F being anti-Hermitian)
//
// Native clover field (caller-owned, hirep_clover_bytes): [parity][tile][c = 0,1][m = 0: H, 1: B][e = i*dR + j][lane]
// complex<T>: 4 dR^2 complex per site, half the bytes of the eight represented links.
//
// Kernels: clover_field_kernel -- a CTA per (part of a) tile, the plaquette leaves as path products W_d1(x) W_d2(x+d1) ... out of
// the gather-layout links (W_d = U_mu(x) / U_mu(x-mu)^dagger) in shared memory; runs once per gauge update like
// links_to_rep.  cphi_site_kernel / cphi_kernel -- out = ((4+m) + c_sw A) in, coalesced 32-lane rows (see there).
#include "hop_ring.cuh"   // DevCache / prepare_launch (opt-in shared-memory size per device)
#include "kernels.h"

namespace hirep {

template <typename T> __device__ __forceinline__ cplx<T> cmul(cplx<T> a, cplx<T> b) { return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <typename T> __device__ __forceinline__ void cfma(cplx<T> &acc, cplx<T> a, cplx<T> b) {
    acc.x += a.x * b.x - a.y * b.y;
    acc.y += a.x * b.y + a.y * b.x;
}
// acc += conj(a) * b
template <typename T> __device__ __forceinline__ void cfma_conj(cplx<T> &acc, cplx<T> a, cplx<T> b) {
    acc.x += a.x * b.x + a.y * b.y;
    acc.y += a.x * b.y - a.y * b.x;
}

__host__ __device__ inline size_t clover_off(int n_tiles, int p, int tile, int c, int m, int e, int lane, int ne) {
    return (((((size_t)p * n_tiles + tile) * 2 + c) * 2 + m) * ne + e) * TILE + lane;
}

// full coordinates of a site walked along a path; no divisions per step (the stencil kernels use neighbour<D> instead)
struct Walker {
    int c[4];
    __device__ void start(const Geo &g, int p, int h) {
        int zh;
        decode_site(g, h, c[0], c[1], c[2], zh);
        c[3] = 2 * zh + ((c[0] + c[1] + c[2] + p) & 1);
    }
    __device__ void step(const Geo &g, int d) {
        const int mu = d & 3, ext = mu == 0 ? g.T : g.L;
        int v = c[mu] + (d < 4 ? 1 : -1);
        v = v == ext ? 0 : (v < 0 ? ext - 1 : v);
        c[mu] = v;
    }
    __device__ int parity() const { return (c[0] + c[1] + c[2] + c[3]) & 1; }
    __device__ int half_index(const Geo &g) const { return encode_site(g, c[0], c[1], c[2], c[3] >> 1); }
};

template <typename T, bool REAL> __device__ __forceinline__ cplx<T> ld_w(const link_elem<T, REAL> *links, size_t off) {
    if constexpr (REAL) return mk<T>(links[off], T(0));
    else return links[off];
}

// blockDim = (S sites, NW entry workers): a CTA owns S consecutive site slots of one tile (S = 32 unless the matrices do
// not fit), thread (s, w) works on the matrix entries e = w, w + NW, ... of site s.  Shared memory [matrix][e][S]:
// W[4 LP] (the links of LP leaves), P[LP], Q[LP] (path products), C (leaf sum), acc[4] = H0, B0, H1, B1.  A global load of
// entry e by the S threads of a row is one contiguous S * 16-byte segment for the site's own links (a gather for the
// neighbours', as in the stencil); shared-memory accesses are conflict free (s is the fastest index).
// DRT > 0 fixes d_R at compile time (inner products unrolled); planes, leaves and path steps are unrolled so that every
// direction is a constant (no local-memory tables, no dynamic indexing of the coordinates).
// multiply-add on path elements: complex for complex links, real for the real (adjoint) links
template <typename T> __device__ __forceinline__ void pfma(cplx<T> &acc, cplx<T> a, cplx<T> b) { cfma<T>(acc, a, b); }
template <typename T> __device__ __forceinline__ void pfma(T &acc, T a, T b) { acc = fma(a, b, acc); }
template <typename T> __device__ __forceinline__ cplx<T> as_cplx(cplx<T> v) { return v; }
template <typename T> __device__ __forceinline__ cplx<T> as_cplx(T v) { return mk<T>(v, T(0)); }
template <typename T> __device__ __forceinline__ void padd(cplx<T> &acc, cplx<T> v) { acc.x += v.x; acc.y += v.y; }
template <typename T> __device__ __forceinline__ void padd(T &acc, T v) { acc += v; }

template <typename T, bool REAL, int LP, int DRT>
__global__ void __launch_bounds__(512) clover_field_kernel(Geo g, int dR_rt, const link_elem<T, REAL> *__restrict__ links, cplx<T> *__restrict__ clover) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // real links (adjoint): the path products are real matrices -- a quarter of the multiply-adds and half the shared memory
    using PT = link_elem<T, REAL>;
    const int dR = DRT ? DRT : dR_rt;
    const int ne = dR * dR, S = blockDim.x, sx = threadIdx.x;
    const size_t mat = (size_t)ne * S;                                  // one matrix for the S sites
    cplx<T> *acc = reinterpret_cast<cplx<T> *>(smem_raw) + sx;          // [4][e][S] complex, then the path matrices
    PT *W = reinterpret_cast<PT *>(smem_raw + 4 * mat * sizeof(cplx<T>)) + sx;
    PT *P = W + 4 * LP * mat, *Q = P + LP * mat, *C = Q + LP * mat;
    const long slot = (long)blockIdx.x * S + sx;                        // padded site slots: [parity][tile][lane]
    const int slots_half = g.n_tiles * TILE;
    const int p = (int)(slot / slots_half), hp = (int)(slot - (long)p * slots_half);
    const bool live = hp < g.Nh;                                        // padding lanes compute site Nh-1 and store zeros
    const int h = live ? hp : g.Nh - 1;
    const int nt = blockDim.y, tid = threadIdx.y;
    // blockDim.y = r * dR: thread (.., tid) owns column j of the rows i0, i0 + r, ... of every matrix
    const int r = nt / dR, i0 = tid / dR, j = tid - i0 * dR;
    Walker w0;
    w0.start(g, p, h);
    for (int e = tid; e < 4 * ne; e += nt) acc[(size_t)e * S] = mk<T>(0, 0);
    constexpr int PL[6][2] = {{0, 1}, {0, 2}, {0, 3}, {1, 2}, {1, 3}, {2, 3}};
#pragma unroll
    for (int pl = 0; pl < 6; ++pl) {
        const int mu = PL[pl][0], nu = PL[pl][1];
        const int seq[4][4] = {{mu, nu, mu + 4, nu + 4}, {nu, mu + 4, nu + 4, mu}, {mu + 4, nu + 4, mu, nu}, {nu + 4, mu, nu, mu + 4}};
        for (int i = i0; i < dR; i += r) C[(size_t)(i * dR + j) * S] = PT{};
#pragma unroll
        for (int lg = 0; lg < 4; lg += LP) {
#pragma unroll
            for (int ll = 0; ll < LP; ++ll) {   // the four links along each closed path x -> x+d1 -> x+d1+d2 -> ... -> x
                Walker w = w0;
                int cp = p, ch = h;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int d = seq[lg + ll][k];
                    const size_t base = link_off(g.n_tiles, cp, ch >> 5, d, 0, ch & 31, ne);
                    PT *dst = W + (size_t)(ll * 4 + k) * mat;
                    for (int i = i0; i < dR; i += r) dst[(size_t)(i * dR + j) * S] = links[base + (size_t)(i * dR + j) * TILE];
                    w.step(g, d);
                    ch = w.half_index(g);
                    cp ^= 1;
                }
            }
            __syncthreads();
#pragma unroll
            for (int ll = 0; ll < LP; ++ll) {
                const PT *A = W + (size_t)(ll * 4) * mat, *B = A + mat;
                for (int i = i0; i < dR; i += r) {
                    const int e = i * dR + j;
                    PT s = PT{};
                    const PT *a = A + (size_t)(i * dR) * S, *b = B + (size_t)j * S;
#pragma unroll
                    for (int l = 0; l < dR; ++l, a += S, b += (size_t)dR * S) pfma<T>(s, *a, *b);
                    P[ll * mat + (size_t)e * S] = s;
                }
            }
            __syncthreads();
#pragma unroll
            for (int ll = 0; ll < LP; ++ll) {
                const PT *A = P + (size_t)ll * mat, *B = W + (size_t)(ll * 4 + 2) * mat;
                for (int i = i0; i < dR; i += r) {
                    const int e = i * dR + j;
                    PT s = PT{};
                    const PT *a = A + (size_t)(i * dR) * S, *b = B + (size_t)j * S;
#pragma unroll
                    for (int l = 0; l < dR; ++l, a += S, b += (size_t)dR * S) pfma<T>(s, *a, *b);
                    Q[ll * mat + (size_t)e * S] = s;
                }
            }
            __syncthreads();
#pragma unroll
            for (int ll = 0; ll < LP; ++ll) {
                const PT *A = Q + (size_t)ll * mat, *B = W + (size_t)(ll * 4 + 3) * mat;
                for (int i = i0; i < dR; i += r) {
                    const int e = i * dR + j;
                    PT s = C[(size_t)e * S];
                    const PT *a = A + (size_t)(i * dR) * S, *b = B + (size_t)j * S;
#pragma unroll
                    for (int l = 0; l < dR; ++l, a += S, b += (size_t)dR * S) pfma<T>(s, *a, *b);
                    C[(size_t)e * S] = s;
                }
            }
            __syncthreads();
        }
        // F = (C - C^+)/8 ; contribution (i/2) F (and for K2, times -i) to H_c / B_c with the signs of the header table
        for (int i = i0; i < dR; i += r) {
            const int e = i * dR + j;
            const cplx<T> a = as_cplx<T>(C[(size_t)e * S]), b = as_cplx<T>(C[(size_t)(j * dR + i) * S]);
            const cplx<T> F = mk<T>((a.x - b.x) * T(0.125), (a.y + b.y) * T(0.125));
            const cplx<T> iF = mk<T>(-T(0.5) * F.y, T(0.5) * F.x);    // (i/2) F
            const cplx<T> hF = mk<T>(T(0.5) * F.x, T(0.5) * F.y);     // -i (i/2) F = F/2
            cplx<T> &H0 = acc[(size_t)e * S], &B0 = acc[mat + (size_t)e * S], &H1 = acc[2 * mat + (size_t)e * S], &B1 = acc[3 * mat + (size_t)e * S];
            switch (pl) {
            case 0: B0.x += iF.x; B0.y += iF.y; B1.x -= iF.x; B1.y -= iF.y; break;   // K1 += +-(i/2) F01
            case 5: B0.x -= iF.x; B0.y -= iF.y; B1.x -= iF.x; B1.y -= iF.y; break;   // K1 -= (i/2) F23
            case 1: B0.x += hF.x; B0.y += hF.y; B1.x -= hF.x; B1.y -= hF.y; break;   // -i K2, K2 += +-(i/2) F02
            case 4: B0.x += hF.x; B0.y += hF.y; B1.x += hF.x; B1.y += hF.y; break;   // -i K2, K2 += (i/2) F13
            case 2: H0.x += iF.x; H0.y += iF.y; H1.x -= iF.x; H1.y -= iF.y; break;   // K3 += +-(i/2) F03
            default: H0.x -= iF.x; H0.y -= iF.y; H1.x -= iF.x; H1.y -= iF.y; break;  // K3 -= (i/2) F12
            }
        }
        __syncthreads();
    }
    const int tile = hp >> 5, lane = hp & 31;
    for (int q = tid; q < 4 * ne; q += nt) {
        const int cm = q / ne, e = q - cm * ne;
        clover[clover_off(g.n_tiles, p, tile, cm >> 1, cm & 1, e, lane, ne)] = live ? acc[(size_t)q * S] : mk<T>(0, 0);
    }
}

// out = (a + csw A) in on `ntile_total` tiles (both parities are contiguous in every native buffer).
// Small d_R (<= 6): one thread per site, one warp per tile, everything unrolled: per chirality the 2 d_R^2 block elements
// stream through once (H serves both spin rows, B serves B psi_1 and B^+ psi_0), all loads independent.
template <typename T, int DR>
__global__ void __launch_bounds__(128) cphi_site_kernel(int ntile_total, T a, T csw, const cplx<T> *__restrict__ clover,
                                                        const cplx<T> *__restrict__ in, cplx<T> *__restrict__ out) {
    constexpr int NE = DR * DR, NCOMP = 4 * DR;
    const int lane = threadIdx.x & 31;
    const int wpb = blockDim.x >> 5;
    for (int tile = blockIdx.x * wpb + (threadIdx.x >> 5); tile < ntile_total; tile += gridDim.x * wpb) {
        const cplx<T> *psi = in + (size_t)tile * NCOMP * TILE + lane;
        const cplx<T> *cl = clover + (size_t)tile * 4 * NE * TILE + lane;
        cplx<T> *o = out + (size_t)tile * NCOMP * TILE + lane;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const cplx<T> *H = cl + (size_t)(2 * c) * NE * TILE, *B = H + (size_t)NE * TILE;
            cplx<T> p0[DR], p1[DR], o0[DR], o1[DR];
#pragma unroll
            for (int j = 0; j < DR; ++j) {
                p0[j] = __ldg(psi + (size_t)((2 * c) * DR + j) * TILE);
                p1[j] = __ldg(psi + (size_t)((2 * c + 1) * DR + j) * TILE);
                o0[j] = mk<T>(0, 0);
                o1[j] = mk<T>(0, 0);
            }
#pragma unroll
            for (int i = 0; i < DR; ++i) {
#pragma unroll
                for (int j = 0; j < DR; ++j) {
                    const cplx<T> h = __ldcs(H + (size_t)(i * DR + j) * TILE);
                    const cplx<T> b = __ldcs(B + (size_t)(i * DR + j) * TILE);
                    cfma<T>(o0[i], h, p0[j]);
                    cfma<T>(o1[i], mk<T>(-h.x, -h.y), p1[j]);
                    cfma<T>(o0[i], b, p1[j]);
                    cfma_conj<T>(o1[j], b, p0[i]);
                }
            }
#pragma unroll
            for (int i = 0; i < DR; ++i) {
                __stcs(o + (size_t)((2 * c) * DR + i) * TILE, mk<T>(a * p0[i].x + csw * o0[i].x, a * p0[i].y + csw * o0[i].y));
                __stcs(o + (size_t)((2 * c + 1) * DR + i) * TILE, mk<T>(a * p1[i].x + csw * o1[i].x, a * p1[i].y + csw * o1[i].y));
            }
        }
    }
}

// Any d_R: block = (32 lanes, WY warps); warp y computes the output rows (2c, i) and (2c+1, i) for the pairs
// (c, i) = y, y + WY, ... of the block's tile: row i of H once for both, row i and column i of B.
template <typename T>
__global__ void __launch_bounds__(256, sizeof(T) == 8 ? 4 : 3) cphi_kernel(int ntile_total, int dR, T a, T csw, const cplx<T> *__restrict__ clover, const cplx<T> *__restrict__ in,
                            cplx<T> *__restrict__ out) {
    const int ne = dR * dR, ncomp = 4 * dR, lane = threadIdx.x;
    for (int tile = blockIdx.x; tile < ntile_total; tile += gridDim.x) {
        const cplx<T> *psi = in + (size_t)tile * ncomp * TILE + lane;
        const cplx<T> *cl = clover + (size_t)tile * 4 * ne * TILE + lane;
        cplx<T> *o = out + (size_t)tile * ncomp * TILE + lane;
        for (int q = threadIdx.y; q < 2 * dR; q += blockDim.y) {
            const int c = q / dR, i = q - c * dR;
            const cplx<T> *H = cl + (size_t)(2 * c) * ne * TILE, *B = H + (size_t)ne * TILE;
            const cplx<T> *p0 = psi + (size_t)(2 * c) * dR * TILE, *p1 = p0 + (size_t)dR * TILE;
            cplx<T> s0 = mk<T>(0, 0), s1 = mk<T>(0, 0), s2 = mk<T>(0, 0), s3 = mk<T>(0, 0);
#pragma unroll 5
            for (int j = 0; j < dR; ++j) {
                const cplx<T> h = __ldg(H + (size_t)(i * dR + j) * TILE), b = __ldg(B + (size_t)(i * dR + j) * TILE);
                const cplx<T> bt = __ldg(B + (size_t)(j * dR + i) * TILE);
                const cplx<T> x0 = __ldg(p0 + (size_t)j * TILE), x1 = __ldg(p1 + (size_t)j * TILE);
                cfma<T>(s0, h, x0);
                cfma<T>(s1, b, x1);
                cfma_conj<T>(s2, bt, x0);
                cfma<T>(s3, h, x1);
            }
            const cplx<T> e0 = __ldg(p0 + (size_t)i * TILE), e1 = __ldg(p1 + (size_t)i * TILE);
            __stcs(o + (size_t)((2 * c) * dR + i) * TILE, mk<T>(a * e0.x + csw * (s0.x + s1.x), a * e0.y + csw * (s0.y + s1.y)));
            __stcs(o + (size_t)((2 * c + 1) * dR + i) * TILE, mk<T>(a * e1.x + csw * (s2.x - s3.x), a * e1.y + csw * (s2.y - s3.y)));
        }
    }
}

// Large d_R (15 ... 35): a warp computes R consecutive rows i of both spin rows of a chirality at once, so that every psi_j it
// loads serves 4 R complex MACs (the row-pair kernel above re-reads the whole chirality half of psi for every row: as many bytes
// through L1 / L2 as the matrices themselves) and 3 R independent matrix loads are in flight per step.  Work units (tile, c, row
// group) are dealt round-robin over all warps of the grid.
template <typename T, int R>
__global__ void __launch_bounds__(256, 2) cphi_rows_kernel(int ntile_total, int dR, T a, T csw, const cplx<T> *__restrict__ clover,
                                                           const cplx<T> *__restrict__ in, cplx<T> *__restrict__ out) {
    const int ne = dR * dR, ncomp = 4 * dR, lane = threadIdx.x & 31;
    const int groups = (dR + R - 1) / R, upt = 2 * groups;               // units per tile
    const long n_units = (long)ntile_total * upt;
    const long gw = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), nw = (long)gridDim.x * (blockDim.x >> 5);
    for (long u = gw; u < n_units; u += nw) {
        const int tile = (int)(u / upt), q = (int)(u - (long)tile * upt), c = q / groups, i0 = (q - c * groups) * R;
        const cplx<T> *psi = in + (size_t)tile * ncomp * TILE + lane;
        const cplx<T> *H = clover + ((size_t)tile * 4 + 2 * c) * ne * TILE + lane, *B = H + (size_t)ne * TILE;
        const cplx<T> *p0 = psi + (size_t)(2 * c) * dR * TILE, *p1 = p0 + (size_t)dR * TILE;
        int row[R];   // rows of this group; a ragged last group repeats row d_R - 1 (computed twice, stored once)
#pragma unroll
        for (int r = 0; r < R; ++r) row[r] = i0 + r < dR ? i0 + r : dR - 1;
        cplx<T> s0[R], s1[R];
#pragma unroll
        for (int r = 0; r < R; ++r) s0[r] = s1[r] = mk<T>(0, 0);
        for (int j = 0; j < dR; ++j) {
            const cplx<T> x0 = __ldg(p0 + (size_t)j * TILE), x1 = __ldg(p1 + (size_t)j * TILE);
            cplx<T> h[R], b[R], bt[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                h[r] = __ldcs(H + (size_t)(row[r] * dR + j) * TILE);
                b[r] = __ldg(B + (size_t)(row[r] * dR + j) * TILE);      // B is read twice (as row and as column): keep it cacheable
                bt[r] = __ldg(B + (size_t)(j * dR + row[r]) * TILE);
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                cfma<T>(s0[r], h[r], x0);
                cfma<T>(s0[r], b[r], x1);
                cfma_conj<T>(s1[r], bt[r], x0);
                cfma<T>(s1[r], mk<T>(-h[r].x, -h[r].y), x1);
            }
        }
        cplx<T> *o = out + (size_t)tile * ncomp * TILE + lane;
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (i0 + r < dR) {
                const int i = i0 + r;
                const cplx<T> e0 = __ldg(p0 + (size_t)i * TILE), e1 = __ldg(p1 + (size_t)i * TILE);
                __stcs(o + (size_t)((2 * c) * dR + i) * TILE, mk<T>(a * e0.x + csw * s0[r].x, a * e0.y + csw * s0[r].y));
                __stcs(o + (size_t)((2 * c + 1) * dR + i) * TILE, mk<T>(a * e1.x + csw * s1[r].x, a * e1.y + csw * s1[r].y));
            }
    }
}

// canonical export: [V][c][2 dR][2 dR] complex, A_c = [[H, B], [B^+, -H]]; one thread per (site, c, row, column)
template <typename T> __global__ void clover_export_kernel(Geo g, int dR, cplx<T> *__restrict__ canon, const cplx<T> *__restrict__ clover) {
    const int n2 = 2 * dR, ne = dR * dR;
    const long per_site = 2L * n2 * n2;
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= 2L * g.Nh * per_site) return;
    const long site = idx / per_site;
    int q = (int)(idx - site * per_site);
    const int c = q / (n2 * n2);
    q -= c * n2 * n2;
    const int I = q / n2, J = q - I * n2;
    const int p = (int)(site / g.Nh), h = (int)(site - (long)p * g.Nh);
    const int tile = h >> 5, lane = h & 31;
    const int bi = I / dR, i = I - bi * dR, bj = J / dR, j = J - bj * dR;
    cplx<T> v;
    if (bi == bj) {
        v = clover[clover_off(g.n_tiles, p, tile, c, 0, i * dR + j, lane, ne)];
        if (bi) { v.x = -v.x; v.y = -v.y; }
    } else if (bi == 0) {
        v = clover[clover_off(g.n_tiles, p, tile, c, 1, i * dR + j, lane, ne)];
    } else {
        v = clover[clover_off(g.n_tiles, p, tile, c, 1, j * dR + i, lane, ne)];
        v.y = -v.y;
    }
    canon[(size_t)canonical_index(g, p, h) * per_site + (size_t)c * n2 * n2 + (size_t)I * n2 + J] = v;
}

// d_R <= 3: one thread per site, every matrix in registers (P, Q path products, C leaf sum, two accumulators).  Planes
// and leaves are run-time loops around ONE unrolled leaf body (a fully unrolled walk would be ~170 KB of code and
// instruction-fetch bound); the direction of step k of leaf l in plane (mu,nu) is s[(l+k)&3] with s = (mu, nu, -mu, -nu),
// the walk keeps the four coordinates in scalar registers.  Plane order 03,12 -> H_c ; 01,23,02,13 -> B_c.
template <typename T, bool REAL, int DR>
__global__ void __launch_bounds__(128) clover_field_site_kernel(Geo g, const link_elem<T, REAL> *__restrict__ links, cplx<T> *__restrict__ clover) {
    constexpr int NE = DR * DR;
    const long slot = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const int slots_half = g.n_tiles * TILE;
    if (slot >= 2L * slots_half) return;
    const int p = (int)(slot / slots_half), hp = (int)(slot - (long)p * slots_half);
    const bool live = hp < g.Nh;
    const int h = live ? hp : g.Nh - 1;
    int t0, x0, y0, zh0;
    decode_site(g, h, t0, x0, y0, zh0);
    const int z0 = 2 * zh0 + ((t0 + x0 + y0 + p) & 1);
    cplx<T> acc0[NE], acc1[NE];
    cplx<T> *dst = clover + clover_off(g.n_tiles, p, hp >> 5, 0, 0, 0, hp & 31, NE);
    for (int q = 0; q < 6; ++q) {
        const int pl = (0x415032 >> (4 * q)) & 7;                  // plane order 2,3,0,5,1,4  (03,12 | 01,23 | 02,13)
        const int mu = (0x211000 >> (4 * pl)) & 3, nu = (0x332321 >> (4 * pl)) & 3;
        if (q == 0 || q == 2) {
#pragma unroll
            for (int e = 0; e < NE; ++e) acc0[e] = acc1[e] = mk<T>(0, 0);
        }
        using PT = link_elem<T, REAL>;   // real links: real path products (a quarter of the multiply-adds)
        PT C[NE];
#pragma unroll
        for (int e = 0; e < NE; ++e) C[e] = PT{};
        for (int leaf = 0; leaf < 4; ++leaf) {
            int t = t0, x = x0, y = y0, z = z0, cp = p, ch = h;
            PT P[NE], Q[NE];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int sq = (leaf + k) & 3;
                const int dmu = (sq & 1) ? nu : mu, d = dmu + ((sq & 2) ? 4 : 0);
                const link_elem<T, REAL> *W = links + link_off(g.n_tiles, cp, ch >> 5, d, 0, ch & 31, NE);
                if (k == 0) {
#pragma unroll
                    for (int e = 0; e < NE; ++e) P[e] = W[(size_t)e * TILE];
                } else {
#pragma unroll
                    for (int e = 0; e < NE; ++e) Q[e] = PT{};
#pragma unroll
                    for (int l = 0; l < DR; ++l)
#pragma unroll
                        for (int j = 0; j < DR; ++j) {
                            const PT w = W[(size_t)(l * DR + j) * TILE];
#pragma unroll
                            for (int i = 0; i < DR; ++i) pfma<T>(Q[i * DR + j], P[i * DR + l], w);
                        }
#pragma unroll
                    for (int e = 0; e < NE; ++e) P[e] = Q[e];
                }
                const int dl = (sq & 2) ? -1 : 1;
                t += dmu == 0 ? dl : 0; x += dmu == 1 ? dl : 0; y += dmu == 2 ? dl : 0; z += dmu == 3 ? dl : 0;
                t = t == g.T ? 0 : (t < 0 ? g.T - 1 : t);
                x = x == g.L ? 0 : (x < 0 ? g.L - 1 : x);
                y = y == g.L ? 0 : (y < 0 ? g.L - 1 : y);
                z = z == g.L ? 0 : (z < 0 ? g.L - 1 : z);
                ch = encode_site(g, t, x, y, z >> 1);
                cp ^= 1;
            }
#pragma unroll
            for (int e = 0; e < NE; ++e) padd<T>(C[e], P[e]);
        }
        // F = (C - C^+)/8; (i/2) F -> K1 (planes 01, 23) or K3 (03, 12); F/2 = -i (i/2) F -> -i K2 (02, 13)
        const T s0 = (pl == 3 || pl == 5) ? T(-1) : T(1);          // c = 0: +F01 -F23 | +F02 +F13 | +F03 -F12
        const T s1 = (pl == 4) ? T(1) : T(-1);                     // c = 1: -F01 -F23 | -F02 +F13 | -F03 -F12
        const bool half = (pl == 1 || pl == 4);
#pragma unroll
        for (int i = 0; i < DR; ++i)
#pragma unroll
            for (int j = 0; j < DR; ++j) {
                const cplx<T> a = as_cplx<T>(C[i * DR + j]), b = as_cplx<T>(C[j * DR + i]);
                const cplx<T> F = mk<T>((a.x - b.x) * T(0.125), (a.y + b.y) * T(0.125));
                const cplx<T> v = half ? mk<T>(T(0.5) * F.x, T(0.5) * F.y) : mk<T>(-T(0.5) * F.y, T(0.5) * F.x);
                acc0[i * DR + j].x += s0 * v.x; acc0[i * DR + j].y += s0 * v.y;
                acc1[i * DR + j].x += s1 * v.x; acc1[i * DR + j].y += s1 * v.y;
            }
        if (q == 1 || q == 5) {                                     // H (m = 0) after 03,12; B (m = 1) after all four
            const int m = q == 1 ? 0 : 1;
#pragma unroll
            for (int e = 0; e < NE; ++e) {
                dst[(size_t)((0 * 2 + m) * NE + e) * TILE] = live ? acc0[e] : mk<T>(0, 0);
                dst[(size_t)((1 * 2 + m) * NE + e) * TILE] = live ? acc1[e] : mk<T>(0, 0);
            }
        }
    }
}
// d_R = 4, 5, 6: the register scheme of clover_field_site_kernel with the ROWS of every matrix split over the NS warps of a CTA
// (CTA = one tile, lane = site, warp w = rows w RP .. w RP + RP - 1).  A path product P <- P W needs, for the rows a thread owns,
// only those rows of P and the whole of W: every element of W is loaded once (coalesced, straight from L1 / L2 -- the NS warps of
// the CTA and the 12 leaves of neighbouring sites that use the same link hit there) and feeds RP complex MACs from registers; no
// shared-memory staging of the matrices at all (the shared-memory kernel above is bound by its two loads per MAC: 10 % of the FP32
// peak at d_R = 6).  Only C^+ in F = (C - C^+)/8 needs the other warps' rows: one exchange of the leaf sum per plane.
template <typename T, bool REAL, int DR, int NS, int MB>
__global__ void __launch_bounds__(32 * NS, MB) clover_field_rows_kernel(Geo g, const link_elem<T, REAL> *__restrict__ links, cplx<T> *__restrict__ clover) {
    static_assert(DR % NS == 0, "the rows must split evenly over the warps");
    constexpr int NE = DR * DR, RP = DR / NS, NR = RP * DR;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    link_elem<T, REAL> *exch = reinterpret_cast<link_elem<T, REAL> *>(smem_raw) + (threadIdx.x & 31);   // leaf sum C of the tile, [e][lane]
    const int lane = threadIdx.x & 31, r0 = (threadIdx.x >> 5) * RP;
    const int p = blockIdx.x / g.n_tiles, tile = blockIdx.x - p * g.n_tiles;
    const int hp = tile * TILE + lane;
    const bool live = hp < g.Nh;
    const int h = live ? hp : g.Nh - 1;
    int t0, x0, y0, zh0;
    decode_site(g, h, t0, x0, y0, zh0);
    const int z0 = 2 * zh0 + ((t0 + x0 + y0 + p) & 1);
    cplx<T> acc0[NR], acc1[NR];
    cplx<T> *dst = clover + clover_off(g.n_tiles, p, tile, 0, 0, 0, lane, NE);
    for (int q = 0; q < 6; ++q) {
        const int pl = (0x415032 >> (4 * q)) & 7;                  // plane order 2,3,0,5,1,4  (03,12 | 01,23 | 02,13)
        const int mu = (0x211000 >> (4 * pl)) & 3, nu = (0x332321 >> (4 * pl)) & 3;
        if (q == 0 || q == 2) {
#pragma unroll
            for (int e = 0; e < NR; ++e) acc0[e] = acc1[e] = mk<T>(0, 0);
        }
        using PT = link_elem<T, REAL>;   // real links: real path products (a quarter of the multiply-adds)
        PT C[NR];
#pragma unroll
        for (int e = 0; e < NR; ++e) C[e] = PT{};
        for (int leaf = 0; leaf < 4; ++leaf) {
            int t = t0, x = x0, y = y0, z = z0, cp = p, ch = h;
            PT P[NR], Q[NR];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int sq = (leaf + k) & 3;
                const int dmu = (sq & 1) ? nu : mu, d = dmu + ((sq & 2) ? 4 : 0);
                const link_elem<T, REAL> *W = links + link_off(g.n_tiles, cp, ch >> 5, d, 0, ch & 31, NE);
                if (k == 0) {
#pragma unroll
                    for (int rr = 0; rr < RP; ++rr)
#pragma unroll
                        for (int j = 0; j < DR; ++j) P[rr * DR + j] = W[(size_t)((r0 + rr) * DR + j) * TILE];
                } else {
#pragma unroll
                    for (int e = 0; e < NR; ++e) Q[e] = PT{};
#pragma unroll
                    for (int l = 0; l < DR; ++l)
#pragma unroll
                        for (int j = 0; j < DR; ++j) {
                            const PT w = W[(size_t)(l * DR + j) * TILE];
#pragma unroll
                            for (int rr = 0; rr < RP; ++rr) pfma<T>(Q[rr * DR + j], P[rr * DR + l], w);
                        }
#pragma unroll
                    for (int e = 0; e < NR; ++e) P[e] = Q[e];
                }
                const int dl = (sq & 2) ? -1 : 1;
                t += dmu == 0 ? dl : 0; x += dmu == 1 ? dl : 0; y += dmu == 2 ? dl : 0; z += dmu == 3 ? dl : 0;
                t = t == g.T ? 0 : (t < 0 ? g.T - 1 : t);
                x = x == g.L ? 0 : (x < 0 ? g.L - 1 : x);
                y = y == g.L ? 0 : (y < 0 ? g.L - 1 : y);
                z = z == g.L ? 0 : (z < 0 ? g.L - 1 : z);
                ch = encode_site(g, t, x, y, z >> 1);
                cp ^= 1;
            }
#pragma unroll
            for (int e = 0; e < NR; ++e) padd<T>(C[e], P[e]);
        }
        // the leaf sum to shared memory: row i of C^+ is column i of C, whose entries the other warps hold
        __syncthreads();                                            // the previous plane's reads are done
#pragma unroll
        for (int rr = 0; rr < RP; ++rr)
#pragma unroll
            for (int j = 0; j < DR; ++j) exch[(size_t)((r0 + rr) * DR + j) * TILE] = C[rr * DR + j];
        __syncthreads();
        // F = (C - C^+)/8; (i/2) F -> K1 (planes 01, 23) or K3 (03, 12); F/2 = -i (i/2) F -> -i K2 (02, 13)
        const T s0 = (pl == 3 || pl == 5) ? T(-1) : T(1);          // c = 0: +F01 -F23 | +F02 +F13 | +F03 -F12
        const T s1 = (pl == 4) ? T(1) : T(-1);                     // c = 1: -F01 -F23 | -F02 +F13 | -F03 -F12
        const bool half = (pl == 1 || pl == 4);
#pragma unroll
        for (int rr = 0; rr < RP; ++rr)
#pragma unroll
            for (int j = 0; j < DR; ++j) {
                const cplx<T> a = as_cplx<T>(C[rr * DR + j]), b = as_cplx<T>(exch[(size_t)(j * DR + r0 + rr) * TILE]);
                const cplx<T> F = mk<T>((a.x - b.x) * T(0.125), (a.y + b.y) * T(0.125));
                const cplx<T> v = half ? mk<T>(T(0.5) * F.x, T(0.5) * F.y) : mk<T>(-T(0.5) * F.y, T(0.5) * F.x);
                acc0[rr * DR + j].x += s0 * v.x; acc0[rr * DR + j].y += s0 * v.y;
                acc1[rr * DR + j].x += s1 * v.x; acc1[rr * DR + j].y += s1 * v.y;
            }
        if (q == 1 || q == 5) {                                     // H (m = 0) after 03,12; B (m = 1) after all four
            const int m = q == 1 ? 0 : 1;
#pragma unroll
            for (int rr = 0; rr < RP; ++rr)
#pragma unroll
                for (int j = 0; j < DR; ++j) {
                    const int e = (r0 + rr) * DR + j;
                    dst[(size_t)((0 * 2 + m) * NE + e) * TILE] = live ? acc0[rr * DR + j] : mk<T>(0, 0);
                    dst[(size_t)((1 * 2 + m) * NE + e) * TILE] = live ? acc1[rr * DR + j] : mk<T>(0, 0);
                }
        }
    }
}
template <typename T, bool REAL, int DR, int NS, int MB = 1> static int clover_field_rows_t(const Geo &g, void *clover, const void *links, cudaStream_t s) {
    auto kern = clover_field_rows_kernel<T, REAL, DR, NS, MB>;
    const size_t smem = (size_t)DR * DR * TILE * sizeof(cplx<T>);
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, smem, cache, n_sm)) return rc;      // d_R = 10 in fp64 needs the opt-in size (51 KB)
    kern<<<2 * g.n_tiles, 32 * NS, smem, s>>>(g, (const link_elem<T, REAL> *)links, (cplx<T> *)clover);
    return (int)cudaGetLastError();
}
template <typename T, bool REAL, int DR> static int clover_field_site_t(const Geo &g, void *clover, const void *links, cudaStream_t s) {
    const long slots = 2L * g.n_tiles * TILE;
    clover_field_site_kernel<T, REAL, DR><<<(unsigned)((slots + 127) / 128), 128, 0, s>>>(g, (const link_elem<T, REAL> *)links, (cplx<T> *)clover);
    return (int)cudaGetLastError();
}

template <typename T, bool REAL> static int clover_field_t(const Geo &g, int dR, void *clover, const void *links, cudaStream_t s) {
    if (dR == 2) return clover_field_site_t<T, REAL, 2>(g, clover, links, s);
    if (dR == 3) return clover_field_site_t<T, REAL, 3>(g, clover, links, s);
    static const int smk = getenv("HIREP_CLOVER_FIELD_SMEM") ? atoi(getenv("HIREP_CLOVER_FIELD_SMEM")) : 0;   // measurement switch: the shared-memory kernel
    if (REAL && !smk) {    // SU(3) adjoint (d_R = 8, real links): two rows per thread in fp32, one in fp64
        if constexpr (REAL) {
            if (dR == 8) return clover_field_rows_t<T, true, 8, sizeof(T) == 4 ? 4 : 8, 1>(g, clover, links, s);
        }
    }
    if (!REAL && !smk) {   // d_R = 4, 5, 6, 10 are complex representations; rows per thread chosen for <= ~200 registers
        if constexpr (!REAL) {
            constexpr bool F32 = sizeof(T) == 4;
            if (dR == 10) return clover_field_rows_t<T, false, 10, F32 ? 5 : 10, 1>(g, clover, links, s);
            if (dR == 4) return clover_field_rows_t<T, false, 4, 2>(g, clover, links, s);
            if (dR == 5) return clover_field_rows_t<T, false, 5, 5>(g, clover, links, s);
            // d_R = 6: fp32 two warps x 3 rows; fp64 six warps x 1 row at two CTAs per SM (three warps x 2 rows need 255 registers: 36.7 vs 24.2 ms
            // for SU(3) SYM on 32^4; the shared-memory kernel: 40.4 ms)
            if (dR == 6) {
                if constexpr (F32) return clover_field_rows_t<T, false, 6, 2, 1>(g, clover, links, s);
                else return clover_field_rows_t<T, false, 6, 6, 2>(g, clover, links, s);
            }
        }
    }
    constexpr int LP = 1;
    const int ne = dR * dR;
    const size_t per_site = (size_t)(6 * LP + 1) * ne * sizeof(link_elem<T, REAL>) + (size_t)4 * ne * sizeof(cplx<T>);   // W[4 LP], P[LP], Q[LP], C + acc[4]
    int S = TILE;
    while (S > 1 && per_site * S > (size_t)200 * 1024) S >>= 1;
    int rows = 512 / S / dR;                       // blockDim.y = rows * dR: each thread owns one column of `rows`-strided rows
    rows = rows < 1 ? 1 : rows > dR ? dR : rows;
    const int nw = rows * dR;
    auto kern = dR == 2 ? clover_field_kernel<T, REAL, LP, 2> : dR == 3 ? clover_field_kernel<T, REAL, LP, 3>
              : dR == 4 ? clover_field_kernel<T, REAL, LP, 4> : dR == 6 ? clover_field_kernel<T, REAL, LP, 6>
              : clover_field_kernel<T, REAL, LP, 0>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_site * S));
    if (e != cudaSuccess) return (int)e;
    kern<<<2 * g.n_tiles * (TILE / S), dim3(S, nw), per_site * S, s>>>(g, dR, (const link_elem<T, REAL> *)links, (cplx<T> *)clover);
    return (int)cudaGetLastError();
}

int k_clover_field(const Geo &g, int prec, int dR, int real, void *clover, const void *links_rep, cudaStream_t s) {
    if (prec == 0) return real ? clover_field_t<double, true>(g, dR, clover, links_rep, s) : clover_field_t<double, false>(g, dR, clover, links_rep, s);
    return real ? clover_field_t<float, true>(g, dR, clover, links_rep, s) : clover_field_t<float, false>(g, dR, clover, links_rep, s);
}

template <typename T, int DR> static int cphi_site_t(int ntile, double a, double csw, const void *clover, const void *in, void *out, cudaStream_t s) {
    const int blocks = (ntile + 3) / 4;
    cphi_site_kernel<T, DR><<<blocks < 148 * 16 ? blocks : 148 * 16, 128, 0, s>>>(ntile, (T)a, (T)csw, (const cplx<T> *)clover, (const cplx<T> *)in,
                                                                                 (cplx<T> *)out);
    return (int)cudaGetLastError();
}
template <typename T> static int cphi_t(int ntile, int dR, double a, double csw, const void *clover, const void *in, void *out, cudaStream_t s) {
    switch (dR) {
    case 2: return cphi_site_t<T, 2>(ntile, a, csw, clover, in, out, s);
    case 3: return cphi_site_t<T, 3>(ntile, a, csw, clover, in, out, s);
    case 4: return cphi_site_t<T, 4>(ntile, a, csw, clover, in, out, s);
    case 5: return cphi_site_t<T, 5>(ntile, a, csw, clover, in, out, s);
    case 6: return cphi_site_t<T, 6>(ntile, a, csw, clover, in, out, s);
    case 8: return cphi_site_t<T, 8>(ntile, a, csw, clover, in, out, s);
    case 10: return cphi_site_t<T, 10>(ntile, a, csw, clover, in, out, s);
    }
    static const int generic = getenv("HIREP_CPHI_GENERIC") ? atoi(getenv("HIREP_CPHI_GENERIC")) : 0;   // measurement switch: the round-1 kernel
    if (dR >= 12 && !generic) {   // row groups: R = 5 where it divides d_R (15, 35), else 4 (24) or 3 (21)
        const int R = dR % 5 == 0 ? 5 : dR % 4 == 0 ? 4 : 3;
        const long units = (long)ntile * 2 * ((dR + R - 1) / R);
        const int grid = (int)((units + 7) / 8 < 148 * 2 ? (units + 7) / 8 : 148 * 2);
        if (R == 5) cphi_rows_kernel<T, 5><<<grid, 256, 0, s>>>(ntile, dR, (T)a, (T)csw, (const cplx<T> *)clover, (const cplx<T> *)in, (cplx<T> *)out);
        else if (R == 4) cphi_rows_kernel<T, 4><<<grid, 256, 0, s>>>(ntile, dR, (T)a, (T)csw, (const cplx<T> *)clover, (const cplx<T> *)in, (cplx<T> *)out);
        else cphi_rows_kernel<T, 3><<<grid, 256, 0, s>>>(ntile, dR, (T)a, (T)csw, (const cplx<T> *)clover, (const cplx<T> *)in, (cplx<T> *)out);
        return (int)cudaGetLastError();
    }
    const int wy = 2 * dR < 8 ? 2 * dR : 8;      // 8 warps per CTA, 3-4 CTAs per SM (one 16-warp CTA per SM was latency bound: 2.9 TB/s)
    int grid = ntile < 148 * 16 ? ntile : 148 * 16;   // (one CTA per SM measured slower: 4.7 vs 4.1 ms at d_R = 35 fp64)
    cphi_kernel<T><<<grid, dim3(TILE, wy), 0, s>>>(ntile, dR, (T)a, (T)csw, (const cplx<T> *)clover, (const cplx<T> *)in, (cplx<T> *)out);
    return (int)cudaGetLastError();
}
// ntile tiles starting at the given pointers (2 n_tiles = full lattice; n_tiles with the parity's offsets = one half)
int k_cphi(int prec, int dR, int ntile, double a, double csw, const void *clover, const void *in, void *out, cudaStream_t s) {
    return prec == 0 ? cphi_t<double>(ntile, dR, a, csw, clover, in, out, s) : cphi_t<float>(ntile, dR, a, csw, clover, in, out, s);
}

// ---- inverse of the diagonal blocks, for the Schur form Eq 43 (L803) with the clover term ---------------------------
// inv field of ONE parity: [tile][c][E = I*2dR + J][lane] complex<T>, the full (2 dR)^2 block of ((4+m) + c_sw A_c)^{-1}.
// One thread per site and chirality: the block is written to the thread's own column of the output buffer (coalesced
// across lanes) and inverted there in place by Gauss-Jordan elimination without pivoting -- the blocks are Hermitian and,
// for the parameters the operator is used with ((4+m) dominates c_sw |A|), positive definite.  Once per gauge update.
// DRT > 0 (small d_R): compile-time d_R, one warp per block, the warp's 32 blocks live in SHARED memory [entry][lane] while they are
// eliminated (each lane its own column: no exchange, no barrier) and are copied out at the end -- the same operations in the same
// order as the in-place form, whose every elimination step is a round trip of the whole block through L2 (C2 fp64 3.4 -> 0.5 ms).
// DRT = 0: run-time d_R, in place in global memory (blocks too large for shared memory).
template <typename T, int DRT>
__global__ void clover_inv_kernel(Geo g, int dR_rt, int parity, T a, T csw, const cplx<T> *__restrict__ clover, cplx<T> *inv, int *flags) {
    const int dR = DRT > 0 ? DRT : dR_rt;
    const int n = 2 * dR, ne = dR * dR;
    const int slot = blockIdx.x * blockDim.x + threadIdx.x;      // padded site slot of the parity
    const int c = blockIdx.y;
    if (slot >= g.n_tiles * TILE) return;
    const int tile = slot >> 5, lane = slot & 31;
    cplx<T> *G = inv + ((size_t)(tile * 2 + c) * n * n) * TILE + lane;
    extern __shared__ __align__(16) unsigned char smem_blk[];
    cplx<T> *M = DRT > 0 ? reinterpret_cast<cplx<T> *>(smem_blk) + (size_t)(threadIdx.x >> 5) * n * n * TILE + lane : G;
    const bool live = slot < g.Nh;
    T scale = 0;                                                  // largest |entry| of the block: the yardstick for the pivots
    for (int I = 0; I < n; ++I)
        for (int J = 0; J < n; ++J) {
            const int bi = I / dR, i = I - bi * dR, bj = J / dR, j = J - bj * dR;
            cplx<T> v;
            if (bi == bj) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 0, i * dR + j, lane, ne)];
                if (bi) { v.x = -v.x; v.y = -v.y; }
            } else if (bi == 0) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, i * dR + j, lane, ne)];
            } else {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, j * dR + i, lane, ne)];
                v.y = -v.y;
            }
            v.x *= csw; v.y *= csw;
            if (I == J) v.x += a;
            if (!live) v = mk<T>(I == J ? T(1) : T(0), T(0));    // padding lanes: identity, inverted harmlessly, zeroed below
            M[(size_t)(I * n + J) * TILE] = v;
            scale = fmax(scale, fmax(fabs(v.x), fabs(v.y)));
        }
    // elimination without pivoting is only safe for well-conditioned (positive definite) blocks: a pivot that is tiny against the
    // block, or not finite, is reported through the geometry's device flags (hirep_sync returns HIREP_EBREAKDOWN)
    const T tiny = scale * (sizeof(T) == 8 ? T(1e-10) : T(1e-4));
    bool bad = false;
    for (int k = 0; k < n; ++k) {
        const cplx<T> d = M[(size_t)(k * n + k) * TILE];
        const T d2 = d.x * d.x + d.y * d.y;
        if (!(d2 > tiny * tiny) || !isfinite(d2)) bad = true;
        const T r = T(1) / d2;
        const cplx<T> p = mk<T>(d.x * r, -d.y * r);
        M[(size_t)(k * n + k) * TILE] = mk<T>(1, 0);
        for (int J = 0; J < n; ++J) M[(size_t)(k * n + J) * TILE] = cmul<T>(M[(size_t)(k * n + J) * TILE], p);
        for (int I = 0; I < n; ++I) {
            if (I == k) continue;
            const cplx<T> f = M[(size_t)(I * n + k) * TILE];
            M[(size_t)(I * n + k) * TILE] = mk<T>(0, 0);
            for (int J = 0; J < n; ++J) {
                const cplx<T> x = M[(size_t)(k * n + J) * TILE];
                cplx<T> y = M[(size_t)(I * n + J) * TILE];
                y.x -= f.x * x.x - f.y * x.y;
                y.y -= f.x * x.y + f.y * x.x;
                M[(size_t)(I * n + J) * TILE] = y;
            }
        }
    }
    if (!live)
        for (int E = 0; E < n * n; ++E) M[(size_t)E * TILE] = mk<T>(0, 0);
    if (DRT > 0)
        for (int E = 0; E < n * n; ++E) G[(size_t)E * TILE] = M[(size_t)E * TILE];
    if (bad && live && flags) atomicOr(flags, 1);
}

// out = block * in per chirality with the full (2 dR)^2 blocks of one parity (n_tiles tiles).
template <typename T, int DR>
__global__ void __launch_bounds__(128) cblock_site_kernel(int ntile, const cplx<T> *__restrict__ blk, const cplx<T> *__restrict__ in,
                                                          cplx<T> *__restrict__ out) {
    constexpr int N = 2 * DR, NCOMP = 4 * DR;
    const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    for (int tile = blockIdx.x * wpb + (threadIdx.x >> 5); tile < ntile; tile += gridDim.x * wpb) {
        const cplx<T> *psi = in + (size_t)tile * NCOMP * TILE + lane;
        cplx<T> *o = out + (size_t)tile * NCOMP * TILE + lane;
#pragma unroll
        for (int c = 0; c < 2; ++c) {
            const cplx<T> *M = blk + (size_t)(tile * 2 + c) * N * N * TILE + lane;
            cplx<T> v[N];
#pragma unroll
            for (int J = 0; J < N; ++J) v[J] = __ldg(psi + (size_t)(c * N + J) * TILE);
#pragma unroll
            for (int I = 0; I < N; ++I) {
                cplx<T> s = mk<T>(0, 0);
#pragma unroll
                for (int J = 0; J < N; ++J) cfma<T>(s, __ldcs(M + (size_t)(I * N + J) * TILE), v[J]);
                __stcs(o + (size_t)(c * N + I) * TILE, s);
            }
        }
    }
}
// any d_R: warp y of block (32, WY) computes rows (c, I) = y, y + WY, ... of the block's tile
template <typename T>
__global__ void __launch_bounds__(256, sizeof(T) == 8 ? 4 : 3) cblock_kernel(int ntile, int dR, const cplx<T> *__restrict__ blk,
                                                                             const cplx<T> *__restrict__ in, cplx<T> *__restrict__ out) {
    const int n = 2 * dR, ncomp = 4 * dR, lane = threadIdx.x;
    for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
        const cplx<T> *psi = in + (size_t)tile * ncomp * TILE + lane;
        cplx<T> *o = out + (size_t)tile * ncomp * TILE + lane;
        for (int q = threadIdx.y; q < 2 * n; q += blockDim.y) {
            const int c = q / n, I = q - c * n;
            const cplx<T> *M = blk + ((size_t)(tile * 2 + c) * n * n + (size_t)I * n) * TILE + lane;
            const cplx<T> *v = psi + (size_t)c * n * TILE;
            cplx<T> s0 = mk<T>(0, 0), s1 = mk<T>(0, 0);
            int J = 0;
#pragma unroll 4
            for (; J + 1 < n; J += 2) {
                cfma<T>(s0, __ldg(M + (size_t)J * TILE), __ldg(v + (size_t)J * TILE));
                cfma<T>(s1, __ldg(M + (size_t)(J + 1) * TILE), __ldg(v + (size_t)(J + 1) * TILE));
            }
            __stcs(o + (size_t)(c * n + I) * TILE, mk<T>(s0.x + s1.x, s0.y + s1.y));
        }
    }
}

// Large d_R: R consecutive rows of a chirality block per warp, one load of v_J serving R rows (see cphi_rows_kernel)
template <typename T, int R>
__global__ void __launch_bounds__(256, 2) cblock_rows_kernel(int ntile, int dR, const cplx<T> *__restrict__ blk, const cplx<T> *__restrict__ in,
                                                             cplx<T> *__restrict__ out) {
    const int n = 2 * dR, ncomp = 4 * dR, lane = threadIdx.x & 31;
    const int groups = (n + R - 1) / R, upt = 2 * groups;
    const long n_units = (long)ntile * upt;
    const long gw = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), nw = (long)gridDim.x * (blockDim.x >> 5);
    for (long u = gw; u < n_units; u += nw) {
        const int tile = (int)(u / upt), q = (int)(u - (long)tile * upt), c = q / groups, I0 = (q - c * groups) * R;
        const cplx<T> *v = in + ((size_t)tile * ncomp + (size_t)c * n) * TILE + lane;
        const cplx<T> *M = blk + ((size_t)(tile * 2 + c) * n * n) * TILE + lane;
        size_t rowoff[R];
#pragma unroll
        for (int r = 0; r < R; ++r) rowoff[r] = (size_t)(I0 + r < n ? I0 + r : n - 1) * n;
        cplx<T> acc[R];
#pragma unroll
        for (int r = 0; r < R; ++r) acc[r] = mk<T>(0, 0);
#pragma unroll 2
        for (int J = 0; J < n; ++J) {
            const cplx<T> x = __ldg(v + (size_t)J * TILE);
            cplx<T> m[R];
#pragma unroll
            for (int r = 0; r < R; ++r) m[r] = __ldcs(M + (rowoff[r] + J) * TILE);
#pragma unroll
            for (int r = 0; r < R; ++r) cfma<T>(acc[r], m[r], x);
        }
        cplx<T> *o = out + ((size_t)tile * ncomp + (size_t)c * n) * TILE + lane;
#pragma unroll
        for (int r = 0; r < R; ++r)
            if (I0 + r < n) __stcs(o + (size_t)(I0 + r) * TILE, acc[r]);
    }
}

template <typename T, int DR> static int cblock_site_t(int ntile, const void *blk, const void *in, void *out, cudaStream_t s) {
    const int blocks = (ntile + 3) / 4;
    cblock_site_kernel<T, DR><<<blocks < 148 * 16 ? blocks : 148 * 16, 128, 0, s>>>(ntile, (const cplx<T> *)blk, (const cplx<T> *)in, (cplx<T> *)out);
    return (int)cudaGetLastError();
}
template <typename T> static int cblock_t(int ntile, int dR, const void *blk, const void *in, void *out, cudaStream_t s) {
    switch (dR) {
    case 2: return cblock_site_t<T, 2>(ntile, blk, in, out, s);
    case 3: return cblock_site_t<T, 3>(ntile, blk, in, out, s);
    case 4: return cblock_site_t<T, 4>(ntile, blk, in, out, s);
    case 5: return cblock_site_t<T, 5>(ntile, blk, in, out, s);
    case 6: return cblock_site_t<T, 6>(ntile, blk, in, out, s);
    }
    static const int generic = getenv("HIREP_CPHI_GENERIC") ? atoi(getenv("HIREP_CPHI_GENERIC")) : 0;   // measurement switch: the round-1 kernel
    if (dR >= 8 && !generic) {   // row groups of 5 where that divides 2 d_R (10, 15, 35), else 6 (21, 24) or 4 (8)
        const int n = 2 * dR, R = n % 5 == 0 ? 5 : n % 6 == 0 ? 6 : 4;
        const long units = (long)ntile * 2 * ((n + R - 1) / R);
        const int grid = (int)((units + 7) / 8 < 148 * 2 ? (units + 7) / 8 : 148 * 2);
        if (R == 5) cblock_rows_kernel<T, 5><<<grid, 256, 0, s>>>(ntile, dR, (const cplx<T> *)blk, (const cplx<T> *)in, (cplx<T> *)out);
        else if (R == 6) cblock_rows_kernel<T, 6><<<grid, 256, 0, s>>>(ntile, dR, (const cplx<T> *)blk, (const cplx<T> *)in, (cplx<T> *)out);
        else cblock_rows_kernel<T, 4><<<grid, 256, 0, s>>>(ntile, dR, (const cplx<T> *)blk, (const cplx<T> *)in, (cplx<T> *)out);
        return (int)cudaGetLastError();
    }
    const int wy = 4 * dR < 8 ? 4 * dR : 8;
    cblock_kernel<T><<<ntile < 148 * 16 ? ntile : 148 * 16, dim3(TILE, wy), 0, s>>>(ntile, dR, (const cplx<T> *)blk, (const cplx<T> *)in, (cplx<T> *)out);
    return (int)cudaGetLastError();
}
int k_cblock(int prec, int dR, int ntile, const void *blk, const void *in, void *out, cudaStream_t s) {
    return prec == 0 ? cblock_t<double>(ntile, dR, blk, in, out, s) : cblock_t<float>(ntile, dR, blk, in, out, s);
}
// Exponential clover (Eq 50): blocks pref * exp(x A_c) of one parity, x = +-c_sw/(4+m0), pref = (4+m0) or 1/(4+m0)
// (the inverse).  Per site and chirality, in the thread's own columns of global memory (S = output, X and Tm = workspace):
// scaling and squaring, exp(Y) = (sum_{k <= K} (Y/2^s)^k / k!)^(2^s) with the sum in Horner form; s = 4, K = 14 covers
// |x A| <= 8 to 1e-16 (truncation 0.5^15/15!) and the four squarings amplify rounding by 16 ulp.
// DRT > 0: compile-time d_R, one warp per block, S, X and the product buffer in shared memory (as clover_inv_kernel; the copy of
// every product back into S is replaced by swapping the two buffers); DRT = 0: run-time d_R in global-memory columns.
template <typename T, int DRT>
__global__ void clover_exp_kernel(Geo g, int dR_rt, int parity, T x, T pref, const cplx<T> *__restrict__ clover, cplx<T> *blocks, cplx<T> *work, int *flags) {
    constexpr int SQ = 4, K = 14;
    const int dR = DRT > 0 ? DRT : dR_rt;
    const int n = 2 * dR, ne = dR * dR;
    const int slot = blockIdx.x * blockDim.x + threadIdx.x;
    const int c = blockIdx.y;
    if (slot >= g.n_tiles * TILE) return;
    const int tile = slot >> 5, lane = slot & 31;
    const size_t off = ((size_t)(tile * 2 + c) * n * n) * TILE + lane;
    extern __shared__ __align__(16) unsigned char smem_blk[];
    cplx<T> *const sm = reinterpret_cast<cplx<T> *>(smem_blk) + (size_t)(threadIdx.x >> 5) * 3 * n * n * TILE + lane;
    cplx<T> *const G = blocks + off;
    cplx<T> *S = DRT > 0 ? sm : G, *X = DRT > 0 ? sm + (size_t)n * n * TILE : work + off;
    cplx<T> *Tm = DRT > 0 ? sm + (size_t)2 * n * n * TILE : work + (size_t)g.n_tiles * 2 * n * n * TILE + off;
    const bool live = slot < g.Nh;
    const T sc = x / T(1 << SQ);
    T norm = 0;                                                   // inf-norm of x A_c: the series below is accurate for <= 8
    for (int I = 0; I < n; ++I) {
        T rowsum = 0;
        for (int J = 0; J < n; ++J) {
            const int bi = I / dR, i = I - bi * dR, bj = J / dR, j = J - bj * dR;
            cplx<T> v;
            if (bi == bj) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 0, i * dR + j, lane, ne)];
                if (bi) { v.x = -v.x; v.y = -v.y; }
            } else if (bi == 0) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, i * dR + j, lane, ne)];
            } else {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, j * dR + i, lane, ne)];
                v.y = -v.y;
            }
            X[(size_t)(I * n + J) * TILE] = mk<T>(sc * v.x, sc * v.y);
            S[(size_t)(I * n + J) * TILE] = mk<T>(I == J ? T(1) : T(0), T(0));
            rowsum += sqrt(v.x * v.x + v.y * v.y);
        }
        norm = fmax(norm, fabs(x) * rowsum);
    }
    if (live && flags && (!(norm <= T(8)) )) atomicOr(flags, 2);   // also catches NaN
    for (int k = K; k >= 1; --k) {            // S <- 1 + (X S)/k
        const T rk = T(1) / T(k);
        for (int I = 0; I < n; ++I) {
            cplx<T> xr[DRT > 0 ? 2 * DRT : 1];     // shared-memory form: row I of the left factor in registers (one load per MAC instead of two)
            if (DRT > 0) {
#pragma unroll
                for (int l = 0; l < 2 * DRT; ++l) xr[l] = X[(size_t)(I * n + l) * TILE];
            }
            for (int J = 0; J < n; ++J) {
                cplx<T> a = mk<T>(0, 0);
#pragma unroll
                for (int l = 0; l < (DRT > 0 ? 2 * DRT : n); ++l) cfma<T>(a, DRT > 0 ? xr[DRT > 0 ? l : 0] : X[(size_t)(I * n + l) * TILE], S[(size_t)(l * n + J) * TILE]);
                Tm[(size_t)(I * n + J) * TILE] = mk<T>(a.x * rk + (I == J ? T(1) : T(0)), a.y * rk);
            }
        }
        if (DRT > 0) { cplx<T> *t_ = S; S = Tm; Tm = t_; }
        else for (int E = 0; E < n * n; ++E) S[(size_t)E * TILE] = Tm[(size_t)E * TILE];
    }
    for (int q = 0; q < SQ; ++q) {            // S <- S S
        for (int I = 0; I < n; ++I) {
            cplx<T> xr[DRT > 0 ? 2 * DRT : 1];
            if (DRT > 0) {
#pragma unroll
                for (int l = 0; l < 2 * DRT; ++l) xr[l] = S[(size_t)(I * n + l) * TILE];
            }
            for (int J = 0; J < n; ++J) {
                cplx<T> a = mk<T>(0, 0);
#pragma unroll
                for (int l = 0; l < (DRT > 0 ? 2 * DRT : n); ++l) cfma<T>(a, DRT > 0 ? xr[DRT > 0 ? l : 0] : S[(size_t)(I * n + l) * TILE], S[(size_t)(l * n + J) * TILE]);
                Tm[(size_t)(I * n + J) * TILE] = a;
            }
        }
        if (DRT > 0) { cplx<T> *t_ = S; S = Tm; Tm = t_; }
        else for (int E = 0; E < n * n; ++E) S[(size_t)E * TILE] = Tm[(size_t)E * TILE];
    }
    for (int E = 0; E < n * n; ++E) {
        const cplx<T> v = S[(size_t)E * TILE];
        G[(size_t)E * TILE] = live ? mk<T>(pref * v.x, pref * v.y) : mk<T>(0, 0);
    }
}
// Row-split form (small d_R): CTA = (tile, chirality), lane = site, warp w owns the rows w RP .. of X, S and of every product.
// A product T = L R needs the thread's rows of L (registers) and all of R: the warps publish their rows of S to ONE shared-memory
// copy [entry][lane], and every element read from there feeds RP complex MACs -- against three full matrices per site in shared
// memory (two warps per SM at d_R = 6 fp32) and two loads per MAC in clover_exp_kernel<T, DRT>.  Same operations in the same order
// per entry: bit-identical results.
template <typename T, int DR, int RP>
__global__ void __launch_bounds__(32 * (2 * DR / RP)) clover_exp_rows_kernel(Geo g, int parity, T x, T pref, const cplx<T> *__restrict__ clover,
                                                                            cplx<T> *blocks, int *flags) {
    constexpr int SQ = 4, K = 14, n = 2 * DR, ne = DR * DR;
    static_assert(n % RP == 0, "rows must split evenly");
    extern __shared__ __align__(16) unsigned char smem_blk[];
    const int lane = threadIdx.x & 31, r0 = (threadIdx.x >> 5) * RP;
    const int tile = blockIdx.x, c = blockIdx.y;
    cplx<T> *R = reinterpret_cast<cplx<T> *>(smem_blk) + lane;               // the right factor S, [I n + J][lane]
    const bool live = tile * TILE + lane < g.Nh;
    const T sc = x / T(1 << SQ);
    cplx<T> X[RP][n], S[RP][n], Tm[RP][n];
    T norm = 0;
#pragma unroll
    for (int rr = 0; rr < RP; ++rr) {
        const int I = r0 + rr, bi = I / DR, i = I - bi * DR;
        T rowsum = 0;
#pragma unroll
        for (int J = 0; J < n; ++J) {
            const int bj = J / DR, j = J - bj * DR;
            cplx<T> v;
            if (bi == bj) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 0, i * DR + j, lane, ne)];
                if (bi) { v.x = -v.x; v.y = -v.y; }
            } else if (bi == 0) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, i * DR + j, lane, ne)];
            } else {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, j * DR + i, lane, ne)];
                v.y = -v.y;
            }
            X[rr][J] = mk<T>(sc * v.x, sc * v.y);
            S[rr][J] = mk<T>(I == J ? T(1) : T(0), T(0));
            rowsum += sqrt(v.x * v.x + v.y * v.y);
        }
        norm = fmax(norm, fabs(x) * rowsum);
    }
    if (live && flags && (!(norm <= T(8)))) atomicOr(flags, 2);   // a row of |x A| beyond the range of the series (also catches NaN)
    auto publish = [&]() {
        __syncthreads();                                            // the previous product's reads are done
#pragma unroll
        for (int rr = 0; rr < RP; ++rr)
#pragma unroll
            for (int J = 0; J < n; ++J) R[(size_t)((r0 + rr) * n + J) * TILE] = S[rr][J];
        __syncthreads();
    };
    for (int k = K; k >= 1; --k) {            // S <- 1 + (X S)/k
        const T rk = T(1) / T(k);
        publish();
#pragma unroll
        for (int J = 0; J < n; ++J) {
            cplx<T> a[RP];
#pragma unroll
            for (int rr = 0; rr < RP; ++rr) a[rr] = mk<T>(0, 0);
#pragma unroll
            for (int l = 0; l < n; ++l) {
                const cplx<T> s = R[(size_t)(l * n + J) * TILE];
#pragma unroll
                for (int rr = 0; rr < RP; ++rr) cfma<T>(a[rr], X[rr][l], s);
            }
#pragma unroll
            for (int rr = 0; rr < RP; ++rr) Tm[rr][J] = mk<T>(a[rr].x * rk + (r0 + rr == J ? T(1) : T(0)), a[rr].y * rk);
        }
#pragma unroll
        for (int rr = 0; rr < RP; ++rr)
#pragma unroll
            for (int J = 0; J < n; ++J) S[rr][J] = Tm[rr][J];
    }
    for (int q = 0; q < SQ; ++q) {            // S <- S S
        publish();
#pragma unroll
        for (int J = 0; J < n; ++J) {
            cplx<T> a[RP];
#pragma unroll
            for (int rr = 0; rr < RP; ++rr) a[rr] = mk<T>(0, 0);
#pragma unroll
            for (int l = 0; l < n; ++l) {
                const cplx<T> s = R[(size_t)(l * n + J) * TILE];
#pragma unroll
                for (int rr = 0; rr < RP; ++rr) cfma<T>(a[rr], S[rr][l], s);
            }
#pragma unroll
            for (int rr = 0; rr < RP; ++rr) Tm[rr][J] = a[rr];
        }
#pragma unroll
        for (int rr = 0; rr < RP; ++rr)
#pragma unroll
            for (int J = 0; J < n; ++J) S[rr][J] = Tm[rr][J];
    }
    cplx<T> *G = blocks + ((size_t)(tile * 2 + c) * n * n) * TILE + lane;
#pragma unroll
    for (int rr = 0; rr < RP; ++rr)
#pragma unroll
        for (int J = 0; J < n; ++J) G[(size_t)((r0 + rr) * n + J) * TILE] = live ? mk<T>(pref * S[rr][J].x, pref * S[rr][J].y) : mk<T>(0, 0);
}
template <typename T, int DR> static int clover_exp_rows(const Geo &g, int parity, double x, double pref, const void *clover, void *blocks, int *flags, cudaStream_t s) {
    constexpr int RP = (sizeof(T) == 4 || DR <= 3) ? 2 : 1;
    auto kern = clover_exp_rows_kernel<T, DR, RP>;
    const size_t smem = (size_t)4 * DR * DR * TILE * sizeof(cplx<T>);
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, smem, cache, n_sm)) return rc;
    kern<<<dim3(g.n_tiles, 2), 32 * (2 * DR / RP), smem, s>>>(g, parity, (T)x, (T)pref, (const cplx<T> *)clover, (cplx<T> *)blocks, flags);
    return (int)cudaGetLastError();
}

// shared-memory form where >= 2 warps' worth of matrices fit an SM (bytes per warp: nbuf x (2 d_R)^2 x 32 lanes x element)
template <typename T, int DRT> static int clover_exp_sm(const Geo &g, int parity, double x, double pref, const void *clover, void *blocks, void *work, int *flags, cudaStream_t s) {
    auto kern = clover_exp_kernel<T, DRT>;
    const size_t smem = (size_t)3 * 4 * DRT * DRT * TILE * sizeof(cplx<T>);
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, smem, cache, n_sm)) return rc;
    kern<<<dim3(g.n_tiles, 2), 32, smem, s>>>(g, DRT, parity, (T)x, (T)pref, (const cplx<T> *)clover, (cplx<T> *)blocks, (cplx<T> *)work, flags);
    return (int)cudaGetLastError();
}
template <typename T> static int clover_exp_t(const Geo &g, int dR, int parity, double x, double pref, const void *clover, void *blocks, void *work, int *flags, cudaStream_t s) {
    static const int glob = getenv("HIREP_CLOVER_GLOBAL") ? atoi(getenv("HIREP_CLOVER_GLOBAL")) : 0;   // measurement switch: 1 = the in-place global-memory form,
    if (glob == 0) {                                                                                      // 2 = the per-site shared-memory form
        switch (dR) {
        case 2: return clover_exp_rows<T, 2>(g, parity, x, pref, clover, blocks, flags, s);
        case 3: return clover_exp_rows<T, 3>(g, parity, x, pref, clover, blocks, flags, s);
        case 4: return clover_exp_rows<T, 4>(g, parity, x, pref, clover, blocks, flags, s);
        case 5: return clover_exp_rows<T, 5>(g, parity, x, pref, clover, blocks, flags, s);
        case 6: return clover_exp_rows<T, 6>(g, parity, x, pref, clover, blocks, flags, s);
        case 8: if constexpr (sizeof(T) == 4) return clover_exp_rows<T, 8>(g, parity, x, pref, clover, blocks, flags, s); break;   // fp64: 3 x 2 x 16 complex doubles per thread do not fit
        }
    }
    if (glob != 1 && (size_t)3 * 4 * dR * dR * TILE * sizeof(cplx<T>) <= 112 * 1024) {
        switch (dR) {
        case 1: return clover_exp_sm<T, 1>(g, parity, x, pref, clover, blocks, work, flags, s);
        case 2: return clover_exp_sm<T, 2>(g, parity, x, pref, clover, blocks, work, flags, s);
        case 3: return clover_exp_sm<T, 3>(g, parity, x, pref, clover, blocks, work, flags, s);
        case 4: return clover_exp_sm<T, 4>(g, parity, x, pref, clover, blocks, work, flags, s);
        case 5: if constexpr (sizeof(T) == 4) return clover_exp_sm<T, 5>(g, parity, x, pref, clover, blocks, work, flags, s); break;
        case 6: if constexpr (sizeof(T) == 4) return clover_exp_sm<T, 6>(g, parity, x, pref, clover, blocks, work, flags, s); break;
        }
    }
    clover_exp_kernel<T, 0><<<dim3((g.n_tiles * TILE + 63) / 64, 2), 64, 0, s>>>(g, dR, parity, (T)x, (T)pref, (const cplx<T> *)clover, (cplx<T> *)blocks,
                                                                              (cplx<T> *)work, flags);
    return (int)cudaGetLastError();
}
int k_clover_exp(const Geo &g, int prec, int dR, int parity, double x, double pref, const void *clover, void *blocks, void *work, int *flags, cudaStream_t s) {
    return prec == 0 ? clover_exp_t<double>(g, dR, parity, x, pref, clover, blocks, work, flags, s) : clover_exp_t<float>(g, dR, parity, x, pref, clover, blocks, work, flags, s);
}

// Row-split Gauss-Jordan (d_R = 2 ... 6): CTA = (tile, chirality), lane = site, warp w holds the rows w RP .. of the block in registers.
// Step k: the warp that owns row k scales it and publishes it to shared memory ([J][lane], double-buffered over k: one barrier per
// step); every warp then eliminates column k from its own rows -- one shared-memory read per RP complex MACs, no global or shared
// round trips of the block.  The same operations per entry as clover_inv_kernel: bit-identical inverse and the same pivot flag.
template <typename T, int DR, int RP>
__global__ void __launch_bounds__(32 * (2 * DR / RP)) clover_inv_rows_kernel(Geo g, int parity, T a, T csw, const cplx<T> *__restrict__ clover, cplx<T> *inv,
                                                                            int *flags) {
    constexpr int n = 2 * DR, ne = DR * DR, NW = n / RP;
    static_assert(n % RP == 0, "rows must split evenly");
    extern __shared__ __align__(16) unsigned char smem_blk[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, r0 = warp * RP;
    const int tile = blockIdx.x, c = blockIdx.y;
    cplx<T> *rowk = reinterpret_cast<cplx<T> *>(smem_blk) + lane;              // [2][n][lane]
    T *smax = reinterpret_cast<T *>(smem_blk + (size_t)2 * n * TILE * sizeof(cplx<T>)) + lane;   // [NW][lane]
    const bool live = tile * TILE + lane < g.Nh;
    cplx<T> M[RP][n];
    T scale = 0;
#pragma unroll
    for (int rr = 0; rr < RP; ++rr) {
        const int I = r0 + rr, bi = I / DR, i = I - bi * DR;
#pragma unroll
        for (int J = 0; J < n; ++J) {
            const int bj = J / DR, j = J - bj * DR;
            cplx<T> v;
            if (bi == bj) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 0, i * DR + j, lane, ne)];
                if (bi) { v.x = -v.x; v.y = -v.y; }
            } else if (bi == 0) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, i * DR + j, lane, ne)];
            } else {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, j * DR + i, lane, ne)];
                v.y = -v.y;
            }
            v.x *= csw; v.y *= csw;
            if (I == J) v.x += a;
            if (!live) v = mk<T>(I == J ? T(1) : T(0), T(0));
            M[rr][J] = v;
            scale = fmax(scale, fmax(fabs(v.x), fabs(v.y)));
        }
    }
    smax[(size_t)warp * TILE] = scale;                              // the yardstick for the pivots is the block's largest entry
    __syncthreads();
#pragma unroll
    for (int w = 0; w < NW; ++w) scale = fmax(scale, smax[(size_t)w * TILE]);
    const T tiny = scale * (sizeof(T) == 8 ? T(1e-10) : T(1e-4));
    bool bad = false;
    static_for<0, n>([&](auto kc) {
        constexpr int k = decltype(kc)::value, kw = k / RP, kk = k % RP;
        cplx<T> *pub = rowk + (size_t)(k & 1) * n * TILE;
        if (warp == kw) {
            const cplx<T> d = M[kk][k];
            const T d2 = d.x * d.x + d.y * d.y;
            if (!(d2 > tiny * tiny) || !isfinite(d2)) bad = true;
            const T r = T(1) / d2;
            const cplx<T> p = mk<T>(d.x * r, -d.y * r);
            M[kk][k] = mk<T>(1, 0);
#pragma unroll
            for (int J = 0; J < n; ++J) {
                M[kk][J] = cmul<T>(M[kk][J], p);
                pub[(size_t)J * TILE] = M[kk][J];
            }
        }
        __syncthreads();
#pragma unroll
        for (int rr = 0; rr < RP; ++rr) {
            if (!(warp == kw && rr == kk)) {
                const cplx<T> f = M[rr][k];
                M[rr][k] = mk<T>(0, 0);
#pragma unroll
                for (int J = 0; J < n; ++J) {
                    const cplx<T> x = pub[(size_t)J * TILE];
                    M[rr][J].x -= f.x * x.x - f.y * x.y;
                    M[rr][J].y -= f.x * x.y + f.y * x.x;
                }
            }
        }
    });
    cplx<T> *G = inv + ((size_t)(tile * 2 + c) * n * n) * TILE + lane;
#pragma unroll
    for (int rr = 0; rr < RP; ++rr)
#pragma unroll
        for (int J = 0; J < n; ++J) G[(size_t)((r0 + rr) * n + J) * TILE] = live ? M[rr][J] : mk<T>(0, 0);
    if (bad && live && flags) atomicOr(flags, 1);
}
template <typename T, int DR> static int clover_inv_rows(const Geo &g, int parity, double a, double csw, const void *clover, void *inv, int *flags, cudaStream_t s) {
    constexpr int RP = 2, n = 2 * DR;
    clover_inv_rows_kernel<T, DR, RP><<<dim3(g.n_tiles, 2), 32 * (n / RP), (size_t)2 * n * TILE * sizeof(cplx<T>) + (size_t)(n / RP) * TILE * sizeof(T), s>>>(
        g, parity, (T)a, (T)csw, (const cplx<T> *)clover, (cplx<T> *)inv, flags);
    return (int)cudaGetLastError();
}

// Large d_R (blocks of 20 x 20 ... 70 x 70): one CTA per (site, chirality), thread = row, the block in shared memory [I][J] with an
// odd row stride (conflict free for "thread I reads M[I][J]", a broadcast for the pivot row).  The per-thread form above sweeps the
// whole block through DRAM once per pivot (2.5 MB per warp at d_R = 35: 418 ms at C5 fp64); here it is read and written once.  The
// site's entries sit 32 elements apart in the native layout: the CTAs of neighbouring lanes run at the same time and share the
// sectors through L2.  Same operations in the same order per entry: bit-identical inverse and pivot flag.
template <typename T, int TPR>   // TPR threads per row, each a contiguous part of the columns (the threads of a row sit in one warp)
__global__ void __launch_bounds__(192) clover_inv_cta_kernel(Geo g, int dR, int parity, T a, T csw, const cplx<T> *__restrict__ clover, cplx<T> *inv, int *flags) {
    extern __shared__ __align__(16) unsigned char smem_blk[];
    const int n = 2 * dR, ne = dR * dR, ld = n + 1;
    cplx<T> *M = reinterpret_cast<cplx<T> *>(smem_blk);
    T *rmax = reinterpret_cast<T *>(M + (size_t)n * ld);
    const int slot = blockIdx.x, c = blockIdx.y, tile = slot >> 5, lane = slot & 31;
    const int I = threadIdx.x / TPR, part = threadIdx.x % TPR, cw = (n + TPR - 1) / TPR;
    const int J0 = part * cw, J1 = J0 + cw < n ? J0 + cw : n;     // this thread's columns
    const bool live = slot < g.Nh, row = I < n;
    cplx<T> *G = inv + ((size_t)(tile * 2 + c) * n * n) * TILE + lane;
    if (!live) {                                                   // padding lanes hold zeros
        if (row)
            for (int J = J0; J < J1; ++J) G[(size_t)(I * n + J) * TILE] = mk<T>(0, 0);
        return;
    }
    if (row) {
        const int bi = I / dR, i = I - bi * dR;
        T m = 0;
        for (int J = J0; J < J1; ++J) {
            const int bj = J / dR, j = J - bj * dR;
            cplx<T> v;
            if (bi == bj) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 0, i * dR + j, lane, ne)];
                if (bi) { v.x = -v.x; v.y = -v.y; }
            } else if (bi == 0) {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, i * dR + j, lane, ne)];
            } else {
                v = clover[clover_off(g.n_tiles, parity, tile, c, 1, j * dR + i, lane, ne)];
                v.y = -v.y;
            }
            v.x *= csw; v.y *= csw;
            if (I == J) v.x += a;
            M[(size_t)I * ld + J] = v;
            m = fmax(m, fmax(fabs(v.x), fabs(v.y)));
        }
        rmax[threadIdx.x] = m;
    }
    __syncthreads();
    T scale = 0;
    for (int r = 0; r < n * TPR; ++r) scale = fmax(scale, rmax[r]);
    const T tiny = scale * (sizeof(T) == 8 ? T(1e-10) : T(1e-4));
    bool bad = false;
    for (int k = 0; k < n; ++k) {
        cplx<T> *Pk = M + (size_t)k * ld;
        cplx<T> *Mi = M + (size_t)(row ? I : 0) * ld;
        // every thread of a row reads the pivot resp. its multiplier before the owner of column k overwrites it
        const cplx<T> dk = Pk[k];
        const cplx<T> f = Mi[k];
        __syncwarp();
        if (I == k) {
            const T d2 = dk.x * dk.x + dk.y * dk.y;
            if (!(d2 > tiny * tiny) || !isfinite(d2)) bad = true;
            const T r = T(1) / d2;
            const cplx<T> p = mk<T>(dk.x * r, -dk.y * r);
            if (k >= J0 && k < J1) Pk[k] = mk<T>(1, 0);
            for (int J = J0; J < J1; ++J) Pk[J] = cmul<T>(Pk[J], p);
        }
        __syncthreads();
        if (row && I != k) {
            if (k >= J0 && k < J1) Mi[k] = mk<T>(0, 0);
#pragma unroll 4
            for (int J = J0; J < J1; ++J) {
                const cplx<T> x = Pk[J];
                cplx<T> y = Mi[J];
                y.x -= f.x * x.x - f.y * x.y;
                y.y -= f.x * x.y + f.y * x.x;
                Mi[J] = y;
            }
        }
        __syncthreads();
    }
    if (row)
        for (int J = J0; J < J1; ++J) G[(size_t)(I * n + J) * TILE] = M[(size_t)I * ld + J];
    if (bad && part == 0 && flags) atomicOr(flags, 1);
}
template <typename T, int TPR> static int clover_inv_cta_launch(const Geo &g, int dR, int parity, double a, double csw, const void *clover, void *inv, int *flags, cudaStream_t s) {
    const int n = 2 * dR;
    const size_t smem = (size_t)n * (n + 1) * sizeof(cplx<T>) + (size_t)n * TPR * sizeof(T);
    auto kern = clover_inv_cta_kernel<T, TPR>;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, (size_t)70 * 71 * sizeof(cplx<T>) + 70 * TPR * sizeof(T), cache, n_sm)) return rc;   // opt-in size for the largest block (d_R = 35)
    kern<<<dim3(g.n_tiles * TILE, 2), (n * TPR + 31) / 32 * 32, smem, s>>>(g, dR, parity, (T)a, (T)csw, (const cplx<T> *)clover, (cplx<T> *)inv, flags);
    return (int)cudaGetLastError();
}
template <typename T> static int clover_inv_cta(const Geo &g, int dR, int parity, double a, double csw, const void *clover, void *inv, int *flags, cudaStream_t s) {
    // two threads per row for the 70 x 70 blocks in fp64 (two CTAs of 80 KB per SM: 140 instead of 70 threads each; C5 154 -> 116 ms); one
    // thread per row elsewhere (measured: fp32 52 vs 57 ms at C5; four threads per row at 30 x 30 in fp64: 9.3 vs 3.5 ms)
    return (2 * dR > 48 && sizeof(T) == 8) ? clover_inv_cta_launch<T, 2>(g, dR, parity, a, csw, clover, inv, flags, s)
                                           : clover_inv_cta_launch<T, 1>(g, dR, parity, a, csw, clover, inv, flags, s);
}

template <typename T, int DRT> static int clover_inv_sm(const Geo &g, int parity, double a, double csw, const void *clover, void *inv, int *flags, cudaStream_t s) {
    auto kern = clover_inv_kernel<T, DRT>;
    const size_t smem = (size_t)4 * DRT * DRT * TILE * sizeof(cplx<T>);
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, smem, cache, n_sm)) return rc;
    kern<<<dim3(g.n_tiles, 2), 32, smem, s>>>(g, DRT, parity, (T)a, (T)csw, (const cplx<T> *)clover, (cplx<T> *)inv, flags);
    return (int)cudaGetLastError();
}
template <typename T> static int clover_inv_t(const Geo &g, int dR, int parity, double a, double csw, const void *clover, void *inv, int *flags, cudaStream_t s) {
    static const int glob = getenv("HIREP_CLOVER_GLOBAL") ? atoi(getenv("HIREP_CLOVER_GLOBAL")) : 0;   // 1 = in place in global memory, 2 = per-site shared-memory form
    if (glob == 0) {
        switch (dR) {
        case 2: return clover_inv_rows<T, 2>(g, parity, a, csw, clover, inv, flags, s);
        case 3: return clover_inv_rows<T, 3>(g, parity, a, csw, clover, inv, flags, s);
        case 4: return clover_inv_rows<T, 4>(g, parity, a, csw, clover, inv, flags, s);
        case 5: return clover_inv_rows<T, 5>(g, parity, a, csw, clover, inv, flags, s);
        case 6: return clover_inv_rows<T, 6>(g, parity, a, csw, clover, inv, flags, s);
        case 8: return clover_inv_rows<T, 8>(g, parity, a, csw, clover, inv, flags, s);
        case 10: if constexpr (sizeof(T) == 4) return clover_inv_rows<T, 10>(g, parity, a, csw, clover, inv, flags, s); break;   // fp64: the unrolled elimination spills (ptxas: 52 KB)
        }
    }
    if (glob != 1 && (size_t)4 * dR * dR * TILE * sizeof(cplx<T>) <= 112 * 1024) {
        switch (dR) {
        case 1: return clover_inv_sm<T, 1>(g, parity, a, csw, clover, inv, flags, s);
        case 2: return clover_inv_sm<T, 2>(g, parity, a, csw, clover, inv, flags, s);
        case 3: return clover_inv_sm<T, 3>(g, parity, a, csw, clover, inv, flags, s);
        case 4: return clover_inv_sm<T, 4>(g, parity, a, csw, clover, inv, flags, s);
        case 5: return clover_inv_sm<T, 5>(g, parity, a, csw, clover, inv, flags, s);
        case 6: return clover_inv_sm<T, 6>(g, parity, a, csw, clover, inv, flags, s);
        case 8: return clover_inv_sm<T, 8>(g, parity, a, csw, clover, inv, flags, s);
        }
    }
    if (glob == 0 && dR >= 10 && dR <= 35) return clover_inv_cta<T>(g, dR, parity, a, csw, clover, inv, flags, s);
    clover_inv_kernel<T, 0><<<dim3((g.n_tiles * TILE + 63) / 64, 2), 64, 0, s>>>(g, dR, parity, (T)a, (T)csw, (const cplx<T> *)clover, (cplx<T> *)inv, flags);
    return (int)cudaGetLastError();
}
int k_clover_inv(const Geo &g, int prec, int dR, int parity, double a, double csw, const void *clover, void *inv, int *flags, cudaStream_t s) {
    return prec == 0 ? clover_inv_t<double>(g, dR, parity, a, csw, clover, inv, flags, s) : clover_inv_t<float>(g, dR, parity, a, csw, clover, inv, flags, s);
}

template <typename T> static int clover_export_t(const Geo &g, int dR, void *canon, const void *clover, cudaStream_t s) {
    const long n = 2L * g.Nh * 2 * (2 * dR) * (2 * dR);
    clover_export_kernel<T><<<(unsigned)((n + 255) / 256), 256, 0, s>>>(g, dR, (cplx<T> *)canon, (const cplx<T> *)clover);
    return (int)cudaGetLastError();
}
int k_clover_export(const Geo &g, int prec, int dR, void *canon, const void *clover, cudaStream_t s) {
    return prec == 0 ? clover_export_t<double>(g, dR, canon, clover, s) : clover_export_t<float>(g, dR, canon, clover, s);
}

}  // namespace hirep
