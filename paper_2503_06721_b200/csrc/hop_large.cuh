// hop_large.cuh -- the hopping stencil for large d_R (d_R >= 8: the link matrix does not fit one thread).
//
// Same operator as hop_small.cuh.  One CTA owns one tile of 32 sites; blockDim = (32 lanes, NG row groups).
// Per direction: (1) the CTA projects the neighbour spinors to half spinors h (2 x d_R complex per site) and
// parks them in shared memory [s][j][lane]; (2) thread (lane, g) multiplies rows i = g*R .. g*R+R-1 of W_d by
// both half-spinor components, reading each W entry once from global memory (coalesced over the 32 lanes) and
// each h_j once from shared memory for all R rows; (3) accumulates into its R rows of the 4 spin components.
// This is the "D_R-site-parallelised" idea of PAPER.md L1532 with R rows per thread instead of one, which cuts
// the re-reads of h by R and keeps 4R independent accumulators per thread.
#pragma once
#include "hop_small.cuh"

namespace hirep {

template <typename T, int DR, bool REAL, int R>
__global__ void __launch_bounds__(32 * ((DR + R - 1) / R)) hop_large_kernel(const Geo g, const HopLaunch L) {
    using C = cplx<T>;
    using E = link_elem<T, REAL>;
    constexpr int NC = 4 * DR, NE = DR * DR, NG = (DR + R - 1) / R;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *hsm = reinterpret_cast<C *>(smem_raw);            // [2 buffers][2][DR][32]
    constexpr int HB = 2 * DR * TILE;

    const HopSet &S = L.set[blockIdx.y];
    const int tile = blockIdx.x, lane = threadIdx.x, grp = threadIdx.y;
    int h = tile * TILE + lane;
    const bool active = h < g.Nh;
    if (!active) h = g.Nh - 1;
    int t, x, y, zh;
    decode_site(g, h, t, x, y, zh);

    const C *__restrict__ in = (const C *)S.in;
    const E *__restrict__ W0 = (const E *)S.links + ((size_t)tile * 8 * NE) * TILE + lane;

    C up[2][R], lo[2][R];
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
        for (int r = 0; r < R; ++r) up[k][r] = lo[k][r] = mk<T>(0, 0);

    static_for<0, 8>([&](auto dc) {
        constexpr int D = decltype(dc)::value;
        using DI = DirInfo<D>;
        C *hb = hsm + (D & 1) * HB;
        const int hn = neighbour<D>(g, S.p_out, t, x, y, zh);
        const C *src = in + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
        // (1) projection: this thread handles colours j = grp, grp+NG, ...
        for (int j = grp; j < DR; j += NG) {
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int q = DI::swap ? 1 - s : s;
                const T cs = (T)(DI::sg * DI::sigma(s));
                const C a = ld_spinor<T>(src + (size_t)(s * DR + j) * TILE);
                const C b = ld_spinor<T>(src + (size_t)((2 + q) * DR + j) * TILE);
                C hv;
                if (DI::imag) hv = mk<T>(fma(-cs, b.y, a.x), fma(cs, b.x, a.y));
                else hv = mk<T>(fma(cs, b.x, a.x), fma(cs, b.y, a.y));
                hb[(s * DR + j) * TILE + lane] = hv;
            }
        }
        __syncthreads();   // double-buffered h: one barrier per direction suffices
        // (2) rows
        C chi[2][R];
#pragma unroll
        for (int k = 0; k < 2; ++k)
#pragma unroll
            for (int r = 0; r < R; ++r) chi[k][r] = mk<T>(0, 0);
        const E *W = W0 + (size_t)D * NE * TILE;
#pragma unroll 5
        for (int j = 0; j < DR; ++j) {
            const C h0 = hb[(0 * DR + j) * TILE + lane];
            const C h1 = hb[(1 * DR + j) * TILE + lane];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int i = grp * R + r;
                if (i < DR) {
                    const E w = ld_link<E>(W + (size_t)(i * DR + j) * TILE);
                    mac<T>(chi[0][r], w, h0);
                    mac<T>(chi[1][r], w, h1);
                }
            }
        }
        // (3) accumulate
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const int q = DI::swap ? 1 - s : s;
            const T cl = (T)(DI::sg * DI::sigma(s));
#pragma unroll
            for (int r = 0; r < R; ++r) {
                up[s][r].x += chi[s][r].x;
                up[s][r].y += chi[s][r].y;
                if (DI::imag) { lo[q][r].x += cl * chi[s][r].y; lo[q][r].y -= cl * chi[s][r].x; }
                else { lo[q][r].x += cl * chi[s][r].x; lo[q][r].y += cl * chi[s][r].y; }
            }
        }
    });

    if (!active) return;
    const T a = (T)L.a, b = (T)L.b;
    const T am = (T)L.am;
    const T g5s = L.g5 ? T(-1) : T(1);
    C *out = (C *)S.out + ((size_t)tile * NC) * TILE + lane;
    const C *self = (const C *)S.self + ((size_t)tile * NC) * TILE + lane;
    const bool use_self = (S.self != nullptr) && (L.a != 0.0);
#pragma unroll
    for (int s = 0; s < 2; ++s)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = grp * R + r;
            if (i >= DR) continue;
            C vu = mk<T>(b * up[s][r].x, b * up[s][r].y);
            C vl = mk<T>(b * lo[s][r].x, b * lo[s][r].y);
            if (use_self) {
                const C su = self[(size_t)(s * DR + i) * TILE];
                const C sl = self[(size_t)((2 + s) * DR + i) * TILE];
                vu.x = fma(a, su.x, vu.x); vu.y = fma(a, su.y, vu.y);
                vl.x = fma(a, sl.x, vl.x); vl.y = fma(a, sl.y, vl.y);
                if (am != T(0)) {   // twisted mass: + i mu gamma_5 self (Eq 51)
                    vu.x = fma(-am, su.y, vu.x); vu.y = fma(am, su.x, vu.y);
                    vl.x = fma(am, sl.y, vl.x); vl.y = fma(-am, sl.x, vl.y);
                }
            }
            out[(size_t)(s * DR + i) * TILE] = vu;
            out[(size_t)((2 + s) * DR + i) * TILE] = mk<T>(g5s * vl.x, g5s * vl.y);
        }
}

template <typename T, int DR, bool REAL, int R>
int launch_hop_large(const Geo &g, const HopLaunch &L, cudaStream_t s) {
    constexpr int NG = (DR + R - 1) / R;
    const size_t smem = 2 * 2 * DR * TILE * sizeof(cplx<T>);
    auto kern = hop_large_kernel<T, DR, REAL, R>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        configured = true;
    }
    dim3 grid(g.n_tiles, L.nsets), block(TILE, NG);
    kern<<<grid, block, smem, s>>>(g, L);
    return (int)cudaGetLastError();
}

}  // namespace hirep
