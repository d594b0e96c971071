// hop_small.cuh -- the Wilson hopping stencil for small d_R (link matrix fits in registers row by row).
//
//   out(x) = a*self(x) + b * sum_{d=0..7} P_d W_d(x) in(nbr_d(x)),   x of parity p_out            (Eq 8)
//
// with P_d = (1 - gamma_mu) for the forward hops d = mu and (1 + gamma_mu) for the backward hops d = 4 + mu.
// In the basis of Eq 1-3 (L171-182), gamma_mu = [[0, e_mu],[e_mu^dagger, 0]], the projectors have rank 2:
//   (1 + sg*gamma_mu) psi = ( h , sg * e_mu^dagger h ),   h = psi_up + sg * e_mu psi_low      (sg = -1 fwd, +1 bwd)
// so only the half spinor h (2 x d_R) is multiplied by the link (steps a2-a4 of SURVEY.md 8(a)).  e_mu has one
// non-zero entry per row: (e_mu v)_s = k_mu(s) v_{q_mu(s)} with
//   mu   q(s)    k(s)
//   0    s       -1
//   1    1-s     -i
//   2    1-s     s==0 ? -1 : +1
//   3    s       s==0 ? -i : +i
// and (e_mu^dagger chi)_{q(s)} = conj(k(s)) chi_s.
//
// Thread mapping: P lanes per site.  P = 1: one thread owns both half-spinor components.  P = 2: lanes (2i, 2i+1)
// own s = 0, 1 of site i; the mu = 1,2 contributions to the lower components belong to the partner lane and are
// exchanged once, at the end, with a single shuffle per accumulator.
#pragma once
#include "kernels.h"

namespace hirep {

template <typename T> __device__ inline cplx<T> ld_spinor(const cplx<T> *p) { return __ldg(p); }
// output spinors are written once and not re-read by the launch: streaming store (L2 evict-first), so that they do
// not compete with the neighbour-spinor lines for L2 (worth 1-2 % on the full-lattice passes)
template <typename C> __device__ __forceinline__ void st_spinor(C *p, const C &v) { __stcs(p, v); }
template <typename E> __device__ inline E ld_link(const E *p) { return __ldcs(p); }   // streamed once: evict-first

template <int D> struct DirInfo {
    static constexpr int mu = D & 3;
    static constexpr bool fwd = D < 4;
    static constexpr int sg = fwd ? -1 : +1;
    static constexpr bool imag = (mu == 1 || mu == 3);
    static constexpr bool swap = (mu == 1 || mu == 2);
    __host__ __device__ static constexpr int sigma(int s) { return (mu < 2) ? -1 : (s ? 1 : -1); }
};

// acc += w * h  for complex or real link element
template <typename T> __device__ __forceinline__ void mac(cplx<T> &acc, const cplx<T> &w, const cplx<T> &h) {
    acc.x = fma(w.x, h.x, acc.x);
    acc.x = fma(-w.y, h.y, acc.x);
    acc.y = fma(w.x, h.y, acc.y);
    acc.y = fma(w.y, h.x, acc.y);
}
template <typename T> __device__ __forceinline__ void mac(cplx<T> &acc, const T &w, const cplx<T> &h) {
    acc.x = fma(w, h.x, acc.x);
    acc.y = fma(w, h.y, acc.y);
}

template <typename T, int DR, bool REAL, int P, int BLOCK>
__global__ void __launch_bounds__(BLOCK) hop_small_kernel(const Geo g, const HopLaunch L) {
    using C = cplx<T>;
    using E = link_elem<T, REAL>;
    constexpr int NC = 4 * DR, NE = DR * DR;
    constexpr int NS = (P == 1) ? 2 : 1;   // half-spinor components owned by this thread

    const HopSet &S = L.set[blockIdx.y];
    const int gt = blockIdx.x * BLOCK + threadIdx.x;
    int h = gt / P;
    const int s_rt = (P == 2) ? (gt & 1) : 0;
    const bool active = h < g.Nh;
    if (!active) h = g.Nh - 1;             // keep the warp converged for the final shuffle; store is predicated
    const int tile = h >> 5, lane = h & 31;
    int t, x, y, zh;
    decode_site(g, h, t, x, y, zh);

    const C *__restrict__ in = (const C *)S.in;
    const E *__restrict__ W0 = (const E *)S.links + ((size_t)tile * 8 * NE) * TILE + lane;

    C up[NS][DR], lo[NS][DR], lx[NS][DR];   // P=1: lo[q] is the lower component q, lx unused
#pragma unroll
    for (int k = 0; k < NS; ++k)
#pragma unroll
        for (int c = 0; c < DR; ++c) up[k][c] = lo[k][c] = lx[k][c] = mk<T>(0, 0);

    static_for<0, 8>([&](auto dc) {
        constexpr int D = decltype(dc)::value;
        using DI = DirInfo<D>;
        const int hn = neighbour<D>(g, S.p_out, t, x, y, zh);
        const C *src = in + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
        C hs[NS][DR];
#pragma unroll
        for (int k = 0; k < NS; ++k) {
            const int s = (P == 1) ? k : s_rt;
            const int q = DI::swap ? 1 - s : s;
            const T cs = (T)(DI::sg * ((DI::mu < 2) ? -1 : (s ? 1 : -1)));
#pragma unroll
            for (int c = 0; c < DR; ++c) {
                const C a = ld_spinor<T>(src + (size_t)(s * DR + c) * TILE);
                const C b = ld_spinor<T>(src + (size_t)((2 + q) * DR + c) * TILE);
                if (DI::imag) hs[k][c] = mk<T>(fma(-cs, b.y, a.x), fma(cs, b.x, a.y));   // a + i cs b
                else hs[k][c] = mk<T>(fma(cs, b.x, a.x), fma(cs, b.y, a.y));             // a + cs b
            }
        }
        const E *W = W0 + (size_t)D * NE * TILE;
#pragma unroll
        for (int i = 0; i < DR; ++i) {
            E w[DR];
#pragma unroll
            for (int j = 0; j < DR; ++j) w[j] = ld_link<E>(W + (size_t)(i * DR + j) * TILE);
#pragma unroll
            for (int k = 0; k < NS; ++k) {
                const int s = (P == 1) ? k : s_rt;
                C chi = mk<T>(0, 0);
#pragma unroll
                for (int j = 0; j < DR; ++j) mac<T>(chi, w[j], hs[k][j]);
                up[k][i].x += chi.x;
                up[k][i].y += chi.y;
                // lower component q(s) += sg * conj(k(s)) * chi
                const T cl = (T)(DI::sg * ((DI::mu < 2) ? -1 : (s ? 1 : -1)));
                C add;
                if (DI::imag) add = mk<T>(cl * chi.y, -cl * chi.x);   // (-i cl) chi
                else add = mk<T>(cl * chi.x, cl * chi.y);
                if constexpr (P == 1) {
                    const int q = DI::swap ? 1 - k : k;
                    lo[q][i].x += add.x;
                    lo[q][i].y += add.y;
                } else if (DI::swap) {
                    lx[0][i].x += add.x;
                    lx[0][i].y += add.y;
                } else {
                    lo[0][i].x += add.x;
                    lo[0][i].y += add.y;
                }
            }
        }
    });

    if constexpr (P == 2) {
#pragma unroll
        for (int i = 0; i < DR; ++i) {
            lo[0][i].x += __shfl_xor_sync(0xffffffffu, lx[0][i].x, 1);
            lo[0][i].y += __shfl_xor_sync(0xffffffffu, lx[0][i].y, 1);
        }
    }
    if (!active) return;

    const T a = (T)L.a, b = (T)L.b;
    const T am = (T)L.am;
    const T g5s = L.g5 ? T(-1) : T(1);
    C *out = (C *)S.out + ((size_t)tile * NC) * TILE + lane;
    const C *self = (const C *)S.self + ((size_t)tile * NC) * TILE + lane;
    const bool use_self = (S.self != nullptr) && (L.a != 0.0);
#pragma unroll
    for (int k = 0; k < NS; ++k) {
        const int s = (P == 1) ? k : s_rt;
#pragma unroll
        for (int c = 0; c < DR; ++c) {
            C vu = mk<T>(b * up[k][c].x, b * up[k][c].y);
            C vl = mk<T>(b * lo[k][c].x, b * lo[k][c].y);
            if (use_self) {
                const C su = self[(size_t)(s * DR + c) * TILE];
                const C sl = self[(size_t)((2 + s) * DR + c) * TILE];
                vu.x = fma(a, su.x, vu.x); vu.y = fma(a, su.y, vu.y);
                vl.x = fma(a, sl.x, vl.x); vl.y = fma(a, sl.y, vl.y);
                if (am != T(0)) {   // twisted mass: + i mu gamma_5 self (Eq 51)
                    vu.x = fma(-am, su.y, vu.x); vu.y = fma(am, su.x, vu.y);
                    vl.x = fma(am, sl.y, vl.x); vl.y = fma(-am, sl.x, vl.y);
                }
            }
            out[(size_t)(s * DR + c) * TILE] = vu;
            out[(size_t)((2 + s) * DR + c) * TILE] = mk<T>(g5s * vl.x, g5s * vl.y);
        }
    }
}

template <typename T, int DR, bool REAL, int P, int BLOCK>
int launch_hop_small(const Geo &g, const HopLaunch &L, cudaStream_t s) {
    const long nthreads = (long)g.n_tiles * TILE * P;
    dim3 grid((unsigned)((nthreads + BLOCK - 1) / BLOCK), L.nsets);
    hop_small_kernel<T, DR, REAL, P, BLOCK><<<grid, BLOCK, 0, s>>>(g, L);
    return (int)cudaGetLastError();
}

}  // namespace hirep
