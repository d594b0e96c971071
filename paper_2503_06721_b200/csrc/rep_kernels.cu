// rep_kernels.cu -- fundamental -> represented links (Eq 7; "functions that translate the
// fundamental gauge field to the represented one", L339-341) with the boundary signs of L945 applied.
//
// Every slot W of the native gather layout is mapped independently:  W^R = s * R(W), R(.) row by row from
// rep_maps.cuh (the same maps the stencil kernels use in link mode REBUILD).  For the backward slots W = U^dagger
// and R(U^dagger) = R(U)^dagger holds identically for all four maps.
//
// Work decomposition: one WARP per (parity, tile, slot) "link block" of 32 sites (lane = site, so every load and
// store is one contiguous 128/256/512-byte row of the layout); the NW warps of a block's team split the d_R rows of
// R (row a goes to warp a % NW), each keeping the fundamental matrix in registers.  NW = 1 for small d_R; for the
// adjoint of SU(4..6) (d_R = 15, 24, 35: thousands of flops per link) NW = 4 keeps the flops per thread and the
// unrolled code size bounded and puts 4x more warps in flight.
#include "kernels.h"
#include "rep_maps.cuh"

namespace hirep {

namespace {

template <typename T, int N, int REP, int NW>
__global__ void __launch_bounds__(128) links_to_rep_kernel(Geo g, typename RepMap<T, N, REP>::E *rep, const cplx<T> *fund, long n_blocks) {
    using Map = RepMap<T, N, REP>;
    using E = typename Map::E;
    constexpr int DR = Map::DR;
    const int lane = threadIdx.x & 31;
    const long gwarp = ((long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long blk = gwarp / NW;              // link block = (p * n_tiles + tile) * 8 + d
    const int wsub = (int)(gwarp % NW);
    if (blk >= n_blocks) return;
    const int d = (int)(blk & 7);
    const long pt = blk >> 3;
    const int tile = (int)(pt % g.n_tiles), p = (int)(pt / g.n_tiles);

    cplx<T> W[N * N];
    const cplx<T> *src = fund + (size_t)blk * (N * N) * TILE + lane;
#pragma unroll
    for (int e = 0; e < N * N; ++e) W[e] = src[(size_t)e * TILE];
    T sgn = 1;
    const int h = tile * TILE + lane;
    if (h < g.Nh) {
        int t, x, y, zh;
        decode_site(g, h, t, x, y, zh);
        sgn = (T)hop_sign(g, p, t, x, y, zh, d);
    }
    E *dst = rep + (size_t)blk * (DR * DR) * TILE + lane;
    static_for<0, DR>([&](auto ac) {
        constexpr int A = decltype(ac)::value;
        if (NW == 1 || (A % NW) == wsub) {
            E w[DR];
            Map::template row<A>(W, w);
#pragma unroll
            for (int B = 0; B < DR; ++B) {
                if constexpr (Map::REAL) dst[(size_t)(A * DR + B) * TILE] = sgn * w[B];
                else dst[(size_t)(A * DR + B) * TILE] = mk<T>(sgn * w[B].x, sgn * w[B].y);
            }
        }
    });
}

template <typename T, int N, int REP> int launch(const Geo &g, void *rep, const void *fund, cudaStream_t s) {
    using Map = RepMap<T, N, REP>;
    constexpr int NW = (Map::DR >= 15) ? 4 : 1;
    const long n_blocks = (long)2 * g.n_tiles * 8;
    const long n_threads = n_blocks * NW * 32;
    const unsigned grid = (unsigned)((n_threads + 127) / 128);
    links_to_rep_kernel<T, N, REP, NW><<<grid, 128, 0, s>>>(g, (typename Map::E *)rep, (const cplx<T> *)fund, n_blocks);
    return (int)cudaGetLastError();
}

template <typename T, int N> int by_rep(const Geo &g, int rep_id, void *rep, const void *fund, cudaStream_t s) {
    switch (rep_id) {
    case 0: return launch<T, N, 0>(g, rep, fund, s);
    case 1: return launch<T, N, 1>(g, rep, fund, s);
    case 2: return launch<T, N, 2>(g, rep, fund, s);
    case 3: return launch<T, N, 3>(g, rep, fund, s);
    }
    return KERR_UNSUPPORTED;
}

template <typename T> int by_n(const Geo &g, int N, int rep_id, void *rep, const void *fund, cudaStream_t s) {
    switch (N) {
    case 2: return by_rep<T, 2>(g, rep_id, rep, fund, s);
    case 3: return by_rep<T, 3>(g, rep_id, rep, fund, s);
    case 4: return by_rep<T, 4>(g, rep_id, rep, fund, s);
    case 5: return by_rep<T, 5>(g, rep_id, rep, fund, s);
    case 6: return by_rep<T, 6>(g, rep_id, rep, fund, s);
    }
    return KERR_UNSUPPORTED;
}

}  // namespace

int k_links_to_rep(const Geo &g, int prec, int N, int rep, void *native_rep, const void *native_fund, cudaStream_t s) {
    return prec == 0 ? by_n<double>(g, N, rep, native_rep, native_fund, s) : by_n<float>(g, N, rep, native_rep, native_fund, s);
}

}  // namespace hirep
