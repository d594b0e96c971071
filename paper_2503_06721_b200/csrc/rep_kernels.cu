// rep_kernels.cu -- fundamental -> represented links (Eq 7; "functions that translate the
// fundamental gauge field to the represented one", L339-341) with the boundary signs of L945 applied.
//
// Every slot W of the native gather layout is mapped independently:  W^R = s * R(W), R(.) row by row from
// rep_maps.cuh (the same maps the stencil kernels use in link mode REBUILD).  For the backward slots W = U^dagger
// and R(U^dagger) = R(U)^dagger holds identically for all four maps.
//
// Work decomposition: one WARP per (parity, tile, slot) "link block" of 32 sites (lane = site, so every load and
// store is one contiguous 128/256/512-byte row of the layout); the NW warps of a block's team split the d_R rows of
// R (row a goes to warp a % NW), each keeping the fundamental matrix in registers.  NW = 1 for small d_R, 4 for
// d_R >= 15.  The adjoints of SU(4..6) (d_R = 15, 24, 35) use links_to_rep_adj_kernel instead: the fully unrolled
// rows are ~280 KB of code at d_R = 35 and the kernel stalled on instruction fetch (ncu: 88 % "no instruction",
// 2.4 TB/s); with a run-time row loop over a shared-memory copy of W it runs at the copy roofline (4.6 -> 1.7 ms).
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

// Large adjoints (SU(4..6)): one warp per link block, W parked in a per-warp shared-memory tile [e][lane], rows of
// R walked by a run-time loop (adj_row_runtime: small code, no instruction-fetch stalls), NW warps split the rows.
template <typename T, int N, int NW>
__global__ void __launch_bounds__(128) links_to_rep_adj_kernel(Geo g, T *rep, const cplx<T> *fund, long n_blocks) {
    constexpr int DR = N * N - 1, WPB = 4;                      // warps per CTA
    extern __shared__ __align__(16) unsigned char smem_l2r[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const long gwarp = (long)blockIdx.x * WPB + wib;
    const long blk = gwarp / NW;
    const int wsub = (int)(gwarp % NW);
    if (blk >= n_blocks) return;
    const int d = (int)(blk & 7);
    const long pt = blk >> 3;
    const int tile = (int)(pt % g.n_tiles), p = (int)(pt / g.n_tiles);
    cplx<T> *Wsm = reinterpret_cast<cplx<T> *>(smem_l2r) + (size_t)wib * (N * N) * TILE + lane;
    const cplx<T> *src = fund + (size_t)blk * (N * N) * TILE + lane;
#pragma unroll
    for (int e = 0; e < N * N; ++e) Wsm[e * TILE] = src[(size_t)e * TILE];
    __syncwarp();
    T sgn = 1;
    const int h = tile * TILE + lane;
    if (h < g.Nh) {
        int t, x, y, zh;
        decode_site(g, h, t, x, y, zh);
        sgn = (T)hop_sign(g, p, t, x, y, zh, d);
    }
    struct Acc_ { const cplx<T> *q; __device__ __forceinline__ cplx<T> operator[](int e) const { return q[e * TILE]; } };
    const Acc_ Wm{Wsm};
    T *dst = rep + (size_t)blk * (DR * DR) * TILE + lane;
#pragma unroll 1
    for (int a = wsub; a < DR; a += NW) {
        T w[DR];
        adj_row_runtime<T, N>(Wm, a, w);
#pragma unroll
        for (int B = 0; B < DR; ++B) dst[(size_t)(a * DR + B) * TILE] = sgn * w[B];
    }
}

template <typename T, int N> int launch_adj_large(const Geo &g, void *rep, const void *fund, cudaStream_t s) {
    constexpr int NW = 4;
    const long n_blocks = (long)2 * g.n_tiles * 8;
    const long n_warps = n_blocks * NW;
    const unsigned grid = (unsigned)((n_warps + 3) / 4);
    const size_t smem = (size_t)4 * N * N * TILE * sizeof(cplx<T>);
    auto kern = links_to_rep_adj_kernel<T, N, NW>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        configured = true;
    }
    kern<<<grid, 128, smem, s>>>(g, (T *)rep, (const cplx<T> *)fund, n_blocks);
    return (int)cudaGetLastError();
}

template <typename T, int N, int REP> int launch(const Geo &g, void *rep, const void *fund, cudaStream_t s) {
    if constexpr (REP == 1 && N >= 4) return launch_adj_large<T, N>(g, rep, fund, s);
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
