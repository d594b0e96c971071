// hop_dispatch.cuh -- maps (N_g, rep, mode, variant) to a stencil-kernel instantiation for one precision T.
// Included by hop_f64.cu and hop_f32.cu so the two precisions compile in parallel.
//
// Variants (hirep_set_kernel_variant):  0 = library default for the instantiation
//   1 = direct-load kernel, one thread per site          (hop_small.cuh, P = 1)
//   2 = direct-load kernel, two lanes per site           (hop_small.cuh, P = 2)
//   3 = persistent kernel, link stream through a per-warp bulk-copy (TMA) ring in shared memory (hop_ring.cuh)
//   4 = the same with two warps per tile, one per half-spinor component (hop_pair.cuh)
// Default for d_R <= 6: variant 3, except fp64 with d_R >= 5 where one thread per site spills: variant 4
// (measured on B200, profiles/).  Large d_R (>= 8) always uses the row-group
// kernel of hop_large.cuh.
#pragma once
#include "hop_large.cuh"
#include "hop_pair.cuh"

namespace hirep {

template <typename T, int DR, bool REAL> int hop_small_variant(const Geo &g, int variant, const HopLaunch &L, cudaStream_t s) {
    if (variant == 0) variant = (sizeof(T) == 8 && DR >= 5) ? 4 : 3;
    switch (variant) {
    case 1: return launch_hop_small<T, DR, REAL, 1, 128>(g, L, s);
    case 2: return launch_hop_small<T, DR, REAL, 2, 128>(g, L, s);
    case 3: return launch_hop_ring<T, DR, REAL>(g, L, s);
    case 4: return launch_hop_pair<T, DR, REAL>(g, L, s);
    }
#ifdef HIREP_SWEEP   // ring-shape sweeps (not part of the library build): variant = 1000*WARPS + 100*STAGES + RPC
    if constexpr (DR == HIREP_SWEEP && !REAL) {
        const bool self = (L.a != 0.0) && L.set[0].self != nullptr;
#define SW(W, S, R)                                                                                          \
    if (variant == 1000 * W + 100 * S + R)                                                                   \
        return self ? launch_hop_ring_cfg<T, DR, REAL, W, S, R, true>(g, L, s) : launch_hop_ring_cfg<T, DR, REAL, W, S, R, false>(g, L, s);
#define SWN(W, S, R)                                                                                         \
    if (variant == 1000 * W + 100 * S + R)                                                                   \
        return self ? launch_hop_ring<T, DR, REAL>(g, L, s) : launch_hop_ring_cfg<T, DR, REAL, W, S, R, false>(g, L, s);
        if constexpr (sizeof(T) == 4) {
            SW(12, 2, 3) SW(12, 4, 2) SWN(11, 2, 6) SWN(10, 2, 6) SW(8, 2, 6) SW(10, 2, 3) SW(11, 2, 3) SW(12, 3, 2) SW(8, 4, 3)
        } else {
            SW(8, 4, 1) SW(8, 2, 2) SW(6, 2, 3) SW(6, 3, 2) SW(4, 4, 3)
        }
#undef SW
#undef SWN
    }
#endif
    return KERR_UNSUPPORTED;
}

template <typename T> int hop_by_config(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s) {
    if (mode != 0) return KERR_UNSUPPORTED;
    const int dR = (rep == 0) ? N : (rep == 1) ? N * N - 1 : (rep == 2) ? N * (N + 1) / 2 : N * (N - 1) / 2;
    const bool real = (rep == 1);
    if (!real) {
        switch (dR) {
        case 2: return hop_small_variant<T, 2, false>(g, variant, L, s);
        case 3: return hop_small_variant<T, 3, false>(g, variant, L, s);
        case 4: return hop_small_variant<T, 4, false>(g, variant, L, s);
        case 5: return hop_small_variant<T, 5, false>(g, variant, L, s);
        case 6: return hop_small_variant<T, 6, false>(g, variant, L, s);
        case 10: return variant == 0 ? launch_hop_large<T, 10, false, 5>(g, L, s) : KERR_UNSUPPORTED;
        case 15: return variant == 0 ? launch_hop_large<T, 15, false, 5>(g, L, s) : KERR_UNSUPPORTED;
        }
    } else {
        switch (dR) {
        case 3: return hop_small_variant<T, 3, true>(g, variant, L, s);
        case 8: return variant == 0 ? launch_hop_large<T, 8, true, 4>(g, L, s) : KERR_UNSUPPORTED;
        case 15: return variant == 0 ? launch_hop_large<T, 15, true, 5>(g, L, s) : KERR_UNSUPPORTED;
        case 35: return variant == 0 ? launch_hop_large<T, 35, true, 5>(g, L, s) : KERR_UNSUPPORTED;
        }
    }
    return KERR_UNSUPPORTED;
}

int k_hop_f64(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s);
int k_hop_f32(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s);

}  // namespace hirep
