// hop_dispatch.cuh -- maps (N_g, rep, mode, variant) to a stencil-kernel instantiation for one precision T.
// Included by hop_f64.cu and hop_f32.cu so the two precisions compile in parallel.
//
// Variants (hirep_set_kernel_variant):  0 = library default for the instantiation
//   1 = direct-load kernel, one thread per site          (hop_small.cuh, P = 1)
//   2 = direct-load kernel, two lanes per site           (hop_small.cuh, P = 2)
//   3 = persistent kernel, link stream through a per-warp bulk-copy (TMA) ring in shared memory (hop_ring.cuh)
//   4 = the same with two warps per tile, one per half-spinor component (hop_pair.cuh)
//   5 = (= 0) full-lattice launches by the tile-pair kernel that stages every forward link once for both of its uses
//       (hop_full.cuh); variants 1-4 force the gather-layout kernels on full-lattice launches too
// Default for d_R <= 6: variant 3, except at d_R >= 5 in fp64 (one thread per site spills) and for the fp32 passes
// with a diagonal term: variant 4 (measured on B200, profiles/).  Link mode REBUILD always runs variant 4.  Large d_R (>= 8) always uses the row-group
// kernel of hop_large.cuh.
#pragma once
#include "hop_large.cuh"
#include "hop_rows.cuh"
#include "hop_pair.cuh"
#include "hop_full.cuh"
#include "hop_adjmf.cuh"

namespace hirep {

// Launches with a site-diagonal matrix term in the epilogue (HopLaunch::diag_mode), stored links, d_R <= 6: the thread-per-site
// ring kernel where one thread can hold the whole spinor of its site (d_R <= 4 in fp64, d_R <= 6 in fp32; variant 3), the pair
// kernel at d_R = 5, 6 (variant 4; default in fp64).  Beyond d_R = 6 the caller applies the blocks in separate launches.
// k_hop_diag_supported (hop_f64.cu) states the same rule to api.cu.
template <typename T, int DR> constexpr bool hop_diag_ring() { return sizeof(T) == 8 ? DR <= 4 : DR <= 6; }
template <typename T, int DR> constexpr bool hop_diag_pair() { return DR >= 5 && DR <= 6; }
template <typename T, int DR> constexpr bool hop_diag_pair_default() { return DR >= 5 && DR <= 6 && sizeof(T) == 8; }

template <typename T, int DR, bool REAL> int hop_small_variant(const Geo &g, int variant, const HopLaunch &L, cudaStream_t s) {
    if (L.diag_mode != DIAG_NONE) {
        if (variant == 0) variant = hop_diag_pair_default<T, DR>() ? 4 : 3;
        if constexpr (hop_diag_ring<T, DR>()) {
            if (variant == 3) return launch_hop_ring<T, DR, REAL>(g, L, s);
        }
        if constexpr (hop_diag_pair<T, DR>()) {
            if (variant == 4) return launch_hop_pair_diag<T, DR, REAL>(g, L, s);
        }
        return KERR_UNSUPPORTED;
    }
    // full-lattice launches whose diagonal term is the other parity's input: every link crosses the SM once (hop_full.cuh)
    // Default where it wins on B200 (profiles/r02_summary.md): complex links at d_R <= 3 in both precisions (C1, C2: 0.26 -> 0.20 ms at C2 fp64,
    // 0.130 -> 0.119 ms in fp32, in bursts; on par under a sustained power-capped load), the real SU(2) adjoint in fp64 (C3: 0.98 -> 0.89 ms) and
    // complex links at d_R = 4, 6 in fp32 (C4: 4.91 -> 4.47 ms; SU(3) SYM 32^4 0.47 -> 0.34 ms; d_R = 5 has only one-row chunks and loses).  In fp64 at d_R >= 4 (half-spinor split over 4 warps: C4 10.7 vs 10.3 ms) and for real
    // links in fp32 the gather-layout kernels are faster; variant 5 forces it anywhere.
    if (L.bi != 0.0 && variant != 0 && variant != 3 && variant != 4 && variant != 5) return KERR_UNSUPPORTED;   // direct-load kernels: no gamma_5 factor on the hop sum
    if (hop_full_eligible(L) && (variant == 5 || (variant == 0 && hop_full_default<T, DR, REAL>()))) return launch_hop_full<T, DR, REAL>(g, L, s);
    // the fused reductions exist in the tile-pair kernel and in the persistent ring / pair kernels (variants 0, 3, 4)
    if (L.red_mode != 0 && variant != 0 && variant != 3 && variant != 4) return KERR_UNSUPPORTED;
    if (variant == 5) variant = 0;
    if (variant == 0) {
        // one thread per site spills in fp64 from d_R = 5 on; in fp32 at d_R >= 5 only the passes with a diagonal
        // term (self block in shared memory, fewer ring stages) run better with two warps per tile (profiles/)
        const bool self = (L.a != 0.0) && L.set[0].self != nullptr;
        variant = (DR >= 5 && (sizeof(T) == 8 || self)) ? 4 : 3;
    }
    if (L.tile_end > 0 && variant < 3) return KERR_UNSUPPORTED;   // slab regions: persistent kernels only
    switch (variant) {
    case 1: return launch_hop_small<T, DR, REAL, 1, 128>(g, L, s);
    case 2: return launch_hop_small<T, DR, REAL, 2, 128>(g, L, s);
    case 3: return launch_hop_ring<T, DR, REAL>(g, L, s);
    case 4: return launch_hop_pair<T, DR, REAL>(g, L, s);
    }
    return KERR_UNSUPPORTED;
}

// d_R >= 8: variant 0 = row-group kernel with bulk-copy rings (hop_rows.cuh; R rows per warp, TP tiles per CTA;
// shapes from a sweep on 32x24^3, profiles/r01b_summary.md),
// variant 1 = the direct-load row-group kernel of round 1 (hop_large.cuh), kept for comparison
template <typename T, int DR, bool REAL, int R, int TP> int hop_large_variant(const Geo &g, int variant, const HopLaunch &L, cudaStream_t s) {
    if (L.red_mode != 0 || L.diag_mode != DIAG_NONE) return KERR_UNSUPPORTED;
    if (variant == 0) return launch_hop_rows<T, DR, REAL, R, TP>(g, L, s);
    if (variant == 1 && L.tile_end == 0 && L.bi == 0.0) return launch_hop_large<T, DR, REAL, R>(g, L, s);
    return KERR_UNSUPPORTED;
}

// link mode REBUILD: the pair kernel with the fundamental block in the ring and R rebuilt row by row (rep_maps.cuh).
// Instantiated for every (N_g, rep) with d_R <= 6; the adjoint of SU(3..6) has its own matrix-free kernel.
template <typename T, int N, int REP> int hop_rebuild(const Geo &g, int variant, const HopLaunch &L, cudaStream_t s) {
    using M = RepMap<T, N, REP>;
    if (variant != 0 && variant != 4) return KERR_UNSUPPORTED;
    return launch_hop_pair<T, M::DR, M::REAL, N, REP>(g, L, s);
}
template <typename T> int hop_rebuild_by_config(const Geo &g, int N, int rep, int variant, const HopLaunch &L, cudaStream_t s) {
    if (L.red_mode != 0 || L.diag_mode != DIAG_NONE) return KERR_UNSUPPORTED;
    switch (rep * 10 + N) {
    case 2: return hop_rebuild<T, 2, 0>(g, variant, L, s);    // FUND
    case 3: return hop_rebuild<T, 3, 0>(g, variant, L, s);
    case 4: return hop_rebuild<T, 4, 0>(g, variant, L, s);
    case 5: return hop_rebuild<T, 5, 0>(g, variant, L, s);
    case 6: return hop_rebuild<T, 6, 0>(g, variant, L, s);
    case 12: return hop_rebuild<T, 2, 1>(g, variant, L, s);   // ADJ SU(2), d_R = 3
    // ADJ SU(3..6), d_R = 8..35: matrix-free, psi^a T^a -> W (psi^a T^a) W^dagger on the fundamental link (hop_adjmf.cuh)
    case 13: return (variant == 0 && L.tile_end == 0) ? launch_hop_adjmf<T, 3>(g, L, s) : KERR_UNSUPPORTED;
    case 14: return (variant == 0 && L.tile_end == 0) ? launch_hop_adjmf<T, 4>(g, L, s) : KERR_UNSUPPORTED;
    case 15: return (variant == 0 && L.tile_end == 0) ? launch_hop_adjmf<T, 5>(g, L, s) : KERR_UNSUPPORTED;
    case 16: return (variant == 0 && L.tile_end == 0) ? launch_hop_adjmf<T, 6>(g, L, s) : KERR_UNSUPPORTED;
    case 22: return hop_rebuild<T, 2, 2>(g, variant, L, s);   // SYM SU(2), SU(3): d_R = 3, 6
    case 23: return hop_rebuild<T, 3, 2>(g, variant, L, s);
    case 32: return hop_rebuild<T, 2, 3>(g, variant, L, s);   // 2AS SU(2), SU(3), SU(4): d_R = 1, 3, 6
    case 33: return hop_rebuild<T, 3, 3>(g, variant, L, s);
    case 34: return hop_rebuild<T, 4, 3>(g, variant, L, s);
    }
    return KERR_UNSUPPORTED;
}

template <typename T> int hop_by_config(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s) {
    if (mode == 1) return hop_rebuild_by_config<T>(g, N, rep, variant, L, s);
    if (mode != 0) return KERR_UNSUPPORTED;
    const int dR = (rep == 0) ? N : (rep == 1) ? N * N - 1 : (rep == 2) ? N * (N + 1) / 2 : N * (N - 1) / 2;
    const bool real = (rep == 1);
    if (!real) {
        switch (dR) {
        case 1: return hop_small_variant<T, 1, false>(g, variant, L, s);   // SU(2) 2AS: R = det U (allowed)
        case 2: return hop_small_variant<T, 2, false>(g, variant, L, s);
        case 3: return hop_small_variant<T, 3, false>(g, variant, L, s);
        case 4: return hop_small_variant<T, 4, false>(g, variant, L, s);
        case 5: return hop_small_variant<T, 5, false>(g, variant, L, s);
        case 6: return hop_small_variant<T, 6, false>(g, variant, L, s);
        case 10: return hop_large_variant<T, 10, false, 2, 2>(g, variant, L, s);   // SU(4) SYM, SU(5) 2AS
        case 15: return hop_large_variant<T, 15, false, 3, 2>(g, variant, L, s);   // SU(5) SYM, SU(6) 2AS
        case 21: return hop_large_variant<T, 21, false, 3, 1>(g, variant, L, s);   // SU(6) SYM
        }
    } else {
        switch (dR) {
        case 3: return hop_small_variant<T, 3, true>(g, variant, L, s);
        case 8: return hop_large_variant<T, 8, true, 4, 4>(g, variant, L, s);      // SU(3) ADJ
        case 15:                                                                   // SU(4) ADJ
            if constexpr (sizeof(T) == 8) return hop_large_variant<T, 15, true, 3, 1>(g, variant, L, s);
            else return hop_large_variant<T, 15, true, 3, 2>(g, variant, L, s);
        case 24: return hop_large_variant<T, 24, true, 4, 1>(g, variant, L, s);    // SU(5) ADJ
        case 35: return hop_large_variant<T, 35, true, 5, 1>(g, variant, L, s);    // SU(6) ADJ
        }
    }
    return KERR_UNSUPPORTED;
}

int k_hop_f64(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s);
int k_hop_f32(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s);

}  // namespace hirep
