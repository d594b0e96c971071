// hop_rows.cuh -- the hopping stencil for large d_R (d_R >= 8: one link matrix no longer fits one thread), with the
// link stream staged through shared memory by the bulk-copy engine.
//
//   out(x) = a*self(x) + b * sum_{d=0..7} P_d W_d(x) in(nbr_d(x)),   x of parity p_out            (Eq 8)
//
// This is the "D_R x site parallel" idea of the paper (L1532: one thread per row of the link matrix) with R rows
// per thread, re-shaped for sm_100a.  A GROUP of NG = d_R / R warps owns one tile of 32 sites (lane = site); warp
// w of the group owns rows i = wR .. wR+R-1 of every link matrix of the tile.  Per direction:
//   (a2) the group projects the neighbour spinor to the half spinor h (2 x d_R complex per site) into shared
//        memory (double buffered, one named barrier per direction); the loads of direction d+1 are issued before
//        the rows of direction d are multiplied, so their latency is hidden by the matvec;
//   (a3) every warp multiplies its R rows by both half-spinor components.  Its part of the link matrix arrives
//        through the warp's own ring of bulk-copy slots: one chunk = R rows x JB columns (R copies of JB x 32
//        contiguous elements on one mbarrier), consumed column by column so that each h_j read from shared memory
//        serves R rows -- without that the h reads would exceed the shared-memory bandwidth;
//   (a4) reconstruct + accumulate into the warp's R rows of the four spin components.
// The kernel is persistent (one CTA per SM, TP groups per CTA); the ring runs across directions and tiles, so the
// link stream (97 % of the bytes at SU(6) adjoint) never waits for the arithmetic.
#pragma once
#include "hop_ring.cuh"

namespace hirep {

template <typename T, int DR, bool REAL, int R, int TP, int JB, int STAGES, bool SELFBUF = false> struct RowsCfg {
    using E = link_elem<T, REAL>;
    static_assert(DR % R == 0 && DR % JB == 0, "row groups and column blocks must divide d_R");
    static constexpr int NG = DR / R, WARPS = NG * TP, NJB = DR / JB;
    static constexpr uint32_t SEG = JB * TILE * sizeof(E);            // one row's part of a chunk (one bulk copy)
    static constexpr uint32_t CHUNK = R * SEG;
    static constexpr uint32_t HBUF = 2 * DR * TILE * sizeof(cplx<T>);  // one half-spinor buffer of one group
    static constexpr size_t RING_BYTES = (size_t)WARPS * STAGES * CHUNK;
    static constexpr uint32_t SELF_BYTES = SELFBUF ? 4 * DR * TILE * sizeof(cplx<T>) : 0;   // the tile's own spinor, per group
    static constexpr size_t H_OFF = RING_BYTES, SELF_OFF = H_OFF + (size_t)TP * 2 * HBUF;
    static constexpr size_t BARS_OFF = SELF_OFF + (size_t)TP * SELF_BYTES;
    static constexpr size_t SMEM = BARS_OFF + (size_t)WARPS * STAGES * 8 + (size_t)TP * 8;
    static_assert(SEG % 16 == 0, "bulk copies move multiples of 16 bytes");
    static_assert(WARPS <= 32 && TP <= 15, "CTA shape");
    static_assert(SMEM <= 227 * 1024, "rings do not fit the 227 KB of shared memory of an sm_100 CTA");
};

__device__ __forceinline__ void group_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

template <typename T, int DR, bool REAL, int R, int TP, int JB, int STAGES, bool SELFBUF>
__global__ void __launch_bounds__(32 * (DR / R) * TP, 1) hop_rows_kernel(const Geo g, const HopLaunch L) {
    using C = cplx<T>;
    using E = link_elem<T, REAL>;
    using Cfg = RowsCfg<T, DR, REAL, R, TP, JB, STAGES, SELFBUF>;
    constexpr int NC = 4 * DR, NE = DR * DR, NG = Cfg::NG, NJB = Cfg::NJB;
    constexpr int CPT = 8 * NJB;                                       // chunks per tile (per warp)
    extern __shared__ __align__(128) unsigned char smem_raw[];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int grp = warp / NG, wg = warp % NG, i0 = wg * R;
    const E *ring = reinterpret_cast<const E *>(smem_raw + (size_t)warp * STAGES * Cfg::CHUNK);
    C *hbuf = reinterpret_cast<C *>(smem_raw + Cfg::H_OFF + (size_t)grp * 2 * Cfg::HBUF);
    const uint32_t ring_s = smem_u32(ring);
    const uint32_t bars_s = smem_u32(smem_raw + Cfg::BARS_OFF) + warp * STAGES * 8;
    const C *selfbuf = reinterpret_cast<const C *>(smem_raw + Cfg::SELF_OFF + (size_t)grp * Cfg::SELF_BYTES);
    const uint32_t self_s = smem_u32(selfbuf);
    const uint32_t selfbar_s = smem_u32(smem_raw + Cfg::BARS_OFF) + Cfg::WARPS * STAGES * 8 + grp * 8;
    if (lane == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(bars_s + 8 * s, 1);
        if (SELFBUF && wg == 0) mbar_init(selfbar_s, 1);
        fence_mbar_init();
    }
    __syncwarp();
    if constexpr (SELFBUF) group_sync(1 + grp, NG * 32);   // the group's self barrier is initialised before anyone waits on it
    pdl_launch_dependents();
    pdl_wait();

    const bool two = L.nsets == 2;
    const int total_tiles = launch_tiles(g, L) * L.nsets;
    const int gg = blockIdx.x * TP + grp, ngr = gridDim.x * TP;
    if (gg >= total_tiles) return;                                     // whole group leaves together
    const int my_tiles = (total_tiles - gg + ngr - 1) / ngr;
    const int my_chunks = my_tiles * CPT;
    const uint64_t pol = l2_policy_evict_first();

    auto locate = [&](int k, int &set_, int &tile_) {
        const int gt = gg + k * ngr;
        set_ = two ? (gt & 1) : 0;
        tile_ = (two ? (gt >> 1) : gt) + L.tile_begin;
    };
    // chunk qi of this warp: tile qi / CPT, direction (qi % CPT) / NJB, column block qi % NJB; R row segments
    auto issue = [&](int qi, int slot) {
        const int kq = qi / CPT, rem = qi - kq * CPT;
        const int step = rem / NJB, jb = rem - step * NJB, d = dir_of<false>(step);   // the walk of common.cuh
        int set_, tile_;
        locate(kq, set_, tile_);
        const E *src = (const E *)(set_ ? L.set[1].links : L.set[0].links) +
                       (((size_t)tile_ * 8 + d) * NE + (size_t)i0 * DR + jb * JB) * TILE;
        const uint32_t bar = bars_s + 8 * slot, dst = ring_s + slot * Cfg::CHUNK;
        mbar_expect_tx(bar, Cfg::CHUNK);
#pragma unroll
        for (int r = 0; r < R; ++r) bulk_g2s(dst + r * Cfg::SEG, src + (size_t)r * DR * TILE, Cfg::SEG, bar, pol);
    };
    if (lane == 0) {
        const int n0 = my_chunks < STAGES ? my_chunks : STAGES;
        for (int qi = 0; qi < n0; ++qi) issue(qi, qi);
    }

    int set, tile, t, x, y, zh, p_out;
    bool active;
    const C *in;
    auto enter_tile = [&](int k) {
        locate(k, set, tile);
        int h = tile * TILE + lane;
        active = h < g.Nh;
        if (!active) h = g.Nh - 1;
        decode_site(g, h, t, x, y, zh);
        p_out = set ? L.set[1].p_out : L.set[0].p_out;
        in = (const C *)(set ? L.set[1].in : L.set[0].in);
    };
    // this warp projects colours j = wg + NG*m, m < R (d_R = NG*R): the 4 spin components of each
    C nb[R][4];
    auto fetch = [&](int hn) {
        const C *src = in + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
#pragma unroll
        for (int m = 0; m < R; ++m)
#pragma unroll
            for (int sp = 0; sp < 4; ++sp) nb[m][sp] = ld_spinor<T>(src + (size_t)(sp * DR + wg + NG * m) * TILE);
    };

    enter_tile(0);
    fetch(neighbour<dir_of<false>(0)>(g, p_out, t, x, y, zh));
    int q = 0, slot = 0;
    uint32_t phase = 0;
    const T a = (T)L.a, b = (T)L.b, bi = (T)L.bi;
    const T am = (T)L.am;
    const T g5s = L.g5 ? T(-1) : T(1);

    for (int k = 0; k < my_tiles; ++k) {
        const int c_set = set, c_tile = tile;
        const bool c_active = active;
        C up[2][R], lo[2][R];
#pragma unroll
        for (int s = 0; s < 2; ++s)
#pragma unroll
            for (int r = 0; r < R; ++r) up[s][r] = lo[s][r] = mk<T>(0, 0);

        static_for<0, 8>([&](auto dc) {
            constexpr int I = decltype(dc)::value, D = dir_of<false>(I);
            using DI = DirInfo<D>;
            C *hb = hbuf + (I & 1) * (2 * DR * TILE);
            // (a2) projection of this warp's colours into the group's half-spinor buffer
#pragma unroll
            for (int m = 0; m < R; ++m)
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    const int qq = DI::swap ? 1 - s : s;
                    const T cs = (T)(DI::sg * DI::sigma(s));
                    const C u = nb[m][s], v = nb[m][2 + qq];
                    C hv;
                    if (DI::imag) hv = mk<T>(fma(-cs, v.y, u.x), fma(cs, v.x, u.y));
                    else hv = mk<T>(fma(cs, v.x, u.x), fma(cs, v.y, u.y));
                    hb[(s * DR + wg + NG * m) * TILE + lane] = hv;
                }
            // prefetch the next neighbour (next direction, or direction 0 of the group's next tile)
            if constexpr (I < 7) {
                fetch(neighbour<dir_of<false>(I + 1)>(g, p_out, t, x, y, zh));
            } else {
                if (k + 1 < my_tiles) {
                    enter_tile(k + 1);
                    fetch(neighbour<dir_of<false>(0)>(g, p_out, t, x, y, zh));
                }
            }
            group_sync(1 + grp, NG * 32);   // h of step I complete; buffer (I&1) was last read at step I-2
            if constexpr (SELFBUF && I == 0) {
                // every warp of the group has passed the previous tile's epilogue: its self block may be overwritten.
                // One bulk copy fetches this tile's own spinor (a contiguous block); it is consumed 7 steps later.
                if (wg == 0 && lane == 0) {
                    fence_proxy_async();
                    const C *sp = (const C *)(c_set ? L.set[1].self : L.set[0].self) + ((size_t)c_tile * NC) * TILE;
                    mbar_expect_tx(selfbar_s, Cfg::SELF_BYTES);
                    bulk_g2s_plain(self_s, sp, Cfg::SELF_BYTES, selfbar_s);
                }
            }
            // (a3) rows i0 .. i0+R-1 times both half-spinor components, column block by column block
            C chi[2][R];
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int r = 0; r < R; ++r) chi[s][r] = mk<T>(0, 0);
#pragma unroll 1
            for (int jb = 0; jb < NJB; ++jb) {
                mbar_wait(bars_s + 8 * slot, phase);
                const E *W = ring + (size_t)slot * (R * JB * TILE) + lane;
                const C *h0 = hb + (jb * JB) * TILE + lane, *h1 = h0 + DR * TILE;
#pragma unroll
                for (int jj = 0; jj < JB; ++jj) {
                    const C x0 = h0[jj * TILE], x1 = h1[jj * TILE];
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const E w = W[(r * JB + jj) * TILE];
                        mac<T>(chi[0][r], w, x0);
                        mac<T>(chi[1][r], w, x1);
                    }
                }
                __syncwarp();
                if (lane == 0 && q + STAGES < my_chunks) {
                    fence_proxy_async();
                    issue(q + STAGES, slot);
                }
                ++q;
                if (++slot == STAGES) { slot = 0; phase ^= 1; }
            }
            // (a4) reconstruct + accumulate
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int qq = DI::swap ? 1 - s : s;
                const T cl = (T)(DI::sg * DI::sigma(s));
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    up[s][r].x += chi[s][r].x;
                    up[s][r].y += chi[s][r].y;
                    if (DI::imag) { lo[qq][r].x += cl * chi[s][r].y; lo[qq][r].y -= cl * chi[s][r].x; }
                    else { lo[qq][r].x += cl * chi[s][r].x; lo[qq][r].y += cl * chi[s][r].y; }
                }
            }
        });

        if constexpr (SELFBUF) mbar_wait(selfbar_s, k & 1);
        if (c_active) {
            C *out = (C *)(c_set ? L.set[1].out : L.set[0].out) + ((size_t)c_tile * NC) * TILE + lane;
            const C *self_base = (const C *)(c_set ? L.set[1].self : L.set[0].self);
            const C *self = SELFBUF ? selfbuf + lane : self_base + ((size_t)c_tile * NC) * TILE + lane;
            const bool use_self = SELFBUF || ((self_base != nullptr) && (L.a != 0.0));
#pragma unroll
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int i = i0 + r;
                    C vu = mk<T>(b * up[s][r].x, b * up[s][r].y);
                    C vl = mk<T>(b * lo[s][r].x, b * lo[s][r].y);
                    if (bi != T(0)) {   // (b + i bi gamma_5) hop
                        vu = mk<T>(fma(-bi, up[s][r].y, vu.x), fma(bi, up[s][r].x, vu.y));
                        vl = mk<T>(fma(bi, lo[s][r].y, vl.x), fma(-bi, lo[s][r].x, vl.y));
                    }
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
                    st_spinor(out + (size_t)(s * DR + i) * TILE, vu);
                    st_spinor(out + (size_t)((2 + s) * DR + i) * TILE, mk<T>(g5s * vl.x, g5s * vl.y));
                }
        }
    }
}

// shape per instantiation: R rows per warp and TP groups per CTA are given; column block = the largest divisor of d_R
// with a chunk of at most 13 KB; as many stages (2..4) as fit next to the half-spinor buffers
template <typename T, int DR, bool REAL, int R, int TP, bool SELFBUF = false> struct RowsPick {
    using E = link_elem<T, REAL>;
    static constexpr int WARPS = (DR / R) * TP;
    static constexpr size_t chunk_of(int c) { return (size_t)R * c * TILE * sizeof(E); }
    static constexpr int stages_of(int c) {
        const size_t fixed = (size_t)TP * (2 * 2 + (SELFBUF ? 4 : 0)) * DR * TILE * sizeof(cplx<T>) + 8 * TP;
        if (fixed >= 226 * 1024) return 0;
        const size_t avail = 226 * 1024 - fixed;
        const int st = (int)(avail / (WARPS * (chunk_of(c) + 8)));
        return st > 4 ? 4 : st;
    }
    static constexpr int pick_jb() {
        int best = 1;
        for (int c = 1; c <= DR; ++c)
            if (DR % c == 0 && chunk_of(c) <= 13 * 1024 && stages_of(c) >= 2) best = c;
        return best;
    }
    static constexpr int JB = pick_jb();
    static constexpr int STAGES = stages_of(JB);
    static constexpr bool FITS = STAGES >= 2;
};

template <typename T, int DR, bool REAL, int R, int TP, bool SELFBUF>
int launch_hop_rows_cfg(const Geo &g, const HopLaunch &L, cudaStream_t s) {
    using P = RowsPick<T, DR, REAL, R, TP, SELFBUF>;
    static_assert(P::FITS, "row ring needs at least two stages");
    using Cfg = RowsCfg<T, DR, REAL, R, TP, P::JB, P::STAGES, SELFBUF>;
    auto kern = hop_rows_kernel<T, DR, REAL, R, TP, P::JB, P::STAGES, SELFBUF>;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, Cfg::SMEM, cache, n_sm)) return rc;
    const int grid = ring_grid(n_sm, L.max_ctas, launch_tiles(g, L) * L.nsets, TP);
    return launch_pdl(kern, grid, Cfg::WARPS * 32, Cfg::SMEM, s, g, L);
}

// passes with a diagonal term stage the tile's own spinor through shared memory when it fits next to two ring stages
// (the epilogue load is otherwise exposed latency -- 45 % of a tile at d_R = 8 in fp32); SU(6) adjoint fp64 does not fit
// and its tiles are long enough (60 us) not to care
template <typename T, int DR, bool REAL, int R, int TP>
int launch_hop_rows(const Geo &g, const HopLaunch &L, cudaStream_t s) {
    const bool self = (L.a != 0.0) && L.set[0].self != nullptr;
    using PS = RowsPick<T, DR, REAL, R, TP, true>;
    using PN = RowsPick<T, DR, REAL, R, TP, false>;
    if constexpr (PS::FITS && PS::JB == PN::JB) {   // only if the ring keeps its chunk size (SU(6) adjoint fp64 would not)
        if (self) return launch_hop_rows_cfg<T, DR, REAL, R, TP, true>(g, L, s);
    }
    return launch_hop_rows_cfg<T, DR, REAL, R, TP, false>(g, L, s);
}

}  // namespace hirep
