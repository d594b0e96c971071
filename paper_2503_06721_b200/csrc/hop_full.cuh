// hop_full.cuh -- the FULL-LATTICE Wilson operator with every represented link crossing the SM once.
//
//   out(x) = a*self(x) + b * sum_{d=0..7} P_d W_d(x) in(nbr_d(x)),   all x (both parities)            (Eq 8)
//
// Why another kernel.  The half-lattice kernels (hop_ring / hop_pair) read the gather block of a tile: 8 matrices per
// site, U_mu(x) and U_mu(x-mu)^dagger.  On the full lattice every U_mu(x) is needed twice -- forward by x, daggered
// backward by x+mu -- so that scheme moves 8K per site where (2S+4K) is compulsory: 1.58x (SU(3), 32^4) to 2.0x the
// compulsory DRAM traffic, 0.59 of the roofline.  It also asks L2 for (10S+8K) per site, 3.2 GB per launch at SU(3) fp64 -- 12 TB/s
// at 0.26 ms, the order of what the L2 slices deliver (B300_MICROARCH.md) -- so the second use of a link is served ON THE SM here
// rather than from L2.
//
// Scheme.  A GROUP of warps owns the tile PAIR (even tile k, odd tile k): the 64 sites (t,x,y,z) with the same half
// index h in both parities.  Those sites are each other's z neighbours (and, for the rows inside the tile, y
// neighbours), so inside the group
//   * the input spinor tiles of both parities are staged ONCE in shared memory (two bulk copies): each is the
//     diagonal term of its own parity and the neighbour data of the other;
//   * only the FORWARD halves U_mu(x) (d < 4) of the gather blocks are streamed (bulk copies, both parities per ring
//     slot).  The forward hop multiplies by the site's own rows; the backward hop of the OTHER parity's site x+mu
//     needs U_mu(x)^dagger and reads the same shared-memory matrix, transposed and conjugated on the fly
//     (column-oriented accumulation: row j of U contributes conj(U_ji) h_j to every chi_i, so both hops consume the
//     matrix row chunk by row chunk);
//   * what is not in the tile pair -- the +-t, +-x (and half of the +-y) neighbours: spinors, and the links of the
//     backward hops -- is GATHERED per lane with cp.async (16/8/4-byte asynchronous copies, no registers) into
//     shared memory: link rows into the gather part of the ring slot they are consumed with (same mbarrier as the
//     bulk part), neighbour spinors into a per-warp buffer one direction ahead -- or (NBREG, complex links) through
//     registers by read-only loads issued half a direction pair ahead, which leaves the shared memory to more groups.
// Requests to L2 per site drop from 10S+8K to about 7S+6.5K (L = 32), DRAM traffic from 2S+8K towards 2S+4K (the
// backward t links of a tile pair were streamed by another group of the same or the previous grid round).
// Optionally (SPLIT) the two half-spinor components are split over two warps as in hop_pair.cuh (fp64, d_R >= 4).
#pragma once
#include "hop_pair.cuh"
#include "reduce.cuh"

namespace hirep {

template <int BYTES> __device__ __forceinline__ void cp_async(uint32_t dst, const void *src) {
    if constexpr (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
    else asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(dst), "l"(src), "n"(BYTES) : "memory");
}
// the executing thread's earlier cp.async copies arrive on the mbarrier when they have landed (the arrival is part
// of the barrier's initial count: .noinc)
__device__ __forceinline__ void cp_async_arrive_noinc(uint32_t bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
// acc += conj(w) * h   (real links: w * h)
template <typename T> __device__ __forceinline__ void macc(cplx<T> &acc, const cplx<T> &w, const cplx<T> &h) {
    acc.x = fma(w.x, h.x, acc.x);
    acc.x = fma(w.y, h.y, acc.x);
    acc.y = fma(w.x, h.y, acc.y);
    acc.y = fma(-w.y, h.x, acc.y);
}
template <typename T> __device__ __forceinline__ void macc(cplx<T> &acc, const T &w, const cplx<T> &h) {
    acc.x = fma(w, h.x, acc.x);
    acc.y = fma(w, h.y, acc.y);
}

template <typename T, int DR, bool REAL, bool SPLIT, int GROUPS, int STAGES, int RPC, bool NBREG = false> struct FullCfg {
    using E = link_elem<T, REAL>;
    using C = cplx<T>;
    static_assert(DR % RPC == 0, "rows per chunk must divide d_R");
    static constexpr int GW = SPLIT ? 4 : 2;                           // warps per group: (parity) x (half-spinor component)
    static constexpr int CPD = DR / RPC, CPT = 4 * CPD;                // chunks per direction pair / per tile pair
    static constexpr uint32_t CH = RPC * DR * TILE * sizeof(E);        // RPC rows of one parity's U_mu
    static constexpr uint32_t SLOT = 4 * CH;                           // forward rows even | odd | gathered rows even | odd
    static constexpr uint32_t SB = 4 * DR * TILE * sizeof(C);          // one spinor tile
    static constexpr int NBC = SPLIT ? 2 * DR : 4 * DR;                // neighbour components a warp stages per direction
    // NBREG: the out-of-pair neighbour spinors travel through registers (read-only loads issued half a direction pair ahead)
    // instead of a per-warp shared-memory buffer: 2 x 4 d_R x 512 B per warp go to the ring (one more stage or one more group)

    static constexpr uint32_t NBD = NBREG ? 0 : NBC * TILE * sizeof(C);   // one direction of a warp's neighbour buffer
    static constexpr uint32_t XB = SPLIT ? 2 * 2 * DR * TILE * sizeof(C) : 0;   // cross contributions [parity][s][d_R][32]
    static constexpr size_t SP_OFF = (size_t)STAGES * SLOT, NB_OFF = SP_OFF + 2 * SB, X_OFF = NB_OFF + (size_t)GW * 2 * NBD;
    static constexpr size_t BAR_OFF = X_OFF + XB;
    static constexpr int NBAR = 2 * STAGES + 2 + GW;                   // full[S], empty[S], spinor full / empty, nbfull[GW]
    static constexpr size_t PER_GROUP = (BAR_OFF + NBAR * 8 + 127) & ~(size_t)127;
    static constexpr size_t SMEM = PER_GROUP * GROUPS;
    static_assert(CH % 16 == 0 && SB % 16 == 0, "bulk copies move multiples of 16 bytes");
    static_assert(STAGES <= CPT, "a chunk issued ahead belongs to this tile pair or the next");
    static_assert(SMEM <= 227 * 1024, "does not fit the 227 KB of shared memory of an sm_100 CTA");
    static_assert(GROUPS * (SPLIT ? 3 : 1) + 1 <= 16, "named barriers");
};

// half spinor h = psi_up + sg e_mu psi_low of one neighbour (step a2), read from shared memory: the other parity's
// staged tile (neighbour inside the tile pair, lane ln) or this warp's gathered copy
template <typename T, int DR, bool SPLIT, typename DI>
__device__ __forceinline__ void project_half(const cplx<T> *spo, const cplx<T> *nbd, bool in_tile, int ln, int lane, int s_rt,
                                             cplx<T> (&h)[SPLIT ? 1 : 2][DR]) {
    using C = cplx<T>;
    constexpr int NSC = SPLIT ? 1 : 2;
#pragma unroll
    for (int kk = 0; kk < NSC; ++kk) {
        const int s = SPLIT ? s_rt : kk;
        const int qq = DI::swap ? 1 - s : s;
        const T cs = (T)(DI::sg * DI::sigma(s));
        const C *pu, *pl;
        if constexpr (SPLIT) {   // gathered copy holds [upper s | lower q(s)] only
            pu = in_tile ? spo + (size_t)(s * DR) * TILE + ln : nbd + lane;
            pl = in_tile ? spo + (size_t)((2 + qq) * DR) * TILE + ln : nbd + (size_t)DR * TILE + lane;
        } else {
            const C *pf = in_tile ? spo + ln : nbd + lane;
            pu = pf + (size_t)(s * DR) * TILE;
            pl = pf + (size_t)((2 + qq) * DR) * TILE;
        }
#pragma unroll
        for (int c = 0; c < DR; ++c) {
            const C u = pu[c * TILE], v = pl[c * TILE];
            if (DI::imag) h[kk][c] = mk<T>(fma(-cs, v.y, u.x), fma(cs, v.x, u.y));   // u + i cs v
            else h[kk][c] = mk<T>(fma(cs, v.x, u.x), fma(cs, v.y, u.y));             // u + cs v
        }
    }
}

// the same with the out-of-pair neighbour in registers (NBREG).  nb holds the components this warp needs: all 4 d_R (one
// thread per site) or [upper s | lower q(s)] (SPLIT)
template <typename T, int DR, bool SPLIT, typename DI>
__device__ __forceinline__ void project_regs(const cplx<T> *spo, const cplx<T> (&nb)[(SPLIT ? 2 : 4) * DR], bool in_tile, int ln, int s_rt,
                                             cplx<T> (&h)[SPLIT ? 1 : 2][DR]) {
    using C = cplx<T>;
    constexpr int NSC = SPLIT ? 1 : 2;
#pragma unroll
    for (int kk = 0; kk < NSC; ++kk) {
        const int s = SPLIT ? s_rt : kk;
        const int qq = DI::swap ? 1 - s : s;
        const T cs = (T)(DI::sg * DI::sigma(s));
#pragma unroll
        for (int c = 0; c < DR; ++c) {
            C u = SPLIT ? nb[c] : nb[kk * DR + c];
            C v = SPLIT ? nb[DR + c] : nb[(2 + (DI::swap ? 1 - kk : kk)) * DR + c];
            if (in_tile) { u = spo[(size_t)(s * DR + c) * TILE + ln]; v = spo[(size_t)((2 + qq) * DR + c) * TILE + ln]; }
            if (DI::imag) h[kk][c] = mk<T>(fma(-cs, v.y, u.x), fma(cs, v.x, u.y));
            else h[kk][c] = mk<T>(fma(cs, v.x, u.x), fma(cs, v.y, u.y));
        }
    }
}

// (a4) reconstruct + accumulate chi = W h of direction DI, row i, component s
template <typename T, int DR, bool SPLIT, typename DI>
__device__ __forceinline__ void accumulate(const cplx<T> &chi, int kk, int s, int i, cplx<T> (&up)[SPLIT ? 1 : 2][DR],
                                           cplx<T> (&lo)[SPLIT ? 1 : 2][DR], cplx<T> (&lx)[SPLIT ? 1 : 2][DR]) {
    up[kk][i].x += chi.x;
    up[kk][i].y += chi.y;
    const T cl = (T)(DI::sg * DI::sigma(s));
    cplx<T> add;   // sg conj(k_mu(s)) chi
    if (DI::imag) add = mk<T>(cl * chi.y, -cl * chi.x);
    else add = mk<T>(cl * chi.x, cl * chi.y);
    if constexpr (SPLIT) {
        if (DI::swap) { lx[0][i].x += add.x; lx[0][i].y += add.y; }
        else { lo[0][i].x += add.x; lo[0][i].y += add.y; }
    } else {
        const int qq = DI::swap ? 1 - s : s;
        lo[qq][i].x += add.x;
        lo[qq][i].y += add.y;
    }
}

template <typename T, int DR, bool REAL, bool SPLIT, int GROUPS, int STAGES, int RPC, bool NBREG>
__global__ void __launch_bounds__(GROUPS * (SPLIT ? 4 : 2) * 32, 1) hop_full_kernel(const Geo g, const HopLaunch L) {
    using C = cplx<T>;
    using E = link_elem<T, REAL>;
    using Cfg = FullCfg<T, DR, REAL, SPLIT, GROUPS, STAGES, RPC, NBREG>;
    constexpr int GW = Cfg::GW, NC = 4 * DR, NE = DR * DR, CPD = Cfg::CPD, CPT = Cfg::CPT, NSC = SPLIT ? 1 : 2;
    constexpr uint32_t CH = Cfg::CH, SLOT = Cfg::SLOT, SB = Cfg::SB, NBD = Cfg::NBD;
    extern __shared__ __align__(128) unsigned char smem_raw[];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int grp = warp / GW, wg = warp % GW;
    const int par = wg & 1, s_rt = wg >> 1;            // this warp: output parity, half-spinor component (SPLIT)
    unsigned char *base = smem_raw + (size_t)grp * Cfg::PER_GROUP;
    const unsigned char *ring = base;
    const C *sp = reinterpret_cast<const C *>(base + Cfg::SP_OFF);                       // [parity][4 d_R][32]
    const C *nbuf = reinterpret_cast<const C *>(base + Cfg::NB_OFF + (size_t)wg * 2 * NBD);   // [+mu | -mu][NBC][32]
    C *xbuf = reinterpret_cast<C *>(base + Cfg::X_OFF);
    const uint32_t ring_s = smem_u32(ring), sp_s = smem_u32(sp), nbuf_s = smem_u32(nbuf);
    const uint32_t full_s = smem_u32(base + Cfg::BAR_OFF), empty_s = full_s + 8 * STAGES;
    const uint32_t spfull_s = empty_s + 8 * STAGES, spempty_s = spfull_s + 8, nbfull_s = spempty_s + 8 + 8 * wg;
    const bool producer = (wg == 0) && (lane == 0);
    if (producer) {
        for (int i = 0; i < STAGES; ++i) {
            mbar_init(full_s + 8 * i, 1 + GW * 32);    // the producer's expect_tx + every thread's gather arrival
            mbar_init(empty_s + 8 * i, GW);
        }
        mbar_init(spfull_s, 1);
        mbar_init(spempty_s, GW);
    }
    if (lane == 0) {
        mbar_init(nbfull_s, 32);
        fence_mbar_init();
    }
    group_sync(1 + grp, GW * 32);
    pdl_launch_dependents();
    pdl_wait();

    const int gg = blockIdx.x * GROUPS + grp, ng = gridDim.x * GROUPS;
    Acc racc{0.0, 0.0, 0.0};                            // fused reduction (HopLaunch::red_mode): this thread's compensated partial sum
    __shared__ Acc red_scratch[32];
    auto red_finish = [&]() {                           // every thread of the CTA calls this exactly once
        if (L.red_mode == 0) return;
        cta_merge(racc, L.red_alg, red_scratch);
        if (threadIdx.x == 0) {
            Acc *part = (Acc *)L.red_partial;
            part[2 * blockIdx.x] = racc;
            part[2 * blockIdx.x + 1] = Acc{0.0, 0.0, 0.0};
        }
    };
    if (gg >= g.n_tiles) { red_finish(); return; }      // the whole group leaves together
    const int my_tiles = (g.n_tiles - gg + ng - 1) / ng;
    const int my_chunks = my_tiles * CPT;

    // set[p] describes output parity p: set[p].in is the spinor on parity 1-p, set[p].links the gather blocks of parity p
    const C *in_nb = (const C *)(par ? L.set[1].in : L.set[0].in);          // neighbours of this warp's sites
    const E *lk_oth = (const E *)(par ? L.set[0].links : L.set[1].links);   // forward links of the other parity

    // ---- link stream: chunk c of a tile pair = rows [rc RPC, (rc+1) RPC) of U_mu, mu = c / CPD, of BOTH parities (bulk), plus,
    // per lane, the same rows of U_mu(x - mu) when that site lies outside the tile pair (cp.async gather)
    int iq_k = 0, iq_c = 0, iq_tile = 0, iq_hn0 = 0, iq_hn1 = 0, iq_hn2 = 0, iq_hn3 = 0;
    auto iq_enter = [&]() {
        iq_tile = gg + iq_k * ng;
        int h = iq_tile * TILE + lane;
        if (h >= g.Nh) h = g.Nh - 1;
        int t_, x_, y_, z_;
        decode_site(g, h, t_, x_, y_, z_);
        iq_hn0 = neighbour<4>(g, par, t_, x_, y_, z_);
        iq_hn1 = neighbour<5>(g, par, t_, x_, y_, z_);
        iq_hn2 = neighbour<6>(g, par, t_, x_, y_, z_);
        iq_hn3 = neighbour<7>(g, par, t_, x_, y_, z_);
    };
    auto issue_chunk = [&](int slot) {
        const int mu = iq_c / CPD, rc = iq_c - mu * CPD;
        const size_t off = (((size_t)iq_tile * 8 + mu) * NE + (size_t)rc * RPC * DR) * TILE;
        const uint32_t dst = ring_s + slot * SLOT, bar = full_s + 8 * slot;
        if (producer) {
            mbar_expect_tx(bar, 2 * CH);
            bulk_g2s_plain(dst, (const E *)L.set[0].links + off, CH, bar);
            bulk_g2s_plain(dst + CH, (const E *)L.set[1].links + off, CH, bar);
        }
        const int hn = mu == 0 ? iq_hn0 : mu == 1 ? iq_hn1 : mu == 2 ? iq_hn2 : iq_hn3;
        if ((hn >> 5) != iq_tile && !((L.dbg >> mu) & 1)) {
            const E *src = lk_oth + (((size_t)(hn >> 5) * 8 + mu) * NE + (size_t)rc * RPC * DR) * TILE + (hn & 31);
            const uint32_t d0 = dst + (2 + par) * CH + lane * (uint32_t)sizeof(E);
            constexpr int NEL = RPC * DR, HALF = (NEL + 1) / 2;
            const int e0 = SPLIT ? (s_rt ? HALF : 0) : 0, e1 = SPLIT ? (s_rt ? NEL : HALF) : NEL;   // the two s-warps share the gather
#pragma unroll
            for (int e = 0; e < NEL; ++e)
                if (e >= e0 && e < e1) cp_async<sizeof(E)>(d0 + e * TILE * (uint32_t)sizeof(E), src + (size_t)e * TILE);
        }
        cp_async_arrive_noinc(bar);
        if (++iq_c == CPT) {
            iq_c = 0;
            if (++iq_k < my_tiles) iq_enter();
        }
    };
    auto issue_sp = [&](int tile_) {   // producer only: both parities' input tiles
        mbar_expect_tx(spfull_s, 2 * SB);
        bulk_g2s_plain(sp_s, (const C *)L.set[1].in + (size_t)tile_ * NC * TILE, SB, spfull_s);        // even sites
        bulk_g2s_plain(sp_s + SB, (const C *)L.set[0].in + (size_t)tile_ * NC * TILE, SB, spfull_s);   // odd sites
    };

    // ---- compute-tile state and the per-warp neighbour staging (one direction pair ahead)
    int tile, t, x, y, zh;
    bool active;
    auto enter_tile = [&](int k) {
        tile = gg + k * ng;
        int h = tile * TILE + lane;
        active = h < g.Nh;
        if (!active) h = g.Nh - 1;
        decode_site(g, h, t, x, y, zh);
    };
    auto stage_dir = [&](int hn, int which, bool swap, int mu_) {
        if ((hn >> 5) != tile && !((L.dbg >> (4 + mu_)) & 1)) {
            const C *src = in_nb + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
            const uint32_t d0 = nbuf_s + which * NBD + lane * (uint32_t)sizeof(C);
            if constexpr (SPLIT) {
                const int ql = swap ? 1 - s_rt : s_rt;
#pragma unroll
                for (int c = 0; c < DR; ++c) {
                    cp_async<sizeof(C)>(d0 + c * TILE * (uint32_t)sizeof(C), src + (size_t)(s_rt * DR + c) * TILE);
                    cp_async<sizeof(C)>(d0 + (DR + c) * TILE * (uint32_t)sizeof(C), src + (size_t)((2 + ql) * DR + c) * TILE);
                }
            } else {
#pragma unroll
                for (int c = 0; c < NC; ++c) cp_async<sizeof(C)>(d0 + c * TILE * (uint32_t)sizeof(C), src + (size_t)c * TILE);
            }
        }
    };
    auto stage_nb = [&](auto muc) {
        constexpr int MU = decltype(muc)::value;
        stage_dir(neighbour<MU>(g, par, t, x, y, zh), 0, DirInfo<MU>::swap, MU);
        stage_dir(neighbour<4 + MU>(g, par, t, x, y, zh), 1, DirInfo<MU>::swap, MU);
        cp_async_arrive_noinc(nbfull_s);
    };

    C nb[NBREG ? Cfg::NBC : 1];
    auto fetch = [&](int hn, int mu_, bool swap) {   // NBREG: the out-of-pair neighbour's components (in-pair ones are read from the staged tiles)
        if constexpr (NBREG) {
            if ((hn >> 5) != tile && !((L.dbg >> (4 + mu_)) & 1)) {
                const C *src = in_nb + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
                if constexpr (SPLIT) {
                    const int ql = swap ? 1 - s_rt : s_rt;
#pragma unroll
                    for (int c = 0; c < DR; ++c) {
                        nb[c] = ld_spinor<T>(src + (size_t)(s_rt * DR + c) * TILE);
                        nb[DR + c] = ld_spinor<T>(src + (size_t)((2 + ql) * DR + c) * TILE);
                    }
                } else {
#pragma unroll
                    for (int c = 0; c < NC; ++c) nb[c] = ld_spinor<T>(src + (size_t)c * TILE);
                }
            }
        }
    };

    // ---- prologue
    iq_enter();
    {
        const int n0 = my_chunks < STAGES ? my_chunks : STAGES;
        for (int i = 0; i < n0; ++i) issue_chunk(i);
    }
    if (producer) issue_sp(gg);
    enter_tile(0);
    if constexpr (NBREG) fetch(neighbour<0>(g, par, t, x, y, zh), 0, DirInfo<0>::swap);
    else stage_nb(IntC<0>{});
    int q = 0, slot = 0;
    uint32_t phase = 0, nbphase = 0;
    const T b = (T)L.b, ab = (T)(L.a / L.b), amb = (T)(L.am / L.b);
    const T g5s = L.g5 ? T(-1) : T(1);

    for (int k = 0; k < my_tiles; ++k) {
        // Round pacing: without it the groups of the grid drift apart (no global synchronisation in a persistent kernel), and a
        // link block or spinor tile gathered from another tile pair has left L2 when the two groups are more than ~20 us apart
        // (6 TB/s turn the 126 MB over that fast).  Leaders are throttled, laggards never wait: a group may start its round k only
        // when the grid as a whole has completed (k - W) rounds' worth of tile pairs (one counter, one poll per group and round).
        if (L.pace_every > 0 && k >= L.pace_every) {
            if (wg == 0 && lane == 0) {
                const unsigned target = (unsigned)(k - L.pace_every) * (unsigned)ng;
                while (*((volatile unsigned *)L.pace) < target) __nanosleep(200);
            }
            group_sync(1 + grp, GW * 32);
        }
        const int c_tile = tile;
        const bool c_active = active;
        // the diagonal term goes into the accumulators first: out = b * ((a/b) self + i (am/b) gamma_5 self + hop), so that the
        // staged tiles are not needed after the last projection and can be refilled during the last direction pair
        C up[NSC][DR], lo[NSC][DR], lx[NSC][DR];   // non-SPLIT: lo[q] = lower component q; SPLIT: lo[0] = lower s, lx[0] = lower 1-s
        mbar_wait(spfull_s, k & 1);
        {
            const C *self = sp + (size_t)par * NC * TILE + lane;
#pragma unroll
            for (int kk = 0; kk < NSC; ++kk) {
                const int s = SPLIT ? s_rt : kk;
#pragma unroll
                for (int c = 0; c < DR; ++c) {
                    const C su = self[(size_t)(s * DR + c) * TILE], sl = self[(size_t)((2 + s) * DR + c) * TILE];
                    up[kk][c] = mk<T>(fma(-amb, su.y, ab * su.x), fma(amb, su.x, ab * su.y));   // (a + i am) psi_up   (Eq 51)
                    lo[kk][c] = mk<T>(fma(amb, sl.y, ab * sl.x), fma(-amb, sl.x, ab * sl.y));   // (a - i am) psi_low
                    lx[kk][c] = mk<T>(0, 0);
                }
            }
        }

        static_for<0, 4>([&](auto mc) {
            constexpr int MU = decltype(mc)::value;
            using DF = DirInfo<MU>;
            using DB = DirInfo<4 + MU>;
            const int hnf = neighbour<MU>(g, par, t, x, y, zh), hnb = neighbour<4 + MU>(g, par, t, x, y, zh);
            const bool inf = (hnf >> 5) == c_tile, inb = (hnb >> 5) == c_tile;
            const int lnb = hnb & 31;
            if constexpr (NBREG) {
                // forward hop of the first chunk while the -mu neighbour is in flight, backward hops while the next +mu one is
                const C *spo = sp + (size_t)(1 - par) * NC * TILE;
                C hp[NSC][DR], hm[NSC][DR];
                project_regs<T, DR, SPLIT, DF>(spo, nb, inf, hnf & 31, s_rt, hp);
                fetch(hnb, MU, DB::swap);
                C chib[NSC][DR];
#pragma unroll
                for (int kk = 0; kk < NSC; ++kk)
#pragma unroll
                    for (int c = 0; c < DR; ++c) chib[kk][c] = mk<T>(0, 0);
                static_for<0, CPD>([&](auto rcc) {
                    constexpr int RC = decltype(rcc)::value;
                    mbar_wait(full_s + 8 * slot, phase);
                    const unsigned char *sl_ = ring + (size_t)slot * SLOT;
                    const E *Wo = reinterpret_cast<const E *>(sl_ + par * CH) + lane;
                    const E *Wb = inb ? reinterpret_cast<const E *>(sl_ + (1 - par) * CH) + lnb : reinterpret_cast<const E *>(sl_ + (2 + par) * CH) + lane;
#pragma unroll
                    for (int r = 0; r < RPC; ++r) {
                        const int i = RC * RPC + r;
                        E w[DR];
#pragma unroll
                        for (int j = 0; j < DR; ++j) w[j] = Wo[(r * DR + j) * TILE];
#pragma unroll
                        for (int kk = 0; kk < NSC; ++kk) {
                            C chi = mk<T>(0, 0);
#pragma unroll
                            for (int j = 0; j < DR; ++j) mac<T>(chi, w[j], hp[kk][j]);
                            accumulate<T, DR, SPLIT, DF>(chi, kk, SPLIT ? s_rt : kk, i, up, lo, lx);
                        }
                    }
                    if constexpr (RC == 0) {
                        project_regs<T, DR, SPLIT, DB>(spo, nb, inb, lnb, s_rt, hm);
                        if constexpr (MU < 3) {
                            fetch(neighbour<MU + 1>(g, par, t, x, y, zh), MU + 1, DirInfo<MU + 1>::swap);
                        } else {
                            __syncwarp();
                            if (lane == 0) mbar_arrive(spempty_s);          // last read of the staged tiles by this warp
                            if (k + 1 < my_tiles) {
                                if (producer) {
                                    mbar_wait(spempty_s, k & 1);
                                    fence_proxy_async();
                                    issue_sp(gg + (k + 1) * ng);
                                }
                                enter_tile(k + 1);
                                fetch(neighbour<0>(g, par, t, x, y, zh), 0, DirInfo<0>::swap);
                            }
                        }
                    }
#pragma unroll
                    for (int r = 0; r < RPC; ++r) {
                        const int i = RC * RPC + r;
                        E w[DR];
#pragma unroll
                        for (int j = 0; j < DR; ++j) w[j] = Wb[(r * DR + j) * TILE];   // row i of U_mu(x-mu)
#pragma unroll
                        for (int kk = 0; kk < NSC; ++kk)
#pragma unroll
                            for (int j = 0; j < DR; ++j) macc<T>(chib[kk][j], w[j], hm[kk][i]);   // chi_j += conj(U_ij) h_i
                    }
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty_s + 8 * slot);
                    if (q + STAGES < my_chunks) {
                        mbar_wait(empty_s + 8 * slot, phase);
                        if (producer) fence_proxy_async();
                        issue_chunk(slot);
                    }
                    ++q;
                    if (++slot == STAGES) { slot = 0; phase ^= 1; }
                });
#pragma unroll
                for (int kk = 0; kk < NSC; ++kk)
#pragma unroll
                    for (int c = 0; c < DR; ++c) accumulate<T, DR, SPLIT, DB>(chib[kk][c], kk, SPLIT ? s_rt : kk, c, up, lo, lx);
            } else {
            // (a2) both half spinors of this direction pair
            mbar_wait(nbfull_s, nbphase);
            nbphase ^= 1;
            C hp[NSC][DR], hm[NSC][DR];
            {
                const C *spo = sp + (size_t)(1 - par) * NC * TILE;
                project_half<T, DR, SPLIT, DF>(spo, nbuf, inf, hnf & 31, lane, s_rt, hp);
                project_half<T, DR, SPLIT, DB>(spo, reinterpret_cast<const C *>(reinterpret_cast<const unsigned char *>(nbuf) + NBD), inb, lnb, lane, s_rt, hm);
            }
            // stage the next direction pair's neighbours (this warp's buffer has just been consumed by its own lanes)
            if constexpr (MU < 3) {
                stage_nb(IntC<MU + 1>{});
            } else {
                __syncwarp();
                if (lane == 0) mbar_arrive(spempty_s);          // last read of the staged tiles by this warp
                if (k + 1 < my_tiles) {
                    if (producer) {
                        mbar_wait(spempty_s, k & 1);            // ... and by every warp of the group
                        fence_proxy_async();
                        issue_sp(gg + (k + 1) * ng);
                    }
                    enter_tile(k + 1);
                    stage_nb(IntC<0>{});
                }
            }
            // (a3) forward hop: rows of U_mu(x) (own parity).  Backward hop: U_mu(x-mu)^dagger, column-oriented from the rows of
            // the other parity's matrix in the same slot (x-mu inside the tile pair) or from the gathered rows
            C chib[NSC][DR];
#pragma unroll
            for (int kk = 0; kk < NSC; ++kk)
#pragma unroll
                for (int c = 0; c < DR; ++c) chib[kk][c] = mk<T>(0, 0);
            static_for<0, CPD>([&](auto rcc) {
                constexpr int RC = decltype(rcc)::value;
                mbar_wait(full_s + 8 * slot, phase);
                const unsigned char *sl_ = ring + (size_t)slot * SLOT;
                const E *Wo = reinterpret_cast<const E *>(sl_ + par * CH) + lane;
                const E *Wb = inb ? reinterpret_cast<const E *>(sl_ + (1 - par) * CH) + lnb : reinterpret_cast<const E *>(sl_ + (2 + par) * CH) + lane;
#pragma unroll
                for (int r = 0; r < RPC; ++r) {
                    const int i = RC * RPC + r;
                    E w[DR];
#pragma unroll
                    for (int j = 0; j < DR; ++j) w[j] = Wo[(r * DR + j) * TILE];
#pragma unroll
                    for (int kk = 0; kk < NSC; ++kk) {
                        C chi = mk<T>(0, 0);
#pragma unroll
                        for (int j = 0; j < DR; ++j) mac<T>(chi, w[j], hp[kk][j]);
                        accumulate<T, DR, SPLIT, DF>(chi, kk, SPLIT ? s_rt : kk, i, up, lo, lx);
                    }
#pragma unroll
                    for (int j = 0; j < DR; ++j) w[j] = Wb[(r * DR + j) * TILE];   // row i of U_mu(x-mu): U_ij, j = 0..d_R-1
#pragma unroll
                    for (int kk = 0; kk < NSC; ++kk)
#pragma unroll
                        for (int j = 0; j < DR; ++j) macc<T>(chib[kk][j], w[j], hm[kk][i]);   // chi_j += conj(U_ij) h_i
                }
                // release the slot; it is refilled (bulk + gather) once every warp of the group has released it
                __syncwarp();
                if (lane == 0) mbar_arrive(empty_s + 8 * slot);
                if (q + STAGES < my_chunks) {
                    mbar_wait(empty_s + 8 * slot, phase);
                    if (producer) fence_proxy_async();
                    issue_chunk(slot);
                }
                ++q;
                if (++slot == STAGES) { slot = 0; phase ^= 1; }
            });
            // (a4) backward hop complete
#pragma unroll
            for (int kk = 0; kk < NSC; ++kk)
#pragma unroll
                for (int c = 0; c < DR; ++c) accumulate<T, DR, SPLIT, DB>(chib[kk][c], kk, SPLIT ? s_rt : kk, c, up, lo, lx);
            }
        });

        if constexpr (SPLIT) {
            // exchange the cross contributions between the two component warps of this parity: lower s += partner's lx
            C *xb = xbuf + (size_t)par * 2 * DR * TILE;
            const int bid = 1 + GROUPS + grp * 2 + par;
            asm volatile("bar.sync %0, 64;" ::"r"(bid) : "memory");   // partner has finished reading the previous tile's exchange
#pragma unroll
            for (int c = 0; c < DR; ++c) xb[(s_rt * DR + c) * TILE + lane] = lx[0][c];
            asm volatile("bar.sync %0, 64;" ::"r"(bid) : "memory");
#pragma unroll
            for (int c = 0; c < DR; ++c) {
                const C o = xb[((1 - s_rt) * DR + c) * TILE + lane];
                lo[0][c].x += o.x;
                lo[0][c].y += o.y;
            }
        }
        if (c_active) {
            const size_t eoff = ((size_t)c_tile * NC) * TILE + lane;
            // fused reductions: the <= 8 d_R squares of ONE site are summed in four independent plain chains (a serial compensated
            // chain per element costs ~10 % of a tile), the site totals enter the thread's compensated accumulator
            double site[4] = {0.0, 0.0, 0.0, 0.0};
            if (L.red_mode == 2) {
                // CG residual update fused into the second stencil pass: r -= alpha (A p), ||r||^2 accumulated; A p is never stored
                C *rp = (C *)L.red_r + (size_t)par * ((size_t)g.n_tiles * NC * TILE) + eoff;
                const T al = (T)__ddiv_rn(L.red_num[0], L.red_den[0]);
#pragma unroll
                for (int kk = 0; kk < NSC; ++kk) {
                    const int s = SPLIT ? s_rt : kk;
#pragma unroll
                    for (int c = 0; c < DR; ++c) {
                        C ru = rp[(size_t)(s * DR + c) * TILE], rl = rp[(size_t)((2 + s) * DR + c) * TILE];
                        ru.x -= al * (b * up[kk][c].x); ru.y -= al * (b * up[kk][c].y);
                        rl.x -= al * (g5s * b * lo[kk][c].x); rl.y -= al * (g5s * b * lo[kk][c].y);
                        rp[(size_t)(s * DR + c) * TILE] = ru;
                        rp[(size_t)((2 + s) * DR + c) * TILE] = rl;
                        site[0] = fma((double)ru.x, (double)ru.x, site[0]); site[1] = fma((double)ru.y, (double)ru.y, site[1]);
                        site[2] = fma((double)rl.x, (double)rl.x, site[2]); site[3] = fma((double)rl.y, (double)rl.y, site[3]);
                    }
                }
                acc_add(racc, (site[0] + site[1]) + (site[2] + site[3]), L.red_alg);
            } else {
                C *out = (C *)(par ? L.set[1].out : L.set[0].out) + eoff;
#pragma unroll
                for (int kk = 0; kk < NSC; ++kk) {
                    const int s = SPLIT ? s_rt : kk;
#pragma unroll
                    for (int c = 0; c < DR; ++c) {
                        const C vu = mk<T>(b * up[kk][c].x, b * up[kk][c].y), vl = mk<T>(g5s * b * lo[kk][c].x, g5s * b * lo[kk][c].y);
                        st_spinor(out + (size_t)(s * DR + c) * TILE, vu);
                        st_spinor(out + (size_t)((2 + s) * DR + c) * TILE, vl);
                        // ||out||^2 (= <p, A p> for A = B^dagger B when out = B p)
                        site[0] = fma((double)vu.x, (double)vu.x, site[0]); site[1] = fma((double)vu.y, (double)vu.y, site[1]);
                        site[2] = fma((double)vl.x, (double)vl.x, site[2]); site[3] = fma((double)vl.y, (double)vl.y, site[3]);
                    }
                }
                if (L.red_mode == 1) acc_add(racc, (site[0] + site[1]) + (site[2] + site[3]), L.red_alg);
            }
        }
        if (L.pace_every > 0 && wg == 0 && lane == 0) atomicAdd(L.pace, 1u);
    }
    red_finish();
}

// shape per instantiation (B200 sweeps, profiles/r02_summary.md): SPLIT in fp64 from d_R = 4 on (one thread per site would hold
// 2 x 4 d_R accumulators, two half spinors and the column accumulators: > 255 registers).  NBREG (out-of-pair neighbours through
// registers) for complex links: the shared memory the neighbour buffers would take buys more groups per SM (d_R = 3: fp64 4 groups =
// 8 warps, fp32 8 groups = 16 warps; C2 fp64 0.224 -> 0.204 ms, fp32 0.144 -> 0.119 ms; d_R = 6 fp32 4 groups: C4 Dphi 5.97 -> 4.47 ms,
// gather-layout kernel 4.91).  For the real SU(2) adjoint on 48^4 (few in-pair neighbours, L/2 = 24 does not divide the tile) the
// buffered version measured faster and is kept.  Rows per chunk = the largest divisor of d_R whose slot (4 parts) stays <= 19 KB
// (SPLIT: 37 KB; NBREG at d_R <= 3: the whole matrix); as many groups per CTA as leave room for two stages; then up to 4 stages.
template <typename T, int DR, bool REAL> struct FullPick {
    using E = link_elem<T, REAL>;
    static constexpr bool SPLIT = sizeof(T) == 8 && DR >= 4;
    static constexpr bool NBREG = !REAL;
    static constexpr int GW = SPLIT ? 4 : 2;
    static constexpr size_t ch_of(int r) { return (size_t)r * DR * TILE * sizeof(E); }
    static constexpr int pick_rpc() {
        if (NBREG && DR <= 3) return DR;
        int best = 1;
        for (int r = 1; r <= DR; ++r)
            if (DR % r == 0 && 4 * ch_of(r) <= (NBREG && SPLIT ? 37 : 19) * 1024) best = r;
        return best;
    }
    static constexpr int RPC = pick_rpc();
    static constexpr size_t FIXED = 2 * (size_t)4 * DR * TILE * sizeof(cplx<T>) + (NBREG ? 0 : (size_t)GW * 2 * (SPLIT ? 2 : 4) * DR * TILE * sizeof(cplx<T>)) +
                                    (SPLIT ? (size_t)4 * DR * TILE * sizeof(cplx<T>) : 0) + 16 * 8 + 128;
    static constexpr int stages_of(int groups) {
        const size_t per = ((226 * 1024) / groups) & ~(size_t)127;
        if (per < FIXED) return 0;
        int st = (int)((per - FIXED) / (4 * ch_of(RPC)));
        const int cpt = 4 * (DR / RPC);
        if (st > cpt) st = cpt;
        return st > 4 ? 4 : st;
    }
    static constexpr int GMAX = sizeof(T) == 8 ? (SPLIT ? 2 : 4) : (NBREG ? (DR <= 3 ? 8 : 4) : 6);
    static constexpr int pick_groups() {
        for (int gr = GMAX; gr >= 1; --gr)
            if (stages_of(gr) >= 2) return gr;
        return 0;
    }
    static constexpr int GROUPS = pick_groups();
    static constexpr int STAGES = GROUPS > 0 ? stages_of(GROUPS) : 0;
    static_assert(GROUPS >= 1 && STAGES >= 2, "full-lattice kernel does not fit shared memory");
};

// the full-lattice kernel applies when both parities are computed in one launch from the stored gather layout and the
// diagonal term of each parity is the other parity's input (plain Dphi / g5 Dphi / twisted mass; not the in-place accumulation
// of the clover passes, whose self field is the output)
inline bool hop_full_eligible(const HopLaunch &L) {
    return L.nsets == 2 && L.set[0].p_out == 0 && L.set[1].p_out == 1 && L.set[0].self == L.set[1].in && L.set[1].self == L.set[0].in &&
           L.b != 0.0 && L.tile_end == 0 && L.diag_mode == DIAG_NONE && L.bi == 0.0;
}
// would a full-lattice launch of this instantiation run hop_full by default?  (the fused CG asks before it relies on the epilogue hooks)
template <typename T, int DR, bool REAL> constexpr bool hop_full_default() {
    return (DR <= 3 && (sizeof(T) == 8 || !REAL)) || (sizeof(T) == 4 && !REAL && DR != 5 && DR <= 6);
}

template <typename T, int DR, bool REAL, bool SPLIT, int GROUPS, int STAGES, int RPC, bool NBREG = false> int launch_hop_full_cfg(const Geo &g, const HopLaunch &L, cudaStream_t s) {
    using Cfg = FullCfg<T, DR, REAL, SPLIT, GROUPS, STAGES, RPC, NBREG>;
    auto kern = hop_full_kernel<T, DR, REAL, SPLIT, GROUPS, STAGES, RPC, NBREG>;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, Cfg::SMEM, cache, n_sm)) return rc;
    const int grid = ring_grid(n_sm, L.max_ctas, g.n_tiles, GROUPS);
    return launch_pdl(kern, grid, GROUPS * Cfg::GW * 32, Cfg::SMEM, s, g, L);
}

template <typename T, int DR, bool REAL> int launch_hop_full(const Geo &g, const HopLaunch &L, cudaStream_t s) {
#ifdef HIREP_FULL_SWEEP   // development: shapes selected by HIREP_DBG bits 8..11
    if constexpr (DR == 6 && !REAL) {
        const int sel = (L.dbg >> 8) & 15;
        if constexpr (sizeof(T) == 8) {
            switch (sel) {
            case 1: return launch_hop_full_cfg<T, DR, REAL, true, 2, 2, 3, true>(g, L, s);
            case 2: return launch_hop_full_cfg<T, DR, REAL, true, 2, 3, 2, true>(g, L, s);
            case 3: return launch_hop_full_cfg<T, DR, REAL, true, 2, 4, 1, true>(g, L, s);
            }
        } else {
            switch (sel) {
            case 1: return launch_hop_full_cfg<T, DR, REAL, false, 4, 2, 3, true>(g, L, s);
            case 2: return launch_hop_full_cfg<T, DR, REAL, false, 4, 3, 2, true>(g, L, s);
            case 3: return launch_hop_full_cfg<T, DR, REAL, false, 2, 2, 6, true>(g, L, s);
            case 4: return launch_hop_full_cfg<T, DR, REAL, true, 4, 2, 3, true>(g, L, s);
            }
        }
    }
    if constexpr (DR == 3) {
        const int sel = (L.dbg >> 8) & 15;
        if constexpr (sizeof(T) == 8 && !REAL) {
            switch (sel) {
            case 1: return launch_hop_full_cfg<T, DR, REAL, true, 2, 3, 3>(g, L, s);
            case 3: return launch_hop_full_cfg<T, DR, REAL, false, 2, 4, 3>(g, L, s);
            case 8: return launch_hop_full_cfg<T, DR, REAL, false, 3, 3, 3, true>(g, L, s);
            case 9: return launch_hop_full_cfg<T, DR, REAL, false, 4, 2, 3, true>(g, L, s);
            }
        } else if constexpr (sizeof(T) == 8 && REAL) {
            switch (sel) {
            case 9: return launch_hop_full_cfg<T, DR, REAL, false, 4, 2, 3, true>(g, L, s);
            case 11: return launch_hop_full_cfg<T, DR, REAL, false, 4, 4, 3, true>(g, L, s);
            case 12: return launch_hop_full_cfg<T, DR, REAL, false, 5, 3, 3, true>(g, L, s);
            case 13: return launch_hop_full_cfg<T, DR, REAL, false, 6, 2, 3, true>(g, L, s);
            }
        } else if constexpr (!REAL) {
            switch (sel) {
            case 9: return launch_hop_full_cfg<T, DR, REAL, false, 4, 2, 3, true>(g, L, s);
            case 11: return launch_hop_full_cfg<T, DR, REAL, false, 6, 3, 3, true>(g, L, s);
            case 12: return launch_hop_full_cfg<T, DR, REAL, false, 8, 2, 3, true>(g, L, s);
            case 13: return launch_hop_full_cfg<T, DR, REAL, false, 4, 4, 3, true>(g, L, s);
            }
        } else {
            switch (sel) {
            case 11: return launch_hop_full_cfg<T, DR, REAL, false, 6, 4, 3, true>(g, L, s);
            case 12: return launch_hop_full_cfg<T, DR, REAL, false, 8, 3, 3, true>(g, L, s);
            }
        }
    }
#endif
    using P = FullPick<T, DR, REAL>;
    using Cfg = FullCfg<T, DR, REAL, P::SPLIT, P::GROUPS, P::STAGES, P::RPC, P::NBREG>;
    auto kern = hop_full_kernel<T, DR, REAL, P::SPLIT, P::GROUPS, P::STAGES, P::RPC, P::NBREG>;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, Cfg::SMEM, cache, n_sm)) return rc;
    const int grid = ring_grid(n_sm, L.max_ctas, g.n_tiles, P::GROUPS);
    kern<<<grid, P::GROUPS * Cfg::GW * 32, Cfg::SMEM, s>>>(g, L);
    return (int)cudaGetLastError();
}

}  // namespace hirep
