// hop_pair.cuh -- the ring stencil kernel with TWO warps per tile: warp s of a pair owns half-spinor component s.
//
//   out(x) = a*self(x) + b * sum_{d=0..7} P_d W_d(x) in(nbr_d(x)),   x of parity p_out            (Eq 8)
//
// Why: with one thread per site (hop_ring.cuh) a thread holds the 4 d_R accumulators, the 2 d_R half spinor, the
// 4 d_R prefetched neighbour and a link row -- 11 d_R + complex numbers, i.e. > 255 registers in fp64 from
// d_R = 5 on (the paper's "register spilling for N_g > 4", L1548).  The two half-spinor components s = 0, 1 of
// (1 -+ gamma_mu) psi are independent through the link multiply (step a3), so two warps share a tile:
//   warp s loads psi_s and the lower component it is combined with (2 d_R numbers instead of 4 d_R), projects
//   h_s (d_R), multiplies by the SAME link rows (read by both warps from one shared ring) and accumulates
//   out_s (upper) and its contributions to the lower components: lo[s] for mu = 0, 3 and lo[1-s] for mu = 1, 2
//   (e_mu is off-diagonal there, hop_small.cuh).  The cross contributions are exchanged once per tile through
//   shared memory.  Per thread: ~5.5 d_R complex numbers -- no spills at d_R = 6 in fp64.
// Data movement is that of hop_ring.cuh: persistent CTAs, one ring of bulk-copy (TMA) slots per PAIR for the link
// stream with full/empty mbarriers (the producer is lane 0 of warp 0 of the pair and refills a slot once BOTH
// warps have released it), register prefetch of the next neighbour, the tile's own spinor by one bulk copy
// (SELF).
//
// Link mode REBUILD (NF > 0): the ring carries the FUNDAMENTAL gather block (N_g x N_g per direction) and each
// row of R(W) is rebuilt in registers by RepMap (rep_maps.cuh) -- "rebuilding the represented field on the fly",
// L343.  The boundary sign (Eq 61), which the stored represented field carries (L945), is applied to the
// half spinor instead.  The pair rebuilds R(W) once per direction: each warp its half of the rows, into a shared-
// memory buffer both then multiply from (two named barriers per direction); for FUND there is nothing to rebuild.
#pragma once
#include "hop_ring.cuh"
#include "rep_maps.cuh"

namespace hirep {

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void pair_sync(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }

// one lane's column of a [e][32 lanes] shared-memory tile, indexable like a register matrix
template <typename T> struct SmemMat {
    const cplx<T> *p;
    __device__ __forceinline__ cplx<T> operator[](int e) const { return p[e * TILE]; }
};

// boundary factor of hop D from the site (Eq 61): bc[mu] if the hop leaves the lattice
template <int D> __device__ __forceinline__ int hop_sign_dir(const Geo &g, int p, int t, int x, int y, int zh) {
    constexpr int mu = D & 3;
    constexpr bool fwd = D < 4;
    if (mu == 0) return t_edge(g, t, fwd) ? g.bc[0] : 1;
    const int c = (mu == 1) ? x : (mu == 2) ? y : 2 * zh + ((t + x + y + p) & 1);
    return (fwd ? (c == g.L - 1) : (c == 0)) ? g.bc[mu] : 1;
}

template <typename T, int DR, bool REAL, int PAIRS, int STAGES, int RPC, bool SELF, int NF, int REP = 0, int DIAG = DIAG_NONE> struct PairCfg {
    using E = link_elem<T, REAL>;                                   // element type of R
    static constexpr bool REBUILD = NF > 0;
    static_assert(DIAG == DIAG_NONE || !REBUILD, "the site-diagonal epilogue exists for stored links only");
    static_assert(DIAG == DIAG_NONE || DIAG == DIAG_POST || SELF, "DIAG_HB / DIAG_PRE act on the self spinor");
    static_assert(DIAG != DIAG_POST || !SELF, "DIAG_POST has no self term");
    static constexpr bool SHARED = REBUILD && REP != 0;             // the pair rebuilds R(W) once, into shared memory
    static constexpr int CPD = REBUILD ? 1 : DR / RPC;              // chunks per direction
    static constexpr uint32_t CHUNK = REBUILD ? NF * NF * TILE * sizeof(cplx<T>) : RPC * DR * TILE * sizeof(E);
    static_assert(REBUILD || DR % RPC == 0, "rows per chunk must divide d_R");
    static constexpr uint32_t SELF_BYTES = SELF ? 4 * DR * TILE * sizeof(cplx<T>) : 0;
    static constexpr uint32_t X_BYTES = 2 * DR * TILE * sizeof(cplx<T>);   // cross contributions of both warps
    static constexpr uint32_t R_BYTES = SHARED ? DR * DR * TILE * sizeof(E) : 0;   // the rebuilt R(W) of one direction
    static constexpr uint32_t NBAR = 2 * STAGES + 2;                // full[S], empty[S], self full, self empty
    // site-diagonal matrices (kernels.h DIAG_*; hop_ring.cuh): NENT complex entries per site in pieces of DE entries, NDC per tile
    static constexpr int NENT = DIAG == DIAG_NONE ? 0 : DIAG == DIAG_HB ? 4 * DR * DR : 8 * DR * DR;
    static constexpr int DE = (int)(CHUNK / (TILE * sizeof(cplx<T>)));
    static constexpr int NDC = DIAG == DIAG_NONE ? 0 : (NENT + DE - 1) / DE;
    static constexpr size_t PER_PAIR = (size_t)STAGES * CHUNK + SELF_BYTES + X_BYTES + R_BYTES + NBAR * 8;
    static constexpr size_t SMEM = PER_PAIR * PAIRS;
    static_assert(CHUNK % 16 == 0 && PER_PAIR % 16 == 0, "bulk copies need 16-byte alignment");
    static_assert(SMEM <= 227 * 1024, "pair rings do not fit the 227 KB of shared memory of an sm_100 CTA");
};

template <typename T, int DR, bool REAL, int PAIRS, int STAGES, int RPC, bool SELF, int NF, int REP, int DIAG = DIAG_NONE>
__global__ void __launch_bounds__(PAIRS * 64, 1) hop_pair_kernel(const Geo g, const HopLaunch L) {
    using C = cplx<T>;
    using E = link_elem<T, REAL>;
    using Cfg = PairCfg<T, DR, REAL, PAIRS, STAGES, RPC, SELF, NF, REP, DIAG>;
    constexpr bool REBUILD = NF > 0, SHARED = Cfg::SHARED;
    constexpr int NC = 4 * DR, CPD = Cfg::CPD, CPT = 8 * CPD + Cfg::NDC;   // chunks per tile: links, then the diagonal matrices
    constexpr int NENT = Cfg::NENT, DE = Cfg::DE;
    constexpr int RPCE = REBUILD ? DR : RPC;                        // rows of R served by one chunk
    extern __shared__ __align__(128) unsigned char smem_raw[];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int pair = warp >> 1, s = warp & 1;                       // s: the half-spinor component this warp owns
    unsigned char *base = smem_raw + (size_t)pair * Cfg::PER_PAIR;
    const unsigned char *ring = base;
    const C *selfbuf = reinterpret_cast<const C *>(base + (size_t)STAGES * Cfg::CHUNK);
    C *xbuf = reinterpret_cast<C *>(base + (size_t)STAGES * Cfg::CHUNK + Cfg::SELF_BYTES);
    const uint32_t ring_s = smem_u32(ring), self_s = smem_u32(selfbuf);
    E *rbuf = reinterpret_cast<E *>(base + (size_t)STAGES * Cfg::CHUNK + Cfg::SELF_BYTES + Cfg::X_BYTES);
    const uint32_t full_s = smem_u32(base + (size_t)STAGES * Cfg::CHUNK + Cfg::SELF_BYTES + Cfg::X_BYTES + Cfg::R_BYTES);
    const uint32_t empty_s = full_s + 8 * STAGES;
    const uint32_t selffull_s = empty_s + 8 * STAGES, selfempty_s = selffull_s + 8;
    const bool producer = (s == 0) && (lane == 0);
    if (producer) {
        for (int i = 0; i < STAGES; ++i) { mbar_init(full_s + 8 * i, 1); mbar_init(empty_s + 8 * i, 2); }
        mbar_init(selffull_s, 1);
        mbar_init(selfempty_s, 2);
        fence_mbar_init();
    }
    pair_sync(1 + pair);
    pdl_launch_dependents();
    pdl_wait();

    const bool two = L.nsets == 2;
    const int total_tiles = launch_tiles(g, L) * L.nsets;
    const int gp = blockIdx.x * PAIRS + pair, np = gridDim.x * PAIRS;
    Acc racc{0.0, 0.0, 0.0};                            // fused reduction (HopLaunch::red_mode): this thread's compensated partial sum
    __shared__ Acc red_scratch[32];
    if (gp >= total_tiles) { red_finish_cta(L.red_mode, L.red_alg, racc, L.red_partial, red_scratch); return; }
    const int my_tiles = (total_tiles - gp + np - 1) / np;
    const int my_chunks = my_tiles * CPT;
    const uint64_t pol = l2_policy_evict_first();

    auto locate = [&](int k, int &set_, int &tile_) {
        const int gt = gp + k * np;
        set_ = two ? (gt & 1) : 0;
        int sq = two ? (gt >> 1) : gt;
        tile_ = sq + L.tile_begin;
    };

    // producer state: the next chunk to issue is chunk iq_c of the pair's iq_k-th tile
    int iq_k = 0, iq_c = 0;
    const unsigned char *iq_base = nullptr;
    const C *iq_diag = nullptr;
    auto iq_enter = [&]() {
        int s_, t_;
        locate(iq_k, s_, t_);
        iq_base = (const unsigned char *)(s_ ? L.set[1].links : L.set[0].links) + (size_t)t_ * (8 * CPD) * Cfg::CHUNK;
        if constexpr (DIAG != DIAG_NONE) iq_diag = (const C *)(s_ ? L.set[1].diag : L.set[0].diag) + (size_t)t_ * NENT * TILE;
    };
    auto issue = [&](int slot) {
        if (DIAG != DIAG_NONE && iq_c >= 8 * CPD) {
            // piece iq_c - 8 CPD of the tile's diagonal matrices: DE entries (the last piece: what is left)
            const int e0 = (iq_c - 8 * CPD) * DE;
            const uint32_t bytes = (uint32_t)((NENT - e0 < DE ? NENT - e0 : DE) * TILE * sizeof(C));
            mbar_expect_tx(full_s + 8 * slot, bytes);
            bulk_g2s(ring_s + slot * Cfg::CHUNK, iq_diag + (size_t)e0 * TILE, bytes, full_s + 8 * slot, pol);
        } else {
        mbar_expect_tx(full_s + 8 * slot, Cfg::CHUNK);
        // chunk iq_c of the tile = step iq_c / CPD of the walk -> direction dir_of<true>(step) of the gather block
        const int step = iq_c / CPD, chunk = dir_of<true>(step) * CPD + (iq_c - step * CPD);
        bulk_g2s(ring_s + slot * Cfg::CHUNK, iq_base + (size_t)chunk * Cfg::CHUNK, Cfg::CHUNK, full_s + 8 * slot, pol);
        }
        if (++iq_c == CPT) {
            iq_c = 0;
            if (++iq_k < my_tiles) iq_enter();
        }
    };
    if (producer) {
        iq_enter();
        const int n0 = my_chunks < STAGES ? my_chunks : STAGES;
        for (int i = 0; i < n0; ++i) issue(i);
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
    // neighbour components this warp needs for direction D: upper s and lower q_D(s)
    C nbu[DR], nbl[DR];
    auto fetch = [&](int hn, bool swap) {
        const int ql = swap ? 1 - s : s;
        const C *src = in + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
#pragma unroll
        for (int c = 0; c < DR; ++c) {
            nbu[c] = ld_spinor<T>(src + (size_t)(s * DR + c) * TILE);
            nbl[c] = ld_spinor<T>(src + (size_t)((2 + ql) * DR + c) * TILE);
        }
    };

    enter_tile(0);
    fetch(neighbour<dir_of<true>(0)>(g, p_out, t, x, y, zh), DirInfo<dir_of<true>(0)>::swap);
    int q = 0, slot = 0;
    uint32_t phase = 0;
    const T a = (T)L.a, b = (T)L.b, bi = (T)L.bi;
    const T am = (T)L.am;
    const T g5s = L.g5 ? T(-1) : T(1);

    for (int k = 0; k < my_tiles; ++k) {
        const int c_set = set, c_tile = tile;
        const bool c_active = active;
        if constexpr (SELF) {
            if (producer) {
                if (k > 0) { mbar_wait(selfempty_s, (k - 1) & 1); fence_proxy_async(); }   // both warps have read the previous tile's block
                const C *sp = (const C *)(c_set ? L.set[1].self : L.set[0].self) + ((size_t)c_tile * NC) * TILE;
                mbar_expect_tx(selffull_s, Cfg::SELF_BYTES);
                bulk_g2s_plain(self_s, sp, Cfg::SELF_BYTES, selffull_s);
            }
        }
        C up[DR], ls[DR], lx[DR];   // out_s ; lower component s (mu = 0,3) ; lower component 1-s (mu = 1,2)
#pragma unroll
        for (int c = 0; c < DR; ++c) up[c] = ls[c] = lx[c] = mk<T>(0, 0);

        static_for<0, 8>([&](auto dc) {
            constexpr int I = decltype(dc)::value, D = dir_of<true>(I);
            using DI = DirInfo<D>;
            // (a2) spin projection: h_s = psi_s + sg e_mu psi_low
            const T cs = (T)(DI::sg * ((DI::mu < 2) ? -1 : (s ? 1 : -1)));
            T sgn = T(1);
            if constexpr (REBUILD) sgn = (T)hop_sign_dir<D>(g, p_out, t, x, y, zh);
            const T cv = cs * sgn;
            C hs[DR];
#pragma unroll
            for (int c = 0; c < DR; ++c) {
                const C u = nbu[c], v = nbl[c];
                if (DI::imag) hs[c] = mk<T>(fma(-cv, v.y, sgn * u.x), fma(cv, v.x, sgn * u.y));   // sgn (u + i cs v)
                else hs[c] = mk<T>(fma(cv, v.x, sgn * u.x), fma(cv, v.y, sgn * u.y));             // sgn (u + cs v)
            }
            if constexpr (I < 7) {
                constexpr int DN = dir_of<true>(I + 1);
                fetch(neighbour<DN>(g, p_out, t, x, y, zh), DirInfo<DN>::swap);
            } else {
                if (k + 1 < my_tiles) {
                    enter_tile(k + 1);
                    fetch(neighbour<dir_of<true>(0)>(g, p_out, t, x, y, zh), DirInfo<dir_of<true>(0)>::swap);
                }
            }
            if constexpr (SHARED) {
                // (a1') REBUILD: the two warps rebuild R(W) ONCE -- each its half of the rows -- from the fundamental
                // chunk into the pair's R buffer, then both multiply all rows from there
                mbar_wait(full_s + 8 * slot, phase);
                {
                    const SmemMat<T> Wm{reinterpret_cast<const C *>(ring + (size_t)slot * Cfg::CHUNK) + lane};
                    constexpr int H = (DR + 1) / 2;
                    static_for<0, DR>([&](auto ic) {
                        constexpr int i = decltype(ic)::value;
                        if ((i < H) == (s == 0)) {
                            E w[DR];
                            RepMap<T, NF, REP>::template row<i>(Wm, w);
#pragma unroll
                            for (int j = 0; j < DR; ++j) rbuf[(i * DR + j) * TILE + lane] = w[j];
                        }
                    });
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(empty_s + 8 * slot);
                if (producer && q + STAGES < my_chunks) {
                    mbar_wait(empty_s + 8 * slot, phase);
                    fence_proxy_async();
                    issue(slot);
                }
                ++q;
                if (++slot == STAGES) { slot = 0; phase ^= 1; }
                pair_sync(1 + pair);   // R(W) of this direction complete
                static_for<0, DR>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    E w[DR];
#pragma unroll
                    for (int j = 0; j < DR; ++j) w[j] = rbuf[(i * DR + j) * TILE + lane];
                    C chi = mk<T>(0, 0);
#pragma unroll
                    for (int j = 0; j < DR; ++j) mac<T>(chi, w[j], hs[j]);
                    up[i].x += chi.x;
                    up[i].y += chi.y;
                    C add;   // sg conj(k_mu(s)) chi
                    if (DI::imag) add = mk<T>(cs * chi.y, -cs * chi.x);
                    else add = mk<T>(cs * chi.x, cs * chi.y);
                    if (DI::swap) { lx[i].x += add.x; lx[i].y += add.y; }
                    else { ls[i].x += add.x; ls[i].y += add.y; }
                });
                pair_sync(1 + pair);   // both warps are done with R before the next direction overwrites it
            } else {
            // (a3) link rows from the pair's ring, (a4) reconstruct + accumulate
            static_for<0, DR>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                if constexpr (i % RPCE == 0) mbar_wait(full_s + 8 * slot, phase);
                E w[DR];
                if constexpr (REBUILD) {
                    const SmemMat<T> Wm{reinterpret_cast<const C *>(ring + (size_t)slot * Cfg::CHUNK) + lane};
                    RepMap<T, NF, REP>::template row<i>(Wm, w);
                } else {
                    const E *W = reinterpret_cast<const E *>(ring + (size_t)slot * Cfg::CHUNK) + lane;
#pragma unroll
                    for (int j = 0; j < DR; ++j) w[j] = W[((i % RPCE) * DR + j) * TILE];
                }
                C chi = mk<T>(0, 0);
#pragma unroll
                for (int j = 0; j < DR; ++j) mac<T>(chi, w[j], hs[j]);
                up[i].x += chi.x;
                up[i].y += chi.y;
                C add;   // sg conj(k_mu(s)) chi
                if (DI::imag) add = mk<T>(cs * chi.y, -cs * chi.x);
                else add = mk<T>(cs * chi.x, cs * chi.y);
                if (DI::swap) { lx[i].x += add.x; lx[i].y += add.y; }
                else { ls[i].x += add.x; ls[i].y += add.y; }
                if constexpr (i % RPCE == RPCE - 1) {
                    // release the slot; the producer refills it once both warps have released it
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty_s + 8 * slot);
                    if (producer && q + STAGES < my_chunks) {
                        mbar_wait(empty_s + 8 * slot, phase);
                        fence_proxy_async();
                        issue(slot);
                    }
                    ++q;
                    if (++slot == STAGES) { slot = 0; phase ^= 1; }
                }
            });
            }
        });

        // exchange the cross contributions: lower component s += partner's lx
        pair_sync(1 + pair);   // partner has finished reading the previous tile's exchange
#pragma unroll
        for (int c = 0; c < DR; ++c) xbuf[(s * DR + c) * TILE + lane] = lx[c];
        pair_sync(1 + pair);
#pragma unroll
        for (int c = 0; c < DR; ++c) {
            const C o = xbuf[((1 - s) * DR + c) * TILE + lane];
            ls[c].x += o.x;
            ls[c].y += o.y;
        }
        if constexpr (SELF) mbar_wait(selffull_s, k & 1);
        if constexpr (DIAG != DIAG_NONE) {
            // Site-diagonal term (kernels.h DIAG_*; the ring kernel's epilogue split over the pair), chirality c = spins 2c, 2c + 1.
            // Clover H, B: warp s computes the rows of spin 2c + s -- H multiplies the warp's own spin, B the partner's, so both
            // warps use every entry that streams by.  Full blocks: warp s computes the rows I = 2r + s of the 2 d_R x 2 d_R block
            // (rows alternate between the warps, so both work on every piece of the stream); the scaled hop sum of the chirality
            // is exchanged through the cross buffer -- as the vector the block multiplies (DIAG_POST) or as the row's start value
            // (DIAG_PRE) -- and the warp stores the rows it computed (FULLROWS below).
            const T csw = (T)L.diag_csw;
            const T sgh = s ? T(-1) : T(1);
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                C o[DR];
                C v[DIAG == DIAG_HB ? DR : 2 * DR], vo[DIAG == DIAG_HB ? DR : 1];   // HB: own spin / partner's spin; full blocks: v = both
#pragma unroll
                for (int j = 0; j < DR; ++j) {
                    const C h = c == 0 ? up[j] : ls[j];
                    o[j] = mk<T>(b * h.x, b * h.y);
                }
                if constexpr (DIAG == DIAG_HB) {
#pragma unroll
                    for (int j = 0; j < DR; ++j) {
                        const C sv = selfbuf[((2 * c + s) * DR + j) * TILE + lane], so = selfbuf[((2 * c + 1 - s) * DR + j) * TILE + lane];
                        o[j].x = fma(a, sv.x, o[j].x); o[j].y = fma(a, sv.y, o[j].y);
                        v[j] = mk<T>(csw * sgh * sv.x, csw * sgh * sv.y);   // +-H on spin 0 / 1 of the chirality block
                        vo[j] = mk<T>(csw * so.x, csw * so.y);
                    }
                } else {
                    pair_sync(1 + pair);   // the partner has read what the buffer held before
#pragma unroll
                    for (int j = 0; j < DR; ++j) xbuf[(s * DR + j) * TILE + lane] = o[j];
                    pair_sync(1 + pair);
#pragma unroll
                    for (int J = 0; J < 2 * DR; ++J)
                        v[J] = DIAG == DIAG_POST ? xbuf[J * TILE + lane] : selfbuf[(2 * c * DR + J) * TILE + lane];
#pragma unroll
                    for (int r = 0; r < DR; ++r) o[r] = DIAG == DIAG_POST ? mk<T>(0, 0) : xbuf[(2 * r + s) * TILE + lane];
                }
#pragma unroll
                for (int e = 0; e < NENT / 2; ++e) {
                    const int ge = c * (NENT / 2) + e;
                    if (ge % DE == 0) mbar_wait(full_s + 8 * slot, phase);
                    const C m = reinterpret_cast<const C *>(ring + (size_t)slot * Cfg::CHUNK)[(ge % DE) * TILE + lane];
                    if constexpr (DIAG == DIAG_HB) {
                        const int i = (e % (DR * DR)) / DR, j = e % DR;
                        if (e < DR * DR) mac<T>(o[i], m, v[j]);
                        else if (s == 0) mac<T>(o[i], m, vo[j]);              // B psi_1 -> spin 0, row i
                        else mac<T>(o[j], mk<T>(m.x, -m.y), vo[i]);            // B^+ psi_0 -> spin 1, row j
                    } else {
                        if (((e / (2 * DR)) & 1) == s) mac<T>(o[(e / (2 * DR)) >> 1], m, v[e % (2 * DR)]);
                    }
                    if (ge % DE == DE - 1 || ge == NENT - 1) {
                        __syncwarp();
                        if (lane == 0) mbar_arrive(empty_s + 8 * slot);
                        if (producer && q + STAGES < my_chunks) {
                            mbar_wait(empty_s + 8 * slot, phase);
                            fence_proxy_async();
                            issue(slot);
                        }
                        ++q;
                        if (++slot == STAGES) { slot = 0; phase ^= 1; }
                    }
                }
#pragma unroll
                for (int j = 0; j < DR; ++j) {
                    if (c == 0) up[j] = o[j];
                    else ls[j] = o[j];
                }
            }
        }
        if (c_active) {
            const size_t eoff = ((size_t)c_tile * NC) * TILE + lane;
            C *out = (C *)(c_set ? L.set[1].out : L.set[0].out) + eoff;
            // fused CG reductions (reduce.cuh): mode 2 updates the residual in place of storing the result
            C *rp = L.red_mode == 2 ? (C *)L.red_r + (size_t)c_set * ((size_t)g.n_tiles * NC * TILE) + eoff : out;
            const T al = L.red_mode == 2 ? (T)__ddiv_rn(L.red_num[0], L.red_den[0]) : T(0);
            double site[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
            for (int c = 0; c < DR; ++c) {
                C vu, vl;
                if constexpr (DIAG != DIAG_NONE) { vu = up[c]; vl = ls[c]; }
                else if (bi != T(0)) {   // (b + i bi gamma_5) hop
                    vu = mk<T>(fma(-bi, up[c].y, b * up[c].x), fma(bi, up[c].x, b * up[c].y));
                    vl = mk<T>(fma(bi, ls[c].y, b * ls[c].x), fma(-bi, ls[c].x, b * ls[c].y));
                } else { vu = mk<T>(b * up[c].x, b * up[c].y); vl = mk<T>(b * ls[c].x, b * ls[c].y); }
                if constexpr (SELF && DIAG == DIAG_NONE) {
                    const C su = selfbuf[(s * DR + c) * TILE + lane];
                    const C sl = selfbuf[((2 + s) * DR + c) * TILE + lane];
                    vu.x = fma(a, su.x, vu.x); vu.y = fma(a, su.y, vu.y);
                    vl.x = fma(a, sl.x, vl.x); vl.y = fma(a, sl.y, vl.y);
                    if (am != T(0)) {   // twisted mass: + i mu gamma_5 self (Eq 51)
                        vu.x = fma(-am, su.y, vu.x); vu.y = fma(am, su.x, vu.y);
                        vl.x = fma(am, sl.y, vl.x); vl.y = fma(-am, sl.x, vl.y);
                    }
                }
                // component of the upper value: spin s, colour c -- or, after a full-block epilogue, row 2c + s of chirality 0
                constexpr bool FULLROWS = DIAG == DIAG_PRE || DIAG == DIAG_POST;
                const int cu = FULLROWS ? 2 * c + s : s * DR + c, cl = 2 * DR + cu;
                red_store(L.red_mode, out + (size_t)cu * TILE, rp + (size_t)cu * TILE, al, vu, site[0], site[1]);
                red_store(L.red_mode, out + (size_t)cl * TILE, rp + (size_t)cl * TILE, al, mk<T>(g5s * vl.x, g5s * vl.y), site[2], site[3]);
            }
            if (L.red_mode != 0) acc_add(racc, (site[0] + site[1]) + (site[2] + site[3]), L.red_alg);
        }
        if constexpr (SELF) {
            __syncwarp();
            if (lane == 0) mbar_arrive(selfempty_s);
        }
    }
    red_finish_cta(L.red_mode, L.red_alg, racc, L.red_partial, red_scratch);
}

template <typename T, int DR, bool REAL, int PAIRS, int STAGES, int RPC, bool SELF, int NF, int REP, int DIAG = DIAG_NONE>
int launch_hop_pair_cfg(const Geo &g, const HopLaunch &L0, cudaStream_t s) {
    using Cfg = PairCfg<T, DR, REAL, PAIRS, STAGES, RPC, SELF, NF, REP, DIAG>;
    auto kern = hop_pair_kernel<T, DR, REAL, PAIRS, STAGES, RPC, SELF, NF, REP, DIAG>;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, Cfg::SMEM, cache, n_sm)) return rc;
    const HopLaunch &L = L0;
    const int grid = ring_grid(n_sm, L.max_ctas, launch_tiles(g, L) * L.nsets, PAIRS);
    return launch_pdl(kern, grid, PAIRS * 64, Cfg::SMEM, s, g, L);
}

// default shape of the pair kernel: PAIRS pairs per CTA; the chunk is the largest whole number of link rows that
// divides d_R, stays <= 13 KB and leaves room for two stages; then as many stages (<= 4) as fit
template <typename T, int DR, bool REAL, bool SELF, int NF, int REP = 0> struct PairPick {
    using E = link_elem<T, REAL>;
    // fp64 pure-hop passes run 3 pairs per CTA: fewer tiles in flight shorten the tile time (bytes per tile / the SM's
    // bandwidth share), which keeps the cross-tile spinor re-use inside what L2 retains (C4 fp64 Dphi_eo: 4 pairs 4.89 ms /
    // 30.4 GB read, 3 pairs 4.52 ms / 28.1 GB, 2 pairs 4.91 ms at 6.4 TB/s); passes with a diagonal term keep 4
    // fp32: 8 pairs (4 warps per scheduler, <= 128 registers); REBUILD 6 pairs (168 registers: the rebuild no longer
    // spills; C4 fp32 rebuilt Dphi_hat 5.05 -> 4.41 ms, below the 4.62 ms of stored links)
    static constexpr int PAIRS = sizeof(T) == 4 ? (NF > 0 ? 6 : 8) : ((SELF || NF > 0) ? 4 : 3);   // warps per SM sub-partition: 4 (fp32, <= 128 registers) or 2 (fp64, <= 255)
    static constexpr size_t FIXED = (SELF ? 4 : 0) * DR * TILE * sizeof(cplx<T>) + 2 * DR * TILE * sizeof(cplx<T>) +
                                    ((NF > 0 && REP != 0) ? DR * DR * TILE * sizeof(E) : 0) + 10 * 8;
    static constexpr size_t chunk_of(int r) { return NF > 0 ? (size_t)NF * NF * TILE * sizeof(cplx<T>) : (size_t)r * DR * TILE * sizeof(E); }
    static constexpr int stages_of(int r) {
        const size_t per_pair = ((226 * 1024) / PAIRS) & ~(size_t)15;
        if (per_pair < FIXED) return 0;
        const int st = (int)((per_pair - FIXED) / chunk_of(r));
        return st > 4 ? 4 : st;
    }
    static constexpr int pick_rpc() {
        if (NF > 0) return DR;
        int best = 1;
        for (int r = 1; r <= DR; ++r)
            if (DR % r == 0 && chunk_of(r) <= 13 * 1024 && stages_of(r) >= 2) best = r;
        return best;
    }
    static constexpr int RPC = pick_rpc();
    static constexpr int STAGES = stages_of(RPC);
    static_assert(STAGES >= 2, "pair ring needs at least two stages");
};

// stored links with the site-diagonal matrices in the epilogue (kernels.h DIAG_*)
template <typename T, int DR, bool REAL> int launch_hop_pair_diag(const Geo &g, const HopLaunch &L, cudaStream_t s) {
    if (L.am != 0.0 || !L.set[0].diag || (L.nsets == 2 && !L.set[1].diag)) return KERR_UNSUPPORTED;
    if (L.diag_mode == DIAG_POST) {
        // the shape of the passes with a self term (4 pairs in fp64): the block epilogue makes a tile long enough that the
        // fourth pair pays, unlike in the pure hop pass
        using P = PairPick<T, DR, REAL, true, 0, 0>;
        return launch_hop_pair_cfg<T, DR, REAL, P::PAIRS, P::STAGES, P::RPC, false, 0, 0, DIAG_POST>(g, L, s);
    }
    if (!L.set[0].self) return KERR_UNSUPPORTED;
    using P = PairPick<T, DR, REAL, true, 0, 0>;
    if (L.diag_mode == DIAG_HB) return launch_hop_pair_cfg<T, DR, REAL, P::PAIRS, P::STAGES, P::RPC, true, 0, 0, DIAG_HB>(g, L, s);
    if (L.diag_mode == DIAG_PRE) return launch_hop_pair_cfg<T, DR, REAL, P::PAIRS, P::STAGES, P::RPC, true, 0, 0, DIAG_PRE>(g, L, s);
    return KERR_UNSUPPORTED;
}

template <typename T, int DR, bool REAL, int NF = 0, int REP = 0> int launch_hop_pair(const Geo &g, const HopLaunch &L, cudaStream_t s) {
    const bool self = (L.a != 0.0) && L.set[0].self != nullptr;
    if (self) {
        using P = PairPick<T, DR, REAL, true, NF, REP>;
        return launch_hop_pair_cfg<T, DR, REAL, P::PAIRS, P::STAGES, P::RPC, true, NF, REP>(g, L, s);
    }
    using P = PairPick<T, DR, REAL, false, NF, REP>;
    return launch_hop_pair_cfg<T, DR, REAL, P::PAIRS, P::STAGES, P::RPC, false, NF, REP>(g, L, s);
}

}  // namespace hirep
