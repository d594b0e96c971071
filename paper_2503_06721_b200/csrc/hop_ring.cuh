// hop_ring.cuh -- the Wilson hopping stencil for small d_R with the link stream staged through shared memory
// by the bulk-copy engine (TMA, cp.async.bulk) -- the sm_100a kernel of this library.
//
//   out(x) = a*self(x) + b * sum_{d=0..7} P_d W_d(x) in(nbr_d(x)),   x of parity p_out            (Eq 8)
//
// Same arithmetic as hop_small.cuh (spin projection to half spinors, d_R x d_R link matvec, reconstruction; steps
// a2-a4 of SURVEY.md 8(a)); what differs is how the bytes move:
//   * The kernel is persistent: one CTA per SM, WARPS warps per CTA, one warp = one tile of 32 sites at a time,
//     tiles dealt round-robin over all warps of the grid (neighbouring tiles run at the same time on different SMs,
//     which is what makes the 8-fold spinor reuse hit in L2).
//   * The 8 link matrices of a tile are ONE contiguous block in the gather layout (common.cuh).  Each warp owns a
//     ring of STAGES shared-memory slots of RPC link-matrix rows each (RPC x d_R x 32 lanes) and keeps it full with
//     cp.async.bulk (global -> shared, completion on an mbarrier, L2 evict_first: links are streamed once).  The
//     bytes in flight per SM are WARPS x (STAGES-1) x slot and cost no registers, so the link stream (75 % of the
//     traffic at SU(3)) no longer depends on occupancy.  The ring runs across tile boundaries.
//   * Neighbour spinors are gathered with plain 128-bit read-only loads; the loads of direction d+1 are issued
//     right after direction d has been projected (the projection frees the registers), so they fly during the
//     link matvec of direction d.  At direction 7 the first neighbour of the warp's next tile is fetched.
//   * When the pass has a diagonal term (a != 0: Dphi, the second pass of Dphi_hat, g5Dphi_sq; template SELF) the
//     tile's own spinor -- one contiguous 4 d_R x 32 block -- is fetched by ONE bulk copy at the start of the tile
//     into a per-warp buffer and read in the epilogue, instead of being loaded (latency exposed) at the end.
// No CTA-wide barrier anywhere: every warp is its own producer/consumer pipeline (lane 0 issues the bulk copies).
#pragma once
#include "hop_small.cuh"
#include "reduce.cuh"

namespace hirep {

// ---- PTX wrappers (mbarrier + bulk async copy, PTX ISA 8.x, sm_90+) ---------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol)
        : "memory");
}

__device__ __forceinline__ void bulk_g2s_plain(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar)
                 : "memory");
}

// cross-proxy hand-off: shared-memory reads through the generic proxy (the consumers' ld.shared, ordered before this point by
// __syncwarp / an mbarrier) must be ordered before the async-proxy write of the bulk copy that refills the same bytes
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Programmatic dependent launch (PTX griddepcontrol): every stencil launch carries the programmatic-stream-serialization attribute,
// so its CTAs may be scheduled while the previous kernel of the stream drains; pdl_wait() -- before the first global read -- blocks
// until that kernel has completed and flushed, pdl_launch_dependents() lets the NEXT launch start its prologue early.  What is
// overlapped is the launch latency, the barrier set-up and the pipeline fill of back-to-back passes (Dphi_hat, g5Dphi_sq, CG).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename K> inline int launch_pdl(K kern, int grid, int block, size_t smem, cudaStream_t s, const Geo &g, const HopLaunch &L) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return (int)cudaLaunchKernelEx(&cfg, kern, g, L);
}

// ring geometry for one instantiation; CHUNK = RPC rows of the link block of one direction of one tile
template <typename T, int DR, bool REAL, int WARPS, int STAGES, int RPC, bool SELF, int DIAG = DIAG_NONE> struct RingCfg {
    using E = link_elem<T, REAL>;
    static constexpr int NE = DR * DR;
    static constexpr int CPD = DR / RPC;                            // chunks per direction
    static constexpr uint32_t CHUNK = RPC * DR * TILE * sizeof(E);  // RPC rows of one link matrix, 32 lanes
    static_assert(DR % RPC == 0, "rows per chunk must divide d_R");
    // site-diagonal matrices (kernels.h DIAG_*): NENT complex entries per site, [entry][lane], streamed through the ring slots
    // after the eight directions of the tile in pieces of DE entries (the whole entries that fit a slot), NDC pieces per tile
    static constexpr int NENT = DIAG == DIAG_NONE ? 0 : DIAG == DIAG_HB ? 4 * NE : 8 * NE;
    static constexpr int DE = (int)(CHUNK / (TILE * sizeof(cplx<T>)));
    static constexpr int NDC = DIAG == DIAG_NONE ? 0 : (NENT + DE - 1) / DE;
    static_assert(DIAG == DIAG_NONE || DE >= 1, "a ring slot must hold at least one entry of the diagonal matrices");
    static_assert(DIAG == DIAG_NONE || DIAG == DIAG_POST || SELF, "DIAG_HB / DIAG_PRE act on the self spinor");
    static_assert(DIAG != DIAG_POST || !SELF, "DIAG_POST has no self term");
    static constexpr uint32_t SELF_BYTES = SELF ? 4 * DR * TILE * sizeof(cplx<T>) : 0;   // one tile of the spinor
    static constexpr size_t RING_BYTES = (size_t)WARPS * STAGES * CHUNK;
    static constexpr size_t BARS_OFF = RING_BYTES + (size_t)WARPS * SELF_BYTES;
    static constexpr size_t SMEM = BARS_OFF + (size_t)WARPS * (STAGES + 1) * sizeof(uint64_t);
    static_assert(CHUNK % 16 == 0, "bulk copies move multiples of 16 bytes");
    static_assert(SMEM <= 227 * 1024, "ring does not fit the 227 KB of shared memory of an sm_100 CTA");
};

// Library default ring shape per instantiation (B200 sweeps: profiles/r01b_summary.md):
//   fp64: 8 warps (the thread-per-site kernel needs ~200 registers); fp32: 16 warps for d_R <= 3, else 12;
//   chunk = the largest whole number of link rows that divides d_R, stays <= 13 KB and leaves room for two stages
//   (large chunks beat deep rings: fewer barrier round trips per byte); then as many stages (<= 4) as fit.
template <typename T, int DR, bool REAL, bool SELF> struct RingPick {
    using E = link_elem<T, REAL>;
    static constexpr int WARPS = sizeof(T) == 4 ? (DR <= 3 ? 16 : 12) : 8;
    static constexpr size_t SELF_BYTES = SELF ? 4 * DR * TILE * sizeof(cplx<T>) : 0;
    static constexpr size_t chunk_of(int r) { return (size_t)r * DR * TILE * sizeof(E); }
    static constexpr int stages_of(int r) {
        const size_t per_warp = (226 * 1024) / WARPS;
        if (per_warp < SELF_BYTES + 8) return 0;
        const int st = (int)((per_warp - SELF_BYTES - 8) / (chunk_of(r) + 8));
        return st > 4 ? 4 : st;
    }
    static constexpr int pick_rpc() {
        int best = 1;
        for (int r = 1; r <= DR; ++r)
            if (DR % r == 0 && chunk_of(r) <= 13 * 1024 && stages_of(r) >= 2) best = r;
        return best;
    }
    static constexpr int RPC = pick_rpc();
    static constexpr int STAGES = stages_of(RPC);
    static_assert(STAGES >= 2, "ring needs at least two stages");
};

template <typename T, int DR, bool REAL, int WARPS, int STAGES, int RPC, bool SELF, int DIAG = DIAG_NONE>
__global__ void __launch_bounds__(WARPS * 32, 1) hop_ring_kernel(const Geo g, const HopLaunch L) {
    using C = cplx<T>;
    using E = link_elem<T, REAL>;
    using Cfg = RingCfg<T, DR, REAL, WARPS, STAGES, RPC, SELF, DIAG>;
    constexpr int NC = 4 * DR, CPD = Cfg::CPD, CPT = 8 * CPD + Cfg::NDC;   // chunks per direction / per tile (links, then diagonal matrices)
    constexpr int NENT = Cfg::NENT, DE = Cfg::DE;
    constexpr int CE = RPC * DR * TILE;                         // link elements per chunk
    constexpr bool IL = !(sizeof(T) == 4 && DR >= 5);           // hop order (common.cuh): the 168-register fp32 kernels
                                                                // at d_R = 5, 6 lose 13 % with the interleaved walk
    extern __shared__ __align__(128) unsigned char smem_raw[];

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const E *ring = reinterpret_cast<const E *>(smem_raw + (size_t)warp * STAGES * Cfg::CHUNK);
    const C *selfbuf = reinterpret_cast<const C *>(smem_raw + Cfg::RING_BYTES + (size_t)warp * Cfg::SELF_BYTES);
    const uint32_t ring_s = smem_u32(ring), self_s = smem_u32(selfbuf);
    const uint32_t bars_s = smem_u32(smem_raw + Cfg::BARS_OFF) + warp * (STAGES + 1) * 8;
    const uint32_t selfbar_s = bars_s + 8 * STAGES;
    if (lane == 0) {
        for (int s = 0; s <= STAGES; ++s) mbar_init(bars_s + 8 * s, 1);
        fence_mbar_init();
    }
    __syncwarp();
    pdl_launch_dependents();
    pdl_wait();   // everything below reads global memory the previous kernel of the stream may have written

    // full-lattice launches (nsets = 2) interleave the two parities tile by tile: the `self` spinor of an even tile is
    // the neighbour data of the odd tiles processed at the same time, so it is served by L2
    const bool two = L.nsets == 2;
    const int total_tiles = launch_tiles(g, L) * L.nsets;
    const int gw = blockIdx.x * WARPS + warp, nw = gridDim.x * WARPS;
    Acc racc{0.0, 0.0, 0.0};                            // fused reduction (HopLaunch::red_mode): this thread's compensated partial sum
    __shared__ Acc red_scratch[32];
    if (gw >= total_tiles) { red_finish_cta(L.red_mode, L.red_alg, racc, L.red_partial, red_scratch); return; }
    const int my_tiles = (total_tiles - gw + nw - 1) / nw;
    const int my_chunks = my_tiles * CPT;
    const uint64_t pol = l2_policy_evict_first();

    // k-th tile of this warp -> (set, tile): tiles are dealt round-robin over all warps of the grid
    auto locate = [&](int k, int &set_, int &tile_) {
        const int gt = gw + k * nw;
        set_ = two ? (gt & 1) : 0;
        int sq = two ? (gt >> 1) : gt;
        tile_ = sq + L.tile_begin;
    };

    // chunk qi of this warp = chunk qi % CPT of its (qi / CPT)-th tile; a tile's chunks are consecutive in memory
    auto issue = [&](int qi, int slot) {
        const int kq = qi / CPT;
        int set_, tile_;
        locate(kq, set_, tile_);
        // chunk c of the tile = step c / CPD of the walk -> direction dir_of<IL>(step) of the gather block
        const int c = qi - kq * CPT;
        if constexpr (DIAG != DIAG_NONE) {
            if (c >= 8 * CPD) {   // piece c - 8 CPD of the tile's diagonal matrices: DE entries (the last piece: what is left)
                const int e0 = (c - 8 * CPD) * DE;
                const uint32_t bytes = (uint32_t)((NENT - e0 < DE ? NENT - e0 : DE) * TILE * sizeof(C));
                const C *src = (const C *)(set_ ? L.set[1].diag : L.set[0].diag) + ((size_t)tile_ * NENT + e0) * TILE;
                mbar_expect_tx(bars_s + 8 * slot, bytes);
                bulk_g2s(ring_s + slot * Cfg::CHUNK, src, bytes, bars_s + 8 * slot, pol);
                return;
            }
        }
        const int step = c / CPD, chunk = dir_of<IL>(step) * CPD + (c - step * CPD);
        const E *src = (const E *)(set_ ? L.set[1].links : L.set[0].links) + ((size_t)tile_ * (8 * CPD) + chunk) * CE;
        mbar_expect_tx(bars_s + 8 * slot, Cfg::CHUNK);
        bulk_g2s(ring_s + slot * Cfg::CHUNK, src, Cfg::CHUNK, bars_s + 8 * slot, pol);
    };

    // per-tile state
    int set, tile, t, x, y, zh, p_out;
    bool active;
    const C *in;
    auto enter_tile = [&]() {   // (set, tile) -> coordinates and pointers
        int h = tile * TILE + lane;
        active = h < g.Nh;
        if (!active) h = g.Nh - 1;
        decode_site(g, h, t, x, y, zh);
        p_out = set ? L.set[1].p_out : L.set[0].p_out;   // selects, not L.set[set]: dynamic indexing would copy the
        in = (const C *)(set ? L.set[1].in : L.set[0].in);   // kernel parameters to local memory
    };
    C nb[NC];
    auto fetch = [&](int hn) {
        const C *src = in + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
#pragma unroll
        for (int c = 0; c < NC; ++c) nb[c] = ld_spinor<T>(src + (size_t)c * TILE);
    };

    if (lane == 0) {
        const int n0 = my_chunks < STAGES ? my_chunks : STAGES;
        for (int qi = 0; qi < n0; ++qi) issue(qi, qi);
    }
    locate(0, set, tile);
    enter_tile();
    fetch(neighbour<dir_of<IL>(0)>(g, p_out, t, x, y, zh));
    int q = 0, slot = 0;
    uint32_t phase = 0;
    const T a = (T)L.a, b = (T)L.b, bi = (T)L.bi;
    const T am = (T)L.am;
    const T g5s = L.g5 ? T(-1) : T(1);

    for (int k = 0; k < my_tiles; ++k) {
        // state of the tile being computed (enter_tile(k+1) below overwrites the shared variables at d = 7)
        const int c_set = set, c_tile = tile;
        const bool c_active = active;
        if constexpr (SELF) {
            // the tile's own spinor: one contiguous block -> one bulk copy, consumed in the epilogue
            __syncwarp();   // every lane has finished reading the buffer in the previous epilogue
            if (lane == 0) {
                fence_proxy_async();
                const C *sp = (const C *)(c_set ? L.set[1].self : L.set[0].self) + ((size_t)c_tile * NC) * TILE;
                mbar_expect_tx(selfbar_s, Cfg::SELF_BYTES);
                bulk_g2s_plain(self_s, sp, Cfg::SELF_BYTES, selfbar_s);
            }
        }
        C up[2][DR], lo[2][DR];
#pragma unroll
        for (int s = 0; s < 2; ++s)
#pragma unroll
            for (int c = 0; c < DR; ++c) up[s][c] = lo[s][c] = mk<T>(0, 0);

        static_for<0, 8>([&](auto dc) {
            constexpr int I = decltype(dc)::value, D = dir_of<IL>(I);
            using DI = DirInfo<D>;
            // (a2) spin projection of the neighbour fetched earlier
            C hs[2][DR];
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int qq = DI::swap ? 1 - s : s;
                const T cs = (T)(DI::sg * DI::sigma(s));
#pragma unroll
                for (int c = 0; c < DR; ++c) {
                    const C u = nb[s * DR + c], v = nb[(2 + qq) * DR + c];
                    if (DI::imag) hs[s][c] = mk<T>(fma(-cs, v.y, u.x), fma(cs, v.x, u.y));   // u + i cs v
                    else hs[s][c] = mk<T>(fma(cs, v.x, u.x), fma(cs, v.y, u.y));             // u + cs v
                }
            }
            // prefetch the next neighbour (next direction, or direction 0 of this warp's next tile)
            if constexpr (I < 7) {
                fetch(neighbour<dir_of<IL>(I + 1)>(g, p_out, t, x, y, zh));
            } else {
                if (k + 1 < my_tiles) {
                    locate(k + 1, set, tile);
                    enter_tile();
                    fetch(neighbour<dir_of<IL>(0)>(g, p_out, t, x, y, zh));
                }
            }
            // (a3) link matvec from the ring, (a4) reconstruct + accumulate
#pragma unroll
            for (int i = 0; i < DR; ++i) {
                if (i % RPC == 0) mbar_wait(bars_s + 8 * slot, phase);
                const E *W = ring + (size_t)slot * CE + lane;
                E w[DR];
#pragma unroll
                for (int j = 0; j < DR; ++j) w[j] = W[((i % RPC) * DR + j) * TILE];
#pragma unroll
                for (int s = 0; s < 2; ++s) {
                    C chi = mk<T>(0, 0);
#pragma unroll
                    for (int j = 0; j < DR; ++j) mac<T>(chi, w[j], hs[s][j]);
                    up[s][i].x += chi.x;
                    up[s][i].y += chi.y;
                    const T cl = (T)(DI::sg * DI::sigma(s));
                    const int qq = DI::swap ? 1 - s : s;
                    if (DI::imag) { lo[qq][i].x += cl * chi.y; lo[qq][i].y -= cl * chi.x; }   // (-i cl) chi
                    else { lo[qq][i].x += cl * chi.x; lo[qq][i].y += cl * chi.y; }
                }
                if (i % RPC == RPC - 1) {
                    // slot consumed by every lane -> refill it with the chunk STAGES ahead
                    __syncwarp();
                    if (lane == 0 && q + STAGES < my_chunks) {
                        fence_proxy_async();
                        issue(q + STAGES, slot);
                    }
                    ++q;
                    if (++slot == STAGES) { slot = 0; phase ^= 1; }
                }
            }
        });

        if constexpr (SELF) mbar_wait(selfbar_s, k & 1);
        if constexpr (DIAG != DIAG_NONE) {
            // Site-diagonal term (kernels.h DIAG_*), chirality by chirality: c = 0 is spin 0, 1 (the `up` accumulators), c = 1 is spin
            // 2, 3 (`lo`).  v = the vector the matrix multiplies (self, or the scaled hop sum), o = the result rows; the matrix
            // entries arrive through the ring in storage order, every lane reads its own site's column of the slot.
            const T csw = (T)L.diag_csw;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                C v[2 * DR], o[2 * DR];
#pragma unroll
                for (int s = 0; s < 2; ++s)
#pragma unroll
                    for (int j = 0; j < DR; ++j) {
                        const C h = c == 0 ? up[s][j] : lo[s][j];
                        const C bh = mk<T>(b * h.x, b * h.y);
                        if constexpr (DIAG == DIAG_POST) {
                            v[s * DR + j] = bh;
                            o[s * DR + j] = mk<T>(0, 0);
                        } else {
                            const C sv = selfbuf[((2 * c + s) * DR + j) * TILE + lane];
                            if constexpr (DIAG == DIAG_HB) {   // (a + csw A) self: the unit term now, A on csw * self below
                                o[s * DR + j] = mk<T>(fma(a, sv.x, bh.x), fma(a, sv.y, bh.y));
                                v[s * DR + j] = mk<T>(csw * sv.x, csw * sv.y);
                            } else {
                                o[s * DR + j] = bh;
                                v[s * DR + j] = sv;
                            }
                        }
                    }
#pragma unroll
                for (int e = 0; e < NENT / 2; ++e) {
                    const int ge = c * (NENT / 2) + e;   // entry of the site's matrices, storage order
                    if (ge % DE == 0) mbar_wait(bars_s + 8 * slot, phase);
                    const C m = reinterpret_cast<const C *>(smem_raw + (size_t)warp * STAGES * Cfg::CHUNK + (size_t)slot * Cfg::CHUNK)[(ge % DE) * TILE + lane];
                    if constexpr (DIAG == DIAG_HB) {
                        const int i = (e % (DR * DR)) / DR, j = e % DR;
                        if (e < DR * DR) {   // H: +H on the upper spin row, -H on the lower
                            mac<T>(o[i], m, v[j]);
                            mac<T>(o[DR + i], mk<T>(-m.x, -m.y), v[DR + j]);
                        } else {             // B: B psi_1 into row i of spin 0, B^+ psi_0 into row j of spin 1
                            mac<T>(o[i], m, v[DR + j]);
                            mac<T>(o[DR + j], mk<T>(m.x, -m.y), v[i]);
                        }
                    } else {
                        mac<T>(o[e / (2 * DR)], m, v[e % (2 * DR)]);
                    }
                    if (ge % DE == DE - 1 || ge == NENT - 1) {
                        __syncwarp();
                        if (lane == 0 && q + STAGES < my_chunks) {
                            fence_proxy_async();
                            issue(q + STAGES, slot);
                        }
                        ++q;
                        if (++slot == STAGES) { slot = 0; phase ^= 1; }
                    }
                }
#pragma unroll
                for (int s = 0; s < 2; ++s)
#pragma unroll
                    for (int j = 0; j < DR; ++j) {
                        if (c == 0) up[s][j] = o[s * DR + j];
                        else lo[s][j] = o[s * DR + j];
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
            for (int s = 0; s < 2; ++s)
#pragma unroll
                for (int c = 0; c < DR; ++c) {
                    C vu, vl;
                    if constexpr (DIAG != DIAG_NONE) { vu = up[s][c]; vl = lo[s][c]; }
                    else if (bi != T(0)) {   // (b + i bi gamma_5) hop: gamma_5 = +1 on the upper, -1 on the lower components
                        vu = mk<T>(fma(-bi, up[s][c].y, b * up[s][c].x), fma(bi, up[s][c].x, b * up[s][c].y));
                        vl = mk<T>(fma(bi, lo[s][c].y, b * lo[s][c].x), fma(-bi, lo[s][c].x, b * lo[s][c].y));
                    } else { vu = mk<T>(b * up[s][c].x, b * up[s][c].y); vl = mk<T>(b * lo[s][c].x, b * lo[s][c].y); }
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
                    red_store(L.red_mode, out + (size_t)(s * DR + c) * TILE, rp + (size_t)(s * DR + c) * TILE, al, vu, site[0], site[1]);
                    red_store(L.red_mode, out + (size_t)((2 + s) * DR + c) * TILE, rp + (size_t)((2 + s) * DR + c) * TILE, al,
                              mk<T>(g5s * vl.x, g5s * vl.y), site[2], site[3]);
                }
            if (L.red_mode != 0) acc_add(racc, (site[0] + site[1]) + (site[2] + site[3]), L.red_alg);
        }
    }
    red_finish_cta(L.red_mode, L.red_alg, racc, L.red_partial, red_scratch);
}

// Per-device launch preparation, cached per kernel instantiation AND per device: the opt-in shared-memory size is a
// per-device function attribute and the persistent grid follows the SM count of the device the launch goes to.
struct DevCache { int sms[64]; };
template <typename K> inline int prepare_launch(K kern, size_t smem, DevCache &c, int &n_sm) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    if (dev < 0 || dev >= 64) return (int)cudaErrorInvalidDevice;
    if (c.sms[dev] == 0) {
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e == cudaSuccess && smem > 0) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        c.sms[dev] = sms;
    }
    n_sm = c.sms[dev];
    return 0;
}

inline int ring_grid(int n_sm, int max_ctas, int total_tiles, int tiles_per_cta) {
    int grid = (total_tiles + tiles_per_cta - 1) / tiles_per_cta;
    if (grid > n_sm) grid = n_sm;
    if (max_ctas > 0 && grid > max_ctas) grid = max_ctas;
    return grid;
}

template <typename T, int DR, bool REAL, int WARPS, int STAGES, int RPC, bool SELF, int DIAG = DIAG_NONE>
int launch_hop_ring_cfg(const Geo &g, const HopLaunch &L0, cudaStream_t s) {
    using Cfg = RingCfg<T, DR, REAL, WARPS, STAGES, RPC, SELF, DIAG>;
    auto kern = hop_ring_kernel<T, DR, REAL, WARPS, STAGES, RPC, SELF, DIAG>;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, Cfg::SMEM, cache, n_sm)) return rc;
    const HopLaunch &L = L0;
    const int grid = ring_grid(n_sm, L.max_ctas, launch_tiles(g, L) * L.nsets, WARPS);
    return launch_pdl(kern, grid, WARPS * 32, Cfg::SMEM, s, g, L);
}

// a pass with a diagonal term (a != 0 and a self spinor) uses the SELF instantiation, a pure hop the plain one
template <typename T, int DR, bool REAL> int launch_hop_ring(const Geo &g, const HopLaunch &L, cudaStream_t s) {
    const bool self = (L.a != 0.0) && L.set[0].self != nullptr;
    if (L.diag_mode != DIAG_NONE) {   // site-diagonal matrices in the epilogue: the self term is the matrix term
        if constexpr (sizeof(T) == 8 && DR > 4) return KERR_UNSUPPORTED;   // one thread per site spills there: the pair kernel's job
        else {
        if (L.am != 0.0 || !L.set[0].diag || (L.nsets == 2 && !L.set[1].diag)) return KERR_UNSUPPORTED;
        if (L.diag_mode == DIAG_POST) {
            using P = RingPick<T, DR, REAL, false>;
            return launch_hop_ring_cfg<T, DR, REAL, P::WARPS, P::STAGES, P::RPC, false, DIAG_POST>(g, L, s);
        }
        if (!L.set[0].self) return KERR_UNSUPPORTED;
        using P = RingPick<T, DR, REAL, true>;
        if (L.diag_mode == DIAG_HB) return launch_hop_ring_cfg<T, DR, REAL, P::WARPS, P::STAGES, P::RPC, true, DIAG_HB>(g, L, s);
        if (L.diag_mode == DIAG_PRE) return launch_hop_ring_cfg<T, DR, REAL, P::WARPS, P::STAGES, P::RPC, true, DIAG_PRE>(g, L, s);
        return KERR_UNSUPPORTED;
        }
    }
    if (self) {
        using P = RingPick<T, DR, REAL, true>;
        return launch_hop_ring_cfg<T, DR, REAL, P::WARPS, P::STAGES, P::RPC, true>(g, L, s);
    }
    using P = RingPick<T, DR, REAL, false>;
    return launch_hop_ring_cfg<T, DR, REAL, P::WARPS, P::STAGES, P::RPC, false>(g, L, s);
}

}  // namespace hirep
