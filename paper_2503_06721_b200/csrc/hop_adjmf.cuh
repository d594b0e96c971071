// hop_adjmf.cuh -- MATRIX-FREE hopping stencil for the adjoint representation (link mode REBUILD at d_R >= 8).
//
//   out(x) = a*self(x) + b * sum_{d=0..7} P_d W^R_d(x) in(nbr_d(x)),   W^R = R_adj(W)                      (Eq 8)
//
// The stored adjoint link is a real d_R x d_R matrix, d_R = N^2 - 1: 9800 B at SU(6) in fp64 against 576 B for the
// fundamental N x N matrix it is a function of (Eq 7; "on-the-fly representation", L343).  The adjoint acts on
// the colour vector psi^a as on the algebra element Psi = psi^a T^a:
//       (R(W) psi)^a = 2 tr( T^a  W Psi W^dagger ),
// so one hop costs two N x N complex matrix products per half-spinor component (2 N^3 complex MACs = 1728 real FMAs at N = 6,
// against 2 d_R^2 = 2450 for the stored real matrix) and reads 17x fewer link bytes: the SU(6) adjoint moves from the HBM
// roofline (0.83 ms per Dphi_eo at C5, fp64) to the FP64 pipe.
//
// Mapping: N consecutive lanes own one site, lane r = row r of every N x N matrix of that site; a warp carries
// SPW = 32 / N sites (5 at N = 6, two lanes idle).  All exchanges between the rows of a site go through a small per-warp
// shared-memory area laid out [entry][site]: the lanes of one site read the same address (a broadcast), so one
// shared-memory wavefront serves a whole warp and the kernel stays on the FP64 / FP32 pipe.  Per direction:
//   1. the neighbour spinor (4 d_R complex, staged by cp.async one direction ahead) is spin-projected on the fly and
//      lane r assembles row r of Psi_s = h_s^a T^a for both half-spinor components s;
//   2. A_s = W Psi_s (row r: W_r. from registers, Psi from shared memory), chi_s = A_s W^dagger (W from shared memory);
//   3. chi_s is written back, each lane projects "its" colours a = r, r+N, ... : chi^a = 2 tr(T^a chi), and accumulates
//      them into the four spin components (step a4).
// The boundary sign (Eq 61) multiplies the half spinor, as in the other REBUILD kernels.  No CTA-wide barrier: a warp is
// its own pipeline.  Generator basis: reading A10 (rep_maps.cuh gen_decode).
#pragma once
#include "hop_full.cuh"

namespace hirep {

__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <typename T, int N> struct AdjMfCfg {
    using C = cplx<T>;
    static constexpr int DR = N * N - 1, NC = 4 * DR, NN = N * N;
    static constexpr int SPW = 32 / N;                       // sites per warp
    static constexpr int NCL = (DR + N - 1) / N;             // colours per lane (a = r + N m)
    static constexpr int NLD = (NC + N - 1) / N;             // neighbour components per lane (c = r + N m)
    static constexpr uint32_t RAW = 4 * NN * SPW * sizeof(C); // staged neighbour spinor [c][site] (4 d_R rows); reused for the 4 result matrices
    static constexpr uint32_t MAT = NN * SPW * sizeof(C);    // one N x N matrix per site [e][site]
    static constexpr uint32_t PER_WARP = RAW + 2 * MAT /* Psi_0, Psi_1 (then chi_0, chi_1) */ + 2 * MAT /* W double buffer */;
    static constexpr int WARPS = sizeof(T) == 8 ? 8 : 12;
    static constexpr size_t SMEM = (size_t)PER_WARP * WARPS;
    static_assert(SMEM <= 227 * 1024, "does not fit shared memory");
};

// index of the generators of reading A10: S_ij, A_ij (i < j) and D_j
__host__ __device__ constexpr int gen_base(int j) { return j * j - 1; }

template <typename T, int N>
__global__ void __launch_bounds__(AdjMfCfg<T, N>::WARPS * 32, 1) hop_adjmf_kernel(const Geo g, const HopLaunch L) {
    using C = cplx<T>;
    using Cfg = AdjMfCfg<T, N>;
    constexpr int DR = Cfg::DR, NC = Cfg::NC, NN = Cfg::NN, SPW = Cfg::SPW, NCL = Cfg::NCL, NLD = Cfg::NLD;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int sl = lane / N, r = lane - sl * N;              // site slot within the warp, matrix row
    const bool lane_on = sl < SPW;
    unsigned char *base = smem_raw + (size_t)warp * Cfg::PER_WARP;
    C *raw = reinterpret_cast<C *>(base);
    C *psi = reinterpret_cast<C *>(base + Cfg::RAW);                          // [s][e][site]
    C *wsm = reinterpret_cast<C *>(base + Cfg::RAW + 2 * Cfg::MAT);           // [buffer][e][site]
    const uint32_t raw_s = smem_u32(raw), wsm_s = smem_u32(wsm);
    const int ssl = lane_on ? sl : 0;                        // idle lanes shadow site slot 0 (reads only, no stores)

    const long n_groups_set = (g.Nh + SPW - 1) / SPW;
    const long n_groups = n_groups_set * L.nsets;
    const long gw = (long)blockIdx.x * Cfg::WARPS + warp, nw = (long)gridDim.x * Cfg::WARPS;
    const T a = (T)L.a, b = (T)L.b, bi = (T)L.bi, am = (T)L.am;
    const T g5s = L.g5 ? T(-1) : T(1);

    for (long grp = gw; grp < n_groups; grp += nw) {
        const int set = L.nsets == 2 ? (int)(grp & 1) : 0;
        const long gs = L.nsets == 2 ? (grp >> 1) : grp;
        int h = (int)(gs * SPW) + ssl;
        const bool active = lane_on && h < g.Nh;
        if (h >= g.Nh) h = g.Nh - 1;
        const int tile = h >> 5, hl = h & 31;
        int t, x, y, zh;
        decode_site(g, h, t, x, y, zh);
        const int p_out = set ? L.set[1].p_out : L.set[0].p_out;
        const C *in = (const C *)(set ? L.set[1].in : L.set[0].in);
        const C *lk = (const C *)(set ? L.set[1].links : L.set[0].links) + ((size_t)tile * 8 * NN) * TILE + hl;   // fundamental gather block

        // the 8 hops run in a RUN-TIME loop: unrolled over the directions the kernel is ~8x the code and stalls on instruction
        // fetch (ncu: 3.7 "no instruction" stalls per issued instruction).  Direction constants of hop_small.cuh at run time:
        auto nbr = [&](int d) {
            switch (d) {
            case 0: return neighbour<0>(g, p_out, t, x, y, zh);
            case 1: return neighbour<1>(g, p_out, t, x, y, zh);
            case 2: return neighbour<2>(g, p_out, t, x, y, zh);
            case 3: return neighbour<3>(g, p_out, t, x, y, zh);
            case 4: return neighbour<4>(g, p_out, t, x, y, zh);
            case 5: return neighbour<5>(g, p_out, t, x, y, zh);
            case 6: return neighbour<6>(g, p_out, t, x, y, zh);
            default: return neighbour<7>(g, p_out, t, x, y, zh);
            }
        };
        // stage direction d: the neighbour spinor (lane r copies components r, r+N, ...) and row r of W_d
        auto stage = [&](int d) {
            const int hn = nbr(d);
            const C *src = in + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
            if (lane_on) {
#pragma unroll
                for (int m = 0; m < NLD; ++m) {
                    const int c = r + N * m;
                    if (c < NC) cp_async<sizeof(C)>(raw_s + (uint32_t)((c * SPW + sl) * sizeof(C)), src + (size_t)c * TILE);
                }
                const uint32_t wb = wsm_s + (d & 1) * Cfg::MAT;
#pragma unroll
                for (int k = 0; k < N; ++k)
                    cp_async<sizeof(C)>(wb + (uint32_t)(((r * N + k) * SPW + sl) * sizeof(C)), lk + (size_t)(d * NN + r * N + k) * TILE);
            }
        };

        // the hop sum is accumulated in the MATRIX basis (row r of the four spin components' N x N matrices): the projection back
        // onto the generators, chi^a = 2 tr(T^a chi), is linear and commutes with the sum over directions and with the spin
        // reconstruction, so it is done once per site instead of once per direction
        C acc[4][N];
#pragma unroll
        for (int sp = 0; sp < 4; ++sp)
#pragma unroll
            for (int k = 0; k < N; ++k) acc[sp][k] = mk<T>(0, 0);

        __syncwarp();                                         // the previous group's last reads of the staging area are done
        stage(0);
#pragma unroll 1
        for (int d = 0; d < 8; ++d) {
            const int mu = d & 3;
            const bool fwd = d < 4, imag = (mu & 1) != 0, swap = (mu == 1 || mu == 2);
            const T sg = fwd ? T(-1) : T(1);
            cp_async_wait_all();
            __syncwarp();
            // boundary factor of the hop (Eq 61), applied to the half spinor
            const int crd = mu == 0 ? t : mu == 1 ? x : mu == 2 ? y : 2 * zh + ((t + x + y + p_out) & 1);
            const int ext = mu == 0 ? g.T : g.L;
            const bool edge = mu == 0 ? t_edge(g, t, fwd) : (fwd ? (crd == ext - 1) : (crd == 0));
            const T sgn = (T)(edge ? g.bc[mu] : 1);
            const C *rw = raw + ssl;
            // (a2) on-the-fly projection h_s^a = sgn (psi_s^a + k psi_low^a), k = cs or i cs, and row r of Psi_s = h_s^a T^a.
            // (Projecting every colour once into shared memory and assembling from there -- each h^a is needed by two rows, the
            // diagonal ones by all N -- was measured slower: two more warp barriers per direction, 0.64 -> 0.68 ms at C5 fp64.)
            C P[2][N];
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int qq = swap ? 1 - s : s;
                const T sig = (mu < 2) ? T(-1) : (s ? T(1) : T(-1));
                const T cs = sg * sig * sgn;
                const T kr = imag ? T(0) : cs, ki = imag ? cs : T(0);
                const C *pu = rw + (size_t)(s * DR) * SPW, *pl = rw + (size_t)((2 + qq) * DR) * SPW;
                auto hval = [&](int aa) {
                    const C u = pu[aa * SPW], v = pl[aa * SPW];
                    return mk<T>(fma(kr, v.x, fma(-ki, v.y, sgn * u.x)), fma(kr, v.y, fma(ki, v.x, sgn * u.y)));
                };
                C dg = mk<T>(0, 0);                           // diagonal entry Psi_rr = sum_j h^{D_j} nrm_j (r < j: 1, r = j: -j)
#pragma unroll
                for (int j = 1; j < N; ++j) {
                    const C hd = hval(gen_base(j) + 2 * j);
                    const T f = (T)diag_norm(j) * (r < j ? T(1) : (r == j ? T(-j) : T(0)));
                    dg.x = fma(f, hd.x, dg.x);
                    dg.y = fma(f, hd.y, dg.y);
                }
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    const int i = k < r ? k : r, j = k < r ? r : k;           // pair (i < j); k = r: unused
                    const int as_ = k == r ? 0 : gen_base(j) + 2 * i;
                    const C hS = hval(as_), hA = hval(as_ + 1);
                    // k > r: Psi_ij = (h^S - i h^A)/2 ;  k < r: Psi_ji = (h^S + i h^A)/2
                    const T sg2 = k > r ? T(1) : T(-1);
                    const C off = mk<T>(T(0.5) * (hS.x + sg2 * hA.y), T(0.5) * (hS.y - sg2 * hA.x));
                    P[s][k] = k == r ? dg : off;
                }
                if (lane_on) {
#pragma unroll
                    for (int k = 0; k < N; ++k) psi[(size_t)((s * NN + r * N + k) * SPW + sl)] = P[s][k];
                }
            }
            const C *wm = wsm + (size_t)(d & 1) * NN * SPW + ssl;
            C wr[N];
#pragma unroll
            for (int k = 0; k < N; ++k) wr[k] = wm[(r * N + k) * SPW];
            __syncwarp();                                     // Psi complete; the staged spinor has been consumed
            if (d < 7) stage(d + 1);
            // (a3) A_s = W Psi_s, chi_s = A_s W^dagger
            C chi[2][N];
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const C *ps = psi + (size_t)(s * NN) * SPW + ssl;
                C A[N];
#pragma unroll
                for (int k = 0; k < N; ++k) A[k] = mk<T>(0, 0);
#pragma unroll
                for (int j = 0; j < N; ++j)
#pragma unroll
                    for (int k = 0; k < N; ++k) mac<T>(A[k], wr[j], ps[(j * N + k) * SPW]);        // A_rk += W_rj Psi_jk
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    C c_ = mk<T>(0, 0);
#pragma unroll
                    for (int j = 0; j < N; ++j) {                                                  // chi_rk += A_rj conj(W_kj)
                        const C w = wm[(k * N + j) * SPW];
                        c_.x = fma(A[j].x, w.x, c_.x); c_.x = fma(A[j].y, w.y, c_.x);
                        c_.y = fma(A[j].y, w.x, c_.y); c_.y = fma(-A[j].x, w.y, c_.y);
                    }
                    chi[s][k] = c_;
                }
            }
            // (a4) reconstruct + accumulate, entry by entry: lower component q(s) += sg conj(k_mu(s)) chi, i.e. times cl or -i cl
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const T sig = (mu < 2) ? T(-1) : (s ? T(1) : T(-1));
                const T cl = sg * sig;
                const bool to0 = (swap ? 1 - s : s) == 0;   // lower component 0 or 1, selected without dynamic register indexing
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    const C v = chi[s][k];
                    const C add = imag ? mk<T>(cl * v.y, -cl * v.x) : mk<T>(cl * v.x, cl * v.y);
                    acc[s][k].x += v.x;
                    acc[s][k].y += v.y;
                    acc[2][k].x += to0 ? add.x : T(0); acc[2][k].y += to0 ? add.y : T(0);
                    acc[3][k].x += to0 ? T(0) : add.x; acc[3][k].y += to0 ? T(0) : add.y;
                }
            }
            __syncwarp();                                     // every row has finished reading Psi and W before they are overwritten
        }

        // the four accumulated matrices -> shared memory (the staging area is free), then each lane projects its colours
        // a = r + N m: out^a = 2 tr(T^a acc)
        if (lane_on) {
#pragma unroll
            for (int sp = 0; sp < 4; ++sp)
#pragma unroll
                for (int k = 0; k < N; ++k) raw[(size_t)((sp * NN + r * N + k) * SPW + sl)] = acc[sp][k];
        }
        __syncwarp();
        C res[4][NCL];
#pragma unroll
        for (int m = 0; m < NCL; ++m) {
            const int aa = r + N * m;
            const GenIdx ga = gen_decode(aa < DR ? aa : 0);
#pragma unroll
            for (int sp = 0; sp < 4; ++sp) {
                const C *cs_ = raw + (size_t)(sp * NN) * SPW + ssl;
                C v;
                if (ga.kind == 2) {
                    C sum = mk<T>(0, 0);
                    for (int q = 0; q < ga.j; ++q) { const C d_ = cs_[(q * N + q) * SPW]; sum.x += d_.x; sum.y += d_.y; }
                    const C dj = cs_[(ga.j * N + ga.j) * SPW];
                    const T f = (T)(2.0 * diag_norm(ga.j));
                    v = mk<T>(f * (sum.x - ga.j * dj.x), f * (sum.y - ga.j * dj.y));
                } else {
                    const C cij = cs_[(ga.i * N + ga.j) * SPW], cji = cs_[(ga.j * N + ga.i) * SPW];
                    if (ga.kind == 0) v = mk<T>(cij.x + cji.x, cij.y + cji.y);              // chi_ij + chi_ji
                    else v = mk<T>(cji.y - cij.y, cij.x - cji.x);                           // -i (chi_ji - chi_ij)
                }
                res[sp][m] = v;
            }
        }

        if (active) {
            C *out = (C *)(set ? L.set[1].out : L.set[0].out) + ((size_t)tile * NC) * TILE + hl;
            const C *self = (const C *)(set ? L.set[1].self : L.set[0].self);
            const bool use_self = self != nullptr && L.a != 0.0;
            if (use_self) self += ((size_t)tile * NC) * TILE + hl;
#pragma unroll
            for (int sp = 0; sp < 4; ++sp)
#pragma unroll
                for (int m = 0; m < NCL; ++m) {
                    const int aa = r + N * m;
                    if (aa < DR) {
                        C v = mk<T>(b * res[sp][m].x, b * res[sp][m].y);
                        if (bi != T(0)) {   // (b + i bi gamma_5) hop
                            const T bs = sp < 2 ? bi : -bi;
                            v = mk<T>(fma(-bs, res[sp][m].y, v.x), fma(bs, res[sp][m].x, v.y));
                        }
                        if (use_self) {
                            const C sv = self[(size_t)(sp * DR + aa) * TILE];
                            const T tm = sp < 2 ? am : -am;                                        // + i mu gamma_5 self (Eq 51)
                            v.x = fma(a, sv.x, v.x); v.y = fma(a, sv.y, v.y);
                            v.x = fma(-tm, sv.y, v.x); v.y = fma(tm, sv.x, v.y);
                        }
                        const T gs_ = sp < 2 ? T(1) : g5s;
                        st_spinor(out + (size_t)(sp * DR + aa) * TILE, mk<T>(gs_ * v.x, gs_ * v.y));
                    }
                }
        }
    }
}

template <typename T, int N> int launch_hop_adjmf(const Geo &g, const HopLaunch &L, cudaStream_t s) {
    using Cfg = AdjMfCfg<T, N>;
    auto kern = hop_adjmf_kernel<T, N>;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, Cfg::SMEM, cache, n_sm)) return rc;
    const long n_groups = (long)((g.Nh + Cfg::SPW - 1) / Cfg::SPW) * L.nsets;
    long grid = (n_groups + Cfg::WARPS - 1) / Cfg::WARPS;
    if (grid > n_sm) grid = n_sm;
    if (L.max_ctas > 0 && grid > L.max_ctas) grid = L.max_ctas;
    kern<<<(unsigned)grid, Cfg::WARPS * 32, Cfg::SMEM, s>>>(g, L);
    return (int)cudaGetLastError();
}

}  // namespace hirep
