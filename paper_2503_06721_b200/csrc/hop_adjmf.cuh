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
    static constexpr uint32_t RAW = NC * SPW * sizeof(C);    // staged neighbour spinor [c][site]
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
    const T a = (T)L.a, b = (T)L.b, am = (T)L.am;
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

        // stage direction D: the neighbour spinor (lane r copies components r, r+N, ...) and row r of W_D
        auto stage = [&](auto dc) {
            constexpr int D = decltype(dc)::value;
            const int hn = neighbour<D>(g, p_out, t, x, y, zh);
            const C *src = in + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
            if (lane_on) {
#pragma unroll
                for (int m = 0; m < NLD; ++m) {
                    const int c = r + N * m;
                    if (c < NC) cp_async<sizeof(C)>(raw_s + (uint32_t)((c * SPW + sl) * sizeof(C)), src + (size_t)c * TILE);
                }
                const uint32_t wb = wsm_s + (D & 1) * Cfg::MAT;
#pragma unroll
                for (int k = 0; k < N; ++k)
                    cp_async<sizeof(C)>(wb + (uint32_t)(((r * N + k) * SPW + sl) * sizeof(C)), lk + (size_t)(D * NN + r * N + k) * TILE);
            }
        };

        C acc[4][NCL];
#pragma unroll
        for (int sp = 0; sp < 4; ++sp)
#pragma unroll
            for (int m = 0; m < NCL; ++m) acc[sp][m] = mk<T>(0, 0);

        __syncwarp();                                         // the previous group's last reads of the staging area are done
        stage(IntC<0>{});
        static_for<0, 8>([&](auto dc) {
            constexpr int D = decltype(dc)::value;
            using DI = DirInfo<D>;
            cp_async_wait_all();
            __syncwarp();
            const T sgn = (T)hop_sign_dir<D>(g, p_out, t, x, y, zh);
            const C *rw = raw + ssl;
            // (a2) on-the-fly projection h_s^a = sgn (psi_s^a + cs psi_low^a) and row r of Psi_s = h_s^a T^a
            C P[2][N];
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int qq = DI::swap ? 1 - s : s;
                const T cs = (T)(DI::sg * DI::sigma(s)) * sgn;
                auto hval = [&](int aa) {
                    const C u = rw[(s * DR + aa) * SPW], v = rw[((2 + qq) * DR + aa) * SPW];
                    return DI::imag ? mk<T>(fma(-cs, v.y, sgn * u.x), fma(cs, v.x, sgn * u.y)) : mk<T>(fma(cs, v.x, sgn * u.x), fma(cs, v.y, sgn * u.y));
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
                    if (k == r) { P[s][k] = dg; continue; }
                    const int i = k < r ? k : r, j = k < r ? r : k;           // pair (i < j)
                    const C hS = hval(gen_base(j) + 2 * i), hA = hval(gen_base(j) + 2 * i + 1);
                    // k > r: Psi_ij = (h^S - i h^A)/2 ;  k < r: Psi_ji = (h^S + i h^A)/2
                    const T sg2 = k > r ? T(1) : T(-1);
                    P[s][k] = mk<T>(T(0.5) * (hS.x + sg2 * hA.y), T(0.5) * (hS.y - sg2 * hA.x));
                }
                if (lane_on) {
#pragma unroll
                    for (int k = 0; k < N; ++k) psi[(size_t)((s * NN + r * N + k) * SPW + sl)] = P[s][k];
                }
            }
            const C *wm = wsm + (size_t)(D & 1) * NN * SPW + ssl;
            C wr[N];
#pragma unroll
            for (int k = 0; k < N; ++k) wr[k] = wm[(r * N + k) * SPW];
            __syncwarp();                                     // Psi complete; the staged spinor has been consumed
            if constexpr (D < 7) stage(IntC<(D < 7 ? D + 1 : 7)>{});
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
            __syncwarp();                                     // every row has finished reading Psi
            if (lane_on) {
#pragma unroll
                for (int s = 0; s < 2; ++s)
#pragma unroll
                    for (int k = 0; k < N; ++k) psi[(size_t)((s * NN + r * N + k) * SPW + sl)] = chi[s][k];
            }
            __syncwarp();
            // chi^a = 2 tr(T^a chi) for this lane's colours a = r + N m, then (a4) reconstruct + accumulate
#pragma unroll
            for (int m = 0; m < NCL; ++m) {
                const int aa = r + N * m;
                if (aa < DR) {
                    const GenIdx ga = gen_decode(aa);
#pragma unroll
                    for (int s = 0; s < 2; ++s) {
                        const C *cs_ = psi + (size_t)(s * NN) * SPW + ssl;
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
                        acc[s][m].x += v.x;
                        acc[s][m].y += v.y;
                        const T cl = (T)(DI::sg * DI::sigma(s));
                        const int qq = DI::swap ? 1 - s : s;
                        if (DI::imag) { acc[2 + qq][m].x += cl * v.y; acc[2 + qq][m].y -= cl * v.x; }
                        else { acc[2 + qq][m].x += cl * v.x; acc[2 + qq][m].y += cl * v.y; }
                    }
                }
            }
            __syncwarp();                                     // chi consumed before the next direction overwrites the area
        });

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
                        C v = mk<T>(b * acc[sp][m].x, b * acc[sp][m].y);
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
