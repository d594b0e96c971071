// force.cu -- fermion force of the hopping term (Eq 20-21).
//
//   T_mu(x)   = tr_spin[ gamma_5 (1 - gamma_mu) { eta(x+mu) (x) xi^dagger(x) + xi(x+mu) (x) eta^dagger(x) } ]        (Eq 20)
//   F^a_mu(x) = -(1/T_FUND) Re tr[ i T_R^a U^R_mu(x) T_mu(x) ] = 2 Im tr[ T_R^a M ],   M = U^R_mu(x) T_mu(x)         (Eq 21, A32)
//
// The same neighbour gather, spin projection and link matvec as the stencil (steps a2-a3), followed by an outer product
// in colour space that is never formed: with the rank-2 structure of gamma_5 (1 - gamma_mu),
//   h^psi_s = psi_up(x+mu) - e_mu psi_low(x+mu)   (the forward projection of the stencil),
//   k^psi_s = psi_up(x)    + e_mu psi_low(x)      (the (1 + gamma_mu) projection of the site's own spinor),
//   M_kj = sum_s [ (U h^eta_s)_k conj(k^xi_s)_j + (U h^xi_s)_k conj(k^eta_s)_j ],
// and the projection onto the algebra runs over the NON-ZERO entries of the represented generators T_R^a only (a sparse
// table built once per geometry: T_R^a = -i dR/d omega^a, taken exactly as the odd part of the polynomial map R, A33).
// One warp per (parity, tile, mu), lane = site; the eight vectors live in shared memory [vector][component][lane]
// (conflict free), all loops run over run-time d_R, so one kernel serves every representation.
#include <vector>

#include "hop_adjmf.cuh"

namespace hirep {
namespace {

// ---- generator table ------------------------------------------------------------------------------------------------
// dense [a][A][B] double2, a < N^2-1, A,B < d_R:  T_R^a = (R(1 + iT^a) - R(1 - iT^a)) / (2i)
template <int N> __device__ void fund_generator(int a, double sgn, cplx<double> *W) {   // W = 1 + sgn * i * T^a
    for (int e = 0; e < N * N; ++e) W[e] = mk<double>(0, 0);
    for (int i = 0; i < N; ++i) W[i * N + i].x = 1.0;
    const GenIdx ga = gen_decode(a);
    if (ga.kind == 0) {            // S_ij = (E_ij + E_ji)/2
        W[ga.i * N + ga.j].y += sgn * 0.5;
        W[ga.j * N + ga.i].y += sgn * 0.5;
    } else if (ga.kind == 1) {     // A_ij = -i (E_ij - E_ji)/2  ->  i A_ij = (E_ij - E_ji)/2
        W[ga.i * N + ga.j].x += sgn * 0.5;
        W[ga.j * N + ga.i].x -= sgn * 0.5;
    } else {                       // D_j = diag(1,..,1 (j times), -j, 0,..) / sqrt(2 j (j+1))
        const double nrm = diag_norm(ga.j);
        for (int r = 0; r < ga.j; ++r) W[r * N + r].y += sgn * nrm;
        W[ga.j * N + ga.j].y -= sgn * nrm * ga.j;
    }
}

struct LocalMat {
    const cplx<double> *p;
    __device__ __forceinline__ cplx<double> operator[](int e) const { return p[e]; }
};

template <int N, int REP> __global__ void rep_generators_kernel(double2 *table) {
    using Map = RepMap<double, N, REP>;
    constexpr int DR = Map::DR, NA = N * N - 1;
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= NA) return;
    cplx<double> Wp[N * N], Wm[N * N];
    fund_generator<N>(a, +1.0, Wp);
    fund_generator<N>(a, -1.0, Wm);
    const LocalMat P{Wp}, M{Wm};
    double2 *out = table + (size_t)a * DR * DR;
    if constexpr (REP == 1) {      // real rows; run-time row index keeps the code small for the large adjoints
#pragma unroll 1
        for (int A = 0; A < DR; ++A) {
            double rp[DR], rm[DR];
            adj_row_runtime<double, N>(P, A, rp);
            adj_row_runtime<double, N>(M, A, rm);
            for (int B = 0; B < DR; ++B) out[A * DR + B] = make_double2(0.0, -0.5 * (rp[B] - rm[B]));   // (r+ - r-)/(2i)
        }
    } else {
        static_for<0, DR>([&](auto ac) {
            constexpr int A = decltype(ac)::value;
            cplx<double> rp[DR], rm[DR];
            Map::template row<A>(P, rp);
            Map::template row<A>(M, rm);
            for (int B = 0; B < DR; ++B) {
                const double dx = rp[B].x - rm[B].x, dy = rp[B].y - rm[B].y;
                out[A * DR + B] = make_double2(0.5 * dy, -0.5 * dx);                                    // (dx + i dy)/(2i)
            }
        });
    }
}

template <int N> int gen_by_rep(int rep, double2 *table, cudaStream_t s) {
    constexpr int NA = N * N - 1;
    const int nb = (NA + 31) / 32;
    switch (rep) {
    case 0: rep_generators_kernel<N, 0><<<nb, 32, 0, s>>>(table); break;
    case 1: rep_generators_kernel<N, 1><<<nb, 32, 0, s>>>(table); break;
    case 2: rep_generators_kernel<N, 2><<<nb, 32, 0, s>>>(table); break;
    case 3: rep_generators_kernel<N, 3><<<nb, 32, 0, s>>>(table); break;
    default: return KERR_UNSUPPORTED;
    }
    return (int)cudaGetLastError();
}

// ---- the force kernel -------------------------------------------------------------------------------------------------
struct ForceTab {
    const int *rowptr;      // [NA + 1] entries of generator a: rowptr[a] .. rowptr[a+1]
    const int *jk;          // packed j * d_R + k of entry T^a_jk
    const double2 *val;     // T^a_jk
    int NA;
};

// psi_up + cs * (i?) psi_low  with the conventions of hop_small.cuh: (e_mu v)_s = k_mu(s) v_{q_mu(s)}
template <typename T> __device__ __forceinline__ cplx<T> proj(const cplx<T> &u, const cplx<T> &v, T cs, bool imag) {
    return imag ? mk<T>(fma(-cs, v.y, u.x), fma(cs, v.x, u.y)) : mk<T>(fma(cs, v.x, u.x), fma(cs, v.y, u.y));
}

template <typename T, bool REAL>
__global__ void __launch_bounds__(256) force_hopping_kernel(const Geo g, int dR, const cplx<T> *eta, const cplx<T> *xi, const void *links_v,
                                                           ForceTab tab, T *force, long n_units, size_t warp_smem) {
    using C = cplx<T>;
    using E = link_elem<T, REAL>;
    extern __shared__ __align__(16) unsigned char smem_force[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const long unit = (long)blockIdx.x * (blockDim.x >> 5) + wib;          // (parity, tile, mu)
    if (unit >= n_units) return;
    const int mu = (int)(unit & 3);
    const long pt = unit >> 2;
    const int tile = (int)(pt % g.n_tiles), p = (int)(pt / g.n_tiles);
    int h = tile * TILE + lane;
    const bool active = h < g.Nh;
    if (!active) h = g.Nh - 1;
    int t, x, y, zh;
    decode_site(g, h, t, x, y, zh);
    const int hn = mu == 0 ? neighbour<0>(g, p, t, x, y, zh) : mu == 1 ? neighbour<1>(g, p, t, x, y, zh)
                 : mu == 2 ? neighbour<2>(g, p, t, x, y, zh) : neighbour<3>(g, p, t, x, y, zh);
    const int NC = 4 * dR;
    const size_t half = (size_t)g.n_tiles * NC * TILE;                     // complex elements of a half-lattice spinor
    // vectors [v][s][c][lane]: v = 0 h^eta, 1 h^xi, 2 k^eta, 3 k^xi, 4 chi^eta = U h^eta, 5 chi^xi
    C *vec = reinterpret_cast<C *>(smem_force + (size_t)wib * warp_smem) + lane;
    auto V = [&](int v, int s, int c) -> C & { return vec[(size_t)((v * 2 + s) * dR + c) * TILE]; };
    const bool imag = (mu & 1), swap = (mu == 1 || mu == 2);
    for (int f = 0; f < 2; ++f) {
        const C *field = f ? xi : eta;
        const C *own = field + (size_t)p * half + ((size_t)tile * NC) * TILE + lane;
        const C *nb = field + (size_t)(1 - p) * half + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
        for (int s = 0; s < 2; ++s) {
            const int qq = swap ? 1 - s : s;
            const T sig = (mu < 2) ? T(-1) : (s ? T(1) : T(-1));           // DirInfo::sigma(s)
            for (int c = 0; c < dR; ++c) {
                V(f, s, c) = proj<T>(nb[(size_t)(s * dR + c) * TILE], nb[(size_t)((2 + qq) * dR + c) * TILE], -sig, imag);       // sg = -1
                V(2 + f, s, c) = proj<T>(own[(size_t)(s * dR + c) * TILE], own[(size_t)((2 + qq) * dR + c) * TILE], sig, imag);  // sg = +1
            }
        }
    }
    // chi = U_mu(x) h: the forward matrix of the gather block (carries the boundary sign, L945)
    const E *W = (const E *)links_v + ((((size_t)p * g.n_tiles + tile) * 8 + mu) * (size_t)dR * dR) * TILE + lane;
    for (int i = 0; i < dR; ++i) {
        C a0 = mk<T>(0, 0), a1 = a0, b0 = a0, b1 = a0;
        for (int j = 0; j < dR; ++j) {
            const E w = W[(size_t)(i * dR + j) * TILE];
            mac<T>(a0, w, V(0, 0, j));
            mac<T>(a1, w, V(0, 1, j));
            mac<T>(b0, w, V(1, 0, j));
            mac<T>(b1, w, V(1, 1, j));
        }
        V(4, 0, i) = a0; V(4, 1, i) = a1; V(5, 0, i) = b0; V(5, 1, i) = b1;
    }
    // F^a = 2 Im sum_{jk} T^a_jk M_kj,  M_kj = sum_s chi^eta_s[k] conj(k^xi_s[j]) + chi^xi_s[k] conj(k^eta_s[j])
    const long ix = canonical_index(g, p, h);
    T *out = force + ((size_t)ix * 4 + mu) * tab.NA;
    for (int a = 0; a < tab.NA; ++a) {
        T acc = 0;
        for (int e = tab.rowptr[a]; e < tab.rowptr[a + 1]; ++e) {
            const int jk = tab.jk[e], j = jk / dR, k = jk - j * dR;
            const double2 tv = tab.val[e];
            T mx = 0, my = 0;
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const C ce = V(4, s, k), kx = V(3, s, j), cx = V(5, s, k), ke = V(2, s, j);
                mx += ce.x * kx.x + ce.y * kx.y + cx.x * ke.x + cx.y * ke.y;       // Re(chi conj(k))
                my += ce.y * kx.x - ce.x * kx.y + cx.y * ke.x - cx.x * ke.y;       // Im(chi conj(k))
            }
            acc += (T)tv.x * my + (T)tv.y * mx;                                   // Im(tv * M_kj)
        }
        if (active) out[a] = 2 * acc;
    }
}

// ---- small d_R: M in registers, one warp per (parity, tile) walks the four mu ---------------------------------------------------
// The site's own eta, xi (needed by all four directions) are staged ONCE per tile in shared memory -- each lane its own column, by
// cp.async: extra register space, not an exchange -- instead of being re-read by four warps; the neighbours and the forward link
// of each mu are loaded as before; M stays in registers.  For the fundamental representation the generators are those of reading
// A10 in closed form (S_ij, A_ij, D_j: F = Im(M_ij + M_ji), Re(M_ij - M_ji), 2 nrm_j Im(sum_{q<j} M_qq - j M_jj)), so nothing is
// read for them; other representations read the dense table from shared memory (a broadcast).  Round 2's first version ran one warp per
// (parity, tile, mu) with the table read through L1: 12 warps per SM, latency bound (C2 fp64 0.67 ms; this one 0.38 ms, C4 fp32 20.9 -> 8.6 ms).
// resident 128-thread blocks per SM the register budget is cut for: the live set grows with d_R^2 x precision
template <typename T, int DR> constexpr int force_minb() { return DR * DR * (int)sizeof(T) <= 64 ? 4 : DR * DR * (int)sizeof(T) <= 100 ? 3 : 2; }
template <typename T, int DR, bool REAL, bool FUND>
__global__ void __launch_bounds__(128, force_minb<T, DR>()) force_tile_kernel(const Geo g, const cplx<T> *eta, const cplx<T> *xi, const void *links_v,
                                                            const double2 *dense, int NA, T *force, int n_pt) {
    using C = cplx<T>;
    using E = link_elem<T, REAL>;
    constexpr int NC = 4 * DR;
    extern __shared__ __align__(16) unsigned char smem_force[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    C *tab = reinterpret_cast<C *>(smem_force + (size_t)4 * 2 * NC * TILE * sizeof(C));
    if constexpr (!FUND) {
        for (int i = threadIdx.x; i < NA * DR * DR; i += blockDim.x) tab[i] = mk<T>((T)dense[i].x, (T)dense[i].y);
        __syncthreads();
    }
    const int pt = blockIdx.x * 4 + wib;
    if (pt >= n_pt) return;
    const int tile = pt % g.n_tiles, p = pt / g.n_tiles;
    int h = tile * TILE + lane;
    const bool active = h < g.Nh;
    if (!active) h = g.Nh - 1;
    int t, x, y, zh;
    decode_site(g, h, t, x, y, zh);
    const size_t half = (size_t)g.n_tiles * NC * TILE;
    // own[f][c][lane]: f = 0 eta, 1 xi of this site
    C *own = reinterpret_cast<C *>(smem_force) + (size_t)wib * 2 * NC * TILE + lane;
    {
        const uint32_t own_s = smem_u32(own);
        const C *e0 = eta + (size_t)p * half + ((size_t)tile * NC) * TILE + lane, *x0 = xi + (size_t)p * half + ((size_t)tile * NC) * TILE + lane;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            cp_async<sizeof(C)>(own_s + (uint32_t)(c * TILE * sizeof(C)), e0 + (size_t)c * TILE);
            cp_async<sizeof(C)>(own_s + (uint32_t)((NC + c) * TILE * sizeof(C)), x0 + (size_t)c * TILE);
        }
    }
    const long ix = canonical_index(g, p, h);
    bool staged = false;
#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) {
        const int hn = mu == 0 ? neighbour<0>(g, p, t, x, y, zh) : mu == 1 ? neighbour<1>(g, p, t, x, y, zh)
                     : mu == 2 ? neighbour<2>(g, p, t, x, y, zh) : neighbour<3>(g, p, t, x, y, zh);
        const bool imag = (mu & 1), swap = (mu == 1 || mu == 2);
        const E *W = (const E *)links_v + ((((size_t)p * g.n_tiles + tile) * 8 + mu) * (size_t)DR * DR) * TILE + lane;
        E w[DR][DR];
#pragma unroll
        for (int k = 0; k < DR; ++k)
#pragma unroll
            for (int j = 0; j < DR; ++j) w[k][j] = W[(size_t)(k * DR + j) * TILE];
        C M[DR][DR];
#pragma unroll
        for (int k = 0; k < DR; ++k)
#pragma unroll
            for (int j = 0; j < DR; ++j) M[k][j] = mk<T>(0, 0);
        // M += (U h^A) (x) (k^B)^dagger for (A, B) = (eta, xi) and (xi, eta)
#pragma unroll
        for (int f = 0; f < 2; ++f) {
            const C *fa = f ? xi : eta;
            const C *nb = fa + (size_t)(1 - p) * half + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
            C nbv[NC];
#pragma unroll
            for (int c = 0; c < NC; ++c) nbv[c] = __ldg(nb + (size_t)c * TILE);
            if (!staged) { cp_async_wait_all(); staged = true; }   // the lane's own column of the staged tile has landed
            const C *ob = own + (size_t)((1 - f) * NC) * TILE;     // k comes from the OTHER field
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int qq = swap ? 1 - s : s;
                const T sig = (mu < 2) ? T(-1) : (s ? T(1) : T(-1));
                C hv[DR], kv[DR];
#pragma unroll
                for (int c = 0; c < DR; ++c) {
                    const C lo_n = qq ? nbv[3 * DR + c] : nbv[2 * DR + c];
                    hv[c] = proj<T>(nbv[s * DR + c], lo_n, -sig, imag);
                    kv[c] = proj<T>(ob[(size_t)(s * DR + c) * TILE], ob[(size_t)((2 + qq) * DR + c) * TILE], sig, imag);
                }
#pragma unroll
                for (int k = 0; k < DR; ++k) {
                    C chi = mk<T>(0, 0);
#pragma unroll
                    for (int j = 0; j < DR; ++j) mac<T>(chi, w[k][j], hv[j]);
#pragma unroll
                    for (int j = 0; j < DR; ++j) {     // M_kj += chi_k conj(k_j)
                        M[k][j].x += chi.x * kv[j].x + chi.y * kv[j].y;
                        M[k][j].y += chi.y * kv[j].x - chi.x * kv[j].y;
                    }
                }
            }
        }
        if (!active) continue;
        T *out = force + ((size_t)ix * 4 + mu) * NA;
        if constexpr (FUND) {
            static_for<1, DR>([&](auto jc) {
                constexpr int j = decltype(jc)::value;
                T dsum = 0;
                static_for<0, j>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    out[gen_base(j) + 2 * i] = M[i][j].y + M[j][i].y;
                    out[gen_base(j) + 2 * i + 1] = M[i][j].x - M[j][i].x;
                    dsum += M[i][i].y;
                });
                out[gen_base(j) + 2 * j] = (T)(2.0 * diag_norm(j)) * (dsum - j * M[j][j].y);
            });
        } else {
            for (int a = 0; a < NA; ++a) {
                const C *ta = tab + (size_t)a * DR * DR;
                T acc = 0;
#pragma unroll
                for (int j = 0; j < DR; ++j)
#pragma unroll
                    for (int k = 0; k < DR; ++k) {
                        const C tv = ta[j * DR + k];                        // T^a_jk, the same address in every lane
                        acc += tv.x * M[k][j].y + tv.y * M[k][j].x;        // Im(T^a_jk M_kj)
                    }
                out[a] = 2 * acc;
            }
        }
    }
}

// ---- d_R = 5, 6 in fp64: the same walk with TWO warps per tile ----------------------------------------------------------------
// One thread cannot hold M (d_R^2 complex doubles) next to the link matrix; warp h of a pair owns the rows k = h RPW .. of M and of
// the link (chi_k = sum_j U_kj h_j needs only row k of U), so a thread holds half of each.  Every generator's sum over (j, k) splits
// by k: both warps write their partial F^a into shared memory ([warp][a][lane], double-buffered over mu), one named barrier, then
// each warp adds and stores the generators a = h, h + 2, ...  Dense generator table from shared memory (a broadcast).  C4 fp64
// (SU(4) 2AS, 96x48^3): 81.5 ms with the generic shared-memory kernel below -> see profiles.
template <int DR>
__global__ void __launch_bounds__(128, 2) force_pair_kernel(const Geo g, const cplx<double> *eta, const cplx<double> *xi, const cplx<double> *links,
                                                            const double2 *dense, int NA, double *force, int n_pt) {
    using T = double;
    using C = cplx<T>;
    constexpr int NC = 4 * DR, RPW = (DR + 1) / 2;
    extern __shared__ __align__(16) unsigned char smem_force[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5, pair = wib >> 1, hh = wib & 1;
    // layout: own spinors [2 pairs][2 fields][NC][32] C | partial forces [2 pairs][2 buffers][2 warps][NA][32] T | table [NA][DR][DR] C
    C *own = reinterpret_cast<C *>(smem_force) + (size_t)pair * 2 * NC * TILE + lane;
    T *fx = reinterpret_cast<T *>(smem_force + (size_t)2 * 2 * NC * TILE * sizeof(C)) + (size_t)pair * 4 * NA * TILE + lane;
    const C *tab = reinterpret_cast<const C *>(smem_force + (size_t)2 * 2 * NC * TILE * sizeof(C) + (size_t)2 * 4 * NA * TILE * sizeof(T));
    {
        C *tw = const_cast<C *>(tab);
        for (int i = threadIdx.x; i < NA * DR * DR; i += blockDim.x) tw[i] = mk<T>(dense[i].x, dense[i].y);
        __syncthreads();
    }
    const int pt = blockIdx.x * 2 + pair;
    if (pt >= n_pt) return;                                   // both warps of the pair leave together
    const int tile = pt % g.n_tiles, p = pt / g.n_tiles;
    int h = tile * TILE + lane;
    const bool active = h < g.Nh;
    if (!active) h = g.Nh - 1;
    int t, x, y, zh;
    decode_site(g, h, t, x, y, zh);
    const size_t half = (size_t)g.n_tiles * NC * TILE;
    {
        const uint32_t own_s = smem_u32(own);
        const C *e0 = eta + (size_t)p * half + ((size_t)tile * NC) * TILE + lane, *x0 = xi + (size_t)p * half + ((size_t)tile * NC) * TILE + lane;
        // the pair shares one staged copy: warp 0 brings eta, warp 1 xi (a pair barrier after the wait, below)
        const C *src = hh ? x0 : e0;
#pragma unroll
        for (int c = 0; c < NC; ++c) cp_async<sizeof(C)>(own_s + (uint32_t)((hh * NC + c) * TILE * sizeof(C)), src + (size_t)c * TILE);
    }
    const long ix = canonical_index(g, p, h);
    const int r0 = hh * RPW;
    bool staged = false;
#pragma unroll 1
    for (int mu = 0; mu < 4; ++mu) {
        const int hn = mu == 0 ? neighbour<0>(g, p, t, x, y, zh) : mu == 1 ? neighbour<1>(g, p, t, x, y, zh)
                     : mu == 2 ? neighbour<2>(g, p, t, x, y, zh) : neighbour<3>(g, p, t, x, y, zh);
        const bool imag = (mu & 1), swap = (mu == 1 || mu == 2);
        const C *W = links + ((((size_t)p * g.n_tiles + tile) * 8 + mu) * (size_t)DR * DR) * TILE + lane;
        C w[RPW][DR];
#pragma unroll
        for (int kk = 0; kk < RPW; ++kk) {
            const int k = r0 + kk < DR ? r0 + kk : DR - 1;     // a ragged last row (d_R = 5) repeats row d_R - 1; it is left out of the sums
#pragma unroll
            for (int j = 0; j < DR; ++j) w[kk][j] = W[(size_t)(k * DR + j) * TILE];
        }
        C M[RPW][DR];
#pragma unroll
        for (int kk = 0; kk < RPW; ++kk)
#pragma unroll
            for (int j = 0; j < DR; ++j) M[kk][j] = mk<T>(0, 0);
#pragma unroll
        for (int f = 0; f < 2; ++f) {
            const C *fa = f ? xi : eta;
            const C *nb = fa + (size_t)(1 - p) * half + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
            const C *ob = own + (size_t)((1 - f) * NC) * TILE;
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                const int qq = swap ? 1 - s : s;
                const T sig = (mu < 2) ? T(-1) : (s ? T(1) : T(-1));
                C nu[DR], nl[DR];
#pragma unroll
                for (int c = 0; c < DR; ++c) {
                    nu[c] = __ldg(nb + (size_t)(s * DR + c) * TILE);
                    nl[c] = __ldg(nb + (size_t)((2 + qq) * DR + c) * TILE);
                }
                if (!staged) { cp_async_wait_all(); pair_sync(1 + pair); staged = true; }
                C hv[DR], kv[DR];
#pragma unroll
                for (int c = 0; c < DR; ++c) {
                    hv[c] = proj<T>(nu[c], nl[c], -sig, imag);
                    kv[c] = proj<T>(ob[(size_t)(s * DR + c) * TILE], ob[(size_t)((2 + qq) * DR + c) * TILE], sig, imag);
                }
#pragma unroll
                for (int kk = 0; kk < RPW; ++kk) {
                    C chi = mk<T>(0, 0);
#pragma unroll
                    for (int j = 0; j < DR; ++j) mac<T>(chi, w[kk][j], hv[j]);
#pragma unroll
                    for (int j = 0; j < DR; ++j) {
                        M[kk][j].x += chi.x * kv[j].x + chi.y * kv[j].y;
                        M[kk][j].y += chi.y * kv[j].x - chi.x * kv[j].y;
                    }
                }
            }
        }
        // partial F^a over this warp's rows k -> shared memory, then the pair adds and stores
        T *mine = fx + (size_t)((mu & 1) * 2 + hh) * NA * TILE;
        for (int a = 0; a < NA; ++a) {
            const C *ta = tab + (size_t)a * DR * DR;
            T acc = 0;
#pragma unroll
            for (int kk = 0; kk < RPW; ++kk) {
                const int k = r0 + kk;
                if (k < DR) {
#pragma unroll
                    for (int j = 0; j < DR; ++j) {
                        const C tv = ta[j * DR + k];
                        acc += tv.x * M[kk][j].y + tv.y * M[kk][j].x;
                    }
                }
            }
            mine[(size_t)a * TILE] = acc;
        }
        pair_sync(1 + pair);
        const T *f0 = fx + (size_t)((mu & 1) * 2) * NA * TILE, *f1 = f0 + (size_t)NA * TILE;
        if (active) {
            T *out = force + ((size_t)ix * 4 + mu) * NA;
            for (int a = hh; a < NA; a += 2) out[a] = 2 * (f0[(size_t)a * TILE] + f1[(size_t)a * TILE]);
        }
    }
}
template <int DR> int launch_force_pair(const Geo &g, const void *eta, const void *xi, const void *links, const void *dense, int NA, void *force, cudaStream_t s) {
    auto kern = force_pair_kernel<DR>;
    auto bytes = [](int na) { return (size_t)2 * 2 * 4 * DR * TILE * sizeof(cplx<double>) + (size_t)2 * 4 * na * TILE * sizeof(double) + (size_t)na * DR * DR * sizeof(cplx<double>); };
    if (NA > 35) return KERR_UNSUPPORTED;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, bytes(35), cache, n_sm)) return rc;
    const int n_pt = 2 * g.n_tiles;
    kern<<<(unsigned)((n_pt + 1) / 2), 128, bytes(NA), s>>>(g, (const cplx<double> *)eta, (const cplx<double> *)xi, (const cplx<double> *)links, (const double2 *)dense, NA,
                                                       (double *)force, n_pt);
    return (int)cudaGetLastError();
}

template <typename T, int DR, bool REAL, bool FUND>
int launch_force_tile(const Geo &g, const void *eta, const void *xi, const void *links, const void *dense, int NA, void *force, cudaStream_t s) {
    auto kern = force_tile_kernel<T, DR, REAL, FUND>;
    const size_t own = (size_t)4 * 2 * 4 * DR * TILE * sizeof(cplx<T>);
    const size_t smem = own + (FUND ? 0 : (size_t)NA * DR * DR * sizeof(cplx<T>));
    // the opt-in size is set once per instantiation and device: for the largest generator table any group has here (SU(6): 35)
    const size_t smem_max = own + (FUND ? 0 : (size_t)35 * DR * DR * sizeof(cplx<T>));
    if (NA > 35) return KERR_UNSUPPORTED;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, smem_max, cache, n_sm)) return rc;
    const int n_pt = 2 * g.n_tiles;
    kern<<<(unsigned)((n_pt + 3) / 4), 128, smem, s>>>(g, (const cplx<T> *)eta, (const cplx<T> *)xi, links, (const double2 *)dense, NA, (T *)force, n_pt);
    return (int)cudaGetLastError();
}
template <typename T, bool REAL>
int force_site_dispatch(const Geo &g, int dR, int fund, const void *eta, const void *xi, const void *links, const void *dense, int NA, void *force,
                        cudaStream_t s) {
#define FT(D)                                                                                                                        \
    do {                                                                                                                             \
        if constexpr (!REAL) { if (fund) return launch_force_tile<T, D, false, true>(g, eta, xi, links, dense, NA, force, s); }       \
        return launch_force_tile<T, D, REAL, false>(g, eta, xi, links, dense, NA, force, s);                                         \
    } while (0)
    switch (dR) {
    case 1: return launch_force_tile<T, 1, REAL, false>(g, eta, xi, links, dense, NA, force, s);
    case 2: FT(2);
    case 3: FT(3);
    case 4: FT(4);
    case 5: if constexpr (sizeof(T) == 4) { FT(5); } else if constexpr (!REAL) return launch_force_pair<5>(g, eta, xi, links, dense, NA, force, s); else return KERR_UNSUPPORTED;
    case 6: if constexpr (sizeof(T) == 4) { FT(6); } else if constexpr (!REAL) return launch_force_pair<6>(g, eta, xi, links, dense, NA, force, s); else return KERR_UNSUPPORTED;
    default: return KERR_UNSUPPORTED;
    }
#undef FT
}

// ---- adjoint representation, matrix-free (link mode REBUILD): the force as a commutator of N x N matrices -----------------------
// (T^a_adj)_bc = -i f^abc, so  k^dagger T^a_adj chi = -2 tr( T^a [K^dagger, X] )  with K = k_b T^b, X = chi_c T^c, and chi = R(W) h means
// X = W H W^dagger (hop_adjmf.cuh).  Hence
//   F^a_mu(x) = -4 Im tr( T^a C ),  C = sum_s [K^xi_s^dagger, W H^eta_s W^dagger] + [K^eta_s^dagger, W H^xi_s W^dagger],
// four N x N products per (field pair, s) on the FUNDAMENTAL link instead of d_R x d_R work per generator: the SU(6) adjoint force
// drops from 50 ms (sparse-generator kernel, one warp per SM) to the cost of a few stencil applications.  Same lane mapping as
// hop_adjmf.cuh: N lanes per site (lane = matrix row), matrices exchanged through a per-warp shared-memory area [entry][site].
template <typename T, int N> struct ForceAdjCfg {
    using C = cplx<T>;
    static constexpr int DR = N * N - 1, NC = 4 * DR, NN = N * N, SPW = 32 / N;
    static constexpr int NCL = (DR + N - 1) / N, NLD = (NC + N - 1) / N;
    static constexpr uint32_t RAW = NC * SPW * sizeof(C), MAT = NN * SPW * sizeof(C);
    static constexpr uint32_t PER_WARP = 2 * RAW + 3 * MAT;        // neighbour spinor, own spinor | X (then C), K, W
    static constexpr int WARPS = (int)((200 * 1024) / PER_WARP) > 8 ? 8 : (int)((200 * 1024) / PER_WARP);
    static constexpr size_t SMEM = (size_t)PER_WARP * WARPS;
};

template <typename T, int N>
__global__ void __launch_bounds__(ForceAdjCfg<T, N>::WARPS * 32) force_adjmf_kernel(const Geo g, const cplx<T> *eta, const cplx<T> *xi, const cplx<T> *links_fund,
                                                                                  T *force, long n_units) {
    using C = cplx<T>;
    using Cfg = ForceAdjCfg<T, N>;
    constexpr int DR = Cfg::DR, NC = Cfg::NC, NN = Cfg::NN, SPW = Cfg::SPW, NCL = Cfg::NCL, NLD = Cfg::NLD;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int sl = lane / N, r = lane - sl * N;
    const bool lane_on = sl < SPW;
    const int ssl = lane_on ? sl : 0;
    unsigned char *base = smem_raw + (size_t)warp * Cfg::PER_WARP;
    C *rawA = reinterpret_cast<C *>(base), *rawB = reinterpret_cast<C *>(base + Cfg::RAW);
    C *mX = reinterpret_cast<C *>(base + 2 * Cfg::RAW), *mK = mX + NN * SPW, *mW = mK + NN * SPW;
    const uint32_t rawA_s = smem_u32(rawA), rawB_s = smem_u32(rawB), mW_s = smem_u32(mW);
    const long n_groups_par = (g.Nh + SPW - 1) / SPW;
    const size_t half = (size_t)g.n_tiles * NC * TILE;

    for (long unit = (long)blockIdx.x * Cfg::WARPS + warp; unit < n_units; unit += (long)gridDim.x * Cfg::WARPS) {
        const int mu = (int)(unit & 3);
        const long gp = unit >> 2;
        const int p = (int)(gp / n_groups_par);
        int h = (int)((gp - p * n_groups_par) * SPW) + ssl;
        const bool active = lane_on && h < g.Nh;
        if (h >= g.Nh) h = g.Nh - 1;
        const int tile = h >> 5, hl = h & 31;
        int t, x, y, zh;
        decode_site(g, h, t, x, y, zh);
        const int hn = mu == 0 ? neighbour<0>(g, p, t, x, y, zh) : mu == 1 ? neighbour<1>(g, p, t, x, y, zh)
                     : mu == 2 ? neighbour<2>(g, p, t, x, y, zh) : neighbour<3>(g, p, t, x, y, zh);
        const bool imag = (mu & 1) != 0, swap = (mu == 1 || mu == 2);
        const int crd = mu == 0 ? t : mu == 1 ? x : mu == 2 ? y : 2 * zh + ((t + x + y + p) & 1);
        const bool edge = mu == 0 ? t_edge(g, t, true) : (crd == g.L - 1);
        const T sgn = (T)(edge ? g.bc[mu] : 1);                  // boundary factor of the forward hop (Eq 61)
        const C *lk = links_fund + ((((size_t)p * g.n_tiles + tile) * 8 + mu) * NN) * TILE + hl;   // U_mu(x), forward matrix of the gather block

        // row r of  sum_a h^a T^a  with h^a = psi_s^a + k psi_low^a  (k = cs or i cs)  from a staged spinor [c][site]
        auto assemble = [&](const C *rw, int s, T sgp, C (&P)[N]) {
            const int qq = swap ? 1 - s : s;
            const T cs = sgp * ((mu < 2) ? T(-1) : (s ? T(1) : T(-1)));
            const T kr = imag ? T(0) : cs, ki = imag ? cs : T(0);
            const C *pu = rw + (size_t)(s * DR) * SPW, *pl = rw + (size_t)((2 + qq) * DR) * SPW;
            auto hval = [&](int aa) {
                const C u = pu[aa * SPW], v = pl[aa * SPW];
                return mk<T>(fma(kr, v.x, fma(-ki, v.y, u.x)), fma(kr, v.y, fma(ki, v.x, u.y)));
            };
            C dg = mk<T>(0, 0);
#pragma unroll
            for (int j = 1; j < N; ++j) {
                const C hd = hval(gen_base(j) + 2 * j);
                const T f = (T)diag_norm(j) * (r < j ? T(1) : (r == j ? T(-j) : T(0)));
                dg.x = fma(f, hd.x, dg.x);
                dg.y = fma(f, hd.y, dg.y);
            }
#pragma unroll
            for (int k = 0; k < N; ++k) {
                const int i = k < r ? k : r, j = k < r ? r : k;
                const int as_ = k == r ? 0 : gen_base(j) + 2 * i;
                const C hS = hval(as_), hA = hval(as_ + 1);
                const T sg2 = k > r ? T(1) : T(-1);
                const C off = mk<T>(T(0.5) * (hS.x + sg2 * hA.y), T(0.5) * (hS.y - sg2 * hA.x));
                P[k] = k == r ? dg : off;
            }
        };

        C Cr[N];                                                 // row r of C
#pragma unroll
        for (int k = 0; k < N; ++k) Cr[k] = mk<T>(0, 0);
        __syncwarp();
        if (lane_on) {
#pragma unroll
            for (int k = 0; k < N; ++k) cp_async<sizeof(C)>(mW_s + (uint32_t)(((r * N + k) * SPW + sl) * sizeof(C)), lk + (size_t)(r * N + k) * TILE);
        }
#pragma unroll 1
        for (int f = 0; f < 2; ++f) {                            // (neighbour field, own field) = (eta, xi), (xi, eta)
            const C *fa = f ? xi : eta, *fb = f ? eta : xi;
            const C *srcA = fa + (size_t)(1 - p) * half + ((size_t)(hn >> 5) * NC) * TILE + (hn & 31);
            const C *srcB = fb + (size_t)p * half + ((size_t)tile * NC) * TILE + hl;
            __syncwarp();                                        // previous readers of the staging areas are done
            if (lane_on) {
#pragma unroll
                for (int m = 0; m < NLD; ++m) {
                    const int c = r + N * m;
                    if (c < NC) {
                        cp_async<sizeof(C)>(rawA_s + (uint32_t)((c * SPW + sl) * sizeof(C)), srcA + (size_t)c * TILE);
                        cp_async<sizeof(C)>(rawB_s + (uint32_t)((c * SPW + sl) * sizeof(C)), srcB + (size_t)c * TILE);
                    }
                }
            }
            cp_async_wait_all();
            __syncwarp();
            C wr[N];
#pragma unroll
            for (int k = 0; k < N; ++k) wr[k] = mW[((r * N + k) * SPW) + ssl];
#pragma unroll 1
            for (int s = 0; s < 2; ++s) {
                C P[N], Kr[N];
                assemble(rawA + ssl, s, T(-1), P);               // H_s: forward projection (1 - gamma_mu) of the neighbour
                assemble(rawB + ssl, s, T(1), Kr);               // K_s: (1 + gamma_mu) projection of the site's own spinor
                __syncwarp();                                    // the previous s has finished reading mX, mK
                if (lane_on) {
#pragma unroll
                    for (int k = 0; k < N; ++k) { mX[((r * N + k) * SPW) + sl] = P[k]; mK[((r * N + k) * SPW) + sl] = Kr[k]; }
                }
                __syncwarp();
                C A[N], X[N];
#pragma unroll
                for (int k = 0; k < N; ++k) A[k] = mk<T>(0, 0);
#pragma unroll
                for (int j = 0; j < N; ++j)
#pragma unroll
                    for (int k = 0; k < N; ++k) mac<T>(A[k], wr[j], mX[((j * N + k) * SPW) + ssl]);          // A = W H
#pragma unroll
                for (int k = 0; k < N; ++k) {
                    C c_ = mk<T>(0, 0);
#pragma unroll
                    for (int j = 0; j < N; ++j) {                                                           // X = A W^dagger
                        const C w = mW[((k * N + j) * SPW) + ssl];
                        c_.x = fma(A[j].x, w.x, c_.x); c_.x = fma(A[j].y, w.y, c_.x);
                        c_.y = fma(A[j].y, w.x, c_.y); c_.y = fma(-A[j].x, w.y, c_.y);
                    }
                    X[k] = c_;
                }
                __syncwarp();                                    // every row has read H
                if (lane_on) {
#pragma unroll
                    for (int k = 0; k < N; ++k) mX[((r * N + k) * SPW) + sl] = X[k];
                }
                __syncwarp();
                // C_r. += (K^dagger X)_r. - (X K^dagger)_r.,   K^dagger_ab = conj(K_ba)
#pragma unroll
                for (int j = 0; j < N; ++j) {
                    const C kjr = mK[((j * N + r) * SPW) + ssl];                                             // K_jr -> K^dagger_rj = conj
#pragma unroll
                    for (int k = 0; k < N; ++k) {
                        const C xv = mX[((j * N + k) * SPW) + ssl];
                        Cr[k].x += kjr.x * xv.x + kjr.y * xv.y;                                              // conj(K_jr) X_jk
                        Cr[k].y += kjr.x * xv.y - kjr.y * xv.x;
                        const C kkj = mK[((k * N + j) * SPW) + ssl];                                         // K^dagger_jk = conj(K_kj)
                        Cr[k].x -= X[j].x * kkj.x + X[j].y * kkj.y;                                          // X_rj conj(K_kj)
                        Cr[k].y -= X[j].y * kkj.x - X[j].x * kkj.y;
                    }
                }
            }
        }
        __syncwarp();
        if (lane_on) {
#pragma unroll
            for (int k = 0; k < N; ++k) mX[((r * N + k) * SPW) + sl] = Cr[k];
        }
        __syncwarp();
        if (active) {
            const long ix = canonical_index(g, p, h);
            T *out = force + ((size_t)ix * 4 + mu) * DR;
            const C *cm = mX + ssl;
#pragma unroll
            for (int m = 0; m < NCL; ++m) {
                const int aa = r + N * m;
                if (aa < DR) {
                    const GenIdx ga = gen_decode(aa);
                    T v;
                    if (ga.kind == 2) {
                        T sum = 0;
                        for (int q = 0; q < ga.j; ++q) sum += cm[(q * N + q) * SPW].y;
                        v = T(-4) * (T)diag_norm(ga.j) * (sum - ga.j * cm[(ga.j * N + ga.j) * SPW].y);
                    } else {
                        const C cij = cm[(ga.i * N + ga.j) * SPW], cji = cm[(ga.j * N + ga.i) * SPW];
                        v = ga.kind == 0 ? T(-2) * (cij.y + cji.y) : T(2) * (cji.x - cij.x);
                    }
                    out[aa] = sgn * v;
                }
            }
        }
    }
}

template <typename T, int N> int launch_force_adjmf(const Geo &g, const void *eta, const void *xi, const void *links_fund, void *force, cudaStream_t s) {
    using Cfg = ForceAdjCfg<T, N>;
    auto kern = force_adjmf_kernel<T, N>;
    static DevCache cache{};
    int n_sm = 0;
    if (const int rc = prepare_launch(kern, Cfg::SMEM, cache, n_sm)) return rc;
    const long n_units = (long)2 * ((g.Nh + Cfg::SPW - 1) / Cfg::SPW) * 4;
    long grid = (n_units + Cfg::WARPS - 1) / Cfg::WARPS;
    if (grid > 4L * n_sm) grid = 4L * n_sm;
    kern<<<(unsigned)grid, Cfg::WARPS * 32, Cfg::SMEM, s>>>(g, (const cplx<T> *)eta, (const cplx<T> *)xi, (const cplx<T> *)links_fund, (T *)force, n_units);
    return (int)cudaGetLastError();
}

}  // namespace

// dense generator table -> device (double2 [NA][dR][dR]); the caller converts it to the sparse form once
int k_rep_generators(int N, int rep, void *table_dev, cudaStream_t s) {
    double2 *t = (double2 *)table_dev;
    switch (N) {
    case 2: return gen_by_rep<2>(rep, t, s);
    case 3: return gen_by_rep<3>(rep, t, s);
    case 4: return gen_by_rep<4>(rep, t, s);
    case 5: return gen_by_rep<5>(rep, t, s);
    case 6: return gen_by_rep<6>(rep, t, s);
    }
    return KERR_UNSUPPORTED;
}

// adjoint representation from the FUNDAMENTAL links (link mode REBUILD)
int k_force_hopping_adj(const Geo &g, int prec, int N, const void *eta, const void *xi, const void *links_fund, void *force, cudaStream_t s) {
#define FA(NN_) (prec == 0 ? launch_force_adjmf<double, NN_>(g, eta, xi, links_fund, force, s) : launch_force_adjmf<float, NN_>(g, eta, xi, links_fund, force, s))
    switch (N) {
    case 2: return FA(2);
    case 3: return FA(3);
    case 4: return FA(4);
    case 5: return FA(5);
    case 6: return FA(6);
    }
#undef FA
    return KERR_UNSUPPORTED;
}

int k_force_hopping(const Geo &g, int prec, int dR, int real, int fund, const void *eta, const void *xi, const void *links, const int *rowptr,
                    const int *jk, const void *val, const void *dense, int NA, void *force, cudaStream_t s) {
    if (dense) {   // d_R <= 4 (fp32: <= 6): the register kernels
        const int rc = prec == 0 ? (real ? force_site_dispatch<double, true>(g, dR, fund, eta, xi, links, dense, NA, force, s)
                                         : force_site_dispatch<double, false>(g, dR, fund, eta, xi, links, dense, NA, force, s))
                                 : (real ? force_site_dispatch<float, true>(g, dR, fund, eta, xi, links, dense, NA, force, s)
                                         : force_site_dispatch<float, false>(g, dR, fund, eta, xi, links, dense, NA, force, s));
        if (rc != KERR_UNSUPPORTED) return rc;
    }
    const size_t w = prec == 0 ? 16 : 8;
    const size_t warp_smem = (size_t)6 * 2 * dR * TILE * w;
    int wpc = (int)((200 * 1024) / warp_smem);
    if (wpc < 1) wpc = 1;
    if (wpc > 8) wpc = 8;
    const long n_units = (long)2 * g.n_tiles * 4;
    const unsigned grid = (unsigned)((n_units + wpc - 1) / wpc);
    const size_t smem = warp_smem * wpc;
    ForceTab tab{rowptr, jk, (const double2 *)val, NA};
    cudaError_t e = cudaSuccess;
#define LAUNCH(TT, RR)                                                                                                              \
    do {                                                                                                                            \
        auto kern = force_hopping_kernel<TT, RR>;                                                                                   \
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);                                     \
        if (e == cudaSuccess)                                                                                                       \
            kern<<<grid, wpc * 32, smem, s>>>(g, dR, (const cplx<TT> *)eta, (const cplx<TT> *)xi, links, tab, (TT *)force, n_units, warp_smem); \
    } while (0)
    if (prec == 0) { if (real) LAUNCH(double, true); else LAUNCH(double, false); }
    else { if (real) LAUNCH(float, true); else LAUNCH(float, false); }
#undef LAUNCH
    if (e != cudaSuccess) return (int)e;
    return (int)cudaGetLastError();
}

}  // namespace hirep
