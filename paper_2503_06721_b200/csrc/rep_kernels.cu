// rep_kernels.cu -- fundamental -> represented links (Eq 7; "functions that translate the
// fundamental gauge field to the represented one", L339-341) with the boundary signs of L945 applied.
//
// Every slot W of the native gather layout is mapped independently:  W^R = s * R(W).  For the backward
// slots W = U^dagger and R(U^dagger) = R(U)^dagger holds identically for all four maps below (cyclicity of
// the trace for ADJ; entrywise conjugation for the polynomial 2-index maps).
//
//   FUND  R(W) = W
//   2AS   R_(ij),(kl) = W_ik W_jl - W_il W_jk,             pairs i<j  in lexicographic order  (A11)
//   SYM   R_(ij),(kl) = c_ij c_kl sum over distinct orderings of W_pr W_qs,  pairs i<=j, c = 1 | 1/sqrt2
//   ADJ   R_ab = 2 Re tr(T^a W T^b W^dagger), T^a = generalised Gell-Mann / 2 in the order of DESIGN.md A10,
//         evaluated from the generators' sparsity: M^b = W T^b W^dagger is built from two columns of W
//         (or a weighted column sum for the diagonal generators) and tr(T^a M) reads two entries of M.
#include "kernels.h"

namespace hirep {

namespace {

template <typename T> __device__ inline cplx<T> cmul(cplx<T> a, cplx<T> b) { return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <typename T> __device__ inline cplx<T> cmulc(cplx<T> a, cplx<T> b) { return mk<T>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }  // a * conj(b)

// generator a of su(N): kind 0 = S_ij, 1 = A_ij, 2 = D_j  (i < j)
__device__ inline void gen_decode(int a, int &kind, int &i, int &j) {
    int base = 0;
    for (int jj = 1;; ++jj) {
        const int cnt = 2 * jj + 1;
        if (a < base + cnt) {
            const int r = a - base;
            j = jj;
            if (r == 2 * jj) { kind = 2; i = 0; }
            else { kind = r & 1; i = r >> 1; }
            return;
        }
        base += cnt;
    }
}

template <typename T, int N, int REP> struct RepMap;

template <typename T, int N> struct RepMap<T, N, 0> {   // FUND
    static constexpr int DR = N;
    static constexpr bool REAL = false;
    __device__ static void apply(const cplx<T> *W, cplx<T> *out, size_t stride, T sgn) {
#pragma unroll
        for (int e = 0; e < N * N; ++e) out[e * stride] = mk<T>(sgn * W[e].x, sgn * W[e].y);
    }
};

template <typename T, int N> struct RepMap<T, N, 3> {   // 2AS
    static constexpr int DR = N * (N - 1) / 2;
    static constexpr bool REAL = false;
    __device__ static void apply(const cplx<T> *W, cplx<T> *out, size_t stride, T sgn) {
        int A = 0;
#pragma unroll
        for (int i = 0; i < N; ++i)
#pragma unroll
            for (int j = i + 1; j < N; ++j) {
                int B = 0;
#pragma unroll
                for (int k = 0; k < N; ++k)
#pragma unroll
                    for (int l = k + 1; l < N; ++l) {
                        const cplx<T> p = cmul<T>(W[i * N + k], W[j * N + l]);
                        const cplx<T> q = cmul<T>(W[i * N + l], W[j * N + k]);
                        out[(size_t)(A * DR + B) * stride] = mk<T>(sgn * (p.x - q.x), sgn * (p.y - q.y));
                        ++B;
                    }
                ++A;
            }
    }
};

template <typename T, int N> struct RepMap<T, N, 2> {   // SYM
    static constexpr int DR = N * (N + 1) / 2;
    static constexpr bool REAL = false;
    __device__ static void apply(const cplx<T> *W, cplx<T> *out, size_t stride, T sgn) {
        const T r2 = T(0.70710678118654752440);
        int A = 0;
#pragma unroll
        for (int i = 0; i < N; ++i)
#pragma unroll
            for (int j = i; j < N; ++j) {
                int B = 0;
#pragma unroll
                for (int k = 0; k < N; ++k)
#pragma unroll
                    for (int l = k; l < N; ++l) {
                        // orderings of (i,j): {(i,j),(j,i)} or {(i,i)}; same for (k,l)
                        cplx<T> v = cmul<T>(W[i * N + k], W[j * N + l]);
                        if (k != l) { const cplx<T> u = cmul<T>(W[i * N + l], W[j * N + k]); v.x += u.x; v.y += u.y; }
                        if (i != j) {
                            cplx<T> u = cmul<T>(W[j * N + k], W[i * N + l]);
                            if (k != l) { const cplx<T> w = cmul<T>(W[j * N + l], W[i * N + k]); u.x += w.x; u.y += w.y; }
                            v.x += u.x; v.y += u.y;
                        }
                        const T c = sgn * (i == j ? T(1) : r2) * (k == l ? T(1) : r2);
                        out[(size_t)(A * DR + B) * stride] = mk<T>(c * v.x, c * v.y);
                        ++B;
                    }
                ++A;
            }
    }
};

template <typename T, int N> struct RepMap<T, N, 1> {   // ADJ (real)
    static constexpr int DR = N * N - 1;
    static constexpr bool REAL = true;
    __device__ static void apply(const cplx<T> *W, T *out, size_t stride, T sgn) {
        cplx<T> M[N * N];
        for (int b = 0; b < DR; ++b) {
            int kind, k, l;
            gen_decode(b, kind, k, l);
            // M = W T^b W^dagger
            if (kind == 2) {
                const T nrm = rsqrt(T(2 * l * (l + 1)));
                for (int p = 0; p < N; ++p)
                    for (int q = 0; q < N; ++q) {
                        cplx<T> acc = mk<T>(0, 0);
                        for (int r = 0; r < l; ++r) { const cplx<T> u = cmulc<T>(W[p * N + r], W[q * N + r]); acc.x += u.x; acc.y += u.y; }
                        const cplx<T> u = cmulc<T>(W[p * N + l], W[q * N + l]);
                        M[p * N + q] = mk<T>(nrm * (acc.x - l * u.x), nrm * (acc.y - l * u.y));
                    }
            } else {
                for (int p = 0; p < N; ++p)
                    for (int q = 0; q < N; ++q) {
                        const cplx<T> u = cmulc<T>(W[p * N + k], W[q * N + l]);   // W_pk conj(W_ql)
                        const cplx<T> v = cmulc<T>(W[p * N + l], W[q * N + k]);   // W_pl conj(W_qk)
                        if (kind == 0) M[p * N + q] = mk<T>(T(0.5) * (u.x + v.x), T(0.5) * (u.y + v.y));
                        else M[p * N + q] = mk<T>(T(0.5) * (u.y - v.y), T(0.5) * (v.x - u.x));   // (-i/2) u + (i/2) v
                    }
            }
            // R_ab = 2 Re tr(T^a M)
            for (int a = 0; a < DR; ++a) {
                int ka, i, j;
                gen_decode(a, ka, i, j);
                T val;
                if (ka == 0) val = M[i * N + j].x + M[j * N + i].x;
                else if (ka == 1) val = M[j * N + i].y - M[i * N + j].y;
                else {
                    T acc = 0;
                    for (int r = 0; r < j; ++r) acc += M[r * N + r].x;
                    val = 2 * rsqrt(T(2 * j * (j + 1))) * (acc - j * M[j * N + j].x);
                }
                out[(size_t)(a * DR + b) * stride] = sgn * val;
            }
        }
    }
};

// one thread per (parity, padded h, d)
template <typename T, int N, int REP>
__global__ void links_to_rep_kernel(Geo g, typename std::conditional<RepMap<T, N, REP>::REAL, T, cplx<T>>::type *rep,
                                    const cplx<T> *fund) {
    using Map = RepMap<T, N, REP>;
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    const int d = blockIdx.y, p = blockIdx.z;
    if (h >= g.n_tiles * TILE) return;
    const int tile = h >> 5, lane = h & 31;
    cplx<T> W[N * N];
#pragma unroll
    for (int e = 0; e < N * N; ++e) W[e] = fund[link_off(g.n_tiles, p, tile, d, e, lane, N * N)];
    T sgn = 1;
    if (h < g.Nh) {
        int t, x, y, zh;
        decode_site(g, h, t, x, y, zh);
        sgn = (T)hop_sign(g, p, t, x, y, zh, d);
    }
    Map::apply(W, rep + link_off(g.n_tiles, p, tile, d, 0, lane, Map::DR * Map::DR), TILE, sgn);
}

template <typename T, int N, int REP> int launch(const Geo &g, void *rep, const void *fund, cudaStream_t s) {
    using Map = RepMap<T, N, REP>;
    using E = typename std::conditional<Map::REAL, T, cplx<T>>::type;
    dim3 grid((g.n_tiles * TILE + 63) / 64, 8, 2);
    links_to_rep_kernel<T, N, REP><<<grid, 64, 0, s>>>(g, (E *)rep, (const cplx<T> *)fund);
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
