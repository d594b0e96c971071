// rep_maps.cuh -- the maps U -> U^R (Eq 7; "functions that translate the fundamental gauge field
// to the represented one", L339-341), one ROW of R(W) at a time, for a fundamental matrix W given by any accessor
// W[e], e = i*N + j (registers, or one lane's column of a shared-memory tile).
//
// Used by links_to_rep (rep_kernels.cu: the stored represented field) and by the stencil kernels in link mode
// REBUILD (R rebuilt in registers from the fundamental field, the "on-the-fly" variant of L343).
//
//   FUND  R(W) = W
//   2AS   R_(ij),(kl) = W_ik W_jl - W_il W_jk,             pairs i<j  in lexicographic order  (A11)
//   SYM   R_(ij),(kl) = c_ij c_kl sum over distinct orderings of W_pr W_qs,  pairs i<=j, c = 1 | 1/sqrt2
//   ADJ   R_ab = 2 Re tr(T^a W T^b W^dagger) = 2 Re tr(Y^a T^b),  Y^a = W^dagger T^a W,
//         T^a = generalised Gell-Mann / 2 in the order of DESIGN.md A10; the generators' sparsity makes Y^a a
//         combination of two rows of W and tr(Y T^b) two entries of Y.
// For the backward gather slots W = U^dagger, and R(U^dagger) = R(U)^dagger holds identically for all four maps.
#pragma once
#include "common.cuh"

namespace hirep {

template <typename T> __device__ __forceinline__ cplx<T> cmul(cplx<T> a, cplx<T> b) { return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <typename T> __device__ __forceinline__ cplx<T> cmulc(cplx<T> a, cplx<T> b) { return mk<T>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }  // a * conj(b)
template <typename T> __device__ __forceinline__ cplx<T> ccmul(cplx<T> a, cplx<T> b) { return mk<T>(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }  // conj(a) * b

// generator a of su(N): kind 0 = S_ij, 1 = A_ij, 2 = D_j  (i < j), order of DESIGN.md A10
struct GenIdx { int kind, i, j; };
__host__ __device__ constexpr GenIdx gen_decode(int a) {
    int base = 0;
    for (int jj = 1;; ++jj) {
        const int cnt = 2 * jj + 1;
        if (a < base + cnt) {
            const int r = a - base;
            if (r == 2 * jj) return GenIdx{2, 0, jj};
            return GenIdx{r & 1, r >> 1, jj};
        }
        base += cnt;
    }
}
// pair (i,j) number A of the 2-index bases: i<j (strict) or i<=j, lexicographic
struct PairIdx { int i, j; };
__host__ __device__ constexpr PairIdx pair_decode(int A, int N, bool strict) {
    int c = 0;
    for (int i = 0; i < N; ++i)
        for (int j = strict ? i + 1 : i; j < N; ++j) {
            if (c == A) return PairIdx{i, j};
            ++c;
        }
    return PairIdx{0, 0};
}
__host__ __device__ constexpr double diag_norm(int j) {   // 1/sqrt(2 j (j+1)) for j = 1..5
    return j == 1 ? 0.5 : j == 2 ? 0.28867513459481288225 : j == 3 ? 0.20412414523193150818
         : j == 4 ? 0.15811388300841896660 : 0.12909944487358056284;
}

template <typename T, int N, int REP> struct RepMap;

template <typename T, int N> struct RepMap<T, N, 0> {   // FUND
    static constexpr int DR = N;
    static constexpr bool REAL = false;
    using E = cplx<T>;
    template <int A, typename WM> __device__ __forceinline__ static void row(const WM &W, E *w) {
#pragma unroll
        for (int B = 0; B < N; ++B) w[B] = W[A * N + B];
    }
};

template <typename T, int N> struct RepMap<T, N, 3> {   // 2AS
    static constexpr int DR = N * (N - 1) / 2;
    static constexpr bool REAL = false;
    using E = cplx<T>;
    template <int A, typename WM> __device__ __forceinline__ static void row(const WM &W, E *w) {
        constexpr PairIdx ij = pair_decode(A, N, true);
        static_for<0, DR>([&](auto bc) {
            constexpr int B = decltype(bc)::value;
            constexpr PairIdx kl = pair_decode(B, N, true);
            const cplx<T> p = cmul<T>(W[ij.i * N + kl.i], W[ij.j * N + kl.j]);
            const cplx<T> q = cmul<T>(W[ij.i * N + kl.j], W[ij.j * N + kl.i]);
            w[B] = mk<T>(p.x - q.x, p.y - q.y);
        });
    }
};

template <typename T, int N> struct RepMap<T, N, 2> {   // SYM
    static constexpr int DR = N * (N + 1) / 2;
    static constexpr bool REAL = false;
    using E = cplx<T>;
    template <int A, typename WM> __device__ __forceinline__ static void row(const WM &W, E *w) {
        constexpr PairIdx ij = pair_decode(A, N, false);
        constexpr int i = ij.i, j = ij.j;
        static_for<0, DR>([&](auto bc) {
            constexpr int B = decltype(bc)::value;
            constexpr PairIdx kl = pair_decode(B, N, false);
            constexpr int k = kl.i, l = kl.j;
            // orderings of (i,j): {(i,j),(j,i)} or {(i,i)}; same for (k,l)
            cplx<T> v = cmul<T>(W[i * N + k], W[j * N + l]);
            if (k != l) { const cplx<T> u = cmul<T>(W[i * N + l], W[j * N + k]); v.x += u.x; v.y += u.y; }
            if (i != j) {
                cplx<T> u = cmul<T>(W[j * N + k], W[i * N + l]);
                if (k != l) { const cplx<T> x = cmul<T>(W[j * N + l], W[i * N + k]); u.x += x.x; u.y += x.y; }
                v.x += u.x; v.y += u.y;
            }
            constexpr double r2 = 0.70710678118654752440;
            const T c = (T)((i == j ? 1.0 : r2) * (k == l ? 1.0 : r2));
            w[B] = mk<T>(c * v.x, c * v.y);
        });
    }
};

template <typename T, int N> struct RepMap<T, N, 1> {   // ADJ (real matrix)
    static constexpr int DR = N * N - 1;
    static constexpr bool REAL = true;
    using E = T;
    // Y = W^dagger T^a W is Hermitian (T^a is), so only its upper triangle is built: Y[p*N+q], p <= q.  Then
    // R_ab = 2 Re tr(Y T^b):  b = S_kl -> 2 Re Y_kl ;  b = A_kl -> -2 Im Y_kl ;  b = D_l -> diagonal combination.
    template <int A, typename WM> __device__ __forceinline__ static void row(const WM &W, E *w) {
        constexpr GenIdx ga = gen_decode(A);
        cplx<T> Y[N * N];
#pragma unroll
        for (int p = 0; p < N; ++p)
#pragma unroll
            for (int q = p; q < N; ++q) {
                if (ga.kind == 2) {
                    cplx<T> acc = mk<T>(0, 0);
#pragma unroll
                    for (int r = 0; r < ga.j; ++r) { const cplx<T> u = ccmul<T>(W[r * N + p], W[r * N + q]); acc.x += u.x; acc.y += u.y; }
                    const cplx<T> u = ccmul<T>(W[ga.j * N + p], W[ga.j * N + q]);
                    const T nrm = (T)diag_norm(ga.j);
                    Y[p * N + q] = mk<T>(nrm * (acc.x - ga.j * u.x), nrm * (acc.y - ga.j * u.y));
                } else {
                    const cplx<T> u = ccmul<T>(W[ga.i * N + p], W[ga.j * N + q]);   // conj(W_ip) W_jq
                    const cplx<T> v = ccmul<T>(W[ga.j * N + p], W[ga.i * N + q]);   // conj(W_jp) W_iq
                    if (ga.kind == 0) Y[p * N + q] = mk<T>(T(0.5) * (u.x + v.x), T(0.5) * (u.y + v.y));
                    else Y[p * N + q] = mk<T>(T(0.5) * (u.y - v.y), T(0.5) * (v.x - u.x));   // (-i/2)(u - v)
                }
            }
        static_for<0, DR>([&](auto bc) {
            constexpr int B = decltype(bc)::value;
            constexpr GenIdx gb = gen_decode(B);
            if constexpr (gb.kind == 0) w[B] = 2 * Y[gb.i * N + gb.j].x;
            else if constexpr (gb.kind == 1) w[B] = -2 * Y[gb.i * N + gb.j].y;
            else {
                T acc = 0;
#pragma unroll
                for (int r = 0; r < gb.j; ++r) acc += Y[r * N + r].x;
                w[B] = (T)(2.0 * diag_norm(gb.j)) * (acc - gb.j * Y[gb.j * N + gb.j].x);
            }
        });
    }
};

// ADJ row with a RUNTIME row index a, for the large adjoints (SU(4..6): d_R = 15, 24, 35).  The compile-time version
// above unrolls d_R rows of ~500 instructions each; at d_R = 35 that is ~280 KB of code and the kernel stalls on
// instruction fetch (ncu: 88 % "no instruction").  Here only the generator (kind, i, j) of row a is a run-time value:
// it selects which rows of W are read (W = any accessor with operator[], e.g. a shared-memory tile), the N x N
// arithmetic and the d_R outputs stay unrolled -- one row body of code.  Same formulas as RepMap<T, N, 1>::row.
template <typename T, int N, typename WM> __device__ __forceinline__ void adj_row_runtime(const WM &W, int a, T *w) {
    constexpr int DR = N * N - 1;
    const GenIdx ga = gen_decode(a);
    cplx<T> Y[N * N];
    if (ga.kind != 2) {
        cplx<T> wi[N], wj[N];
#pragma unroll
        for (int q = 0; q < N; ++q) { wi[q] = W[ga.i * N + q]; wj[q] = W[ga.j * N + q]; }
#pragma unroll
        for (int p = 0; p < N; ++p)
#pragma unroll
            for (int q = p; q < N; ++q) {
                const cplx<T> u = ccmul<T>(wi[p], wj[q]);   // conj(W_ip) W_jq
                const cplx<T> v = ccmul<T>(wj[p], wi[q]);   // conj(W_jp) W_iq
                if (ga.kind == 0) Y[p * N + q] = mk<T>(T(0.5) * (u.x + v.x), T(0.5) * (u.y + v.y));
                else Y[p * N + q] = mk<T>(T(0.5) * (u.y - v.y), T(0.5) * (v.x - u.x));   // (-i/2)(u - v)
            }
    } else {
#pragma unroll
        for (int p = 0; p < N; ++p)
#pragma unroll
            for (int q = p; q < N; ++q) Y[p * N + q] = mk<T>(0, 0);
        for (int r = 0; r <= ga.j; ++r) {
            cplx<T> wr[N];
#pragma unroll
            for (int q = 0; q < N; ++q) wr[q] = W[r * N + q];
            const T f = (r < ga.j) ? T(1) : T(-ga.j);
#pragma unroll
            for (int p = 0; p < N; ++p)
#pragma unroll
                for (int q = p; q < N; ++q) {
                    const cplx<T> u = ccmul<T>(wr[p], wr[q]);
                    Y[p * N + q].x += f * u.x;
                    Y[p * N + q].y += f * u.y;
                }
        }
        const T nrm = (T)diag_norm(ga.j);
#pragma unroll
        for (int p = 0; p < N; ++p)
#pragma unroll
            for (int q = p; q < N; ++q) { Y[p * N + q].x *= nrm; Y[p * N + q].y *= nrm; }
    }
    static_for<0, DR>([&](auto bc) {
        constexpr int B = decltype(bc)::value;
        constexpr GenIdx gb = gen_decode(B);
        if constexpr (gb.kind == 0) w[B] = 2 * Y[gb.i * N + gb.j].x;
        else if constexpr (gb.kind == 1) w[B] = -2 * Y[gb.i * N + gb.j].y;
        else {
            T acc = 0;
#pragma unroll
            for (int r = 0; r < gb.j; ++r) acc += Y[r * N + r].x;
            w[B] = (T)(2.0 * diag_norm(gb.j)) * (acc - gb.j * Y[gb.j * N + gb.j].x);
        }
    });
}

}  // namespace hirep
