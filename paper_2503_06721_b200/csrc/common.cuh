// common.cuh -- geometry, native layout addressing and small complex helpers shared by the CUDA kernels.
//
// Native layout (private to the library):
//   parity p of site (t,x,y,z) = (t+x+y+z) & 1
//   half index   h = ((t*L + x)*L + y)*(L/2) + zh,   z = 2*zh + ((t+x+y+p)&1)
//   tiles of 32 consecutive h;  Nh = T*L^3/2 sites per parity, n_tiles = ceil(Nh/32)
//   spinor (half lattice)  [tile][comp = spin*d_R + colour][lane]        complex<T>
//   spinor (full lattice)  even half followed by odd half
//   links                  [parity][tile][d = 0..7][e = i*d + j][lane]   complex<T> or T (real adjoint)
//       W_d, d < 4 : U_mu(x),   mu = d      -- multiplies psi(x+mu)   (forward hop of Eq 8)
//       W_d, d >= 4: U_mu(x-mu)^dagger, mu = d-4 -- multiplies psi(x-mu)
//   so a warp-wide access to one (tile, comp) or (tile, d, e) row is one contiguous 128/256/512-byte segment.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace hirep {

constexpr int TILE = 32;

struct Geo {
    int T, L, Lh;   // Lh = L/2
    int Nh;         // sites per parity
    int n_tiles;    // ceil(Nh / 32)
    int bc[4];      // +-1 per direction (Eq 58-63)
    // Slab of a lattice that is block-partitioned in t over several GPUs (Fig 1): local slice t holds global slice
    // (t + t0) mod Tg.  The boundary factor of direction 0 sits where the GLOBAL lattice closes (only the ranks owning global
    // slices Tg-1 / 0 see it); the local wrap in t is never used by an owned site (ghost slices at both ends).  Undivided
    // lattice: t0 = 0, Tg = T.
    int t0, Tg;
};
// does the hop from local slice t in direction 0 cross the edge of the GLOBAL lattice?
__host__ __device__ inline bool t_edge(const Geo &g, int t, bool fwd) {
    int tg = t + g.t0;
    if (tg >= g.Tg) tg -= g.Tg;
    return fwd ? (tg == g.Tg - 1) : (tg == 0);
}

template <typename T> struct CplxOf;
template <> struct CplxOf<double> { using type = double2; };
template <> struct CplxOf<float> { using type = float2; };
template <typename T> using cplx = typename CplxOf<T>::type;
template <typename T, bool REAL> using link_elem = std::conditional_t<REAL, T, cplx<T>>;

template <typename T> __host__ __device__ inline cplx<T> mk(T re, T im) { cplx<T> r; r.x = re; r.y = im; return r; }

// compile-time loop: f(IntC<B>{}), ..., f(IntC<E-1>{})
template <int I> struct IntC { static constexpr int value = I; };
template <int B, int E, typename F> __device__ __forceinline__ void static_for(F &&f) {
    if constexpr (B < E) {
        f(IntC<B>{});
        static_for<B + 1, E>(f);
    }
}

// Order in which the persistent kernels walk the 8 hops of a tile: step I -> direction dir_of<IL>(I).
// IL = false: storage order 0..7 (+t,+x,+y,+z,-t,-x,-y,-z).
// IL = true : interleaved (+z,-z,+y,-y,+x,-x,+t,-t).  The spinor line of a site is read as the +mu neighbour of one
// tile and as the -mu neighbour of another tile of the same grid round; putting the two reads in adjacent steps
// shortens their distance in L2 from half a tile time to an eighth (C4 fp64: DRAM reads of a Dphi_eo launch 30.3 ->
// 28.8 GB, 4.85 -> 4.6-4.7 ms).  z and y first: those neighbours live in the tile's own rows, which a full-lattice
// launch has just touched as the `self` block.  Which kernels use it is a measured choice.
template <bool IL> __host__ __device__ constexpr int dir_of(int I) { return IL ? ((3 - (I >> 1)) | ((I & 1) << 2)) : I; }

// ---- site <-> coordinates ------------------------------------------------------------------
__host__ __device__ inline void decode_site(const Geo &g, int h, int &t, int &x, int &y, int &zh) {
    zh = h % g.Lh;
    int r = h / g.Lh;
    y = r % g.L;
    r /= g.L;
    x = r % g.L;
    t = r / g.L;
}
__host__ __device__ inline int encode_site(const Geo &g, int t, int x, int y, int zh) {
    return ((t * g.L + x) * g.L + y) * g.Lh + zh;
}
// canonical lexicographic index of native site (parity p, half index h)
__host__ __device__ inline long canonical_index(const Geo &g, int p, int h) {
    int t, x, y, zh;
    decode_site(g, h, t, x, y, zh);
    const int z = 2 * zh + ((t + x + y + p) & 1);
    return (((long)t * g.L + x) * g.L + y) * g.L + z;
}

// Half index (in the OTHER parity's ordering) of the neighbour of site (p; t,x,y,zh) in direction
// D: D < 4 -> x + mu (mu = D), D >= 4 -> x - mu (mu = D-4).  Periodic wrap; the boundary sign lives in the links.
template <int D> __host__ __device__ inline int neighbour(const Geo &g, int p, int t, int x, int y, int zh) {
    constexpr int mu = D & 3;
    constexpr bool fwd = D < 4;
    if (mu == 0) {
        const int tn = fwd ? (t + 1 == g.T ? 0 : t + 1) : (t == 0 ? g.T - 1 : t - 1);
        return encode_site(g, tn, x, y, zh);
    } else if (mu == 1) {
        const int xn = fwd ? (x + 1 == g.L ? 0 : x + 1) : (x == 0 ? g.L - 1 : x - 1);
        return encode_site(g, t, xn, y, zh);
    } else if (mu == 2) {
        const int yn = fwd ? (y + 1 == g.L ? 0 : y + 1) : (y == 0 ? g.L - 1 : y - 1);
        return encode_site(g, t, x, yn, zh);
    } else {
        // z = 2 zh + r with r = (t+x+y+p)&1; the neighbour has the other parity, so its r' = 1-r:
        //   r = 0: z+1 -> zh' = zh,   z-1 -> zh' = zh-1 ;   r = 1: z+1 -> zh' = zh+1,   z-1 -> zh' = zh
        const int r = (t + x + y + p) & 1;
        int zn;
        if (fwd) zn = r ? (zh + 1 == g.Lh ? 0 : zh + 1) : zh;
        else zn = r ? zh : (zh == 0 ? g.Lh - 1 : zh - 1);
        return encode_site(g, t, x, y, zn);
    }
}

// boundary factor of the hop from site (p; t,x,y,zh) in direction d (Eq 61): bc[mu] if it crosses the edge
__host__ __device__ inline int hop_sign(const Geo &g, int p, int t, int x, int y, int zh, int d) {
    const int mu = d & 3;
    const bool fwd = d < 4;
    const int z = 2 * zh + ((t + x + y + p) & 1);
    if (mu == 0) return t_edge(g, t, fwd) ? g.bc[0] : 1;
    const int c = (mu == 1) ? x : (mu == 2) ? y : z;
    const bool cross = fwd ? (c == g.L - 1) : (c == 0);
    return cross ? g.bc[mu] : 1;
}

// ---- element offsets (in elements of the respective type) -------------------------------------
__host__ __device__ inline size_t spinor_off(int tile, int comp, int lane, int ncomp) {
    return ((size_t)tile * ncomp + comp) * TILE + lane;
}
__host__ __device__ inline size_t link_off(int n_tiles, int p, int tile, int d, int e, int lane, int nelem) {
    return ((((size_t)p * n_tiles + tile) * 8 + d) * nelem + e) * TILE + lane;
}

}  // namespace hirep
