// layout_kernels.cu -- canonical <-> native conversion kernels (off the hot path; used by tests, bench set-up
// and hirep_apply_host).  Canonical layout: include/hirep_b200.h; native layout: common.cuh.
#include "kernels.h"

namespace hirep {

// one thread per native site (parity p, half index h); copies the 4*dR complex components
template <typename T, bool IMPORT>
__global__ void spinor_convert_kernel(Geo g, int dR, cplx<T> *native, cplx<T> *canon, int which) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    const int py = blockIdx.y;                       // 0 or (for FULL) 0/1
    const int p = (which == 2) ? py : which;
    if (h >= g.Nh) return;
    const int ncomp = 4 * dR;
    const long ix = canonical_index(g, p, h);
    // canonical row: FULL -> ix ; half lattice -> rank of ix among the sites of that parity (= ix/2: sites of a
    // given parity alternate along z, and L is even, so exactly one of (2k, 2k+1) has the parity)
    const long row = (which == 2) ? ix : (ix >> 1);
    cplx<T> *nat = native + (which == 2 ? (size_t)p * g.n_tiles * ncomp * TILE : 0);
    const int tile = h >> 5, lane = h & 31;
    for (int c = 0; c < ncomp; ++c) {
        const size_t no = spinor_off(tile, c, lane, ncomp);
        const size_t co = (size_t)row * ncomp + c;
        if (IMPORT) nat[no] = canon[co];
        else canon[co] = nat[no];
    }
}

// zero the padding lanes of the last tile so that padded sites never hold garbage
template <typename T> __global__ void spinor_pad_zero_kernel(Geo g, int dR, cplx<T> *native, int nhalves) {
    const int ncomp = 4 * dR;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;   // over ncomp * 32
    if (idx >= ncomp * TILE) return;
    const int c = idx / TILE, lane = idx % TILE;
    const int tile = g.n_tiles - 1;
    if (tile * TILE + lane < g.Nh) return;
    for (int p = 0; p < nhalves; ++p)
        native[(size_t)p * g.n_tiles * ncomp * TILE + spinor_off(tile, c, lane, ncomp)] = mk<T>(0, 0);
}

// one thread per (parity, h, d): gathers the matrix that multiplies the neighbour in direction d
//   d < 4 : U_mu(x) ; d >= 4 : U_mu(x - mu)^dagger         (Eq 8)
template <typename T> __global__ void links_import_kernel(Geo g, int N, cplx<T> *native, const cplx<T> *canon) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    const int d = blockIdx.y, p = blockIdx.z;
    if (h >= g.n_tiles * TILE) return;
    const int tile = h >> 5, lane = h & 31, ne = N * N;
    if (h >= g.Nh) {   // padding lanes: identity-free zeros
        for (int e = 0; e < ne; ++e) native[link_off(g.n_tiles, p, tile, d, e, lane, ne)] = mk<T>(0, 0);
        return;
    }
    int t, x, y, zh;
    decode_site(g, h, t, x, y, zh);
    const int mu = d & 3;
    long ix;
    if (d < 4) ix = canonical_index(g, p, h);
    else {
        int hn;
        switch (mu) {
        case 0: hn = neighbour<4>(g, p, t, x, y, zh); break;
        case 1: hn = neighbour<5>(g, p, t, x, y, zh); break;
        case 2: hn = neighbour<6>(g, p, t, x, y, zh); break;
        default: hn = neighbour<7>(g, p, t, x, y, zh); break;
        }
        ix = canonical_index(g, 1 - p, hn);
    }
    const cplx<T> *U = canon + ((size_t)ix * 4 + mu) * ne;
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j) {
            cplx<T> v;
            if (d < 4) v = U[i * N + j];
            else { v = U[j * N + i]; v.y = -v.y; }
            native[link_off(g.n_tiles, p, tile, d, i * N + j, lane, ne)] = v;
        }
}

// one thread per (parity, h, mu): writes W_mu (bwd = 0) or W_{4+mu} (bwd = 1) to canonical [ix][mu][i][j]
template <typename E> __global__ void links_rep_export_kernel(Geo g, int dR, E *canon, const E *native, int bwd) {
    const int h = blockIdx.x * blockDim.x + threadIdx.x;
    const int mu = blockIdx.y, p = blockIdx.z;
    if (h >= g.Nh) return;
    const int tile = h >> 5, lane = h & 31, ne = dR * dR;
    const long ix = canonical_index(g, p, h);
    E *dst = canon + ((size_t)ix * 4 + mu) * ne;
    for (int e = 0; e < ne; ++e) dst[e] = native[link_off(g.n_tiles, p, tile, mu + 4 * bwd, e, lane, ne)];
}

template <typename T> static int spinor_convert(const Geo &g, int dR, void *native, const void *canon, int which, bool imp, cudaStream_t s) {
    dim3 grid((g.Nh + 127) / 128, which == 2 ? 2 : 1);
    if (imp) {
        spinor_convert_kernel<T, true><<<grid, 128, 0, s>>>(g, dR, (cplx<T> *)native, (cplx<T> *)canon, which);
        if (g.Nh % TILE) spinor_pad_zero_kernel<T><<<(4 * dR * TILE + 127) / 128, 128, 0, s>>>(g, dR, (cplx<T> *)native, which == 2 ? 2 : 1);
    } else
        spinor_convert_kernel<T, false><<<grid, 128, 0, s>>>(g, dR, (cplx<T> *)native, (cplx<T> *)canon, which);
    return (int)cudaGetLastError();
}

int k_spinor_import(const Geo &g, int prec, int dR, void *native, const void *canon, int which, cudaStream_t s) {
    return prec == 0 ? spinor_convert<double>(g, dR, native, canon, which, true, s)
                     : spinor_convert<float>(g, dR, native, canon, which, true, s);
}
int k_spinor_export(const Geo &g, int prec, int dR, void *canon, const void *native, int which, cudaStream_t s) {
    return prec == 0 ? spinor_convert<double>(g, dR, const_cast<void *>(native), canon, which, false, s)
                     : spinor_convert<float>(g, dR, const_cast<void *>(native), canon, which, false, s);
}
int k_links_import(const Geo &g, int prec, int N, void *native_fund, const void *canon, cudaStream_t s) {
    dim3 grid((g.n_tiles * TILE + 127) / 128, 8, 2);
    if (prec == 0) links_import_kernel<double><<<grid, 128, 0, s>>>(g, N, (double2 *)native_fund, (const double2 *)canon);
    else links_import_kernel<float><<<grid, 128, 0, s>>>(g, N, (float2 *)native_fund, (const float2 *)canon);
    return (int)cudaGetLastError();
}
int k_links_rep_export(const Geo &g, int prec, int dR, int real, void *canon, const void *native, int bwd, cudaStream_t s) {
    dim3 grid((g.Nh + 127) / 128, 4, 2);
    if (prec == 0 && real) links_rep_export_kernel<double><<<grid, 128, 0, s>>>(g, dR, (double *)canon, (const double *)native, bwd);
    else if (prec == 0) links_rep_export_kernel<double2><<<grid, 128, 0, s>>>(g, dR, (double2 *)canon, (const double2 *)native, bwd);
    else if (real) links_rep_export_kernel<float><<<grid, 128, 0, s>>>(g, dR, (float *)canon, (const float *)native, bwd);
    else links_rep_export_kernel<float2><<<grid, 128, 0, s>>>(g, dR, (float2 *)canon, (const float2 *)native, bwd);
    return (int)cudaGetLastError();
}

// ---- slab halo: projected half-spinor faces (L624: "send only the projected half spinors") ---------------------------
// The face of a slab = one time slice of one parity = the contiguous half-index range [t_f S, (t_f + 1) S), S = L^3/2.
// face 0: first owned slice (t_f = 1), h = psi_up - e_0 psi_low = psi_up + psi_low : what (1 - gamma_0) needs at the previous rank
// face 1: last owned slice (t_f = T-2), h = psi_up + e_0 psi_low = psi_up - psi_low : what (1 + gamma_0) needs at the next rank
// Message layout [s * d_R + c][site of the slice]: 2 d_R complex per face site.  unpack writes the ghost spinor (h, 0): the
// stencil's own projection of it returns h, so the kernels need no second code path for halo sites.
template <typename T> __global__ void halo_pack_kernel(Geo g, int dR, int face, cplx<T> *buf, const cplx<T> *sp) {
    const int S = g.L * g.L * g.Lh;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S) return;
    const int h = (face ? g.T - 2 : 1) * S + i, ncomp = 4 * dR;
    const T sg = face ? T(-1) : T(1);
    for (int c = 0; c < 2 * dR; ++c) {
        const cplx<T> u = sp[spinor_off(h >> 5, c, h & 31, ncomp)], v = sp[spinor_off(h >> 5, 2 * dR + c, h & 31, ncomp)];
        buf[(size_t)c * S + i] = mk<T>(u.x + sg * v.x, u.y + sg * v.y);
    }
}
template <typename T> __global__ void halo_unpack_kernel(Geo g, int dR, int face, cplx<T> *sp, const cplx<T> *buf) {
    const int S = g.L * g.L * g.Lh;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= S) return;
    const int h = (face ? 0 : g.T - 1) * S + i, ncomp = 4 * dR;   // face-0 data (next rank's first slice) -> ghost slice T-1
    for (int c = 0; c < 2 * dR; ++c) {
        sp[spinor_off(h >> 5, c, h & 31, ncomp)] = buf[(size_t)c * S + i];
        sp[spinor_off(h >> 5, 2 * dR + c, h & 31, ncomp)] = mk<T>(0, 0);
    }
}
int k_halo_pack(const Geo &g, int prec, int dR, int parity, int face, void *buf, const void *spinor_half, cudaStream_t s) {
    (void)parity;
    const int S = g.L * g.L * g.Lh, nb = (S + 127) / 128;
    if (prec == 0) halo_pack_kernel<double><<<nb, 128, 0, s>>>(g, dR, face, (cplx<double> *)buf, (const cplx<double> *)spinor_half);
    else halo_pack_kernel<float><<<nb, 128, 0, s>>>(g, dR, face, (cplx<float> *)buf, (const cplx<float> *)spinor_half);
    return (int)cudaGetLastError();
}
int k_halo_unpack(const Geo &g, int prec, int dR, int parity, int face, void *spinor_half, const void *buf, cudaStream_t s) {
    (void)parity;
    const int S = g.L * g.L * g.Lh, nb = (S + 127) / 128;
    if (prec == 0) halo_unpack_kernel<double><<<nb, 128, 0, s>>>(g, dR, face, (cplx<double> *)spinor_half, (const cplx<double> *)buf);
    else halo_unpack_kernel<float><<<nb, 128, 0, s>>>(g, dR, face, (cplx<float> *)spinor_half, (const cplx<float> *)buf);
    return (int)cudaGetLastError();
}

}  // namespace hirep
