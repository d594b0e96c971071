// reduce.cuh -- compensated accumulators shared by the reductions of linalg.cu and the reductions fused into the stencil
// epilogues (hop_full.cuh): Neumaier (Algorithm 2), second-order Neumaier (Algorithm 3), double-double
// (Algorithm 4); partial sums are merged with the branch-free two-sum (L654).
#pragma once
#include "common.cuh"

namespace hirep {

// running compensated sum.  ALG selects the paper's accumulation algorithm (L636: "different algorithms for the
// accumulation are available"):  2 = Neumaier (Algorithm 2, the default): value = s + c
//                                3 = second-order Neumaier (Algorithm 3):  value = s + (c + c2)
//                                4 = double-double (Algorithm 4):          value = s, with (s, c) a normalised pair
struct Acc {
    double s, c, c2;
};
__device__ __forceinline__ void two_sum(double a, double b, double &s, double &e) {   // branch-free variant of Alg 1
    s = __dadd_rn(a, b);
    const double bb = __dsub_rn(s, a);
    e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}
__device__ __forceinline__ void acc_add(Acc &A, double x, int alg) {   // one loop iteration of Algorithm 2 / 3 / 4
    double s, e;
    two_sum(A.s, x, s, e);
    if (alg == 2) {
        A.s = s;
        A.c = __dadd_rn(A.c, e);
    } else if (alg == 3) {
        double c, e2;
        two_sum(A.c, e, c, e2);
        A.s = s;
        A.c = c;
        A.c2 = __dadd_rn(A.c2, e2);
    } else {
        two_sum(s, __dadd_rn(A.c, e), A.s, A.c);
    }
}
// merge two partial sums of the same algorithm (lanes, warps, blocks): the partner's components enter as terms
__device__ __forceinline__ void acc_merge(Acc &A, const Acc &B, int alg) {
    double s, e;
    two_sum(A.s, B.s, s, e);
    if (alg == 2) {
        A.s = s;
        A.c = __dadd_rn(__dadd_rn(A.c, B.c), e);
    } else if (alg == 3) {
        double c, e2, c3, e3;
        two_sum(A.c, B.c, c, e2);
        two_sum(c, e, c3, e3);
        A.s = s;
        A.c = c3;
        A.c2 = __dadd_rn(__dadd_rn(A.c2, B.c2), __dadd_rn(e2, e3));
    } else {
        two_sum(s, __dadd_rn(__dadd_rn(A.c, B.c), e), A.s, A.c);
    }
}
__device__ __forceinline__ double acc_value(const Acc &A, int alg) {
    return alg == 2 ? __dadd_rn(A.s, A.c) : alg == 3 ? __dadd_rn(A.s, __dadd_rn(A.c, A.c2)) : A.s;
}
__device__ __forceinline__ Acc acc_shfl_down(const Acc &A, int off) {
    Acc B;
    B.s = __shfl_down_sync(0xffffffffu, A.s, off);
    B.c = __shfl_down_sync(0xffffffffu, A.c, off);
    B.c2 = __shfl_down_sync(0xffffffffu, A.c2, off);
    return B;
}
// CTA-wide merge for kernels of any block size (<= 32 warps): lanes by shuffles, warps through `scratch` (>= 32 Acc in shared
// memory), fixed order -> deterministic.  Every thread of the CTA must call it (it contains barrier 0); result valid in thread 0.
__device__ inline void cta_merge(Acc &a, int alg, Acc *scratch) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const Acc b = acc_shfl_down(a, off);
        acc_merge(a, b, alg);
    }
    if (lane == 0) scratch[warp] = a;
    __syncthreads();
    if (threadIdx.x == 0)
        for (int w = 1; w < nwarp; ++w) acc_merge(a, scratch[w], alg);
}


// Reductions fused into a stencil epilogue (HopLaunch::red_mode), shared by hop_ring.cuh and hop_pair.cuh; one output element v:
//   mode 0: out = v                                 mode 1: out = v, (s0, s1) += (re v)^2, (im v)^2
//   mode 2: r -= alpha v, (s0, s1) += (re r)^2, (im r)^2; v itself is not stored (the CG's A p)
// s0, s1 are PLAIN per-site chains (<= 8 d_R terms); the site total enters the thread's compensated accumulator once.
template <typename C, typename T>
__device__ __forceinline__ void red_store(int mode, C *out, C *rp, T alpha, const C &v, double &s0, double &s1) {
    if (mode == 2) {
        C r = *rp;
        r.x -= alpha * v.x; r.y -= alpha * v.y;
        *rp = r;
        s0 = fma((double)r.x, (double)r.x, s0); s1 = fma((double)r.y, (double)r.y, s1);
    } else {
        __stcs(out, v);
        if (mode == 1) { s0 = fma((double)v.x, (double)v.x, s0); s1 = fma((double)v.y, (double)v.y, s1); }
    }
}
// end of a kernel with a fused reduction: EVERY thread of the CTA calls this exactly once (also the ones that leave early)
__device__ inline void red_finish_cta(int mode, int alg, Acc &a, void *partial, Acc *scratch) {
    if (mode == 0) return;
    cta_merge(a, alg, scratch);
    if (threadIdx.x == 0) {
        Acc *part = (Acc *)partial;
        part[2 * blockIdx.x] = a;
        part[2 * blockIdx.x + 1] = Acc{0.0, 0.0, 0.0};
    }
}

}  // namespace hirep
