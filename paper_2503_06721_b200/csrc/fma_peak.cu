// fma_peak.cu -- register-resident FMA microbenchmark ("FP64/FP32 FMA peaks must be measured by a
// register-resident DFMA/FFMA microbenchmark on the box").  Not on the hot path: it gives the ALU roofline the
// stencil's pipe utilisation (and the REBUILD link mode, which is ALU-bound in fp64) is read against.
#include "kernels.h"

namespace hirep {

namespace {
template <typename T> __global__ void __launch_bounds__(256) fma_peak_kernel(T *sink, int iters, T seed) {
    constexpr int CH = 16;   // independent chains per thread: covers the FMA latency at 8 warps per scheduler
    T x[CH];
#pragma unroll
    for (int c = 0; c < CH; ++c) x[c] = seed + (T)(threadIdx.x + c);
    const T m = (T)0.999, a = (T)1e-3;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int c = 0; c < CH; ++c) x[c] = fma(x[c], m, a);
    }
    T s = 0;
#pragma unroll
    for (int c = 0; c < CH; ++c) s += x[c];
    if (s == (T)-12345) sink[0] = s;   // never true: keeps the chains alive
}
}  // namespace

// returns 0 and the achieved TFLOP/s (2 flops per FMA), or a cudaError_t
int k_fma_peak(int prec, double *tflops, cudaStream_t stream) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return (int)e;
    void *sink = nullptr;
    if ((e = cudaMalloc(&sink, 16)) != cudaSuccess) return (int)e;
    const int blocks = sms * 8, threads = 256, iters = 4096;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0);
    cudaEventCreate(&t1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {   // first repetition is the warm-up
        cudaEventRecord(t0, stream);
        if (prec == 0) fma_peak_kernel<double><<<blocks, threads, 0, stream>>>((double *)sink, iters, 1.0);
        else fma_peak_kernel<float><<<blocks, threads, 0, stream>>>((float *)sink, iters, 1.0f);
        cudaEventRecord(t1, stream);
        if ((e = cudaEventSynchronize(t1)) != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, t0, t1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(t0);
    cudaEventDestroy(t1);
    cudaFree(sink);
    if (e != cudaSuccess) return (int)e;
    if ((e = cudaGetLastError()) != cudaSuccess) return (int)e;
    *tflops = 2.0 * 16 * (double)iters * threads * blocks / (best * 1e-3) / 1e12;
    return 0;
}

}  // namespace hirep
