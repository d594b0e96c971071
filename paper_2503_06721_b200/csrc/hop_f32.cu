// hop_f32.cu -- single-precision instantiations of the stencil kernels.
#include "hop_dispatch.cuh"
namespace hirep {
int k_hop_f32(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s) {
    return hop_by_config<float>(g, N, rep, mode, variant, L, s);
}
}  // namespace hirep
