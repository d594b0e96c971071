// hop_f64.cu -- double-precision instantiations of the stencil kernels.
#include "hop_dispatch.cuh"
namespace hirep {
int k_hop_f64(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s) {
    return hop_by_config<double>(g, N, rep, mode, variant, L, s);
}
}  // namespace hirep
