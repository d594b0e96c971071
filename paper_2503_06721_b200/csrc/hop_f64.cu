// hop_f64.cu -- double-precision instantiations of the stencil kernels.
#include "hop_dispatch.cuh"
namespace hirep {
int k_hop_f64(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s) {
    return hop_by_config<double>(g, N, rep, mode, variant, L, s);
}
// the rules of hop_diag_ring / hop_diag_pair in hop_dispatch.cuh, for the host code that chooses between the fused and the composed form
bool k_hop_diag_supported(int prec, int dR, int real, int mode, int variant) {
    if (mode != 0 || dR > 6 || (real && dR != 3)) return false;
    const bool ring = prec == 0 ? dR <= 4 : true, pair = dR >= 5;
    return variant == 0 || (variant == 3 && ring) || (variant == 4 && pair);
}
}  // namespace hirep
