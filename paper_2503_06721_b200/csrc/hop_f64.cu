// hop_f64.cu -- double-precision instantiations of the stencil kernels.
#include "hop_dispatch.cuh"
namespace hirep {
int k_hop_f64(const Geo &g, int N, int rep, int mode, int variant, const HopLaunch &L, cudaStream_t s) {
    return hop_by_config<double>(g, N, rep, mode, variant, L, s);
}
// the rule of hop_diag_ring<T, DR>() in hop_dispatch.cuh, for the host code that chooses between the fused and the composed form
bool k_hop_diag_supported(int prec, int dR, int real, int mode, int variant) {
    if (mode != 0 || (variant != 0 && variant != 3)) return false;
    if (real && dR != 3) return false;
    return prec == 0 ? dR <= 4 : dR <= 6;
}
}  // namespace hirep
