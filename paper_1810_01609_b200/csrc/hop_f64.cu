// csrc/hop_f64.cu -- hop_kernel instantiations for double storage (see mdwf_hop.cuh).
#include "mdwf_hop_launch.cuh"
namespace mdwf {
int launch_hop_f64(mdwf_ctx* c, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st) {
    return launch_hop_S<double>(c, recon, dagger, fused, a, st);
}
}  // namespace mdwf
