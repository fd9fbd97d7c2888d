// csrc/hop_f32.cu -- hop_kernel instantiations for float storage (see mdwf_hop.cuh).
#include "mdwf_hop_launch.cuh"
namespace mdwf {
int launch_hop_f32(mdwf_ctx* c, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st) {
    return launch_hop_S<float>(c, recon, dagger, fused, a, st);
}
}  // namespace mdwf
