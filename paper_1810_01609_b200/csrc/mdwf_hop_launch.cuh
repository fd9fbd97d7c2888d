// csrc/mdwf_hop_launch.cuh -- launcher template for hop_kernel (fp32/fp64 storage); instantiated per storage precision
// in hop_f64.cu / hop_f32.cu so they compile in parallel.  The fp16 stencil has its own unit (hop16.cu).
#pragma once
#include "mdwf_host.h"

namespace mdwf {

template <typename K>
static inline int launch_with_smem(mdwf_ctx* c, K kern, int grid, int block, size_t smem, cudaStream_t st,
                                   const Geom& g, const HopArgs& a) {
    if (smem > 48 * 1024 && !c->attr_raised.count((const void*)kern)) {
        MDWF_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        c->attr_raised.insert((const void*)kern);
    }
    kern<<<grid, block, smem, st>>>(g, a);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

template <typename S, int R>
static int launch_hop_SR(mdwf_ctx* c, int dagger, int fused, HopArgs& a, cudaStream_t st) {
    typedef typename Store<S>::real T;
    const int cls = sizeof(S) == 4 ? 1 : 2;
    const Geom& gh = hop_geom(c, cls, a.nact);
    const int grid = c->nblk_cls[cls] * a.nact, blk = c->blk_cls[cls];
    size_t smem = 0;
    if (fused) {
        smem = (size_t)blk * sizeof(double);
        if (a.op.kind) smem = std::max(smem, (size_t)smem_reals_G<T>(c->g.Ls, blk) * sizeof(T));
    }
    if (a.partial) c->partial_nblk = c->nblk_cls[cls];
    smem += smem_bytes_links<T>(blk / c->g.Ls);
    if (fused) {
        if (dagger) return launch_with_smem(c, hop_kernel<S, R, true, true>, grid, blk, smem, st, gh, a);
        return launch_with_smem(c, hop_kernel<S, R, false, true>, grid, blk, smem, st, gh, a);
    }
    if (dagger) return launch_with_smem(c, hop_kernel<S, R, true, false>, grid, blk, smem, st, gh, a);
    return launch_with_smem(c, hop_kernel<S, R, false, false>, grid, blk, smem, st, gh, a);
}

template <typename S>
static int launch_hop_S(mdwf_ctx* c, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st) {
    switch (recon) {
        case 18: return launch_hop_SR<S, 18>(c, dagger, fused, a, st);
        case 12: return launch_hop_SR<S, 12>(c, dagger, fused, a, st);
        case 8: return launch_hop_SR<S, 8>(c, dagger, fused, a, st);
    }
    MDWF_FAIL(c, MDWF_EINVAL, "recon must be 18, 12 or 8 (got %d)", recon);
}

int launch_hop_f64(mdwf_ctx* c, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st);
int launch_hop_f32(mdwf_ctx* c, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st);
int launch_hop_f16(mdwf_ctx* c, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st);

}  // namespace mdwf
