// csrc/mdwf_hop_tile.cuh -- the Dslash stencil over compact 4D tiles with the neighbour spinors staged in shared
// memory (same operator and arguments as hop_kernel in mdwf_hop.cuh).
//
// Why: in hop_kernel every output site gathers its 8 neighbours from L2 (L1 only merges the two x-legs), i.e. 8 x
// 24 reals per output cross the L2->SM fabric, which is what limits the fp32 kernel on B200 (profiles/README.md).
// Here a block owns a box of Lx x Ly x Lz x Lt lattice sites (its nsite = volume/2 sites of the output parity);
// the box's input sites -- the other-parity sites inside the box plus the one-site halo -- are copied ONCE into
// shared memory with cp.async (all Ls slices), so only (nsite + halo)/nsite ~ 4 spinors per output are fetched.
// Tiles are congruent up to the parity of their origin, so the local geometry (which local sites are outputs,
// which are input slots, and the slot of every leg) is tabulated on the host for the two patterns (Geom.q4*).
#pragma once
#include <cuda_pipeline.h>
#include "mdwf_hop.cuh"

namespace mdwf {

template <typename S> __host__ __device__ inline size_t smem_bytes_tile(int nsite, int nslot, int Ls) {
    typedef typename Store<S>::real T;
    size_t b = (size_t)nslot * Store<S>::NV * Ls * 16;                 // spinors [slot][row][s]
    if (Store<S>::HALF) b += (((size_t)nslot * Ls * 4) + 15) & ~(size_t)15;   // scales [slot][s]
    b += (size_t)nsite * MDWF_LSITE * sizeof(T);                     // links
    b += (((size_t)(nslot + nsite) * 4) + 15) & ~(size_t)15;           // slot -> xh, output -> xh
    return b;
}

// neighbour spinor from shared memory: rows of Ls x 16 bytes per (slot, vector index)
template <typename S>
__device__ __forceinline__ void load_smem(const unsigned char* spin, const float* scl, int k, int s, int Ls,
                                          typename Store<S>::real v[24], typename Store<S>::real& sc);
template <>
__device__ __forceinline__ void load_smem<float>(const unsigned char* spin, const float*, int k, int s, int Ls,
                                                 float v[24], float& sc) {
    const float4* p = reinterpret_cast<const float4*>(spin) + (k * 6) * Ls + s;
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        const float4 t = p[c * Ls];
        v[4 * c] = t.x; v[4 * c + 1] = t.y; v[4 * c + 2] = t.z; v[4 * c + 3] = t.w;
    }
    sc = 1.0f;
}
template <>
__device__ __forceinline__ void load_smem<__half>(const unsigned char* spin, const float* scl, int k, int s, int Ls,
                                                  float v[24], float& sc) {
    const uint4* p = reinterpret_cast<const uint4*>(spin) + (k * 3) * Ls + s;
    sc = scl[k * Ls + s];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const uint4 t = p[c * Ls];
        float2 a = h2f(t.x), b = h2f(t.y), cc = h2f(t.z), d = h2f(t.w);
        v[8 * c] = a.x; v[8 * c + 1] = a.y; v[8 * c + 2] = b.x; v[8 * c + 3] = b.y;
        v[8 * c + 4] = cc.x; v[8 * c + 5] = cc.y; v[8 * c + 6] = d.x; v[8 * c + 7] = d.y;
    }
}
template <>
__device__ __forceinline__ void load_smem<double>(const unsigned char* spin, const float*, int k, int s, int Ls,
                                                  double v[24], double& sc) {
    const double2* p = reinterpret_cast<const double2*>(spin) + (k * 12) * Ls + s;
#pragma unroll
    for (int c = 0; c < 12; ++c) {
        const double2 t = p[c * Ls];
        v[2 * c] = t.x; v[2 * c + 1] = t.y;
    }
    sc = 1.0;
}

template <typename S, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void leg3(const unsigned char* spin, const float* scl, int k, int s, int Ls,
                                     const typename Store<S>::real* __restrict__ Us, typename Store<S>::real acc[24]) {
    typedef typename Store<S>::real T;
    T v[24], sc;
    load_smem<S>(spin, scl, k, s, Ls, v, sc);
    leg_core<T, MU, FWD, DAG>(v, sc, Us, acc);
}

__device__ __forceinline__ int wrapc(int c, int L) { return c < 0 ? c + L : (c >= L ? c - L : c); }

template <typename S, int R, bool DAG, bool FUSED>
__global__ void __launch_bounds__(256, (sizeof(S) == 8 ? 1 : sizeof(S) == 4 ? MDWF_TILE_MINB32 : MDWF_TILE_MINB16))
hop_tile_kernel(const Geom g, const HopArgs a) {
    typedef typename Store<S>::real T;
    typedef Pack16<T> P;
    constexpr int NV = Store<S>::NV;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int Ls = g.Ls, nsite = g.q4nsite, nslot = g.q4nslot;
    unsigned char* spin = smem_raw;
    size_t off = (size_t)nslot * NV * Ls * 16;
    float* scl = reinterpret_cast<float*>(smem_raw + off);
    if (Store<S>::HALF) off += (((size_t)nslot * Ls * 4) + 15) & ~(size_t)15;
    T* links = reinterpret_cast<T*>(smem_raw + off);
    off += (size_t)nsite * MDWF_LSITE * sizeof(T);
    int* slotXh = reinterpret_cast<int*>(smem_raw + off);
    int* outXh = slotXh + nslot;
    const int slot_r = blockIdx.x % a.nact;
    const int tile = blockIdx.x / a.nact;
    const int rhs = a.rhs_list[slot_r];
    // tile origin (full-lattice coordinates) and parity pattern
    uint32_t q, r, tX, tY, tZ, tT;
    g.q4dTx.divmod((uint32_t)tile, q, tX);
    g.q4dTy.divmod(q, r, tY);
    g.q4dTzs.divmod(r, q, tZ);
    g.q4dTt.divmod(q, r, tT);                    // r = z-slab index
    const int ox = tX * g.q4L[0], oy = tY * g.q4L[1], oz = r * g.zc + tZ * g.q4L[2], ot = tT * g.q4L[3];
    const int pat = (ox + oy + oz + ot + a.par) & 1;
    // ---- phase A: index tables and links ----------------------------------------------------------------
    for (int k = threadIdx.x; k < nslot; k += blockDim.x) {
        const int pk = __ldg(g.q4slot[pat] + k);
        const int x = wrapc(ox + (pk & 255) - 1, g.X), y = wrapc(oy + ((pk >> 8) & 255) - 1, g.Y);
        const int z = wrapc(oz + ((pk >> 16) & 255) - 1, g.Z), t = wrapc(ot + ((pk >> 24) & 255) - 1, g.T);
        slotXh[k] = (x >> 1) + g.XH * (y + g.Y * (z + g.Z * t));
    }
    for (int task = threadIdx.x; task < nsite * 8; task += blockDim.x) {
        const int i = task >> 3, l = task & 7;
        const int pk = __ldg(g.q4out[pat] + i);
        SiteCoord c;
        const int x = ox + (pk & 255);
        c.y = oy + ((pk >> 8) & 255); c.z = oz + ((pk >> 16) & 255); c.t = ot + ((pk >> 24) & 255);
        c.xx = x >> 1; c.o = x & 1;
        c.xh = c.xx + g.XH * (c.y + g.Y * (c.z + g.Z * c.t));
        T V[MDWF_LROW];
        stage_link<S, R>(g, a.g, a.par, c, l, V);
        P* dst = reinterpret_cast<P*>(links + i * MDWF_LSITE + l * MDWF_LROW);
#pragma unroll
        for (int qq = 0; qq < MDWF_LROW / P::N; ++qq) {
            P t;
#pragma unroll
            for (int e = 0; e < P::N; ++e) t.d[e] = V[qq * P::N + e];
            dst[qq] = t;
        }
        if (l == 0) outXh[i] = c.xh;
    }
    __syncthreads();
    // ---- phase B: copy the box's input sites (all s) into shared memory ------------------------------------
    for (int task = threadIdx.x; task < nslot * Ls; task += blockDim.x) {
        const int k = (int)g.dLs.div((uint32_t)task), s = task - k * Ls;
        const int idx = slotXh[k] * Ls + s;
        const char* src = site_ptr<S>(a.in, rhs, idx);
        unsigned char* dst = spin + ((size_t)(k * NV) * Ls + s) * 16;
#pragma unroll
        for (int c = 0; c < NV; ++c) __pipeline_memcpy_async(dst + (size_t)c * Ls * 16, src + c * 512, 16);
        if (Store<S>::HALF) __pipeline_memcpy_async(scl + task, src - (idx & 31) * 12 + 3 * 512, 4);
    }
    __pipeline_commit();
    __pipeline_wait_prior(0);
    __syncthreads();
    // ---- phase C: the stencil from shared memory -----------------------------------------------------------
    const int grp = (int)g.dLs.div(threadIdx.x), s = threadIdx.x - grp * Ls;
    const bool live = grp < nsite;
    T acc[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0;
    int idx = 0;
    if (live) {
        const uint2 nb = __ldg(reinterpret_cast<const uint2*>(g.q4nbr[pat]) + grp);
        idx = outXh[grp] * Ls + s;
        const T* Ub = links + grp * MDWF_LSITE;
        leg3<S, 0, true, DAG>(spin, scl, nb.x & 255, s, Ls, Ub + 0 * MDWF_LROW, acc);
        leg3<S, 0, false, DAG>(spin, scl, (nb.x >> 8) & 255, s, Ls, Ub + 1 * MDWF_LROW, acc);
        leg3<S, 1, true, DAG>(spin, scl, (nb.x >> 16) & 255, s, Ls, Ub + 2 * MDWF_LROW, acc);
        leg3<S, 1, false, DAG>(spin, scl, (nb.x >> 24) & 255, s, Ls, Ub + 3 * MDWF_LROW, acc);
        leg3<S, 2, true, DAG>(spin, scl, nb.y & 255, s, Ls, Ub + 4 * MDWF_LROW, acc);
        leg3<S, 2, false, DAG>(spin, scl, (nb.y >> 8) & 255, s, Ls, Ub + 5 * MDWF_LROW, acc);
        leg3<S, 3, true, DAG>(spin, scl, (nb.y >> 16) & 255, s, Ls, Ub + 6 * MDWF_LROW, acc);
        leg3<S, 3, false, DAG>(spin, scl, (nb.y >> 24) & 255, s, Ls, Ub + 7 * MDWF_LROW, acc);
    }
    if (!FUSED) {
        if (live) store_spinor<S, MDWF_HOP_STCS>(a.out, rhs, idx, g.N5h, acc);
        return;
    }
    // ---- fused epilogue (the staged spinors are dead: their shared memory is reused) ------------------------
    __syncthreads();
    unsigned char* smem_epi = smem_raw;
    fused_epilogue<S>(g, a, acc, live, rhs, idx, slot_r, tile, smem_epi);
}

}  // namespace mdwf
