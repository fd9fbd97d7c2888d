// csrc/mdwf_blas.cuh -- 4D-site-local kernels: the Ls-direction operators (A = "M4pre", M5, M5^-1 and
// their products are one Ls x Ls real matrix per chirality, SURVEY 8 Notation), the fused BLAS-1 of the
// CG iteration with fp64 fixed-order reductions ("all reductions are done in double precision",
// PAPER.md:183), precision conversion and canonical<->packed packing.
// One thread per 5D site (s fastest), one rhs per block, blockIdx.x = tile*nact + slot.
#pragma once
#include "mdwf_hop.cuh"

namespace mdwf {

// The rhs a launch works on.  Plain mode (ril == 0): one rhs per block, blockIdx.x = tile*nact + slot.  Grouped mode
// (launches whose fields are fp16: the rhs are interleaved in groups of 1 << ril inside a 4D site, mdwf_device.cuh):
// blockIdx.x = tile*ng + group, and consecutive threads walk the (rhs in group, s) rows of consecutive 4D sites, i.e.
// consecutive 16-byte pieces of memory; the Ls threads of one (site, rhs) are still consecutive.
struct RhsList {
    int nact;
    int rhs[64];
    int ril, ng;
    unsigned char grp[64], gmask[64], slot_of[64];
};
struct RowWork {
    int rhs, idx, slot, tile, nblk, ri, grp;
    bool live;
};
__device__ __forceinline__ RowWork map_work(const Geom& g, const RhsList& rl) {
    RowWork w;
    if (rl.ril == 0 && rl.ng == 0) {
        w.slot = blockIdx.x % rl.nact; w.tile = blockIdx.x / rl.nact; w.rhs = rl.rhs[w.slot];
        w.idx = w.tile * blockDim.x + threadIdx.x; w.live = w.idx < g.N5h; w.nblk = gridDim.x / rl.nact; w.ri = 0; w.grp = w.rhs;
    } else {
        const int gi = blockIdx.x % rl.ng;
        w.tile = blockIdx.x / rl.ng; w.nblk = gridDim.x / rl.ng; w.grp = rl.grp[gi];
        const uint32_t v = (uint32_t)w.tile * blockDim.x + threadIdx.x;
        const uint32_t q = g.dLs.div(v);                 // = xh * RI + ri
        const int xh = (int)(q >> rl.ril);
        w.ri = (int)(q & ((1u << rl.ril) - 1u));
        w.rhs = (w.grp << rl.ril) + w.ri;
        w.idx = xh * g.Ls + (int)(v - q * g.Ls);
        w.live = xh < g.Vh && ((rl.gmask[gi] >> w.ri) & 1);
        w.slot = rl.slot_of[w.rhs & 63];
    }
    return w;
}
// fixed-order block sums per rhs of the block: plain mode one sum, grouped mode one per active rhs of the group
__device__ __forceinline__ void block_sum_rhs(double v, const RowWork& w, const RhsList& rl, unsigned char* smem_raw, double* partial, int g_Ls) {
    if (rl.ril == 0 && rl.ng == 0) {
        block_sum_store(v, smem_raw, partial + (long long)w.slot * w.nblk + w.tile);
        return;
    }
    // grouped mode: one pass through shared memory, then thread j < RI sums the entries of rhs j in thread order (the
    // Ls threads of a (site, rhs) are consecutive and the rhs of a site follow each other, so thread t belongs to rhs
    // (first + t / Ls) mod RI): two barriers instead of 4 RI
    // (no barrier before the first write: every earlier user of smem_raw in these kernels ends with one -- apply_ls -- or
    // there is none; and none after the sums: the callers either end here or synchronise themselves)
    double* red = reinterpret_cast<double*>(smem_raw);
    red[threadIdx.x] = w.live ? v : 0.0;
    __syncthreads();
    const int RI = 1 << rl.ril;
    if ((int)threadIdx.x < RI) {
        const int gm = rl.gmask[blockIdx.x % rl.ng], j = threadIdx.x;
        if ((gm >> j) & 1) {
            const int Ls = (int)g_Ls, ngrp = (int)blockDim.x / Ls;          // (site, rhs) groups of Ls threads in the block
            const int first = (int)(((unsigned)w.tile * blockDim.x / (unsigned)Ls) & (unsigned)(RI - 1));   // rhs-in-group of thread 0
            double tot = 0.0;
            for (int q = (j - first) & (RI - 1); q < ngrp; q += RI)
                for (int t = q * Ls; t < q * Ls + Ls; ++t) tot += red[t];
            partial[(long long)rl.slot_of[((w.grp << rl.ril) + j) & 63] * w.nblk + w.tile] = tot;
        }
    }
}
// 1 / scale of an fp16 output for this thread's rhs (see block_out_scale); grouped mode evaluates the rule once per rhs
// of the group
// (SLOT: a kernel that evaluates two rules uses a different slot for each, so that no barrier is needed before the write)
template <typename S, int SLOT = 0>
__device__ __forceinline__ typename Store<S>::real work_out_scale(const ScaleRule& sr, const RowWork& w, const RhsList& rl) {
    if constexpr (!Store<S>::HALF) return 1;
    else {
        if (rl.ril == 0 && rl.ng == 0) return block_out_scale<S>(sr, w.rhs, w.tile == 0);
        __shared__ float s_oinv4[4];
        if (threadIdx.x < (1u << rl.ril)) {
            const int gm = rl.gmask[blockIdx.x % rl.ng];
            s_oinv4[threadIdx.x] = (gm >> threadIdx.x) & 1 ? 1.0f / eval_scale(sr, (w.grp << rl.ril) + (int)threadIdx.x, w.tile == 0) : 1.0f;
        }
        __syncthreads();
        return s_oinv4[w.ri];
    }
}

// out = cx*xin + ch * G in   (G == nullptr: identity), optional sum |out|^2, optional no store
struct LsArgs {
    SpinorView out, in, xin;
    LsOp op;
    double cx, ch;
    double* partial;
    int write;
    RhsList rl;
    ScaleRule sr;       // fp16 output only
    const int* stop;    // optional: non-zero -> no-op (see HopArgs)
};
template <typename S>
__global__ void __launch_bounds__(256) ls_kernel(const Geom g, const LsArgs a) {
    typedef typename Store<S>::real T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (a.stop != nullptr && *a.stop != 0) return;
    const RowWork w = map_work(g, a.rl);
    const int rhs = w.rhs, idx = w.idx;
    const bool live = w.live;
    T acc[24];
    if (live) load_spinor<S>(a.in, rhs, idx, g.N5h, acc);
    else {
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = 0;
    }
    if (a.op.kind != 0) apply_ls<T>(acc, a.op, g.Ls, smem_raw);
    const T ch = (T)a.ch, cx = (T)a.cx;
    if (a.xin.v != nullptr && live) {
        T xv[24];
        load_spinor<S>(a.xin, rhs, idx, g.N5h, xv);
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = cx * xv[i] + ch * acc[i];
    } else {
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] *= ch;
    }
    if (a.write) {
        const T oinv = work_out_scale<S>(a.sr, w, a.rl);
        if (live) store_spinor<S>(a.out, rhs, idx, g.N5h, acc, oinv);
    }
    if (a.partial != nullptr) {
        double s2 = 0.0;
        if (live) {
#pragma unroll
            for (int i = 0; i < 24; ++i) s2 += (double)acc[i] * (double)acc[i];
        }
        block_sum_rhs(s2, w, a.rl, smem_raw, a.partial, g.Ls);
    }
}

// out = ca*a + cb*b with independent storage types (conversion, x_hi += x_lo, r = bhat - y, ...);
// a or b may be absent (v == nullptr); optional sum |out|^2.
struct AxpbyArgs {
    SpinorView out, a, b;
    double ca, cb;
    double* partial;
    RhsList rl;
    ScaleRule sr;       // fp16 output only
};
template <typename SO, typename SA, typename SB>
__global__ void __launch_bounds__(256) axpby_kernel(const Geom g, const AxpbyArgs p) {
    typedef typename Store<SO>::real TO;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const RowWork w = map_work(g, p.rl);
    const int rhs = w.rhs, idx = w.idx;
    const bool live = w.live;
    double s2 = 0.0;
    const TO oinv = work_out_scale<SO>(p.sr, w, p.rl);
    if (live) {
        double o[24];
#pragma unroll
        for (int i = 0; i < 24; ++i) o[i] = 0.0;
        if (p.a.v != nullptr) {
            typename Store<SA>::real v[24];
            load_spinor<SA>(p.a, rhs, idx, g.N5h, v);
#pragma unroll
            for (int i = 0; i < 24; ++i) o[i] = p.ca * (double)v[i];
        }
        if (p.b.v != nullptr) {
            typename Store<SB>::real v[24];
            load_spinor<SB>(p.b, rhs, idx, g.N5h, v);
#pragma unroll
            for (int i = 0; i < 24; ++i) o[i] += p.cb * (double)v[i];
        }
        TO w[24];
#pragma unroll
        for (int i = 0; i < 24; ++i) {
            w[i] = (TO)o[i];
            s2 += o[i] * o[i];
        }
        store_spinor<SO>(p.out, rhs, idx, g.N5h, w, oinv);
    }
    if (p.partial != nullptr) block_sum_rhs(s2, w, p.rl, smem_raw, p.partial, g.Ls);
}

// CG step, part 1:  alpha = rr/pAp ;  x += alpha p ;  r -= alpha Ap ;  partial |r|^2
struct CgXrArgs {
    SpinorView x, r, p, Ap;
    const double* rr;     // [64] by rhs id
    const double* pAp;    // [64]
    double* partial;
    RhsList rl;
    ScaleRule sr;         // fp16 r only: scale of the updated r
    const int* stop;      // optional: non-zero -> no-op
};
template <typename SX, typename S>
__global__ void __launch_bounds__(256) cg_update_xr_kernel(const Geom g, const CgXrArgs a) {
    typedef typename Store<S>::real T;
    typedef typename Store<SX>::real TX;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (a.stop != nullptr && *a.stop != 0) return;
    const RowWork w = map_work(g, a.rl);
    const int rhs = w.rhs, idx = w.idx;
    const bool live = w.live;
    double s2 = 0.0;
    const T oinv = work_out_scale<S>(a.sr, w, a.rl);
    if (live) {
        const double alpha_d = a.rr[rhs] / a.pAp[rhs];
        T pv[24], rv[24], av[24];
        TX xv[24];
        load_spinor<S>(a.p, rhs, idx, g.N5h, pv);
        load_spinor<S>(a.Ap, rhs, idx, g.N5h, av);
        load_spinor<S>(a.r, rhs, idx, g.N5h, rv);
        load_spinor<SX>(a.x, rhs, idx, g.N5h, xv);
        const T al = (T)alpha_d;
        const TX alx = (TX)alpha_d;
#pragma unroll
        for (int i = 0; i < 24; ++i) {
            xv[i] += alx * (TX)pv[i];
            rv[i] -= al * av[i];
            s2 += (double)rv[i] * (double)rv[i];
        }
        store_spinor<SX>(a.x, rhs, idx, g.N5h, xv);
        store_spinor<S>(a.r, rhs, idx, g.N5h, rv, oinv);
    }
    block_sum_rhs(s2, w, a.rl, smem_raw, a.partial, g.Ls);
}

// CG step, part 2:  beta = rr_new/rr_old ;  p = r + beta p ;  optionally also q = G p (G = A or M5^-dag:
// the leading s-direction factor of the next operator application, fused to save one pass)
struct CgPArgs {
    SpinorView p, r, q;
    LsOp op;
    const double* rr_new;
    const double* rr_old;
    double* partial;      // optional |p_new|^2 partials (fp16: refreshes p's norm bound)
    RhsList rl;
    ScaleRule sr_p, sr_q; // fp16 only: scales of the updated p and of q
    const int* stop;      // optional: non-zero -> no-op
};
template <typename S>
__global__ void __launch_bounds__(256) cg_update_p_kernel(const Geom g, const CgPArgs a) {
    typedef typename Store<S>::real T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (a.stop != nullptr && *a.stop != 0) return;
    const RowWork w = map_work(g, a.rl);
    const int rhs = w.rhs, idx = w.idx;
    const bool live = w.live;
    T pv[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) pv[i] = 0;
    const T oinv_p = work_out_scale<S>(a.sr_p, w, a.rl);
    if (live) {
        const T beta = (T)(a.rr_new[rhs] / a.rr_old[rhs]);
        T rv[24];
        load_spinor<S>(a.p, rhs, idx, g.N5h, pv);
        load_spinor<S>(a.r, rhs, idx, g.N5h, rv);
#pragma unroll
        for (int i = 0; i < 24; ++i) pv[i] = rv[i] + beta * pv[i];
        store_spinor<S>(a.p, rhs, idx, g.N5h, pv, oinv_p);
    }
    if (a.partial != nullptr) {
        double s2 = 0.0;
#pragma unroll
        for (int i = 0; i < 24; ++i) s2 += (double)pv[i] * (double)pv[i];
        block_sum_rhs(s2, w, a.rl, smem_raw, a.partial, g.Ls);
        __syncthreads();
    }
    if (a.op.kind != 0) {
        apply_ls<T>(pv, a.op, g.Ls, smem_raw);
        const T oinv_q = work_out_scale<S, 1>(a.sr_q, w, a.rl);
        if (live) store_spinor<S>(a.q, rhs, idx, g.N5h, pv, oinv_q);
    }
}

// out[rhs] = sum_b partial[slot][b] in a fixed order; optionally mirrored to (mapped) host memory.
// With `ctl` the kernel is the loop control of the inner CG (solver.cu): after |r|^2 of every active rhs is known it
// decides ON THE DEVICE whether the inner loop must be left (reliable update due, target reached, breakdown, iteration
// cap) and raises ctl->stop, which turns every kernel queued behind it into a no-op; the host, which runs a few
// iterations ahead, only polls the pinned mirror.  Iteration counts are therefore exactly those of a loop that
// synchronises after every iteration.
struct CgCtl {
    int stop;            // device flag read by the gated kernels
    int done_blocks;     // blocks of the current finish launch that are through
    int iters;           // iterations completed since the flag was cleared
    int iter_cap;        // leave the loop when iters reaches this
    double delta;
    double stop_nr[64], maxr[64];
};
struct CgCtlHost {       // pinned mirror, written by the last block of every loop-control launch
    volatile int seq;    // sequence number of the last loop-control launch that ran (also when it was a no-op)
    volatile int stop;
    volatile int iters;
};
struct FinishArgs {
    const double* partial;
    int nblk;
    double* out;        // [64] by rhs id
    double* out2;       // optional second destination (e.g. host-mapped), may be nullptr
    double* nb;         // optional: norm bound of the fp16 field that was just measured, nb[rhs] = sqrt(sum) (1 + 2^-9)
    RhsList rl;
    const int* stop;    // optional: non-zero -> no-op
    CgCtl* ctl;         // optional: loop control (this launch finishes |r|^2)
    CgCtlHost* hctl;
    const double* pap;  // loop control: <p, A p> of the iteration (breakdown check)
    int seq;
};
static __global__ void __launch_bounds__(1024) finish_sum_kernel(const FinishArgs a) {
    __shared__ double red[1024];
    const int slot = blockIdx.x, rhs = a.rl.rhs[slot];
    const bool skip = a.stop != nullptr && *a.stop != 0;
    bool want_stop = false;
    if (!skip) {
        const double* p = a.partial + (long long)slot * a.nblk;
        double s = 0.0;
        for (int i = threadIdx.x; i < a.nblk; i += 1024) s += p[i];
        red[threadIdx.x] = s;
        __syncthreads();
        for (int o = 512; o > 0; o >>= 1) {
            if ((int)threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            a.out[rhs] = red[0];
            if (a.out2) a.out2[rhs] = red[0];
            if (a.nb) a.nb[rhs] = sqrt(red[0]) * 1.001953125;
            if (a.ctl) {
                const double rn = sqrt(red[0]), pap = a.pap[rhs];
                want_stop = !(rn == rn) || !(pap > 0.0) || rn <= a.ctl->stop_nr[rhs] || rn < a.ctl->delta * a.ctl->maxr[rhs] ||
                            a.ctl->iters + 1 >= a.ctl->iter_cap;
                if (rn > a.ctl->maxr[rhs]) a.ctl->maxr[rhs] = rn;
            }
        }
    }
    if (a.ctl && threadIdx.x == 0) {
        if (want_stop) atomicExch(&a.ctl->stop, 1);
        __threadfence();
        if (atomicAdd(&a.ctl->done_blocks, 1) == (int)gridDim.x - 1) {      // last block of this launch
            a.ctl->done_blocks = 0;
            if (!skip) a.ctl->iters += 1;
            __threadfence();
            a.hctl->iters = a.ctl->iters;
            a.hctl->stop = *(volatile int*)&a.ctl->stop;
            __threadfence_system();
            a.hctl->seq = a.seq;
        }
    }
}

// canonical fp64 <-> packed.  Canonical site index: half-lattice (full == 0): xh; full lattice: x4 = 2*xh + o.
struct PackArgs {
    SpinorView f;
    double* canon;          // [rhs][s][Vc][24]
    long long Vc;           // Vh or V4
    int full, par, nrhs;
    int rhs0;               // packed rhs index = rhs0 + r for canonical rhs r
    int s0, ns;             // ns > 0: `canon` holds only the s-slices [s0, s0 + ns) of each rhs, [rhs][ns][Vc][24]
    double* partial;        // NORM pass only: [nrhs][gridDim.x] sums of squares of the canonical data
    ScaleRule sr;           // fp16 pack only
};
__device__ __forceinline__ long long canon_site(const Geom& g, int full, int par, int xh) {
    if (!full) return xh;
    uint32_t row, xx, r2, y, t, z;
    g.dXH.divmod((uint32_t)xh, row, xx);
    g.dY.divmod(row, r2, y);
    g.dZ.divmod(r2, t, z);
    const int o = (par + y + z + t) & 1;
    return 2ll * xh + o;
}
// fp16 packing needs |field|_2 before it can choose the scale: first pass over the canonical data
static __global__ void __launch_bounds__(256) pack_norm_kernel(const Geom g, const PackArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int rhs = blockIdx.y;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    double s2 = 0.0;
    if (idx < g.N5h) {
        uint32_t xh, s;
        g.dLs.divmod((uint32_t)idx, xh, s);
        const long long xs = canon_site(g, a.full, a.par, (int)xh);
        const double* c = a.canon + (((long long)rhs * g.Ls + s) * a.Vc + xs) * 24;
#pragma unroll
        for (int i = 0; i < 12; ++i) {
            const double2 t = reinterpret_cast<const double2*>(c)[i];
            s2 += t.x * t.x + t.y * t.y;
        }
    }
    block_sum_store(s2, smem_raw, a.partial + (long long)rhs * gridDim.x + blockIdx.x);
}
template <typename S, bool UNPACK>
__global__ void __launch_bounds__(256) pack_kernel(const Geom g, const PackArgs a) {
    typedef typename Store<S>::real T;
    const int rhs = blockIdx.y;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    T oinv = 1;
    if (!UNPACK) oinv = block_out_scale<S>(a.sr, a.rhs0 + rhs, blockIdx.x == 0);
    if (idx >= g.N5h) return;
    uint32_t xh, s;
    g.dLs.divmod((uint32_t)idx, xh, s);
    if (a.ns > 0 && ((int)s < a.s0 || (int)s >= a.s0 + a.ns)) return;
    const long long xs = canon_site(g, a.full, a.par, (int)xh);
    double* c = a.canon + ((a.ns > 0 ? (long long)rhs * a.ns + ((int)s - a.s0) : (long long)rhs * g.Ls + s) * a.Vc + xs) * 24;
    T v[24];
    if (UNPACK) {
        load_spinor<S>(a.f, a.rhs0 + rhs, idx, g.N5h, v);
#pragma unroll
        for (int i = 0; i < 12; ++i) reinterpret_cast<double2*>(c)[i] = make_double2((double)v[2 * i], (double)v[2 * i + 1]);
    } else {
#pragma unroll
        for (int i = 0; i < 12; ++i) {
            const double2 t = reinterpret_cast<const double2*>(c)[i];
            v[2 * i] = (T)t.x;
            v[2 * i + 1] = (T)t.y;
        }
        store_spinor<S>(a.f, a.rhs0 + rhs, idx, g.N5h, v, oinv);
    }
}

}  // namespace mdwf
