// csrc/mdwf_hop.cuh -- the even-odd MDWF Dslash stencil kernel ("red-black preconditioned Domain-wall
// stencil") with its fused Ls-direction epilogue.
//
//   out(x,s) = cx * xin(x,s) + ch * sum_{s'} G_chi[s][s'] * (H_{p<-pbar} in)(x,s')       (FUSED)
//   out(x,s) = (H_{p<-pbar} in)(x,s)                                                     (PLAIN)
//   (H psi)(x) = sum_mu [ (1 - g_mu) U_mu(x) psi(x+mu) + (1 + g_mu) U_mu(x-mu)^dag psi(x-mu) ]   (SURVEY 8
//   Notation; dagger swaps the projector signs; a hop across the mu boundary is multiplied by bc_mu).
// G_chi is an Ls x Ls real matrix per chirality (A M5^-1, M5^-1, A^dag, M5^-dag A^dag ...: every
// s-direction factor of the Schur operators is such a matrix, so "kernel fusion to minimize memory
// traffic", turns Mhat into two of these launches).  gamma matrices: DeGrand-Rossi chiral
// basis written out below from SURVEY 8 Notation (gamma5 = diag(1,1,-1,-1): P+ = spins 0,1).
//
// One thread per 5D site (s fastest), one rhs per block; blocks run chunk-major (z-slab x timeslice of tiles), then
// rhs, then tile, so the rhs sharing a chunk's links run back to back; sites are traversed in z-slabs so that
// t-neighbours are re-read from L2, not HBM.  The block's links are reconstructed once into shared
// memory and read from there by all Ls threads of a site.
#pragma once
#include "mdwf_device.cuh"

namespace mdwf {

// (1 + SGN*gamma_MU) psi -> upper two rows h[12]; lower rows follow by the relations in recon()
template <int MU, int SGN, typename T>
__device__ __forceinline__ void project(const T v[24], T h[12]) {
#define VR(a, c) v[((a) * 3 + (c)) * 2]
#define VI(a, c) v[((a) * 3 + (c)) * 2 + 1]
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        T r0r, r0i, r1r, r1i;
        if (MU == 0) {        // r0 = psi0 + s*i*psi3 ; r1 = psi1 + s*i*psi2
            r0r = VR(0, c) - SGN * VI(3, c); r0i = VI(0, c) + SGN * VR(3, c);
            r1r = VR(1, c) - SGN * VI(2, c); r1i = VI(1, c) + SGN * VR(2, c);
        } else if (MU == 1) { // r0 = psi0 - s*psi3 ; r1 = psi1 + s*psi2
            r0r = VR(0, c) - SGN * VR(3, c); r0i = VI(0, c) - SGN * VI(3, c);
            r1r = VR(1, c) + SGN * VR(2, c); r1i = VI(1, c) + SGN * VI(2, c);
        } else if (MU == 2) { // r0 = psi0 + s*i*psi2 ; r1 = psi1 - s*i*psi3
            r0r = VR(0, c) - SGN * VI(2, c); r0i = VI(0, c) + SGN * VR(2, c);
            r1r = VR(1, c) + SGN * VI(3, c); r1i = VI(1, c) - SGN * VR(3, c);
        } else {              // r0 = psi0 + s*psi2 ; r1 = psi1 + s*psi3
            r0r = VR(0, c) + SGN * VR(2, c); r0i = VI(0, c) + SGN * VI(2, c);
            r1r = VR(1, c) + SGN * VR(3, c); r1i = VI(1, c) + SGN * VI(3, c);
        }
        h[c * 2] = r0r; h[c * 2 + 1] = r0i;
        h[6 + c * 2] = r1r; h[6 + c * 2 + 1] = r1i;
    }
#undef VR
#undef VI
}

// acc += cf * (full spinor rebuilt from the half spinor w):  rows 2,3 from rows 0,1:
//  MU0: r2 = -s*i*r1, r3 = -s*i*r0 ; MU1: r2 = s*r1, r3 = -s*r0 ; MU2: r2 = -s*i*r0, r3 = s*i*r1 ; MU3: r2 = s*r0, r3 = s*r1
template <int MU, int SGN, typename T>
__device__ __forceinline__ void recon(const T w[12], T cf, T acc[24]) {
    const T cs = cf * (T)SGN;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T w0r = w[c * 2], w0i = w[c * 2 + 1], w1r = w[6 + c * 2], w1i = w[6 + c * 2 + 1];
        acc[(0 * 3 + c) * 2] += cf * w0r; acc[(0 * 3 + c) * 2 + 1] += cf * w0i;
        acc[(1 * 3 + c) * 2] += cf * w1r; acc[(1 * 3 + c) * 2 + 1] += cf * w1i;
        if (MU == 0) {        // r2 = -s*i*r1 = s*(w1i, -w1r) ; r3 = s*(w0i, -w0r)
            acc[(2 * 3 + c) * 2] += cs * w1i; acc[(2 * 3 + c) * 2 + 1] -= cs * w1r;
            acc[(3 * 3 + c) * 2] += cs * w0i; acc[(3 * 3 + c) * 2 + 1] -= cs * w0r;
        } else if (MU == 1) { // r2 = s*r1 ; r3 = -s*r0
            acc[(2 * 3 + c) * 2] += cs * w1r; acc[(2 * 3 + c) * 2 + 1] += cs * w1i;
            acc[(3 * 3 + c) * 2] -= cs * w0r; acc[(3 * 3 + c) * 2 + 1] -= cs * w0i;
        } else if (MU == 2) { // r2 = -s*i*r0 = s*(w0i, -w0r) ; r3 = s*i*r1 = s*(-w1i, w1r)
            acc[(2 * 3 + c) * 2] += cs * w0i; acc[(2 * 3 + c) * 2 + 1] -= cs * w0r;
            acc[(3 * 3 + c) * 2] -= cs * w1i; acc[(3 * 3 + c) * 2 + 1] += cs * w1r;
        } else {              // r2 = s*r0 ; r3 = s*r1
            acc[(2 * 3 + c) * 2] += cs * w0r; acc[(2 * 3 + c) * 2 + 1] += cs * w0i;
            acc[(3 * 3 + c) * 2] += cs * w1r; acc[(3 * 3 + c) * 2 + 1] += cs * w1i;
        }
    }
}

// w = U h (ADJ = false) or U^dag h (ADJ = true) for the two spin rows of a half spinor
template <bool ADJ, typename T>
__device__ __forceinline__ void su3_mul(const T U[18], const T h[12], T w[12]) {
#pragma unroll
    for (int k = 0; k < 2; ++k)
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            T re, im;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const T ur = ADJ ? U[(j * 3 + i) * 2] : U[(i * 3 + j) * 2];
                const T ui = ADJ ? -U[(j * 3 + i) * 2 + 1] : U[(i * 3 + j) * 2 + 1];
                const T hr = h[k * 6 + j * 2], hi = h[k * 6 + j * 2 + 1];
                if (j == 0) { re = ur * hr; im = ur * hi; }
                else { re = fma_<T>(ur, hr, re); im = fma_<T>(ur, hi, im); }
                re = fma_<T>(-ui, hi, re);
                im = fma_<T>(ui, hr, im);
            }
            w[k * 6 + i * 2] = re;
            w[k * 6 + i * 2 + 1] = im;
        }
}

template <typename T> struct alignas(16) Pack16 {
    static constexpr int N = 16 / sizeof(T);
    T d[N];
};

// s-direction operator of a fused epilogue / site-local kernel (SURVEY 8 Notation):
//   kind 1:  out = c0 v + c1 L v      (A = b5 + c5 L, M5 = a + d L;  dag: L -> L^dag)
//   kind 2:  out = c0 v + c1 M5^-1 v  (M5^-1, and A M5^-1 = c5/d + (b5 - c5 a/d) M5^-1;  dag: M5^-dag)
// with (L v)_s = P- v_{s+1} + P+ v_{s-1}, wraps multiplied by -mf, and M5^-1 through its closed form as a
// first-order recurrence: for the "forward" chirality  P_s = v_s + kappa P_{s-1},  T = P_{Ls-1},
//   (M5^-1 v)_s = P_s / a - gfac kappa^{s+1} T,   gfac = mf / (a (1 + mf kappa^Ls)),  kappa = -d/a,
// and mirrored in s for the other chirality (P+ is forward for M5^-1, P- for M5^-dag).  O(Ls) work per site
// instead of the O(Ls^2) of a dense Ls x Ls multiply.
struct LsOp {
    int kind, dag;
    double c0, c1, kappa, inv_a, gfac, mf;
};
// shared memory: Ls reals (kappa powers) rounded up, then one 28-real row per thread (+4 per site group)
template <typename T> __host__ __device__ inline int smem_reals_G(int Ls, int nthreads) {
    return ((Ls + 3) & ~3) + (nthreads / Ls) * (Ls * 28 + 4);
}
// Every thread of the block must call it (block-wide barriers); blockDim.x is a multiple of Ls; the Ls threads of
// a (site, rhs) group are consecutive.
template <typename T>
__device__ __forceinline__ void apply_ls(T acc[24], const LsOp& op, int Ls, unsigned char* smem_raw) {
    typedef Pack16<T> P;
    constexpr int NP = 24 / P::N;
    T* kp = reinterpret_cast<T*>(smem_raw);
    T* buf = kp + ((Ls + 3) & ~3);
    const int grp = threadIdx.x / Ls, sl = threadIdx.x - grp * Ls;
    const int gstride = Ls * 28 + 4;   // 28-real rows (+4 per group): conflict-free 16-byte accesses
    T* grow = buf + grp * gstride;
    P* mine = reinterpret_cast<P*>(grow + sl * 28);
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        P t;
#pragma unroll
        for (int e = 0; e < P::N; ++e) t.d[e] = acc[q * P::N + e];
        mine[q] = t;
    }
    if (op.kind == 2 && (int)threadIdx.x < Ls) {
        T v = (T)op.kappa;
        for (int i = 0; i < (int)threadIdx.x; ++i) v *= (T)op.kappa;
        kp[threadIdx.x] = v;            // kappa^{k+1}
    }
    __syncthreads();
    const T c0 = (T)op.c0, c1 = (T)op.c1;
    if (op.kind == 1) {
        const int sm = sl == 0 ? Ls - 1 : sl - 1, sp = sl == Ls - 1 ? 0 : sl + 1;
        const T fm = c1 * (sl == 0 ? (T)(-op.mf) : (T)1), fp = c1 * (sl == Ls - 1 ? (T)(-op.mf) : (T)1);
        const P* up = reinterpret_cast<const P*>(grow + (op.dag ? sp : sm) * 28);   // source row of the P+ components
        const P* lo = reinterpret_cast<const P*>(grow + (op.dag ? sm : sp) * 28);   // source row of the P- components
        const T fu = op.dag ? fp : fm, fl = op.dag ? fm : fp;
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            const bool plus = q * P::N < 12;
            const P t = plus ? up[q] : lo[q];
#pragma unroll
            for (int e = 0; e < P::N; ++e) acc[q * P::N + e] = c0 * acc[q * P::N + e] + (plus ? fu : fl) * t.d[e];
        }
    } else {
        const T kap = (T)op.kappa;
        for (int col = sl; col < NP; col += Ls) {
            const bool fwd = (col * P::N < 12) != (op.dag != 0);
            P run;
#pragma unroll
            for (int e = 0; e < P::N; ++e) run.d[e] = 0;
            for (int k = 0; k < Ls; ++k) {
                P* row = reinterpret_cast<P*>(grow + (fwd ? k : Ls - 1 - k) * 28) + col;
                const P v = *row;
#pragma unroll
                for (int e = 0; e < P::N; ++e) run.d[e] = v.d[e] + kap * run.d[e];
                *row = run;
            }
        }
        __syncthreads();
        const T ia = c1 * (T)op.inv_a;
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            const bool fwd = (q * P::N < 12) != (op.dag != 0);
            const P ps = mine[q];
            const P tt = reinterpret_cast<const P*>(grow + (fwd ? Ls - 1 : 0) * 28)[q];
            const T gk = -c1 * (T)op.gfac * kp[fwd ? sl : Ls - 1 - sl];
#pragma unroll
            for (int e = 0; e < P::N; ++e) acc[q * P::N + e] = c0 * acc[q * P::N + e] + ia * ps.d[e] + gk * tt.d[e];
        }
    }
    __syncthreads();
}

// fixed-order block sum (same order every run -> bit-reproducible); thread 0 stores.  Two-level: 32 strided
// partial sums, then one serial pass.  smem needed: blockDim.x doubles.  Every thread of the block must call it.
__device__ __forceinline__ void block_sum_store(double v, unsigned char* smem_raw, double* dst) {
    double* red = reinterpret_cast<double*>(smem_raw);
    __syncthreads();
    red[threadIdx.x] = v;
    __syncthreads();
    double a = 0.0;
    if (threadIdx.x < 32)
        for (int i = threadIdx.x; i < (int)blockDim.x; i += 32) a += red[i];
    __syncthreads();
    if (threadIdx.x < 32) red[threadIdx.x] = a;
    __syncthreads();
    if (threadIdx.x == 0) {
        double tot = 0.0;
        const int n = blockDim.x < 32 ? (int)blockDim.x : 32;
        for (int i = 0; i < n; ++i) tot += red[i];
        *dst = tot;
    }
}

// ---- links staged in shared memory ------------------------------------------------------------------
// Per block: for each of its 4D sites the 8 stencil links, reconstructed to 18 reals of the compute type,
// already daggered for the backward legs and multiplied by the boundary sign, plus the 8 neighbour
// half-indices and the site's own half-index.  Every thread of a site (all Ls slices) then reads the same
// link rows (broadcast) -- "staging of links reused across the Ls slices" (north_star).
//   smem link row: 20 reals (16-byte aligned); site stride 8*20+4 reals (keeps 16-byte reads of the sites
//   of one warp in different banks); index table: 12 ints per site (8 neighbours, own xh, pad).
#ifndef MDWF_HOP_STCS
#define MDWF_HOP_STCS true
#endif
#ifndef MDWF_HOP_MINB
#define MDWF_HOP_MINB 3      // fp16 storage: 80 registers, 3 blocks/SM
#endif
#ifndef MDWF_HOP_MINB32
#define MDWF_HOP_MINB32 4    // fp32: 64 registers, 4 blocks/SM (measured faster: latency-bound gathers)
#endif
#ifndef MDWF_HOP_MINB64
#define MDWF_HOP_MINB64 2    // fp64: 128 registers, 2 blocks/SM (measured: 6.6 -> 5.8 ms on 48^3x64x10)
#endif
#define MDWF_LROW 20
#define MDWF_LSITE (8 * MDWF_LROW + 4)
template <typename T> __host__ __device__ inline size_t smem_bytes_links(int nsite) {
    return (size_t)nsite * (MDWF_LSITE * sizeof(T) + 12 * sizeof(int));
}

// one stencil leg from staged data: neighbour spinor v (unscaled, scale sc), U (smem, already U or U^dag, bc sign
// folded): acc += sc * rebuild( U * project(v) )
template <typename T, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void leg_core(const T v[24], T sc, const T* __restrict__ Us, T acc[24]) {
    constexpr int SGN = (FWD ? -1 : 1) * (DAG ? -1 : 1);
    T h[12], w[12], U[MDWF_LROW];
    project<MU, SGN, T>(v, h);
    typedef Pack16<T> P;
#pragma unroll
    for (int q = 0; q < MDWF_LROW / P::N; ++q) {
        if (q * P::N >= 18) break;
        const P t = reinterpret_cast<const P*>(Us)[q];
#pragma unroll
        for (int e = 0; e < P::N; ++e) U[q * P::N + e] = t.d[e];
    }
    su3_mul<false, T>(U, h, w);
    // acc += sc * (rebuilt spinor), explicit FMAs (24 per leg)
    const T cs = sc * (T)SGN;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const T w0r = w[c * 2], w0i = w[c * 2 + 1], w1r = w[6 + c * 2], w1i = w[6 + c * 2 + 1];
        acc[c * 2] = fma_<T>(sc, w0r, acc[c * 2]); acc[c * 2 + 1] = fma_<T>(sc, w0i, acc[c * 2 + 1]);
        acc[6 + c * 2] = fma_<T>(sc, w1r, acc[6 + c * 2]); acc[6 + c * 2 + 1] = fma_<T>(sc, w1i, acc[6 + c * 2 + 1]);
        if (MU == 0) {
            acc[12 + c * 2] = fma_<T>(cs, w1i, acc[12 + c * 2]); acc[12 + c * 2 + 1] = fma_<T>(-cs, w1r, acc[12 + c * 2 + 1]);
            acc[18 + c * 2] = fma_<T>(cs, w0i, acc[18 + c * 2]); acc[18 + c * 2 + 1] = fma_<T>(-cs, w0r, acc[18 + c * 2 + 1]);
        } else if (MU == 1) {
            acc[12 + c * 2] = fma_<T>(cs, w1r, acc[12 + c * 2]); acc[12 + c * 2 + 1] = fma_<T>(cs, w1i, acc[12 + c * 2 + 1]);
            acc[18 + c * 2] = fma_<T>(-cs, w0r, acc[18 + c * 2]); acc[18 + c * 2 + 1] = fma_<T>(-cs, w0i, acc[18 + c * 2 + 1]);
        } else if (MU == 2) {
            acc[12 + c * 2] = fma_<T>(cs, w0i, acc[12 + c * 2]); acc[12 + c * 2 + 1] = fma_<T>(-cs, w0r, acc[12 + c * 2 + 1]);
            acc[18 + c * 2] = fma_<T>(-cs, w1i, acc[18 + c * 2]); acc[18 + c * 2 + 1] = fma_<T>(cs, w1r, acc[18 + c * 2 + 1]);
        } else {
            acc[12 + c * 2] = fma_<T>(cs, w0r, acc[12 + c * 2]); acc[12 + c * 2 + 1] = fma_<T>(cs, w0i, acc[12 + c * 2 + 1]);
            acc[18 + c * 2] = fma_<T>(cs, w1r, acc[18 + c * 2]); acc[18 + c * 2 + 1] = fma_<T>(cs, w1i, acc[18 + c * 2 + 1]);
        }
    }
}

// the same with the neighbour gathered from global memory (5D index nidx)
template <typename S, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void leg2(const SpinorView& in, int rhs, int N5h, int nidx,
                                     const typename Store<S>::real* __restrict__ Us,
                                     typename Store<S>::real acc[24]) {
    typedef typename Store<S>::real T;
    T v[24], sc;
    load_raw<S>(in, rhs, nidx, N5h, v, sc);
    leg_core<T, MU, FWD, DAG>(v, sc, Us, acc);
}

struct HopArgs {
    SpinorView out, in, xin;   // xin.v == nullptr -> no xpay term
    GaugeView g;
    LsOp op;                   // s-direction factor applied to H(in); kind 0 -> none
    double cx, ch;
    double* partial;           // nullptr or [nact][nblk_per_rhs] per-block sum |out|^2 (fixed order)
    int par;                   // parity of the output sites
    int nact;                  // active rhs count; blockIdx.x = tile*nact + slot
    int rhs_list[64];
    ScaleRule sr;              // fp16 output only (mdwf_hop16.cuh)
    const int* stop;           // optional device flag: non-zero -> the launch is a no-op (CG iterations queued behind the
                               // point where the device decided to leave the inner loop, solver.cu)
};

// (tile, site-in-tile) -> coordinates; see Geom for the traversal order
struct SiteCoord { int xh, xx, y, z, t, o; };
__device__ __forceinline__ SiteCoord decode_site(const Geom& g, int par, uint32_t tile, uint32_t i) {
    SiteCoord c;
    uint32_t q, tT, tZ, tY, tX, ix, iy, iz, it, r;
    g.dnTx.divmod(tile, q, tX);
    g.dnTy.divmod(q, r, tY);
    g.dnTzs.divmod(r, q, tZ);
    g.dnTt.divmod(q, r, tT);            // r = slab index
    g.dtxh.divmod(i, q, ix);
    g.dty.divmod(q, it, iy);
    g.dtz.divmod(it, it, iz);
    c.xx = tX * g.txh + ix; c.y = tY * g.ty + iy; c.z = r * g.zc + tZ * g.tz + iz; c.t = tT * g.tt + it;
    c.o = (par + c.y + c.z + c.t) & 1;                 // x = 2*xx + o
    c.xh = c.xx + g.XH * (c.y + g.Y * (c.z + g.Z * c.t));
    return c;
}

// Fused epilogue of hop_kernel:  out = cx * xin + ch * op(acc), streaming store, optional fixed-order |out|^2
// partial.  ch is folded into the s-direction coefficients, so the xpay costs 24 FMAs.
template <typename S>
__device__ __forceinline__ void fused_epilogue(const Geom& g, const HopArgs& a, typename Store<S>::real acc[24], bool live,
                                               int rhs, int idx, int slot, int tile, unsigned char* smem_epi) {
    typedef typename Store<S>::real T;
    if (a.op.kind != 0) {
        LsOp op = a.op;
        op.c0 *= a.ch;
        op.c1 *= a.ch;
        apply_ls<T>(acc, op, g.Ls, smem_epi);
    } else {
        const T ch = (T)a.ch;
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] *= ch;
    }
    if (a.xin.v != nullptr && live) {
        T xv[24], sc;
        load_raw<S>(a.xin, rhs, idx, g.N5h, xv, sc);
        const T cxs = (T)a.cx * sc;
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] = fma_<T>(cxs, xv[i], acc[i]);
    }
    if (live) store_spinor<S, MDWF_HOP_STCS>(a.out, rhs, idx, g.N5h, acc);
    if (a.partial != nullptr) {
        // the 24 squares of one site are summed in the compute type, everything above in fp64
        T s24 = 0;
        if (live) {
#pragma unroll
            for (int i = 0; i < 24; ++i) s24 = fma_<T>(acc[i], acc[i], s24);
        }
        block_sum_store((double)s24, smem_epi, a.partial + (long long)slot * (gridDim.x / a.nact) + tile);
    }
}

// Leg l (mu = l>>1, forward for even l) of site c: the link as the stencil multiplies it -- reconstructed from
// the packed format, daggered for backward legs, times the boundary sign -- as 18 (+2 pad) reals; returns the
// neighbour's half-index.
template <typename S, int R>
__device__ __forceinline__ int stage_link(const Geom& g, const GaugeView& gv, int par, const SiteCoord& c, int l,
                                          typename Store<S>::real V[MDWF_LROW]) {
    typedef typename Store<S>::real T;
    const int mu = l >> 1, xh = c.xh;
    const bool fwd = (l & 1) == 0;
    int n;
    bool wrap;
    if (mu == 0) {
        if (fwd) { wrap = (c.o == 1 && c.xx == g.XH - 1); n = wrap ? xh - (g.XH - 1) : xh + c.o; }
        else { wrap = (c.o == 0 && c.xx == 0); n = wrap ? xh + (g.XH - 1) : xh - (1 - c.o); }
    } else {
        const int cm = mu == 1 ? c.y : mu == 2 ? c.z : c.t;
        const int Lm = mu == 1 ? g.Y : mu == 2 ? g.Z : g.T;
        const int sm = mu == 1 ? g.XH : mu == 2 ? g.XH * g.Y : g.XH * g.Y * g.Z;
        if (fwd) { wrap = cm == Lm - 1; n = wrap ? xh - (Lm - 1) * sm : xh + sm; }
        else { wrap = cm == 0; n = wrap ? xh + (Lm - 1) * sm : xh - sm; }
    }
    const T sgn = wrap ? (T)g.bc[mu] : (T)1;
    T U[18];
    load_link<S, R>(fwd ? gv.v[par] : gv.v[1 - par], mu, fwd ? xh : n, g.Vh, U);
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) {
            V[(r * 3 + cc) * 2] = sgn * (fwd ? U[(r * 3 + cc) * 2] : U[(cc * 3 + r) * 2]);
            V[(r * 3 + cc) * 2 + 1] = sgn * (fwd ? U[(r * 3 + cc) * 2 + 1] : -U[(cc * 3 + r) * 2 + 1]);
        }
    V[18] = V[19] = 0;
    return n;
}

template <typename S, int R, bool DAG, bool FUSED>
__global__ void __launch_bounds__(256, (sizeof(S) == 8 ? MDWF_HOP_MINB64 : sizeof(S) == 4 ? MDWF_HOP_MINB32 : MDWF_HOP_MINB)) hop_kernel(const Geom g, const HopArgs a) {
    typedef typename Store<S>::real T;
    typedef Pack16<T> P;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (a.stop != nullptr && *a.stop != 0) return;
    const int Ls = g.Ls;
    const int nsite = g.nsite;
    T* links = reinterpret_cast<T*>(smem_raw);
    int* tab = reinterpret_cast<int*>(smem_raw + (size_t)nsite * MDWF_LSITE * sizeof(T));
    unsigned char* smem_epi = smem_raw + smem_bytes_links<T>(nsite);
    // block order: chunk (z-slab x tile-timeslice) slowest, then rhs, then the tiles of the chunk -- all rhs of a
    // chunk run back to back (their links stay in L2) while each rhs streams through its own slab working set
    uint32_t bq, tin;
    g.dntc.divmod(blockIdx.x, bq, tin);
    const int slot = bq % a.nact;
    const int tile = (bq / a.nact) * g.ntc + tin;
    const int rhs = a.rhs_list[slot];
    // ---- stage the block's links and neighbour table --------------------------------------------------
    {
        for (int task = threadIdx.x; task < nsite * 8; task += blockDim.x) {
            const int i = task >> 3, l = task & 7;
            const SiteCoord c = decode_site(g, a.par, (uint32_t)tile, (uint32_t)i);
            T V[MDWF_LROW];
            const int n = stage_link<S, R>(g, a.g, a.par, c, l, V);
            P* dst = reinterpret_cast<P*>(links + i * MDWF_LSITE + l * MDWF_LROW);
#pragma unroll
            for (int q = 0; q < MDWF_LROW / P::N; ++q) {
                P t;
#pragma unroll
                for (int e = 0; e < P::N; ++e) t.d[e] = V[q * P::N + e];
                dst[q] = t;
            }
            tab[i * 12 + l] = n;
            if (l == 0) tab[i * 12 + 8] = c.xh;
        }
    }
    __syncthreads();
    // ---- the stencil: one thread per (site, s) -----------------------------------------------------------
    const int grp = (int)g.dLs.div(threadIdx.x), s = threadIdx.x - grp * Ls;
    const bool live = grp < nsite;
    T acc[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0;
    int idx = 0;
    if (live) {
        const int4 n0 = reinterpret_cast<const int4*>(tab + grp * 12)[0];
        const int4 n1 = reinterpret_cast<const int4*>(tab + grp * 12)[1];
        idx = tab[grp * 12 + 8] * Ls + s;
        const T* Ub = links + grp * MDWF_LSITE;
        const int N5h = g.N5h;
        leg2<S, 0, true, DAG>(a.in, rhs, N5h, n0.x * Ls + s, Ub + 0 * MDWF_LROW, acc);
        leg2<S, 0, false, DAG>(a.in, rhs, N5h, n0.y * Ls + s, Ub + 1 * MDWF_LROW, acc);
        leg2<S, 1, true, DAG>(a.in, rhs, N5h, n0.z * Ls + s, Ub + 2 * MDWF_LROW, acc);
        leg2<S, 1, false, DAG>(a.in, rhs, N5h, n0.w * Ls + s, Ub + 3 * MDWF_LROW, acc);
        leg2<S, 2, true, DAG>(a.in, rhs, N5h, n1.x * Ls + s, Ub + 4 * MDWF_LROW, acc);
        leg2<S, 2, false, DAG>(a.in, rhs, N5h, n1.y * Ls + s, Ub + 5 * MDWF_LROW, acc);
        leg2<S, 3, true, DAG>(a.in, rhs, N5h, n1.z * Ls + s, Ub + 6 * MDWF_LROW, acc);
        leg2<S, 3, false, DAG>(a.in, rhs, N5h, n1.w * Ls + s, Ub + 7 * MDWF_LROW, acc);
    }
    if (!FUSED) {
        if (live) store_spinor<S, MDWF_HOP_STCS>(a.out, rhs, idx, g.N5h, acc);
        return;
    }
    fused_epilogue<S>(g, a, acc, live, rhs, idx, slot, tile, smem_epi);
}

}  // namespace mdwf
