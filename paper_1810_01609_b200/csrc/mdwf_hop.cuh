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
// One thread per 5D site (s fastest), one rhs per block; blocks are ordered rhs-fastest so the blocks
// that share a tile's links run together and hit L2; sites are traversed in z-slabs so t-neighbours
// are reused from L2.  Links are loaded through L1 (all Ls threads of a site read the
// same vectors: one broadcast sector per warp).
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
            T re = 0, im = 0;
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const T ur = ADJ ? U[(j * 3 + i) * 2] : U[(i * 3 + j) * 2];
                const T ui = ADJ ? -U[(j * 3 + i) * 2 + 1] : U[(i * 3 + j) * 2 + 1];
                const T hr = h[k * 6 + j * 2], hi = h[k * 6 + j * 2 + 1];
                re += ur * hr - ui * hi;
                im += ur * hi + ui * hr;
            }
            w[k * 6 + i * 2] = re;
            w[k * 6 + i * 2 + 1] = im;
        }
}

// one of the eight stencil legs.  FWD: neighbour x+mu, link U_mu(x) (parity p array at xh);
// !FWD: neighbour x-mu, link U_mu(x-mu)^dag (parity pbar array at the neighbour's xh).
template <typename S, int R, int MU, bool FWD, bool DAG>
__device__ __forceinline__ void leg(const SpinorView& in, const GaugeView& gv, int rhs, int N5h, int Ls, int Vh,
                                    int par, int xh, int nxh, int s, typename Store<S>::real bcs,
                                    typename Store<S>::real acc[24]) {
    typedef typename Store<S>::real T;
    constexpr int SGN = (FWD ? -1 : 1) * (DAG ? -1 : 1);
    T v[24], sc;
    load_raw<S>(in, rhs, nxh * Ls + s, N5h, v, sc);
    T h[12], w[12], U[18];
    project<MU, SGN, T>(v, h);
    if (FWD) load_link<S, R>(gv.v[par], MU, xh, Vh, U);
    else load_link<S, R>(gv.v[1 - par], MU, nxh, Vh, U);
    su3_mul<!FWD, T>(U, h, w);
    recon<MU, SGN, T>(w, sc * bcs, acc);
}

template <typename T> struct alignas(16) Pack16 {
    static constexpr int N = 16 / sizeof(T);
    T d[N];
};

// acc(s) <- sum_{s'} G_chi[s][s'] acc(s') over the Ls threads of one (site, rhs) group, through shared
// memory.  G: device Gt[chi][s'][s] (chi = 0: spins 0,1 = P+, chi = 1: spins 2,3 = P-).  Every thread of
// the block must call it (block-wide barriers); blockDim.x is a multiple of Ls.
// smem needed: smem_bytes_G<T>(Ls, nthreads).
template <typename T> __host__ __device__ inline int smem_reals_G(int Ls, int nthreads) {
    return ((2 * Ls * Ls + 3) & ~3) + (nthreads / Ls) * (Ls * 28 + 4);
}
template <typename T>
__device__ __forceinline__ void apply_G(T acc[24], const void* G, int Ls, unsigned char* smem_raw) {
    T* Gs = reinterpret_cast<T*>(smem_raw);
    const int gsz = (2 * Ls * Ls + 3) & ~3;
    T* buf = Gs + gsz;
    for (int i = threadIdx.x; i < 2 * Ls * Ls; i += blockDim.x) Gs[i] = reinterpret_cast<const T*>(G)[i];
    const int grp = threadIdx.x / Ls, sl = threadIdx.x - grp * Ls;
    const int gstride = Ls * 28 + 4;   // 28-real rows (+4 per group): conflict-free 16-byte accesses
    typedef Pack16<T> P;
    constexpr int NP = 24 / P::N;
    P* mine = reinterpret_cast<P*>(buf + grp * gstride + sl * 28);
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        P t;
#pragma unroll
        for (int e = 0; e < P::N; ++e) t.d[e] = acc[q * P::N + e];
        mine[q] = t;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0;
    const T* grow = buf + grp * gstride;
    for (int sp = 0; sp < Ls; ++sp) {
        const T gp = Gs[sp * Ls + sl], gm = Gs[Ls * Ls + sp * Ls + sl];
        const P* src = reinterpret_cast<const P*>(grow + sp * 28);
#pragma unroll
        for (int q = 0; q < NP; ++q) {
            const P t = src[q];
#pragma unroll
            for (int e = 0; e < P::N; ++e) acc[q * P::N + e] += (q * P::N + e < 12 ? gp : gm) * t.d[e];
        }
    }
    __syncthreads();
}

// fixed-order block sum (shared-memory tree: same order every run -> bit-reproducible); thread 0 stores.
// smem needed: blockDim.x doubles.  Every thread of the block must call it.
__device__ __forceinline__ void block_sum_store(double v, unsigned char* smem_raw, double* dst) {
    double* red = reinterpret_cast<double*>(smem_raw);
    __syncthreads();
    red[threadIdx.x] = v;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o && (int)threadIdx.x + o < (int)blockDim.x) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *dst = red[0];
}

struct HopArgs {
    SpinorView out, in, xin;   // xin.v == nullptr -> no xpay term
    GaugeView g;
    const void* G;             // device: 2*Ls*Ls reals of the compute type, Gt[chi][s'][s]; nullptr -> identity
    double cx, ch;
    double* partial;           // nullptr or [nact][nblk_per_rhs] per-block sum |out|^2 (fixed order)
    int par;                   // parity of the output sites
    int nact;                  // active rhs count; blockIdx.x = tile*nact + slot
    int rhs_list[64];
};

// thread linear index within a rhs -> (xh, s, coordinates) through the slab traversal
struct SiteCoord { int xh, s, xx, y, z, t, o; };
__device__ __forceinline__ SiteCoord decode_site(const Geom& g, int par, uint32_t j) {
    SiteCoord c;
    uint32_t site, s;
    g.dLs.divmod(j, site, s);
    uint32_t zcI, rem, t, rem2, row, xx, zl, y;
    g.dTslab.divmod(site, zcI, rem);
    g.dSlab.divmod(rem, t, rem2);
    g.dXH.divmod(rem2, row, xx);
    g.dY.divmod(row, zl, y);
    c.s = s; c.xx = xx; c.y = y; c.z = zcI * g.zc + zl; c.t = t;
    c.o = (par + c.y + c.z + c.t) & 1;                 // x = 2*xx + o
    c.xh = xx + g.XH * (c.y + g.Y * (c.z + g.Z * c.t));
    return c;
}

template <typename S, int R, bool DAG, bool FUSED>
__global__ void __launch_bounds__(256) hop_kernel(const Geom g, const HopArgs a) {
    typedef typename Store<S>::real T;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int slot = blockIdx.x % a.nact;
    const int tile = blockIdx.x / a.nact;
    const int rhs = a.rhs_list[slot];
    const uint32_t j = (uint32_t)tile * blockDim.x + threadIdx.x;
    const bool live = j < (uint32_t)g.N5h;
    T acc[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) acc[i] = 0;
    int idx = 0;
    if (live) {
        const SiteCoord c = decode_site(g, a.par, j);
        const int xh = c.xh, s = c.s, Ls = g.Ls, Vh = g.Vh, N5h = g.N5h;
        idx = xh * Ls + s;
        const int sy = g.XH, sz = g.XH * g.Y, st = g.XH * g.Y * g.Z;
        // x: neighbours live in the other parity's half-index space
        {
            int nf = xh + c.o, nb = xh - (1 - c.o);
            T bf = 1, bb = 1;
            if (c.o == 1 && c.xx == g.XH - 1) { nf = xh - (g.XH - 1); bf = (T)g.bc[0]; }
            if (c.o == 0 && c.xx == 0) { nb = xh + (g.XH - 1); bb = (T)g.bc[0]; }
            leg<S, R, 0, true, DAG>(a.in, a.g, rhs, N5h, Ls, Vh, a.par, xh, nf, s, bf, acc);
            leg<S, R, 0, false, DAG>(a.in, a.g, rhs, N5h, Ls, Vh, a.par, xh, nb, s, bb, acc);
        }
        {
            int nf = xh + sy, nb = xh - sy;
            T bf = 1, bb = 1;
            if (c.y == g.Y - 1) { nf = xh - (g.Y - 1) * sy; bf = (T)g.bc[1]; }
            if (c.y == 0) { nb = xh + (g.Y - 1) * sy; bb = (T)g.bc[1]; }
            leg<S, R, 1, true, DAG>(a.in, a.g, rhs, N5h, Ls, Vh, a.par, xh, nf, s, bf, acc);
            leg<S, R, 1, false, DAG>(a.in, a.g, rhs, N5h, Ls, Vh, a.par, xh, nb, s, bb, acc);
        }
        {
            int nf = xh + sz, nb = xh - sz;
            T bf = 1, bb = 1;
            if (c.z == g.Z - 1) { nf = xh - (g.Z - 1) * sz; bf = (T)g.bc[2]; }
            if (c.z == 0) { nb = xh + (g.Z - 1) * sz; bb = (T)g.bc[2]; }
            leg<S, R, 2, true, DAG>(a.in, a.g, rhs, N5h, Ls, Vh, a.par, xh, nf, s, bf, acc);
            leg<S, R, 2, false, DAG>(a.in, a.g, rhs, N5h, Ls, Vh, a.par, xh, nb, s, bb, acc);
        }
        {
            int nf = xh + st, nb = xh - st;
            T bf = 1, bb = 1;
            if (c.t == g.T - 1) { nf = xh - (g.T - 1) * st; bf = (T)g.bc[3]; }
            if (c.t == 0) { nb = xh + (g.T - 1) * st; bb = (T)g.bc[3]; }
            leg<S, R, 3, true, DAG>(a.in, a.g, rhs, N5h, Ls, Vh, a.par, xh, nf, s, bf, acc);
            leg<S, R, 3, false, DAG>(a.in, a.g, rhs, N5h, Ls, Vh, a.par, xh, nb, s, bb, acc);
        }
    }
    if (!FUSED) {
        if (live) store_spinor<S>(a.out, rhs, idx, g.N5h, acc);
        return;
    }
    // ---- fused epilogue: s-direction matrix, xpay, optional |out|^2 ---------------------------
    if (a.G != nullptr) apply_G<T>(acc, a.G, g.Ls, smem_raw);
    const T ch = (T)a.ch;
    if (a.xin.v != nullptr) {
        if (live) {
            T xv[24];
            load_spinor<S>(a.xin, rhs, idx, g.N5h, xv);
            const T cx = (T)a.cx;
#pragma unroll
            for (int i = 0; i < 24; ++i) acc[i] = cx * xv[i] + ch * acc[i];
        }
    } else {
#pragma unroll
        for (int i = 0; i < 24; ++i) acc[i] *= ch;
    }
    if (live) store_spinor<S>(a.out, rhs, idx, g.N5h, acc);
    if (a.partial != nullptr) {
        double s2 = 0.0;
        if (live) {
#pragma unroll
            for (int i = 0; i < 24; ++i) s2 += (double)acc[i] * (double)acc[i];
        }
        block_sum_store(s2, smem_raw, a.partial + (long long)slot * (gridDim.x / a.nact) + tile);
    }
}

}  // namespace mdwf
