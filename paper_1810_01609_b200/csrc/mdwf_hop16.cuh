// csrc/mdwf_hop16.cuh -- the even-odd MDWF Dslash stencil for 16-bit storage on the tensor cores
// ("16-bit precision ... storage (utilizing single-precision computation)"; the stencil itself: PAPER.md:77,
// 90, 175; "SU(3) x (4 Ls nrhs spin-columns) as a batched small-K MMA ... exact w.r.t. 16-bit
// storage / fp32 accumulate").
//
//   out(x,s) = cx * xin(x,s) + ch * sum_{s'} G[s][s'] (H_{p<-pbar} in)(x,s')        (same contract as hop_kernel)
//   (H psi)(x) = sum_mu [ (1 - g_mu) U_mu(x) psi(x+mu) + (1 + g_mu) U_mu(x-mu)^dag psi(x-mu) ]   (SURVEY 8 Notation)
//
// Formulation.  For one output site x and one leg l the map psi(neighbour) -> contribution is the REAL 24 x 24 matrix
// M_l = Gamma_l (x) U_l (Gamma_l = 1 -+ gamma_mu, entries 0, +-1, +-i; U_l the link or its adjoint, boundary sign
// folded).  It is the same for all Ls slices, so the site's hop is the dense contraction
//       out[s][24] = sum_l  psi_l[s][24] . M_l^T          (M = Ls rows, N = 24, K = 8 legs x 24)
// executed as mma.sync m16n8k16 / m16n8k8 (f16 x f16 -> f32): A = the neighbours' stored halves exactly as they sit in
// memory (no cvt, no projection arithmetic), B = +-Re/Im U entries in half precision, accumulation over all 8 legs
// in the fp32 accumulator.  Products of halves are exact in fp32, so this is "16-bit storage, fp32 compute" up to
// summation order; the spin projection and reconstruction cost nothing (they are zeros and signs inside M_l).
//
// Data movement.  A block owns a 4D tile of output sites.  All input sites the tile needs (interior of the other
// parity + one-site halo, each used by up to 8 outputs) are fetched ONCE per (tile, rhs) into shared memory with bulk
// async copies (cp.async.bulk + mbarrier; a 4D site is Ls*48 contiguous bytes in the fp16 layout, x-runs are fetched
// as one copy), double-buffered across the rhs of the tile, so the L2->SM gather traffic drops from 8 to ni/ns (~4)
// site reads per output.  A-fragments come from there with ldmatrix (row = one 5D site's 16-byte colour chunk; the
// 48-byte row stride is bank-conflict free).  The tile's 8*ns links are reconstructed once per tile (12/8-real
// formats), rounded to half and parked in shared memory as the four sign/swap variants (u, i u, -u, -i u in real
// 2x2 form) that the 32 lanes of a B-fragment need, and are reused by every Ls slice and every rhs of the tile
// (north_star: "staging of links reused across the Ls slices and across multiple right-hand sides").
// Epilogue: accumulators -> per-warp shared tile -> s-direction operator (LsOp: c0 + c1 L or c0 + c1 M5^-1 as the
// first-order recurrence of mdwf_hop.cuh) -> xpay -> |out|^2 partial -> half conversion -> 16-byte coalesced stores.
#pragma once
#include "mdwf_hop.cuh"

namespace mdwf {

#define MDWF_H16_HDR 2560          // fixed header of the dynamic shared memory (barriers, per-rhs coefficients, sums)
#define MDWF_H16_LREC 192          // bytes per staged link: 4 variants x 12 words
#define MDWF_H16_MAXW 16           // warps per block

struct Tile16 {
    int L[4];                       // box extents in lattice sites (L[0] even), dividing the lattice
    int nT[4];                      // tiles per direction
    int ns;                         // output sites per tile
    int nip[2], nrun[2];            // input slots / copy runs per parity pattern of the box
    int ntiles;
    int zc_t;                       // z-tiles per slab of the tile traversal (x, y, z-in-slab, t, slab)
    FastDiv dTx, dTy, dTzs, dTt;
    const int* outc[2];             // [ns] packed local coordinates x | y<<8 | z<<16 | t<<24 of the output sites
    const int4* run[2];             // [nrun] {packed local coordinates + 1 of the first site, sites, first slot, 0}
    const unsigned short* nbr[2];   // [ns*8] input slot of each leg
    int off_nbr, off_oxh, off_links, off_zero, off_stage, stage_bytes, off_epi, smem_total;
    uint32_t vcode[2][32];          // [dagger][lane]: 4 bits per leg = variant of the lane's B words (4 = zero)
};
struct Tile16Host {                 // host-side owner of the device tables
    Tile16 t;
    void* dev[6];
    int nw;                         // warps per block
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t mbar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(mbar), "r"(parity) : "memory");
    } while (!done);
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t mbar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(mbar) : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t r[4], uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(addr) : "memory");
}
__device__ __forceinline__ void ldsm_x2(uint32_t r[2], uint32_t addr) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x2.shared.b16 {%0,%1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(addr) : "memory");
}
__device__ __forceinline__ void mma_16816(float c[4], const uint32_t a[4], uint32_t b0, uint32_t b1) {
    asm("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void mma_1688(float c[4], const uint32_t a[2], uint32_t b0) {
    asm("mma.sync.aligned.m16n8k8.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5}, {%6}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3]) : "r"(a[0]), "r"(a[1]), "r"(b0));
}

// origin (lattice coordinates of the box corner) of tile `tile`; tiles run x, y, z inside a z-slab, t, slab
__device__ __forceinline__ void tile16_origin(const Tile16& tl, int tile, int o[4]) {
    uint32_t q, tx, ty, tzs, tt, slab;
    tl.dTx.divmod((uint32_t)tile, q, tx);
    tl.dTy.divmod(q, q, ty);
    tl.dTzs.divmod(q, q, tzs);
    tl.dTt.divmod(q, slab, tt);
    o[0] = tx * tl.L[0]; o[1] = ty * tl.L[1]; o[2] = (slab * tl.zc_t + tzs) * tl.L[2]; o[3] = tt * tl.L[3];
}

// One warp issues the bulk copies of (tile, rhs) into a staging buffer: every x-run of input sites is one copy of
// n*Ls*48 bytes (split where the run wraps around the lattice).
__device__ __forceinline__ void hop16_issue(const Geom& g, const Tile16& tl, const HopArgs& a, int tile, int rhs,
                                            uint32_t stage, uint32_t mbar, int lane) {
    int o[4];
    tile16_origin(tl, tile, o);
    const int pat = (a.par + o[1] + o[2] + o[3]) & 1;
    const uint32_t sb = (uint32_t)g.Ls * 48u;
    if (lane == 0) mbar_expect_tx(mbar, (uint32_t)tl.nip[pat] * sb);
    __syncwarp();
    const char* base = reinterpret_cast<const char*>(a.in.v) + (long long)rhs * a.in.rs;
    const int4* runs = tl.run[pat];
    for (int r = lane; r < tl.nrun[pat]; r += 32) {
        const int4 q = __ldg(runs + r);
        const int lx = (q.x & 255) - 1, ly = ((q.x >> 8) & 255) - 1, lz = ((q.x >> 16) & 255) - 1, lt = ((q.x >> 24) & 255) - 1;
        int gy = o[1] + ly, gz = o[2] + lz, gt = o[3] + lt;
        gy = gy < 0 ? gy + g.Y : gy >= g.Y ? gy - g.Y : gy;
        gz = gz < 0 ? gz + g.Z : gz >= g.Z ? gz - g.Z : gz;
        gt = gt < 0 ? gt + g.T : gt >= g.T ? gt - g.T : gt;
        const int row = g.XH * (gy + g.Y * (gz + g.Z * gt));
        int first = (o[0] + lx) >> 1;            // -1 for the x = -1 halo of the first tile of a row
        const int last = first + q.y - 1;
        int slot = q.z;
        if (first < 0) {
            bulk_g2s(stage + (uint32_t)slot * sb, base + (long long)(row + g.XH - 1) * sb, sb, mbar);
            ++first; ++slot;
        }
        const int lastc = last >= g.XH ? g.XH - 1 : last;
        if (lastc >= first) {
            bulk_g2s(stage + (uint32_t)slot * sb, base + (long long)(row + first) * sb, (uint32_t)(lastc - first + 1) * sb, mbar);
            slot += lastc - first + 1;
        }
        if (last >= g.XH) bulk_g2s(stage + (uint32_t)slot * sb, base + (long long)row * sb, sb, mbar);
    }
}

// Links of the tile -> shared memory: per (site, leg) the matrix the stencil multiplies (reconstructed, daggered for
// backward legs, boundary sign folded: stage_link of mdwf_hop.cuh), rounded to half, in the four variants
//   V0 = (ur, -ui)   V1 = (ui, ur)   V2 = -V0   V3 = -V1        (word a*3+b of each 12-word variant block)
// which are the (k even, k odd) pairs of Re/Im parts of Gamma*u that a B-fragment lane needs for Gamma = 1, -1, i, -i.
template <int R>
__device__ __forceinline__ void hop16_stage_links(const Geom& g, const Tile16& tl, const HopArgs& a, const int o[4], int pat,
                                                  unsigned char* sm) {
    const int* outc = tl.outc[pat];
    int* oxh = reinterpret_cast<int*>(sm + tl.off_oxh);
    for (int task = threadIdx.x; task < tl.ns * 8; task += blockDim.x) {
        const int i = task >> 3, l = task & 7;
        const int pc = __ldg(outc + i);
        const int gx = o[0] + (pc & 255);
        SiteCoord c;
        c.xx = gx >> 1; c.o = gx & 1;
        c.y = o[1] + ((pc >> 8) & 255); c.z = o[2] + ((pc >> 16) & 255); c.t = o[3] + ((pc >> 24) & 255);
        c.xh = c.xx + g.XH * (c.y + g.Y * (c.z + g.Z * c.t));
        float V[MDWF_LROW];
        stage_link<__half, R>(g, a.g, a.par, c, l, V);
        uint32_t w[4][12];
#pragma unroll
        for (int e = 0; e < 9; ++e) {
            const uint32_t h = f2h(V[2 * e], V[2 * e + 1]);      // (ur, ui)
            const uint32_t sw = __byte_perm(h, 0, 0x1032);       // (ui, ur)
            w[0][e] = h ^ 0x80000000u;
            w[1][e] = sw;
            w[2][e] = h ^ 0x00008000u;
            w[3][e] = sw ^ 0x80008000u;
        }
#pragma unroll
        for (int v = 0; v < 4; ++v) { w[v][9] = 0; w[v][10] = 0; w[v][11] = 0; }
        uint4* dst = reinterpret_cast<uint4*>(sm + tl.off_links + task * MDWF_H16_LREC);
#pragma unroll
        for (int v = 0; v < 4; ++v)
#pragma unroll
            for (int q = 0; q < 3; ++q) dst[v * 3 + q] = make_uint4(w[v][4 * q], w[v][4 * q + 1], w[v][4 * q + 2], w[v][4 * q + 3]);
        if (l == 0) oxh[i] = c.xh;
    }
}

// MT = m16 tiles per site: ceil(Ls / 16)
template <int MT>
__global__ void __launch_bounds__(32 * MDWF_H16_MAXW, 1) hop16_kernel(const Geom g, const Tile16 tl, const HopArgs a, const int recon,
                                                                    const int dag) {
    extern __shared__ __align__(128) unsigned char sm[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nw = blockDim.x >> 5;
    const int Ls = g.Ls;
    const uint32_t sbase = smem_u32(sm);
    // header: [0,16) two mbarriers | float4 cf[64] | double e2[64] | double part[64] | double wsum[2][16] | float kp[32]
    float4* s_cf = reinterpret_cast<float4*>(sm + 16);
    double* s_e2 = reinterpret_cast<double*>(sm + 16 + 1024);
    double* s_part = s_e2 + 64;
    double* s_wsum = s_part + 64;
    float* s_kp = reinterpret_cast<float*>(s_wsum + 32);
    const unsigned short* s_nbr = reinterpret_cast<const unsigned short*>(sm + tl.off_nbr);
    const int* s_oxh = reinterpret_cast<const int*>(sm + tl.off_oxh);

    if (tid == 0) {
        mbar_init(sbase, 1);
        mbar_init(sbase + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (tid < a.nact) {
        const int rhs = a.rhs_list[tid];
        const float eo = eval_scale(a.sr, rhs, blockIdx.x == 0);
        const float ei = a.in.m->e[rhs];
        const float ex = a.xin.v != nullptr ? a.xin.m->e[rhs] : 0.f;
        s_cf[tid] = make_float4(ei / eo, ex / eo, 0.f, 0.f);
        s_e2[tid] = (double)eo * (double)eo;
        s_part[tid] = 0.0;
    }
    if (tid < 32) {
        float v = (float)a.op.kappa;
        for (int i = 0; i < tid; ++i) v *= (float)a.op.kappa;
        s_kp[tid] = v;                                  // kappa^{k+1}
    }
    if (tid < 12) reinterpret_cast<uint32_t*>(sm + tl.off_zero)[tid] = 0u;
    __syncthreads();

    const int G = gridDim.x;
    const int nmy = (tl.ntiles - (int)blockIdx.x + G - 1) / G;
    const int nitems = nmy * a.nact;
    if (warp == 0)
        for (int k = 0; k < 2 && k < nitems; ++k)
            hop16_issue(g, tl, a, blockIdx.x + (k / a.nact) * G, a.rhs_list[k % a.nact], sbase + tl.off_stage + k * tl.stage_bytes,
                        sbase + 8 * k, lane);

    // per-lane constants of the fragments
    const int gq = lane >> 2, tq = lane & 3;
    const uint32_t vc = tl.vcode[dag ? 1 : 0][lane];
    uint32_t rowoff4[MT], rowoff2[MT];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        int r4 = mt * 16 + (lane & 7) + 8 * ((lane >> 3) & 1), r2 = mt * 16 + (lane & 15);
        r4 = r4 < Ls ? r4 : Ls - 1;
        r2 = r2 < Ls ? r2 : Ls - 1;
        rowoff4[mt] = (uint32_t)r4 * 48u + (uint32_t)(lane >> 4) * 16u;
        rowoff2[mt] = (uint32_t)r2 * 48u + 32u;
    }
    const uint32_t site_bytes = (uint32_t)Ls * 48u;
    const uint32_t links_addr = sbase + tl.off_links, zero_addr = sbase + tl.off_zero;
    float* E = reinterpret_cast<float*>(sm + tl.off_epi) + warp * (MT * 16 * 24);
    const LsOp op = a.op;
    const float mf = (float)op.mf, kap = (float)op.kappa;

    int cur_tile = -1;
    for (int k = 0; k < nitems; ++k) {
        const int tile = blockIdx.x + (k / a.nact) * G, slot = k % a.nact, rhs = a.rhs_list[slot], buf = k & 1;
        if (tile != cur_tile) {       // new tile: neighbour table, output sites and links (the previous item ended with a barrier)
            int o[4];
            tile16_origin(tl, tile, o);
            const int pat = (a.par + o[1] + o[2] + o[3]) & 1;
            unsigned short* wn = reinterpret_cast<unsigned short*>(sm + tl.off_nbr);
            for (int i = tid; i < tl.ns * 8; i += blockDim.x) wn[i] = __ldg(tl.nbr[pat] + i);
            if (recon == 18) hop16_stage_links<18>(g, tl, a, o, pat, sm);
            else if (recon == 12) hop16_stage_links<12>(g, tl, a, o, pat, sm);
            else hop16_stage_links<8>(g, tl, a, o, pat, sm);
            __syncthreads();
            cur_tile = tile;
        }
        mbar_wait(sbase + 8 * buf, (uint32_t)((k >> 1) & 1));
        const float4 cf = s_cf[slot];
        const uint32_t stg = sbase + tl.off_stage + buf * tl.stage_bytes;
        const float chc = (float)a.ch * cf.x;                       // ch * e_in / e_out
        const float c0f = (float)op.c0 * chc, c1f = (float)op.c1 * chc;
        const float cxs = (float)a.cx * cf.y;                       // cx * e_x / e_out
        const char* xbase = a.xin.v != nullptr ? reinterpret_cast<const char*>(a.xin.v) + (long long)rhs * a.xin.rs : nullptr;
        char* obase = reinterpret_cast<char*>(a.out.v) + (long long)rhs * a.out.rs;
        double s2w = 0.0;
        for (int i = warp; i < tl.ns; i += nw) {
            float acc[MT][3][4];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int n = 0; n < 3; ++n)
#pragma unroll
                    for (int e = 0; e < 4; ++e) acc[mt][n][e] = 0.f;
#pragma unroll
            for (int l = 0; l < 8; ++l) {
                const uint32_t in_addr = stg + (uint32_t)s_nbr[i * 8 + l] * site_bytes;
                const uint32_t code = (vc >> (4 * l)) & 7u;
                const uint32_t baddr = code == 4u ? zero_addr : links_addr + (uint32_t)(i * 8 + l) * MDWF_H16_LREC + code * 48u;
                uint32_t w[12];
#pragma unroll
                for (int q = 0; q < 3; ++q)
                    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];"
                                 : "=r"(w[4 * q]), "=r"(w[4 * q + 1]), "=r"(w[4 * q + 2]), "=r"(w[4 * q + 3]) : "r"(baddr + 16u * q));
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    uint32_t A[4], A2[2];
                    ldsm_x4(A, in_addr + rowoff4[mt]);
                    ldsm_x2(A2, in_addr + rowoff2[mt]);
#pragma unroll
                    for (int n = 0; n < 3; ++n) {
                        mma_16816(acc[mt][n], A, w[3 * n], w[3 * n + 1]);
                        mma_1688(acc[mt][n], A2, w[3 * n + 2]);
                    }
                }
            }
            // ---- epilogue of site i: accumulators -> E[row][colour*8 + spin*2 + reim] ------------------------------
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int n = 0; n < 3; ++n) {
                    float* e0 = E + (mt * 16 + gq) * 24 + (n * 4 + tq) * 2;
                    *reinterpret_cast<float2*>(e0) = make_float2(acc[mt][n][0], acc[mt][n][1]);
                    *reinterpret_cast<float2*>(e0 + 8 * 24) = make_float2(acc[mt][n][2], acc[mt][n][3]);
                }
            __syncwarp();
            constexpr int NQ = (MT * 16 * 3 + 31) / 32;
            float v[NQ][8];
#pragma unroll
            for (int qi = 0; qi < NQ; ++qi) {
                const int q = lane + 32 * qi;
                if (q < Ls * 3) {
                    const int s = (q * 43) >> 7, c = q - 3 * s;
                    const float4 lo = *reinterpret_cast<const float4*>(E + s * 24 + c * 8);
                    const float4 hi = *reinterpret_cast<const float4*>(E + s * 24 + c * 8 + 4);
                    v[qi][0] = lo.x; v[qi][1] = lo.y; v[qi][2] = lo.z; v[qi][3] = lo.w;
                    v[qi][4] = hi.x; v[qi][5] = hi.y; v[qi][6] = hi.z; v[qi][7] = hi.w;
                }
            }
            if (op.kind == 2) {
                // closed form of M5^-1 as a first-order recurrence along s (mdwf_hop.cuh, LsOp), one lane per column
                __syncwarp();
                if (lane < 24) {
                    const bool fwd = ((lane & 7) < 4) != (op.dag != 0);
                    float run = 0.f;
                    for (int kk = 0; kk < Ls; ++kk) {
                        float* p = E + (fwd ? kk : Ls - 1 - kk) * 24 + lane;
                        run = *p + kap * run;
                        *p = run;
                    }
                }
                __syncwarp();
            }
            const long long idx0 = (long long)s_oxh[i] * Ls;
#pragma unroll
            for (int qi = 0; qi < NQ; ++qi) {
                const int q = lane + 32 * qi;
                if (q < Ls * 3) {
                    const int s = (q * 43) >> 7, c = q - 3 * s;
                    float o8[8];
                    if (op.kind == 0) {
#pragma unroll
                        for (int e = 0; e < 8; ++e) o8[e] = chc * v[qi][e];
                    } else if (op.kind == 1) {
                        const int sm1 = s == 0 ? Ls - 1 : s - 1, sp1 = s == Ls - 1 ? 0 : s + 1;
                        const float fm = c1f * (s == 0 ? -mf : 1.f), fp = c1f * (s == Ls - 1 ? -mf : 1.f);
                        const float4 up = *reinterpret_cast<const float4*>(E + (op.dag ? sp1 : sm1) * 24 + c * 8);       // P+ elements
                        const float4 dn = *reinterpret_cast<const float4*>(E + (op.dag ? sm1 : sp1) * 24 + c * 8 + 4);   // P- elements
                        const float fu = op.dag ? fp : fm, fl = op.dag ? fm : fp;
                        o8[0] = c0f * v[qi][0] + fu * up.x; o8[1] = c0f * v[qi][1] + fu * up.y;
                        o8[2] = c0f * v[qi][2] + fu * up.z; o8[3] = c0f * v[qi][3] + fu * up.w;
                        o8[4] = c0f * v[qi][4] + fl * dn.x; o8[5] = c0f * v[qi][5] + fl * dn.y;
                        o8[6] = c0f * v[qi][6] + fl * dn.z; o8[7] = c0f * v[qi][7] + fl * dn.w;
                    } else {
                        const bool fwdp = op.dag == 0;         // P+ columns run forward for M5^-1, backward for its adjoint
                        const float4 pp = *reinterpret_cast<const float4*>(E + s * 24 + c * 8);
                        const float4 pm = *reinterpret_cast<const float4*>(E + s * 24 + c * 8 + 4);
                        const float4 tp = *reinterpret_cast<const float4*>(E + (fwdp ? Ls - 1 : 0) * 24 + c * 8);
                        const float4 tm = *reinterpret_cast<const float4*>(E + (fwdp ? 0 : Ls - 1) * 24 + c * 8 + 4);
                        const float ia = c1f * (float)op.inv_a;
                        const float gp = -c1f * (float)op.gfac * s_kp[fwdp ? s : Ls - 1 - s];
                        const float gm = -c1f * (float)op.gfac * s_kp[fwdp ? Ls - 1 - s : s];
                        o8[0] = c0f * v[qi][0] + ia * pp.x + gp * tp.x; o8[1] = c0f * v[qi][1] + ia * pp.y + gp * tp.y;
                        o8[2] = c0f * v[qi][2] + ia * pp.z + gp * tp.z; o8[3] = c0f * v[qi][3] + ia * pp.w + gp * tp.w;
                        o8[4] = c0f * v[qi][4] + ia * pm.x + gm * tm.x; o8[5] = c0f * v[qi][5] + ia * pm.y + gm * tm.y;
                        o8[6] = c0f * v[qi][6] + ia * pm.z + gm * tm.z; o8[7] = c0f * v[qi][7] + ia * pm.w + gm * tm.w;
                    }
                    const long long off = (idx0 + s) * 48 + c * 16;
                    if (xbase != nullptr) {
                        const uint4 xv = ldg(reinterpret_cast<const uint4*>(xbase + off));
                        const float2 x0 = h2f(xv.x), x1 = h2f(xv.y), x2 = h2f(xv.z), x3 = h2f(xv.w);
                        o8[0] = fmaf(cxs, x0.x, o8[0]); o8[1] = fmaf(cxs, x0.y, o8[1]);
                        o8[2] = fmaf(cxs, x1.x, o8[2]); o8[3] = fmaf(cxs, x1.y, o8[3]);
                        o8[4] = fmaf(cxs, x2.x, o8[4]); o8[5] = fmaf(cxs, x2.y, o8[5]);
                        o8[6] = fmaf(cxs, x3.x, o8[6]); o8[7] = fmaf(cxs, x3.y, o8[7]);
                    }
                    float s8 = 0.f;
#pragma unroll
                    for (int e = 0; e < 8; ++e) s8 = fmaf(o8[e], o8[e], s8);
                    s2w += (double)s8;
                    uint4 t;
                    t.x = f2h_sat(o8[0], o8[1]); t.y = f2h_sat(o8[2], o8[3]); t.z = f2h_sat(o8[4], o8[5]); t.w = f2h_sat(o8[6], o8[7]);
                    __stcs(reinterpret_cast<uint4*>(obase + off), t);
                }
            }
            __syncwarp();
        }
        if (a.partial != nullptr) {
            // fixed-order sums: lanes (shuffle tree) -> warps (serial) -> this block's running sum for the rhs
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s2w += __shfl_down_sync(0xffffffffu, s2w, o);
            if (lane == 0) s_wsum[buf * 16 + warp] = s2w;
        }
        __syncthreads();          // every warp is done with stage[buf] (and with the links if the tile changes)
        if (warp == 0) {
            if (k + 2 < nitems)
                hop16_issue(g, tl, a, blockIdx.x + ((k + 2) / a.nact) * G, a.rhs_list[(k + 2) % a.nact], stg, sbase + 8 * buf, lane);
            if (a.partial != nullptr && lane == 0) {
                double t = 0.0;
                for (int w2 = 0; w2 < nw; ++w2) t += s_wsum[buf * 16 + w2];
                s_part[slot] += t;
            }
        }
    }
    __syncthreads();
    if (a.partial != nullptr && tid < a.nact) a.partial[(long long)tid * G + blockIdx.x] = s_part[tid] * s_e2[tid];
}

}  // namespace mdwf
