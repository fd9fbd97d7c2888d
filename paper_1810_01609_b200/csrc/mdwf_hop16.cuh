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

#define MDWF_H16_HDR 4096          // fixed header of the dynamic shared memory (barriers, per-rhs coefficients, kappa powers)
#define MDWF_H16_LREC 272          // bytes per staged link: 4 variants + a zero block of 12 words each (240 B), padded so that
                                   // the 8 records of a site start 4 banks apart (conflict-free staging stores)
#define MDWF_H16_SREC (8 * MDWF_H16_LREC + 16)   // per site: 8 link records + the site index
#define MDWF_H16_MAXW 16           // warps per block
#define MDWF_H16_MAXST 4           // staging buffers

struct Tile16 {
    int L[4];                       // box extents in lattice sites (L[0] even), dividing the lattice
    int nT[4];                      // tiles per direction
    int ns;                         // output sites per tile
    int spw;                        // sites per consumer warp = ceil(ns / warps)
    int nst;                        // staging buffers (2..4)
    int nip[2], nrun[2];            // input slots / copy runs per parity pattern of the box
    int ntiles;
    int zc_t;                       // z-tiles per slab of the tile traversal (x, y, z-in-slab, t, slab)
    FastDiv dTx, dTy, dTzs, dTt;
    const int* outc[2];             // [ns] packed local coordinates x | y<<8 | z<<16 | t<<24 of the output sites
    const int4* run[2];             // [nrun] {packed local coordinates + 1 of the first site, sites, first slot, 0}
    const unsigned short* nbr[2];   // [ns*8] input slot of each leg
    int off_nbr, off_links, off_stage, stage_bytes, off_epi, off_wpart, smem_total;
    uint32_t vcode[2][32];          // [dagger][lane]: 4 bits per leg = variant of the lane's B words (4 = zero)
};
struct Tile16Host {                 // host-side owner of the device tables
    Tile16 t;
    void* dev[6];
    int nw;                         // consumer warps per block
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

// One warp issues the bulk copies of (tile, rhs group) into a staging buffer: every x-run of input sites is one copy
// of n*RI*Ls*48 bytes (split where the run wraps around the lattice).
__device__ __forceinline__ void hop16_issue(const Geom& g, const Tile16& tl, const HopArgs& a, int tile, int grp,
                                            uint32_t stage, uint32_t mbar, int lane) {
    int o[4];
    tile16_origin(tl, tile, o);
    const int pat = (a.par + o[1] + o[2] + o[3]) & 1;
    const uint32_t sb = ((uint32_t)g.Ls * 48u) << a.in.ril;      // all rhs of the group at one 4D site
    if (lane == 0) mbar_expect_tx(mbar, (uint32_t)tl.nip[pat] * sb);
    __syncwarp();
    const char* base = reinterpret_cast<const char*>(a.in.v) + (long long)grp * a.in.rs;
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

__device__ __forceinline__ void mbar_arrive(uint32_t mbar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
    return r;
}
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t r;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(addr));
    return r;
}

// Persistent kernel without block barriers in steady state.  The (tile, rhs group) items of a block stream through
// `nst` staging buffers filled by bulk async copies ("full" mbarriers); the warp that finishes an item LAST (shared
// counter) refills its buffer with item k + nst.  Each warp owns `spw` output sites of every tile, prepares the links
// of ITS sites itself (from the prepared half-precision link table, fetched one tile ahead into registers) and runs
// stencil + epilogue on them.  The M rows of a site are (rhs in group, s): RI*Ls rows = MT m16 tiles that share one
// set of B fragments per leg.
//   link record of a (site, leg), 4 variants + zeros, 12 words each:  V0 = (ur, -ui)  V1 = (ui, ur)  V2 = -V0  V3 = -V1
//   per U entry u = U[a][b]: the (k even, k odd) pairs of Re/Im parts of Gamma*u that a B-fragment lane needs for
//   Gamma = 1, -1, i, -i (0: the zero block).  Word order inside a variant: B00 B01 B10 B11 | B20 B21 B02 B12 | B22,
//   so that the k16 operand pairs of the three n-tiles (= output colours) are aligned register pairs of two 16-byte
//   loads; the five blocks sit in disjoint banks, so the 32 lanes of a fragment load never conflict.
// MT = m16 tiles per site: ceil(RI * Ls / 16) <= 3
template <int MT>
__global__ void __launch_bounds__(32 * MDWF_H16_MAXW, 1) hop16_kernel(const Geom g, const Tile16 tl, const HopArgs a, const int dag) {
    extern __shared__ __align__(128) unsigned char sm[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nwc = (int)(blockDim.x >> 5);
    const int Ls = g.Ls, nst = tl.nst, ns = tl.ns, spw = tl.spw;
    const int ril = a.in.ril, RI = 1 << ril, rows = Ls << ril;
    const uint32_t sbase = smem_u32(sm);
    // header: full[4] mbarriers | int done[4] | float4 cf[64] (by rhs id) | double e2[64] | float kp[32] | groups
    int* s_done = reinterpret_cast<int*>(sm + 32);
    int* s_ngrp = reinterpret_cast<int*>(sm + 48);
    float4* s_cf = reinterpret_cast<float4*>(sm + 64);
    double* s_e2 = reinterpret_cast<double*>(sm + 1088);
    float* s_kp = reinterpret_cast<float*>(sm + 1600);
    int* s_grp = reinterpret_cast<int*>(sm + 1728);           // [64] group ids with an active rhs
    int* s_gmask = s_grp + 64;                                // [64] active rhs of the group (bit per rhs in group)
    int* s_slot = s_gmask + 64;                               // [64] rhs id -> position in the active list
    uint32_t* s_nbr = reinterpret_cast<uint32_t*>(sm + tl.off_nbr);       // [2][ns*8] byte offsets inside a staging buffer
    int* s_outc = reinterpret_cast<int*>(s_nbr + 2 * ns * 8);              // [2][ns]
    double* s_wpart = reinterpret_cast<double*>(sm + tl.off_wpart);        // [64 rhs][nwc]
    const uint32_t site_bytes = (uint32_t)rows * 48u;

    if (tid == 0) {
        for (int st = 0; st < nst; ++st) { mbar_init(sbase + 8 * st, 1); s_done[st] = 0; }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        int ng = 0;
        for (int k = 0; k < a.nact; ++k) {
            const int rhs = a.rhs_list[k], gr = rhs >> ril;
            int j = 0;
            while (j < ng && s_grp[j] != gr) ++j;
            if (j == ng) { s_grp[ng] = gr; s_gmask[ng] = 0; ++ng; }
            s_gmask[j] |= 1 << (rhs & (RI - 1));
            s_slot[rhs] = k;
        }
        *s_ngrp = ng;
    }
    if (tid < a.nact) {
        const int rhs = a.rhs_list[tid];
        const float eo = eval_scale(a.sr, rhs, blockIdx.x == 0);
        const float ei = a.in.m->e[rhs];
        const float ex = a.xin.v != nullptr ? a.xin.m->e[rhs] : 0.f;
        s_cf[rhs] = make_float4(ei / eo, ex / eo, 0.f, 0.f);
        s_e2[rhs] = (double)eo * (double)eo;
    }
    if (tid < 32) {
        float v = (float)a.op.kappa;
        for (int i = 0; i < tid; ++i) v *= (float)a.op.kappa;
        s_kp[tid] = v;                                  // kappa^{k+1}
    }
    for (int i = tid; i < 2 * ns * 8; i += blockDim.x) {
        const int pat = i >= ns * 8 ? 1 : 0;
        s_nbr[i] = (uint32_t)__ldg(tl.nbr[pat] + (i - pat * ns * 8)) * site_bytes;
    }
    for (int i = tid; i < 2 * ns; i += blockDim.x) {
        const int pat = i >= ns ? 1 : 0;
        s_outc[i] = __ldg(tl.outc[pat] + (i - pat * ns));
    }
    for (int i = tid; i < nwc * spw * 8 * 12; i += blockDim.x) {      // the zero block of every link record
        const int rec = i / 12;
        reinterpret_cast<uint32_t*>(sm + tl.off_links + (rec >> 3) * MDWF_H16_SREC + (rec & 7) * MDWF_H16_LREC + 192)[i % 12] = 0u;
    }
    for (int i = tid; i < 64 * nwc; i += blockDim.x) s_wpart[i] = 0.0;
    __syncthreads();

    const int G = gridDim.x, ngrp = *s_ngrp;
    const int nmy = (tl.ntiles - (int)blockIdx.x + G - 1) / G;
    const int nitems = nmy * ngrp;
    if (warp == 0)
        for (int k = 0; k < nst && k < nitems; ++k)
            hop16_issue(g, tl, a, blockIdx.x + (k / ngrp) * G, s_grp[k % ngrp], sbase + tl.off_stage + k * tl.stage_bytes, sbase + 8 * k, lane);

    const int gq = lane >> 2, tq = lane & 3;
    const uint32_t vc = tl.vcode[dag ? 1 : 0][lane];
    uint32_t cl[8];                       // offset of the lane's variant block (or the zero block) inside a site record
#pragma unroll
    for (int l = 0; l < 8; ++l) cl[l] = (uint32_t)l * MDWF_H16_LREC + ((vc >> (4 * l)) & 7u) * 48u;
    uint32_t rowoff4[MT], rowoff2[MT];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt) {
        int r4 = mt * 16 + (lane & 7) + 8 * ((lane >> 3) & 1), r2 = mt * 16 + (lane & 15);
        r4 = r4 < rows ? r4 : rows - 1;
        r2 = r2 < rows ? r2 : rows - 1;
        rowoff4[mt] = (uint32_t)r4 * 48u + (uint32_t)(lane >> 4) * 16u;
        rowoff2[mt] = (uint32_t)r2 * 48u + 32u;
    }
    constexpr int NQ = (MT * 16 * 3 + 31) / 32;
    unsigned char* wl = sm + tl.off_links + warp * spw * MDWF_H16_SREC;      // this warp's site records
    const uint32_t wl_addr = smem_u32(wl);
    float* E = reinterpret_cast<float*>(sm + tl.off_epi) + warp * (MT * 16 * 24);
    const LsOp op = a.op;
    const float mf = (float)op.mf, kap = (float)op.kappa;
    const int il_me = lane >> 3, l_me = lane & 7;
    const bool has_link = il_me < spw && warp * spw + il_me < ns;
    const uint32_t* plt = a.g.pl[a.par];

    uint32_t raw[9];
    int rxh = 0, rpat = 0;
    // prepared links (and output site index) of this lane's (site, leg) in tile `tile`
    auto fetch_links = [&](int tile) {
        int o[4];
        tile16_origin(tl, tile, o);
        rpat = (a.par + o[1] + o[2] + o[3]) & 1;
        if (has_link) {
            const int pc = s_outc[rpat * ns + warp * spw + il_me];
            const int gx = o[0] + (pc & 255);
            rxh = (gx >> 1) + g.XH * (o[1] + ((pc >> 8) & 255) + g.Y * (o[2] + ((pc >> 16) & 255) + g.Z * (o[3] + ((pc >> 24) & 255))));
            const uint32_t* p = plt + (long long)rxh * 72 + l_me;
#pragma unroll
            for (int e = 0; e < 9; ++e) raw[e] = __ldg(p + e * 8);
        }
    };
    if (nitems > 0) fetch_links(blockIdx.x);

    int st = 0, use = 0, tix = 0, gi = 0, pat = 0;
    for (int k = 0; k < nitems; ++k) {
        if (gi == 0) {
            // ---- new tile: this warp's link records from the fetched words, then fetch the next tile's ------------
            pat = rpat;
            if (has_link) {
                uint32_t w[4][12];
#pragma unroll
                for (int e = 0; e < 9; ++e) {
                    constexpr int pos[9] = {0, 1, 6, 2, 3, 7, 4, 5, 8};     // e = a*3 + b -> word
                    const uint32_t h = raw[e];                               // (ur, ui)
                    const uint32_t sw = __byte_perm(h, 0, 0x1032);           // (ui, ur)
                    w[0][pos[e]] = h ^ 0x80000000u;
                    w[1][pos[e]] = sw;
                    w[2][pos[e]] = h ^ 0x00008000u;
                    w[3][pos[e]] = sw ^ 0x80008000u;
                }
#pragma unroll
                for (int v = 0; v < 4; ++v) { w[v][9] = 0; w[v][10] = 0; w[v][11] = 0; }
                uint4* dst = reinterpret_cast<uint4*>(wl + il_me * MDWF_H16_SREC + l_me * MDWF_H16_LREC);
#pragma unroll
                for (int v = 0; v < 4; ++v)
#pragma unroll
                    for (int q = 0; q < 3; ++q) dst[v * 3 + q] = make_uint4(w[v][4 * q], w[v][4 * q + 1], w[v][4 * q + 2], w[v][4 * q + 3]);
                if (l_me == 0) *reinterpret_cast<int*>(wl + il_me * MDWF_H16_SREC + 8 * MDWF_H16_LREC) = rxh;
            }
            __syncwarp();
            if (tix + 1 < nmy) fetch_links(blockIdx.x + (tix + 1) * G);
        }
        const int grp = s_grp[gi], gmask = s_gmask[gi];
        mbar_wait(sbase + 8 * st, (uint32_t)(use & 1));
        const uint32_t stg = sbase + tl.off_stage + st * tl.stage_bytes;
        const char* xbase = a.xin.v != nullptr ? reinterpret_cast<const char*>(a.xin.v) + (long long)grp * a.xin.rs : nullptr;
        char* obase = reinterpret_cast<char*>(a.out.v) + (long long)grp * a.out.rs;
        float s2r[4] = {0.f, 0.f, 0.f, 0.f};
        for (int il = 0; il < spw; ++il) {
            const int i = warp * spw + il;
            if (i >= ns) break;
            const uint32_t srec = wl_addr + il * MDWF_H16_SREC;
            const uint4 n0 = lds128(sbase + tl.off_nbr + (uint32_t)(pat * ns + i) * 32u);
            const uint4 n1 = lds128(sbase + tl.off_nbr + (uint32_t)(pat * ns + i) * 32u + 16u);
            const uint32_t noff[8] = {n0.x, n0.y, n0.z, n0.w, n1.x, n1.y, n1.z, n1.w};
            float acc[MT][3][4];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int n = 0; n < 3; ++n)
#pragma unroll
                    for (int e = 0; e < 4; ++e) acc[mt][n][e] = 0.f;
#pragma unroll
            for (int l = 0; l < 8; ++l) {
                const uint32_t in_addr = stg + noff[l];
                const uint32_t baddr = srec + cl[l];
                const uint4 b0 = lds128(baddr), b1 = lds128(baddr + 16u);
                const uint32_t b2 = lds32(baddr + 32u);
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    uint32_t A[4], A2[2];
                    ldsm_x4(A, in_addr + rowoff4[mt]);
                    ldsm_x2(A2, in_addr + rowoff2[mt]);
                    mma_16816(acc[mt][0], A, b0.x, b0.y);
                    mma_16816(acc[mt][1], A, b0.z, b0.w);
                    mma_16816(acc[mt][2], A, b1.x, b1.y);
                    mma_1688(acc[mt][0], A2, b1.z);
                    mma_1688(acc[mt][1], A2, b1.w);
                    mma_1688(acc[mt][2], A2, b2);
                }
            }
            // ---- epilogue of site i: accumulators -> E[row][colour*8 + spin*2 + reim], row = rhs-in-group * Ls + s -----
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int n = 0; n < 3; ++n) {
                    float* e0 = E + (mt * 16 + gq) * 24 + (n * 4 + tq) * 2;
                    *reinterpret_cast<float2*>(e0) = make_float2(acc[mt][n][0], acc[mt][n][1]);
                    *reinterpret_cast<float2*>(e0 + 8 * 24) = make_float2(acc[mt][n][2], acc[mt][n][3]);
                }
            __syncwarp();
            if (op.kind == 2) {
                // closed form of M5^-1 as a first-order recurrence along s (mdwf_hop.cuh, LsOp), one lane per column of a rhs:
                // P_s = v_s + kappa P_{s-1} in place (forward for one chirality, backward for the other)
                for (int j = lane; j < RI * 24; j += 32) {
                    const int rj = j / 24, col = j - rj * 24;
                    const bool fwd = ((col & 7) < 4) != (op.dag != 0);
                    float run = 0.f;
                    float* base = E + rj * Ls * 24 + col;
                    for (int kk = 0; kk < Ls; ++kk) {
                        float* p = base + (fwd ? kk : Ls - 1 - kk) * 24;
                        run = *p + kap * run;
                        *p = run;
                    }
                }
                __syncwarp();
            }
            const long long idx0 = (long long)*reinterpret_cast<const int*>(wl + il * MDWF_H16_SREC + 8 * MDWF_H16_LREC) * site_bytes;
#pragma unroll
            for (int qi = 0; qi < NQ; ++qi) {
                const int q = lane + 32 * qi;
                if (q < rows * 3) {
                    const int row = (q * 171) >> 9, c = q - 3 * row;
                    const int ri = (row >= Ls) + (row >= 2 * Ls) + (row >= 3 * Ls), s = row - ri * Ls;
                    if ((gmask >> ri) & 1) {
                        const float4 cf = s_cf[(grp << ril) + ri];
                        const float chc = (float)a.ch * cf.x;                       // ch * e_in / e_out
                        const float* Er = E + ri * Ls * 24 + c * 8;                 // this rhs, this colour chunk, row s at + s*24
                        float o8[8];
                        if (op.kind == 0) {
                            const float4 lo = *reinterpret_cast<const float4*>(Er + s * 24);
                            const float4 hi = *reinterpret_cast<const float4*>(Er + s * 24 + 4);
                            o8[0] = chc * lo.x; o8[1] = chc * lo.y; o8[2] = chc * lo.z; o8[3] = chc * lo.w;
                            o8[4] = chc * hi.x; o8[5] = chc * hi.y; o8[6] = chc * hi.z; o8[7] = chc * hi.w;
                        } else if (op.kind == 1) {
                            const float c0f = (float)op.c0 * chc, c1f = (float)op.c1 * chc;
                            const int sm1 = s == 0 ? Ls - 1 : s - 1, sp1 = s == Ls - 1 ? 0 : s + 1;
                            const float fm = c1f * (s == 0 ? -mf : 1.f), fp = c1f * (s == Ls - 1 ? -mf : 1.f);
                            const float4 lo = *reinterpret_cast<const float4*>(Er + s * 24);
                            const float4 hi = *reinterpret_cast<const float4*>(Er + s * 24 + 4);
                            const float4 up = *reinterpret_cast<const float4*>(Er + (op.dag ? sp1 : sm1) * 24);       // P+ elements
                            const float4 dn = *reinterpret_cast<const float4*>(Er + (op.dag ? sm1 : sp1) * 24 + 4);   // P- elements
                            const float fu = op.dag ? fp : fm, fl = op.dag ? fm : fp;
                            o8[0] = c0f * lo.x + fu * up.x; o8[1] = c0f * lo.y + fu * up.y;
                            o8[2] = c0f * lo.z + fu * up.z; o8[3] = c0f * lo.w + fu * up.w;
                            o8[4] = c0f * hi.x + fl * dn.x; o8[5] = c0f * hi.y + fl * dn.y;
                            o8[6] = c0f * hi.z + fl * dn.z; o8[7] = c0f * hi.w + fl * dn.w;
                        } else {
                            // (c0 + c1 M5^-1) v from the in-place P:  v_s = P_s - kappa P_prev,  M5^-1 v = P_s / a - g kappa^{k+1} T
                            const float c0f = (float)op.c0 * chc, c1f = (float)op.c1 * chc;
                            const bool fwdp = op.dag == 0;         // P+ columns run forward for M5^-1, backward for its adjoint
                            const int sprev_p = fwdp ? s - 1 : s + 1, sprev_m = fwdp ? s + 1 : s - 1;
                            const float4 pp = *reinterpret_cast<const float4*>(Er + s * 24);
                            const float4 pm = *reinterpret_cast<const float4*>(Er + s * 24 + 4);
                            float4 qp = make_float4(0.f, 0.f, 0.f, 0.f), qm = qp;
                            if (sprev_p >= 0 && sprev_p < Ls) qp = *reinterpret_cast<const float4*>(Er + sprev_p * 24);
                            if (sprev_m >= 0 && sprev_m < Ls) qm = *reinterpret_cast<const float4*>(Er + sprev_m * 24 + 4);
                            const float4 tp = *reinterpret_cast<const float4*>(Er + (fwdp ? Ls - 1 : 0) * 24);
                            const float4 tm = *reinterpret_cast<const float4*>(Er + (fwdp ? 0 : Ls - 1) * 24 + 4);
                            const float ia = c0f + c1f * (float)op.inv_a, ck = -c0f * kap;
                            const float gp = -c1f * (float)op.gfac * s_kp[fwdp ? s : Ls - 1 - s];
                            const float gm = -c1f * (float)op.gfac * s_kp[fwdp ? Ls - 1 - s : s];
                            o8[0] = ia * pp.x + ck * qp.x + gp * tp.x; o8[1] = ia * pp.y + ck * qp.y + gp * tp.y;
                            o8[2] = ia * pp.z + ck * qp.z + gp * tp.z; o8[3] = ia * pp.w + ck * qp.w + gp * tp.w;
                            o8[4] = ia * pm.x + ck * qm.x + gm * tm.x; o8[5] = ia * pm.y + ck * qm.y + gm * tm.y;
                            o8[6] = ia * pm.z + ck * qm.z + gm * tm.z; o8[7] = ia * pm.w + ck * qm.w + gm * tm.w;
                        }
                        const long long off = idx0 + row * 48 + c * 16;
                        if (xbase != nullptr) {
                            const float cxs = (float)a.cx * cf.y;                   // cx * e_x / e_out
                            const uint4 xv = ldg(reinterpret_cast<const uint4*>(xbase + off));
                            const float2 x0 = h2f(xv.x), x1 = h2f(xv.y), x2 = h2f(xv.z), x3 = h2f(xv.w);
                            o8[0] = fmaf(cxs, x0.x, o8[0]); o8[1] = fmaf(cxs, x0.y, o8[1]);
                            o8[2] = fmaf(cxs, x1.x, o8[2]); o8[3] = fmaf(cxs, x1.y, o8[3]);
                            o8[4] = fmaf(cxs, x2.x, o8[4]); o8[5] = fmaf(cxs, x2.y, o8[5]);
                            o8[6] = fmaf(cxs, x3.x, o8[6]); o8[7] = fmaf(cxs, x3.y, o8[7]);
                        }
                        if (a.partial != nullptr) {
                            float s8 = 0.f;
#pragma unroll
                            for (int e = 0; e < 8; ++e) s8 = fmaf(o8[e], o8[e], s8);
#pragma unroll
                            for (int rr = 0; rr < 4; ++rr) s2r[rr] += ri == rr ? s8 : 0.f;
                        }
                        uint4 t;
                        t.x = f2h_sat(o8[0], o8[1]); t.y = f2h_sat(o8[2], o8[3]); t.z = f2h_sat(o8[4], o8[5]); t.w = f2h_sat(o8[6], o8[7]);
                        __stcs(reinterpret_cast<uint4*>(obase + off), t);
                    }
                }
            }
            __syncwarp();
        }
        // this warp is done with the staging buffer; the last warp to get here refills it with item k + nst
        int last = 0;
        if (lane == 0) {
            __threadfence_block();
            last = atomicAdd(&s_done[st], 1) == nwc - 1;
            if (last) s_done[st] = 0;
        }
        last = __shfl_sync(0xffffffffu, last, 0);
        if (last && k + nst < nitems) {
            const int k2 = k + nst;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            hop16_issue(g, tl, a, blockIdx.x + (k2 / ngrp) * G, s_grp[k2 % ngrp], stg, sbase + 8 * st, lane);
        }
        if (a.partial != nullptr) {
            // fixed-order sums: lanes (shuffle tree) -> this warp's running sum per rhs -> warps (serial, at the end)
#pragma unroll
            for (int rr = 0; rr < 4; ++rr) {
                if (rr < RI && ((gmask >> rr) & 1)) {
                    double d = (double)s2r[rr];
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) d += __shfl_down_sync(0xffffffffu, d, o);
                    if (lane == 0) s_wpart[((grp << ril) + rr) * nwc + warp] += d;
                }
            }
        }
        if (++st == nst) { st = 0; ++use; }
        if (++gi == ngrp) { gi = 0; ++tix; }
    }
    if (a.partial != nullptr) {
        __syncthreads();
        if (tid < a.nact) {
            const int rhs = a.rhs_list[tid];
            double t = 0.0;
            for (int w2 = 0; w2 < nwc; ++w2) t += s_wpart[rhs * nwc + w2];
            a.partial[(long long)tid * G + blockIdx.x] = t * s_e2[rhs];
        }
    }
}

}  // namespace mdwf
