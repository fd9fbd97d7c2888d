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
// folded).  It is the same for all Ls slices and all right-hand sides, so the site's hop is the dense contraction
//       out[row][24] = sum_l  psi_l[row][24] . M_l^T       (M = RI*Ls rows (rhs in group, s), N = 24, K = 8 legs x 24)
// executed as mma.sync m16n8k16 / m16n8k8 (f16 x f16 -> f32): A = the neighbours' stored halves exactly as they sit in
// memory (no cvt, no projection arithmetic), B = +-Re/Im U entries in half precision, accumulation over all 8 legs
// in the fp32 accumulator.  Products of halves are exact in fp32, so this is "16-bit storage, fp32 compute" up to
// summation order; the spin projection and reconstruction cost nothing (they are zeros and signs inside M_l).
//
// Data movement.  The fp16 field layout IS the A-fragment order (mdwf_device.cuh): the 16 rows x 24 halves of an m16
// tile are six 128-byte lines, each read by one coalesced LDG.32 straight into the fragment registers (through L1,
// where the other legs of the block's 4D tile find them again) -- no shared-memory staging, so shared memory only
// holds the link records and the epilogue tile and 16 warps per SM stay resident.  A block owns a 4D tile of output
// sites (one warp per site, or a few sites per warp); the 8 links of a site come from the stencil-ready half-precision
// link table (gauge.cu: decoded from the 18/12/8-real format, daggered, boundary sign folded, at load time), are
// fetched one item ahead and parked in shared memory as the four sign/swap variants (u, i u, -u, -i u in real 2x2
// form) plus zeros that the 32 lanes of a B fragment need; they serve every Ls slice and every rhs of the group
// (north_star: "staging of links reused across the Ls slices and across multiple right-hand sides").
// Epilogue: accumulators -> per-warp shared tile -> s-direction operator (LsOp: c0 + c1 L or c0 + c1 M5^-1 as the
// first-order recurrence of mdwf_hop.cuh) -> xpay -> |out|^2 partial -> half conversion -> 16-byte coalesced stores.
#pragma once
#include "mdwf_hop.cuh"

namespace mdwf {

#define MDWF_H16_HDR 1408          // fixed header of the dynamic shared memory (kappa powers, per-rhs coefficients, lane codes)
#define MDWF_H16_LREC 272          // bytes per staged link: 4 variants + a zero block of 12 words each (240 B), padded so that
                                   // the 8 records of a site start 4 banks apart (conflict-free staging stores)
#define MDWF_H16_SREC (8 * MDWF_H16_LREC + 48)   // per site: 8 link records + the site index + the 8 neighbour indices
#define MDWF_H16_MAXW 16           // warps per block
#define MDWF_H16_PLW 80            // words per site of the stencil-ready link table: 9 x 8 link words + 8 neighbours

struct Tile16 {
    int L[4];                       // box extents in lattice sites (L[0] even), dividing the lattice
    int nT[4];                      // tiles per direction
    int ns;                         // output sites per tile
    int spw;                        // sites per warp = ceil(ns / warps)
    int ntiles;
    int zc_t;                       // z-tiles per slab of the tile traversal (x, y, z-in-slab, t, slab)
    FastDiv dTx, dTy, dTzs, dTt, dng;
    const int* outc[2];             // [ns] packed local coordinates x | y<<8 | z<<16 | t<<24 of the output sites, per parity pattern
    int off_links, off_epi, off_wpart, smem_total;
    int ngrp;                       // rhs groups with an active rhs, their ids and active-rhs masks
    unsigned char grp[64], gmask[64];
    uint32_t vcode[2][32];          // [dagger][lane]: 4 bits per leg = variant of the lane's B words (4 = zero)
};
struct Tile16Host {                 // host-side owner of the device tables
    Tile16 t;
    void* dev[2];
    int nw;                         // warps per block
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
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

// Persistent kernel: block b processes the (tile, rhs group) items b, b + G, ...; there is no block barrier in the item
// loop.  Each warp owns `spw` output sites of the tile and prepares the link records of ITS sites itself:
//   link record of a (site, leg), 4 variants + zeros, 12 words each:  V0 = (ur, -ui)  V1 = (ui, ur)  V2 = -V0  V3 = -V1
//   per U entry u = U[a][b]: the (k even, k odd) pairs of Re/Im parts of Gamma*u that a B-fragment lane needs for
//   Gamma = 1, -1, i, -i (0: the zero block).  Word order inside a variant: B00 B01 B10 B11 | B20 B21 B02 B12 | B22,
//   so that the k16 operand pairs of the three n-tiles (= output colours) are aligned register pairs of two 16-byte
//   loads; the five blocks sit in disjoint banks, so the 32 lanes of a fragment load never conflict.
// MT = m16 tiles per site: ceil(RI * Ls / 16) <= 3
// KIND = LsOp kind of the fused epilogue (0: none, 1: c0 + c1 L, 2: c0 + c1 M5^-1), a template parameter so that each
// instantiation carries only its own epilogue (registers, code size)
template <int MT, int PF, int MINB, int KIND>
__global__ void __launch_bounds__(PF ? 32 * MDWF_H16_MAXW : 256, MINB) hop16_kernel(const Geom g, const Tile16 tl, const HopArgs a, const int dag) {
    extern __shared__ __align__(128) unsigned char sm[];
    if (a.stop != nullptr && *a.stop != 0) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nwc = (int)(blockDim.x >> 5);
    const int Ls = g.Ls, ns = tl.ns, spw = tl.spw;
    const int ril = a.in.ril, RI = 1 << ril, rows = Ls << ril, nrb = (rows + 7) >> 3;
    const uint32_t sb = (uint32_t)a.in.sb;                    // bytes of a 4D site of one rhs group
    float* s_kp = reinterpret_cast<float*>(sm);               // [32] kappa^{k+1}
    float2* s_cf = reinterpret_cast<float2*>(sm + 128);       // [64] by rhs id: (e_in / e_out, e_x / e_out)
    double* s_e2 = reinterpret_cast<double*>(sm + 640);       // [64] e_out^2
    uint32_t* s_vc = reinterpret_cast<uint32_t*>(sm + 1152);  // [32] per lane: variant code of each leg (4 bits per leg)
    double* s_wpart = reinterpret_cast<double*>(sm + tl.off_wpart);        // [64 rhs][nwc]
    if (tid < 32) {
        float v = (float)a.op.kappa;
        for (int i = 0; i < tid; ++i) v *= (float)a.op.kappa;
        s_kp[tid] = v;
        s_vc[tid] = tl.vcode[dag ? 1 : 0][tid];
    }
    for (int i = tid; i < nwc * spw * 8 * 12; i += blockDim.x) {      // the zero block of every link record
        const int rec = i / 12;
        reinterpret_cast<uint32_t*>(sm + tl.off_links + (rec >> 3) * MDWF_H16_SREC + (rec & 7) * MDWF_H16_LREC + 192)[i % 12] = 0u;
    }
    if (a.partial != nullptr)
        for (int i = tid; i < 64 * nwc; i += blockDim.x) s_wpart[i] = 0.0;
    // the scale of the output: every block evaluates the rule (same inputs, same result); block 0 stores it
    if (tid < a.nact) {
        const int rhs = a.rhs_list[tid];
        const float eo = eval_scale(a.sr, rhs, blockIdx.x == 0);
        const float ei = a.in.m->e[rhs];
        const float ex = a.xin.v != nullptr ? a.xin.m->e[rhs] : 0.f;
        s_cf[rhs] = make_float2(ei / eo, ex / eo);
        s_e2[rhs] = (double)eo * (double)eo;
    }
    __syncthreads();

    const int G = gridDim.x, ngrp = tl.ngrp;
    const int nitems = tl.ntiles * ngrp;
    const int gq = lane >> 2, tq = lane & 3;
    const uint32_t vc = s_vc[lane];
    uint32_t cl[8];                       // offset of the lane's variant block (or the zero block) inside a site record
#pragma unroll
    for (int l = 0; l < 8; ++l) cl[l] = (uint32_t)l * MDWF_H16_LREC + ((vc >> (4 * l)) & 7u) * 48u;
    // A-fragment addressing inside a site: row block rb at rb*384, chunk c at + c*128, this lane at + gq*16 + tq*4.
    // Row blocks 2*mt and 2*mt + 1 are read at compile-time offsets; rows beyond the site's last row block are zeros.
    const uint32_t lane_off = (uint32_t)gq * 16u + (uint32_t)tq * 4u;
    constexpr int NQ = (MT * 48 + 31) / 32;
    // epilogue work items of this lane: 16-byte piece q = lane + 32 qi of the site in memory order (row block q / 24,
    // colour chunk (q % 24) / 8, row q % 8), packed as  E offset of (rhs, chunk) | s << 16 | rhs-in-group << 24, or -1
    int qd[NQ];
#pragma unroll
    for (int qi = 0; qi < NQ; ++qi) {
        const int q = lane + 32 * qi;
        const int rb = (q * 171) >> 12, rem = q - rb * 24, c = rem >> 3, row = rb * 8 + (rem & 7);
        const int ri = (row >= Ls) + (row >= 2 * Ls) + (row >= 3 * Ls), s = row - ri * Ls;
        qd[qi] = (row < rows && q < nrb * 24) ? ((ri * Ls * 24 + c * 8) | (s << 16) | (ri << 24)) : -1;
    }
    unsigned char* wl = sm + tl.off_links + warp * spw * MDWF_H16_SREC;      // this warp's site records
    const uint32_t wl_addr = smem_u32(wl);
    float* E = reinterpret_cast<float*>(sm + tl.off_epi) + warp * (MT * 16 * 24);
    const LsOp op = a.op;
    const float mf = (float)op.mf, kap = (float)op.kappa;
    const int il_me = lane >> 3, l_me = lane & 7;
    const bool has_link = il_me < spw && warp * spw + il_me < ns;
    const uint32_t* plt = a.g.pl[a.par];

    uint32_t raw[9];
    int rxh = 0, rnb = 0, rtile = -1;
    // stencil-ready links, neighbour index and output site index of this lane's (site, leg) in tile `tile`
    auto fetch_links = [&](int tile) {
        rtile = tile;
        if (has_link) {
            int o[4];
            tile16_origin(tl, tile, o);
            const int pat = (a.par + o[1] + o[2] + o[3]) & 1;
            const int pc = __ldg(tl.outc[pat] + warp * spw + il_me);
            const int gx = o[0] + (pc & 255);
            rxh = (gx >> 1) + g.XH * (o[1] + ((pc >> 8) & 255) + g.Y * (o[2] + ((pc >> 16) & 255) + g.Z * (o[3] + ((pc >> 24) & 255))));
            const uint32_t* p = plt + (long long)rxh * MDWF_H16_PLW + l_me;
#pragma unroll
            for (int e = 0; e < 9; ++e) raw[e] = __ldg(p + e * 8);
            rnb = (int)__ldg(p + 72);
        }
    };
    int cur_tile = -1;
    if ((int)blockIdx.x < nitems) fetch_links((int)tl.dng.div(blockIdx.x));

    for (int k = blockIdx.x; k < nitems; k += G) {
        uint32_t tile_u, gi_u;
        tl.dng.divmod((uint32_t)k, tile_u, gi_u);
        const int tile = (int)tile_u, grp = tl.grp[gi_u], gmask = tl.gmask[gi_u];
        if (tile != cur_tile) {
            // ---- new tile: this warp's link records from the fetched words, then fetch the next item's ------------
            if (rtile != tile) fetch_links(tile);
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
                int* meta = reinterpret_cast<int*>(wl + il_me * MDWF_H16_SREC + 8 * MDWF_H16_LREC);
                meta[4 + l_me] = rnb;
                if (l_me == 0) meta[0] = rxh;
            }
            __syncwarp();
            cur_tile = tile;
            const int k2 = k + G;
            if (k2 < nitems) {
                const int t2 = (int)tl.dng.div((uint32_t)k2);
                if (t2 != tile) fetch_links(t2);
            }
        }
        const char* ibase = reinterpret_cast<const char*>(a.in.v) + (long long)grp * a.in.rs;
        const char* xbase = a.xin.v != nullptr ? reinterpret_cast<const char*>(a.xin.v) + (long long)grp * a.xin.rs : nullptr;
        char* obase = reinterpret_cast<char*>(a.out.v) + (long long)grp * a.out.rs;
        float s2r[4] = {0.f, 0.f, 0.f, 0.f};
        uint32_t A[2][MT][6];
        bool a0_ready = false;          // A[0] already holds leg 0 of this site (issued during the previous site's last leg)
        for (int il = 0; il < spw; ++il) {
            const int i = warp * spw + il;
            if (i >= ns) break;
            const uint32_t srec = wl_addr + il * MDWF_H16_SREC;
            const int* smeta = reinterpret_cast<const int*>(wl + il * MDWF_H16_SREC + 8 * MDWF_H16_LREC);
            const int4 nb0 = *reinterpret_cast<const int4*>(smeta + 4), nb1 = *reinterpret_cast<const int4*>(smeta + 8);
            const int nxh[8] = {nb0.x, nb0.y, nb0.z, nb0.w, nb1.x, nb1.y, nb1.z, nb1.w};
            float acc[MT][3][4];
#pragma unroll
            for (int mt = 0; mt < MT; ++mt)
#pragma unroll
                for (int n = 0; n < 3; ++n)
#pragma unroll
                    for (int e = 0; e < 4; ++e) acc[mt][n][e] = 0.f;
            // A fragments of one leg: per m16 tile six 128-byte lines (rows 0-7 / 8-15 x colour chunk 0, 1, 2)
            auto load_A = [&](int nx, uint32_t (&dst)[MT][6]) {
                const uint32_t* np = reinterpret_cast<const uint32_t*>(ibase + ((long long)nx * sb + lane_off));
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    dst[mt][0] = __ldg(np + mt * 192); dst[mt][2] = __ldg(np + mt * 192 + 32); dst[mt][4] = __ldg(np + mt * 192 + 64);
                    if (2 * mt + 1 < nrb) {      // rows 8-15 of the tile exist (the site has an odd number of row blocks otherwise)
                        dst[mt][1] = __ldg(np + mt * 192 + 96); dst[mt][3] = __ldg(np + mt * 192 + 128); dst[mt][5] = __ldg(np + mt * 192 + 160);
                    } else {
                        dst[mt][1] = 0u; dst[mt][3] = 0u; dst[mt][5] = 0u;
                    }
                }
            };
            if (PF && !a0_ready) load_A(nxh[0], A[0]);
            a0_ready = false;
            const long long idx0 = (long long)smeta[0] * sb;
#pragma unroll
            for (int l = 0; l < 8; ++l) {
                if (PF) {
                    if (l < 7) load_A(nxh[l + 1], A[(l + 1) & 1]);
                    else if (il + 1 < spw && i + 1 < ns) {
                        // leg 0 of the warp's next site of this tile: in flight during this site's last MMAs and its epilogue
                        load_A(reinterpret_cast<const int*>(wl + (il + 1) * MDWF_H16_SREC + 8 * MDWF_H16_LREC)[4], A[0]);
                        a0_ready = true;
                    }
                } else load_A(nxh[l], A[l & 1]);
                const uint4 b0 = *reinterpret_cast<const uint4*>(wl + il * MDWF_H16_SREC + cl[l]);
                const uint4 b1 = *reinterpret_cast<const uint4*>(wl + il * MDWF_H16_SREC + cl[l] + 16);
                const uint32_t b2 = *reinterpret_cast<const uint32_t*>(wl + il * MDWF_H16_SREC + cl[l] + 32);
#pragma unroll
                for (int mt = 0; mt < MT; ++mt) {
                    const uint32_t* Ac = A[l & 1][mt];
                    mma_16816(acc[mt][0], Ac, b0.x, b0.y);
                    mma_16816(acc[mt][1], Ac, b0.z, b0.w);
                    mma_16816(acc[mt][2], Ac, b1.x, b1.y);
                    mma_1688(acc[mt][0], Ac + 4, b1.z);
                    mma_1688(acc[mt][1], Ac + 4, b1.w);
                    mma_1688(acc[mt][2], Ac + 4, b2);
                }
            }
            (void)srec;
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
            if (KIND == 2) {
                // closed form of M5^-1 as a first-order recurrence along s (mdwf_hop.cuh, LsOp), one lane per column of a rhs:
                // P_s = v_s + kappa P_{s-1} in place (forward for one chirality, backward for the other)
                // (up to three columns per lane, advanced together so that their dependent load-fma-store chains overlap)
                float* cb[3];
                bool cf[3], cv[3];
                float run[3] = {0.f, 0.f, 0.f};
#pragma unroll
                for (int u = 0; u < 3; ++u) {
                    const int j = lane + 32 * u, rj = j / 24, col = j - rj * 24;
                    cv[u] = j < RI * 24;
                    cf[u] = ((col & 7) < 4) != (op.dag != 0);
                    cb[u] = E + rj * Ls * 24 + col;
                }
                for (int kk = 0; kk < Ls; ++kk) {
#pragma unroll
                    for (int u = 0; u < 3; ++u) {
                        if (cv[u]) {
                            float* p = cb[u] + (cf[u] ? kk : Ls - 1 - kk) * 24;
                            run[u] = *p + kap * run[u];
                            *p = run[u];
                        }
                    }
                }
                __syncwarp();
            }
#pragma unroll
            for (int qi = 0; qi < NQ; ++qi) {
                const int q = lane + 32 * qi;
                if (qd[qi] >= 0) {
                    const int ri = qd[qi] >> 24, s = (qd[qi] >> 16) & 255;
                    if ((gmask >> ri) & 1) {
                        const float2 cf = s_cf[(grp << ril) + ri];
                        const float chc = (float)a.ch * cf.x;                       // ch * e_in / e_out
                        const float* Er = E + (qd[qi] & 0xffff);                    // this rhs, this colour chunk, row s at + s*24
                        float o8[8];
                        if (KIND == 0) {
                            const float4 lo = *reinterpret_cast<const float4*>(Er + s * 24);
                            const float4 hi = *reinterpret_cast<const float4*>(Er + s * 24 + 4);
                            o8[0] = chc * lo.x; o8[1] = chc * lo.y; o8[2] = chc * lo.z; o8[3] = chc * lo.w;
                            o8[4] = chc * hi.x; o8[5] = chc * hi.y; o8[6] = chc * hi.z; o8[7] = chc * hi.w;
                        } else if (KIND == 1) {
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
                        const long long off = idx0 + q * 16;
                        if (xbase != nullptr) {
                            const float cxs = (float)a.cx * cf.y;                   // cx * e_x / e_out
                            // (loading the xpay input ahead of the s-direction operator was tried: +5 registers' worth of spills, 30 % slower)
                            const uint4 xv = __ldcs(reinterpret_cast<const uint4*>(xbase + off));
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
