// csrc/hop16.cu -- host side of the tensor-core fp16 stencil (mdwf_hop16.cuh): 4D tile tables, shared-memory plan,
// tile choice and launch.
#include "mdwf_hop_launch.cuh"
#include "mdwf_hop16.cuh"
#include <algorithm>
#include <cmath>

namespace mdwf {

// gamma matrices of SURVEY 8 Notation (DeGrand-Rossi): entry code 0 = 0, 1 = +1, 2 = -1, 3 = +i, 4 = -i
static const int kGamma[4][4][4] = {
    {{0, 0, 0, 3}, {0, 0, 3, 0}, {0, 4, 0, 0}, {4, 0, 0, 0}},      // gamma_x
    {{0, 0, 0, 2}, {0, 0, 1, 0}, {0, 1, 0, 0}, {2, 0, 0, 0}},      // gamma_y
    {{0, 0, 3, 0}, {0, 0, 0, 4}, {4, 0, 0, 0}, {0, 3, 0, 0}},      // gamma_z
    {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}}};     // gamma_t
static int negate_code(int c) { return c == 1 ? 2 : c == 2 ? 1 : c == 3 ? 4 : c == 4 ? 3 : 0; }

// B-fragment lane (g, t): column n = g <-> (out spin al = g >> 1, re/im = g & 1), k rows <-> in spin be = t.  The words
// it needs for leg l are variant v of the link record:  Gamma = (1 -+ gamma_mu)[al][be],
//   Gamma = 1: re -> V0, im -> V1;  -1: V2, V3;  i: V3, V0;  -i: V1, V2;  0: zero block (code 4)   (mdwf_hop16.cuh)
static void build_vcode(uint32_t vcode[2][32]) {
    for (int dag = 0; dag < 2; ++dag)
        for (int lane = 0; lane < 32; ++lane) {
            const int g = lane >> 2, be = lane & 3, al = g >> 1, ri = g & 1;
            uint32_t packed = 0;
            for (int l = 0; l < 8; ++l) {
                const int mu = l >> 1, fwd = (l & 1) == 0;
                const int sgn = (fwd ? -1 : 1) * (dag ? -1 : 1);
                int gc = al == be ? 1 : kGamma[mu][al][be];
                if (al != be && sgn < 0) gc = negate_code(gc);
                int v;
                switch (gc) {
                    case 1: v = ri ? 1 : 0; break;
                    case 2: v = ri ? 3 : 2; break;
                    case 3: v = ri ? 0 : 3; break;
                    case 4: v = ri ? 2 : 1; break;
                    default: v = 4;
                }
                packed |= (uint32_t)v << (4 * l);
            }
            vcode[dag][lane] = packed;
        }
}

static inline int pack4(int x, int y, int z, int t) { return x | (y << 8) | (z << 16) | (t << 24); }

// shared memory of a block: header | link records of every warp's sites | per-warp epilogue tile | per-warp partial sums
struct Plan16 { int ns, spw; size_t off_links, off_epi, off_wpart, smem; };
static Plan16 plan_tile16(const int L[4], int rows, int nw) {      // rows = RI * Ls of one site
    Plan16 p;
    p.ns = L[0] * L[1] * L[2] * L[3] / 2;
    p.spw = (p.ns + nw - 1) / nw;
    const int MT = (rows + 15) / 16;
    size_t off = MDWF_H16_HDR;
    p.off_links = off; off += (size_t)nw * p.spw * MDWF_H16_SREC;
    off = (off + 15) / 16 * 16;
    p.off_epi = off; off += (size_t)nw * MT * 16 * 24 * 4;
    p.off_wpart = off; off += (size_t)64 * nw * 8;
    p.smem = off;
    return p;
}

static int build_tile16(mdwf_ctx* c, const int L[4], int rows, int nw, Tile16Host* th) {
    const Geom& g = c->g;
    Tile16& tl = th->t;
    memset(&tl, 0, sizeof(tl));
    const int dims[4] = {g.X, g.Y, g.Z, g.T};
    for (int d = 0; d < 4; ++d) { tl.L[d] = L[d]; tl.nT[d] = dims[d] / L[d]; }
    tl.ns = L[0] * L[1] * L[2] * L[3] / 2;
    tl.ntiles = tl.nT[0] * tl.nT[1] * tl.nT[2] * tl.nT[3];
    th->nw = nw;
    th->dev[0] = th->dev[1] = nullptr;
    for (int pat = 0; pat < 2; ++pat) {
        std::vector<int> outc;
        for (int t = 0; t < L[3]; ++t) for (int z = 0; z < L[2]; ++z) for (int y = 0; y < L[1]; ++y) for (int x = 0; x < L[0]; ++x)
            if (((x + y + z + t) & 1) == pat) outc.push_back(pack4(x, y, z, t));
        if ((int)outc.size() != tl.ns) MDWF_FAIL(c, MDWF_EINVAL, "internal: fp16 tile has %zu output sites, expected %d", outc.size(), tl.ns);
        void* d0;
        MDWF_CUDA(c, cudaMalloc(&d0, outc.size() * 4));
        MDWF_CUDA(c, cudaMemcpy(d0, outc.data(), outc.size() * 4, cudaMemcpyHostToDevice));
        th->dev[pat] = d0;
        tl.outc[pat] = (const int*)d0;
    }
    const Plan16 pl = plan_tile16(L, rows, nw);
    tl.spw = pl.spw;
    tl.off_links = (int)pl.off_links; tl.off_epi = (int)pl.off_epi; tl.off_wpart = (int)pl.off_wpart; tl.smem_total = (int)pl.smem;
    tl.dTx = make_fastdiv(tl.nT[0]); tl.dTy = make_fastdiv(tl.nT[1]); tl.dTt = make_fastdiv(tl.nT[3]);
    tl.zc_t = tl.nT[2]; tl.dTzs = make_fastdiv(tl.zc_t);
    build_vcode(tl.vcode);
    return MDWF_OK;
}

void free_tile16(Tile16Host* th) {
    for (int i = 0; i < 2; ++i) if (th->dev[i]) { cudaFree(th->dev[i]); th->dev[i] = nullptr; }
}

// Tile choice.  The block's tile decides how often an input site is found again in L1 by another leg (a 2^4 box has 8
// output sites and 40 distinct inputs: 5 fetches per output instead of 8; 4x4x2x2 has 32 and 128: 4), and with several
// sites per warp all 32 lanes share the link staging of a tile.  Measured on B200 (48^3x64x10, 4 rhs; profiles/README.md):
// 4x4x2x2 with 8 warps (4 sites per warp, two blocks per SM) is ~10 % faster than one site per warp.  Default: extents
// (4, 4, 2, 2) reduced to divisors of the lattice, 8 warps.  mdwf_set_hop16_tile forces a box / warp count (tuning).
static int choose_tile16(mdwf_ctx* c, int rows, int L[4], int* nw_out) {
    const Geom& g = c->g;
    const int dims[4] = {g.X, g.Y, g.Z, g.T};
    const size_t cap = 227 * 1024 - 256;
    if (c->tile16_forced[0] > 0) {
        for (int d = 0; d < 4; ++d) L[d] = c->tile16_forced[d];
        for (int d = 0; d < 4; ++d) if (L[d] < 1 || L[d] > 16 || dims[d] % L[d] || (d == 0 && (L[d] & 1))) MDWF_FAIL(c, MDWF_EINVAL, "forced fp16 tile does not divide the lattice");
        const int ns = L[0] * L[1] * L[2] * L[3] / 2;
        const int nw = c->tile16_nw > 0 ? c->tile16_nw : std::min(ns, MDWF_H16_MAXW);
        const Plan16 pf = plan_tile16(L, rows, nw);
        if (pf.smem > cap || pf.spw > 4) MDWF_FAIL(c, MDWF_EINVAL, "forced fp16 tile does not fit in shared memory (or has more than 4 sites per warp)");
        *nw_out = nw;
        return MDWF_OK;
    }
    auto tu = c->tune.find(tune_key_tile16(c, rows));
    if (tu != c->tune.end() && tu->second.size() == 5) {        // found by mdwf_autotune (or loaded): use it if it is admissible here
        bool ok = true;
        for (int d = 0; d < 4; ++d) {
            L[d] = tu->second[d];
            if (L[d] < 1 || L[d] > 16 || dims[d] % L[d] || (d == 0 && (L[d] & 1))) ok = false;
        }
        const int nw = tu->second[4];
        if (ok && nw >= 1 && nw <= MDWF_H16_MAXW) {
            const Plan16 pt = plan_tile16(L, rows, nw);
            if (pt.smem <= cap && pt.spw <= 4) { *nw_out = nw; return MDWF_OK; }
        }
    }
    const int want[4] = {4, 4, 2, 2};
    for (int d = 0; d < 4; ++d) {
        L[d] = want[d];
        while (dims[d] % L[d]) L[d] >>= 1;
    }
    if (L[0] < 2) L[0] = 2;
    for (;;) {
        const int ns = L[0] * L[1] * L[2] * L[3] / 2;
        *nw_out = std::min(std::max(ns / 4, std::min(ns, 8)), MDWF_H16_MAXW);
        const Plan16 p = plan_tile16(L, rows, *nw_out);
        if (p.smem <= cap / 2 && p.spw <= 4) return MDWF_OK;          // two blocks per SM
        int d = 3;
        while (d >= 0 && L[d] <= (d == 0 ? 2 : 1)) --d;
        if (d < 0) {
            if (p.smem <= cap && p.spw <= 4) return MDWF_OK;
            MDWF_FAIL(c, MDWF_EINVAL, "fp16 stencil tile does not fit in shared memory (%d rows per site)", rows);
        }
        L[d] >>= 1;
    }
}

// tiles are cached per rhs interleave (the epilogue tile holds RI * Ls rows per site)
int get_tile16(mdwf_ctx* c, int ril, Tile16Host** out) {
    if (ril < 0 || ril > 2) MDWF_FAIL(c, MDWF_EINVAL, "internal: bad rhs interleave");
    if (!c->tile16[ril]) {
        const int rows = c->g.Ls << ril;
        int L[4], nw = 0;
        int rc = choose_tile16(c, rows, L, &nw);
        if (rc) return rc;
        Tile16Host* th = new Tile16Host;
        rc = build_tile16(c, L, rows, nw, th);
        if (rc) { free_tile16(th); delete th; return rc; }
        c->tile16[ril] = th;
    }
    *out = c->tile16[ril];
    return MDWF_OK;
}

// z-tiles per slab: the three t-consecutive layers (x, y, slab depth, one tile in t) of every rhs in flight should stay
// in L2, budget ~60 MB
static int pick_zc16(const Geom& g, const Tile16& tl, int sb, int ngrp) {
    int best = 1;
    for (int z = 1; z <= tl.nT[2]; ++z) {
        if (tl.nT[2] % z) continue;
        const double layer = (double)g.XH * g.Y * (z * tl.L[2]) * tl.L[3] * (double)sb * ngrp;
        if (3.0 * layer <= 60.0e6) best = z;
    }
    return best;
}

int launch_hop_f16(mdwf_ctx* c, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st) {
    (void)fused;
    (void)recon;       // the stencil-ready links were decoded from the (prec 16, recon) format at load time
    Tile16Host* th;
    int rc = get_tile16(c, a.in.ril, &th);
    if (rc) return rc;
    if (!a.g.pl[0] || !a.g.pl[1]) MDWF_FAIL(c, MDWF_ESTATE, "internal: stencil-ready fp16 links missing");
    if (!a.in.m || !a.out.m || (a.xin.v && !a.xin.m) || a.sr.n < 1) MDWF_FAIL(c, MDWF_EINVAL, "internal: fp16 hop without field scales");
    if (a.out.ril != a.in.ril || (a.xin.v && a.xin.ril != a.in.ril)) MDWF_FAIL(c, MDWF_EINVAL, "internal: fp16 hop on fields with different rhs interleave");
    const int rows = c->g.Ls << a.in.ril;
    if (rows > 48) MDWF_FAIL(c, MDWF_EINVAL, "internal: %d rows per site", rows);
    Tile16 tl = th->t;
    // rhs groups with an active rhs
    tl.ngrp = 0;
    for (int k = 0; k < a.nact; ++k) {
        const int gr = a.rhs_list[k] >> a.in.ril;
        int j = 0;
        while (j < tl.ngrp && tl.grp[j] != gr) ++j;
        if (j == tl.ngrp) { tl.grp[j] = (unsigned char)gr; tl.gmask[j] = 0; ++tl.ngrp; }
        tl.gmask[j] |= (unsigned char)(1 << (a.rhs_list[k] & ((1 << a.in.ril) - 1)));
    }
    tl.dng = make_fastdiv(tl.ngrp);
    tl.zc_t = c->zc_forced > 0 && c->zc_forced % tl.L[2] == 0 && tl.nT[2] % (c->zc_forced / tl.L[2]) == 0 ? c->zc_forced / tl.L[2]
                                                                                                        : pick_zc16(c->g, tl, a.in.sb, tl.ngrp);
    tl.dTzs = make_fastdiv(tl.zc_t);
    const int block = th->nw * 32;
    const int regs = 128;
    const int per_sm = std::max(1, std::min(2048 / block, (int)((227 * 1024) / (tl.smem_total + 1024))));
    const int grid = (int)std::min<long long>((long long)tl.ntiles * tl.ngrp, (long long)c->sm_count * std::min(per_sm, 65536 / (regs * block)) );
    typedef void (*Kern16)(const Geom, const Tile16, const HopArgs, const int);
    // (templating on the xpay input / the norm output as well was measured: no gain)
    static const Kern16 kerns[3][3] = {{hop16_kernel<1, 1, 1, 0>, hop16_kernel<1, 1, 1, 1>, hop16_kernel<1, 1, 1, 2>},
                                       {hop16_kernel<2, 1, 1, 0>, hop16_kernel<2, 1, 1, 1>, hop16_kernel<2, 1, 1, 2>},
                                       {hop16_kernel<3, 1, 1, 0>, hop16_kernel<3, 1, 1, 1>, hop16_kernel<3, 1, 1, 2>}};
    if (a.op.kind < 0 || a.op.kind > 2) MDWF_FAIL(c, MDWF_EINVAL, "internal: bad epilogue kind %d", a.op.kind);
    const Kern16 kern = kerns[rows <= 16 ? 0 : rows <= 32 ? 1 : 2][a.op.kind];
    if (!c->attr_raised.count((const void*)kern)) {
        MDWF_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        c->attr_raised.insert((const void*)kern);
    }
    if ((size_t)grid > c->partial_cap) MDWF_FAIL(c, MDWF_EINVAL, "internal: partial buffer too small");
    kern<<<std::max(grid, 1), block, tl.smem_total, st>>>(c->g, tl, a, dagger ? 1 : 0);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    c->partial_nblk = std::max(grid, 1);
    return MDWF_OK;
}

}  // namespace mdwf
