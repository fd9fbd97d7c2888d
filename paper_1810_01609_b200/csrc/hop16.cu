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

struct Plan16 { int ns, spw, nst, nip[2], nrun[2]; size_t off_nbr, off_links, off_wpart, off_stage, stage, off_epi, smem; };
// counts and shared-memory need of a box without building tables
static Plan16 plan_tile16(const int L[4], int rows, int nw) {      // rows = RI * Ls of one site
    Plan16 p;
    const int vol = L[0] * L[1] * L[2] * L[3];
    p.ns = vol / 2;
    for (int pat = 0; pat < 2; ++pat) {
        int ni = 0, nr = 0;
        for (int t = -1; t <= L[3]; ++t) for (int z = -1; z <= L[2]; ++z) for (int y = -1; y <= L[1]; ++y) {
            const int out = (y < 0 || y >= L[1]) + (z < 0 || z >= L[2]) + (t < 0 || t >= L[3]);
            if (out >= 2) continue;
            const int x0 = out ? 0 : -1, x1 = out ? L[0] - 1 : L[0];
            int n = 0;
            for (int x = x0; x <= x1; ++x) if (((x + y + z + t) & 1) != pat) ++n;
            if (n) { ni += n; ++nr; }
        }
        p.nip[pat] = ni; p.nrun[pat] = nr;
    }
    const int MT = (rows + 15) / 16;
    p.spw = (p.ns + nw - 1) / nw;
    size_t off = MDWF_H16_HDR;
    p.off_nbr = off; off += ((size_t)2 * p.ns * 8 * 4 + (size_t)2 * p.ns * 4 + 15) / 16 * 16;
    p.off_links = off; off += (size_t)nw * p.spw * MDWF_H16_SREC;
    p.off_wpart = off; off += (size_t)64 * nw * 8;
    p.off_epi = off; off += (size_t)nw * MT * 16 * 24 * 4;
    off = (off + 127) / 128 * 128;
    p.off_stage = off;
    p.stage = ((size_t)std::max(p.nip[0], p.nip[1]) * rows * 48 + 127) / 128 * 128;
    const size_t cap = 227 * 1024 - 256;
    p.nst = off + 2 * p.stage > cap ? 2 : (int)std::min<size_t>(MDWF_H16_MAXST, (cap - off) / p.stage);
    p.smem = off + (size_t)p.nst * p.stage;
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
    for (int i = 0; i < 6; ++i) th->dev[i] = nullptr;
    for (int pat = 0; pat < 2; ++pat) {
        std::vector<int> outc;
        std::vector<int4> runs;
        std::map<int, int> slot_of;
        int nslot = 0;
        for (int t = -1; t <= L[3]; ++t) for (int z = -1; z <= L[2]; ++z) for (int y = -1; y <= L[1]; ++y) {
            const int out = (y < 0 || y >= L[1]) + (z < 0 || z >= L[2]) + (t < 0 || t >= L[3]);
            if (out >= 2) continue;
            const int x0 = out ? 0 : -1, x1 = out ? L[0] - 1 : L[0];
            int first = 1 << 30, n = 0;
            for (int x = x0; x <= x1; ++x)
                if (((x + y + z + t) & 1) != pat) {
                    if (n == 0) first = x;
                    slot_of[pack4(x + 1, y + 1, z + 1, t + 1)] = nslot + n;
                    ++n;
                }
            if (n) { runs.push_back(make_int4(pack4(first + 1, y + 1, z + 1, t + 1), n, nslot, 0)); nslot += n; }
        }
        std::vector<unsigned short> nbr;
        for (int t = 0; t < L[3]; ++t) for (int z = 0; z < L[2]; ++z) for (int y = 0; y < L[1]; ++y) for (int x = 0; x < L[0]; ++x) {
            if (((x + y + z + t) & 1) != pat) continue;
            outc.push_back(pack4(x, y, z, t));
            for (int l = 0; l < 8; ++l) {
                int cc[4] = {x, y, z, t};
                cc[l >> 1] += (l & 1) == 0 ? 1 : -1;
                const auto it = slot_of.find(pack4(cc[0] + 1, cc[1] + 1, cc[2] + 1, cc[3] + 1));
                if (it == slot_of.end()) MDWF_FAIL(c, MDWF_EINVAL, "internal: fp16 tile table is inconsistent");
                nbr.push_back((unsigned short)it->second);
            }
        }
        if ((int)outc.size() != tl.ns) MDWF_FAIL(c, MDWF_EINVAL, "internal: fp16 tile has %zu output sites, expected %d", outc.size(), tl.ns);
        tl.nip[pat] = nslot; tl.nrun[pat] = (int)runs.size();
        void *d0, *d1, *d2;
        MDWF_CUDA(c, cudaMalloc(&d0, outc.size() * 4));
        MDWF_CUDA(c, cudaMalloc(&d1, runs.size() * sizeof(int4)));
        MDWF_CUDA(c, cudaMalloc(&d2, nbr.size() * 2));
        MDWF_CUDA(c, cudaMemcpy(d0, outc.data(), outc.size() * 4, cudaMemcpyHostToDevice));
        MDWF_CUDA(c, cudaMemcpy(d1, runs.data(), runs.size() * sizeof(int4), cudaMemcpyHostToDevice));
        MDWF_CUDA(c, cudaMemcpy(d2, nbr.data(), nbr.size() * 2, cudaMemcpyHostToDevice));
        th->dev[3 * pat] = d0; th->dev[3 * pat + 1] = d1; th->dev[3 * pat + 2] = d2;
        tl.outc[pat] = (const int*)d0; tl.run[pat] = (const int4*)d1; tl.nbr[pat] = (const unsigned short*)d2;
    }
    const Plan16 pl = plan_tile16(L, rows, nw);
    tl.spw = pl.spw; tl.nst = pl.nst;
    tl.off_nbr = (int)pl.off_nbr; tl.off_links = (int)pl.off_links; tl.off_wpart = (int)pl.off_wpart; tl.off_epi = (int)pl.off_epi;
    tl.off_stage = (int)pl.off_stage; tl.stage_bytes = (int)pl.stage; tl.smem_total = (int)pl.smem;
    tl.dTx = make_fastdiv(tl.nT[0]); tl.dTy = make_fastdiv(tl.nT[1]); tl.dTt = make_fastdiv(tl.nT[3]);
    tl.zc_t = tl.nT[2]; tl.dTzs = make_fastdiv(tl.zc_t);
    build_vcode(tl.vcode);
    return MDWF_OK;
}

void free_tile16(Tile16Host* th) {
    for (int i = 0; i < 6; ++i) if (th->dev[i]) { cudaFree(th->dev[i]); th->dev[i] = nullptr; }
}

// Tile choice: among the boxes that divide the lattice and fit in shared memory (with at least two staging buffers),
// the one with the fewest input-site fetches per output site (ni/ns: 8 without any reuse, 5 for a 2^4 box, 4 for
// 4x4x2x2).  Warps per block: one per output site up to 16 (then 2..4 sites per warp).  mdwf_set_hop16_tile forces a box.
static int warps_for(int ns) { return ns >= 16 ? 16 : ns >= 8 ? 8 : 4; }
static int choose_tile16(mdwf_ctx* c, int rows, int L[4], int* nw_out) {
    const Geom& g = c->g;
    const int dims[4] = {g.X, g.Y, g.Z, g.T};
    const size_t cap = 227 * 1024 - 256;
    if (c->tile16_forced[0] > 0) {
        for (int d = 0; d < 4; ++d) L[d] = c->tile16_forced[d];
        for (int d = 0; d < 4; ++d) if (L[d] < 1 || dims[d] % L[d] || (d == 0 && (L[d] & 1))) MDWF_FAIL(c, MDWF_EINVAL, "forced fp16 tile does not divide the lattice");
        const int nw = c->tile16_nw > 0 ? c->tile16_nw : warps_for(L[0] * L[1] * L[2] * L[3] / 2);
        const Plan16 pf = plan_tile16(L, rows, nw);
        if (pf.smem > cap || pf.spw > 4) MDWF_FAIL(c, MDWF_EINVAL, "forced fp16 tile does not fit in shared memory (or has more than 4 sites per warp)");
        *nw_out = nw;
        return MDWF_OK;
    }
    double best = 1e30;
    L[0] = 0;
    for (int lx = 2; lx <= 8; lx += 2) for (int ly = 1; ly <= 8; ++ly) for (int lz = 1; lz <= 8; ++lz) for (int lt = 1; lt <= 8; ++lt) {
        if (dims[0] % lx || dims[1] % ly || dims[2] % lz || dims[3] % lt) continue;
        const int cand[4] = {lx, ly, lz, lt};
        const int nw = warps_for(lx * ly * lz * lt / 2);
        const Plan16 p = plan_tile16(cand, rows, nw);
        if (p.spw > 4 || p.smem > cap) continue;
        const double fetch = (double)std::max(p.nip[0], p.nip[1]) / p.ns;
        const double imbal = (double)((p.ns + nw - 1) / nw * nw) / p.ns;
        const double cost = fetch * (1.0 + 0.25 * (imbal - 1.0));
        if (cost < best - 1e-12) { best = cost; L[0] = lx; L[1] = ly; L[2] = lz; L[3] = lt; *nw_out = nw; }
    }
    if (!L[0]) MDWF_FAIL(c, MDWF_EINVAL, "no fp16 stencil tile fits in shared memory (%d rows per site)", rows);
    return MDWF_OK;
}

// tiles are cached per rhs interleave (the staging buffers hold RI * Ls rows per site)
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
// in L2, budget ~40 MB
static int pick_zc16(const Geom& g, const Tile16& tl, int nact) {
    int best = 1;
    for (int z = 1; z <= tl.nT[2]; ++z) {
        if (tl.nT[2] % z) continue;
        const double layer = (double)g.XH * g.Y * (z * tl.L[2]) * tl.L[3] * g.Ls * 48.0 * nact;   // nact rhs = groups x RI
        if (3.0 * layer <= 40.0e6) best = z;
    }
    return best;
}

int launch_hop_f16(mdwf_ctx* c, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st) {
    (void)fused;
    Tile16Host* th;
    int rc = get_tile16(c, a.in.ril, &th);
    if (rc) return rc;
    (void)recon;       // the stencil-ready links were decoded from the (prec 16, recon) format at load time
    if (!a.g.pl[0] || !a.g.pl[1]) MDWF_FAIL(c, MDWF_ESTATE, "internal: stencil-ready fp16 links missing");
    if (!a.in.m || !a.out.m || (a.xin.v && !a.xin.m) || a.sr.n < 1) MDWF_FAIL(c, MDWF_EINVAL, "internal: fp16 hop without field scales");
    if (a.out.ril != a.in.ril || (a.xin.v && a.xin.ril != a.in.ril)) MDWF_FAIL(c, MDWF_EINVAL, "internal: fp16 hop on fields with different rhs interleave");
    const int rows = c->g.Ls << a.in.ril;
    Tile16 tl = th->t;
    tl.zc_t = c->zc_forced > 0 && c->zc_forced % tl.L[2] == 0 && tl.nT[2] % (c->zc_forced / tl.L[2]) == 0 ? c->zc_forced / tl.L[2]
                                                                                                        : pick_zc16(c->g, tl, a.nact);
    tl.dTzs = make_fastdiv(tl.zc_t);
    const int grid = std::min(tl.ntiles, c->sm_count), block = th->nw * 32;
    auto kern = rows <= 16 ? hop16_kernel<1> : rows <= 32 ? hop16_kernel<2> : hop16_kernel<3>;
    if (rows > 48) MDWF_FAIL(c, MDWF_EINVAL, "internal: %d rows per site", rows);
    if (!c->attr_raised.count((const void*)kern)) {
        MDWF_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
        c->attr_raised.insert((const void*)kern);
    }
    kern<<<grid, block, tl.smem_total, st>>>(c->g, tl, a, dagger ? 1 : 0);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    c->partial_nblk = grid;
    return MDWF_OK;
}

}  // namespace mdwf
