// csrc/api.cu -- the C-ABI entry points declared in include/mdwf.h (context, gauge load, Dslash family,
// packed fields) and the composite even-odd operators built from the fused kernels.
#include "mdwf_host.h"
#include "mdwf_hop16.cuh"
#include <cmath>
#include <cstring>
#include <algorithm>
#include <map>
#include <cstdlib>

using namespace mdwf;

// ---------------------------------------------------------------------------------------------
// Ls x Ls chirality blocks (SURVEY 8 Notation): L+ [s][s-1] = 1, L+ [0][Ls-1] = -mf ; L- [s][s+1] = 1,
// L- [Ls-1][0] = -mf ; A = b5 + c5 L ; M5 = a + d L ; M5^-1 by its closed form
//   (M5^-1)+[s][s'] = kappa^{(s-s') mod Ls} (s >= s' ? 1 : -mf) / (a (1 + mf kappa^Ls)),  kappa = -d/a
//   (M5^-1)-[s][s'] = kappa^{(s'-s) mod Ls} (s' >= s ? 1 : -mf) / (a (1 + mf kappa^Ls)).
// dagger = transpose inside each chirality block.
// ---------------------------------------------------------------------------------------------
static void build_matrices(int Ls, double M5, double b5, double c5, double mf, std::vector<double> mats[MAT_COUNT]) {
    const double a = b5 * (4.0 - M5) + 1.0, d = c5 * (4.0 - M5) - 1.0, kappa = -d / a;
    const int n = Ls * Ls;
    std::vector<double> L[2], A[2], M[2], Mi[2], AMi[2];
    for (int ch = 0; ch < 2; ++ch) {
        L[ch].assign(n, 0.0);
        for (int s = 0; s < Ls; ++s) {
            if (ch == 0) { if (s >= 1) L[0][s * Ls + s - 1] += 1.0; else L[0][0 * Ls + Ls - 1] += -mf; }
            else { if (s + 1 < Ls) L[1][s * Ls + s + 1] += 1.0; else L[1][(Ls - 1) * Ls + 0] += -mf; }
        }
        A[ch].assign(n, 0.0);
        M[ch].assign(n, 0.0);
        Mi[ch].assign(n, 0.0);
        AMi[ch].assign(n, 0.0);
        const double den = a * (1.0 + mf * std::pow(kappa, Ls));
        for (int s = 0; s < Ls; ++s)
            for (int t = 0; t < Ls; ++t) {
                const double id = s == t ? 1.0 : 0.0;
                A[ch][s * Ls + t] = b5 * id + c5 * L[ch][s * Ls + t];
                M[ch][s * Ls + t] = a * id + d * L[ch][s * Ls + t];
                const int k = ch == 0 ? ((s - t) % Ls + Ls) % Ls : ((t - s) % Ls + Ls) % Ls;
                const bool nowrap = ch == 0 ? (s >= t) : (t >= s);
                Mi[ch][s * Ls + t] = std::pow(kappa, k) * (nowrap ? 1.0 : -mf) / den;
            }
        for (int s = 0; s < Ls; ++s)
            for (int t = 0; t < Ls; ++t) {
                double acc = 0.0;
                for (int k = 0; k < Ls; ++k) acc += A[ch][s * Ls + k] * Mi[ch][k * Ls + t];
                AMi[ch][s * Ls + t] = acc;
            }
    }
    // device layout Gt[chi][s'][s] = Mat_chi[s][s'] ; dagger: Mat_chi[s'][s]
    std::vector<double>* src[4] = {A, M, Mi, AMi};
    const int ids[4] = {MAT_A, MAT_M5, MAT_M5INV, MAT_AM5INV};
    for (int m = 0; m < 4; ++m) {
        mats[ids[m]].assign(2 * n, 0.0);
        mats[ids[m] + 4].assign(2 * n, 0.0);
        for (int ch = 0; ch < 2; ++ch)
            for (int s = 0; s < Ls; ++s)
                for (int t = 0; t < Ls; ++t) {
                    mats[ids[m]][ch * n + t * Ls + s] = src[m][ch][s * Ls + t];
                    mats[ids[m] + 4][ch * n + t * Ls + s] = src[m][ch][t * Ls + s];
                }
    }
}

// The structured form of the same operators that the kernels apply (LsOp, mdwf_hop.cuh).
static void build_lsops(int Ls, double M5, double b5, double c5, double mf, LsOp ops[MAT_COUNT]) {
    const double a = b5 * (4.0 - M5) + 1.0, d = c5 * (4.0 - M5) - 1.0, kappa = -d / a;
    LsOp base;
    base.kind = 1; base.dag = 0; base.c0 = 0; base.c1 = 0;
    base.kappa = kappa; base.inv_a = 1.0 / a; base.mf = mf;
    base.gfac = mf / (a * (1.0 + mf * std::pow(kappa, Ls)));
    for (int dag = 0; dag < 2; ++dag) {
        LsOp o = base;
        o.dag = dag;
        o.kind = 1; o.c0 = b5; o.c1 = c5; ops[MAT_A + 4 * dag] = o;
        o.kind = 1; o.c0 = a; o.c1 = d; ops[MAT_M5 + 4 * dag] = o;
        o.kind = 2; o.c0 = 0.0; o.c1 = 1.0; ops[MAT_M5INV + 4 * dag] = o;
        // (b5 + c5 L)/(a + d L) = c5/d + (b5 - c5 a/d) M5^-1 (d != 0; mdwf_create refuses 0 < |d| < 1e-4 |a|, where the two
        // coefficients would cancel to fewer digits than the fp32 epilogues carry);  d == 0: M5 = a, so A M5^-1 = A / a
        if (d != 0.0) { o.kind = 2; o.c0 = c5 / d; o.c1 = b5 - c5 * a / d; }
        else { o.kind = 1; o.c0 = b5 / a; o.c1 = c5 / a; }
        ops[MAT_AM5INV + 4 * dag] = o;
    }
}
// 2-norm bounds of the same operators (used only to choose fp16 scales, mdwf_device.cuh ScaleRule): |L| <= max(1, mf);
// |M5^-1| <= sqrt(|.|_1 |.|_inf) = max(1, mf) sum_k |kappa|^k / |a (1 + mf kappa^Ls)| from the closed form.
static void build_lsop_norms(int Ls, double M5, double b5, double c5, double mf, const LsOp ops[MAT_COUNT], double nrm[MAT_COUNT]) {
    const double a = b5 * (4.0 - M5) + 1.0, d = c5 * (4.0 - M5) - 1.0, kappa = -d / a;
    const double lmax = std::max(1.0, std::fabs(mf));
    double geo = 0.0;
    for (int k = 0; k < Ls; ++k) geo += std::pow(std::fabs(kappa), k);
    const double minv = lmax * geo / std::fabs(a * (1.0 + mf * std::pow(kappa, Ls)));
    for (int i = 0; i < MAT_COUNT; ++i)
        nrm[i] = std::fabs(ops[i].c0) + std::fabs(ops[i].c1) * (ops[i].kind == 2 ? minv : lmax);
}
// host emulation of apply_ls on one chirality column (for the self-test): out = op(v), v[s], chi 0 = P+
static void lsop_host(const LsOp& op, int Ls, int chi, const std::vector<double>& v, std::vector<double>& out) {
    out.assign(Ls, 0.0);
    if (op.kind == 1) {
        for (int s = 0; s < Ls; ++s) {
            const int sm = s == 0 ? Ls - 1 : s - 1, sp = s == Ls - 1 ? 0 : s + 1;
            const double fm = s == 0 ? -op.mf : 1.0, fp = s == Ls - 1 ? -op.mf : 1.0;
            const bool take_minus = (chi == 0) != (op.dag != 0);      // P+ takes s-1 (L), s+1 (L^dag)
            out[s] = op.c0 * v[s] + op.c1 * (take_minus ? fm * v[sm] : fp * v[sp]);
        }
        return;
    }
    const bool fwd = (chi == 0) != (op.dag != 0);
    std::vector<double> P(Ls);
    double run = 0.0;
    for (int k = 0; k < Ls; ++k) { const int s = fwd ? k : Ls - 1 - k; run = v[s] + op.kappa * run; P[s] = run; }
    const double T = P[fwd ? Ls - 1 : 0];
    for (int s = 0; s < Ls; ++s) {
        const int k = fwd ? s : Ls - 1 - s;
        out[s] = op.c0 * v[s] + op.c1 * (op.inv_a * P[s] - op.gfac * std::pow(op.kappa, k + 1) * T);
    }
}

// z-slab depth (per storage precision): largest multiple of the tile depth tz dividing Z whose input slab
// XH*Y*zc*Ls*(bytes per site) stays under ~9 MB, so that the three t-consecutive slabs a row of tiles touches (plus
// the streamed output) live in L2 (measured on B200, 48^3x64 Ls=10: fp32 fastest at zc = 8,
// fp64 at zc = 4, fp16 flat between 2 and 16)
static int pick_zc(const mdwf_ctx* c, const Geom& g, int want, double site_bytes) {
    (void)c;
    if (want > 0 && g.Z % want == 0 && want % g.tz == 0) return want;
    int best = 0;
    for (int z = g.tz; z <= g.Z; z += g.tz)
        if (g.Z % z == 0 && (best == 0 || (double)g.XH * g.Y * z * g.Ls * site_bytes <= 9.0e6)) best = z;
    return best;
}
static void fill_zc(mdwf_ctx* c, Geom& g, int zc) {
    g.zc = zc;
    g.dZc = make_fastdiv(zc);
    g.dSlab = make_fastdiv((uint32_t)(g.XH * g.Y * zc));
    g.dTslab = make_fastdiv((uint32_t)(g.XH * g.Y * zc) * (uint32_t)g.T);
    g.dnTzs = make_fastdiv((uint32_t)(zc / g.tz));
    g.ntc = (g.XH / g.txh) * (g.Y / g.ty) * (zc / g.tz);
    g.dntc = make_fastdiv((uint32_t)g.ntc);
    (void)c;
}
static const double kSiteBytes[3] = {48.0, 96.0, 192.0};
namespace mdwf {
void set_zc(mdwf_ctx* c, int want) {
    c->zc_forced = want > 0 ? want : 0;
    c->ghop_multi.clear();
    for (int cls = 0; cls < 3; ++cls) fill_zc(c, c->ghop[cls], pick_zc(c, c->ghop[cls], want, kSiteBytes[cls]));
    c->g = c->ghop[1];
}
// Geometry of a hop launch.  Slab depth: forced (mdwf_set_tiling) > tuned (mdwf_autotune) > heuristic; with nact rhs in
// flight the slab working set is nact times larger, so the heuristic is evaluated for nact * (bytes per site)
const Geom& hop_geom(mdwf_ctx* c, int cls, int nact) {
    if (c->zc_forced > 0) return c->ghop[cls];
    const int key = cls * 100 + nact;
    auto it = c->ghop_multi.find(key);
    if (it != c->ghop_multi.end()) return it->second;
    auto tu = c->tune.find(tune_key_zc(c, cls, nact));
    if (tu == c->tune.end() && nact <= 1) return c->ghop[cls];
    Geom g = c->ghop[cls];
    const int want = tu != c->tune.end() && !tu->second.empty() ? tu->second[0] : 0;   // pick_zc ignores an inadmissible value
    fill_zc(c, g, pick_zc(c, g, want, kSiteBytes[cls] * std::max(1, nact)));
    return c->ghop_multi.emplace(key, g).first->second;
}
}  // namespace mdwf
// Sites of a block: a box txh*ty*tz*tt (x fastest) that divides the lattice, filled greedily along x, then y, z, t
// up to `cap` sites, i.e. (nearly) whole x-rows in storage order.  Compact 4D boxes (e.g. 4x4x2x2) were measured
// SLOWER on B200 (profiles/README.md, "tile shape").  cap: min(256/Ls, 32) sites for fp32/fp64 storage, min(128/Ls, 32)
// for fp16 -- the issue-bound fp16 kernels stall less at their block barriers with ~128-thread blocks (measured
// -5..7 % on the fused kernels), while fp32 prefers the larger ones.
static void pick_tile(Geom& g, int cap) {
    cap = std::max(1, cap);
    int best[4] = {1, 1, 1, 1};
    const int ext[4] = {g.XH, g.Y, g.Z, g.T};
    int n = 1;
    for (int d = 0; d < 4; ++d) {
        int pick = 1;
        for (int k = 1; k <= ext[d] && n * k <= cap; ++k)
            if (ext[d] % k == 0) pick = k;
        best[d] = pick;
        n *= pick;
        if (pick != ext[d]) break;   // only extend into the next direction when this one is covered completely
    }
    g.txh = best[0]; g.ty = best[1]; g.tz = best[2]; g.tt = best[3];
    g.nsite = g.txh * g.ty * g.tz * g.tt;
    g.dtxh = make_fastdiv(g.txh); g.dty = make_fastdiv(g.ty); g.dtz = make_fastdiv(g.tz);
    g.dnTx = make_fastdiv(g.XH / g.txh); g.dnTy = make_fastdiv(g.Y / g.ty); g.dnTt = make_fastdiv(g.T / g.tt);
}

static void prof_drain(mdwf_ctx* c) {
    for (size_t i = 0; i < c->prof_pending.size(); ++i) {
        mdwf_ctx::ProfRec& r = c->prof_pending[i];
        float ms = 0.f;
        if (cudaEventSynchronize(r.e1) == cudaSuccess && cudaEventElapsedTime(&ms, r.e0, r.e1) == cudaSuccess) {
            c->prof_ms[r.cls] += ms; c->prof_bytes[r.cls] += r.bytes; c->prof_flops[r.cls] += r.flops; c->prof_n[r.cls]++;
        }
        c->prof_pool.push_back(r.e0);
        c->prof_pool.push_back(r.e1);
    }
    c->prof_pending.clear();
}

extern "C" {

int mdwf_create(mdwf_ctx** out, const mdwf_geometry* geo, double M5, double b5, double c5, double mf) {
    if (!out || !geo) return MDWF_EINVAL;
    *out = nullptr;
    mdwf_ctx* c = new mdwf_ctx;
    c->geo = *geo;
    c->M5 = M5; c->b5 = b5; c->c5 = c5; c->mf = mf;
    c->partial = nullptr; c->dscal = nullptr; c->hscal = nullptr; c->launches = 0; c->prof_on = 0; c->zc_forced = 0;
    c->tile16[0] = c->tile16[1] = c->tile16[2] = nullptr; c->tile16_nw = 0; c->partial_nblk = 0; c->partial_cap = 0;
    c->ws = nullptr; c->ws_bytes = 0; c->ws_external = false;
    c->dctl = nullptr; c->hctl_stage = nullptr; c->hctl = nullptr;
    for (int i = 0; i < 4; ++i) c->tile16_forced[i] = 0;
    for (int i = 0; i < 8; ++i) { c->prof_ms[i] = c->prof_bytes[i] = c->prof_flops[i] = 0.0; c->prof_n[i] = 0; }
    *out = c;   // returned even on failure so that mdwf_last_error can be read; caller destroys it
    long long v4 = 1;
    for (int m = 0; m < 4; ++m) {
        if (geo->dims[m] < 2 || (geo->dims[m] & 1)) MDWF_FAIL(c, MDWF_EINVAL, "extent %d of direction %d must be even and >= 2", geo->dims[m], m);
        if (geo->bc[m] != 1 && geo->bc[m] != -1) MDWF_FAIL(c, MDWF_EINVAL, "bc[%d] must be +1 or -1", m);
        v4 *= geo->dims[m];
    }
    if (geo->Ls < 1 || geo->Ls > 32) MDWF_FAIL(c, MDWF_EINVAL, "Ls must be in 1..32 (got %d)", geo->Ls);
    if (v4 / 2 * geo->Ls >= (1ll << 31) / 2) MDWF_FAIL(c, MDWF_EINVAL, "lattice too large for 32-bit 5D site indices");
    const double a = b5 * (4.0 - M5) + 1.0, dd = c5 * (4.0 - M5) - 1.0;
    if (a == 0.0) MDWF_FAIL(c, MDWF_EINVAL, "b5(4-M5)+1 must be non-zero");
    // M5 = a + d L is inverted through its closed form: kappa = -d/a must contract and 1 + mf kappa^Ls must not vanish
    if (!(std::fabs(dd / a) < 1.0)) MDWF_FAIL(c, MDWF_EINVAL, "|c5(4-M5)-1| must be smaller than |b5(4-M5)+1| (kappa = %.4g)", -dd / a);
    if (!(std::fabs(1.0 + mf * std::pow(-dd / a, geo->Ls)) > 1e-8)) MDWF_FAIL(c, MDWF_EINVAL, "1 + mf kappa^Ls vanishes: M5 is singular");
    if (dd != 0.0 && std::fabs(dd) < 1e-4 * std::fabs(a)) MDWF_FAIL(c, MDWF_EINVAL, "c5(4-M5)-1 = %.3g is too close to (but not) zero for the fused A M5^-1 epilogue", dd);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        MDWF_FAIL(c, MDWF_ECUDA, "no CUDA device: libmdwf has no CPU fallback");
    }
    if (geo->device < 0 || geo->device >= ndev) MDWF_FAIL(c, MDWF_EINVAL, "device %d out of range (%d devices)", geo->device, ndev);
    MDWF_CUDA(c, cudaSetDevice(geo->device));
    cudaDeviceProp prop;
    MDWF_CUDA(c, cudaGetDeviceProperties(&prop, geo->device));
    c->sm_count = prop.multiProcessorCount;
    Geom& g = c->g;
    g.X = geo->dims[0]; g.Y = geo->dims[1]; g.Z = geo->dims[2]; g.T = geo->dims[3];
    g.XH = g.X / 2; g.Ls = geo->Ls;
    g.Vh = (int)(v4 / 2);
    g.N5h = g.Vh * g.Ls;
    for (int m = 0; m < 4; ++m) g.bc[m] = geo->bc[m];
    g.dLs = make_fastdiv(g.Ls); g.dXH = make_fastdiv(g.XH); g.dY = make_fastdiv(g.Y); g.dZ = make_fastdiv(g.Z);
    pick_tile(g, std::min(256 / g.Ls, 32));
    int max_nblk = 0;
    for (int cls = 0; cls < 3; ++cls) {
        c->ghop[cls] = g;
        if (cls == 0) pick_tile(c->ghop[cls], std::min(128 / g.Ls, 32));   // blocks of the site-local fp16 kernels (measured: ~128 threads)
        c->blk_cls[cls] = c->ghop[cls].nsite * g.Ls;
        c->nblk_cls[cls] = g.Vh / c->ghop[cls].nsite;
        max_nblk = std::max(max_nblk, c->nblk_cls[cls]);
    }
    c->block = c->blk_cls[1];
    c->nblk = c->nblk_cls[1];
    set_zc(c, 0);
    c->partial_cap = std::max<size_t>((size_t)max_nblk, (size_t)(g.N5h + 255) / 256 + 1);
    c->partial_cap = std::max<size_t>(c->partial_cap, (size_t)c->sm_count * 4);
    MDWF_CUDA(c, cudaMalloc(&c->partial, sizeof(double) * 64 * c->partial_cap));
    MDWF_CUDA(c, cudaMalloc(&c->dscal, sizeof(double) * 16 * 64));
    MDWF_CUDA(c, cudaMemset(c->dscal, 0, sizeof(double) * 16 * 64));
    MDWF_CUDA(c, cudaHostAlloc(&c->hscal, sizeof(double) * 16 * 64, cudaHostAllocDefault));
    MDWF_CUDA(c, cudaMalloc(&c->dctl, sizeof(CgCtl)));
    MDWF_CUDA(c, cudaMemset(c->dctl, 0, sizeof(CgCtl)));
    MDWF_CUDA(c, cudaHostAlloc(&c->hctl_stage, sizeof(CgCtl), cudaHostAllocDefault));
    MDWF_CUDA(c, cudaHostAlloc(&c->hctl, sizeof(CgCtlHost), cudaHostAllocDefault));
    memset((void*)c->hctl, 0, sizeof(CgCtlHost));
    build_lsops(g.Ls, M5, b5, c5, mf, c->lsop);
    build_lsop_norms(g.Ls, M5, b5, c5, mf, c->lsop, c->lsop_norm);
    return MDWF_OK;
}

int mdwf_destroy(mdwf_ctx* c) {
    if (!c) return MDWF_OK;
    for (size_t i = 0; i < c->gauges.size(); ++i) free_gauge(&c->gauges[i]);
    for (auto& kv : c->temps) for (mdwf_field* f : kv.second) free_field(f);
    for (int i = 0; i < 3; ++i) if (c->tile16[i]) { free_tile16(c->tile16[i]); delete c->tile16[i]; c->tile16[i] = nullptr; }
    if (c->ws && !c->ws_external) cudaFree(c->ws);
    if (c->dctl) cudaFree(c->dctl);
    if (c->hctl_stage) cudaFreeHost(c->hctl_stage);
    if (c->hctl) cudaFreeHost((void*)c->hctl);
    prof_drain(c);
    for (cudaEvent_t e : c->prof_pool) cudaEventDestroy(e);
    if (c->partial) cudaFree(c->partial);
    if (c->dscal) cudaFree(c->dscal);
    if (c->hscal) cudaFreeHost(c->hscal);
    delete c;
    return MDWF_OK;
}

const char* mdwf_last_error(const mdwf_ctx* c) { return c ? c->err.c_str() : "null context"; }
int64_t mdwf_launch_count(const mdwf_ctx* c) { return c ? c->launches : 0; }

int mdwf_profile(mdwf_ctx* c, int enable) {
    MDWF_ENTER(c);
    prof_drain(c);
    if (enable) for (int i = 0; i < 8; ++i) { c->prof_ms[i] = c->prof_bytes[i] = c->prof_flops[i] = 0.0; c->prof_n[i] = 0; }
    c->prof_on = enable ? 1 : 0;
    return MDWF_OK;
}
int mdwf_profile_read(mdwf_ctx* c, int cls, double* ms, double* bytes, double* flops, int64_t* launches) {
    MDWF_ENTER(c);
    if (cls < 0 || cls > 7 || !ms || !bytes || !flops || !launches) return MDWF_EINVAL;
    prof_drain(c);
    *ms = c->prof_ms[cls]; *bytes = c->prof_bytes[cls]; *flops = c->prof_flops[cls]; *launches = c->prof_n[cls];
    return MDWF_OK;
}

int mdwf_selftest_host(double M5, double b5, double c5, double mf) {
    // 1: fast division
    const uint32_t ds[] = {1, 2, 3, 4, 5, 6, 7, 8, 10, 12, 16, 21, 24, 25, 32, 48, 96, 250, 1152, 9216, 55296, 442368, 3538944};
    for (uint32_t d : ds) {
        const FastDiv f = make_fastdiv(d);
        for (uint32_t n = 0; n < 3000000u; ++n) if (f.div(n) != n / d) return 1;
        for (uint64_t n = 3000000u; n < (1ull << 31); n += 9973) if (f.div((uint32_t)n) != (uint32_t)n / d) return 1;
        if (f.div((1u << 31) - 1) != ((1u << 31) - 1) / d) return 1;
    }
    // 2, 3: s-direction blocks
    const double a = b5 * (4.0 - M5) + 1.0, d = c5 * (4.0 - M5) - 1.0;
    (void)a; (void)d;
    for (int Ls = 1; Ls <= 32; ++Ls) {
        std::vector<double> m[MAT_COUNT];
        build_matrices(Ls, M5, b5, c5, mf, m);
        const int n = Ls * Ls;
        for (int ch = 0; ch < 2; ++ch)
            for (int s = 0; s < Ls; ++s)
                for (int t = 0; t < Ls; ++t) {
                    double acc = 0.0, acc2 = 0.0;   // (M5 M5inv)[s][t], (A M5inv)[s][t]; Gt[chi][s'][s] = Mat[s][s']
                    for (int k = 0; k < Ls; ++k) {
                        acc += m[MAT_M5][ch * n + k * Ls + s] * m[MAT_M5INV][ch * n + t * Ls + k];
                        acc2 += m[MAT_A][ch * n + k * Ls + s] * m[MAT_M5INV][ch * n + t * Ls + k];
                    }
                    if (std::fabs(acc - (s == t ? 1.0 : 0.0)) > 1e-13) return 2;
                    if (std::fabs(acc2 - m[MAT_AM5INV][ch * n + t * Ls + s]) > 1e-13) return 2;
                    for (int id = 0; id < 4; ++id)
                        if (m[id + 4][ch * n + t * Ls + s] != m[id][ch * n + s * Ls + t]) return 3;
                }
        // 4: the structured operators the kernels apply reproduce the dense blocks column by column
        LsOp ops[MAT_COUNT];
        build_lsops(Ls, M5, b5, c5, mf, ops);
        for (int id = 0; id < MAT_COUNT; ++id)
            for (int ch = 0; ch < 2; ++ch)
                for (int t = 0; t < Ls; ++t) {
                    std::vector<double> e(Ls, 0.0), o;
                    e[t] = 1.0;
                    lsop_host(ops[id], Ls, ch, e, o);
                    for (int s = 0; s < Ls; ++s)
                        if (std::fabs(o[s] - m[id][ch * n + t * Ls + s]) > 1e-12) return 4;
                }
    }
    return 0;
}

int mdwf_set_tiling(mdwf_ctx* c, int zc) {
    MDWF_ENTER(c);
    if (zc < 0 || (zc > 0 && (c->g.Z % zc != 0 || zc % c->ghop[1].tz != 0 || zc % c->ghop[2].tz != 0)))
        MDWF_FAIL(c, MDWF_EINVAL, "zc = %d must divide Z = %d and be a multiple of the tile depth %d", zc, c->g.Z, c->g.tz);
    set_zc(c, zc);
    return MDWF_OK;
}

int mdwf_load_gauge(mdwf_ctx* c, const void* U, int store_prec, int recon, void* stream) {
    MDWF_ENTER(c);
    if (!U) MDWF_FAIL(c, MDWF_EINVAL, "null gauge pointer");
    GaugeSet gs;
    int rc = pack_gauge(c, U, store_prec, recon, &gs, (cudaStream_t)stream);
    if (rc) return rc;
    for (size_t i = 0; i < c->gauges.size(); ++i)
        if (c->gauges[i].prec == store_prec && c->gauges[i].recon == recon) {
            free_gauge(&c->gauges[i]);
            c->gauges[i] = gs;
            return MDWF_OK;
        }
    c->gauges.push_back(gs);
    return MDWF_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
namespace mdwf {

static SpinorView no_view() {
    SpinorView v;
    memset(&v, 0, sizeof(v));
    return v;
}

int op_ls(const OpCtx& o, mdwf_field* out, const mdwf_field* in, int mat, const mdwf_field* xin, double cx,
          double ch, const RhsList& rl, double* partial, int write) {
    LsArgs a;
    a.out = out->view(); a.in = in->view();
    a.xin = xin ? xin->view() : no_view();
    if (mat >= 0) a.op = o.c->lsop[mat]; else a.op.kind = 0;
    a.cx = cx; a.ch = ch; a.partial = partial; a.write = write; a.rl = rl; a.stop = o.stop;
    a.sr = write ? rule_lin(out, in, std::fabs(ch) * (mat >= 0 ? o.c->lsop_norm[mat] : 1.0), xin, std::fabs(cx)) : rule_lin(nullptr, nullptr, 0.0);
    const int rc = launch_ls(o.c, o.prec, a, o.st);
    if (write) out->flip();
    return rc;
}

int op_hop(const OpCtx& o, mdwf_field* out, const mdwf_field* in, int out_par, int dagger, int mat,
           const mdwf_field* xin, double cx, double ch, const RhsList& rl, double* partial) {
    HopArgs a;
    a.out = out->view(); a.in = in->view();
    a.xin = xin ? xin->view() : no_view();
    a.g.v[0] = o.gs->v[0]; a.g.v[1] = o.gs->v[1];
    a.g.pl[0] = o.gs->pl[0]; a.g.pl[1] = o.gs->pl[1];
    if (mat >= 0) a.op = o.c->lsop[mat]; else { a.op = o.c->lsop[0]; a.op.kind = 0; }
    a.cx = cx; a.ch = ch; a.partial = partial; a.par = out_par; a.nact = rl.nact; a.stop = o.stop;
    for (int i = 0; i < 64; ++i) a.rhs_list[i] = rl.rhs[i];
    // |H_{p<-pbar}| <= 8: each of the 8 legs is (1 -+ gamma_mu) x unitary = 2 x (projector x unitary)
    a.sr = rule_lin(out, in, 8.0 * std::fabs(ch) * (mat >= 0 ? o.c->lsop_norm[mat] : 1.0), xin, std::fabs(cx));
    const int fused = (mat >= 0 || xin || partial || ch != 1.0) ? 1 : 0;
    const int rc = launch_hop(o.c, o.prec, o.recon, dagger, fused, a, o.st);
    out->flip();
    return rc;
}

// Dhat = M5 - 1/4 H A M5^-1 H A,  Mhat = M5^-1 Dhat,  and their adjoints (SURVEY 8 "Even-odd form"):
//   Mhat v     : t1 = A v ; t2 = (A M5^-1) H t1 ; out = v - 1/4 M5^-1 H t2
//   Dhat v     : t1 = A v ; t2 = (A M5^-1) H t1 ; t1 = M5 v ; out = t1 - 1/4 H t2
//   Mhat^dag v : t1 = M5^-dag v ; t2 = (A M5^-1)^dag H^dag t1 ; out = v - 1/4 A^dag H^dag t2
//   Dhat^dag v : t2 = (A M5^-1)^dag H^dag v ; t1 = M5^dag v ; out = t1 - 1/4 A^dag H^dag t2
int op_schur(const OpCtx& o, mdwf_field* out, const mdwf_field* in, int par, int dagger, int symmetric,
             mdwf_field* t1, mdwf_field* t2, const RhsList& rl, double* partial, int first_factor_done) {
    int rc;
    if (!dagger) {
        if (!first_factor_done && (rc = op_ls(o, t1, in, MAT_A, nullptr, 0.0, 1.0, rl))) return rc;
        if ((rc = op_hop(o, t2, t1, 1 - par, 0, MAT_AM5INV, nullptr, 0.0, 1.0, rl))) return rc;
        if (symmetric) return op_hop(o, out, t2, par, 0, MAT_M5INV, in, 1.0, -0.25, rl, partial);
        if ((rc = op_ls(o, t1, in, MAT_M5, nullptr, 0.0, 1.0, rl))) return rc;
        return op_hop(o, out, t2, par, 0, -1, t1, 1.0, -0.25, rl, partial);
    }
    if (symmetric) {
        if ((rc = op_ls(o, t1, in, MAT_M5INV_D, nullptr, 0.0, 1.0, rl))) return rc;
        if ((rc = op_hop(o, t2, t1, 1 - par, 1, MAT_AM5INV_D, nullptr, 0.0, 1.0, rl))) return rc;
        return op_hop(o, out, t2, par, 1, MAT_A_D, in, 1.0, -0.25, rl, partial);
    }
    if ((rc = op_hop(o, t2, in, 1 - par, 1, MAT_AM5INV_D, nullptr, 0.0, 1.0, rl))) return rc;
    if ((rc = op_ls(o, t1, in, MAT_M5_D, nullptr, 0.0, 1.0, rl))) return rc;
    return op_hop(o, out, t2, par, 1, MAT_A_D, t1, 1.0, -0.25, rl, partial);
}

static int make_opctx(mdwf_ctx* c, int prec, int recon, cudaStream_t st, OpCtx* o) {
    o->c = c; o->prec = prec; o->recon = recon; o->st = st;
    o->gs = c->find_gauge(prec, recon);
    if (!o->gs) MDWF_FAIL(c, MDWF_ESTATE, "gauge format (prec %d, recon %d) not loaded: call mdwf_load_gauge first", prec, recon);
    return MDWF_OK;
}

static int dslash_packed_impl(mdwf_ctx* c, int op, int parity, int dagger, int recon, mdwf_field* out,
                              const mdwf_field* in, cudaStream_t st) {
    if (!out || !in) MDWF_FAIL(c, MDWF_EINVAL, "null field");
    if (out->prec != in->prec || out->nrhs != in->nrhs) MDWF_FAIL(c, MDWF_EINVAL, "in/out fields differ in precision or nrhs");
    if (out->v == in->v) MDWF_FAIL(c, MDWF_EINVAL, "out must not alias in");
    if (parity != 0 && parity != 1) MDWF_FAIL(c, MDWF_EINVAL, "parity must be 0 or 1");
    const int prec = in->prec, nrhs = in->nrhs;
    const RhsList rl = all_rhs(nrhs);
    OpCtx o;
    o.c = c; o.prec = prec; o.recon = recon; o.st = st; o.gs = nullptr;
    const bool needs_gauge = !(op == MDWF_OP_M4PRE || op == MDWF_OP_M5 || op == MDWF_OP_M5INV);
    int rc;
    if (needs_gauge && (rc = make_opctx(c, prec, recon, st, &o))) return rc;
    const int dg = dagger ? 4 : 0;
    switch (op) {
        case MDWF_OP_HOP: return op_hop(o, out, in, parity, dagger, -1, nullptr, 0.0, 1.0, rl);
        case MDWF_OP_M4PRE: return op_ls(o, out, in, MAT_A + dg, nullptr, 0.0, 1.0, rl);
        case MDWF_OP_M5: return op_ls(o, out, in, MAT_M5 + dg, nullptr, 0.0, 1.0, rl);
        case MDWF_OP_M5INV: return op_ls(o, out, in, MAT_M5INV + dg, nullptr, 0.0, 1.0, rl);
        case MDWF_OP_DHAT_ASYM:
        case MDWF_OP_DHAT_SYM: {
            mdwf_field *t1, *t2;
            if ((rc = temp_field(c, prec, nrhs, 2, &t1)) || (rc = temp_field(c, prec, nrhs, 3, &t2))) return rc;
            return op_schur(o, out, in, parity, dagger, op == MDWF_OP_DHAT_SYM, t1, t2, rl);
        }
        case MDWF_OP_NORMAL_ASYM:
        case MDWF_OP_NORMAL_SYM: {
            mdwf_field *t1, *t2, *t3;
            if ((rc = temp_field(c, prec, nrhs, 2, &t1)) || (rc = temp_field(c, prec, nrhs, 3, &t2)) ||
                (rc = temp_field(c, prec, nrhs, 4, &t3))) return rc;
            const int sym = op == MDWF_OP_NORMAL_SYM;
            if ((rc = op_schur(o, t3, in, parity, 0, sym, t1, t2, rl))) return rc;
            return op_schur(o, out, t3, parity, 1, sym, t1, t2, rl);
        }
    }
    MDWF_FAIL(c, MDWF_EINVAL, "unknown or non-packed op %d", op);
}

}  // namespace mdwf

namespace mdwf {
// canonical fp64 <-> packed field (half lattice: full = 0; one parity of a full-lattice field: full = 1)
int pack_field(mdwf_field* f, const double* canon, int full, int par, cudaStream_t st) {
    PackArgs a;
    memset(&a, 0, sizeof(a));
    a.f = f->view(); a.canon = const_cast<double*>(canon); a.Vc = (full ? 2ll : 1ll) * f->ctx->g.Vh; a.full = full; a.par = par;
    a.nrhs = f->nrhs; a.rhs0 = 0;
    a.sr.out = f->wmeta();
    const int rc = launch_pack(f->ctx, f->prec, false, a, st);
    f->flip();
    return rc;
}
// one rhs column, s-slices [s0, s0 + ns) of one parity <-> a full-lattice canonical buffer [ns][V][4][3] (host-buffer solves
// stream a right-hand side through a small staging buffer this way); fp64 / fp32 fields only
int pack_slices(mdwf_field* f, int rhs, double* stage, int s0, int ns, int par, bool unpack, cudaStream_t st) {
    mdwf_ctx* c = f->ctx;
    if (f->prec == 16 || rhs < 0 || rhs >= f->nrhs || s0 < 0 || ns < 1 || s0 + ns > c->g.Ls) MDWF_FAIL(c, MDWF_EINVAL, "internal: bad slice pack");
    PackArgs a;
    memset(&a, 0, sizeof(a));
    a.f = f->view(); a.canon = stage; a.Vc = 2ll * c->g.Vh; a.full = 1; a.par = par; a.nrhs = 1; a.rhs0 = rhs; a.s0 = s0; a.ns = ns;
    return launch_pack(c, f->prec, unpack, a, st);
}
int unpack_field(const mdwf_field* f, double* canon, int full, int par, cudaStream_t st) {
    PackArgs a;
    memset(&a, 0, sizeof(a));
    a.f = f->view(); a.canon = canon; a.Vc = (full ? 2ll : 1ll) * f->ctx->g.Vh; a.full = full; a.par = par; a.nrhs = f->nrhs; a.rhs0 = 0;
    return launch_pack(f->ctx, f->prec, true, a, st);
}
}  // namespace mdwf

extern "C" {

int mdwf_set_hop16_tile(mdwf_ctx* c, int lx, int ly, int lz, int lt, int warps) {
    MDWF_ENTER(c);
    if (warps < 0 || warps > MDWF_H16_MAXW) MDWF_FAIL(c, MDWF_EINVAL, "warps must be in 0..%d", MDWF_H16_MAXW);
    for (int i = 0; i < 3; ++i) if (c->tile16[i]) { free_tile16(c->tile16[i]); delete c->tile16[i]; c->tile16[i] = nullptr; }
    c->tile16_forced[0] = lx; c->tile16_forced[1] = ly; c->tile16_forced[2] = lz; c->tile16_forced[3] = lt;
    c->tile16_nw = warps;
    return MDWF_OK;     // checked when the next fp16 stencil launch builds its tables
}

int mdwf_field_create(mdwf_ctx* c, int prec, int nrhs, mdwf_field** out) {
    MDWF_ENTER(c);
    if (!out) return MDWF_EINVAL;
    return alloc_field(c, prec, nrhs, out);
}
int mdwf_field_destroy(mdwf_field* f) {
    free_field(f);
    return MDWF_OK;
}
int mdwf_field_pack(mdwf_field* f, const void* canonical, void* stream) {
    if (!f || !canonical) return MDWF_EINVAL;
    return pack_field(f, (const double*)canonical, 0, 0, (cudaStream_t)stream);
}
int mdwf_field_unpack(const mdwf_field* f, void* canonical, void* stream) {
    if (!f || !canonical) return MDWF_EINVAL;
    return unpack_field(f, (double*)canonical, 0, 0, (cudaStream_t)stream);
}
// one column at a time (so that a large multi-rhs field can be filled from a single-rhs canonical buffer)
static int pack_one(mdwf_field* f, int rhs, double* canonical, bool unpack, cudaStream_t st) {
    mdwf_ctx* c = f->ctx;
    if (rhs < 0 || rhs >= f->nrhs) MDWF_FAIL(c, MDWF_EINVAL, "rhs %d out of range", rhs);
    if (f->prec == 16) MDWF_FAIL(c, MDWF_EINVAL, "column-wise packing is for fp64/fp32 fields (an fp16 field is scaled as a whole)");
    PackArgs a;
    memset(&a, 0, sizeof(a));
    a.f = f->view(); a.canon = canonical; a.Vc = c->g.Vh; a.full = 0; a.par = 0; a.nrhs = 1; a.rhs0 = rhs;
    return launch_pack(c, f->prec, unpack, a, st);
}
int mdwf_field_pack_rhs(mdwf_field* f, int rhs, const void* canonical, void* stream) {
    if (!f || !canonical) return MDWF_EINVAL;
    return pack_one(f, rhs, (double*)canonical, false, (cudaStream_t)stream);
}
int mdwf_field_unpack_rhs(const mdwf_field* f, int rhs, void* canonical, void* stream) {
    if (!f || !canonical) return MDWF_EINVAL;
    return pack_one(const_cast<mdwf_field*>(f), rhs, (double*)canonical, true, (cudaStream_t)stream);
}

int mdwf_dslash_packed(mdwf_ctx* c, int op, int parity, int dagger, int recon, mdwf_field* out,
                       const mdwf_field* in, void* stream) {
    MDWF_ENTER(c);
    return dslash_packed_impl(c, op, parity, dagger, recon, out, in, (cudaStream_t)stream);
}

int mdwf_dslash(mdwf_ctx* c, int op, int parity, int dagger, int prec, int recon, void* out, const void* in,
                int nrhs, void* stream) {
    MDWF_ENTER(c);
    if (!out || !in) MDWF_FAIL(c, MDWF_EINVAL, "null field pointer");
    if (nrhs < 1 || nrhs > MDWF_MAX_RHS) MDWF_FAIL(c, MDWF_EINVAL, "nrhs must be in 1..%d", MDWF_MAX_RHS);
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    if (op != MDWF_OP_FULL) {
        mdwf_field *fi, *fo;
        if ((rc = temp_field(c, prec, nrhs, 0, &fi)) || (rc = temp_field(c, prec, nrhs, 1, &fo))) return rc;
        if ((rc = mdwf_field_pack(fi, in, stream))) return rc;
        if ((rc = dslash_packed_impl(c, op, parity, dagger, recon, fo, fi, st))) return rc;
        return mdwf_field_unpack(fo, out, stream);
    }
    // FULL: D = M5 - 1/2 H A ; D^dag = M5^dag - 1/2 A^dag H^dag  (SURVEY 8 "Even-odd form")
    OpCtx o;
    if ((rc = make_opctx(c, prec, recon, st, &o))) return rc;
    mdwf_field *f[2], *fo, *t1, *t2;
    if ((rc = temp_field(c, prec, nrhs, 0, &f[0])) || (rc = temp_field(c, prec, nrhs, 5, &f[1])) ||
        (rc = temp_field(c, prec, nrhs, 1, &fo)) || (rc = temp_field(c, prec, nrhs, 2, &t1)) ||
        (rc = temp_field(c, prec, nrhs, 3, &t2))) return rc;
    const RhsList rl = all_rhs(nrhs);
    for (int p = 0; p < 2; ++p)
        if ((rc = pack_field(f[p], (const double*)in, 1, p, st))) return rc;
    for (int p = 0; p < 2; ++p) {
        mdwf_field *same = f[p], *other = f[1 - p];
        if (!dagger) {
            if ((rc = op_ls(o, t1, other, MAT_A, nullptr, 0.0, 1.0, rl))) return rc;
            if ((rc = op_ls(o, t2, same, MAT_M5, nullptr, 0.0, 1.0, rl))) return rc;
            if ((rc = op_hop(o, fo, t1, p, 0, -1, t2, 1.0, -0.5, rl))) return rc;
        } else {
            if ((rc = op_ls(o, t2, same, MAT_M5_D, nullptr, 0.0, 1.0, rl))) return rc;
            if ((rc = op_hop(o, fo, other, p, 1, MAT_A_D, t2, 1.0, -0.5, rl))) return rc;
        }
        if ((rc = unpack_field(fo, (double*)out, 1, p, st))) return rc;
    }
    return MDWF_OK;
}

// per 5D site and rhs, w = bytes per real,
//   hop: 1320 flop, 2*24*w + 8*R*w/(Ls*nrhs) bytes;  A, M5: 72 flop;  M5^-1: 48*Ls flop;
//   site-local ops: 2*24*w bytes;  Dhat/Mhat: 2832 + 96*Ls flop, fused floor 5 spinor passes + 2 link passes.
int mdwf_dslash_cost(const mdwf_ctx* c, int op, int prec, int recon, int nrhs, double* bytes, double* flops) {
    if (!c || !bytes || !flops) return MDWF_EINVAL;
    const double w = prec / 8.0, n5 = (double)c->g.N5h * nrhs, Ls = c->g.Ls;
    const double pass = 24.0 * w;
    const double links = 8.0 * recon * w * c->g.Vh;
    switch (op) {
        case MDWF_OP_HOP: *bytes = 2 * pass * n5 + links; *flops = 1320.0 * n5; return MDWF_OK;
        case MDWF_OP_M4PRE:
        case MDWF_OP_M5: *bytes = 2 * pass * n5; *flops = 72.0 * n5; return MDWF_OK;
        case MDWF_OP_M5INV: *bytes = 2 * pass * n5; *flops = 48.0 * Ls * n5; return MDWF_OK;
        case MDWF_OP_DHAT_ASYM:
        case MDWF_OP_DHAT_SYM: *bytes = 5 * pass * n5 + 2 * links; *flops = (2832.0 + 96.0 * Ls) * n5; return MDWF_OK;
        case MDWF_OP_NORMAL_ASYM:
        case MDWF_OP_NORMAL_SYM: *bytes = 2 * (5 * pass * n5 + 2 * links); *flops = 2 * (2832.0 + 96.0 * Ls) * n5; return MDWF_OK;
        case MDWF_OP_FULL: *bytes = 2 * (3 * pass * n5 + links); *flops = 2 * (1320.0 + 72.0 * 2 + 48.0) * n5; return MDWF_OK;
    }
    return MDWF_EINVAL;
}

}  // extern "C"
