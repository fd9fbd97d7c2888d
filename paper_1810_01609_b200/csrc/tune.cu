// csrc/tune.cu -- run-time launch-parameter autotuner with a cache ("GPU kernel autotuning ... QUDA performs a brute-force
// search over the launch parameters the first time a kernel is called and stores the optimum in a std::map ... written to
// disk", PAPER.md:92-94 IV).  Here the free launch parameters of the Dslash stencil are
//   fp16 storage (hop16_kernel):  the 4D tile of output sites a block owns and the warps per block,
//   fp32 / fp64 (hop_kernel):     the z-slab depth of the tile traversal (how much of the lattice one sweep keeps in L2),
// and the search is explicit (mdwf_autotune) instead of hidden in the first launch, so that no timed call ever contains
// it.  Candidates are timed with CUDA events on scratch fields of the real size -- the plain hop plus the fused hop of the
// CG iteration (M5^-1 epilogue, xpay, norm) -- and the fastest is kept in ctx->tune (std::map), used by every later
// launch (hop16.cu choose_tile16, api.cu hop_geom) and saved / loaded as text by mdwf_tune_save / mdwf_tune_load.
#include "mdwf_host.h"
#include "mdwf_hop16.cuh"
#include <cstdio>
#include <cstring>
#include <algorithm>
#include <sstream>
#include <fstream>

namespace mdwf {

static std::string lattice_key(const mdwf_ctx* c) {
    char b[96];
    snprintf(b, sizeof(b), "%dx%dx%dx%d/Ls%d", c->g.X, c->g.Y, c->g.Z, c->g.T, c->g.Ls);
    return b;
}
std::string tune_key_tile16(const mdwf_ctx* c, int rows) {
    return "hop16/" + lattice_key(c) + "/rows" + std::to_string(rows);
}
std::string tune_key_zc(const mdwf_ctx* c, int cls, int nact) {
    return std::string(cls == 1 ? "hop32/" : cls == 2 ? "hop64/" : "hop16zc/") + lattice_key(c) + "/rhs" + std::to_string(nact);
}
void tune_invalidate(mdwf_ctx* c) {
    c->ghop_multi.clear();
    for (int i = 0; i < 3; ++i)
        if (c->tile16[i]) { free_tile16(c->tile16[i]); delete c->tile16[i]; c->tile16[i] = nullptr; }
}

namespace {
struct Scratch {
    mdwf_field *in = nullptr, *out = nullptr, *x = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    ~Scratch() {
        free_field(in); free_field(out); free_field(x);
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    }
};
// finite, harmless contents: every byte 0x3c (half 1.06, float 0.0115, double 1.6e-15); fp16 scales and norm bounds 1
int fill(mdwf_ctx* c, mdwf_field* f, cudaStream_t st) {
    MDWF_CUDA(c, cudaMemsetAsync(f->v, 0x3c, f->bytes, st));
    if (f->meta) {
        FieldMeta m;
        for (int i = 0; i < 64; ++i) { m.e[i] = 1.0f; m.nb[i] = 1.0; }
        for (int k = 0; k < 2; ++k) MDWF_CUDA(c, cudaMemcpyAsync(f->meta + k, &m, sizeof(m), cudaMemcpyHostToDevice, st));
        MDWF_CUDA(c, cudaStreamSynchronize(st));        // `m` is on the stack
    }
    return MDWF_OK;
}
// milliseconds of `reps` x (plain hop + fused hop of the CG iteration) with the launch parameters in force
int time_hops(const OpCtx& o, Scratch& S, const RhsList& rl, int reps, float* ms) {
    mdwf_ctx* c = o.c;
    int rc;
    MDWF_CUDA(c, cudaEventRecord(S.e0, o.st));
    for (int k = 0; k < reps; ++k) {
        if ((rc = op_hop(o, S.out, S.in, 0, 0, -1, nullptr, 0.0, 1.0, rl))) return rc;
        if ((rc = op_hop(o, S.out, S.in, 0, 1, MAT_M5INV, S.x, 1.0, -0.25, rl, c->partial))) return rc;
    }
    MDWF_CUDA(c, cudaEventRecord(S.e1, o.st));
    MDWF_CUDA(c, cudaEventSynchronize(S.e1));
    MDWF_CUDA(c, cudaEventElapsedTime(ms, S.e0, S.e1));
    return MDWF_OK;
}
}  // namespace

int autotune_impl(mdwf_ctx* c, int prec, int recon, int nrhs, cudaStream_t st) {
    if (prec != 64 && prec != 32 && prec != 16) MDWF_FAIL(c, MDWF_EINVAL, "prec must be 64, 32 or 16");
    if (nrhs < 1 || nrhs > MDWF_MAX_RHS) MDWF_FAIL(c, MDWF_EINVAL, "nrhs must be in 1..%d", MDWF_MAX_RHS);
    OpCtx o;
    o.c = c; o.prec = prec; o.recon = recon; o.st = st;
    o.gs = c->find_gauge(prec, recon);
    if (!o.gs) MDWF_FAIL(c, MDWF_ESTATE, "gauge format (prec %d, recon %d) not loaded: call mdwf_load_gauge first", prec, recon);
    Scratch S;
    int rc;
    if ((rc = alloc_field(c, prec, nrhs, &S.in)) || (rc = alloc_field(c, prec, nrhs, &S.out)) || (rc = alloc_field(c, prec, nrhs, &S.x))) return rc;
    if ((rc = fill(c, S.in, st)) || (rc = fill(c, S.out, st)) || (rc = fill(c, S.x, st))) return rc;
    MDWF_CUDA(c, cudaEventCreate(&S.e0));
    MDWF_CUDA(c, cudaEventCreate(&S.e1));
    const RhsList rl = all_rhs(nrhs);
    // repetitions per candidate: at least 3, and enough for ~20 ms per candidate on small lattices (first candidate's time)
    int reps = 3;
    float best_ms = -1.f, ms = 0.f;
    auto set_reps = [&](float one_ms) { if (one_ms > 0.f) reps = std::max(3, std::min(100, (int)(20.f / one_ms))); };
    bool reps_set = false;
    std::vector<int> best;

    if (prec == 16) {
        const int rows = c->g.Ls << half_ril(nrhs, c->g.Ls);
        const std::string key = tune_key_tile16(c, rows);
        int saved[5];
        for (int d = 0; d < 4; ++d) saved[d] = c->tile16_forced[d];
        saved[4] = c->tile16_nw;
        static const int tiles[][4] = {{4, 4, 2, 2}, {4, 2, 2, 2}, {2, 2, 2, 2}, {8, 2, 2, 2}, {4, 4, 4, 2}, {8, 4, 2, 2}, {4, 4, 2, 4}, {2, 4, 2, 2}};
        static const int warps[] = {4, 8, 16};
        const int dims[4] = {c->g.X, c->g.Y, c->g.Z, c->g.T};
        for (const auto& t : tiles)
            for (int nw : warps) {
                bool ok = true;
                for (int d = 0; d < 4; ++d) ok = ok && dims[d] % t[d] == 0;
                const int ns = t[0] * t[1] * t[2] * t[3] / 2;
                if (!ok || nw > ns || (ns + nw - 1) / nw > 4) continue;
                for (int d = 0; d < 4; ++d) c->tile16_forced[d] = t[d];
                c->tile16_nw = nw;
                tune_invalidate(c);
                // a candidate that does not fit (shared memory) is refused by the launcher: skip it
                if (time_hops(o, S, rl, 1, &ms) != MDWF_OK) { cudaGetLastError(); c->err.clear(); continue; }
                if (!reps_set) { if (time_hops(o, S, rl, 1, &ms) == MDWF_OK) set_reps(ms); reps_set = true; }
                if (time_hops(o, S, rl, reps, &ms) != MDWF_OK) { cudaGetLastError(); c->err.clear(); continue; }
                if (best_ms < 0.f || ms < best_ms) { best_ms = ms; best = {t[0], t[1], t[2], t[3], nw}; }
            }
        for (int d = 0; d < 4; ++d) c->tile16_forced[d] = saved[d];
        c->tile16_nw = saved[4];
        tune_invalidate(c);
        if (best.empty()) MDWF_FAIL(c, MDWF_ESTATE, "autotune: no admissible fp16 tile for this lattice");
        c->tune[key] = best;
    } else {
        const int cls = cls_of(prec);
        const std::string key = tune_key_zc(c, cls, nrhs);
        const int saved = c->zc_forced, tz = c->ghop[cls].tz;
        for (int zc = tz; zc <= c->g.Z; zc += tz) {
            if (c->g.Z % zc || zc % c->ghop[1].tz || zc % c->ghop[2].tz) continue;
            set_zc(c, zc);
            if ((rc = time_hops(o, S, rl, 1, &ms))) { set_zc(c, saved); return rc; }
            if (!reps_set) { if ((rc = time_hops(o, S, rl, 1, &ms))) { set_zc(c, saved); return rc; } set_reps(ms); reps_set = true; }
            if ((rc = time_hops(o, S, rl, reps, &ms))) { set_zc(c, saved); return rc; }
            if (best_ms < 0.f || ms < best_ms) { best_ms = ms; best = {zc}; }
        }
        set_zc(c, saved);
        if (best.empty()) MDWF_FAIL(c, MDWF_ESTATE, "autotune: no admissible slab depth");
        c->tune[key] = best;
        c->ghop_multi.clear();
    }
    return MDWF_OK;
}

}  // namespace mdwf

extern "C" {

int mdwf_autotune(mdwf_ctx* c, int prec, int recon, int nrhs, void* stream) {
    MDWF_ENTER(c);
    return mdwf::autotune_impl(c, prec, recon, nrhs, (cudaStream_t)stream);
}

int mdwf_tune_save(mdwf_ctx* c, const char* path) {
    if (!c || !path) return MDWF_EINVAL;
    std::ofstream f(path);
    if (!f) MDWF_FAIL(c, MDWF_EINVAL, "cannot write %s", path);
    f << "# libmdwf launch parameters (mdwf_autotune): key values...\n";
    for (const auto& kv : c->tune) {
        f << kv.first;
        for (int v : kv.second) f << ' ' << v;
        f << '\n';
    }
    return f.good() ? MDWF_OK : MDWF_EINVAL;
}

int mdwf_tune_load(mdwf_ctx* c, const char* path) {
    if (!c || !path) return MDWF_EINVAL;
    std::ifstream f(path);
    if (!f) MDWF_FAIL(c, MDWF_EINVAL, "cannot read %s", path);
    std::string line;
    while (std::getline(f, line)) {
        if (line.empty() || line[0] == '#') continue;
        std::istringstream is(line);
        std::string key;
        is >> key;
        std::vector<int> v;
        int x;
        while (is >> x) v.push_back(x);
        if (key.empty() || v.empty() || v.size() > 8) MDWF_FAIL(c, MDWF_EINVAL, "malformed line in %s: %s", path, line.c_str());
        c->tune[key] = v;       // entries for other lattices are kept and simply never match
    }
    mdwf::tune_invalidate(c);
    return MDWF_OK;
}

int mdwf_tune_get(mdwf_ctx* c, const char* key, int* values, int cap) {
    if (!c || !key || !values) return MDWF_EINVAL;
    auto it = c->tune.find(key);
    if (it == c->tune.end()) return 0;
    const int n = (int)it->second.size();
    for (int i = 0; i < n && i < cap; ++i) values[i] = it->second[i];
    return n;
}

}
