// csrc/blas.cu -- launchers of the 4D-site-local kernels in mdwf_blas.cuh and the packed-field allocator.
#include "mdwf_hop_launch.cuh"
#include <cstring>

namespace mdwf {

// fp16: rhs interleave of a field with nrhs columns (log2): groups of RI = 4 when there are at least 3 rhs, of 2 for two,
// else 1, as far as the RI * Ls rows of a site stay within 48 = three m16 tiles of the tensor-core stencil.  Three rhs
// take a group of 4 with one padding slot: the stencil's cost per group grows much more slowly than its rows (measured at
// 48^3x64x10: 3.8 / 6.3 / 9.4 ms for groups of 1 / 2 / 4), so one padded group beats two groups of 2.
int half_ril(int nrhs, int Ls) {
    for (int ril = 2; ril > 0; --ril)
        if ((1 << ril) < 2 * nrhs && (Ls << ril) <= 48) return ril;
    return 0;
}
int half_site_bytes(int nrhs, int Ls) { return (((Ls << half_ril(nrhs, Ls)) + 7) / 8) * 384; }
static size_t rhs_bytes(const Geom& g, int prec, int nrhs) {      // stride between rhs (fp16: between rhs groups)
    // (+ 1536 bytes: the tensor-core stencil reads an even number of row blocks per site, mdwf_hop16.cuh)
    if (prec == 16) return ((size_t)g.Vh * half_site_bytes(nrhs, g.Ls) + 1536 + 255) / 256 * 256;
    const size_t nb = ((size_t)g.N5h + 31) / 32;
    return nb * (size_t)((24 * (prec / 8) / 16) * 512);
}
size_t field_bytes(const Geom& g, int prec, int nrhs) {
    if (prec == 16) {
        const int ri = 1 << half_ril(nrhs, g.Ls);
        return rhs_bytes(g, prec, nrhs) * ((nrhs + ri - 1) / ri);
    }
    return rhs_bytes(g, prec, nrhs) * nrhs;
}

static int make_field(mdwf_ctx* c, int prec, int nrhs, void* mem, void* meta_mem, mdwf_field** out) {
    if (prec != 64 && prec != 32 && prec != 16) MDWF_FAIL(c, MDWF_EINVAL, "prec must be 64, 32 or 16 (got %d)", prec);
    if (nrhs < 1 || nrhs > MDWF_MAX_RHS) MDWF_FAIL(c, MDWF_EINVAL, "nrhs must be in 1..%d (got %d)", MDWF_MAX_RHS, nrhs);
    mdwf_field* f = new mdwf_field;
    f->ctx = c;
    f->prec = prec;
    f->nrhs = nrhs;
    f->bytes = field_bytes(c->g, prec, nrhs);
    f->v = mem;
    f->meta = nullptr;
    f->cur = 0;
    f->rhs0 = 0;
    f->owns = mem == nullptr;
    f->owns_meta = false;
    f->rs = rhs_bytes(c->g, prec, nrhs);
    if (!mem) {
        cudaError_t e = cudaMalloc(&f->v, f->bytes);
        if (e == cudaErrorMemoryAllocation && c->ws && !c->ws_external) {
            // the solver workspace the library keeps between solves is only a cache: give it back and try again
            cudaGetLastError();
            cudaFree(c->ws);
            c->ws = nullptr; c->ws_bytes = 0;
            e = cudaMalloc(&f->v, f->bytes);
        }
        if (e == cudaSuccess && prec == 16) e = cudaMemset(f->v, 0, f->bytes);     // padding rhs of the last group
        if (e != cudaSuccess) {
            const size_t want = f->bytes;
            delete f;
            cudaGetLastError();
            MDWF_FAIL(c, MDWF_ENOMEM, "cudaMalloc of %zu bytes for a packed field failed: %s", want, cudaGetErrorString(e));
        }
    }
    if (prec == 16 && meta_mem) f->meta = reinterpret_cast<FieldMeta*>(meta_mem);
    else if (prec == 16) {
        f->owns_meta = true;
        cudaError_t e = cudaMalloc(&f->meta, 2 * sizeof(FieldMeta));
        if (e == cudaSuccess) e = cudaMemset(f->meta, 0, 2 * sizeof(FieldMeta));
        if (e != cudaSuccess) {
            if (f->owns) cudaFree(f->v);
            delete f;
            cudaGetLastError();
            MDWF_FAIL(c, MDWF_ENOMEM, "cudaMalloc of field scales failed: %s", cudaGetErrorString(e));
        }
    }
    *out = f;
    return MDWF_OK;
}
int alloc_field(mdwf_ctx* c, int prec, int nrhs, mdwf_field** out) { return make_field(c, prec, nrhs, nullptr, nullptr, out); }
int wrap_field(mdwf_ctx* c, int prec, int nrhs, void* mem, void* meta_mem, mdwf_field** out) { return make_field(c, prec, nrhs, mem, meta_mem, out); }
void free_field(mdwf_field* f) {
    if (!f) return;
    if (f->v && f->owns) cudaFree(f->v);
    if (f->meta && f->owns_meta) cudaFree(f->meta);
    delete f;
}
int temp_field(mdwf_ctx* c, int prec, int nrhs, int slot, mdwf_field** out) {
    std::vector<mdwf_field*>& v = c->temps[(long long)prec * 1000 + nrhs];
    while ((int)v.size() <= slot) v.push_back(nullptr);
    if (!v[slot]) {
        int rc = alloc_field(c, prec, nrhs, &v[slot]);
        if (rc) return rc;
    }
    *out = v[slot];
    return MDWF_OK;
}

ScaleRule rule_lin(const mdwf_field* out, const mdwf_field* a, double ca, const mdwf_field* b, double cb) {
    ScaleRule r;
    memset(&r, 0, sizeof(r));
    if (!out || !out->meta) return r;
    r.out = out->wmeta();
    if (a && a->meta) { r.t[r.n].nb = a->nb(); r.t[r.n].coef = ca; ++r.n; }
    if (b && b->meta) { r.t[r.n].nb = b->nb(); r.t[r.n].coef = cb; ++r.n; }
    return r;
}

// Grouped mode of a launch whose fields are fp16 with the rhs interleaved in groups of 1 << ril (mdwf_blas.cuh RhsList):
// the groups that hold an active rhs, their masks, and the blocks per group.
static int group_rhs(const Geom& g, RhsList& rl, int ril, int blk) {
    rl.ril = ril;
    rl.ng = 0;
    if (ril == 0) return -1;
    for (int k = 0; k < rl.nact; ++k) {
        const int gr = rl.rhs[k] >> ril;
        int j = 0;
        while (j < rl.ng && rl.grp[j] != gr) ++j;
        if (j == rl.ng) { rl.grp[j] = (unsigned char)gr; rl.gmask[j] = 0; ++rl.ng; }
        rl.gmask[j] |= (unsigned char)(1 << (rl.rhs[k] & ((1 << ril) - 1)));
        rl.slot_of[rl.rhs[k]] = (unsigned char)k;
    }
    const long long rows = (long long)g.Vh * (g.Ls << ril);
    return (int)((rows + blk - 1) / blk);      // blocks per group
}
// grid / partials per rhs of a site-local launch at storage precision `prec` whose fp16 fields have interleave ril
static void site_grid(mdwf_ctx* c, int prec, RhsList& rl, int ril, int* grid, int* blk, int* nblk) {
    *blk = c->blk_cls[cls_of(prec)];
    const int per_group = prec == 16 || ril > 0 ? group_rhs(c->g, rl, ril, *blk) : -1;
    if (per_group > 0) { *grid = per_group * rl.ng; *nblk = per_group; }
    else { rl.ril = 0; rl.ng = 0; *grid = c->nblk_cls[cls_of(prec)] * rl.nact; *nblk = c->nblk_cls[cls_of(prec)]; }
}

#define LAUNCH(kern, grid, blk, smem, ...)                              \
    do {                                                                \
        kern<<<(grid), (blk), (smem), st>>>(__VA_ARGS__);               \
        MDWF_CUDA(c, cudaGetLastError());                               \
        c->launches++;                                                  \
    } while (0)

template <typename K, typename A>
static int launch_big_smem(mdwf_ctx* c, K kern, int grid, int blk, size_t smem, cudaStream_t st, const A& a) {
    if (smem > 48 * 1024 && !c->attr_raised.count((const void*)kern)) {
        MDWF_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        c->attr_raised.insert((const void*)kern);
    }
    kern<<<grid, blk, smem, st>>>(c->g, a);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

template <typename S> static size_t g_smem(mdwf_ctx* c, bool useG) {
    typedef typename Store<S>::real T;
    const int blk = c->blk_cls[sizeof(S) == 2 ? 0 : sizeof(S) == 4 ? 1 : 2];
    size_t smem = (size_t)blk * sizeof(double);
    if (useG) smem = std::max(smem, (size_t)smem_reals_G<T>(c->g.Ls, blk) * sizeof(T));
    return smem;
}

int launch_ls(mdwf_ctx* c, int prec, LsArgs& a, cudaStream_t st) {
    ProfScope ps(c, 3, st);
    int grid, blk, nblk;
    site_grid(c, prec, a.rl, prec == 16 ? a.in.ril : 0, &grid, &blk, &nblk);
    if (a.partial) c->partial_nblk = nblk;
    switch (prec) {
        case 64: return launch_big_smem(c, ls_kernel<double>, grid, blk, g_smem<double>(c, a.op.kind != 0), st, a);
        case 32: return launch_big_smem(c, ls_kernel<float>, grid, blk, g_smem<float>(c, a.op.kind != 0), st, a);
        case 16: return launch_big_smem(c, ls_kernel<__half>, grid, blk, g_smem<__half>(c, a.op.kind != 0), st, a);
    }
    MDWF_FAIL(c, MDWF_EINVAL, "bad precision %d", prec);
}

static int launch_hop_raw(mdwf_ctx* c, int prec, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st) {
    switch (prec) {
        case 64: return launch_hop_f64(c, recon, dagger, fused, a, st);
        case 32: return launch_hop_f32(c, recon, dagger, fused, a, st);
        case 16: return launch_hop_f16(c, recon, dagger, fused, a, st);
    }
    MDWF_FAIL(c, MDWF_EINVAL, "bad precision %d", prec);
}
int launch_hop(mdwf_ctx* c, int prec, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st) {
    if (!c->prof_on) return launch_hop_raw(c, prec, recon, dagger, fused, a, st);
    mdwf_ctx::ProfRec r;
    for (int k = 0; k < 2; ++k) {
        cudaEvent_t e;
        if (!c->prof_pool.empty()) { e = c->prof_pool.back(); c->prof_pool.pop_back(); }
        else MDWF_CUDA(c, cudaEventCreate(&e));
        (k ? r.e1 : r.e0) = e;
    }
    const double w = prec / 8.0, n5 = (double)c->g.N5h * a.nact;
    const double pass = 24.0 * w;
    r.cls = prec == 16 ? 0 : prec == 32 ? 1 : 2;
    r.bytes = (2.0 + (a.xin.v ? 1.0 : 0.0)) * pass * n5 + 8.0 * recon * w * c->g.Vh;
    r.flops = 1320.0 * n5;
    cudaEventRecord(r.e0, st);
    int rc = launch_hop_raw(c, prec, recon, dagger, fused, a, st);
    cudaEventRecord(r.e1, st);
    c->prof_pending.push_back(r);
    return rc;
}

ProfScope::ProfScope(mdwf_ctx* c_, int cls, cudaStream_t st_) : c(c_), st(st_), on(c_->prof_on != 0) {
    if (!on) return;
    for (int k = 0; k < 2; ++k) {
        cudaEvent_t e;
        if (!c->prof_pool.empty()) { e = c->prof_pool.back(); c->prof_pool.pop_back(); }
        else if (cudaEventCreate(&e) != cudaSuccess) { on = false; return; }
        (k ? r.e1 : r.e0) = e;
    }
    r.cls = cls; r.bytes = 0.0; r.flops = 0.0;
    cudaEventRecord(r.e0, st);
}
ProfScope::~ProfScope() {
    if (!on) return;
    cudaEventRecord(r.e1, st);
    c->prof_pending.push_back(r);
}

template <typename SO, typename SA>
static int axpby_b(mdwf_ctx* c, int pb, AxpbyArgs& a, cudaStream_t st) {
    // blocked like the output's storage class; grouped when any field is fp16 (they share one interleave)
    const int ril = sizeof(SO) == 2 ? a.out.ril : sizeof(SA) == 2 && a.a.v ? a.a.ril : pb == 16 && a.b.v ? a.b.ril : 0;
    int grid, blk, nblk;
    site_grid(c, sizeof(SO) == 2 ? 16 : sizeof(SO) == 4 ? 32 : 64, a.rl, ril, &grid, &blk, &nblk);
    const size_t smem = (size_t)blk * sizeof(double);
    if (a.partial) c->partial_nblk = nblk;
    switch (pb) {
        case 64: LAUNCH((axpby_kernel<SO, SA, double>), grid, blk, smem, c->g, a); return MDWF_OK;
        case 32: LAUNCH((axpby_kernel<SO, SA, float>), grid, blk, smem, c->g, a); return MDWF_OK;
        case 16: LAUNCH((axpby_kernel<SO, SA, __half>), grid, blk, smem, c->g, a); return MDWF_OK;
    }
    MDWF_FAIL(c, MDWF_EINVAL, "bad precision %d", pb);
}
template <typename SO>
static int axpby_a(mdwf_ctx* c, int pa, int pb, AxpbyArgs& a, cudaStream_t st) {
    switch (pa) {
        case 64: return axpby_b<SO, double>(c, pb, a, st);
        case 32: return axpby_b<SO, float>(c, pb, a, st);
        case 16: return axpby_b<SO, __half>(c, pb, a, st);
    }
    MDWF_FAIL(c, MDWF_EINVAL, "bad precision %d", pa);
}
int launch_axpby(mdwf_ctx* c, int po, int pa, int pb, AxpbyArgs& a, cudaStream_t st) {
    ProfScope ps(c, 7, st);
    switch (po) {
        case 64: return axpby_a<double>(c, pa, pb, a, st);
        case 32: return axpby_a<float>(c, pa, pb, a, st);
        case 16: return axpby_a<__half>(c, pa, pb, a, st);
    }
    MDWF_FAIL(c, MDWF_EINVAL, "bad precision %d", po);
}

int launch_cg_xr(mdwf_ctx* c, int prec_x, int prec, CgXrArgs& a, cudaStream_t st) {
    ProfScope ps(c, 4, st);
    int grid, blk, nblk;
    site_grid(c, prec, a.rl, prec == 16 ? a.r.ril : 0, &grid, &blk, &nblk);
    const size_t smem = (size_t)blk * sizeof(double);
    c->partial_nblk = nblk;
    if (prec == 64 && prec_x == 64) { LAUNCH((cg_update_xr_kernel<double, double>), grid, blk, smem, c->g, a); return MDWF_OK; }
    if (prec == 32 && prec_x == 32) { LAUNCH((cg_update_xr_kernel<float, float>), grid, blk, smem, c->g, a); return MDWF_OK; }
    if (prec == 16 && prec_x == 32) { LAUNCH((cg_update_xr_kernel<float, __half>), grid, blk, smem, c->g, a); return MDWF_OK; }
    MDWF_FAIL(c, MDWF_EINVAL, "unsupported CG precision pair x=%d, r=%d", prec_x, prec);
}

int launch_cg_p(mdwf_ctx* c, int prec, CgPArgs& a, cudaStream_t st) {
    ProfScope ps(c, 5, st);
    int grid, blk, nblk;
    site_grid(c, prec, a.rl, prec == 16 ? a.p.ril : 0, &grid, &blk, &nblk);
    if (a.partial) c->partial_nblk = nblk;
    switch (prec) {
        case 64: return launch_big_smem(c, cg_update_p_kernel<double>, grid, blk, g_smem<double>(c, a.op.kind != 0), st, a);
        case 32: return launch_big_smem(c, cg_update_p_kernel<float>, grid, blk, g_smem<float>(c, a.op.kind != 0), st, a);
        case 16: return launch_big_smem(c, cg_update_p_kernel<__half>, grid, blk, g_smem<__half>(c, a.op.kind != 0), st, a);
    }
    MDWF_FAIL(c, MDWF_EINVAL, "bad precision %d", prec);
}

int launch_finish(mdwf_ctx* c, const RhsList& rl, double* out, double* out2, cudaStream_t st, double* nb, const FinishCtl* fc) {
    ProfScope ps(c, 6, st);
    FinishArgs f;
    memset(&f, 0, sizeof(f));
    if (fc) { f.stop = fc->stop; f.ctl = fc->ctl; f.hctl = fc->hctl; f.pap = fc->pap; f.seq = fc->seq; }
    f.partial = c->partial;
    f.nblk = c->partial_nblk;
    f.out = out;
    f.out2 = out2;
    f.nb = nb;
    f.rl = rl;
    finish_sum_kernel<<<rl.nact, 1024, 0, st>>>(f);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

int launch_pack(mdwf_ctx* c, int prec, bool unpack, PackArgs& a, cudaStream_t st) {
    dim3 grid((c->g.N5h + 255) / 256, a.nrhs);
    if (prec == 16 && !unpack) {
        // the scale of an fp16 field follows from its 2-norm: measure it first (R11).  a.sr.out is set by the caller.
        if ((size_t)grid.x > c->partial_cap) MDWF_FAIL(c, MDWF_EINVAL, "internal: partial buffer too small for the pack norm");
        PackArgs n = a;
        n.partial = c->partial;
        pack_norm_kernel<<<grid, 256, 256 * sizeof(double), st>>>(c->g, n);
        MDWF_CUDA(c, cudaGetLastError());
        c->launches++;
        c->partial_nblk = grid.x;
        RhsList rl = all_rhs(a.nrhs);
        double* dn = c->dscal + 64 * 7;
        if (a.rhs0 != 0) MDWF_FAIL(c, MDWF_EINVAL, "internal: fp16 pack with a rhs offset");
        int rc = launch_finish(c, rl, dn, nullptr, st);
        if (rc) return rc;
        a.sr.n = 1;
        a.sr.t[0].nb = dn; a.sr.t[0].num = nullptr; a.sr.t[0].den = nullptr; a.sr.t[0].coef = 1.0009765625; a.sr.t[0].sq = 1;
    }
#define PK(S, U) pack_kernel<S, U><<<grid, 256, 0, st>>>(c->g, a)
    if (prec == 64) { if (unpack) PK(double, true); else PK(double, false); }
    else if (prec == 32) { if (unpack) PK(float, true); else PK(float, false); }
    else if (prec == 16) { if (unpack) PK(__half, true); else PK(__half, false); }
    else MDWF_FAIL(c, MDWF_EINVAL, "bad precision %d", prec);
#undef PK
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

}  // namespace mdwf

mdwf::SpinorView mdwf_field::view() const {
    mdwf::SpinorView s;
    s.rs = (long long)rs;
    s.v = reinterpret_cast<char*>(v) - (long long)rhs0 * s.rs;
    s.m = rmeta();
    s.ril = prec == 16 ? mdwf::half_ril(nrhs, ctx->g.Ls) : 0;
    s.Ls = ctx->g.Ls;
    s.sb = prec == 16 ? mdwf::half_site_bytes(nrhs, ctx->g.Ls) : 0;
    s.dLs = ctx->g.dLs;
    return s;
}
