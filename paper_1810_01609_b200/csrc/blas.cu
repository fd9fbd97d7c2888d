// csrc/blas.cu -- launchers of the 4D-site-local kernels in mdwf_blas.cuh and the packed-field allocator.
#include "mdwf_hop_launch.cuh"

namespace mdwf {

static size_t rhs_bytes(const Geom& g, int prec) {
    const size_t nb = ((size_t)g.N5h + 31) / 32;
    return nb * (size_t)((24 * (prec / 8) / 16) * 512 + (prec == 16 ? 128 : 0));
}
size_t field_bytes(const Geom& g, int prec, int nrhs, size_t* norm_off) {
    if (norm_off) *norm_off = 0;
    return rhs_bytes(g, prec) * nrhs;
}

int alloc_field(mdwf_ctx* c, int prec, int nrhs, mdwf_field** out) {
    if (prec != 64 && prec != 32 && prec != 16) MDWF_FAIL(c, MDWF_EINVAL, "prec must be 64, 32 or 16 (got %d)", prec);
    if (nrhs < 1 || nrhs > MDWF_MAX_RHS) MDWF_FAIL(c, MDWF_EINVAL, "nrhs must be in 1..%d (got %d)", MDWF_MAX_RHS, nrhs);
    mdwf_field* f = new mdwf_field;
    f->ctx = c;
    f->prec = prec;
    f->nrhs = nrhs;
    size_t noff = 0;
    f->bytes = field_bytes(c->g, prec, nrhs, &noff);
    f->v = nullptr;
    cudaError_t e = cudaMalloc(&f->v, f->bytes);
    if (e != cudaSuccess) {
        delete f;
        cudaGetLastError();
        MDWF_FAIL(c, MDWF_ENOMEM, "cudaMalloc of %zu bytes for a packed field failed: %s", f->bytes, cudaGetErrorString(e));
    }
    f->n = nullptr;
    *out = f;
    return MDWF_OK;
}
void free_field(mdwf_field* f) {
    if (!f) return;
    if (f->v) cudaFree(f->v);
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

#define LAUNCH(kern, grid, blk, smem, ...)                              \
    do {                                                                \
        kern<<<(grid), (blk), (smem), st>>>(__VA_ARGS__);               \
        MDWF_CUDA(c, cudaGetLastError());                               \
        c->launches++;                                                  \
    } while (0)

template <typename K, typename A>
static int launch_big_smem(mdwf_ctx* c, K kern, int grid, int blk, size_t smem, cudaStream_t st, const A& a) {
    static std::set<const void*> raised;
    if (smem > 48 * 1024 && !raised.count((const void*)kern)) {
        MDWF_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
        raised.insert((const void*)kern);
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
    const int grid = c->nblk_cls[cls_of(prec)] * a.rl.nact, blk = c->blk_cls[cls_of(prec)];
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
    const double pass = 24.0 * w + (prec == 16 ? 4.0 : 0.0);
    r.cls = prec == 16 ? 0 : prec == 32 ? 1 : 2;
    r.bytes = (2.0 + (a.xin.v ? 1.0 : 0.0)) * pass * n5 + 8.0 * recon * w * c->g.Vh;
    r.flops = 1320.0 * n5;
    cudaEventRecord(r.e0, st);
    int rc = launch_hop_raw(c, prec, recon, dagger, fused, a, st);
    cudaEventRecord(r.e1, st);
    c->prof_pending.push_back(r);
    return rc;
}

template <typename SO, typename SA>
static int axpby_b(mdwf_ctx* c, int pb, AxpbyArgs& a, cudaStream_t st) {
    const int cls = sizeof(SO) == 2 ? 0 : sizeof(SO) == 4 ? 1 : 2;      // blocked like the output's storage class
    const int grid = c->nblk_cls[cls] * a.rl.nact, blk = c->blk_cls[cls];
    const size_t smem = (size_t)blk * sizeof(double);
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
    switch (po) {
        case 64: return axpby_a<double>(c, pa, pb, a, st);
        case 32: return axpby_a<float>(c, pa, pb, a, st);
        case 16: return axpby_a<__half>(c, pa, pb, a, st);
    }
    MDWF_FAIL(c, MDWF_EINVAL, "bad precision %d", po);
}

int launch_cg_xr(mdwf_ctx* c, int prec_x, int prec, CgXrArgs& a, cudaStream_t st) {
    const int grid = c->nblk_cls[cls_of(prec)] * a.rl.nact, blk = c->blk_cls[cls_of(prec)];
    const size_t smem = (size_t)blk * sizeof(double);
    if (prec == 64 && prec_x == 64) { LAUNCH((cg_update_xr_kernel<double, double>), grid, blk, smem, c->g, a); return MDWF_OK; }
    if (prec == 32 && prec_x == 32) { LAUNCH((cg_update_xr_kernel<float, float>), grid, blk, smem, c->g, a); return MDWF_OK; }
    if (prec == 16 && prec_x == 32) { LAUNCH((cg_update_xr_kernel<float, __half>), grid, blk, smem, c->g, a); return MDWF_OK; }
    if (prec == 16 && prec_x == 16) { LAUNCH((cg_update_xr_kernel<__half, __half>), grid, blk, smem, c->g, a); return MDWF_OK; }
    MDWF_FAIL(c, MDWF_EINVAL, "unsupported CG precision pair x=%d, r=%d", prec_x, prec);
}

int launch_cg_p(mdwf_ctx* c, int prec, CgPArgs& a, cudaStream_t st) {
    const int grid = c->nblk_cls[cls_of(prec)] * a.rl.nact, blk = c->blk_cls[cls_of(prec)];
    switch (prec) {
        case 64: return launch_big_smem(c, cg_update_p_kernel<double>, grid, blk, g_smem<double>(c, a.op.kind != 0), st, a);
        case 32: return launch_big_smem(c, cg_update_p_kernel<float>, grid, blk, g_smem<float>(c, a.op.kind != 0), st, a);
        case 16: return launch_big_smem(c, cg_update_p_kernel<__half>, grid, blk, g_smem<__half>(c, a.op.kind != 0), st, a);
    }
    MDWF_FAIL(c, MDWF_EINVAL, "bad precision %d", prec);
}

int launch_finish(mdwf_ctx* c, int prec, const RhsList& rl, double* out, double* out2, cudaStream_t st) {
    FinishArgs f;
    f.partial = c->partial;
    f.nblk = c->nblk_cls[cls_of(prec)];
    f.out = out;
    f.out2 = out2;
    f.rl = rl;
    finish_sum_kernel<<<rl.nact, 256, 0, st>>>(f);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

int launch_pack(mdwf_ctx* c, int prec, bool unpack, PackArgs& a, cudaStream_t st) {
    dim3 grid((c->g.N5h + 255) / 256, a.nrhs);
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
    s.v = v;
    s.n = nullptr;
    s.rs = (long long)(bytes / nrhs);
    s.rn = 0;
    return s;
}
