// csrc/gauge.cu -- gauge-field packing (north_star "gauge-field ... layout/packing, with optional
// 12/8-parameter link reconstruction and fp16/fp32 storage").  Canonical fp64 U[mu][x4][3][3][re,im] ->
// per (parity of the base site, mu): vec[c][xh] in {fp64,fp32,fp16} x {18,12,8 reals} (formats: SURVEY A12).
// The boundary sign is never stored (the 8/12-real formats need an SU(3) matrix); hop_kernel applies it.
#include "mdwf_host.h"

namespace mdwf {

struct GaugePackArgs {
    const double* U;     // canonical
    void* out[2];
    int* bad;            // count of links the 8-real format cannot represent
    long long V4;
};

template <typename S, int R>
__global__ void __launch_bounds__(256) gauge_pack_kernel(const Geom g, const GaugePackArgs a) {
    const int xh = blockIdx.x * blockDim.x + threadIdx.x;
    const int mu = blockIdx.y, par = blockIdx.z;
    if (xh >= g.Vh) return;
    const long long x4 = canon_site(g, 1, par, xh);
    const double* u = a.U + ((long long)mu * a.V4 + x4) * 18;
    double gq[20];
#pragma unroll
    for (int i = 0; i < 20; ++i) gq[i] = 0.0;
    if (R == 18 || R == 12) {
#pragma unroll
        for (int i = 0; i < R; ++i) gq[i] = u[i];
    } else {
        // rows (a1,a2,a3),(b1,..),(c1,..): keep a2, a3, b1, arg a1, arg c1
        gq[0] = u[2]; gq[1] = u[3]; gq[2] = u[4]; gq[3] = u[5];
        gq[4] = u[6]; gq[5] = u[7];
        gq[6] = atan2(u[1], u[0]);
        gq[7] = atan2(u[13], u[12]);
        const double N = u[2] * u[2] + u[3] * u[3] + u[4] * u[4] + u[5] * u[5];
        if (!(N > 1e-8)) atomicAdd(a.bad, 1);
        if (Store<S>::HALF) { gq[6] *= 0.31830988618379067154; gq[7] *= 0.31830988618379067154; }
    }
    constexpr int NG = GaugeFmt<S, R>::NGV;
    typedef typename GaugeFmt<S, R>::vec V;
    V* o = reinterpret_cast<V*>(a.out[par]) + (long long)mu * NG * g.Vh + xh;
#pragma unroll
    for (int c = 0; c < NG; ++c) {
        V* dst = o + (long long)c * g.Vh;
        if (sizeof(S) == 8) {
            *reinterpret_cast<double2*>(dst) = make_double2(gq[2 * c], gq[2 * c + 1]);
        } else if (sizeof(S) == 4) {
            *reinterpret_cast<float4*>(dst) = make_float4((float)gq[4 * c], (float)gq[4 * c + 1], (float)gq[4 * c + 2], (float)gq[4 * c + 3]);
        } else {
            uint2 t;
            t.x = f2h((float)gq[4 * c], (float)gq[4 * c + 1]);
            t.y = f2h((float)gq[4 * c + 2], (float)gq[4 * c + 3]);
            *reinterpret_cast<uint2*>(dst) = t;
        }
    }
}

// Stencil-ready links for 16-bit storage (GaugeView::pl): for every output site of parity `par` and leg l the matrix
// exactly as the stencil multiplies it -- decoded from the packed fp16 format (18/12/8 reals), daggered for backward
// legs, boundary sign folded (stage_link, mdwf_hop.cuh) -- rounded to half, and the neighbour's site index.  320 bytes per site; it replaces the
// per-block reconstruction (and makes the 12/8-real decode a load-time cost) for the tensor-core stencil.
template <int R>
__global__ void __launch_bounds__(256) gauge_prepare16_kernel(const Geom g, GaugeView gv, uint32_t* pl, int par) {
    const int task = blockIdx.x * blockDim.x + threadIdx.x;
    if (task >= g.Vh * 8) return;
    const int xh = task >> 3, l = task & 7;
    SiteCoord c;
    uint32_t row, xx, r2, y, t, z;
    g.dXH.divmod((uint32_t)xh, row, xx);
    g.dY.divmod(row, r2, y);
    g.dZ.divmod(r2, t, z);
    c.xh = xh; c.xx = xx; c.y = y; c.z = z; c.t = t;
    c.o = (par + y + z + t) & 1;
    float V[MDWF_LROW];
    const int n = stage_link<__half, R>(g, gv, par, c, l, V);
    uint32_t* dst = pl + (long long)xh * 80 + l;            // [xh][9 link words + neighbour index][leg 8]
#pragma unroll
    for (int e = 0; e < 9; ++e) dst[e * 8] = f2h(V[2 * e], V[2 * e + 1]);
    dst[72] = (uint32_t)n;
}

void free_gauge(GaugeSet* gs) {
    for (int p = 0; p < 2; ++p) {
        if (gs->v[p]) cudaFree(gs->v[p]);
        if (gs->pl[p]) cudaFree(gs->pl[p]);
        gs->v[p] = nullptr; gs->pl[p] = nullptr;
    }
}

template <typename S>
static int pack_gauge_S(mdwf_ctx* c, int recon, const GaugePackArgs& a, cudaStream_t st) {
    dim3 grid((c->g.Vh + 255) / 256, 4, 2);
    switch (recon) {
        case 18: gauge_pack_kernel<S, 18><<<grid, 256, 0, st>>>(c->g, a); break;
        case 12: gauge_pack_kernel<S, 12><<<grid, 256, 0, st>>>(c->g, a); break;
        case 8: gauge_pack_kernel<S, 8><<<grid, 256, 0, st>>>(c->g, a); break;
        default: MDWF_FAIL(c, MDWF_EINVAL, "recon must be 18, 12 or 8 (got %d)", recon);
    }
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

int pack_gauge(mdwf_ctx* c, const void* U, int prec, int recon, GaugeSet* gs, cudaStream_t st) {
    int ngv, vbytes;
    if (prec == 64) { ngv = (recon + 1) / 2; vbytes = 16; }
    else if (prec == 32) { ngv = (recon + 3) / 4; vbytes = 16; }
    else if (prec == 16) { ngv = (recon + 3) / 4; vbytes = 8; }
    else MDWF_FAIL(c, MDWF_EINVAL, "store_prec must be 64, 32 or 16 (got %d)", prec);
    if (recon != 18 && recon != 12 && recon != 8) MDWF_FAIL(c, MDWF_EINVAL, "recon must be 18, 12 or 8 (got %d)", recon);
    gs->prec = prec;
    gs->recon = recon;
    gs->bytes_per_parity = (size_t)4 * ngv * c->g.Vh * vbytes;
    gs->v[0] = gs->v[1] = nullptr;
    gs->pl[0] = gs->pl[1] = nullptr;
    int* bad = nullptr;
    for (int p = 0; p < 2; ++p) {
        cudaError_t e = cudaMalloc(&gs->v[p], gs->bytes_per_parity);
        if (e != cudaSuccess) {
            cudaGetLastError();
            if (gs->v[0]) cudaFree(gs->v[0]);
            MDWF_FAIL(c, MDWF_ENOMEM, "cudaMalloc of %zu bytes for packed links failed", gs->bytes_per_parity);
        }
    }
    MDWF_CUDA(c, cudaMalloc(&bad, sizeof(int)));
    MDWF_CUDA(c, cudaMemsetAsync(bad, 0, sizeof(int), st));
    GaugePackArgs a;
    a.U = reinterpret_cast<const double*>(U);
    a.out[0] = gs->v[0];
    a.out[1] = gs->v[1];
    a.bad = bad;
    a.V4 = 2ll * c->g.Vh;
    int rc = prec == 64 ? pack_gauge_S<double>(c, recon, a, st)
             : prec == 32 ? pack_gauge_S<float>(c, recon, a, st) : pack_gauge_S<__half>(c, recon, a, st);
    int nbad = 0;
    if (rc == MDWF_OK) {
        cudaError_t e = cudaMemcpyAsync(&nbad, bad, sizeof(int), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) { c->err = std::string("gauge pack: ") + cudaGetErrorString(e); rc = MDWF_ECUDA; }
    }
    cudaFree(bad);
    if (rc == MDWF_OK && nbad > 0) {
        char b[256];
        snprintf(b, sizeof(b), "8-real link format cannot represent %d links with |U01|^2+|U02|^2 -> 0 (SURVEY A12); use recon 12 or 18", nbad);
        c->err = b;
        rc = MDWF_EINVAL;
    }
    if (rc == MDWF_OK && prec == 16) {
        GaugeView gv;
        gv.v[0] = gs->v[0]; gv.v[1] = gs->v[1];
        gv.pl[0] = gv.pl[1] = nullptr;
        const int ntask = c->g.Vh * 8, grid = (ntask + 255) / 256;
        for (int p = 0; p < 2 && rc == MDWF_OK; ++p) {
            if (cudaMalloc(&gs->pl[p], (size_t)c->g.Vh * 320) != cudaSuccess) {
                cudaGetLastError();
                c->err = "cudaMalloc of the stencil-ready fp16 links failed";
                rc = MDWF_ENOMEM;
                break;
            }
            if (recon == 18) gauge_prepare16_kernel<18><<<grid, 256, 0, st>>>(c->g, gv, gs->pl[p], p);
            else if (recon == 12) gauge_prepare16_kernel<12><<<grid, 256, 0, st>>>(c->g, gv, gs->pl[p], p);
            else gauge_prepare16_kernel<8><<<grid, 256, 0, st>>>(c->g, gv, gs->pl[p], p);
            if (cudaGetLastError() != cudaSuccess) { c->err = "gauge_prepare16_kernel launch failed"; rc = MDWF_ECUDA; }
            c->launches++;
        }
    }
    if (rc != MDWF_OK) free_gauge(gs);
    return rc;
}

}  // namespace mdwf
