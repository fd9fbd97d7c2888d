// csrc/smear.cu -- the fuller Feynman-Hellmann workload: gauge-covariant Gaussian
// smearing of 4D spin-colour fields at source and sink, and the effective derivative of the FH correlator ratio.
// The paper names smeared sources but prints no formula; R25 fixes the reading
//     psi' = (1 + sigma^2/(4 N) Lap)^N psi,
//     (Lap psi)(x) = sum_{j=x,y,z} [ U_j(x) psi(x+j) + U_j(x-j)^dag psi(x-j) - 2 psi(x) ]     (3D, every timeslice on its own),
// hops that wrap multiplied by the geometry's boundary sign.  Fields are canonical fp64 [col][x4][4][3] (the layout of
// mdwf_seq_source / mdwf_nucleon_2pt); links are the loaded fp64 18-real format.
//
// One step = one launch.  A block owns NS consecutive 4D sites: phase 0 parks their 6 spatial links in shared memory as
// the 3x3 matrices the step multiplies (backward legs daggered, boundary sign and the step size folded) together with the 6 neighbour
// indices; phase 1 runs over (column, site, spin) items -- a lane owns one colour 3-vector (48 contiguous bytes), a warp 8
// consecutive sites of one column, all 6 neighbour vectors in flight at once -- so the links are read from HBM once per step and shared by all columns (the same idea as
// the link staging of the Dslash stencil, north_star).  Algorithmic bytes per step: 2 x 192 B per site and column plus
// 3 x 144 B of links per site; HBM-bound.
#include "mdwf_host.h"
#include <cstring>
#include <cmath>

namespace mdwf {

#define MDWF_SMEAR_NS 32          // sites per block
#define MDWF_SMEAR_THREADS 256

struct SmearArgs {
    const double2* in;
    double2* out;
    GaugeView g;
    long long V4;
    int ncol;
    double a;                     // sigma^2 / (4 N)
};

__global__ void __launch_bounds__(MDWF_SMEAR_THREADS) smear_step_kernel(const Geom g, const SmearArgs a) {
    __shared__ double2 s_link[MDWF_SMEAR_NS][6][9];
    __shared__ int s_nb[MDWF_SMEAR_NS][6];
    const long long x0 = (long long)blockIdx.x * MDWF_SMEAR_NS;
    // ---- phase 0: links and neighbours of the block's sites ---------------------------------------------------
    for (int k = threadIdx.x; k < MDWF_SMEAR_NS * 6; k += blockDim.x) {
        const int s = k / 6, l = k - 6 * s, j = l >> 1, bwd = l & 1;
        const long long x4 = x0 + s;
        if (x4 >= a.V4) continue;
        unsigned r = (unsigned)x4;
        const int cx = (int)(r % (unsigned)g.X); r /= (unsigned)g.X;
        const int cy = (int)(r % (unsigned)g.Y); r /= (unsigned)g.Y;
        const int cz = (int)(r % (unsigned)g.Z); r /= (unsigned)g.Z;
        const int par = (cx + cy + cz + (int)r) & 1;
        const int cj = j == 0 ? cx : j == 1 ? cy : cz, ext = j == 0 ? g.X : j == 1 ? g.Y : g.Z;
        const long long stride = j == 0 ? 1 : j == 1 ? g.X : (long long)g.X * g.Y;
        const int cn = bwd ? (cj == 0 ? ext - 1 : cj - 1) : (cj == ext - 1 ? 0 : cj + 1);
        const bool wrap = bwd ? cj == 0 : cj == ext - 1;
        const long long xn = x4 + (cn - cj) * stride;
        s_nb[s][l] = (int)xn;
        double U[18];
        if (!bwd) load_link<double, 18>(a.g.v[par], j, (int)(x4 >> 1), g.Vh, U);
        else load_link<double, 18>(a.g.v[1 - par], j, (int)(xn >> 1), g.Vh, U);
        const double sg = a.a * (wrap ? (double)(j == 0 ? g.bc[0] : j == 1 ? g.bc[1] : g.bc[2]) : 1.0);   // a = sigma^2/(4N) folded in
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                // forward: M = U_j(x);  backward: M = U_j(x - j)^dag
                const double re = bwd ? U[2 * (c * 3 + r)] : U[2 * (r * 3 + c)];
                const double im = bwd ? -U[2 * (c * 3 + r) + 1] : U[2 * (r * 3 + c) + 1];
                s_link[s][l][r * 3 + c] = make_double2(sg * re, sg * im);
            }
    }
    __syncthreads();
    // ---- phase 1: (column, site, spin) items: a lane owns one colour 3-vector, 4 lanes a site, a warp 8 consecutive sites -------
    const double diag = 1.0 - 6.0 * a.a;
    for (int it = threadIdx.x; it < MDWF_SMEAR_NS * 4 * a.ncol; it += blockDim.x) {
        const int col = it / (MDWF_SMEAR_NS * 4), rem = it - col * (MDWF_SMEAR_NS * 4), s = rem >> 2, sp = rem & 3;
        const long long x4 = x0 + s;
        if (x4 >= a.V4) continue;
        const double2* base = a.in + (long long)col * a.V4 * 12 + 3 * sp;
        double2 acc[3];
        {
            const double2* p = base + x4 * 12;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double2 v = __ldg(p + c);
                acc[c] = make_double2(diag * v.x, diag * v.y);
            }
        }
        double2 v[6][3];
#pragma unroll
        for (int l = 0; l < 6; ++l) {
            const double2* p = base + (long long)s_nb[s][l] * 12;
#pragma unroll
            for (int c = 0; c < 3; ++c) v[l][c] = __ldg(p + c);
        }
#pragma unroll
        for (int l = 0; l < 6; ++l)
#pragma unroll
            for (int r = 0; r < 3; ++r)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const double2 m = s_link[s][l][r * 3 + c];
                    const double2 w = v[l][c];
                    acc[r].x = fma(m.x, w.x, fma(-m.y, w.y, acc[r].x));
                    acc[r].y = fma(m.x, w.y, fma(m.y, w.x, acc[r].y));
                }
        double2* o = a.out + ((long long)col * a.V4 + x4) * 12 + 3 * sp;
#pragma unroll
        for (int c = 0; c < 3; ++c) o[c] = acc[c];
    }
}

// g_eff(t) = R(t+1) - R(t),  R = C_FH / C_2pt (complex), t = 0 .. T-2
__global__ void fh_effective_derivative_kernel(double2* geff, const double2* c2, const double2* cfh, int T) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T - 1) return;
    double2 R[2];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const double2 n = cfh[t + k], d = c2[t + k];
        const double den = d.x * d.x + d.y * d.y;
        R[k] = make_double2((n.x * d.x + n.y * d.y) / den, (n.y * d.x - n.x * d.y) / den);
    }
    geff[t] = make_double2(R[1].x - R[0].x, R[1].y - R[0].y);
}

}  // namespace mdwf

using namespace mdwf;

extern "C" {

int mdwf_smear_gaussian(mdwf_ctx* c, void* out4d, const void* in4d, int ncol, double width, int n_iter, void* stream) {
    MDWF_ENTER(c);
    if (!out4d || !in4d) MDWF_FAIL(c, MDWF_EINVAL, "null pointer");
    if (out4d == in4d) MDWF_FAIL(c, MDWF_EINVAL, "mdwf_smear_gaussian: out4d must not alias in4d");
    if (ncol < 1 || ncol > 4096) MDWF_FAIL(c, MDWF_EINVAL, "ncol must be in 1..4096 (got %d)", ncol);
    if (n_iter < 0 || !(width >= 0.0) || !std::isfinite(width)) MDWF_FAIL(c, MDWF_EINVAL, "need n_iter >= 0 and a finite width >= 0");
    const GaugeSet* gs = c->find_gauge(64, 18);
    if (!gs) MDWF_FAIL(c, MDWF_ESTATE, "mdwf_smear_gaussian needs the fp64 18-real links: call mdwf_load_gauge(U, 64, 18) first");
    cudaStream_t st = (cudaStream_t)stream;
    const long long V4 = 2ll * c->g.Vh;
    const size_t bytes = (size_t)ncol * V4 * 12 * sizeof(double2);
    if (n_iter == 0) {
        MDWF_CUDA(c, cudaMemcpyAsync(out4d, in4d, bytes, cudaMemcpyDeviceToDevice, st));
        return MDWF_OK;
    }
    SmearArgs a;
    memset(&a, 0, sizeof(a));
    a.g.v[0] = gs->v[0]; a.g.v[1] = gs->v[1];
    a.V4 = V4; a.ncol = ncol; a.a = width * width / (4.0 * n_iter);
    void* tmp = nullptr;
    if (n_iter > 1) MDWF_CUDA(c, cudaMallocAsync(&tmp, bytes, st));
    // ping-pong between out and tmp so that the last step lands in out:  n odd: in -> out -> tmp -> out ...;  n even: in -> tmp -> out ...
    const void* src = in4d;
    const unsigned grid = (unsigned)((V4 + MDWF_SMEAR_NS - 1) / MDWF_SMEAR_NS);
    for (int k = 0; k < n_iter; ++k) {
        void* dst = ((n_iter - k) & 1) ? out4d : tmp;
        a.in = (const double2*)src; a.out = (double2*)dst;
        smear_step_kernel<<<grid, MDWF_SMEAR_THREADS, 0, st>>>(c->g, a);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) {
            if (tmp) cudaFreeAsync(tmp, st);
            MDWF_FAIL(c, MDWF_ECUDA, "smear_step_kernel: %s", cudaGetErrorString(e));
        }
        c->launches++;
        src = dst;
    }
    if (tmp) MDWF_CUDA(c, cudaFreeAsync(tmp, st));
    return MDWF_OK;
}

int mdwf_fh_effective_derivative(mdwf_ctx* c, double* geff, const double* c2pt, const double* cfh, void* stream) {
    MDWF_ENTER(c);
    if (!geff || !c2pt || !cfh) MDWF_FAIL(c, MDWF_EINVAL, "null pointer");
    const int T = c->g.T;
    fh_effective_derivative_kernel<<<(T + 63) / 64, 64, 0, (cudaStream_t)stream>>>((double2*)geff, (const double2*)c2pt, (const double2*)cfh, T);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

}  // extern "C"
