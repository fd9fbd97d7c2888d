// csrc/meas.cu -- 4D <-> 5D wall maps, the Feynman-Hellmann sequential source
// and the nucleon two-point contraction.
#include "mdwf_host.h"
#include <cstring>

namespace mdwf {

// packed 5D wall field of parity `par`:  w(x, s=0) = P+ eta(x),  w(x, s=Ls-1) = P- eta(x)  (both if Ls = 1)
__global__ void __launch_bounds__(256) wall_pack_kernel(const Geom g, SpinorView out, const double* eta, int par) {
    const int rhs = blockIdx.y;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= g.N5h) return;
    uint32_t xh, s;
    g.dLs.divmod((uint32_t)idx, xh, s);
    double v[24];
#pragma unroll
    for (int i = 0; i < 24; ++i) v[i] = 0.0;
    if (s == 0 || (int)s == g.Ls - 1) {
        const long long x4 = canon_site(g, 1, par, (int)xh);
        const double* e = eta + ((long long)rhs * 2 * g.Vh + x4) * 24;
        if (s == 0) {
#pragma unroll
            for (int i = 0; i < 12; ++i) v[i] = e[i];
        }
        if ((int)s == g.Ls - 1) {
#pragma unroll
            for (int i = 12; i < 24; ++i) v[i] = e[i];
        }
    }
    store_spinor<double>(out, rhs, idx, g.N5h, v);
}

// q(x) = P- psi(x, 0) + P+ psi(x, Ls-1) for the sites of parity `par`, written into the canonical 4D field
__global__ void __launch_bounds__(256) wall_unpack_kernel(const Geom g, double* q4, SpinorView in, int par) {
    const int rhs = blockIdx.y;
    const int xh = blockIdx.x * blockDim.x + threadIdx.x;
    if (xh >= g.Vh) return;
    double lo[24], hi[24];
    load_spinor<double>(in, rhs, xh * g.Ls + 0, g.N5h, lo);
    load_spinor<double>(in, rhs, xh * g.Ls + g.Ls - 1, g.N5h, hi);
    const long long x4 = canon_site(g, 1, par, xh);
    double* q = q4 + ((long long)rhs * 2 * g.Vh + x4) * 24;
#pragma unroll
    for (int i = 0; i < 12; ++i) q[i] = hi[i];
#pragma unroll
    for (int i = 12; i < 24; ++i) q[i] = lo[i];
}

int launch_wall_pack(mdwf_ctx* c, const SpinorView& out, const double* eta4, int par, int ncol, cudaStream_t st) {
    dim3 grid((c->g.N5h + 255) / 256, ncol);
    wall_pack_kernel<<<grid, 256, 0, st>>>(c->g, out, eta4, par);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}
int launch_wall_unpack(mdwf_ctx* c, double* q4, const SpinorView& in, int par, int ncol, cudaStream_t st) {
    dim3 grid((c->g.Vh + 255) / 256, ncol);
    wall_unpack_kernel<<<grid, 256, 0, st>>>(c->g, q4, in, par);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

// canonical full-lattice projection q[col][x4] from psi5[col][s][x4]
__global__ void __launch_bounds__(256) wall_project_kernel(double2* q4, const double2* psi5, long long V4, int Ls, int ncol) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // over ncol*V4*12 complex
    if (i >= (long long)ncol * V4 * 12) return;
    const int k = (int)(i % 12);
    const long long cx = i / 12, x = cx % V4, col = cx / V4;
    const int s = k < 6 ? Ls - 1 : 0;   // spins 0,1 (P+) from s = Ls-1 ; spins 2,3 (P-) from s = 0
    q4[i] = psi5[((col * Ls + s) * V4 + x) * 12 + k];
}

// eta_seq[col](x) = Gamma . S[col](x) for t_min <= t <= t_max, else 0.  One thread per (col, x4, colour).
struct SeqArgs {
    double2* out;
    const double2* in;
    long long V4, V3;
    int ncol, t_min, t_max;
    double G[32];
};
__global__ void __launch_bounds__(256) seq_source_kernel(const SeqArgs a) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // over ncol*V4*3
    if (i >= (long long)a.ncol * a.V4 * 3) return;
    const int col3 = (int)(i % 3);
    const long long cx = i / 3, x = cx % a.V4;
    const int t = (int)(x / a.V3);
    const double2* s = a.in + cx * 12 + col3;
    double2* o = a.out + cx * 12 + col3;
    const bool on = t >= a.t_min && t <= a.t_max;
    double2 v[4];
#pragma unroll
    for (int b = 0; b < 4; ++b) v[b] = on ? s[3 * b] : make_double2(0.0, 0.0);
#pragma unroll
    for (int al = 0; al < 4; ++al) {
        double re = 0.0, im = 0.0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const double gr = a.G[2 * (4 * al + b)], gi = a.G[2 * (4 * al + b) + 1];
            re += gr * v[b].x - gi * v[b].y;
            im += gr * v[b].y + gi * v[b].x;
        }
        o[3 * al] = make_double2(re, im);
    }
}

// ---------------------------------------------------------------------------------------------
// Nucleon 2-pt (SURVEY O4 C-def), in the trace form
//   C(t) = sum_x eps_{abc} eps_{a'b'c'} { tr[Q^{bb'} (Su1^{aa'})^T] tr[P Su2^{cc'}] - tr[(Q^{bb'})^T Su1^{ac'} P Su2^{ca'}] },
//   Q^{bb'} = G Sd^{bb'} Gt,  G = C gamma5,  Gt = gamma_t G^dag gamma_t,  S^{ab}_{al be}(x) = S[3 be + b][x][al][a].
// One warp per site; the 144 work items (colour-permutation pair e1,e2 ; spin index al') are spread over the lanes.
struct NucArgs {
    const double2 *Su1, *Sd, *Su2;
    double* partial;       // [T][nblk_t][2]
    long long V4, V3;
    int nblk_t;            // blocks per timeslice
    double G[32], Gt[32], P[32];
};
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 cfma(double2 a, double2 b, double2 c) {
    return make_double2(c.x + a.x * b.x - a.y * b.y, c.y + a.x * b.y + a.y * b.x);
}

#define MDWF_NUC_WARPS 8      // warps per block
#define MDWF_NUC_WPS 2        // warps per site (they meet at a named barrier)
__constant__ int c_perm[6][3] = {{0, 1, 2}, {1, 2, 0}, {2, 0, 1}, {0, 2, 1}, {2, 1, 0}, {1, 0, 2}};
__constant__ double c_psign[6] = {1, 1, 1, -1, -1, -1};
__global__ void __launch_bounds__(32 * MDWF_NUC_WARPS) nucleon_kernel(const NucArgs a) {
    // MDWF_NUC_WPS warps per site (named barriers only); 144 work items per phase are spread over their lanes.
    // prop element (sink spin al, sink colour ca, source spin be, source colour cb) at S[(3*be+cb)*12 + 3*al+ca]
    extern __shared__ __align__(16) unsigned char nuc_smem[];
    constexpr int GT = 32 * MDWF_NUC_WPS;                     // threads per site group
    const int grp = threadIdx.x / GT, lane = threadIdx.x % GT;
    double2* base = reinterpret_cast<double2*>(nuc_smem) + grp * (5 * 144 + 16);
#define NUC_SYNC() asm volatile("bar.sync %0, %1;" ::"r"(grp + 1), "r"(GT) : "memory")
    double2 *s1 = base, *sd = base + 144, *s2 = base + 288, *Q = base + 432, *W = base + 576, *trP = base + 720;
    const int t = blockIdx.y;
    double accr = 0.0, acci = 0.0;
    constexpr int GPB = MDWF_NUC_WARPS / MDWF_NUC_WPS;         // site groups per block
    const int gid = blockIdx.x * GPB + grp, ng = a.nblk_t * GPB;
    for (long long xs = gid; xs < a.V3; xs += ng) {
        const long long x = (long long)t * a.V3 + xs;
        for (int i = lane; i < 144; i += GT) {
            const int col = i / 12, k = i - col * 12;
            const long long off = ((long long)col * a.V4 + x) * 12 + k;
            s1[i] = __ldg(a.Su1 + off);
            sd[i] = __ldg(a.Sd + off);
            s2[i] = __ldg(a.Su2 + off);
        }
        NUC_SYNC();
        for (int e = lane; e < 144; e += GT) {
            // e -> (b, b', al, al'):  Q^{bb'}_{al al'} = sum_{be,be'} G[al][be] Sd^{bb'}_{be be'} Gt[be'][al']
            const int b = e / 48, bp = (e / 16) % 3, al = (e / 4) % 4, alp = e % 4;
            double2 q = make_double2(0.0, 0.0);
#pragma unroll
            for (int be = 0; be < 4; ++be) {
                const double2 g1 = make_double2(a.G[2 * (4 * al + be)], a.G[2 * (4 * al + be) + 1]);
                if (g1.x == 0.0 && g1.y == 0.0) continue;
#pragma unroll
                for (int bep = 0; bep < 4; ++bep) {
                    const double2 g2 = make_double2(a.Gt[2 * (4 * bep + alp)], a.Gt[2 * (4 * bep + alp) + 1]);
                    if (g2.x == 0.0 && g2.y == 0.0) continue;
                    q = cfma(cmul(g1, g2), sd[(3 * bep + bp) * 12 + 3 * be + b], q);
                }
            }
            Q[e] = q;     // index ((b*3+bp)*4+al)*4+alp
            // W^{c a'}_{ga' al'} = sum_ga P[ga'][ga] Su2^{c a'}_{ga al'}   (same index pattern: c, a', ga', al')
            double2 w = make_double2(0.0, 0.0);
#pragma unroll
            for (int ga = 0; ga < 4; ++ga) {
                const double2 pp = make_double2(a.P[2 * (4 * al + ga)], a.P[2 * (4 * al + ga) + 1]);
                if (pp.x == 0.0 && pp.y == 0.0) continue;
                w = cfma(pp, s2[(3 * alp + bp) * 12 + 3 * ga + b], w);
            }
            W[e] = w;     // index ((c*3+a')*4+ga')*4+al'
        }
        if (lane < 9) {
            const int c = lane / 3, cp = lane % 3;
            double2 tr = make_double2(0.0, 0.0);
            for (int gap = 0; gap < 4; ++gap)
                for (int ga = 0; ga < 4; ++ga)
                    tr = cfma(make_double2(a.P[2 * (4 * gap + ga)], a.P[2 * (4 * gap + ga) + 1]),
                              s2[(3 * gap + cp) * 12 + 3 * ga + c], tr);
            trP[lane] = tr;
        }
        NUC_SYNC();
        for (int wi = lane; wi < 144; wi += GT) {
            const int e = wi / 4, alp = wi % 4, e1 = e / 6, e2 = e % 6;
            const int ca = c_perm[e1][0], cb = c_perm[e1][1], cc = c_perm[e1][2];
            const int cap = c_perm[e2][0], cbp = c_perm[e2][1], ccp = c_perm[e2][2];
            const double sg = c_psign[e1] * c_psign[e2];
            const double2* q = Q + (cb * 3 + cbp) * 16;
            // direct: sum_al Q_{al al'} Su1^{aa'}_{al al'}  * tr[P Su2^{cc'}]
            double2 d = make_double2(0.0, 0.0);
#pragma unroll
            for (int al = 0; al < 4; ++al) d = cfma(q[al * 4 + alp], s1[(3 * alp + cap) * 12 + 3 * al + ca], d);
            d = cmul(d, trP[cc * 3 + ccp]);
            // exchange: sum_{al, ga'} Q_{al al'} Su1^{ac'}_{al ga'} W^{ca'}_{ga' al'}
            const double2* w = W + (cc * 3 + cap) * 16;
            double2 ex = make_double2(0.0, 0.0);
#pragma unroll
            for (int al = 0; al < 4; ++al) {
                double2 u = make_double2(0.0, 0.0);
#pragma unroll
                for (int gap = 0; gap < 4; ++gap) u = cfma(s1[(3 * gap + ccp) * 12 + 3 * al + ca], w[gap * 4 + alp], u);
                ex = cfma(q[al * 4 + alp], u, ex);
            }
            accr += sg * (d.x - ex.x);
            acci += sg * (d.y - ex.y);
        }
        NUC_SYNC();
    }
    // fixed-order warp sum, one partial per warp
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        accr += __shfl_down_sync(0xffffffffu, accr, o);
        acci += __shfl_down_sync(0xffffffffu, acci, o);
    }
    if ((threadIdx.x & 31) == 0) {
        const int wid = blockIdx.x * MDWF_NUC_WARPS + (threadIdx.x >> 5), nw = a.nblk_t * MDWF_NUC_WARPS;
        a.partial[((long long)t * nw + wid) * 2] = accr;
        a.partial[((long long)t * nw + wid) * 2 + 1] = acci;
    }
#undef NUC_SYNC
}

__global__ void nucleon_finish_kernel(double* corr, const double* partial, int nblk_t, int T, int t0) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    double sr = 0.0, si = 0.0;
    for (int b = 0; b < nblk_t; ++b) { sr += partial[((long long)t * nblk_t + b) * 2]; si += partial[((long long)t * nblk_t + b) * 2 + 1]; }
    const int k = ((t - t0) % T + T) % T;
    corr[2 * k] = sr;
    corr[2 * k + 1] = si;
}

static void mat4mul(const double* A, const double* B, double* C) {   // complex 4x4 row-major [re,im]
    double T[32];
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) {
            double re = 0, im = 0;
            for (int k = 0; k < 4; ++k) {
                const double ar = A[2 * (4 * i + k)], ai = A[2 * (4 * i + k) + 1], br = B[2 * (4 * k + j)], bi = B[2 * (4 * k + j) + 1];
                re += ar * br - ai * bi;
                im += ar * bi + ai * br;
            }
            T[2 * (4 * i + j)] = re;
            T[2 * (4 * i + j) + 1] = im;
        }
    memcpy(C, T, sizeof(T));
}

}  // namespace mdwf

using namespace mdwf;

extern "C" {

int mdwf_wall_inject(mdwf_ctx* c, void* b5, const void* eta4, int ncol, int recon, void* stream) {
    MDWF_ENTER(c);
    if (!b5 || !eta4) MDWF_FAIL(c, MDWF_EINVAL, "null pointer");
    if (ncol < 1 || ncol > MDWF_MAX_RHS) MDWF_FAIL(c, MDWF_EINVAL, "ncol must be in 1..%d", MDWF_MAX_RHS);
    cudaStream_t st = (cudaStream_t)stream;
    OpCtx o;
    o.c = c; o.prec = 64; o.recon = recon; o.st = st; o.gs = c->find_gauge(64, recon);
    if (!o.gs) MDWF_FAIL(c, MDWF_ESTATE, "gauge format (prec 64, recon %d) not loaded", recon);
    mdwf_field *w[2], *fo;
    int rc;
    if ((rc = temp_field(c, 64, ncol, 0, &w[0])) || (rc = temp_field(c, 64, ncol, 5, &w[1])) || (rc = temp_field(c, 64, ncol, 1, &fo))) return rc;
    for (int p = 0; p < 2; ++p)
        if ((rc = launch_wall_pack(c, w[p]->view(), (const double*)eta4, p, ncol, st))) return rc;
    const double d = c->c5 * (4.0 - c->M5) - 1.0;
    const RhsList rl = all_rhs(ncol);
    for (int p = 0; p < 2; ++p) {
        if ((rc = op_hop(o, fo, w[1 - p], p, 0, -1, w[p], -d, 0.5 * c->c5, rl))) return rc;
        if ((rc = unpack_field(fo, (double*)b5, 1, p, st))) return rc;
    }
    return MDWF_OK;
}

int mdwf_wall_project(mdwf_ctx* c, void* q4, const void* psi5, int ncol, void* stream) {
    MDWF_ENTER(c);
    if (!q4 || !psi5 || ncol < 1) MDWF_FAIL(c, MDWF_EINVAL, "bad argument");
    const long long V4 = 2ll * c->g.Vh, n = (long long)ncol * V4 * 12;
    wall_project_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>((double2*)q4, (const double2*)psi5, V4, c->g.Ls, ncol);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

int mdwf_seq_source(mdwf_ctx* c, void* out4d, const void* prop4d, int ncol, const double* Gamma_host, int t_min,
                    int t_max, void* stream) {
    MDWF_ENTER(c);
    if (!out4d || !prop4d || !Gamma_host || ncol < 1) MDWF_FAIL(c, MDWF_EINVAL, "bad argument");
    SeqArgs a;
    a.out = (double2*)out4d; a.in = (const double2*)prop4d;
    a.V4 = 2ll * c->g.Vh; a.V3 = a.V4 / c->g.T; a.ncol = ncol; a.t_min = t_min; a.t_max = t_max;
    memcpy(a.G, Gamma_host, sizeof(a.G));
    const long long n = (long long)ncol * a.V4 * 3;
    seq_source_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(a);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches++;
    return MDWF_OK;
}

int mdwf_nucleon_2pt(mdwf_ctx* c, double* corr, const void* S_u1, const void* S_d, const void* S_u2,
                     const double* proj_host, int t0, void* stream) {
    MDWF_ENTER(c);
    if (!corr || !S_u1 || !S_d || !S_u2 || !proj_host) MDWF_FAIL(c, MDWF_EINVAL, "null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    NucArgs a;
    a.Su1 = (const double2*)S_u1; a.Sd = (const double2*)S_d; a.Su2 = (const double2*)S_u2;
    a.V4 = 2ll * c->g.Vh; a.V3 = a.V4 / c->g.T;
    const int T = c->g.T;
    const int gpb = MDWF_NUC_WARPS / MDWF_NUC_WPS;
    a.nblk_t = (int)std::min<long long>((a.V3 + gpb - 1) / gpb, std::max(1, (c->sm_count * 16) / T));
    // C = gamma_y gamma_t, G = C gamma5, Gt = gamma_t G^dag gamma_t in the DeGrand-Rossi basis (SURVEY 8 Notation)
    const double gy[32] = {0,0, 0,0, 0,0, -1,0,   0,0, 0,0, 1,0, 0,0,   0,0, 1,0, 0,0, 0,0,   -1,0, 0,0, 0,0, 0,0};
    const double gt[32] = {0,0, 0,0, 1,0, 0,0,   0,0, 0,0, 0,0, 1,0,   1,0, 0,0, 0,0, 0,0,   0,0, 1,0, 0,0, 0,0};
    const double g5[32] = {1,0, 0,0, 0,0, 0,0,   0,0, 1,0, 0,0, 0,0,   0,0, 0,0, -1,0, 0,0,   0,0, 0,0, 0,0, -1,0};
    double C[32], G[32], Gd[32], Gt[32];
    mat4mul(gy, gt, C);
    mat4mul(C, g5, G);
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) { Gd[2 * (4 * i + j)] = G[2 * (4 * j + i)]; Gd[2 * (4 * i + j) + 1] = -G[2 * (4 * j + i) + 1]; }
    mat4mul(gt, Gd, Gt);
    mat4mul(Gt, gt, Gt);
    memcpy(a.G, G, sizeof(G));
    memcpy(a.Gt, Gt, sizeof(Gt));
    memcpy(a.P, proj_host, sizeof(a.P));
    double* partial = nullptr;
    const int npart = a.nblk_t * MDWF_NUC_WARPS;
    MDWF_CUDA(c, cudaMallocAsync(&partial, sizeof(double) * 2 * T * npart, st));
    a.partial = partial;
    dim3 grid(a.nblk_t, T);
    const size_t nsm = (size_t)gpb * (5 * 144 + 16) * sizeof(double2);
    if (!c->attr_raised.count((const void*)nucleon_kernel)) {
        MDWF_CUDA(c, cudaFuncSetAttribute(nucleon_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)nsm));
        c->attr_raised.insert((const void*)nucleon_kernel);
    }
    nucleon_kernel<<<grid, 32 * MDWF_NUC_WARPS, nsm, st>>>(a);
    MDWF_CUDA(c, cudaGetLastError());
    nucleon_finish_kernel<<<(T + 63) / 64, 64, 0, st>>>(corr, partial, npart, T, t0);
    MDWF_CUDA(c, cudaGetLastError());
    MDWF_CUDA(c, cudaFreeAsync(partial, st));
    c->launches += 2;
    return MDWF_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// mdwf_nucleon_2pt_noalloc: the same contraction for callers that must not allocate (CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc).  mdwf_nucleon_2pt takes its per-warp partial sums from cudaMallocAsync; here they
// live in a file-scope device array of fixed size that every GPU loading the library holds until exit.
// In HOST code the array's name is only a host-side stand-in, never a device address: the address is asked for once per
// device, with that device current, by cudaGetSymbolAddress, and that pointer is what the kernels get.
// All calls share the array (it keeps the previous call's contents): calls that overlap on the GPU -- different
// streams, or two contexts on one device -- race; serialise them.
// ---------------------------------------------------------------------------------------------
#define MDWF_NUC_SCRATCH_DOUBLES 65536        // 512 KiB: 2 x T x (blocks per timeslice) x MDWF_NUC_WARPS doubles must fit
static __device__ __align__(256) double g_nuc_scratch[MDWF_NUC_SCRATCH_DOUBLES];

#define MDWF_NUC_MAX_DEVICES 64
static double* g_nuc_scratch_ptr[MDWF_NUC_MAX_DEVICES];      // device address of g_nuc_scratch on device d, nullptr = not set up

// once per device, with that device current (MDWF_ENTER): the array's device address and the kernel's shared-memory limit
static int nuc_noalloc_setup(mdwf_ctx* c, size_t nsm, double** ptr) {
    const int dev = c->geo.device;
    if (dev < 0 || dev >= MDWF_NUC_MAX_DEVICES) MDWF_FAIL(c, MDWF_EINVAL, "mdwf_nucleon_2pt_noalloc: device %d outside 0..%d", dev, MDWF_NUC_MAX_DEVICES - 1);
    if (!g_nuc_scratch_ptr[dev]) {
        double* p = nullptr;
        MDWF_CUDA(c, cudaGetSymbolAddress((void**)&p, g_nuc_scratch));
        if (!p) MDWF_FAIL(c, MDWF_ECUDA, "mdwf_nucleon_2pt_noalloc: cudaGetSymbolAddress returned a null address");
        MDWF_CUDA(c, cudaFuncSetAttribute(nucleon_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)nsm));
        g_nuc_scratch_ptr[dev] = p;
    }
    *ptr = g_nuc_scratch_ptr[dev];
    return MDWF_OK;
}

extern "C" {

int64_t mdwf_nucleon_2pt_noalloc_max_bytes(void) { return (int64_t)sizeof(double) * MDWF_NUC_SCRATCH_DOUBLES; }

int mdwf_nucleon_2pt_noalloc(mdwf_ctx* c, double* corr, const void* S_u1, const void* S_d, const void* S_u2,
                             const double* proj_host, int t0, void* stream) {
    MDWF_ENTER(c);
    if (!corr || !S_u1 || !S_d || !S_u2 || !proj_host) MDWF_FAIL(c, MDWF_EINVAL, "null pointer");
    cudaStream_t st = (cudaStream_t)stream;
    NucArgs a;
    a.Su1 = (const double2*)S_u1; a.Sd = (const double2*)S_d; a.Su2 = (const double2*)S_u2;
    a.V4 = 2ll * c->g.Vh; a.V3 = a.V4 / c->g.T;
    const int T = c->g.T;
    const int gpb = MDWF_NUC_WARPS / MDWF_NUC_WPS;
    // the launch shape of mdwf_nucleon_2pt, so that the fixed-order sums are the same sums
    a.nblk_t = (int)std::min<long long>((a.V3 + gpb - 1) / gpb, std::max(1, (c->sm_count * 16) / T));
    const int npart = a.nblk_t * MDWF_NUC_WARPS;
    const long long need = 2ll * T * npart;
    if (need > MDWF_NUC_SCRATCH_DOUBLES)
        MDWF_FAIL(c, MDWF_EINVAL, "mdwf_nucleon_2pt_noalloc: T = %d with %d blocks per timeslice needs %lld bytes of scratch, the "
                  "static array holds %lld (use mdwf_nucleon_2pt)", T, a.nblk_t, need * 8, (long long)sizeof(double) * MDWF_NUC_SCRATCH_DOUBLES);
    // C = gamma_y gamma_t, G = C gamma5, Gt = gamma_t G^dag gamma_t in the DeGrand-Rossi basis (SURVEY 8 Notation)
    const double gy[32] = {0,0, 0,0, 0,0, -1,0,   0,0, 0,0, 1,0, 0,0,   0,0, 1,0, 0,0, 0,0,   -1,0, 0,0, 0,0, 0,0};
    const double gt[32] = {0,0, 0,0, 1,0, 0,0,   0,0, 0,0, 0,0, 1,0,   1,0, 0,0, 0,0, 0,0,   0,0, 1,0, 0,0, 0,0};
    const double g5[32] = {1,0, 0,0, 0,0, 0,0,   0,0, 1,0, 0,0, 0,0,   0,0, 0,0, -1,0, 0,0,   0,0, 0,0, 0,0, -1,0};
    double C[32], G[32], Gd[32], Gt[32];
    mat4mul(gy, gt, C);
    mat4mul(C, g5, G);
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) { Gd[2 * (4 * i + j)] = G[2 * (4 * j + i)]; Gd[2 * (4 * i + j) + 1] = -G[2 * (4 * j + i) + 1]; }
    mat4mul(gt, Gd, Gt);
    mat4mul(Gt, gt, Gt);
    memcpy(a.G, G, sizeof(G));
    memcpy(a.Gt, Gt, sizeof(Gt));
    memcpy(a.P, proj_host, sizeof(a.P));
    const size_t nsm = (size_t)gpb * (5 * 144 + 16) * sizeof(double2);
    double* scratch = nullptr;
    int rc = nuc_noalloc_setup(c, nsm, &scratch);
    if (rc) return rc;
    a.partial = scratch;
    // every slot the finish kernel reads is written by nucleon_kernel of this call; the clear only keeps a kernel that
    // failed to launch from passing off the previous call's sums as its own
    MDWF_CUDA(c, cudaMemsetAsync(scratch, 0, sizeof(double) * (size_t)need, st));
    dim3 grid(a.nblk_t, T);
    nucleon_kernel<<<grid, 32 * MDWF_NUC_WARPS, nsm, st>>>(a);
    MDWF_CUDA(c, cudaGetLastError());
    nucleon_finish_kernel<<<(T + 63) / 64, 64, 0, st>>>(corr, scratch, npart, T, t0);
    MDWF_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return MDWF_OK;
}

}  // extern "C"
