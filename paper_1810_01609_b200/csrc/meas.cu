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
struct NucArgs {
    const double2 *Su1, *Sd, *Su2;
    double* partial;       // [T][nblk_t][2]
    long long V4, V3;
    int nblk_t;            // blocks per timeslice
    double G[32], Gt[32], P[32];
    // G = C gamma5 and Gt = gamma_t G^dag gamma_t are signed permutation matrices (one non-zero per row and column; checked
    // on the host): Q_{al al'} = sum G[al][be] Sd_{be be'} Gt[be'][al'] = qc[al][al'] Sd_{gb[al] gtb[al']}
    int gb[4], gtb[4];
    double qc[32];         // qc[al][al'] = G[al][gb[al]] * Gt[gtb[al']][al'], complex
};
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 cfma(double2 a, double2 b, double2 c) {
    return make_double2(c.x + a.x * b.x - a.y * b.y, c.y + a.x * b.y + a.y * b.x);
}

#define MDWF_NUC_SPB 4        // sites per block and pass
#define MDWF_NUC_WARPS 5      // warps per block: 36 lanes per site (one per pair of colour permutations) = 144 of the 160 threads
#define MDWF_NUC_BLK 17       // stride of a 4x4 spin block in shared memory (double2): 8 consecutive blocks cover all banks once
#define MDWF_NUC_SITE (5 * 9 * MDWF_NUC_BLK)                 // per site: Su1, Sd, Su2, Q, W as 9 colour-pair blocks each
#define MDWF_NUC_SMEM ((MDWF_NUC_SPB * MDWF_NUC_SITE + 32) * sizeof(double2))   // + qc, P
__constant__ int c_perm[6][3] = {{0, 1, 2}, {1, 2, 0}, {2, 0, 1}, {0, 2, 1}, {2, 1, 0}, {1, 0, 2}};
__constant__ double c_psign[6] = {1, 1, 1, -1, -1, -1};
// A block handles MDWF_NUC_SPB sites per pass in three phases separated by block barriers (three blocks per SM overlap
// each other's phases):
//  1. the three propagators of the sites -> shared memory as 4x4 spin blocks per colour pair,
//     B^{xy}[al*4 + be] = S^{xy}_{al be} = S[col 3 be + y][site][3 al + x]   (x sink colour, y source colour);
//  2. Q^{bb'} = G Sd^{bb'} Gt and W^{ca'} = P Su2^{ca'} for the 9 colour pairs (tr[P Su2^{cc'}] is the trace of W^{cc'});
//  3. one lane per (site, e1, e2), e1 = (a b c), e2 = (a' b' c') colour permutations: W^{ca'} stays in registers while the
//     rows of Q^{bb'}, Su1^{ac'} and Su1^{aa'} stream through: 96 complex multiply-adds for 68 16-byte loads.
__global__ void __launch_bounds__(32 * MDWF_NUC_WARPS, 3) nucleon_kernel(const NucArgs a) {
    extern __shared__ __align__(16) unsigned char nuc_smem[];
    double2* sm = reinterpret_cast<double2*>(nuc_smem);
    double2* sC = sm + MDWF_NUC_SPB * MDWF_NUC_SITE;          // qc[16], P[16]
    const int tid = threadIdx.x, NT = 32 * MDWF_NUC_WARPS;
    int gb_me = 0, gtb_me = 0;                                // phase 2: this thread's element is (al, al') = ((tid >> 2) & 3, tid & 3)
    if (tid < 32) {
        const double* src = tid < 16 ? a.qc : a.P;
        const int k = tid & 15;
        double re = 0.0, im = 0.0;
#pragma unroll
        for (int q = 0; q < 16; ++q)
            if (q == k) { re = src[2 * q]; im = src[2 * q + 1]; }      // (no dynamic indexing of the kernel parameters)
        sC[tid] = make_double2(re, im);
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (q == ((tid >> 2) & 3)) gb_me = a.gb[q];
        if (q == (tid & 3)) gtb_me = a.gtb[q];
    }
    const int t = blockIdx.y;
    double accr = 0.0, acci = 0.0;
    const int my_site = tid / 36, item = tid - 36 * my_site, e1 = (item / 6) % 6, e2 = item % 6;
    const int ca = c_perm[e1][0], cb = c_perm[e1][1], cc = c_perm[e1][2];
    const int cap = c_perm[e2][0], cbp = c_perm[e2][1], ccp = c_perm[e2][2];
    const double sg = c_psign[e1] * c_psign[e2];
    constexpr int NEL = 3 * 12 * MDWF_NUC_SPB * 12;            // propagator elements per pass
    constexpr int NLD = (NEL + 32 * MDWF_NUC_WARPS - 1) / (32 * MDWF_NUC_WARPS);
    for (long long xs0 = (long long)blockIdx.x * MDWF_NUC_SPB; xs0 < a.V3; xs0 += (long long)a.nblk_t * MDWF_NUC_SPB) {
        const int nsite = (int)min((long long)MDWF_NUC_SPB, a.V3 - xs0);
        const long long x0 = (long long)t * a.V3 + xs0;
        // ---- phase 1: element i -> (prop, col, site, k): runs of SPB * 192 contiguous bytes per (prop, col); all loads of a
        // thread are issued before the first store
        double2 v[NLD];
#pragma unroll
        for (int n = 0; n < NLD; ++n) {
            const int i = tid + NT * n;
            const int k = i % 12, r = i / 12, site = r % MDWF_NUC_SPB, pc = r / MDWF_NUC_SPB, col = pc % 12, prop = pc / 12;
            const double2* src = prop == 0 ? a.Su1 : prop == 1 ? a.Sd : a.Su2;
            v[n] = (i < NEL && site < nsite) ? __ldg(src + ((long long)col * a.V4 + x0 + site) * 12 + k) : make_double2(0.0, 0.0);
        }
        __syncthreads();                                       // the previous pass is through with the blocks
#pragma unroll
        for (int n = 0; n < NLD; ++n) {
            const int i = tid + NT * n;
            const int k = i % 12, r = i / 12, site = r % MDWF_NUC_SPB, pc = r / MDWF_NUC_SPB, col = pc % 12, prop = pc / 12;
            const int be = col / 3, y = col - 3 * be, al = k / 3, x = k - 3 * al;
            if (i < NEL) sm[site * MDWF_NUC_SITE + (prop * 9 + x * 3 + y) * MDWF_NUC_BLK + al * 4 + be] = v[n];
        }
        __syncthreads();
        // ---- phase 2: Q (array 3) and W (array 4): element j -> (site, Q|W, colour pair, al, al'), (al, al') = j & 15 is the
        // same for every element of a thread (NT is a multiple of 16)
        for (int j = tid; j < MDWF_NUC_SPB * 288; j += NT) {
            const int site = j / 288, e = j - 288 * site, isW = e >= 144, blk = (e - 144 * isW) >> 4, al = (j >> 2) & 3, alp = j & 3;
            double2* S = sm + site * MDWF_NUC_SITE;
            if (!isW) {
                S[(27 + blk) * MDWF_NUC_BLK + al * 4 + alp] = cmul(sC[al * 4 + alp], S[(9 + blk) * MDWF_NUC_BLK + gb_me * 4 + gtb_me]);
            } else {
                const double2* B = S + (18 + blk) * MDWF_NUC_BLK;                   // Su2^{ca'}
                double2 r = make_double2(0.0, 0.0);
#pragma unroll
                for (int ga = 0; ga < 4; ++ga) r = cfma(sC[16 + al * 4 + ga], B[ga * 4 + alp], r);
                S[(36 + blk) * MDWF_NUC_BLK + al * 4 + alp] = r;
            }
        }
        __syncthreads();
        // ---- phase 3
        if (my_site < nsite) {
            const double2* S = sm + my_site * MDWF_NUC_SITE;
            const double2* Wb = S + (36 + cc * 3 + cap) * MDWF_NUC_BLK;
            const double2* Wt = S + (36 + cc * 3 + ccp) * MDWF_NUC_BLK;
            const double2* Qb = S + (27 + cb * 3 + cbp) * MDWF_NUC_BLK;
            const double2* Sx = S + (ca * 3 + ccp) * MDWF_NUC_BLK;                  // Su1^{ac'}
            const double2* Sdr = S + (ca * 3 + cap) * MDWF_NUC_BLK;                 // Su1^{aa'}
            double2 w[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) w[i] = Wb[i];
            const double2 trp = cadd(cadd(Wt[0], Wt[5]), cadd(Wt[10], Wt[15]));
            double2 d = make_double2(0.0, 0.0), ex = make_double2(0.0, 0.0);
#pragma unroll
            for (int al = 0; al < 4; ++al) {
                double2 q[4], sx[4], sd[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) { q[i] = Qb[al * 4 + i]; sx[i] = Sx[al * 4 + i]; sd[i] = Sdr[al * 4 + i]; }
#pragma unroll
                for (int alp = 0; alp < 4; ++alp) {
                    double2 u = make_double2(0.0, 0.0);
#pragma unroll
                    for (int gap = 0; gap < 4; ++gap) u = cfma(sx[gap], w[gap * 4 + alp], u);
                    ex = cfma(q[alp], u, ex);
                    d = cfma(q[alp], sd[alp], d);
                }
            }
            d = cmul(d, trp);
            accr += sg * (d.x - ex.x);
            acci += sg * (d.y - ex.y);
        }
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

// C = gamma_y gamma_t, G = C gamma5, Gt = gamma_t G^dag gamma_t in the DeGrand-Rossi basis (SURVEY 8 Notation), the projector,
// and the signed-permutation form of G and Gt that the kernel's phase 2 uses
static int nuc_fill_args(mdwf_ctx* c, NucArgs& a, const double* proj_host) {
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
    for (int i = 0; i < 4; ++i) {
        int nr = 0, ncol = 0;
        for (int j = 0; j < 4; ++j) {
            if (G[2 * (4 * i + j)] != 0.0 || G[2 * (4 * i + j) + 1] != 0.0) { a.gb[i] = j; ++nr; }          // row i of G
            if (Gt[2 * (4 * j + i)] != 0.0 || Gt[2 * (4 * j + i) + 1] != 0.0) { a.gtb[i] = j; ++ncol; }     // column i of Gt
        }
        if (nr != 1 || ncol != 1) MDWF_FAIL(c, MDWF_ECUDA, "internal: C gamma5 is not a signed permutation in this basis");
    }
    for (int al = 0; al < 4; ++al)
        for (int alp = 0; alp < 4; ++alp) {
            const double gr = G[2 * (4 * al + a.gb[al])], gi = G[2 * (4 * al + a.gb[al]) + 1];
            const double hr = Gt[2 * (4 * a.gtb[alp] + alp)], hi = Gt[2 * (4 * a.gtb[alp] + alp) + 1];
            a.qc[2 * (4 * al + alp)] = gr * hr - gi * hi;
            a.qc[2 * (4 * al + alp) + 1] = gr * hi + gi * hr;
        }
    return MDWF_OK;
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
    const int gpb = MDWF_NUC_SPB;
    a.nblk_t = (int)std::min<long long>((a.V3 + gpb - 1) / gpb, std::max(1, (c->sm_count * 16) / T));
    { const int rcf = nuc_fill_args(c, a, proj_host); if (rcf) return rcf; }
    double* partial = nullptr;
    const int npart = a.nblk_t * MDWF_NUC_WARPS;
    MDWF_CUDA(c, cudaMallocAsync(&partial, sizeof(double) * 2 * T * npart, st));
    a.partial = partial;
    dim3 grid(a.nblk_t, T);
    const size_t nsm = MDWF_NUC_SMEM;
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
    const int gpb = MDWF_NUC_SPB;
    // the launch shape of mdwf_nucleon_2pt, so that the fixed-order sums are the same sums
    a.nblk_t = (int)std::min<long long>((a.V3 + gpb - 1) / gpb, std::max(1, (c->sm_count * 16) / T));
    const int npart = a.nblk_t * MDWF_NUC_WARPS;
    const long long need = 2ll * T * npart;
    if (need > MDWF_NUC_SCRATCH_DOUBLES)
        MDWF_FAIL(c, MDWF_EINVAL, "mdwf_nucleon_2pt_noalloc: T = %d with %d blocks per timeslice needs %lld bytes of scratch, the "
                  "static array holds %lld (use mdwf_nucleon_2pt)", T, a.nblk_t, need * 8, (long long)sizeof(double) * MDWF_NUC_SCRATCH_DOUBLES);
    { const int rcf = nuc_fill_args(c, a, proj_host); if (rcf) return rcf; }
    const size_t nsm = MDWF_NUC_SMEM;
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
