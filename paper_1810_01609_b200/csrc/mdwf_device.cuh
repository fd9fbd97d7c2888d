// csrc/mdwf_device.cuh -- device-side layout, storage traits and spinor/link accessors of the CUDA
// product path (sm_100a).  Private to csrc/.  Shares nothing with oracle/.
//
// Packed layouts:
//   spinor fp64/fp32, one parity, one rhs:  blocks of 32 consecutive 5D sites, each block = vec[c][lane]
//        c = 0..NV-1, 16-byte vectors; 5D site idx = xh*Ls + s (s fastest)
//        fp64: NV = 12 x double2     fp32: NV = 6 x float4
//        reals inside a site are in canonical order r = ((spin*3 + colour)*2 + reim), vector c holds
//        r = c*RPV .. c*RPV+RPV-1.  A thread owns one 5D site idx = xh*Ls + s (s fastest), so a warp
//        reads 512 contiguous bytes per vector index.  rhs are separate fields (stride in bytes).
//   spinor fp16 ("16-bit storage, single-precision computation"; reading R11):
//        48 bytes per 5D site: half[colour 3][spin 4][re,im] -- one 16-byte chunk per colour -- stored in the
//        FRAGMENT ORDER of the tensor-core stencil (mdwf_hop16.cuh).  The rhs are interleaved in groups of RI = 1,
//        2 or 4 inside a 4D site; the RI*Ls "rows" (rhs in group, s) of a site are cut into blocks of 8 rows and a
//        block is stored as [colour chunk 3][row 8][16 B] = 3 x 128 bytes:
//           [group][xh][row block][chunk][row in block][16 B]        (rows padded to a multiple of 8)
//        so (a) the A operand of an m16n8k16 / m16n8k8 MMA is read with six perfectly coalesced 128-byte LDG.32
//        per 16 rows, register <- memory with no conversion, shuffle or shared-memory staging, (b) all rows of a
//        site share one set of link fragments (north_star: links "reused across the Ls slices and across multiple
//        right-hand sides"), (c) one-thread-per-5D-site kernels still read 16 contiguous bytes per lane.
//        One power-of-two fp32 scale per (field, rhs): value = e * half.
//   gauge, per (site parity, mu): vec[c][xh]   fp64: double2 x ceil(R/2), fp32: float4 x ceil(R/4),
//        fp16: 4 x half (8 bytes) x ceil(R/4);  R = 18 | 12 | 8 reals.
#pragma once
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <stdint.h>

namespace mdwf {

// ---------------------------------------------------------------------------------------------
// division by a run-time constant: q = (umulhi(M, n) + n) >> l, exact for 0 <= n < 2^31, 1 <= d < 2^31
// (Granlund-Montgomery round-up method).  Checked exhaustively on the host in tests (fastdiv_selftest).
struct FastDiv {
    uint32_t d, M, l;
    __host__ __device__ __forceinline__ uint32_t div(uint32_t n) const {
#ifdef __CUDA_ARCH__
        return (__umulhi(M, n) + n) >> l;
#else
        return (uint32_t)((((uint64_t)M * n) >> 32) + n) >> l;
#endif
    }
    __host__ __device__ __forceinline__ void divmod(uint32_t n, uint32_t& q, uint32_t& r) const {
        q = div(n);
        r = n - q * d;
    }
};
inline FastDiv make_fastdiv(uint32_t d) {
    FastDiv f;
    f.d = d;
    uint32_t l = 0;
    while ((1ull << l) < d) ++l;
    f.l = l;
    f.M = (uint32_t)((((1ull << l) - d) << 32) / d + 1);
    return f;
}

// ---------------------------------------------------------------------------------------------
struct Geom {
    int X, Y, Z, T, XH;       // XH = X/2
    int Ls;
    int Vh;                   // sites per parity
    int N5h;                  // Vh*Ls = 5D sites per parity (thread count per rhs)
    int bc[4];
    int zc;                   // z-slab depth of the hop traversal (divides Z)
    FastDiv dLs, dXH, dY, dZ;       // canonical decode of xh
    FastDiv dZc, dSlab, dTslab;     // (unused by the tiled traversal; kept for the linear one)
    // 4D tiles of the hop kernel: a block owns txh*ty*tz*tt sites (x fastest); tiles are ordered x, y, z within a
    // z-slab of depth zc, then t, then slab, so that t-neighbours are re-used from L2 and in-tile neighbours from L1
    int txh, ty, tz, tt, nsite;
    int ntc;                            // tiles per (z-slab, timeslice-of-tiles) chunk: blocks run chunk-major, then rhs, then tile
    FastDiv dntc;
    FastDiv dtxh, dty, dtz;             // in-tile decode
    FastDiv dnTx, dnTy, dnTzs, dnTt;    // tile-index decode: tiles per row, per column, per slab depth, per T
};

// fp16 fields carry, per rhs, a power-of-two scale e (value = e * stored half) and a bound nb >= |field|_2 from which
// the scale of whatever is computed from the field is derived ON THE DEVICE (no host round trip): a kernel that writes
// an fp16 field evaluates a ScaleRule  nb_out = sum_i coef_i |num_i/den_i| (sq_i ? sqrt(nb_i) : nb_i)  -- operator-norm
// bounds times the inputs' bounds, refreshed by measured norms wherever a reduction exists -- and stores with
// e_out = 2^ceil(log2(nb_out / 2^15)), so |stored| <= |field|_2 / e_out <= 2^15 can never overflow a half.
struct FieldMeta {
    float e[64];
    double nb[64];
};
struct ScaleTerm {
    const double* nb;      // [64] by rhs id: a norm bound, or (sq != 0) a squared norm
    const double* num;     // optional device scalars [64]: the term is multiplied by |num/den|
    const double* den;
    double coef;
    int sq;
};
struct ScaleRule {
    ScaleTerm t[3];
    int n;                 // 0: the output is not an fp16 field
    FieldMeta* out;        // meta slot of the output field (written by one thread per rhs)
};
__device__ __forceinline__ float eval_scale(const ScaleRule& r, int rhs, bool write) {
    double nb = 0.0;
    for (int i = 0; i < r.n; ++i) {
        const ScaleTerm& t = r.t[i];
        double v = t.nb[rhs];
        if (t.sq) v = sqrt(fmax(v, 0.0));
        double s = t.coef;
        if (t.num) s *= fabs(t.num[rhs]);
        if (t.den) s /= fabs(t.den[rhs]);
        nb += fabs(s) * v;
    }
    float e = 1.0f;
    if (nb > 1e-300 && nb < 1e300) {
        int k;
        frexp(nb * (1.0 / 32768.0), &k);     // nb/2^15 = m 2^k, m in [0.5, 1)  ->  2^k >= nb/2^15
        k = k < -120 ? -120 : k > 120 ? 120 : k;
        e = (float)ldexp(1.0, k);
    }
    if (write && r.out) { r.out->e[rhs] = e; r.out->nb[rhs] = nb; }
    return e;
}

// one packed spinor field set (nrhs fields of one parity)
struct SpinorView {
    void* v;          // vectors
    FieldMeta* m;     // fp16 only: scales / norm bounds of the CURRENT content (read side)
    long long rs;     // rhs stride in BYTES (fp16: stride of a GROUP of 1 << ril rhs)
    int ril;          // fp16 only: log2 of the rhs interleave RI
    int Ls;           // fp16 only
    int sb;           // fp16 only: bytes of one 4D site of a group = ceil(RI*Ls / 8) * 384
    FastDiv dLs;      // fp16 only: idx -> (xh, s)
};

struct GaugeView {
    const void* v[2];   // per parity of the link's base site; [mu][c][xh] vectors
    // fp16 storage only: per parity of the OUTPUT site, the 8 stencil links of every site as the half-precision matrices
    // the stencil multiplies (reconstructed, daggered for backward legs, boundary sign folded): word (re, im) of entry e
    // of leg l at [xh][e 9][l 8]
    const uint32_t* pl[2];
};

// ---------------------------------------------------------------------------------------------
template <typename S> struct Store;
template <> struct Store<double> {
    typedef double real;
    typedef double2 vec;
    static constexpr int NV = 12, RPV = 2, BYTES = 8;
    static constexpr bool HALF = false;
};
template <> struct Store<float> {
    typedef float real;
    typedef float4 vec;
    static constexpr int NV = 6, RPV = 4, BYTES = 4;
    static constexpr bool HALF = false;
};
template <> struct Store<__half> {
    typedef float real;
    typedef uint4 vec;
    static constexpr int NV = 3, RPV = 8, BYTES = 2;
    static constexpr bool HALF = true;
};

__device__ __forceinline__ double2 ldg(const double2* p) { return __ldg(p); }
__device__ __forceinline__ float4 ldg(const float4* p) { return __ldg(p); }
__device__ __forceinline__ uint4 ldg(const uint4* p) { return __ldg(p); }
__device__ __forceinline__ uint2 ldg(const uint2* p) { return __ldg(p); }

__device__ __forceinline__ float2 h2f(uint32_t w) {
    __half2 h = *reinterpret_cast<__half2*>(&w);
    return __half22float2(h);
}
__device__ __forceinline__ uint32_t f2h(float a, float b) {
    __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<uint32_t*>(&h);
}

// Blocked layout: 32 consecutive 5D sites form one block of NV rows of 32 x 16 bytes (+ 32 fp32 scales for
// fp16), so all vectors of a site sit within BLK bytes (one DRAM page, constant offsets between rows).
template <typename S> struct Blk { static constexpr int BYTES = Store<S>::NV * 512; };
template <typename S>
__device__ __forceinline__ const char* site_ptr(const SpinorView& f, int r, int idx) {
    if (Store<S>::HALF) {
        uint32_t xh, sl;
        f.dLs.divmod((uint32_t)idx, xh, sl);
        const int row = (r & ((1 << f.ril) - 1)) * f.Ls + (int)sl;      // chunk c of the site at + c*128
        return reinterpret_cast<const char*>(f.v) + (long long)(r >> f.ril) * f.rs + (long long)xh * f.sb + (row >> 3) * 384 + (row & 7) * 16;
    }
    return reinterpret_cast<const char*>(f.v) + (long long)r * f.rs + (long long)(idx >> 5) * Blk<S>::BYTES + (idx & 31) * 16;
}

// load the 24 reals of 5D site `idx` of rhs `r`.  fp16: returns the UNSCALED values and the scale
// (callers fold the scale into a later multiply); other types: scale = 1.
template <typename S>
__device__ __forceinline__ void load_raw(const SpinorView& f, int r, int idx, int N5h,
                                         typename Store<S>::real v[24], typename Store<S>::real& scale);

template <>
__device__ __forceinline__ void load_raw<double>(const SpinorView& f, int r, int idx, int N5h, double v[24],
                                                 double& scale) {
    const char* p = site_ptr<double>(f, r, idx);
#pragma unroll
    for (int c = 0; c < 12; ++c) {
        double2 t = ldg(reinterpret_cast<const double2*>(p + c * 512));
        v[2 * c] = t.x;
        v[2 * c + 1] = t.y;
    }
    scale = 1.0;
}
template <>
__device__ __forceinline__ void load_raw<float>(const SpinorView& f, int r, int idx, int N5h, float v[24],
                                                float& scale) {
    const char* p = site_ptr<float>(f, r, idx);
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        float4 t = ldg(reinterpret_cast<const float4*>(p + c * 512));
        v[4 * c] = t.x;
        v[4 * c + 1] = t.y;
        v[4 * c + 2] = t.z;
        v[4 * c + 3] = t.w;
    }
    scale = 1.0f;
}
template <>
__device__ __forceinline__ void load_raw<__half>(const SpinorView& f, int r, int idx, int N5h, float v[24],
                                                 float& scale) {
    const char* p = site_ptr<__half>(f, r, idx);
    scale = f.m->e[r];
#pragma unroll
    for (int c = 0; c < 3; ++c) {        // chunk c = colour c: spins 0..3 (re, im)
        uint4 t = ldg(reinterpret_cast<const uint4*>(p + c * 128));
        float2 a = h2f(t.x), b = h2f(t.y), cc = h2f(t.z), d = h2f(t.w);
        v[(0 * 3 + c) * 2] = a.x; v[(0 * 3 + c) * 2 + 1] = a.y;
        v[(1 * 3 + c) * 2] = b.x; v[(1 * 3 + c) * 2 + 1] = b.y;
        v[(2 * 3 + c) * 2] = cc.x; v[(2 * 3 + c) * 2 + 1] = cc.y;
        v[(3 * 3 + c) * 2] = d.x; v[(3 * 3 + c) * 2 + 1] = d.y;
    }
}

// load with the scale applied
template <typename S>
__device__ __forceinline__ void load_spinor(const SpinorView& f, int r, int idx, int N5h,
                                            typename Store<S>::real v[24]) {
    typename Store<S>::real sc;
    load_raw<S>(f, r, idx, N5h, v, sc);
    if (Store<S>::HALF) {
#pragma unroll
        for (int i = 0; i < 24; ++i) v[i] *= sc;
    }
}

// st_<CS>: plain store, or streaming store (evict-first: the stencil's output is not re-read before it has
// left L2, so it should not displace the input sites that neighbouring blocks are about to gather)
template <bool CS, typename V> __device__ __forceinline__ void st_(V* p, V v) {
    if (CS) __stcs(p, v); else *p = v;
}
// two floats -> packed half2, round to nearest, saturating to +-65504 (an overflow becomes a rounding error that the
// next reliable update removes, never an Inf)
__device__ __forceinline__ uint32_t f2h_sat(float a, float b) {
    uint32_t r;
    asm("cvt.rn.satfinite.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(b), "f"(a));
    return r;
}
// store the 24 reals of 5D site `idx`.  fp16 ("16-bit storage, single-precision computation"; DESIGN.md
// R11): stored half = v * oinv with oinv = 1 / (scale of the output field, see ScaleRule); other types ignore oinv.
template <typename S, bool CS = false>
__device__ __forceinline__ void store_spinor(const SpinorView& f, int r, int idx, int N5h,
                                             const typename Store<S>::real v[24], typename Store<S>::real oinv = 1) {
    char* p = const_cast<char*>(site_ptr<S>(f, r, idx));
    if constexpr (sizeof(S) == 8) {
#pragma unroll
        for (int c = 0; c < 12; ++c) st_<CS>(reinterpret_cast<double2*>(p + c * 512), make_double2(v[2 * c], v[2 * c + 1]));
    } else if constexpr (sizeof(S) == 4) {
#pragma unroll
        for (int c = 0; c < 6; ++c)
            st_<CS>(reinterpret_cast<float4*>(p + c * 512), make_float4(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]));
    } else {
#pragma unroll
        for (int c = 0; c < 3; ++c) {      // chunk c = colour c: spins 0..3 (re, im)
            uint4 t;
            t.x = f2h_sat(v[(0 * 3 + c) * 2] * oinv, v[(0 * 3 + c) * 2 + 1] * oinv);
            t.y = f2h_sat(v[(1 * 3 + c) * 2] * oinv, v[(1 * 3 + c) * 2 + 1] * oinv);
            t.z = f2h_sat(v[(2 * 3 + c) * 2] * oinv, v[(2 * 3 + c) * 2 + 1] * oinv);
            t.w = f2h_sat(v[(3 * 3 + c) * 2] * oinv, v[(3 * 3 + c) * 2 + 1] * oinv);
            st_<CS>(reinterpret_cast<uint4*>(p + c * 128), t);
        }
    }
}
// Scale of an fp16 output: thread 0 evaluates the rule, everybody gets 1/e through shared memory (one barrier).
// `writer` blocks (one per rhs) also store the new meta.  No-op (returns 1) for fp32/fp64 outputs.
template <typename S>
__device__ __forceinline__ typename Store<S>::real block_out_scale(const ScaleRule& sr, int rhs, bool writer) {
    if constexpr (!Store<S>::HALF) return 1;
    else {
        __shared__ float s_oinv;
        if (threadIdx.x == 0) s_oinv = 1.0f / eval_scale(sr, rhs, writer);
        __syncthreads();
        return s_oinv;
    }
}

// ---------------------------------------------------------------------------------------------
// Links.  NGV = vectors per link; U[18] = [row][col][re,im] after reconstruction.
template <typename S, int R> struct GaugeFmt;
template <int R> struct GaugeFmt<double, R> { static constexpr int NGV = (R + 1) / 2; typedef double2 vec; };
template <int R> struct GaugeFmt<float, R> { static constexpr int NGV = (R + 3) / 4; typedef float4 vec; };
template <int R> struct GaugeFmt<__half, R> { static constexpr int NGV = (R + 3) / 4; typedef uint2 vec; };

template <typename S, int R>
__device__ __forceinline__ void load_link_raw(const void* base, int mu, int xh, int Vh, typename Store<S>::real g[20]);

#define MDWF_LINK_LOADERS(R)                                                                              \
    template <>                                                                                           \
    __device__ __forceinline__ void load_link_raw<double, R>(const void* base, int mu, int xh, int Vh,    \
                                                             double g[20]) {                              \
        constexpr int NG = GaugeFmt<double, R>::NGV;                                                      \
        const double2* p = reinterpret_cast<const double2*>(base) + (long long)mu * NG * Vh + xh;         \
        _Pragma("unroll") for (int c = 0; c < NG; ++c) {                                                  \
            double2 t = ldg(p + (long long)c * Vh);                                                       \
            g[2 * c] = t.x;                                                                               \
            g[2 * c + 1] = t.y;                                                                           \
        }                                                                                                 \
    }                                                                                                     \
    template <>                                                                                           \
    __device__ __forceinline__ void load_link_raw<float, R>(const void* base, int mu, int xh, int Vh,     \
                                                            float g[20]) {                                \
        constexpr int NG = GaugeFmt<float, R>::NGV;                                                       \
        const float4* p = reinterpret_cast<const float4*>(base) + (long long)mu * NG * Vh + xh;           \
        _Pragma("unroll") for (int c = 0; c < NG; ++c) {                                                  \
            float4 t = ldg(p + (long long)c * Vh);                                                        \
            g[4 * c] = t.x; g[4 * c + 1] = t.y; g[4 * c + 2] = t.z; g[4 * c + 3] = t.w;                   \
        }                                                                                                 \
    }                                                                                                     \
    template <>                                                                                           \
    __device__ __forceinline__ void load_link_raw<__half, R>(const void* base, int mu, int xh, int Vh,    \
                                                             float g[20]) {                               \
        constexpr int NG = GaugeFmt<__half, R>::NGV;                                                      \
        const uint2* p = reinterpret_cast<const uint2*>(base) + (long long)mu * NG * Vh + xh;             \
        _Pragma("unroll") for (int c = 0; c < NG; ++c) {                                                  \
            uint2 t = ldg(p + (long long)c * Vh);                                                         \
            float2 a = h2f(t.x), b = h2f(t.y);                                                            \
            g[4 * c] = a.x; g[4 * c + 1] = a.y; g[4 * c + 2] = b.x; g[4 * c + 3] = b.y;                   \
        }                                                                                                 \
    }
MDWF_LINK_LOADERS(18)
MDWF_LINK_LOADERS(12)
MDWF_LINK_LOADERS(8)
#undef MDWF_LINK_LOADERS

template <typename T> __device__ __forceinline__ T fma_(T a, T b, T c);
template <> __device__ __forceinline__ float fma_<float>(float a, float b, float c) { return __fmaf_rn(a, b, c); }
template <> __device__ __forceinline__ double fma_<double>(double a, double b, double c) { return __fma_rn(a, b, c); }

template <typename T> __device__ __forceinline__ void sincos_(T a, T& s, T& c);
template <> __device__ __forceinline__ void sincos_<double>(double a, double& s, double& c) { sincos(a, &s, &c); }
template <> __device__ __forceinline__ void sincos_<float>(float a, float& s, float& c) { sincosf(a, &s, &c); }
template <typename T> __device__ __forceinline__ T sqrt_(T a);
template <> __device__ __forceinline__ double sqrt_<double>(double a) { return sqrt(a); }
template <> __device__ __forceinline__ float sqrt_<float>(float a) { return sqrtf(a); }

// rows 0,1 known -> row 2 = conj(row0 x row1)   (SURVEY A12, 12-real format)
template <typename T> __device__ __forceinline__ void row2_from_rows01(T U[18]) {
#define RE(r, c) U[((r) * 3 + (c)) * 2]
#define IM(r, c) U[((r) * 3 + (c)) * 2 + 1]
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int c1 = (c + 1) % 3, c2 = (c + 2) % 3;
        // (row0 x row1)_c = r0[c1]*r1[c2] - r0[c2]*r1[c1]; conj -> negate imaginary part
        const T re = RE(0, c1) * RE(1, c2) - IM(0, c1) * IM(1, c2) - RE(0, c2) * RE(1, c1) + IM(0, c2) * IM(1, c1);
        const T im = RE(0, c1) * IM(1, c2) + IM(0, c1) * RE(1, c2) - RE(0, c2) * IM(1, c1) - IM(0, c2) * RE(1, c1);
        RE(2, c) = re;
        IM(2, c) = -im;
    }
#undef RE
#undef IM
}

// 8-real format: g = {a2.re,a2.im,a3.re,a3.im,b1.re,b1.im, arg a1, arg c1}; fp16 stores the
// two phases divided by pi.  rows: (a1,a2,a3), (b1,b2,b3), (c1,c2,c3).
template <typename T, bool PHASE_OVER_PI>
__device__ __forceinline__ void reconstruct8(const T g[8], T U[18]) {
    const T a2r = g[0], a2i = g[1], a3r = g[2], a3i = g[3], b1r = g[4], b1i = g[5];
    T tha = g[6], thc = g[7];
    if (PHASE_OVER_PI) { tha *= (T)3.14159265358979323846; thc *= (T)3.14159265358979323846; }
    const T N = a2r * a2r + a2i * a2i + a3r * a3r + a3i * a3i;
    const T ma = sqrt_<T>(fmax((T)0, (T)1 - N));
    const T mc = sqrt_<T>(fmax((T)0, N - b1r * b1r - b1i * b1i));
    T sa, ca, sc, cc;
    sincos_<T>(tha, sa, ca);
    sincos_<T>(thc, sc, cc);
    const T a1r = ma * ca, a1i = ma * sa, c1r = mc * cc, c1i = mc * sc;
    const T iN = (T)1 / N;
    // p = conj(a1)*b1, q = conj(a1)*c1
    const T pr = a1r * b1r + a1i * b1i, pi = a1r * b1i - a1i * b1r;
    const T qr = a1r * c1r + a1i * c1i, qi = a1r * c1i - a1i * c1r;
    // b2 = -(p a2 + conj(c1) conj(a3))/N ; b3 = (-p a3 + conj(c1) conj(a2))/N
    // c2 = (-q a2 + conj(b1) conj(a3))/N ; c3 = -(q a3 + conj(b1) conj(a2))/N
    // conj(u) conj(v) = conj(u v)
    const T c1a3r = c1r * a3r - c1i * a3i, c1a3i = c1r * a3i + c1i * a3r;
    const T c1a2r = c1r * a2r - c1i * a2i, c1a2i = c1r * a2i + c1i * a2r;
    const T b1a3r = b1r * a3r - b1i * a3i, b1a3i = b1r * a3i + b1i * a3r;
    const T b1a2r = b1r * a2r - b1i * a2i, b1a2i = b1r * a2i + b1i * a2r;
    U[0] = a1r; U[1] = a1i; U[2] = a2r; U[3] = a2i; U[4] = a3r; U[5] = a3i;
    U[6] = b1r; U[7] = b1i;
    U[8] = -((pr * a2r - pi * a2i) + c1a3r) * iN;
    U[9] = -((pr * a2i + pi * a2r) - c1a3i) * iN;
    U[10] = (-(pr * a3r - pi * a3i) + c1a2r) * iN;
    U[11] = (-(pr * a3i + pi * a3r) - c1a2i) * iN;
    U[12] = c1r; U[13] = c1i;
    U[14] = (-(qr * a2r - qi * a2i) + b1a3r) * iN;
    U[15] = (-(qr * a2i + qi * a2r) - b1a3i) * iN;
    U[16] = -((qr * a3r - qi * a3i) + b1a2r) * iN;
    U[17] = -((qr * a3i + qi * a3r) - b1a2i) * iN;
}

template <typename S, int R>
__device__ __forceinline__ void load_link(const void* base, int mu, int xh, int Vh, typename Store<S>::real U[18]) {
    typedef typename Store<S>::real T;
    T g[20];
    load_link_raw<S, R>(base, mu, xh, Vh, g);
    if (R == 18) {
#pragma unroll
        for (int i = 0; i < 18; ++i) U[i] = g[i];
    } else if (R == 12) {
#pragma unroll
        for (int i = 0; i < 12; ++i) U[i] = g[i];
        row2_from_rows01<T>(U);
    } else {
        reconstruct8<T, Store<S>::HALF>(g, U);
    }
}

}  // namespace mdwf
