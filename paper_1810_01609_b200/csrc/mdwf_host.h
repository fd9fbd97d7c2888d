// csrc/mdwf_host.h -- host-side context and launcher prototypes of libmdwf.so (private to csrc/).
#pragma once
#include <string>
#include <vector>
#include <map>
#include <set>
#include <cstdio>
#include <cstddef>
#include <cstring>
#include "../../include/mdwf.h"
#include "mdwf_blas.cuh"

// Ls x Ls chirality-block matrices kept on the device (fp64 and fp32 copies), layout Gt[chi][s'][s]
enum MatId { MAT_A = 0, MAT_M5, MAT_M5INV, MAT_AM5INV, MAT_A_D, MAT_M5_D, MAT_M5INV_D, MAT_AM5INV_D, MAT_COUNT };

struct GaugeSet {
    int prec, recon;
    void* v[2];
    size_t bytes_per_parity;
    uint32_t* pl[2];    // prec 16: stencil-ready half-precision links (GaugeView::pl), else nullptr
};

// A packed field set.  fp16 fields own two FieldMeta slots (scales / norm bounds, mdwf_device.cuh): readers use slot
// `cur`, the kernel that rewrites the field fills the other one (so in-place updates never race) and the host then
// calls flip().
struct mdwf_field {
    mdwf_ctx* ctx;
    int prec, nrhs;
    void* v;
    mdwf::FieldMeta* meta;     // device, [2]; nullptr unless prec == 16
    int cur;
    int rhs0;                  // rhs id of slot 0 (temporaries that serve a window of a larger batch), normally 0
    size_t bytes;
    size_t rs;                 // bytes between rhs (fp16: between rhs groups)
    bool owns, owns_meta;      // v / meta were cudaMalloc'ed by alloc_field (else they live in a workspace)
    mdwf::SpinorView view() const;
    mdwf::FieldMeta* rmeta() const { return meta ? meta + cur : nullptr; }
    mdwf::FieldMeta* wmeta() const { return meta ? meta + (cur ^ 1) : nullptr; }
    void flip() { if (meta) cur ^= 1; }
    const double* nb() const { return meta ? reinterpret_cast<const double*>(reinterpret_cast<const char*>(meta + cur) + offsetof(mdwf::FieldMeta, nb)) : nullptr; }
    double* nb_w() const { return meta ? reinterpret_cast<double*>(reinterpret_cast<char*>(meta + cur) + offsetof(mdwf::FieldMeta, nb)) : nullptr; }
};

namespace mdwf { struct Tile16Host; }

struct mdwf_ctx {
    mdwf_geometry geo;
    double M5, b5, c5, mf;
    mdwf::Geom g;
    mdwf::Geom ghop[3];
    std::map<int, mdwf::Geom> ghop_multi;   // the same for launches with several rhs (key cls*100 + nact): shallower slabs
    int zc_forced;             // > 0: mdwf_set_tiling fixed the slab depth        // the same with the hop traversal's z-slab depth for fp16 / fp32 / fp64 storage
    int block;                 // threads per block (fp32 class): a multiple of Ls, <= 256
    int nblk;                  // blocks per rhs = N5h / block (fp32 class)
    int blk_cls[3], nblk_cls[3];   // the same per storage class (0 fp16, 1 fp32, 2 fp64): fp16 uses smaller blocks
    std::vector<GaugeSet> gauges;
    mdwf::LsOp lsop[MAT_COUNT];
    double* partial;           // [64][nblk] per-block partial sums
    double* dscal;             // device scalars [8][64]
    double* hscal;             // pinned host mirror [8][64]
    std::map<long long, std::vector<mdwf_field*> > temps;   // cached work fields keyed by prec*1000+nrhs
    std::string err;
    long long launches;
    // optional per-launch timing of the hop kernel (CUDA events on the launching stream), by class:
    // 0 = fp16 storage, 1 = fp32, 2 = fp64
    int prof_on;
    struct ProfRec { cudaEvent_t e0, e1; int cls; double bytes, flops; };
    std::vector<ProfRec> prof_pending;
    std::vector<cudaEvent_t> prof_pool;
    // classes 0..2: hop by storage class; 3: s-direction kernel, 4: x/r update, 5: p update, 6: reduction finish, 7: axpby/convert
    double prof_ms[8], prof_bytes[8], prof_flops[8];
    long long prof_n[8];
    int sm_count;
    double lsop_norm[MAT_COUNT];   // 2-norm bounds of the s-direction operators (fp16 scale rules)
    mdwf::Tile16Host* tile16[3];   // tile tables of the fp16 tensor-core stencil per rhs interleave (built on first use)
    int tile16_forced[4], tile16_nw;
    std::set<const void*> attr_raised;   // kernels whose dynamic shared-memory limit was raised on THIS device
    int partial_nblk;              // partial sums per rhs written by the last kernel that filled `partial`
    size_t partial_cap;            // doubles per rhs in `partial`
    mdwf::CgCtl* dctl;             // device-side loop control of the inner CG (mdwf_blas.cuh) and its pinned staging copy / mirror
    mdwf::CgCtl* hctl_stage;
    mdwf::CgCtlHost* hctl;
    // launch parameters found by mdwf_autotune (tune.cu), keyed by kernel / lattice / Ls / rows or rhs in flight:
    // "hop16/..." -> {lx, ly, lz, lt, warps}; "hop32/..." and "hop64/..." -> {zc}
    std::map<std::string, std::vector<int> > tune;
    void* ws;                      // solver workspace: library-owned (kept between calls) or caller-supplied
    size_t ws_bytes;
    bool ws_external;
    const GaugeSet* find_gauge(int prec, int recon) const {
        for (size_t i = 0; i < gauges.size(); ++i)
            if (gauges[i].prec == prec && gauges[i].recon == recon) return &gauges[i];
        return nullptr;
    }
};

#define MDWF_FAIL(ctx, code, ...)                          \
    do {                                                   \
        char _b[512];                                      \
        snprintf(_b, sizeof(_b), __VA_ARGS__);             \
        (ctx)->err = _b;                                   \
        return (code);                                     \
    } while (0)
// every entry point runs on the context's device, whatever the caller's current device is
#define MDWF_ENTER(ctx)                                                                                   \
    do {                                                                                                  \
        if (!(ctx)) return MDWF_EINVAL;                                                                   \
        if (cudaSetDevice((ctx)->geo.device) != cudaSuccess) { cudaGetLastError(); (ctx)->err = "cudaSetDevice failed"; return MDWF_ECUDA; } \
    } while (0)
#define MDWF_CUDA(ctx, expr)                                                                             \
    do {                                                                                                 \
        cudaError_t _e = (expr);                                                                         \
        if (_e != cudaSuccess) MDWF_FAIL(ctx, MDWF_ECUDA, "%s: %s (%s:%d)", #expr, cudaGetErrorString(_e), \
                                         __FILE__, __LINE__);                                            \
    } while (0)

namespace mdwf {

inline RhsList all_rhs(int n) {
    RhsList r;
    memset(&r, 0, sizeof(r));
    r.nact = n;
    for (int i = 0; i < 64; ++i) r.rhs[i] = i < n ? i : 0;
    return r;
}

size_t field_bytes(const Geom& g, int prec, int nrhs);
int half_ril(int nrhs, int Ls);
int half_site_bytes(int nrhs, int Ls);
int alloc_field(mdwf_ctx* c, int prec, int nrhs, mdwf_field** out);
// a field whose vectors live at `mem` (field_bytes() bytes, 256-byte aligned) instead of their own allocation
int wrap_field(mdwf_ctx* c, int prec, int nrhs, void* mem, void* meta_mem, mdwf_field** out);
void free_field(mdwf_field* f);
// cached temporaries: slot-th work field of (prec, nrhs)
int temp_field(mdwf_ctx* c, int prec, int nrhs, int slot, mdwf_field** out);

// ---- launchers (each returns MDWF_OK or an error code with ctx->err set) --------------------------
// out = H in (fused == 0) or cx*xin + ch*G*(H in) (fused != 0; G/xin optional; partial optional)
int launch_hop(mdwf_ctx* c, int prec, int recon, int dagger, int fused, HopArgs& a, cudaStream_t st);
int launch_ls(mdwf_ctx* c, int prec, LsArgs& a, cudaStream_t st);
int launch_axpby(mdwf_ctx* c, int prec_out, int prec_a, int prec_b, AxpbyArgs& a, cudaStream_t st);
int launch_cg_xr(mdwf_ctx* c, int prec_x, int prec, CgXrArgs& a, cudaStream_t st);
int launch_cg_p(mdwf_ctx* c, int prec, CgPArgs& a, cudaStream_t st);
// sums the partials of the LAST kernel that wrote them (c->partial_nblk per rhs); nb: optional norm-bound slot of the
// fp16 field that was just measured
struct FinishCtl { const int* stop; CgCtl* ctl; CgCtlHost* hctl; const double* pap; int seq; };
int launch_finish(mdwf_ctx* c, const RhsList& rl, double* out, double* out2, cudaStream_t st, double* nb = nullptr,
                  const FinishCtl* fc = nullptr);
inline int cls_of(int prec) { return prec == 16 ? 0 : prec == 32 ? 1 : 2; }
// per-launch event timing of a site-local kernel while mdwf_profile is on (classes 3..7)
struct ProfScope {
    mdwf_ctx* c; cudaStream_t st; mdwf_ctx::ProfRec r; bool on;
    ProfScope(mdwf_ctx* c_, int cls, cudaStream_t st_);
    ~ProfScope();
};
int launch_pack(mdwf_ctx* c, int prec, bool unpack, PackArgs& a, cudaStream_t st);
int pack_field(mdwf_field* f, const double* canon, int full, int par, cudaStream_t st);
int unpack_field(const mdwf_field* f, double* canon, int full, int par, cudaStream_t st);
int pack_slices(mdwf_field* f, int rhs, double* stage, int s0, int ns, int par, bool unpack, cudaStream_t st);
const mdwf::Geom& hop_geom(mdwf_ctx* c, int cls, int nact);
void set_zc(mdwf_ctx* c, int want);                       // force (want > 0) or release (0) the z-slab depth of hop_kernel
std::string tune_key_tile16(const mdwf_ctx* c, int rows); // rows = (rhs per interleave group) * Ls
std::string tune_key_zc(const mdwf_ctx* c, int cls, int nact);
void tune_invalidate(mdwf_ctx* c);                        // drop the launch tables built from forced / tuned parameters
int pack_gauge(mdwf_ctx* c, const void* U, int prec, int recon, GaugeSet* gs, cudaStream_t st);
void free_gauge(GaugeSet* gs);

// ---- composite operators on packed fields (solver + API) ------------------------------------------
struct OpCtx {
    mdwf_ctx* c;
    int prec, recon;
    const GaugeSet* gs;
    cudaStream_t st;
    const int* stop = nullptr;   // gate of the launches (HopArgs::stop)
};
// simple helpers: out = cx*xin + ch*G*in ; out = cx*xin + ch*G*H(in).  All fields of one call have precision o.prec;
// for fp16 the scale rule of the output is built here (operator-norm bounds x the inputs' norm bounds) and the
// output's meta slot is flipped after the launch.
int op_ls(const OpCtx& o, mdwf_field* out, const mdwf_field* in, int mat, const mdwf_field* xin, double cx,
          double ch, const RhsList& rl, double* partial = nullptr, int write = 1);
int op_hop(const OpCtx& o, mdwf_field* out, const mdwf_field* in, int out_par, int dagger, int mat,
           const mdwf_field* xin, double cx, double ch, const RhsList& rl, double* partial = nullptr);
// Schur operator: out = Dhat/Mhat (dagger) in, parity p; t1, t2 are work fields; if partial != nullptr the
// per-block |out|^2 sums are written there (to be finished with launch_finish)
int op_schur(const OpCtx& o, mdwf_field* out, const mdwf_field* in, int par, int dagger, int symmetric,
             mdwf_field* t1, mdwf_field* t2, const RhsList& rl, double* partial = nullptr,
             int first_factor_done = 0);   // non-dagger only: t1 already holds A*in (fused into the CG p-update)
// fp16 scale rule  nb_out = ca nb(a) + cb nb(b)  (b optional); n = 0 when out is not fp16
ScaleRule rule_lin(const mdwf_field* out, const mdwf_field* a, double ca, const mdwf_field* b = nullptr, double cb = 0.0);
int get_tile16(mdwf_ctx* c, int ril, Tile16Host** out);
void free_tile16(Tile16Host* th);

int solve_impl(mdwf_ctx* c, void* x, const void* b, int nrhs, const mdwf_solve_opts* opts, mdwf_solve_info* info,
               cudaStream_t st, bool host_buffers);
int solve_packed_impl(mdwf_ctx* c, mdwf_field* even, mdwf_field* odd, const mdwf_solve_opts* opts, mdwf_solve_info* info,
                      cudaStream_t st);
}  // namespace mdwf
