/* include/mdwf.h -- C-ABI boundary of the B200-native MDWF hot path (libmdwf.so).
 *
 * What it is.  The paper (reference PAPER.md) names its method only: "Moebius Domain-Wall
 * discretization", a "radius-one stencil" with "12x12 dense" spin-colour blocks,
 * a "red-black preconditioned" operator solved by "CG on the normal equations" in "double-half"
 * mixed precision with "reliable updates", Feynman-Hellmann propagators
 * and nucleon contractions.  The operator definitions used here
 * are the readings fixed in SURVEY.md section 8 ("Notation", A1-A23) and restated in DESIGN.md.
 *
 * Conventions for every call
 *  - returns int: 0 = MDWF_OK, <0 = error, >0 = soft status.  Nothing throws or exits.
 *    mdwf_last_error(ctx) gives a message owned by ctx (valid until the next call on ctx).
 *  - every data pointer is a DEVICE pointer owned by the caller unless the name ends in _host.
 *    The library never frees or retains caller memory past the call; mdwf_load_gauge and
 *    mdwf_field_pack make their own packed copies.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls are
 *    asynchronous on it, except mdwf_solve* (host-visible info => synchronises before returning)
 *    and the *_host variants.
 *  - canonical interchange layouts (fp64, x fastest): x4 = x + X*(y + Y*(z + Z*t));
 *      5D spinor  psi[rhs][s][site][spin 4][colour 3][re,im]   site = x4 (full lattice) or
 *                                                              xh = x4>>1 over the sites of one parity
 *      gauge      U[mu][x4][row 3][col 3][re,im]               U_mu(x) = link from x to x+mu
 *      4D field   eta[col][x4][spin][colour][re,im]            col = 3*spin_src + colour_src
 *  - there is no CPU fallback: every entry point needs a CUDA device.
 *  - a context (and the fields created from it) must not be used from two host threads at the same time; separate
 *    contexts are independent.
 */
#ifndef MDWF_H
#define MDWF_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define MDWF_OK 0
#define MDWF_EINVAL (-1)
#define MDWF_ENOMEM (-2)
#define MDWF_ECUDA (-3)
#define MDWF_ESTATE (-4)
#define MDWF_NOT_CONVERGED 1
#define MDWF_BREAKDOWN 2

/* operators of mdwf_dslash (SURVEY 8 "Even-odd form"; a = b5(4-M5)+1, d = c5(4-M5)-1):
 *   HOP        H_{p <- pbar}                 4D Wilson hopping stencil on every s slice
 *   M4PRE      A  = b5 + c5 L                (s-direction, 4D-site local)
 *   M5         M5 = a + d L                  ("Ls-direction M5/mass coupling", north_star)
 *   M5INV      M5^-1
 *   DHAT_ASYM  Dhat = M5 - 1/4 H A M5^-1 H A          (red-black Schur complement)
 *   DHAT_SYM   Mhat = M5^-1 Dhat
 *   NORMAL_ASYM / NORMAL_SYM   Dhat^dag Dhat / Mhat^dag Mhat   (the CG operator)
 *   FULL       D = M5 - 1/2 H A on the full lattice (both parities)                        */
enum { MDWF_OP_HOP = 0, MDWF_OP_M4PRE = 1, MDWF_OP_M5 = 2, MDWF_OP_M5INV = 3, MDWF_OP_DHAT_ASYM = 4,
       MDWF_OP_DHAT_SYM = 5, MDWF_OP_NORMAL_ASYM = 6, MDWF_OP_NORMAL_SYM = 7, MDWF_OP_FULL = 8 };

typedef struct mdwf_ctx mdwf_ctx;
typedef struct mdwf_field mdwf_field;

typedef struct {
    int32_t dims[4]; /* X,Y,Z,T: all even, >= 2                                   */
    int32_t Ls;      /* >= 1, <= 32                                               */
    int32_t bc[4];   /* +1 periodic, -1 antiperiodic (runs use {1,1,1,-1})        */
    int32_t device;  /* CUDA device ordinal                                       */
} mdwf_geometry;

/* Create a context for one lattice geometry and one set of Moebius parameters (north_star:
 * mdwf_create(geometry, M5, b5, c5, mf)).  Precomputes the Ls x Ls chirality blocks of A, M5, M5^-1
 * (closed form, SURVEY 8 Notation) and their products.  EINVAL: odd/too small extent, Ls out of range. */
int mdwf_create(mdwf_ctx** out, const mdwf_geometry* g, double M5, double b5, double c5, double mf);
int mdwf_destroy(mdwf_ctx* ctx);
const char* mdwf_last_error(const mdwf_ctx* ctx);

/* Pack the canonical fp64 gauge field (device pointer) into the even/odd-split device format
 * {store_prec 64|32|16} x {recon 18|12|8 reals per link} (north_star "gauge-field ... layout/packing,
 * with optional 12/8-parameter link reconstruction and fp16/fp32 storage"; formats: SURVEY A12).
 * May be called repeatedly: each (store_prec, recon) pair stays resident until destroy.
 * The boundary sign bc is never stored in a link; kernels apply it after reconstruction.
 * recon 8 cannot represent links with |U01|^2+|U02|^2 -> 0 (e.g. unit links): EINVAL, nothing loaded. */
int mdwf_load_gauge(mdwf_ctx* ctx, const void* U, int store_prec, int recon, void* stream);

/* out = op(in) on `nrhs` canonical fp64 fields (device).  Half-lattice ops (everything but FULL)
 * take/return half-lattice fields [rhs][s][xh][4][3][2]; `parity` is the parity of the OUTPUT sites
 * (HOP reads the other parity, all other ops read the same parity).  FULL takes/returns
 * full-lattice fields [rhs][s][x4][4][3][2] and ignores parity.  `prec` 64|32|16 selects the storage
 * precision of every packed spinor and of the links (compute is fp64 for 64, fp32 otherwise);
 * (prec, recon) must have been loaded.  This is pack -> packed kernels -> unpack; the parity tests
 * call it.  For NORMAL_* `dagger` is ignored. */
int mdwf_dslash(mdwf_ctx* ctx, int op, int parity, int dagger, int prec, int recon, void* out,
                const void* in, int nrhs, void* stream);

/* Packed fields for timing loops (canonical<->packed conversion stays outside the timed region). */
int mdwf_field_create(mdwf_ctx* ctx, int prec, int nrhs, mdwf_field** out);
int mdwf_field_destroy(mdwf_field* f);
/* canonical half-lattice fp64 [rhs][s][xh][4][3][2] (device) <-> packed */
int mdwf_field_pack(mdwf_field* f, const void* canonical, void* stream);
int mdwf_field_unpack(const mdwf_field* f, void* canonical, void* stream);
/* the same for column `rhs` alone (canonical [s][xh][4][3][2] of one rhs); fp64 / fp32 fields only */
int mdwf_field_pack_rhs(mdwf_field* f, int rhs, const void* canonical, void* stream);
int mdwf_field_unpack_rhs(const mdwf_field* f, int rhs, void* canonical, void* stream);
/* out = op(in) on packed half-lattice fields of equal prec/nrhs (op != FULL); out must not alias in. */
int mdwf_dslash_packed(mdwf_ctx* ctx, int op, int parity, int dagger, int recon, mdwf_field* out,
                       const mdwf_field* in, void* stream);
/* algorithmic bytes / flops of one mdwf_dslash_packed(op) call under DESIGN.md's convention
 * (SURVEY 8(d), A19): returns 0 and fills *bytes, *flops. */
int mdwf_dslash_cost(const mdwf_ctx* ctx, int op, int prec, int recon, int nrhs, double* bytes, double* flops);

typedef struct {
    double tol;          /* target ||b - D psi|| / ||b|| (full system, fp64)                        */
    int32_t max_iter;    /* cap on inner CG iterations per rhs                                       */
    int32_t inner_prec;  /* 64 | 32 | 16: storage precision of the inner CG vectors and links        */
    int32_t recon;       /* link format used by the inner operator (outer fp64 uses 18 if loaded,
                            else the same recon)                                                     */
    int32_t parity;      /* parity p that is solved (the other one is reconstructed)                 */
    int32_t symmetric;   /* 0: Dhat, 1: Mhat = M5^-1 Dhat                                            */
    double delta;        /* reliable-update threshold, <=0 -> 0.1                       */
    int32_t src_kind;    /* 0: b is a 5D full-lattice field; 1: b is a 4D source, wall-injected (O3) */
    int32_t out_kind;    /* 0: x is the 5D solution; 1: x is the 4D wall projection q (O3)           */
    int32_t batch;       /* max rhs solved concurrently (0 = as many as fit in free device memory)   */
    int32_t check_every; /* host convergence check period in iterations (<=0 -> 1)                   */
} mdwf_solve_opts;

#define MDWF_MAX_RHS 64
typedef struct {
    int32_t iters[MDWF_MAX_RHS];
    int32_t reliable_updates[MDWF_MAX_RHS];
    int32_t status[MDWF_MAX_RHS];      /* MDWF_OK | MDWF_NOT_CONVERGED | MDWF_BREAKDOWN per rhs */
    double true_resid[MDWF_MAX_RHS];   /* ||bhat - Dhat psi_p|| / ||b|| in fp64 = full-system residual */
    double seconds;                    /* device time of the whole call (CUDA events)                 */
    double seconds_inner;              /* device time spent in inner (low precision) iterations       */
    int64_t kernel_launches;           /* kernels launched by this call                               */
    int32_t batch;                     /* rhs that were in flight together (the launches' n_active)    */
} mdwf_solve_info;

/* Solve D psi = b for nrhs (<= MDWF_MAX_RHS) right-hand sides by even-odd preconditioning +
 * batched mixed-precision CG on the normal equations with reliable updates (
 * SURVEY 8(a) a7-a9, A9, A10, A20).  b, x: canonical fp64 device fields; 5D full-lattice
 * [rhs][s][x4][4][3][2] or 4D [rhs][x4][4][3][2] per src_kind/out_kind.  x may alias b only if both are
 * 5D.  Returns MDWF_OK, or MDWF_NOT_CONVERGED / MDWF_BREAKDOWN if any rhs ended that way. */
int mdwf_solve(mdwf_ctx* ctx, void* x, const void* b, int nrhs, const mdwf_solve_opts* opts,
               mdwf_solve_info* info, void* stream);
/* Same with HOST buffers (pageable or pinned; pinned lets the copies overlap the packing): all copies are inside the
 * call.  5D right-hand sides and solutions are never held in canonical form on the device: they stream through two
 * staging chunks of whole s-slices (<= 1.5 GB each, cudaMalloc'ed for the duration of the call) on a copy stream and are
 * packed / unpacked as they pass, so as many right-hand sides are in flight as in mdwf_solve_packed (4 at 48^3x64x10).
 * 4D sources / solutions (src_kind / out_kind = 1) are staged whole per batch.  x_host may alias b_host only if both are
 * 5D.  MDWF_ENOMEM if workspace plus staging buffers do not fit. */
int mdwf_solve_host(mdwf_ctx* ctx, void* x_host, const void* b_host, int nrhs, const mdwf_solve_opts* opts,
                    mdwf_solve_info* info, void* stream);

/* The same solve on PACKED fp64 half-lattice fields, in place: psi_even / psi_odd (mdwf_field_create(ctx, 64, nrhs),
 * filled with mdwf_field_pack) hold b on entry and the solution on exit.  No canonical copies are involved, so a
 * whole batch of large-volume rhs fits on the device at once (config 5: 4 rhs in flight, SURVEY 8(a) A20
 * "batched multi-RHS").  5D sources / solutions only. */
int mdwf_solve_packed(mdwf_ctx* ctx, mdwf_field* psi_even, mdwf_field* psi_odd, const mdwf_solve_opts* opts,
                      mdwf_solve_info* info, void* stream);
/* Solver workspace: by default the library allocates it on first use and keeps it until destroy (it grows
 * when a larger batch asks for more).  mdwf_workspace_bytes: bytes a batch of `nrhs` rhs needs with the fp64 temporaries
 * of the reliable updates shared one rhs at a time (packed != 0: for mdwf_solve_packed, whose sources live in the
 * caller's fields).  mdwf_set_workspace hands the library a caller-owned device buffer (e.g. from PyTorch's allocator)
 * to use instead -- it must stay valid until replaced or destroy; mem = NULL returns to library-owned memory. */
int mdwf_workspace_bytes(mdwf_ctx* ctx, int nrhs, int inner_prec, int packed, int64_t* bytes);
int mdwf_set_workspace(mdwf_ctx* ctx, void* mem, int64_t bytes);

/* Feynman-Hellmann sequential source:
 * out4d[col](x) = Gamma . prop4d[col](x) on timeslices t_min <= t <= t_max (all t = "sum over t"),
 * zero elsewhere.  Gamma: 4x4 complex, row-major [re,im], HOST pointer.  ncol columns of
 * canonical 4D fields [col][x4][4][3][2] fp64 (device).  out4d may alias prop4d. */
int mdwf_seq_source(mdwf_ctx* ctx, void* out4d, const void* prop4d, int ncol, const double* Gamma_host,
                    int t_min, int t_max, void* stream);

/* Nucleon two-point function (SURVEY a11, O4 C-def, A15).  Three 12-column 4D
 * propagators (device, canonical): S_u1 (diquark u), S_d, S_u2 (spectator u); proj: 4x4 complex
 * HOST; corr: device double [T][2], index (t - t0) mod T, overwritten. */
int mdwf_nucleon_2pt(mdwf_ctx* ctx, double* corr, const void* S_u1, const void* S_d, const void* S_u2,
                     const double* proj_host, int t0, void* stream);

/* The same contraction (same arguments, same launch shape, same fixed-order sums, hence the same numbers) for callers that
 * cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  The call makes
 * no cudaMalloc / cudaMallocAsync / cudaFree and calls no allocating library routine: the per-warp partial sums that
 * mdwf_nucleon_2pt takes from the stream-ordered allocator live in a file-scope `static __device__` array of
 * mdwf_nucleon_2pt_noalloc_max_bytes() = 512 KiB, which every GPU that loads the library holds until the process exits.
 * Limit: 10 * T * min(ceil(X*Y*Z / 4), max(1, 16 * SMs / T)) doubles must fit in it (on a 148-SM GPU every T <= 2368 with
 * any spatial volume does, e.g. all BASELINE configs); beyond that the call returns MDWF_EINVAL with the sizes in
 * mdwf_last_error and touches nothing.  The array is shared by every call on that GPU and keeps the last call's contents
 * (the call clears the part it uses first): calls that overlap on the GPU -- two streams, or two contexts on one device
 * -- race on it and must be serialised by the caller; calls on one stream are ordered and safe.  The first call on a
 * device looks up the array's device address (cudaGetSymbolAddress, that device current) and raises the kernel's
 * shared-memory limit; neither allocates device memory. */
int mdwf_nucleon_2pt_noalloc(mdwf_ctx* ctx, double* corr, const void* S_u1, const void* S_d, const void* S_u2,
                             const double* proj_host, int t0, void* stream);
int64_t mdwf_nucleon_2pt_noalloc_max_bytes(void);

/* Gauge-covariant Gaussian smearing of 4D spin-colour fields, for sources and sinks of the Feynman-Hellmann workload
 * (PAPER.md:98-102 names smeared sources, no formula; R25):
 *     out = (1 + width^2 / (4 n_iter) Lap)^n_iter in,
 *     (Lap psi)(x) = sum_{j=x,y,z} [ U_j(x) psi(x+j) + U_j(x-j)^dag psi(x-j) - 2 psi(x) ]   (every timeslice on its own),
 * hops that wrap multiplied by the geometry's bc_j.  in4d / out4d: ncol canonical 4D fields [col][x4][4][3][2] fp64
 * (device); out4d must not alias in4d (EINVAL).  Needs the fp64 18-real links (mdwf_load_gauge(U, 64, 18); ESTATE
 * otherwise).  n_iter = 0 copies; n_iter > 1 takes one temporary of the fields' size from the stream-ordered allocator
 * for the duration of the call.  For a positive kernel keep 6 width^2 / (4 n_iter) < 1.  Stream-ordered, no host sync. */
int mdwf_smear_gaussian(mdwf_ctx* ctx, void* out4d, const void* in4d, int ncol, double width, int n_iter, void* stream);

/* Feynman-Hellmann effective derivative (Fig. 1; R25): with R(t) = C_FH(t) / C_2pt(t) (complex
 * division), geff[t] = R(t+1) - R(t) for t = 0 .. T-2.  c2pt, cfh: device double [T][2] as written by mdwf_nucleon_2pt;
 * geff: device double [T-1][2], overwritten. */
int mdwf_fh_effective_derivative(mdwf_ctx* ctx, double* geff, const double* c2pt, const double* cfh, void* stream);

/* 4D <-> 5D maps of SURVEY O3 as stand-alone calls (used by the tests; mdwf_solve applies them
 * itself for src_kind/out_kind = 1):  b5 = -D_- (P+ eta @ s=0 (+) P- eta @ s=Ls-1),
 * q = P- psi_0 + P+ psi_{Ls-1}.  Full-lattice canonical fp64 device fields. */
int mdwf_wall_inject(mdwf_ctx* ctx, void* b5, const void* eta4, int ncol, int recon, void* stream);
int mdwf_wall_project(mdwf_ctx* ctx, void* q4, const void* psi5, int ncol, void* stream);

/* number of kernels this context has launched so far (bench.py's gpu_launches) */
int64_t mdwf_launch_count(const mdwf_ctx* ctx);
/* Per-launch timing of the hop (Dslash stencil) kernel with CUDA events on the launching stream.
 * mdwf_profile(ctx, 1) clears the counters and starts recording, mdwf_profile(ctx, 0) stops.
 * mdwf_profile_read synchronises the recorded events and returns, for class cls (hop kernel by storage class 0: fp16,
 * 1: fp32, 2: fp64; time only for the site-local kernels 3: s-direction, 4: CG x/r update, 5: CG p update, 6: reduction
 * finish, 7: axpby/convert), the summed device time [ms], algorithmic bytes and flops (DESIGN.md cost convention: per 5D
 * site 24*w bytes per spinor pass, 2 passes (+1 with an xpay input), links once per launch; 1320 flop)
 * and the launch count. */
int mdwf_profile(mdwf_ctx* ctx, int enable);
int mdwf_profile_read(mdwf_ctx* ctx, int cls, double* ms, double* bytes, double* flops, int64_t* launches);
/* force the z-slab depth of the fp32 / fp64 hop kernel's site traversal (L2 tiling); 0 = back to the tuned
 * (mdwf_autotune) or heuristic value.  zc must divide Z and be a multiple of the block's z extent (else EINVAL). */
int mdwf_set_tiling(mdwf_ctx* ctx, int zc);

/* Run-time autotuner ("GPU kernel autotuning ... brute-force search ... stored in a std::map", PAPER.md:92-94 IV).
 * mdwf_autotune times, on scratch fields of the real size (3 fields of `nrhs` columns in precision `prec` are allocated
 * for the duration of the call; ENOMEM if they do not fit), the free launch parameters of the Dslash stencil for the
 * loaded gauge format (prec, recon) (ESTATE if it is not loaded) with `nrhs` right-hand sides per launch -- prec 16: the
 * 4D tile and warps per block of the tensor-core kernel; prec 32 / 64: the z-slab depth -- keeps the fastest in the
 * context and uses it for every later launch of that (lattice, Ls, prec, rhs count).  Results never depend on these
 * parameters beyond the order of fp32 partial sums.  The call synchronises the stream.  Forced values
 * (mdwf_set_tiling, mdwf_set_hop16_tile) take precedence over tuned ones.
 * mdwf_tune_save / mdwf_tune_load write / read all entries as a text file ("key v0 v1 ..." per line; entries of other
 * lattices are kept and never match); EINVAL if the file cannot be opened or parsed.
 * mdwf_tune_get copies the values of one entry (keys: "hop16/XxYxZxT/LsN/rowsR" -> lx ly lz lt warps;
 * "hop32/.../rhsN", "hop64/.../rhsN" -> zc) into values[0..cap) and returns their number, 0 if there is no such entry,
 * < 0 on a null argument. */
int mdwf_autotune(mdwf_ctx* ctx, int prec, int recon, int nrhs, void* stream);
int mdwf_tune_save(mdwf_ctx* ctx, const char* path);
int mdwf_tune_load(mdwf_ctx* ctx, const char* path);
int mdwf_tune_get(mdwf_ctx* ctx, const char* key, int* values, int cap);

/* Tuning control of the fp16 tensor-core stencil (mdwf_hop16.cuh): the 4D box of output sites one block owns
 * (lx even; each extent divides the lattice) and the warps per block (0 = default).  lx = 0 returns to the tuned (mdwf_autotune)
 * or default choice.  Results do not depend on it beyond fp32 summation order.  EINVAL if the box does not fit in shared memory. */
int mdwf_set_hop16_tile(mdwf_ctx* ctx, int lx, int ly, int lz, int lt, int warps);

/* Host-only self-test (needs no GPU): the run-time-constant division used for site decoding (exhaustive over
 * the index ranges in use), the closed-form M5^-1 blocks against M5 (M5 * M5^-1 = 1) and dagger = transpose,
 * for Ls = 1..32 at the given parameters.  Returns 0 on success, else the number of the failed check. */
int mdwf_selftest_host(double M5, double b5, double c5, double mf);

#ifdef __cplusplus
}
#endif
#endif
