// csrc/solver.cu -- batched multi-rhs mixed-precision CG on the normal equations of the even-odd
// preconditioned MDWF operator, with reliable updates to fp64 ("red-black preconditioned double-half CG
// ... iterated in 16-bit storage / single-precision computation with occasional reliable updates to full
// double precision"; "CG on the normal equations"; readings SURVEY A6, A9, A10, A20).
//
//   S = Mhat (symmetric) or Dhat;  solve S psi_p = rhs  through  S^dag S psi_p = S^dag rhs
//   rhs = bhat (asym) or M5^-1 bhat (sym),  bhat = b_p + 1/2 H A M5^-1 b_pbar
//   psi_pbar = M5^-1 ( b_pbar + 1/2 H A psi_p )
// Inner iteration (storage precision `inner_prec`, fp32/fp64 arithmetic, fp64 reductions):
//   t = S p ; pAp = |t|^2 ; Ap = S^dag t ; alpha = rr/pAp ; x += alpha p ; r -= alpha Ap ; rr' = |r|^2 ;
//   beta = rr'/rr ; p = r + beta p.
// Reliable update (fp64): x_hi += x_lo ; x_lo = 0 ; rho = rhs - S x_hi ; r = S^dag rho ; the acceptance test is
// on the true residual |bhat - Dhat x_hi| / |b| ( = |M5 rho| / |b| in the symmetric form), SURVEY A9.
#include "mdwf_host.h"
#include <cmath>
#include <algorithm>
#include <cstring>
#include <string>

namespace mdwf {

int launch_wall_pack(mdwf_ctx* c, const SpinorView& out, const double* eta4, int par, int ncol, cudaStream_t st);
int launch_wall_unpack(mdwf_ctx* c, double* q4, const SpinorView& in, int par, int ncol, cudaStream_t st);

namespace {

struct Fields {
    std::vector<mdwf_field*> all;
    ~Fields() { for (size_t i = 0; i < all.size(); ++i) free_field(all[i]); }
    int make(mdwf_ctx* c, int prec, int nrhs, mdwf_field** f) {
        int rc = alloc_field(c, prec, nrhs, f);
        if (rc == MDWF_OK) all.push_back(*f);
        return rc;
    }
};

enum { SC_RR_A = 0, SC_RR_B = 1, SC_PAP = 2, SC_TMP = 3, SC_TMP2 = 4 };

struct Solver {
    mdwf_ctx* c;
    cudaStream_t st;
    OpCtx hi, lo;
    int nb, par, sym, prec, px;
    double tol, delta;
    int max_iter, check_every;

    double* dsc(int k) { return c->dscal + 64 * k; }
    double* hsc(int k) { return c->hscal + 64 * k; }

    // out[rhs] (device + pinned host mirror) = sum |f|^2
    int norm2(const OpCtx& o, const SpinorView& f, const RhsList& rl, int k) {
        int rc = op_ls(o, f, f, -1, nullptr, 0.0, 1.0, rl, c->partial, 0);
        if (rc) return rc;
        return launch_finish(c, o.prec, rl, dsc(k), hsc(k), st);
    }
    int sync() {
        MDWF_CUDA(c, cudaStreamSynchronize(st));
        return MDWF_OK;
    }
};

size_t per_rhs_bytes(const Geom& g, int prec, int px) {
    const size_t f64 = (size_t)g.N5h * 24 * 8;
    const size_t flo = (size_t)g.N5h * (24 * (prec / 8) + (prec == 16 ? 4 : 0));
    const size_t fx = (size_t)g.N5h * 24 * (px / 8);
    return 5 * f64 + 5 * flo + fx;
}

}  // namespace

// build the packed fp64 source halves of one batch: src_kind 0: pack the canonical 5D field;
// src_kind 1: wall-inject the 4D source, b5 = -D_- w = -d w + (c5/2) H w  (D_- = c5 D_W - 1)
static int make_source(Solver& S, const double* b, int src_kind, int which_par, const SpinorView& out,
                       const SpinorView& tmp_same, const SpinorView& tmp_other) {
    mdwf_ctx* c = S.c;
    const RhsList rl = all_rhs(S.nb);
    if (src_kind == 0) {
        PackArgs a;
        a.f = out; a.canon = const_cast<double*>(b); a.Vc = 2ll * c->g.Vh; a.full = 1; a.par = which_par; a.nrhs = S.nb; a.rhs0 = 0;
        return launch_pack(c, 64, false, a, S.st);
    }
    int rc;
    if ((rc = launch_wall_pack(c, tmp_same, b, which_par, S.nb, S.st))) return rc;
    if ((rc = launch_wall_pack(c, tmp_other, b, 1 - which_par, S.nb, S.st))) return rc;
    const double d = c->c5 * (4.0 - c->M5) - 1.0;
    return op_hop(S.hi, out, tmp_other, which_par, 0, -1, &tmp_same, -d, 0.5 * c->c5, rl);
}

static int solve_batch(Solver& S, double* x, const double* b, const mdwf_solve_opts* opts, mdwf_solve_info* info,
                       int r0, double* t_inner_ms) {
    mdwf_ctx* c = S.c;
    const Geom& g = c->g;
    const int nb = S.nb, par = S.par, sym = S.sym;
    cudaStream_t st = S.st;
    int rc;
    Fields F;
    mdwf_field *f_rhs, *f_x, *f_t2, *f_t3, *f_t4, *f_r, *f_p, *f_t, *f_a, *f_b, *f_xl;
    if ((rc = F.make(c, 64, nb, &f_rhs)) || (rc = F.make(c, 64, nb, &f_x)) || (rc = F.make(c, 64, nb, &f_t2)) ||
        (rc = F.make(c, 64, nb, &f_t3)) || (rc = F.make(c, 64, nb, &f_t4)) || (rc = F.make(c, S.prec, nb, &f_r)) ||
        (rc = F.make(c, S.prec, nb, &f_p)) || (rc = F.make(c, S.prec, nb, &f_t)) || (rc = F.make(c, S.prec, nb, &f_a)) ||
        (rc = F.make(c, S.prec, nb, &f_b)) || (rc = F.make(c, S.px, nb, &f_xl)))
        return rc;
    const SpinorView rhs = f_rhs->view(), xh = f_x->view(), t2 = f_t2->view(), t3 = f_t3->view(), t4 = f_t4->view(),
                     r = f_r->view(), p = f_p->view(), t = f_t->view(), wa = f_a->view(), wb = f_b->view(),
                     xl = f_xl->view();
    const RhsList all = all_rhs(nb);
    const size_t x4d = (size_t)2 * g.Vh * 24, x5d = x4d * g.Ls;
    const double* bsrc = b + (size_t)r0 * (opts->src_kind ? x4d : x5d);
    SpinorView none;
    none.v = nullptr; none.n = nullptr; none.rs = none.rn = 0;

    // ---- source: b_p -> rhs, b_pbar -> t3 ; |b|^2 ; bhat ; (sym) M5^-1 bhat ------------------------
    if ((rc = make_source(S, bsrc, opts->src_kind, par, rhs, t2, t4))) return rc;
    if ((rc = make_source(S, bsrc, opts->src_kind, 1 - par, t3, t2, t4))) return rc;
    if ((rc = S.norm2(S.hi, rhs, all, SC_TMP)) || (rc = S.norm2(S.hi, t3, all, SC_TMP2)) || (rc = S.sync())) return rc;
    double bnorm[MDWF_MAX_RHS], stop_nr[MDWF_MAX_RHS], maxr[MDWF_MAX_RHS];
    int status[MDWF_MAX_RHS], iters[MDWF_MAX_RHS], nrel[MDWF_MAX_RHS];
    double tres[MDWF_MAX_RHS];
    for (int i = 0; i < nb; ++i) {
        bnorm[i] = std::sqrt(S.hsc(SC_TMP)[i] + S.hsc(SC_TMP2)[i]);
        status[i] = -100;   // active
        iters[i] = 0; nrel[i] = 0; tres[i] = 0.0; stop_nr[i] = 0.0; maxr[i] = 0.0;
    }
    if ((rc = op_ls(S.hi, t2, t3, MAT_AM5INV, nullptr, 0.0, 1.0, all))) return rc;
    if ((rc = op_hop(S.hi, rhs, t2, par, 0, -1, &rhs, 1.0, 0.5, all))) return rc;           // bhat
    if (sym && (rc = op_ls(S.hi, rhs, rhs, MAT_M5INV, nullptr, 0.0, 1.0, all))) return rc;   // M5^-1 bhat
    MDWF_CUDA(c, cudaMemsetAsync(f_x->v, 0, f_x->bytes, st));
    MDWF_CUDA(c, cudaMemsetAsync(f_xl->v, 0, f_xl->bytes, st));

    RhsList act = all;
    int rrOld = SC_RR_A, rrNew = SC_RR_B;

    // reliable update over the active list: refreshes r (low precision), dsc(rrNew) = |r_hi|^2,
    // tres[] / status[]; first == true: x_hi = 0 so rho = rhs.
    auto reliable = [&](bool first) -> int {
        int rc2;
        AxpbyArgs d;
        d.out = t3; d.a = rhs; d.ca = 1.0; d.partial = sym ? nullptr : c->partial; d.rl = act;
        if (!first) {
            AxpbyArgs a;
            a.out = xh; a.a = xh; a.b = xl; a.ca = 1.0; a.cb = 1.0; a.partial = nullptr; a.rl = act;
            if ((rc2 = launch_axpby(c, 64, 64, S.px, a, st))) return rc2;
            MDWF_CUDA(c, cudaMemsetAsync(f_xl->v, 0, f_xl->bytes, st));
            if ((rc2 = op_schur(S.hi, t3, xh, par, 0, sym, t3, t2, act))) return rc2;
            d.b = t3; d.cb = -1.0;
        } else {
            d.b = none; d.cb = 0.0;
        }
        if ((rc2 = launch_axpby(c, 64, 64, 64, d, st))) return rc2;                                   // rho -> t3
        if (sym && (rc2 = op_ls(S.hi, t3, t3, MAT_M5, nullptr, 0.0, 1.0, act, c->partial, 0))) return rc2;   // |M5 rho|^2
        if ((rc2 = launch_finish(c, 64, act, S.dsc(SC_TMP), S.hsc(SC_TMP), st))) return rc2;
        if ((rc2 = op_schur(S.hi, t4, t3, par, 1, sym, t4, t2, act, c->partial))) return rc2;         // r = S^dag rho
        if ((rc2 = launch_finish(c, 64, act, S.dsc(rrNew), S.hsc(rrNew), st))) return rc2;
        AxpbyArgs cv;
        cv.out = r; cv.a = t4; cv.b = none; cv.ca = 1.0; cv.cb = 0.0; cv.partial = nullptr; cv.rl = act;
        if ((rc2 = launch_axpby(c, S.prec, 64, 64, cv, st))) return rc2;
        if ((rc2 = S.sync())) return rc2;
        RhsList na;
        na.nact = 0;
        for (int k = 0; k < 64; ++k) na.rhs[k] = 0;
        for (int k = 0; k < act.nact; ++k) {
            const int i = act.rhs[k];
            const double tn = std::sqrt(S.hsc(SC_TMP)[i]);
            const double rn = std::sqrt(S.hsc(rrNew)[i]);
            tres[i] = bnorm[i] > 0 ? tn / bnorm[i] : 0.0;
            if (!first) nrel[i]++;
            if (!(tn == tn) || !(rn == rn)) status[i] = MDWF_BREAKDOWN;
            else if (tres[i] <= S.tol) status[i] = MDWF_OK;
            else if (iters[i] >= S.max_iter) status[i] = MDWF_NOT_CONVERGED;
            else {
                // normal-equation residual matching the target true residual, with a safety margin (A9)
                stop_nr[i] = 0.5 * (rn / tn) * S.tol * bnorm[i];
                maxr[i] = rn;
                na.rhs[na.nact++] = i;
            }
        }
        act = na;
        return MDWF_OK;
    };

    if ((rc = reliable(true))) return rc;
    if (act.nact > 0) {
        AxpbyArgs cp;
        cp.out = p; cp.a = r; cp.b = none; cp.ca = 1.0; cp.cb = 0.0; cp.partial = nullptr; cp.rl = act;
        if ((rc = launch_axpby(c, S.prec, S.prec, S.prec, cp, st))) return rc;
        if ((rc = op_ls(S.lo, t, p, MAT_A, nullptr, 0.0, 1.0, act))) return rc;   // q = A p (later fused into the p-update)
        std::swap(rrOld, rrNew);   // dsc(rrOld) = |r_0|^2
    }
    cudaEvent_t e0, e1;
    MDWF_CUDA(c, cudaEventCreate(&e0));
    MDWF_CUDA(c, cudaEventCreate(&e1));
    int since_check = 0;
    bool open = false;
    rc = MDWF_OK;
    while (act.nact > 0 && rc == MDWF_OK) {
        if (!open) { cudaEventRecord(e0, st); open = true; }
        // t = S p, pAp = |t|^2 ; Ap = S^dag t   (out may alias the first work field, see op_schur)
        if ((rc = op_schur(S.lo, t, p, par, 0, sym, t, wb, act, c->partial, 1))) break;   // t holds A p on entry
        if ((rc = launch_finish(c, S.prec, act, S.dsc(SC_PAP), S.hsc(SC_PAP), st))) break;
        if ((rc = op_schur(S.lo, wa, t, par, 1, sym, wa, wb, act))) break;
        CgXrArgs u;
        u.x = xl; u.r = r; u.p = p; u.Ap = wa; u.rr = S.dsc(rrOld); u.pAp = S.dsc(SC_PAP); u.partial = c->partial; u.rl = act;
        if ((rc = launch_cg_xr(c, S.px, S.prec, u, st))) break;
        if ((rc = launch_finish(c, S.prec, act, S.dsc(rrNew), S.hsc(rrNew), st))) break;
        for (int k = 0; k < act.nact; ++k) iters[act.rhs[k]]++;
        bool need_update = false;
        if (++since_check >= S.check_every) {
            since_check = 0;
            if ((rc = S.sync())) break;
            for (int k = 0; k < act.nact; ++k) {
                const int i = act.rhs[k];
                const double rn = std::sqrt(S.hsc(rrNew)[i]), pap = S.hsc(SC_PAP)[i];
                if (!(rn == rn) || !(pap > 0.0)) need_update = true;          // breakdown: let the fp64 update decide
                if (rn <= stop_nr[i] || rn < S.delta * maxr[i] || iters[i] >= S.max_iter) need_update = true;
                if (rn > maxr[i]) maxr[i] = rn;
            }
        }
        if (need_update) {
            cudaEventRecord(e1, st);
            cudaEventSynchronize(e1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            *t_inner_ms += ms;
            open = false;
            const int before = act.nact;
            if ((rc = reliable(false))) break;
            (void)before;
            if (act.nact == 0) break;
        }
        CgPArgs q;
        q.p = p; q.r = r; q.q = t; q.op = c->lsop[MAT_A]; q.rr_new = S.dsc(rrNew); q.rr_old = S.dsc(rrOld); q.rl = act;
        if ((rc = launch_cg_p(c, S.prec, q, st))) break;
        std::swap(rrOld, rrNew);
    }
    if (open) {
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        *t_inner_ms += ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc) return rc;

    // ---- reconstruct psi_pbar = M5^-1 ( b_pbar + 1/2 H A psi_p ) and write the result ---------------
    if ((rc = make_source(S, bsrc, opts->src_kind, 1 - par, t3, t2, t4))) return rc;   // b_pbar again (not kept: memory)
    if ((rc = op_ls(S.hi, t2, xh, MAT_A, nullptr, 0.0, 1.0, all))) return rc;
    if ((rc = op_hop(S.hi, t3, t2, 1 - par, 0, -1, &t3, 1.0, 0.5, all))) return rc;
    if ((rc = op_ls(S.hi, t3, t3, MAT_M5INV, nullptr, 0.0, 1.0, all))) return rc;
    if (opts->out_kind == 0) {
        double* xo = x + (size_t)r0 * x5d;
        PackArgs a;
        a.canon = xo; a.Vc = 2ll * g.Vh; a.full = 1; a.nrhs = nb; a.rhs0 = 0;
        a.f = xh; a.par = par;
        if ((rc = launch_pack(c, 64, true, a, st))) return rc;
        a.f = t3; a.par = 1 - par;
        if ((rc = launch_pack(c, 64, true, a, st))) return rc;
    } else {
        double* xo = x + (size_t)r0 * x4d;
        if ((rc = launch_wall_unpack(c, xo, xh, par, nb, st))) return rc;
        if ((rc = launch_wall_unpack(c, xo, t3, 1 - par, nb, st))) return rc;
    }
    if ((rc = S.sync())) return rc;
    for (int i = 0; i < nb; ++i) {
        info->iters[r0 + i] = iters[i];
        info->reliable_updates[r0 + i] = nrel[i];
        info->status[r0 + i] = status[i] == -100 ? MDWF_NOT_CONVERGED : status[i];
        info->true_resid[r0 + i] = tres[i];
    }
    return MDWF_OK;
}

int solve_impl(mdwf_ctx* c, void* x, const void* b, int nrhs, const mdwf_solve_opts* opts, mdwf_solve_info* info,
               cudaStream_t st, bool host_buffers) {
    if (!x || !b || !opts || !info) MDWF_FAIL(c, MDWF_EINVAL, "null argument");
    if (nrhs < 1 || nrhs > MDWF_MAX_RHS) MDWF_FAIL(c, MDWF_EINVAL, "nrhs must be in 1..%d (got %d)", MDWF_MAX_RHS, nrhs);
    if (!(opts->tol > 0.0)) MDWF_FAIL(c, MDWF_EINVAL, "tol must be > 0");
    if (opts->parity != 0 && opts->parity != 1) MDWF_FAIL(c, MDWF_EINVAL, "parity must be 0 or 1");
    const int prec = opts->inner_prec;
    if (prec != 64 && prec != 32 && prec != 16) MDWF_FAIL(c, MDWF_EINVAL, "inner_prec must be 64, 32 or 16");
    if (opts->src_kind == 0 && opts->out_kind == 0) { /* x may alias b */ }
    else if (x == b) MDWF_FAIL(c, MDWF_EINVAL, "x may alias b only for 5D source and 5D solution");
    Solver S;
    S.c = c; S.st = st;
    S.prec = prec;
    S.px = prec == 16 ? 32 : prec;
    S.par = opts->parity; S.sym = opts->symmetric ? 1 : 0;
    S.tol = opts->tol;
    S.delta = opts->delta > 0.0 ? opts->delta : 0.1;
    S.max_iter = opts->max_iter > 0 ? opts->max_iter : 100000;
    S.check_every = opts->check_every > 0 ? opts->check_every : 1;
    S.lo.c = c; S.lo.prec = prec; S.lo.recon = opts->recon; S.lo.st = st;
    S.lo.gs = c->find_gauge(prec, opts->recon);
    if (!S.lo.gs) MDWF_FAIL(c, MDWF_ESTATE, "inner gauge format (prec %d, recon %d) not loaded", prec, opts->recon);
    S.hi.c = c; S.hi.prec = 64; S.hi.st = st;
    S.hi.recon = 18;
    S.hi.gs = c->find_gauge(64, 18);
    if (!S.hi.gs) { S.hi.recon = opts->recon; S.hi.gs = c->find_gauge(64, opts->recon); }
    if (!S.hi.gs) MDWF_FAIL(c, MDWF_ESTATE, "outer fp64 gauge format (recon 18 or %d) not loaded", opts->recon);

    const Geom& g = c->g;
    const size_t in_per = (size_t)2 * g.Vh * 24 * 8 * (opts->src_kind ? 1 : g.Ls);
    const size_t out_per = (size_t)2 * g.Vh * 24 * 8 * (opts->out_kind ? 1 : g.Ls);
    int nb = opts->batch > 0 ? std::min(opts->batch, nrhs) : nrhs;
    if (opts->batch <= 0) {
        size_t fr = 0, tot = 0;
        MDWF_CUDA(c, cudaMemGetInfo(&fr, &tot));
        const size_t per = per_rhs_bytes(g, S.prec, S.px) + (host_buffers ? 2 * (in_per + out_per) : 0);
        const size_t fit = (size_t)(0.92 * (double)fr) / per;
        if (fit < 1) MDWF_FAIL(c, MDWF_ENOMEM, "not enough free device memory for one rhs (%zu needed, %zu free)", per, fr);
        nb = (int)std::min<size_t>(fit, (size_t)nrhs);
    }
    memset(info, 0, sizeof(*info));
    cudaEvent_t e0, e1;
    MDWF_CUDA(c, cudaEventCreate(&e0));
    MDWF_CUDA(c, cudaEventCreate(&e1));
    MDWF_CUDA(c, cudaEventRecord(e0, st));
    const long long l0 = c->launches;
    double inner_ms = 0.0;
    int rc = MDWF_OK;
    if (!host_buffers) {
        for (int r0 = 0; r0 < nrhs && rc == MDWF_OK; r0 += nb) {
            S.nb = std::min(nb, nrhs - r0);
            rc = solve_batch(S, (double*)x, (const double*)b, opts, info, r0, &inner_ms);
        }
    } else {
        // Host buffers: every batch is staged through device buffers; the copies are part of the call (mdwf.h).
        // Two buffer sets and a copy stream: the upload of batch k+1 and the download of batch k-1 overlap the
        // solve of batch k (true overlap needs pinned host memory; pageable memory still gives correct results).
        void *din[2] = {nullptr, nullptr}, *dout[2] = {nullptr, nullptr};
        cudaStream_t cs = nullptr;
        cudaEvent_t up[2] = {nullptr, nullptr}, down[2] = {nullptr, nullptr}, solved = nullptr;
        const int nbatch = (nrhs + nb - 1) / nb, nset = nbatch > 1 ? 2 : 1;
        cudaError_t e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
        for (int k = 0; k < nset && e == cudaSuccess; ++k) {
            e = cudaMalloc(&din[k], in_per * nb);
            if (e == cudaSuccess) e = cudaMalloc(&dout[k], out_per * nb);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&up[k], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&down[k], cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&solved, cudaEventDisableTiming);
        if (e != cudaSuccess) {
            cudaGetLastError();
            c->err = std::string("staging buffers for host-buffer solve: ") + cudaGetErrorString(e);
            rc = MDWF_ENOMEM;
        }
        auto upload = [&](int k) -> cudaError_t {     // batch k -> din[k % nset] on the copy stream
            const int r0 = k * nb, n = std::min(nb, nrhs - r0);
            cudaError_t ee = cudaMemcpyAsync(din[k % nset], (const char*)b + in_per * r0, in_per * n, cudaMemcpyHostToDevice, cs);
            if (ee == cudaSuccess) ee = cudaEventRecord(up[k % nset], cs);
            return ee;
        };
        if (rc == MDWF_OK && (e = upload(0)) != cudaSuccess) { c->err = cudaGetErrorString(e); rc = MDWF_ECUDA; }
        for (int k = 0; k < nbatch && rc == MDWF_OK; ++k) {
            const int r0 = k * nb, set = k % nset;
            S.nb = std::min(nb, nrhs - r0);
            e = cudaStreamWaitEvent(st, up[set], 0);                           // batch k is on the device
            if (e == cudaSuccess && k >= nset) e = cudaStreamWaitEvent(st, down[set], 0);   // dout[set] has been drained
            // din[(k+1) % nset] was last read by batch k-1, which has completed (solve_batch returns synchronised)
            if (e == cudaSuccess && k + 1 < nbatch) e = upload(k + 1);
            if (e != cudaSuccess) { c->err = cudaGetErrorString(e); rc = MDWF_ECUDA; break; }
            mdwf_solve_info tmp;
            memset(&tmp, 0, sizeof(tmp));
            rc = solve_batch(S, (double*)dout[set], (const double*)din[set], opts, &tmp, 0, &inner_ms);
            if (rc) break;
            for (int i = 0; i < S.nb; ++i) {
                info->iters[r0 + i] = tmp.iters[i]; info->reliable_updates[r0 + i] = tmp.reliable_updates[i];
                info->status[r0 + i] = tmp.status[i]; info->true_resid[r0 + i] = tmp.true_resid[i];
            }
            e = cudaEventRecord(solved, st);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(cs, solved, 0);
            if (e == cudaSuccess) e = cudaMemcpyAsync((char*)x + out_per * r0, dout[set], out_per * S.nb, cudaMemcpyDeviceToHost, cs);
            if (e == cudaSuccess) e = cudaEventRecord(down[set], cs);
            if (e != cudaSuccess) { c->err = cudaGetErrorString(e); rc = MDWF_ECUDA; break; }
        }
        if (cs) {
            e = cudaStreamSynchronize(cs);
            if (e != cudaSuccess && rc == MDWF_OK) { c->err = cudaGetErrorString(e); rc = MDWF_ECUDA; }
        }
        for (int k = 0; k < 2; ++k) {
            if (din[k]) cudaFree(din[k]);
            if (dout[k]) cudaFree(dout[k]);
            if (up[k]) cudaEventDestroy(up[k]);
            if (down[k]) cudaEventDestroy(down[k]);
        }
        if (solved) cudaEventDestroy(solved);
        if (cs) cudaStreamDestroy(cs);
    }
    cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    info->seconds = ms * 1e-3;
    info->seconds_inner = inner_ms * 1e-3;
    info->kernel_launches = c->launches - l0;
    if (rc) return rc;
    int worst = MDWF_OK;
    for (int i = 0; i < nrhs; ++i) worst = std::max(worst, info->status[i]);
    return worst;
}

}  // namespace mdwf

extern "C" {
int mdwf_solve(mdwf_ctx* c, void* x, const void* b, int nrhs, const mdwf_solve_opts* opts, mdwf_solve_info* info,
               void* stream) {
    if (!c) return MDWF_EINVAL;
    return mdwf::solve_impl(c, x, b, nrhs, opts, info, (cudaStream_t)stream, false);
}
int mdwf_solve_host(mdwf_ctx* c, void* x, const void* b, int nrhs, const mdwf_solve_opts* opts,
                    mdwf_solve_info* info, void* stream) {
    if (!c) return MDWF_EINVAL;
    return mdwf::solve_impl(c, x, b, nrhs, opts, info, (cudaStream_t)stream, true);
}
}
