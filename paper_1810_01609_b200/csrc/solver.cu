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
//
// Memory plan.  Per rhs of a batch: three fp64 half-lattice fields (rhs, x_hi and the other
// parity's source, which becomes the other parity's solution), five inner-precision fields (r, p, t, Ap, work) and
// x_lo (fp32 for 16-bit inner vectors); the three fp64 temporaries of the reliable updates are shared by `nhi` <= batch
// rhs at a time.  Everything lives in one workspace (library-owned and kept between calls, or supplied by the caller
// through mdwf_set_workspace).  The inner loop never waits for the host: the decision to leave it is taken on the
// device (finish_sum_kernel with loop control) and the kernels of iterations already queued behind that point turn
// into no-ops, so iteration counts equal those of a loop that synchronises after every iteration.
#include "mdwf_host.h"
#include <cmath>
#include <algorithm>
#include <cstring>
#include <cstdlib>
#include <string>

namespace mdwf {

int launch_wall_pack(mdwf_ctx* c, const SpinorView& out, const double* eta4, int par, int ncol, cudaStream_t st);
int launch_wall_unpack(mdwf_ctx* c, double* q4, const SpinorView& in, int par, int ncol, cudaStream_t st);

namespace {

enum { SC_RR_A = 0, SC_RR_B = 1, SC_PAP = 2, SC_TMP = 3, SC_TMP2 = 4, SC_PP = 5, SC_STOPNR = 8, SC_MAXR = 9 };

struct Arena {
    char* base;
    size_t cap, off;
    void* take(size_t n) {
        off = (off + 255) / 256 * 256;
        void* p = base ? base + off : nullptr;
        off += n;
        return p;
    }
};

struct Work {
    std::vector<mdwf_field*> all;
    mdwf_field *rhs, *xh, *opar, *t2, *t3, *t4, *r, *p, *t, *wa, *wb, *xl;
    bool rhs_external;      // rhs / opar are the caller's packed fields (mdwf_solve_packed)
    ~Work() { for (size_t i = 0; i < all.size(); ++i) free_field(all[i]); }
};

struct Solver {
    mdwf_ctx* c;
    cudaStream_t st;
    OpCtx hi, lo;
    int nb, nhi, par, sym, prec, px;
    double tol, delta;
    int max_iter, check_every;
    int seq = 0;        // sequence number of the loop-control launches (CgCtlHost::seq)

    double* dsc(int k) { return c->dscal + 64 * k; }
    double* hsc(int k) { return c->hscal + 64 * k; }

    // out[rhs] (device + pinned host mirror) = sum |f|^2
    int norm2(const OpCtx& o, mdwf_field* f, const RhsList& rl, int k) {
        int rc = op_ls(o, f, f, -1, nullptr, 0.0, 1.0, rl, c->partial, 0);
        if (rc) return rc;
        return launch_finish(c, rl, dsc(k), hsc(k), st);
    }
    int sync() {
        MDWF_CUDA(c, cudaStreamSynchronize(st));
        return MDWF_OK;
    }
};

// bytes of the workspace of one batch (nb rhs in flight, nhi rhs of fp64 temporaries); own_src: rhs/opar inside
size_t work_bytes(const Geom& g, int prec, int px, int nb, int nhi, bool own_src) {
    auto al = [](size_t n) { return (n + 255) / 256 * 256; };
    size_t n = 0;
    n += (own_src ? 3 : 1) * al(field_bytes(g, 64, nb));
    n += 3 * al(field_bytes(g, 64, nhi));
    n += 5 * al(field_bytes(g, prec, nb));
    n += al(field_bytes(g, px, nb));
    n += 16 * al(2 * sizeof(FieldMeta));
    return n + 4096;
}

int ensure_workspace(mdwf_ctx* c, size_t need) {
    if (c->ws_bytes >= need) return MDWF_OK;
    if (c->ws_external) MDWF_FAIL(c, MDWF_ENOMEM, "caller-supplied workspace of %zu bytes is too small (%zu needed)", c->ws_bytes, need);
    if (c->ws) { cudaFree(c->ws); c->ws = nullptr; c->ws_bytes = 0; }
    cudaError_t e = cudaMalloc(&c->ws, need);
    if (e != cudaSuccess) {
        cudaGetLastError();
        c->ws = nullptr;
        MDWF_FAIL(c, MDWF_ENOMEM, "cudaMalloc of the %zu-byte solver workspace failed: %s", need, cudaGetErrorString(e));
    }
    c->ws_bytes = need;
    return MDWF_OK;
}

int make_work(Solver& S, Work& W, mdwf_field* ext_rhs, mdwf_field* ext_opar) {
    mdwf_ctx* c = S.c;
    const Geom& g = c->g;
    W.rhs_external = ext_rhs != nullptr;
    const size_t need = work_bytes(g, S.prec, S.px, S.nb, S.nhi, !W.rhs_external);
    int rc = ensure_workspace(c, need);
    if (rc) return rc;
    Arena A;
    A.base = (char*)c->ws; A.cap = c->ws_bytes; A.off = 0;
    auto mk = [&](int prec, int n, mdwf_field** f) -> int {
        void* mem = A.take(field_bytes(g, prec, n));
        void* meta = prec == 16 ? A.take(2 * sizeof(FieldMeta)) : nullptr;
        int r2 = wrap_field(c, prec, n, mem, meta, f);
        if (r2 == MDWF_OK) {
            W.all.push_back(*f);
            if (meta) MDWF_CUDA(c, cudaMemsetAsync(meta, 0, 2 * sizeof(FieldMeta), S.st));
            // padding rhs of the last interleave group and padding rows of a site must hold finite numbers
            if (prec == 16 && ((n & ((1 << half_ril(n, g.Ls)) - 1)) || ((g.Ls << half_ril(n, g.Ls)) & 7)))
                MDWF_CUDA(c, cudaMemsetAsync(mem, 0, field_bytes(g, prec, n), S.st));
        }
        return r2;
    };
    if (W.rhs_external) { W.rhs = ext_rhs; W.opar = ext_opar; }
    else if ((rc = mk(64, S.nb, &W.rhs)) || (rc = mk(64, S.nb, &W.opar))) return rc;
    if ((rc = mk(64, S.nb, &W.xh)) || (rc = mk(64, S.nhi, &W.t2)) || (rc = mk(64, S.nhi, &W.t3)) || (rc = mk(64, S.nhi, &W.t4)) ||
        (rc = mk(S.prec, S.nb, &W.r)) || (rc = mk(S.prec, S.nb, &W.p)) || (rc = mk(S.prec, S.nb, &W.t)) ||
        (rc = mk(S.prec, S.nb, &W.wa)) || (rc = mk(S.prec, S.nb, &W.wb)) || (rc = mk(S.px, S.nb, &W.xl)))
        return rc;
    if (A.off > A.cap) MDWF_FAIL(c, MDWF_ENOMEM, "internal: workspace plan exceeds its size");
    return MDWF_OK;
}

// the rhs ids of `act` that fall into [c0, c0 + n)
RhsList chunk_of(const RhsList& act, int c0, int n) {
    RhsList r;
    memset(&r, 0, sizeof(r));
    for (int k = 0; k < act.nact; ++k)
        if (act.rhs[k] >= c0 && act.rhs[k] < c0 + n) r.rhs[r.nact++] = act.rhs[k];
    return r;
}

SpinorView no_view() {
    SpinorView v;
    memset(&v, 0, sizeof(v));
    return v;
}

}  // namespace

// build the packed fp64 source halves of one batch from canonical data: src_kind 0: pack the canonical 5D field;
// src_kind 1: wall-inject the 4D source, b5 = -D_- w = -d w + (c5/2) H w  (D_- = c5 D_W - 1)
static int make_source(Solver& S, Work& W, const double* b, int src_kind, int which_par, mdwf_field* out) {
    mdwf_ctx* c = S.c;
    if (src_kind == 0) return pack_field(out, b, 1, which_par, S.st);
    int rc;
    const double d = c->c5 * (4.0 - c->M5) - 1.0;
    const size_t x4d = (size_t)2 * c->g.Vh * 24;
    for (int c0 = 0; c0 < S.nb; c0 += S.nhi) {          // temporaries hold nhi columns at a time
        const int n = std::min(S.nhi, S.nb - c0);
        W.t2->rhs0 = W.t4->rhs0 = 0;
        if ((rc = launch_wall_pack(c, W.t2->view(), b + c0 * x4d, which_par, n, S.st))) return rc;
        if ((rc = launch_wall_pack(c, W.t4->view(), b + c0 * x4d, 1 - which_par, n, S.st))) return rc;
        W.t2->rhs0 = W.t4->rhs0 = c0;
        RhsList rl = chunk_of(all_rhs(S.nb), c0, n);
        if ((rc = op_hop(S.hi, out, W.t4, which_par, 0, -1, W.t2, -d, 0.5 * c->c5, rl))) return rc;
    }
    return MDWF_OK;
}

// The solve proper on packed fp64 halves: on entry W.rhs = b_p, W.opar = b_pbar; on exit W.xh = psi_p, W.opar = psi_pbar.
static int solve_core(Solver& S, Work& W, mdwf_solve_info* info, int r0, double* t_inner_ms) {
    mdwf_ctx* c = S.c;
    const int nb = S.nb, par = S.par, sym = S.sym;
    cudaStream_t st = S.st;
    int rc;
    const RhsList all = all_rhs(nb);
    mdwf_field *rhs = W.rhs, *xh = W.xh, *opar = W.opar, *t2 = W.t2, *t3 = W.t3, *t4 = W.t4, *r = W.r, *p = W.p, *t = W.t,
               *wa = W.wa, *wb = W.wb, *xl = W.xl;
    auto set_chunk = [&](int c0) { t2->rhs0 = t3->rhs0 = t4->rhs0 = c0; };

    // ---- |b|^2 ; bhat ; (sym) M5^-1 bhat ----------------------------------------------------------------
    if ((rc = S.norm2(S.hi, rhs, all, SC_TMP)) || (rc = S.norm2(S.hi, opar, all, SC_TMP2)) || (rc = S.sync())) return rc;
    double bnorm[MDWF_MAX_RHS], stop_nr[MDWF_MAX_RHS], maxr[MDWF_MAX_RHS];
    int status[MDWF_MAX_RHS], iters[MDWF_MAX_RHS], nrel[MDWF_MAX_RHS];
    double tres[MDWF_MAX_RHS];
    for (int i = 0; i < nb; ++i) {
        bnorm[i] = std::sqrt(S.hsc(SC_TMP)[i] + S.hsc(SC_TMP2)[i]);
        status[i] = -100;   // active
        iters[i] = 0; nrel[i] = 0; tres[i] = 0.0; stop_nr[i] = 0.0; maxr[i] = 0.0;
    }
    for (int c0 = 0; c0 < nb; c0 += S.nhi) {
        const RhsList rl = chunk_of(all, c0, S.nhi);
        set_chunk(c0);
        if ((rc = op_ls(S.hi, t2, opar, MAT_AM5INV, nullptr, 0.0, 1.0, rl))) return rc;
        if ((rc = op_hop(S.hi, rhs, t2, par, 0, -1, rhs, 1.0, 0.5, rl))) return rc;           // bhat
    }
    if (sym && (rc = op_ls(S.hi, rhs, rhs, MAT_M5INV, nullptr, 0.0, 1.0, all))) return rc;   // M5^-1 bhat
    MDWF_CUDA(c, cudaMemsetAsync(xh->v, 0, xh->bytes, st));
    MDWF_CUDA(c, cudaMemsetAsync(xl->v, 0, xl->bytes, st));

    RhsList act = all;
    int rrOld = SC_RR_A, rrNew = SC_RR_B;

    // reliable update over the active list: refreshes r (low precision), dsc(rrNew) = |r_hi|^2,
    // tres[] / status[]; first == true: x_hi = 0 so rho = rhs.  The fp64 temporaries serve nhi rhs at a time.
    auto reliable = [&](bool first) -> int {
        int rc2;
        if (!first) {
            AxpbyArgs a;
            memset(&a, 0, sizeof(a));
            a.out = xh->view(); a.a = xh->view(); a.b = xl->view(); a.ca = 1.0; a.cb = 1.0; a.partial = nullptr; a.rl = act;
            if ((rc2 = launch_axpby(c, 64, 64, S.px, a, st))) return rc2;
            MDWF_CUDA(c, cudaMemsetAsync(xl->v, 0, xl->bytes, st));
        }
        for (int c0 = 0; c0 < nb; c0 += S.nhi) {
            const RhsList rl = chunk_of(act, c0, S.nhi);
            if (rl.nact == 0) continue;
            set_chunk(c0);
            AxpbyArgs d;
            memset(&d, 0, sizeof(d));
            d.out = t3->view(); d.a = rhs->view(); d.ca = 1.0; d.partial = sym ? nullptr : c->partial; d.rl = rl;
            if (!first) {
                if ((rc2 = op_schur(S.hi, t3, xh, par, 0, sym, t3, t2, rl))) return rc2;
                d.b = t3->view(); d.cb = -1.0;
            } else {
                d.b = no_view(); d.cb = 0.0;
            }
            if ((rc2 = launch_axpby(c, 64, 64, 64, d, st))) return rc2;                                   // rho -> t3
            if (sym && (rc2 = op_ls(S.hi, t3, t3, MAT_M5, nullptr, 0.0, 1.0, rl, c->partial, 0))) return rc2;   // |M5 rho|^2
            if ((rc2 = launch_finish(c, rl, S.dsc(SC_TMP), S.hsc(SC_TMP), st))) return rc2;
            if ((rc2 = op_schur(S.hi, t4, t3, par, 1, sym, t4, t2, rl, c->partial))) return rc2;         // r = S^dag rho
            if ((rc2 = launch_finish(c, rl, S.dsc(rrNew), S.hsc(rrNew), st))) return rc2;
            AxpbyArgs cv;
            memset(&cv, 0, sizeof(cv));
            cv.out = r->view(); cv.a = t4->view(); cv.b = no_view(); cv.ca = 1.0; cv.cb = 0.0; cv.partial = nullptr; cv.rl = rl;
            if (r->meta) {       // scale of the fp16 residual from its measured norm
                cv.sr.n = 1; cv.sr.out = r->wmeta();
                cv.sr.t[0].nb = S.dsc(rrNew); cv.sr.t[0].sq = 1; cv.sr.t[0].coef = 1.001953125;
            }
            if ((rc2 = launch_axpby(c, S.prec, 64, 64, cv, st))) return rc2;
        }
        // every chunk wrote r through the same write slot: flip once
        r->flip();
        if ((rc2 = S.sync())) return rc2;
        RhsList na;
        memset(&na, 0, sizeof(na));
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
    // fp16 only: the r slot that readers see must carry the scales of ALL rhs, also of those that are no longer
    // active (they are never read again), so nothing else is needed after the flip above.

    if ((rc = reliable(true))) return rc;
    if (act.nact > 0) {
        AxpbyArgs cp;
        memset(&cp, 0, sizeof(cp));
        cp.out = p->view(); cp.a = r->view(); cp.b = no_view(); cp.ca = 1.0; cp.cb = 0.0; cp.partial = nullptr; cp.rl = act;
        cp.sr = rule_lin(p, r, 1.0);
        if ((rc = launch_axpby(c, S.prec, S.prec, S.prec, cp, st))) return rc;
        p->flip();
        if ((rc = op_ls(S.lo, t, p, MAT_A, nullptr, 0.0, 1.0, act))) return rc;   // q = A p (later fused into the p-update)
        std::swap(rrOld, rrNew);   // dsc(rrOld) = |r_0|^2
    }
    cudaEvent_t e0, e1;
    MDWF_CUDA(c, cudaEventCreate(&e0));
    MDWF_CUDA(c, cudaEventCreate(&e1));
    rc = MDWF_OK;
    // Inner loop.  The host queues iterations a few ahead of the device and never waits for a result: the last kernel
    // of an iteration (finish_sum_kernel with loop control) decides on the device whether the loop must be left and
    // turns everything queued behind it into no-ops (gate `ctl->stop`).  One cycle = arm the control block, (pending
    // p-update), iterations until the gate closes, drain, fp64 reliable update.
    const int* gate = &c->dctl->stop;
    // iterations the host may be ahead: enough to hide the launch latency of tiny lattices; on large ones an iteration takes
    // tens of milliseconds and every iteration queued behind a closed gate costs ~3 ms of empty million-block launches
    const int kRunAhead = (double)c->g.N5h * nb > 2.0e7 ? 2 : 6;
    bool pending_p = false;
    auto p_update = [&](const int* stop) -> int {
        int rc2;
        CgPArgs q;
        memset(&q, 0, sizeof(q));
        q.p = p->view(); q.r = r->view(); q.q = t->view(); q.op = c->lsop[MAT_A]; q.rr_new = S.dsc(rrNew); q.rr_old = S.dsc(rrOld); q.rl = act;
        q.stop = stop;
        if (p->meta) {      // |r + beta p| <= |r| + beta |p| ; |A p| <= |A| |p| ; p's bound is then refreshed by its measured norm
            for (int w = 0; w < 2; ++w) {
                ScaleRule& sr = w ? q.sr_q : q.sr_p;
                const double f = w ? c->lsop_norm[MAT_A] : 1.0;
                sr.n = 2; sr.out = w ? t->wmeta() : p->wmeta();
                sr.t[0].nb = S.dsc(rrNew); sr.t[0].sq = 1; sr.t[0].coef = 1.001953125 * f;
                sr.t[1].nb = p->nb(); sr.t[1].coef = f; sr.t[1].num = S.dsc(rrNew); sr.t[1].den = S.dsc(rrOld);
            }
            q.partial = c->partial;
        }
        if ((rc2 = launch_cg_p(c, S.prec, q, st))) return rc2;
        p->flip();
        t->flip();
        if (p->meta) {
            FinishCtl fc;
            memset(&fc, 0, sizeof(fc));
            fc.stop = stop;
            if ((rc2 = launch_finish(c, act, S.dsc(SC_PP), nullptr, st, p->nb_w(), &fc))) return rc2;
        }
        std::swap(rrOld, rrNew);
        return MDWF_OK;
    };
    while (act.nact > 0 && rc == MDWF_OK) {
        // ---- arm the loop control ------------------------------------------------------------------------------
        CgCtl* hs = c->hctl_stage;
        memset(hs, 0, sizeof(*hs));
        hs->delta = S.delta;
        int cap = 1 << 30;
        for (int k = 0; k < act.nact; ++k) {
            const int i = act.rhs[k];
            hs->stop_nr[i] = stop_nr[i];
            hs->maxr[i] = maxr[i];
            cap = std::min(cap, std::max(1, S.max_iter - iters[i]));
        }
        hs->iter_cap = cap;
        MDWF_CUDA(c, cudaMemcpyAsync(c->dctl, hs, sizeof(CgCtl), cudaMemcpyHostToDevice, st));
        c->hctl->stop = 0;
        c->hctl->iters = 0;
        cudaEventRecord(e0, st);
        if (pending_p && (rc = p_update(nullptr))) break;
        pending_p = false;
        S.lo.stop = gate;
        // meta slots / rr slots as they are before the first iteration of this cycle (flips of no-op launches are undone below)
        const int cur0[5] = {r->cur, p->cur, t->cur, wa->cur, wb->cur};
        const int rrOld0 = rrOld, rrNew0 = rrNew;
        int queued = 0;
        std::vector<size_t> pmark;               // profile records at the start of each queued iteration
        while (rc == MDWF_OK) {
            if (c->prof_on) pmark.push_back(c->prof_pending.size());
            // t = S p, pAp = |t|^2 ; Ap = S^dag t   (out may alias the first work field, see op_schur)
            FinishCtl fg;
            memset(&fg, 0, sizeof(fg));
            fg.stop = gate;
            if ((rc = op_schur(S.lo, t, p, par, 0, sym, t, wb, act, c->partial, 1))) break;   // t holds A p on entry
            if ((rc = launch_finish(c, act, S.dsc(SC_PAP), S.hsc(SC_PAP), st, t->nb_w(), &fg))) break;
            if ((rc = op_schur(S.lo, wa, t, par, 1, sym, wa, wb, act))) break;
            CgXrArgs u;
            memset(&u, 0, sizeof(u));
            u.x = xl->view(); u.r = r->view(); u.p = p->view(); u.Ap = wa->view(); u.rr = S.dsc(rrOld); u.pAp = S.dsc(SC_PAP);
            u.partial = c->partial; u.rl = act; u.stop = gate;
            if (r->meta) {      // |r - alpha Ap| <= |r| + |alpha| |Ap|
                u.sr.n = 2; u.sr.out = r->wmeta();
                u.sr.t[0].nb = r->nb(); u.sr.t[0].coef = 1.0;
                u.sr.t[1].nb = wa->nb(); u.sr.t[1].coef = 1.0; u.sr.t[1].num = S.dsc(rrOld); u.sr.t[1].den = S.dsc(SC_PAP);
            }
            if ((rc = launch_cg_xr(c, S.px, S.prec, u, st))) break;
            r->flip();
            FinishCtl fc;
            memset(&fc, 0, sizeof(fc));
            fc.stop = gate; fc.ctl = c->dctl; fc.hctl = c->hctl; fc.pap = S.dsc(SC_PAP); fc.seq = ++S.seq;
            if ((rc = launch_finish(c, act, S.dsc(rrNew), S.hsc(rrNew), st, r->nb_w(), &fc))) break;
            ++queued;
            if ((rc = p_update(gate))) break;           // a no-op if this iteration closed the gate: redone after the update
            while (S.seq - c->hctl->seq > kRunAhead && cudaStreamQuery(st) == cudaErrorNotReady) {}
            if (c->hctl->stop) break;
        }
        S.lo.stop = nullptr;
        if (rc) break;
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        *t_inner_ms += ms;
        const int done = c->hctl->iters;          // iterations that really ran; the last one is complete up to its |r|^2
        if (done < 1 || done > queued) { c->err = "internal: inner-loop control out of step"; rc = MDWF_ECUDA; break; }
        // host-side bookkeeping as if only `done` iterations had been queued: `done` x-r updates, done - 1 p-updates
        r->cur = cur0[0] ^ (done & 1);
        p->cur = cur0[1] ^ ((done - 1) & 1);
        // t: written once (Mhat) or twice (Dhat: M5 p, then the hop) per operator application and once per p-update (q = A p)
        t->cur = cur0[2] ^ ((done * (sym ? 1 : 2) + done - 1) & 1);
        wa->cur = cur0[3]; wb->cur = cur0[4];      // an even number of flips per iteration
        if ((done - 1) & 1) { rrOld = rrNew0; rrNew = rrOld0; } else { rrOld = rrOld0; rrNew = rrNew0; }
        for (int k = 0; k < act.nact; ++k) iters[act.rhs[k]] += done;
        // launches queued behind the closed gate did no work: they are not part of the per-launch profile
        if (c->prof_on && done < (int)pmark.size()) {
            for (size_t k = pmark[done]; k < c->prof_pending.size(); ++k) {
                c->prof_pool.push_back(c->prof_pending[k].e0);
                c->prof_pool.push_back(c->prof_pending[k].e1);
            }
            c->prof_pending.resize(pmark[done]);
        }
        if ((rc = reliable(false))) break;
        pending_p = true;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc) return rc;

    // ---- reconstruct psi_pbar = M5^-1 ( b_pbar + 1/2 H A psi_p ), in place in opar -----------------------
    for (int c0 = 0; c0 < nb; c0 += S.nhi) {
        const RhsList rl = chunk_of(all, c0, S.nhi);
        set_chunk(c0);
        if ((rc = op_ls(S.hi, t2, xh, MAT_A, nullptr, 0.0, 1.0, rl))) return rc;
        if ((rc = op_hop(S.hi, opar, t2, 1 - par, 0, -1, opar, 1.0, 0.5, rl))) return rc;
    }
    if ((rc = op_ls(S.hi, opar, opar, MAT_M5INV, nullptr, 0.0, 1.0, all))) return rc;
    for (int i = 0; i < nb; ++i) {
        info->iters[r0 + i] = iters[i];
        info->reliable_updates[r0 + i] = nrel[i];
        info->status[r0 + i] = status[i] == -100 ? MDWF_NOT_CONVERGED : status[i];
        info->true_resid[r0 + i] = tres[i];
    }
    return MDWF_OK;
}

// one batch through canonical device buffers
static int solve_batch(Solver& S, double* x, const double* b, const mdwf_solve_opts* opts, mdwf_solve_info* info,
                       int r0, double* t_inner_ms) {
    mdwf_ctx* c = S.c;
    const Geom& g = c->g;
    Work W;
    int rc = make_work(S, W, nullptr, nullptr);
    if (rc) return rc;
    const size_t x4d = (size_t)2 * g.Vh * 24, x5d = x4d * g.Ls;
    const double* bsrc = b + (size_t)r0 * (opts->src_kind ? x4d : x5d);
    if ((rc = make_source(S, W, bsrc, opts->src_kind, S.par, W.rhs))) return rc;
    if ((rc = make_source(S, W, bsrc, opts->src_kind, 1 - S.par, W.opar))) return rc;
    if ((rc = solve_core(S, W, info, r0, t_inner_ms))) return rc;
    if (opts->out_kind == 0) {
        double* xo = x + (size_t)r0 * x5d;
        if ((rc = unpack_field(W.xh, xo, 1, S.par, S.st))) return rc;
        if ((rc = unpack_field(W.opar, xo, 1, 1 - S.par, S.st))) return rc;
    } else {
        double* xo = x + (size_t)r0 * x4d;
        if ((rc = launch_wall_unpack(c, xo, W.xh->view(), S.par, S.nb, S.st))) return rc;
        if ((rc = launch_wall_unpack(c, xo, W.opar->view(), 1 - S.par, S.nb, S.st))) return rc;
    }
    return S.sync();
}

// Host-buffer solves (mdwf_solve_host): the copies are part of the call.  A 5D right-hand side is never held in canonical
// form on the device: it streams, a few s-slices at a time, through two staging chunks on a copy stream and is packed into
// (unpacked from) the batch's fp64 half-lattice fields as it arrives, so the device holds the same fields as a packed
// in-place solve and the same number of right-hand sides stays in flight.  True copy/pack overlap needs pinned host
// memory; pageable memory still gives correct results.
struct HostStage {
    cudaStream_t cs = nullptr;
    void* stage[2] = {nullptr, nullptr};
    cudaEvent_t filled[2] = {nullptr, nullptr}, drained[2] = {nullptr, nullptr};
    void *d4in = nullptr, *d4out = nullptr;     // whole-batch buffers of 4D sources / 4D solutions
    size_t slice_bytes = 0;
    int ns = 1, k = 0;
    int acquire(mdwf_ctx* c, size_t chunk, size_t in4, size_t out4) {
        cudaError_t e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
        for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
            if (chunk) e = cudaMalloc(&stage[i], chunk);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&filled[i], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&drained[i], cudaEventDisableTiming);
        }
        if (e == cudaSuccess && in4) e = cudaMalloc(&d4in, in4);
        if (e == cudaSuccess && out4) e = cudaMalloc(&d4out, out4);
        if (e != cudaSuccess) {
            cudaGetLastError();
            c->err = std::string("staging buffers for host-buffer solve: ") + cudaGetErrorString(e);
            return MDWF_ENOMEM;
        }
        return MDWF_OK;
    }
    void release() {
        for (int i = 0; i < 2; ++i) {
            if (stage[i]) cudaFree(stage[i]);
            if (filled[i]) cudaEventDestroy(filled[i]);
            if (drained[i]) cudaEventDestroy(drained[i]);
            stage[i] = nullptr; filled[i] = drained[i] = nullptr;
        }
        if (d4in) cudaFree(d4in);
        if (d4out) cudaFree(d4out);
        d4in = d4out = nullptr;
        if (cs) cudaStreamDestroy(cs);
        cs = nullptr;
    }
};

// column `col` of the two half-lattice fields <-> one canonical 5D host field, chunk by chunk
static int stream_rhs(Solver& S, HostStage& H, mdwf_field* fpar, mdwf_field* fopar, int col, char* host, bool download) {
    mdwf_ctx* c = S.c;
    int rc;
    for (int s0 = 0; s0 < c->g.Ls; s0 += H.ns, ++H.k) {
        const int n = std::min(H.ns, c->g.Ls - s0), set = H.k & 1;
        const size_t bytes = (size_t)n * H.slice_bytes;
        double* stg = (double*)H.stage[set];
        if (!download) {
            MDWF_CUDA(c, cudaStreamWaitEvent(H.cs, H.drained[set], 0));       // the pack that last read this chunk is done
            MDWF_CUDA(c, cudaMemcpyAsync(stg, host + (size_t)s0 * H.slice_bytes, bytes, cudaMemcpyHostToDevice, H.cs));
            MDWF_CUDA(c, cudaEventRecord(H.filled[set], H.cs));
            MDWF_CUDA(c, cudaStreamWaitEvent(S.st, H.filled[set], 0));
            if ((rc = pack_slices(fpar, col, stg, s0, n, S.par, false, S.st))) return rc;
            if ((rc = pack_slices(fopar, col, stg, s0, n, 1 - S.par, false, S.st))) return rc;
            MDWF_CUDA(c, cudaEventRecord(H.drained[set], S.st));
        } else {
            MDWF_CUDA(c, cudaStreamWaitEvent(S.st, H.drained[set], 0));       // the copy that last read this chunk is done
            if ((rc = pack_slices(fpar, col, stg, s0, n, S.par, true, S.st))) return rc;
            if ((rc = pack_slices(fopar, col, stg, s0, n, 1 - S.par, true, S.st))) return rc;
            MDWF_CUDA(c, cudaEventRecord(H.filled[set], S.st));
            MDWF_CUDA(c, cudaStreamWaitEvent(H.cs, H.filled[set], 0));
            MDWF_CUDA(c, cudaMemcpyAsync(host + (size_t)s0 * H.slice_bytes, stg, bytes, cudaMemcpyDeviceToHost, H.cs));
            MDWF_CUDA(c, cudaEventRecord(H.drained[set], H.cs));
        }
    }
    return MDWF_OK;
}

// one batch from / to host buffers
static int solve_batch_host(Solver& S, HostStage& H, char* x, const char* b, const mdwf_solve_opts* opts, mdwf_solve_info* info,
                            int r0, double* t_inner_ms) {
    mdwf_ctx* c = S.c;
    const Geom& g = c->g;
    Work W;
    int rc = make_work(S, W, nullptr, nullptr);
    if (rc) return rc;
    const size_t x4d = (size_t)2 * g.Vh * 24 * 8, x5d = x4d * g.Ls;
    if (opts->src_kind == 0) {
        for (int i = 0; i < S.nb; ++i)
            if ((rc = stream_rhs(S, H, W.rhs, W.opar, i, const_cast<char*>(b) + (size_t)(r0 + i) * x5d, false))) return rc;
    } else {
        MDWF_CUDA(c, cudaMemcpyAsync(H.d4in, b + (size_t)r0 * x4d, x4d * S.nb, cudaMemcpyHostToDevice, S.st));
        if ((rc = make_source(S, W, (const double*)H.d4in, 1, S.par, W.rhs))) return rc;
        if ((rc = make_source(S, W, (const double*)H.d4in, 1, 1 - S.par, W.opar))) return rc;
    }
    mdwf_solve_info tmp;
    memset(&tmp, 0, sizeof(tmp));
    if ((rc = solve_core(S, W, &tmp, 0, t_inner_ms))) return rc;
    for (int i = 0; i < S.nb; ++i) {
        info->iters[r0 + i] = tmp.iters[i]; info->reliable_updates[r0 + i] = tmp.reliable_updates[i];
        info->status[r0 + i] = tmp.status[i]; info->true_resid[r0 + i] = tmp.true_resid[i];
    }
    if (opts->out_kind == 0) {
        for (int i = 0; i < S.nb; ++i)
            if ((rc = stream_rhs(S, H, W.xh, W.opar, i, x + (size_t)(r0 + i) * x5d, true))) return rc;
        MDWF_CUDA(c, cudaStreamSynchronize(H.cs));
    } else {
        if ((rc = launch_wall_unpack(c, (double*)H.d4out, W.xh->view(), S.par, S.nb, S.st))) return rc;
        if ((rc = launch_wall_unpack(c, (double*)H.d4out, W.opar->view(), 1 - S.par, S.nb, S.st))) return rc;
        MDWF_CUDA(c, cudaMemcpyAsync(x + (size_t)r0 * x4d, H.d4out, x4d * S.nb, cudaMemcpyDeviceToHost, S.st));
    }
    return S.sync();
}

static int setup_solver(mdwf_ctx* c, Solver& S, const mdwf_solve_opts* opts, cudaStream_t st) {
    if (!(opts->tol > 0.0)) MDWF_FAIL(c, MDWF_EINVAL, "tol must be > 0");
    if (opts->parity != 0 && opts->parity != 1) MDWF_FAIL(c, MDWF_EINVAL, "parity must be 0 or 1");
    const int prec = opts->inner_prec;
    if (prec != 64 && prec != 32 && prec != 16) MDWF_FAIL(c, MDWF_EINVAL, "inner_prec must be 64, 32 or 16");
    S.c = c; S.st = st;
    S.prec = prec;
    // x_lo, the solution accumulated since the last reliable update, stays in fp32 under the fp16 inner solve: fp16 rounding
    // of x (2^-11 per element and iteration) is noise in all directions, which A = Mhat^dag Mhat amplifies by its average
    // eigenvalue while x itself sits in the low modes -- at the condition numbers of the production workload that noise
    // floor is above the residual the cycle is supposed to reach and the solve stalls (tried, measured, reverted)
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
    return MDWF_OK;
}

// Batch size nb and number of rhs served by the fp64 temporaries (nhi) for `avail` bytes (beyond `extra_per_rhs` each).
// As many rhs in flight as fit (that is what the kernels gain from); the temporaries only save a few chunked passes at
// the reliable updates, so they may grow only while the workspace stays within half of `avail` -- a library-owned
// workspace is cached between calls and must not starve the caller's own allocations.
static int plan_batch(mdwf_ctx* c, const Solver& S, int nrhs, int want, size_t avail, size_t extra_per_rhs, bool own_src,
                      int* nb_out, int* nhi_out) {
    const Geom& g = c->g;
    int nb = want > 0 ? std::min(want, nrhs) : nrhs;
    for (; nb >= 1; --nb) {
        if (work_bytes(g, S.prec, S.px, nb, 1, own_src) + extra_per_rhs * nb <= avail) {
            int nhi = 1;
            while (nhi < nb) {
                const int next = std::min(nb, nhi * 2);
                const size_t need = work_bytes(g, S.prec, S.px, nb, next, own_src) + extra_per_rhs * nb;
                if (need > avail || (!c->ws_external && need > avail / 2)) break;
                nhi = next;
            }
            *nb_out = nb; *nhi_out = nhi;
            return MDWF_OK;
        }
        if (want > 0) break;    // an explicit batch is honoured or refused
    }
    MDWF_FAIL(c, MDWF_ENOMEM, "not enough device memory for a batch of %d rhs (%zu bytes available)", std::max(1, want), avail);
}

static size_t avail_bytes(mdwf_ctx* c) {
    if (c->ws_external) return c->ws_bytes;
    size_t fr = 0, tot = 0;
    if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) { cudaGetLastError(); return 0; }
    return (size_t)(0.97 * (double)(fr + c->ws_bytes));     // our own cached workspace can be re-used or re-sized
}

int solve_impl(mdwf_ctx* c, void* x, const void* b, int nrhs, const mdwf_solve_opts* opts, mdwf_solve_info* info,
               cudaStream_t st, bool host_buffers) {
    if (!x || !b || !opts || !info) MDWF_FAIL(c, MDWF_EINVAL, "null argument");
    if (nrhs < 1 || nrhs > MDWF_MAX_RHS) MDWF_FAIL(c, MDWF_EINVAL, "nrhs must be in 1..%d (got %d)", MDWF_MAX_RHS, nrhs);
    if (opts->src_kind == 0 && opts->out_kind == 0) { /* x may alias b */ }
    else if (x == b) MDWF_FAIL(c, MDWF_EINVAL, "x may alias b only for 5D source and 5D solution");
    Solver S;
    int rc = setup_solver(c, S, opts, st);
    if (rc) return rc;
    const Geom& g = c->g;
    const size_t in_per = (size_t)2 * g.Vh * 24 * 8 * (opts->src_kind ? 1 : g.Ls);
    const size_t out_per = (size_t)2 * g.Vh * 24 * 8 * (opts->out_kind ? 1 : g.Ls);
    int nb = 1, nhi = 1;
    HostStage H;
    size_t avail = avail_bytes(c), per_rhs = 0;
    if (host_buffers) {
        // 5D fields stream through two staging chunks of whole s-slices (<= ~1.5 GB each); 4D fields (wall sources, wall-projected
        // solutions) are small and staged whole
        const size_t slice = (size_t)2 * g.Vh * 24 * 8;
        H.slice_bytes = slice;
        H.ns = (int)std::max<size_t>(1, std::min<size_t>((size_t)g.Ls, ((size_t)3 << 29) / slice));
        // test hook: MDWF_STAGE_SLICES=n forces chunks of n s-slices, so that small lattices exercise the chunked, double-buffered path
        if (const char* ev = getenv("MDWF_STAGE_SLICES")) {
            const int n = atoi(ev);
            if (n >= 1) H.ns = std::min(n, g.Ls);
        }
        if (opts->src_kind == 0 || opts->out_kind == 0) avail = avail > 2 * H.ns * slice ? avail - 2 * H.ns * slice : 0;
        per_rhs = (opts->src_kind ? in_per : 0) + (opts->out_kind ? out_per : 0);
    }
    if ((rc = plan_batch(c, S, nrhs, opts->batch, avail, per_rhs, true, &nb, &nhi))) return rc;
    if (host_buffers) {
        // the workspace first, so that the staging buffers cannot starve it
        if ((rc = ensure_workspace(c, work_bytes(g, S.prec, S.px, nb, nhi, true)))) return rc;
        if ((rc = H.acquire(c, (opts->src_kind == 0 || opts->out_kind == 0) ? H.ns * H.slice_bytes : 0,
                            opts->src_kind ? in_per * nb : 0, opts->out_kind ? out_per * nb : 0))) { H.release(); return rc; }
    }
    memset(info, 0, sizeof(*info));
    cudaEvent_t e0, e1;
    MDWF_CUDA(c, cudaEventCreate(&e0));
    MDWF_CUDA(c, cudaEventCreate(&e1));
    MDWF_CUDA(c, cudaEventRecord(e0, st));
    const long long l0 = c->launches;
    double inner_ms = 0.0;
    S.nhi = nhi;
    if (!host_buffers) {
        for (int r0 = 0; r0 < nrhs && rc == MDWF_OK; r0 += nb) {
            S.nb = std::min(nb, nrhs - r0);
            S.nhi = std::min(nhi, S.nb);
            rc = solve_batch(S, (double*)x, (const double*)b, opts, info, r0, &inner_ms);
        }
    } else {
        for (int r0 = 0; r0 < nrhs && rc == MDWF_OK; r0 += nb) {
            S.nb = std::min(nb, nrhs - r0);
            S.nhi = std::min(nhi, S.nb);
            rc = solve_batch_host(S, H, (char*)x, (const char*)b, opts, info, r0, &inner_ms);
        }
        H.release();
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
    info->batch = nb;
    if (rc) return rc;
    int worst = MDWF_OK;
    for (int i = 0; i < nrhs; ++i) worst = std::max(worst, info->status[i]);
    return worst;
}

// Packed in-place solve: psi[par] / psi[1-par] hold b on entry and the solution on exit (fp64 packed half-lattice
// fields of nrhs columns each).  No canonical copies exist, so a whole batch of large-volume rhs fits on the device.
int solve_packed_impl(mdwf_ctx* c, mdwf_field* even, mdwf_field* odd, const mdwf_solve_opts* opts, mdwf_solve_info* info,
                      cudaStream_t st) {
    if (!even || !odd || !opts || !info) MDWF_FAIL(c, MDWF_EINVAL, "null argument");
    if (even->prec != 64 || odd->prec != 64 || even->nrhs != odd->nrhs || even->ctx != c || odd->ctx != c)
        MDWF_FAIL(c, MDWF_EINVAL, "mdwf_solve_packed needs two fp64 fields of this context with equal nrhs");
    if (opts->src_kind != 0 || opts->out_kind != 0) MDWF_FAIL(c, MDWF_EINVAL, "mdwf_solve_packed handles 5D sources and solutions only");
    const int nrhs = even->nrhs;
    Solver S;
    int rc = setup_solver(c, S, opts, st);
    if (rc) return rc;
    int nb = 1, nhi = 1;
    if ((rc = plan_batch(c, S, nrhs, nrhs, avail_bytes(c), 0, false, &nb, &nhi))) return rc;
    memset(info, 0, sizeof(*info));
    cudaEvent_t e0, e1;
    MDWF_CUDA(c, cudaEventCreate(&e0));
    MDWF_CUDA(c, cudaEventCreate(&e1));
    MDWF_CUDA(c, cudaEventRecord(e0, st));
    const long long l0 = c->launches;
    double inner_ms = 0.0;
    S.nb = nb; S.nhi = nhi;
    {
        Work W;
        mdwf_field* fp = S.par == 0 ? even : odd;
        mdwf_field* fo = S.par == 0 ? odd : even;
        rc = make_work(S, W, fp, fo);
        if (rc == MDWF_OK) rc = solve_core(S, W, info, 0, &inner_ms);
        if (rc == MDWF_OK) {      // psi_p: x_hi -> the caller's field
            MDWF_CUDA(c, cudaMemcpyAsync(fp->v, W.xh->v, fp->bytes, cudaMemcpyDeviceToDevice, st));
            rc = S.sync();
        }
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
    info->batch = nb;
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
    if (cudaSetDevice(c->geo.device) != cudaSuccess) return MDWF_ECUDA;
    return mdwf::solve_impl(c, x, b, nrhs, opts, info, (cudaStream_t)stream, false);
}
int mdwf_solve_host(mdwf_ctx* c, void* x, const void* b, int nrhs, const mdwf_solve_opts* opts,
                    mdwf_solve_info* info, void* stream) {
    if (!c) return MDWF_EINVAL;
    if (cudaSetDevice(c->geo.device) != cudaSuccess) return MDWF_ECUDA;
    return mdwf::solve_impl(c, x, b, nrhs, opts, info, (cudaStream_t)stream, true);
}
int mdwf_solve_packed(mdwf_ctx* c, mdwf_field* psi_even, mdwf_field* psi_odd, const mdwf_solve_opts* opts,
                      mdwf_solve_info* info, void* stream) {
    if (!c) return MDWF_EINVAL;
    if (cudaSetDevice(c->geo.device) != cudaSuccess) return MDWF_ECUDA;
    return mdwf::solve_packed_impl(c, psi_even, psi_odd, opts, info, (cudaStream_t)stream);
}
int mdwf_workspace_bytes(mdwf_ctx* c, int nrhs, int inner_prec, int packed, int64_t* bytes) {
    if (!c || !bytes) return MDWF_EINVAL;
    if (nrhs < 1 || nrhs > MDWF_MAX_RHS || (inner_prec != 64 && inner_prec != 32 && inner_prec != 16)) MDWF_FAIL(c, MDWF_EINVAL, "bad nrhs or precision");
    *bytes = (int64_t)mdwf::work_bytes(c->g, inner_prec, inner_prec == 16 ? 32 : inner_prec, nrhs, 1, !packed);
    return MDWF_OK;
}
int mdwf_set_workspace(mdwf_ctx* c, void* mem, int64_t bytes) {
    if (!c) return MDWF_EINVAL;
    if (c->ws && !c->ws_external) cudaFree(c->ws);
    c->ws = mem; c->ws_bytes = mem ? (size_t)bytes : 0; c->ws_external = mem != nullptr;
    return MDWF_OK;
}
}
