// oracle/mdwf_oracle_dwf.cpp -- ORACLE (test infrastructure only): Moebius domain-wall operator,
// its even-odd Schur complements, and the plain fp64 CG solves.  See mdwf_oracle.cpp for the
// header notes; definitions are the readings of SURVEY.md section 8 ("Notation", A1-A10).
#include "mdwf_oracle.h"
#include <vector>
#include <cmath>
#include <cstdio>
#include <functional>

typedef std::vector<cd> vec;

static int64_t vol4(const int* dims) { return (int64_t)dims[0] * dims[1] * dims[2] * dims[3]; }

static double norm2(const cd* a, int64_t n) {
    double s = 0.0;
#pragma omp parallel for reduction(+ : s) schedule(static)
    for (int64_t i = 0; i < n; ++i) s += std::norm(a[i]);
    return s;
}
static cd cdot(const cd* a, const cd* b, int64_t n) {   // <a,b> = sum conj(a) b
    double re = 0.0, im = 0.0;
#pragma omp parallel for reduction(+ : re, im) schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        cd t = std::conj(a[i]) * b[i];
        re += t.real();
        im += t.imag();
    }
    return cd(re, im);
}

extern "C" {

// ---------------------------------------------------------------------------------------------
// Moebius DWF (SURVEY 8 Notation, reading A1):  D_+ = b5 D_W + 1,  D_- = c5 D_W - 1,
//   D psi     = D_+ psi + D_- (L psi)
//   D^dag psi = D_+^dag psi + L^dag (D_-^dag psi),   D_W^dag = (4-M5) - 1/2 H^dag
// ---------------------------------------------------------------------------------------------
int oracle_D(cd* out, const cd* in, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
             const double* params, int dagger) {
    const double M5 = params[0], b5 = params[1], c5 = params[2], mf = params[3];
    const int64_t V4 = vol4(dims), n = (int64_t)nrhs * Ls * V4 * 12;
    const int n5 = nrhs * Ls;
    vec dw(n), t(n), dwt(n);
    if (!dagger) {
        oracle_ls_hop(t.data(), in, V4, Ls, nrhs, mf, 0.0, 1.0, 0);           // t = L psi
        oracle_wilson(dw.data(), in, U, dims, bc, n5, M5, 0);                   // D_W psi
        oracle_wilson(dwt.data(), t.data(), U, dims, bc, n5, M5, 0);            // D_W L psi
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) out[i] = (b5 * dw[i] + in[i]) + (c5 * dwt[i] - t[i]);
    } else {
        oracle_wilson(dw.data(), in, U, dims, bc, n5, M5, 1);                   // D_W^dag psi
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) t[i] = c5 * dw[i] - in[i];             // D_-^dag psi
        oracle_ls_hop(dwt.data(), t.data(), V4, Ls, nrhs, mf, 0.0, 1.0, 1);     // L^dag D_-^dag psi
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) out[i] = (b5 * dw[i] + in[i]) + dwt[i];
    }
    return 0;
}

// D_- = c5 D_W - 1 on every s-slice (needed for the 4D source injection, O3, and for the A8 pins)
int oracle_Dminus(cd* out, const cd* in, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
                  const double* params, int dagger) {
    const double M5 = params[0], c5 = params[2];
    const int64_t V4 = vol4(dims), n = (int64_t)nrhs * Ls * V4 * 12;
    vec dw(n);
    oracle_wilson(dw.data(), in, U, dims, bc, nrhs * Ls, M5, dagger);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) out[i] = c5 * dw[i] - in[i];
    return 0;
}

// ---------------------------------------------------------------------------------------------
// Even-odd form (SURVEY 8 "Even-odd form", readings A6, A7), all on FULL-lattice arrays whose
// other-parity sites are zero:   a = b5(4-M5)+1, d = c5(4-M5)-1, M5op = a + d L, A = b5 + c5 L
//   Dhat      = M5op - 1/4 H_{p pbar} A M5op^-1 H_{pbar p} A
//   Dhat^dag  = M5op^dag - 1/4 A^dag (H^dag)_{p pbar} M5op^-dag A^dag (H^dag)_{pbar p}
//   Mhat      = M5op^-1 Dhat,   Mhat^dag = Dhat^dag M5op^-dag              (symmetric = 1)
// H_{q <- q'} is "apply H to a field supported on q', keep parity q" (oracle_hop's out_parity).
// ---------------------------------------------------------------------------------------------
int oracle_schur(cd* out, const cd* in_, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
                 const double* params, int parity, int dagger, int symmetric) {
    const double M5 = params[0], b5 = params[1], c5 = params[2], mf = params[3];
    const double a = b5 * (4.0 - M5) + 1.0, d = c5 * (4.0 - M5) - 1.0;
    const int64_t V4 = vol4(dims), n = (int64_t)nrhs * Ls * V4 * 12;
    const int n5 = nrhs * Ls, p = parity, pb = 1 - parity;
    vec in(in_, in_ + n), t1(n), t2(n);
    oracle_mask(in.data(), dims, n5, p);
    if (!dagger) {
        oracle_ls_hop(t1.data(), in.data(), V4, Ls, nrhs, mf, b5, c5, 0);        // A x
        oracle_hop(t2.data(), t1.data(), U, dims, bc, n5, 0, pb);                // H_{pbar p}
        oracle_ls_inv(t1.data(), t2.data(), V4, Ls, nrhs, mf, a, d, 0);          // M5^-1
        oracle_ls_hop(t2.data(), t1.data(), V4, Ls, nrhs, mf, b5, c5, 0);        // A
        oracle_hop(t1.data(), t2.data(), U, dims, bc, n5, 0, p);                 // H_{p pbar}
        oracle_ls_hop(t2.data(), in.data(), V4, Ls, nrhs, mf, a, d, 0);          // M5 x
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) t2[i] = t2[i] - 0.25 * t1[i];           // Dhat x
        if (symmetric) oracle_ls_inv(out, t2.data(), V4, Ls, nrhs, mf, a, d, 0);
        else std::copy(t2.begin(), t2.end(), out);
    } else {
        vec y(in);
        if (symmetric) oracle_ls_inv(y.data(), in.data(), V4, Ls, nrhs, mf, a, d, 1);   // M5^-dag x
        oracle_hop(t1.data(), y.data(), U, dims, bc, n5, 1, pb);                 // (H^dag)_{pbar p}
        oracle_ls_hop(t2.data(), t1.data(), V4, Ls, nrhs, mf, b5, c5, 1);        // A^dag
        oracle_ls_inv(t1.data(), t2.data(), V4, Ls, nrhs, mf, a, d, 1);          // M5^-dag
        oracle_hop(t2.data(), t1.data(), U, dims, bc, n5, 1, p);                 // (H^dag)_{p pbar}
        oracle_ls_hop(t1.data(), t2.data(), V4, Ls, nrhs, mf, b5, c5, 1);        // A^dag
        oracle_ls_hop(t2.data(), y.data(), V4, Ls, nrhs, mf, a, d, 1);           // M5^dag y
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) out[i] = t2[i] - 0.25 * t1[i];
    }
    return 0;
}

// bhat_p = b_p + 1/2 H_{p pbar} A M5^-1 b_pbar   (full-lattice array, zero on pbar)
int oracle_prepare_source(cd* bhat, const cd* b, const cd* U, const int* dims, const int* bc, int Ls,
                          int nrhs, const double* params, int parity) {
    const double M5 = params[0], b5 = params[1], c5 = params[2], mf = params[3];
    const double a = b5 * (4.0 - M5) + 1.0, d = c5 * (4.0 - M5) - 1.0;
    const int64_t V4 = vol4(dims), n = (int64_t)nrhs * Ls * V4 * 12;
    const int n5 = nrhs * Ls;
    vec bp(b, b + n), bq(b, b + n), t(n);
    oracle_mask(bp.data(), dims, n5, parity);
    oracle_mask(bq.data(), dims, n5, 1 - parity);
    oracle_ls_inv(t.data(), bq.data(), V4, Ls, nrhs, mf, a, d, 0);
    oracle_ls_hop(bq.data(), t.data(), V4, Ls, nrhs, mf, b5, c5, 0);
    oracle_hop(t.data(), bq.data(), U, dims, bc, n5, 0, parity);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) bhat[i] = bp[i] + 0.5 * t[i];
    return 0;
}

// psi = psi_p (+) M5^-1 ( b_pbar + 1/2 H_{pbar p} A psi_p )
int oracle_reconstruct(cd* psi, const cd* psi_p_, const cd* b, const cd* U, const int* dims, const int* bc,
                       int Ls, int nrhs, const double* params, int parity) {
    const double M5 = params[0], b5 = params[1], c5 = params[2], mf = params[3];
    const double a = b5 * (4.0 - M5) + 1.0, d = c5 * (4.0 - M5) - 1.0;
    const int64_t V4 = vol4(dims), n = (int64_t)nrhs * Ls * V4 * 12;
    const int n5 = nrhs * Ls;
    vec pp(psi_p_, psi_p_ + n), bq(b, b + n), t(n), t2(n);
    oracle_mask(pp.data(), dims, n5, parity);
    oracle_mask(bq.data(), dims, n5, 1 - parity);
    oracle_ls_hop(t.data(), pp.data(), V4, Ls, nrhs, mf, b5, c5, 0);
    oracle_hop(t2.data(), t.data(), U, dims, bc, n5, 0, 1 - parity);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) t2[i] = bq[i] + 0.5 * t2[i];
    oracle_ls_inv(t.data(), t2.data(), V4, Ls, nrhs, mf, a, d, 0);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) psi[i] = pp[i] + t[i];
    return 0;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// Plain CG on a hermitian positive operator N (textbook; "CG on the normal equations").
// x0 = 0.  Stops when ||r||/||rhs|| <= tol (recursive residual) or after max_iter.
// ---------------------------------------------------------------------------------------------
static int cg(const std::function<void(cd*, const cd*)>& N, cd* x, const cd* rhs, int64_t n, double tol,
              int max_iter, double* rel_out) {
    vec r(rhs, rhs + n), p(rhs, rhs + n), Ap(n);
    std::fill(x, x + n, cd(0, 0));
    const double b2 = norm2(rhs, n);
    double r2 = b2;
    int it = 0;
    if (b2 == 0.0) { *rel_out = 0.0; return 0; }
    while (it < max_iter && std::sqrt(r2 / b2) > tol) {
        N(Ap.data(), p.data());
        const double pAp = cdot(p.data(), Ap.data(), n).real();
        const double alpha = r2 / pAp;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) { x[i] += alpha * p[i]; r[i] -= alpha * Ap[i]; }
        const double r2n = norm2(r.data(), n);
        const double beta = r2n / r2;
        r2 = r2n;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
        ++it;
    }
    *rel_out = std::sqrt(r2 / b2);
    return it;
}

extern "C" {

// Variant A: CG on D^dag D psi = D^dag b on the full unpreconditioned 5D lattice.
int oracle_solve_full(cd* x, const cd* b, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
                      const double* params, double tol, int max_iter, int* iters, double* resid) {
    const int64_t n1 = (int64_t)Ls * vol4(dims) * 12;
    for (int r = 0; r < nrhs; ++r) {
        vec rhs(n1), tmp(n1);
        oracle_D(rhs.data(), b + r * n1, U, dims, bc, Ls, 1, params, 1);
        auto N = [&](cd* o, const cd* i) {
            oracle_D(tmp.data(), i, U, dims, bc, Ls, 1, params, 0);
            oracle_D(o, tmp.data(), U, dims, bc, Ls, 1, params, 1);
        };
        iters[r] = cg(N, x + r * n1, rhs.data(), n1, tol, max_iter, &resid[r]);
    }
    return 0;
}

// Variant B: the oracle's own even-odd route.  Solve (S^dag S) psi_p = S^dag rhs with
// S = Dhat (rhs = bhat) or S = Mhat (rhs = M5^-1 bhat), then reconstruct psi_pbar.
int oracle_solve_eo(cd* x, const cd* b, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
                    const double* params, int parity, int symmetric, double tol, int max_iter, int* iters,
                    double* resid) {
    const double M5 = params[0], b5 = params[1], c5 = params[2], mf = params[3];
    const double a = b5 * (4.0 - M5) + 1.0, d = c5 * (4.0 - M5) - 1.0;
    const int64_t V4 = vol4(dims), n1 = (int64_t)Ls * V4 * 12;
    for (int r = 0; r < nrhs; ++r) {
        vec bhat(n1), rhs(n1), tmp(n1), xp(n1);
        oracle_prepare_source(bhat.data(), b + r * n1, U, dims, bc, Ls, 1, params, parity);
        if (symmetric) {
            oracle_ls_inv(tmp.data(), bhat.data(), V4, Ls, 1, mf, a, d, 0);
            bhat = tmp;
        }
        oracle_schur(rhs.data(), bhat.data(), U, dims, bc, Ls, 1, params, parity, 1, symmetric);
        auto N = [&](cd* o, const cd* i) {
            oracle_schur(tmp.data(), i, U, dims, bc, Ls, 1, params, parity, 0, symmetric);
            oracle_schur(o, tmp.data(), U, dims, bc, Ls, 1, params, parity, 1, symmetric);
        };
        iters[r] = cg(N, xp.data(), rhs.data(), n1, tol, max_iter, &resid[r]);
        oracle_reconstruct(x + r * n1, xp.data(), b + r * n1, U, dims, bc, Ls, 1, params, parity);
    }
    return 0;
}

}  // extern "C"
