// oracle/mdwf_oracle_meas.cpp -- ORACLE (test infrastructure only): 4D<->5D maps, the
// Feynman-Hellmann sequential source and the nucleon two-point contraction, written as the
// literal index sums of SURVEY.md 8(c) O3, O4 (readings A3, A13-A15).  The paper only names these
// steps ("new type of propagator", "contractions").
#include "mdwf_oracle.h"
#include <vector>
#include <cmath>

typedef std::vector<cd> vec;
static int64_t vol4(const int* dims) { return (int64_t)dims[0] * dims[1] * dims[2] * dims[3]; }

static void get_gamma(int mu, cd g[4][4]) {
    double buf[32];
    oracle_gamma(mu, buf);
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) g[a][b] = cd(buf[2 * (4 * a + b)], buf[2 * (4 * a + b) + 1]);
}
static void matmul4(const cd A[4][4], const cd B[4][4], cd C[4][4]) {
    cd T[4][4];
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
        cd s = 0.0;
        for (int k = 0; k < 4; ++k) s += A[a][k] * B[k][b];
        T[a][b] = s;
    }
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) C[a][b] = T[a][b];
}

extern "C" {

// O3 / A13: b5D = -D_- ( P+ eta at s=0  (+)  P- eta at s=Ls-1 ).   eta4[col][x4][4][3] -> b5[col][s][x4][4][3]
int oracle_wall_inject(cd* b5, const cd* eta4, const cd* U, const int* dims, const int* bc, int Ls, int ncol,
                       const double* params) {
    const int64_t V4 = vol4(dims), n = (int64_t)ncol * Ls * V4 * 12;
    vec w(n, cd(0, 0)), t(n);
    for (int c = 0; c < ncol; ++c)
        for (int64_t x = 0; x < V4; ++x)
            for (int a = 0; a < 4; ++a)
                for (int i = 0; i < 3; ++i) {
                    const cd e = eta4[((int64_t)c * V4 + x) * 12 + 3 * a + i];
                    if (a < 2) w[(((int64_t)c * Ls + 0) * V4 + x) * 12 + 3 * a + i] += e;          // P+ at s=0
                    else       w[(((int64_t)c * Ls + (Ls - 1)) * V4 + x) * 12 + 3 * a + i] += e;   // P- at s=Ls-1
                }
    oracle_Dminus(t.data(), w.data(), U, dims, bc, Ls, ncol, params, 0);
    for (int64_t i = 0; i < n; ++i) b5[i] = -t[i];
    return 0;
}

// O3 / A3: q = P- psi_0 + P+ psi_{Ls-1}
int oracle_wall_project(cd* q4, const cd* psi5, int64_t V4, int Ls, int ncol) {
    for (int c = 0; c < ncol; ++c)
        for (int64_t x = 0; x < V4; ++x)
            for (int a = 0; a < 4; ++a)
                for (int i = 0; i < 3; ++i) {
                    const int s = (a < 2) ? (Ls - 1) : 0;   // P+ rows from s=Ls-1, P- rows from s=0
                    q4[((int64_t)c * V4 + x) * 12 + 3 * a + i] = psi5[(((int64_t)c * Ls + s) * V4 + x) * 12 + 3 * a + i];
                }
    return 0;
}

// A14: eta_seq(x)[col] = Gamma . S(x)[col] on every site with t_min <= t <= t_max, zero elsewhere.
int oracle_seq_source(cd* out4, const cd* prop4, const double* Gamma32, const int* dims, int ncol, int t_min,
                      int t_max) {
    const int64_t V4 = vol4(dims), V3 = V4 / dims[3];
    cd G[4][4];
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) G[a][b] = cd(Gamma32[2 * (4 * a + b)], Gamma32[2 * (4 * a + b) + 1]);
    for (int c = 0; c < ncol; ++c)
        for (int64_t x = 0; x < V4; ++x) {
            const int t = (int)(x / V3);
            const bool on = (t >= t_min && t <= t_max);
            for (int a = 0; a < 4; ++a)
                for (int i = 0; i < 3; ++i) {
                    cd s = 0.0;
                    if (on) for (int b = 0; b < 4; ++b) s += G[a][b] * prop4[((int64_t)c * V4 + x) * 12 + 3 * b + i];
                    out4[((int64_t)c * V4 + x) * 12 + 3 * a + i] = s;
                }
        }
    return 0;
}

// O4 (C-def), reading A15.  S^{ab}_{alpha beta}(x) = S[col = 3*beta + b][x][alpha][a].
//   C(t) = sum_x eps_{abc} eps_{a'b'c'} G_{al be} Gt_{be' al'} P_{ga' ga} Sd^{bb'}_{be be'}
//          [ Su1^{aa'}_{al al'} Su2^{cc'}_{ga ga'}  -  Su1^{ac'}_{al ga'} Su2^{ca'}_{ga al'} ]
//   G = C gamma5, C = gamma_y gamma_t;  Gt = gamma_t G^dag gamma_t.   corr index = (t - t0) mod T.
// Only timeslices t_lo <= t <= t_hi are computed (others set to 0) so that large lattices can be
// sampled; the sums skip zero entries of G, Gt, P and are otherwise the literal loops.
int oracle_nucleon_2pt(double* corr, const cd* Su1, const cd* Sd, const cd* Su2, const double* proj32,
                       const int* dims, int t0, int t_lo, int t_hi) {
    const int T = dims[3];
    const int64_t V4 = vol4(dims), V3 = V4 / T;
    cd gy[4][4], gt[4][4], g5[4][4], C[4][4], G[4][4], Gd[4][4], Gt[4][4], P[4][4];
    get_gamma(1, gy); get_gamma(3, gt); get_gamma(4, g5);
    matmul4(gy, gt, C);
    matmul4(C, g5, G);
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) Gd[a][b] = std::conj(G[b][a]);
    matmul4(gt, Gd, Gt);
    matmul4(Gt, gt, Gt);
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) P[a][b] = cd(proj32[2 * (4 * a + b)], proj32[2 * (4 * a + b) + 1]);
    static const int perm[6][3] = {{0, 1, 2}, {1, 2, 0}, {2, 0, 1}, {0, 2, 1}, {2, 1, 0}, {1, 0, 2}};
    static const double psign[6] = {1, 1, 1, -1, -1, -1};
    for (int t = 0; t < T; ++t) { corr[2 * t] = 0.0; corr[2 * t + 1] = 0.0; }
    auto S = [&](const cd* prop, int64_t x, int al, int a, int be, int b) -> cd {
        return prop[((int64_t)(3 * be + b) * V4 + x) * 12 + 3 * al + a];
    };
    for (int t = t_lo; t <= t_hi && t < T; ++t) {
        double sre = 0.0, sim = 0.0;
#pragma omp parallel for reduction(+ : sre, sim) schedule(static)
        for (int64_t xs = 0; xs < V3; ++xs) {
            const int64_t x = (int64_t)t * V3 + xs;
            cd acc = 0.0;
            for (int e1 = 0; e1 < 6; ++e1)
                for (int e2 = 0; e2 < 6; ++e2) {
                    const int a = perm[e1][0], b = perm[e1][1], c = perm[e1][2];
                    const int ap = perm[e2][0], bp = perm[e2][1], cp = perm[e2][2];
                    const double eps = psign[e1] * psign[e2];
                    for (int al = 0; al < 4; ++al) for (int be = 0; be < 4; ++be) {
                        if (G[al][be] == cd(0, 0)) continue;
                        for (int bep = 0; bep < 4; ++bep) for (int alp = 0; alp < 4; ++alp) {
                            if (Gt[bep][alp] == cd(0, 0)) continue;
                            const cd d = S(Sd, x, be, b, bep, bp);
                            for (int gap = 0; gap < 4; ++gap) for (int ga = 0; ga < 4; ++ga) {
                                if (P[gap][ga] == cd(0, 0)) continue;
                                const cd direct = S(Su1, x, al, a, alp, ap) * S(Su2, x, ga, c, gap, cp);
                                const cd exch = S(Su1, x, al, a, gap, cp) * S(Su2, x, ga, c, alp, ap);
                                acc += eps * G[al][be] * Gt[bep][alp] * P[gap][ga] * d * (direct - exch);
                            }
                        }
                    }
                }
            sre += acc.real();
            sim += acc.imag();
        }
        const int k = ((t - t0) % T + T) % T;
        corr[2 * k] = sre;
        corr[2 * k + 1] = sim;
    }
    return 0;
}

}  // extern "C"
