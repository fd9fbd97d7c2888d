// oracle/mdwf_oracle.cpp -- plain, slow, fp64 CPU ORACLE for the MDWF hot path.
//
// TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this library.  It shares no code, header, table or constant with
// paper_1810_01609_b200/csrc (the CUDA product path) and neither includes the other.
//
// What it follows.  The paper (reference PAPER.md) only NAMES its method: "Moebius Domain-Wall
// discretization", "radius-one stencil", "12x12 dense" blocks, "red-black
// preconditioned" operator solved by CG on the normal equations in "double-half" precision with
// "reliable updates", Feynman-Hellmann propagators and nucleon
// contractions.  It prints no operator, so the definitions written out here are
// the readings fixed in SURVEY.md section 8 "Notation" and 8(c) A1-A23 (listed again in DESIGN.md).
// Every function cites the reading it implements.  Each is pinned in tests/test_oracle_pins.py
// by something other than itself (free-field spectrum, gamma5-hermiticity, gauge covariance,
// Shamir limit vs an independently coded operator, dense brute force, overlap identity, ...).
//
// Style: the plain definition, full 4x4 gamma matrices, full 3x3 links, no half-spinor trick, no
// blocking or fusion.  Even-odd objects are derived by masking full-lattice operators.
// OpenMP "parallel for" over sites only (it doubles as the timed CPU baseline).
//
// Canonical layouts:  x4 = x + X*(y + Y*(z + Z*t));
//   spinor psi[k][x4][spin(4)][colour(3)]   k = slice index (rhs*Ls + s), complex<double>
//   gauge  U[mu][x4][row][col]              U_mu(x) is the link from x to x+mu
#include <complex>
#include <vector>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <cstdio>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
static const cd I_(0.0, 1.0);

// ---------------------------------------------------------------------------------------------
// gamma matrices: DeGrand-Rossi chiral basis (SURVEY 8 Notation, reading A2).  mu = 0..3 <-> x,y,z,t
// gamma5 = gx gy gz gt = diag(+1,+1,-1,-1).  Pinned by the Clifford-algebra test.
// ---------------------------------------------------------------------------------------------
static const cd GAMMA[4][4][4] = {
    // gamma_x
    {{0, 0, 0, I_}, {0, 0, I_, 0}, {0, -I_, 0, 0}, {-I_, 0, 0, 0}},
    // gamma_y
    {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    // gamma_z
    {{0, 0, I_, 0}, {0, 0, 0, -I_}, {-I_, 0, 0, 0}, {0, I_, 0, 0}},
    // gamma_t
    {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}},
};
static const double GAMMA5[4] = {1.0, 1.0, -1.0, -1.0};

struct Geom {
    int L[4];
    int bc[4];
    int64_t V4;
};
static Geom make_geom(const int* dims, const int* bc) {
    Geom g;
    g.V4 = 1;
    for (int m = 0; m < 4; ++m) { g.L[m] = dims[m]; g.bc[m] = bc[m]; g.V4 *= dims[m]; }
    return g;
}
static inline void coords(const Geom& g, int64_t x4, int c[4]) {
    c[0] = (int)(x4 % g.L[0]); x4 /= g.L[0];
    c[1] = (int)(x4 % g.L[1]); x4 /= g.L[1];
    c[2] = (int)(x4 % g.L[2]); x4 /= g.L[2];
    c[3] = (int)x4;
}
static inline int64_t lin(const Geom& g, const int c[4]) {
    return c[0] + (int64_t)g.L[0] * (c[1] + (int64_t)g.L[1] * (c[2] + (int64_t)g.L[2] * c[3]));
}
static inline int site_parity(const int c[4]) { return (c[0] + c[1] + c[2] + c[3]) & 1; }

extern "C" {

// gamma matrices exported so the tests can check the algebra (pin: Clifford, hermiticity, gamma5).
void oracle_gamma(int mu, double* out32 /* [4][4][re,im] */) {
    for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b) {
            cd v = (mu < 4) ? GAMMA[mu][a][b] : ((a == b) ? cd(GAMMA5[a], 0) : cd(0, 0));
            out32[2 * (4 * a + b)] = v.real();
            out32[2 * (4 * a + b) + 1] = v.imag();
        }
}

int oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// ---------------------------------------------------------------------------------------------
// Wilson hop (SURVEY 8 Notation; reading A1, A4, A21):
//   (H psi)(x)   = sum_mu [ (1 - g_mu) U_mu(x) psi(x+mu) + (1 + g_mu) U_mu(x-mu)^dag psi(x-mu) ]
//   (H^dag psi)  = same with (1 - g_mu) <-> (1 + g_mu)
// A hop that crosses the mu boundary is multiplied by bc_mu.  Acts identically on each of the
// n5 slices.  out_parity = -1: every site; 0/1: only sites of that 4D parity are computed and the
// others are set to zero (this IS "apply H, then keep parity p").
// ---------------------------------------------------------------------------------------------
int oracle_hop(cd* out, const cd* in, const cd* U, const int* dims, const int* bc, int n5, int dagger,
               int out_parity) {
    const Geom g = make_geom(dims, bc);
    const double sgn = dagger ? -1.0 : 1.0;   // (1 - sgn*g_mu) forward, (1 + sgn*g_mu) backward
#pragma omp parallel for schedule(static)
    for (int64_t x4 = 0; x4 < g.V4; ++x4) {
        int c[4];
        coords(g, x4, c);
        const bool keep = (out_parity < 0) || (site_parity(c) == out_parity);
        for (int k = 0; k < n5; ++k) {
            cd acc[4][3];
            for (int a = 0; a < 4; ++a) for (int i = 0; i < 3; ++i) acc[a][i] = 0.0;
            if (keep) {
                for (int mu = 0; mu < 4; ++mu) {
                    // forward neighbour x+mu, link U_mu(x)
                    int cf[4] = {c[0], c[1], c[2], c[3]};
                    double ff = 1.0;
                    cf[mu] += 1;
                    if (cf[mu] == g.L[mu]) { cf[mu] = 0; ff = (double)g.bc[mu]; }
                    const int64_t xf = lin(g, cf);
                    const cd* Uf = U + ((int64_t)mu * g.V4 + x4) * 9;
                    const cd* pf = in + ((int64_t)k * g.V4 + xf) * 12;
                    // backward neighbour x-mu, link U_mu(x-mu)^dagger
                    int cb[4] = {c[0], c[1], c[2], c[3]};
                    double fb = 1.0;
                    cb[mu] -= 1;
                    if (cb[mu] < 0) { cb[mu] = g.L[mu] - 1; fb = (double)g.bc[mu]; }
                    const int64_t xb = lin(g, cb);
                    const cd* Ub = U + ((int64_t)mu * g.V4 + xb) * 9;
                    const cd* pb = in + ((int64_t)k * g.V4 + xb) * 12;
                    cd wf[4][3], wb[4][3];
                    for (int a = 0; a < 4; ++a)
                        for (int i = 0; i < 3; ++i) {
                            cd sf = 0.0, sb = 0.0;
                            for (int j = 0; j < 3; ++j) {
                                sf += Uf[3 * i + j] * pf[3 * a + j];
                                sb += std::conj(Ub[3 * j + i]) * pb[3 * a + j];
                            }
                            wf[a][i] = ff * sf;
                            wb[a][i] = fb * sb;
                        }
                    for (int a = 0; a < 4; ++a)
                        for (int i = 0; i < 3; ++i) {
                            cd gf = 0.0, gb = 0.0;
                            for (int b = 0; b < 4; ++b) {
                                gf += GAMMA[mu][a][b] * wf[b][i];
                                gb += GAMMA[mu][a][b] * wb[b][i];
                            }
                            acc[a][i] += (wf[a][i] - sgn * gf) + (wb[a][i] + sgn * gb);
                        }
                }
            }
            cd* o = out + ((int64_t)k * g.V4 + x4) * 12;
            for (int a = 0; a < 4; ++a) for (int i = 0; i < 3; ++i) o[3 * a + i] = acc[a][i];
        }
    }
    return 0;
}

// D_W = (4 - M5) - 1/2 H   (SURVEY 8 Notation, reading A5); dagger: H -> H^dag.
int oracle_wilson(cd* out, const cd* in, const cd* U, const int* dims, const int* bc, int n5, double M5,
                  int dagger) {
    const Geom g = make_geom(dims, bc);
    oracle_hop(out, in, U, dims, bc, n5, dagger, -1);
    const int64_t n = (int64_t)n5 * g.V4 * 12;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) out[i] = (4.0 - M5) * in[i] - 0.5 * out[i];
    return 0;
}

// ---------------------------------------------------------------------------------------------
// s-direction hop with mass (SURVEY 8 Notation, reading A3):
//   (L psi)_s     = P- psi_{s+1} + P+ psi_{s-1},  psi_{Ls} = -mf psi_0,  psi_{-1} = -mf psi_{Ls-1}
//   (L^dag psi)_s = P+ psi_{s+1} + P- psi_{s-1}   with the same -mf wraps
// P+ keeps spin rows 0,1, P- keeps rows 2,3 (gamma5 diagonal).   out = c0*psi + c1*L psi.
// (c0,c1) = (a,d) gives M5, (b5,c5) gives A = "M4pre" (SURVEY 8 "Even-odd form").
// ---------------------------------------------------------------------------------------------
int oracle_ls_hop(cd* out, const cd* in, int64_t V4, int Ls, int nrhs, double mf, double c0, double c1,
                  int dagger) {
#pragma omp parallel for schedule(static)
    for (int64_t x4 = 0; x4 < V4; ++x4)
        for (int r = 0; r < nrhs; ++r)
            for (int s = 0; s < Ls; ++s) {
                const int sp = (s + 1) % Ls, sm = (s + Ls - 1) % Ls;
                const double fp = (s + 1 == Ls) ? -mf : 1.0;   // factor on psi_{s+1}
                const double fm = (s == 0) ? -mf : 1.0;        // factor on psi_{s-1}
                const cd* up = in + (((int64_t)r * Ls + sp) * V4 + x4) * 12;
                const cd* dn = in + (((int64_t)r * Ls + sm) * V4 + x4) * 12;
                const cd* me = in + (((int64_t)r * Ls + s) * V4 + x4) * 12;
                cd* o = out + (((int64_t)r * Ls + s) * V4 + x4) * 12;
                for (int a = 0; a < 4; ++a) {
                    const bool plus = GAMMA5[a] > 0;     // spin row belongs to P+
                    // not dagger: P+ rows take psi_{s-1}, P- rows take psi_{s+1}; dagger swaps
                    const bool take_up = dagger ? plus : !plus;
                    for (int i = 0; i < 3; ++i) {
                        const cd l = take_up ? fp * up[3 * a + i] : fm * dn[3 * a + i];
                        o[3 * a + i] = c0 * me[3 * a + i] + c1 * l;
                    }
                }
            }
    return 0;
}

// ---------------------------------------------------------------------------------------------
// M5^{-1} (reading A7: the oracle uses a GENERIC dense LU, not the closed form).
// M5 = a + d L is diagonal in the 4D site and in colour and couples only s within one chirality,
// so per chirality it is one real Ls x Ls matrix.  The matrix is built by applying oracle_ls_hop
// to unit vectors, factored by Gaussian elimination with partial pivoting, and the triangular
// solves are applied to every (site, spin, colour) column.
// ---------------------------------------------------------------------------------------------
static void lu_factor(std::vector<double>& A, std::vector<int>& piv, int n) {
    piv.resize(n);
    for (int k = 0; k < n; ++k) {
        int p = k;
        for (int i = k + 1; i < n; ++i) if (std::fabs(A[i * n + k]) > std::fabs(A[p * n + k])) p = i;
        piv[k] = p;
        if (p != k) for (int j = 0; j < n; ++j) std::swap(A[k * n + j], A[p * n + j]);
        for (int i = k + 1; i < n; ++i) {
            A[i * n + k] /= A[k * n + k];
            for (int j = k + 1; j < n; ++j) A[i * n + j] -= A[i * n + k] * A[k * n + j];
        }
    }
}
static void lu_solve(const std::vector<double>& A, const std::vector<int>& piv, int n, cd* x) {
    for (int k = 0; k < n; ++k) if (piv[k] != k) std::swap(x[k], x[piv[k]]);
    for (int i = 0; i < n; ++i) for (int j = 0; j < i; ++j) x[i] -= A[i * n + j] * x[j];
    for (int i = n - 1; i >= 0; --i) {
        for (int j = i + 1; j < n; ++j) x[i] -= A[i * n + j] * x[j];
        x[i] /= A[i * n + i];
    }
}

int oracle_ls_inv(cd* out, const cd* in, int64_t V4, int Ls, int nrhs, double mf, double c0, double c1,
                  int dagger) {
    // build the two chirality blocks from the definition (one site, one rhs)
    std::vector<double> Mat[2];
    std::vector<int> piv[2];
    for (int ch = 0; ch < 2; ++ch) Mat[ch].assign((size_t)Ls * Ls, 0.0);
    {
        std::vector<cd> e((size_t)Ls * 12), Me((size_t)Ls * 12);
        for (int sc = 0; sc < Ls; ++sc)
            for (int ch = 0; ch < 2; ++ch) {
                std::fill(e.begin(), e.end(), cd(0, 0));
                const int spin = ch == 0 ? 0 : 2;     // a P+ row / a P- row
                e[(size_t)sc * 12 + 3 * spin] = 1.0;
                oracle_ls_hop(Me.data(), e.data(), 1, Ls, 1, mf, c0, c1, dagger);
                for (int sr = 0; sr < Ls; ++sr) Mat[ch][(size_t)sr * Ls + sc] = Me[(size_t)sr * 12 + 3 * spin].real();
            }
    }
    for (int ch = 0; ch < 2; ++ch) lu_factor(Mat[ch], piv[ch], Ls);
#pragma omp parallel for schedule(static)
    for (int64_t x4 = 0; x4 < V4; ++x4) {
        std::vector<cd> col(Ls);
        for (int r = 0; r < nrhs; ++r)
            for (int a = 0; a < 4; ++a)
                for (int i = 0; i < 3; ++i) {
                    const int ch = GAMMA5[a] > 0 ? 0 : 1;
                    for (int s = 0; s < Ls; ++s) col[s] = in[(((int64_t)r * Ls + s) * V4 + x4) * 12 + 3 * a + i];
                    lu_solve(Mat[ch], piv[ch], Ls, col.data());
                    for (int s = 0; s < Ls; ++s) out[(((int64_t)r * Ls + s) * V4 + x4) * 12 + 3 * a + i] = col[s];
                }
    }
    return 0;
}

// zero every site whose 4D parity differs from `keep` (keep = 0/1)
int oracle_mask(cd* f, const int* dims, int n5, int keep) {
    const int bcd[4] = {1, 1, 1, 1};
    const Geom g = make_geom(dims, bcd);
#pragma omp parallel for schedule(static)
    for (int64_t x4 = 0; x4 < g.V4; ++x4) {
        int c[4];
        coords(g, x4, c);
        if (site_parity(c) != keep)
            for (int k = 0; k < n5; ++k) {
                cd* p = f + ((int64_t)k * g.V4 + x4) * 12;
                for (int j = 0; j < 12; ++j) p[j] = 0.0;
            }
    }
    return 0;
}

}  // extern "C"
