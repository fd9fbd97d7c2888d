// oracle/mdwf_oracle.h -- prototypes of the CPU ORACLE (test infrastructure only; see
// mdwf_oracle.cpp).  Private to oracle/: nothing under paper_1810_01609_b200/ may include it.
#pragma once
#include <complex>
#include <cstdint>
typedef std::complex<double> cd;

extern "C" {
void oracle_gamma(int mu, double* out32);
int oracle_num_threads(void);
int oracle_hop(cd* out, const cd* in, const cd* U, const int* dims, const int* bc, int n5, int dagger,
               int out_parity);
int oracle_wilson(cd* out, const cd* in, const cd* U, const int* dims, const int* bc, int n5, double M5,
                  int dagger);
int oracle_ls_hop(cd* out, const cd* in, int64_t V4, int Ls, int nrhs, double mf, double c0, double c1,
                  int dagger);
int oracle_ls_inv(cd* out, const cd* in, int64_t V4, int Ls, int nrhs, double mf, double c0, double c1,
                  int dagger);
int oracle_mask(cd* f, const int* dims, int n5, int keep);

// params = {M5, b5, c5, mf}
int oracle_D(cd* out, const cd* in, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
             const double* params, int dagger);
int oracle_Dminus(cd* out, const cd* in, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
                  const double* params, int dagger);
int oracle_schur(cd* out, const cd* in, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
                 const double* params, int parity, int dagger, int symmetric);
int oracle_prepare_source(cd* bhat, const cd* b, const cd* U, const int* dims, const int* bc, int Ls,
                          int nrhs, const double* params, int parity);
int oracle_reconstruct(cd* psi, const cd* psi_p, const cd* b, const cd* U, const int* dims, const int* bc,
                       int Ls, int nrhs, const double* params, int parity);
int oracle_solve_full(cd* x, const cd* b, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
                      const double* params, double tol, int max_iter, int* iters, double* resid);
int oracle_solve_eo(cd* x, const cd* b, const cd* U, const int* dims, const int* bc, int Ls, int nrhs,
                    const double* params, int parity, int symmetric, double tol, int max_iter, int* iters,
                    double* resid);
int oracle_wall_inject(cd* b5, const cd* eta4, const cd* U, const int* dims, const int* bc, int Ls, int ncol,
                       const double* params);
int oracle_wall_project(cd* q4, const cd* psi5, int64_t V4, int Ls, int ncol);
int oracle_seq_source(cd* out4, const cd* prop4, const double* Gamma32, const int* dims, int ncol, int t_min,
                      int t_max);
int oracle_nucleon_2pt(double* corr /* [T][2] */, const cd* Su1, const cd* Sd, const cd* Su2,
                       const double* proj32, const int* dims, int t0, int t_lo, int t_hi);
}
