// ORACLE — TEST INFRASTRUCTURE ONLY (see grid.hpp).  Declarations of the solver steps.
#pragma once
#include "grid.hpp"

namespace orc {

enum { ST_OK = 0, ST_NOT_CONVERGED = 1, ST_BREAKDOWN = 2 };

// One colour half-sweep of red-black SOR (colour 0 = red = (i+j+k) even, 1 = black).  PAPER.md:59-63.
template <typename T>
void rbsor_half(const Grid& g, T* phi, const T* rhs, T omega, int colour, bool use_ghost);
// nsweeps full sweeps: red then black (PAPER.md:74 footnote: a sweep is one complete round of updates).
template <typename T>
void rbsor(const Grid& g, T* phi, const T* rhs, T omega, int nsweeps, bool use_ghost);

// Row f4 (Eq. 6-7): Chebyshev-accelerated omega sequence and its position-dependent variant.
double jacobi_radius(const Grid& g);
double local_jacobi_radius(const Grid& g, int i, int j);
double cheby_next(double rJ, int n_next, double omega_n);
void rbsor_cheby(const Grid& g, double* phi, const double* rhs, double rJ, int nsweeps, int start_n, bool use_ghost,
                 double* omegas /* nullable, 2 nsweeps */);
void rbsor_local(const Grid& g, double* phi, const double* rhs, int nsweeps, int start_n, bool use_ghost);

// Conjugate gradient, Saad Alg. 6.18 on A = -L_h (SPD), b = -rhs.  PAPER.md:95-105.
int cg(const Grid& g, double* x, const double* rhs, double rtol, int max_iter, int fixed_iters, int* iters,
       double* relres, double* history /* nullable, max_iter+1 relative residuals */);

// Row f3 (Eq. 9-10): z = B^-1 v with B the colour-block lower-triangular part of the operator
// (sign = +1: of L_h; -1: of A = -L_h), i.e. one red-black Gauss-Seidel sweep from zero; symmetric: red, black, red.
void gs_precond(const Grid& g, const double* v, double* z, int sign, bool symmetric);
// Preconditioned CG (Saad Alg. 9.1) on A = -L_h with M^-1 = the symmetrised red-black Gauss-Seidel sweep.
int pcg(const Grid& g, double* x, const double* rhs, double rtol, int max_iter, int fixed_iters, int* iters,
        double* relres, double* history);

// BiCGSTAB, Saad Alg. 7.7, right-preconditioned: jacobi = 0 none, 1 Jacobi scaling (reading C4/C10),
// 2 the red-black Gauss-Seidel preconditioner of Eq. 10.  PAPER.md:105, 107-123.
int bicgstab(const Grid& g, double* x, const double* rhs, double rtol, int max_iter, int fixed_iters, int jacobi,
             int* iters, double* relres, double* history);
// Near-breakdown threshold (default 1e-12; reading C4) and the counts of the last call: restarts taken,
// true-residual confirmations that failed.
void set_bicgstab_restart_eps(double eps);
void bicgstab_stats(int* restarts, int* confirm_failed);

// Geometric multigrid V-cycles (Eq. 11-13; reading C7).
//   restriction: 0 = transpose of trilinear (1/8)[1 3 3 1]^3, 1 = mean of the 8 children
//   precision:   0 = fp64, 1 = mixed (fp64 residual + correction, fp32 error-equation V-cycle)
int vcycle(const Grid& g, double* phi, const double* rhs, int nu1, int nu2, int coarsest_n, int coarsest_sweeps,
           int precision, int restriction, int ncycles, double* resnorms /* nullable, ncycles+1 */);

// Transfer operators exposed for the pins (R 1 = 1, P 1 = 1, <Pu,v> = 8 <u,Rv>).
template <typename T>
void restrict_fw(const Grid& fine, const Grid& coarse, const T* r, T* fc, int restriction);
template <typename T>
void prolong_add(const Grid& fine, const Grid& coarse, const T* ec, T* phi);
Grid coarsen(const Grid& fine, int level_of_coarse);

// ---- the paper's own multigrid (mgv.cpp): vertex-centred, Galerkin, SPAI smoother, CG coarsest; PAPER.md:125-205 -------
// spai[5] = {omega, alpha, beta, gamma, delta} of Eq. 15-16 (Table 1).
void spai_smooth(const Grid& g, double* phi, const double* rhs, const double spai[5], int nsteps, int order = 2);
// compact radius-1 discretisations of order 2 / 4 / 6: the operator and its right-hand-side transform
int compact_apply(const Grid& g, int order, const double* v, double* out);
int compact_rhs(const int n[3], int order, const double* f_ext, double* out);
int mgv_vcycle(const Grid& g, double* phi, const double* rhs, int nu1, int nu2, int coarsest_n, const double spai[5],
               double cg_rtol, int storage_f32, int ncycles, double* resnorms /* nullable, ncycles+1 */, int order = 2);
int mgv_galerkin_stencil(const Grid& g, int level, int I, int J, int K, double* out27, int order = 2);
void mgv_restrict(const Grid& g, const double* r, double* bc);
void mgv_prolong_add(const Grid& g, const double* ec, double* x);

// Multipole boundary condition, Eq. 19-20.  Fills g.ghost[] on Dirichlet faces.
void multipole_moments(const Grid& g, const double* rho, int lmax, double* q /* (lmax+1)^2, index l*l+l+m */);
double multipole_potential(const double* q, int lmax, double G, double x, double y, double z);
void multipole_bc(Grid& g, const double* rho, double G, int lmax, double* moments /* nullable */,
                  double* inner_moments = nullptr /* nullable */);
// Inner expansion for a spherical grid with r_in > 0 (Eq. 21-22).
void multipole_inner_moments(const Grid& g, const double* rho, int lmax, double* qbar);
double multipole_inner_potential(const double* qbar, int lmax, double G, double x, double y, double z);

}  // namespace orc
