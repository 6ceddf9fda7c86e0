// ORACLE — TEST INFRASTRUCTURE ONLY (see grid.hpp).
// Red-black Gauss-Seidel / SOR.  PAPER.md:59-63: "red and black cells of a 3D checkerboard pattern are alternately
// updated"; "Each SOR update amplifies the corresponding Gauss-Seidel update by the factor omega"; omega = 1 is
// Gauss-Seidel.  Reading: red = (i+j+k) even, red first then black; one sweep = both colours.
//   gs  = (sum_nb c_nb phi_nb - rhs) / d        (the value that zeroes the residual of row ijk)
//   phi <- phi + omega (gs - phi)
#include <cmath>
#include <vector>

#include "solvers.hpp"

namespace orc {

template <typename T>
void rbsor_half(const Grid& g, T* phi, const T* rhs, T omega, int colour, bool use_ghost) {
    // With a radius-1 stencil points of one colour are independent, so the k-loop may run in parallel with
    // identical results.  For radius 3 the two-colouring is not independent: keep it serial.
#pragma omp parallel for schedule(static) if (g.order == 2)
    for (int k = 0; k < g.n[2]; ++k)
        for (int j = 0; j < g.n[1]; ++j)
            for (int i = 0; i < g.n[0]; ++i) {
                if (((i + j + k) & 1) != colour) continue;
                size_t p = g.idx(i, j, k);
                T s = offsum(g, phi, i, j, k, use_ghost);
                T d = diag<T>(g, i, j, k);
                T gs = (s - rhs[p]) / d;
                phi[p] = fma_(omega, gs - phi[p], phi[p]);
            }
}
template void rbsor_half<double>(const Grid&, double*, const double*, double, int, bool);
template void rbsor_half<float>(const Grid&, float*, const float*, float, int, bool);

template <typename T>
void rbsor(const Grid& g, T* phi, const T* rhs, T omega, int nsweeps, bool use_ghost) {
    for (int s = 0; s < nsweeps; ++s) {
        rbsor_half(g, phi, rhs, omega, 0, use_ghost);
        rbsor_half(g, phi, rhs, omega, 1, use_ghost);
    }
}
template void rbsor<double>(const Grid&, double*, const double*, double, int, bool);
template void rbsor<float>(const Grid&, float*, const float*, float, int, bool);

// ---- Chebyshev-accelerated and position-dependent omega (Eq. 6-7) -----------------
// Spectral radius of the Jacobi iteration, Eq. 4, with N = n + 1 intervals for n unknowns per axis (C0: the
// exact value for ghost-Dirichlet faces, consistent with omega_opt = 2/(1 + sin(pi/(n+1))) of Eq. 3).
double jacobi_radius(const Grid& g) {
    double num = 0.0, den = 0.0;
    for (int a = 0; a < 3; ++a) {
        const double c = 1.0 / (g.h[a] * g.h[a]);
        num += c * std::cos(M_PI / (g.n[a] + 1));
        den += c;
    }
    return num / den;
}

// Eq. 6: omega_0 = 1, omega_1 = 1/(1 - rJ^2/2), omega_{n+1} = 1/(1 - rJ^2 omega_n/4).
double cheby_next(double rJ, int n_next, double omega_n) {
    if (n_next == 0) return 1.0;
    if (n_next == 1) return 1.0 / (1.0 - 0.5 * rJ * rJ);
    return 1.0 / (1.0 - 0.25 * rJ * rJ * omega_n);
}

// nsweeps full sweeps; colour half-sweep number m (0, 1, 2, ...: red, black, red, ...) uses omega_{m + start_n}
// (Press et al. Eq. 20.5.30 as cited at PAPER.md:86: omega changes every half-sweep; start_n = 1 skips omega_0 = 1,
// the variant the paper uses).  omegas (nullable, 2 nsweeps) receives the sequence used.
void rbsor_cheby(const Grid& g, double* phi, const double* rhs, double rJ, int nsweeps, int start_n, bool use_ghost,
                 double* omegas) {
    double om = 1.0;
    for (int n = 0; n <= start_n; ++n) om = cheby_next(rJ, n, om);  // omega_{start_n}
    for (int m = 0; m < 2 * nsweeps; ++m) {
        if (omegas) omegas[m] = om;
        rbsor_half(g, phi, rhs, om, m & 1, use_ghost);
        om = cheby_next(rJ, m + start_n + 1, om);
    }
}

// Eq. 7: local Jacobi radius of the spherical (or nonuniform Cartesian) grid at (i, j); independent of k for uniform phi.
double local_jacobi_radius(const Grid& g, int i, int j) {
    if (g.coord != SPHERICAL) return jacobi_radius(g);
    const double dr = g.edge[0][i + 1] - g.edge[0][i], dth = g.edge[1][j + 1] - g.edge[1][j];
    const double dph = g.edge[2][1] - g.edge[2][0];
    const double r = g.ctr[0][i], st = std::sin(g.ctr[1][j]);
    const double a = 1.0 / (dr * dr), b = 1.0 / ((r * dth) * (r * dth)), c = 1.0 / ((r * st * dph) * (r * st * dph));
    return (std::cos(M_PI / g.n[0]) * a + std::cos(M_PI / g.n[1]) * b + std::cos(M_PI / g.n[2]) * c) / (a + b + c);
}

// Red-black SOR with the position-dependent sequence omega_n(i,j) of Eq. 6 driven by the local r_J of Eq. 7
// ("a variant in which the values of omega_n are not uniform, but depend on position on the grid"),
// starting from n = start_n; advanced after every colour half-sweep.
void rbsor_local(const Grid& g, double* phi, const double* rhs, int nsweeps, int start_n, bool use_ghost) {
    const int n0 = g.n[0], n1 = g.n[1];
    std::vector<double> rj((size_t)n0 * n1), om((size_t)n0 * n1, 1.0);
    for (int j = 0; j < n1; ++j)
        for (int i = 0; i < n0; ++i) {
            rj[(size_t)j * n0 + i] = local_jacobi_radius(g, i, j);
            for (int n = 0; n <= start_n; ++n) om[(size_t)j * n0 + i] = cheby_next(rj[(size_t)j * n0 + i], n, om[(size_t)j * n0 + i]);
        }
    for (int m = 0; m < 2 * nsweeps; ++m) {
        const int colour = m & 1;
#pragma omp parallel for schedule(static)
        for (int k = 0; k < g.n[2]; ++k)
            for (int j = 0; j < n1; ++j)
                for (int i = 0; i < n0; ++i) {
                    if (((i + j + k) & 1) != colour) continue;
                    const size_t p = g.idx(i, j, k);
                    const double s = offsum(g, phi, i, j, k, use_ghost);
                    const double d = diag<double>(g, i, j, k);
                    const double gs = (s - rhs[p]) / d;
                    phi[p] = fma_(om[(size_t)j * n0 + i], gs - phi[p], phi[p]);
                }
        for (size_t q = 0; q < om.size(); ++q) om[q] = cheby_next(rj[q], m + start_n + 1, om[q]);
    }
}

}  // namespace orc
