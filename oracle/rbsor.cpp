// ORACLE — TEST INFRASTRUCTURE ONLY (see grid.hpp).
// Red-black Gauss-Seidel / SOR.  PAPER.md:59-63: "red and black cells of a 3D checkerboard pattern are alternately
// updated"; "Each SOR update amplifies the corresponding Gauss-Seidel update by the factor omega"; omega = 1 is
// Gauss-Seidel.  Reading: red = (i+j+k) even, red first then black; one sweep = both colours.
//   gs  = (sum_nb c_nb phi_nb - rhs) / d        (the value that zeroes the residual of row ijk)
//   phi <- phi + omega (gs - phi)
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

}  // namespace orc
