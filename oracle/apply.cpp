// ORACLE — TEST INFRASTRUCTURE ONLY (see grid.hpp).
// Stencil apply out = L_h phi, residual norm, dot products, spherical coefficient set-up.
//   PAPER.md:43-49 (Eq. 1, 2), 55 ("residual (difference between the left and right hand side ...)"), 105.
#include "grid.hpp"

namespace orc {

template <typename T>
void apply(const Grid& g, const T* v, T* out, bool use_ghost) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
        for (int j = 0; j < g.n[1]; ++j)
            for (int i = 0; i < g.n[0]; ++i) out[g.idx(i, j, k)] = row_apply(g, v, i, j, k, use_ghost);
}
template void apply<double>(const Grid&, const double*, double*, bool);
template void apply<float>(const Grid&, const float*, float*, bool);

template <typename T>
double residual_norm(const Grid& g, const T* v, const T* rhs, bool use_ghost) {
    std::vector<long double> part(g.n[2]);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k) {
        long double s = 0;
        for (int j = 0; j < g.n[1]; ++j)
            for (int i = 0; i < g.n[0]; ++i) {
                T r = rhs[g.idx(i, j, k)] - row_apply(g, v, i, j, k, use_ghost);
                s += (long double)r * (long double)r;
            }
        part[k] = s;
    }
    long double tot = 0;
    for (int k = 0; k < g.n[2]; ++k) tot += part[k];
    return (double)sqrtl(tot);
}
template double residual_norm<double>(const Grid&, const double*, const double*, bool);
template double residual_norm<float>(const Grid&, const float*, const float*, bool);

double dot(const Grid& g, const double* a, const double* b) {
    std::vector<long double> part(g.n[2]);
    size_t plane = (size_t)g.n[0] * g.n[1];
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k) {
        long double s = 0;
        for (size_t q = 0; q < plane; ++q) s += (long double)a[k * plane + q] * (long double)b[k * plane + q];
        part[k] = s;
    }
    long double tot = 0;
    for (int k = 0; k < g.n[2]; ++k) tot += part[k];
    return (double)tot;
}

double sum(const Grid& g, const double* a) {
    std::vector<long double> part(g.n[2]);
    size_t plane = (size_t)g.n[0] * g.n[1];
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k) {
        long double s = 0;
        for (size_t q = 0; q < plane; ++q) s += (long double)a[k * plane + q];
        part[k] = s;
    }
    long double tot = 0;
    for (int k = 0; k < g.n[2]; ++k) tot += part[k];
    return (double)tot;
}

// Spherical grid of DESIGN.md reading C5 (Eq. 2; 397-405 for the log grid with geometric-mean
// centres).  Axis 0 = r (edges given), axis 1 = theta, axis 2 = phi.
//   (L Phi)_ijk = [ r^2_{i+1/2}(Phi_{i+1}-Phi_i)/(r_{i+1}-r_i) - r^2_{i-1/2}(Phi_i-Phi_{i-1})/(r_i-r_{i-1}) ]/(r_i^2 dr_i)
//               + [ sin th_{j+1/2}(Phi_{j+1}-Phi_j) - sin th_{j-1/2}(Phi_j-Phi_{j-1}) ]/(r_i^2 sin th_j dth^2)
//               + (Phi_{k+1} - 2 Phi_k + Phi_{k-1})/(r_i^2 sin^2 th_j dph^2)
void setup_spherical(Grid& g) {
    const int nr = g.n[0], nt = g.n[1], np = g.n[2];
    const std::vector<double>&re = g.edge[0], &te = g.edge[1], &pe = g.edge[2];
    g.ctr[0].resize(nr);
    g.ctr[1].resize(nt);
    g.ctr[2].resize(np);
    for (int i = 0; i < nr; ++i) g.ctr[0][i] = std::sqrt(re[i] * re[i + 1]);  // geometric mean
    for (int j = 0; j < nt; ++j) g.ctr[1][j] = 0.5 * (te[j] + te[j + 1]);
    for (int k = 0; k < np; ++k) g.ctr[2][k] = 0.5 * (pe[k] + pe[k + 1]);
    // ghost shell centres continue the geometric progression of the outermost / innermost cell
    g.r_ghost_out = re[nr] * std::sqrt(re[nr] / re[nr - 1]);
    const double r_ghost_in = re[0] * std::sqrt(re[0] / re[1]);
    g.ar_m.assign(nr, 0.0);
    g.ar_p.assign(nr, 0.0);
    g.ir2.assign(nr, 0.0);
    g.dr.assign(nr, 0.0);
    for (int i = 0; i < nr; ++i) {
        double ri = g.ctr[0][i], dri = re[i + 1] - re[i];
        double rm = (i > 0) ? g.ctr[0][i - 1] : r_ghost_in;
        double rp = (i < nr - 1) ? g.ctr[0][i + 1] : g.r_ghost_out;
        g.ir2[i] = 1.0 / (ri * ri);
        g.ar_m[i] = (re[i] * re[i]) / ((ri - rm) * (ri * ri) * dri);
        g.ar_p[i] = (re[i + 1] * re[i + 1]) / ((rp - ri) * (ri * ri) * dri);
        if (i == 0 && g.bc[0] == BC_NEUMANN0) g.ar_m[i] = 0.0;        // zero flux through the inner face
        if (i == nr - 1 && g.bc[1] == BC_NEUMANN0) g.ar_p[i] = 0.0;
        g.dr[i] = g.ar_m[i] + g.ar_p[i];
    }
    g.at_m.assign(nt, 0.0);
    g.at_p.assign(nt, 0.0);
    g.cp.assign(nt, 0.0);
    g.dt.assign(nt, 0.0);
    const double dph = pe[1] - pe[0];
    for (int j = 0; j < nt; ++j) {
        double dth = te[j + 1] - te[j];
        double st = std::sin(g.ctr[1][j]);
        g.at_m[j] = std::sin(te[j]) / (st * dth * dth);
        g.at_p[j] = std::sin(te[j + 1]) / (st * dth * dth);
        if (j == 0 && g.bc[2] == BC_AXIS) g.at_m[j] = 0.0;            // face area vanishes on the axis
        if (j == nt - 1 && g.bc[3] == BC_AXIS) g.at_p[j] = 0.0;
        g.cp[j] = 1.0 / (st * st * dph * dph);
        g.dt[j] = (g.at_m[j] + g.at_p[j]) + 2.0 * g.cp[j];
    }
}

}  // namespace orc
