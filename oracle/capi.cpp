// ORACLE — TEST INFRASTRUCTURE ONLY (see grid.hpp).  C entry points for the ctypes harness (oracle/pyoracle.py).
// All pointers are host pointers; arrays are contiguous, axis 0 fastest.
#include <cstring>
#ifdef _OPENMP
#include <omp.h>
#endif

#include "solvers.hpp"

using namespace orc;

extern "C" {

void* orc_create(const int* shape, const double* spacing, const double* origin, const double* const* edges,
                 int coord, int order, const int* bc) {
    Grid* g = new Grid;
    for (int a = 0; a < 3; ++a) {
        g->n[a] = shape[a];
        g->h[a] = spacing ? spacing[a] : 1.0;
        g->origin[a] = origin ? origin[a] : 0.0;
    }
    g->coord = coord;
    g->order = order;
    g->R = (order == 6) ? 3 : 1;
    for (int f = 0; f < 6; ++f) g->bc[f] = bc[f];
    for (int f = 0; f < 6; ++f)
        if (g->bc[f] == BC_DIRICHLET_GHOST) g->ghost[f].assign(g->face_len(f), 0.0);
    if (coord == SPHERICAL) {
        for (int a = 0; a < 3; ++a) g->edge[a].assign(edges[a], edges[a] + shape[a] + 1);
        setup_spherical(*g);
    }
    return g;
}

void orc_destroy(void* h) { delete (Grid*)h; }

void orc_set_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int orc_get_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_gamma(void* h, double gamma) { ((Grid*)h)->gamma = gamma; }

long orc_face_len(void* h, int f) { return (long)((Grid*)h)->face_len(f); }

void orc_set_ghost_face(void* h, int f, const double* v) {
    Grid* g = (Grid*)h;
    g->ghost[f].assign(v, v + g->face_len(f));
}
void orc_get_ghost_face(void* h, int f, double* v) {
    Grid* g = (Grid*)h;
    if (g->ghost[f].empty()) return;
    std::memcpy(v, g->ghost[f].data(), g->ghost[f].size() * sizeof(double));
}

void orc_apply(void* h, const double* phi, double* out, int use_ghost) { apply(*(Grid*)h, phi, out, use_ghost != 0); }
void orc_apply_f32(void* h, const float* phi, float* out, int use_ghost) { apply(*(Grid*)h, phi, out, use_ghost != 0); }
void orc_diag(void* h, double* out) {
    Grid* g = (Grid*)h;
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i) out[g->idx(i, j, k)] = diag<double>(*g, i, j, k);
}
double orc_residual_norm(void* h, const double* phi, const double* rhs) {
    return residual_norm(*(Grid*)h, phi, rhs, true);
}

void orc_rbsor_half(void* h, double* phi, const double* rhs, double omega, int colour) {
    rbsor_half(*(Grid*)h, phi, rhs, omega, colour, true);
}
void orc_rbsor(void* h, double* phi, const double* rhs, double omega, int nsweeps, double* resnorm) {
    rbsor(*(Grid*)h, phi, rhs, omega, nsweeps, true);
    if (resnorm) *resnorm = residual_norm(*(Grid*)h, phi, rhs, true);
}
void orc_rbsor_f32(void* h, float* phi, const float* rhs, float omega, int nsweeps) {
    rbsor(*(Grid*)h, phi, rhs, omega, nsweeps, true);
}

int orc_cg(void* h, double* phi, const double* rhs, double rtol, int max_iter, int fixed_iters, int* iters,
           double* relres, double* history) {
    return cg(*(Grid*)h, phi, rhs, rtol, max_iter, fixed_iters, iters, relres, history);
}
int orc_bicgstab(void* h, double* phi, const double* rhs, double rtol, int max_iter, int fixed_iters, int jacobi,
                 int* iters, double* relres, double* history) {
    return bicgstab(*(Grid*)h, phi, rhs, rtol, max_iter, fixed_iters, jacobi, iters, relres, history);
}
int orc_pcg(void* h, double* phi, const double* rhs, double rtol, int max_iter, int fixed_iters, int* iters,
            double* relres, double* history) {
    return pcg(*(Grid*)h, phi, rhs, rtol, max_iter, fixed_iters, iters, relres, history);
}
void orc_gs_precond(void* h, const double* v, double* z, int sign, int symmetric) {
    gs_precond(*(Grid*)h, v, z, sign, symmetric != 0);
}
double orc_jacobi_radius(void* h) { return jacobi_radius(*(Grid*)h); }
double orc_local_jacobi_radius(void* h, int i, int j) { return local_jacobi_radius(*(Grid*)h, i, j); }
void orc_rbsor_cheby(void* h, double* phi, const double* rhs, double rJ, int nsweeps, int start_n, double* omegas) {
    rbsor_cheby(*(Grid*)h, phi, rhs, rJ, nsweeps, start_n, true, omegas);
}
void orc_rbsor_local(void* h, double* phi, const double* rhs, int nsweeps, int start_n) {
    rbsor_local(*(Grid*)h, phi, rhs, nsweeps, start_n, true);
}
void orc_multipole_bc2(void* h, const double* rho, double G, int lmax, double* moments, double* inner_moments) {
    multipole_bc(*(Grid*)h, rho, G, lmax, moments, inner_moments);
}
void orc_multipole_inner_moments(void* h, const double* rho, int lmax, double* qbar) {
    multipole_inner_moments(*(Grid*)h, rho, lmax, qbar);
}
double orc_multipole_inner_potential(const double* qbar, int lmax, double G, double x, double y, double z) {
    return multipole_inner_potential(qbar, lmax, G, x, y, z);
}
void orc_set_bicgstab_restart_eps(double eps) { set_bicgstab_restart_eps(eps); }
void orc_bicgstab_stats(int* restarts, int* confirm_failed) { bicgstab_stats(restarts, confirm_failed); }
int orc_vcycle(void* h, double* phi, const double* rhs, int nu1, int nu2, int coarsest_n, int coarsest_sweeps,
               int precision, int restriction, int ncycles, double* resnorms) {
    return vcycle(*(Grid*)h, phi, rhs, nu1, nu2, coarsest_n, coarsest_sweeps, precision, restriction, ncycles,
                  resnorms);
}

// transfer operators between this grid (fine) and its first coarse level, for the pins
void orc_restrict(void* h, const double* r, double* fc, int restriction) {
    Grid* g = (Grid*)h;
    Grid c = coarsen(*g, 1);
    restrict_fw(*g, c, r, fc, restriction);
}
void orc_prolong_add(void* h, const double* ec, double* phi, double coarse_gamma) {
    Grid* g = (Grid*)h;
    Grid c = coarsen(*g, 1);
    c.gamma = coarse_gamma;
    prolong_add(*g, c, ec, phi);
}

void orc_spai_smooth(void* h, double* phi, const double* rhs, const double* spai, int nsteps, int order) {
    spai_smooth(*(Grid*)h, phi, rhs, spai, nsteps, order);
}
int orc_mgv_vcycle(void* h, double* phi, const double* rhs, int nu1, int nu2, int coarsest_n, const double* spai,
                   double cg_rtol, int storage_f32, int ncycles, double* resnorms, int order) {
    return mgv_vcycle(*(Grid*)h, phi, rhs, nu1, nu2, coarsest_n, spai, cg_rtol, storage_f32, ncycles, resnorms, order);
}
int orc_compact_apply(void* h, int order, const double* v, double* out) { return compact_apply(*(Grid*)h, order, v, out); }
int orc_compact_rhs(const int* n, int order, const double* f_ext, double* out) { return compact_rhs(n, order, f_ext, out); }
int orc_mgv_galerkin_stencil(void* h, int level, int I, int J, int K, double* out27, int order) {
    return mgv_galerkin_stencil(*(Grid*)h, level, I, J, K, out27, order);
}
void orc_mgv_restrict(void* h, const double* r, double* bc) { mgv_restrict(*(Grid*)h, r, bc); }
void orc_mgv_prolong_add(void* h, const double* ec, double* x) { mgv_prolong_add(*(Grid*)h, ec, x); }

void orc_multipole_moments(void* h, const double* rho, int lmax, double* q) {
    multipole_moments(*(Grid*)h, rho, lmax, q);
}
double orc_multipole_potential(const double* q, int lmax, double G, double x, double y, double z) {
    return multipole_potential(q, lmax, G, x, y, z);
}
void orc_multipole_bc(void* h, const double* rho, double G, int lmax, double* moments) {
    multipole_bc(*(Grid*)h, rho, G, lmax, moments);
}

// spherical helpers for the harness: centres and the outer ghost radius
void orc_centres(void* h, int axis, double* out) {
    Grid* g = (Grid*)h;
    if (g->coord == SPHERICAL)
        std::memcpy(out, g->ctr[axis].data(), g->ctr[axis].size() * sizeof(double));
    else
        for (int i = 0; i < g->n[axis]; ++i) out[i] = g->coordinate(axis, i);
}
double orc_r_ghost_out(void* h) { return ((Grid*)h)->r_ghost_out; }

}  // extern "C"
