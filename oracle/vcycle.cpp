// ORACLE — TEST INFRASTRUCTURE ONLY (see grid.hpp).
// Geometric multigrid V-cycle.  PAPER.md:125-136 (Eq. 11-12: pre-smooth, coarse-grid correction, post-smooth,
// recursively; coarsest level solved), 138-142 (Eq. 13: full weighting; P = c R^T preserving constants), 205
// (mixed precision).  BASELINE.json config 3 fixes the variant: cell-centred 2:1 coarsening 256^3 -> 8^3,
// red-black Gauss-Seidel smoothing (nu1, nu2), full-weighting restriction, trilinear prolongation, coarsest
// level by SOR sweeps, fp64 or "fp32 smoothing, fp64 residual/correction".  Readings: DESIGN.md C7.
#include <cmath>
#include <vector>

#include "solvers.hpp"

namespace orc {

// Level l >= 1 of the hierarchy below `fine` (level l-1): half the cells, twice the spacing, cell-centred, 7-point
// rediscretisation.  Its homogeneous Dirichlet condition sits at the finest grid's ghost centres (h_0/2 outside
// the face), which in terms of its own ghost cell reads ghost = -gamma_l * adjacent, gamma_l = (2^l-1)/(2^l+1).
Grid coarsen(const Grid& fine, int level_of_coarse) {
    Grid c;
    c.coord = CARTESIAN;
    c.order = 2;
    c.R = 1;
    for (int a = 0; a < 3; ++a) {
        c.n[a] = fine.n[a] / 2;
        c.h[a] = 2.0 * fine.h[a];
        c.origin[a] = fine.origin[a] + 0.5 * fine.h[a];  // centre of the union of fine cells 0 and 1
    }
    for (int f = 0; f < 6; ++f) c.bc[f] = fine.bc[f];
    const double s = std::ldexp(1.0, level_of_coarse);
    c.gamma = (s - 1.0) / (s + 1.0);
    return c;
}

// f_c = R r.  restriction 0: 1-D weights (1/8)[1 3 3 1] on fine cells 2I-1..2I+2, tensor product, out-of-range
// residual = 0 (the transpose of trilinear interpolation divided by 8: P = 8 R^T).
// restriction 1: mean of the 8 children.
template <typename T>
void restrict_fw(const Grid& fine, const Grid& coarse, const T* r, T* fc, int restriction) {
    static const double W[4] = {0.125, 0.375, 0.375, 0.125};
#pragma omp parallel for schedule(static)
    for (int K = 0; K < coarse.n[2]; ++K)
        for (int J = 0; J < coarse.n[1]; ++J)
            for (int I = 0; I < coarse.n[0]; ++I) {
                T acc = 0;
                if (restriction == 1) {
                    for (int c = 0; c < 2; ++c)
                        for (int b = 0; b < 2; ++b)
                            for (int a = 0; a < 2; ++a) acc += r[fine.idx(2 * I + a, 2 * J + b, 2 * K + c)];
                    acc *= (T)0.125;
                } else {
                    for (int c = 0; c < 4; ++c)
                        for (int b = 0; b < 4; ++b)
                            for (int a = 0; a < 4; ++a) {
                                int i = 2 * I - 1 + a, j = 2 * J - 1 + b, k = 2 * K - 1 + c;
                                if (i < 0 || i >= fine.n[0] || j < 0 || j >= fine.n[1] || k < 0 || k >= fine.n[2])
                                    continue;
                                acc += (T)(W[a] * W[b] * W[c]) * r[fine.idx(i, j, k)];
                            }
                }
                fc[coarse.idx(I, J, K)] = acc;
            }
}
template void restrict_fw<double>(const Grid&, const Grid&, const double*, double*, int);
template void restrict_fw<float>(const Grid&, const Grid&, const float*, float*, int);

// Coarse value with the level's ghost closure applied axis by axis: out-of-range index -> -gamma * clamped value.
template <typename T>
static inline T coarse_val(const Grid& c, const T* e, int I, int J, int K) {
    T sgn = 1;
    int q[3] = {I, J, K};
    for (int a = 0; a < 3; ++a) {
        if (q[a] < 0) {
            q[a] = 0;
            sgn *= (T)(-c.gamma);
        } else if (q[a] >= c.n[a]) {
            q[a] = c.n[a] - 1;
            sgn *= (T)(-c.gamma);
        }
    }
    return sgn * e[c.idx(q[0], q[1], q[2])];
}

// phi += P e_c, P = trilinear interpolation for cell-centred 2:1 refinement: per axis fine 2I <- 3/4 e_I + 1/4
// e_{I-1}, fine 2I+1 <- 3/4 e_I + 1/4 e_{I+1}; evaluated as a tensor product, x then y then z.
template <typename T>
void prolong_add(const Grid& fine, const Grid& coarse, const T* ec, T* phi) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < fine.n[2]; ++k)
        for (int j = 0; j < fine.n[1]; ++j)
            for (int i = 0; i < fine.n[0]; ++i) {
                int I = i >> 1, J = j >> 1, K = k >> 1;
                int In = I + ((i & 1) ? 1 : -1), Jn = J + ((j & 1) ? 1 : -1), Kn = K + ((k & 1) ? 1 : -1);
                T ey[2];
                for (int c = 0; c < 2; ++c) {
                    int KK = c ? Kn : K;
                    T ex[2];
                    for (int b = 0; b < 2; ++b) {
                        int JJ = b ? Jn : J;
                        T near = coarse_val(coarse, ec, I, JJ, KK), far = coarse_val(coarse, ec, In, JJ, KK);
                        ex[b] = fma_((T)0.75, near, (T)0.25 * far);
                    }
                    ey[c] = fma_((T)0.75, ex[0], (T)0.25 * ex[1]);
                }
                T v = fma_((T)0.75, ey[0], (T)0.25 * ey[1]);
                phi[fine.idx(i, j, k)] += v;
            }
}
template void prolong_add<double>(const Grid&, const Grid&, const double*, double*);
template void prolong_add<float>(const Grid&, const Grid&, const float*, float*);

template <typename T>
static void vcycle_rec(const std::vector<Grid>& lv, size_t l, T* phi, const T* rhs, bool use_ghost, int nu1, int nu2,
                       int coarsest_sweeps, int restriction) {
    const Grid& g = lv[l];
    if (l + 1 == lv.size()) {
        // coarsest level: SOR sweeps with the omega_opt of Eq. 3-4 for n unknowns per axis
        const double om = 2.0 / (1.0 + std::sin(M_PI / (g.n[0] + 1)));
        rbsor(g, phi, rhs, (T)om, coarsest_sweeps, use_ghost);
        return;
    }
    rbsor(g, phi, rhs, (T)1, nu1, use_ghost);  // pre-smoothing: red-black Gauss-Seidel
    const Grid& c = lv[l + 1];
    std::vector<T> r(g.size()), fc(c.size()), ec(c.size(), (T)0);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
        for (int j = 0; j < g.n[1]; ++j)
            for (int i = 0; i < g.n[0]; ++i) r[g.idx(i, j, k)] = rhs[g.idx(i, j, k)] - row_apply(g, phi, i, j, k, use_ghost);
    restrict_fw(g, c, r.data(), fc.data(), restriction);
    vcycle_rec(lv, l + 1, ec.data(), fc.data(), false, nu1, nu2, coarsest_sweeps, restriction);
    prolong_add(g, c, ec.data(), phi);
    rbsor(g, phi, rhs, (T)1, nu2, use_ghost);  // post-smoothing
}

int vcycle(const Grid& g, double* phi, const double* rhs, int nu1, int nu2, int coarsest_n, int coarsest_sweeps,
           int precision, int restriction, int ncycles, double* resnorms) {
    std::vector<Grid> lv;
    lv.push_back(g);
    int level = 0;
    while (lv.back().n[0] > coarsest_n && lv.back().n[0] % 2 == 0 && lv.back().n[1] % 2 == 0 &&
           lv.back().n[2] % 2 == 0) {
        ++level;
        lv.push_back(coarsen(lv.back(), level));
    }
    if (resnorms) resnorms[0] = residual_norm(g, phi, rhs, true);
    const size_t n = g.size();
    for (int c = 0; c < ncycles; ++c) {
        if (precision == 0) {
            vcycle_rec<double>(lv, 0, phi, rhs, true, nu1, nu2, coarsest_sweeps, restriction);
        } else {
            // iterative-refinement form: r = rhs - L phi in fp64; one fp32 V-cycle on L e = r from e = 0 with
            // homogeneous ghosts on every level (gamma_0 = 0); phi += e in fp64.
            std::vector<double> r(n);
            apply(g, phi, r.data(), true);
            std::vector<float> r32(n), e32(n, 0.0f);
            for (size_t m = 0; m < n; ++m) r32[m] = (float)(rhs[m] - r[m]);
            vcycle_rec<float>(lv, 0, e32.data(), r32.data(), false, nu1, nu2, coarsest_sweeps, restriction);
            for (size_t m = 0; m < n; ++m) phi[m] += (double)e32[m];
        }
        if (resnorms) resnorms[c + 1] = residual_norm(g, phi, rhs, true);
    }
    return ST_OK;
}

}  // namespace orc
