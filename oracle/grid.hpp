// ORACLE — TEST INFRASTRUCTURE ONLY.  Plain, slow CPU statement of what the hot path computes.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
// It shares no code with the CUDA path (paper_2605_03563_b200/csrc) and neither includes the other.
//
// grid.hpp: the discrete operator as a matrix row (off-diagonal sum, diagonal) on a 3-D structured grid.
//   Cartesian 7-point 2nd-order Laplacian          PAPER.md:43-45 (Eq. 1), 67-69 (Eq. 4 uses the same coefficients)
//   Cartesian 19-point radius-3 "naive" 6th-order  PAPER.md:172 ("naive stencils ... radii of two and three")
//   Spherical (r,theta,phi) direct finite differences of Eq. (2), nonsymmetric (row-scaled) PAPER.md:47-49, 105
//   ghost zones hold the Dirichlet boundary potential
// Readings the paper leaves open are those of SURVEY.md §8(c) C0/C1/C5/C7 and are restated in DESIGN.md.
// Pins: tests/test_oracle_*.py.  Parity unpinned: only the converged config-5 solution's absolute accuracy (krylov.cpp).
#pragma once
#include <cmath>
#include <cstddef>
#include <vector>

namespace orc {

enum { CARTESIAN = 0, SPHERICAL = 1 };
enum { BC_DIRICHLET_GHOST = 0, BC_PERIODIC = 1, BC_NEUMANN0 = 2, BC_AXIS = 3 };

inline double fma_(double a, double b, double c) { return std::fma(a, b, c); }
inline float fma_(float a, float b, float c) { return std::fmaf(a, b, c); }

// Unknowns: n[0] x n[1] x n[2] points, index (i,j,k), i fastest.
// Faces: 0 = axis0 low, 1 = axis0 high, 2 = axis1 low, 3 = axis1 high, 4 = axis2 low, 5 = axis2 high.
struct Grid {
    int n[3] = {0, 0, 0};
    int coord = CARTESIAN;
    int order = 2;   // 2 -> radius 1, 6 -> radius 3
    int R = 1;       // stencil radius = number of ghost layers on Dirichlet faces
    int bc[6] = {0, 0, 0, 0, 0, 0};
    double h[3] = {1, 1, 1};       // Cartesian spacing
    double origin[3] = {0, 0, 0};  // Cartesian coordinate of unknown (0,0,0)
    // Multigrid coarse-level closure (reading C7): on a Dirichlet face the homogeneous ghost value is
    // -gamma * (adjacent interior value); in matrix form the diagonal grows by gamma*c on every such face touched.
    double gamma = 0.0;
    // Ghost values on Dirichlet faces, R layers each.  Face on axis a, layer l (distance l+1 from the domain):
    //   index = (l * n[a2] + q2) * n[a1] + q1, (a1,a2) = the two other axes in increasing order, q1 fastest.
    std::vector<double> ghost[6];
    // Spherical: edges (n+1 per axis) and the derived 1-D coefficient arrays of DESIGN.md reading C5.
    std::vector<double> edge[3], ctr[3];
    std::vector<double> ar_m, ar_p, ir2, at_m, at_p, cp, dr, dt;
    double r_ghost_out = 0.0;  // centre radius of the outer ghost shell

    size_t size() const { return (size_t)n[0] * n[1] * n[2]; }
    size_t idx(int i, int j, int k) const { return ((size_t)k * n[1] + j) * n[0] + i; }
    size_t face_len(int f) const {
        int a = f / 2, a1 = (a == 0) ? 1 : 0, a2 = (a == 2) ? 1 : 2;
        return (size_t)R * n[a1] * n[a2];
    }
    double ghost_at(int f, int layer, int q1, int q2) const {
        int a = f / 2, a1 = (a == 0) ? 1 : 0, a2 = (a == 2) ? 1 : 2;
        (void)a2;
        return ghost[f][((size_t)layer * n[a2] + q2) * n[a1] + q1];
    }
    double coordinate(int a, int i) const {  // Cartesian point coordinate along axis a (i may be a ghost index)
        return origin[a] + i * h[a];
    }
};

// Value of the neighbour at offset s (may be out of range) along axis a of point (i,j,k).
//   in range          -> v[...]
//   periodic face     -> wrapped value
//   Dirichlet face    -> ghost value if use_ghost (inhomogeneous operator), else 0 (search directions, error equations)
//   Neumann0 / axis   -> 0 here: their effect lives in the diagonal / in zero coefficients (see diag())
template <typename T>
inline T nbr(const Grid& g, const T* v, int i, int j, int k, int a, int s, bool use_ghost) {
    int q[3] = {i, j, k};
    int p = q[a] + s;
    if (p >= 0 && p < g.n[a]) {
        q[a] = p;
        return v[g.idx(q[0], q[1], q[2])];
    }
    int f = 2 * a + (p < 0 ? 0 : 1);
    if (g.bc[f] == BC_PERIODIC) {
        q[a] = ((p % g.n[a]) + g.n[a]) % g.n[a];
        return v[g.idx(q[0], q[1], q[2])];
    }
    if (g.bc[f] == BC_DIRICHLET_GHOST && use_ghost && g.gamma == 0.0 && !g.ghost[f].empty()) {
        int layer = (p < 0) ? (-1 - p) : (p - g.n[a]);
        int a1 = (a == 0) ? 1 : 0, a2 = (a == 2) ? 1 : 2;
        return (T)g.ghost_at(f, layer, q[a1], q[a2]);
    }
    return (T)0;
}

static const double W6[4] = {-49.0 / 18.0, 3.0 / 2.0, -3.0 / 20.0, 1.0 / 90.0};  // 6th-order second difference

// Diagonal entry d of the row, defined so that (L v)_ijk = offsum - d * v_ijk.
template <typename T>
inline T diag(const Grid& g, int i, int j, int k) {
    if (g.coord == SPHERICAL) {
        (void)k;
        return fma_((T)g.ir2[i], (T)g.dt[j], (T)g.dr[i]);
    }
    T c[3] = {(T)(1.0 / (g.h[0] * g.h[0])), (T)(1.0 / (g.h[1] * g.h[1])), (T)(1.0 / (g.h[2] * g.h[2]))};
    if (g.order == 6) return (T)(-W6[0]) * ((c[0] + c[1]) + c[2]);
    T d = (T)2 * ((c[0] + c[1]) + c[2]);
    int q[3] = {i, j, k};
    for (int a = 0; a < 3; ++a) {
        if (q[a] == 0) {
            if (g.bc[2 * a] == BC_DIRICHLET_GHOST && g.gamma != 0.0) d = fma_((T)g.gamma, c[a], d);
            if (g.bc[2 * a] == BC_NEUMANN0) d -= c[a];
        }
        if (q[a] == g.n[a] - 1) {
            if (g.bc[2 * a + 1] == BC_DIRICHLET_GHOST && g.gamma != 0.0) d = fma_((T)g.gamma, c[a], d);
            if (g.bc[2 * a + 1] == BC_NEUMANN0) d -= c[a];
        }
    }
    return d;
}

// Off-diagonal part of the row: sum over neighbours of coefficient * value, in the canonical order of DESIGN.md.
template <typename T>
inline T offsum(const Grid& g, const T* v, int i, int j, int k, bool use_ghost) {
    if (g.coord == SPHERICAL) {
        T vrm = nbr(g, v, i, j, k, 0, -1, use_ghost), vrp = nbr(g, v, i, j, k, 0, +1, use_ghost);
        T vtm = nbr(g, v, i, j, k, 1, -1, use_ghost), vtp = nbr(g, v, i, j, k, 1, +1, use_ghost);
        T vpm = nbr(g, v, i, j, k, 2, -1, use_ghost), vpp = nbr(g, v, i, j, k, 2, +1, use_ghost);
        T s = (T)g.ar_m[i] * vrm;
        s = fma_((T)g.ar_p[i], vrp, s);
        T t = (T)g.at_m[j] * vtm;
        t = fma_((T)g.at_p[j], vtp, t);
        t = fma_((T)g.cp[j], vpm + vpp, t);
        return fma_((T)g.ir2[i], t, s);
    }
    T c[3] = {(T)(1.0 / (g.h[0] * g.h[0])), (T)(1.0 / (g.h[1] * g.h[1])), (T)(1.0 / (g.h[2] * g.h[2]))};
    if (g.order == 6) {
        T t[3];
        for (int a = 0; a < 3; ++a) {
            T p1 = nbr(g, v, i, j, k, a, -1, use_ghost) + nbr(g, v, i, j, k, a, +1, use_ghost);
            T p2 = nbr(g, v, i, j, k, a, -2, use_ghost) + nbr(g, v, i, j, k, a, +2, use_ghost);
            T p3 = nbr(g, v, i, j, k, a, -3, use_ghost) + nbr(g, v, i, j, k, a, +3, use_ghost);
            T u = (T)W6[1] * p1;
            u = fma_((T)W6[2], p2, u);
            u = fma_((T)W6[3], p3, u);
            t[a] = u;
        }
        T s = t[0] * c[0];
        s = fma_(t[1], c[1], s);
        s = fma_(t[2], c[2], s);
        return s;
    }
    T px = nbr(g, v, i, j, k, 0, -1, use_ghost) + nbr(g, v, i, j, k, 0, +1, use_ghost);
    T py = nbr(g, v, i, j, k, 1, -1, use_ghost) + nbr(g, v, i, j, k, 1, +1, use_ghost);
    T pz = nbr(g, v, i, j, k, 2, -1, use_ghost) + nbr(g, v, i, j, k, 2, +1, use_ghost);
    T s = px * c[0];
    s = fma_(py, c[1], s);
    s = fma_(pz, c[2], s);
    return s;
}

// (L v)_ijk = offsum - d v_ijk (single rounding of the last step).
template <typename T>
inline T row_apply(const Grid& g, const T* v, int i, int j, int k, bool use_ghost) {
    return fma_(-diag<T>(g, i, j, k), v[g.idx(i, j, k)], offsum(g, v, i, j, k, use_ghost));
}

// out = L v over the whole grid.
template <typename T>
void apply(const Grid& g, const T* v, T* out, bool use_ghost);

// ||rhs - L v||_2 (long double accumulation, plane partial sums added in k order).
template <typename T>
double residual_norm(const Grid& g, const T* v, const T* rhs, bool use_ghost);

// long-double dot product, plane partial sums added in k order (deterministic, thread-count independent).
double dot(const Grid& g, const double* a, const double* b);
double sum(const Grid& g, const double* a);

void setup_spherical(Grid& g);  // fills ctr[], coefficient arrays from edge[] (reading C5)

}  // namespace orc
