// ORACLE — TEST INFRASTRUCTURE ONLY (see grid.hpp).
// The paper's own multigrid, step by step in the paper's notation:
//   PAPER.md:125-136  Eq. 11-12   V-cycle: nu1 smoothing steps, coarse-grid correction, nu2 smoothing steps; A_N solved
//   PAPER.md:138-142  Eq. 13      full weighting R = R1d (x) R1d (x) R1d, R1d = 1/4 [1 2 1]; P = c R^T preserving constants
//   PAPER.md:144-150  Eq. 14      Galerkin coarse operators, radius one, 27 coefficients per point, built "by applying
//                                 their definition to a grid point (i,j,k)"
//   PAPER.md:146                  CG on the coarsest level
//   PAPER.md:152                  vertex-centred grids of 2^N k - 1 points per axis (odd sizes)
//   PAPER.md:154-184  Eq. 15-16   SPAI smoother x <- (I - omega M A) x + omega M b, M = h^2 {alpha; beta on the 6 faces;
//                                 gamma on the 12 edges; delta on the 8 corners}, Table 1 (order 2 row)
//   PAPER.md:205                  mixed precision: coarse-level data STORED in fp32, all arithmetic in fp64
// Conventions: A is the paper's SPD matrix, A = -L_h (grid.hpp), b = -rhs; unknowns are the interior vertices of a
// uniform isotropic grid, Dirichlet values on the boundary vertices (the ghost faces of grid.hpp on level 0, zero on the
// error-equation levels).  Readings (C12-C14): c = 8, i.e. P = trilinear interpolation; the Galerkin product
// is taken as R A P (Eq. 14 writes R A R^T: the constant c of P = c R^T is left out there — with R A R^T and P the
// correction would be 8 times too large); the same Table-1 coefficients serve every level with h_l = 2^l h.
// Everything is written for general per-point coefficients (27 per point), as the paper stores them; that the Galerkin
// stencils of this constant-coefficient problem come out identical at every point is a pin, not an assumption.
#include <cmath>
#include <cstring>
#include <vector>

#include "solvers.hpp"

namespace orc {

namespace {

struct VLevel {
    int n[3];
    double h;
    std::vector<double> coef;  // 27 per point: index ((dk+1)*3 + (dj+1))*3 + (di+1)
    size_t size() const { return (size_t)n[0] * n[1] * n[2]; }
    size_t idx(int i, int j, int k) const { return ((size_t)k * n[1] + j) * n[0] + i; }
    bool in(int i, int j, int k) const { return i >= 0 && i < n[0] && j >= 0 && j < n[1] && k >= 0 && k < n[2]; }
};

// (A v)_ijk with zero Dirichlet values outside.
inline double row27(const VLevel& L, const double* v, int i, int j, int k) {
    const double* c = &L.coef[L.idx(i, j, k) * 27];
    double s = 0.0;
    for (int dk = -1; dk <= 1; ++dk)
        for (int dj = -1; dj <= 1; ++dj)
            for (int di = -1; di <= 1; ++di) {
                if (!L.in(i + di, j + dj, k + dk)) continue;
                s += c[((dk + 1) * 3 + (dj + 1)) * 3 + (di + 1)] * v[L.idx(i + di, j + dj, k + dk)];
            }
    return s;
}

// The compact radius-1 discretisations of the Laplacian ("compact stencils of radius unity even for
// fourth order, or, assuming isotropic spacing, even for sixth order (Spotz & Carey 1996)").  PAPER.md prints no
// coefficients; they follow from the Taylor expansion (reading C19).  With the 1-D second difference d_a^2
// (= h^2 D_a^2 + h^4 D_a^4 / 12 + h^6 D_a^6 / 360 + ...) and S1 = sum_a d_a^2, S2 = sum_{a<b} d_a^2 d_b^2,
// S3 = d_x^2 d_y^2 d_z^2:
//   order 2:  L_h = S1 / h^2                        = lap + O(h^2)                                      7 points
//   order 4:  L_h = (S1 + S2/6) / h^2               = lap + h^2/12 lap^2 + O(h^4)                       19 points
//   order 6:  L_h = (S1 + S2/6 + S3/30) / h^2       = lap + h^2/12 lap^2 + h^4/360 [lap^3 + 2 (D_x^2 D_y^2 + D_y^2 D_z^2
//                                                     + D_z^2 D_x^2) lap] + O(h^6)                      27 points
// so that L_h u = (the same operators applied to f) for lap u = f: see compact_rhs below.  In weights per number of
// non-zero offsets (centre, 6 faces, 12 edges, 8 corners) x 1/h^2:
//   order 2: -6, 1, 0, 0      order 4: -4, 1/3, 1/6, 0  (= (-24, 2, 1, 0)/6)
//   order 6: -64/15, 7/15, 1/10, 1/30  (= (-128, 14, 3, 1)/30)
bool compact_weights(int order, double w[4]) {
    if (order == 2) { w[0] = -6.0; w[1] = 1.0; w[2] = 0.0; w[3] = 0.0; return true; }
    if (order == 4) { w[0] = -4.0; w[1] = 1.0 / 3.0; w[2] = 1.0 / 6.0; w[3] = 0.0; return true; }
    if (order == 6) { w[0] = -64.0 / 15.0; w[1] = 7.0 / 15.0; w[2] = 1.0 / 10.0; w[3] = 1.0 / 30.0; return true; }
    return false;
}

// Level 0: A = -L_h as 27 coefficients per point (PAPER.md:43-45 with the sign of PAPER.md:105); order 2: 7-point.
VLevel level0(const Grid& g, int order = 2) {
    VLevel L;
    for (int a = 0; a < 3; ++a) L.n[a] = g.n[a];
    L.h = g.h[0];
    L.coef.assign(L.size() * 27, 0.0);
    const double c = 1.0 / (L.h * L.h);
    double w[4];
    compact_weights(order, w);
    for (size_t p = 0; p < L.size(); ++p) {
        double* q = &L.coef[p * 27];
        for (int dk = -1; dk <= 1; ++dk)
            for (int dj = -1; dj <= 1; ++dj)
                for (int di = -1; di <= 1; ++di)
                    q[((dk + 1) * 3 + (dj + 1)) * 3 + (di + 1)] = -w[(di != 0) + (dj != 0) + (dk != 0)] * c;
    }
    return L;
}

// 1-D full-weighting weights of Eq. 13 and the interpolation weights of P = 8 R^T (per axis 2 R1d^T = [1/2 1 1/2]).
const double R1[3] = {0.25, 0.5, 0.25};
const double P1[3] = {0.5, 1.0, 0.5};

// Coarse point I sits on fine point 2I+1 (zero-based interior indices; fine n = 2 nc + 1).
// Eq. 14 by its definition: column J of A_c is R A P e_J; the 27 coefficients of row I are read off for J = I + offset.
VLevel galerkin(const VLevel& F) {
    VLevel C;
    for (int a = 0; a < 3; ++a) C.n[a] = (F.n[a] - 1) / 2;
    C.h = 2.0 * F.h;
    C.coef.assign(C.size() * 27, 0.0);
#pragma omp parallel for schedule(static)
    for (int K = 0; K < C.n[2]; ++K) {
        std::vector<double> pe(125), ape(27);
        for (int J = 0; J < C.n[1]; ++J)
            for (int I = 0; I < C.n[0]; ++I)
                for (int ok = -1; ok <= 1; ++ok)
                    for (int oj = -1; oj <= 1; ++oj)
                        for (int oi = -1; oi <= 1; ++oi) {
                            const int Ic = I + oi, Jc = J + oj, Kc = K + ok;  // the coarse column
                            if (Ic < 0 || Ic >= C.n[0] || Jc < 0 || Jc >= C.n[1] || Kc < 0 || Kc >= C.n[2]) continue;
                            // P e_J on the fine points within distance 2 of fine(I) = (2I+1, 2J+1, 2K+1)
                            const int fi = 2 * I + 1, fj = 2 * J + 1, fk = 2 * K + 1;
                            const int ci = 2 * Ic + 1, cj = 2 * Jc + 1, ck = 2 * Kc + 1;
                            for (int c = -2; c <= 2; ++c)
                                for (int b = -2; b <= 2; ++b)
                                    for (int a = -2; a <= 2; ++a) {
                                        const int di = fi + a - ci, dj = fj + b - cj, dk = fk + c - ck;
                                        double w = 0.0;
                                        if (di >= -1 && di <= 1 && dj >= -1 && dj <= 1 && dk >= -1 && dk <= 1 &&
                                            F.in(fi + a, fj + b, fk + c))
                                            w = P1[di + 1] * P1[dj + 1] * P1[dk + 1];
                                        pe[((c + 2) * 5 + (b + 2)) * 5 + (a + 2)] = w;
                                    }
                            // A (P e_J) on the 27 fine points around fine(I)
                            for (int c = -1; c <= 1; ++c)
                                for (int b = -1; b <= 1; ++b)
                                    for (int a = -1; a <= 1; ++a) {
                                        double s = 0.0;
                                        if (F.in(fi + a, fj + b, fk + c)) {
                                            const double* q = &F.coef[F.idx(fi + a, fj + b, fk + c) * 27];
                                            for (int dk = -1; dk <= 1; ++dk)
                                                for (int dj = -1; dj <= 1; ++dj)
                                                    for (int di = -1; di <= 1; ++di)
                                                        s += q[((dk + 1) * 3 + (dj + 1)) * 3 + (di + 1)] *
                                                             pe[((c + dk + 2) * 5 + (b + dj + 2)) * 5 + (a + di + 2)];
                                        }
                                        ape[((c + 1) * 3 + (b + 1)) * 3 + (a + 1)] = s;
                                    }
                            // R at coarse point I
                            double s = 0.0;
                            for (int c = -1; c <= 1; ++c)
                                for (int b = -1; b <= 1; ++b)
                                    for (int a = -1; a <= 1; ++a)
                                        s += R1[a + 1] * R1[b + 1] * R1[c + 1] * ape[((c + 1) * 3 + (b + 1)) * 3 + (a + 1)];
                            C.coef[C.idx(I, J, K) * 27 + ((ok + 1) * 3 + (oj + 1)) * 3 + (oi + 1)] = s;
                        }
    }
    return C;
}

// b_c = R r (Eq. 13), r = 0 outside.
void restrict_v(const VLevel& F, const VLevel& C, const double* r, double* bc) {
#pragma omp parallel for schedule(static)
    for (int K = 0; K < C.n[2]; ++K)
        for (int J = 0; J < C.n[1]; ++J)
            for (int I = 0; I < C.n[0]; ++I) {
                double s = 0.0;
                for (int c = -1; c <= 1; ++c)
                    for (int b = -1; b <= 1; ++b)
                        for (int a = -1; a <= 1; ++a)
                            s += R1[a + 1] * R1[b + 1] * R1[c + 1] * r[F.idx(2 * I + 1 + a, 2 * J + 1 + b, 2 * K + 1 + c)];
                bc[C.idx(I, J, K)] = s;
            }
}

// x += P e_c, P = 8 R^T = trilinear interpolation from the coarse vertices (zero on the boundary).
void prolong_v(const VLevel& F, const VLevel& C, const double* ec, double* x) {
    auto cv = [&](int I, int J, int K) -> double {
        return (I < 0 || I >= C.n[0] || J < 0 || J >= C.n[1] || K < 0 || K >= C.n[2]) ? 0.0 : ec[C.idx(I, J, K)];
    };
#pragma omp parallel for schedule(static)
    for (int k = 0; k < F.n[2]; ++k)
        for (int j = 0; j < F.n[1]; ++j)
            for (int i = 0; i < F.n[0]; ++i) {
                // fine index q: odd q sits on coarse (q-1)/2; even q lies half-way between coarse q/2-1 and q/2
                const int I0 = (i - 1) >> 1, J0 = (j - 1) >> 1, K0 = (k - 1) >> 1;  // floor, -1 for q = 0
                const int ni = (i & 1) ? 1 : 2, nj = (j & 1) ? 1 : 2, nk = (k & 1) ? 1 : 2;
                double s = 0.0;
                for (int c = 0; c < nk; ++c)
                    for (int b = 0; b < nj; ++b)
                        for (int a = 0; a < ni; ++a) s += cv(I0 + a, J0 + b, K0 + c);
                x[F.idx(i, j, k)] += s / (double)(ni * nj * nk);
            }
}

// One SPAI step x <- x + omega M (b - A x) (Eq. 15); M of Eq. 16 with h = the level's spacing; r = 0 outside.
// A x is supplied by the caller through `r` (so that level 0 can use the ghost-carrying operator of grid.hpp).
void spai_update(const VLevel& L, double* x, const double* r, const double sp[5]) {
    const double om = sp[0], h2 = L.h * L.h;
    const double w[4] = {sp[1] * h2, sp[2] * h2, sp[3] * h2, sp[4] * h2};  // by number of non-zero offsets: 0,1,2,3
    auto rv = [&](int i, int j, int k) -> double { return L.in(i, j, k) ? r[L.idx(i, j, k)] : 0.0; };
    std::vector<double> xn(L.size());
#pragma omp parallel for schedule(static)
    for (int k = 0; k < L.n[2]; ++k)
        for (int j = 0; j < L.n[1]; ++j)
            for (int i = 0; i < L.n[0]; ++i) {
                double m = 0.0;
                for (int dk = -1; dk <= 1; ++dk)
                    for (int dj = -1; dj <= 1; ++dj)
                        for (int di = -1; di <= 1; ++di)
                            m += w[(di != 0) + (dj != 0) + (dk != 0)] * rv(i + di, j + dj, k + dk);
                xn[L.idx(i, j, k)] = x[L.idx(i, j, k)] + om * m;
            }
    std::memcpy(x, xn.data(), L.size() * sizeof(double));
}

// r = b - A x on a coarse (homogeneous) level.
void residual27(const VLevel& L, const double* x, const double* b, double* r) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < L.n[2]; ++k)
        for (int j = 0; j < L.n[1]; ++j)
            for (int i = 0; i < L.n[0]; ++i) r[L.idx(i, j, k)] = b[L.idx(i, j, k)] - row27(L, x, i, j, k);
}

// r = b - A x on level 0: A = -L_h with the Dirichlet boundary values of the grid's ghost faces, b = -rhs.
void residual0(const Grid& g, const double* x, const double* rhs, double* r) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k)
        for (int j = 0; j < g.n[1]; ++j)
            for (int i = 0; i < g.n[0]; ++i) r[g.idx(i, j, k)] = row_apply(g, x, i, j, k, true) - rhs[g.idx(i, j, k)];
}

long double dotv(const std::vector<double>& a, const std::vector<double>& b) {
    long double s = 0;
    for (size_t m = 0; m < a.size(); ++m) s += (long double)a[m] * (long double)b[m];
    return s;
}

// Coarsest level: CG (Saad Alg. 6.18) from e = 0 to ||r|| <= rtol ||b|| or max_iter iterations.
void cg_coarse(const VLevel& L, double* e, const double* b, double rtol, int max_iter) {
    const size_t n = L.size();
    std::vector<double> r(b, b + n), p(b, b + n), q(n);
    std::memset(e, 0, n * sizeof(double));
    long double rr = dotv(r, r);
    const long double rr0 = rr;
    if (rr0 == 0) return;
    for (int it = 0; it < max_iter; ++it) {
        for (int k = 0; k < L.n[2]; ++k)
            for (int j = 0; j < L.n[1]; ++j)
                for (int i = 0; i < L.n[0]; ++i) q[L.idx(i, j, k)] = row27(L, p.data(), i, j, k);
        const double alpha = (double)(rr / dotv(p, q));
        for (size_t m = 0; m < n; ++m) {
            e[m] += alpha * p[m];
            r[m] -= alpha * q[m];
        }
        const long double rn = dotv(r, r);
        if (sqrtl(rn) <= (long double)rtol * sqrtl(rr0)) break;
        const double beta = (double)(rn / rr);
        rr = rn;
        for (size_t m = 0; m < n; ++m) p[m] = r[m] + beta * p[m];
    }
}

inline void store(std::vector<double>& v, bool f32) {  // coarse-level data live in fp32
    if (!f32) return;
    for (double& x : v) x = (double)(float)x;
}

struct Hier {
    std::vector<VLevel> lv;
    int nu1, nu2, cg_max;
    double sp[5], cg_rtol;
    bool f32;
};

// Error-equation levels l >= 1: A_l e = b_l from e = 0.
void cycle_coarse(const Hier& H, size_t l, std::vector<double>& e, std::vector<double>& b) {
    const VLevel& L = H.lv[l];
    store(b, H.f32);
    if (l + 1 == H.lv.size()) {
        cg_coarse(L, e.data(), b.data(), H.cg_rtol, H.cg_max);
        store(e, H.f32);
        return;
    }
    std::vector<double> r(L.size());
    for (int s = 0; s < H.nu1; ++s) {
        residual27(L, e.data(), b.data(), r.data());
        spai_update(L, e.data(), r.data(), H.sp);
        store(e, H.f32);
    }
    residual27(L, e.data(), b.data(), r.data());
    const VLevel& C = H.lv[l + 1];
    std::vector<double> bc(C.size()), ec(C.size(), 0.0);
    restrict_v(L, C, r.data(), bc.data());
    cycle_coarse(H, l + 1, ec, bc);
    prolong_v(L, C, ec.data(), e.data());
    store(e, H.f32);
    for (int s = 0; s < H.nu2; ++s) {
        residual27(L, e.data(), b.data(), r.data());
        spai_update(L, e.data(), r.data(), H.sp);
        store(e, H.f32);
    }
}

Hier build(const Grid& g, int nu1, int nu2, int coarsest_n, const double spai[5], double cg_rtol, int f32, int order) {
    Hier H;
    H.nu1 = nu1;
    H.nu2 = nu2;
    H.cg_rtol = cg_rtol;
    H.f32 = f32 != 0;
    for (int c = 0; c < 5; ++c) H.sp[c] = spai[c];
    H.lv.push_back(level0(g, order));
    while (true) {
        const VLevel& F = H.lv.back();
        bool ok = true;
        for (int a = 0; a < 3; ++a) ok = ok && (F.n[a] % 2 == 1) && (F.n[a] - 1) / 2 >= coarsest_n;
        if (!ok) break;
        VLevel C = galerkin(F);
        if (H.f32)
            for (double& q : C.coef) q = (double)(float)q;
        H.lv.push_back(std::move(C));
    }
    H.cg_max = 4 * (int)H.lv.back().size() + 10;
    return H;
}

}  // namespace

// x <- x + omega M (rhs-form residual) on the user's grid: nsteps SPAI steps of Eq. 15 for L_h phi = rhs.
// order 2: the grid's 7-point operator with its ghost faces; order 4 / 6: the compact operator with ZERO Dirichlet values
// (boundary data belong in the right-hand side there) and rhs = the transformed right-hand side of compact_rhs.
void residual_level0(const Grid& g, const VLevel& L0, int order, const double* x, const double* rhs, double* r) {
    if (order == 2) {
        residual0(g, x, rhs, r);
        return;
    }
    std::vector<double> b(L0.size());
    for (size_t m = 0; m < b.size(); ++m) b[m] = -rhs[m];
    residual27(L0, x, b.data(), r);
}

void spai_smooth(const Grid& g, double* phi, const double* rhs, const double spai[5], int nsteps, int order) {
    VLevel L0 = level0(g, order);
    std::vector<double> r(L0.size());
    for (int s = 0; s < nsteps; ++s) {
        residual_level0(g, L0, order, phi, rhs, r.data());
        spai_update(L0, phi, r.data(), spai);
    }
}

// out = L_h v, the compact Laplacian of the given order with zero Dirichlet values outside the grid.
int compact_apply(const Grid& g, int order, const double* v, double* out) {
    double w[4];
    if (!compact_weights(order, w) || g.h[0] != g.h[1] || g.h[0] != g.h[2]) return -1;
    VLevel L0 = level0(g, order);
    for (int k = 0; k < g.n[2]; ++k)
        for (int j = 0; j < g.n[1]; ++j)
            for (int i = 0; i < g.n[0]; ++i) out[L0.idx(i, j, k)] = -row27(L0, v, i, j, k);
    return 0;
}

// Right-hand side of the compact schemes: for lap u = f the discrete equation is L_h u = B f with
//   order 4:  B f = f + h^2/12 lap f                                   -> f + S1 f / 12
//   order 6:  B f = f + h^2/12 lap f + h^4/360 [lap^2 f + 2 (f_xxyy + f_yyzz + f_zzxx)]
//                 -> f + S1 f / 12 - (sum_a d_a^4 f) / 240 + S2 f / 90
// (lap f = S1 f / h^2 - h^2/12 sum_a D_a^4 f + O(h^4) moves -1/144 + 1/360 = -1/240 onto the fourth differences, which
// reach two points out; lap^2 f + 2 (...) = sum_a D_a^4 f + 4 sum_{a<b} D_a^2 D_b^2 f.)
// f_ext: f on the grid extended by TWO layers per side, (n0+4)(n1+4)(n2+4) values, x fastest; order 2: a copy.
int compact_rhs(const int n[3], int order, const double* f_ext, double* out) {
    if (order != 2 && order != 4 && order != 6) return -1;
    const int e0 = n[0] + 4, e1 = n[1] + 4;
    auto F = [&](int i, int j, int k) -> double { return f_ext[((size_t)(k + 2) * e1 + (j + 2)) * e0 + (i + 2)]; };
    for (int k = 0; k < n[2]; ++k)
        for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
                const double f0 = F(i, j, k);
                double v = f0;
                if (order >= 4) {
                    const double s1 = (F(i - 1, j, k) + F(i + 1, j, k)) + (F(i, j - 1, k) + F(i, j + 1, k)) +
                                      (F(i, j, k - 1) + F(i, j, k + 1)) - 6.0 * f0;
                    v += s1 / 12.0;
                }
                if (order == 6) {
                    auto d4 = [&](int di, int dj, int dk) -> double {
                        return F(i - 2 * di, j - 2 * dj, k - 2 * dk) - 4.0 * F(i - di, j - dj, k - dk) + 6.0 * f0 -
                               4.0 * F(i + di, j + dj, k + dk) + F(i + 2 * di, j + 2 * dj, k + 2 * dk);
                    };
                    // d_a^2 d_b^2 f: the 9-point cross difference in the plane of axes a, b
                    auto d22 = [&](int ai, int aj, int ak, int bi, int bj, int bk) -> double {
                        double s = 0.0;
                        const double c1[3] = {1.0, -2.0, 1.0};
                        for (int p = -1; p <= 1; ++p)
                            for (int q = -1; q <= 1; ++q)
                                s += c1[p + 1] * c1[q + 1] * F(i + p * ai + q * bi, j + p * aj + q * bj, k + p * ak + q * bk);
                        return s;
                    };
                    v -= (d4(1, 0, 0) + d4(0, 1, 0) + d4(0, 0, 1)) / 240.0;
                    v += (d22(1, 0, 0, 0, 1, 0) + d22(0, 1, 0, 0, 0, 1) + d22(0, 0, 1, 1, 0, 0)) / 90.0;
                }
                out[((size_t)k * n[1] + j) * n[0] + i] = v;
            }
    return 0;
}

// Galerkin stencil of coarse level `level` (>= 1) at coarse point (I,J,K): 27 coefficients.
int mgv_galerkin_stencil(const Grid& g, int level, int I, int J, int K, double* out27, int order) {
    VLevel L = level0(g, order);
    for (int l = 0; l < level; ++l) {
        for (int a = 0; a < 3; ++a)
            if (L.n[a] % 2 == 0 || L.n[a] < 3) return -1;
        L = galerkin(L);
    }
    if (!L.in(I, J, K)) return -1;
    std::memcpy(out27, &L.coef[L.idx(I, J, K) * 27], 27 * sizeof(double));
    return 0;
}

void mgv_restrict(const Grid& g, const double* r, double* bc) {
    VLevel F = level0(g), C;
    for (int a = 0; a < 3; ++a) C.n[a] = (F.n[a] - 1) / 2;
    restrict_v(F, C, r, bc);
}
void mgv_prolong_add(const Grid& g, const double* ec, double* x) {
    VLevel F = level0(g), C;
    for (int a = 0; a < 3; ++a) C.n[a] = (F.n[a] - 1) / 2;
    prolong_v(F, C, ec, x);
}

// ncycles V-cycles (Eq. 11) on L_h phi = rhs; storage_f32: coarse levels stored in fp32.
// resnorms (nullable, ncycles+1): ||rhs - L_h phi||_2 before the first and after every cycle (for Eq. 18).
// order: the level-0 discretisation (2: the grid's 7-point operator and ghost faces; 4, 6: compact, zero boundary values,
// rhs = compact_rhs output; the norms are then those of the compact residual).
int mgv_vcycle(const Grid& g, double* phi, const double* rhs, int nu1, int nu2, int coarsest_n, const double spai[5],
               double cg_rtol, int storage_f32, int ncycles, double* resnorms, int order) {
    if (g.coord != CARTESIAN || g.order != 2 || g.h[0] != g.h[1] || g.h[0] != g.h[2]) return -1;
    if (order != 2 && order != 4 && order != 6) return -1;
    for (int f = 0; f < 6; ++f)
        if (g.bc[f] != BC_DIRICHLET_GHOST) return -1;
    Hier H = build(g, nu1, nu2, coarsest_n, spai, cg_rtol, storage_f32, order);
    const VLevel& L0 = H.lv[0];
    std::vector<double> r(L0.size());
    auto residual0 = [&](const Grid& gg, const double* x, const double* f, double* out) {
        residual_level0(gg, L0, order, x, f, out);
    };
    auto norm0 = [&]() -> double {
        if (order == 2) return residual_norm(g, phi, rhs, true);
        std::vector<double> t(L0.size());
        residual0(g, phi, rhs, t.data());
        return (double)sqrtl(dotv(t, t));
    };
    if (resnorms) resnorms[0] = norm0();
    for (int c = 0; c < ncycles; ++c) {
        if (H.lv.size() == 1) {
            // no coarse level: the "coarsest solve" is CG on the error equation A e = r
            residual0(g, phi, rhs, r.data());
            std::vector<double> e(L0.size());
            cg_coarse(L0, e.data(), r.data(), cg_rtol, H.cg_max);
            for (size_t m = 0; m < e.size(); ++m) phi[m] += e[m];
        } else {
            for (int s = 0; s < nu1; ++s) {
                residual0(g, phi, rhs, r.data());
                spai_update(L0, phi, r.data(), H.sp);
            }
            residual0(g, phi, rhs, r.data());
            const VLevel& C = H.lv[1];
            std::vector<double> bc(C.size()), ec(C.size(), 0.0);
            restrict_v(L0, C, r.data(), bc.data());
            cycle_coarse(H, 1, ec, bc);
            prolong_v(L0, C, ec.data(), phi);
            for (int s = 0; s < nu2; ++s) {
                residual0(g, phi, rhs, r.data());
                spai_update(L0, phi, r.data(), H.sp);
            }
        }
        if (resnorms) resnorms[c + 1] = norm0();
    }
    return ST_OK;
}

}  // namespace orc
