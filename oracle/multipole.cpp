// ORACLE — TEST INFRASTRUCTURE ONLY (see grid.hpp).
// Multipole-expansion open boundary, PAPER.md:213-222:
//   Phi(x)  = -G sum_{l,m} q_lm / r^{l+1} * sqrt(4 pi/(2l+1)) Y_lm(x)                       (Eq. 19)
//   q_lm    = int dV' sqrt(4 pi/(2l+1)) rho(x') r'^l Y_lm(x')   ("sums over cells")          (Eq. 20)
// with real spherical harmonics, cosine harmonics for m >= 0 and sine harmonics for m < 0.
// Written out in trigonometric / associated-Legendre form (reading C6):
//   S_lm = sqrt(4 pi/(2l+1)) Y_lm ;  S_l0 = P_l(cos th) ;  m > 0: S_{l,m} = N_lm P_l^m(cos th) cos(m ph),
//   S_{l,-m} = N_lm P_l^m(cos th) sin(m ph), N_lm = sqrt(2 (l-m)!/(l+m)!).
// Expansion centre = coordinate origin.  Moment index: l*l + l + m.
#include <cmath>
#include <vector>

#include "solvers.hpp"

namespace orc {

static const int LMAX_CAP = 16;

// S_lm(theta, phi) for 0 <= l <= lmax, |m| <= l, into S[l*l+l+m].
static void real_harmonics(int lmax, long double ct, long double st, long double ph, long double* S) {
    // associated Legendre functions without the Condon-Shortley phase:
    // P_m^m = (2m-1)!! sin^m th ; P_{m+1}^m = (2m+1) cos th P_m^m ;
    // (l-m) P_l^m = (2l-1) cos th P_{l-1}^m - (l+m-1) P_{l-2}^m.
    long double P[LMAX_CAP + 1][LMAX_CAP + 1];
    for (int m = 0; m <= lmax; ++m) {
        long double pmm = 1;
        for (int q = 1; q <= m; ++q) pmm *= (2 * q - 1) * st;
        P[m][m] = pmm;
        if (m + 1 <= lmax) P[m + 1][m] = (2 * m + 1) * ct * pmm;
        for (int l = m + 2; l <= lmax; ++l)
            P[l][m] = ((2 * l - 1) * ct * P[l - 1][m] - (l + m - 1) * P[l - 2][m]) / (long double)(l - m);
    }
    for (int l = 0; l <= lmax; ++l) {
        S[l * l + l] = P[l][0];
        for (int m = 1; m <= l; ++m) {
            long double ratio = 1;  // (l-m)!/(l+m)!
            for (int q = l - m + 1; q <= l + m; ++q) ratio /= (long double)q;
            long double N = sqrtl(2 * ratio);
            S[l * l + l + m] = N * P[l][m] * cosl(m * ph);
            S[l * l + l - m] = N * P[l][m] * sinl(m * ph);
        }
    }
}

static void to_spherical(long double x, long double y, long double z, long double& r, long double& ct, long double& st,
                         long double& ph) {
    r = sqrtl(x * x + y * y + z * z);
    if (r == 0) {
        ct = 1;
        st = 0;
        ph = 0;
        return;
    }
    ct = z / r;
    st = sqrtl(x * x + y * y) / r;
    ph = atan2l(y, x);
}

void multipole_moments(const Grid& g, const double* rho, int lmax, double* q) {
    const int nq = (lmax + 1) * (lmax + 1);
    std::vector<std::vector<long double>> part(g.n[2], std::vector<long double>(nq, 0.0L));
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k) {
        long double S[(LMAX_CAP + 1) * (LMAX_CAP + 1)];
        for (int j = 0; j < g.n[1]; ++j)
            for (int i = 0; i < g.n[0]; ++i) {
                long double r, ct, st, ph, dV;
                if (g.coord == CARTESIAN) {
                    to_spherical(g.coordinate(0, i), g.coordinate(1, j), g.coordinate(2, k), r, ct, st, ph);
                    dV = (long double)g.h[0] * g.h[1] * g.h[2];
                } else {
                    r = g.ctr[0][i];
                    ct = cosl((long double)g.ctr[1][j]);
                    st = sinl((long double)g.ctr[1][j]);
                    ph = g.ctr[2][k];
                    // exact cell volume (reading C6)
                    long double r0 = g.edge[0][i], r1 = g.edge[0][i + 1];
                    dV = (r1 * r1 * r1 - r0 * r0 * r0) / 3.0L *
                         (cosl((long double)g.edge[1][j]) - cosl((long double)g.edge[1][j + 1])) *
                         ((long double)g.edge[2][k + 1] - (long double)g.edge[2][k]);
                }
                real_harmonics(lmax, ct, st, ph, S);
                long double w = (long double)rho[g.idx(i, j, k)] * dV, rl = 1;
                for (int l = 0; l <= lmax; ++l) {
                    for (int m = -l; m <= l; ++m) part[k][l * l + l + m] += w * rl * S[l * l + l + m];
                    rl *= r;
                }
            }
    }
    for (int s = 0; s < nq; ++s) {
        long double tot = 0;
        for (int k = 0; k < g.n[2]; ++k) tot += part[k][s];
        q[s] = (double)tot;
    }
}

double multipole_potential(const double* q, int lmax, double G, double x, double y, double z) {
    long double r, ct, st, ph;
    to_spherical(x, y, z, r, ct, st, ph);
    long double S[(LMAX_CAP + 1) * (LMAX_CAP + 1)];
    real_harmonics(lmax, ct, st, ph, S);
    long double acc = 0, rinv = 1 / r, rp = rinv;  // rp = r^-(l+1)
    for (int l = 0; l <= lmax; ++l) {
        long double sl = 0;
        for (int m = -l; m <= l; ++m) sl += (long double)q[l * l + l + m] * S[l * l + l + m];
        acc += sl * rp;
        rp *= rinv;
    }
    return (double)(-(long double)G * acc);
}

// Inner multipoles, Eq. 22: qbar_lm = sum_cells rho r'^-(l+1) S_lm dV (spherical grids with r_in > 0).
void multipole_inner_moments(const Grid& g, const double* rho, int lmax, double* qbar) {
    const int nq = (lmax + 1) * (lmax + 1);
    std::vector<std::vector<long double>> part(g.n[2], std::vector<long double>(nq, 0.0L));
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g.n[2]; ++k) {
        long double S[(LMAX_CAP + 1) * (LMAX_CAP + 1)];
        for (int j = 0; j < g.n[1]; ++j)
            for (int i = 0; i < g.n[0]; ++i) {
                long double r, ct, st, ph, dV;
                if (g.coord == CARTESIAN) {
                    to_spherical(g.coordinate(0, i), g.coordinate(1, j), g.coordinate(2, k), r, ct, st, ph);
                    dV = (long double)g.h[0] * g.h[1] * g.h[2];
                } else {
                    r = g.ctr[0][i];
                    ct = cosl((long double)g.ctr[1][j]);
                    st = sinl((long double)g.ctr[1][j]);
                    ph = g.ctr[2][k];
                    long double r0 = g.edge[0][i], r1 = g.edge[0][i + 1];
                    dV = (r1 * r1 * r1 - r0 * r0 * r0) / 3.0L *
                         (cosl((long double)g.edge[1][j]) - cosl((long double)g.edge[1][j + 1])) *
                         ((long double)g.edge[2][k + 1] - (long double)g.edge[2][k]);
                }
                if (rho[g.idx(i, j, k)] == 0.0 || r == 0) continue;
                real_harmonics(lmax, ct, st, ph, S);
                long double w = (long double)rho[g.idx(i, j, k)] * dV, rl = 1 / r;  // r^-(l+1)
                for (int l = 0; l <= lmax; ++l) {
                    for (int m = -l; m <= l; ++m) part[k][l * l + l + m] += w * rl * S[l * l + l + m];
                    rl /= r;
                }
            }
    }
    for (int s = 0; s < nq; ++s) {
        long double tot = 0;
        for (int k = 0; k < g.n[2]; ++k) tot += part[k][s];
        qbar[s] = (double)tot;
    }
}

// Eq. 21: Phi(x) = -G sum_lm qbar_lm r^l S_lm(x), valid inside all the mass.
double multipole_inner_potential(const double* qbar, int lmax, double G, double x, double y, double z) {
    long double r, ct, st, ph;
    to_spherical(x, y, z, r, ct, st, ph);
    long double S[(LMAX_CAP + 1) * (LMAX_CAP + 1)];
    real_harmonics(lmax, ct, st, ph, S);
    long double acc = 0, rp = 1;  // r^l
    for (int l = 0; l <= lmax; ++l) {
        long double sl = 0;
        for (int m = -l; m <= l; ++m) sl += (long double)qbar[l * l + l + m] * S[l * l + l + m];
        acc += sl * rp;
        rp *= r;
    }
    return (double)(-(long double)G * acc);
}

// Fill the ghost zones of every Dirichlet face with Eq. 19 ("We use this formula for all
// boundaries in Cartesian coordinates, and for the outer boundary r = r_out in spherical coordinates").
void multipole_bc(Grid& g, const double* rho, double G, int lmax, double* moments, double* inner_moments) {
    std::vector<double> q((lmax + 1) * (lmax + 1)), qbar;
    multipole_moments(g, rho, lmax, q.data());
    if (moments)
        for (size_t s = 0; s < q.size(); ++s) moments[s] = q[s];
    // a spherical grid whose inner radial face is a ghost-Dirichlet face also needs the inner expansion, Eq. 21-22
    const bool inner = g.coord == SPHERICAL && g.bc[0] == BC_DIRICHLET_GHOST;
    if (inner) {
        qbar.resize(q.size());
        multipole_inner_moments(g, rho, lmax, qbar.data());
        if (inner_moments)
            for (size_t s = 0; s < qbar.size(); ++s) inner_moments[s] = qbar[s];
    }
    for (int f = 0; f < 6; ++f) {
        if (g.bc[f] != BC_DIRICHLET_GHOST) continue;
        int a = f / 2, a1 = (a == 0) ? 1 : 0, a2 = (a == 2) ? 1 : 2;
        g.ghost[f].assign(g.face_len(f), 0.0);
        for (int layer = 0; layer < g.R; ++layer)
            for (int q2 = 0; q2 < g.n[a2]; ++q2)
                for (int q1 = 0; q1 < g.n[a1]; ++q1) {
                    double x, y, z;
                    if (g.coord == CARTESIAN) {
                        int id[3];
                        id[a] = (f & 1) ? g.n[a] + layer : -1 - layer;
                        id[a1] = q1;
                        id[a2] = q2;
                        x = g.coordinate(0, id[0]);
                        y = g.coordinate(1, id[1]);
                        z = g.coordinate(2, id[2]);
                    } else {
                        if (f > 1) continue;  // only the radial shells carry Eq. 19 / Eq. 21
                        // ghost shell centres continue the geometric progression of the radial centres
                        double r = f == 1 ? g.r_ghost_out : g.edge[0][0] * std::sqrt(g.edge[0][0] / g.edge[0][1]);
                        double th = g.ctr[1][q1], ph = g.ctr[2][q2];
                        x = r * std::sin(th) * std::cos(ph);
                        y = r * std::sin(th) * std::sin(ph);
                        z = r * std::cos(th);
                    }
                    g.ghost[f][((size_t)layer * g.n[a2] + q2) * g.n[a1] + q1] =
                        (inner && f == 0) ? multipole_inner_potential(qbar.data(), lmax, G, x, y, z)
                                          : multipole_potential(q.data(), lmax, G, x, y, z);
                }
    }
}

}  // namespace orc
