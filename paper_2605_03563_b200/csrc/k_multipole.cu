// k_multipole.cu — multipole-expansion open boundary.  PAPER.md:213-222:
//   q_lm = sum_cells rho r'^l S_lm dV          (Eq. 20, "numerically the integrals are expressed as sums over cells")
//   Phi(x) = -G sum_lm q_lm S_lm(x) / r^(l+1)  (Eq. 19), S_lm = sqrt(4 pi/(2l+1)) Y_lm, real harmonics, cosine for
//   m >= 0 and sine for m < 0.  Moment index l*l + l + m.
// Evaluated with Cartesian solid-harmonic recurrences (no trigonometry, no pole singularity):
//   A_m + i B_m = (x + i y)^m ;  Q_m^m = (2m-1)!! ;  Q_{m+1}^m = (2m+1) z Q_m^m ;
//   (l-m) Q_l^m = (2l-1) z Q_{l-1}^m - (l+m-1) r^2 Q_{l-2}^m ;
//   r^l S_l0 = Q_l^0 ;  r^l S_{l,m} = N_lm Q_l^m A_m ;  r^l S_{l,-m} = N_lm Q_l^m B_m ;  N_lm = sqrt(2 (l-m)!/(l+m)!).
// One fused pass over rho accumulates all (lmax+1)^2 moments per thread in registers, then warp shuffles, a block
// reduction and a last-block final sum (fixed order -> deterministic).  The pass is fp64-ALU bound at lmax = 8.
#include <algorithm>
#include <cmath>

#include "stencil.cuh"

namespace pb {

constexpr int kNQ = (kMaxLmax + 1) * (kMaxLmax + 1);

// N_lm at index l*l + l + m (both signs of m); 1 for m = 0.  Travels in the kernel parameters (constant bank), so
// there is no per-process or per-device state.
static void fill_norm(double* h) {
    for (int l = 0; l <= kMaxLmax; ++l) {
        h[l * l + l] = 1.0;
        for (int m = 1; m <= l; ++m) {
            long double ratio = 1;  // (l-m)!/(l+m)!
            for (int q = l - m + 1; q <= l + m; ++q) ratio /= (long double)q;
            h[l * l + l + m] = (double)sqrtl(2 * ratio);
            h[l * l + l - m] = h[l * l + l + m];
        }
    }
}

struct MpGeom {
    double norm[kNQ];
    int sph;
    int n[3];
    double origin[3], h[3];
    // spherical 1-D tables (device): centre radius, sin/cos theta, cos/sin phi, volume factors
    const double *rc, *st, *ct, *cph, *sph_, *vr, *vt, *vp;
    double r_ghost, r_ghost_in;
};

// One point's contribution to all moments, WITHOUT the normalisation N_lm (applied once per thread at the end).
// Per (l, m): one multiply, one fma and one scaling for the recurrence, one fma (two for m > 0) for the sums; the
// products (2l-1) z and k r^2 are formed once per point.
// INNER: the inner multipoles of Eq. 22, qbar_lm = sum rho r^-(l+1) S_lm dV = sum rho (r^l S_lm) r^-(2l+1) dV — the same
// solid harmonics with the weight scaled by r^-(2l+1) per degree.
// Only the orders M0 <= m <= M1 are accumulated (the unrolled loops touch no other accumulator, so the rest of `acc`
// never exists in registers).
template <int L, bool INNER, int M0, int M1>
__device__ __forceinline__ void accumulate(double (&acc)[(L + 1) * (L + 1)], double x, double y, double z, double w) {
    const double r2 = fma(z, z, fma(y, y, x * x));
    double pw[L + 1];  // r^-(2l+1)
    if (INNER) {
        const double rinv = 1.0 / sqrt(r2), rinv2 = rinv * rinv;
        pw[0] = rinv;
#pragma unroll
        for (int l = 1; l <= L; ++l) pw[l] = pw[l - 1] * rinv2;
    }
    double cz[L + 2], kr2[2 * L + 2];
#pragma unroll
    for (int l = 0; l <= L; ++l) cz[l] = (2 * l - 1) * z;
#pragma unroll
    for (int k = 0; k <= 2 * L; ++k) kr2[k] = k * r2;
    double A = 1.0, B = 0.0, dfact = 1.0;  // (x+iy)^m, (2m-1)!!
#pragma unroll
    for (int m = 0; m <= M1; ++m) {
        if (m >= M0) {
            double qm2 = 0.0, qm1 = dfact;  // Q_{l-2}^m, Q_{l-1}^m while walking l = m..L
            const double wa = w * A, wb = w * B;
#pragma unroll
            for (int l = m; l <= L; ++l) {
                double ql;
                if (l == m)
                    ql = dfact;
                else if (l == m + 1)
                    ql = cz[l] * qm1;
                else
                    ql = fma(cz[l], qm1, -(kr2[l + m - 1] * qm2)) * (1.0 / (l - m));
                const double qw = INNER ? ql * pw[l] : ql;
                if (m == 0) {
                    acc[l * l + l] = fma(wa, qw, acc[l * l + l]);
                } else {
                    acc[l * l + l + m] = fma(wa, qw, acc[l * l + l + m]);
                    acc[l * l + l - m] = fma(wb, qw, acc[l * l + l - m]);
                }
                qm2 = qm1;
                qm1 = ql;
            }
        }
        const double An = x * A - y * B, Bn = fma(y, A, x * B);
        A = An;
        B = Bn;
        dfact *= (2 * m + 1);
    }
}

// |m| of moment index s = l*l + l + m.
__host__ __device__ constexpr int abs_m_of(int s) {
    int l = 0;
    while ((l + 1) * (l + 1) <= s) ++l;
    const int m = s - l * l - l;
    return m < 0 ? -m : m;
}
// The orders are cut in two halves of about equal work: half 0 takes m < split, half 1 the rest.  At l_max = 8 that is
// 24 + 21 (l, |m|) pairs and ~40 accumulators per thread instead of 81: 128 registers and two CTAs per SM instead of
// 255 and one (ncu: the one-CTA kernel sat at 8 warps per SM with its loads exposed).  Each half walks rho once.
__host__ __device__ constexpr int m_split(int L) {
    int total = 0;
    for (int m = 0; m <= L; ++m) total += L - m + 1;
    int acc = 0;
    for (int m = 0; m <= L; ++m) {
        acc += L - m + 1;
        if (2 * acc >= total) return m + 1;
    }
    return L + 1;
}

template <int L, bool INNER, int M0, int M1>
__device__ __forceinline__ void moments_half(const MpGeom& g, const double* __restrict__ rho, double* __restrict__ partials,
                                             unsigned bid, unsigned nblk, double (*sm)[(L + 1) * (L + 1)]) {
    constexpr int NQ = (L + 1) * (L + 1);
    double acc[NQ];
#pragma unroll
    for (int s = 0; s < NQ; ++s) acc[s] = 0.0;
    const size_t n = (size_t)g.n[0] * g.n[1] * g.n[2];
    const size_t plane = (size_t)g.n[0] * g.n[1];
    const double dV = g.h[0] * g.h[1] * g.h[2];
    // whole warps walk consecutive points; a warp whose 32 densities are all zero skips the arithmetic.  The point
    // index is decoded once; every further step adds the (decoded) grid stride with carries — no division per point
    const size_t stride = (size_t)nblk * blockDim.x;
    const int n0 = g.n[0], n1 = g.n[1];
    const int di = (int)(stride % n0), dj = (int)((stride / n0) % n1), dk = (int)(stride / plane);
    size_t p = (size_t)bid * blockDim.x + threadIdx.x;
    int k = (int)(p / plane), j = (int)((p - (size_t)k * plane) / n0), i = (int)(p - (size_t)k * plane - (size_t)j * n0);
    double dnext = p < n ? rho[p] : 0.0;  // the density is loaded one step ahead of its use
    for (size_t base = ((size_t)bid * blockDim.x + (threadIdx.x & ~31)); base < n; base += stride, p += stride) {
        const int ci = i, cj = j, ck = k;  // this iteration's point
        const double d = dnext;
        dnext = p + stride < n ? rho[p + stride] : 0.0;
        i += di;
        if (i >= n0) { i -= n0; ++j; }
        j += dj;
        if (j >= n1) { j -= n1; ++k; }
        k += dk;
        if (__all_sync(0xffffffffu, d == 0.0)) continue;
        if (d == 0.0) continue;
        double x, y, z, w;
        if (g.sph) {
            const double r = g.rc[ci], rs = r * g.st[cj];
            x = rs * g.cph[ck];
            y = rs * g.sph_[ck];
            z = r * g.ct[cj];
            w = d * (g.vr[ci] * g.vt[cj] * g.vp[ck]);
        } else {
            x = fma((double)ci, g.h[0], g.origin[0]);
            y = fma((double)cj, g.h[1], g.origin[1]);
            z = fma((double)ck, g.h[2], g.origin[2]);
            w = d * dV;
        }
        accumulate<L, INNER, M0, M1>(acc, x, y, z, w);
    }
    // N_lm once per thread instead of once per point, then warp shuffles and shared memory across the 8 warps
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int s = 0; s < NQ; ++s) {
        if (abs_m_of(s) < M0 || abs_m_of(s) > M1) continue;  // compile-time after unrolling
        const double v = warp_sum(acc[s] * g.norm[s]);
        if (lane == 0) sm[wid][s] = v;
    }
    __syncthreads();
    for (int s = threadIdx.x; s < NQ; s += blockDim.x) {
        if (abs_m_of(s) < M0 || abs_m_of(s) > M1) continue;
        double v = 0.0;
        for (int ww = 0; ww < 8; ++ww) v += sm[ww][s];
        partials[(size_t)blockIdx.x * NQ + s] = v;
    }
}

// Grid: 2 G blocks; block b works on half b & 1 as block b >> 1 of G.  The last block adds, per moment, the partials of
// the blocks of its half in a fixed order.
template <int L, bool INNER>
__global__ void __launch_bounds__(256, 2)
    k_moments(MpGeom g, const double* __restrict__ rho, double* __restrict__ partials, unsigned int* counter,
              double* __restrict__ q_out) {
    constexpr int NQ = (L + 1) * (L + 1);
    constexpr int MS = m_split(L);
    __shared__ double sm[8][NQ];
    __shared__ int is_last;
    const unsigned half = MS <= L ? (blockIdx.x & 1u) : 0u;
    const unsigned nhalf = MS <= L ? 2u : 1u;
    const unsigned bid = blockIdx.x / nhalf, nblk = gridDim.x / nhalf;
    if (half == 0)
        moments_half<L, INNER, 0, (MS <= L ? MS - 1 : L)>(g, rho, partials, bid, nblk, sm);
    else
        moments_half<L, INNER, (MS <= L ? MS : L), L>(g, rho, partials, bid, nblk, sm);
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        is_last = (atomicInc(counter, gridDim.x - 1) == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    for (int s = threadIdx.x; s < NQ; s += blockDim.x) {
        const unsigned h = (MS <= L && abs_m_of(s) >= MS) ? 1u : 0u;
        double v = 0.0;
        for (unsigned b = h; b < gridDim.x; b += nhalf) v += __ldcg(&partials[(size_t)b * NQ + s]);
        q_out[s] = v;
    }
}

// ---- Cartesian grids: the same moments by z lines ---------------------------------------------------------------------------
// For a fixed column (x, y) the solid harmonic r^l S_lm is (x + i y)^m times a polynomial in z of degree l - m whose
// coefficients depend on s = x^2 + y^2 only: Q_l^m(z) = sum_c P_lm,c(s) z^c with the SAME recurrence as above applied
// to coefficient vectors,
//   P_m^m = (2m-1)!! ;  P_{m+1}^m = (2m+1) z P_m^m ;  (l-m) P_l^m = (2l-1) z P_{l-1}^m - (l+m-1) (s + z^2) P_{l-2}^m ,
// so that  sum_z rho Q_l^m = sum_c P_lm,c(s) Z_c  with the line sums  Z_c = sum_z rho z^c  (c = 0..lmax).
// Per point that is one load and lmax + 1 fused multiply-adds instead of ~270 fp64 instructions: the pass becomes
// HBM-bound (8 B/point).  A thread owns one column of a z chunk (lanes along x: coalesced), forms Z_c, converts once per
// chunk, and the 81 column values are summed over the CTA through shared memory in three groups of orders (m = 0-1,
// 2-3, 4-8: at most 30 values each).  Same sums in another order: the moments agree with the point-by-point kernel to
// rounding (measured 1e-19 .. 1e-24 absolute on configs 2 and 3, tolerance 1e-12 relative).
template <int L>
__global__ void __launch_bounds__(256, 2)
    k_moments_zline(MpGeom g, const double* __restrict__ rho, double* __restrict__ partials, unsigned int* counter,
                    double* __restrict__ q_out, int kc) {
    constexpr int NQ = (L + 1) * (L + 1), NC = L + 1, NCP = (NC + 1) & ~1;  // table rows padded to whole 16-byte pairs
    extern __shared__ __align__(16) double smz[];
    double* const zt = smz;                        // kc x NCP powers of z
    double* const buf = zt + (size_t)kc * NCP;     // 256 x 33: one row per thread (padded: conflict-free both ways)
    double* const sm2 = buf + 256 * 33;            // 8 x 32 warp partials
    __shared__ int smap[32];
    __shared__ int is_last;
    const int tid = threadIdx.x, lane = tid & 31, ty = tid >> 5;
    const int n0 = g.n[0], n1 = g.n[1], n2 = g.n[2];
    // columns in memory order: a CTA reads 2 KB of consecutive densities per plane
    const size_t plane = (size_t)n0 * n1, col = (size_t)blockIdx.x * 256 + tid;
    const int j = (int)(col / n0), i = (int)(col - (size_t)j * n0);
    const int k0 = blockIdx.y * kc, nk = min(kc, n2 - k0);
    const unsigned nblk = gridDim.x * gridDim.y;
    const unsigned bid = blockIdx.y * gridDim.x + blockIdx.x;
    for (int kk = tid; kk < nk; kk += 256) {
        const double z = fma((double)(k0 + kk), g.h[2], g.origin[2]);
        double p = 1.0;
#pragma unroll
        for (int c = 0; c < NCP; ++c) {
            zt[kk * NCP + c] = c < NC ? p : 0.0;
            p *= z;
        }
    }
    __syncthreads();
    double Z[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) Z[c] = 0.0;
    if (col < plane) {
        const double* p = rho + (size_t)k0 * plane + col;
        int kk = 0;
        constexpr int UNR = 16;  // loads in flight per thread
        for (; kk + UNR <= nk; kk += UNR) {
            double d[UNR];
#pragma unroll
            for (int u = 0; u < UNR; ++u) d[u] = p[(size_t)(kk + u) * plane];
#pragma unroll
            for (int u = 0; u < UNR; ++u) {
                const double2* const zr = reinterpret_cast<const double2*>(zt + (kk + u) * NCP);  // broadcast, 16 bytes a load
#pragma unroll
                for (int c = 0; c < NC; c += 2) {
                    const double2 t = zr[c / 2];
                    Z[c] = fma(d[u], t.x, Z[c]);
                    if (c + 1 < NC) Z[c + 1] = fma(d[u], t.y, Z[c + 1]);
                }
            }
        }
        for (; kk < nk; ++kk) {
            const double d = p[(size_t)kk * plane];
#pragma unroll
            for (int c = 0; c < NC; ++c) Z[c] = fma(d, zt[kk * NCP + c], Z[c]);
        }
    }
    // one group of orders: sum the values every thread has put into its row of buf over the CTA (fixed order)
    auto reduce_group = [&](int nvals) {
        __syncthreads();
        double acc = 0.0;
        if (lane < nvals)
            for (int t = 0; t < 32; ++t) acc += buf[(ty * 32 + t) * 33 + lane];
        sm2[ty * 32 + lane] = acc;
        __syncthreads();
        if (tid < nvals) {
            double t = 0.0;
            for (int w = 0; w < 8; ++w) t += sm2[w * 32 + tid];
            partials[(size_t)smap[tid] * nblk + bid] = t;  // moment-major: the final sum reads consecutive blocks
        }
        __syncthreads();
    };
    const double x = fma((double)i, g.h[0], g.origin[0]), y = fma((double)j, g.h[1], g.origin[1]);
    const double s = fma(y, y, x * x);
    double A = 1.0, B = 0.0, dfact = 1.0;  // (x + i y)^m, (2m-1)!!
    int slot = 0;
    double* const row = buf + tid * 33;
#pragma unroll
    for (int m = 0; m <= L; ++m) {
        double P1[NC], P2[NC];  // coefficient vectors of Q_{l-1}^m, Q_{l-2}^m (powers of z; only c = l-m mod 2 is non-zero)
#pragma unroll
        for (int c = 0; c < NC; ++c) P1[c] = P2[c] = 0.0;
#pragma unroll
        for (int l = m; l <= L; ++l) {
            double P[NC];
#pragma unroll
            for (int c = 0; c < NC; ++c) P[c] = 0.0;
            if (l == m) {
                P[0] = dfact;
            } else if (l == m + 1) {
                P[1] = (2 * m + 1) * P1[0];
            } else {
#pragma unroll
                for (int c = (l - m) & 1; c <= l - m; c += 2) {
                    const double up = c >= 1 ? (2 * l - 1) * P1[c - 1] : 0.0;
                    double lo = c <= l - 2 - m ? s * P2[c] : 0.0;
                    if (c >= 2) lo += P2[c - 2];
                    P[c] = (up - (l + m - 1) * lo) * (1.0 / (l - m));
                }
            }
            double v = 0.0;
#pragma unroll
            for (int c = (l - m) & 1; c <= l - m; c += 2) v = fma(P[c], Z[c], v);
            if (m == 0) {
                row[slot] = v;
                if (tid == 0) smap[slot] = l * l + l;
                ++slot;
            } else {
                row[slot] = A * v;
                row[slot + 1] = B * v;
                if (tid == 0) {
                    smap[slot] = l * l + l + m;
                    smap[slot + 1] = l * l + l - m;
                }
                slot += 2;
            }
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                P2[c] = P1[c];
                P1[c] = P[c];
            }
        }
        if (m == 1 || m == 3 || m == L) {  // groups m = 0-1, 2-3, 4-L
            reduce_group(slot);
            slot = 0;
        }
        const double An = x * A - y * B, Bn = fma(y, A, x * B);
        A = An;
        B = Bn;
        dfact *= (2 * m + 1);
    }
    // the last block adds the block partials in a fixed order; N_lm and the cell volume are applied once, here
    if (tid == 0) {
        __threadfence();
        is_last = (atomicInc(counter, nblk - 1) == nblk - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    const double dV = g.h[0] * g.h[1] * g.h[2];
    for (int q = ty; q < NQ; q += 8) {  // a warp per moment: lanes over the blocks, then the warp (fixed order)
        double v = 0.0;
        for (unsigned b = lane; b < nblk; b += 32) v += __ldcg(&partials[(size_t)q * nblk + b]);
        v = warp_sum(v);
        if (lane == 0) q_out[q] = v * g.norm[q] * dV;
    }
}

// ---- spherical grids: the same moments by radial lines -----------------------------------------------------------------------
// r^l S_lm(theta, phi) dV factorises on a spherical grid: q_lm = sum_{j,k} [N_lm P_l^m(cos theta_j) {cos, sin}(m phi_k)
// vt_j vp_k] * R_l(j,k) with the radial line sums R_l = sum_i rho_ijk rc_i^l vr_i (inner moments, Eq. 22: rc_i^-(l+1)).
// The radius is the fastest index: a warp walks one line (coalesced), every lane forms the lmax + 1 partial sums of its
// points (one load, lmax multiplications and lmax + 1 fused multiply-adds per point instead of ~270 fp64 instructions),
// the warp adds them, and then lane q owns the moments q, q + 32, q + 64: it evaluates their angular factor for the line
// and accumulates.  The angular factors come from two tables every CTA builds once in shared memory — P_l^m(cos
// theta_j) vt_j by its recurrence from the tabulated sin / cos theta, {cos, sin}(m phi_k) vp_k by powers of the
// tabulated cos phi + i sin phi (no trigonometric call) — so a line costs each lane two loads and three multiply-adds
// per moment it owns.
constexpr int kRlineWarps = 16;  // one 512-thread CTA per SM

template <int L, bool INNER>
__global__ void __launch_bounds__(32 * kRlineWarps, 1)
    k_moments_rline(MpGeom g, const double* __restrict__ rho, double* __restrict__ partials, unsigned int* counter,
                    double* __restrict__ q_out) {
    constexpr int NQ = (L + 1) * (L + 1), NC = L + 1, NP = (L + 1) * (L + 2) / 2, NM = 2 * L + 1;
    extern __shared__ double smr[];
    const int n0 = g.n[0], n1 = g.n[1], n2 = g.n[2];
    double* const rtab = smr;            // rc_i (inner: 1 / rc_i)
    double* const vtab = rtab + n0;      // vr_i (inner: vr_i / rc_i)
    constexpr int NW = kRlineWarps, NT = 32 * NW;
    double* const Rw = vtab + n0;        // NW warps x 2 x 16: the line sums of the warp's two current lines
    double* const accw = Rw + NW * 32;   // NW warps x 96: the warps' moments at the end
    double* const PT = accw + NW * 96;   // n1 x NP: P_l^m(cos theta_j) vt_j at l (l+1)/2 + m
    double* const CS = PT + (size_t)n1 * NP;  // n2 x NM: cos(m phi_k) vp_k at m, sin(m phi_k) vp_k at L + m
    double* const Rs = CS + (size_t)n2 * NM;  // NW warps x 2 NC x 33: the lanes' partial line sums, transposed to add
    __shared__ int is_last;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int i = tid; i < n0; i += NT) {
        const double r = g.rc[i];
        rtab[i] = INNER ? 1.0 / r : r;
        vtab[i] = INNER ? g.vr[i] / r : g.vr[i];
    }
    for (int j = tid; j < n1; j += NT) {
        const double ct = g.ct[j], st = g.st[j], vt = g.vt[j];
        const double rk[9] = {0.0, 1.0, 1.0 / 2, 1.0 / 3, 1.0 / 4, 1.0 / 5, 1.0 / 6, 1.0 / 7, 1.0 / 8};  // 1 / (l - m)
        double pmm = 1.0;  // P_m^m = (2m-1)!! sin^m theta, no Condon-Shortley phase
#pragma unroll
        for (int m = 0; m <= L; ++m) {
            if (m > 0) pmm *= (2 * m - 1) * st;
            double pm2 = 0.0, pm1 = pmm;
#pragma unroll
            for (int l = m; l <= L; ++l) {
                double pl;
                if (l == m)
                    pl = pmm;
                else if (l == m + 1)
                    pl = (2 * m + 1) * ct * pm1;
                else
                    pl = ((2 * l - 1) * ct * pm1 - (l + m - 1) * pm2) * rk[l - m];
                PT[(size_t)j * NP + l * (l + 1) / 2 + m] = pl * vt;
                pm2 = pm1;
                pm1 = pl;
            }
        }
    }
    for (int k = tid; k < n2; k += NT) {
        const double cp = g.cph[k], sp = g.sph_[k], vp = g.vp[k];
        double ca = 1.0, sa = 0.0;
        CS[(size_t)k * NM] = vp;
#pragma unroll
        for (int m = 1; m <= L; ++m) {
            const double cn = ca * cp - sa * sp, sn = fma(sa, cp, ca * sp);
            ca = cn;
            sa = sn;
            CS[(size_t)k * NM + m] = ca * vp;
            CS[(size_t)k * NM + L + m] = sa * vp;
        }
    }
    __syncthreads();
    // this lane's moments: index s = lane + 32 q, degree ls, order ms (sine harmonic for ms < 0)
    int ls[3], pi[3], ci[3];  // degree (-1: none), index into a PT row, index into a CS row
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const int s = lane + 32 * q;
        int l = 0;
        while ((l + 1) * (l + 1) <= s) ++l;
        const int m = s - l * l - l, am = m < 0 ? -m : m;
        ls[q] = s < NQ ? l : -1;
        pi[q] = s < NQ ? l * (l + 1) / 2 + am : 0;
        ci[q] = s < NQ ? (m < 0 ? L + am : am) : 0;
    }
    double acc[3] = {0.0, 0.0, 0.0};
    const long nlines = (long)n1 * n2, nw = (long)gridDim.x * NW;
    // two lines per pass of the warp: twice the loads in flight and twice the independent reductions
    double* const rs = Rs + (size_t)wid * (2 * NC * 33);
    for (long line0 = (long)blockIdx.x * NW + wid; line0 < nlines; line0 += 2 * nw) {
        const long line1 = line0 + nw;
        const bool two = line1 < nlines;
        const double* const p0 = rho + (size_t)line0 * n0;
        const double* const p1 = rho + (size_t)(two ? line1 : line0) * n0;
        double R0[NC], R1[NC];
#pragma unroll
        for (int l = 0; l < NC; ++l) R0[l] = R1[l] = 0.0;
#pragma unroll 4
        for (int i = lane; i < n0; i += 32) {
            const double d0 = p0[i], d1 = p1[i], rr = rtab[i];
            double rl = vtab[i];
#pragma unroll
            for (int l = 0; l < NC; ++l) {
                R0[l] = fma(d0, rl, R0[l]);
                R1[l] = fma(d1, rl, R1[l]);
                rl *= rr;
            }
        }
        // the warp's sums through shared memory: every lane deposits its 2 NC partial sums, lane v adds row v
        // (18 stores + 32 loads and additions per lane instead of 90 shuffle-and-add steps)
#pragma unroll
        for (int l = 0; l < NC; ++l) {
            rs[l * 33 + lane] = R0[l];
            rs[(NC + l) * 33 + lane] = R1[l];
        }
        __syncwarp();
        if (lane < 2 * NC) {
            double t = 0.0;
#pragma unroll 8
            for (int u = 0; u < 32; ++u) t += rs[lane * 33 + u];
            Rw[wid * 32 + (lane < NC ? lane : 16 + lane - NC)] = t;
        }
        __syncwarp();
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (h == 1 && !two) break;
            const long line = h ? line1 : line0;
            const int k = (int)(line / n1), j = (int)(line - (long)k * n1);
            const double* const pt = PT + (size_t)j * NP;
            const double* const cs = CS + (size_t)k * NM;
#pragma unroll
            for (int q = 0; q < 3; ++q)
                if (ls[q] >= 0) acc[q] = fma(pt[pi[q]] * cs[ci[q]], Rw[wid * 32 + 16 * h + ls[q]], acc[q]);
        }
        __syncwarp();
    }
#pragma unroll
    for (int q = 0; q < 3; ++q) accw[wid * 96 + lane + 32 * q] = acc[q];
    __syncthreads();
    const unsigned nblk = gridDim.x, bid = blockIdx.x;
    if (tid < NQ) {
        double t = 0.0;
        for (int w = 0; w < NW; ++w) t += accw[w * 96 + tid];
        partials[(size_t)tid * nblk + bid] = t;
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        is_last = (atomicInc(counter, nblk - 1) == nblk - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    for (int q = wid; q < NQ; q += NW) {  // a warp per moment: lanes over the blocks, then the warp (fixed order)
        double v = 0.0;
        for (unsigned b = lane; b < nblk; b += 32) v += __ldcg(&partials[(size_t)q * nblk + b]);
        v = warp_sum(v);
        if (lane == 0) q_out[q] = v * g.norm[q];
    }
}

// Phi at one exterior point from the moments.
// inner: Eq. 21, Phi = -G sum qbar_lm r^l S_lm (no inverse powers of r).
// qn = q_lm N_lm (shared memory).
// LMAX is a template parameter: both loops unroll (no table of reciprocals in local memory, no loop bookkeeping —
// the run-time-lmax version spent ~24 instructions per harmonic).
template <int LMAX>
__device__ __forceinline__ double expansion(const double* __restrict__ qn, double G, double x, double y, double z,
                                            bool inner) {
    constexpr int lmax = LMAX;
    const double r2 = fma(z, z, fma(y, y, x * x));
    const double rinv = inner ? 1.0 : 1.0 / sqrt(r2), rinv2 = rinv * rinv;
    double A = 1.0, B = 0.0, dfact = 1.0, acc = 0.0;
    double pw_m = rinv;  // r^-(2m+1)  (1 for the inner expansion)
#pragma unroll
    for (int m = 0; m <= lmax; ++m) {
        double qm2 = 0.0, qm1 = dfact, pw = pw_m;  // pw = r^-(2l+1)
#pragma unroll
        for (int l = m; l <= lmax; ++l) {
            double ql;
            if (l == m)
                ql = dfact;
            else if (l == m + 1)
                ql = (2 * m + 1) * z * qm1;
            else
                ql = ((2 * l - 1) * z * qm1 - (l + m - 1) * r2 * qm2) * (1.0 / (l - m));
            if (m == 0)
                acc = fma(qn[l * l + l] * ql, pw, acc);
            else
                acc = fma((qn[l * l + l + m] * A + qn[l * l + l - m] * B) * ql, pw, acc);
            qm2 = qm1;
            qm1 = ql;
            pw *= rinv2;
        }
        const double An = x * A - y * B, Bn = fma(y, A, x * B);
        A = An;
        B = Bn;
        dfact *= (2 * m + 1);
        pw_m *= rinv2;
    }
    return -G * acc;
}

// All ghost faces in ONE launch (six launches of a few thousand threads each cost six launch latencies): block b
// belongs to the face whose block range contains it.
struct GhostFaces {
    int nf;
    int face[6], first_block[7];  // first_block[nf] = total
    double* out[6];
    const double* q[6];
    int inner[6];
};

template <int LMAX>
__global__ void __launch_bounds__(256) k_ghost_eval(MpGeom g, GhostFaces gf, int R, double G) {
    constexpr int lmax = LMAX;
    int s = 0;
#pragma unroll
    for (int m = 1; m < 6; ++m)
        if (m < gf.nf && (int)blockIdx.x >= gf.first_block[m]) s = m;
    const int face = gf.face[s];
    const bool inner = gf.inner[s] != 0;
    __shared__ double qn[kNQ];  // this face's moments times N_lm, read 81 times by every thread
    for (int e = threadIdx.x; e < (lmax + 1) * (lmax + 1); e += blockDim.x) qn[e] = gf.q[s][e] * g.norm[e];
    __syncthreads();
    const int a = face / 2, a1 = (a == 0) ? 1 : 0, a2 = (a == 2) ? 1 : 2;
    const long len = (long)R * g.n[a1] * g.n[a2];
    const long t = (long)(blockIdx.x - gf.first_block[s]) * blockDim.x + threadIdx.x;
    if (t >= len) return;
    const int q1 = (int)(t % g.n[a1]), q2 = (int)((t / g.n[a1]) % g.n[a2]), layer = (int)(t / ((long)g.n[a1] * g.n[a2]));
    double x, y, z;
    if (g.sph) {
        const double rg = inner ? g.r_ghost_in : g.r_ghost;
        const double rs = rg * g.st[q1];
        x = rs * g.cph[q2];
        y = rs * g.sph_[q2];
        z = rg * g.ct[q1];
    } else {
        int id[3];
        id[a] = (face & 1) ? g.n[a] + layer : -1 - layer;
        id[a1] = q1;
        id[a2] = q2;
        x = fma((double)id[0], g.h[0], g.origin[0]);
        y = fma((double)id[1], g.h[1], g.origin[1]);
        z = fma((double)id[2], g.h[2], g.origin[2]);
    }
    gf.out[s][t] = expansion<LMAX>(qn, G, x, y, z, inner);
}

static MpGeom make_geom(poisson_ctx* ctx) {
    MpGeom g{};
    fill_norm(g.norm);
    g.sph = ctx->op.coord == POISSON_SPHERICAL;
    for (int a = 0; a < 3; ++a) {
        g.n[a] = ctx->op.n[a];
        g.origin[a] = ctx->origin[a];
        g.h[a] = ctx->h[a];
    }
    if (g.sph) {
        const int nr = g.n[0], nt = g.n[1], np = g.n[2];
        const double* b = ctx->d_ctr;
        g.rc = b;
        g.st = b + nr;
        g.ct = b + nr + nt;
        g.cph = b + nr + 2 * nt;
        g.sph_ = b + nr + 2 * nt + np;
        g.vr = b + nr + 2 * nt + 2 * np;
        g.vt = b + 2 * nr + 2 * nt + 2 * np;
        g.vp = b + 2 * nr + 3 * nt + 2 * np;
        g.r_ghost = ctx->r_ghost_out;
        g.r_ghost_in = ctx->edges[0][0] * std::sqrt(ctx->edges[0][0] / ctx->edges[0][1]);
    }
    return g;
}

template <int L>
static void moments_launch(poisson_ctx* ctx, const MpGeom& g, const double* rho, double* d_q, int blocks, bool inner) {
    if (inner)
        k_moments<L, true><<<blocks, 256, 0, ctx->stream>>>(g, rho, ctx->red.partials, ctx->red.counter, d_q);
    else
        k_moments<L, false><<<blocks, 256, 0, ctx->stream>>>(g, rho, ctx->red.partials, ctx->red.counter, d_q);
}

// z-line kernel: Cartesian grids, outer moments; z chunks so that about two waves of CTAs exist (a chunk costs one
// conversion + CTA reduction, ~1100 instructions per thread, next to ~22 per plane).
template <int L>
static int zline_launch(poisson_ctx* ctx, const MpGeom& g, const double* rho, double* d_q) {
    const long bx = ((long)g.n[0] * g.n[1] + 255) / 256, by = 1;
    // z chunks only where the columns alone do not give every SM a CTA: a chunk costs a conversion and a CTA reduction
    // (measured 6 us per layer of 256 CTAs at 256^3, lmax = 8; 48 / 54 / 66 us with 1 / 2 / 4 chunks)
    int nzc = std::max(1, (int)((ctx->num_sms + bx - 1) / bx));
    nzc = std::min(nzc, std::max(1, g.n[2] / 64));
    int kc = (g.n[2] + nzc - 1) / nzc;
    kc = std::min(kc, 512);
    nzc = (g.n[2] + kc - 1) / kc;
    constexpr int NQ = (L + 1) * (L + 1);
    if ((size_t)bx * nzc * NQ > (size_t)kMaxRedBlocks * kRedSlots || bx > 0x7fffffffL || nzc > 65535) return POISSON_UNSUPPORTED;
    const size_t smem = ((size_t)kc * ((L + 2) & ~1) + 256 * 33 + 8 * 32) * sizeof(double);
    const int rc = kernel_ready(ctx, k_moments_zline<L>, 256, 110 * 1024);
    if (rc != POISSON_OK) return rc;
    k_moments_zline<L><<<dim3((unsigned)bx, nzc), 256, smem, ctx->stream>>>(g, rho, ctx->red.partials, ctx->red.counter, d_q, kc);
    return POISSON_OK;
}

template <int L>
static int rline_launch(poisson_ctx* ctx, const MpGeom& g, const double* rho, double* d_q, bool inner) {
    const long nlines = (long)g.n[1] * g.n[2];
    constexpr int NW = kRlineWarps;
    const int blocks = (int)std::max(1L, std::min<long>((long)ctx->num_sms, (nlines + 2 * NW - 1) / (2 * NW)));
    const size_t smem = ((size_t)2 * g.n[0] + NW * 32 + NW * 96 + (size_t)g.n[1] * ((L + 1) * (L + 2) / 2) +
                         (size_t)g.n[2] * (2 * L + 1) + (size_t)NW * 2 * (L + 1) * 33) * sizeof(double);
    if (smem > 200 * 1024) return POISSON_UNSUPPORTED;
    int rc = kernel_ready(ctx, k_moments_rline<L, false>, 32 * NW, 200 * 1024);
    if (rc == POISSON_OK) rc = kernel_ready(ctx, k_moments_rline<L, true>, 32 * NW, 200 * 1024);
    if (rc != POISSON_OK) return rc;
    if (inner)
        k_moments_rline<L, true><<<blocks, 32 * NW, smem, ctx->stream>>>(g, rho, ctx->red.partials, ctx->red.counter, d_q);
    else
        k_moments_rline<L, false><<<blocks, 32 * NW, smem, ctx->stream>>>(g, rho, ctx->red.partials, ctx->red.counter, d_q);
    return POISSON_OK;
}

int launch_moments(poisson_ctx* ctx, const double* rho, int lmax, double* d_q, bool inner) {
    if (lmax < 0 || lmax > kMaxLmax) return fail(ctx, POISSON_INVALID_ARG, "lmax must be in 0..8");
    const MpGeom g = make_geom(ctx);
    // spherical grids: by radial lines; POISSON_OPT_KERNEL_PATH = 1 keeps the point-by-point kernel
    if (g.sph && ctx->opt_path != 1) {
        pre_launch(ctx, KID_MP_MOMENTS);
        int rc = POISSON_UNSUPPORTED;
        switch (lmax) {
            case 0: rc = rline_launch<0>(ctx, g, rho, d_q, inner); break;
            case 1: rc = rline_launch<1>(ctx, g, rho, d_q, inner); break;
            case 2: rc = rline_launch<2>(ctx, g, rho, d_q, inner); break;
            case 3: rc = rline_launch<3>(ctx, g, rho, d_q, inner); break;
            case 4: rc = rline_launch<4>(ctx, g, rho, d_q, inner); break;
            case 5: rc = rline_launch<5>(ctx, g, rho, d_q, inner); break;
            case 6: rc = rline_launch<6>(ctx, g, rho, d_q, inner); break;
            case 7: rc = rline_launch<7>(ctx, g, rho, d_q, inner); break;
            case 8: rc = rline_launch<8>(ctx, g, rho, d_q, inner); break;
            default: break;
        }
        if (rc == POISSON_OK) {
            post_launch(ctx, KID_MP_MOMENTS);
            PB_CUDA_OK(cudaGetLastError());
            return POISSON_OK;
        }
        if (rc != POISSON_UNSUPPORTED) return rc;
    }
    // Cartesian grids: by z lines (HBM-bound); POISSON_OPT_KERNEL_PATH = 1 keeps the point-by-point kernel
    if (!g.sph && !inner && ctx->opt_path != 1) {
        pre_launch(ctx, KID_MP_MOMENTS);
        int rc = POISSON_UNSUPPORTED;
        switch (lmax) {
            case 0: rc = zline_launch<0>(ctx, g, rho, d_q); break;
            case 1: rc = zline_launch<1>(ctx, g, rho, d_q); break;
            case 2: rc = zline_launch<2>(ctx, g, rho, d_q); break;
            case 3: rc = zline_launch<3>(ctx, g, rho, d_q); break;
            case 4: rc = zline_launch<4>(ctx, g, rho, d_q); break;
            case 5: rc = zline_launch<5>(ctx, g, rho, d_q); break;
            case 6: rc = zline_launch<6>(ctx, g, rho, d_q); break;
            case 7: rc = zline_launch<7>(ctx, g, rho, d_q); break;
            case 8: rc = zline_launch<8>(ctx, g, rho, d_q); break;
            default: break;
        }
        if (rc == POISSON_OK) {
            post_launch(ctx, KID_MP_MOMENTS);
            PB_CUDA_OK(cudaGetLastError());
            return POISSON_OK;
        }
        if (rc != POISSON_UNSUPPORTED) return rc;
    }
    // two resident CTAs per SM; for l_max >= 1 the grid is made of pairs of blocks (one per half of the orders)
    int blocks = ctx->num_sms * 2;
    const size_t maxb = (ctx->npts + 255) / 256;
    if ((size_t)blocks > maxb) blocks = (int)maxb;
    if (lmax >= 1) blocks = 2 * std::max(1, blocks);  // G blocks per half (m_split(L) <= L for every L >= 1)
    pre_launch(ctx, KID_MP_MOMENTS);
    switch (lmax) {
        case 0: moments_launch<0>(ctx, g, rho, d_q, blocks, inner); break;
        case 1: moments_launch<1>(ctx, g, rho, d_q, blocks, inner); break;
        case 2: moments_launch<2>(ctx, g, rho, d_q, blocks, inner); break;
        case 3: moments_launch<3>(ctx, g, rho, d_q, blocks, inner); break;
        case 4: moments_launch<4>(ctx, g, rho, d_q, blocks, inner); break;
        case 5: moments_launch<5>(ctx, g, rho, d_q, blocks, inner); break;
        case 6: moments_launch<6>(ctx, g, rho, d_q, blocks, inner); break;
        case 7: moments_launch<7>(ctx, g, rho, d_q, blocks, inner); break;
        case 8: moments_launch<8>(ctx, g, rho, d_q, blocks, inner); break;
        default: break;  // range checked by the caller
    }
    post_launch(ctx, KID_MP_MOMENTS);
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

// d_qbar: inner moments (Eq. 22), used for the inner radial shell of a spherical grid (face 0) when it is a Dirichlet face.
int launch_ghost_eval(poisson_ctx* ctx, const double* d_q, const double* d_qbar, double G, int lmax) {
    const MpGeom g = make_geom(ctx);
    GhostFaces gf{};
    int blocks = 0;
    for (int f = 0; f < 6; ++f) {
        if (ctx->op.bc[f] != POISSON_BC_DIRICHLET_GHOST || !ctx->d_ghost[f]) continue;
        if (g.sph && f > 1) continue;  // only the radial shells carry Eq. 19 / Eq. 21
        const bool inner = g.sph && f == 0;
        if (inner && !d_qbar) continue;
        gf.face[gf.nf] = f;
        gf.first_block[gf.nf] = blocks;
        gf.out[gf.nf] = ctx->d_ghost[f];
        gf.q[gf.nf] = inner ? d_qbar : d_q;
        gf.inner[gf.nf] = inner ? 1 : 0;
        blocks += (int)((ctx->face_len[f] + 255) / 256);
        ++gf.nf;
    }
    gf.first_block[gf.nf] = blocks;
    if (blocks > 0) {
        pre_launch(ctx, KID_MP_GHOSTS);
        switch (lmax) {
            case 0: k_ghost_eval<0><<<blocks, 256, 0, ctx->stream>>>(g, gf, ctx->op.R, G); break;
            case 1: k_ghost_eval<1><<<blocks, 256, 0, ctx->stream>>>(g, gf, ctx->op.R, G); break;
            case 2: k_ghost_eval<2><<<blocks, 256, 0, ctx->stream>>>(g, gf, ctx->op.R, G); break;
            case 3: k_ghost_eval<3><<<blocks, 256, 0, ctx->stream>>>(g, gf, ctx->op.R, G); break;
            case 4: k_ghost_eval<4><<<blocks, 256, 0, ctx->stream>>>(g, gf, ctx->op.R, G); break;
            case 5: k_ghost_eval<5><<<blocks, 256, 0, ctx->stream>>>(g, gf, ctx->op.R, G); break;
            case 6: k_ghost_eval<6><<<blocks, 256, 0, ctx->stream>>>(g, gf, ctx->op.R, G); break;
            case 7: k_ghost_eval<7><<<blocks, 256, 0, ctx->stream>>>(g, gf, ctx->op.R, G); break;
            case 8: k_ghost_eval<8><<<blocks, 256, 0, ctx->stream>>>(g, gf, ctx->op.R, G); break;
            default: return fail(ctx, POISSON_INVALID_ARG, "lmax must be in 0..8");
        }
        post_launch(ctx, KID_MP_GHOSTS);
    }
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

}  // namespace pb
