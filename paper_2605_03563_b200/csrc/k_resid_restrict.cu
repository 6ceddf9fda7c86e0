// k_resid_restrict.cu — V-cycle downward leg in one pass: coarse right-hand side f_c = R (f - L phi) without ever
// writing the fine residual to memory.  PAPER.md:125-142 (Eq. 11-13: residual, restriction R; P = c R^T).
// Reads phi and f (16 B per fine point), writes f_c (1 B per fine point).
//
// Structure = k_apply7.cu (a thread owns a 16-byte pair of x-adjacent fine columns (2I, 2I+1) = the two x children of
// coarse column I, keeps planes k-1, k, k+1 of phi in registers, publishes the arriving plane to a ring of three
// shared-memory planes).  The tile carries two halo rows / one halo pair of phi on each side so that the residual is
// available one fine cell beyond the valid tile, which is what the (1/8)[1 3 3 1]^3 weights of coarse cell (I,J,K) —
// fine cells 2I-1..2I+2 per axis — reach.  The restriction runs axis by axis (fw_acc, stencil.cuh) as a three-stage
// pipeline behind the residual, one barrier per fine plane: in the iteration that forms the residual of plane k, the
// x sums of plane k-1 are taken (own pair + one value of each neighbour pair, from a two-plane residual ring) and the
// y sums of plane k-2 (own row + three rows of a two-plane ring of x sums) are added into the z sums of the two coarse
// planes that fine plane touches, which live in the registers of the thread that owns fine row 2J.  Same bits as the
// residual kernel followed by k_restrict.  Work items are (tile, COARSE plane).
#include <algorithm>
#include <cstdlib>

#include "pairq.cuh"

namespace pb {

struct RRGeom {
    int ntx, nty;
    long items;
};

template <int PXN_, int EY_>
struct RRTile {
    static constexpr int PXN = PXN_, EY = EY_;
    static constexpr int NT = ((PXN * EY + 31) / 32) * 32;
    static constexpr int SW = 2 * PXN, SLOT = SW * EY;
    static constexpr int VX = 2 * PXN - 4, VY = EY - 4;   // valid fine tile (both even)
    static constexpr int NC = (VX / 2) * (VY / 2);         // coarse cells per tile plane
};

template <typename T, class Cfg, bool PLAIN>
__global__ void __launch_bounds__(Cfg::NT, 1)
    k_resid_restrict(const Op op, const Op cop, const T* __restrict__ v, const T* __restrict__ rhs,
                     T* __restrict__ fc, const bool ug_in, const int restriction, const RRGeom g) {
    using P2 = typename P2T<T>::type;
    constexpr int SW = Cfg::SW, SLOT = Cfg::SLOT, PXN = Cfg::PXN, EY = Cfg::EY;
    extern __shared__ __align__(16) unsigned char smraw[];
    T* const ring = reinterpret_cast<T*>(smraw);   // 3 planes of phi
    T* const rres = ring + 3 * SLOT;               // 2 planes of residual (pairs, the layout of the phi ring)
    constexpr int XSLOT = PXN * EY;
    T* const xbuf = rres + 2 * SLOT;               // 2 planes of x sums (one value per pair)
    const int n0 = op.n[0], n1 = op.n[1], n2 = op.n[2], nc2 = cop.n[2];
    const int tid = threadIdx.x;
    const bool live = tid < PXN * EY;
    const int lx = live ? tid % PXN : 0, ly = live ? tid / PXN : 0;
    const bool ug = ug_in && op.gamma == 0.0;
    const T c0 = (T)op.c[0], c1 = (T)op.c[1], c2 = (T)op.c[2];
    const T dplain = (T)2 * ((c0 + c1) + c2);
    const size_t plane = (size_t)n0 * n1;
    const int so = ly * SW + 2 * lx;
    T* const mine = ring + so;
    const bool rrow = live && ly >= 1 && ly < EY - 1;  // rows on which the residual is formed
    // shared-memory offsets of the x neighbours, clamped inside the row (the clamped ones feed only unused residuals)
    const int o_xl = lx > 0 ? -1 : 0, o_xr = lx < PXN - 1 ? 2 : 1;
    // the pair of thread lx = cI + 1 is the pair of x children (2I, 2I+1) of the tile's coarse column cI
    const bool xth = live && lx >= 1 && lx <= PXN - 2;

    const long total = (long)g.ntx * g.nty * nc2;
    long pos = (long)blockIdx.x * g.items;
    const long end = min(total, pos + g.items);
    while (pos < end) {
        const int t = (int)(pos / nc2), K0 = (int)(pos % nc2);
        const int K1 = (int)min((long)nc2, (long)K0 + (end - pos));
        pos += K1 - K0;
        const int tx = t % g.ntx, ty = t / g.ntx;
        const int i = tx * Cfg::VX - 2 + 2 * lx, j = ty * Cfg::VY - 2 + ly;
        const bool col_in = live && i >= 0 && i < n0 && j >= 0 && j < n1;
        const bool rown = col_in && rrow;
        int kind = 0;
        const T* vp = v;
        ptrdiff_t vs = 0;
        if (col_in) {
            kind = 1;
            vp = v + (size_t)j * n0 + i;
            vs = (ptrdiff_t)plane;
        } else if (live && ug && sizeof(T) == sizeof(double)) {
            const bool jin = j >= 0 && j < n1;
            int f = -1;
            if (jin && i == -2) { f = 0; kind = 2; }
            else if (jin && i == n0) { f = 1; kind = 3; }
            else if (i >= 0 && i < n0 && (j == -1 || j == n1)) { f = j < 0 ? 2 : 3; kind = 4; }
            if (f >= 0 && op.bc[f] == POISSON_BC_DIRICHLET_GHOST && op.ghost[f] != nullptr) {
                vp = reinterpret_cast<const T*>(op.ghost[f]) + (f < 2 ? j : i);
                vs = f < 2 ? n1 : n0;
            } else {
                kind = 0;
            }
        }
        const T* zlo = nullptr;
        const T* zhi = nullptr;
        if (col_in && ug && sizeof(T) == sizeof(double)) {
            if (op.bc[4] == POISSON_BC_DIRICHLET_GHOST && op.ghost[4]) zlo = reinterpret_cast<const T*>(op.ghost[4]) + (size_t)j * n0 + i;
            if (op.bc[5] == POISSON_BC_DIRICHLET_GHOST && op.ghost[5]) zhi = reinterpret_cast<const T*>(op.ghost[5]) + (size_t)j * n0 + i;
        }
        T dx = dplain, dy = dplain;
        if (!PLAIN && rown) {
            dx = a7_diag_xy<T>(op, i, j);
            dy = a7_diag_xy<T>(op, i + 1, j);
        }
        // fine planes 2K0-2 .. 2K1+1 of phi pass through; the residual of plane kin-1 is formed in iteration kin
        const int kbeg = 2 * K0 - 2, kend = 2 * K1 + 1;
        vp += (ptrdiff_t)kbeg * vs;
        const T* prh = rhs + (rown ? (size_t)j * n0 + i : 0) + (ptrdiff_t)(kbeg + 1) * (ptrdiff_t)plane;
        auto loadv = [&](int kk) -> P2 {
            P2 w = P2T<T>::make((T)0, (T)0);
            if (kk >= 0 && kk < n2) {
                if (kind == 1 || kind == 4) w = *reinterpret_cast<const P2*>(vp);
                else if (kind == 2) w.y = *vp;
                else if (kind == 3) w.x = *vp;
            } else if (kk == -1) {
                if (zlo) w = *reinterpret_cast<const P2*>(zlo);
            } else if (kk == n2) {
                if (zhi) w = *reinterpret_cast<const P2*>(zhi);
            }
            return w;
        };
        P2 q[3];
        q[0] = q[1] = q[2] = P2T<T>::make((T)0, (T)0);
        constexpr int PF = 3;
        P2 nvq[PF], frq[3];
#pragma unroll
        for (int m = 0; m < PF; ++m) {
            nvq[m] = P2T<T>::make((T)0, (T)0);
            if (kbeg + m <= kend) nvq[m] = loadv(kbeg + m);
            vp += vs;
        }
        frq[0] = frq[1] = frq[2] = P2T<T>::make((T)0, (T)0);
        // restriction state of this thread: its residual pair of the previous plane, its x sum of the plane before,
        // and the z sums of the two coarse planes the current fine plane contributes to
        P2 res_prev = P2T<T>::make((T)0, (T)0);
        T x_prev = (T)0, zA = (T)0, zB = (T)0;
        const bool xrow = xth && rrow && col_in;                    // forms x sums (fine columns 2I, 2I+1 = its own pair)
        const bool own = xrow && (ly & 1) == 0 && ly >= 2 && ly <= EY - 4;  // fine row 2J: forms y and z sums, stores
        const bool has_l = i - 1 >= 0, has_r = i + 2 < n0, has_d = j - 1 >= 0, has_u = j + 2 < n1;
        T* const fcp = own ? fc + (size_t)(j >> 1) * cop.n[0] + (i >> 1) : fc;
        const size_t cplane = (size_t)cop.n[0] * cop.n[1];
        __syncthreads();  // the previous segment's readers are done with the rings
        for (int kin0 = kbeg; kin0 <= kend + 2; kin0 += 3) {
#pragma unroll
            for (int u = 0; u < 3; ++u) {
                const int kin = kin0 + u;
                if (kin > kend + 2) break;
                if (kin <= kend) {
                    const P2 nv = nvq[u % PF];
                    q[u] = nv;
                    if (live) *reinterpret_cast<P2*>(mine + u * SLOT) = nv;
                    if (kin + PF <= kend) nvq[u % PF] = loadv(kin + PF);
                }
                vp += vs;
                // rhs of plane kin + 1 (used two iterations later)
                frq[(u + 1) % 3] = P2T<T>::make((T)0, (T)0);
                if (rown && kin + 1 >= 0 && kin + 1 < n2 && kin + 1 <= kend - 1) frq[(u + 1) % 3] = *reinterpret_cast<const P2*>(prh);
                prh += plane;
                const P2 f = frq[(u + 2) % 3];  // rhs of plane kin - 1
                __syncthreads();
                const int k = kin - 1;          // residual plane of this iteration
                // (c) y and z sums of plane k - 2, whose x sums were published one iteration ago
                {
                    const int kz = k - 2;
                    if (own && kz > kbeg && kz < kend && kz >= 0 && kz < n2) {
                        const T* const xs = xbuf + ((kz + 8) & 1) * XSLOT + ly * PXN + lx;
                        if (restriction == 1) {
                            const T y = x_prev + xs[PXN];
                            if (kz & 1) {
                                const int K = kz >> 1;
                                if (K >= K0 && K < K1) fcp[(size_t)K * cplane] = (zA + y) * (T)0.125;
                            } else {
                                zA = y;
                            }
                        } else {
                            T y = (T)0;
                            if (has_d) y = fw_acc<T>(y, 0, xs[-PXN]);
                            y = fw_acc<T>(y, 1, x_prev);
                            y = fw_acc<T>(y, 2, xs[PXN]);
                            if (has_u) y = fw_acc<T>(y, 3, xs[2 * PXN]);
                            if (kz & 1) {  // fine plane 2m+1: weight 2 of coarse plane m, weight 0 of m + 1
                                zA = fw_acc<T>(zA, 2, y);
                                zB = fw_acc<T>((T)0, 0, y);
                                const int K = kz >> 1;
                                if (kz == n2 - 1 && K >= K0 && K < K1) fcp[(size_t)K * cplane] = zA;
                            } else {       // fine plane 2m: weight 3 of coarse plane m - 1 (now complete), weight 1 of m
                                zA = fw_acc<T>(zA, 3, y);
                                const int K = (kz >> 1) - 1;
                                if (K >= K0 && K < K1) fcp[(size_t)K * cplane] = zA;
                                zA = fw_acc<T>(zB, 1, y);
                                zB = (T)0;
                            }
                        }
                    }
                }
                // (b) x sums of plane k - 1, whose residuals were published one iteration ago
                {
                    const int kx = k - 1;
                    if (xrow && kx > kbeg && kx < kend && kx >= 0 && kx < n2) {
                        const T* const rp = rres + ((kx + 8) & 1) * SLOT + so;
                        T x = (T)0;
                        if (restriction == 1) {
                            x = res_prev.x + res_prev.y;
                        } else {
                            if (has_l) x = fw_acc<T>(x, 0, rp[-1]);
                            x = fw_acc<T>(x, 1, res_prev.x);
                            x = fw_acc<T>(x, 2, res_prev.y);
                            if (has_r) x = fw_acc<T>(x, 3, rp[2]);
                        }
                        xbuf[((kx + 8) & 1) * XSLOT + ly * PXN + lx] = x;
                        x_prev = x;
                    }
                }
                // (a) residual of plane k
                if (kin > kbeg && kin <= kend && live) {
                    P2 res = P2T<T>::make((T)0, (T)0);
                    if (rown && k >= 0 && k < n2 && kin >= kbeg + 2) {
                        const T* const sp = mine + ((u + 2) % 3) * SLOT;
                        const P2 C = q[(u + 2) % 3], zm = q[(u + 1) % 3], zp = q[u];
                        const T xl = sp[o_xl], xr = sp[o_xr];
                        const P2 ym = *reinterpret_cast<const P2*>(sp - SW), yp = *reinterpret_cast<const P2*>(sp + SW);
                        T d0 = PLAIN ? dplain : dx, d1 = PLAIN ? dplain : dy;
                        if (!PLAIN && (k == 0 || k == n2 - 1)) {
                            d0 = a7_diag_z<T>(op, d0, k);
                            d1 = a7_diag_z<T>(op, d1, k);
                        }
                        T s = (xl + C.y) * c0;
                        s = fma_(ym.x + yp.x, c1, s);
                        s = fma_(zm.x + zp.x, c2, s);
                        res.x = f.x - fma_(-d0, C.x, s);
                        s = (C.x + xr) * c0;
                        s = fma_(ym.y + yp.y, c1, s);
                        s = fma_(zm.y + zp.y, c2, s);
                        res.y = f.y - fma_(-d1, C.y, s);
                    }
                    *reinterpret_cast<P2*>(rres + ((k + 8) & 1) * SLOT + so) = res;
                    res_prev = res;
                }
            }
        }
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------------
bool resid_restrict_ok(const poisson_ctx* ctx, const Op& fine, const Op& coarse) {
    if (ctx->opt_path == 1) return false;
    if (fine.coord != POISSON_CARTESIAN || fine.order != 2) return false;
    for (int a = 0; a < 3; ++a)
        if (fine.n[a] != 2 * coarse.n[a]) return false;
    for (int f = 0; f < 6; ++f)
        if (fine.bc[f] == POISSON_BC_PERIODIC) return false;
    if (ctx->opt_path == 2) return true;
    return (size_t)fine.n[0] * fine.n[1] * fine.n[2] >= (size_t)1 << 15;
}

template <typename T, class Cfg>
static int rr_launch(poisson_ctx* ctx, const Op& fine, const Op& coarse, const T* phi, const T* rhs, T* fc, bool ug) {
    bool plain = fine.gamma == 0.0;
    for (int f = 0; f < 6; ++f) plain = plain && fine.bc[f] != POISSON_BC_NEUMANN0;
    RRGeom g;
    g.ntx = (fine.n[0] + Cfg::VX - 1) / Cfg::VX;
    g.nty = (fine.n[1] + Cfg::VY - 1) / Cfg::VY;
    const long total = (long)g.ntx * g.nty * coarse.n[2];
    g.items = std::max(2L, (total + ctx->num_sms - 1) / ctx->num_sms);
    const int grid = (int)((total + g.items - 1) / g.items);
    const size_t smem = (size_t)6 * Cfg::SLOT * sizeof(T);
    int rc = kernel_ready(ctx, k_resid_restrict<T, Cfg, true>, Cfg::NT, smem);
    if (rc == POISSON_OK) rc = kernel_ready(ctx, k_resid_restrict<T, Cfg, false>, Cfg::NT, smem);
    if (rc != POISSON_OK) return rc;
    if (plain)
        PB_LAUNCH(ctx, KID_MG_RESTRICT, (k_resid_restrict<T, Cfg, true><<<grid, Cfg::NT, smem, ctx->stream>>>(fine, coarse, phi, rhs, fc, ug, ctx->opt_restriction, g)));
    else
        PB_LAUNCH(ctx, KID_MG_RESTRICT, (k_resid_restrict<T, Cfg, false><<<grid, Cfg::NT, smem, ctx->stream>>>(fine, coarse, phi, rhs, fc, ug, ctx->opt_restriction, g)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

template <typename T>
static int rr_t(poisson_ctx* ctx, const Op& fine, const Op& coarse, const T* phi, const T* rhs, T* fc, bool ug) {
    using CA = RRTile<34, 20>;  // 64 x 16 valid, 680 threads
    using CB = RRTile<18, 20>;  // 32 x 16 valid, 360 threads (small levels)
    if ((size_t)fine.n[0] * fine.n[1] * fine.n[2] >= ((size_t)1 << 21)) return rr_launch<T, CA>(ctx, fine, coarse, phi, rhs, fc, ug);
    return rr_launch<T, CB>(ctx, fine, coarse, phi, rhs, fc, ug);
}

int resid_restrict(poisson_ctx* ctx, const Op& fine, const Op& coarse, const double* phi, const double* rhs, double* fc,
                   bool ug) {
    return rr_t<double>(ctx, fine, coarse, phi, rhs, fc, ug);
}
int resid_restrict32(poisson_ctx* ctx, const Op& fine, const Op& coarse, const float* phi, const float* rhs, float* fc) {
    return rr_t<float>(ctx, fine, coarse, phi, rhs, fc, false);
}

}  // namespace pb
