// k_apply7.cu — lean 7-point (Cartesian, radius 1) stencil apply / residual for non-periodic grids, fp64 and fp32:
//   out = L v   or   out = rhs - L v   (+ fp32 copy, + sum(out^2), sum(out)).      PAPER.md:43-45 (Eq. 1), 55, 57.
// 2.5-D blocking with a register queue along z: a thread owns one 16-byte pair of x-adjacent columns of one row and
// keeps planes k-1, k, k+1 of it in registers; the plane that has just arrived is published to a ring of three
// shared-memory planes so that the neighbouring threads can read their x/y neighbours — one __syncthreads per plane,
// every shared-memory offset a compile-time constant (the z loop is unrolled by the ring size).  The tile carries one
// halo row above/below and one halo pair left/right whose threads only load and publish; on a domain boundary they hold
// the ghost-face values (or zero), fetched through one pointer + stride per thread.  Work is split among the resident
// CTAs as equal runs of (tile, plane) items.  Arithmetic order = stencil.cuh row_apply<KIND_CART2> (C1b).
#include <algorithm>
#include <cstdlib>

#include "pairq.cuh"

namespace pb {

struct A7Geom {
    int ntx, nty;
    long items;
};

template <int PXN_, int EY_, int MINB_, int PF_ = 1>
struct A7Tile {
    static constexpr int PXN = PXN_, EY = EY_, MINB = MINB_, PF = PF_;  // PF = planes of load prefetch: 1 or 3  // MINB = resident CTAs per SM asked of the compiler
    static constexpr int NT = ((PXN * EY + 31) / 32) * 32;
    static constexpr int SW = 2 * PXN, SLOT = SW * EY, NS = 3;
    static constexpr int VX = 2 * PXN - 4, VY = EY - 2;
};

template <typename T, class Cfg, int MODE, bool RED, bool PLAIN>
__global__ void __launch_bounds__(Cfg::NT, Cfg::MINB)
    k_apply7(const Op op, const T* __restrict__ v, const T* __restrict__ rhs, T* __restrict__ out,
             float* __restrict__ out32, const bool ug_in, const A7Geom g, RedBuf rb, double* scal) {
    using P2 = typename P2T<T>::type;
    constexpr int SW = Cfg::SW, SLOT = Cfg::SLOT, PXN = Cfg::PXN, EY = Cfg::EY, NS = Cfg::NS;
    extern __shared__ __align__(16) unsigned char smraw[];
    T* const ring = reinterpret_cast<T*>(smraw);
    const int n0 = op.n[0], n1 = op.n[1], n2 = op.n[2];
    const int tid = threadIdx.x;
    const bool live = tid < PXN * EY;
    const int lx = live ? tid % PXN : 0, ly = live ? tid / PXN : 0;
    const bool ug = ug_in && op.gamma == 0.0;
    const T c0 = (T)op.c[0], c1 = (T)op.c[1], c2 = (T)op.c[2];
    const T dplain = (T)2 * ((c0 + c1) + c2);
    const size_t plane = (size_t)n0 * n1;
    T* const mine = ring + ly * SW + 2 * lx;
    const bool inner = live && lx >= 1 && lx < PXN - 1 && ly >= 1 && ly < EY - 1;  // not a halo thread
    double s2 = 0.0, s1 = 0.0;

    const long total = (long)g.ntx * g.nty * n2;
    long pos = (long)blockIdx.x * g.items;
    const long end = min(total, pos + g.items);
    while (pos < end) {
        const int t = (int)(pos / n2), k0 = (int)(pos % n2);
        const int k1 = (int)min((long)n2, (long)k0 + (end - pos));
        pos += k1 - k0;
        const int tx = t % g.ntx, ty = t / g.ntx;
        const int i = tx * Cfg::VX - 2 + 2 * lx, j = ty * Cfg::VY - 1 + ly;
        const bool col_in = live && i >= 0 && i < n0 && j >= 0 && j < n1;
        const bool own = col_in && inner;
        // where the pair of plane kk comes from (see k_sor_fused.cu): 1 = the array, 2 / 3 = an x ghost face into
        // .y / .x, 4 = a y ghost face pair, 0 = zeros; planes -1 and n2 of in-domain columns are the z ghost faces
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
        if (!PLAIN && own) {
            dx = a7_diag_xy<T>(op, i, j);
            dy = a7_diag_xy<T>(op, i + 1, j);
        }
        const int kbeg = k0 - 1, kend = k1;  // planes kbeg .. kend pass through; plane kin - 1 is computed in iteration kin
        vp += (ptrdiff_t)kbeg * vs;
        const size_t cb = own ? (size_t)j * n0 + i : 0;
        const T* prh = rhs + cb + (ptrdiff_t)k0 * (ptrdiff_t)plane;  // rhs of plane kin + 1; only used when MODE != 0
        size_t po = cb + (size_t)k0 * plane;                           // output index of the next computed plane
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
        // loads run PF planes ahead of their use (PF = 1 or 3): nvq[u % PF] holds plane kin at unrolled iteration u;
        // the right-hand side of plane p sits in frq[(p - kbeg) % 3] and is loaded two iterations before its use
        constexpr int PF = Cfg::PF;
        P2 nvq[PF], frq[3];
#pragma unroll
        for (int m = 0; m < PF; ++m) {
            nvq[m] = P2T<T>::make((T)0, (T)0);
            if (kbeg + m <= kend) nvq[m] = loadv(kbeg + m);
            vp += vs;
        }
        frq[0] = frq[1] = frq[2] = P2T<T>::make((T)0, (T)0);
        __syncthreads();  // the previous segment's readers are done with the ring
        for (int kin0 = kbeg; kin0 <= kend; kin0 += 3) {
#pragma unroll
            for (int u = 0; u < 3; ++u) {
                const int kin = kin0 + u;
                if (kin > kend) break;
                const P2 nv = nvq[u % PF];
                q[u] = nv;
                if (live) *reinterpret_cast<P2*>(mine + u * SLOT) = nv;
                if (kin + PF <= kend) nvq[u % PF] = loadv(kin + PF);
                vp += vs;
                if (MODE != 0 && own && kin + 1 < k1) frq[(u + 1) % 3] = *reinterpret_cast<const P2*>(prh);
                prh += plane;
                const P2 f = frq[(u + 2) % 3];  // rhs of plane kin - 1
                __syncthreads();
                const int k = kin - 1;
                if (own && k >= k0 && k < k1) {
                    const T* const sp = mine + ((u + 2) % 3) * SLOT;
                    const P2 C = q[(u + 2) % 3], zm = q[(u + 1) % 3], zp = q[u];
                    const T xl = sp[-1], xr = sp[2];
                    const P2 ym = *reinterpret_cast<const P2*>(sp - SW), yp = *reinterpret_cast<const P2*>(sp + SW);
                    T d0 = PLAIN ? dplain : dx, d1 = PLAIN ? dplain : dy;
                    if (!PLAIN && (k == 0 || k == n2 - 1)) {
                        d0 = a7_diag_z<T>(op, d0, k);
                        d1 = a7_diag_z<T>(op, d1, k);
                    }
                    T s = (xl + C.y) * c0;
                    s = fma_(ym.x + yp.x, c1, s);
                    s = fma_(zm.x + zp.x, c2, s);
                    const T lx0 = fma_(-d0, C.x, s);
                    s = (C.x + xr) * c0;
                    s = fma_(ym.y + yp.y, c1, s);
                    s = fma_(zm.y + zp.y, c2, s);
                    const T lx1 = fma_(-d1, C.y, s);
                    const T o0 = MODE ? f.x - lx0 : lx0, o1 = MODE ? f.y - lx1 : lx1;
                    if (out) *reinterpret_cast<P2*>(out + po) = P2T<T>::make(o0, o1);
                    if (out32) *reinterpret_cast<float2*>(out32 + po) = make_float2((float)o0, (float)o1);
                    if (RED) {
                        s2 = fma((double)o0, (double)o0, s2);
                        s1 += (double)o0;
                        s2 = fma((double)o1, (double)o1, s2);
                        s1 += (double)o1;
                    }
                    po += plane;
                }
            }
        }
    }
    if (RED) {
        double vals[2] = {s2, s1};
        grid_reduce<2>(vals, rb, [=](const double* t) {
            scal[0] = t[0];
            scal[1] = t[1];
        });
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------------
bool apply7_ok(const poisson_ctx* ctx, const Op& op) {
    if (ctx->opt_path == 1) return false;
    if (op.coord != POISSON_CARTESIAN || op.order != 2 || op.n[0] % 2 != 0) return false;
    for (int f = 0; f < 6; ++f)
        if (op.bc[f] == POISSON_BC_PERIODIC) return false;
    if (ctx->opt_path == 2) return true;
    return (size_t)op.n[0] * op.n[1] * op.n[2] >= (size_t)1 << 15;
}

template <typename T, class Cfg, int MODE, bool RED>
static int apply7_launch(poisson_ctx* ctx, const Op& op, const T* v, const T* rhs, T* out, float* out32, bool ug,
                         int per_sm) {
    bool plain = op.gamma == 0.0;
    for (int f = 0; f < 6; ++f) plain = plain && op.bc[f] != POISSON_BC_NEUMANN0;
    A7Geom g;
    g.ntx = (op.n[0] + Cfg::VX - 1) / Cfg::VX;
    g.nty = (op.n[1] + Cfg::VY - 1) / Cfg::VY;
    const long total = (long)g.ntx * g.nty * op.n[2];
    const long slots = (long)ctx->num_sms * per_sm;
    g.items = std::max(4L, (total + slots - 1) / slots);
    const int grid = (int)((total + g.items - 1) / g.items);
    if (grid > kMaxRedBlocks) return fail(ctx, POISSON_UNSUPPORTED, "grid too large for the reduction buffer");
    const size_t smem = (size_t)Cfg::NS * Cfg::SLOT * sizeof(T);
    int rc = kernel_ready(ctx, k_apply7<T, Cfg, MODE, RED, true>, Cfg::NT, smem);
    if (rc == POISSON_OK) rc = kernel_ready(ctx, k_apply7<T, Cfg, MODE, RED, false>, Cfg::NT, smem);
    if (rc != POISSON_OK) return rc;
    if (plain)
        PB_LAUNCH(ctx, KID_APPLY, (k_apply7<T, Cfg, MODE, RED, true><<<grid, Cfg::NT, smem, ctx->stream>>>(op, v, rhs, out, out32, ug, g, ctx->red, ctx->d_scal)));
    else
        PB_LAUNCH(ctx, KID_APPLY, (k_apply7<T, Cfg, MODE, RED, false><<<grid, Cfg::NT, smem, ctx->stream>>>(op, v, rhs, out, out32, ug, g, ctx->red, ctx->d_scal)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

template <typename T, int MODE, bool RED>
static int apply7_cfg(poisson_ctx* ctx, const Op& op, const T* v, const T* rhs, T* out, float* out32, bool ug) {
    // measured at 256^3 fp64 on B200 (us per apply): CE 82.7, CA 85.1, CB 87.4, whole-row tiles 107
    using CE = A7Tile<34, 10, 2, 3>;  // 64 x 8 valid, 340 threads, two CTAs per SM, loads 3 planes ahead
    using CA = A7Tile<34, 18, 1, 3>;  // 64 x 16 valid, 612 threads, one CTA per SM
    using CC = A7Tile<18, 14, 4>;     // 32 x 12 valid, 252 threads (small grids)
    int c = (size_t)op.n[0] * op.n[1] * op.n[2] >= ((size_t)1 << 21) ? 0 : 2;
    const int ov = ctx->opt_tile_cfg;
    if (ov >= 0 && ov < 3) c = ov;
    switch (c) {
        case 0: return apply7_launch<T, CE, MODE, RED>(ctx, op, v, rhs, out, out32, ug, 2);
        case 1: return apply7_launch<T, CA, MODE, RED>(ctx, op, v, rhs, out, out32, ug, 1);
        default: return apply7_launch<T, CC, MODE, RED>(ctx, op, v, rhs, out, out32, ug, 4);
    }
}

template <typename T>
static int apply7_t(poisson_ctx* ctx, const Op& op, const T* v, const T* rhs, T* out, float* out32, int mode, bool ug,
                    bool reduce) {
    if (mode == 0) return apply7_cfg<T, 0, false>(ctx, op, v, rhs, out, out32, ug);
    if (!reduce) return apply7_cfg<T, 1, false>(ctx, op, v, rhs, out, out32, ug);
    return apply7_cfg<T, 1, true>(ctx, op, v, rhs, out, out32, ug);
}

int apply7(poisson_ctx* ctx, const Op& op, const double* v, const double* rhs, double* out, float* out32, int mode,
           bool ug, bool reduce) {
    return apply7_t<double>(ctx, op, v, rhs, out, out32, mode, ug, reduce);
}
int apply7_32(poisson_ctx* ctx, const Op& op, const float* v, const float* rhs, float* out, int mode) {
    return apply7_t<float>(ctx, op, v, rhs, out, nullptr, mode, false, false);
}

}  // namespace pb
