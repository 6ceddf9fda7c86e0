// k_sor_fused.cu — red-black SOR / Gauss-Seidel with both colour half-sweeps of a full sweep (or of two sweeps) fused
// into ONE pass over HBM: temporal blocking of NHS = 2 or 4 colour half-steps by a z wavefront.  PAPER.md:59-63.
//
// A CTA owns an extended xy tile (valid tile + NHS halo columns/rows on every side that is not a domain boundary) and
// marches z.  A thread owns one 16-byte pair of x-adjacent columns (i, i+1) of one row and keeps their last NHS+2
// planes in a register queue.  In iteration `kin` (plane kin has just arrived) half-step h = 1..NHS updates plane
// kin-h: because the colour of (i,j,k) is (i+j+k)&1 and half-step h updates colour (h-1)&1, the SAME column of the
// pair — the one with (i+j+kin) odd — is the updated one in every half-step of the iteration, so the whole chain
//   plane kin-1 (red) -> plane kin-2 (black) [-> kin-3 (red) -> kin-4 (black)]
// runs in registers: z neighbours come from the thread's own queue, the x neighbour inside the pair from the partner
// queue, and only the outer x neighbour and the two y neighbours come from shared memory, where every thread
// publishes what it changes (a ring of NHS+2 planes).  The columns read from shared memory are the ones that are NOT
// updated in this iteration, so one __syncthreads per plane is enough.  After iteration kin plane kin-NHS is final
// and is written out.  Halo points are recomputed by the neighbouring CTA (overlapped tiling), hence input and output
// are different arrays (ping-pong) — the byte count per sweep is unchanged: read phi, rhs; write phi = 24 B/point.
// Work is split among the resident CTAs as equal runs of (tile, plane) items, so all SMs stay busy for any grid.
// Arithmetic and its order are those of k_rbsor_half / DESIGN.md C1b, C2: results are bit-identical to the unfused
// half-sweep kernels.
#include <algorithm>
#include <cstdlib>

#include "stencil.cuh"

namespace pb {

struct SorGeom {
    int pxn, ey;    // extended tile: pxn pairs x ey rows (threads in use = pxn * ey)
    int vx, vy;     // valid tile
    int ntx, nty;   // tiles per axis
    long items;     // (tile, plane) items per CTA
};

template <bool B>
struct FastTag {
    static constexpr bool value = B;
};

template <typename T>
struct PairT {};
template <>
struct PairT<double> {
    using type = double2;
    static __device__ __forceinline__ double2 make(double a, double b) { return make_double2(a, b); }
};
template <>
struct PairT<float> {
    using type = float2;
    static __device__ __forceinline__ float2 make(float a, float b) { return make_float2(a, b); }
};

// Value seen at an out-of-domain position: the ghost-face value when exactly one index is one step outside a
// Dirichlet face (a star stencil reads nothing else), zero otherwise.
template <typename T>
__device__ __forceinline__ T sor_bval(const Op& op, int i, int j, int k, bool ug) {
    const bool ox = i < 0 || i >= op.n[0], oy = j < 0 || j >= op.n[1], oz = k < 0 || k >= op.n[2];
    if (!ug || (int)ox + (int)oy + (int)oz != 1) return (T)0;
    int f;
    size_t idx;
    if (ox) {
        if (i != -1 && i != op.n[0]) return (T)0;
        f = i < 0 ? 0 : 1;
        idx = (size_t)k * op.n[1] + j;
    } else if (oy) {
        if (j != -1 && j != op.n[1]) return (T)0;
        f = j < 0 ? 2 : 3;
        idx = (size_t)k * op.n[0] + i;
    } else {
        if (k != -1 && k != op.n[2]) return (T)0;
        f = k < 0 ? 4 : 5;
        idx = (size_t)j * op.n[0] + i;
    }
    if (op.bc[f] != POISSON_BC_DIRICHLET_GHOST || op.ghost[f] == nullptr) return (T)0;
    return (T)op.ghost[f][idx];
}

// x/y part of row_diag (same order of operations), then the z part per plane.
template <typename T>
__device__ __forceinline__ T sor_diag_xy(const Op& op, int i, int j) {
    const T c0 = (T)op.c[0], c1 = (T)op.c[1], c2 = (T)op.c[2];
    T d = (T)2 * ((c0 + c1) + c2);
    const T g = (T)op.gamma;
    const bool closure = op.gamma != 0.0;
    if (i == 0) {
        if (op.bc[0] == POISSON_BC_DIRICHLET_GHOST && closure) d = fma_(g, c0, d);
        if (op.bc[0] == POISSON_BC_NEUMANN0) d -= c0;
    }
    if (i == op.n[0] - 1) {
        if (op.bc[1] == POISSON_BC_DIRICHLET_GHOST && closure) d = fma_(g, c0, d);
        if (op.bc[1] == POISSON_BC_NEUMANN0) d -= c0;
    }
    if (j == 0) {
        if (op.bc[2] == POISSON_BC_DIRICHLET_GHOST && closure) d = fma_(g, c1, d);
        if (op.bc[2] == POISSON_BC_NEUMANN0) d -= c1;
    }
    if (j == op.n[1] - 1) {
        if (op.bc[3] == POISSON_BC_DIRICHLET_GHOST && closure) d = fma_(g, c1, d);
        if (op.bc[3] == POISSON_BC_NEUMANN0) d -= c1;
    }
    return d;
}
template <typename T>
__device__ __forceinline__ T sor_diag_z(const Op& op, T d, int k) {
    const T c2 = (T)op.c[2], g = (T)op.gamma;
    const bool closure = op.gamma != 0.0;
    if (k == 0) {
        if (op.bc[4] == POISSON_BC_DIRICHLET_GHOST && closure) d = fma_(g, c2, d);
        if (op.bc[4] == POISSON_BC_NEUMANN0) d -= c2;
    }
    if (k == op.n[2] - 1) {
        if (op.bc[5] == POISSON_BC_DIRICHLET_GHOST && closure) d = fma_(g, c2, d);
        if (op.bc[5] == POISSON_BC_NEUMANN0) d -= c2;
    }
    return d;
}

template <typename T>
__device__ __forceinline__ typename PairT<T>::type sor_bpair(const Op& op, int i, int j, int k, bool ug) {
    return PairT<T>::make(sor_bval<T>(op, i, j, k, ug), sor_bval<T>(op, i + 1, j, k, ug));
}

// Tile configuration: extended tile of PXN pairs x EY rows (threads in use = PXN * EY), NHS colour half-steps per pass.
// NACT <= NHS of the half-steps do work (the rest are no-ops that only delay the plane: the three-half-step symmetric
// Gauss-Seidel sweep of the CG preconditioner runs in the four-half-step geometry, whose even depth the colour
// bookkeeping needs); the y halo is NACT rows, the x halo stays NHS columns (16-byte pairs start at even columns).
// ZIN: the input field is known to be zero and is not read.  DOT: the kernel also forms sum rhs . out over the grid
// (r . z of preconditioned CG) from the values it holds when it stores a plane.
template <int NHS_, int PXN_, int EY_, int PF_ = 1, int NACT_ = NHS_, bool ZIN_ = false, bool DOT_ = false>
struct SorTile {
    static constexpr int NHS = NHS_, PXN = PXN_, EY = EY_, PF = PF_;  // PF = planes of load prefetch (1 or 2)
    static constexpr int NACT = NACT_, HY = NACT_;
    static constexpr bool ZIN = ZIN_, DOT = DOT_;
    static constexpr int D = NHS + 2;                       // queue depth = ring slots
    static constexpr int NT = ((PXN * EY + 31) / 32) * 32;  // threads per CTA
    static constexpr int SW = 2 * PXN, SLOT = SW * EY;
    static constexpr int VX = 2 * PXN - 2 * NHS, VY = EY - 2 * HY;
    static constexpr int MINB = (NT <= 320) ? 2 : 1;  // fp64 needs ~105 registers per thread
};

// One overrelaxation factor per colour half-step of the pass (constant omega: all equal; the Chebyshev sequence of
// PAPER.md:81-88 Eq. 6: consecutive members; a factor of 0 turns a half-step into a no-op, which makes the
// red-black-red symmetric Gauss-Seidel sweep of the CG preconditioner out of a four-half-step pass).
template <typename T>
struct OmegaSet {
    T w[4];
};

template <typename T, class Cfg, bool PLAIN>
__global__ void __launch_bounds__(Cfg::NT, Cfg::MINB)
    k_sor_fused(const Op op, const T* __restrict__ in, T* __restrict__ out, const T* __restrict__ rhs,
                const OmegaSet<T> om, const bool ug_in, const SorGeom g, KrylovCtl* const ctl, const RedBuf rb) {
    using P2 = typename PairT<T>::type;
    constexpr int NHS = Cfg::NHS, D = Cfg::D, SW = Cfg::SW, SLOT = Cfg::SLOT, PXN = Cfg::PXN, EY = Cfg::EY;
    extern __shared__ __align__(16) unsigned char smraw[];
    T* const ring = reinterpret_cast<T*>(smraw);
    const int n0 = op.n[0], n1 = op.n[1], n2 = op.n[2];
    const int tid = threadIdx.x;
    const bool live = tid < PXN * EY;  // threads padding the last warp only take part in the barriers
    const int lx = live ? tid % PXN : 0, ly = live ? tid / PXN : 0;
    const bool ug = ug_in && op.gamma == 0.0;
    const T c0 = (T)op.c[0], c1 = (T)op.c[1], c2 = (T)op.c[2];
    const T dplain = (T)2 * ((c0 + c1) + c2);
    const T rdplain = (T)1 / dplain;
    const size_t plane = (size_t)n0 * n1;
    // Shared-memory planes are stored de-interleaved: row = [even columns | odd columns], so that the 8-byte reads of
    // one column parity by consecutive lanes are consecutive words (no bank conflicts; the interleaved layout had 2-way)
    T* const mine = ring + ly * SW + lx;  // column 0 of this thread's pair in slot 0; column 1 is PXN words further

    [[maybe_unused]] double dot = 0.0;
    const long total = (long)g.ntx * g.nty * n2;
    long pos = (long)blockIdx.x * g.items;
    const long end = min(total, pos + g.items);
    while (pos < end) {
        const int t = (int)(pos / n2), k0 = (int)(pos % n2);
        const int k1 = (int)min((long)n2, (long)k0 + (end - pos));
        pos += k1 - k0;
        const int tx = t % g.ntx, ty = t / g.ntx;
        const int i = tx * Cfg::VX - NHS + 2 * lx, j = ty * Cfg::VY - Cfg::HY + ly;
        const bool col_in = live && i >= 0 && i < n0 && j >= 0 && j < n1;
        const bool st_ok = col_in && i >= tx * Cfg::VX && i < (tx + 1) * Cfg::VX && j >= ty * Cfg::VY &&
                           j < (ty + 1) * Cfg::VY;
        // Column A of the pair is the one updated when kin is even, column B when kin is odd:
        // (i + c + j + kin) odd with i even  ->  cA = 1 - (j & 1).
        const int cA = 1 - (j & 1);
        // shared-memory offsets (relative to `mine`) of each column's own cell and of its three outside neighbours
        const int selfA = cA * PXN, selfB = (1 - cA) * PXN;
        // outer x neighbour: left of column 0 = column 1 of the pair to the left; right of column 1 = column 0 of the next
        const int xo0 = lx > 0 ? PXN - 1 : 0, xo1 = lx < PXN - 1 ? 1 : PXN;
        const int xoA = cA ? xo1 : xo0, xoB = cA ? xo0 : xo1;
        const int ymA = selfA + (ly > 0 ? -SW : 0), ypA = selfA + (ly < EY - 1 ? SW : 0);
        const int ymB = selfB + (ly > 0 ? -SW : 0), ypB = selfB + (ly < EY - 1 ? SW : 0);
        T* const mineA = mine + selfA;
        T* const mineB = mine + selfB;
        T dA = dplain, dB = dplain, rdA = rdplain, rdB = rdplain;
        if (!PLAIN && col_in) {
            dA = sor_diag_xy<T>(op, i + cA, j);
            dB = sor_diag_xy<T>(op, i + 1 - cA, j);
            rdA = (T)1 / dA;
            rdB = (T)1 / dB;
        }
        const int kbeg = max(k0 - NHS, -1), kend = k1 - 1 + NHS;
        const int kstart = kbeg & ~1;  // even: column A is the active one in unrolled iterations 0, 2, ...
        // Where this thread's pair of plane kk comes from: kind 1 = the array itself (16-byte load), kinds 2 / 3 = one
        // ghost-face value per plane into .y / .x (the pair straddles an x face), kind 4 = a pair of a y ghost face,
        // kind 0 = nothing.  One pointer + one stride per thread; planes -1 and n2 of in-domain columns are the z faces.
        int kind = 0;
        const T* vp = in;
        ptrdiff_t vs = 0;
        if (col_in) {
            kind = 1;
            vp = in + (size_t)j * n0 + i;
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
        vp += (ptrdiff_t)kstart * vs;  // vp / prh always point at the next plane to load
        const T* prh = rhs + (col_in ? (size_t)j * n0 + i : 0) + (ptrdiff_t)kstart * (ptrdiff_t)plane;
        T* pout = out + (col_in ? (size_t)j * n0 + i : 0) + ((ptrdiff_t)kstart - NHS - 1) * (ptrdiff_t)plane;
        // vp / prh point at plane kk (the next plane to load); they are only dereferenced when that plane exists
        auto loadv = [&](int kk) -> P2 {
            P2 v = PairT<T>::make((T)0, (T)0);
            if (Cfg::ZIN) return v;
            if (kk >= 0 && kk < n2) {
                if (kind == 1 || kind == 4) v = *reinterpret_cast<const P2*>(vp);
                else if (kind == 2) v.y = *vp;
                else if (kind == 3) v.x = *vp;
            } else if (kk == -1) {
                if (zlo) v = *reinterpret_cast<const P2*>(zlo);
            } else if (kk == n2) {
                if (zhi) v = *reinterpret_cast<const P2*>(zhi);
            }
            return v;
        };
        auto loadr = [&](int kk) -> P2 {
            if (kind == 1 && kk >= 0 && kk < n2) return *reinterpret_cast<const P2*>(prh);
            return PairT<T>::make((T)0, (T)0);
        };
        // the same loads for a plane known to exist (FAST blocks)
        auto loadv_in = [&]() -> P2 {
            P2 v = PairT<T>::make((T)0, (T)0);
            if (Cfg::ZIN) return v;
            if (kind == 1 || kind == 4) v = *reinterpret_cast<const P2*>(vp);
            else if (kind == 2) v.y = *vp;
            else if (kind == 3) v.x = *vp;
            return v;
        };
        auto loadr_in = [&]() -> P2 {
            if (kind == 1) return *reinterpret_cast<const P2*>(prh);
            return PairT<T>::make((T)0, (T)0);
        };
        // register queues; the value of plane kin - m sits at index (m - u) mod D in unrolled iteration u
        T qA[D], qB[D], fA[D], fB[D];
#pragma unroll
        for (int m = 0; m < D; ++m) qA[m] = qB[m] = fA[m] = fB[m] = (T)0;
        // loads run PF planes ahead of their use: nvq[m] / nrq[m] hold plane (next plane to consume) + m
        constexpr int PF = Cfg::PF;
        P2 nvq[PF], nrq[PF];
#pragma unroll
        for (int m = 0; m < PF; ++m) {
            nvq[m] = loadv(kstart + m);
            nrq[m] = loadr(kstart + m);
            vp += vs;
            prh += plane;
        }
        __syncthreads();  // the previous segment's readers are done with the ring
        // One block = D unrolled iterations.  FAST blocks lie strictly inside the z range (every plane touched exists,
        // none is a boundary plane, every finished plane belongs to this run): no range tests, no z-closure of the
        // diagonal — the same arithmetic with ~20 % fewer instructions; the lead-in / lead-out blocks take the full path.
        auto block = [&](auto fast_tag, const int kin0) {
            constexpr bool FAST = decltype(fast_tag)::value;
#pragma unroll
            for (int u = 0; u < D; ++u) {
                const int kin = kin0 + u;
                if (!FAST && kin > kend) break;
                const int p0 = (D - u) % D;  // index of plane kin (m = 0)
                const P2 nv = nvq[u % PF], nr = nrq[u % PF];
                qA[p0] = cA ? nv.y : nv.x;
                qB[p0] = cA ? nv.x : nv.y;
                fA[p0] = cA ? nr.y : nr.x;
                fB[p0] = cA ? nr.x : nr.y;
                if (live) {  // slot of plane kin is u
                    mine[u * SLOT] = nv.x;
                    mine[u * SLOT + PXN] = nv.y;
                }
                pout += plane;
                if (FAST) {
                    nvq[u % PF] = loadv_in();
                    nrq[u % PF] = loadr_in();
                } else if (kin + PF <= kend) {
                    nvq[u % PF] = loadv(kin + PF);
                    nrq[u % PF] = loadr(kin + PF);
                }
                vp += vs;
                prh += plane;
                __syncthreads();
                // (1) everything that does not depend on this iteration's updates: the shared-memory neighbours belong
                // to columns that are not updated now, so the x/y part of every half-step can be formed up front
                const bool actA = (u % 2) == 0;
                T sxy[NHS];
#pragma unroll
                for (int h = 1; h <= Cfg::NACT; ++h) {
                    const T* const sp = mine + ((u - h + D) % D) * SLOT;
                    const int ph = (h - u + 2 * D) % D;
                    const T partner = actA ? qB[ph] : qA[ph];
                    const T outer = sp[actA ? xoA : xoB];
                    const T ym = sp[actA ? ymA : ymB], yp = sp[actA ? ypA : ypB];
                    sxy[h - 1] = fma_(ym + yp, c1, (outer + partner) * c0);
                }
                // (2) the dependent chain plane kin-1 -> kin-2 -> ... through the z neighbours, in registers
#pragma unroll
                for (int h = 1; h <= Cfg::NACT; ++h) {
                    const int kz = kin - h;
                    const bool upd = FAST ? col_in : (col_in && kz >= 0 && kz < n2);
                    const int ph = (h - u + 2 * D) % D, pm = (h + 1 - u + 2 * D) % D, pp = (h - 1 - u + 2 * D) % D;
                    const T zp = actA ? qA[pp] : qB[pp], zm = actA ? qA[pm] : qB[pm];
                    const T old = actA ? qA[ph] : qB[ph];
                    const T f = actA ? fA[ph] : fB[ph];
                    T d = PLAIN ? dplain : (actA ? dA : dB), rd = PLAIN ? rdplain : (actA ? rdA : rdB);
                    if (!PLAIN && !FAST && (kz == 0 || kz == n2 - 1)) {
                        d = sor_diag_z<T>(op, d, kz);
                        rd = (T)1 / d;
                    }
                    const T s = fma_(zm + zp, c2, sxy[h - 1]);
                    const T gs = div_by<T>(s - f, d, rd);
                    const T nw = fma_(om.w[h - 1], gs - old, old);
                    if (upd) {
                        if (actA) qA[ph] = nw; else qB[ph] = nw;
                        (actA ? mineA : mineB)[((u - h + D) % D) * SLOT] = nw;
                    }
                }
                const int ko = kin - NHS;
                if (FAST ? st_ok : (st_ok && ko >= k0 && ko < k1)) {
                    const int po = (NHS - u + 2 * D) % D;
                    *reinterpret_cast<P2*>(pout) = cA ? PairT<T>::make(qB[po], qA[po]) : PairT<T>::make(qA[po], qB[po]);
                    if constexpr (Cfg::DOT) dot = fma((double)fB[po], (double)qB[po], fma((double)fA[po], (double)qA[po], dot));
                }
            }
        };
        for (int kin0 = kstart; kin0 <= kend; kin0 += D) {
            const bool fast = kin0 - NHS >= 1 && kin0 + D - 1 + PF <= n2 - 1 && kin0 + D - 1 + PF <= kend &&
                              kin0 - NHS >= k0 && kin0 + D - 1 - NHS < k1;
            if (fast) block(FastTag<true>{}, kin0);
            else block(FastTag<false>{}, kin0);
        }
    }
    if constexpr (Cfg::DOT) {  // beta = rz_new / rz_old (0 before the first iteration), Saad Alg. 9.1
        double vals[1] = {dot};
        grid_reduce<1>(vals, rb, [=](const double* t) {
            if (ctl->done) return;
            const double rz_new = t[0];
            if (!isfinite(rz_new) || rz_new == 0.0) {
                ctl->done = 1;
                ctl->status = POISSON_BREAKDOWN;
                return;
            }
            ctl->beta = ctl->it == 0 ? 0.0 : rz_new / ctl->rz;
            ctl->rz = rz_new;
        });
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------------
template <class Cfg>
static double sor_cfg_cost(const poisson_ctx* ctx, const Op& op, size_t esize, SorGeom* g, int* grid) {
    SorGeom s;
    s.pxn = Cfg::PXN;
    s.ey = Cfg::EY;
    s.vx = Cfg::VX;
    s.vy = Cfg::VY;
    s.ntx = (op.n[0] + Cfg::VX - 1) / Cfg::VX;
    s.nty = (op.n[1] + Cfg::VY - 1) / Cfg::VY;
    const size_t smem = (size_t)Cfg::D * Cfg::SLOT * esize;
    const int per_sm = std::max(1, std::min(Cfg::MINB, (int)((220 * 1024) / smem)));
    if (Cfg::NT > 1024 || smem > 220 * 1024) return 1e300;
    const long slots = (long)ctx->num_sms * per_sm;
    const long total = (long)s.ntx * s.nty * op.n[2];
    s.items = std::max(1L, (total + slots - 1) / slots);
    const long ctas = (total + s.items - 1) / s.items;
    const long conc = std::min<long>(per_sm, (ctas + ctx->num_sms - 1) / ctx->num_sms);
    *g = s;
    *grid = (int)ctas;
    // time per plane ~ threads per SM; narrow tiles move shorter row segments (measured ~15 % slower per point)
    // (the constant stands for the planes a run spends filling and draining the wavefront)
    return (double)(s.items + 2 * Cfg::NHS + 8) * Cfg::NT * conc * (Cfg::PXN < 32 ? 1.2 : 1.0);
}

template <typename T, class Cfg>
static int sor_launch_cfg(poisson_ctx* ctx, const Op& op, const T* in, T* out, const T* rhs, const OmegaSet<T>& omega,
                          bool ug, const SorGeom& g, int grid) {
    bool plain = op.gamma == 0.0;
    for (int f = 0; f < 6; ++f) plain = plain && op.bc[f] != POISSON_BC_NEUMANN0;
    const size_t smem = (size_t)Cfg::D * Cfg::SLOT * sizeof(T);
    if (Cfg::DOT && grid > kMaxRedBlocks) return POISSON_UNSUPPORTED;
    int rc = kernel_ready(ctx, k_sor_fused<T, Cfg, true>, Cfg::NT, smem);
    if (rc == POISSON_OK) rc = kernel_ready(ctx, k_sor_fused<T, Cfg, false>, Cfg::NT, smem);
    if (rc != POISSON_OK) return rc;
    if (plain)
        PB_LAUNCH(ctx, KID_RBSOR, (k_sor_fused<T, Cfg, true><<<grid, Cfg::NT, smem, ctx->stream>>>(op, in, out, rhs, omega, ug, g, ctx->d_ctl, ctx->red)));
    else
        PB_LAUNCH(ctx, KID_RBSOR, (k_sor_fused<T, Cfg, false><<<grid, Cfg::NT, smem, ctx->stream>>>(op, in, out, rhs, omega, ug, g, ctx->d_ctl, ctx->red)));
    return POISSON_OK;
}

// Tile choice: the compiled configuration with the smallest estimated pass time (POISSON_OPT_TILE_CFG overrides).
template <typename T, int NHS, int NACT = NHS, bool ZIN = false, bool DOT = false>
static int sor_fused_pass(poisson_ctx* ctx, const Op& op, const T* in, T* out, const T* rhs, const OmegaSet<T>& omega,
                          bool ug) {
    // Configuration 0 is sized for 7 warps per scheduler: the register file is split over the SM's four schedulers
    // (16384 registers each), so 25..28 warps all get 72 registers per thread and the kernel, which is latency-bound,
    // wants as many as fit.  Four half-steps: 36 x 24 threads = 27 warps, 64 x 16 valid (measured at 256^3, us per
    // sweep: 22 rows 109.4, 24 rows 99.5, 28 rows at 64 registers 104.3); two half-steps: 34 x 26 threads = 28 warps,
    // 64 x 22 valid (18 rows 136.0, 22 rows 124.9, 26 rows 108.5, 30 rows at 64 registers 115.2)
    constexpr int V0 = NHS == 4 ? (NACT < NHS ? 18 : 16) : 22;
    using C0 = SorTile<NHS, 32 + NHS, V0 + 2 * NACT, 1, NACT, ZIN, DOT>;  // 64 x V0 valid (best at 256^3 on B200)
    using C1 = SorTile<NHS, 16 + NHS, 28 + 2 * NACT, 1, NACT, ZIN, DOT>;  // 32 x 28 valid, 576 threads
    using C2 = SorTile<NHS, 16 + NHS, 10 + 2 * NACT, 1, NACT, ZIN, DOT>;  // 32 x 10 valid, 252 threads, two CTAs per SM
    using C3 = SorTile<NHS, 32 + NHS, 8 + 2 * NACT, 1, NACT, ZIN, DOT>;   // 64 x 8 valid, 408 threads
    SorGeom g[4];
    int grid[4];
    double cost[4] = {sor_cfg_cost<C0>(ctx, op, sizeof(T), &g[0], &grid[0]), sor_cfg_cost<C1>(ctx, op, sizeof(T), &g[1], &grid[1]),
                      sor_cfg_cost<C2>(ctx, op, sizeof(T), &g[2], &grid[2]), sor_cfg_cost<C3>(ctx, op, sizeof(T), &g[3], &grid[3])};
    int best = 0;
    for (int c = 1; c < 4; ++c)
        if (cost[c] < cost[best]) best = c;
    const int ov = ctx->opt_tile_cfg;
    if (ov >= 0 && ov < 4) best = ov;
    switch (best) {
        case 0: return sor_launch_cfg<T, C0>(ctx, op, in, out, rhs, omega, ug, g[0], grid[0]);
        case 1: return sor_launch_cfg<T, C1>(ctx, op, in, out, rhs, omega, ug, g[1], grid[1]);
        case 2: return sor_launch_cfg<T, C2>(ctx, op, in, out, rhs, omega, ug, g[2], grid[2]);
        default: return sor_launch_cfg<T, C3>(ctx, op, in, out, rhs, omega, ug, g[3], grid[3]);
    }
}

bool sor_fused_ok(const poisson_ctx* ctx, const Op& op) {
    if (ctx->opt_path == 1) return false;
    if (op.coord != POISSON_CARTESIAN || op.order != 2 || op.n[0] % 2 != 0) return false;
    for (int f = 0; f < 6; ++f)
        if (op.bc[f] == POISSON_BC_PERIODIC) return false;
    if (ctx->opt_path == 2) return true;
    return (size_t)op.n[0] * op.n[1] * op.n[2] >= (size_t)1 << 15;
}

// nsweeps full sweeps phi -> phi through the ping-pong buffer tmp (same size as phi).
// omegas == nullptr: the constant `omega`; else 2 nsweeps factors, one per colour half-sweep (red, black, red, ...).
template <typename T>
static int sor_fused_t(poisson_ctx* ctx, const Op& op, T* phi, T* tmp, const T* rhs, T omega, int nsweeps, bool ug,
                       T** result, const double* omegas = nullptr) {
    T *src = phi, *dst = tmp;
    int left = nsweeps;
    // two sweeps per pass (NHS = 4) pay from 2^21 points (128^3: 22.9 vs 24.8 us per sweep in fp64; 256^3: 109 vs 138;
    // 64^3: the same either way); 0 = this automatic choice
    const bool two = ctx->opt_sor_nhs == 4 ||
                     (ctx->opt_sor_nhs == 0 && (size_t)op.n[0] * op.n[1] * op.n[2] >= ((size_t)1 << 21));
    // Plan: n4 passes of two sweeps + n2 passes of one.  An odd number of passes ends in the ping-pong buffer and costs
    // a copy back (16 B/point): in fp64 one two-sweep pass is then split into two one-sweep passes instead
    // (measured: 2 x NHS=2 beats NHS=4 + copy at 256^3; in fp32 the single pass + copy is the faster one).
    int n4 = two ? nsweeps / 2 : 0;
    if (!result && sizeof(T) == 8 && n4 > 0 && ((n4 + (nsweeps - 2 * n4)) & 1)) --n4;
    int half = 0;  // colour half-sweeps done so far
    while (left > 0) {
        int rc;
        OmegaSet<T> os;
        for (int h = 0; h < 4; ++h) os.w[h] = omegas ? (half + h < 2 * nsweeps ? (T)omegas[half + h] : (T)0) : omega;
        if (n4 > 0) {
            --n4;
            rc = sor_fused_pass<T, 4>(ctx, op, src, dst, rhs, os, ug);
            left -= 2;
            half += 4;
        } else {
            rc = sor_fused_pass<T, 2>(ctx, op, src, dst, rhs, os, ug);
            left -= 1;
            half += 2;
        }
        if (rc != POISSON_OK) return rc;
        std::swap(src, dst);
    }
    PB_CUDA_OK(cudaGetLastError());
    if (result) {
        *result = src;  // the caller carries on with whichever buffer holds the result (V-cycle: no copy back)
    } else if (src != phi) {
        const size_t bytes = (size_t)op.n[0] * op.n[1] * op.n[2] * sizeof(T);
        PB_CUDA_OK(cudaMemcpyAsync(phi, src, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    }
    return POISSON_OK;
}

int sor_fused(poisson_ctx* ctx, const Op& op, double* phi, double* tmp, const double* rhs, double omega, int nsweeps,
              bool ug, double** result) {
    return sor_fused_t<double>(ctx, op, phi, tmp, rhs, omega, nsweeps, ug, result);
}
int sor_fused_seq(poisson_ctx* ctx, const Op& op, double* phi, double* tmp, const double* rhs, const double* omegas,
                  int nsweeps, bool ug, double** result) {
    return sor_fused_t<double>(ctx, op, phi, tmp, rhs, 1.0, nsweeps, ug, result, omegas);
}
// z = (symmetric ? red-black-red : red-black) Gauss-Seidel sweep on L z = f from z = 0 (zin must hold zeros): the
// multi-colour preconditioner of PAPER.md:107-123 Eq. 10 in ONE pass over HBM.  The result lands in zout.
// with_rz: the pass also leaves r . z and beta in the Krylov control block (what k_pcg_dot does as a pass of its own).
int sor_fused_precond(poisson_ctx* ctx, const Op& op, const double* zin, double* zout, const double* f, bool symmetric,
                      bool with_rz) {
    OmegaSet<double> os;
    os.w[0] = os.w[1] = 1.0;
    os.w[2] = symmetric ? 1.0 : 0.0;
    os.w[3] = 0.0;
    if (with_rz && !symmetric) return POISSON_INVALID_ARG;
    const int rc = !symmetric ? sor_fused_pass<double, 2, 2, true>(ctx, op, zin, zout, f, os, false)
                   : with_rz  ? sor_fused_pass<double, 4, 3, true, true>(ctx, op, zin, zout, f, os, false)
                              : sor_fused_pass<double, 4, 3, true>(ctx, op, zin, zout, f, os, false);
    if (rc != POISSON_OK) return rc;
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}
int sor_fused32(poisson_ctx* ctx, const Op& op, float* phi, float* tmp, const float* rhs, float omega, int nsweeps,
                float** result) {
    return sor_fused_t<float>(ctx, op, phi, tmp, rhs, omega, nsweeps, false, result);
}

}  // namespace pb
