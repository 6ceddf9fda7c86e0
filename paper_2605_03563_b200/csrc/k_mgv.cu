// k_mgv.cu — the paper's own multigrid on vertex-centred grids of 2^N k - 1 points per axis:
//   SPAI smoother   x <- x + omega M (b - A x), M = h^2 {alpha | beta faces | gamma edges | delta corners}   PAPER.md:154-184 Eq. 15-16, Table 1
//   full weighting  R = (1/4 [1 2 1])^(x)3, P = 8 R^T (trilinear)                                         PAPER.md:138-142 Eq. 13
//   Galerkin        A_{l+1} = R A_l P, radius one                                                         PAPER.md:144-150 Eq. 14
//   coarsest level  CG
//   mixed precision coarse-level data stored in fp32, all arithmetic in fp64
// A is the paper's SPD matrix (A = -L_h), b = -rhs.  The operator has constant coefficients and zero Dirichlet values
// on the boundary vertices of every level (level 0: the ghost values are folded into the right-hand side once per
// call), so every Galerkin product is one fully symmetric 27-point stencil: four numbers per level
// (centre | face | edge | corner), formed on the device from the definition R A P.
//
// Hot kernel k_spai: one pass over HBM per smoothing step (read x, b; write x: 24 B/point in fp64, 12 in fp32 storage).
// A CTA of 32 x NTY threads owns an xy tile of 32 x (NTY RY) residual points (output tile + 1 halo) and marches z; a
// thread owns RY consecutive rows of one column.  Both 27-point applications are evaluated from in-plane sums,
//   Q0 = v(c), Q1 = sum of the 4 in-plane face neighbours, Q2 = sum of the 4 in-plane diagonal neighbours,
//   (S v)(k) = C(k) + U(k-1) + U(k+1),  C = s0 Q0 + s1 Q1 + s2 Q2,  U = s1 Q0 + s2 Q1 + s3 Q2,
// so a plane contributes to three output planes through two numbers per point, the running sums live in registers
// along z (two doubles per point and operator), only ONE plane of x and ONE plane of r is shared at a time
// (double-buffered, two barriers per plane), and the in-plane sums of the RY rows share their row loads:
// 3 (RY + 2) / RY shared-memory loads per point and operator instead of 27.
#include <algorithm>
#include <functional>

#include "stencil.cuh"

namespace pb {

namespace mgv {

constexpr int NTX = 32, NTY = 8, RY = 3;   // threads; rows per thread (ms per SPAI step at 255^3 / 511^3, 7-point A: 8x3 0.143 / 0.900, 8x2 0.140 / 0.920, 8x4 0.177 / 1.259 (128 registers, two CTAs per SM); V(1,1) cycle 0.728 / 3.81, 0.744 / 4.01, 0.902 / 5.10; earlier: 4x4, 16x1, 16x2 all 13-25 % behind 8x2)
constexpr int TY = NTY * RY;               // residual tile NTX x TY; output tile (NTX-2) x (TY-2)
constexpr int VX = NTX - 2, VY = TY - 2;
constexpr int XW = NTX + 2, XH = TY + 2;   // x plane with its halo (and the r plane with an unused zero border)
constexpr int NHALO = 2 * XW + 2 * TY;     // ring of x points around the residual tile
constexpr int NT = NTX * NTY;

template <typename S>
__device__ __forceinline__ double ldv(const S* p) { return (double)*p; }

struct Plan {
    int n0, n1, n2;
    int ntx, nty, nz, kc;  // tiles and z chunks (MODE 2: chunks of kc COARSE planes)
    int nc0, nc1, nc2;     // MODE 2: the coarse grid
};

constexpr int NS = 5, PD = 3;  // planes in the staging rings; loads run PD planes ahead (a slot is reused NS - PD = 2 barriers later)

// 4- or 8-byte asynchronous copy global -> shared (LDGSTS); `ok` false zero-fills the destination instead.
template <typename S>
__device__ __forceinline__ void cp_async_fast(unsigned d, const void* gsrc) {  // d: shared-window address
    if constexpr (sizeof(S) == 8)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
template <typename S>
__device__ __forceinline__ void cp_async(S* smem_dst, const S* gsrc, bool ok) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int nbytes = ok ? (int)sizeof(S) : 0;
    if constexpr (sizeof(S) == 8)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(gsrc), "r"(nbytes) : "memory");
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(d), "l"(gsrc), "r"(nbytes) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// In-plane sums of the RY owned rows from a shared plane (row pitch XW): rows row0 .. row0+RY+1, columns tx .. tx+2.
template <typename S>
__device__ __forceinline__ void plane_sums(const S* pl, int tx, int row0, double (&q0)[RY], double (&q1)[RY],
                                           double (&q2)[RY], bool want_q2) {
    double h[RY + 2], c[RY + 2];
#pragma unroll
    for (int w = 0; w < RY + 2; ++w) {
        const S* rowp = pl + (row0 + w) * XW;
        c[w] = (double)rowp[tx + 1];
        h[w] = (double)rowp[tx] + (double)rowp[tx + 2];
    }
#pragma unroll
    for (int r = 0; r < RY; ++r) {
        q0[r] = c[r + 1];
        q1[r] = h[r + 1] + (c[r] + c[r + 2]);
        q2[r] = want_q2 ? h[r] + h[r + 2] : 0.0;
    }
}

template <typename SX, typename SB>
constexpr size_t spai_smem() {
    return (size_t)NS * XH * XW * sizeof(SX) + (size_t)NS * TY * NTX * sizeof(SB) + (size_t)2 * XH * XW * sizeof(double);
}

// MODE 0: out = x + omega M (bsign b - A x)      (one SPAI step, Eq. 15)
// MODE 1: out = bsign b - A x                    (residual)
// MODE 2: out = R (bsign b - A x) on the coarse grid (residual + full weighting Eq. 13 in one pass: the fine residual
//         never goes to memory; the in-plane part of R is the same partial sums, W = P0/4 + P1/8 + P2/16 at the fine
//         vertices that carry a coarse vertex, and b_c(K) = W(2K)/4 + W(2K+1)/2 + W(2K+2)/4 is a running sum along z)
// SEVEN: A has no edge / corner coefficients (level 0: the 7-point operator).
// Planes of x (with halo) and b are staged by asynchronous copies PD planes ahead of their use: no staging registers,
// PD planes of loads in flight per CTA.
template <typename SX, typename SB, typename SO, int MODE, bool SEVEN>
__global__ void __launch_bounds__(NT)
    k_spai(const Plan pl, const SX* __restrict__ x, const SB* __restrict__ b, SO* __restrict__ out,
           const double* __restrict__ a4 /* A: centre, face, edge, corner */, const double bsign, const double omega,
           const double m0, const double m1, const double m2, const double m3) {
    extern __shared__ __align__(16) unsigned char smraw[];
    double* const rs = reinterpret_cast<double*>(smraw);                       // [2][XH][XW]
    SX* const xs = reinterpret_cast<SX*>(rs + 2 * XH * XW);                    // [NS][XH][XW]
    SB* const bs = reinterpret_cast<SB*>(xs + NS * XH * XW);                   // [NS][TY][NTX]
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * NTX + tx;
    const int tile = blockIdx.x % (pl.ntx * pl.nty), zc = blockIdx.x / (pl.ntx * pl.nty);
    const int i0 = (tile % pl.ntx) * VX, j0 = (tile / pl.ntx) * VY;
    // output planes [k0, k1): fine planes (MODE 0, 1) or coarse planes (MODE 2); r planes needed: [kr_first, kr_last]
    const int k0 = zc * pl.kc, k1 = min(MODE == 2 ? pl.nc2 : pl.n2, k0 + pl.kc);
    const int kr_first = MODE == 0 ? k0 - 1 : (MODE == 1 ? k0 : 2 * k0);
    const int kr_last = MODE == 0 ? k1 : (MODE == 1 ? k1 - 1 : 2 * k1);
    const int n0 = pl.n0, n1 = pl.n1, n2 = pl.n2;
    const int i = i0 - 1 + tx, jb = j0 - 1 + ty * RY;  // this thread's residual points: (i, jb + r)
    const size_t plane = (size_t)n0 * n1;
    bool in[RY], owner[RY];
    size_t col[RY];
#pragma unroll
    for (int r = 0; r < RY; ++r) {
        const int j = jb + r, row = ty * RY + r;
        in[r] = i >= 0 && i < n0 && j >= 0 && j < n1;
        owner[r] = in[r] && tx >= 1 && tx <= VX && row >= 1 && row <= VY;
        col[r] = in[r] ? (size_t)j * n0 + i : 0;
    }
    // this thread's halo point of the x plane (ring around the residual tile), if any
    int hx = -1, hy = -1;
    if (tid < NHALO) {
        if (tid < XW) { hx = tid; hy = 0; }
        else if (tid < 2 * XW) { hx = tid - XW; hy = XH - 1; }
        else if (tid < 2 * XW + TY) { hx = 0; hy = 1 + tid - 2 * XW; }
        else { hx = XW - 1; hy = 1 + tid - 2 * XW - TY; }
    }
    const int hi = i0 - 2 + hx, hj = j0 - 2 + hy;
    const bool hin = hx >= 0 && hi >= 0 && hi < n0 && hj >= 0 && hj < n1;
    const size_t hcol = hin ? (size_t)hj * n0 + hi : 0;
    const double s0 = a4[0], s1 = a4[1], s2 = SEVEN ? 0.0 : a4[2], s3 = SEVEN ? 0.0 : a4[3];
    for (int e = tid; e < 2 * XH * XW; e += NT) rs[e] = 0.0;  // the border of the r planes stays zero

    // stage x plane kk (own points + halo ring) and b plane kk-1 (consumed in the same iteration) into ring slot
    // `slot` (= kk mod NS); planes outside the grid and points outside the domain are zero-filled.  One commit group
    // per call, always (uniform group counting).  The slot written in iteration kx was last read in iteration kx-2:
    // the barrier of iteration kx-1 lies in between.  Tiles whose points (halo ring included) all lie in the domain
    // take a path without per-copy predicates when both planes exist.
    bool tile_inside = hx < 0 || hin;
#pragma unroll
    for (int r = 0; r < RY; ++r) tile_inside = tile_inside && in[r];
    tile_inside = __syncthreads_and(tile_inside);
    SX* const xown = xs + (ty * RY + 1) * XW + tx + 1;
    SB* const bown = bs + (ty * RY) * NTX + tx;
    SX* const xhal = xs + (hx >= 0 ? hy * XW + hx : 0);
    // fast path state: shared-window addresses of slot 0 and running global pointers of the next plane to stage
    const unsigned sx0 = (unsigned)__cvta_generic_to_shared(xown), sb0 = (unsigned)__cvta_generic_to_shared(bown),
                   sh0 = (unsigned)__cvta_generic_to_shared(xhal);
    const int kx0 = kr_first - 1;
    const char* gx = reinterpret_cast<const char*>(x) + ((ptrdiff_t)kx0 * (ptrdiff_t)plane + (ptrdiff_t)col[0]) * (ptrdiff_t)sizeof(SX);
    const char* gh = reinterpret_cast<const char*>(x) + ((ptrdiff_t)kx0 * (ptrdiff_t)plane + (ptrdiff_t)hcol) * (ptrdiff_t)sizeof(SX);
    const char* gb = reinterpret_cast<const char*>(b) + ((ptrdiff_t)(kx0 - 1) * (ptrdiff_t)plane + (ptrdiff_t)col[0]) * (ptrdiff_t)sizeof(SB);
    const size_t pbx = plane * sizeof(SX), pbb = plane * sizeof(SB), rbx = (size_t)n0 * sizeof(SX), rbb = (size_t)n0 * sizeof(SB);
    // stage(kk, slot) must be called for consecutive kk starting at kx0 (the running pointers advance by one plane)
    auto stage = [&](int kk, int slot) {
        const bool kin = kk >= 0 && kk < n2, kbin = kk - 1 >= 0 && kk - 1 < n2;
        if (tile_inside && kin && kbin) {
            const unsigned ox = slot * (unsigned)(XH * XW * sizeof(SX)), ob = slot * (unsigned)(TY * NTX * sizeof(SB));
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                cp_async_fast<SX>(sx0 + ox + r * (unsigned)(XW * sizeof(SX)), gx + r * rbx);
                cp_async_fast<SB>(sb0 + ob + r * (unsigned)(NTX * sizeof(SB)), gb + r * rbb);
            }
            if (hx >= 0) cp_async_fast<SX>(sh0 + ox, gh);
        } else {
            SX* const xp = xown + slot * (XH * XW);
            SB* const bp = bown + slot * (TY * NTX);
            const size_t off = kin ? (size_t)kk * plane : 0, offb = kbin ? (size_t)(kk - 1) * plane : 0;
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                cp_async(xp + r * XW, x + off + col[r], kin && in[r]);
                cp_async(bp + r * NTX, b + offb + col[r], kbin && in[r]);
            }
            if (hx >= 0) cp_async(xhal + slot * (XH * XW), x + off + hcol, kin && hin);
        }
        gx += pbx;
        gh += pbx;
        gb += pbb;
        cp_commit();
    };

    double accA[RY], uA[RY], accM[RY], uM[RY], x1[RY], x2[RY];  // running sums along z; x of planes kx-1, kx-2
#pragma unroll
    for (int r = 0; r < RY; ++r) accA[r] = uA[r] = accM[r] = uM[r] = x1[r] = x2[r] = 0.0;
    const int kx_end = kr_last + 1;
    double accR[RY];  // MODE 2: running z sum of the restriction
#pragma unroll
    for (int r = 0; r < RY; ++r) accR[r] = 0.0;
#pragma unroll
    for (int d = 0; d < PD; ++d) stage(kx0 + d, d);
    int slot = 0, slot_pd = PD;  // ring slots of planes kx and kx + PD
    size_t oo = (size_t)(kx0 - (MODE == 0 ? 2 : 1)) * plane;  // offset of the fine plane written in this iteration (MODE 0, 1)
    for (int kx = kx0; kx <= kx_end; ++kx, oo += plane) {
        stage(kx + PD, slot_pd);
        cp_wait<PD>();   // everything up to plane kx has landed (this thread's copies)
        __syncthreads();  // ... and everybody else's
        const SX* const xp = xs + slot * (XH * XW);
        const SB* const bp = bs + slot * (TY * NTX);
        slot = slot + 1 == NS ? 0 : slot + 1;
        slot_pd = slot_pd + 1 == NS ? 0 : slot_pd + 1;
        const int par = kx & 1;
        double q0[RY], q1[RY], q2[RY], rv[RY];
        plane_sums<SX>(xp, tx, ty * RY, q0, q1, q2, !SEVEN);
        const int kr = kx - 1;
        const bool krin = kr >= 0 && kr < n2;
#pragma unroll
        for (int r = 0; r < RY; ++r) {
            // residual of plane kx-1 (zero outside the domain: Dirichlet vertices carry no residual)
            double u = s1 * q0[r], c = fma(s1, q1[r], s0 * q0[r]);
            if (!SEVEN) {
                u = fma(s3, q2[r], fma(s2, q1[r], u));
                c = fma(s2, q2[r], c);
            }
            const double ax = accA[r] + u;  // C(kx-1) + U(kx-2) + U(kx)
            accA[r] = c + uA[r];
            uA[r] = u;
            rv[r] = (in[r] && krin) ? bsign * (double)bp[(ty * RY + r) * NTX + tx] - ax : 0.0;
        }
        if (MODE == 1) {
#pragma unroll
            for (int r = 0; r < RY; ++r)
                if (owner[r] && kr >= k0 && kr < k1) out[oo + col[r]] = (SO)rv[r];
        } else if (MODE == 2) {
            double* const rp = rs + par * (XH * XW);
#pragma unroll
            for (int r = 0; r < RY; ++r) rp[(ty * RY + r + 1) * XW + tx + 1] = rv[r];
            __syncthreads();
            double p0[RY], p1[RY], p2[RY];
            plane_sums<double>(rp, tx, ty * RY, p0, p1, p2, true);
            const int K = kr >> 1;  // kr even: the plane between coarse planes K-1 and K; odd: the plane of coarse K
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                const double w = fma(0.0625, p2[r], fma(0.125, p1[r], 0.25 * p0[r]));
                if (kr & 1) {
                    accR[r] = fma(0.5, w, accR[r]);
                } else {
                    const int j = jb + r;
                    if (owner[r] && (i & 1) && (j & 1) && K - 1 >= k0 && K - 1 < k1)
                        out[((size_t)(K - 1) * pl.nc1 + (j >> 1)) * pl.nc0 + (i >> 1)] = (SO)fma(0.25, w, accR[r]);
                    accR[r] = 0.25 * w;
                }
            }
        } else {
            double* const rp = rs + par * (XH * XW);
#pragma unroll
            for (int r = 0; r < RY; ++r) rp[(ty * RY + r + 1) * XW + tx + 1] = rv[r];
            __syncthreads();
            double p0[RY], p1[RY], p2[RY];
            plane_sums<double>(rp, tx, ty * RY, p0, p1, p2, true);
            const int ko = kx - 2;
            const bool koin = ko >= k0 && ko < k1;
#pragma unroll
            for (int r = 0; r < RY; ++r) {
                const double u = fma(m3, p2[r], fma(m2, p1[r], m1 * p0[r]));
                const double c = fma(m2, p2[r], fma(m1, p1[r], m0 * p0[r]));
                const double mr = accM[r] + u;  // (M r)(kx-2)
                accM[r] = c + uM[r];
                uM[r] = u;
                if (owner[r] && koin) out[oo + col[r]] = (SO)fma(omega, mr, x2[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < RY; ++r) {
            x2[r] = x1[r];
            x1[r] = q0[r];
        }
    }
    cp_wait<0>();
}

// x += P e_c, P = 8 R^T: odd fine indices sit on a coarse vertex, even ones half-way between two (zero beyond the boundary).
// One thread per coarse slot (I,J,K), 0 <= I <= nc: it reads the 2 x 2 x 2 coarse values e(I-1..I, J-1..J, K-1..K) once and
// updates its (up to) 8 fine points (2I+a, 2J+b, 2K+c): per axis an even fine index averages the two coarse
// neighbours, an odd one copies the coarse vertex it sits on.
template <typename SX, typename SE>
__global__ void __launch_bounds__(256)
    k_prolong27(int n0, int n1, int n2, int nc0, int nc1, int nc2, const SE* __restrict__ ec, SX* __restrict__ x) {
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    if (I > nc0 || J > nc1) return;
    double e[2][2][2];  // [gamma][beta][alpha]
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int bb = 0; bb < 2; ++bb)
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                const int Ic = I - 1 + a, Jc = J - 1 + bb, Kc = K - 1 + c;
                const bool ok = Ic >= 0 && Ic < nc0 && Jc >= 0 && Jc < nc1 && Kc >= 0 && Kc < nc2;
                e[c][bb][a] = ok ? ldv(ec + ((size_t)Kc * nc1 + Jc) * nc0 + Ic) : 0.0;
            }
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int bb = 0; bb < 2; ++bb)
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                const int i = 2 * I + a, j = 2 * J + bb, k = 2 * K + c;
                if (i >= n0 || j >= n1 || k >= n2) continue;
                // even index: both coarse neighbours (in the oracle's order: gamma, beta, alpha ascending); odd: the upper one
                double sum = 0.0;
#pragma unroll
                for (int g = (c ? 1 : 0); g < 2; ++g)
#pragma unroll
                    for (int bt = (bb ? 1 : 0); bt < 2; ++bt)
#pragma unroll
                        for (int al = (a ? 1 : 0); al < 2; ++al) sum += e[g][bt][al];
                const double w = (a ? 1.0 : 0.5) * (bb ? 1.0 : 0.5) * (c ? 1.0 : 0.5);
                const size_t p = ((size_t)k * n1 + j) * n0 + i;
                x[p] = (SX)(ldv(x + p) + sum * w);
            }
}

// Galerkin product of a constant symmetric 27-point stencil (Eq. 14 with P = 8 R^T), from its definition: entry O of
// R A P is sum over the restriction offset a and the operator offset d of R(a) A(d) P(a + d - 2 O).  One thread per O.
__global__ void k_galerkin27(const double* __restrict__ fine4, double* __restrict__ coarse4, int round_f32) {
    const int t = threadIdx.x;
    if (t >= 4) return;
    const int O[3] = {t >= 1 ? 1 : 0, t >= 2 ? 1 : 0, t >= 3 ? 1 : 0};  // centre, face, edge, corner representatives
    const double R1[3] = {0.25, 0.5, 0.25}, P1[3] = {0.5, 1.0, 0.5};
    double s = 0.0;
    for (int a2 = -1; a2 <= 1; ++a2)
        for (int a1 = -1; a1 <= 1; ++a1)
            for (int a0 = -1; a0 <= 1; ++a0)
                for (int d2 = -1; d2 <= 1; ++d2)
                    for (int d1 = -1; d1 <= 1; ++d1)
                        for (int d0 = -1; d0 <= 1; ++d0) {
                            const int f0 = a0 + d0 - 2 * O[0], f1 = a1 + d1 - 2 * O[1], f2 = a2 + d2 - 2 * O[2];
                            if (f0 < -1 || f0 > 1 || f1 < -1 || f1 > 1 || f2 < -1 || f2 > 1) continue;
                            const double ad = fine4[(d0 != 0) + (d1 != 0) + (d2 != 0)];
                            s += (R1[a0 + 1] * R1[a1 + 1] * R1[a2 + 1]) * ad * (P1[f0 + 1] * P1[f1 + 1] * P1[f2 + 1]);
                        }
    coarse4[t] = round_f32 ? (double)(float)s : s;
}

// Level 0 right-hand side with the Dirichlet boundary values folded in: bt = rhs - L_h [ghost-only field].
__global__ void __launch_bounds__(256) k_fold_ghosts(Op op, const double* __restrict__ rhs, double* __restrict__ bt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= op.n[0] || j >= op.n[1]) return;
    struct ZeroLd {
        __device__ __forceinline__ double operator()(size_t, int, int, int) const { return 0.0; }
    };
    const size_t p = gidx(op, i, j, k);
    double g = 0.0;
    if (i == 0 || j == 0 || k == 0 || i == op.n[0] - 1 || j == op.n[1] - 1 || k == op.n[2] - 1)
        g = row_offsum<double, KIND_CART2>(op, ZeroLd{}, i, j, k, true);
    bt[p] = rhs[p] - g;
}

// Right-hand side of the compact schemes (reading C19): out = B f with
//   order 4: B f = f + S1 f / 12;   order 6: B f = f + S1 f / 12 - (sum_a d_a^4 f) / 240 + S2 f / 90,
// S1 = sum_a d_a^2, S2 = sum_{a<b} d_a^2 d_b^2 (second differences), d_a^4 = (d_a^2)^2 reaching two points out.
// f_ext carries two extra layers per side: (n0+4)(n1+4)(n2+4) values.  One pass, done once per right-hand side.
template <int ORDER>
__global__ void __launch_bounds__(256)
    k_compact_rhs(int n0, int n1, int n2, const double* __restrict__ fe, double* __restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= n0 || j >= n1) return;
    const ptrdiff_t sx = 1, sy = n0 + 4, sz = (ptrdiff_t)(n0 + 4) * (n1 + 4);
    const double* const c = fe + (k + 2) * sz + (j + 2) * sy + (i + 2);
    const double f0 = c[0];
    double v = f0;
    if (ORDER >= 4) {
        const double s1 = fma(-6.0, f0, ((c[-sx] + c[sx]) + (c[-sy] + c[sy])) + (c[-sz] + c[sz]));
        v = fma(s1, 1.0 / 12.0, v);
    }
    if (ORDER == 6) {
        auto d4 = [&](ptrdiff_t s) { return fma(6.0, f0, fma(-4.0, c[-s] + c[s], c[-2 * s] + c[2 * s])); };
        auto d22 = [&](ptrdiff_t a, ptrdiff_t b) {
            const double corners = (c[-a - b] + c[a + b]) + (c[-a + b] + c[a - b]);
            const double faces = (c[-a] + c[a]) + (c[-b] + c[b]);
            return fma(4.0, f0, fma(-2.0, faces, corners));
        };
        v = fma(-(d4(sx) + d4(sy) + d4(sz)), 1.0 / 240.0, v);
        v = fma(d22(sx, sy) + d22(sy, sz) + d22(sz, sx), 1.0 / 90.0, v);
    }
    out[((size_t)k * n1 + j) * n0 + i] = v;
}

__global__ void __launch_bounds__(256) k_norm2(size_t n, const double* __restrict__ r, double* scal, RedBuf rb) {
    double s = 0.0;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x)
        s = fma(r[q], r[q], s);
    double vals[1] = {s};
    grid_reduce<1>(vals, rb, [=](const double* t) { scal[0] = t[0]; });
}

// Coarsest level: CG (Saad Alg. 6.18) from e = 0 in ONE CTA, vectors in shared memory, to ||r|| <= rtol ||b|| or max_it.
template <typename S>
__global__ void __launch_bounds__(512)
    k_cg_coarse27(int n0, int n1, int n2, const double* __restrict__ a4, const S* __restrict__ b, S* __restrict__ e,
                  double rtol, int max_it) {
    extern __shared__ double sm[];
    const int n = n0 * n1 * n2, tid = threadIdx.x, nt = blockDim.x;
    double *ev = sm, *r = sm + n, *p = sm + 2 * n, *q = sm + 3 * n;
    __shared__ double red[16];
    __shared__ double scal;
    auto bsum = [&](double v) -> double {
        v = warp_sum(v);
        __syncthreads();
        if ((tid & 31) == 0) red[tid >> 5] = v;
        __syncthreads();
        if (tid == 0) {
            double s = 0.0;
            for (int w = 0; w < (nt + 31) / 32; ++w) s += red[w];
            scal = s;
        }
        __syncthreads();
        return scal;
    };
    double part = 0.0;
    for (int m = tid; m < n; m += nt) {
        const double v = (double)b[m];
        ev[m] = 0.0;
        r[m] = v;
        p[m] = v;
        part = fma(v, v, part);
    }
    double rr = bsum(part);
    const double rr0 = rr;
    const double s0 = a4[0], s1 = a4[1], s2 = a4[2], s3 = a4[3];
    for (int it = 0; it < max_it && rr0 > 0.0; ++it) {
        part = 0.0;
        for (int m = tid; m < n; m += nt) {
            const int i = m % n0, j = (m / n0) % n1, k = m / (n0 * n1);
            double acc = 0.0;
            for (int dk = -1; dk <= 1; ++dk)
                for (int dj = -1; dj <= 1; ++dj)
                    for (int di = -1; di <= 1; ++di) {
                        const int ii = i + di, jj = j + dj, kk = k + dk;
                        if (ii < 0 || ii >= n0 || jj < 0 || jj >= n1 || kk < 0 || kk >= n2) continue;
                        const int nz = (di != 0) + (dj != 0) + (dk != 0);
                        acc += (nz == 0 ? s0 : nz == 1 ? s1 : nz == 2 ? s2 : s3) * p[(kk * n1 + jj) * n0 + ii];
                    }
            q[m] = acc;
            part = fma(p[m], acc, part);
        }
        const double alpha = rr / bsum(part);
        part = 0.0;
        for (int m = tid; m < n; m += nt) {
            ev[m] = fma(alpha, p[m], ev[m]);
            const double rn = fma(-alpha, q[m], r[m]);
            r[m] = rn;
            part = fma(rn, rn, part);
        }
        const double rn2 = bsum(part);
        if (sqrt(rn2) <= rtol * sqrt(rr0)) break;
        const double beta = rn2 / rr;
        rr = rn2;
        for (int m = tid; m < n; m += nt) p[m] = fma(beta, p[m], r[m]);
        __syncthreads();
    }
    for (int m = tid; m < n; m += nt) e[m] = (S)ev[m];
}

}  // namespace mgv

// ---- host side ---------------------------------------------------------------------------------------------------------
using mgv::Plan;

// z chunks: the number of chunks that minimises (waves of resident CTAs) x (planes marched per CTA, 4 lead-in planes
// included) — a partly filled last wave costs as much as a full one.
static Plan make_plan(const poisson_ctx* ctx, const int n[3], int resident, const int* nc = nullptr) {
    Plan pl;
    pl.n0 = n[0];
    pl.n1 = n[1];
    pl.n2 = n[2];
    pl.nc0 = pl.nc1 = pl.nc2 = 0;
    if (nc) {  // residual + restriction: chunks of coarse planes, each costing two fine planes
        pl.nc0 = nc[0];
        pl.nc1 = nc[1];
        pl.nc2 = nc[2];
    }
    const int nplanes = nc ? nc[2] : n[2], per = nc ? 2 : 1;
    pl.ntx = (n[0] + mgv::VX - 1) / mgv::VX;
    pl.nty = (n[1] + mgv::VY - 1) / mgv::VY;
    const long tiles = (long)pl.ntx * pl.nty, slots = (long)ctx->num_sms * std::max(1, resident);
    double best = 1e300;
    pl.kc = n[2];
    pl.nz = 1;
    pl.kc = nplanes;
    for (int nz = 1; nz <= std::max(1, per * nplanes / 2); ++nz) {  // chunks down to two fine planes: small levels are latency-bound
        const int kc = (nplanes + nz - 1) / nz, nzz = (nplanes + kc - 1) / kc;
        const double cost = (double)((tiles * nzz + slots - 1) / slots) * (per * kc + 4 + 2);
        if (cost < best - 1e-9) {
            best = cost;
            pl.kc = kc;
            pl.nz = nzz;
        }
    }
    return pl;
}

template <typename SX, typename SB, typename SO, int MODE, bool SEVEN>
static int spai_launch_k(poisson_ctx* ctx, int kid, const int n[3], const SX* x, const SB* b, SO* out, const double* a4,
                         double bsign, const double spai[5], double h, const int* nc) {
    auto kern = mgv::k_spai<SX, SB, SO, MODE, SEVEN>;
    constexpr size_t smem = mgv::spai_smem<SX, SB>();
    int resident = 0;
    const int rc = kernel_ready(ctx, kern, mgv::NT, smem, &resident);
    if (rc != POISSON_OK) return rc;
    const Plan pl = make_plan(ctx, n, resident, nc);
    const dim3 blk(mgv::NTX, mgv::NTY), grid((unsigned)(pl.ntx * pl.nty * pl.nz));
    const double h2 = h * h, om = spai ? spai[0] : 0.0;
    const double m0 = spai ? spai[1] * h2 : 0, m1 = spai ? spai[2] * h2 : 0, m2 = spai ? spai[3] * h2 : 0,
                 m3 = spai ? spai[4] * h2 : 0;
    PB_LAUNCH(ctx, kid, (kern<<<grid, blk, smem, ctx->stream>>>(pl, x, b, out, a4, bsign, om, m0, m1, m2, m3)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

template <typename SX, typename SB, typename SO, int MODE>
static int spai_launch(poisson_ctx* ctx, int kid, const int n[3], bool seven, const SX* x, const SB* b, SO* out,
                       const double* a4, double bsign, const double spai[5], double h, const int* nc = nullptr) {
    if (seven) return spai_launch_k<SX, SB, SO, MODE, true>(ctx, kid, n, x, b, out, a4, bsign, spai, h, nc);
    return spai_launch_k<SX, SB, SO, MODE, false>(ctx, kid, n, x, b, out, a4, bsign, spai, h, nc);
}

// Level bookkeeping lives in the handle (common.cuh MgvLevel); built lazily, rebuilt when the parameters change.
static void mgv_free(poisson_ctx* ctx) {
    for (auto& L : ctx->vlevels) {
        cudaFree(L.x);
        cudaFree(L.b);
        cudaFree(L.t);
    }
    ctx->vlevels.clear();
    cudaFree(ctx->v_sten);
    ctx->v_sten = nullptr;
    ctx->v_key[0] = ctx->v_key[1] = ctx->v_key[2] = -1;
}

void mgv_destroy(poisson_ctx* ctx) { mgv_free(ctx); }

static int mgv_build(poisson_ctx* ctx, int coarsest_n, int f32) {
    const int order = ctx->opt_compact_order;
    if (ctx->v_key[0] == coarsest_n && ctx->v_key[1] == f32 && ctx->v_key[2] == order && !ctx->vlevels.empty())
        return POISSON_OK;
    mgv_free(ctx);
    MgvLevel L0;
    for (int a = 0; a < 3; ++a) L0.n[a] = ctx->op.n[a];
    L0.h = ctx->h[0];
    L0.npts = ctx->npts;
    ctx->vlevels.push_back(L0);
    for (;;) {
        const MgvLevel& F = ctx->vlevels.back();
        bool ok = true;
        for (int a = 0; a < 3; ++a) ok = ok && (F.n[a] % 2 == 1) && (F.n[a] - 1) / 2 >= coarsest_n;
        if (!ok) break;
        MgvLevel C;
        C.npts = 1;
        for (int a = 0; a < 3; ++a) {
            C.n[a] = (F.n[a] - 1) / 2;
            C.npts *= (size_t)C.n[a];
        }
        C.h = 2.0 * F.h;
        ctx->vlevels.push_back(C);
    }
    const size_t nl = ctx->vlevels.size();
    PB_CUDA_OK(cudaMalloc((void**)&ctx->v_sten, nl * 4 * sizeof(double)));
    const double c = 1.0 / (ctx->h[0] * ctx->h[0]);
    // A = -L_h as a symmetric 27-point stencil (centre, faces, edges, corners): the 7-point operator, or the compact
    // radius-1 discretisation of order 4 / 6: L_h = (S1 + S2/6 [+ S3/30]) / h^2 in second differences,
    // i.e. (-24, 2, 1, 0)/6 and (-128, 14, 3, 1)/30 (reading C19)
    const double s0[4] = {order == 2 ? 6.0 * c : order == 4 ? 4.0 * c : (64.0 / 15.0) * c,
                          order == 2 ? -c : order == 4 ? -c / 3.0 : -(7.0 / 15.0) * c,
                          order == 2 ? 0.0 : order == 4 ? -c / 6.0 : -c / 10.0, order == 6 ? -c / 30.0 : 0.0};
    PB_CUDA_OK(cudaMemcpyAsync(ctx->v_sten, s0, sizeof(s0), cudaMemcpyHostToDevice, ctx->stream));
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));  // s0 is a stack array
    for (size_t l = 1; l < nl; ++l)
        PB_LAUNCH(ctx, KID_MGV_SETUP, (mgv::k_galerkin27<<<1, 32, 0, ctx->stream>>>(ctx->v_sten + 4 * (l - 1), ctx->v_sten + 4 * l, f32)));
    PB_CUDA_OK(cudaGetLastError());
    const size_t es = f32 ? sizeof(float) : sizeof(double);
    for (size_t l = 0; l < nl; ++l) {
        MgvLevel& L = ctx->vlevels[l];
        // level 0: b = folded right-hand side (fp64), t = ping-pong / residual buffer (fp64); x is the caller's array.
        // coarse levels: x, b in the storage type; t fp64 (residual) and a second x buffer for the Jacobi ping-pong
        PB_CUDA_OK(cudaMalloc(&L.b, L.npts * (l == 0 ? sizeof(double) : es)));
        PB_CUDA_OK(cudaMalloc(&L.t, L.npts * sizeof(double)));
        if (l > 0) PB_CUDA_OK(cudaMalloc(&L.x, 2 * L.npts * es));
    }
    ctx->v_key[0] = coarsest_n;
    ctx->v_key[1] = f32;
    ctx->v_key[2] = order;
    return POISSON_OK;
}

// PAPER.md:176-182 Table 1.  The delta of row 6 is printed as 0.0909 (a copy of the mu column): 0.0150, the middle of
// the interval on which the smoothing factor of Eq. 17 is smallest with the other printed values (reading C20).
static const double kSpaiOrder2[5] = {1.3699, 0.1432, 0.0284, 0.0081, 0.0025};
static const double kSpaiOrder4[5] = {0.9363, 0.2807, 0.0329, 0.0166, 0.0044};
static const double kSpaiOrder6[5] = {0.3543, 0.7064, 0.1005, 0.0363, 0.0150};
static const double* default_spai(const poisson_ctx* ctx) {
    return ctx->opt_compact_order == 4 ? kSpaiOrder4 : ctx->opt_compact_order == 6 ? kSpaiOrder6 : kSpaiOrder2;
}

// Level-0 right-hand side.  Order 2: the Dirichlet values of the ghost faces folded in (into bt).  Orders 4 / 6: the
// caller's array as it is — a 27-point stencil would need ghost values on the edges and corners of the shell, which the
// face arrays do not hold, so boundary data belong in the right-hand side there and the ghosts must be zero.
static int fold_ghosts(poisson_ctx* ctx, const double* rhs, double* bt, const double** use) {
    if (ctx->opt_compact_order != 2) {
        if (ctx->ghost_nonzero)
            return fail(ctx, POISSON_UNSUPPORTED, "compact order 4 / 6: ghost values are not used — fold the boundary data into the right-hand side");
        *use = rhs;
        return POISSON_OK;
    }
    *use = bt;
    const Op& op = ctx->op;
    const dim3 blk(64, 4), grid((op.n[0] + 63) / 64, (op.n[1] + 3) / 4, op.n[2]);
    PB_LAUNCH(ctx, KID_MGV_SETUP, (mgv::k_fold_ghosts<<<grid, blk, 0, ctx->stream>>>(op, rhs, bt)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

// Error-equation levels l >= 1: A_l e = b_l from e = 0 (storage type S).  L.x holds two buffers; the result is left in
// *res.
template <typename S>
static int mgv_cycle(poisson_ctx* ctx, size_t l, int nu1, int nu2, const double* spai, double cg_rtol, S** res) {
    MgvLevel& L = ctx->vlevels[l];
    S* xa = (S*)L.x;
    S* xb = xa + L.npts;
    const S* b = (const S*)L.b;
    const double* a4 = ctx->v_sten + 4 * l;
    int rc;
    if (l + 1 == ctx->vlevels.size()) {
        const int n = (int)L.npts;
        const size_t smem = (size_t)4 * n * sizeof(double);
        if (smem > 200 * 1024) return fail(ctx, POISSON_UNSUPPORTED, "coarsest level too large for the one-CTA CG (lower coarsest_n)");
        if ((rc = kernel_ready(ctx, mgv::k_cg_coarse27<S>, 512, 200 * 1024)) != POISSON_OK) return rc;  // the limit, once
        PB_LAUNCH(ctx, KID_MGV_COARSE, (mgv::k_cg_coarse27<S><<<1, 512, smem, ctx->stream>>>(L.n[0], L.n[1], L.n[2], a4, b, xa, cg_rtol, 4 * n + 10)));
        PB_CUDA_OK(cudaGetLastError());
        *res = xa;
        return POISSON_OK;
    }
    PB_CUDA_OK(cudaMemsetAsync(xa, 0, L.npts * sizeof(S), ctx->stream));
    S *cur = xa, *oth = xb;
    for (int s = 0; s < nu1; ++s) {
        if ((rc = spai_launch<S, S, S, 0>(ctx, KID_MGV_SMOOTH, L.n, false, cur, b, oth, a4, 1.0, spai, L.h)) != POISSON_OK) return rc;
        std::swap(cur, oth);
    }
    MgvLevel& C = ctx->vlevels[l + 1];
    // residual + full weighting in one pass: b_c = R (b - A x)
    if ((rc = spai_launch<S, S, S, 2>(ctx, KID_MGV_RESTRICT, L.n, false, cur, b, (S*)C.b, a4, 1.0, nullptr, L.h, C.n)) != POISSON_OK) return rc;
    S* ec = nullptr;
    if ((rc = mgv_cycle<S>(ctx, l + 1, nu1, nu2, spai, cg_rtol, &ec)) != POISSON_OK) return rc;
    {
        const dim3 blk(32, 8), grid((C.n[0] + 1 + 31) / 32, (C.n[1] + 1 + 7) / 8, C.n[2] + 1);
        PB_LAUNCH(ctx, KID_MGV_PROLONG, (mgv::k_prolong27<S, S><<<grid, blk, 0, ctx->stream>>>(L.n[0], L.n[1], L.n[2], C.n[0], C.n[1], C.n[2], ec, cur)));
    }
    for (int s = 0; s < nu2; ++s) {
        if ((rc = spai_launch<S, S, S, 0>(ctx, KID_MGV_SMOOTH, L.n, false, cur, b, oth, a4, 1.0, spai, L.h)) != POISSON_OK) return rc;
        std::swap(cur, oth);
    }
    PB_CUDA_OK(cudaGetLastError());
    *res = cur;
    return POISSON_OK;
}

static int mgv_check(poisson_ctx* ctx) {
    if (ctx->kind != KIND_CART2) return fail(ctx, POISSON_UNSUPPORTED, "SPAI / Galerkin multigrid: Cartesian 7-point operator only");
    if (ctx->h[0] != ctx->h[1] || ctx->h[0] != ctx->h[2])
        return fail(ctx, POISSON_UNSUPPORTED, "the SPAI smoother is restricted to isotropic spacing (PAPER.md:162)");
    for (int f = 0; f < 6; ++f)
        if (ctx->op.bc[f] != POISSON_BC_DIRICHLET_GHOST)
            return fail(ctx, POISSON_UNSUPPORTED, "SPAI / Galerkin multigrid: Dirichlet (ghost) faces only");
    return POISSON_OK;
}

// nsteps SPAI steps on the user's grid (row f1).  The steps ping-pong between phi and the handle's buffer.
int mgv_spai_smooth(poisson_ctx* ctx, double* phi, const double* rhs, const double* spai, int nsteps) {
    int rc;
    if ((rc = mgv_check(ctx)) != POISSON_OK) return rc;
    if ((rc = mgv_build(ctx, ctx->v_key[0] < 0 ? 3 : ctx->v_key[0], ctx->v_key[1] < 0 ? 0 : ctx->v_key[1])) != POISSON_OK) return rc;
    if (!spai) spai = default_spai(ctx);
    const bool seven = ctx->opt_compact_order == 2;
    MgvLevel& L0 = ctx->vlevels[0];
    const double* bt = nullptr;
    if ((rc = fold_ghosts(ctx, rhs, (double*)L0.b, &bt)) != POISSON_OK) return rc;
    double *cur = phi, *oth = (double*)L0.t;
    for (int s = 0; s < nsteps; ++s) {
        // level 0: b = -rhs~ (bsign = -1), A = -L_h
        if ((rc = spai_launch<double, double, double, 0>(ctx, KID_MGV_SMOOTH, L0.n, seven, cur, bt, oth, ctx->v_sten, -1.0, spai, L0.h)) != POISSON_OK) return rc;
        std::swap(cur, oth);
    }
    if (cur != phi) PB_CUDA_OK(cudaMemcpyAsync(phi, cur, ctx->npts * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    return POISSON_OK;
}

template <typename S>
static int mgv_vcycles_t(poisson_ctx* ctx, double* phi, const double* rhs, int nu1, int nu2, const double* spai,
                         double cg_rtol, int ncycles, const std::function<int(int)>& record) {
    int rc;
    const bool seven = ctx->opt_compact_order == 2;
    MgvLevel& L0 = ctx->vlevels[0];
    const double* bt = nullptr;
    if ((rc = fold_ghosts(ctx, rhs, (double*)L0.b, &bt)) != POISSON_OK) return rc;
    for (int c = 0; c < ncycles; ++c) {
        double *cur = phi, *oth = (double*)L0.t;
        if (ctx->vlevels.size() == 1) {
            return fail(ctx, POISSON_UNSUPPORTED, "the grid admits no coarse level (sizes must be 2^N k - 1 >= 2 coarsest_n + 1, PAPER.md:152)");
        }
        for (int s = 0; s < nu1; ++s) {
            if ((rc = spai_launch<double, double, double, 0>(ctx, KID_MGV_SMOOTH, L0.n, seven, cur, bt, oth, ctx->v_sten, -1.0, spai, L0.h)) != POISSON_OK) return rc;
            std::swap(cur, oth);
        }
        MgvLevel& C = ctx->vlevels[1];
        if ((rc = spai_launch<double, double, S, 2>(ctx, KID_MGV_RESTRICT, L0.n, seven, cur, bt, (S*)C.b, ctx->v_sten, -1.0, nullptr, L0.h, C.n)) != POISSON_OK) return rc;
        S* ec = nullptr;
        if ((rc = mgv_cycle<S>(ctx, 1, nu1, nu2, spai, cg_rtol, &ec)) != POISSON_OK) return rc;
        {
            const dim3 blk(32, 8), grid((C.n[0] + 1 + 31) / 32, (C.n[1] + 1 + 7) / 8, C.n[2] + 1);
            PB_LAUNCH(ctx, KID_MGV_PROLONG, (mgv::k_prolong27<double, S><<<grid, blk, 0, ctx->stream>>>(L0.n[0], L0.n[1], L0.n[2], C.n[0], C.n[1], C.n[2], ec, cur)));
        }
        for (int s = 0; s < nu2; ++s) {
            if ((rc = spai_launch<double, double, double, 0>(ctx, KID_MGV_SMOOTH, L0.n, seven, cur, bt, oth, ctx->v_sten, -1.0, spai, L0.h)) != POISSON_OK) return rc;
            std::swap(cur, oth);
        }
        if (cur != phi) PB_CUDA_OK(cudaMemcpyAsync(phi, cur, ctx->npts * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
        PB_CUDA_OK(cudaGetLastError());
        if ((rc = record(c + 1)) != POISSON_OK) return rc;
    }
    return POISSON_OK;
}

int mgv_vcycles(poisson_ctx* ctx, double* phi, const double* rhs, int nu1, int nu2, int coarsest_n, const double* spai,
                double cg_rtol, int storage_f32, int ncycles, const std::function<int(int)>& record) {
    int rc;
    if ((rc = mgv_check(ctx)) != POISSON_OK) return rc;
    if ((rc = mgv_build(ctx, coarsest_n, storage_f32 ? 1 : 0)) != POISSON_OK) return rc;
    if (!spai) spai = default_spai(ctx);
    if (storage_f32) return mgv_vcycles_t<float>(ctx, phi, rhs, nu1, nu2, spai, cg_rtol, ncycles, record);
    return mgv_vcycles_t<double>(ctx, phi, rhs, nu1, nu2, spai, cg_rtol, ncycles, record);
}

// ||B f - L_h phi||_2^2 of the compact operator (orders 4 / 6) into d_scal[0]: residual pass + one reduction.
int mgv_residual_norm2(poisson_ctx* ctx, const double* phi, const double* rhs, int coarsest_n, int storage_f32) {
    int rc;
    if ((rc = mgv_check(ctx)) != POISSON_OK) return rc;
    if ((rc = mgv_build(ctx, coarsest_n, storage_f32 ? 1 : 0)) != POISSON_OK) return rc;
    MgvLevel& L0 = ctx->vlevels[0];
    const double* bt = nullptr;
    if ((rc = fold_ghosts(ctx, rhs, (double*)L0.b, &bt)) != POISSON_OK) return rc;
    double* r = (double*)L0.t;
    if ((rc = spai_launch<double, double, double, 1>(ctx, KID_MGV_SMOOTH, L0.n, ctx->opt_compact_order == 2, phi, bt, r,
                                                     ctx->v_sten, -1.0, nullptr, L0.h)) != POISSON_OK)
        return rc;
    const int blocks = (int)std::min<size_t>((ctx->npts + 255) / 256, (size_t)ctx->num_sms * 8);
    PB_LAUNCH(ctx, KID_MGV_SMOOTH, (mgv::k_norm2<<<blocks, 256, 0, ctx->stream>>>(ctx->npts, r, ctx->d_scal, ctx->red)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

// out = B f (compact right-hand side of the handle's compact order) from f on the grid extended by two layers per side.
int mgv_compact_rhs(poisson_ctx* ctx, const double* f_ext, double* out) {
    const Op& op = ctx->op;
    const dim3 blk(64, 4), grid((op.n[0] + 63) / 64, (op.n[1] + 3) / 4, op.n[2]);
    switch (ctx->opt_compact_order) {
        case 4: PB_LAUNCH(ctx, KID_MGV_SETUP, (mgv::k_compact_rhs<4><<<grid, blk, 0, ctx->stream>>>(op.n[0], op.n[1], op.n[2], f_ext, out))); break;
        case 6: PB_LAUNCH(ctx, KID_MGV_SETUP, (mgv::k_compact_rhs<6><<<grid, blk, 0, ctx->stream>>>(op.n[0], op.n[1], op.n[2], f_ext, out))); break;
        default: PB_LAUNCH(ctx, KID_MGV_SETUP, (mgv::k_compact_rhs<2><<<grid, blk, 0, ctx->stream>>>(op.n[0], op.n[1], op.n[2], f_ext, out))); break;
    }
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

}  // namespace pb
