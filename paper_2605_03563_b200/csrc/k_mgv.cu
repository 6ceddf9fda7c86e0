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
// A CTA of NTX x NTY threads owns the xy tile of residual points (output tile + 1 halo) and marches z.  Both
// 27-point applications are evaluated from per-plane partial sums kept in registers along z,
//   Q0 = v(c), Q1 = sum of the 4 in-plane face neighbours, Q2 = sum of the 4 in-plane diagonal neighbours,
//   (S v)(k) = s0 Q0(k) + s1 [Q1(k) + Q0(k-1) + Q0(k+1)] + s2 [Q2(k) + Q1(k-1) + Q1(k+1)] + s3 [Q2(k-1) + Q2(k+1)],
// so only ONE plane of x and ONE plane of r is shared at a time (double-buffered, two barriers per plane) and a
// point costs 9 + 9 shared-memory loads instead of 27 + 27.
#include <algorithm>
#include <functional>

#include "stencil.cuh"

namespace pb {

namespace mgv {

constexpr int NTX = 32, NTY = 16;          // threads = residual tile; output tile (NTX-2) x (NTY-2)
constexpr int VX = NTX - 2, VY = NTY - 2;
constexpr int XW = NTX + 2, XH = NTY + 2;  // x plane with its halo
constexpr int NHALO = 2 * XW + 2 * NTY;    // ring of x points around the residual tile

template <typename S>
__device__ __forceinline__ double ldv(const S* p) { return (double)*p; }

struct Sten {  // symmetric 27-point stencil: centre, face, edge, corner
    double s0, s1, s2, s3;
};

struct Plan {
    int n0, n1, n2;
    int ntx, nty, nz, kc;  // tiles and z chunks
};

// MODE 0: out = x + omega M (bsign b - A x)      (one SPAI step, Eq. 15)
// MODE 1: out = bsign b - A x                    (residual, for the restriction)
// SEVEN: A has no edge / corner coefficients (level 0: the 7-point operator).
template <typename SX, typename SB, typename SO, int MODE, bool SEVEN>
__global__ void __launch_bounds__(NTX* NTY)
    k_spai(const Plan pl, const SX* __restrict__ x, const SB* __restrict__ b, SO* __restrict__ out,
           const double* __restrict__ a4 /* A: centre, face, edge, corner */, const double bsign, const double omega,
           const double m0, const double m1, const double m2, const double m3) {
    __shared__ double xs[2][XH][XW];
    __shared__ double rs[2][NTY][NTX];
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * NTX + tx;
    const int tile = blockIdx.x % (pl.ntx * pl.nty), zc = blockIdx.x / (pl.ntx * pl.nty);
    const int i0 = (tile % pl.ntx) * VX, j0 = (tile / pl.ntx) * VY;
    const int k0 = zc * pl.kc, k1 = min(pl.n2, k0 + pl.kc);
    const int n0 = pl.n0, n1 = pl.n1, n2 = pl.n2;
    const int i = i0 - 1 + tx, j = j0 - 1 + ty;  // this thread's residual point
    const bool in = i >= 0 && i < n0 && j >= 0 && j < n1;
    const bool owner = in && tx >= 1 && tx <= VX && ty >= 1 && ty <= VY;
    const size_t plane = (size_t)n0 * n1;
    const size_t col = in ? (size_t)j * n0 + i : 0;
    // this thread's halo point of the x plane (ring around the residual tile), if any
    int hx = -1, hy = -1;
    if (tid < NHALO) {
        if (tid < XW) { hx = tid; hy = 0; }
        else if (tid < 2 * XW) { hx = tid - XW; hy = XH - 1; }
        else if (tid < 2 * XW + NTY) { hx = 0; hy = 1 + tid - 2 * XW; }
        else { hx = XW - 1; hy = 1 + tid - 2 * XW - NTY; }
    }
    const int hi = i0 - 2 + hx, hj = j0 - 2 + hy;
    const bool hin = hx >= 0 && hi >= 0 && hi < n0 && hj >= 0 && hj < n1;
    const size_t hcol = hin ? (size_t)hj * n0 + hi : 0;
    const double s0 = a4[0], s1 = a4[1], s2 = SEVEN ? 0.0 : a4[2], s3 = SEVEN ? 0.0 : a4[3];

    double q0m = 0, q1m = 0, q2m = 0, q0c = 0, q1c = 0, q2c = 0;  // x partial sums of planes kx-2, kx-1
    double p0m = 0, p1m = 0, p2m = 0, p0c = 0, p1c = 0, p2c = 0;  // r partial sums of planes kx-3, kx-2
    // software pipeline: the values of plane kx are loaded one iteration before they are shared
    auto ldx = [&](int kk, bool ok, size_t c) -> double {
        return (ok && kk >= 0 && kk < n2) ? ldv(x + (size_t)kk * plane + c) : 0.0;
    };
    auto ldb = [&](int kk) -> double { return (in && kk >= 0 && kk < n2) ? bsign * ldv(b + (size_t)kk * plane + col) : 0.0; };
    const int kx0 = (MODE == 0 ? k0 - 2 : k0 - 1);
    double xn = ldx(kx0, in, col), hn = ldx(kx0, hin, hcol), bn = ldb(kx0 - 1);
    for (int kx = kx0; kx <= k1 + (MODE == 0 ? 1 : 0); ++kx) {
        const int par = kx & 1;
        xs[par][ty + 1][tx + 1] = xn;
        if (hx >= 0) xs[par][hy][hx] = hn;
        const double bcur = bn;  // b of plane kx-1
        xn = ldx(kx + 1, in, col);
        hn = ldx(kx + 1, hin, hcol);
        bn = ldb(kx);
        __syncthreads();
        // partial sums of x plane kx at this thread's residual point
        const double q0p = xs[par][ty + 1][tx + 1];
        const double q1p = (xs[par][ty + 1][tx] + xs[par][ty + 1][tx + 2]) + (xs[par][ty][tx + 1] + xs[par][ty + 2][tx + 1]);
        double q2p = 0.0;
        if (!SEVEN) q2p = (xs[par][ty][tx] + xs[par][ty][tx + 2]) + (xs[par][ty + 2][tx] + xs[par][ty + 2][tx + 2]);
        // residual of plane kx-1 (zero outside the domain: Dirichlet vertices carry no residual)
        const int kr = kx - 1;
        double r = 0.0;
        if (in && kr >= 0 && kr < n2) {
            double ax = s0 * q0c;
            ax = fma(s1, q1c + (q0m + q0p), ax);
            if (!SEVEN) {
                ax = fma(s2, q2c + (q1m + q1p), ax);
                ax = fma(s3, q2m + q2p, ax);
            }
            r = bcur - ax;
        }
        if (MODE == 1) {
            if (owner && kr >= k0 && kr < k1) out[(size_t)kr * plane + col] = (SO)r;
        } else {
            rs[par][ty][tx] = r;
            __syncthreads();
            if (owner) {  // only owners have all their in-plane neighbours inside the tile
                const double p0p = r;
                const double p1p = (rs[par][ty][tx - 1] + rs[par][ty][tx + 1]) + (rs[par][ty - 1][tx] + rs[par][ty + 1][tx]);
                const double p2p = (rs[par][ty - 1][tx - 1] + rs[par][ty - 1][tx + 1]) +
                                   (rs[par][ty + 1][tx - 1] + rs[par][ty + 1][tx + 1]);
                const int ko = kx - 2;
                if (ko >= k0 && ko < k1) {
                    double mr = m0 * p0c;
                    mr = fma(m1, p1c + (p0m + p0p), mr);
                    mr = fma(m2, p2c + (p1m + p1p), mr);
                    mr = fma(m3, p2m + p2p, mr);
                    out[(size_t)ko * plane + col] = (SO)fma(omega, mr, q0m);  // q0m = x of plane kx-2
                }
                p0m = p0c; p1m = p1c; p2m = p2c;
                p0c = p0p; p1c = p1p; p2c = p2p;
            }
        }
        q0m = q0c; q1m = q1c; q2m = q2c;
        q0c = q0p; q1c = q1p; q2c = q2p;
    }
}

// b_c = R r (Eq. 13): coarse vertex I sits on fine vertex 2I+1; all 27 fine points are interior.
template <typename SO>
__global__ void __launch_bounds__(256)
    k_restrict27(int nc0, int nc1, int nc2, int n0, int n1, const double* __restrict__ r, SO* __restrict__ bc) {
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    if (I >= nc0 || J >= nc1 || K >= nc2) return;
    const double w[3] = {0.25, 0.5, 0.25};
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int bb = 0; bb < 3; ++bb) {
            const double* row = r + ((size_t)(2 * K + c) * n1 + (2 * J + bb)) * n0 + 2 * I;
            s = fma(w[bb] * w[c], fma(0.25, row[0] + row[2], 0.5 * row[1]), s);
        }
    bc[((size_t)K * nc1 + J) * nc0 + I] = (SO)s;
}

// x += P e_c, P = 8 R^T: odd fine indices sit on a coarse vertex, even ones half-way between two (zero beyond the boundary).
template <typename SX, typename SE>
__global__ void __launch_bounds__(256)
    k_prolong27(int n0, int n1, int n2, int nc0, int nc1, int nc2, const SE* __restrict__ ec, SX* __restrict__ x) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= n0 || j >= n1 || k >= n2) return;
    const int I0 = (i - 1) >> 1, J0 = (j - 1) >> 1, K0 = (k - 1) >> 1;
    const int ni = (i & 1) ? 1 : 2, nj = (j & 1) ? 1 : 2, nk = (k & 1) ? 1 : 2;
    double s = 0.0;
    for (int c = 0; c < nk; ++c)
        for (int bb = 0; bb < nj; ++bb)
            for (int a = 0; a < ni; ++a) {
                const int I = I0 + a, J = J0 + bb, K = K0 + c;
                if (I >= 0 && I < nc0 && J >= 0 && J < nc1 && K >= 0 && K < nc2) s += ldv(ec + ((size_t)K * nc1 + J) * nc0 + I);
            }
    const size_t p = ((size_t)k * n1 + j) * n0 + i;
    x[p] = (SX)(ldv(x + p) + s / (double)(ni * nj * nk));
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

static Plan make_plan(const poisson_ctx* ctx, const int n[3]) {
    Plan pl;
    pl.n0 = n[0];
    pl.n1 = n[1];
    pl.n2 = n[2];
    pl.ntx = (n[0] + mgv::VX - 1) / mgv::VX;
    pl.nty = (n[1] + mgv::VY - 1) / mgv::VY;
    // z chunks: enough CTAs for ~3 waves of 4 resident CTAs per SM, chunks of at least 16 planes (4 lead-in planes each)
    const long tiles = (long)pl.ntx * pl.nty, want = 12L * ctx->num_sms;
    int nz = (int)std::max(1L, std::min((long)std::max(1, n[2] / 16), (want + tiles - 1) / tiles));
    pl.kc = (n[2] + nz - 1) / nz;
    pl.nz = (n[2] + pl.kc - 1) / pl.kc;
    return pl;
}

template <typename SX, typename SB, typename SO, int MODE>
static int spai_launch(poisson_ctx* ctx, int kid, const int n[3], bool seven, const SX* x, const SB* b, SO* out,
                       const double* a4, double bsign, const double spai[5], double h) {
    const Plan pl = make_plan(ctx, n);
    const dim3 blk(mgv::NTX, mgv::NTY), grid((unsigned)(pl.ntx * pl.nty * pl.nz));
    const double h2 = h * h, om = spai ? spai[0] : 0.0;
    const double m0 = spai ? spai[1] * h2 : 0, m1 = spai ? spai[2] * h2 : 0, m2 = spai ? spai[3] * h2 : 0,
                 m3 = spai ? spai[4] * h2 : 0;
    if (seven)
        PB_LAUNCH(ctx, kid, (mgv::k_spai<SX, SB, SO, MODE, true><<<grid, blk, 0, ctx->stream>>>(pl, x, b, out, a4, bsign, om, m0, m1, m2, m3)));
    else
        PB_LAUNCH(ctx, kid, (mgv::k_spai<SX, SB, SO, MODE, false><<<grid, blk, 0, ctx->stream>>>(pl, x, b, out, a4, bsign, om, m0, m1, m2, m3)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
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
    ctx->v_key[0] = ctx->v_key[1] = -1;
}

void mgv_destroy(poisson_ctx* ctx) { mgv_free(ctx); }

static int mgv_build(poisson_ctx* ctx, int coarsest_n, int f32) {
    if (ctx->v_key[0] == coarsest_n && ctx->v_key[1] == f32 && !ctx->vlevels.empty()) return POISSON_OK;
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
    const double s0[4] = {6.0 * c, -c, 0.0, 0.0};  // A = -L_h: the 7-point operator as a symmetric 27-point stencil
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
    return POISSON_OK;
}

static const double kSpaiOrder2[5] = {1.3699, 0.1432, 0.0284, 0.0081, 0.0025};  // PAPER.md:176-182 Table 1, order 2

static int fold_ghosts(poisson_ctx* ctx, const double* rhs, double* bt) {
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
    double* r = (double*)L.t;
    if ((rc = spai_launch<S, S, double, 1>(ctx, KID_MGV_RESTRICT, L.n, false, cur, b, r, a4, 1.0, nullptr, L.h)) != POISSON_OK) return rc;
    MgvLevel& C = ctx->vlevels[l + 1];
    {
        const dim3 blk(32, 8), grid((C.n[0] + 31) / 32, (C.n[1] + 7) / 8, C.n[2]);
        PB_LAUNCH(ctx, KID_MGV_RESTRICT, (mgv::k_restrict27<S><<<grid, blk, 0, ctx->stream>>>(C.n[0], C.n[1], C.n[2], L.n[0], L.n[1], r, (S*)C.b)));
    }
    S* ec = nullptr;
    if ((rc = mgv_cycle<S>(ctx, l + 1, nu1, nu2, spai, cg_rtol, &ec)) != POISSON_OK) return rc;
    {
        const dim3 blk(64, 4), grid((L.n[0] + 63) / 64, (L.n[1] + 3) / 4, L.n[2]);
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
    if (!spai) spai = kSpaiOrder2;
    MgvLevel& L0 = ctx->vlevels[0];
    double* bt = (double*)L0.b;
    if ((rc = fold_ghosts(ctx, rhs, bt)) != POISSON_OK) return rc;
    double *cur = phi, *oth = (double*)L0.t;
    for (int s = 0; s < nsteps; ++s) {
        // level 0: b = -rhs~ (bsign = -1), A = -L_h
        if ((rc = spai_launch<double, double, double, 0>(ctx, KID_MGV_SMOOTH, L0.n, true, cur, bt, oth, ctx->v_sten, -1.0, spai, L0.h)) != POISSON_OK) return rc;
        std::swap(cur, oth);
    }
    if (cur != phi) PB_CUDA_OK(cudaMemcpyAsync(phi, cur, ctx->npts * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
    return POISSON_OK;
}

template <typename S>
static int mgv_vcycles_t(poisson_ctx* ctx, double* phi, const double* rhs, int nu1, int nu2, const double* spai,
                         double cg_rtol, int ncycles, const std::function<int(int)>& record) {
    int rc;
    MgvLevel& L0 = ctx->vlevels[0];
    double* bt = (double*)L0.b;
    if ((rc = fold_ghosts(ctx, rhs, bt)) != POISSON_OK) return rc;
    for (int c = 0; c < ncycles; ++c) {
        double *cur = phi, *oth = (double*)L0.t;
        if (ctx->vlevels.size() == 1) {
            return fail(ctx, POISSON_UNSUPPORTED, "the grid admits no coarse level (sizes must be 2^N k - 1 >= 2 coarsest_n + 1, PAPER.md:152)");
        }
        for (int s = 0; s < nu1; ++s) {
            if ((rc = spai_launch<double, double, double, 0>(ctx, KID_MGV_SMOOTH, L0.n, true, cur, bt, oth, ctx->v_sten, -1.0, spai, L0.h)) != POISSON_OK) return rc;
            std::swap(cur, oth);
        }
        if ((rc = spai_launch<double, double, double, 1>(ctx, KID_MGV_RESTRICT, L0.n, true, cur, bt, oth, ctx->v_sten, -1.0, nullptr, L0.h)) != POISSON_OK) return rc;
        MgvLevel& C = ctx->vlevels[1];
        {
            const dim3 blk(32, 8), grid((C.n[0] + 31) / 32, (C.n[1] + 7) / 8, C.n[2]);
            PB_LAUNCH(ctx, KID_MGV_RESTRICT, (mgv::k_restrict27<S><<<grid, blk, 0, ctx->stream>>>(C.n[0], C.n[1], C.n[2], L0.n[0], L0.n[1], oth, (S*)C.b)));
        }
        S* ec = nullptr;
        if ((rc = mgv_cycle<S>(ctx, 1, nu1, nu2, spai, cg_rtol, &ec)) != POISSON_OK) return rc;
        {
            const dim3 blk(64, 4), grid((L0.n[0] + 63) / 64, (L0.n[1] + 3) / 4, L0.n[2]);
            PB_LAUNCH(ctx, KID_MGV_PROLONG, (mgv::k_prolong27<double, S><<<grid, blk, 0, ctx->stream>>>(L0.n[0], L0.n[1], L0.n[2], C.n[0], C.n[1], C.n[2], ec, cur)));
        }
        for (int s = 0; s < nu2; ++s) {
            if ((rc = spai_launch<double, double, double, 0>(ctx, KID_MGV_SMOOTH, L0.n, true, cur, bt, oth, ctx->v_sten, -1.0, spai, L0.h)) != POISSON_OK) return rc;
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
    if (!spai) spai = kSpaiOrder2;
    if (storage_f32) return mgv_vcycles_t<float>(ctx, phi, rhs, nu1, nu2, spai, cg_rtol, ncycles, record);
    return mgv_vcycles_t<double>(ctx, phi, rhs, nu1, nu2, spai, cg_rtol, ncycles, record);
}

}  // namespace pb
