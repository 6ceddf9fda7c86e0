// k_mg.cu — multigrid transfer operators and the coarsest-level solver.  PAPER.md:125-152 (Eq. 11-13), 205.
// Variant fixed by BASELINE.json config 3 / DESIGN.md reading C7: cell-centred 2:1 coarsening, full-weighting
// restriction as the transpose of trilinear interpolation ((1/8)[1 3 3 1] per axis, P = 8 R^T),
// trilinear prolongation with the level's ghost closure, coarsest level by red-black SOR sweeps in shared memory.
#include "stencil.cuh"

namespace pb {

template <typename T>
struct Vec2 {};
template <>
struct Vec2<double> {
    using type = double2;
};
template <>
struct Vec2<float> {
    using type = float2;
};

// One coarse value, axis by axis (fw_acc in stencil.cuh): the order every restriction kernel follows.
template <typename T>
__device__ __forceinline__ T restrict_cell(const Op& fine, const T* __restrict__ r, int I, int J, int K, int restriction) {
    T z = 0;
    if (restriction == 1) {
        T y[2];
        for (int c = 0; c < 2; ++c) {
            T x[2];
            for (int b = 0; b < 2; ++b)
                x[b] = r[gidx(fine, 2 * I, 2 * J + b, 2 * K + c)] + r[gidx(fine, 2 * I + 1, 2 * J + b, 2 * K + c)];
            y[c] = x[0] + x[1];
        }
        return (y[0] + y[1]) * (T)0.125;
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int k = 2 * K - 1 + c;
        if (k < 0 || k >= fine.n[2]) continue;
        T y = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int j = 2 * J - 1 + b;
            if (j < 0 || j >= fine.n[1]) continue;
            T x = 0;
#pragma unroll
            for (int a = 0; a < 4; ++a) {
                const int i = 2 * I - 1 + a;
                if (i < 0 || i >= fine.n[0]) continue;
                x = fw_acc<T>(x, a, r[gidx(fine, i, j, k)]);
            }
            y = fw_acc<T>(y, b, x);
        }
        z = fw_acc<T>(z, c, y);
    }
    return z;
}

template <typename T>
__global__ void __launch_bounds__(256)
    k_restrict(Op fine, Op coarse, const T* __restrict__ r, T* __restrict__ fc, int restriction) {
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    if (I >= coarse.n[0] || J >= coarse.n[1]) return;
    fc[gidx(coarse, I, J, K)] = restrict_cell<T>(fine, r, I, J, K, restriction);
}

// The same restriction ((1/8)[1 3 3 1]^3, the same axis-by-axis sums) for fine.n = 2 coarse.n and 32 x 8 thread
// blocks: a warp is 32 consecutive coarse cells of one row, every thread loads the aligned fine pair (2I, 2I+1) of each
// of the 16 fine rows it needs with one 16-byte access and takes r[2I-1] / r[2I+2] from its neighbour lanes (warp edges:
// one extra scalar load) — 16 load instructions per coarse cell instead of 64 half-used ones.  (A version that walked
// the fine planes of 8 coarse planes with running z sums, 10 loads per coarse cell, measured 89 us against 72 us at
// 256^3: one short block per coarse plane keeps more independent loads in flight.)
template <typename T>
__global__ void __launch_bounds__(256)
    k_restrict_v(Op fine, Op coarse, const T* __restrict__ r, T* __restrict__ fc) {
    using V2 = typename Vec2<T>::type;
    const int lane = threadIdx.x;
    const int I = blockIdx.x * 32 + lane, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    const bool in = I < coarse.n[0] && J < coarse.n[1];
    const bool has_l = 2 * I - 1 >= 0, has_r = 2 * I + 2 < fine.n[0];
    T z = 0;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int k = 2 * K - 1 + c;
        const bool kin = k >= 0 && k < fine.n[2];
        T y = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int j = 2 * J - 1 + b;
            const bool row = in && kin && j >= 0 && j < fine.n[1];
            V2 v;
            v.x = v.y = (T)0;
            const T* const p = r + gidx(fine, 2 * I, j, k);
            if (row) v = *reinterpret_cast<const V2*>(p);
            T left = __shfl_up_sync(0xffffffffu, v.y, 1), right = __shfl_down_sync(0xffffffffu, v.x, 1);
            if (row && lane == 0 && has_l) left = p[-1];
            if (row && lane == 31 && has_r) right = p[2];
            if (row) {
                T x = 0;
                if (has_l) x = fw_acc<T>(x, 0, left);
                x = fw_acc<T>(x, 1, v.x);
                x = fw_acc<T>(x, 2, v.y);
                if (has_r) x = fw_acc<T>(x, 3, right);
                y = fw_acc<T>(y, b, x);
            }
        }
        if (kin) z = fw_acc<T>(z, c, y);
    }
    if (in) fc[gidx(coarse, I, J, K)] = z;
}

// coarse value with the ghost closure applied axis by axis: out-of-range index -> -gamma * clamped value
template <typename T>
__device__ __forceinline__ T coarse_val(const Op& c, const T* __restrict__ e, int I, int J, int K) {
    T sgn = 1;
    const T mg = (T)(-c.gamma);
    if (I < 0) { I = 0; sgn *= mg; } else if (I >= c.n[0]) { I = c.n[0] - 1; sgn *= mg; }
    if (J < 0) { J = 0; sgn *= mg; } else if (J >= c.n[1]) { J = c.n[1] - 1; sgn *= mg; }
    if (K < 0) { K = 0; sgn *= mg; } else if (K >= c.n[2]) { K = c.n[2] - 1; sgn *= mg; }
    return sgn * e[gidx(c, I, J, K)];
}

// phi += P e_c (trilinear, "P = c R^T").  One thread per COARSE cell: it reads the 3 x 3 x 3 coarse
// neighbourhood once (ghost closure applied by coarse_val) and updates its 8 fine children, two x-adjacent ones per
// 16-byte (fp64) access.  Per fine point the arithmetic is exactly
//   ex = fma(3/4, e[I], 1/4 e[I +- 1]) ; ey = fma(3/4, ex[J], 1/4 ex[J +- 1]) ; v = fma(3/4, ey[K], 1/4 ey[K +- 1]).
template <typename T>
__global__ void __launch_bounds__(256)
    k_prolong_add(Op fine, Op coarse, const T* __restrict__ ec, T* __restrict__ phi) {
    using V2 = typename Vec2<T>::type;
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    if (I >= coarse.n[0] || J >= coarse.n[1]) return;
    // the four 16-byte pairs of phi this thread updates: loaded first, so that they are in flight during the interpolation
    // (taking the x neighbours from the neighbour lanes by shuffles instead of loading them was measured slower)
    V2* const q0 = reinterpret_cast<V2*>(phi + gidx(fine, 2 * I, 2 * J, 2 * K));
    const size_t qsj = (size_t)fine.n[0] / 2, qsk = qsj * fine.n[1];  // strides in pairs
    V2 w[2][2];
#pragma unroll
    for (int pk = 0; pk < 2; ++pk)
#pragma unroll
        for (int pj = 0; pj < 2; ++pj) w[pk][pj] = q0[pk * qsk + pj * qsj];
    T ex[2][3][3];  // [x parity][dJ][dK]
    // Rows J +- 1 and planes K +- 1 all inside the coarse grid (true for whole warps, and for all but the boundary
    // layers): no closure in y and z, and the x closure (clamped index, factor -gamma) is worked out once per thread —
    // the same values as coarse_val delivers (1 * e and (-gamma) * e) with an eighth of its integer instructions.
    const bool jk_inside = J >= 1 && J + 1 < coarse.n[1] && K >= 1 && K + 1 < coarse.n[2];
    if (jk_inside) {
        const T mg = (T)(-coarse.gamma);
        const int Im = I > 0 ? I - 1 : 0, Ip = I + 1 < coarse.n[0] ? I + 1 : coarse.n[0] - 1;
        const T sm = I > 0 ? (T)1 : mg, sp = I + 1 < coarse.n[0] ? (T)1 : mg;
        const size_t sj = (size_t)coarse.n[0], sk = sj * coarse.n[1];
        const T* const c0 = ec + gidx(coarse, 0, J - 1, K - 1);
#pragma unroll
        for (int dk = 0; dk < 3; ++dk)
#pragma unroll
            for (int dj = 0; dj < 3; ++dj) {
                const T* const row = c0 + dk * sk + dj * sj;
                const T em = sm * row[Im], e0 = row[I], ep = sp * row[Ip];
                ex[0][dj][dk] = fma_((T)0.75, e0, (T)0.25 * em);
                ex[1][dj][dk] = fma_((T)0.75, e0, (T)0.25 * ep);
            }
    } else {
#pragma unroll
        for (int dk = 0; dk < 3; ++dk)
#pragma unroll
            for (int dj = 0; dj < 3; ++dj) {
                const T em = coarse_val(coarse, ec, I - 1, J + dj - 1, K + dk - 1);
                const T e0 = coarse_val(coarse, ec, I, J + dj - 1, K + dk - 1);
                const T ep = coarse_val(coarse, ec, I + 1, J + dj - 1, K + dk - 1);
                ex[0][dj][dk] = fma_((T)0.75, e0, (T)0.25 * em);
                ex[1][dj][dk] = fma_((T)0.75, e0, (T)0.25 * ep);
            }
    }
#pragma unroll
    for (int pk = 0; pk < 2; ++pk)
#pragma unroll
        for (int pj = 0; pj < 2; ++pj) {
            T v[2];
#pragma unroll
            for (int pi = 0; pi < 2; ++pi) {
                // y: near row J (dj = 1), far row J - 1 (even fine j) or J + 1 (odd); same in z
                const int fj = pj ? 2 : 0, fk = pk ? 2 : 0;
                const T ey_near = fma_((T)0.75, ex[pi][1][1], (T)0.25 * ex[pi][fj][1]);
                const T ey_far = fma_((T)0.75, ex[pi][1][fk], (T)0.25 * ex[pi][fj][fk]);
                v[pi] = fma_((T)0.75, ey_near, (T)0.25 * ey_far);
            }
            V2 o = w[pk][pj];
            o.x += v[0];
            o.y += v[1];
            q0[pk * qsk + pj * qsj] = o;
        }
}

__global__ void __launch_bounds__(256) k_add32to64(size_t n, const float* __restrict__ e, double* __restrict__ phi) {
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x)
        phi[q] += (double)e[q];
}

// Coarsest level: the whole grid lives in shared memory of one CTA; nsweeps red-black SOR sweeps, one
// __syncthreads per colour.
template <typename T>
__global__ void __launch_bounds__(512)
    k_coarse_solve(Op op, T* __restrict__ phi, const T* __restrict__ rhs, T omega, int nsweeps) {
    extern __shared__ unsigned char smraw[];
    T* s = reinterpret_cast<T*>(smraw);
    const int n0 = op.n[0], n1 = op.n[1], n2 = op.n[2], n = n0 * n1 * n2;
    for (int q = threadIdx.x; q < n; q += blockDim.x) s[q] = phi[q];
    __syncthreads();
    const ArrLd<T> ld{s};
    for (int sw = 0; sw < nsweeps; ++sw)
        for (int colour = 0; colour < 2; ++colour) {
            for (int q = threadIdx.x; q < n; q += blockDim.x) {
                const int i = q % n0, j = (q / n0) % n1, k = q / (n0 * n1);
                if (((i + j + k) & 1) != colour) continue;
                const T sum = row_offsum<T, KIND_CART2>(op, ld, i, j, k, false);
                const T d = row_diag<T, KIND_CART2>(op, i, j, k);
                const T gs = (sum - rhs[q]) / d;
                const T old = s[q];
                s[q] = fma_(omega, gs - old, old);
            }
            __syncthreads();
        }
    for (int q = threadIdx.x; q < n; q += blockDim.x) phi[q] = s[q];
}

// ---- the bottom of the V-cycle in one CTA ---------------------------------------------------------------------------------
// Levels of at most 16^3 points are launch-latency bound (a dozen kernels of ~10 us each, plus 2 x 50 colour
// half-sweeps on the coarsest grid).  This kernel runs the whole sub-cycle below such a level — pre-smoothing,
// residual, restriction, recursion, coarsest-level SOR, prolongation + correction, post-smoothing — in the shared memory
// of a single CTA, with the same arithmetic (row_offsum / row_diag, restriction and interpolation weights, order of
// operations) as the per-level kernels above, so the results are bit-identical to the multi-launch path.
constexpr int kBottomMaxLevels = 4;
struct BottomArgs {
    Op op[kBottomMaxLevels];
    int nlev;
    int nu1, nu2, csweeps, restriction;
    double omega_c;
};

// nsweeps red-black sweeps on a grid of at most 4 x 1024 points held in shared memory.  Every thread first works out,
// once, what its (up to four) points need — which neighbours exist, the diagonal and its reciprocal, the right-hand side
// — so that a colour half-sweep is a handful of shared-memory reads and one exact division (div_by).
template <typename T>
__device__ void bottom_smooth(const Op& op, T* phi, const T* rhs, T omega, int nsweeps) {
    constexpr int MP = 4;
    const int n0 = op.n[0], n1 = op.n[1], n2 = op.n[2], n01 = n0 * n1, n = n01 * n2;
    const T c0 = (T)op.c[0], c1 = (T)op.c[1], c2 = (T)op.c[2];
    int msk[MP];
    T dd[MP], rd[MP], f[MP];
#pragma unroll
    for (int m = 0; m < MP; ++m) {
        const int q = threadIdx.x + m * 1024;
        msk[m] = 0;
        dd[m] = rd[m] = f[m] = (T)1;
        if (q < n) {
            const int i = q % n0, j = (q / n0) % n1, k = q / n01;
            msk[m] = (i > 0 ? 1 : 0) | (i < n0 - 1 ? 2 : 0) | (j > 0 ? 4 : 0) | (j < n1 - 1 ? 8 : 0) | (k > 0 ? 16 : 0) |
                     (k < n2 - 1 ? 32 : 0) | (((i + j + k) & 1) << 6) | 128;
            dd[m] = row_diag<T, KIND_CART2>(op, i, j, k);
            rd[m] = (T)1 / dd[m];
            f[m] = rhs[q];
        }
    }
    for (int sw = 0; sw < nsweeps; ++sw)
        for (int colour = 0; colour < 2; ++colour) {
#pragma unroll
            for (int m = 0; m < MP; ++m) {
                const int q = threadIdx.x + m * 1024, k = msk[m];
                if (!(k & 128) || ((k >> 6) & 1) != colour) continue;
                const T xm = (k & 1) ? phi[q - 1] : (T)0, xp = (k & 2) ? phi[q + 1] : (T)0;
                const T ym = (k & 4) ? phi[q - n0] : (T)0, yp = (k & 8) ? phi[q + n0] : (T)0;
                const T zm = (k & 16) ? phi[q - n01] : (T)0, zp = (k & 32) ? phi[q + n01] : (T)0;
                T s = (xm + xp) * c0;
                s = fma_(ym + yp, c1, s);
                s = fma_(zm + zp, c2, s);
                const T gs = div_by<T>(s - f[m], dd[m], rd[m]);
                const T old = phi[q];
                phi[q] = fma_(omega, gs - old, old);
            }
            __syncthreads();
        }
}

template <typename T>
__global__ void __launch_bounds__(1024) k_mg_bottom(const BottomArgs a, T* __restrict__ g_phi, const T* __restrict__ g_rhs) {
    extern __shared__ __align__(16) unsigned char smraw[];
    T* base = reinterpret_cast<T*>(smraw);
    T *phi[kBottomMaxLevels], *rhs[kBottomMaxLevels], *res[kBottomMaxLevels];
    int npt[kBottomMaxLevels];
    for (int l = 0; l < a.nlev; ++l) {
        npt[l] = a.op[l].n[0] * a.op[l].n[1] * a.op[l].n[2];
        phi[l] = base;
        rhs[l] = base + npt[l];
        res[l] = base + 2 * npt[l];
        base += 3 * npt[l];
    }
    for (int q = threadIdx.x; q < npt[0]; q += blockDim.x) {
        phi[0][q] = g_phi[q];
        rhs[0][q] = g_rhs[q];
    }
    __syncthreads();
    // downward leg
    for (int l = 0; l + 1 < a.nlev; ++l) {
        const Op& f = a.op[l];
        const Op& c = a.op[l + 1];
        bottom_smooth<T>(f, phi[l], rhs[l], (T)1, a.nu1);
        const ArrLd<T> ld{phi[l]};
        for (int q = threadIdx.x; q < npt[l]; q += blockDim.x) {
            const int i = q % f.n[0], j = (q / f.n[0]) % f.n[1], k = q / (f.n[0] * f.n[1]);
            res[l][q] = rhs[l][q] - row_apply<T, KIND_CART2>(f, ld, i, j, k, false);
        }
        __syncthreads();
        for (int q = threadIdx.x; q < npt[l + 1]; q += blockDim.x) {
            const int I = q % c.n[0], J = (q / c.n[0]) % c.n[1], K = q / (c.n[0] * c.n[1]);
            rhs[l + 1][q] = restrict_cell<T>(f, res[l], I, J, K, a.restriction);
            phi[l + 1][q] = (T)0;
        }
        __syncthreads();
    }
    // coarsest level
    {
        const int l = a.nlev - 1;
        bottom_smooth<T>(a.op[l], phi[l], rhs[l], (T)a.omega_c, a.csweeps);
    }
    // upward leg
    for (int l = a.nlev - 2; l >= 0; --l) {
        const Op& f = a.op[l];
        const Op& c = a.op[l + 1];
        for (int q = threadIdx.x; q < npt[l]; q += blockDim.x) {
            const int i = q % f.n[0], j = (q / f.n[0]) % f.n[1], k = q / (f.n[0] * f.n[1]);
            const int I = i >> 1, J = j >> 1, K = k >> 1;
            const int In = I + ((i & 1) ? 1 : -1), Jn = J + ((j & 1) ? 1 : -1), Kn = K + ((k & 1) ? 1 : -1);
            T ey[2];
            for (int cc = 0; cc < 2; ++cc) {
                const int KK = cc ? Kn : K;
                T ex[2];
                for (int b = 0; b < 2; ++b) {
                    const int JJ = b ? Jn : J;
                    const T nearv = coarse_val(c, phi[l + 1], I, JJ, KK), farv = coarse_val(c, phi[l + 1], In, JJ, KK);
                    ex[b] = fma_((T)0.75, nearv, (T)0.25 * farv);
                }
                ey[cc] = fma_((T)0.75, ex[0], (T)0.25 * ex[1]);
            }
            phi[l][q] += fma_((T)0.75, ey[0], (T)0.25 * ey[1]);
        }
        __syncthreads();
        bottom_smooth<T>(f, phi[l], rhs[l], (T)1, a.nu2);
    }
    for (int q = threadIdx.x; q < npt[0]; q += blockDim.x) g_phi[q] = phi[0][q];
}

// Runs levels first..last of the hierarchy (ops[] = their operators) in one CTA; UNSUPPORTED if they do not fit.
template <typename T>
static int bottom_t(poisson_ctx* ctx, const Op* ops, int nlev, T* phi, const T* rhs, int nu1, int nu2, int csweeps,
                    double omega_c) {
    if (nlev < 1 || nlev > kBottomMaxLevels) return POISSON_UNSUPPORTED;
    BottomArgs a;
    size_t elems = 0;
    for (int l = 0; l < nlev; ++l) {
        a.op[l] = ops[l];
        elems += 3 * (size_t)ops[l].n[0] * ops[l].n[1] * ops[l].n[2];
    }
    const size_t bytes = elems * sizeof(T);
    if (bytes > 200 * 1024) return POISSON_UNSUPPORTED;
    a.nlev = nlev;
    a.nu1 = nu1;
    a.nu2 = nu2;
    a.csweeps = csweeps;
    a.restriction = ctx->opt_restriction;
    a.omega_c = omega_c;
    const int rc = kernel_ready(ctx, k_mg_bottom<T>, 1024, 200 * 1024);
    if (rc != POISSON_OK) return rc;
    PB_LAUNCH(ctx, KID_MG_COARSE, (k_mg_bottom<T><<<1, 1024, bytes, ctx->stream>>>(a, phi, rhs)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}
int launch_mg_bottom(poisson_ctx* ctx, const Op* ops, int nlev, double* phi, const double* rhs, int nu1, int nu2,
                     int csweeps, double omega_c) {
    return bottom_t<double>(ctx, ops, nlev, phi, rhs, nu1, nu2, csweeps, omega_c);
}
int launch_mg_bottom32(poisson_ctx* ctx, const Op* ops, int nlev, float* phi, const float* rhs, int nu1, int nu2,
                       int csweeps, double omega_c) {
    return bottom_t<float>(ctx, ops, nlev, phi, rhs, nu1, nu2, csweeps, omega_c);
}

template <typename T>
static int restrict_t(poisson_ctx* ctx, const Op& fine, const Op& coarse, const T* r, T* fc, int restriction) {
    dim3 b(32, 8), g((coarse.n[0] + 31) / 32, (coarse.n[1] + 7) / 8, coarse.n[2]);
    const bool two_to_one = fine.n[0] == 2 * coarse.n[0] && fine.n[1] == 2 * coarse.n[1] && fine.n[2] == 2 * coarse.n[2];
    if (restriction == 0 && two_to_one && ctx->opt_path != 1)
        PB_LAUNCH(ctx, KID_MG_RESTRICT, (k_restrict_v<T><<<g, b, 0, ctx->stream>>>(fine, coarse, r, fc)));
    else
        PB_LAUNCH(ctx, KID_MG_RESTRICT, (k_restrict<T><<<g, b, 0, ctx->stream>>>(fine, coarse, r, fc, restriction)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}
int launch_restrict(poisson_ctx* ctx, const Op& f, const Op& c, const double* r, double* fc, int rs) {
    return restrict_t<double>(ctx, f, c, r, fc, rs);
}
int launch_restrict32(poisson_ctx* ctx, const Op& f, const Op& c, const float* r, float* fc, int rs) {
    return restrict_t<float>(ctx, f, c, r, fc, rs);
}

template <typename T>
static int prolong_t(poisson_ctx* ctx, const Op& fine, const Op& coarse, const T* ec, T* phi) {
    dim3 b(32, 8), g((coarse.n[0] + 31) / 32, (coarse.n[1] + 7) / 8, coarse.n[2]);
    PB_LAUNCH(ctx, KID_MG_PROLONG, (k_prolong_add<T><<<g, b, 0, ctx->stream>>>(fine, coarse, ec, phi)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}
int launch_prolong_add(poisson_ctx* ctx, const Op& f, const Op& c, const double* ec, double* phi) {
    return prolong_t<double>(ctx, f, c, ec, phi);
}
int launch_prolong_add32(poisson_ctx* ctx, const Op& f, const Op& c, const float* ec, float* phi) {
    return prolong_t<float>(ctx, f, c, ec, phi);
}

int launch_add32to64(poisson_ctx* ctx, size_t n, const float* e, double* phi) {
    size_t blocks = (n + 2047) / 2048;
    if (blocks > (size_t)ctx->num_sms * 16) blocks = (size_t)ctx->num_sms * 16;
    PB_LAUNCH(ctx, KID_MG_AXPY, (k_add32to64<<<(int)blocks, 256, 0, ctx->stream>>>(n, e, phi)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

template <typename T>
static int coarse_t(poisson_ctx* ctx, const Op& op, T* phi, const T* rhs, T omega, int nsweeps) {
    const size_t n = (size_t)op.n[0] * op.n[1] * op.n[2];
    const size_t bytes = n * sizeof(T);
    if (bytes > 200 * 1024) return POISSON_UNSUPPORTED;  // caller falls back to per-colour launches
    if (bytes > 48 * 1024)
        PB_CUDA_OK(cudaFuncSetAttribute(k_coarse_solve<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    PB_LAUNCH(ctx, KID_MG_COARSE, (k_coarse_solve<T><<<1, 512, bytes, ctx->stream>>>(op, phi, rhs, omega, nsweeps)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}
int launch_coarse_solve(poisson_ctx* ctx, const Op& op, double* phi, const double* rhs, double omega, int nsweeps) {
    return coarse_t<double>(ctx, op, phi, rhs, omega, nsweeps);
}
int launch_coarse_solve32(poisson_ctx* ctx, const Op& op, float* phi, const float* rhs, float omega, int nsweeps) {
    return coarse_t<float>(ctx, op, phi, rhs, omega, nsweeps);
}

}  // namespace pb
