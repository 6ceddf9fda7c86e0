// k_mg.cu — multigrid transfer operators and the coarsest-level solver.  PAPER.md:125-152 (Eq. 11-13), 205.
// Variant fixed by BASELINE.json config 3 / DESIGN.md reading C7: cell-centred 2:1 coarsening, full-weighting
// restriction as the transpose of trilinear interpolation ((1/8)[1 3 3 1] per axis, P = 8 R^T),
// trilinear prolongation with the level's ghost closure, coarsest level by red-black SOR sweeps in shared memory.
#include "stencil.cuh"

namespace pb {

template <typename T>
__global__ void __launch_bounds__(256)
    k_restrict(Op fine, Op coarse, const T* __restrict__ r, T* __restrict__ fc, int restriction) {
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    if (I >= coarse.n[0] || J >= coarse.n[1]) return;
    const double W[4] = {0.125, 0.375, 0.375, 0.125};
    T acc = 0;
    if (restriction == 1) {
        for (int c = 0; c < 2; ++c)
            for (int b = 0; b < 2; ++b)
                for (int a = 0; a < 2; ++a) acc += r[gidx(fine, 2 * I + a, 2 * J + b, 2 * K + c)];
        acc *= (T)0.125;
    } else {
#pragma unroll
        for (int c = 0; c < 4; ++c)
#pragma unroll
            for (int b = 0; b < 4; ++b)
#pragma unroll
                for (int a = 0; a < 4; ++a) {
                    const int i = 2 * I - 1 + a, j = 2 * J - 1 + b, k = 2 * K - 1 + c;
                    if (i < 0 || i >= fine.n[0] || j < 0 || j >= fine.n[1] || k < 0 || k >= fine.n[2]) continue;
                    acc += (T)(W[a] * W[b] * W[c]) * r[gidx(fine, i, j, k)];
                }
    }
    fc[gidx(coarse, I, J, K)] = acc;
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

template <typename T>
__global__ void __launch_bounds__(256)
    k_prolong_add(Op fine, Op coarse, const T* __restrict__ ec, T* __restrict__ phi) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= fine.n[0] || j >= fine.n[1]) return;
    const int I = i >> 1, J = j >> 1, K = k >> 1;
    const int In = I + ((i & 1) ? 1 : -1), Jn = J + ((j & 1) ? 1 : -1), Kn = K + ((k & 1) ? 1 : -1);
    T ey[2];
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        const int KK = c ? Kn : K;
        T ex[2];
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const int JJ = b ? Jn : J;
            const T nearv = coarse_val(coarse, ec, I, JJ, KK), farv = coarse_val(coarse, ec, In, JJ, KK);
            ex[b] = fma_((T)0.75, nearv, (T)0.25 * farv);
        }
        ey[c] = fma_((T)0.75, ex[0], (T)0.25 * ex[1]);
    }
    const T v = fma_((T)0.75, ey[0], (T)0.25 * ey[1]);
    phi[gidx(fine, i, j, k)] += v;
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

template <typename T>
static int restrict_t(poisson_ctx* ctx, const Op& fine, const Op& coarse, const T* r, T* fc, int restriction) {
    dim3 b(32, 8), g((coarse.n[0] + 31) / 32, (coarse.n[1] + 7) / 8, coarse.n[2]);
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
    dim3 b(64, 4), g((fine.n[0] + 63) / 64, (fine.n[1] + 3) / 4, fine.n[2]);
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
