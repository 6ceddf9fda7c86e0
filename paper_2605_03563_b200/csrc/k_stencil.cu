// k_stencil.cu — generic (any shape, direct global loads) stencil apply / residual and red-black SOR kernels.
// Each thread owns a column (i,j) and marches a chunk of k planes, so x/y neighbours come from L1 and the previous
// planes from L1/L2.  Used for small or odd-shaped grids (multigrid levels, 32^3) and as the always-available path;
// large aligned grids take the plane-pipeline kernels of k_plane.cu.
//   apply:   PAPER.md:43-49 (Eq. 1-2), 57        residual: PAPER.md:55        red-black SOR: PAPER.md:59-63
#include "stencil.cuh"

namespace pb {

constexpr int BX = 64, BY = 4;

static inline int pick_kc(const Op& op, int sms) {
    // enough blocks to fill the machine a few times, few enough that the last-block reduction stays short
    const long cols = (long)((op.n[0] + BX - 1) / BX) * ((op.n[1] + BY - 1) / BY);
    int kc = op.n[2];
    while (kc > 8 && cols * ((op.n[2] + kc - 1) / kc) < 8L * sms) kc = (kc + 1) / 2;
    return kc;
}

// MODE 0: out = L v.  MODE 1: out = rhs - L v.  RED: sum(out^2), sum(out) -> scal[0], scal[1].
template <typename T, int KIND, int MODE, bool RED>
__global__ void __launch_bounds__(BX* BY)
    k_apply(Op op, const T* __restrict__ v, const T* __restrict__ rhs, T* __restrict__ out, float* __restrict__ out32,
            bool ug, int kc, RedBuf rb, double* scal) {
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    double s2 = 0.0, s1 = 0.0;
    if (i < op.n[0] && j < op.n[1]) {
        for (int k = k0; k < k1; ++k) {
            const size_t p = gidx(op, i, j, k);
            const T lv = row_apply<T, KIND>(op, ArrLd<T>{v}, i, j, k, ug);
            const T o = MODE ? (rhs[p] - lv) : lv;
            if (out) out[p] = o;
            if (out32) out32[p] = (float)o;
            if (RED) {
                s2 = fma((double)o, (double)o, s2);
                s1 += (double)o;
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

template <typename T, int KIND>
__global__ void __launch_bounds__(BX* BY)
    k_rbsor_half(Op op, T* phi, const T* __restrict__ rhs, T omega, int colour, bool ug, int kc) {
    const int ti = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    if (j >= op.n[1]) return;
    for (int k = k0; k < k1; ++k) {
        const int i = 2 * ti + ((j + k + colour) & 1);
        if (i >= op.n[0]) continue;
        const size_t p = gidx(op, i, j, k);
        const T s = row_offsum<T, KIND>(op, ArrLd<T>{phi}, i, j, k, ug);
        const T d = row_diag<T, KIND>(op, i, j, k);
        const T gs = (s - rhs[p]) / d;
        const T old = phi[p];
        phi[p] = fma_(omega, gs - old, old);
    }
}

// The same half-sweep with a position-dependent factor omega(i,j) (Eq. 7: "the values of omega_n are not
// uniform, but depend on position on the grid"); om holds the current member of the sequence of Eq. 6 per (i,j).
template <typename T, int KIND>
__global__ void __launch_bounds__(BX* BY)
    k_rbsor_half_local(Op op, T* phi, const T* __restrict__ rhs, const double* __restrict__ om, int colour, bool ug, int kc) {
    const int ti = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    if (j >= op.n[1]) return;
    for (int k = k0; k < k1; ++k) {
        const int i = 2 * ti + ((j + k + colour) & 1);
        if (i >= op.n[0]) continue;
        const size_t p = gidx(op, i, j, k);
        const T s = row_offsum<T, KIND>(op, ArrLd<T>{phi}, i, j, k, ug);
        const T d = row_diag<T, KIND>(op, i, j, k);
        const T gs = (s - rhs[p]) / d;
        const T old = phi[p];
        phi[p] = fma_((T)om[(size_t)j * op.n[0] + i], gs - old, old);
    }
}

// Eq. 6 advanced by one member per (i,j): omega_0 = 1, omega_1 = 1/(1 - rJ^2/2), omega_{n+1} = 1/(1 - rJ^2 omega_n/4).
__global__ void __launch_bounds__(256) k_omega_advance(size_t n, const double* __restrict__ rj, double* __restrict__ om, int n_next) {
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n) return;
    const double r = rj[q];
    om[q] = n_next == 0 ? 1.0 : (n_next == 1 ? 1.0 / (1.0 - 0.5 * r * r) : 1.0 / (1.0 - 0.25 * r * r * om[q]));
}

static dim3 grid_for(const Op& op, int kc, bool half_x) {
    const int nxe = half_x ? (op.n[0] + 1) / 2 : op.n[0];
    return dim3((nxe + BX - 1) / BX, (op.n[1] + BY - 1) / BY, (op.n[2] + kc - 1) / kc);
}

template <typename T, int KIND>
static int apply_dispatch(poisson_ctx* ctx, const Op& op, const T* v, const T* rhs, T* out, float* out32, int mode,
                          bool ug, bool reduce) {
    const int kc = pick_kc(op, ctx->num_sms);
    const dim3 g = grid_for(op, kc, false), b(BX, BY);
    if ((size_t)g.x * g.y * g.z > (size_t)kMaxRedBlocks) return fail(ctx, POISSON_UNSUPPORTED, "grid too large for the reduction buffer");
    cudaStream_t s = ctx->stream;
    pre_launch(ctx, KID_APPLY);
    if (mode == 0)
        k_apply<T, KIND, 0, false><<<g, b, 0, s>>>(op, v, rhs, out, out32, ug, kc, ctx->red, ctx->d_scal);
    else if (!reduce)
        k_apply<T, KIND, 1, false><<<g, b, 0, s>>>(op, v, rhs, out, out32, ug, kc, ctx->red, ctx->d_scal);
    else
        k_apply<T, KIND, 1, true><<<g, b, 0, s>>>(op, v, rhs, out, out32, ug, kc, ctx->red, ctx->d_scal);
    post_launch(ctx, KID_APPLY);
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

int launch_apply(poisson_ctx* ctx, const Op& op, int kind, const double* v, const double* rhs, double* out, int mode,
                 bool ug, bool reduce) {
    if (kind == KIND_CART2 && apply_bulk_ok(ctx, op)) {
        const int rc = apply_bulk(ctx, op, v, rhs, out, nullptr, mode, ug, reduce);
        if (rc != POISSON_UNSUPPORTED) return rc;  // no tensor-map encoder in this driver: thread-staged kernel
    }
    if (kind == KIND_CART2 && apply7_ok(ctx, op)) return apply7(ctx, op, v, rhs, out, nullptr, mode, ug, reduce);
    if (plane_ok(ctx, op)) return plane_apply(ctx, op, kind, v, rhs, out, nullptr, mode, ug, reduce);
    switch (kind) {
        case KIND_CART2: return apply_dispatch<double, KIND_CART2>(ctx, op, v, rhs, out, nullptr, mode, ug, reduce);
        case KIND_CART6: return apply_dispatch<double, KIND_CART6>(ctx, op, v, rhs, out, nullptr, mode, ug, reduce);
        default: return apply_dispatch<double, KIND_SPH>(ctx, op, v, rhs, out, nullptr, mode, ug, reduce);
    }
}

int launch_apply32(poisson_ctx* ctx, const Op& op, const float* v, const float* rhs, float* out, int mode) {
    if (apply7_ok(ctx, op)) return apply7_32(ctx, op, v, rhs, out, mode);
    return apply_dispatch<float, KIND_CART2>(ctx, op, v, rhs, out, nullptr, mode, false, false);
}

int launch_residual_to32(poisson_ctx* ctx, const Op& op, const double* v, const double* rhs, float* out32, bool ug) {
    if (apply_bulk_ok(ctx, op)) {
        const int rc = apply_bulk(ctx, op, v, rhs, nullptr, out32, 1, ug, true);
        if (rc != POISSON_UNSUPPORTED) return rc;
    }
    if (apply7_ok(ctx, op)) return apply7(ctx, op, v, rhs, nullptr, out32, 1, ug, true);
    if (plane_ok(ctx, op)) return plane_apply(ctx, op, KIND_CART2, v, rhs, nullptr, out32, 1, ug, true);
    return apply_dispatch<double, KIND_CART2>(ctx, op, v, rhs, nullptr, out32, 1, ug, true);
}

template <typename T, int KIND>
static int rbsor_dispatch(poisson_ctx* ctx, const Op& op, T* phi, const T* rhs, T omega, int nsweeps, bool ug) {
    const int kc = pick_kc(op, ctx->num_sms);
    const dim3 g = grid_for(op, kc, true), b(BX, BY);
    for (int s = 0; s < nsweeps; ++s)
        for (int colour = 0; colour < 2; ++colour) {
            PB_LAUNCH(ctx, KID_RBSOR, (k_rbsor_half<T, KIND><<<g, b, 0, ctx->stream>>>(op, phi, rhs, omega, colour, ug, kc)));
        }
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

// One colour half-sweep with the generic kernel (building block of the preconditioner and of the omega sequences).
int launch_rbsor_half(poisson_ctx* ctx, const Op& op, int kind, double* phi, const double* rhs, double omega, int colour,
                      bool ug, int kid) {
    if (kind == KIND_CART6)
        return fail(ctx, POISSON_UNSUPPORTED, "red-black sweeps need a radius-1 stencil (two colours, PAPER.md:61)");
    const int kc = pick_kc(op, ctx->num_sms);
    const dim3 g = grid_for(op, kc, true), b(BX, BY);
    if (kind == KIND_CART2)
        PB_LAUNCH(ctx, kid, (k_rbsor_half<double, KIND_CART2><<<g, b, 0, ctx->stream>>>(op, phi, rhs, omega, colour, ug, kc)));
    else
        PB_LAUNCH(ctx, kid, (k_rbsor_half<double, KIND_SPH><<<g, b, 0, ctx->stream>>>(op, phi, rhs, omega, colour, ug, kc)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

// nsweeps sweeps with one factor per colour half-sweep: omegas[0 .. 2 nsweeps) (Eq. 6).
int launch_rbsor_seq(poisson_ctx* ctx, const Op& op, int kind, double* phi, const double* rhs, const double* omegas,
                     int nsweeps, bool ug) {
    if (kind == KIND_CART2 && nsweeps > 0 && sor_fused_ok(ctx, op)) {
        double* tmp = (double*)sor_scratch(ctx, (size_t)op.n[0] * op.n[1] * op.n[2] * sizeof(double));
        if (!tmp) return POISSON_OUT_OF_MEMORY;
        return sor_fused_seq(ctx, op, phi, tmp, rhs, omegas, nsweeps, ug, nullptr);
    }
    for (int m = 0; m < 2 * nsweeps; ++m) {
        const int rc = launch_rbsor_half(ctx, op, kind, phi, rhs, omegas[m], m & 1, ug, KID_RBSOR);
        if (rc != POISSON_OK) return rc;
    }
    return POISSON_OK;
}

// nsweeps sweeps with the position-dependent sequence: d_rj = local Jacobi radius per (i,j), d_om = work array.
int launch_rbsor_local(poisson_ctx* ctx, const Op& op, int kind, double* phi, const double* rhs, const double* d_rj,
                       double* d_om, int nsweeps, int start_n, bool ug) {
    if (kind == KIND_CART6)
        return fail(ctx, POISSON_UNSUPPORTED, "red-black sweeps need a radius-1 stencil (two colours, PAPER.md:61)");
    const size_t n2d = (size_t)op.n[0] * op.n[1];
    const int ob = (int)((n2d + 255) / 256);
    for (int n = 0; n <= start_n; ++n)
        PB_LAUNCH(ctx, KID_RBSOR, (k_omega_advance<<<ob, 256, 0, ctx->stream>>>(n2d, d_rj, d_om, n)));
    const int kc = pick_kc(op, ctx->num_sms);
    const dim3 g = grid_for(op, kc, true), b(BX, BY);
    for (int m = 0; m < 2 * nsweeps; ++m) {
        if (kind == KIND_CART2)
            PB_LAUNCH(ctx, KID_RBSOR, (k_rbsor_half_local<double, KIND_CART2><<<g, b, 0, ctx->stream>>>(op, phi, rhs, d_om, m & 1, ug, kc)));
        else
            PB_LAUNCH(ctx, KID_RBSOR, (k_rbsor_half_local<double, KIND_SPH><<<g, b, 0, ctx->stream>>>(op, phi, rhs, d_om, m & 1, ug, kc)));
        PB_LAUNCH(ctx, KID_RBSOR, (k_omega_advance<<<ob, 256, 0, ctx->stream>>>(n2d, d_rj, d_om, m + start_n + 1)));
    }
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

int launch_rbsor(poisson_ctx* ctx, const Op& op, int kind, double* phi, const double* rhs, double omega, int nsweeps,
                 bool ug) {
    if (kind == KIND_CART2 && nsweeps > 0 && sor_fused_ok(ctx, op)) {
        double* tmp = (double*)sor_scratch(ctx, (size_t)op.n[0] * op.n[1] * op.n[2] * sizeof(double));
        if (!tmp) return POISSON_OUT_OF_MEMORY;
        return sor_fused(ctx, op, phi, tmp, rhs, omega, nsweeps, ug);
    }
    if (kind == KIND_CART2) return rbsor_dispatch<double, KIND_CART2>(ctx, op, phi, rhs, omega, nsweeps, ug);
    if (kind == KIND_SPH) return rbsor_dispatch<double, KIND_SPH>(ctx, op, phi, rhs, omega, nsweeps, ug);
    return fail(ctx, POISSON_UNSUPPORTED,
                "red-black SOR needs a radius-1 stencil: two colours are not independent for order 6");
}

int launch_rbsor32(poisson_ctx* ctx, const Op& op, float* phi, const float* rhs, float omega, int nsweeps) {
    if (nsweeps > 0 && sor_fused_ok(ctx, op)) {
        float* tmp = (float*)sor_scratch(ctx, (size_t)op.n[0] * op.n[1] * op.n[2] * sizeof(float));
        if (!tmp) return POISSON_OUT_OF_MEMORY;
        return sor_fused32(ctx, op, phi, tmp, rhs, omega, nsweeps);
    }
    return rbsor_dispatch<float, KIND_CART2>(ctx, op, phi, rhs, omega, nsweeps, false);
}

int launch_rbsor_pp(poisson_ctx* ctx, const Op& op, double** cur, double* a, double* b, const double* rhs, double omega,
                    int nsweeps, bool ug) {
    if (nsweeps > 0 && a && b && sor_fused_ok(ctx, op))
        return sor_fused(ctx, op, *cur, *cur == a ? b : a, rhs, omega, nsweeps, ug, cur);
    return launch_rbsor(ctx, op, KIND_CART2, *cur, rhs, omega, nsweeps, ug);
}

int launch_rbsor_pp32(poisson_ctx* ctx, const Op& op, float** cur, float* a, float* b, const float* rhs, float omega,
                      int nsweeps) {
    if (nsweeps > 0 && a && b && sor_fused_ok(ctx, op))
        return sor_fused32(ctx, op, *cur, *cur == a ? b : a, rhs, omega, nsweeps, cur);
    return launch_rbsor32(ctx, op, *cur, rhs, omega, nsweeps);
}

}  // namespace pb
