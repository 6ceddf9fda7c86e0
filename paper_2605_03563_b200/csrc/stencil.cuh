// stencil.cuh — device functions: matrix rows of the discrete Laplacian (direct global-memory form) and the
// single-pass deterministic grid reduction.  Evaluation order is the canonical one of DESIGN.md ("Arithmetic
// order"), so pointwise results agree with an IEEE implementation of the same formulas to the last bit.
// Compiled with -fmad=false: every fused multiply-add below is explicit.
#pragma once
#include "common.cuh"

namespace pb {

__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }

__device__ __forceinline__ size_t gidx(const Op& op, int i, int j, int k) {
    return ((size_t)k * op.n[1] + j) * op.n[0] + i;
}

// Neighbour of (i,j,k) at offset s along axis A; out-of-range handled per face type (include/poisson.h).
// `ld(p,i,j,k)` returns the value of the vector at point (i,j,k), linear index p: a plain array (ArrLd) or a vector formed on the fly
// (e.g. p_new = r + beta p_old inside the fused CG pass).
template <typename T>
struct ArrLd {
    const T* v;
    __device__ __forceinline__ T operator()(size_t p, int, int, int) const { return v[p]; }
};

template <typename T, int A, class Ld>
__device__ __forceinline__ T nb(const Op& op, const Ld& v, int i, int j, int k, int s, bool use_ghost) {
    const int n = op.n[A];
    int q = (A == 0 ? i : (A == 1 ? j : k)) + s;
    if (q >= 0 && q < n)
        return v(gidx(op, A == 0 ? q : i, A == 1 ? q : j, A == 2 ? q : k), A == 0 ? q : i, A == 1 ? q : j, A == 2 ? q : k);
    const int f = 2 * A + (q < 0 ? 0 : 1);
    const int bc = op.bc[f];
    if (bc == POISSON_BC_PERIODIC) {
        q = q < 0 ? q + n : q - n;
        return v(gidx(op, A == 0 ? q : i, A == 1 ? q : j, A == 2 ? q : k), A == 0 ? q : i, A == 1 ? q : j, A == 2 ? q : k);
    }
    if (bc == POISSON_BC_DIRICHLET_GHOST && use_ghost && op.ghost[f] != nullptr) {
        const int layer = q < 0 ? (-1 - q) : (q - n);
        constexpr int A1 = (A == 0) ? 1 : 0, A2 = (A == 2) ? 1 : 2;
        const int q1 = (A1 == 0 ? i : j), q2 = (A2 == 1 ? j : k);
        return (T)op.ghost[f][((size_t)layer * op.n[A2] + q2) * op.n[A1] + q1];
    }
    return (T)0;
}

// Diagonal d of the row: (L v)_ijk = offsum - d v_ijk.
template <typename T, int KIND>
__device__ __forceinline__ T row_diag(const Op& op, int i, int j, int k) {
    if (KIND == KIND_SPH) return fma_((T)op.ir2[i], (T)op.dt[j], (T)op.dr[i]);
    const T c0 = (T)op.c[0], c1 = (T)op.c[1], c2 = (T)op.c[2];
    if (KIND == KIND_CART6) return (T)(49.0 / 18.0) * ((c0 + c1) + c2);
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

template <typename T, int A, class Ld>
__device__ __forceinline__ T axis6(const Op& op, const Ld& v, int i, int j, int k, bool ug) {
    const T p1 = nb<T, A>(op, v, i, j, k, -1, ug) + nb<T, A>(op, v, i, j, k, +1, ug);
    const T p2 = nb<T, A>(op, v, i, j, k, -2, ug) + nb<T, A>(op, v, i, j, k, +2, ug);
    const T p3 = nb<T, A>(op, v, i, j, k, -3, ug) + nb<T, A>(op, v, i, j, k, +3, ug);
    T u = (T)(3.0 / 2.0) * p1;
    u = fma_((T)(-3.0 / 20.0), p2, u);
    u = fma_((T)(1.0 / 90.0), p3, u);
    return u;
}

// Off-diagonal part of the row.  When closure (gamma != 0) is active Dirichlet ghosts contribute nothing here.
template <typename T, int KIND, class Ld>
__device__ __forceinline__ T row_offsum(const Op& op, const Ld& v, int i, int j, int k, bool use_ghost) {
    const bool ug = use_ghost && op.gamma == 0.0;
    if (KIND == KIND_SPH) {
        const T vrm = nb<T, 0>(op, v, i, j, k, -1, ug), vrp = nb<T, 0>(op, v, i, j, k, +1, ug);
        const T vtm = nb<T, 1>(op, v, i, j, k, -1, ug), vtp = nb<T, 1>(op, v, i, j, k, +1, ug);
        const T vpm = nb<T, 2>(op, v, i, j, k, -1, ug), vpp = nb<T, 2>(op, v, i, j, k, +1, ug);
        T s = (T)op.ar_m[i] * vrm;
        s = fma_((T)op.ar_p[i], vrp, s);
        T t = (T)op.at_m[j] * vtm;
        t = fma_((T)op.at_p[j], vtp, t);
        t = fma_((T)op.cp[j], vpm + vpp, t);
        return fma_((T)op.ir2[i], t, s);
    }
    const T c0 = (T)op.c[0], c1 = (T)op.c[1], c2 = (T)op.c[2];
    if (KIND == KIND_CART6) {
        const T t0 = axis6<T, 0>(op, v, i, j, k, ug);
        const T t1 = axis6<T, 1>(op, v, i, j, k, ug);
        const T t2 = axis6<T, 2>(op, v, i, j, k, ug);
        T s = t0 * c0;
        s = fma_(t1, c1, s);
        s = fma_(t2, c2, s);
        return s;
    }
    const T px = nb<T, 0>(op, v, i, j, k, -1, ug) + nb<T, 0>(op, v, i, j, k, +1, ug);
    const T py = nb<T, 1>(op, v, i, j, k, -1, ug) + nb<T, 1>(op, v, i, j, k, +1, ug);
    const T pz = nb<T, 2>(op, v, i, j, k, -1, ug) + nb<T, 2>(op, v, i, j, k, +1, ug);
    T s = px * c0;
    s = fma_(py, c1, s);
    s = fma_(pz, c2, s);
    return s;
}

template <typename T, int KIND, class Ld>
__device__ __forceinline__ T row_apply(const Op& op, const Ld& v, int i, int j, int k, bool use_ghost) {
    return fma_(-row_diag<T, KIND>(op, i, j, k), v(gidx(op, i, j, k), i, j, k),
                row_offsum<T, KIND>(op, v, i, j, k, use_ghost));
}

// ---- division by a repeated divisor --------------------------------------------------------------------------------
// Correctly rounded a / d from the correctly rounded reciprocal rd = 1/d: two Markstein corrections (exact residuals
// by fma).  Same result as IEEE division (no overflow / underflow on this path) without its slow-path branches.
template <typename T>
__device__ __forceinline__ T div_by(T a, T d, T rd) {
    T q = a * rd;
    T r = fma_(-d, q, a);
    q = fma_(r, rd, q);
    r = fma_(-d, q, a);
    return fma_(r, rd, q);
}

// ---- full-weighting restriction, one axis at a time -------------------------------------------------------------------
// R = (1/8)[1 3 3 1] per axis (cell-centred 2:1 coarsening, the transpose of trilinear interpolation).
// Every restriction kernel evaluates it axis by axis — x, then y, then z — each axis as acc = fma(w_a, v_a, acc) over
// a = 0..3 from acc = 0, cells outside the domain skipped: 12 multiply-adds per coarse cell instead of the 64 of the
// tensor-product sum, and the same bits from every kernel (the one-kernel-per-operator path, the bottom-of-the-cycle
// kernel, the fused residual + restriction pass, whose z sum runs along with the planes).  The values differ from the
// 64-term sum only by the rounding of the partial sums.  The 8-cell average sums pairs the same way: x, y, z, then / 8.
template <typename T>
__device__ __forceinline__ T fw_acc(T acc, int a, T v) {
    return fma_((a == 0 || a == 3) ? (T)0.125 : (T)0.375, v, acc);
}

// ---- single-pass grid reduction -------------------------------------------------------------------------------------
__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// Every thread of every block calls this with its NRED partial sums.  Warp shuffles -> shared memory -> one set of
// per-block partials in global memory -> the last block to arrive adds all block partials in a fixed order and
// calls epi(totals) from one thread.  Deterministic for a given launch configuration; no second kernel, no host sync.
template <int NRED, class Epi>
__device__ __forceinline__ void grid_reduce(double (&v)[NRED], RedBuf rb, Epi epi) {
    __shared__ double sm[NRED][32];
    __shared__ int is_last;
    const int nthr = blockDim.x * blockDim.y * blockDim.z;
    const int tid = (threadIdx.z * blockDim.y + threadIdx.y) * blockDim.x + threadIdx.x;
    const int lane = tid & 31, w = tid >> 5, nw = (nthr + 31) >> 5;
    const unsigned nblk = gridDim.x * gridDim.y * gridDim.z;
    const unsigned bid = (blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
#pragma unroll
    for (int r = 0; r < NRED; ++r) {
        const double x = warp_sum(v[r]);
        if (lane == 0) sm[r][w] = x;
    }
    __syncthreads();
    if (w == 0) {
#pragma unroll
        for (int r = 0; r < NRED; ++r) {
            double x = lane < nw ? sm[r][lane] : 0.0;
            x = warp_sum(x);
            if (lane == 0) rb.partials[(size_t)bid * NRED + r] = x;
        }
    }
    if (tid == 0) {
        __threadfence();
        const unsigned prev = atomicInc(rb.counter, nblk - 1);
        is_last = (prev == nblk - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double tot[NRED];
#pragma unroll
    for (int r = 0; r < NRED; ++r) {
        double acc = 0.0;
        for (unsigned b = tid; b < nblk; b += nthr) acc += __ldcg(&rb.partials[(size_t)b * NRED + r]);
        acc = warp_sum(acc);
        if (lane == 0) sm[r][w] = acc;
    }
    __syncthreads();
    if (w == 0) {
#pragma unroll
        for (int r = 0; r < NRED; ++r) {
            double x = lane < nw ? sm[r][lane] : 0.0;
            tot[r] = warp_sum(x);
        }
        if (lane == 0) epi(tot);
    }
}

// Scalars after the initial-residual pass (t[0] = sum r^2, t[1] = sum r).  With ctl->confirm set the pass was the
// true-residual check of a BiCGSTAB solution the recurrence calls converged: accept, or carry on from the true
// residual as from a fresh start (r^_0 := r was stored by the pass, beta = 0 gives p := r), keeping it and rr0.
__device__ __forceinline__ void krylov_init_finish(KrylovCtl* ctl, double* hist, const double* t) {
    const double mu = ctl->project ? t[1] / ctl->npoints : 0.0;
    const double rr = ctl->project ? fma(-ctl->npoints * mu, mu, t[0]) : t[0];
    ctl->mu = mu;
    ctl->rr = rr;
    ctl->rho = rr;
    ctl->r0n2 = rr;
    ctl->restart = 0;
    ctl->beta = 0.0;
    if (ctl->confirm) {
        ctl->confirm = 0;
        const bool fin = isfinite(rr);
        const bool ok = fin && sqrt(rr) <= sqrt(ctl->tol2) * sqrt(ctl->rr0);
        // rtol below the attainable accuracy: the recurrence keeps converging, the true residual never does
        if (!ok) ctl->nconf_failed += 1;
        const bool stall = ctl->nconf_failed > kMaxBicgConfirm;
        ctl->done = (ok || !fin || stall || ctl->it >= ctl->max_it) ? 1 : 0;
        ctl->status = ok ? POISSON_OK : (fin ? POISSON_NOT_CONVERGED : POISSON_BREAKDOWN);
        return;
    }
    ctl->rr0 = rr;
    ctl->nconf_failed = 0;
    ctl->nrestarts = 0;
    ctl->alpha = 0.0;
    ctl->omega = 0.0;
    ctl->it = 0;
    // a zero initial residual is convergence; a non-finite one (NaN/Inf in rhs or in the initial guess) is BREAKDOWN in
    // both modes — `!(rr > 0)` would call NaN converged
    const bool fin = isfinite(rr);
    const int trivially_done = (!ctl->fixed && rr == 0.0) ? 1 : 0;
    ctl->done = (trivially_done || !fin) ? 1 : 0;
    ctl->status = !fin ? POISSON_BREAKDOWN : ((ctl->fixed || trivially_done) ? POISSON_OK : POISSON_NOT_CONVERGED);
    if (ctl->record && hist) hist[0] = 1.0;
}

}  // namespace pb
