// k_krylov.cu — generic (direct global load) fused passes of CG and BiCGSTAB.  PAPER.md:95-105; Saad Alg. 6.18, 7.7.
// Scalars (alpha, beta, omega, rho, ||r||^2, iteration counter, convergence flag) stay in device memory; the last
// block of each fused reduction computes the next ones, so an iteration never crosses to the host.
//   CG        pass A: x += alpha_prev p_old ; p = r + beta p_old ; q = L p ; sum p.q        -> alpha
//             pass B: r -= alpha q ; sum r^2 (and sum r for the periodic null-space projection) -> beta, convergence
//   BiCGSTAB  pass 1: p = r + beta (p - omega v) ; v = L D^-1 p ; sum r0^.v                  -> alpha
//             pass 2: s = r - alpha v ; t = L D^-1 s ; sum t.s, t.t                           -> omega
//             pass 3: x += alpha D^-1 p + omega D^-1 s ; r = s - omega t ; sum r.r, r0^.r     -> beta, convergence
// Vectors whose stencil is taken in the pass that forms them (p, v, s) are recomputed in the halo from read-only
// inputs and written to a different buffer (ping-pong), so no block reads what another block is writing.
#include <algorithm>

#include "stencil.cuh"

namespace pb {

constexpr int BX = 64, BY = 4;

static inline int pick_kc(const Op& op, int sms) {
    const long cols = (long)((op.n[0] + BX - 1) / BX) * ((op.n[1] + BY - 1) / BY);
    int kc = op.n[2];
    while (kc > 8 && cols * ((op.n[2] + kc - 1) / kc) < 8L * sms) kc = (kc + 1) / 2;
    return kc;
}
// The reduction buffer holds one set of partials per block: lengthen the z chunks until the grid fits, or refuse.
static int fit_grid(poisson_ctx* ctx, const Op& op, int nx_eff, int* kc, dim3* g) {
    for (;;) {
        *g = dim3((nx_eff + BX - 1) / BX, (op.n[1] + BY - 1) / BY, (op.n[2] + *kc - 1) / *kc);
        if ((size_t)g->x * g->y * g->z <= (size_t)kMaxRedBlocks) return POISSON_OK;
        if (*kc >= op.n[2]) return fail(ctx, POISSON_UNSUPPORTED, "grid too large for the reduction buffer");
        *kc = std::min(op.n[2], *kc * 2);
    }
}

__device__ __forceinline__ void finish_iteration(KrylovCtl* c, double* hist, double rr_new) {
    // shared tail of CG pass B and BiCGSTAB pass 3: count the iteration, record, test convergence
    const int it = c->it + 1;
    c->it = it;
    if (c->record && hist) hist[it] = sqrt(rr_new / c->rr0);
}

// ---- initial residual -----------------------------------------------------------------------------------------------
template <int KIND>
__global__ void __launch_bounds__(BX* BY)
    k_krylov_init(Op op, const double* __restrict__ x, const double* __restrict__ rhs, double* __restrict__ r,
                  double* __restrict__ r0hat, KrylovCtl* ctl, double* hist, int kc, RedBuf rb) {
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    double s2 = 0.0, s1 = 0.0;
    if (i < op.n[0] && j < op.n[1])
        for (int k = k0; k < k1; ++k) {
            const size_t p = gidx(op, i, j, k);
            const double o = rhs[p] - row_apply<double, KIND>(op, ArrLd<double>{x}, i, j, k, true);
            r[p] = o;
            if (r0hat) r0hat[p] = o;
            s2 = fma(o, o, s2);
            s1 += o;
        }
    double vals[2] = {s2, s1};
    grid_reduce<2>(vals, rb, [=](const double* t) { krylov_init_finish(ctl, hist, t); });
}

// ---- CG ---------------------------------------------------------------------------------------------------------------
struct PnewLd {  // p_new = (r - mu) + beta p_old, formed on the fly (also in the halo)
    const double* r;
    const double* p;
    double beta, mu;
    __device__ __forceinline__ double operator()(size_t q, int, int, int) const { return fma(beta, p[q], r[q] - mu); }
};

template <int KIND>
__global__ void __launch_bounds__(BX* BY)
    k_cg_passA(Op op, const double* __restrict__ r, const double* __restrict__ p_old, double* __restrict__ p_new,
               double* __restrict__ q, double* __restrict__ x, KrylovCtl* ctl, int kc, RedBuf rb) {
    if (ctl->done) return;
    const double beta = ctl->beta, mu = ctl->mu, alpha_prev = ctl->alpha;
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    const PnewLd ld{r, p_old, beta, mu};
    double acc = 0.0;
    if (i < op.n[0] && j < op.n[1])
        for (int k = k0; k < k1; ++k) {
            const size_t p = gidx(op, i, j, k);
            const double pn = ld(p, i, j, k);
            const double qv = row_apply<double, KIND>(op, ld, i, j, k, false);
            x[p] = fma(alpha_prev, p_old[p], x[p]);  // deferred x-update of the previous iteration
            p_new[p] = pn;
            q[p] = qv;
            acc = fma(pn, qv, acc);
        }
    double vals[1] = {acc};
    grid_reduce<1>(vals, rb, [=](const double* t) {
        ctl->pq = t[0];
        ctl->alpha = (ctl->pcg ? ctl->rz : ctl->rr) / t[0];
    });
}

__global__ void __launch_bounds__(256)
    k_cg_passB(size_t n, double* __restrict__ r, const double* __restrict__ q, KrylovCtl* ctl, double* hist, RedBuf rb) {
    if (ctl->done) return;
    const double alpha = ctl->alpha;
    double s2 = 0.0, s1 = 0.0;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (size_t)gridDim.x * blockDim.x) {
        const double rn = fma(-alpha, q[p], r[p]);
        r[p] = rn;
        s2 = fma(rn, rn, s2);
        s1 += rn;
    }
    double vals[2] = {s2, s1};
    grid_reduce<2>(vals, rb, [=](const double* t) {
        const double mu = ctl->project ? t[1] / ctl->npoints : 0.0;
        const double rr_new = ctl->project ? fma(-ctl->npoints * mu, mu, t[0]) : t[0];
        finish_iteration(ctl, hist, rr_new);
        const bool conv = !ctl->fixed && sqrt(rr_new) <= sqrt(ctl->tol2) * sqrt(ctl->rr0);
        if (conv) {
            ctl->done = 1;
            ctl->status = POISSON_OK;
        } else if (ctl->it >= ctl->max_it) {
            ctl->done = 1;
        } else if (!ctl->pcg) {
            ctl->beta = rr_new / ctl->rr;  // preconditioned CG takes beta from r.z after the preconditioner (k_pcg_dot)
        }
        ctl->rr = rr_new;
        ctl->mu = mu;
    });
}

// Preconditioned CG (Saad Alg. 9.1): rz = r . z after z = M^-1 r; beta = rz_new / rz_old (0 before the first iteration).
__global__ void __launch_bounds__(256)
    k_pcg_dot(size_t n, const double* __restrict__ r, const double* __restrict__ z, KrylovCtl* ctl, RedBuf rb) {
    if (ctl->done) return;
    double s = 0.0;
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (size_t)gridDim.x * blockDim.x)
        s = fma(r[p], z[p], s);
    double vals[1] = {s};
    grid_reduce<1>(vals, rb, [=](const double* t) {
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

__global__ void __launch_bounds__(256) k_cg_final(size_t n, double* __restrict__ x, const double* __restrict__ p,
                                                    const KrylovCtl* ctl) {
    const double alpha = ctl->alpha;
    if (ctl->it == 0) return;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x)
        x[q] = fma(alpha, p[q], x[q]);
}

__global__ void __launch_bounds__(256) k_sum(size_t n, const double* __restrict__ x, KrylovCtl* ctl, RedBuf rb) {
    double s = 0.0;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) s += x[q];
    double vals[1] = {s};
    grid_reduce<1>(vals, rb, [=](const double* t) { ctl->sum_x = t[0]; });
}
__global__ void __launch_bounds__(256) k_sub_mean(size_t n, double* __restrict__ x, const KrylovCtl* ctl) {
    const double mu = ctl->sum_x / ctl->npoints;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) x[q] -= mu;
}

// ---- BiCGSTAB ---------------------------------------------------------------------------------------------------------
// D = diag(A) with A = L: entry -d (right Jacobi scaling p^ = D^-1 p), or 1 when scaling is off.
template <int KIND>
__device__ __forceinline__ double jac(const Op& op, int i, int j, int k, int jacobi) {
    return jacobi ? -row_diag<double, KIND>(op, i, j, k) : 1.0;
}

template <int KIND>
struct PhatLd {  // p_new = r + beta (p_old - omega v_old) ; p^ = p_new / D
    const Op& op;
    const double* r;
    const double* p;
    const double* v;
    double beta, omega;
    int jacobi;
    __device__ __forceinline__ double pnew(size_t q) const { return fma(beta, fma(-omega, v[q], p[q]), r[q]); }
    __device__ __forceinline__ double operator()(size_t q, int i, int j, int k) const {
        return pnew(q) / jac<KIND>(op, i, j, k, jacobi);
    }
};

template <int KIND>
struct ShatLd {  // s = r - alpha v ; s^ = s / D
    const Op& op;
    const double* r;
    const double* v;
    double alpha;
    int jacobi;
    __device__ __forceinline__ double s(size_t q) const { return fma(-alpha, v[q], r[q]); }
    __device__ __forceinline__ double operator()(size_t q, int i, int j, int k) const {
        return s(q) / jac<KIND>(op, i, j, k, jacobi);
    }
};

template <int KIND>
__global__ void __launch_bounds__(BX* BY)
    k_bicg_pass1(Op op, const double* __restrict__ r, const double* __restrict__ p_old,
                 const double* __restrict__ v_old, const double* r0, double* __restrict__ p_new,
                 double* __restrict__ v_new, KrylovCtl* ctl, int jacobi, int kc, RedBuf rb) {
    if (ctl->done) return;
    const int restart = ctl->restart;
    double* const r0w = const_cast<double*>(r0);
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    const PhatLd<KIND> ld{op, r, p_old, v_old, ctl->beta, ctl->omega, jacobi};
    double acc = 0.0;
    if (i < op.n[0] && j < op.n[1])
        for (int k = k0; k < k1; ++k) {
            const size_t p = gidx(op, i, j, k);
            const double vn = row_apply<double, KIND>(op, ld, i, j, k, false);
            p_new[p] = ld.pnew(p);
            v_new[p] = vn;
            double r0p = r0[p];
            if (restart) {  // r^_0 := r
                r0p = r[p];
                r0w[p] = r0p;
            }
            acc = fma(r0p, vn, acc);
        }
    double vals[1] = {acc};
    grid_reduce<1>(vals, rb, [=](const double* t) {
        const double r0v = t[0];
        ctl->r0v = r0v;
        if (!(fabs(r0v) > 0.0) || !isfinite(r0v) || !(fabs(ctl->rho) > 0.0)) {
            ctl->status = POISSON_BREAKDOWN;
            ctl->done = 1;
        } else {
            ctl->alpha = ctl->rho / r0v;
        }
    });
}

template <int KIND>
__global__ void __launch_bounds__(BX* BY)
    k_bicg_pass2(Op op, const double* __restrict__ r, const double* __restrict__ v, double* __restrict__ s,
                 double* __restrict__ t, KrylovCtl* ctl, int jacobi, int kc, RedBuf rb) {
    if (ctl->done) return;
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    const ShatLd<KIND> ld{op, r, v, ctl->alpha, jacobi};
    double a_ts = 0.0, a_tt = 0.0;
    if (i < op.n[0] && j < op.n[1])
        for (int k = k0; k < k1; ++k) {
            const size_t p = gidx(op, i, j, k);
            const double tv = row_apply<double, KIND>(op, ld, i, j, k, false);
            const double sv = ld.s(p);
            s[p] = sv;
            t[p] = tv;
            a_ts = fma(tv, sv, a_ts);
            a_tt = fma(tv, tv, a_tt);
        }
    double vals[2] = {a_ts, a_tt};
    grid_reduce<2>(vals, rb, [=](const double* tot) {
        ctl->ts = tot[0];
        ctl->tt = tot[1];
        if (!(tot[1] > 0.0) || !isfinite(tot[1])) {
            ctl->status = POISSON_BREAKDOWN;
            ctl->done = 1;
        } else {
            ctl->omega = tot[0] / tot[1];
        }
    });
}

__device__ __forceinline__ void bicg_finish_iteration(KrylovCtl* ctl, double* hist, const double* tot) {
    const double rr = tot[0];
    finish_iteration(ctl, hist, rr);
    ctl->rr = rr;
    if (!isfinite(rr)) {
        ctl->status = POISSON_BREAKDOWN;
        ctl->done = 1;
    } else if (!ctl->fixed && sqrt(rr) <= sqrt(ctl->tol2) * sqrt(ctl->rr0)) {
        ctl->status = POISSON_OK;
        ctl->done = 1;
    } else if (!(fabs(ctl->omega) > 0.0)) {
        ctl->status = POISSON_BREAKDOWN;
        ctl->done = 1;
    } else if (ctl->it >= ctl->max_it) {
        ctl->done = 1;
    } else {
        const double rho_new = tot[1];
        if (fabs(rho_new) <= ctl->eps_bd * sqrt(ctl->r0n2 * rr)) {
            // near-breakdown (r has become orthogonal to r^_0 up to rounding): restart with r^_0 := r, p := r
            ctl->restart = 1;
            ctl->nrestarts += 1;
            ctl->beta = 0.0;
            ctl->rho = rr;
            ctl->r0n2 = rr;
        } else {
            ctl->restart = 0;
            ctl->beta = (rho_new / ctl->rho) * (ctl->alpha / ctl->omega);
            ctl->rho = rho_new;
        }
    }
}

template <int KIND>
__global__ void __launch_bounds__(BX* BY)
    k_bicg_pass3(Op op, double* __restrict__ x, const double* __restrict__ p, const double* __restrict__ s,
                 const double* __restrict__ t, const double* __restrict__ r0, double* __restrict__ r, KrylovCtl* ctl,
                 double* hist, int jacobi, int kc, RedBuf rb) {
    if (ctl->done) return;
    const double alpha = ctl->alpha, omega = ctl->omega;
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    double a_rr = 0.0, a_r0r = 0.0;
    if (i < op.n[0] && j < op.n[1])
#pragma unroll 4
        for (int k = k0; k < k1; ++k) {
            const size_t q = gidx(op, i, j, k);
            const double dg = jac<KIND>(op, i, j, k, jacobi);
            const double rdg = 1.0 / dg;  // one division; the two quotients by div_by are still correctly rounded
            const double sv = s[q];
            const double ph = div_by<double>(p[q], dg, rdg), sh = div_by<double>(sv, dg, rdg);
            x[q] = fma(omega, sh, fma(alpha, ph, x[q]));
            const double rn = fma(-omega, t[q], sv);
            r[q] = rn;
            a_rr = fma(rn, rn, a_rr);
            a_r0r = fma(r0[q], rn, a_r0r);
        }
    double vals[2] = {a_rr, a_r0r};
    grid_reduce<2>(vals, rb, [=](const double* tot) { bicg_finish_iteration(ctl, hist, tot); });
}

// Pair version for even n0: 16-byte accesses; the spherical diagonal does not depend on k, so it and its reciprocal are
// formed once per column (the quotients by div_by stay correctly rounded, i.e. equal to p / D and s / D).
template <int KIND>
__global__ void __launch_bounds__(BX* BY)
    k_bicg_pass3_pair(Op op, double* __restrict__ x, const double* __restrict__ p, const double* __restrict__ s,
                      const double* __restrict__ t, const double* __restrict__ r0, double* __restrict__ r,
                      KrylovCtl* ctl, double* hist, int jacobi, int kc, RedBuf rb) {
    if (ctl->done) return;
    const double alpha = ctl->alpha, omega = ctl->omega;
    const int i = 2 * (blockIdx.x * BX + threadIdx.x), j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    double a_rr = 0.0, a_r0r = 0.0;
    if (i < op.n[0] && j < op.n[1]) {
        double d0 = jac<KIND>(op, i, j, k0, jacobi), d1 = jac<KIND>(op, i + 1, j, k0, jacobi);
        double rd0 = 1.0 / d0, rd1 = 1.0 / d1;
        const size_t plane = (size_t)op.n[0] * op.n[1];
        size_t q = gidx(op, i, j, k0);
#pragma unroll 4
        for (int k = k0; k < k1; ++k, q += plane) {
            if (KIND != KIND_SPH) {
                d0 = jac<KIND>(op, i, j, k, jacobi);
                d1 = jac<KIND>(op, i + 1, j, k, jacobi);
                rd0 = 1.0 / d0;
                rd1 = 1.0 / d1;
            }
            const double2 pv = *reinterpret_cast<const double2*>(p + q), sv = *reinterpret_cast<const double2*>(s + q);
            const double2 tv = *reinterpret_cast<const double2*>(t + q), zv = *reinterpret_cast<const double2*>(r0 + q);
            double2 xv = *reinterpret_cast<const double2*>(x + q);
            xv.x = fma(omega, div_by<double>(sv.x, d0, rd0), fma(alpha, div_by<double>(pv.x, d0, rd0), xv.x));
            xv.y = fma(omega, div_by<double>(sv.y, d1, rd1), fma(alpha, div_by<double>(pv.y, d1, rd1), xv.y));
            *reinterpret_cast<double2*>(x + q) = xv;
            const double2 rn = make_double2(fma(-omega, tv.x, sv.x), fma(-omega, tv.y, sv.y));
            *reinterpret_cast<double2*>(r + q) = rn;
            a_rr = fma(rn.x, rn.x, a_rr);
            a_r0r = fma(zv.x, rn.x, a_r0r);
            a_rr = fma(rn.y, rn.y, a_rr);
            a_r0r = fma(zv.y, rn.y, a_r0r);
        }
    }
    double vals[2] = {a_rr, a_r0r};
    grid_reduce<2>(vals, rb, [=](const double* tot) { bicg_finish_iteration(ctl, hist, tot); });
}

// ---- BiCGSTAB right-preconditioned by the multi-colour Gauss-Seidel sweep of PAPER.md:107-123 Eq. 10 (row f3) ---------
// The preconditioner solve p^ = B^-1 p is a red-black sweep over the grid (k_sor_fused / k_rbsor_half), so the
// iteration is cut at it:  p = r + beta (p - omega v) | p^ = B^-1 p | v = L p^, r0^.v -> alpha | s = r - alpha v |
// s^ = B^-1 s | t = L s^, t.s, t.t -> omega | x += alpha p^ + omega s^, r = s - omega t, r.r, r0^.r -> beta.
__global__ void __launch_bounds__(256)
    k_gsb_p(size_t n, const double* __restrict__ r, double* __restrict__ p, const double* __restrict__ v,
            double* __restrict__ r0, KrylovCtl* ctl) {
    if (ctl->done) return;
    const double beta = ctl->beta, omega = ctl->omega;
    const int restart = ctl->restart;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) {
        const double rv = r[q];
        p[q] = fma(beta, fma(-omega, v[q], p[q]), rv);
        if (restart) r0[q] = rv;  // near-breakdown restart: r^_0 := r (reading C4)
    }
}

__global__ void __launch_bounds__(256)
    k_gsb_s(size_t n, const double* __restrict__ r, const double* __restrict__ v, double* __restrict__ s, const KrylovCtl* ctl) {
    if (ctl->done) return;
    const double alpha = ctl->alpha;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x)
        s[q] = fma(-alpha, v[q], r[q]);
}

// out = L in (homogeneous ghosts).  WHICH 1: sum other.out (other = r^_0) -> alpha; WHICH 2: sum out.other, out.out
// (other = s) -> omega.
template <int KIND, int WHICH>
__global__ void __launch_bounds__(BX* BY)
    k_gsb_matvec(Op op, const double* __restrict__ in, double* __restrict__ out, const double* __restrict__ other,
                 KrylovCtl* ctl, int kc, RedBuf rb) {
    if (ctl->done) return;
    const int i = blockIdx.x * BX + threadIdx.x, j = blockIdx.y * BY + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(op.n[2], k0 + kc);
    double a0 = 0.0, a1 = 0.0;
    if (i < op.n[0] && j < op.n[1])
        for (int k = k0; k < k1; ++k) {
            const size_t q = gidx(op, i, j, k);
            const double o = row_apply<double, KIND>(op, ArrLd<double>{in}, i, j, k, false);
            out[q] = o;
            a0 = fma(other[q], o, a0);
            if (WHICH == 2) a1 = fma(o, o, a1);
        }
    double vals[2] = {a0, a1};
    grid_reduce<2>(vals, rb, [=](const double* t) {
        if (WHICH == 1) {
            const double r0v = t[0];
            ctl->r0v = r0v;
            if (!(fabs(r0v) > 0.0) || !isfinite(r0v) || !(fabs(ctl->rho) > 0.0)) {
                ctl->status = POISSON_BREAKDOWN;
                ctl->done = 1;
            } else {
                ctl->alpha = ctl->rho / r0v;
            }
        } else {
            ctl->ts = t[0];
            ctl->tt = t[1];
            if (!(t[1] > 0.0) || !isfinite(t[1])) {
                ctl->status = POISSON_BREAKDOWN;
                ctl->done = 1;
            } else {
                ctl->omega = t[0] / t[1];
            }
        }
    });
}

__global__ void __launch_bounds__(256)
    k_gsb_update(size_t n, double* __restrict__ x, const double* __restrict__ ph, const double* __restrict__ sh,
                 const double* __restrict__ s, const double* __restrict__ t, const double* __restrict__ r0,
                 double* __restrict__ r, KrylovCtl* ctl, double* hist, RedBuf rb) {
    if (ctl->done) return;
    const double alpha = ctl->alpha, omega = ctl->omega;
    double a_rr = 0.0, a_r0r = 0.0;
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (size_t)gridDim.x * blockDim.x) {
        x[q] = fma(omega, sh[q], fma(alpha, ph[q], x[q]));
        const double rn = fma(-omega, t[q], s[q]);
        r[q] = rn;
        a_rr = fma(rn, rn, a_rr);
        a_r0r = fma(r0[q], rn, a_r0r);
    }
    double vals[2] = {a_rr, a_r0r};
    grid_reduce<2>(vals, rb, [=](const double* tot) { bicg_finish_iteration(ctl, hist, tot); });
}

// ---- launch wrappers --------------------------------------------------------------------------------------------------
#define KIND_SWITCH(kind, CALL)                       \
    switch (kind) {                                   \
        case KIND_CART2: { constexpr int K = KIND_CART2; CALL; } break; \
        case KIND_CART6: { constexpr int K = KIND_CART6; CALL; } break; \
        default:         { constexpr int K = KIND_SPH;   CALL; } break; \
    }

static int stream_blocks(poisson_ctx* ctx, size_t n) {
    size_t b = (n + 256 * 8 - 1) / (256 * 8);
    size_t cap = (size_t)ctx->num_sms * 16;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (int)b;
}

int launch_krylov_init(poisson_ctx* ctx, const double* x, const double* rhs, double* r, bool bicg, double* r0hat) {
    const Op& op = ctx->op;
    if (plane_ok(ctx, op)) return plane_krylov_init(ctx, x, rhs, r, bicg ? r0hat : nullptr);
    int kc = pick_kc(op, ctx->num_sms);
    dim3 g;
    const dim3 b(BX, BY);
    const int rcg = fit_grid(ctx, op, op.n[0], &kc, &g);
    if (rcg != POISSON_OK) return rcg;
    pre_launch(ctx, KID_KRYLOV_INIT);
    KIND_SWITCH(ctx->kind, (k_krylov_init<K><<<g, b, 0, ctx->stream>>>(op, x, rhs, r, bicg ? r0hat : nullptr, ctx->d_ctl,
                                                                         ctx->d_hist, kc, ctx->red)));
    post_launch(ctx, KID_KRYLOV_INIT);
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

int launch_cg_passA(poisson_ctx* ctx, const double* r, const double* p_old, double* p_new, double* q, double* x) {
    const Op& op = ctx->op;
    if (plane_ok(ctx, op)) return plane_cg_passA(ctx, r, p_old, p_new, q, x);
    int kc = pick_kc(op, ctx->num_sms);
    dim3 g;
    const dim3 b(BX, BY);
    const int rcg = fit_grid(ctx, op, op.n[0], &kc, &g);
    if (rcg != POISSON_OK) return rcg;
    pre_launch(ctx, KID_CG_PASS_A);
    KIND_SWITCH(ctx->kind,
                (k_cg_passA<K><<<g, b, 0, ctx->stream>>>(op, r, p_old, p_new, q, x, ctx->d_ctl, kc, ctx->red)));
    post_launch(ctx, KID_CG_PASS_A);
    return POISSON_OK;
}

int launch_cg_passB(poisson_ctx* ctx, double* r, const double* q) {
    PB_LAUNCH(ctx, KID_CG_PASS_B, (k_cg_passB<<<stream_blocks(ctx, ctx->npts), 256, 0, ctx->stream>>>(
                                      ctx->npts, r, q, ctx->d_ctl, ctx->d_hist, ctx->red)));
    return POISSON_OK;
}

int launch_pcg_dot(poisson_ctx* ctx, const double* r, const double* z) {
    PB_LAUNCH(ctx, KID_PCG_PRECOND,
              (k_pcg_dot<<<stream_blocks(ctx, ctx->npts), 256, 0, ctx->stream>>>(ctx->npts, r, z, ctx->d_ctl, ctx->red)));
    return POISSON_OK;
}

int launch_cg_final(poisson_ctx* ctx, double* x, const double* p_last) {
    PB_LAUNCH(ctx, KID_CG_FINAL,
              (k_cg_final<<<stream_blocks(ctx, ctx->npts), 256, 0, ctx->stream>>>(ctx->npts, x, p_last, ctx->d_ctl)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

int launch_sub_mean(poisson_ctx* ctx, double* x) {
    PB_LAUNCH(ctx, KID_CG_FINAL,
              (k_sum<<<stream_blocks(ctx, ctx->npts), 256, 0, ctx->stream>>>(ctx->npts, x, ctx->d_ctl, ctx->red)));
    PB_LAUNCH(ctx, KID_CG_FINAL,
              (k_sub_mean<<<stream_blocks(ctx, ctx->npts), 256, 0, ctx->stream>>>(ctx->npts, x, ctx->d_ctl)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

int launch_bicg_pass1(poisson_ctx* ctx, const double* r, const double* p_old, const double* v_old, const double* r0,
                      double* p_new, double* v_new) {
    const Op& op = ctx->op;
    if (plane_ok(ctx, op)) return plane_bicg_pass1(ctx, r, p_old, v_old, r0, p_new, v_new);
    int kc = pick_kc(op, ctx->num_sms);
    dim3 g;
    const dim3 b(BX, BY);
    const int rcg = fit_grid(ctx, op, op.n[0], &kc, &g);
    if (rcg != POISSON_OK) return rcg;
    pre_launch(ctx, KID_BICG_PASS1);
    KIND_SWITCH(ctx->kind, (k_bicg_pass1<K><<<g, b, 0, ctx->stream>>>(op, r, p_old, v_old, r0, p_new, v_new, ctx->d_ctl,
                                                                        ctx->opt_jacobi, kc, ctx->red)));
    post_launch(ctx, KID_BICG_PASS1);
    return POISSON_OK;
}

int launch_bicg_pass2(poisson_ctx* ctx, const double* r, const double* v, double* s, double* t) {
    const Op& op = ctx->op;
    if (plane_ok(ctx, op)) return plane_bicg_pass2(ctx, r, v, s, t);
    int kc = pick_kc(op, ctx->num_sms);
    dim3 g;
    const dim3 b(BX, BY);
    const int rcg = fit_grid(ctx, op, op.n[0], &kc, &g);
    if (rcg != POISSON_OK) return rcg;
    pre_launch(ctx, KID_BICG_PASS2);
    KIND_SWITCH(ctx->kind, (k_bicg_pass2<K><<<g, b, 0, ctx->stream>>>(op, r, v, s, t, ctx->d_ctl, ctx->opt_jacobi, kc,
                                                                        ctx->red)));
    post_launch(ctx, KID_BICG_PASS2);
    return POISSON_OK;
}

int launch_gsb_p(poisson_ctx* ctx, const double* r, double* p, const double* v, double* r0) {
    PB_LAUNCH(ctx, KID_BICG_PASS1, (k_gsb_p<<<stream_blocks(ctx, ctx->npts), 256, 0, ctx->stream>>>(ctx->npts, r, p, v, r0, ctx->d_ctl)));
    return POISSON_OK;
}
int launch_gsb_s(poisson_ctx* ctx, const double* r, const double* v, double* s) {
    PB_LAUNCH(ctx, KID_BICG_PASS2, (k_gsb_s<<<stream_blocks(ctx, ctx->npts), 256, 0, ctx->stream>>>(ctx->npts, r, v, s, ctx->d_ctl)));
    return POISSON_OK;
}
int launch_gsb_matvec(poisson_ctx* ctx, int which, const double* in, double* out, const double* other) {
    const Op& op = ctx->op;
    int kc = pick_kc(op, ctx->num_sms);
    dim3 g;
    const dim3 b(BX, BY);
    const int rcg = fit_grid(ctx, op, op.n[0], &kc, &g);
    if (rcg != POISSON_OK) return rcg;
    const int kid = which == 1 ? KID_BICG_PASS1 : KID_BICG_PASS2;
    pre_launch(ctx, kid);
    if (which == 1) {
        KIND_SWITCH(ctx->kind, (k_gsb_matvec<K, 1><<<g, b, 0, ctx->stream>>>(op, in, out, other, ctx->d_ctl, kc, ctx->red)));
    } else {
        KIND_SWITCH(ctx->kind, (k_gsb_matvec<K, 2><<<g, b, 0, ctx->stream>>>(op, in, out, other, ctx->d_ctl, kc, ctx->red)));
    }
    post_launch(ctx, kid);
    return POISSON_OK;
}
int launch_gsb_update(poisson_ctx* ctx, double* x, const double* ph, const double* sh, const double* s, const double* t,
                      const double* r0, double* r) {
    PB_LAUNCH(ctx, KID_BICG_PASS3, (k_gsb_update<<<stream_blocks(ctx, ctx->npts), 256, 0, ctx->stream>>>(
                                       ctx->npts, x, ph, sh, s, t, r0, r, ctx->d_ctl, ctx->d_hist, ctx->red)));
    return POISSON_OK;
}

int launch_bicg_pass3(poisson_ctx* ctx, double* x, const double* p, const double* s, const double* t,
                      const double* r0, double* r) {
    const Op& op = ctx->op;
    int kc = pick_kc(op, ctx->num_sms);
    const bool pair = op.n[0] % 2 == 0 && ctx->opt_path != 1;
    dim3 g;
    const dim3 b(BX, BY);
    const int rcg = fit_grid(ctx, op, pair ? op.n[0] / 2 : op.n[0], &kc, &g);
    if (rcg != POISSON_OK) return rcg;
    pre_launch(ctx, KID_BICG_PASS3);
    if (pair) {
        KIND_SWITCH(ctx->kind, (k_bicg_pass3_pair<K><<<g, b, 0, ctx->stream>>>(op, x, p, s, t, r0, r, ctx->d_ctl,
                                                                                 ctx->d_hist, ctx->opt_jacobi, kc, ctx->red)));
    } else {
        KIND_SWITCH(ctx->kind, (k_bicg_pass3<K><<<g, b, 0, ctx->stream>>>(op, x, p, s, t, r0, r, ctx->d_ctl, ctx->d_hist,
                                                                            ctx->opt_jacobi, kc, ctx->red)));
    }
    post_launch(ctx, KID_BICG_PASS3);
    return POISSON_OK;
}

}  // namespace pb
