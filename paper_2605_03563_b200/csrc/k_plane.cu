// k_plane.cu — instances of the plane-pipeline engine (plane.cuh) for large, pair-aligned grids:
//   stencil apply / residual / residual norm
//   initial Krylov residual
//   CG pass A       x += alpha p_old ; p = r + beta p_old ; q = L p ; sum p.q
//   BiCGSTAB pass 1 p = r + beta (p - omega v) ; v = L D^-1 p ; sum r0^.v
//   BiCGSTAB pass 2 s = r - alpha v ; t = L D^-1 s ; sum t.s, t.t
// Same arithmetic, same order as the generic kernels (k_stencil.cu, k_krylov.cu); only the data movement differs.
#include <cstdlib>

#include "plane.cuh"

namespace pb {

// ---- loaders ------------------------------------------------------------------------------------------------------------
struct LdArr {  // v itself
    static constexpr bool PLAIN = true, SIDE = false, USES_DIAG = false;
    const double* v;
    struct Raw {
        double2 a;
    };
    __device__ __forceinline__ void prepare() {}
    __device__ __forceinline__ Raw load(size_t p) const { return Raw{ld2(v + p)}; }
    __device__ __forceinline__ Raw load_own(size_t p) const { return load(p); }
    __device__ __forceinline__ void prefetch_own(size_t p) const { asm volatile("prefetch.global.L2 [%0];" ::"l"(v + p)); }
    __device__ __forceinline__ void side(const Raw&, size_t) const {}
    __device__ __forceinline__ double2 form(const Op&, const Raw& r, int, int, int) const { return r.a; }
    __device__ __forceinline__ double at(const Op&, size_t p, int, int, int) const { return v[p]; }
};

struct LdPnew {  // p_new = (r - mu) + beta p_old; side effect on owned points: x += alpha_prev p_old (deferred x-update)
    static constexpr bool PLAIN = false, SIDE = true, USES_DIAG = false;
    const double* r;
    const double* p;
    double* x;
    const KrylovCtl* ctl;
    double beta, mu, alpha_prev;
    struct Raw {
        double2 r, p, x;
    };
    __device__ __forceinline__ void prepare() {
        beta = ctl->beta;
        mu = ctl->mu;
        alpha_prev = ctl->alpha;
    }
    __device__ __forceinline__ Raw load(size_t q) const { return Raw{ld2(r + q), ld2(p + q), mk2(0.0, 0.0)}; }
    __device__ __forceinline__ Raw load_own(size_t q) const { return Raw{ld2(r + q), ld2(p + q), ld2(x + q)}; }
    __device__ __forceinline__ void prefetch_own(size_t q) const {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(r + q));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(p + q));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(x + q));
    }
    __device__ __forceinline__ void side(const Raw& w, size_t q) const {
        st2(x + q, mk2(fma(alpha_prev, w.p.x, w.x.x), fma(alpha_prev, w.p.y, w.x.y)));
    }
    __device__ __forceinline__ double2 form(const Op&, const Raw& w, int, int, int) const {
        return mk2(fma(beta, w.p.x, w.r.x - mu), fma(beta, w.p.y, w.r.y - mu));
    }
    __device__ __forceinline__ double at(const Op&, size_t q, int, int, int) const {
        return fma(beta, p[q], r[q] - mu);
    }
};

template <int KIND>
__device__ __forceinline__ double jac_(const Op& op, int i, int j, int k, int jacobi) {
    return jacobi ? -row_diag<double, KIND>(op, i, j, k) : 1.0;
}

template <int KIND>
struct LdPhat {  // p^ = (r + beta (p_old - omega v_old)) / D; side effect on owned points: store p_new
    static constexpr bool PLAIN = false, SIDE = true, USES_DIAG = true;
    const double* r;
    const double* p;
    const double* v;
    double* p_new;
    double* r0w;  // r^_0, rewritten with r on a restart
    const KrylovCtl* ctl;
    int jacobi;
    double beta, omega;
    int restart;
    struct Raw {
        double2 r, p, v;
    };
    __device__ __forceinline__ void prepare() {
        beta = ctl->beta;
        omega = ctl->omega;
        restart = ctl->restart;
    }
    __device__ __forceinline__ Raw load(size_t q) const { return Raw{ld2(r + q), ld2(p + q), ld2(v + q)}; }
    __device__ __forceinline__ Raw load_own(size_t q) const { return load(q); }
    __device__ __forceinline__ void prefetch_own(size_t q) const {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(r + q));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(p + q));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(v + q));
    }
    __device__ __forceinline__ void side(const Raw& w, size_t q) const {
        st2(p_new + q, mk2(fma(beta, fma(-omega, w.v.x, w.p.x), w.r.x), fma(beta, fma(-omega, w.v.y, w.p.y), w.r.y)));
        if (restart) st2(r0w + q, w.r);  // r^_0 := r; the epilogue of this same thread reads it back for r^_0 . v
    }
    __device__ __forceinline__ double2 form(const Op& op, const Raw& w, int i, int j, int k) const {
        return mk2(fma(beta, fma(-omega, w.v.x, w.p.x), w.r.x) / jac_<KIND>(op, i, j, k, jacobi),
                   fma(beta, fma(-omega, w.v.y, w.p.y), w.r.y) / jac_<KIND>(op, i + 1, j, k, jacobi));
    }
    __device__ __forceinline__ double2 form_own(const Raw& w, double d0, double d1) const {  // d = row diagonal
        return mk2(fma(beta, fma(-omega, w.v.x, w.p.x), w.r.x) / (jacobi ? -d0 : 1.0),
                   fma(beta, fma(-omega, w.v.y, w.p.y), w.r.y) / (jacobi ? -d1 : 1.0));
    }
    __device__ __forceinline__ double at(const Op& op, size_t q, int i, int j, int k) const {
        return fma(beta, fma(-omega, v[q], p[q]), r[q]) / jac_<KIND>(op, i, j, k, jacobi);
    }
};

template <int KIND>
struct LdShat {  // s^ = (r - alpha v) / D; side effect on owned points: store s
    static constexpr bool PLAIN = false, SIDE = true, USES_DIAG = true;
    const double* r;
    const double* v;
    double* s;
    const KrylovCtl* ctl;
    int jacobi;
    double alpha;
    struct Raw {
        double2 r, v;
    };
    __device__ __forceinline__ void prepare() { alpha = ctl->alpha; }
    __device__ __forceinline__ Raw load(size_t q) const { return Raw{ld2(r + q), ld2(v + q)}; }
    __device__ __forceinline__ Raw load_own(size_t q) const { return load(q); }
    __device__ __forceinline__ void prefetch_own(size_t q) const {
        asm volatile("prefetch.global.L2 [%0];" ::"l"(r + q));
        asm volatile("prefetch.global.L2 [%0];" ::"l"(v + q));
    }
    __device__ __forceinline__ void side(const Raw& w, size_t q) const {
        st2(s + q, mk2(fma(-alpha, w.v.x, w.r.x), fma(-alpha, w.v.y, w.r.y)));
    }
    __device__ __forceinline__ double2 form(const Op& op, const Raw& w, int i, int j, int k) const {
        return mk2(fma(-alpha, w.v.x, w.r.x) / jac_<KIND>(op, i, j, k, jacobi),
                   fma(-alpha, w.v.y, w.r.y) / jac_<KIND>(op, i + 1, j, k, jacobi));
    }
    __device__ __forceinline__ double2 form_own(const Raw& w, double d0, double d1) const {
        return mk2(fma(-alpha, w.v.x, w.r.x) / (jacobi ? -d0 : 1.0), fma(-alpha, w.v.y, w.r.y) / (jacobi ? -d1 : 1.0));
    }
    // the same quotients from a divisor that does not change along z and its reciprocal (div_by: correctly rounded)
    static constexpr bool RECIP = true;
    __device__ __forceinline__ double divisor(double d) const { return jacobi ? -d : 1.0; }
    __device__ __forceinline__ double2 form_own_rd(const Raw& w, double v0, double v1, double r0, double r1) const {
        return mk2(div_by<double>(fma(-alpha, w.v.x, w.r.x), v0, r0), div_by<double>(fma(-alpha, w.v.y, w.r.y), v1, r1));
    }
    __device__ __forceinline__ double at(const Op& op, size_t q, int i, int j, int k) const {
        return fma(-alpha, v[q], r[q]) / jac_<KIND>(op, i, j, k, jacobi);
    }
};

// ---- epilogues ----------------------------------------------------------------------------------------------------------
// out = L v (MODE 0) or rhs - L v (MODE 1); optional fp32 copy; optional sum(out^2), sum(out) -> scal[0..1]
template <int MODE, bool RED>
struct EpApply {
    static constexpr int NRED = RED ? 2 : 0;
    const double* rhs;
    double* out;
    float* out32;
    double* scal;
    struct Raw {
        double2 f;
    };
    __device__ __forceinline__ bool skip() const { return false; }
    __device__ __forceinline__ void prepare() {}
    __device__ __forceinline__ Raw load(size_t p) const {
        Raw w;
        if (MODE) w.f = ld2(rhs + p);
        return w;
    }
    __device__ __forceinline__ void apply(const Raw& w, size_t p, int, int, int, double2, double2 lv,
                                          double* acc) const {
        double2 o = lv;
        if (MODE) o = mk2(w.f.x - lv.x, w.f.y - lv.y);
        if (out) st2(out + p, o);
        if (out32) *reinterpret_cast<float2*>(out32 + p) = make_float2((float)o.x, (float)o.y);
        if (RED) {
            acc[0] = fma(o.x, o.x, acc[0]);
            acc[1] += o.x;
            acc[0] = fma(o.y, o.y, acc[0]);
            acc[1] += o.y;
        }
    }
    __device__ __forceinline__ void finish(const double* t) const {
        scal[0] = t[0];
        scal[1] = t[1];
    }
};

struct EpInit {  // r = rhs - L x (ghosts included); r0^ = r; first scalars of the Krylov recurrences
    static constexpr int NRED = 2;
    const double* rhs;
    double* r;
    double* r0hat;
    KrylovCtl* ctl;
    double* hist;
    struct Raw {
        double2 f;
    };
    __device__ __forceinline__ bool skip() const { return false; }
    __device__ __forceinline__ void prepare() {}
    __device__ __forceinline__ Raw load(size_t p) const { return Raw{ld2(rhs + p)}; }
    __device__ __forceinline__ void apply(const Raw& w, size_t p, int, int, int, double2, double2 lv,
                                          double* acc) const {
        const double2 o = mk2(w.f.x - lv.x, w.f.y - lv.y);
        st2(r + p, o);
        if (r0hat) st2(r0hat + p, o);
        acc[0] = fma(o.x, o.x, acc[0]);
        acc[1] += o.x;
        acc[0] = fma(o.y, o.y, acc[0]);
        acc[1] += o.y;
    }
    __device__ __forceinline__ void finish(const double* t) const { krylov_init_finish(ctl, hist, t); }
};

struct EpCgA {  // stores p_new and q = L p_new, sum p.q -> alpha (the x-update rides on the loader, LdPnew::side)
    static constexpr int NRED = 1;
    double* p_new;
    double* q;
    KrylovCtl* ctl;
    struct Raw {};
    __device__ __forceinline__ bool skip() const { return ctl->done != 0; }
    __device__ __forceinline__ void prepare() {}
    __device__ __forceinline__ Raw load(size_t) const { return Raw{}; }
    __device__ __forceinline__ void apply(const Raw&, size_t m, int, int, int, double2 pn, double2 lv, double* acc) const {
        st2(p_new + m, pn);
        st2(q + m, lv);
        acc[0] = fma(pn.x, lv.x, acc[0]);
        acc[0] = fma(pn.y, lv.y, acc[0]);
    }
    __device__ __forceinline__ void finish(const double* t) const {
        ctl->pq = t[0];
        ctl->alpha = (ctl->pcg ? ctl->rz : ctl->rr) / t[0];
    }
};

struct EpBicg1 {  // v_new = L p^, sum r0^.v -> alpha (p_new is stored by the loader, LdPhat::side)
    static constexpr int NRED = 1;
    const double* r0;
    double* v_new;
    KrylovCtl* ctl;
    struct Raw {
        double2 r0;
    };
    __device__ __forceinline__ bool skip() const { return ctl->done != 0; }
    __device__ __forceinline__ void prepare() {}
    __device__ __forceinline__ Raw load(size_t m) const { return Raw{ld2(r0 + m)}; }
    __device__ __forceinline__ void apply(const Raw& w, size_t m, int, int, int, double2, double2 lv,
                                          double* acc) const {
        st2(v_new + m, lv);
        acc[0] = fma(w.r0.x, lv.x, acc[0]);
        acc[0] = fma(w.r0.y, lv.y, acc[0]);
    }
    __device__ __forceinline__ void finish(const double* t) const {
        const double r0v = t[0];
        ctl->r0v = r0v;
        if (!(fabs(r0v) > 0.0) || !isfinite(r0v) || !(fabs(ctl->rho) > 0.0)) {
            ctl->status = POISSON_BREAKDOWN;
            ctl->done = 1;
        } else {
            ctl->alpha = ctl->rho / r0v;
        }
    }
};

struct EpBicg2 {  // t = L s^, sum t.s, t.t -> omega (s was stored by the loader of this same thread, LdShat::side)
    static constexpr int NRED = 2;
    const double* s;
    double* t;
    KrylovCtl* ctl;
    struct Raw {
        double2 s;
    };
    __device__ __forceinline__ bool skip() const { return ctl->done != 0; }
    __device__ __forceinline__ void prepare() {}
    __device__ __forceinline__ Raw load(size_t m) const { return Raw{ld2(s + m)}; }
    __device__ __forceinline__ void apply(const Raw& w, size_t m, int, int, int, double2, double2 lv,
                                          double* acc) const {
        st2(t + m, lv);
        acc[0] = fma(lv.x, w.s.x, acc[0]);
        acc[1] = fma(lv.x, lv.x, acc[1]);
        acc[0] = fma(lv.y, w.s.y, acc[0]);
        acc[1] = fma(lv.y, lv.y, acc[1]);
    }
    __device__ __forceinline__ void finish(const double* tot) const {
        ctl->ts = tot[0];
        ctl->tt = tot[1];
        if (!(tot[1] > 0.0) || !isfinite(tot[1])) {
            ctl->status = POISSON_BREAKDOWN;
            ctl->done = 1;
        } else {
            ctl->omega = tot[0] / tot[1];
        }
    }
};

#define KIND_SWITCH(kind, CALL)                                         \
    switch (kind) {                                                     \
        case KIND_CART2: { constexpr int K = KIND_CART2; CALL; } break; \
        case KIND_CART6: { constexpr int K = KIND_CART6; CALL; } break; \
        default:         { constexpr int K = KIND_SPH;   CALL; } break; \
    }

template <int KIND>
static int apply_k(poisson_ctx* ctx, const Op& op, const double* v, const double* rhs, double* out, float* out32,
                   int mode, bool ug, bool reduce) {
    const LdArr ld{v};
    int rc;
    if (mode == 0)
        rc = launch_plane<KIND>(ctx, op, ld, EpApply<0, false>{rhs, out, out32, ctx->d_scal}, ug, KID_APPLY);
    else if (!reduce)
        rc = launch_plane<KIND>(ctx, op, ld, EpApply<1, false>{rhs, out, out32, ctx->d_scal}, ug, KID_APPLY);
    else
        rc = launch_plane<KIND>(ctx, op, ld, EpApply<1, true>{rhs, out, out32, ctx->d_scal}, ug, KID_APPLY);
    if (rc != POISSON_OK) return rc;
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

bool plane_ok(const poisson_ctx* ctx, const Op& op) { return plane_eligible(ctx, op); }

int plane_apply(poisson_ctx* ctx, const Op& op, int kind, const double* v, const double* rhs, double* out,
                float* out32, int mode, bool ug, bool reduce) {
    int rc = POISSON_OK;
    KIND_SWITCH(kind, rc = apply_k<K>(ctx, op, v, rhs, out, out32, mode, ug, reduce));
    return rc;
}

int plane_krylov_init(poisson_ctx* ctx, const double* x, const double* rhs, double* r, double* r0hat) {
    int rc = POISSON_OK;
    KIND_SWITCH(ctx->kind, rc = launch_plane<K>(ctx, ctx->op, LdArr{x}, EpInit{rhs, r, r0hat, ctx->d_ctl, ctx->d_hist},
                                                true, KID_KRYLOV_INIT));
    if (rc != POISSON_OK) return rc;
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

int plane_cg_passA(poisson_ctx* ctx, const double* r, const double* p_old, double* p_new, double* q, double* x) {
    int rc = POISSON_OK;
    const LdPnew ld{r, p_old, x, ctx->d_ctl, 0.0, 0.0, 0.0};
    const EpCgA ep{p_new, q, ctx->d_ctl};
    KIND_SWITCH(ctx->kind, rc = launch_plane<K>(ctx, ctx->op, ld, ep, false, KID_CG_PASS_A));
    return rc;
}

int plane_bicg_pass1(poisson_ctx* ctx, const double* r, const double* p_old, const double* v_old, const double* r0,
                     double* p_new, double* v_new) {
    int rc = POISSON_OK;
    const EpBicg1 ep{r0, v_new, ctx->d_ctl};
    KIND_SWITCH(ctx->kind, rc = launch_plane<K>(ctx, ctx->op, LdPhat<K>{r, p_old, v_old, p_new, const_cast<double*>(r0), ctx->d_ctl, ctx->opt_jacobi, 0.0, 0.0, 0},
                                                ep, false, KID_BICG_PASS1));
    return rc;
}

int plane_bicg_pass2(poisson_ctx* ctx, const double* r, const double* v, double* s, double* t) {
    int rc = POISSON_OK;
    const EpBicg2 ep{s, t, ctx->d_ctl};
    KIND_SWITCH(ctx->kind, rc = launch_plane<K>(ctx, ctx->op, LdShat<K>{r, v, s, ctx->d_ctl, ctx->opt_jacobi, 0.0}, ep, false,
                                                KID_BICG_PASS2));
    return rc;
}

}  // namespace pb
