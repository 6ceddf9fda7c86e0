// api.cu — the C ABI of include/poisson.h: context set-up and the host-side solver drivers.
// Drivers only enqueue kernels and poll a device flag; all arithmetic of the path runs in the kernels.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>

#include "common.cuh"

using namespace pb;

static std::string g_create_error;

namespace pb {

int fail(poisson_ctx* ctx, int code, const std::string& msg) {
    if (ctx)
        ctx->err = msg;
    else
        g_create_error = msg;
    return code;
}

int fail_cuda(poisson_ctx* ctx, cudaError_t e, const char* what, const char* file, int line) {
    char buf[512];
    snprintf(buf, sizeof(buf), "CUDA error %s (%s) at %s:%d in %s", cudaGetErrorName(e), cudaGetErrorString(e), file,
             line, what);
    cudaGetLastError();
    return fail(ctx, e == cudaErrorMemoryAllocation ? POISSON_OUT_OF_MEMORY : POISSON_CUDA_ERROR, buf);
}

double* scratch(poisson_ctx* ctx, int slot) {
    if ((int)ctx->vec.size() <= slot) ctx->vec.resize(slot + 1, nullptr);
    if (!ctx->vec[slot]) {
        void* p = nullptr;
        if (cudaMalloc(&p, ctx->npts * sizeof(double)) != cudaSuccess) {
            cudaGetLastError();
            fail(ctx, POISSON_OUT_OF_MEMORY, "out of device memory for a scratch vector");
            return nullptr;
        }
        ctx->vec[slot] = (double*)p;
    }
    return ctx->vec[slot];
}

void* sor_scratch(poisson_ctx* ctx, size_t bytes) {
    if (ctx->sor_tmp_bytes < bytes) {
        cudaFree(ctx->sor_tmp);
        ctx->sor_tmp = nullptr;
        ctx->sor_tmp_bytes = 0;
        if (cudaMalloc(&ctx->sor_tmp, bytes) != cudaSuccess) {
            cudaGetLastError();
            fail(ctx, POISSON_OUT_OF_MEMORY, "out of device memory for the red-black ping-pong buffer");
            return nullptr;
        }
        ctx->sor_tmp_bytes = bytes;
    }
    return ctx->sor_tmp;
}

void pre_launch(poisson_ctx* ctx, int kid) {
    if (ctx->time_kid != kid && ctx->time_kid != -2) return;
    if (ctx->ev_used + 2 > ctx->ev_pool.size()) {
        cudaEvent_t a = nullptr, b = nullptr;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) {
            cudaGetLastError();
            return;
        }
        ctx->ev_pool.push_back(a);
        ctx->ev_pool.push_back(b);
        ctx->ev_kid.push_back(kid);
    } else {
        ctx->ev_kid[ctx->ev_used / 2] = kid;
    }
    cudaEventRecord(ctx->ev_pool[ctx->ev_used], ctx->stream);
}

void post_launch(poisson_ctx* ctx, int kid) {
    ctx->launches++;
    ctx->launches_by_kid[kid]++;
    if (ctx->time_kid != kid && ctx->time_kid != -2) return;
    if (ctx->ev_used + 2 > ctx->ev_pool.size()) return;
    cudaEventRecord(ctx->ev_pool[ctx->ev_used + 1], ctx->stream);
    ctx->ev_used += 2;
}

}  // namespace pb

static const char* const kKernelNames[pb::KID_COUNT] = {
    "apply", "rbsor", "krylov_init", "cg_pass_a", "cg_pass_b", "cg_final", "bicg_pass1", "bicg_pass2", "bicg_pass3",
    "mg_restrict", "mg_prolong", "mg_coarse", "mg_axpy", "mp_moments", "mp_ghosts",
    "mgv_smooth", "mgv_restrict", "mgv_prolong", "mgv_coarse", "mgv_setup", "pcg_precond"};

static void free_levels(poisson_ctx* ctx) {
    for (auto& L : ctx->levels) {
        cudaFree(L.phi);
        cudaFree(L.rhs);
        cudaFree(L.res);
        cudaFree(L.phi32);
        cudaFree(L.rhs32);
        cudaFree(L.res32);
        cudaFree(L.alt);
        cudaFree(L.alt32);
    }
    ctx->levels.clear();
    ctx->mg_coarsest_n = -1;
}

// Spherical coefficient arrays of DESIGN.md reading C5 (Eq. 2 by direct finite differences on
// (r,theta,phi) with geometric-mean radial centres).
static int setup_spherical(poisson_ctx* ctx) {
    const int nr = ctx->op.n[0], nt = ctx->op.n[1], np = ctx->op.n[2];
    const std::vector<double>&re = ctx->edges[0], &te = ctx->edges[1], &pe = ctx->edges[2];
    std::vector<double>&rc = ctx->ctr[0], &tc = ctx->ctr[1], &pc = ctx->ctr[2];
    rc.resize(nr);
    tc.resize(nt);
    pc.resize(np);
    for (int i = 0; i < nr; ++i) rc[i] = std::sqrt(re[i] * re[i + 1]);
    for (int j = 0; j < nt; ++j) tc[j] = 0.5 * (te[j] + te[j + 1]);
    for (int k = 0; k < np; ++k) pc[k] = 0.5 * (pe[k] + pe[k + 1]);
    ctx->r_ghost_out = re[nr] * std::sqrt(re[nr] / re[nr - 1]);
    const double r_ghost_in = re[0] * std::sqrt(re[0] / re[1]);
    std::vector<double> coef(4 * nr + 4 * nt);
    double *ar_m = coef.data(), *ar_p = ar_m + nr, *ir2 = ar_p + nr, *dr = ir2 + nr;
    double *at_m = dr + nr, *at_p = at_m + nt, *cp = at_p + nt, *dt = cp + nt;
    for (int i = 0; i < nr; ++i) {
        const double ri = rc[i], dri = re[i + 1] - re[i];
        const double rm = (i > 0) ? rc[i - 1] : r_ghost_in;
        const double rp = (i < nr - 1) ? rc[i + 1] : ctx->r_ghost_out;
        ir2[i] = 1.0 / (ri * ri);
        ar_m[i] = (re[i] * re[i]) / ((ri - rm) * (ri * ri) * dri);
        ar_p[i] = (re[i + 1] * re[i + 1]) / ((rp - ri) * (ri * ri) * dri);
        if (i == 0 && ctx->op.bc[0] == POISSON_BC_NEUMANN0) ar_m[i] = 0.0;
        if (i == nr - 1 && ctx->op.bc[1] == POISSON_BC_NEUMANN0) ar_p[i] = 0.0;
        dr[i] = ar_m[i] + ar_p[i];
    }
    const double dph = pe[1] - pe[0];
    for (int j = 0; j < nt; ++j) {
        const double dth = te[j + 1] - te[j], st = std::sin(tc[j]);
        at_m[j] = std::sin(te[j]) / (st * dth * dth);
        at_p[j] = std::sin(te[j + 1]) / (st * dth * dth);
        if (j == 0 && ctx->op.bc[2] == POISSON_BC_AXIS) at_m[j] = 0.0;
        if (j == nt - 1 && ctx->op.bc[3] == POISSON_BC_AXIS) at_p[j] = 0.0;
        cp[j] = 1.0 / (st * st * dph * dph);
        dt[j] = (at_m[j] + at_p[j]) + 2.0 * cp[j];
    }
    PB_CUDA_OK(cudaMalloc((void**)&ctx->d_coef, coef.size() * sizeof(double)));
    PB_CUDA_OK(cudaMemcpyAsync(ctx->d_coef, coef.data(), coef.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    Op& op = ctx->op;
    op.ar_m = ctx->d_coef;
    op.ar_p = op.ar_m + nr;
    op.ir2 = op.ar_p + nr;
    op.dr = op.ir2 + nr;
    op.at_m = op.dr + nr;
    op.at_p = op.at_m + nt;
    op.cp = op.at_p + nt;
    op.dt = op.cp + nt;
    // tables for the multipole kernels: rc, sin th, cos th, cos ph, sin ph, and the exact cell-volume factors
    std::vector<double> tab(2 * nr + 3 * nt + 3 * np);
    double* b = tab.data();
    for (int i = 0; i < nr; ++i) b[i] = rc[i];
    for (int j = 0; j < nt; ++j) {
        b[nr + j] = std::sin(tc[j]);
        b[nr + nt + j] = std::cos(tc[j]);
    }
    for (int k = 0; k < np; ++k) {
        b[nr + 2 * nt + k] = std::cos(pc[k]);
        b[nr + 2 * nt + np + k] = std::sin(pc[k]);
    }
    double* vr = b + nr + 2 * nt + 2 * np;
    double* vt = vr + nr;
    double* vp = vt + nt;
    for (int i = 0; i < nr; ++i) vr[i] = (re[i + 1] * re[i + 1] * re[i + 1] - re[i] * re[i] * re[i]) / 3.0;
    for (int j = 0; j < nt; ++j) vt[j] = std::cos(te[j]) - std::cos(te[j + 1]);
    for (int k = 0; k < np; ++k) vp[k] = pe[k + 1] - pe[k];
    PB_CUDA_OK(cudaMalloc((void**)&ctx->d_ctr, tab.size() * sizeof(double)));
    PB_CUDA_OK(cudaMemcpyAsync(ctx->d_ctr, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));  // coef and tab are local vectors; the uploads are ordered on the handle's stream
    return POISSON_OK;
}

extern "C" {

const char* poisson_last_error(poisson_t h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int poisson_destroy(poisson_t ctx) {
    const DeviceGuard on_device(ctx);
    if (!ctx) return POISSON_INVALID_ARG;
    cudaStreamSynchronize(ctx->stream);
    free_levels(ctx);
    mgv_destroy(ctx);
    for (double* v : ctx->vec) cudaFree(v);
    for (int f = 0; f < 6; ++f) cudaFree(ctx->d_ghost[f]);
    cudaFree(ctx->sor_tmp);
    cudaFree(ctx->d_coef);
    cudaFree(ctx->d_ctr);
    cudaFree(ctx->d_rj);
    cudaFree(ctx->red.partials);
    cudaFree(ctx->red.counter);
    cudaFree(ctx->d_ctl);
    cudaFreeHost(ctx->h_ctl);
    cudaFree(ctx->d_hist);
    cudaFree(ctx->d_scal);
    cudaFreeHost(ctx->h_scal);
    for (double* s : ctx->d_stage) cudaFree(s);
    for (cudaEvent_t e : ctx->ev_pool) cudaEventDestroy(e);
    delete ctx;
    return POISSON_OK;
}

int poisson_create(poisson_t* out, const int shape[3], const double spacing[3], const double origin[3],
                   const double* const edges[3], int coord_system, int stencil_order, const int bc[6],
                   void* cuda_stream) {
    if (!out || !shape || !bc) return fail(nullptr, POISSON_INVALID_ARG, "null argument");
    *out = nullptr;
    if (coord_system != POISSON_CARTESIAN && coord_system != POISSON_SPHERICAL)
        return fail(nullptr, POISSON_INVALID_ARG, "coord_system must be POISSON_CARTESIAN or POISSON_SPHERICAL");
    if (stencil_order != 2 && stencil_order != 6)
        return fail(nullptr, POISSON_INVALID_ARG, "stencil_order must be 2 or 6");
    if (coord_system == POISSON_SPHERICAL && stencil_order != 2)
        return fail(nullptr, POISSON_UNSUPPORTED, "the spherical operator is 2nd order (7-point)");
    const int R = stencil_order == 6 ? 3 : 1;
    for (int a = 0; a < 3; ++a) {
        if (shape[a] < 1 || shape[a] > (1 << 14)) return fail(nullptr, POISSON_INVALID_ARG, "shape out of range");
        if ((bc[2 * a] == POISSON_BC_PERIODIC) != (bc[2 * a + 1] == POISSON_BC_PERIODIC))
            return fail(nullptr, POISSON_INVALID_ARG, "periodic faces come in pairs");
        if (bc[2 * a] == POISSON_BC_PERIODIC && shape[a] < R)
            return fail(nullptr, POISSON_INVALID_ARG, "periodic axis shorter than the stencil radius");
        for (int s = 0; s < 2; ++s)
            if (bc[2 * a + s] < 0 || bc[2 * a + s] > 3) return fail(nullptr, POISSON_INVALID_ARG, "bad boundary type");
    }
    if (coord_system == POISSON_CARTESIAN) {
        if (!spacing || !origin) return fail(nullptr, POISSON_INVALID_ARG, "spacing/origin required");
        for (int a = 0; a < 3; ++a)
            if (!(spacing[a] > 0)) return fail(nullptr, POISSON_INVALID_ARG, "spacing must be positive");
        for (int f = 0; f < 6; ++f)
            if (bc[f] == POISSON_BC_AXIS) return fail(nullptr, POISSON_INVALID_ARG, "BC_AXIS is spherical-only");
        if (stencil_order == 6)
            for (int f = 0; f < 6; ++f)
                if (bc[f] == POISSON_BC_NEUMANN0)
                    return fail(nullptr, POISSON_UNSUPPORTED, "Neumann faces need the 2nd-order stencil");
    } else {
        if (!edges || !edges[0] || !edges[1] || !edges[2])
            return fail(nullptr, POISSON_INVALID_ARG, "spherical grids need edges[3]");
        for (int a = 0; a < 3; ++a)
            for (int i = 0; i < shape[a]; ++i)
                if (!(edges[a][i + 1] > edges[a][i]))
                    return fail(nullptr, POISSON_INVALID_ARG, "cell edges must increase strictly");
        if (!(edges[0][0] > 0.0)) return fail(nullptr, POISSON_INVALID_ARG, "spherical grids need r_in > 0");
        if (edges[1][0] < -1e-12 || edges[1][shape[1]] > M_PI + 1e-12)
            return fail(nullptr, POISSON_INVALID_ARG, "theta edges must lie in [0, pi]");
        // the theta and phi differences are taken with one cell width (reading C5): uniform angles only
        for (int a = 1; a < 3; ++a) {
            const double w0 = (edges[a][shape[a]] - edges[a][0]) / shape[a];
            for (int i = 0; i < shape[a]; ++i)
                if (std::fabs((edges[a][i + 1] - edges[a][i]) - w0) > 1e-10 * w0)
                    return fail(nullptr, POISSON_UNSUPPORTED, "nonuniform theta / phi edges are not supported (only r may be nonuniform)");
        }
        if (bc[2] == POISSON_BC_AXIS && std::fabs(edges[1][0]) > 1e-12)
            return fail(nullptr, POISSON_INVALID_ARG, "BC_AXIS on the low theta face needs theta_edge[0] = 0");
        if (bc[3] == POISSON_BC_AXIS && std::fabs(edges[1][shape[1]] - M_PI) > 1e-12)
            return fail(nullptr, POISSON_INVALID_ARG, "BC_AXIS on the high theta face needs theta_edge[n] = pi");
        if (bc[0] == POISSON_BC_AXIS || bc[1] == POISSON_BC_AXIS || bc[4] == POISSON_BC_AXIS || bc[5] == POISSON_BC_AXIS)
            return fail(nullptr, POISSON_INVALID_ARG, "BC_AXIS applies to the theta faces only");
    }
    poisson_ctx* ctx = new poisson_ctx;
    ctx->stream = (cudaStream_t)cuda_stream;
    Op& op = ctx->op;
    std::memset(&op, 0, sizeof(op));
    ctx->npts = 1;
    for (int a = 0; a < 3; ++a) {
        op.n[a] = shape[a];
        ctx->npts *= (size_t)shape[a];
        ctx->h[a] = spacing ? spacing[a] : 1.0;
        ctx->origin[a] = origin ? origin[a] : 0.0;
        op.c[a] = 1.0 / (ctx->h[a] * ctx->h[a]);
    }
    op.coord = coord_system;
    op.order = stencil_order;
    op.R = R;
    for (int f = 0; f < 6; ++f) op.bc[f] = bc[f];
    ctx->kind = coord_system == POISSON_SPHERICAL ? KIND_SPH : (stencil_order == 6 ? KIND_CART6 : KIND_CART2);
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    ctx->device = dev;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) {
        int rc = fail_cuda(nullptr, e, "cudaGetDevice", __FILE__, __LINE__);
        delete ctx;
        return rc;
    }
#define CREATE_OK(call)                                                            \
    do {                                                                           \
        cudaError_t e2 = (call);                                                   \
        if (e2 != cudaSuccess) {                                                   \
            int rc2 = fail_cuda(nullptr, e2, #call, __FILE__, __LINE__);           \
            poisson_destroy(ctx);                                                  \
            return rc2;                                                            \
        }                                                                          \
    } while (0)
    for (int f = 0; f < 6; ++f) {
        const int a = f / 2, a1 = (a == 0) ? 1 : 0, a2 = (a == 2) ? 1 : 2;
        ctx->face_len[f] = (long)R * shape[a1] * shape[a2];
        if (bc[f] == POISSON_BC_DIRICHLET_GHOST) {
            CREATE_OK(cudaMalloc((void**)&ctx->d_ghost[f], ctx->face_len[f] * sizeof(double)));
            CREATE_OK(cudaMemset(ctx->d_ghost[f], 0, ctx->face_len[f] * sizeof(double)));
            op.ghost[f] = ctx->d_ghost[f];
        }
    }
    CREATE_OK(cudaMalloc((void**)&ctx->red.partials, (size_t)kMaxRedBlocks * kRedSlots * sizeof(double)));
    CREATE_OK(cudaMalloc((void**)&ctx->red.counter, sizeof(unsigned int)));
    CREATE_OK(cudaMemset(ctx->red.counter, 0, sizeof(unsigned int)));
    CREATE_OK(cudaMalloc((void**)&ctx->d_ctl, sizeof(KrylovCtl)));
    CREATE_OK(cudaMemset(ctx->d_ctl, 0, sizeof(KrylovCtl)));
    CREATE_OK(cudaMallocHost((void**)&ctx->h_ctl, sizeof(KrylovCtl)));
    CREATE_OK(cudaMalloc((void**)&ctx->d_scal, 512 * sizeof(double)));
    CREATE_OK(cudaMemset(ctx->d_scal, 0, 512 * sizeof(double)));
    CREATE_OK(cudaMallocHost((void**)&ctx->h_scal, 512 * sizeof(double)));
    if (coord_system == POISSON_SPHERICAL) {
        for (int a = 0; a < 3; ++a) ctx->edges[a].assign(edges[a], edges[a] + shape[a] + 1);
        int rc = setup_spherical(ctx);
        if (rc != POISSON_OK) {
            g_create_error = ctx->err;
            poisson_destroy(ctx);
            return rc;
        }
    }
    CREATE_OK(cudaDeviceSynchronize());  // the set-up copies and fills are complete whatever stream the caller uses next
    *out = ctx;
    return POISSON_OK;
}

int poisson_set_option(poisson_t ctx, int option, int value) {
    if (!ctx) return POISSON_INVALID_ARG;
    switch (option) {
        case POISSON_OPT_KERNEL_PATH:
            if (value < 0 || value > 2) return fail(ctx, POISSON_INVALID_ARG, "kernel path must be 0, 1 or 2");
            ctx->opt_path = value;
            return POISSON_OK;
        case POISSON_OPT_RESTRICTION:
            if (value < 0 || value > 1) return fail(ctx, POISSON_INVALID_ARG, "restriction must be 0 or 1");
            ctx->opt_restriction = value;
            return POISSON_OK;
        case POISSON_OPT_POLL_INTERVAL:
            if (value < 1) return fail(ctx, POISSON_INVALID_ARG, "poll interval must be >= 1");
            ctx->opt_poll = value;
            return POISSON_OK;
        case POISSON_OPT_JACOBI:
            if (value < 0 || value > 2) return fail(ctx, POISSON_INVALID_ARG, "BiCGSTAB preconditioner must be 0, 1 or 2");
            ctx->opt_jacobi = value;
            return POISSON_OK;
        case POISSON_OPT_RECORD_HISTORY:
            ctx->opt_history = value ? 1 : 0;
            return POISSON_OK;
        case POISSON_OPT_SOR_HALFSTEPS:
            if (value != 0 && value != 2 && value != 4)
                return fail(ctx, POISSON_INVALID_ARG, "half-steps per pass must be 0 (auto), 2 or 4");
            ctx->opt_sor_nhs = value;
            return POISSON_OK;
        case POISSON_OPT_FUSED_RESTRICT:
            if (value < 0 || value > 2) return fail(ctx, POISSON_INVALID_ARG, "fused restriction must be 0, 1 or 2");
            ctx->opt_fused_restrict = value;
            return POISSON_OK;
        case POISSON_OPT_TILE_CFG:
            ctx->opt_tile_cfg = value < 0 ? -1 : value;
            return POISSON_OK;
        case POISSON_OPT_PLANE_SPLIT:
            ctx->opt_plane_split = value < 0 ? -1 : (value ? 1 : 0);
            return POISSON_OK;
        case POISSON_OPT_APPLY_BULK:
            ctx->opt_apply_bulk = value < 0 ? -1 : (value ? 1 : 0);
            return POISSON_OK;
        case POISSON_OPT_COMPACT_ORDER:
            if (value != 2 && value != 4 && value != 6) return fail(ctx, POISSON_INVALID_ARG, "compact order must be 2, 4 or 6");
            if (value != 2 && (ctx->kind != KIND_CART2 || ctx->h[0] != ctx->h[1] || ctx->h[0] != ctx->h[2]))
                return fail(ctx, POISSON_UNSUPPORTED, "compact orders 4 / 6: Cartesian grid with isotropic spacing, created with stencil order 2 (PAPER.md:172)");
            ctx->opt_compact_order = value;
            return POISSON_OK;
        case POISSON_OPT_TIME_KERNELS:
            if (value < -2 || value >= KID_COUNT) return fail(ctx, POISSON_INVALID_ARG, "bad kernel class");
            ctx->time_kid = value;
            return POISSON_OK;
    }
    return fail(ctx, POISSON_INVALID_ARG, "unknown option");
}

int poisson_set_option_f64(poisson_t ctx, int option, double value) {
    if (!ctx) return POISSON_INVALID_ARG;
    switch (option) {
        case POISSON_OPT_BICG_RESTART_EPS:
            if (!(value >= 0.0)) return fail(ctx, POISSON_INVALID_ARG, "restart threshold must be >= 0");
            ctx->opt_bicg_restart_eps = value;
            return POISSON_OK;
    }
    return fail(ctx, POISSON_INVALID_ARG, "unknown floating-point option");
}

int poisson_bicgstab_stats(poisson_t ctx, int* restarts, int* confirm_failed) {
    if (!ctx) return POISSON_INVALID_ARG;
    if (restarts) *restarts = ctx->last_restarts;
    if (confirm_failed) *confirm_failed = ctx->last_confirm_failed;
    return POISSON_OK;
}

long poisson_face_len(poisson_t ctx, int face) { return (ctx && face >= 0 && face < 6) ? ctx->face_len[face] : -1; }
long poisson_kernel_launches(poisson_t ctx) { return ctx ? ctx->launches : -1; }

int poisson_kernel_classes(void) { return KID_COUNT; }
const char* poisson_kernel_name(int kernel_class) {
    return (kernel_class >= 0 && kernel_class < KID_COUNT) ? kKernelNames[kernel_class] : "";
}
long poisson_kernel_class_launches(poisson_t ctx, int kernel_class) {
    return (ctx && kernel_class >= 0 && kernel_class < KID_COUNT) ? ctx->launches_by_kid[kernel_class] : -1;
}
int poisson_kernel_time(poisson_t ctx, int kernel_class, double* h_ms_total, long* h_count) {
    const DeviceGuard on_device(ctx);
    if (!ctx || kernel_class < 0 || kernel_class >= KID_COUNT) return POISSON_INVALID_ARG;
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
    double tot = 0;
    long cnt = 0;
    for (size_t i = 0; i + 1 < ctx->ev_used; i += 2) {
        if (ctx->ev_kid[i / 2] != kernel_class) continue;
        float ms = 0;
        PB_CUDA_OK(cudaEventElapsedTime(&ms, ctx->ev_pool[i], ctx->ev_pool[i + 1]));
        tot += ms;
        ++cnt;
    }
    if (h_ms_total) *h_ms_total = tot;
    if (h_count) *h_count = cnt;
    return POISSON_OK;
}
int poisson_reset_kernel_times(poisson_t ctx) {
    const DeviceGuard on_device(ctx);
    if (!ctx) return POISSON_INVALID_ARG;
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
    ctx->ev_used = 0;
    return POISSON_OK;
}

int poisson_set_ghost_faces(poisson_t ctx, const double* const d_faces[6]) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_faces) return POISSON_INVALID_ARG;
    for (int f = 0; f < 6; ++f) {
        if (!d_faces[f]) continue;
        if (!ctx->d_ghost[f]) return fail(ctx, POISSON_INVALID_ARG, "ghost values given for a non-Dirichlet face");
        PB_CUDA_OK(cudaMemcpyAsync(ctx->d_ghost[f], d_faces[f], ctx->face_len[f] * sizeof(double),
                                   cudaMemcpyDeviceToDevice, ctx->stream));
    }
    ctx->ghost_nonzero = true;
    return POISSON_OK;
}

int poisson_get_ghost_face(poisson_t ctx, int face, double* d_out) {
    const DeviceGuard on_device(ctx);
    if (!ctx || face < 0 || face > 5 || !d_out) return POISSON_INVALID_ARG;
    if (!ctx->d_ghost[face]) return fail(ctx, POISSON_INVALID_ARG, "not a Dirichlet face");
    PB_CUDA_OK(cudaMemcpyAsync(d_out, ctx->d_ghost[face], ctx->face_len[face] * sizeof(double),
                               cudaMemcpyDeviceToDevice, ctx->stream));
    return POISSON_OK;
}

int poisson_apply_laplacian(poisson_t ctx, const double* d_phi, double* d_out) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_out || d_phi == d_out) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    return launch_apply(ctx, ctx->op, ctx->kind, d_phi, nullptr, d_out, 0, true, false);
}

// The last block of the fused residual reduction writes the scalar straight into pinned host memory (device-visible
// under unified addressing); the host spins on the word instead of paying for a copy and a stream synchronisation.
// A NaN sentinel marks "not written yet"; if the stream drains and the word is still NaN the norm itself is NaN.
static int residual_norm_sync(poisson_ctx* ctx, const double* d_phi, const double* d_rhs, double* h_norm) {
    volatile double* mail = ctx->h_scal + 500;
    mail[0] = std::nan("");
    double* const keep = ctx->d_scal;
    ctx->d_scal = ctx->h_scal + 500;  // the reduction epilogue writes scal[0] = sum r^2, scal[1] = sum r
    const int rc = launch_apply(ctx, ctx->op, ctx->kind, d_phi, d_rhs, nullptr, 1, true, true);
    ctx->d_scal = keep;
    if (rc != POISSON_OK) return rc;
    for (long spin = 0;; ++spin) {
        if (mail[0] == mail[0]) break;
        if ((spin & 1023) == 1023) {
            const cudaError_t q = cudaStreamQuery(ctx->stream);
            if (q == cudaSuccess) break;  // drained: whatever is there is the answer (a genuine NaN included)
            if (q != cudaErrorNotReady) return fail_cuda(ctx, q, "cudaStreamQuery", __FILE__, __LINE__);
        }
    }
    *h_norm = std::sqrt(mail[0]);
    return POISSON_OK;
}

int poisson_residual_norm(poisson_t ctx, const double* d_phi, const double* d_rhs, double* h_norm) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs || !h_norm) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    return residual_norm_sync(ctx, d_phi, d_rhs, h_norm);
}

int poisson_rbsor_sweep(poisson_t ctx, double* d_phi, const double* d_rhs, double omega, int nsweeps,
                        double* h_resnorm) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs || nsweeps < 0) return fail(ctx, POISSON_INVALID_ARG, "bad arguments");
    if (!(omega > 0.0 && omega < 2.0)) return fail(ctx, POISSON_INVALID_ARG, "omega must lie in (0,2) (PAPER.md:63)");
    int rc = launch_rbsor(ctx, ctx->op, ctx->kind, d_phi, d_rhs, omega, nsweeps, true);
    if (rc != POISSON_OK) return rc;
    if (h_resnorm) return residual_norm_sync(ctx, d_phi, d_rhs, h_resnorm);
    return POISSON_OK;
}

// ---- Krylov drivers ---------------------------------------------------------------------------------------------------
static int krylov_setup(poisson_ctx* ctx, double rtol, int max_iter, int fixed_iters, bool project, bool pcg = false) {
    const int nit = fixed_iters > 0 ? fixed_iters : max_iter;
    KrylovCtl* c = ctx->h_ctl;
    std::memset(c, 0, sizeof(*c));
    c->tol2 = rtol * rtol;
    c->fixed = fixed_iters > 0 ? 1 : 0;
    c->max_it = nit;
    c->project = project ? 1 : 0;
    c->record = ctx->opt_history;
    c->npoints = (double)ctx->npts;
    c->eps_bd = ctx->opt_bicg_restart_eps;
    c->pcg = pcg ? 1 : 0;
    if (ctx->opt_history) {
        if (ctx->hist_cap < nit + 1) {
            cudaFree(ctx->d_hist);
            ctx->d_hist = nullptr;
            PB_CUDA_OK(cudaMalloc((void**)&ctx->d_hist, (size_t)(nit + 1) * sizeof(double)));
            ctx->hist_cap = nit + 1;
        }
        PB_CUDA_OK(cudaMemsetAsync(ctx->d_hist, 0, (size_t)(nit + 1) * sizeof(double), ctx->stream));
    }
    PB_CUDA_OK(cudaMemcpyAsync(ctx->d_ctl, c, sizeof(*c), cudaMemcpyHostToDevice, ctx->stream));
    return POISSON_OK;
}

static int read_ctl(poisson_ctx* ctx) {
    PB_CUDA_OK(cudaMemcpyAsync(ctx->h_ctl, ctx->d_ctl, sizeof(KrylovCtl), cudaMemcpyDeviceToHost, ctx->stream));
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
    return POISSON_OK;
}

static bool all_periodic(const poisson_ctx* ctx) {
    for (int f = 0; f < 6; ++f)
        if (ctx->op.bc[f] != POISSON_BC_PERIODIC) return false;
    return ctx->op.coord == POISSON_CARTESIAN;
}

int poisson_cg_solve(poisson_t ctx, double* d_phi, const double* d_rhs, double rtol, int max_iter, int fixed_iters,
                     int* iters, double* relres) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    if (fixed_iters <= 0 && (max_iter < 1 || !(rtol > 0))) return fail(ctx, POISSON_INVALID_ARG, "bad rtol/max_iter");
    if (ctx->kind == KIND_SPH)
        return fail(ctx, POISSON_UNSUPPORTED, "CG needs a symmetric operator; use BiCGSTAB on spherical grids");
    const bool project = all_periodic(ctx);
    double *r = scratch(ctx, 0), *P[2] = {scratch(ctx, 1), scratch(ctx, 2)}, *q = scratch(ctx, 3);
    if (!r || !P[0] || !P[1] || !q) return POISSON_OUT_OF_MEMORY;
    int rc = krylov_setup(ctx, rtol, max_iter, fixed_iters, project);
    if (rc != POISSON_OK) return rc;
    PB_CUDA_OK(cudaMemsetAsync(P[0], 0, ctx->npts * sizeof(double), ctx->stream));
    PB_CUDA_OK(cudaMemsetAsync(P[1], 0, ctx->npts * sizeof(double), ctx->stream));
    rc = launch_krylov_init(ctx, d_phi, d_rhs, r, false, nullptr);
    if (rc != POISSON_OK) return rc;
    const int nit = fixed_iters > 0 ? fixed_iters : max_iter;
    for (int j = 0; j < nit;) {
        const int chunk = std::min(ctx->opt_poll, nit - j);
        for (int c = 0; c < chunk; ++c, ++j) {
            if ((rc = launch_cg_passA(ctx, r, P[j & 1], P[(j + 1) & 1], q, d_phi)) != POISSON_OK) return rc;
            if ((rc = launch_cg_passB(ctx, r, q)) != POISSON_OK) return rc;
        }
        PB_CUDA_OK(cudaGetLastError());
        if (fixed_iters <= 0) {
            rc = read_ctl(ctx);
            if (rc != POISSON_OK) return rc;
            if (ctx->h_ctl->done) break;
        }
    }
    rc = read_ctl(ctx);
    if (rc != POISSON_OK) return rc;
    const KrylovCtl c = *ctx->h_ctl;
    rc = launch_cg_final(ctx, d_phi, P[c.it & 1]);  // the x-update of the last iteration is still pending
    if (rc != POISSON_OK) return rc;
    if (project) {
        rc = launch_sub_mean(ctx, d_phi);
        if (rc != POISSON_OK) return rc;
    }
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
    ctx->hist_len = c.it + 1;
    if (iters) *iters = c.it;
    if (relres) *relres = c.rr0 > 0 ? std::sqrt(c.rr / c.rr0) : 0.0;
    if (c.status == POISSON_NOT_CONVERGED) ctx->err = "CG: residual threshold not reached within max_iter iterations";
    return c.status;
}

// z = B^-1 f, B = the colour-block lower-triangular part of L_h (Eq. 10): one red-black Gauss-Seidel sweep
// on L_h z = f from z = 0; symmetric: a second red half-sweep (the CG preconditioner).  One fused pass where the fused
// kernel applies (zeros = an all-zero vector it reads as the initial guess), else half-sweep kernels.
// with_rz (preconditioned CG): r . z and beta follow in the control block, inside the fused pass or by k_pcg_dot.
static int gs_precond_apply(poisson_ctx* ctx, const double* f, double* z, const double* zeros, bool symmetric,
                            bool with_rz = false) {
    if (ctx->kind == KIND_CART2 && sor_fused_ok(ctx, ctx->op))
        return sor_fused_precond(ctx, ctx->op, zeros, z, f, symmetric, with_rz);
    PB_CUDA_OK(cudaMemsetAsync(z, 0, ctx->npts * sizeof(double), ctx->stream));
    for (int h = 0; h < (symmetric ? 3 : 2); ++h) {
        const int rc = launch_rbsor_half(ctx, ctx->op, ctx->kind, z, f, 1.0, h & 1, false, KID_PCG_PRECOND);
        if (rc != POISSON_OK) return rc;
    }
    return with_rz ? launch_pcg_dot(ctx, f, z) : POISSON_OK;
}

int poisson_bicgstab_solve(poisson_t ctx, double* d_phi, const double* d_rhs, double rtol, int max_iter,
                           int fixed_iters, int* iters, double* relres) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    if (fixed_iters <= 0 && (max_iter < 1 || !(rtol > 0))) return fail(ctx, POISSON_INVALID_ARG, "bad rtol/max_iter");
    double *r = scratch(ctx, 0), *r0 = scratch(ctx, 1), *P[2] = {scratch(ctx, 2), scratch(ctx, 3)},
           *V[2] = {scratch(ctx, 4), scratch(ctx, 5)}, *s = scratch(ctx, 6), *t = scratch(ctx, 7);
    if (!r || !r0 || !P[0] || !P[1] || !V[0] || !V[1] || !s || !t) return POISSON_OUT_OF_MEMORY;
    const bool gs = ctx->opt_jacobi == 2;  // right-preconditioned by the Gauss-Seidel sweep of Eq. 10
    double *ph = nullptr, *sh = nullptr, *zeros = nullptr;
    if (gs) {
        if (ctx->kind == KIND_CART6)
            return fail(ctx, POISSON_UNSUPPORTED, "the two-colour Gauss-Seidel preconditioner needs a radius-1 stencil (PAPER.md:113)");
        ph = scratch(ctx, 8);
        sh = scratch(ctx, 9);
        zeros = scratch(ctx, 10);
        if (!ph || !sh || !zeros) return POISSON_OUT_OF_MEMORY;
        PB_CUDA_OK(cudaMemsetAsync(zeros, 0, ctx->npts * sizeof(double), ctx->stream));
    }
    int rc = krylov_setup(ctx, rtol, max_iter, fixed_iters, false);
    if (rc != POISSON_OK) return rc;
    for (double* z : {P[0], P[1], V[0], V[1]}) PB_CUDA_OK(cudaMemsetAsync(z, 0, ctx->npts * sizeof(double), ctx->stream));
    rc = launch_krylov_init(ctx, d_phi, d_rhs, r, true, r0);
    if (rc != POISSON_OK) return rc;
    const int nit = fixed_iters > 0 ? fixed_iters : max_iter;
    int nconfirm_failed = 0;
    for (int j = 0; j < nit;) {
        const int chunk = std::min(ctx->opt_poll, nit - j);
        for (int c = 0; c < chunk; ++c, ++j) {
            const int o = j & 1, n = (j + 1) & 1;
            if (gs) {  // p and v are updated in place (P[0], V[0]): nothing reads a neighbour of the vector being written
                if ((rc = launch_gsb_p(ctx, r, P[0], V[0], r0)) != POISSON_OK) return rc;
                if ((rc = gs_precond_apply(ctx, P[0], ph, zeros, false)) != POISSON_OK) return rc;
                if ((rc = launch_gsb_matvec(ctx, 1, ph, V[0], r0)) != POISSON_OK) return rc;
                if ((rc = launch_gsb_s(ctx, r, V[0], s)) != POISSON_OK) return rc;
                if ((rc = gs_precond_apply(ctx, s, sh, zeros, false)) != POISSON_OK) return rc;
                if ((rc = launch_gsb_matvec(ctx, 2, sh, t, s)) != POISSON_OK) return rc;
                if ((rc = launch_gsb_update(ctx, d_phi, ph, sh, s, t, r0, r)) != POISSON_OK) return rc;
                continue;
            }
            if ((rc = launch_bicg_pass1(ctx, r, P[o], V[o], r0, P[n], V[n])) != POISSON_OK) return rc;
            if ((rc = launch_bicg_pass2(ctx, r, V[n], s, t)) != POISSON_OK) return rc;
            if ((rc = launch_bicg_pass3(ctx, d_phi, P[n], s, t, r0, r)) != POISSON_OK) return rc;
        }
        PB_CUDA_OK(cudaGetLastError());
        if (fixed_iters <= 0) {
            rc = read_ctl(ctx);
            if (rc != POISSON_OK) return rc;
            if (!ctx->h_ctl->done) continue;
            if (ctx->h_ctl->status != POISSON_OK || !(ctx->h_ctl->rr0 > 0.0)) break;
            // The recurrence says converged: confirm with the true residual r = rhs - L x (the recursively updated r
            // drifts away from it over thousands of iterations); if it is not there yet the pass has restarted the
            // iteration from it (r^_0 := r, p := r) and cleared done.  DESIGN.md reading C4.
            static const int one = 1;
            PB_CUDA_OK(cudaMemcpyAsync(&ctx->d_ctl->confirm, &one, sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
            rc = launch_krylov_init(ctx, d_phi, d_rhs, r, true, r0);
            if (rc != POISSON_OK) return rc;
            rc = read_ctl(ctx);
            if (rc != POISSON_OK) return rc;
            if (ctx->h_ctl->done) break;
            nconfirm_failed += 1;
            j = ctx->h_ctl->it;
        }
    }
    rc = read_ctl(ctx);
    if (rc != POISSON_OK) return rc;
    const KrylovCtl c = *ctx->h_ctl;
    ctx->hist_len = c.it + 1;
    if (iters) *iters = c.it;
    if (relres) *relres = c.rr0 > 0 ? std::sqrt(c.rr / c.rr0) : 0.0;
    if (c.status == POISSON_NOT_CONVERGED) ctx->err = "BiCGSTAB: residual threshold not reached within max_iter";
    ctx->last_restarts = c.nrestarts;
    ctx->last_confirm_failed = nconfirm_failed;
    if (c.status == POISSON_BREAKDOWN) ctx->err = "BiCGSTAB: breakdown (rho, omega or r0.v vanished or is not finite)";
    return c.status;
}

int poisson_get_history(poisson_t ctx, double* h_out, int n) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !h_out || n < 0) return POISSON_INVALID_ARG;
    if (!ctx->d_hist || n > ctx->hist_cap) return fail(ctx, POISSON_INVALID_ARG, "no history recorded / n too large");
    PB_CUDA_OK(cudaMemcpyAsync(h_out, ctx->d_hist, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
    return POISSON_OK;
}

// ---- multigrid --------------------------------------------------------------------------------------------------------
static int build_levels(poisson_ctx* ctx, int coarsest_n, bool mixed) {
    if (ctx->mg_coarsest_n != coarsest_n) {
        free_levels(ctx);
        MgLevel L0;
        L0.op = ctx->op;
        L0.npts = ctx->npts;
        ctx->levels.push_back(L0);
        double hl[3] = {ctx->h[0], ctx->h[1], ctx->h[2]};
        int lev = 0;
        while (ctx->levels.back().op.n[0] > coarsest_n && ctx->levels.back().op.n[0] % 2 == 0 &&
               ctx->levels.back().op.n[1] % 2 == 0 && ctx->levels.back().op.n[2] % 2 == 0) {
            ++lev;
            MgLevel L;
            L.op = ctx->levels.back().op;
            L.npts = 1;
            for (int a = 0; a < 3; ++a) {
                L.op.n[a] /= 2;
                hl[a] *= 2.0;
                L.op.c[a] = 1.0 / (hl[a] * hl[a]);
                L.npts *= (size_t)L.op.n[a];
            }
            const double s = std::ldexp(1.0, lev);
            L.op.gamma = (s - 1.0) / (s + 1.0);  // ghost closure of DESIGN.md reading C7
            for (int f = 0; f < 6; ++f) L.op.ghost[f] = nullptr;
            ctx->levels.push_back(L);
        }
        ctx->mg_coarsest_n = coarsest_n;
    }
    for (size_t l = 0; l < ctx->levels.size(); ++l) {
        MgLevel& L = ctx->levels[l];
        const size_t b64 = L.npts * sizeof(double), b32 = L.npts * sizeof(float);
        if (!mixed) {
            if (l > 0 && !L.phi) PB_CUDA_OK(cudaMalloc((void**)&L.phi, b64));
            if (l > 0 && !L.rhs) PB_CUDA_OK(cudaMalloc((void**)&L.rhs, b64));
            if (!L.res) PB_CUDA_OK(cudaMalloc((void**)&L.res, b64));
            if (!L.alt) PB_CUDA_OK(cudaMalloc((void**)&L.alt, b64));
        } else {
            if (!L.phi32) PB_CUDA_OK(cudaMalloc((void**)&L.phi32, b32));
            if (!L.rhs32) PB_CUDA_OK(cudaMalloc((void**)&L.rhs32, b32));
            if (!L.res32) PB_CUDA_OK(cudaMalloc((void**)&L.res32, b32));
            if (!L.alt32) PB_CUDA_OK(cudaMalloc((void**)&L.alt32, b32));
        }
    }
    return POISSON_OK;
}

// One V-cycle on level l and below.  The field of the level starts in `phi`; the red-black passes ping-pong between it
// and the level's second buffer, and *result tells the caller which of the two holds the outcome (no copies).
static int cycle64(poisson_ctx* ctx, size_t l, double* phi, const double* rhs, bool ug, int nu1, int nu2, int csweeps,
                   double** result) {
    MgLevel& L = ctx->levels[l];
    int rc;
    *result = phi;
    if (!ug && L.npts <= 4096 && ctx->opt_path != 1) {  // the rest of the cycle fits one CTA's shared memory
        Op ops[8];
        const size_t nl = ctx->levels.size() - l;
        if (nl <= 4) {
            for (size_t m = 0; m < nl; ++m) ops[m] = ctx->levels[l + m].op;
            const double omc = 2.0 / (1.0 + std::sin(M_PI / (ops[nl - 1].n[0] + 1)));
            rc = launch_mg_bottom(ctx, ops, (int)nl, phi, rhs, nu1, nu2, csweeps, omc);
            if (rc != POISSON_UNSUPPORTED) return rc;
        }
    }
    if (l + 1 == ctx->levels.size()) {
        const double om = 2.0 / (1.0 + std::sin(M_PI / (L.op.n[0] + 1)));  // Eq. 3-4 for n unknowns per axis
        rc = ug ? POISSON_UNSUPPORTED : launch_coarse_solve(ctx, L.op, phi, rhs, om, csweeps);
        if (rc == POISSON_UNSUPPORTED) rc = launch_rbsor(ctx, L.op, KIND_CART2, phi, rhs, om, csweeps, ug);
        return rc;
    }
    MgLevel& C = ctx->levels[l + 1];
    double* cur = phi;
    if ((rc = launch_rbsor_pp(ctx, L.op, &cur, phi, L.alt, rhs, 1.0, nu1, ug)) != POISSON_OK) return rc;
    // residual and restriction in one pass (no fine residual in memory).  fp64, measured: 13 / 12 us against 20 / 18 us
    // for the two kernels at 64^3 / 32^3, the same at 128^3, 181 against 153 us at 256^3 (one 704-thread CTA per SM
    // with a barrier per plane, against the TMA-staged residual kernel with three small CTAs): fused below 2^21 points
    const bool fuse = ctx->opt_fused_restrict == 1 || (ctx->opt_fused_restrict == 0 && L.npts < ((size_t)1 << 21));
    if (fuse && resid_restrict_ok(ctx, L.op, C.op)) {
        if ((rc = resid_restrict(ctx, L.op, C.op, cur, rhs, C.rhs, ug)) != POISSON_OK) return rc;
    } else {
        if ((rc = launch_apply(ctx, L.op, KIND_CART2, cur, rhs, L.res, 1, ug, false)) != POISSON_OK) return rc;
        if ((rc = launch_restrict(ctx, L.op, C.op, L.res, C.rhs, ctx->opt_restriction)) != POISSON_OK) return rc;
    }
    PB_CUDA_OK(cudaMemsetAsync(C.phi, 0, C.npts * sizeof(double), ctx->stream));
    double* ec = C.phi;
    if ((rc = cycle64(ctx, l + 1, C.phi, C.rhs, false, nu1, nu2, csweeps, &ec)) != POISSON_OK) return rc;
    if ((rc = launch_prolong_add(ctx, L.op, C.op, ec, cur)) != POISSON_OK) return rc;
    if ((rc = launch_rbsor_pp(ctx, L.op, &cur, phi, L.alt, rhs, 1.0, nu2, ug)) != POISSON_OK) return rc;
    *result = cur;
    return POISSON_OK;
}

static int cycle32(poisson_ctx* ctx, size_t l, int nu1, int nu2, int csweeps, float** result) {
    MgLevel& L = ctx->levels[l];
    int rc;
    *result = L.phi32;
    if (L.npts <= 4096 && ctx->opt_path != 1) {
        Op ops[8];
        const size_t nl = ctx->levels.size() - l;
        if (nl <= 4) {
            for (size_t m = 0; m < nl; ++m) ops[m] = ctx->levels[l + m].op;
            const double omc = 2.0 / (1.0 + std::sin(M_PI / (ops[nl - 1].n[0] + 1)));
            rc = launch_mg_bottom32(ctx, ops, (int)nl, L.phi32, L.rhs32, nu1, nu2, csweeps, omc);
            if (rc != POISSON_UNSUPPORTED) return rc;
        }
    }
    if (l + 1 == ctx->levels.size()) {
        const float om = (float)(2.0 / (1.0 + std::sin(M_PI / (L.op.n[0] + 1))));
        rc = launch_coarse_solve32(ctx, L.op, L.phi32, L.rhs32, om, csweeps);
        if (rc == POISSON_UNSUPPORTED) rc = launch_rbsor32(ctx, L.op, L.phi32, L.rhs32, om, csweeps);
        return rc;
    }
    MgLevel& C = ctx->levels[l + 1];
    float* cur = L.phi32;
    if ((rc = launch_rbsor_pp32(ctx, L.op, &cur, L.phi32, L.alt32, L.rhs32, 1.0f, nu1)) != POISSON_OK) return rc;
    if (ctx->opt_fused_restrict != 2 && resid_restrict_ok(ctx, L.op, C.op)) {
        if ((rc = resid_restrict32(ctx, L.op, C.op, cur, L.rhs32, C.rhs32)) != POISSON_OK) return rc;
    } else {
        if ((rc = launch_apply32(ctx, L.op, cur, L.rhs32, L.res32, 1)) != POISSON_OK) return rc;
        if ((rc = launch_restrict32(ctx, L.op, C.op, L.res32, C.rhs32, ctx->opt_restriction)) != POISSON_OK) return rc;
    }
    PB_CUDA_OK(cudaMemsetAsync(C.phi32, 0, C.npts * sizeof(float), ctx->stream));
    float* ec = C.phi32;
    if ((rc = cycle32(ctx, l + 1, nu1, nu2, csweeps, &ec)) != POISSON_OK) return rc;
    if ((rc = launch_prolong_add32(ctx, L.op, C.op, ec, cur)) != POISSON_OK) return rc;
    if ((rc = launch_rbsor_pp32(ctx, L.op, &cur, L.phi32, L.alt32, L.rhs32, 1.0f, nu2)) != POISSON_OK) return rc;
    *result = cur;
    return POISSON_OK;
}

int poisson_mg_vcycle(poisson_t ctx, double* d_phi, const double* d_rhs, int nu1, int nu2, int coarsest_n,
                      int coarsest_sweeps, int precision, int ncycles, double* h_resnorms) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    if (nu1 < 0 || nu2 < 0 || coarsest_n < 1 || coarsest_sweeps < 0 || ncycles < 0 ||
        (precision != POISSON_F64 && precision != POISSON_MIXED))
        return fail(ctx, POISSON_INVALID_ARG, "bad V-cycle parameters");
    if (ctx->kind != KIND_CART2) return fail(ctx, POISSON_UNSUPPORTED, "multigrid: Cartesian 7-point operator only");
    for (int f = 0; f < 6; ++f)
        if (ctx->op.bc[f] != POISSON_BC_DIRICHLET_GHOST)
            return fail(ctx, POISSON_UNSUPPORTED, "multigrid: Dirichlet (ghost) faces only");
    int rc = build_levels(ctx, coarsest_n, precision == POISSON_MIXED);
    if (rc != POISSON_OK) return rc;
    // the last-block reductions write squared norms to d_scal[16 + c]; one copy at the end, no per-cycle sync
    auto record_norm = [&](int slot) -> int {
        if (!h_resnorms) return POISSON_OK;
        int r2 = launch_apply(ctx, ctx->op, ctx->kind, d_phi, d_rhs, nullptr, 1, true, true);
        if (r2 != POISSON_OK) return r2;
        PB_CUDA_OK(cudaMemcpyAsync(ctx->d_scal + 16 + slot, ctx->d_scal, sizeof(double), cudaMemcpyDeviceToDevice,
                                   ctx->stream));
        return POISSON_OK;
    };
    if (ncycles + 1 > 200) return fail(ctx, POISSON_INVALID_ARG, "ncycles too large");
    if ((rc = record_norm(0)) != POISSON_OK) return rc;
    for (int c = 0; c < ncycles; ++c) {
        if (precision == POISSON_F64) {
            double* res = d_phi;
            rc = cycle64(ctx, 0, d_phi, d_rhs, true, nu1, nu2, coarsest_sweeps, &res);
            if (rc == POISSON_OK && res != d_phi)  // an odd number of ping-pong passes on level 0
                PB_CUDA_OK(cudaMemcpyAsync(d_phi, res, ctx->npts * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream));
        } else {
            MgLevel& L0 = ctx->levels[0];
            rc = launch_residual_to32(ctx, ctx->op, d_phi, d_rhs, L0.rhs32, true);
            if (rc != POISSON_OK) return rc;
            PB_CUDA_OK(cudaMemsetAsync(L0.phi32, 0, L0.npts * sizeof(float), ctx->stream));
            float* e32 = L0.phi32;
            rc = cycle32(ctx, 0, nu1, nu2, coarsest_sweeps, &e32);
            if (rc != POISSON_OK) return rc;
            rc = launch_add32to64(ctx, L0.npts, e32, d_phi);
        }
        if (rc != POISSON_OK) return rc;
        if ((rc = record_norm(c + 1)) != POISSON_OK) return rc;
    }
    if (h_resnorms) {
        PB_CUDA_OK(cudaMemcpyAsync(ctx->h_scal, ctx->d_scal + 16, (ncycles + 1) * sizeof(double),
                                   cudaMemcpyDeviceToHost, ctx->stream));
        PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
        for (int c = 0; c <= ncycles; ++c) h_resnorms[c] = std::sqrt(ctx->h_scal[c]);
    }
    return POISSON_OK;
}

// ---- the paper's own multigrid: SPAI smoother, vertex-centred Galerkin hierarchy (rows f1, f2) -------------------------------
int poisson_spai_smooth(poisson_t ctx, double* d_phi, const double* d_rhs, const double* spai, int nsteps) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs || nsteps < 0) return fail(ctx, POISSON_INVALID_ARG, "bad arguments");
    return mgv_spai_smooth(ctx, d_phi, d_rhs, spai, nsteps);
}

int poisson_mgv_vcycle(poisson_t ctx, double* d_phi, const double* d_rhs, int nu1, int nu2, int coarsest_n,
                       const double* spai, double cg_rtol, int precision, int ncycles, double* h_resnorms) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    if (nu1 < 0 || nu2 < 0 || coarsest_n < 1 || ncycles < 0 || ncycles + 1 > 200 || !(cg_rtol > 0) ||
        (precision != POISSON_F64 && precision != POISSON_MIXED))
        return fail(ctx, POISSON_INVALID_ARG, "bad V-cycle parameters");
    auto record_norm = [&](int slot) -> int {
        if (!h_resnorms) return POISSON_OK;
        // order 2: the handle's 7-point residual with its ghosts; compact orders: the residual of the compact operator
        int r2 = ctx->opt_compact_order == 2
                     ? launch_apply(ctx, ctx->op, ctx->kind, d_phi, d_rhs, nullptr, 1, true, true)
                     : mgv_residual_norm2(ctx, d_phi, d_rhs, coarsest_n, precision == POISSON_MIXED);
        if (r2 != POISSON_OK) return r2;
        PB_CUDA_OK(cudaMemcpyAsync(ctx->d_scal + 16 + slot, ctx->d_scal, sizeof(double), cudaMemcpyDeviceToDevice,
                                   ctx->stream));
        return POISSON_OK;
    };
    int rc = record_norm(0);
    if (rc != POISSON_OK) return rc;
    rc = mgv_vcycles(ctx, d_phi, d_rhs, nu1, nu2, coarsest_n, spai, cg_rtol, precision == POISSON_MIXED, ncycles,
                     record_norm);
    if (rc != POISSON_OK) return rc;
    if (h_resnorms) {
        PB_CUDA_OK(cudaMemcpyAsync(ctx->h_scal, ctx->d_scal + 16, (ncycles + 1) * sizeof(double),
                                   cudaMemcpyDeviceToHost, ctx->stream));
        PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
        for (int c = 0; c <= ncycles; ++c) h_resnorms[c] = std::sqrt(ctx->h_scal[c]);
    }
    return POISSON_OK;
}

int poisson_compact_rhs(poisson_t ctx, const double* d_f_ext, double* d_out) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_f_ext || !d_out) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    if (ctx->kind != KIND_CART2 || ctx->h[0] != ctx->h[1] || ctx->h[0] != ctx->h[2])
        return fail(ctx, POISSON_UNSUPPORTED, "compact right-hand side: Cartesian grid with isotropic spacing (PAPER.md:172)");
    return mgv_compact_rhs(ctx, d_f_ext, d_out);
}

// ---- multipole boundary -------------------------------------------------------------------------------------------------
int poisson_multipole_bc(poisson_t ctx, const double* d_rho, double G, int lmax, double* h_moments) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_rho) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    if (lmax < 0 || lmax > kMaxLmax) return fail(ctx, POISSON_INVALID_ARG, "lmax must be in 0..8");
    double* d_q = ctx->d_scal + 128;
    int rc = launch_moments(ctx, d_rho, lmax, d_q, false);
    if (rc != POISSON_OK) return rc;
    // a spherical grid whose inner radial face is a Dirichlet face also takes the inner expansion (Eq. 21-22)
    double* d_qbar = nullptr;
    if (ctx->op.coord == POISSON_SPHERICAL && ctx->op.bc[0] == POISSON_BC_DIRICHLET_GHOST) {
        d_qbar = ctx->d_scal + 300;
        if ((rc = launch_moments(ctx, d_rho, lmax, d_qbar, true)) != POISSON_OK) return rc;
    }
    ctx->inner_lmax = d_qbar ? lmax : -1;
    rc = launch_ghost_eval(ctx, d_q, d_qbar, G, lmax);
    if (rc != POISSON_OK) return rc;
    ctx->ghost_nonzero = true;
    if (h_moments) {
        const int nq = (lmax + 1) * (lmax + 1);
        PB_CUDA_OK(cudaMemcpyAsync(ctx->h_scal + 128, d_q, nq * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
        PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
        std::memcpy(h_moments, ctx->h_scal + 128, nq * sizeof(double));
    }
    return POISSON_OK;
}

int poisson_multipole_inner_moments(poisson_t ctx, double* h_qbar, int lmax) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !h_qbar) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    if (ctx->inner_lmax < 0 || lmax != ctx->inner_lmax)
        return fail(ctx, POISSON_INVALID_ARG, "no inner moments of this order: call poisson_multipole_bc on a spherical grid "
                                              "with a Dirichlet inner face first");
    const int nq = (lmax + 1) * (lmax + 1);
    PB_CUDA_OK(cudaMemcpyAsync(ctx->h_scal + 300, ctx->d_scal + 300, nq * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
    std::memcpy(h_qbar, ctx->h_scal + 300, nq * sizeof(double));
    return POISSON_OK;
}

// ---- rows f3, f4: omega sequences, position-dependent omega, Gauss-Seidel-preconditioned CG ------------------------------
// Eq. 4 with N = n + 1 intervals (exact for ghost-Dirichlet faces; reading C0).
static double jacobi_radius_eq4(const poisson_ctx* ctx) {
    double num = 0.0, den = 0.0;
    for (int a = 0; a < 3; ++a) {
        num += ctx->op.c[a] * std::cos(M_PI / (ctx->op.n[a] + 1));
        den += ctx->op.c[a];
    }
    return num / den;
}

int poisson_rbsor_cheby(poisson_t ctx, double* d_phi, const double* d_rhs, double r_jacobi, int nsweeps, int start_n,
                        double* h_resnorm) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs || nsweeps < 0 || start_n < 0) return fail(ctx, POISSON_INVALID_ARG, "bad arguments");
    if (!(r_jacobi > 0.0)) {
        if (ctx->kind != KIND_CART2) return fail(ctx, POISSON_INVALID_ARG, "r_jacobi must be given on this grid (Eq. 4 is Cartesian)");
        r_jacobi = jacobi_radius_eq4(ctx);
    }
    if (!(r_jacobi < 1.0)) return fail(ctx, POISSON_INVALID_ARG, "the Jacobi spectral radius must lie in (0,1)");
    // Eq. 6: omega_0 = 1, omega_1 = 1/(1 - rJ^2/2), omega_{n+1} = 1/(1 - rJ^2 omega_n/4); half-sweep m uses omega_{m+start_n}
    std::vector<double> om((size_t)2 * nsweeps);
    double w = 1.0;
    for (int n = 1; n <= start_n; ++n) w = n == 1 ? 1.0 / (1.0 - 0.5 * r_jacobi * r_jacobi) : 1.0 / (1.0 - 0.25 * r_jacobi * r_jacobi * w);
    for (int m = 0; m < 2 * nsweeps; ++m) {
        om[m] = w;
        const int nn = m + start_n + 1;
        w = nn == 1 ? 1.0 / (1.0 - 0.5 * r_jacobi * r_jacobi) : 1.0 / (1.0 - 0.25 * r_jacobi * r_jacobi * w);
    }
    int rc = launch_rbsor_seq(ctx, ctx->op, ctx->kind, d_phi, d_rhs, om.data(), nsweeps, true);
    if (rc != POISSON_OK) return rc;
    if (h_resnorm) return residual_norm_sync(ctx, d_phi, d_rhs, h_resnorm);
    return POISSON_OK;
}

int poisson_rbsor_local(poisson_t ctx, double* d_phi, const double* d_rhs, int nsweeps, int start_n, double* h_resnorm) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs || nsweeps < 0 || start_n < 0) return fail(ctx, POISSON_INVALID_ARG, "bad arguments");
    if (ctx->kind == KIND_CART6) return fail(ctx, POISSON_UNSUPPORTED, "red-black sweeps need a radius-1 stencil");
    const int n0 = ctx->op.n[0], n1 = ctx->op.n[1];
    const size_t n2d = (size_t)n0 * n1;
    if (!ctx->d_rj) {
        // Eq. 7: the local Jacobi radius from the grid metric (a coefficient array like those of setup_spherical)
        std::vector<double> rj(n2d);
        for (int j = 0; j < n1; ++j)
            for (int i = 0; i < n0; ++i) {
                if (ctx->kind == KIND_SPH) {
                    const double dr = ctx->edges[0][i + 1] - ctx->edges[0][i], dth = ctx->edges[1][j + 1] - ctx->edges[1][j];
                    const double dph = ctx->edges[2][1] - ctx->edges[2][0];
                    const double r = ctx->ctr[0][i], st = std::sin(ctx->ctr[1][j]);
                    const double a = 1.0 / (dr * dr), b = 1.0 / ((r * dth) * (r * dth)), c = 1.0 / ((r * st * dph) * (r * st * dph));
                    rj[(size_t)j * n0 + i] = (std::cos(M_PI / n0) * a + std::cos(M_PI / n1) * b + std::cos(M_PI / ctx->op.n[2]) * c) / (a + b + c);
                } else {
                    rj[(size_t)j * n0 + i] = jacobi_radius_eq4(ctx);
                }
            }
        PB_CUDA_OK(cudaMalloc((void**)&ctx->d_rj, 2 * n2d * sizeof(double)));
        PB_CUDA_OK(cudaMemcpyAsync(ctx->d_rj, rj.data(), n2d * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
        PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));  // rj is a local vector
    }
    int rc = launch_rbsor_local(ctx, ctx->op, ctx->kind, d_phi, d_rhs, ctx->d_rj, ctx->d_rj + n2d, nsweeps, start_n, true);
    if (rc != POISSON_OK) return rc;
    if (h_resnorm) return residual_norm_sync(ctx, d_phi, d_rhs, h_resnorm);
    return POISSON_OK;
}

static int gs_precond(poisson_ctx* ctx, const double* r, double* z, const double* zeros) {
    return gs_precond_apply(ctx, r, z, zeros, true, true);  // red, black, red; then r . z
}

int poisson_pcg_solve(poisson_t ctx, double* d_phi, const double* d_rhs, double rtol, int max_iter, int fixed_iters,
                      int* iters, double* relres) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !d_phi || !d_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    if (fixed_iters <= 0 && (max_iter < 1 || !(rtol > 0))) return fail(ctx, POISSON_INVALID_ARG, "bad rtol/max_iter");
    if (ctx->kind != KIND_CART2)
        return fail(ctx, POISSON_UNSUPPORTED, "Gauss-Seidel-preconditioned CG: Cartesian 7-point operator (two colours, PAPER.md:113)");
    for (int f = 0; f < 6; ++f)
        if (ctx->op.bc[f] == POISSON_BC_PERIODIC)
            return fail(ctx, POISSON_UNSUPPORTED, "Gauss-Seidel-preconditioned CG: non-periodic faces only");
    double *r = scratch(ctx, 0), *P[2] = {scratch(ctx, 1), scratch(ctx, 2)}, *q = scratch(ctx, 3), *z = scratch(ctx, 4),
           *zeros = scratch(ctx, 5);
    if (!r || !P[0] || !P[1] || !q || !z || !zeros) return POISSON_OUT_OF_MEMORY;
    int rc = krylov_setup(ctx, rtol, max_iter, fixed_iters, false, true);
    if (rc != POISSON_OK) return rc;
    for (double* v : {P[0], P[1], zeros}) PB_CUDA_OK(cudaMemsetAsync(v, 0, ctx->npts * sizeof(double), ctx->stream));
    if ((rc = launch_krylov_init(ctx, d_phi, d_rhs, r, false, nullptr)) != POISSON_OK) return rc;
    if ((rc = gs_precond(ctx, r, z, zeros)) != POISSON_OK) return rc;
    const int nit = fixed_iters > 0 ? fixed_iters : max_iter;
    for (int j = 0; j < nit;) {
        const int chunk = std::min(ctx->opt_poll, nit - j);
        for (int c = 0; c < chunk; ++c, ++j) {
            // pass A with z in the place of r: p = z + beta p_old, q = L p, alpha = r.z / p.q (+ deferred x-update)
            if ((rc = launch_cg_passA(ctx, z, P[j & 1], P[(j + 1) & 1], q, d_phi)) != POISSON_OK) return rc;
            if ((rc = launch_cg_passB(ctx, r, q)) != POISSON_OK) return rc;
            if ((rc = gs_precond(ctx, r, z, zeros)) != POISSON_OK) return rc;
        }
        PB_CUDA_OK(cudaGetLastError());
        if (fixed_iters <= 0) {
            if ((rc = read_ctl(ctx)) != POISSON_OK) return rc;
            if (ctx->h_ctl->done) break;
        }
    }
    if ((rc = read_ctl(ctx)) != POISSON_OK) return rc;
    const KrylovCtl c = *ctx->h_ctl;
    if ((rc = launch_cg_final(ctx, d_phi, P[c.it & 1])) != POISSON_OK) return rc;
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
    ctx->hist_len = c.it + 1;
    if (iters) *iters = c.it;
    if (relres) *relres = c.rr0 > 0 ? std::sqrt(c.rr / c.rr0) : 0.0;
    if (c.status == POISSON_NOT_CONVERGED) ctx->err = "PCG: residual threshold not reached within max_iter iterations";
    return c.status;
}

// ---- end-to-end with host buffers -----------------------------------------------------------------------------------------
// Each call copies its inputs host->device on the handle's stream, runs the device entry point above, copies the
// result back and synchronises.  Host buffers should be pinned for full PCIe speed; pageable memory also works.
static int stage(poisson_ctx* ctx, int slot, const double* h_src) {
    const size_t bytes = ctx->npts * sizeof(double);
    if (!ctx->d_stage[slot]) PB_CUDA_OK(cudaMalloc((void**)&ctx->d_stage[slot], bytes));
    if (h_src) PB_CUDA_OK(cudaMemcpyAsync(ctx->d_stage[slot], h_src, bytes, cudaMemcpyHostToDevice, ctx->stream));
    return POISSON_OK;
}
static int unstage(poisson_ctx* ctx, int slot, double* h_dst) {
    PB_CUDA_OK(cudaMemcpyAsync(h_dst, ctx->d_stage[slot], ctx->npts * sizeof(double), cudaMemcpyDeviceToHost,
                               ctx->stream));
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
    return POISSON_OK;
}
#define STAGE_OK(call)                  \
    do {                                \
        int rc__ = (call);              \
        if (rc__ != POISSON_OK) return rc__; \
    } while (0)

int poisson_apply_laplacian_host(poisson_t ctx, const double* h_phi, double* h_out) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !h_phi || !h_out) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    STAGE_OK(stage(ctx, 0, h_phi));
    STAGE_OK(stage(ctx, 1, nullptr));
    const int rc = poisson_apply_laplacian(ctx, ctx->d_stage[0], ctx->d_stage[1]);
    if (rc < 0) return rc;
    return unstage(ctx, 1, h_out);
}

int poisson_rbsor_sweep_host(poisson_t ctx, double* h_phi, const double* h_rhs, double omega, int nsweeps,
                             double* h_resnorm) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !h_phi || !h_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    STAGE_OK(stage(ctx, 0, h_phi));
    STAGE_OK(stage(ctx, 1, h_rhs));
    const int rc = poisson_rbsor_sweep(ctx, ctx->d_stage[0], ctx->d_stage[1], omega, nsweeps, h_resnorm);
    if (rc < 0) return rc;
    return unstage(ctx, 0, h_phi);
}

int poisson_cg_solve_host(poisson_t ctx, double* h_phi, const double* h_rhs, double rtol, int max_iter,
                          int fixed_iters, int* iters, double* relres) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !h_phi || !h_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    STAGE_OK(stage(ctx, 0, h_phi));
    STAGE_OK(stage(ctx, 1, h_rhs));
    const int rc = poisson_cg_solve(ctx, ctx->d_stage[0], ctx->d_stage[1], rtol, max_iter, fixed_iters, iters, relres);
    if (rc < 0) return rc;
    const int rc2 = unstage(ctx, 0, h_phi);
    return rc2 != POISSON_OK ? rc2 : rc;
}

int poisson_bicgstab_solve_host(poisson_t ctx, double* h_phi, const double* h_rhs, double rtol, int max_iter,
                                int fixed_iters, int* iters, double* relres) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !h_phi || !h_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    STAGE_OK(stage(ctx, 0, h_phi));
    STAGE_OK(stage(ctx, 1, h_rhs));
    const int rc =
        poisson_bicgstab_solve(ctx, ctx->d_stage[0], ctx->d_stage[1], rtol, max_iter, fixed_iters, iters, relres);
    if (rc < 0) return rc;
    const int rc2 = unstage(ctx, 0, h_phi);
    return rc2 != POISSON_OK ? rc2 : rc;
}

int poisson_mg_vcycle_host(poisson_t ctx, double* h_phi, const double* h_rhs, int nu1, int nu2, int coarsest_n,
                           int coarsest_sweeps, int precision, int ncycles, double* h_resnorms) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !h_phi || !h_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    STAGE_OK(stage(ctx, 0, h_phi));
    STAGE_OK(stage(ctx, 1, h_rhs));
    const int rc = poisson_mg_vcycle(ctx, ctx->d_stage[0], ctx->d_stage[1], nu1, nu2, coarsest_n, coarsest_sweeps,
                                     precision, ncycles, h_resnorms);
    if (rc < 0) return rc;
    return unstage(ctx, 0, h_phi);
}

int poisson_mgv_vcycle_host(poisson_t ctx, double* h_phi, const double* h_rhs, int nu1, int nu2, int coarsest_n,
                            const double* spai, double cg_rtol, int precision, int ncycles, double* h_resnorms) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !h_phi || !h_rhs) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    STAGE_OK(stage(ctx, 0, h_phi));
    STAGE_OK(stage(ctx, 1, h_rhs));
    const int rc = poisson_mgv_vcycle(ctx, ctx->d_stage[0], ctx->d_stage[1], nu1, nu2, coarsest_n, spai, cg_rtol,
                                      precision, ncycles, h_resnorms);
    if (rc < 0) return rc;
    return unstage(ctx, 0, h_phi);
}

int poisson_multipole_bc_host(poisson_t ctx, const double* h_rho, double G, int lmax, double* h_moments) {
    const DeviceGuard on_device(ctx);
    if (!ctx || !h_rho) return fail(ctx, POISSON_INVALID_ARG, "bad pointers");
    STAGE_OK(stage(ctx, 1, h_rho));
    const int rc = poisson_multipole_bc(ctx, ctx->d_stage[1], G, lmax, h_moments);
    if (rc < 0) return rc;
    PB_CUDA_OK(cudaStreamSynchronize(ctx->stream));
    return rc;
}

}  // extern "C"
