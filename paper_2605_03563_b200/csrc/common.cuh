// common.cuh — context, device-side operator descriptor and the single-pass grid reduction shared by all kernels.
// CUDA path of the Poisson hot path (arxiv/paper_2605_03563).  Shares no code with oracle/.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <functional>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/poisson.h"

namespace pb {

constexpr int kMaxLmax = 8;
constexpr int kRedSlots = 4;          // doubles per block in the partials buffer
constexpr int kMaxRedBlocks = 1 << 16;

// Operator descriptor, passed by value to kernels (lives in the constant bank).
struct Op {
    int n[3];
    int coord, order, R;
    int bc[6];
    double c[3];   // 1/h^2 per axis (Cartesian)
    double gamma;  // multigrid coarse-level ghost closure (0 on the user's grid)
    // spherical 1-D coefficient arrays (device): ar_m, ar_p, ir2, dr (len n0); at_m, at_p, cp, dt (len n1)
    const double* ar_m;
    const double* ar_p;
    const double* ir2;
    const double* dr;
    const double* at_m;
    const double* at_p;
    const double* cp;
    const double* dt;
    const double* ghost[6];  // device ghost-face arrays (nullptr on non-Dirichlet faces)
};

enum { KIND_CART2 = 0, KIND_CART6 = 1, KIND_SPH = 2 };

// Kernel classes, for launch counting and the optional per-class CUDA-event timing (POISSON_OPT_TIME_KERNELS).
enum KernelId {
    KID_APPLY = 0,      // stencil apply / residual (a1, a7)
    KID_RBSOR,          // red-black SOR sweeps (a2)
    KID_KRYLOV_INIT,    // initial residual of CG / BiCGSTAB
    KID_CG_PASS_A,      // p-update + matvec + p.Ap (+ deferred x-update) (a3)
    KID_CG_PASS_B,      // r-update + ||r||^2 (a3)
    KID_CG_FINAL,       // pending x-update / mean removal
    KID_BICG_PASS1,     // (a4)
    KID_BICG_PASS2,
    KID_BICG_PASS3,
    KID_MG_RESTRICT,    // residual + restriction (a5)
    KID_MG_PROLONG,     // prolongation + correction (+ smoothing) (a5)
    KID_MG_COARSE,      // coarsest-level solver (a5)
    KID_MG_AXPY,        // mixed path: phi += (double) e32
    KID_MP_MOMENTS,     // multipole moments (a6)
    KID_MP_GHOSTS,      // ghost-zone evaluation (a6)
    KID_MGV_SMOOTH,     // SPAI smoothing step (f1)
    KID_MGV_RESTRICT,   // vertex-centred residual + full weighting (f2)
    KID_MGV_PROLONG,    // vertex-centred trilinear prolongation + correction (f2)
    KID_MGV_COARSE,     // coarsest-level CG (f2)
    KID_MGV_SETUP,      // Galerkin stencils, boundary folding (f2)
    KID_PCG_PRECOND,    // red-black Gauss-Seidel preconditioner sweeps (f3)
    KID_COUNT
};

// Device-resident scalars of the Krylov solvers: nothing crosses to the host inside an iteration.
constexpr int kMaxBicgConfirm = 30;

struct KrylovCtl {
    double rr, rr0, pq, alpha, beta, mu, rho, omega, r0v, ts, tt, tol2;
    double sum_x;
    int it, done, status, fixed;
    int max_it, project, record, restart;  // restart: BiCGSTAB takes r^_0 := r in the next pass 1 (near-breakdown)
    double npoints;
    double r0n2, eps_bd;  // ||r^_0||^2 and the near-breakdown threshold on |rho| / (||r^_0|| ||r||)
    int nconf_failed, pad3;  // true-residual confirmations that failed so far (at most kMaxBicgConfirm)
    int nrestarts, confirm;                 // confirm: the next initial-residual pass re-checks convergence (BiCGSTAB)
    double rz;                              // preconditioned CG: r . M^-1 r
    int pcg, pad4;                          // pcg: alpha = rz / p.q and beta = rz_new / rz_old (Saad Alg. 9.1)
};

struct RedBuf {
    double* partials;       // kMaxRedBlocks * kRedSlots
    unsigned int* counter;  // self-resetting (atomicInc wraps)
};

#define PB_CUDA_OK(call)                                                                      \
    do {                                                                                      \
        cudaError_t e__ = (call);                                                             \
        if (e__ != cudaSuccess) return pb::fail_cuda(ctx, e__, #call, __FILE__, __LINE__);    \
    } while (0)

struct MgLevel {
    Op op;
    size_t npts = 0;
    double *phi = nullptr, *rhs = nullptr, *res = nullptr;     // fp64 storage (levels >= 1; level 0 uses caller's)
    float *phi32 = nullptr, *rhs32 = nullptr, *res32 = nullptr;  // fp32 storage (mixed path, all levels)
    double* alt = nullptr;   // second buffer of the level's field for the ping-pong red-black sweeps
    float* alt32 = nullptr;
};

// One level of the vertex-centred Galerkin hierarchy (k_mgv.cu): constant symmetric 27-point operator, spacing h.
struct MgvLevel {
    int n[3] = {0, 0, 0};
    double h = 0.0;
    size_t npts = 0;
    void *x = nullptr, *b = nullptr, *t = nullptr;  // x: two buffers (coarse levels); b; t: fp64 residual / ping-pong
};

}  // namespace pb

struct poisson_ctx {
    pb::Op op;
    int kind = 0;
    cudaStream_t stream = nullptr;
    size_t npts = 0;
    double h[3] = {1, 1, 1}, origin[3] = {0, 0, 0};
    std::vector<double> edges[3], ctr[3];
    double r_ghost_out = 0;
    double* d_coef = nullptr;       // spherical coefficient arrays, one allocation
    double* d_ctr = nullptr;        // spherical centres + cos/sin tables for the multipole kernels
    double* d_rj = nullptr;         // local Jacobi radius per (i,j) (Eq. 7) and the omega work array behind it (2 n0 n1)
    double* d_ghost[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    long face_len[6] = {0, 0, 0, 0, 0, 0};
    bool ghost_nonzero = false;
    int inner_lmax = -1;            // order of the inner multipole moments held in d_scal + 300 (-1: none)
    // scratch vectors (lazily allocated)
    std::vector<double*> vec;
    pb::RedBuf red{nullptr, nullptr};
    pb::KrylovCtl* d_ctl = nullptr;
    pb::KrylovCtl* h_ctl = nullptr;  // pinned
    double* d_hist = nullptr;
    int hist_cap = 0, hist_len = 0;
    double* d_scal = nullptr;        // small device scalar scratch (moments, norms)
    double* h_scal = nullptr;        // pinned
    std::vector<pb::MgLevel> levels;
    int mg_coarsest_n = -1;
    std::vector<pb::MgvLevel> vlevels;  // the paper's vertex-centred hierarchy
    double* v_sten = nullptr;           // 4 stencil coefficients per level (device)
    int v_key[3] = {-1, -1, -1};        // (coarsest_n, fp32 storage, compact order) the hierarchy was built for
    int opt_compact_order = 2;          // level-0 discretisation of the SPAI / Galerkin multigrid: 2, 4 or 6
    // options
    int opt_path = 0, opt_restriction = 0, opt_poll = 16, opt_jacobi = 1, opt_history = 0;
    int opt_sor_nhs = 0;             // colour half-steps fused per HBM pass of the red-black kernel (2, 4; 0 = auto)
    double opt_bicg_restart_eps = 1e-12;  // BiCGSTAB restart threshold (0 = never), reading C4
    int opt_fused_restrict = 0;      // V-cycle residual + restriction in one kernel: 0 auto (fp32 levels; fp64 levels below 2^21 points), 1 always, 2 never
    void* sor_tmp = nullptr;         // ping-pong buffer of the fused red-black kernel
    size_t sor_tmp_bytes = 0;
    long launches = 0;
    long launches_by_kid[pb::KID_COUNT] = {0};
    // optional event timing of one kernel class (or all with -2): pairs of events around every such launch
    int time_kid = -1;
    std::vector<cudaEvent_t> ev_pool;           // start/stop pairs, reused after poisson_reset_kernel_times
    std::vector<int> ev_kid;                    // kernel class of pair i
    size_t ev_used = 0;
    int num_sms = 148;
    int device = 0;                  // the device the handle was created on; every entry point runs on it
    // kernels whose dynamic shared-memory limit has been raised on this handle's device -> resident CTAs per SM
    std::unordered_map<const void*, int> kern_resident;
    // tuning overrides (poisson_set_option): -1 = automatic
    int opt_tile_cfg = -1, opt_plane_split = -1, opt_apply_bulk = -1;
    int last_restarts = 0, last_confirm_failed = 0;  // of the last BiCGSTAB solve (poisson_bicgstab_stats)
    std::string err;
    // pinned staging for the host-buffer entry points
    double* d_stage[2] = {nullptr, nullptr};
};

namespace pb {

int fail(poisson_ctx* ctx, int code, const std::string& msg);
int fail_cuda(poisson_ctx* ctx, cudaError_t e, const char* what, const char* file, int line);
double* scratch(poisson_ctx* ctx, int slot);  // lazily allocated npts-sized vector; nullptr on OOM
void pre_launch(poisson_ctx* ctx, int kid);
void post_launch(poisson_ctx* ctx, int kid);

// Raise the kernel's dynamic shared-memory limit (a per-device attribute) once per handle and report how many CTAs of
// it fit on an SM.  Handles are bound to one device and are not thread-safe, so the cache lives in the handle.
template <class K>
inline int kernel_ready(poisson_ctx* ctx, K kern, int nthreads, size_t smem, int* resident = nullptr) {
    const void* key = reinterpret_cast<const void*>(kern);
    auto it = ctx->kern_resident.find(key);
    if (it == ctx->kern_resident.end()) {
        PB_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int r = 0;
        PB_CUDA_OK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&r, kern, nthreads, smem));
        it = ctx->kern_resident.emplace(key, r).first;
    }
    if (resident) *resident = it->second;
    return POISSON_OK;
}

// Entry points run on the handle's device whatever the caller's current device is.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const poisson_ctx* ctx) {
        if (!ctx) return;
        if (cudaGetDevice(&prev) == cudaSuccess && prev != ctx->device) switched = cudaSetDevice(ctx->device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};

// Every kernel launch of the library goes through this: counts it and, when asked, brackets it with CUDA events.
#define PB_LAUNCH(ctx, kid, ...)       \
    do {                               \
        pb::pre_launch((ctx), (kid));  \
        __VA_ARGS__;                   \
        pb::post_launch((ctx), (kid)); \
    } while (0)

// ---- launch wrappers (definitions in the k_*.cu files) --------------------------------------------------------------
// out = L v (mode 0) or out = rhs - L v (mode 1).  red != 0: also reduce sum(out^2), sum(out) into d_scal[0..1].
int launch_apply(poisson_ctx* ctx, const Op& op, int kind, const double* v, const double* rhs, double* out, int mode,
                 bool use_ghost, bool reduce);
int launch_apply32(poisson_ctx* ctx, const Op& op, const float* v, const float* rhs, float* out, int mode);
// mixed path: out32 = (float)(rhs - L v) in fp64 arithmetic, sum(r^2) into d_scal[0]
int launch_residual_to32(poisson_ctx* ctx, const Op& op, const double* v, const double* rhs, float* out32,
                         bool use_ghost);
int launch_rbsor(poisson_ctx* ctx, const Op& op, int kind, double* phi, const double* rhs, double omega, int nsweeps,
                 bool use_ghost);
int launch_rbsor32(poisson_ctx* ctx, const Op& op, float* phi, const float* rhs, float omega, int nsweeps);

// Krylov passes
int launch_krylov_init(poisson_ctx* ctx, const double* x, const double* rhs, double* r, bool bicg, double* r0hat);
int launch_cg_passA(poisson_ctx* ctx, const double* r, const double* p_old, double* p_new, double* q, double* x);
int launch_cg_passB(poisson_ctx* ctx, double* r, const double* q);
int launch_cg_final(poisson_ctx* ctx, double* x, const double* p_last);
int launch_sub_mean(poisson_ctx* ctx, double* x);
int launch_bicg_pass1(poisson_ctx* ctx, const double* r, const double* p_old, const double* v_old, const double* r0,
                      double* p_new, double* v_new);
int launch_bicg_pass2(poisson_ctx* ctx, const double* r, const double* v, double* s, double* t);
int launch_bicg_pass3(poisson_ctx* ctx, double* x, const double* p, const double* s, const double* t,
                      const double* r0, double* r);

// Fused red-black sweeps (k_sor_fused.cu): both colours (or two sweeps) per HBM pass, ping-pong through tmp
bool sor_fused_ok(const poisson_ctx* ctx, const Op& op);
// result == nullptr: the sweeps end in phi (copy back if needed); else *result = the buffer (phi or tmp) that holds them
int sor_fused(poisson_ctx* ctx, const Op& op, double* phi, double* tmp, const double* rhs, double omega, int nsweeps,
              bool ug, double** result = nullptr);
int sor_fused32(poisson_ctx* ctx, const Op& op, float* phi, float* tmp, const float* rhs, float omega, int nsweeps,
                float** result = nullptr);
// V-cycle smoothing: nsweeps sweeps of the field in *cur (one of the level's two buffers a, b); *cur then points at the
// buffer that holds the result — never a copy back
int launch_rbsor_pp(poisson_ctx* ctx, const Op& op, double** cur, double* a, double* b, const double* rhs, double omega,
                    int nsweeps, bool ug);
int launch_rbsor_pp32(poisson_ctx* ctx, const Op& op, float** cur, float* a, float* b, const float* rhs, float omega,
                      int nsweeps);
void* sor_scratch(poisson_ctx* ctx, size_t bytes);  // nullptr on OOM
int sor_fused_seq(poisson_ctx* ctx, const Op& op, double* phi, double* tmp, const double* rhs, const double* omegas,
                  int nsweeps, bool ug, double** result);
int sor_fused_precond(poisson_ctx* ctx, const Op& op, const double* zin, double* zout, const double* f, bool symmetric,
                      bool with_rz);
int launch_rbsor_half(poisson_ctx* ctx, const Op& op, int kind, double* phi, const double* rhs, double omega, int colour,
                      bool ug, int kid);
int launch_rbsor_seq(poisson_ctx* ctx, const Op& op, int kind, double* phi, const double* rhs, const double* omegas,
                     int nsweeps, bool ug);
int launch_rbsor_local(poisson_ctx* ctx, const Op& op, int kind, double* phi, const double* rhs, const double* d_rj,
                       double* d_om, int nsweeps, int start_n, bool ug);
int launch_pcg_dot(poisson_ctx* ctx, const double* r, const double* z);
// BiCGSTAB right-preconditioned by the Gauss-Seidel sweep of Eq. 10: the pieces between the preconditioner solves
int launch_gsb_p(poisson_ctx* ctx, const double* r, double* p, const double* v, double* r0);
int launch_gsb_s(poisson_ctx* ctx, const double* r, const double* v, double* s);
int launch_gsb_matvec(poisson_ctx* ctx, int which, const double* in, double* out, const double* other);
int launch_gsb_update(poisson_ctx* ctx, double* x, const double* ph, const double* sh, const double* s, const double* t,
                      const double* r0, double* r);

// Lean 7-point apply / residual for non-periodic Cartesian grids (k_apply7.cu), fp64 and fp32
bool apply7_ok(const poisson_ctx* ctx, const Op& op);
int apply7(poisson_ctx* ctx, const Op& op, const double* v, const double* rhs, double* out, float* out32, int mode,
           bool ug, bool reduce);
int apply7_32(poisson_ctx* ctx, const Op& op, const float* v, const float* rhs, float* out, int mode);

// Fused residual + restriction (k_resid_restrict.cu): f_c = R (rhs - L phi) without storing the fine residual
bool resid_restrict_ok(const poisson_ctx* ctx, const Op& fine, const Op& coarse);
int resid_restrict(poisson_ctx* ctx, const Op& fine, const Op& coarse, const double* phi, const double* rhs, double* fc,
                   bool ug);
int resid_restrict32(poisson_ctx* ctx, const Op& fine, const Op& coarse, const float* phi, const float* rhs, float* fc);

// 7-point apply / residual with planes staged by bulk async copies (k_apply_bulk.cu), fp64
bool apply_bulk_ok(const poisson_ctx* ctx, const Op& op);
int apply_bulk(poisson_ctx* ctx, const Op& op, const double* v, const double* rhs, double* out, float* out32, int mode,
               bool ug, bool reduce);

// Plane-pipeline versions (k_plane.cu) for pair-aligned grids; same results, bit for bit
int plane_apply(poisson_ctx* ctx, const Op& op, int kind, const double* v, const double* rhs, double* out,
                float* out32, int mode, bool ug, bool reduce);
int plane_krylov_init(poisson_ctx* ctx, const double* x, const double* rhs, double* r, double* r0hat);
int plane_cg_passA(poisson_ctx* ctx, const double* r, const double* p_old, double* p_new, double* q, double* x);
int plane_bicg_pass1(poisson_ctx* ctx, const double* r, const double* p_old, const double* v_old, const double* r0,
                     double* p_new, double* v_new);
int plane_bicg_pass2(poisson_ctx* ctx, const double* r, const double* v, double* s, double* t);
bool plane_ok(const poisson_ctx* ctx, const Op& op);

// Multigrid transfer
int launch_restrict(poisson_ctx* ctx, const Op& fine, const Op& coarse, const double* r, double* fc, int restriction);
int launch_restrict32(poisson_ctx* ctx, const Op& fine, const Op& coarse, const float* r, float* fc, int restriction);
int launch_prolong_add(poisson_ctx* ctx, const Op& fine, const Op& coarse, const double* ec, double* phi);
int launch_prolong_add32(poisson_ctx* ctx, const Op& fine, const Op& coarse, const float* ec, float* phi);
int launch_add32to64(poisson_ctx* ctx, size_t n, const float* e, double* phi);
int launch_coarse_solve(poisson_ctx* ctx, const Op& op, double* phi, const double* rhs, double omega, int nsweeps);
int launch_coarse_solve32(poisson_ctx* ctx, const Op& op, float* phi, const float* rhs, float omega, int nsweeps);
// levels first..last (nlev operators) of the V-cycle in one CTA's shared memory; UNSUPPORTED when they do not fit
int launch_mg_bottom(poisson_ctx* ctx, const Op* ops, int nlev, double* phi, const double* rhs, int nu1, int nu2,
                     int csweeps, double omega_c);
int launch_mg_bottom32(poisson_ctx* ctx, const Op* ops, int nlev, float* phi, const float* rhs, int nu1, int nu2,
                       int csweeps, double omega_c);

// The paper's own multigrid (k_mgv.cu): SPAI smoother, vertex-centred transfers, Galerkin stencils, CG coarsest
int mgv_spai_smooth(poisson_ctx* ctx, double* phi, const double* rhs, const double* spai, int nsteps);
int mgv_vcycles(poisson_ctx* ctx, double* phi, const double* rhs, int nu1, int nu2, int coarsest_n, const double* spai,
                double cg_rtol, int storage_f32, int ncycles, const std::function<int(int)>& record);
void mgv_destroy(poisson_ctx* ctx);
int mgv_residual_norm2(poisson_ctx* ctx, const double* phi, const double* rhs, int coarsest_n, int storage_f32);
int mgv_compact_rhs(poisson_ctx* ctx, const double* f_ext, double* out);

// Multipole
int launch_moments(poisson_ctx* ctx, const double* rho, int lmax, double* d_q, bool inner);
int launch_ghost_eval(poisson_ctx* ctx, const double* d_q, const double* d_qbar, double G, int lmax);

}  // namespace pb
