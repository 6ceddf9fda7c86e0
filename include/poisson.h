/* poisson.h — C ABI of the B200-native matrix-free Poisson solvers (hot path of arxiv/paper_2605_03563,
 * "Iterative Poisson Solvers for Self-gravity with the GPU Code Astaroth").
 *
 * The library solves  L_h phi = rhs  on a 3-D structured grid, where L_h is the finite-difference Laplacian
 * (Eq. 1-2) and rhs = 4 pi G rho for self-gravity.  Every step of every call runs in hand-written
 * CUDA kernels for sm_100a; there is no CPU fallback.  All work is enqueued on the stream given at create time.
 *
 * Conventions (DESIGN.md "Boundary" and readings C0):
 *  - Unknowns: shape[0] x shape[1] x shape[2] points, index (i,j,k), axis 0 fastest; arrays are contiguous,
 *    exactly shape[0]*shape[1]*shape[2] elements, 16-byte aligned.  Cartesian: axis 0,1,2 = x,y,z and point
 *    coordinate = origin[a] + i*spacing[a].  Spherical: axis 0,1,2 = r,theta,phi given by cell edges.
 *  - `d_*` arguments are DEVICE pointers owned by the caller; `h_*` arguments are HOST pointers.
 *  - Faces: 0 = axis0 low, 1 = axis0 high, 2 = axis1 low, 3 = axis1 high, 4 = axis2 low, 5 = axis2 high.
 *  - Ghost zones ("the multipole expansion of Phi in the ghost zones") are kept in the handle as six
 *    face arrays with R = stencil radius layers (R = 1 for order 2, 3 for order 6).  Face on axis a, layer l
 *    (distance l+1 outside the domain): index (l*n[a2] + q2)*n[a1] + q1 with (a1,a2) the other two axes in
 *    increasing order, q1 fastest.  Only face ghosts exist: a star stencil never reads edge or corner ghosts.
 *  - L_h is the Laplacian itself (negative definite); the SPD matrix "A" of the paper is -L_h.
 *  - Return value: 0 OK; >0 soft status (1 NOT_CONVERGED: "warning ... if the threshold is not achieved
 *    within a maximum number of iterations"; 2 BREAKDOWN); <0 error.  No exceptions, no aborts.
 *  - Calls that return host scalars synchronise the stream; the others only enqueue work.
 *  - A non-zero initial guess in d_phi is honoured (warm start).
 */
#ifndef POISSON_B200_H
#define POISSON_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct poisson_ctx* poisson_t; /* opaque; owns scratch vectors, MG levels, face-ghost arrays */

enum { POISSON_CARTESIAN = 0, POISSON_SPHERICAL = 1 };
enum {
    POISSON_BC_DIRICHLET_GHOST = 0, /* ghost values supplied by poisson_multipole_bc or poisson_set_ghost_faces */
    POISSON_BC_PERIODIC = 1,
    POISSON_BC_NEUMANN0 = 2,        /* zero normal flux through the face */
    POISSON_BC_AXIS = 3             /* spherical theta faces on the polar axis: zero face area */
};
enum { POISSON_F64 = 0, POISSON_MIXED = 1 };
enum {
    POISSON_OK = 0,
    POISSON_NOT_CONVERGED = 1,
    POISSON_BREAKDOWN = 2,
    POISSON_INVALID_ARG = -1,
    POISSON_UNSUPPORTED = -2,
    POISSON_CUDA_ERROR = -3,
    POISSON_OUT_OF_MEMORY = -4
};
/* options for poisson_set_option */
enum {
    POISSON_OPT_KERNEL_PATH = 0,   /* 0 auto, 1 force the generic (direct global load) kernels, 2 force the
                                      plane-pipeline (bulk-copy staged) kernels where they exist */
    POISSON_OPT_RESTRICTION = 1,   /* V-cycle restriction: 0 = (1/8)[1 3 3 1]^3 (transpose of trilinear),
                                      1 = mean of the 8 children (reading C7) */
    POISSON_OPT_POLL_INTERVAL = 2, /* Krylov solvers poll the device convergence flag every this many iterations */
    POISSON_OPT_JACOBI = 3,        /* BiCGSTAB right preconditioner: 1 (default) Jacobi scaling (reading C10),
                                      0 none, 2 the multi-colour Gauss-Seidel preconditioner of PAPER.md:107-123
                                      Eq. 10 (p^ = B^-1 p by one red-black Gauss-Seidel sweep from zero; radius-1
                                      stencils, Cartesian or spherical) */
    POISSON_OPT_RECORD_HISTORY = 4,/* 1: record ||r_k||/||r_0|| per Krylov iteration for poisson_get_history */
    POISSON_OPT_SOR_HALFSTEPS = 6, /* red-black colour half-steps fused per HBM pass (temporal blocking): 2 = one
                                      full sweep per pass, 4 = two sweeps per pass, 0 = automatic (default: 4 on
                                      grids of >= 2^21 points, else 2); the results do not depend on it */
    POISSON_OPT_FUSED_RESTRICT = 7,/* V-cycle: residual + restriction fused into one pass over the level (no fine residual
                                      in memory): 0 = automatic (fp32 levels of the mixed cycle, fp64 levels below 2^21 points),
                                      1 = always, 2 = never;
                                      the results do not depend on it */
    POISSON_OPT_TIME_KERNELS = 5,  /* bracket every launch of one kernel class (0..poisson_kernel_classes()-1) with
                                      CUDA events on the handle's stream; -2 = every class, -1 = off (default) */
    /* tuning overrides for measurements; the results do not depend on them; -1 = automatic (default) */
    POISSON_OPT_TILE_CFG = 9,      /* index of the compiled tile configuration of the fused SOR / lean apply kernels */
    POISSON_OPT_PLANE_SPLIT = 10,  /* plane engine: 1 = always split the (tile, plane) items linearly, 0 = never */
    POISSON_OPT_APPLY_BULK = 11,   /* TMA-staged 7-point apply: 1 = whenever eligible, 0 = never */
    POISSON_OPT_COMPACT_ORDER = 12,/* level-0 discretisation of poisson_spai_smooth / poisson_mgv_vcycle: 2 (default; the
                                      handle's 7-point operator with its ghost faces), 4 or 6 = the compact radius-1
                                      19- / 27-point discretisations of PAPER.md:172 (see poisson_compact_rhs) */
    /* floating-point options (poisson_set_option_f64) */
    POISSON_OPT_BICG_RESTART_EPS = 8 /* BiCGSTAB near-breakdown restart threshold on |r0^.r| / (|r0^| |r|); default
                                      1e-12 (reading C4), 0 = never restart */
};

/* Create a solver context for one grid + operator ("uniform and nonuniform grids in spherical and
 * Cartesian coordinates"; 41-57).
 *   shape[3], spacing[3], origin[3]: Cartesian geometry (spacing/origin ignored for spherical).
 *   edges: NULL for Cartesian; for spherical three HOST arrays of shape[a]+1 strictly increasing cell-edge
 *          coordinates (r, theta, phi), r_in > 0, theta within [0, pi].  Only r may be nonuniform (radial centres are
 *          the geometric means of the edges); theta and phi edges must be uniform (UNSUPPORTED
 *          otherwise) and a BC_AXIS face must lie on the polar axis (theta edge 0 or pi).
 *   coord_system: POISSON_CARTESIAN | POISSON_SPHERICAL.
 *   stencil_order: 2 (7-point, radius 1) or 6 (19-point star, radius 3; Cartesian only) — PAPER.md:172.
 *   bc[6]: boundary type per face.
 *   cuda_stream: a cudaStream_t (NULL = default stream).
 * The handle is bound to the CUDA device that is current at create time (every call runs there whatever the
 * caller's current device is) and must not be used from two threads at once.
 * Errors: INVALID_ARG (bad shape/order/bc/edges), UNSUPPORTED, OUT_OF_MEMORY, CUDA_ERROR. */
int poisson_create(poisson_t* out, const int shape[3], const double spacing[3], const double origin[3],
                   const double* const edges[3], int coord_system, int stencil_order, const int bc[6],
                   void* cuda_stream);
int poisson_destroy(poisson_t h);
/* Static string describing the last error of this handle (or of create when h is NULL). */
const char* poisson_last_error(poisson_t h);
int poisson_set_option(poisson_t h, int option, int value);
int poisson_set_option_f64(poisson_t h, int option, double value);

/* out = L_h phi with the handle's ghost values on Dirichlet faces.  d_out must not alias d_phi. */
int poisson_apply_laplacian(poisson_t h, const double* d_phi, double* d_out);

/* nsweeps full red-black SOR sweeps in place: red = (i+j+k) even first, then black; omega = 1 is Gauss-Seidel
 * (PAPER.md:59-63).  h_resnorm (nullable) receives ||rhs - L phi||_2 after the last sweep. */
int poisson_rbsor_sweep(poisson_t h, double* d_phi, const double* d_rhs, double omega, int nsweeps,
                        double* h_resnorm);

/* Red-black SOR with the Chebyshev-accelerated sequence of PAPER.md:81-88 Eq. 6 instead of a fixed omega:
 *   omega_0 = 1, omega_1 = 1/(1 - rJ^2/2), omega_{n+1} = 1/(1 - rJ^2 omega_n/4)  ->  omega_opt of Eq. 3,
 * one member per colour half-sweep (Press et al. Eq. 20.5.30, as cited there): half-sweep m = 0, 1, 2, ... (red, black,
 * red, ...) uses omega_{m + start_n}; start_n = 1 is the variant the paper uses ("starting from n = 1").
 * r_jacobi: spectral radius of the Jacobi iteration; <= 0 selects Eq. 4 with N = n + 1 intervals (Cartesian grids).
 * Each call starts the sequence afresh.  h_resnorm as in poisson_rbsor_sweep. */
int poisson_rbsor_cheby(poisson_t h, double* d_phi, const double* d_rhs, double r_jacobi, int nsweeps, int start_n,
                        double* h_resnorm);

/* The position-dependent variant for spherical (and nonuniform) grids, Eq. 7: every point (i,j) runs
 * the sequence of Eq. 6 with its own local Jacobi radius
 *   rJ(i,j) = [cos(pi/Nr) dr_i^-2 + cos(pi/Nth) (r_i dth)^-2 + cos(pi/Nph) (r_i sin th_j dph)^-2] / [sum of the three],
 * advanced after every colour half-sweep.  On a Cartesian grid rJ is that of Eq. 4 everywhere. */
int poisson_rbsor_local(poisson_t h, double* d_phi, const double* d_rhs, int nsweeps, int start_n, double* h_resnorm);

/* Conjugate gradient preconditioned by the multi-colour Gauss-Seidel preconditioner of PAPER.md:107-123 Eq. 9-10
 * (two colours for the 7-point operator): z = M^-1 r is one red-black Gauss-Seidel sweep on L_h z = r from z = 0 —
 * the block lower-triangular solve B^-1 of Eq. 10 — followed by a second red half-sweep, which makes M the symmetric
 * Gauss-Seidel splitting a CG iteration needs (reading C15); Saad Alg. 9.1.  The sweep is ONE fused pass
 * over HBM.  Same stopping rule (on the unpreconditioned residual), statuses and outputs as poisson_cg_solve.
 * Cartesian 7-point operator, non-periodic faces. */
int poisson_pcg_solve(poisson_t h, double* d_phi, const double* d_rhs, double rtol, int max_iter, int fixed_iters,
                      int* iters, double* relres);

/* Unpreconditioned conjugate gradient on A = -L_h (Saad Alg. 6.18), fused as
 * {p-update + matvec + p.Ap} and {r-update + ||r||^2}.  Stops when ||r_k|| <= rtol ||r_0|| (r_0 from the initial
 * guess) or after max_iter iterations (-> NOT_CONVERGED).  fixed_iters > 0 runs exactly that many iterations.
 * For an all-periodic grid the constant null space is projected out every iteration and phi is returned with
 * zero mean (reading C3).  iters / relres are nullable host outputs. */
int poisson_cg_solve(poisson_t h, double* d_phi, const double* d_rhs, double rtol, int max_iter, int fixed_iters,
                     int* iters, double* relres);

/* BiCGSTAB (Saad Alg. 7.7) with right Jacobi scaling, for the nonsymmetric spherical operator;
 * same stopping rule.  Near-breakdown restart (reading C4): when |r0^.r| <= 1e-12 |r0^| |r| at the beta
 * step the shadow residual is replaced by r (rho = r.r, beta = 0); POISSON_OPT_BICG_RESTART_EPS overrides the
 * threshold, 0 disables the rule.  When the recurrence's residual meets rtol the
 * true residual rhs - L phi is recomputed: OK (and *relres the true figure) only if it meets rtol as well, otherwise
 * the iteration carries on from it; NOT_CONVERGED also after 30 such checks have failed (rtol below the attainable
 * accuracy).  fixed_iters > 0 runs exactly that many iterations without any check.
 * BREAKDOWN when rho, omega or r0^.v vanish or turn non-finite. */
int poisson_bicgstab_solve(poisson_t h, double* d_phi, const double* d_rhs, double rtol, int max_iter,
                           int fixed_iters, int* iters, double* relres);

/* ncycles geometric-multigrid V-cycles (Eq. 11-12) in the CELL-CENTRED variant BASELINE.json config 3
 * fixes (reading C7) — not the paper's own vertex-centred Eq. 13-14 operators, for which see
 * poisson_mgv_vcycle below: nu1/nu2 red-black Gauss-Seidel sweeps, restriction = transpose of trilinear
 * (1/8)[1 3 3 1]^3 ("full weighting" for cell centres; P = 8 R^T), trilinear prolongation, 7-point
 * rediscretisation on 2:1 coarsened cells down to coarsest_n points per axis, coarsest level by coarsest_sweeps SOR
 * sweeps at omega_opt of Eq. 3-4.  precision = POISSON_F64 or POISSON_MIXED (fp64 residual
 * and correction, fp32 error-equation cycle).  Cartesian, order 2, Dirichlet faces only.
 * h_resnorms (nullable, ncycles+1): ||rhs - L phi||_2 before the first and after every cycle. */
int poisson_mg_vcycle(poisson_t h, double* d_phi, const double* d_rhs, int nu1, int nu2, int coarsest_n,
                      int coarsest_sweeps, int precision, int ncycles, double* h_resnorms);

/* The paper's own multigrid ingredients, for vertex-centred grids of 2^N k - 1 points per
 * axis with isotropic spacing and Dirichlet (ghost) faces, 7-point operator.
 *
 * poisson_spai_smooth: nsteps steps of the SPAI smoother  x <- x + omega M (b - A x)  (Eq. 15) on
 *   A = -L_h, b = -rhs, with M = h^2 {alpha at the centre, beta on the 6 faces, gamma on the 12 edges, delta on the
 *   8 corners} (Eq. 16).  spai = {omega, alpha, beta, gamma, delta}; NULL = Table 1, order 2:
 *   {1.3699, 0.1432, 0.0284, 0.0081, 0.0025}.  Works on any shape (it is level 0 of the hierarchy below).
 *
 * poisson_mgv_vcycle: ncycles V-cycles (Eq. 11-12) with nu1/nu2 SPAI steps, full-weighting restriction
 *   R = (1/4 [1 2 1])^(x)3 (Eq. 13), prolongation P = 8 R^T (trilinear, "c adjusted such that P preserves constant
 *   functions"), Galerkin coarse operators R A P (Eq. 14; reading C13 on the constant), coarsening while
 *   every axis is odd and the coarse level keeps >= coarsest_n points per axis (coarsest_n = 3 gives the paper's seven
 *   coarse levels at 511^3), coarsest level by CG to relative residual cg_rtol (at most 15^3 unknowns).
 *   precision = POISSON_F64, or POISSON_MIXED = the paper's mixed precision: all coarse-level data stored
 *   in fp32, all arithmetic in fp64.  UNSUPPORTED when the grid admits no coarse level.
 *   h_resnorms (nullable, ncycles+1): ||rhs - L phi||_2 before the first and after every cycle (for Eq. 18). */
int poisson_spai_smooth(poisson_t h, double* d_phi, const double* d_rhs, const double* spai, int nsteps);
/* Compact discretisations (radius-1 stencils of 4th and, on isotropic grids, 6th order; the paper
 * prints no coefficients — DESIGN.md reading C19).  With POISSON_OPT_COMPACT_ORDER = 4 or 6, poisson_spai_smooth and
 * poisson_mgv_vcycle work on L_h phi = d_rhs with
 *   L_h = (S1 + S2/6 [+ S3/30]) / h^2,  S1 = sum_a d_a^2, S2 = sum_{a<b} d_a^2 d_b^2, S3 = d_x^2 d_y^2 d_z^2
 * (stencil weights (-24, 2, 1, 0)/6h^2 and (-128, 14, 3, 1)/30h^2 on centre, faces, edges, corners), ZERO values on the
 * boundary vertices (the handle's ghost faces must be unset: fold boundary data into the right-hand side), the SPAI
 * rows 4 / 6 of Table 1 by default (delta of row 6: 0.0150, reading C20), and d_rhs = the TRANSFORMED right-hand side
 * that poisson_compact_rhs computes for lap u = f:
 *   order 4: f + S1 f / 12;   order 6: f + S1 f / 12 - (sum_a d_a^4 f) / 240 + S2 f / 90;   order 2: f.
 * d_f_ext: DEVICE array of (n0+4)(n1+4)(n2+4) doubles, f on the grid extended by two layers per side (x fastest);
 * d_out: DEVICE array of n0 n1 n2 doubles.  The residual norms poisson_mgv_vcycle reports are then those of this
 * operator.  Errors: INVALID_ARG, UNSUPPORTED (non-Cartesian, anisotropic, ghosts set). */
int poisson_compact_rhs(poisson_t h, const double* d_f_ext, double* d_out);
int poisson_mgv_vcycle(poisson_t h, double* d_phi, const double* d_rhs, int nu1, int nu2, int coarsest_n,
                       const double* spai, double cg_rtol, int precision, int ncycles, double* h_resnorms);

/* Multipole-expansion open boundary (Eq. 19-20): moments q_lm = sum_cells rho r^l S_lm dV for
 * 0 <= l <= lmax (<= 8), |m| <= l in one fused reduction over d_rho, then Phi_ghost = -G sum q_lm S_lm / r^(l+1)
 * written into the handle's ghost faces (all Dirichlet faces in Cartesian, the outer radial shell in spherical).
 * Expansion centre = coordinate origin.  h_moments (nullable): (lmax+1)^2 values, index l*l + l + m, cosine
 * harmonics m >= 0, sine harmonics m < 0. */
int poisson_multipole_bc(poisson_t h, const double* d_rho, double G, int lmax, double* h_moments);
/* Spherical grids whose inner radial face (face 0) is POISSON_BC_DIRICHLET_GHOST: poisson_multipole_bc also forms the
 * inner multipoles qbar_lm = sum_cells rho r^-(l+1) S_lm dV and writes Phi = -G sum qbar_lm r^l S_lm into the inner
 * ghost shell (Eq. 21-22).  This call returns those moments, (lmax+1)^2 values, same indexing. */
int poisson_multipole_inner_moments(poisson_t h, double* h_qbar, int lmax);

/* Helpers. */
/* Copy caller-supplied ghost values (DEVICE arrays, layout above; NULL entries = leave that face) into the handle. */
int poisson_set_ghost_faces(poisson_t h, const double* const d_faces[6]);
/* Copy the handle's ghost face f into a DEVICE array of poisson_face_len(h,f) doubles. */
int poisson_get_ghost_face(poisson_t h, int face, double* d_out);
long poisson_face_len(poisson_t h, int face);
/* ||rhs - L phi||_2 with the handle's ghosts. */
int poisson_residual_norm(poisson_t h, const double* d_phi, const double* d_rhs, double* h_norm);
/* The same norm for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): no handle, and NO cudaMalloc / cudaFree / allocating library call inside.  L is the Cartesian 7-point
 * Laplacian (Eq. 1) of the grid `shape` (x fastest) with spacing `spacing`, phi = 0 outside the grid
 * (what a fresh handle with six DIRICHLET_GHOST faces computes).  d_phi, d_rhs: DEVICE arrays of shape[0] shape[1]
 * shape[2] doubles on the current device (the caller's; not modified); d_norm: DEVICE double, receives the norm when
 * the work queued on `cuda_stream` (a cudaStream_t, NULL = default stream) has run — the call does not synchronise.
 * The block partial sums live in a static 256 KiB device array of the library (every GPU that loads the library holds
 * it until exit): ceil(shape[0]/32) ceil(shape[1]/8) ceil(shape[2]/16) must not exceed 32768 (512^3 points fit) —
 * larger grids return UNSUPPORTED.  All calls on a device share that array: calls that overlap on the GPU (different
 * streams, two threads) race; calls queued on one stream do not.  The first call on a device resolves the array's
 * address (make it before starting a capture).  Errors: INVALID_ARG (NULL / host / other-device pointers, bad shape),
 * UNSUPPORTED, CUDA_ERROR; poisson_residual_norm_static_error() describes the calling thread's last one. */
int poisson_residual_norm_static(const int shape[3], const double spacing[3], const double* d_phi,
                                 const double* d_rhs, double* d_norm, void* cuda_stream);
const char* poisson_residual_norm_static_error(void);
/* Relative residual history of the last Krylov solve (needs POISSON_OPT_RECORD_HISTORY): h_out[0..n-1]. */
int poisson_get_history(poisson_t h, double* h_out, int n);
/* Near-breakdown restarts taken and true-residual confirmations that failed in the last BiCGSTAB solve (nullable). */
int poisson_bicgstab_stats(poisson_t h, int* restarts, int* confirm_failed);
/* Number of kernels this handle has launched so far (bench bookkeeping). */
long poisson_kernel_launches(poisson_t h);

/* Kernel-class bookkeeping for the bench: the classes are the rows of the hot path
 * (apply, rbsor, cg_pass_a, ...).  poisson_kernel_time synchronises the stream and returns the summed CUDA-event
 * duration (ms) and the number of timed launches of one class since the last reset. */
int poisson_kernel_classes(void);
const char* poisson_kernel_name(int kernel_class);
long poisson_kernel_class_launches(poisson_t h, int kernel_class);
int poisson_kernel_time(poisson_t h, int kernel_class, double* h_ms_total, long* h_count);
int poisson_reset_kernel_times(poisson_t h);

/* End-to-end variants with HOST buffers (all h_* below, including the fields): host->device copy of the inputs on
 * the handle's stream, the device entry point of the same name, device->host copy of the result, synchronise.
 * Same arguments, statuses and errors as the device versions.  Pinned host memory gives full PCIe speed. */
int poisson_apply_laplacian_host(poisson_t h, const double* h_phi, double* h_out);
int poisson_rbsor_sweep_host(poisson_t h, double* h_phi, const double* h_rhs, double omega, int nsweeps,
                             double* h_resnorm);
int poisson_cg_solve_host(poisson_t h, double* h_phi, const double* h_rhs, double rtol, int max_iter,
                          int fixed_iters, int* iters, double* relres);
int poisson_bicgstab_solve_host(poisson_t h, double* h_phi, const double* h_rhs, double rtol, int max_iter,
                                int fixed_iters, int* iters, double* relres);
int poisson_mg_vcycle_host(poisson_t h, double* h_phi, const double* h_rhs, int nu1, int nu2, int coarsest_n,
                           int coarsest_sweeps, int precision, int ncycles, double* h_resnorms);
int poisson_multipole_bc_host(poisson_t h, const double* h_rho, double G, int lmax, double* h_moments);
int poisson_mgv_vcycle_host(poisson_t h, double* h_phi, const double* h_rhs, int nu1, int nu2, int coarsest_n,
                            const double* spai, double cg_rtol, int precision, int ncycles, double* h_resnorms);

#ifdef __cplusplus
}
#endif
#endif /* POISSON_B200_H */
