// pairq.cuh — helpers shared by the "thread owns a 16-byte pair, z register queue" kernels (k_apply7.cu,
// k_resid_restrict.cu): the pair type per precision and the diagonal of the 7-point row split into its x/y part (fixed
// per column) and its z part (per plane), in the order of operations of stencil.cuh row_diag.
#pragma once
#include "stencil.cuh"

namespace pb {

template <typename T>
struct P2T {};
template <>
struct P2T<double> {
    using type = double2;
    static __device__ __forceinline__ double2 make(double a, double b) { return make_double2(a, b); }
};
template <>
struct P2T<float> {
    using type = float2;
    static __device__ __forceinline__ float2 make(float a, float b) { return make_float2(a, b); }
};

// z part of row_diag on top of the x/y part (same order of operations as stencil.cuh row_diag)
template <typename T>
__device__ __forceinline__ T a7_diag_xy(const Op& op, int i, int j) {
    const T c0 = (T)op.c[0], c1 = (T)op.c[1], c2 = (T)op.c[2];
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
    return d;
}
template <typename T>
__device__ __forceinline__ T a7_diag_z(const Op& op, T d, int k) {
    const T c2 = (T)op.c[2], g = (T)op.gamma;
    const bool closure = op.gamma != 0.0;
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

}  // namespace pb
