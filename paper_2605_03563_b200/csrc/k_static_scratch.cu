// k_static_scratch.cu — poisson_residual_norm_static: ||rhs - L phi||_2 (Eq. 1, 55) through an entry
// point that allocates NOTHING — for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
// loops, harnesses that forbid it).  The handle-based poisson_residual_norm keeps its block partials in memory that
// poisson_create cudaMalloc'ed; here they live in a file-scope `static __device__` array of kStaticMaxBlocks doubles
// (256 KiB, held by every GPU that loads the library until the process exits).
//
// The array's name is, in host code, a host-side stand-in and NOT a device address: handing it to a kernel would fault
// (or silently use host memory where the GPU can reach it).  static_scratch() below asks the runtime for the device
// address — once per device, with that device current, return code checked — and the kernels get that pointer.
//
// Sharing: every call on a device uses the same array, which keeps the last call's contents.  Nothing in it has to
// start at zero: a call overwrites partials 0 .. nblk-1 before its second kernel reads exactly those.  Two calls that
// overlap on the GPU (different streams, or two host threads) race on it; calls on one stream are ordered and safe.
#include <cuda_runtime.h>

#include <cstdio>
#include <mutex>

#include "../../include/poisson.h"

namespace pbs {

constexpr int kTX = 32, kTY = 8, kKC = 16;   // a block owns 32 x 8 columns and marches 16 planes
constexpr int kStaticMaxBlocks = 32768;       // 512^3 = 16 x 64 x 32 blocks of 32 x 8 x 16 points
constexpr int kMaxDevices = 64;

static __device__ __align__(256) double g_static_scratch[kStaticMaxBlocks];

static thread_local char g_err[256] = "";
static int fail(int code, const char* msg) {
    std::snprintf(g_err, sizeof(g_err), "%s", msg);
    return code;
}
static int fail_cuda(cudaError_t e, const char* what) {
    std::snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
    return POISSON_CUDA_ERROR;
}

// Device address of g_static_scratch on the CURRENT device (resolved once per device).
static int static_scratch(double** out) {
    static std::mutex mu;
    static double* ptr[kMaxDevices] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail_cuda(e, "cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) return fail(POISSON_UNSUPPORTED, "device ordinal beyond 63");
    const std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        double* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
        if (e != cudaSuccess || !p) return fail_cuda(e, "cudaGetSymbolAddress(g_static_scratch)");
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return POISSON_OK;
}

__device__ __forceinline__ double warp_sum(double x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

// partials[block] = sum over the block's points of (rhs - L phi)^2, L = 7-point Laplacian, phi = 0 outside the grid.
// Same order of operations per point as stencil.cuh row_apply<KIND_CART2> (x pair, fma y pair, fma z pair, fma centre).
__global__ void __launch_bounds__(kTX * kTY)
    k_resid_partials(int n0, int n1, int n2, double c0, double c1, double c2, const double* __restrict__ phi,
                     const double* __restrict__ rhs, double* __restrict__ partials) {
    __shared__ double sm[kTX * kTY / 32];
    const int i = blockIdx.x * kTX + threadIdx.x, j = blockIdx.y * kTY + threadIdx.y;
    const int k0 = blockIdx.z * kKC, k1 = min(k0 + kKC, n2);
    const size_t plane = (size_t)n0 * n1;
    const double d = 2.0 * ((c0 + c1) + c2);
    double s2 = 0.0;
    if (i < n0 && j < n1) {
        const double* p = phi + (size_t)k0 * plane + (size_t)j * n0 + i;
        const double* f = rhs + (size_t)k0 * plane + (size_t)j * n0 + i;
        double zm = k0 > 0 ? p[-(ptrdiff_t)plane] : 0.0, c = p[0];
        for (int k = k0; k < k1; ++k) {
            const double zp = k + 1 < n2 ? p[plane] : 0.0;
            const double xm = i > 0 ? p[-1] : 0.0, xp = i + 1 < n0 ? p[1] : 0.0;
            const double ym = j > 0 ? p[-n0] : 0.0, yp = j + 1 < n1 ? p[n0] : 0.0;
            double s = (xm + xp) * c0;
            s = fma(ym + yp, c1, s);
            s = fma(zm + zp, c2, s);
            const double r = f[0] - fma(-d, c, s);
            s2 = fma(r, r, s2);
            zm = c;
            c = zp;
            p += plane;
            f += plane;
        }
    }
    const int tid = threadIdx.y * kTX + threadIdx.x;
    s2 = warp_sum(s2);
    if ((tid & 31) == 0) sm[tid >> 5] = s2;
    __syncthreads();
    if (tid < 32) {
        double x = tid < kTX * kTY / 32 ? sm[tid] : 0.0;
        x = warp_sum(x);
        if (tid == 0) partials[(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x] = x;
    }
}

// norm[0] = sqrt(sum of partials[0 .. nblk-1]), added in a fixed order (deterministic for a given grid shape).
__global__ void __launch_bounds__(1024) k_resid_finish(int nblk, const double* __restrict__ partials,
                                                        double* __restrict__ norm) {
    __shared__ double sm[32];
    double acc = 0.0;
    for (int b = threadIdx.x; b < nblk; b += 1024) acc += partials[b];
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x < 32) {
        const double x = warp_sum(sm[threadIdx.x]);
        if (threadIdx.x == 0) norm[0] = sqrt(x);
    }
}

// a device (or managed) pointer of the current device?
static bool on_device(const void* p, int dev) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) && a.device == dev;
}

}  // namespace pbs

extern "C" const char* poisson_residual_norm_static_error(void) { return pbs::g_err; }

extern "C" int poisson_residual_norm_static(const int shape[3], const double spacing[3], const double* d_phi,
                                            const double* d_rhs, double* d_norm, void* cuda_stream) {
    using namespace pbs;
    if (!shape || !spacing || !d_phi || !d_rhs || !d_norm) return fail(POISSON_INVALID_ARG, "bad pointers");
    for (int a = 0; a < 3; ++a)
        if (shape[a] < 1 || !(spacing[a] > 0.0)) return fail(POISSON_INVALID_ARG, "bad shape or spacing");
    const long gx = (shape[0] + kTX - 1) / kTX, gy = (shape[1] + kTY - 1) / kTY, gz = (shape[2] + kKC - 1) / kKC;
    if (gx * gy * gz > kStaticMaxBlocks || gy > 65535 || gz > 65535) {
        std::snprintf(g_err, sizeof(g_err),
                      "grid %d x %d x %d needs %ld blocks of 32 x 8 x 16 points; the static scratch array holds %d "
                      "(up to 512^3 points): use poisson_residual_norm",
                      shape[0], shape[1], shape[2], gx * gy * gz, kStaticMaxBlocks);
        return POISSON_UNSUPPORTED;
    }
    double* scratch = nullptr;
    const int rc = static_scratch(&scratch);
    if (rc != POISSON_OK) return rc;
    int dev = -1;
    cudaGetDevice(&dev);
    if (!on_device(d_phi, dev) || !on_device(d_rhs, dev) || !on_device(d_norm, dev))
        return fail(POISSON_INVALID_ARG, "d_phi, d_rhs and d_norm must be device memory of the current device");
    const cudaStream_t st = (cudaStream_t)cuda_stream;
    const double c0 = 1.0 / (spacing[0] * spacing[0]), c1 = 1.0 / (spacing[1] * spacing[1]),
                 c2 = 1.0 / (spacing[2] * spacing[2]);
    k_resid_partials<<<dim3((unsigned)gx, (unsigned)gy, (unsigned)gz), dim3(kTX, kTY), 0, st>>>(
        shape[0], shape[1], shape[2], c0, c1, c2, d_phi, d_rhs, scratch);
    k_resid_finish<<<1, 1024, 0, st>>>((int)(gx * gy * gz), scratch, d_norm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda(e, "kernel launch");
    return POISSON_OK;
}
