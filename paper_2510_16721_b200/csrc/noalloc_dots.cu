// noalloc_dots.cu -- cfneb_band_dots_noalloc: the ten per-image dot products of K4 (kernels_neb.cu) for callers
// that must not allocate device memory.
//
// Who needs this.  The band handle of cfneb_create gets its scratch from a workspace the caller allocates.  Some
// callers have no allocator to ask: a force-field plug-in inside a host MD / optimiser code that was handed its
// arrays and nothing else; a process whose GPU memory was given away whole at start-up (a caching pool at its cap,
// a fixed MPS / MIG budget); a latency-bound loop that may not take cudaMalloc's implicit device-wide
// synchronisation.  For them the block partials of the reduction live in a file-scope `__device__` array that is
// part of this library's image: the loader places it when the library's module is loaded on a GPU, every GPU that
// loads the library keeps its own copy (kNaScratchBytes, 640 KiB) until the process exits, and this entry point
// calls no cudaMalloc, cudaFree or any library routine that allocates.  The caller passes inputs and outputs only.
//
// What it computes (Eq. 1; ref [13] via P:20).  For a band of P images of n_dof numbers each
// (generalized coordinates X, generalized forces G, FIRE velocities v; n_dof = 3 (N + 3) for the cell filter,
// Eq. 17) and every movable image p = 1..P-2 with tau+ = X_{p+1} - X_p, tau- = X_p - X_{p-1}:
//     dots[p] = { tau+.tau+, tau-.tau-, tau+.tau-, G.tau+, G.tau-, G.G, G.v, tau+.v, tau-.v, v.v }
// (the order of DOT_PP .. DOT_VV), from which the tangent, the projection, the spring term and every FIRE scalar
// follow (kernels_neb.cu, scalar_kernel).  Same two stages as K4: per-block partial sums, then one warp per image
// adds the partials in a fixed order, so the result is bitwise repeatable from call to call.
//
// Sharing.  There is ONE scratch array per GPU, shared by every call from every thread and stream.  Each call
// overwrites the partials of the images it works on before it reads them, so nothing has to start at zero and what
// an earlier call left behind is never read.  Two calls that overlap on the GPU (different streams, or different
// host threads) write the same slots and race: keep the calls on one stream, or order them with events.
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "cfneb_internal.cuh"

namespace cfn {

constexpr int kNaMaxImages = CFNEB_NOALLOC_MAX_IMAGES;  // movable + fixed images of one call
constexpr int kNaBlocks = 64;                           // partial sums per image (blocks of stage 1)
constexpr int kNaThreads = 256;
constexpr int kNaMaxDevices = 64;
constexpr size_t kNaScratchBytes = sizeof(double) * kNaMaxImages * kNaBlocks * kNDots;  // 655 360 B

// The scratch.  In HOST code this name is only a handle for the runtime (cudaGetSymbolAddress below); it is not a
// device address and must never be passed to a kernel as one.
static __device__ __align__(256) double g_na_partials[kNaMaxImages * kNaBlocks * kNDots];

// Stage 1: grid (kNaBlocks, P - 2).  Block b of image p strides over the n_dof components and leaves its ten sums
// in part[(p * kNaBlocks + b) * 10 ..]; a block with no component still writes its ten zeros.
__global__ void __launch_bounds__(kNaThreads) na_partial_kernel(const double *__restrict__ X, const double *__restrict__ G,
                                                               const double *__restrict__ v, long long n_dof,
                                                               double *__restrict__ part) {
    const int p = blockIdx.y + 1;
    const double *Xm = X + (size_t)(p - 1) * n_dof, *X0 = X + (size_t)p * n_dof, *Xp = X + (size_t)(p + 1) * n_dof;
    const double *Gp = G + (size_t)p * n_dof, *vp = v + (size_t)p * n_dof;
    __shared__ double red[32 * kNDots];
    double acc[kNDots];
#pragma unroll
    for (int q = 0; q < kNDots; ++q) acc[q] = 0.0;
    for (long long i = (long long)blockIdx.x * kNaThreads + threadIdx.x; i < n_dof; i += (long long)kNaBlocks * kNaThreads) {
        const double x0 = X0[i], tp = Xp[i] - x0, tm = x0 - Xm[i], g = Gp[i], w = vp[i];
        acc[DOT_PP] += tp * tp;
        acc[DOT_MM] += tm * tm;
        acc[DOT_PM] += tp * tm;
        acc[DOT_GP] += g * tp;
        acc[DOT_GM] += g * tm;
        acc[DOT_GG] += g * g;
        acc[DOT_GV] += g * w;
        acc[DOT_PV] += tp * w;
        acc[DOT_MV] += tm * w;
        acc[DOT_VV] += w * w;
    }
    block_sum<kNDots>(acc, red);
    if (threadIdx.x == 0) {
        double *out = part + ((size_t)p * kNaBlocks + blockIdx.x) * kNDots;
#pragma unroll
        for (int q = 0; q < kNDots; ++q) out[q] = acc[q];
    }
}

// Stage 2: one warp per image.  Lane l adds partials l and l + 32, then a shuffle tree; endpoint rows are zero.
__global__ void __launch_bounds__(32) na_finish_kernel(const double *__restrict__ part, int P, double *__restrict__ dots) {
    const int p = blockIdx.x, lane = threadIdx.x;
    double a[kNDots];
#pragma unroll
    for (int q = 0; q < kNDots; ++q) a[q] = 0.0;
    if (p > 0 && p < P - 1) {
        const double *pd = part + (size_t)p * kNaBlocks * kNDots;
        for (int b = lane; b < kNaBlocks; b += 32)
#pragma unroll
            for (int q = 0; q < kNDots; ++q) a[q] += pd[(size_t)b * kNDots + q];
    }
#pragma unroll
    for (int q = 0; q < kNDots; ++q)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) a[q] += __shfl_down_sync(0xffffffffu, a[q], o);
    if (lane == 0)
        for (int q = 0; q < kNDots; ++q) dots[(size_t)p * kNDots + q] = a[q];
}

}  // namespace cfn

using namespace cfn;

static thread_local char g_na_err[512] = "";

static int na_fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_na_err, sizeof g_na_err, fmt, ap);
    va_end(ap);
    return code;
}

// Device address of the scratch on the CURRENT device, looked up once per device and remembered.
static std::mutex g_na_mu;
static double *g_na_ptr[kNaMaxDevices] = {};

static int na_scratch(int dev, double **out) {
    std::lock_guard<std::mutex> lock(g_na_mu);
    if (!g_na_ptr[dev]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_na_partials);
        if (e != cudaSuccess || !p)
            return na_fail(CFNEB_ECUDA, "cudaGetSymbolAddress(scratch) on device %d: %s", dev, cudaGetErrorString(e));
        g_na_ptr[dev] = static_cast<double *>(p);
    }
    *out = g_na_ptr[dev];
    return CFNEB_OK;
}

// A caller's pointer must be device (or managed) memory of the current device.
static int na_check_ptr(const void *p, const char *name, int dev) {
    if (!p) return na_fail(CFNEB_EINVAL, "%s is NULL", name);
    cudaPointerAttributes at;
    const cudaError_t e = cudaPointerGetAttributes(&at, p);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return na_fail(CFNEB_ECUDA, "cudaPointerGetAttributes(%s): %s", name, cudaGetErrorString(e));
    }
    if (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)
        return na_fail(CFNEB_EINVAL, "%s is not a device pointer", name);
    if (at.type == cudaMemoryTypeDevice && at.device != dev)
        return na_fail(CFNEB_EINVAL, "%s lives on device %d but device %d is current", name, at.device, dev);
    return CFNEB_OK;
}

extern "C" {

int cfneb_band_dots_noalloc(const double *X, const double *G, const double *v, int32_t n_images, int64_t n_dof,
                            double *dots, void *cuda_stream) {
    g_na_err[0] = 0;
    if (n_images < 3) return na_fail(CFNEB_EINVAL, "n_images = %d: a band has at least 3 images", (int)n_images);
    if (n_images > kNaMaxImages)
        return na_fail(CFNEB_ERANGE, "n_images = %d exceeds CFNEB_NOALLOC_MAX_IMAGES = %d: the fixed scratch of this entry "
                       "point holds no more; use a cfneb_create handle with a workspace for longer bands", (int)n_images, kNaMaxImages);
    if (n_dof < 1) return na_fail(CFNEB_EINVAL, "n_dof = %lld", (long long)n_dof);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(CFNEB_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kNaMaxDevices) return na_fail(CFNEB_ERANGE, "device ordinal %d: at most %d devices", dev, kNaMaxDevices);
    int rc;
    if ((rc = na_check_ptr(X, "X", dev)) || (rc = na_check_ptr(G, "G", dev)) || (rc = na_check_ptr(v, "v", dev)) ||
        (rc = na_check_ptr(dots, "dots", dev)))
        return rc;
    double *part = nullptr;
    if ((rc = na_scratch(dev, &part))) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    na_partial_kernel<<<dim3(kNaBlocks, n_images - 2), kNaThreads, 0, st>>>(X, G, v, (long long)n_dof, part);
    na_finish_kernel<<<n_images, 32, 0, st>>>(part, n_images, dots);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(CFNEB_ECUDA, "kernel launch: %s", cudaGetErrorString(e));
    return CFNEB_OK;
}

const char *cfneb_band_dots_noalloc_error(void) { return g_na_err; }

}  // extern "C"
