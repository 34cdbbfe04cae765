// cbct_tv_value_noalloc (include/cbct.h): the TV term of the energy (O3) for callers that must not allocate.
//
// The energy monitor's tv_value_kernel (tv.cu) leaves one fp64 partial sum per block in a scratch array that the handle
// allocates with cudaMalloc on first use.  Some users of this library cannot make that call:
//   - a reconstruction service that hands ALL device memory to its own pool at start-up (PyTorch's caching allocator with a
//     fixed budget, a scanner console with a per-scan memory contract): a raw cudaMalloc from inside a library bypasses the
//     pool's accounting and can fail although the pool still has room;
//   - a monitoring thread that watches the TV term while a c5-sized reconstruction (512^3 volume, 363 views) has filled the
//     card on purpose: there may be nothing left to allocate from;
//   - a latency-bound loop: cudaMalloc / cudaFree serialise against the whole device, so one call from a side thread stalls
//     the kernels of every other stream.
// For them the partial sums live in the file-scope device array below instead.  It exists from the moment the library is
// loaded on a GPU until the process exits, on every GPU that loads the library, whether or not this entry point is ever
// called: kNoAllocMaxBlocks doubles = 128 KiB per GPU.  That size fixes the largest volume the entry point accepts.
#include <mutex>

#include "cbct_internal.h"

namespace {
constexpr int kNoAllocThreads = 256;
constexpr int kNoAllocPerThread = 32;
constexpr unsigned long long kNoAllocVoxPerBlock = (unsigned long long)kNoAllocThreads * kNoAllocPerThread;   // 8192
constexpr int kNoAllocMaxBlocks = 16384;                                                                       // 128 KiB of doubles
constexpr unsigned long long kNoAllocMaxVox = kNoAllocVoxPerBlock * kNoAllocMaxBlocks;                        // 2^27 = 512^3

// The scratch itself.  In HOST code this name is only a stand-in for the symbol: it is not a device address, and a kernel
// handed `s_tv_partial` by the host would read and write somewhere else entirely.  Host code below therefore asks the
// runtime for the real address (cudaGetSymbolAddress) once per device and passes that to the kernels.
static __device__ __align__(256) double s_tv_partial[kNoAllocMaxBlocks];

// Variant of tv_value_kernel (tv.cu): same per-voxel arithmetic (forward differences over the spacing, zero at the far
// faces, sqrtf of the fp32 sum of squares plus eps^2, accumulated in fp64), but a block owns a fixed run of 8192 voxels so
// that the number of partials, and with it the scratch a call needs, is known from the volume size alone.
__global__ void __launch_bounds__(kNoAllocThreads)
tv_value_noalloc_kernel(const float *__restrict__ f, int nx, int ny, int nz, float ihx, float ihy, float ihz, float eps2,
                        double *__restrict__ partial)
{
    const unsigned long long n = (unsigned long long)nx * ny * nz, sxy = (unsigned long long)nx * ny;
    const unsigned long long base = (unsigned long long)blockIdx.x * kNoAllocVoxPerBlock;
    double acc = 0.0;
#pragma unroll 4
    for (int m = 0; m < kNoAllocPerThread; ++m) {
        const unsigned long long o = base + (unsigned long long)m * kNoAllocThreads + threadIdx.x;
        if (o >= n) break;
        const int i = (int)(o % nx), j = (int)((o / nx) % ny), k = (int)(o / sxy);
        const float c = __ldg(f + o);
        const float dx = (i + 1 < nx) ? (__ldg(f + o + 1) - c) * ihx : 0.f;
        const float dy = (j + 1 < ny) ? (__ldg(f + o + nx) - c) * ihy : 0.f;
        const float dz = (k + 1 < nz) ? (__ldg(f + o + sxy) - c) * ihz : 0.f;
        acc += (double)sqrtf(fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2))));
    }
    __shared__ double sh[kNoAllocThreads];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = kNoAllocThreads / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];        // every block of the grid writes its slot: no slot needs clearing
}

// Second stage: one block adds the first n_blocks partials in a fixed order and writes the caller's output.
__global__ void __launch_bounds__(kNoAllocThreads)
tv_value_noalloc_final_kernel(const double *__restrict__ partial, int n_blocks, double *__restrict__ out)
{
    __shared__ double sh[kNoAllocThreads];
    double acc = 0.0;
    for (int q = threadIdx.x; q < n_blocks; q += kNoAllocThreads) acc += partial[q];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int s = kNoAllocThreads / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sh[0];
}

// Device address of s_tv_partial per CUDA device ordinal, looked up on the first call made with that device current.
constexpr int kMaxDevices = 64;
std::mutex s_setup_mutex;
double *s_partial_addr[kMaxDevices] = {};

cbct_status scratch_address(double **out)
{
    int dev = -1;
    CBCT_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) {
        cbct_set_error("cbct_tv_value_noalloc: device ordinal %d outside 0..%d", dev, kMaxDevices - 1);
        return CBCT_ERR_CUDA;
    }
    std::lock_guard<std::mutex> lock(s_setup_mutex);
    if (!s_partial_addr[dev]) {
        double *p = nullptr;
        CBCT_CUDA(cudaGetSymbolAddress((void **)&p, s_tv_partial));     // the copy of the array on the CURRENT device
        if (!p) {
            cbct_set_error("cbct_tv_value_noalloc: cudaGetSymbolAddress returned a null address on device %d", dev);
            return CBCT_ERR_CUDA;
        }
        s_partial_addr[dev] = p;
    }
    *out = s_partial_addr[dev];
    return CBCT_OK;
}
}  // namespace

extern "C" cbct_status cbct_tv_value_noalloc(const float *d_f, int nx, int ny, int nz, double hx_mm, double hy_mm,
                                             double hz_mm, float eps, double *d_out, void *stream)
{
    if (!d_f || !d_out) {
        cbct_set_error("cbct_tv_value_noalloc: NULL argument");
        return CBCT_ERR_INVALID_ARG;
    }
    if (nx <= 0 || ny <= 0 || nz <= 0 || !(hx_mm > 0.0) || !(hy_mm > 0.0) || !(hz_mm > 0.0) || !(eps >= 0.f)) {
        cbct_set_error("cbct_tv_value_noalloc: non-positive dimension or spacing, or eps < 0");
        return CBCT_ERR_INVALID_ARG;
    }
    const unsigned long long n = (unsigned long long)nx * (unsigned long long)ny * (unsigned long long)nz;
    if (nx > 16384 || ny > 16384 || nz > 16384 || n > kNoAllocMaxVox) {
        cbct_set_error("cbct_tv_value_noalloc: volume %d x %d x %d has %llu voxels, more than the %llu (= 512^3) the fixed "
                       "128 KiB scratch array covers; use cbct_energy on a handle for larger volumes",
                       nx, ny, nz, n, kNoAllocMaxVox);
        return CBCT_ERR_SHAPE;
    }
    double *partial = nullptr;
    CBCT_TRY(scratch_address(&partial));
    cudaStream_t st = (cudaStream_t)stream;
    const int n_blocks = (int)((n + kNoAllocVoxPerBlock - 1) / kNoAllocVoxPerBlock);
    tv_value_noalloc_kernel<<<n_blocks, kNoAllocThreads, 0, st>>>(d_f, nx, ny, nz, (float)(1.0 / hx_mm), (float)(1.0 / hy_mm),
                                                                  (float)(1.0 / hz_mm), eps * eps, partial);
    CBCT_LAUNCH_CHECK();
    tv_value_noalloc_final_kernel<<<1, kNoAllocThreads, 0, st>>>(partial, n_blocks, d_out);
    CBCT_LAUNCH_CHECK();
    return CBCT_OK;
}
